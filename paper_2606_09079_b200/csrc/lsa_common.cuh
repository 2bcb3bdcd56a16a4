// lsa_common.cuh - device-side state and small helpers shared by the LSA kernels (sm_100a).
// Nothing here is shared with oracle/ (the CPU oracle is independent numpy code).
#pragma once

#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace lsa {

constexpr int kMaxK = 1024;            // top-k bound (lsa_config.k)
constexpr int kSortCap = 4096;         // u64 keys sorted in shared memory by one block
constexpr int kPageBits = 20;          // LRU key = last_used << 20 | page  -> hot_pages <= 2^20
constexpr int kFireMax = 64;           // sequences per trigger launch

// Per-sequence device record.  Fields below `-- mutable --` are written by kernels only
// (prestep / residency), in stream order; the host keeps deterministic mirrors.
struct SeqDev {
  const void* cold;        // device-mapped address of the pinned-host cold pool [n_chunks][2][C][D]
  const void* emb;         // [n_chunks][E]
  const void* hca_k;       // [n_hca][D]
  const void* hca_v;
  void* win_k;             // ring [W][D]
  void* win_v;
  long long n_csa;
  int n_chunks;
  int n_hca;
  int k_eff;               // min(k, n_chunks)
  int page_of_off;         // offset of this sequence in page_of[]
  // -- mutable --
  int w_len;
  int w_head;
  int cur_buf;             // which of the two table buffers is attended
  int pending;             // a staged table sits in buffer 1-cur_buf
  int n_tbl[2];            // entries per table buffer
  // -- growth (lsa_append_compressed, DESIGN R29-R33); static contexts: cap_hca = n_hca, tier_page0 = -1 --
  int cap_hca;             // rows hca_k / hca_v can hold (tensor maps are made over this many)
  int tier_page0;          // first of this sequence's two reserved hot-pool pages, or -1
  const float* cold_scale; // FP8 cold pool: [n_chunks][2] (K scale, V scale), else null
  unsigned int grow_epoch; // lsa_append_compressed calls applied to this sequence so far (released after the rows are written)
  unsigned int app_epoch;  // ring rows appended so far; bumped with release semantics AFTER the row is written, so a
                           // launch that does not wait for its predecessor (lsa_attn_tc_small.cuh) can order its reads
};

struct PoolDev {
  int* page_of;                 // [sum n_chunks]  chunk -> page or -1
  int* owner_seq;               // [P] -1 = never used
  int* owner_chunk;             // [P]
  unsigned long long* last_used;// [P] 0 = never used
  unsigned int* pin_mark;       // [P] == epoch -> pinned during this residency pass
  int* tbl_chunk;               // [B][2][k]
  int* tbl_page;                // [B][2][k]
  // fetch list of the current trigger launch
  const void** fetch_src;       // [B*k]
  int* fetch_page;              // [B*k]
  const float** fetch_scale;    // [B*k] FP8 cold pool: the page's two block scales
  // scalars
  unsigned long long* counters; // [8]: tick, triggers, hits, misses, evictions, bytes, fetch_count, error
  unsigned int* epoch;
};

enum Counter { C_TICK = 0, C_TRIGGERS, C_HITS, C_MISSES, C_EVICTIONS, C_BYTES, C_FETCH_COUNT, C_ERROR };

struct FireList {
  int n;
  int ids[kFireMax];
};

// ---- element load helpers -------------------------------------------------------------
template <typename T> struct Elem;
template <> struct Elem<float> {
  static constexpr int kVec = 4;  // elements per 16 bytes
  static __device__ __forceinline__ void load16(const float* p, float* out) {
    float4 v = *reinterpret_cast<const float4*>(p);
    out[0] = v.x; out[1] = v.y; out[2] = v.z; out[3] = v.w;
  }
  static __device__ __forceinline__ void unpack16(const uint4& v, float* out) {
    out[0] = __uint_as_float(v.x); out[1] = __uint_as_float(v.y); out[2] = __uint_as_float(v.z); out[3] = __uint_as_float(v.w);
  }
  static __device__ __forceinline__ float to_f(float x) { return x; }
  static __device__ __forceinline__ float from_f(float x) { return x; }
};
template <> struct Elem<__nv_bfloat16> {
  static constexpr int kVec = 8;
  static __device__ __forceinline__ void load16(const __nv_bfloat16* p, float* out) {
    uint4 v = *reinterpret_cast<const uint4*>(p);
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      out[2 * i] = __uint_as_float(w[i] << 16);
      out[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
    }
  }
  static __device__ __forceinline__ void unpack16(const uint4& v, float* out) {
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      out[2 * i] = __uint_as_float(w[i] << 16);
      out[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
    }
  }
  static __device__ __forceinline__ float to_f(__nv_bfloat16 x) { return __bfloat162float(x); }
  static __device__ __forceinline__ __nv_bfloat16 from_f(float x) { return __float2bfloat16_rn(x); }
};

// ---- programmatic dependent launch: the kernels of the trigger side band are chained so that the launch and
// prologue of each overlap the tail of its predecessor.  pdl_wait(): everything written by earlier kernels of
// the stream is visible after it (no-op without the launch attribute).
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

#ifdef __CUDACC__
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t lc{};
  lc.gridDim = grid; lc.blockDim = block; lc.dynamicSmemBytes = smem; lc.stream = st;
  lc.attrs = attr; lc.numAttrs = 1;
  return cudaLaunchKernelEx(&lc, kernel, static_cast<KArgs>(args)...);
}
#endif

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// Monotone map float -> uint32 (larger float -> larger uint); -0 is canonicalised to +0, NaN -> -inf.
__device__ __forceinline__ uint32_t float_to_ordered(float f) {
  if (f != f) f = -INFINITY;
  if (f == 0.f) f = 0.f;
  uint32_t b = __float_as_uint(f);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float ordered_to_float(uint32_t u) {
  uint32_t b = (u & 0x80000000u) ? (u & 0x7fffffffu) : ~u;
  return __uint_as_float(b);
}

}  // namespace lsa
