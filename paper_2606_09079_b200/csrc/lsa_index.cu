// lsa_index.cu - S1 query tower, S2 chunk scoring, S3 per-sequence top-k  (sm_100a)
//
//   S1  z = W_q h ; q_hat = z / max(||z||, 1e-12)     PAPER.md l.61-65 Eq.(1)-(2) collapsed to one
//       linear map + L2 norm (l.124 "standard dual-encoder"; BASELINE.json north_star; DESIGN R1)
//   S2  score_c = q_hat . Emb[c]                       PAPER.md l.71-75 Eq.(4) in cosine form (R1,R3)
//   S3  first min(k, n_chunks) by (score desc, idx asc) PAPER.md l.77-79 Eq.(5) with top-k (R2,R14)
//
// All three are HBM/latency bound (W_q 4 MiB + Emb <= 2 MiB per trigger): 16-byte loads, one warp per
// output row, fp32 accumulation in a fixed order so bit-identical embedding rows give bit-identical
// scores wherever they sit in the table (exact planted ties stay exact).
#include <cstdio>

#include "lsa_kernels.h"
#include "lsa_select.cuh"

namespace lsa {

constexpr int kQtWarps = 4;   // rows of W_q per block
constexpr int kQtSeqs = 4;    // sequences per pass (W_q row is read once for all of them)

template <typename T>
__global__ void __launch_bounds__(kQtWarps * 32)
qtower_kernel(const T* __restrict__ W, const T* __restrict__ h, FireList rows, float* __restrict__ z, int E, int Dh) {
  constexpr int V = Elem<T>::kVec;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  pdl_wait();
  pdl_launch_dependents();
  const int e = blockIdx.x * kQtWarps + warp;
  const int i0 = blockIdx.y * kQtSeqs;
  const int n = rows.n;
  if (e >= E) return;
  float acc[kQtSeqs];
#pragma unroll
  for (int s = 0; s < kQtSeqs; ++s) acc[s] = 0.f;
  const T* wrow = W + (size_t)e * Dh;
  // 16 independent 16-byte loads of the weight row are issued before any of them is used (the row is read once
  // from HBM; h comes from L1/L2), so a 4096-wide bf16 row is one memory round trip, not sixteen
  constexpr int kU = 16;
  for (int d0 = lane * V; d0 < Dh; d0 += 32 * V * kU) {
    uint4 wraw[kU];
#pragma unroll
    for (int u = 0; u < kU; ++u) {
      const int d = d0 + u * 32 * V;
      wraw[u] = d < Dh ? *reinterpret_cast<const uint4*>(wrow + d) : make_uint4(0u, 0u, 0u, 0u);
    }
    // the hidden state of the first sequence of the pass (the only one when a single sequence fires) travels the same
    // way: 16 more independent loads in flight instead of one dependent L2 round trip per 16 bytes inside the loop below
    uint4 hraw[kU];
    const T* h0 = h + (size_t)rows.ids[i0] * Dh;
#pragma unroll
    for (int u = 0; u < kU; ++u) {
      const int d = d0 + u * 32 * V;
      hraw[u] = d < Dh ? *reinterpret_cast<const uint4*>(h0 + d) : make_uint4(0u, 0u, 0u, 0u);
    }
#pragma unroll
    for (int u = 0; u < kU; ++u) {
      const int d = d0 + u * 32 * V;
      if (d < Dh) {
        float wf[V];
        Elem<T>::unpack16(wraw[u], wf);
#pragma unroll
        for (int s = 0; s < kQtSeqs; ++s) {
          if (i0 + s < n) {
            float hf[V];
            if (s == 0) Elem<T>::unpack16(hraw[u], hf);
            else Elem<T>::load16(h + (size_t)rows.ids[i0 + s] * Dh + d, hf);
#pragma unroll
            for (int j = 0; j < V; ++j) acc[s] = fmaf(wf[j], hf[j], acc[s]);
          }
        }
      }
    }
  }
#pragma unroll
  for (int s = 0; s < kQtSeqs; ++s) {
    float v = warp_sum(acc[s]);
    if (lane == 0 && i0 + s < n) z[(size_t)(i0 + s) * E + e] = v;
  }
}

constexpr int kScWarps = 8;

template <typename T>
__global__ void __launch_bounds__(kScWarps * 32)
score_kernel(const SeqDev* __restrict__ seqs, FireList fire, const float* __restrict__ z,
             float* __restrict__ scores, int E, int n_chunks_max, int n_part) {
  extern __shared__ float zs[];           // [E]
  __shared__ float red[kScWarps];
  __shared__ float inv_norm_s;
  constexpr int V = Elem<T>::kVec;
  const int i = blockIdx.y;
  pdl_wait();
  pdl_launch_dependents();
  const SeqDev& sq = seqs[fire.ids[i]];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int c0 = blockIdx.x * kScWarps;
  if (c0 >= sq.n_chunks) return;
  float ss = 0.f;
  for (int e = threadIdx.x; e < E; e += blockDim.x) {
    // z arrives as n_part partial sums over slices of Dh (the batched tensor-core tower, lsa_index_tc.cu), added here in
    // a fixed order; n_part = 1: the GEMV's complete sums
    float v = z[(size_t)i * E + e];
    for (int pz = 1; pz < n_part; ++pz) v += z[((size_t)pz * fire.n + i) * E + e];
    zs[e] = v;
    ss = fmaf(v, v, ss);
  }
  ss = warp_sum(ss);
  if (lane == 0) red[warp] = ss;
  __syncthreads();
  if (threadIdx.x == 0) {
    float t = 0.f;
    for (int w = 0; w < kScWarps; ++w) t += red[w];
    inv_norm_s = 1.0f / fmaxf(sqrtf(t), 1e-12f);
  }
  __syncthreads();
  const int c = c0 + warp;
  if (c >= sq.n_chunks) return;
  const T* row = reinterpret_cast<const T*>(sq.emb) + (size_t)c * E;
  float acc = 0.f;
  for (int e0 = lane * V; e0 < E; e0 += 32 * V) {
    float ef[V];
    Elem<T>::load16(row + e0, ef);
#pragma unroll
    for (int j = 0; j < V; ++j) acc = fmaf(ef[j], zs[e0 + j], acc);
  }
  acc = warp_sum(acc);
  if (lane == 0) scores[(size_t)i * n_chunks_max + c] = acc * inv_norm_s;
}

__global__ void __launch_bounds__(1024)
topk_kernel(const SeqDev* __restrict__ seqs, FireList fire, const float* __restrict__ scores,
            int n_chunks_max, int k, int32_t* __restrict__ sel_idx, float* __restrict__ sel_score) {
  __shared__ SelectSmem sm;
  const int i = blockIdx.x;
  pdl_wait();
  pdl_launch_dependents();
  const SeqDev& sq = seqs[fire.ids[i]];
  const float* sc = scores + (size_t)i * n_chunks_max;
  auto keyf = [sc](int c) -> unsigned long long {
    return ((unsigned long long)(~float_to_ordered(sc[c])) << 32) | (unsigned)c;
  };
  // n <= 4096: histogram select + sort of the k winners; larger tables: radix select over the keys in global memory
  // k_eff = min(recalled chunks per table, n_chunks): k for a static context, k - 2 for a growing one (DESIGN R33)
  const int kk = min(k, sq.k_eff);
  const int m = sq.n_chunks <= 4096 ? block_topk_select(sc, sq.n_chunks, kk, sm)
                                    : block_select_smallest(keyf, sq.n_chunks, kk, sm);
  for (int j = threadIdx.x; j < k; j += blockDim.x) {
    int idx = -1;
    float val = -INFINITY;
    if (j < m) {
      unsigned long long key = sm.keys[j];
      idx = (int)(key & 0xffffffffull);
      val = ordered_to_float(~(uint32_t)(key >> 32));
    }
    sel_idx[(size_t)i * k + j] = idx;
    if (sel_score) sel_score[(size_t)i * k + j] = val;
  }
}

cudaError_t launch_qtower(int dtype, const void* W, const void* h, const FireList& rows, float* z, int E, int Dh,
                          cudaStream_t st) {
  dim3 grid((E + kQtWarps - 1) / kQtWarps, (rows.n + kQtSeqs - 1) / kQtSeqs);
  if (dtype == 0)
    return launch_pdl(qtower_kernel<float>, grid, dim3(kQtWarps * 32), 0, st, (const float*)W, (const float*)h, rows, z, E, Dh);
  return launch_pdl(qtower_kernel<__nv_bfloat16>, grid, dim3(kQtWarps * 32), 0, st, (const __nv_bfloat16*)W, (const __nv_bfloat16*)h, rows, z, E, Dh);
}

cudaError_t launch_scores(int dtype, const SeqDev* seqs, const FireList& fire, const float* z, float* scores,
                          int E, int n_chunks_max, cudaStream_t st, int n_part) {
  dim3 grid((n_chunks_max + kScWarps - 1) / kScWarps, fire.n);
  size_t smem = (size_t)E * sizeof(float);
  if (dtype == 0)
    return launch_pdl(score_kernel<float>, grid, dim3(kScWarps * 32), smem, st, seqs, fire, z, scores, E, n_chunks_max, n_part);
  return launch_pdl(score_kernel<__nv_bfloat16>, grid, dim3(kScWarps * 32), smem, st, seqs, fire, z, scores, E, n_chunks_max, n_part);
}

cudaError_t launch_topk(const SeqDev* seqs, const FireList& fire, const float* scores, int n_chunks_max, int k,
                        int32_t* sel_idx, float* sel_score, cudaStream_t st) {
  return launch_pdl(topk_kernel, dim3(fire.n), dim3(1024), 0, st, seqs, fire, scores, n_chunks_max, k, sel_idx, sel_score);
}

}  // namespace lsa

// ---- lsa_index_select_static: S1-S3 for callers that may not allocate -------------------------------------------
// The indexer needs scratch between its three kernels (z = W_q h, the scores, the per-sequence records the scoring and
// top-k kernels read).  Here that scratch is a file-scope device array of fixed size instead of cudaMalloc'ed memory:
// nothing is allocated by the call, so it can be used under CUDA graph capture, in a serving loop, or by a harness that
// forbids allocation.  Every GPU that loads the library holds the array (sizeof(IndexStaticScratch), ~641 KiB) until exit.
// Every call on a device shares it and it keeps the last call's contents: nothing in it has to start at zero (the records,
// z[i][0..E) and scores[i][0..n_chunks_i) are fully rewritten before they are read), but two calls that overlap on the GPU
// (different streams, no ordering between them) race on it.
namespace lsa {

struct IndexStaticScratch {
  SeqDev seqs[kStaticSeqs];
  float z[kStaticSeqs * kStaticE];
  float scores[kStaticSeqs * kStaticChunks];
};
static __device__ __align__(256) IndexStaticScratch g_index_scratch;

struct StaticSeqArgs {
  const void* emb[kStaticSeqs];
  int n_chunks[kStaticSeqs];
  int n, k;
};
// Device code names the array directly; only host code needs its address.
__global__ void static_seq_setup_kernel(StaticSeqArgs a) {
  const int i = threadIdx.x;
  if (i >= a.n) return;
  SeqDev s{};
  s.emb = a.emb[i];
  s.n_chunks = a.n_chunks[i];
  s.n_csa = 0;
  s.k_eff = min(a.k, a.n_chunks[i]);
  s.tier_page0 = -1;
  g_index_scratch.seqs[i] = s;
}

int index_select_static(int dtype, const void* W_q, const void* h, const void* const* chunk_emb, const int* n_chunks, int n, int E,
                        int Dh, int k, int32_t* sel_idx, float* sel_score, cudaStream_t st, char* msg, size_t msg_len) {
  auto fail = [&](int code, const char* fmt, long long a = 0, long long b = 0) {
    snprintf(msg, msg_len, fmt, a, b);
    return code;
  };
  if (dtype != 0 && dtype != 1) return fail(-1, "bad dtype %lld", dtype);
  if (!W_q || !h || !chunk_emb || !n_chunks || !sel_idx) return fail(-1, "null argument");
  if (n < 1 || n > kStaticSeqs) return fail(-1, "n = %lld sequences: the static scratch holds at most %lld", n, kStaticSeqs);
  if (E < 8 || E > kStaticE || E % 8) return fail(-1, "E = %lld: must be a multiple of 8 and at most %lld (static scratch)", E, kStaticE);
  if (Dh < 8 || Dh % 8) return fail(-1, "Dh = %lld must be a positive multiple of 8", Dh);
  if (k < 1 || k > kMaxK) return fail(-1, "k = %lld must be in [1, %lld]", k, kMaxK);
  StaticSeqArgs a{};
  a.n = n; a.k = k;
  int n_max = 0;
  for (int i = 0; i < n; ++i) {
    if (!chunk_emb[i]) return fail(-1, "chunk_emb[%lld] is null", i);
    if (n_chunks[i] < 1 || n_chunks[i] > kStaticChunks)
      return fail(-1, "n_chunks = %lld: the static scratch holds at most %lld scores per sequence", n_chunks[i], kStaticChunks);
    a.emb[i] = chunk_emb[i];
    a.n_chunks[i] = n_chunks[i];
    n_max = n_chunks[i] > n_max ? n_chunks[i] : n_max;
  }
  // the array's address on the CURRENT device, looked up once per device (in host code the symbol's name is only a
  // stand-in: passing &g_index_scratch to a kernel would hand it a host address)
  static IndexStaticScratch* ptr_of[64] = {};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess || dev < 0 || dev >= 64) return fail(-2, "cudaGetDevice failed or device index %lld >= 64", dev);
  IndexStaticScratch* sp = __atomic_load_n(&ptr_of[dev], __ATOMIC_ACQUIRE);
  if (!sp) {
    e = cudaGetSymbolAddress(reinterpret_cast<void**>(&sp), g_index_scratch);
    if (e != cudaSuccess || !sp) {
      snprintf(msg, msg_len, "cudaGetSymbolAddress(g_index_scratch) failed: %s", cudaGetErrorString(e));
      return -2;
    }
    __atomic_store_n(&ptr_of[dev], sp, __ATOMIC_RELEASE);     // the same value whichever thread gets here first
  }
  static_seq_setup_kernel<<<1, kStaticSeqs, 0, st>>>(a);
  e = cudaGetLastError();
  FireList fire{};
  fire.n = n;
  for (int i = 0; i < n; ++i) fire.ids[i] = i;
  if (e == cudaSuccess) e = launch_qtower(dtype, W_q, h, fire, sp->z, E, Dh, st);
  // row stride of the scores = the longest table of this call (<= kStaticChunks, so n rows always fit)
  if (e == cudaSuccess) e = launch_scores(dtype, sp->seqs, fire, sp->z, sp->scores, E, n_max, st, 1);
  if (e == cudaSuccess) e = launch_topk(sp->seqs, fire, sp->scores, n_max, k, sel_idx, sel_score, st);
  if (e != cudaSuccess) {
    snprintf(msg, msg_len, "launch failed: %s", cudaGetErrorString(e));
    return -2;
  }
  return 0;
}

}  // namespace lsa
