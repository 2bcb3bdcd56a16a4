// lsa_attn_tc.cu - host side of the tcgen05 attention (tensor maps, launch) and the S8 combine kernel.
// Kernel: lsa_attn_tc_kernel.cuh.  Design notes: lsa_attn_tc_defs.cuh.
#include "lsa_attn_tc_kernel.cuh"

namespace lsa {

// ---- S8: merge the split partials of one sequence  ----------------------------------------------
//   m* = max m_i ; l* = sum l_i 2^(m_i-m*) ; out = sum o_i 2^(m_i-m*) / l* ; lse = ln2 (m* + log2 l*)
// grid (2*H, B), 256 threads: block = one head, one half of D; thread = one output element.
__global__ void __launch_bounds__(256)
combine_tc_kernel(TcParams p, int n_cta, __nv_bfloat16* __restrict__ out, float* __restrict__ lse) {
  __shared__ float w_s[256];
  __shared__ int red_i[8][3];
  __shared__ float red_f[8];
  __shared__ int s_lo, s_hi;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int h = blockIdx.x >> 1, d = (blockIdx.x & 1) * 256 + tid, b = blockIdx.y;
  // group counts: before b, of b, total
  int pre = 0, mine = 0, tot = 0;
  for (int i = tid; i < p.B; i += 256) {
    const int g = seq_groups(p.seqs[i]);
    tot += g;
    if (i < b) pre += g;
    if (i == b) mine = g;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    pre += __shfl_xor_sync(0xffffffffu, pre, o);
    mine += __shfl_xor_sync(0xffffffffu, mine, o);
    tot += __shfl_xor_sync(0xffffffffu, tot, o);
  }
  if (lane == 0) { red_i[warp][0] = pre; red_i[warp][1] = mine; red_i[warp][2] = tot; }
  __syncthreads();
  pre = mine = tot = 0;
  for (int w = 0; w < 8; ++w) { pre += red_i[w][0]; mine += red_i[w][1]; tot += red_i[w][2]; }
  // which CTAs hold a piece of sequence b (same partition arithmetic as PieceCursor)
  bool active = false;
  if (tid < n_cta && mine > 0) {
    const int f0 = (int)((long long)tid * tot / n_cta), f1 = (int)((long long)(tid + 1) * tot / n_cta);
    active = f0 < f1 && f0 < pre + mine && f1 > pre;
  }
  const size_t slot = (size_t)tid + b;
  const float mi = active ? p.part_m[slot * kTcH + h] : -INFINITY;
  float mmax = mi;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mmax = fmaxf(mmax, __shfl_xor_sync(0xffffffffu, mmax, o));
  if (tid == 0) { s_lo = 1 << 30; s_hi = -1; }
  __syncthreads();
  if (lane == 0) red_f[warp] = mmax;
  if (active) { atomicMin(&s_lo, tid); atomicMax(&s_hi, tid); }
  __syncthreads();
  float m_star = red_f[0];
  for (int w = 1; w < 8; ++w) m_star = fmaxf(m_star, red_f[w]);
  const float wi = (active && mi != -INFINITY) ? exp2f(mi - m_star) : 0.f;
  w_s[tid] = wi;
  float lsum = active ? wi * p.part_l[slot * kTcH + h] : 0.f;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) lsum += __shfl_xor_sync(0xffffffffu, lsum, o);
  __syncthreads();
  if (lane == 0) red_f[warp] = lsum;
  __syncthreads();
  float l_star = 0.f;
  for (int w = 0; w < 8; ++w) l_star += red_f[w];
  const bool empty = !(l_star > 0.f);
  float acc = 0.f;
  const int lo = s_lo, hi = s_hi;
  const float* po = p.part_o + ((size_t)b * kTcH + h) * kTcD + d;     // slot i+b -> + i * H * D
#pragma unroll 4
  for (int i = lo; i <= hi; ++i) {
    const float w = w_s[i];                       // 0 for CTAs without a piece: their slot is never read
    if (w != 0.f) acc = fmaf(w, po[(size_t)i * (kTcH * kTcD)], acc);
  }
  out[((size_t)b * kTcH + h) * kTcD + d] = __float2bfloat16_rn(empty ? 0.f : acc / l_star);
  if (lse && (blockIdx.x & 1) == 0 && tid == 0)
    lse[(size_t)b * kTcH + h] = empty ? -INFINITY : (m_star + log2f(l_star)) * 0.6931471805599453f;
}

// ---- host ------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct TcPlan {
  TcInit init{};
  EncodeTiledFn encode = nullptr;
  CUtensorMap map_pool{}, map_q{};
  const void* q_cached = nullptr;
  CUtensorMap* d_maps = nullptr;
  TcParams params{};
  int grid = 0;
  size_t smem = 0;
};

bool tc_supported(int dtype, int H, int D, int C) { return dtype == 1 && H == kTcH && D == kTcD && C == kTcC; }

static bool encode_rows(EncodeTiledFn enc, CUtensorMap* m, const void* ptr, uint64_t rows, uint32_t box_rows, std::string* msg) {
  cuuint64_t dims[2] = {(cuuint64_t)kTcD, rows};
  cuuint64_t strides[1] = {(cuuint64_t)kTcD * 2};
  cuuint32_t box[2] = {64, box_rows};
  cuuint32_t es[2] = {1, 1};
  CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(ptr), dims, strides, box, es,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    *msg = "cuTensorMapEncodeTiled failed with CUresult " + std::to_string((int)r);
    return false;
  }
  return true;
}

#define TC_CUDA(expr)                                                               \
  do {                                                                              \
    cudaError_t _e = (expr);                                                        \
    if (_e != cudaSuccess) {                                                        \
      *msg = std::string(#expr) + ": " + cudaGetErrorString(_e);                    \
      return -2;                                                                    \
    }                                                                               \
  } while (0)

int tc_create(const TcInit& init, TcPlan** out, std::string* msg) {
  if (init.B > kTcMaxB) { *msg = "tcgen05 attention supports at most 256 sequences per context"; return -6; }
  TcPlan* pl = new TcPlan();
  pl->init = init;
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
  if (e != cudaSuccess || !fn) { *msg = "cuTensorMapEncodeTiled entry point not found"; delete pl; return -2; }
  pl->encode = (EncodeTiledFn)fn;
  pl->grid = init.max_ctas > 0 ? std::min(init.max_ctas, init.n_sms) : init.n_sms;
  if (pl->grid > 256) pl->grid = 256;
  if (!encode_rows(pl->encode, &pl->map_pool, init.hot_pool, (uint64_t)init.P * 2 * kTcC, 32, msg)) { delete pl; return -2; }
  std::vector<CUtensorMap> maps((size_t)init.B * 4);
  for (int b = 0; b < init.B; ++b) {
    const SeqDev& s = init.seq_host[b];
    const void* ptrs[4] = {s.hca_k, s.hca_v, s.win_k, s.win_v};
    const uint64_t rows[4] = {(uint64_t)s.n_hca, (uint64_t)s.n_hca, (uint64_t)init.W, (uint64_t)init.W};
    for (int j = 0; j < 4; ++j) {
      const bool none = rows[j] == 0 || ptrs[j] == nullptr;     // never referenced: point at the pool
      if (!encode_rows(pl->encode, &maps[(size_t)b * 4 + j], none ? init.hot_pool : ptrs[j], none ? 32 : rows[j], 32, msg)) {
        delete pl;
        return -2;
      }
    }
    // rows of the window ring that are not attended yet must hold finite values (they are multiplied by P = 0)
    if (init.W > s.w_len && s.win_k && s.win_v) {
      const size_t off = (size_t)s.w_len * kTcD * 2, n = (size_t)(init.W - s.w_len) * kTcD * 2;
      TC_CUDA(cudaMemset((char*)s.win_k + off, 0, n));
      TC_CUDA(cudaMemset((char*)s.win_v + off, 0, n));
    }
  }
  TC_CUDA(cudaMalloc(&pl->d_maps, maps.size() * sizeof(CUtensorMap)));
  TC_CUDA(cudaMemcpy(pl->d_maps, maps.data(), maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice));
  const size_t slots = (size_t)pl->grid + init.B;
  TcParams& p = pl->params;
  p.seqs = init.d_seqs; p.tbl_chunk = init.pool.tbl_chunk; p.tbl_page = init.pool.tbl_page; p.seq_maps = pl->d_maps;
  p.B = init.B; p.k = init.k; p.pool_rows = init.P * 2 * kTcC;
  p.scale_log2 = init.sm_scale * 1.4426950408889634f;
  TC_CUDA(cudaMalloc(&p.part_o, slots * kTcH * kTcD * sizeof(float)));
  TC_CUDA(cudaMalloc(&p.part_m, slots * kTcH * sizeof(float)));
  TC_CUDA(cudaMalloc(&p.part_l, slots * kTcH * sizeof(float)));
  pl->smem = sizeof(TcSmem) + 1024;
  TC_CUDA(cudaFuncSetAttribute(attn_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl->smem));
  *out = pl;
  return 0;
}

int tc_attention(TcPlan* pl, const void* q, void* out, float* lse, cudaStream_t st, int* launches, int* ctas,
                 std::string* msg) {
  if (q != pl->q_cached) {
    if (!encode_rows(pl->encode, &pl->map_q, q, (uint64_t)pl->init.B * kTcH, 64, msg)) return -2;
    pl->q_cached = q;
  }
  attn_tc_kernel<<<pl->grid, kTcThreads, pl->smem, st>>>(pl->map_pool, pl->map_q, pl->params);
  TC_CUDA(cudaGetLastError());
  combine_tc_kernel<<<dim3(kTcH * 2, pl->init.B), 256, 0, st>>>(pl->params, pl->grid, (__nv_bfloat16*)out, lse);
  TC_CUDA(cudaGetLastError());
  *launches = 2;
  *ctas = pl->grid;
  return 0;
}

void tc_destroy(TcPlan* pl) {
  if (!pl) return;
  cudaFree(pl->d_maps);
  cudaFree(pl->params.part_o);
  cudaFree(pl->params.part_m);
  cudaFree(pl->params.part_l);
  delete pl;
}

}  // namespace lsa
