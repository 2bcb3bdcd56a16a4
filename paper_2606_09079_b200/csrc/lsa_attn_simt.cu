// lsa_attn_simt.cu - S7 split-K decode attention (plain-FMA implementation) and S8 combine (sm_100a)
//
//   S7  per head h: s_j = sm_scale * q_h . K_j over HCA rows (+) valid rows of every page of the
//       current table (+) window rows; fp32 online softmax (running max m, sum l); o = sum p_j V_j;
//       each split emits (m, l, o).        PAPER.md l.85, l.185, l.197; BASELINE.json north_star
//   S8  m* = max m_i ; l* = sum l_i 2^{m_i-m*} ; out = sum o_i 2^{m_i-m*} / l*        (north_star)
//
// This is the shape-generic path: fp32 inputs (BASELINE.json cfg 1: "plain FMA") and any bf16 shape
// the tcgen05 kernel (lsa_attn_tc.cu) does not cover.  One CTA = 8 warps owns a contiguous range of
// the sequence's virtual key list; warp w owns heads [w*H/8, (w+1)*H/8): QK^T with lane <-> key,
// PV with lane <-> D/32 contiguous dims, so neither phase needs a cross-warp reduction.
// Logits are kept in the log2 domain: s2 = s * log2(e), p = 2^(s2 - m2).
#include "lsa_kernels.h"

namespace lsa {

constexpr int kSimtWarps = 8;
constexpr int kSimtThreads = kSimtWarps * 32;
constexpr int kSimtTile = 32;   // keys per tile (lane <-> key)

template <typename T, int N>
__device__ __forceinline__ void load_contig(const T* p, float* out) {
  constexpr int bytes = N * (int)sizeof(T);
  if constexpr (bytes % 16 == 0) {
#pragma unroll
    for (int i = 0; i < bytes / 16; ++i) Elem<T>::load16(p + i * Elem<T>::kVec, out + i * Elem<T>::kVec);
  } else {
#pragma unroll
    for (int i = 0; i < N; ++i) out[i] = Elem<T>::to_f(p[i]);
  }
}

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

template <typename T, int H, int D>
struct SimtLayout {
  static constexpr int V = Elem<T>::kVec;
  static constexpr int HPW = H / kSimtWarps;
  static constexpr int DPL = D / 32;
  static constexpr int KROW = D + V;                        // +16 B: conflict-free lane<->row reads
  static constexpr size_t q_bytes = (size_t)H * D * sizeof(T);
  static constexpr size_t k_bytes = (size_t)kSimtTile * KROW * sizeof(T);
  static constexpr size_t v_bytes = (size_t)kSimtTile * D * sizeof(T);
  static constexpr size_t p_bytes = (size_t)H * kSimtTile * sizeof(float);
  static size_t total(int k) { return q_bytes + k_bytes + v_bytes + p_bytes + (size_t)2 * k * sizeof(int); }
};

template <typename T, int H, int D>
__global__ void __launch_bounds__(kSimtThreads)
attn_simt_kernel(const SeqDev* __restrict__ seqs, PoolDev pool, const T* __restrict__ hot_pool,
                 const T* __restrict__ q, float scale_log2, int C, int k, int keys_per_cta, int s_max,
                 float* __restrict__ part_o, float* __restrict__ part_ml) {
  using L = SimtLayout<T, H, D>;
  constexpr int V = L::V, HPW = L::HPW, DPL = L::DPL, KROW = L::KROW, TK = kSimtTile;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* qs = reinterpret_cast<T*>(smem_raw);
  T* Ks = reinterpret_cast<T*>(smem_raw + L::q_bytes);
  T* Vs = reinterpret_cast<T*>(smem_raw + L::q_bytes + L::k_bytes);
  float* ps = reinterpret_cast<float*>(smem_raw + L::q_bytes + L::k_bytes + L::v_bytes);
  int* tblc = reinterpret_cast<int*>(smem_raw + L::q_bytes + L::k_bytes + L::v_bytes + L::p_bytes);
  int* tblp = tblc + k;

  const int b = blockIdx.y, s = blockIdx.x;
  const SeqDev& sq = seqs[b];
  const int n_hca = sq.n_hca, cur = sq.cur_buf, n_cur = sq.n_tbl[cur], w_len = sq.w_len;
  const int n_virtual = n_hca + n_cur * C + w_len;
  const int v_begin = s * keys_per_cta;
  if (v_begin >= n_virtual) return;
  const int v_end = min(n_virtual, v_begin + keys_per_cta);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

  for (int i = tid; i < n_cur; i += kSimtThreads) {
    tblc[i] = pool.tbl_chunk[((size_t)b * 2 + cur) * k + i];
    tblp[i] = pool.tbl_page[((size_t)b * 2 + cur) * k + i];
  }
  {
    const T* qg = q + (size_t)b * H * D;
    for (int i = tid * V; i < H * D; i += kSimtThreads * V)
      *reinterpret_cast<uint4*>(qs + i) = *reinterpret_cast<const uint4*>(qg + i);
  }
  __syncthreads();

  const T* hca_k = reinterpret_cast<const T*>(sq.hca_k);
  const T* hca_v = reinterpret_cast<const T*>(sq.hca_v);
  const T* win_k = reinterpret_cast<const T*>(sq.win_k);
  const T* win_v = reinterpret_cast<const T*>(sq.win_v);
  const long long n_csa = sq.n_csa;

  float o[HPW][DPL];
  float m_run[HPW], l_run[HPW];
#pragma unroll
  for (int hh = 0; hh < HPW; ++hh) {
    m_run[hh] = -INFINITY;
    l_run[hh] = 0.f;
#pragma unroll
    for (int dd = 0; dd < DPL; ++dd) o[hh][dd] = 0.f;
  }

  for (int v0 = v_begin; v0 < v_end; v0 += TK) {
    // ---- stage K/V rows [v0, v0+TK) ; rows that are not attended are zero-filled ----
    constexpr int CPR = D / V;  // 16-byte chunks per row
    for (int idx = tid; idx < TK * CPR; idx += kSimtThreads) {
      const int r = idx / CPR, ch = idx % CPR;
      int v = v0 + r;
      const T* kp = nullptr;
      const T* vp = nullptr;
      if (v < v_end) {
        if (v < n_hca) {
          kp = hca_k + (size_t)v * D;
          vp = hca_v + (size_t)v * D;
        } else {
          v -= n_hca;
          if (v < n_cur * C) {
            const int slot = v / C, row = v % C;
            const long long valid = n_csa - (long long)tblc[slot] * C;
            if (row < valid) {
              kp = hot_pool + ((size_t)tblp[slot] * 2 * C + row) * D;
              vp = kp + (size_t)C * D;
            }
          } else {
            v -= n_cur * C;
            kp = win_k + (size_t)v * D;
            vp = win_v + (size_t)v * D;
          }
        }
      }
      T* kd = Ks + r * KROW + ch * V;
      T* vd = Vs + r * D + ch * V;
      if (kp) {
        cp_async16(kd, kp + ch * V);
        cp_async16(vd, vp + ch * V);
      } else {
        *reinterpret_cast<uint4*>(kd) = make_uint4(0, 0, 0, 0);
        *reinterpret_cast<uint4*>(vd) = make_uint4(0, 0, 0, 0);
      }
    }
    // validity of the key this lane scores (same resolution, without pointers)
    bool key_ok = false;
    {
      int v = v0 + lane;
      if (v < v_end) {
        if (v < n_hca) key_ok = true;
        else {
          v -= n_hca;
          if (v < n_cur * C) key_ok = (v % C) < (n_csa - (long long)tblc[v / C] * C);
          else key_ok = true;
        }
      }
    }
    cp_async_wait_all();
    __syncthreads();

    // ---- S = q K^T : lane <-> key, warp <-> HPW heads ----
    float sc[HPW];
#pragma unroll
    for (int hh = 0; hh < HPW; ++hh) sc[hh] = 0.f;
    const T* krow = Ks + lane * KROW;
#pragma unroll 4
    for (int d0 = 0; d0 < D; d0 += V) {
      float kf[V];
      Elem<T>::load16(krow + d0, kf);
#pragma unroll
      for (int hh = 0; hh < HPW; ++hh) {
        float qf[V];
        Elem<T>::load16(qs + (warp * HPW + hh) * D + d0, qf);
#pragma unroll
        for (int j = 0; j < V; ++j) sc[hh] = fmaf(kf[j], qf[j], sc[hh]);
      }
    }
    // ---- online softmax (log2 domain) ----
    float alpha[HPW];
#pragma unroll
    for (int hh = 0; hh < HPW; ++hh) {
      const float s2 = key_ok ? sc[hh] * scale_log2 : -INFINITY;
      const float m_new = fmaxf(m_run[hh], warp_max(s2));
      float p = 0.f;
      alpha[hh] = 1.f;
      if (m_new != -INFINITY) {
        p = exp2f(s2 - m_new);
        alpha[hh] = exp2f(m_run[hh] - m_new);
      }
      l_run[hh] = l_run[hh] * alpha[hh] + warp_sum(p);
      m_run[hh] = m_new;
      ps[(warp * HPW + hh) * TK + lane] = p;
    }
    __syncwarp();
    // ---- O = alpha O + P V : lane <-> DPL contiguous dims ----
#pragma unroll
    for (int hh = 0; hh < HPW; ++hh)
#pragma unroll
      for (int dd = 0; dd < DPL; ++dd) o[hh][dd] *= alpha[hh];
#pragma unroll 2
    for (int j0 = 0; j0 < TK; j0 += 4) {
      float4 p4[HPW];
#pragma unroll
      for (int hh = 0; hh < HPW; ++hh)
        p4[hh] = *reinterpret_cast<const float4*>(ps + (warp * HPW + hh) * TK + j0);
#pragma unroll
      for (int jj = 0; jj < 4; ++jj) {
        float vf[DPL];
        load_contig<T, DPL>(Vs + (j0 + jj) * D + lane * DPL, vf);
#pragma unroll
        for (int hh = 0; hh < HPW; ++hh) {
          const float pj = jj == 0 ? p4[hh].x : jj == 1 ? p4[hh].y : jj == 2 ? p4[hh].z : p4[hh].w;
#pragma unroll
          for (int dd = 0; dd < DPL; ++dd) o[hh][dd] = fmaf(pj, vf[dd], o[hh][dd]);
        }
      }
    }
    __syncthreads();   // tile buffers are reused
  }

  // ---- emit the split partial (m, l, o) ----
  const size_t slot = (size_t)b * s_max + s;
#pragma unroll
  for (int hh = 0; hh < HPW; ++hh) {
    const int h = warp * HPW + hh;
    float* po = part_o + (slot * H + h) * D + lane * DPL;
#pragma unroll
    for (int dd = 0; dd < DPL; ++dd) po[dd] = o[hh][dd];
    if (lane == 0) {
      part_ml[(slot * H + h) * 2 + 0] = m_run[hh];
      part_ml[(slot * H + h) * 2 + 1] = l_run[hh];
    }
  }
}

// ---- S8 combine: grid (H, B), 128 threads -------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(128)
combine_kernel(const SeqDev* __restrict__ seqs, int H, int D, int C, int keys_per_cta, int s_max,
               const float* __restrict__ part_o, const float* __restrict__ part_ml, T* __restrict__ out,
               float* __restrict__ lse) {
  extern __shared__ float wsm[];   // [s_max] weights
  __shared__ float red_m[4], red_l[4];
  const int h = blockIdx.x, b = blockIdx.y;
  const SeqDev& sq = seqs[b];
  const int n_virtual = sq.n_hca + sq.n_tbl[sq.cur_buf] * C + sq.w_len;
  const int n_split = min(s_max, (n_virtual + keys_per_cta - 1) / keys_per_cta);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const size_t base = (size_t)b * s_max;

  float m_loc = -INFINITY;
  for (int i = tid; i < n_split; i += blockDim.x) m_loc = fmaxf(m_loc, part_ml[((base + i) * H + h) * 2]);
  m_loc = warp_max(m_loc);
  if (lane == 0) red_m[warp] = m_loc;
  __syncthreads();
  const float m_star = fmaxf(fmaxf(red_m[0], red_m[1]), fmaxf(red_m[2], red_m[3]));
  float l_loc = 0.f;
  for (int i = tid; i < n_split; i += blockDim.x) {
    const float mi = part_ml[((base + i) * H + h) * 2];
    const float w = (mi == -INFINITY) ? 0.f : exp2f(mi - m_star);
    wsm[i] = w;
    l_loc += w * part_ml[((base + i) * H + h) * 2 + 1];
  }
  l_loc = warp_sum(l_loc);
  if (lane == 0) red_l[warp] = l_loc;
  __syncthreads();
  const float l_star = (red_l[0] + red_l[1]) + (red_l[2] + red_l[3]);
  const bool empty = (n_split == 0) || !(l_star > 0.f);
  const float inv_l = empty ? 0.f : 1.f / l_star;
  for (int d = tid; d < D; d += blockDim.x) {
    float acc = 0.f;
    for (int i = 0; i < n_split; ++i) acc = fmaf(wsm[i], part_o[((base + i) * H + h) * D + d], acc);
    out[((size_t)b * H + h) * D + d] = Elem<T>::from_f(acc * inv_l);
  }
  if (lse && tid == 0)
    lse[(size_t)b * H + h] = empty ? -INFINITY : (m_star + log2f(l_star)) * 0.6931471805599453f;
}

// ---- dispatch ---------------------------------------------------------------------------------
#define LSA_SIMT_SHAPES(X) \
  X(8, 64) X(8, 128) X(16, 64) X(16, 128) X(16, 512) X(64, 64) X(64, 128) X(64, 512)

template <typename T, int H, int D>
static cudaError_t simt_prepare(size_t smem) {
  return cudaFuncSetAttribute(attn_simt_kernel<T, H, D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
}

bool simt_supported(int dtype, int H, int D) {
  (void)dtype;
#define X(h, d) if (H == h && D == d) return true;
  LSA_SIMT_SHAPES(X)
#undef X
  return false;
}
int simt_tile_keys() { return kSimtTile; }

template <typename T>
static cudaError_t smem_bytes_t(int H, int D, int k, size_t* bytes) {
#define X(h, d) if (H == h && D == d) { *bytes = SimtLayout<T, h, d>::total(k); return cudaSuccess; }
  LSA_SIMT_SHAPES(X)
#undef X
  return cudaErrorInvalidValue;
}

cudaError_t simt_smem_bytes(int dtype, int H, int D, int k, size_t* bytes) {
  return dtype == 0 ? smem_bytes_t<float>(H, D, k, bytes) : smem_bytes_t<__nv_bfloat16>(H, D, k, bytes);
}

template <typename T>
static cudaError_t occ_t(int H, int D, int k, int* ctas) {
#define X(h, d)                                                                                          \
  if (H == h && D == d) {                                                                                \
    size_t sm = SimtLayout<T, h, d>::total(k);                                                           \
    cudaError_t e = simt_prepare<T, h, d>(sm);                                                           \
    if (e != cudaSuccess) return e;                                                                      \
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas, attn_simt_kernel<T, h, d>, kSimtThreads, sm); \
  }
  LSA_SIMT_SHAPES(X)
#undef X
  return cudaErrorInvalidValue;
}

cudaError_t simt_max_ctas_per_sm(int dtype, int H, int D, int k, int* ctas) {
  return dtype == 0 ? occ_t<float>(H, D, k, ctas) : occ_t<__nv_bfloat16>(H, D, k, ctas);
}

template <typename T>
static cudaError_t launch_simt_t(int H, int D, int C, int k, const SeqDev* seqs, PoolDev pool, const void* hot_pool,
                                 const void* q, float sm_scale, AttnGeom g, int B, float* part_o, float* part_ml,
                                 cudaStream_t st) {
  const float scale_log2 = sm_scale * 1.4426950408889634f;
  dim3 grid(g.s_max, B);
#define X(h, d)                                                                                             \
  if (H == h && D == d) {                                                                                   \
    size_t sm = SimtLayout<T, h, d>::total(k);                                                              \
    cudaError_t e = simt_prepare<T, h, d>(sm);                                                              \
    if (e != cudaSuccess) return e;                                                                         \
    attn_simt_kernel<T, h, d><<<grid, kSimtThreads, sm, st>>>(seqs, pool, (const T*)hot_pool, (const T*)q,  \
                                                              scale_log2, C, k, g.keys_per_cta, g.s_max,    \
                                                              part_o, part_ml);                             \
    return cudaGetLastError();                                                                              \
  }
  LSA_SIMT_SHAPES(X)
#undef X
  return cudaErrorInvalidValue;
}

cudaError_t launch_attn_simt(int dtype, int H, int D, int C, int k, const SeqDev* seqs, PoolDev pool,
                             const void* hot_pool, const void* q, float sm_scale, AttnGeom g, int B, float* part_o,
                             float* part_ml, cudaStream_t st) {
  return dtype == 0 ? launch_simt_t<float>(H, D, C, k, seqs, pool, hot_pool, q, sm_scale, g, B, part_o, part_ml, st)
                    : launch_simt_t<__nv_bfloat16>(H, D, C, k, seqs, pool, hot_pool, q, sm_scale, g, B, part_o,
                                                   part_ml, st);
}

cudaError_t launch_combine(int dtype, int H, int D, int C, const SeqDev* seqs, AttnGeom g, int B, const float* part_o,
                           const float* part_ml, void* out, float* lse, cudaStream_t st) {
  dim3 grid(H, B);
  size_t sm = (size_t)g.s_max * sizeof(float);
  if (dtype == 0)
    combine_kernel<float><<<grid, 128, sm, st>>>(seqs, H, D, C, g.keys_per_cta, g.s_max, part_o, part_ml, (float*)out, lse);
  else
    combine_kernel<__nv_bfloat16><<<grid, 128, sm, st>>>(seqs, H, D, C, g.keys_per_cta, g.s_max, part_o, part_ml,
                                                         (__nv_bfloat16*)out, lse);
  return cudaGetLastError();
}

}  // namespace lsa
