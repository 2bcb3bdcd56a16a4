// lsa_attn_tc.cu - S7 split-K decode attention on tcgen05 tensor cores + TMA, and S8 combine (sm_100a)
//
// Shape: bf16, H = 64 query heads sharing ONE K and ONE V of D = 512 (MQA, DESIGN R19),
// pages of C = 128 rows (BASELINE.json configs 2-5).  Per key the path moves 2 KiB and does
// 4*H*D = 131 kFLOP (64 flop/B), so it is HBM-bound only if tensor cores carry the two contractions.
//
// Formulation ("keys on M"): with only 64 heads a head-major MMA would run at M = 64, i.e. half rate, and
// its 64x512 fp32 accumulator would fill all 512 TMEM columns.  Instead each 128-key tile computes
//     S^T[128 keys x 64 heads] = K_tile[128 x 512] . Q^T            (A = K, K-major;  B = Q, K-major)
//     O^T[512 x 64 heads]     += V_tile^T[512 x 128] . P^T           (A = V, MN-major; B = P, K-major)
//     L  [128 x 64 heads]     += 1[128 x 128]        . P^T           (row sums of P for free)
// all at M = 128, N = 64: every K and V byte is read from shared memory exactly once, straight from the
// swizzled TMA landing buffers, and O^T needs only 4 x 64 TMEM columns.
//
// One persistent CTA per SM owns a contiguous range of 32-key groups of the batch's flat key list
// (HCA rows, pages of the current table, window rows - per sequence, in that order) and emits one
// (m, l, o) partial per sequence it touches; lsa_combine_tc merges them (S8).
//   warp 0   : TMA producer   - Q tile, then K/V stages (4-deep ring of 32 KiB = 128 keys x 128 dims)
//   warp 1   : MMA issuer     - one elected thread issues tcgen05.mma / tcgen05.commit
//   warps 2-5: softmax        - thread <-> key: TMEM -> regs, masked scale, cross-lane max via
//                               redux.sync, 2^(x-m) -> bf16 P tile in swizzled smem; lazy O rescale;
//                               epilogue TMEM -> partial in global memory
#pragma once
#include <cuda.h>

#include <vector>

#include "lsa_attn_tc.h"
#include "lsa_tc_ptx.cuh"

namespace lsa {
using namespace ptx;

constexpr int kTcH = 64, kTcD = 512, kTcC = 128;
constexpr int kTcStages = 4;
constexpr int kTcStageBytes = 32768;
constexpr int kTcThreads = 192;
constexpr int kTcMaxB = 256;
constexpr float kRescaleThreshold = 8.0f;   // log2 units: P may grow to 2^8 before O is rescaled

struct TcSmem {
  alignas(1024) unsigned char q[65536];                       // [8 d-blocks][64 heads][128 B], SW128
  alignas(1024) unsigned char stage[kTcStages][kTcStageBytes];// [2 d-blocks][128 keys][128 B], SW128
  alignas(1024) unsigned char p[16384];                       // [2 key-blocks][64 heads][128 B], SW128
  alignas(1024) unsigned char ones[4096];                     // 128 x 16 bf16 ones, no swizzle
  float wmax[2][kTcH][4];                                     // per-warp tile maxima (ordered ints)
  int gpre[kTcMaxB + 1];                                      // prefix of 32-key groups per sequence
  uint64_t full[kTcStages], empty[kTcStages];
  uint64_t q_full, q_empty, s_full[2], s_empty[2], p_full, pv_done, o_empty;
  uint32_t tmem_base;
};

struct TcParams {
  const SeqDev* seqs;
  const int* tbl_chunk;
  const int* tbl_page;
  const CUtensorMap* seq_maps;   // [B][4]: hca_k, hca_v, win_k, win_v
  int B, k, pool_rows;
  float scale_log2;
  float* part_o;                 // [slots][H][D]
  float* part_m;                 // [slots][H]   (log2 domain)
  float* part_l;                 // [slots][H]
};

__device__ __forceinline__ int seq_groups(const SeqDev& s) {
  return (s.n_hca + 31) / 32 + s.n_tbl[s.cur_buf] * (kTcC / 32) + (s.w_len + 31) / 32;
}

// where a 32-key group of a sequence lives
struct GroupSrc {
  const CUtensorMap* mk;
  const CUtensorMap* mv;
  int row_k, row_v, n_valid;
};

struct SeqView {
  int b, g_hca, n_cur, n_hca, w_len, cur;
  long long n_csa;
};

__device__ __forceinline__ SeqView make_view(const TcParams& p, int b) {
  const SeqDev& s = p.seqs[b];
  SeqView v;
  v.b = b; v.n_hca = s.n_hca; v.g_hca = (s.n_hca + 31) / 32; v.cur = s.cur_buf; v.n_cur = s.n_tbl[s.cur_buf];
  v.w_len = s.w_len; v.n_csa = s.n_csa;
  return v;
}

__device__ __forceinline__ GroupSrc resolve_group(const TcParams& p, const CUtensorMap* map_pool, const SeqView& v, int g,
                                                  int g_end) {
  GroupSrc r;
  if (g >= g_end) {                       // beyond this CTA's range: whole box out of bounds -> TMA zero fill
    r.mk = r.mv = map_pool; r.row_k = r.row_v = p.pool_rows; r.n_valid = 0;
    return r;
  }
  if (g < v.g_hca) {
    r.mk = p.seq_maps + v.b * 4 + 0; r.mv = p.seq_maps + v.b * 4 + 1;
    r.row_k = r.row_v = g * 32; r.n_valid = min(32, v.n_hca - g * 32);
    return r;
  }
  g -= v.g_hca;
  if (g < v.n_cur * 4) {
    const int slot = g >> 2, r0 = (g & 3) * 32;
    const size_t ti = ((size_t)v.b * 2 + v.cur) * p.k + slot;
    const int chunk = p.tbl_chunk[ti], page = p.tbl_page[ti];
    const long long valid_rows = v.n_csa - (long long)chunk * kTcC;
    r.mk = r.mv = map_pool;
    r.row_k = page * (2 * kTcC) + r0; r.row_v = r.row_k + kTcC;
    r.n_valid = (int)max(0ll, min(32ll, valid_rows - r0));
    return r;
  }
  g -= v.n_cur * 4;
  r.mk = p.seq_maps + v.b * 4 + 2; r.mv = p.seq_maps + v.b * 4 + 3;
  r.row_k = r.row_v = g * 32; r.n_valid = min(32, v.w_len - g * 32);
  return r;
}

// Iterates the (sequence, group range) pieces of this CTA's share [f0, f1) of the flat group list.
struct PieceCursor {
  const int* gpre;
  int B, f, f1, b;
  __device__ PieceCursor(const int* gpre_, int B_, int cta, int n_cta) : gpre(gpre_), B(B_) {
    const long long T = gpre_[B_];
    f = (int)((long long)cta * T / n_cta);
    f1 = (int)((long long)(cta + 1) * T / n_cta);
    b = 0;
  }
  // returns false when exhausted; else fills b_out and the group range [g0, g1) inside sequence b_out
  __device__ bool next(int& b_out, int& g0, int& g1) {
    if (f >= f1) return false;
    while (gpre[b + 1] <= f) ++b;
    b_out = b;
    g0 = f - gpre[b];
    const int end = min(f1, gpre[b + 1]);
    g1 = end - gpre[b];
    f = end;
    return true;
  }
};

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ int float_ordered_s32(float f) {   // monotone float -> signed int
  int b = __float_as_int(f);
  return b >= 0 ? b : (b ^ 0x7fffffff);
}
__device__ __forceinline__ float s32_ordered_float(int i) { return __int_as_float(i >= 0 ? i : (i ^ 0x7fffffff)); }

}  // namespace lsa
