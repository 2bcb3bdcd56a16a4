// lsa_attn_tc_defs.cuh - S7 split-K decode attention on tcgen05 tensor cores + TMA, and S8 combine (sm_100a)
//
// Shape: bf16, H = 64 query heads sharing ONE K and ONE V of D = 512 (MQA, DESIGN R19),
// pages of C = 128 rows (BASELINE.json configs 2-5).  Per key the path moves 2 KiB and does
// 4*H*D = 131 kFLOP (64 flop/B), so it is HBM-bound only if tensor cores carry the two contractions.
//
// Formulation ("keys on M"): with only 64 heads a head-major MMA would run at M = 64, i.e. half rate, and
// its 64x512 fp32 accumulator would fill all 512 TMEM columns.  Instead each 128-key tile computes
//     S^T[128 keys x 64 heads] = K_tile[128 x 512] . Q^T            (A = K, K-major;  B = Q, K-major)
//     O^T[512 x 64 heads]     += V_tile^T[512 x 128] . P^T           (A = V, MN-major; B = P, MN-major)
//     L  [128 x 64 heads]     += 1[128 x 128]        . P^T           (row sums of P for free)
// all at M = 128, N = 64: every K and V byte is read from shared memory exactly once, straight from the
// swizzled TMA landing buffers, and O^T needs only 4 x 64 TMEM columns.  At N = 64 one MMA reads
// 4 KiB of A + 2 KiB of B from shared memory, i.e. it is paced by the 128 B/clk shared-memory port
// (48 clk per MMA, measured) - 3456 clk per 128-key tile against >= 5700 clk of TMA time per tile.
//
// Work unit: a TILE = 128 consecutive rows of one tensor (HCA rows [128j, 128j+128), one page of the
// current table, window rows [128j, ...)), so every TMA box is one 32 KiB [2 d-blocks][128 rows][128 B]
// image (3-D tensor map: 64 columns x rows x 8 d-blocks).  The flat tile list of the batch (per sequence:
// HCA tiles, pages in table order, window tiles) is cut into n_attn contiguous ranges (n_attn <= SM count,
// chosen so every CTA gets the same number of whole tiles); a CTA emits one (m, l, o) partial per sequence it
// touches and a combine kernel (lsa_attn_tc.cu) merges them (S8).  S6 and the window append ride on the launch
// on steps without a trigger (make_view / commit_state below).
//   warp 0    : TMA producer  - Q tile (one 64 KiB box), then K/V stages (4-deep ring of 32 KiB)
//   warp 1    : MMA issuer    - one elected thread issues tcgen05.mma / tcgen05.commit
//   warps 2-9 : softmax       - thread <-> (key, half of the heads): TMEM -> regs, masked scale,
//                               2^(x-m) -> bf16 P tile (8 heads per 16-byte store, swizzled);
//                               the running maximum is exact on the first tile of a piece and kept
//                               until a logit exceeds it by 2^8 (one OR-reduction barrier per tile);
//                               epilogue TMEM -> partial in global memory
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>

#include <vector>

#include "lsa_attn_tc.h"
#include "lsa_tc_ptx.cuh"

namespace lsa {
using namespace ptx;

constexpr int kTcH = 64, kTcD = 512, kTcC = 128;
constexpr int kTcTile = 128;                // keys per tile
constexpr int kTcStages = 4;
constexpr int kTcStageBytes = 32768;        // [2 d-blocks][128 rows][128 B]
constexpr int kTcSoftmaxWarps = 8;
constexpr int kTcThreads = 64 + 32 * kTcSoftmaxWarps;
constexpr int kTcMaxB = 256;
constexpr float kRescaleThreshold = 8.0f;   // log2 units: P may grow to 2^8 before O is rescaled

// ---- split-K partial format --------------------------------------------------------------------
// The un-normalised O^T of a piece goes to the workspace as fp16 with one power-of-two scale per warp of the
// epilogue (32 d-rows x 32 heads): the block's largest magnitude lands in [2^14, 2^15), so every element within
// 2^-28 of it keeps fp16's 11-bit mantissa (relative error <= 2^-12, 8x below the rounding of the bf16 result)
// and smaller ones keep an absolute error below 2^-39 of the block maximum.  Half the bytes of fp32 partials:
// both the store at the end of the attention kernel (per-SM store bandwidth) and the combine kernel's read
// (L2 bandwidth) are bound by them at small B.  m and l stay fp32.
constexpr int kTcPartScales = 32;           // scales per slot: [4 d-blocks m][2 head halves hh][4 lane quarters]
__device__ __forceinline__ int part_scale_idx(size_t slot, int m, int hh, int q4) {
  return (int)(((slot * 4 + m) * 2 + hh) * 4 + q4);
}
// amax = largest |value| of the block.  Returns the multiplier (2^e) applied before the fp16 conversion and,
// through *inv, its exact inverse 2^-e; both are normal fp32 numbers for every amax (0, denormal, inf, NaN too).
__device__ __forceinline__ float part_scale(float amax, float* inv) {
  const int eb = (int)((__float_as_uint(amax) >> 23) & 0xffu);      // biased exponent of amax
  int sb = 268 - eb;                                                // 127 + 14 - (eb - 127)
  sb = sb > 253 ? 253 : sb;                                         // tiny or zero blocks: keep the inverse normal
  *inv = __uint_as_float((uint32_t)(254 - sb) << 23);
  return __uint_as_float((uint32_t)sb << 23);
}

// per-sequence shape as of this launch
struct SeqView {
  int b, t_hca, n_cur, n_hca, w_len, cur;
  int app_tile, app_slot;      // tile of this sequence holding the ring slot written by this launch (-1: no append)
  long long n_csa;
};

struct TcSmem {
  alignas(1024) unsigned char q[65536];                       // [8 d-blocks][64 heads][128 B], SW128
  alignas(1024) unsigned char stage[kTcStages][kTcStageBytes];// [2 d-blocks][128 keys][128 B], SW128
  alignas(1024) unsigned char p[16384];                       // [128 keys][64 heads] bf16, SW128 (MN-major B)
  alignas(1024) unsigned char ones[4096];                     // 128 x 16 bf16 ones, no swizzle
  alignas(16) float wmax[2][32][4];                           // [head half][head][lane quarter] tile maxima
  alignas(16) float mtile[2][4][32];                          // [head half][lane quarter][head] merged tile maxima
  SeqView view[kTcMaxB];                                      // per-sequence shape, read once by warp 0
  int gpre[kTcMaxB + 1];                                      // prefix of tiles per sequence
  uint64_t full[kTcStages], empty[kTcStages];
  uint64_t q_full, q_empty, s_full[2], s_empty[2], p_full, pv_done, o_full[4], o_empty, setup, app_done;
  uint32_t tmem_base;
};

struct TcParams {
  const SeqDev* seqs;
  const int* tbl_chunk;
  const int* tbl_page;
  const CUtensorMap* seq_maps;   // [B][4]: hca_k, hca_v, win_k, win_v
  int B, k;
  float scale_log2;
  uint2* part_o;                 // [slots][4 d-blocks m][2 head halves hh][8 head quads g][128 d][4 heads] fp16, scaled:
  float* part_s;                 // [slots][m][hh][4 lane quarters]: o = fp16 value * part_s (a power of two), see part_scale()
  float* part_m;                 // [slots][H]   (log2 domain)
  float* part_l;                 // [slots][H]
  int2* piece_info;              // [grid]: (first sequence, number of sequences) this CTA wrote partials for
  // S6 + window append folded into this launch (steps without a trigger): every CTA applies them to its VIEW of
  // the per-sequence records; the records themselves are updated once, after the grid, by commit_state()
  SeqDev* seqs_mut;
  unsigned int swap[kTcMaxB / 32];   // bit b: sequence b's staged table becomes current (if one is pending)
  const __nv_bfloat16* k_new;        // [B][D] or null: row b is written to ring slot w_head of sequence b
  const __nv_bfloat16* v_new;
  int W;                             // ring capacity
  // Level 2 (Eq.(6); lsa_l2.cu): key mask of the pages of the current table, [B][k][4] words (bit r of word
  // r / 32 = row r of the page is one of the Top-k entries), or null: every valid row is attended
  const uint32_t* l2_mask;
  // fused S8 (small batches): the grid meets at a counter barrier and merges the partials itself
  int fused;                     // 1: no combine kernel follows
  int n_attn;                    // CTAs that own tiles (the remaining CTAs of the grid only help with the merge)
  unsigned int* grid_ctr;        // monotonically increasing arrival counter
  unsigned int grid_target;      // value of the counter once every CTA of this launch has arrived
  __nv_bfloat16* out;            // [B][H][D]      (fused mode)
  float* lse;                    // [B][H] or null (fused mode)
  // profiling only (null otherwise): [0] = min over CTAs of %globaltimer once past the launch dependency,
  // [1] = max over CTAs at exit - the kernel's own working time, with programmatic overlap left intact
  unsigned long long* ktime;
};

__device__ __forceinline__ SeqView make_view(const TcParams& p, int b) {
  const SeqDev& s = p.seqs[b];
  SeqView v;
  const bool swap = ((p.swap[b >> 5] >> (b & 31)) & 1u) && s.pending;
  v.b = b; v.n_hca = s.n_hca; v.t_hca = (s.n_hca + kTcTile - 1) / kTcTile;
  v.cur = swap ? 1 - s.cur_buf : s.cur_buf;
  v.n_cur = s.n_tbl[v.cur];
  v.n_csa = s.n_csa;
  v.w_len = s.w_len; v.app_tile = -1; v.app_slot = 0;
  if (p.k_new) {
    v.app_slot = s.w_head;
    v.w_len = min(p.W, s.w_len + 1);
    v.app_tile = v.t_hca + v.n_cur + s.w_head / kTcTile;
  }
  return v;
}

// The per-sequence records catch up with the view: one thread per sequence, after the whole grid has finished.
__device__ __forceinline__ void commit_state(const TcParams& p, int b) {
  SeqDev& s = p.seqs_mut[b];
  if (((p.swap[b >> 5] >> (b & 31)) & 1u) && s.pending) { s.cur_buf = 1 - s.cur_buf; s.pending = 0; }
  if (p.k_new) {
    const int slot = s.w_head;
    s.w_head = (slot + 1 == p.W) ? 0 : slot + 1;
    s.w_len = min(p.W, s.w_len + 1);
    s.app_epoch += 1;          // the row was written by the attention grid, which has completed
  }
}

// where tile t of a sequence lives
struct TileSrc {
  const CUtensorMap* mk;
  const CUtensorMap* mv;
  int row_k, row_v;
};

__device__ __forceinline__ TileSrc tile_src(const TcParams& p, const CUtensorMap* map_pool, const SeqView& v, int t) {
  TileSrc r;
  if (t < v.t_hca) {
    r.mk = p.seq_maps + v.b * 4 + 0; r.mv = p.seq_maps + v.b * 4 + 1;
    r.row_k = r.row_v = t * kTcTile;
    return r;
  }
  t -= v.t_hca;
  if (t < v.n_cur) {
    const int page = p.tbl_page[((size_t)v.b * 2 + v.cur) * p.k + t];
    r.mk = r.mv = map_pool;
    r.row_k = page * (2 * kTcC); r.row_v = r.row_k + kTcC;
    return r;
  }
  t -= v.n_cur;
  r.mk = p.seq_maps + v.b * 4 + 2; r.mv = p.seq_maps + v.b * 4 + 3;
  r.row_k = r.row_v = t * kTcTile;
  return r;
}

// attended rows of tile t (the rest of its 128 rows is masked)
__device__ __forceinline__ int tile_valid(const TcParams& p, const SeqView& v, int t) {
  if (t < v.t_hca) return min(kTcTile, v.n_hca - t * kTcTile);
  t -= v.t_hca;
  if (t < v.n_cur) {
    const int chunk = p.tbl_chunk[((size_t)v.b * 2 + v.cur) * p.k + t];
    return (int)max(0ll, min((long long)kTcC, v.n_csa - (long long)chunk * kTcC));
  }
  t -= v.n_cur;
  return min(kTcTile, v.w_len - t * kTcTile);
}

// Level-2 key mask of tile t for the 32 rows [32 * q4, 32 * q4 + 32): all ones outside the page segment
__device__ __forceinline__ uint32_t tile_keymask(const TcParams& p, const SeqView& v, int t, int q4) {
  if (!p.l2_mask) return 0xffffffffu;
  t -= v.t_hca;
  if (t < 0 || t >= v.n_cur) return 0xffffffffu;
  return p.l2_mask[((size_t)v.b * p.k + t) * 4 + q4];
}

// Iterates the (sequence, tile range) pieces of this CTA's share [f0, f1) of the flat tile list.
// 32-bit arithmetic: T < 2^21 tiles, n_cta <= 256.
struct PieceCursor {
  const int* gpre;
  int B, f, f1, b;
  __device__ PieceCursor(const int* gpre_, int B_, int cta, int n_cta) : gpre(gpre_), B(B_) {
    const unsigned T = (unsigned)gpre_[B_];
    f = (int)((unsigned)cta * T / (unsigned)n_cta);
    f1 = (int)((unsigned)(cta + 1) * T / (unsigned)n_cta);
    if (cta >= n_cta) f = f1 = 0;                 // helper CTA: no tiles
    b = 0;
  }
  // returns false when exhausted; else fills b_out and the tile range [t0, t1) inside sequence b_out
  __device__ bool next(int& b_out, int& t0, int& t1) {
    if (f >= f1) return false;
    while (gpre[b + 1] <= f) ++b;
    b_out = b;
    t0 = f - gpre[b];
    const int end = min(f1, gpre[b + 1]);
    t1 = end - gpre[b];
    f = end;
    return true;
  }
};

__device__ __forceinline__ unsigned long long gtime() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
  return t;
}

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

}  // namespace lsa
