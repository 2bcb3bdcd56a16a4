// lsa_l1.cu - the paper-exact Level-1 Memory Indexer (Eq.(1)-(5), l.142 Eq.(13))
//
//   Eq.(1) c^Q = h W^DQ        Eq.(2) q = c^Q W^IUQ (n_h heads of c^I)        Eq.(3) w = h W^w
//   Eq.(4) I_s = sigmoid( sum_h w_h ReLU(q_h . K_s^IComp) )  for every compressed entry s
//   Eq.(5) recall { s : I_s >= 0.5 }, bounded by K_max;   Eq.(13) OR-union over the indexer layers
// Page-granular recall (l.185): chunk c is recalled iff any of its entries qualifies in any layer; if more
// than K_max chunks qualify the K_max best by (score desc, chunk id asc) are kept (DESIGN "NEXT-1 readings").
//
// Kernels
//   l1_gemv_kernel      Eq.(1)-(3): one warp per output row, 16-byte loads, fp32 accumulation.  c^Q stays fp32;
//                       q is rounded to bf16 (it is the B operand of the tensor-core match below).  Two launches
//                       per trigger: Eq.(1)+(3) of every layer, then Eq.(2) of every layer.
//   l1_score_kernel     Eq.(4) over all entries, the only heavy part: 64 MiB of index keys per layer at 1M
//                       context against 4.3 GFLOP -> HBM-bound with the match on tensor cores.  Same
//                       "entries on M" formulation as the attention kernel: per 128-entry tile
//                       S^T[128 entries x 64 heads] = K_tile[128 x 128] . q^T  (8 tcgen05.mma, M=128 N=64 K=16),
//                       TMA boxes of 32 KiB through a 6-deep ring, S^T double-buffered in TMEM.  A thread owns
//                       one entry: ReLU, head-weighted sum and the validity mask are thread-local, and because
//                       a tile is exactly one chunk (C = 128) the chunk maximum is one redux + one 4-way max.
//   l1_select_kernel    Eq.(5)/(13) + K_max: max over layers, threshold on the pre-activation
//                       (sigmoid is monotone: I >= thr  <=>  pre >= logit(thr)), block-wide select.
#include <cuda.h>
#include <cuda_bf16.h>

#include <cmath>
#include <string>
#include <vector>

#include "lsa_kernels.h"
#include "lsa_l1.h"
#include "lsa_select.cuh"
#include "lsa_tc_ptx.cuh"

namespace lsa {
using namespace ptx;

constexpr int kL1H = 64, kL1C = 128, kL1CI = 128;   // indexer heads, entries per chunk (= tile), index-key dim
constexpr int kL1Stages = 6;
constexpr int kL1StageBytes = 32768;                 // [2 d-blocks][128 entries][128 B]
constexpr int kL1Threads = 64 + 128;                 // producer warp, MMA warp, 4 epilogue warps
constexpr int kL1MaxPieces = 4 * kFireMax;           // (sequence, layer) pairs per launch

// ---- Eq.(1)-(3): y[i][e] = sum_d W[e][d] x[i][d] ------------------------------------------------------------
template <typename XT> struct L1X;
template <> struct L1X<__nv_bfloat16> {
  static __device__ __forceinline__ void load8(const __nv_bfloat16* p, float* out) { Elem<__nv_bfloat16>::load16(p, out); }
};
template <> struct L1X<float> {
  static __device__ __forceinline__ void load8(const float* p, float* out) {
    const float4 a = *reinterpret_cast<const float4*>(p), b = *reinterpret_cast<const float4*>(p + 4);
    out[0] = a.x; out[1] = a.y; out[2] = a.z; out[3] = a.w; out[4] = b.x; out[5] = b.y; out[6] = b.z; out[7] = b.w;
  }
};
template <typename OT> __device__ __forceinline__ OT l1_out(float v);
template <> __device__ __forceinline__ float l1_out<float>(float v) { return v; }
template <> __device__ __forceinline__ __nv_bfloat16 l1_out<__nv_bfloat16>(float v) { return __float2bfloat16_rn(v); }

constexpr int kGvWarps = 4, kGvSeqs = 4;

// W bf16 [E][Din]; x rows of stride ldx (input i is row xrows.ids[i]); out [n][ldo] (row i at out + i*ldo).
// One launch carries several independent products that share Din ("jobs": the three layers' Eq.(1) and Eq.(3) in
// one launch, their Eq.(2) in another) - a single layer's matrix is one wave of blocks and leaves HBM half idle.
// Blocks are persistent: a block stages its (up to 4) x rows in shared memory ONCE - read from L2 inside the
// FMA loop they would be 16 dependent round trips per lane - and its warps then walk weight rows r, r + stride,
// ... with all loads of a row in flight; the other warps of the SM cover a warp's latency.
//   shared_x = 1: every job reads the same x; the rows of all jobs form one flat list, gridDim.z = 1
//   shared_x = 0: job = blockIdx.z has its own x
constexpr int kGvMaxJobs = 8;
struct GvJobs {
  const __nv_bfloat16* W[kGvMaxJobs];   // [E][Din]
  const void* x[kGvMaxJobs];            // input rows (XT)
  void* out[kGvMaxJobs];                // row i at out + i * ldo (OT)
  long long ldo[kGvMaxJobs];
  int E[kGvMaxJobs];
  int n_jobs, shared_x;
  long long lo_off;                     // bf16 outputs only, 0 = off: element e also gets its rounding residual
                                        // bf16(v - float(bf16(v))) at out + lo_off, so that hi + lo carries ~16 bits
};

constexpr int kGvU = 8;                       // 16-byte loads per lane and batch: one batch = 2048 weights of a row
constexpr int kGvBatch = kGvU * 256;

// The warp's rows as a sequence of batches (row, d0); batch t+1 is loaded into the other register buffer before
// batch t is multiplied, so a warp always has 4 KiB in flight.  NS = sequences handled per block (1: the common
// single-trigger case without the 4x predicated code; 4: rows i0 .. i0+3, those >= n masked).
__device__ __forceinline__ void gv_locate(const GvJobs& jobs, int j_lo, int j_hi, int rr, int& j, int& e) {
  j = j_lo; e = rr;                                        // row rr of the flat list -> (job, row inside the job)
  while (j + 1 < j_hi && e >= jobs.E[j]) { e -= jobs.E[j]; ++j; }
}
__device__ __forceinline__ void gv_load(uint4* w, const __nv_bfloat16* wrow, int d0, int Din, int lane) {
#pragma unroll
  for (int u = 0; u < kGvU; ++u) {
    const int d = d0 + lane * 8 + u * 256;
    w[u] = d < Din ? *reinterpret_cast<const uint4*>(wrow + d) : make_uint4(0u, 0u, 0u, 0u);
  }
}

// wa holds batch 0 of row r0 = (j, e) already (loaded by the caller before the launch dependency resolved).
template <typename XT, typename OT, int NS>
__device__ __forceinline__ void gv_rows(const GvJobs& jobs, const XT* xs, int j_lo, int j_hi, int total, int stride, int r0,
                                        int i0, int n, int Din, int lane, uint4 (&wa)[kGvU], int j, int e) {
  auto locate = [&](int rr, int& jj, int& ee) { gv_locate(jobs, j_lo, j_hi, rr, jj, ee); };
  auto load = [&](uint4* w, const __nv_bfloat16* wrow, int d0) { gv_load(w, wrow, d0, Din, lane); };
  float acc[NS][2];
#pragma unroll
  for (int s = 0; s < NS; ++s) acc[s][0] = acc[s][1] = 0.f;
  auto mul = [&](const uint4* w, int d0) {
#pragma unroll
    for (int u = 0; u < kGvU; ++u) {
      const int d = d0 + lane * 8 + u * 256;
      if (d < Din) {
        float wf[8];
        Elem<__nv_bfloat16>::unpack16(w[u], wf);
#pragma unroll
        for (int s = 0; s < NS; ++s) {
          if (NS == 1 || i0 + s < n) {
            float xf[8];
            L1X<XT>::load8(xs + (size_t)s * Din + d, xf);
#pragma unroll
            for (int jj = 0; jj < 8; ++jj) acc[s][jj & 1] = fmaf(wf[jj], xf[jj], acc[s][jj & 1]);
          }
        }
      }
    }
  };
  auto finish = [&](int j, int e) {
    OT* out = reinterpret_cast<OT*>(jobs.out[j]);
#pragma unroll
    for (int s = 0; s < NS; ++s) {
      const float v = warp_sum(acc[s][0] + acc[s][1]);
      if (lane == 0 && i0 + s < n) {
        const OT hi = l1_out<OT>(v);
        out[(size_t)(i0 + s) * jobs.ldo[j] + e] = hi;
        if constexpr (sizeof(OT) == 2) {
          if (jobs.lo_off) out[(size_t)(i0 + s) * jobs.ldo[j] + e + jobs.lo_off] = __float2bfloat16_rn(v - __bfloat162float(hi));
        }
      }
      acc[s][0] = acc[s][1] = 0.f;
    }
  };
  // state of the batch in flight / being multiplied
  int r = r0, d0 = 0;
  const __nv_bfloat16* wrow = r < total ? jobs.W[j] + (size_t)e * Din : nullptr;
  uint4 wb[kGvU];
  // one step: issue the loads of the next batch into `nxt`, multiply `cur`
  auto step = [&](uint4* cur, uint4* nxt) {
    int r2 = r, d2 = d0 + kGvBatch, j2 = j, e2 = e;
    const __nv_bfloat16* wrow2 = wrow;
    if (d2 >= Din) {
      r2 = r + stride; d2 = 0;
      if (r2 < total) { locate(r2, j2, e2); wrow2 = jobs.W[j2] + (size_t)e2 * Din; }
    }
    if (r2 < total) load(nxt, wrow2, d2);
    mul(cur, d0);
    if (r2 != r) finish(j, e);
    r = r2; d0 = d2; j = j2; e = e2; wrow = wrow2;
  };
  while (r < total) {
    step(wa, wb);
    if (r >= total) break;
    step(wb, wa);
  }
}

template <typename XT, typename OT>
__global__ void __launch_bounds__(kGvWarps * 32, 4)
l1_gemv_kernel(GvJobs jobs, long long ldx, FireList xrows, int n, int Din) {
  extern __shared__ __align__(16) unsigned char gv_smem[];
  XT* xs = reinterpret_cast<XT*>(gv_smem);                 // [kGvSeqs][Din]
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int i0 = blockIdx.y * kGvSeqs;
  const int j_lo = jobs.shared_x ? 0 : (int)blockIdx.z, j_hi = jobs.shared_x ? jobs.n_jobs : j_lo + 1;
  int total = 0;
  for (int j = j_lo; j < j_hi; ++j) total += jobs.E[j];
  const int stride = gridDim.x * kGvWarps, r0 = blockIdx.x * kGvWarps + warp;
  uint4 wa[kGvU];
  int j0 = j_lo, e0 = 0;
  if (r0 < total) {                                         // weights never depend on the previous kernel
    gv_locate(jobs, j_lo, j_hi, r0, j0, e0);
    gv_load(wa, jobs.W[j0] + (size_t)e0 * Din, 0, Din, lane);
  }
  pdl_wait();
  pdl_launch_dependents();
  constexpr int kPer16 = 16 / (int)sizeof(XT);
  const XT* x = reinterpret_cast<const XT*>(jobs.x[j_lo]);
  for (int s = 0; s < kGvSeqs; ++s)
    if (i0 + s < n)
      for (int d = threadIdx.x * kPer16; d < Din; d += kGvWarps * 32 * kPer16)
        *reinterpret_cast<uint4*>(xs + (size_t)s * Din + d) = *reinterpret_cast<const uint4*>(x + (size_t)xrows.ids[i0 + s] * ldx + d);
  __syncthreads();
  if (n - i0 == 1) gv_rows<XT, OT, 1>(jobs, xs, j_lo, j_hi, total, stride, r0, i0, n, Din, lane, wa, j0, e0);
  else gv_rows<XT, OT, kGvSeqs>(jobs, xs, j_lo, j_hi, total, stride, r0, i0, n, Din, lane, wa, j0, e0);
}

// ---- Eq.(4): entry scoring on tensor cores -----------------------------------------------------------------
struct L1Piece {
  int n_entries;     // valid compressed entries of the sequence
  int tile0;         // first tile of this (sequence, layer) piece in the launch's flat tile list
  int n_tiles;       // = n_chunks of the sequence
  int map_idx;       // tensor map of this (sequence, layer)'s index keys
};

struct L1ScoreParams {
  const CUtensorMap* k_maps;     // [B * n_layers]: index keys [n_entries][128] bf16 as (64, rows, 2 d-blocks)
  const float* wbuf;             // [n_pieces][64] head weights (Eq.3)
  float* chunk_pre;              // [n_pieces][n_chunks_max] max over the chunk's entries of the pre-activation
  int n_pieces, total_tiles, n_chunks_max;
  L1Piece pieces[kL1MaxPieces / 4];
};

struct L1Smem {
  alignas(1024) unsigned char q[32768];                          // [2 d-blocks][hi: 64 heads, lo: 64 heads][128 B], SW128
  alignas(1024) unsigned char stage[kL1Stages][kL1StageBytes];   // [2 d-blocks][128 entries][128 B], SW128
  float wm[2][4];                                                // per S buffer: the 4 warps' maxima
  uint64_t full[kL1Stages], empty[kL1Stages];
  uint64_t q_full, q_empty, s_full[2], s_empty[2];
  uint32_t tmem_base;
};

// pieces of this CTA's share [f0, f1) of the flat tile list
struct L1Cursor {
  const L1ScoreParams& p;
  int f, f1, pi;
  __device__ L1Cursor(const L1ScoreParams& p_, int cta, int n_cta) : p(p_) {
    f = (int)((unsigned)cta * (unsigned)p_.total_tiles / (unsigned)n_cta);
    f1 = (int)((unsigned)(cta + 1) * (unsigned)p_.total_tiles / (unsigned)n_cta);
    pi = 0;
  }
  __device__ bool next(int& piece, int& t0, int& t1) {
    if (f >= f1) return false;
    while (p.pieces[pi].tile0 + p.pieces[pi].n_tiles <= f) ++pi;
    piece = pi;
    t0 = f - p.pieces[pi].tile0;
    const int end = min(f1, p.pieces[pi].tile0 + p.pieces[pi].n_tiles);
    t1 = end - p.pieces[pi].tile0;
    f = end;
    return true;
  }
};

__global__ void __launch_bounds__(kL1Threads, 1)
l1_score_kernel(const __grid_constant__ CUtensorMap map_q, const __grid_constant__ L1ScoreParams p) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  L1Smem& sm = *reinterpret_cast<L1Smem*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int cta = blockIdx.x, n_cta = gridDim.x;
  if (tid == 0) {
    for (int i = 0; i < kL1Stages; ++i) { mbar_init(&sm.full[i], 1); mbar_init(&sm.empty[i], 1); }
    mbar_init(&sm.q_full, 1); mbar_init(&sm.q_empty, 1);
    for (int i = 0; i < 2; ++i) { mbar_init(&sm.s_full[i], 1); mbar_init(&sm.s_empty[i], 4); }
    fence_mbar_init();
    prefetch_tmap(&map_q);
  }
  if (warp == 1) tmem_alloc(&sm.tmem_base, 128);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  griddep_wait();                 // q, w and the piece list come from the kernels before this one
  griddep_launch_dependents();
  const uint32_t tS = sm.tmem_base;

  if (warp == 0) {
    // =========================== TMA producer ===========================
    if (elect_one()) {
      L1Cursor cur(p, cta, n_cta);
      int piece, t0, t1, item = 0;
      uint32_t ring = 0;
      while (cur.next(piece, t0, t1)) {
        if (item > 0) mbar_wait(&sm.q_empty, (item - 1) & 1, 40);
        mbar_arrive_expect_tx(&sm.q_full, 32768);
        tma_load_3d(sm.q, &map_q, 0, piece * 2 * kL1H, 0, &sm.q_full);
        const CUtensorMap* mk = p.k_maps + p.pieces[piece].map_idx;
        for (int t = t0; t < t1; ++t) {
          const int st = ring % kL1Stages;
          mbar_wait(&sm.empty[st], ((ring / kL1Stages) & 1) ^ 1, 41);
          mbar_arrive_expect_tx(&sm.full[st], kL1StageBytes);
          tma_load_3d(sm.stage[st], mk, 0, t * kL1C, 0, &sm.full[st]);
          ++ring;
        }
        ++item;
      }
    }
  } else if (warp == 1) {
    // =========================== MMA issuer ===========================
    if (elect_one()) {
      constexpr uint32_t id_s = make_idesc_bf16(128, 64, 0, 0);    // A = key tile (K-major), B = q (K-major)
      const uint64_t dk0 = make_sdesc(smem_u32(sm.stage[0]), 16, 1024, kLayoutSw128);
      const uint64_t dq0 = make_sdesc(smem_u32(sm.q), 16, 1024, kLayoutSw128);
      L1Cursor cur(p, cta, n_cta);
      int piece, t0, t1, item = 0;
      uint32_t ring = 0, n_s = 0;
      while (cur.next(piece, t0, t1)) {
        mbar_wait(&sm.q_full, item & 1, 42);
        tc_fence_after();
        for (int t = t0; t < t1; ++t) {
          const int buf = n_s & 1, st = ring % kL1Stages;
          mbar_wait(&sm.s_empty[buf], ((n_s >> 1) & 1) ^ 1, 43);
          mbar_wait(&sm.full[st], (ring / kL1Stages) & 1, 44);
          tc_fence_after();
          const uint64_t a0 = dk0 + (uint64_t)(st * (kL1StageBytes >> 4));
          // the query is kept as two bf16 terms (q = hi + lo, the Eq.(2) kernel writes both): K . hi, then K . lo into
          // the same accumulator - the match then carries the fp32 query, not its 8-bit rounding
#pragma unroll
          for (int ks = 0; ks < 16; ++ks) {
            const int kk = ks & 7, part = ks >> 3;
            const uint64_t off_a = (uint64_t)(((kk >> 2) * 16384 + (kk & 3) * 32) >> 4);
            const uint64_t off_b = (uint64_t)(((kk >> 2) * 16384 + part * 8192 + (kk & 3) * 32) >> 4);
            umma_bf16(tS + buf * 64, a0 + off_a, dq0 + off_b, id_s, ks != 0);
          }
          umma_commit(&sm.empty[st]);
          umma_commit(&sm.s_full[buf]);
          if (t == t1 - 1) umma_commit(&sm.q_empty);
          ++ring; ++n_s;
        }
        ++item;
      }
    }
  } else {
    // =========================== gate + reduce (4 warps, thread = entry) ===========================
    const int q4 = warp & 3;
    const uint32_t lane_addr = (uint32_t)(q4 * 32) << 16;
    const int row = q4 * 32 + lane;
    L1Cursor cur(p, cta, n_cta);
    int piece, t0, t1;
    uint32_t n_s = 0;
    while (cur.next(piece, t0, t1)) {
      float w[kL1H];
      const float4* wp = reinterpret_cast<const float4*>(p.wbuf + (size_t)piece * kL1H);
#pragma unroll
      for (int j = 0; j < kL1H / 4; ++j) { const float4 t4 = wp[j]; w[4 * j] = t4.x; w[4 * j + 1] = t4.y; w[4 * j + 2] = t4.z; w[4 * j + 3] = t4.w; }
      const int n_entries = p.pieces[piece].n_entries;
      for (int t = t0; t < t1; ++t) {
        const int buf = n_s & 1;
        float x[kL1H];
        mbar_wait(&sm.s_full[buf], (n_s >> 1) & 1, 45);
        tc_fence_after();
        tmem_ld32(tS + buf * 64 + lane_addr, reinterpret_cast<uint32_t*>(x));
        tmem_ld32(tS + buf * 64 + 32 + lane_addr, reinterpret_cast<uint32_t*>(x) + 32);
        tmem_wait_ld();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&sm.s_empty[buf]);
        float pre = 0.f;
#pragma unroll
        for (int h = 0; h < kL1H; ++h) pre = fmaf(w[h], fmaxf(x[h], 0.f), pre);          // Eq.(4) before the sigmoid
        if (t * kL1C + row >= n_entries) pre = -INFINITY;                                  // rows past the last entry
        const float wmax = redux_max_f32(pre);
        if (lane == 0) sm.wm[buf][q4] = wmax;
        named_bar_sync(1, 128);
        if (tid == 64) {
          const float m4 = fmaxf(fmaxf(sm.wm[buf][0], sm.wm[buf][1]), fmaxf(sm.wm[buf][2], sm.wm[buf][3]));
          p.chunk_pre[(size_t)piece * p.n_chunks_max + t] = m4;
        }
        ++n_s;
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(sm.tmem_base, 128);
  }
}

// ---- Eq.(5), (13), K_max ---------------------------------------------------------------------------------------
// one block per firing sequence; chunk_pre [(i * L + l)][n_chunks_max]
__global__ void __launch_bounds__(1024)
l1_select_kernel(const SeqDev* __restrict__ seqs, FireList fire, const float* __restrict__ chunk_pre, int n_layers, int n_chunks_max,
                 float logit_thr, int k, int32_t* __restrict__ sel_idx, float* __restrict__ sel_score) {
  __shared__ SelectSmem sm;
  const int i = blockIdx.x;
  pdl_wait();
  pdl_launch_dependents();
  const SeqDev& sq = seqs[fire.ids[i]];
  const float* base = chunk_pre + (size_t)i * n_layers * n_chunks_max;
  auto score = [base, n_layers, n_chunks_max](int c) -> float {      // Eq.(13): OR over layers = max over layers
    float s = base[c];
    for (int l = 1; l < n_layers; ++l) s = fmaxf(s, base[(size_t)l * n_chunks_max + c]);
    return s;
  };
  auto keyf = [score, logit_thr](int c) -> unsigned long long {      // Eq.(5): I >= thr  <=>  pre >= logit(thr)
    const float s = score(c);
    return s >= logit_thr ? (((unsigned long long)(~float_to_ordered(s)) << 32) | (unsigned)c) : kKeyMax;
  };
  const int m = block_select_smallest(keyf, sq.n_chunks, min(k, sq.n_chunks), sm);
  for (int j = threadIdx.x; j < k; j += blockDim.x) {
    int idx = -1;
    float val = -INFINITY;
    if (j < m && sm.keys[j] != kKeyMax) {
      idx = (int)(sm.keys[j] & 0xffffffffull);
      const float pre = ordered_to_float(~(uint32_t)(sm.keys[j] >> 32));
      val = 1.0f / (1.0f + __expf(-pre));
    }
    sel_idx[(size_t)i * k + j] = idx;
    if (sel_score) sel_score[(size_t)i * k + j] = val;
  }
}

// ---- host -------------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct L1Plan {
  L1Init init{};
  EncodeTiledFn encode = nullptr;
  CUtensorMap* d_maps = nullptr;       // [B * L]
  CUtensorMap map_q{};
  float* cq = nullptr;                 // [L][cap][d_c]
  __nv_bfloat16* q = nullptr;          // [cap * L][2: hi, lo][64 * 128]
  float* wbuf = nullptr;               // [cap * L][64]
  float* chunk_pre = nullptr;          // [cap * L][n_chunks_max]
  int cap = 0;                         // sequences per launch
  size_t smem = 0;
  int n_sms = 0;
  int occ13 = 1, occ2 = 1;             // resident GEMV blocks per SM (Eq.(1)+(3) launch, Eq.(2) launch)
};

// [rows][128] bf16 seen as (64 columns, rows, 2 d-blocks): a box lands as [2][box_rows][128 B], 128-byte swizzle
static bool l1_encode(EncodeTiledFn enc, CUtensorMap* m, const void* ptr, uint64_t rows, uint32_t box_rows, std::string* msg) {
  cuuint64_t dims[3] = {64, rows, 2};
  cuuint64_t strides[2] = {(cuuint64_t)kL1CI * 2, 128};
  cuuint32_t box[3] = {64, box_rows, 2};
  cuuint32_t es[3] = {1, 1, 1};
  CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(ptr), dims, strides, box, es,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { *msg = "cuTensorMapEncodeTiled failed with CUresult " + std::to_string((int)r); return false; }
  return true;
}

#define L1_CUDA(expr)                                                               \
  do {                                                                              \
    cudaError_t _e = (expr);                                                        \
    if (_e != cudaSuccess) {                                                        \
      *msg = std::string(#expr) + ": " + cudaGetErrorString(_e);                    \
      return -2;                                                                    \
    }                                                                               \
  } while (0)

bool l1_supported(int dtype, int C, int c_I, int n_h) { return dtype == 1 && C == kL1C && c_I == kL1CI && n_h == kL1H; }

int l1_create(const L1Init& init, L1Plan** out, std::string* msg) {
  L1Plan* pl = new L1Plan();
  pl->init = init;
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) {
    *msg = "cuTensorMapEncodeTiled entry point not found"; delete pl; return -2;
  }
  pl->encode = (EncodeTiledFn)fn;
  const int L = init.n_layers, B = init.B;
  pl->cap = std::max(1, std::min(kFireMax, (kL1MaxPieces / 4) / L));
  pl->n_sms = init.n_sms;
  std::vector<CUtensorMap> maps((size_t)B * L);
  for (int b = 0; b < B; ++b)
    for (int l = 0; l < L; ++l) {
      const void* ptr = init.index_k[(size_t)b * L + l];
      const long long rows = init.seq_host[b].n_csa;
      if (rows > 0 && !ptr) { *msg = "null index_k pointer"; delete pl; return -1; }
      if (!l1_encode(pl->encode, &maps[(size_t)b * L + l], rows > 0 ? ptr : init.layers[0].W_dq, rows > 0 ? (uint64_t)rows : kL1C, kL1C, msg)) {
        delete pl; return -2;
      }
    }
  L1_CUDA(cudaMalloc(&pl->d_maps, maps.size() * sizeof(CUtensorMap)));
  L1_CUDA(cudaMemcpy(pl->d_maps, maps.data(), maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice));
  const size_t pieces = (size_t)pl->cap * L;
  L1_CUDA(cudaMalloc(&pl->cq, (size_t)L * pl->cap * init.d_c * sizeof(float)));
  L1_CUDA(cudaMalloc(&pl->q, pieces * 2 * kL1H * kL1CI * sizeof(__nv_bfloat16)));
  L1_CUDA(cudaMalloc(&pl->wbuf, pieces * kL1H * sizeof(float)));
  L1_CUDA(cudaMalloc(&pl->chunk_pre, pieces * (size_t)std::max(init.n_chunks_max, 1) * sizeof(float)));
  if (!l1_encode(pl->encode, &pl->map_q, pl->q, pieces * 2 * kL1H, 2 * kL1H, msg)) { delete pl; return -2; }
  pl->smem = sizeof(L1Smem) + 1024;
  L1_CUDA(cudaFuncSetAttribute(l1_score_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl->smem));
  if ((size_t)kGvSeqs * init.Dh * 2 > 200 * 1024 || (size_t)kGvSeqs * init.d_c * 4 > 200 * 1024) { *msg = "Dh / d_c too large for the staged projections"; delete pl; return -6; }
  L1_CUDA(cudaFuncSetAttribute(l1_gemv_kernel<__nv_bfloat16, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
  L1_CUDA(cudaFuncSetAttribute(l1_gemv_kernel<float, __nv_bfloat16>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
  // persistent GEMV blocks: exactly one resident wave (a second, partial wave would double the kernel's time)
  L1_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&pl->occ13, l1_gemv_kernel<__nv_bfloat16, float>, kGvWarps * 32, (size_t)kGvSeqs * init.Dh * 2));
  L1_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&pl->occ2, l1_gemv_kernel<float, __nv_bfloat16>, kGvWarps * 32, (size_t)kGvSeqs * init.d_c * 4));
  *out = pl;
  return 0;
}

void l1_destroy(L1Plan* pl) {
  if (!pl) return;
  cudaFree(pl->d_maps); cudaFree(pl->cq); cudaFree(pl->q); cudaFree(pl->wbuf); cudaFree(pl->chunk_pre);
  delete pl;
}

// h DEVICE rows of Dh (row hrows[i] belongs to sequence ids[i]); sel_idx DEVICE [n][k]
int l1_select(L1Plan* pl, const SeqDev* d_seqs, const void* h, const int* ids, const int* hrows, int n, int k, float threshold,
              int32_t* sel_idx, float* sel_score, cudaStream_t st, int* launches, std::string* msg) {
  const L1Init& in = pl->init;
  const int L = in.n_layers, Dh = in.Dh, d_c = in.d_c;
  const float logit_thr = (float)std::log((double)threshold / (1.0 - (double)threshold));
  const __nv_bfloat16* hb = reinterpret_cast<const __nv_bfloat16*>(h);
  for (int off = 0; off < n; off += pl->cap) {
    const int m = std::min(pl->cap, n - off);
    const dim3 blk(kGvWarps * 32);
    FireList hr{}, ident{};
    hr.n = ident.n = m;
    for (int i = 0; i < m; ++i) { hr.ids[i] = hrows[off + i]; ident.ids[i] = i; }
    // Eq.(1) c^Q [m][d_c] fp32 and Eq.(3) w -> piece (i, l), all layers in one launch (both read h)
    GvJobs j13{}, j2{};
    for (int l = 0; l < L; ++l) {
      float* cq = pl->cq + (size_t)l * pl->cap * d_c;
      j13.W[l] = reinterpret_cast<const __nv_bfloat16*>(in.layers[l].W_dq);
      j13.x[l] = hb; j13.out[l] = cq; j13.ldo[l] = d_c; j13.E[l] = d_c;
      j13.W[L + l] = reinterpret_cast<const __nv_bfloat16*>(in.layers[l].W_w);
      j13.x[L + l] = hb; j13.out[L + l] = pl->wbuf + (size_t)l * kL1H; j13.ldo[L + l] = (long long)L * kL1H; j13.E[L + l] = kL1H;
      // Eq.(2): q -> piece (i, l) as two bf16 terms (hi, lo)
      j2.W[l] = reinterpret_cast<const __nv_bfloat16*>(in.layers[l].W_iuq);
      j2.x[l] = cq; j2.out[l] = pl->q + (size_t)l * 2 * kL1H * kL1CI; j2.ldo[l] = (long long)L * 2 * kL1H * kL1CI; j2.E[l] = kL1H * kL1CI;
    }
    j13.n_jobs = 2 * L; j13.shared_x = 1;
    j2.n_jobs = L; j2.shared_x = 0; j2.lo_off = (long long)kL1H * kL1CI;
    const unsigned gy = (unsigned)((m + kGvSeqs - 1) / kGvSeqs);
    // persistent blocks: as many as fit on the machine at once (shared memory bounds the occupancy)
    auto blocks_x = [&](int per_sm, int rows, int z) {
      const int fit = std::max(1, pl->n_sms * std::max(1, per_sm) / (int)(gy * z));
      return (unsigned)std::max(1, std::min(fit, (rows + kGvWarps - 1) / kGvWarps));
    };
    const size_t sm13 = (size_t)kGvSeqs * Dh * 2, sm2 = (size_t)kGvSeqs * d_c * 4;
    L1_CUDA(launch_pdl(l1_gemv_kernel<__nv_bfloat16, float>, dim3(blocks_x(pl->occ13, L * (d_c + kL1H), 1), gy, 1), blk, sm13, st, j13,
                       (long long)Dh, hr, m, Dh));
    L1_CUDA(launch_pdl(l1_gemv_kernel<float, __nv_bfloat16>, dim3(blocks_x(pl->occ2, kL1H * kL1CI, L), gy, L), blk, sm2, st, j2,
                       (long long)d_c, ident, m, d_c));
    *launches += 2;
    L1ScoreParams sp{};
    sp.k_maps = pl->d_maps; sp.wbuf = pl->wbuf; sp.chunk_pre = pl->chunk_pre;
    sp.n_pieces = m * L; sp.n_chunks_max = std::max(in.n_chunks_max, 1);
    int tiles = 0;
    FireList fire{};
    fire.n = m;
    for (int i = 0; i < m; ++i) {
      const int b = ids[off + i];
      fire.ids[i] = b;
      for (int l = 0; l < L; ++l) {
        L1Piece& pc = sp.pieces[i * L + l];
        pc.n_entries = (int)in.seq_host[b].n_csa;
        pc.n_tiles = in.seq_host[b].n_chunks;
        pc.tile0 = tiles;
        pc.map_idx = b * L + l;
        tiles += pc.n_tiles;
      }
    }
    sp.total_tiles = tiles;
    if (tiles > 0) {
      const int grid = std::max(1, std::min(pl->n_sms, tiles));
      L1_CUDA(launch_pdl(l1_score_kernel, dim3(grid), dim3(kL1Threads), pl->smem, st, pl->map_q, sp));
      *launches += 1;
    }
    L1_CUDA(launch_pdl(l1_select_kernel, dim3(m), dim3(1024), 0, st, d_seqs, fire, (const float*)pl->chunk_pre, L, sp.n_chunks_max, logit_thr, k,
                       sel_idx + (size_t)off * k, sel_score ? sel_score + (size_t)off * k : (float*)nullptr));
    *launches += 1;
  }
  return 0;
}

}  // namespace lsa
