// lsa_attn_tc_small.cuh - S7/S8 for small batches (B <= 4): the latency-bound regime (BASELINE cfg 2, cfg 3).
//
// At B = 1 the attended set of a 1M-token context is 24 576 keys = 48 MiB: 7.7 us at the measured HBM peak, i.e. the
// same order as a kernel launch, a dependency flush and the merge of the split partials.  Three things differ
// from the general kernel (lsa_attn_tc_kernel.cuh), whose tcgen05 / TMA pipeline this kernel keeps:
//
// 1. Pieces are cut at HALF tiles (64 rows).  The flat list of 64-row half tiles (per sequence: HCA rows, two
//    halves per page of the current table, window rows) is cut into gridDim.x contiguous ranges, so all 148 SMs
//    pull from HBM (whole 128-row tiles allow only 96 equal shares at cfg 3).  Adjacent halves of one source are
//    merged back into a 128-row sub-tile; a lone half is a 64-row TMA box (its own tensor map) that fills the
//    first half of a stage: S^T is still one M = 128 MMA per k-step (rows 64.. are stale shared memory, masked by
//    the softmax threads), PV and the row sums run 4 instead of 8 k-steps.
//
// 2. Nothing the LIBRARY wrote for the previous step is read before the K/V stream starts: the per-sequence shape
//    arrives BY VALUE from the host's deterministic mirrors (SmSeq), the split partials alternate between two
//    workspace buffers, and the one true cross-launch dependency - the window row the previous step appended
//     - is ordered by a release / acquire counter in the sequence record (SeqDev::app_epoch).  Launched with
//    programmatic stream serialization, its CTAs start on an SM the moment the previous step's CTA leaves it and
//    fill their 128 KiB stage ring with K rows while that step's partials are still being merged.  What remains is
//    the CALLER's data: q, k_new and v_new are whatever the stream produced last, so the producer thread (before
//    the Q tile) and the appending threads execute griddepcontrol.wait first (wait_inputs = 1, the default).
//    A caller whose inputs do not depend on the previous step's output (lsa_config.step_overlap) drops that wait
//    too: the whole kernel then runs underneath the previous step's merge.
//
// 3. The merge (combine_small_kernel) needs 4 KiB of shared memory and < 64 registers per thread, so its blocks are
//    co-resident with attention CTAs (which leave ~12 KiB of an SM's shared memory free): it waits for ITS
//    attention grid with griddepcontrol.wait and runs underneath the next step's attention kernel instead of
//    between the two.  A counter the combine blocks bump on exit (comb_ctr) protects the buffer reuse two launches
//    later and orders consecutive combines (they write the same records and, typically, the same `out`).
#pragma once
#include <type_traits>

#include "lsa_attn_tc_defs.cuh"

namespace lsa {

constexpr int kSmB = 4;                     // sequences per context on this path
constexpr int kSmHalf = 64;                 // rows per half tile: the granularity of the split

// per-sequence shape as of this launch (host mirror)
struct SmSeq {
  int n_hca;
  int cur;                  // table buffer attended by this launch
  int n_cur;                // entries of that table, or -1: read SeqDev::n_tbl[cur] (written at the last trigger)
  int w_len;                // attended ring rows, this launch's append included
  int app_slot;             // ring slot this launch writes k_new / v_new to, or -1
  unsigned int app_count;   // appends enqueued before this launch: SeqDev::app_epoch reaches it before ring rows are read
  long long n_csa;
};

struct SmParams {
  SmSeq seq[kSmB];
  SeqDev* seqs;                  // device records: n_tbl (read), win_k / win_v (append), app_epoch
  const int* tbl_chunk;
  const int* tbl_page;
  const CUtensorMap* seq_maps;   // [B][8]: (hca_k, hca_v, win_k, win_v) with 128-row boxes, then with 64-row boxes
  int B, k, n_attn;
  float scale_log2;
  uint2* part_o;                 // the workspace buffer of this launch (same layout as TcParams)
  float* part_s;
  float* part_m;
  float* part_l;
  int2* piece_info;
  const unsigned int* comb_ctr;  // combine blocks finished so far on this workspace
  unsigned int comb_need;        // value it must have reached before this launch may overwrite its buffer
  const __nv_bfloat16* k_new;    // [B][D] or null
  const __nv_bfloat16* v_new;
  int wait_inputs;               // 1: griddepcontrol.wait before q / k_new / v_new are read
  unsigned long long* ktime;     // profiling only, see TcParams
};

struct SmSmem {
  alignas(1024) unsigned char q[65536];                       // [8 d-blocks][64 heads][128 B], SW128
  alignas(1024) unsigned char stage[kTcStages][kTcStageBytes];// [2 d-blocks][rows][128 B], SW128; rows = 128 or 64
  alignas(1024) unsigned char p[16384];                       // [128 keys][64 heads] bf16, SW128 (MN-major B)
  alignas(1024) unsigned char ones[4096];                     // 128 x 16 bf16 ones, no swizzle
  alignas(16) float wmax[2][32][4];
  alignas(16) float mtile[2][4][32];
  SmSeq seq[kSmB];
  int hh_hca[kSmB], hh_pg[kSmB];                              // half tiles of the HCA rows / of the pages
  int gpre[kSmB + 1];                                         // prefix of half tiles per sequence
  uint64_t full[kTcStages], empty[kTcStages];
  uint64_t q_full, q_empty, s_full[2], s_empty[2], p_full, pv_done, o_full[4], o_empty, setup, app_done;
  uint32_t tmem_base;
};

__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_u32(unsigned int* p, unsigned int v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void red_release_add_u32(unsigned int* p, unsigned int v) {
  asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// Bounded wait for a monotonically increasing counter (wrap-safe); normally satisfied by the first load.
static __device__ __noinline__ void wait_counter_slow(const unsigned int* p, unsigned int need, int tag) {
  const long long t0 = clock64();
  while ((int)(ld_acquire_u32(p) - need) < 0) {
    if (clock64() - t0 > 4000000000ll) {
      printf("lsa tc kernel: counter timeout tag=%d block=%d need=%u have=%u\n", tag, blockIdx.x, need, ld_acquire_u32(p));
      __trap();
    }
  }
}
__device__ __forceinline__ void wait_counter(const unsigned int* p, unsigned int need, int tag) {
  if ((int)(ld_acquire_u32(p) - need) >= 0) return;
  wait_counter_slow(p, need, tag);
}

// One unit of the pipeline: `rows` (64 or 128) consecutive rows of one source.
struct SubTile {
  int b;
  int kind;        // 0 = HCA rows, 1 = page of the current table, 2 = window rows
  int t;           // kind 1: position in the table
  int row0;        // first row inside the source (inside the page for kind 1)
  int rows;
  bool first, last;   // of this CTA's piece of sequence b
};

// Iterates the sub-tiles of this CTA's share [f0, f1) of the flat half-tile list; every role runs its own copy.
struct SubCursor {
  const SmSmem& sm;
  int B, f, f1, b, prev_b;
  __device__ SubCursor(const SmSmem& sm_, int B_, int cta, int n_cta) : sm(sm_), B(B_) {
    const unsigned T = (unsigned)sm_.gpre[B_];
    f = (int)((unsigned)cta * T / (unsigned)n_cta);
    f1 = (int)((unsigned)(cta + 1) * T / (unsigned)n_cta);
    b = 0; prev_b = -1;
  }
  __device__ bool next(SubTile& s) {
    if (f >= f1) return false;
    while (sm.gpre[b + 1] <= f) ++b;
    const int u = f - sm.gpre[b];
    const int end_b = min(f1, sm.gpre[b + 1]) - sm.gpre[b];
    const int hca = sm.hh_hca[b], pg = sm.hh_pg[b];
    int n;
    if (u < hca) {
      n = min(2, min(end_b, hca) - u);
      s.kind = 0; s.t = 0; s.row0 = u * kSmHalf;
    } else if (u < hca + pg) {
      const int up = u - hca;
      n = ((up & 1) == 0 && u + 1 < end_b) ? 2 : 1;           // both halves of one page
      s.kind = 1; s.t = up >> 1; s.row0 = (up & 1) * kSmHalf;
    } else {
      const int uw = u - hca - pg;
      n = min(2, end_b - u);
      s.kind = 2; s.t = 0; s.row0 = uw * kSmHalf;
    }
    s.b = b; s.rows = n * kSmHalf;
    s.first = (b != prev_b);
    prev_b = b;
    f += n;
    s.last = (f >= f1) || (f >= sm.gpre[b + 1]);
    return true;
  }
};

// attended rows of a sub-tile (the rest of its rows is masked)
__device__ __forceinline__ int sub_valid(const SmParams& p, const SmSmem& sm, const SubTile& s) {
  const SmSeq& q = sm.seq[s.b];
  if (s.kind == 0) return min(s.rows, q.n_hca - s.row0);
  if (s.kind == 2) return min(s.rows, q.w_len - s.row0);
  const int chunk = p.tbl_chunk[((size_t)s.b * 2 + q.cur) * p.k + s.t];
  const int vc = (int)max(0ll, min((long long)kTcC, q.n_csa - (long long)chunk * kTcC));
  return max(0, min(s.rows, vc - s.row0));
}

__global__ void __launch_bounds__(kTcThreads, 1)
attn_tc_small_kernel(const __grid_constant__ CUtensorMap map_pool, const __grid_constant__ CUtensorMap map_pool64,
                     const __grid_constant__ CUtensorMap map_q, const __grid_constant__ SmParams p) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  SmSmem& sm = *reinterpret_cast<SmSmem*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int cta = blockIdx.x, n_cta = p.n_attn;

  if (tid == 0) {
    for (int i = 0; i < kTcStages; ++i) { mbar_init(&sm.full[i], 1); mbar_init(&sm.empty[i], 1); }
    mbar_init(&sm.q_full, 1); mbar_init(&sm.q_empty, 1);
    for (int i = 0; i < 2; ++i) { mbar_init(&sm.s_full[i], 1); mbar_init(&sm.s_empty[i], kTcSoftmaxWarps); }
    mbar_init(&sm.p_full, kTcSoftmaxWarps); mbar_init(&sm.pv_done, 1); mbar_init(&sm.o_empty, kTcSoftmaxWarps);
    for (int i = 0; i < 4; ++i) mbar_init(&sm.o_full[i], 1);
    mbar_init(&sm.setup, kTcThreads / 32);
    mbar_init(&sm.app_done, kTcSoftmaxWarps);
    fence_mbar_init();
    prefetch_tmap(&map_pool);
    prefetch_tmap(&map_pool64);
    prefetch_tmap(&map_q);
  }
  __syncthreads();
  griddep_launch_dependents();    // the combine blocks of this step (and, behind them, the next step's CTAs) may be placed
  if (p.ktime && tid == 0) atomicMin(p.ktime, gtime());
  if (warp == 0) {
    // per-sequence shape -> half tiles per segment and their prefix (B <= 4); ring rows appended by earlier
    // launches are visible once app_epoch has caught up with the host's count
    int g = 0;
    if (lane < p.B) {
      SmSeq q = p.seq[lane];
      if (q.n_cur < 0) q.n_cur = __ldcg(&p.seqs[lane].n_tbl[q.cur]);
      wait_counter(&p.seqs[lane].app_epoch, q.app_count, 50);
      sm.seq[lane] = q;
      const int hca = (q.n_hca + kSmHalf - 1) / kSmHalf, pg = 2 * q.n_cur, win = (q.w_len + kSmHalf - 1) / kSmHalf;
      sm.hh_hca[lane] = hca; sm.hh_pg[lane] = pg;
      g = hca + pg + win;
    }
    int incl = g;
#pragma unroll
    for (int o = 1; o < kSmB; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += t;
    }
    if (lane < p.B) sm.gpre[lane + 1] = incl;
    if (lane == 0) sm.gpre[0] = 0;
    __syncwarp();
    if (lane == 0) mbar_arrive(&sm.setup);
  } else if (warp == 1) {
    tmem_alloc(&sm.tmem_base, 512);
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive(&sm.setup);
  } else {
    for (int i = tid - 64; i < 2048; i += kTcThreads - 64) reinterpret_cast<uint16_t*>(sm.ones)[i] = 0x3f80;   // bf16 1.0
    fence_proxy_async_smem();
    // the partials of two launches ago (same buffer) have been merged
    if (tid == 64) wait_counter(p.comb_ctr, p.comb_need, 51);
    __syncwarp();
    if (lane == 0) mbar_arrive(&sm.setup);
  }

  if (warp == 0) {
    // =========================== TMA producer ===========================
    if (elect_one()) {
      fence_proxy_async_all();                            // ring rows written by other CTAs' generic stores -> TMA reads
      SubCursor cur(sm, p.B, cta, n_cta);
      SubTile s, nx;
      uint32_t ring = 0;
      int item = 0;
      bool app_seen = false, waited = false;
      auto src_of = [&](const SubTile& t, const CUtensorMap*& mk, const CUtensorMap*& mv, int& rk, int& rv) {
        const int big = t.rows == kTcTile ? 0 : 4;
        if (t.kind == 1) {
          const int page = p.tbl_page[((size_t)t.b * 2 + sm.seq[t.b].cur) * p.k + t.t];
          mk = mv = (t.rows == kTcTile ? &map_pool : &map_pool64);
          rk = page * (2 * kTcC) + t.row0; rv = rk + kTcC;
        } else {
          mk = p.seq_maps + t.b * 8 + big + (t.kind == 0 ? 0 : 2);
          mv = mk + 1;
          rk = rv = t.row0;
        }
      };
      // the sub-tile holding this launch's new ring row is loaded only after the softmax warps have written it;
      // the row is then published for the launches that follow
      auto app_gate = [&](const SubTile& t) {
        const SmSeq& q = sm.seq[t.b];
        if (t.kind == 2 && p.k_new && q.app_slot >= t.row0 && q.app_slot < t.row0 + t.rows) {
          if (!app_seen) { mbar_wait(&sm.app_done, 0, 12); app_seen = true; }   // every row of this CTA is written by then
          st_release_u32(&p.seqs[t.b].app_epoch, q.app_count + 1u);
          fence_proxy_async_all();
        }
      };
      auto issue4 = [&](const CUtensorMap* m, int row, int rows) {
#pragma unroll 1
        for (int s4 = 0; s4 < 4; ++s4) {
          const int st = ring % kTcStages;
          mbar_wait(&sm.empty[st], ((ring / kTcStages) & 1) ^ 1, 11);
          mbar_arrive_expect_tx(&sm.full[st], (uint32_t)rows * 256u);
          tma_load_3d(sm.stage[st], m, 0, row, s4 * 2, &sm.full[st]);
          ++ring;
        }
      };
      bool have = cur.next(s);
      while (have) {
        const CUtensorMap *mk, *mv;
        int rk, rv;
        src_of(s, mk, mv, rk, rv);
        if (s.first) {
          app_gate(s);
          issue4(mk, rk, s.rows);                          // K of the piece's first sub-tile: in flight before Q is known
          if (item > 0) mbar_wait(&sm.q_empty, (item - 1) & 1, 10);
          if (p.wait_inputs && !waited) { griddep_wait(); waited = true; }   // q is the caller's: whatever the stream ran last
          mbar_arrive_expect_tx(&sm.q_full, 65536);
          tma_load_3d(sm.q, &map_q, 0, s.b * kTcH, 0, &sm.q_full);
        }
        have = cur.next(nx);
        if (!s.last) {                                     // K runs one sub-tile ahead of V inside a piece
          const CUtensorMap *nk, *nv;
          int nrk, nrv;
          src_of(nx, nk, nv, nrk, nrv);
          app_gate(nx);
          issue4(nk, nrk, nx.rows);
        }
        issue4(mv, rv, s.rows);
        if (s.last) ++item;
        s = nx;
      }
    }
  } else if (warp == 1) {
    // =========================== MMA issuer ===========================
    if (elect_one()) {
      constexpr uint32_t id_s = make_idesc_bf16(128, 64, 0, 0);    // A = K tile (K-major),  B = Q   (K-major)
      constexpr uint32_t id_pv = make_idesc_bf16(128, 64, 1, 1);   // A = V tile (MN-major), B = P^T (MN-major)
      constexpr uint32_t id_l = make_idesc_bf16(128, 64, 0, 1);    // A = ones   (K-major),  B = P^T (MN-major)
      mbar_wait(&sm.setup, 0, 19);
      tc_fence_after();
      const uint32_t tmem = sm.tmem_base;
      const uint32_t tS = tmem, tO = tmem + 128, tL = tmem + 384;
      const uint64_t dk0 = make_sdesc(smem_u32(sm.stage[0]), 16, 1024, kLayoutSw128);
      const uint64_t dv128 = make_sdesc(smem_u32(sm.stage[0]), 16384, 1024, kLayoutSw128);   // d-block stride = rows * 128 B
      const uint64_t dv64 = make_sdesc(smem_u32(sm.stage[0]), 8192, 1024, kLayoutSw128);
      const uint64_t dq0 = make_sdesc(smem_u32(sm.q), 16, 1024, kLayoutSw128);
      const uint64_t dp0 = make_sdesc(smem_u32(sm.p), 16384, 1024, kLayoutSw128);
      const uint64_t ones_desc = make_sdesc(smem_u32(sm.ones), 128, 256, kLayoutNone);
      SubCursor cur(sm, p.B, cta, n_cta);
      SubTile s, nx;
      uint32_t ring = 0, n_s = 0, n_pv = 0;
      int item = 0;
      // S^T(sub-tile n_s) = K Q^T into S buffer n_s & 1.  A 64-row sub-tile still runs M = 128: rows 64.. of the
      // stage are stale and the softmax threads mask them.
      auto issue_s = [&](int rows, bool last_of_piece) {
        const int buf = n_s & 1;
        const uint64_t dbs = (uint64_t)((rows * 128) >> 4);         // second d-block of a stage
        mbar_wait(&sm.s_empty[buf], ((n_s >> 1) & 1) ^ 1, 21);
        tc_fence_after();
#pragma unroll 1
        for (int s4 = 0; s4 < 4; ++s4) {
          const int st = ring % kTcStages;
          mbar_wait(&sm.full[st], (ring / kTcStages) & 1, 22);
          tc_fence_after();
          const uint64_t a0 = dk0 + (uint64_t)(st * (kTcStageBytes >> 4));
          const uint64_t b0 = dq0 + (uint64_t)(s4 * (16384 >> 4));
#pragma unroll
          for (int ks = 0; ks < 8; ++ks) {
            const uint64_t a = a0 + (ks >> 2 ? dbs : 0ull) + (uint64_t)(((ks & 3) * 32) >> 4);
            const uint64_t bq = b0 + (uint64_t)(((ks >> 2) * 8192 + (ks & 3) * 32) >> 4);
            umma_bf16(tS + buf * 64, a, bq, id_s, (s4 | ks) != 0);
          }
          umma_commit(&sm.empty[st]);
          ++ring;
        }
        umma_commit(&sm.s_full[buf]);
        if (last_of_piece) umma_commit(&sm.q_empty);
        ++n_s;
      };
      // O^T (+)= V^T P^T ; L (+)= 1 P^T over rows / 16 k-steps
      auto issue_pv = [&](auto nks_c, bool first_of_piece, bool last_of_piece) {
        constexpr int kKs = decltype(nks_c)::value;
        const uint64_t dv0 = kKs == 8 ? dv128 : dv64;
        mbar_wait(&sm.p_full, n_pv & 1, 23);
        tc_fence_after();
        if (first_of_piece && item > 0) {                 // the previous piece's epilogue has drained O and L
          mbar_wait(&sm.o_empty, (item - 1) & 1, 24);
          tc_fence_after();
        }
        const uint32_t acc = first_of_piece ? 0u : 1u;
#pragma unroll
        for (int ks = 0; ks < kKs; ++ks) umma_bf16(tL, ones_desc, dp0 + (uint64_t)((ks * 2048) >> 4), id_l, acc | (ks != 0));
#pragma unroll 1
        for (int m = 0; m < 4; ++m) {
          const int st = ring % kTcStages;
          mbar_wait(&sm.full[st], (ring / kTcStages) & 1, 25);
          tc_fence_after();
          const uint64_t a0 = dv0 + (uint64_t)(st * (kTcStageBytes >> 4));
#pragma unroll
          for (int ks = 0; ks < kKs; ++ks)
            umma_bf16(tO + m * 64, a0 + (uint64_t)((ks * 2048) >> 4), dp0 + (uint64_t)((ks * 2048) >> 4), id_pv, acc | (ks != 0));
          umma_commit(&sm.empty[st]);
          if (last_of_piece) umma_commit(&sm.o_full[m]);
          ++ring;
        }
        umma_commit(&sm.pv_done);
        ++n_pv;
      };
      bool have = cur.next(s);
      while (have) {
        if (s.first) {
          mbar_wait(&sm.q_full, item & 1, 20);
          tc_fence_after();
          issue_s(s.rows, s.last);
        }
        have = cur.next(nx);
        if (!s.last) issue_s(nx.rows, nx.last);
        if (s.rows == kTcTile) issue_pv(std::integral_constant<int, 8>{}, s.first, s.last);
        else issue_pv(std::integral_constant<int, 4>{}, s.first, s.last);
        if (s.last) ++item;
        s = nx;
      }
    }
  } else {
    // =========================== softmax + epilogue (8 warps) ===========================
    const int q4 = warp & 3;                              // TMEM lane quarter this warp may access
    const int hh = (warp - 2) >> 2;                       // half of the heads owned by this warp
    const uint32_t lane_addr = (uint32_t)(q4 * 32) << 16;
    const int key = q4 * 32 + lane;                       // key row of the sub-tile owned by this thread
    mbar_wait(&sm.setup, 0, 29);
    tc_fence_after();
    const uint32_t tmem = sm.tmem_base;
    const uint32_t tS = tmem, tO = tmem + 128, tL = tmem + 384;
    if (p.k_new) {
      // window append ("decoded tokens stay resident"; DESIGN R6): the CTA that owns the sub-tile holding
      // ring slot w_head of a sequence writes k_new / v_new there before its producer loads that sub-tile
      SubCursor pc(sm, p.B, cta, n_cta);
      SubTile a;
      const int t = tid - 64;
      bool waited = false;
      while (pc.next(a)) {
        const SmSeq& q = sm.seq[a.b];
        if (a.kind == 2 && q.app_slot >= a.row0 && q.app_slot < a.row0 + a.rows && t < 128) {
          if (p.wait_inputs && !waited) { griddep_wait(); waited = true; }   // k_new / v_new are the caller's
          const SeqDev& sd = p.seqs[a.b];
          const uint4* src = reinterpret_cast<const uint4*>((t < 64 ? p.k_new : p.v_new) + (size_t)a.b * kTcD) + (t & 63);
          uint4* dst = reinterpret_cast<uint4*>(reinterpret_cast<__nv_bfloat16*>(t < 64 ? sd.win_k : sd.win_v) + (size_t)q.app_slot * kTcD) + (t & 63);
          *dst = *src;
        }
      }
      fence_proxy_async_all();                            // generic-proxy stores -> later TMA (async proxy) reads
      __syncwarp();
      if (lane == 0) mbar_arrive(&sm.app_done);
    }
    SubCursor cur(sm, p.B, cta, n_cta);
    SubTile s;
    uint32_t tcount = 0, piece = 0;
    int b_first = -1, b_last = -1;
    float m_run[32];
    auto tile_max = [&](const float (&x)[32], float (&mt)[32]) {
      float mine = -INFINITY;
#pragma unroll
      for (int h = 0; h < 32; ++h) {
        const float r = redux_max_f32(x[h]);
        if (lane == h) mine = r;
      }
      sm.wmax[hh][lane][q4] = mine;
      named_bar_sync(1, 32 * kTcSoftmaxWarps);
      const float4 w = *reinterpret_cast<const float4*>(sm.wmax[hh][lane]);
      sm.mtile[hh][q4][lane] = fmaxf(fmaxf(w.x, w.y), fmaxf(w.z, w.w));
      __syncwarp();
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const float4 t4 = *reinterpret_cast<const float4*>(&sm.mtile[hh][q4][4 * j]);
        mt[4 * j] = t4.x; mt[4 * j + 1] = t4.y; mt[4 * j + 2] = t4.z; mt[4 * j + 3] = t4.w;
      }
      __syncwarp();
    };
    bool have = cur.next(s);
    int nv_next = have ? sub_valid(p, sm, s) : 0;
    while (have) {
      const int b = s.b;
      if (s.first) {
        if (b_first < 0) b_first = b;
        // sequences without keys between two pieces of this CTA get an empty partial (weight 0 in S8)
        for (int e = b_last + 1; b_last >= 0 && e < b; ++e)
          if (tid < 64 + kTcH) { p.part_m[((size_t)cta + e) * kTcH + tid - 64] = -INFINITY; p.part_l[((size_t)cta + e) * kTcH + tid - 64] = 0.f; }
        b_last = b;
      }
      const bool first = s.first, last = s.last;
      const int buf = tcount & 1;
      const bool valid = key < nv_next;
      have = cur.next(s);                                 // global look-ups of the next sub-tile overlap the wait below
      if (have) nv_next = sub_valid(p, sm, s);
      float x[32];
      mbar_wait(&sm.s_full[buf], (tcount >> 1) & 1, 30);
      tc_fence_after();
      tmem_ld32(tS + buf * 64 + hh * 32 + lane_addr, reinterpret_cast<uint32_t*>(x));
      tmem_wait_ld();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&sm.s_empty[buf]);
      // masked, scaled logits (log2 domain); a select, not arithmetic: masked rows may hold anything
#pragma unroll
      for (int h = 0; h < 32; ++h) x[h] = valid ? x[h] * p.scale_log2 : -INFINITY;
      bool rescale = false;
      float f[32];
      if (first) {
        tile_max(x, m_run);
        // a first sub-tile without any attended key (partial last chunk) leaves -inf: keep the maximum finite so
        // that 2^(x - m) is 0, not NaN; the first real logit then takes the rescale path
#pragma unroll
        for (int h = 0; h < 32; ++h) m_run[h] = fmaxf(m_run[h], -1e30f);
      } else {
        bool over = false;
#pragma unroll
        for (int h = 0; h < 32; ++h) over |= (x[h] > m_run[h] + kRescaleThreshold);
        rescale = named_bar_red_or(1, 32 * kTcSoftmaxWarps, over);
        if (rescale) {                      // rare: adopt the new maximum, O^T and L are rescaled below
          float mt[32];
          tile_max(x, mt);
#pragma unroll
          for (int h = 0; h < 32; ++h) {
            const float mn = fmaxf(m_run[h], mt[h]);
            f[h] = ex2_approx(m_run[h] - mn);
            m_run[h] = mn;
          }
        }
      }
      uint32_t pw[16];
#pragma unroll
      for (int e = 0; e < 16; ++e) pw[e] = pack_bf16x2(ex2_approx(x[2 * e] - m_run[2 * e]), ex2_approx(x[2 * e + 1] - m_run[2 * e + 1]));
      // the P tile buffer (and O) are free once the previous sub-tile's PV MMAs have completed
      if (tcount > 0) {
        mbar_wait(&sm.pv_done, (tcount - 1) & 1, 31);
        tc_fence_after();
      }
      if (rescale) {
#pragma unroll 1
        for (int c = 0; c < 5; ++c) {             // 4 x 64 O columns + 64 L columns; this warp's 32 of each
          uint32_t vreg[32];
          const uint32_t addr = tO + c * 64 + hh * 32 + lane_addr;
          tmem_ld32(addr, vreg);
          tmem_wait_ld();
#pragma unroll
          for (int j = 0; j < 32; ++j) vreg[j] = __float_as_uint(__uint_as_float(vreg[j]) * f[j]);
          tmem_st32(addr, vreg);
        }
        tmem_wait_st();
      }
      {
        unsigned char* prow = sm.p + key * 128;
#pragma unroll
        for (int j = 0; j < 4; ++j)
          *reinterpret_cast<uint4*>(prow + (((hh * 4 + j) ^ (key & 7)) << 4)) = make_uint4(pw[4 * j], pw[4 * j + 1], pw[4 * j + 2], pw[4 * j + 3]);
      }
      fence_proxy_async_smem();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&sm.p_full);
      ++tcount;
      if (!last) continue;
      // ---- epilogue: O^T, L, m -> partial slot (cta + b) ----
      const size_t slot = (size_t)cta + b;
      uint2* po = p.part_o + slot * (kTcH * kTcD / 4) + (size_t)hh * (8 * 128) + key;
#pragma unroll 1
      for (int m = 0; m < 4; ++m) {               // d = m * 128 + key
        uint32_t vreg[32];
        mbar_wait(&sm.o_full[m], piece & 1, 32);
        tc_fence_after();
        tmem_ld32(tO + m * 64 + hh * 32 + lane_addr, vreg);
        tmem_wait_ld();
        float amax = 0.f;
#pragma unroll
        for (int j = 0; j < 32; ++j) amax = fmaxf(amax, fabsf(__uint_as_float(vreg[j])));
        float inv;
        const float sc = part_scale(redux_max_f32(amax), &inv);   // one scale per warp: 32 d-rows x 32 heads
        if (lane == 0) p.part_s[part_scale_idx(slot, m, hh, q4)] = inv;
#pragma unroll
        for (int g = 0; g < 8; ++g)
          po[(size_t)m * (2 * 8 * 128) + g * 128] =
              make_uint2(pack_f16x2(__uint_as_float(vreg[4 * g]) * sc, __uint_as_float(vreg[4 * g + 1]) * sc),
                         pack_f16x2(__uint_as_float(vreg[4 * g + 2]) * sc, __uint_as_float(vreg[4 * g + 3]) * sc));
      }
      if (q4 == 0) {                              // every lane of L holds the same row sums: lane 0 writes them
        uint32_t vreg[32];
        tmem_ld32(tL + hh * 32 + lane_addr, vreg);
        tmem_wait_ld();
        if (lane == 0) {
#pragma unroll
          for (int j = 0; j < 32; ++j) {
            p.part_l[slot * kTcH + hh * 32 + j] = __uint_as_float(vreg[j]);
            p.part_m[slot * kTcH + hh * 32 + j] = m_run[j] <= -1e30f ? -INFINITY : m_run[j];   // no attended key: S8 skips the slot
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&sm.o_empty);
      ++piece;
    }
    if (tid == 64) p.piece_info[cta] = make_int2(b_first < 0 ? 0 : b_first, b_first < 0 ? 0 : b_last - b_first + 1);
  }
  // ---- teardown ----
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(sm.tmem_base, 512);
  }
  if (p.ktime && tid == 0) atomicMax(p.ktime + 1, gtime());
}

// ---- S8 under the next step's attention ---------------------------------------------------------------------------
// grid (128, B) x 128 threads; block = (m, hh, g, dh) = 512 contiguous bytes (64 d x 4 heads fp16) of every slot, as in
// combine_tc_kernel.  A warp reads a whole 512-byte row per load (16 bytes per lane = 2 d x 4 heads), the four warps take
// slots w, w+4, ...; weights and scales go through 4 KiB of shared memory.
constexpr int kCombSmThreads = 128;
constexpr int kCombSmUnroll = 8;

struct SmCombParams {
  const uint2* part_o;
  const float* part_s;
  const float* part_m;
  const float* part_l;
  const int2* piece_info;
  unsigned int* comb_ctr;
  unsigned int comb_prev;        // blocks of every earlier combine on this workspace: they have finished before this one writes
  SeqDev* seqs_mut;              // S6 / window append folded into the attention launch: the records catch up here
  unsigned int swap;             // bit b: sequence b's staged table became current in this step
  int append;                    // 1: the step appended a ring row
  int W;
};

__global__ void __launch_bounds__(kCombSmThreads)
combine_small_kernel(const __grid_constant__ SmCombParams p, int n_cta, __nv_bfloat16* __restrict__ out, float* __restrict__ lse) {
  __shared__ float4 w_s[256];                     // weights by CTA; reused for the cross-warp sum at the end
  __shared__ float2 sc_s[256];
  __shared__ float4 red_f[4];
  float4 (*acc_s)[32][2] = reinterpret_cast<float4 (*)[32][2]>(w_s);   // [4 warps][32 lanes][2]
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int dh = blockIdx.x & 1, g = (blockIdx.x >> 1) & 7, hh = (blockIdx.x >> 4) & 1, m = blockIdx.x >> 5, b = blockIdx.y;
  const int h0 = hh * 32 + g * 4;
  griddep_launch_dependents();                    // the next step's attention CTAs may be placed as SMs free up
  griddep_wait();                                 // this step's partials and piece_info are final from here on
  if (tid == 0) wait_counter(p.comb_ctr, p.comb_prev, 52);   // every earlier combine has finished (records, `out`)
  __syncthreads();
  if (blockIdx.x == 0 && tid == 0) {              // the per-sequence record catches up with the launch's view
    SeqDev& s = p.seqs_mut[b];
    if (((p.swap >> b) & 1u) && s.pending) { s.cur_buf = 1 - s.cur_buf; s.pending = 0; }
    if (p.append) {
      const int slot = s.w_head;
      s.w_head = (slot + 1 == p.W) ? 0 : slot + 1;
      s.w_len = min(p.W, s.w_len + 1);
    }
  }
  // thread c (and c + 128) looks at CTA c: did it write a partial for sequence b?  (n_cta <= 256)
  float4 mi[2], li[2];
  float2 s2[2];
  bool act[2];
  float4 mmax = make_float4(-INFINITY, -INFINITY, -INFINITY, -INFINITY);
#pragma unroll
  for (int r = 0; r < 2; ++r) {
    const int c = tid + r * kCombSmThreads;
    mi[r] = make_float4(-INFINITY, -INFINITY, -INFINITY, -INFINITY);
    li[r] = make_float4(0.f, 0.f, 0.f, 0.f);
    s2[r] = make_float2(0.f, 0.f);
    act[r] = false;
    if (c < n_cta) {
      const size_t slot = (size_t)c + b;
      const int2 info = __ldcg(p.piece_info + c);
      const float4 m4 = __ldcg(reinterpret_cast<const float4*>(p.part_m + slot * kTcH + h0));
      const float4 l4 = __ldcg(reinterpret_cast<const float4*>(p.part_l + slot * kTcH + h0));
      s2[r] = __ldcg(reinterpret_cast<const float2*>(p.part_s + part_scale_idx(slot, m, hh, dh * 2)));
      // a piece without valid keys (m = -inf for every head) wrote no O: its slot is skipped like an inactive one
      act[r] = info.x <= b && b < info.x + info.y && m4.x != -INFINITY;
      if (act[r]) { mi[r] = m4; li[r] = l4; }
    }
    mmax.x = fmaxf(mmax.x, mi[r].x); mmax.y = fmaxf(mmax.y, mi[r].y); mmax.z = fmaxf(mmax.z, mi[r].z); mmax.w = fmaxf(mmax.w, mi[r].w);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    mmax.x = fmaxf(mmax.x, __shfl_xor_sync(0xffffffffu, mmax.x, o));
    mmax.y = fmaxf(mmax.y, __shfl_xor_sync(0xffffffffu, mmax.y, o));
    mmax.z = fmaxf(mmax.z, __shfl_xor_sync(0xffffffffu, mmax.z, o));
    mmax.w = fmaxf(mmax.w, __shfl_xor_sync(0xffffffffu, mmax.w, o));
  }
  if (lane == 0) red_f[warp] = mmax;
  __syncthreads();
  float4 m_star = red_f[0];
#pragma unroll
  for (int w = 1; w < 4; ++w) {
    const float4 r = red_f[w];
    m_star.x = fmaxf(m_star.x, r.x); m_star.y = fmaxf(m_star.y, r.y); m_star.z = fmaxf(m_star.z, r.z); m_star.w = fmaxf(m_star.w, r.w);
  }
  float4 lsum = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
  for (int r = 0; r < 2; ++r) {
    const int c = tid + r * kCombSmThreads;
    float4 wi = make_float4(0.f, 0.f, 0.f, 0.f);
    if (act[r]) {
      wi.x = mi[r].x == -INFINITY ? 0.f : exp2f(mi[r].x - m_star.x);
      wi.y = mi[r].y == -INFINITY ? 0.f : exp2f(mi[r].y - m_star.y);
      wi.z = mi[r].z == -INFINITY ? 0.f : exp2f(mi[r].z - m_star.z);
      wi.w = mi[r].w == -INFINITY ? 0.f : exp2f(mi[r].w - m_star.w);
    }
    // an inactive slot keeps scale 0: its (possibly stale) data is multiplied by 0 weights below only if finite,
    // so it is skipped by the scale test instead
    if (c < 256) { w_s[c] = wi; sc_s[c] = act[r] ? s2[r] : make_float2(0.f, 0.f); }
    lsum.x += wi.x * li[r].x; lsum.y += wi.y * li[r].y; lsum.z += wi.z * li[r].z; lsum.w += wi.w * li[r].w;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    lsum.x += __shfl_xor_sync(0xffffffffu, lsum.x, o);
    lsum.y += __shfl_xor_sync(0xffffffffu, lsum.y, o);
    lsum.z += __shfl_xor_sync(0xffffffffu, lsum.z, o);
    lsum.w += __shfl_xor_sync(0xffffffffu, lsum.w, o);
  }
  __syncthreads();                                // red_f is reused; w_s / sc_s are complete
  if (lane == 0) red_f[warp] = lsum;
  __syncthreads();
  float4 l_star = red_f[0];
#pragma unroll
  for (int w = 1; w < 4; ++w) {
    const float4 r = red_f[w];
    l_star.x += r.x; l_star.y += r.y; l_star.z += r.z; l_star.w += r.w;
  }
  // ---- weighted sum: lane = d pair (dh*64 + 2*lane, +1) x 4 heads; warp w takes slots w, w+4, ... ----
  const uint4* rows = reinterpret_cast<const uint4*>(p.part_o) + ((((size_t)m * 2 + hh) * 8 + g) * 2 + dh) * 32 + lane;
  constexpr size_t kSlot16 = (size_t)kTcH * kTcD * 2 / 16;          // 16-byte units per slot
  float a0[4] = {0.f, 0.f, 0.f, 0.f}, a1[4] = {0.f, 0.f, 0.f, 0.f};
  const bool hi = lane >= 16;                                       // lane quarter of this d pair (scale block)
  for (int c0 = warp; c0 < n_cta; c0 += 4 * kCombSmUnroll) {
    uint4 v[kCombSmUnroll];
#pragma unroll
    for (int j = 0; j < kCombSmUnroll; ++j) {
      const int c = c0 + 4 * j;
      const float2 sc = c < n_cta ? sc_s[c] : make_float2(0.f, 0.f);
      v[j] = (hi ? sc.y : sc.x) != 0.f ? __ldcg(rows + ((size_t)c + b) * kSlot16) : make_uint4(0u, 0u, 0u, 0u);
    }
#pragma unroll
    for (int j = 0; j < kCombSmUnroll; ++j) {
      const int c = c0 + 4 * j;
      if (c < n_cta) {
        const float2 sc2 = sc_s[c];
        const float sc = hi ? sc2.y : sc2.x;
        if (sc != 0.f) {
          const float4 w = w_s[c];
          const float2 x01 = unpack_f16x2(v[j].x), x23 = unpack_f16x2(v[j].y), y01 = unpack_f16x2(v[j].z), y23 = unpack_f16x2(v[j].w);
          a0[0] = fmaf(w.x * sc, x01.x, a0[0]); a0[1] = fmaf(w.y * sc, x01.y, a0[1]);
          a0[2] = fmaf(w.z * sc, x23.x, a0[2]); a0[3] = fmaf(w.w * sc, x23.y, a0[3]);
          a1[0] = fmaf(w.x * sc, y01.x, a1[0]); a1[1] = fmaf(w.y * sc, y01.y, a1[1]);
          a1[2] = fmaf(w.z * sc, y23.x, a1[2]); a1[3] = fmaf(w.w * sc, y23.y, a1[3]);
        }
      }
    }
  }
  __syncthreads();                                // every warp is done with w_s
  acc_s[warp][lane][0] = make_float4(a0[0], a0[1], a0[2], a0[3]);
  acc_s[warp][lane][1] = make_float4(a1[0], a1[1], a1[2], a1[3]);
  __syncthreads();
  {                                               // thread = (head e, d pair): 4 heads x 32 pairs
    const int e = tid >> 5;
    float s0 = 0.f, s1 = 0.f;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      s0 += reinterpret_cast<const float*>(&acc_s[w][lane][0])[e];
      s1 += reinterpret_cast<const float*>(&acc_s[w][lane][1])[e];
    }
    const float ls = e == 0 ? l_star.x : e == 1 ? l_star.y : e == 2 ? l_star.z : l_star.w;
    __nv_bfloat162 o2;
    o2.x = __float2bfloat16_rn(ls > 0.f ? s0 / ls : 0.f);
    o2.y = __float2bfloat16_rn(ls > 0.f ? s1 / ls : 0.f);
    *reinterpret_cast<__nv_bfloat162*>(out + ((size_t)b * kTcH + h0 + e) * kTcD + m * 128 + dh * 64 + 2 * lane) = o2;
  }
  if (lse && m == 0 && dh == 0 && tid < 4) {
    const float ls = tid == 0 ? l_star.x : tid == 1 ? l_star.y : tid == 2 ? l_star.z : l_star.w;
    const float ms = tid == 0 ? m_star.x : tid == 1 ? m_star.y : tid == 2 ? m_star.z : m_star.w;
    lse[(size_t)b * kTcH + h0 + tid] = ls > 0.f ? (ms + log2f(ls)) * 0.6931471805599453f : -INFINITY;
  }
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    red_release_add_u32(p.comb_ctr, 1u);
  }
}

}  // namespace lsa
