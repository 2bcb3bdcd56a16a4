// lsa_attn_tc_small.cuh - S7/S8 for small batches (B <= 4): the latency-bound regime (BASELINE cfg 2, cfg 3).
//
// At B = 1 the attended set of a 1M-token context is 24 576 keys = 48 MiB: 7.7 us at the measured HBM peak, i.e. the
// same order as a kernel launch, a dependency flush and the merge of the split partials.  Three things differ
// from the general kernel (lsa_attn_tc_kernel.cuh), whose tcgen05 / TMA pipeline this kernel keeps:
//
// 1. Pieces are cut at HALF tiles (64 rows).  The flat list of 64-row half tiles (per sequence: HCA rows, two
//    halves per page of the current table, window rows) is cut into gridDim.x contiguous ranges of equal length (whole
//    128-row tiles allow only 96 equal shares at cfg 3; the host picks an even length where it can).  Adjacent halves of one source are
//    merged back into a 128-row sub-tile; a lone half is a 64-row TMA box (its own tensor map) that fills the
//    first half of a stage: S^T is still one M = 128 MMA per k-step (rows 64.. are stale shared memory, masked by
//    the softmax threads), PV and the row sums run 4 instead of 8 k-steps.
//
// 2. Nothing the LIBRARY wrote for the previous step is read before the K/V stream starts: the per-sequence shape
//    arrives BY VALUE from the host's deterministic mirrors (SmSeq), the split partials rotate through three
//    workspace buffers, and the one true cross-launch dependency - the window row the previous step appended
//     - is ordered by a release / acquire counter in the sequence record (SeqDev::app_epoch).  Launched with
//    programmatic stream serialization, its CTAs start on an SM the moment the previous step's CTA leaves it and
//    fill their 128 KiB stage ring with K rows while that step's partials are still being merged.  What remains is
//    the CALLER's data: q, k_new and v_new are whatever the stream produced last, so the producer thread (before
//    the Q tile) and the appending threads execute griddepcontrol.wait first (wait_inputs = 1, the default).
//    A caller whose inputs do not depend on the previous step's output (lsa_config.step_overlap) drops that wait
//    too: the whole kernel then runs underneath the previous step's merge.
//
// 3. S8 runs inside the launch.  A second kernel in the programmatic chain must sit resident and wait for the attention
//    grid; measured, those waiting blocks pile up on the SMs the next step's CTAs need, and the host pays a second
//    launch.  Instead every CTA publishes its partials and takes an arrival number from a counter (one per workspace
//    buffer).  The launch's LAST n_mrg arrivals (32 of 48 at cfg 3) stay and merge: they wait for the stragglers among
//    themselves, request the fp16 partials of their output units by TMA, weigh and sum them (unit = 4 heads x 32 d, one
//    per warp and round).  Every earlier arrival LEAVES at once and its SM goes to the next launch's CTA.  A per-CTA
//    timeline (%globaltimer at ten points, %smid) showed why: with every CTA waiting at a barrier for the slowest and
//    then merging, a CTA spent 10 of its 26 us of residence not streaming, and the step time was SM residence / 148,
//    not bytes / bandwidth (cfg 3: 12.45 -> 10.85 us per step, 10.0 with the changes that followed).
//    A second counter (done_ctr, mergers only) orders the merges of consecutive launches (records, `out`) and protects
//    the reuse of a workspace buffer three launches later.
//    Mergers wait only for CTAs of their own launch and for mergers of EARLIER launches; every CTA of a launch has
//    started before the next launch's first CTA starts (programmatic launch), so the only CTAs that can hold an SM
//    while an unstarted CTA still needs one are that launch's own mergers - at most 32 SMs - and the waits cannot
//    starve (a launch that runs alone lets all its CTAs merge: grid <= SM count, one CTA per SM, all resident);
//    they are bounded and trap.  Contexts that run CONCURRENTLY on different streams could each hold part of the SMs
//    and wait for the rest: such contexts must share stream_compute (they then share the workspace) or be run in turn.
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
  unsigned int grow_count;  // lsa_append_compressed calls enqueued before this launch (SeqDev::grow_epoch), see grow_wait
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
  uint2* part_o;                 // the workspace buffer of this launch: O^T partials in TcParams' layout ...
  float* part_s;                 // ... but m, l and the block scales TRANSPOSED, [64 heads][n_slots] / [32 blocks][n_slots]:
  float* part_m;                 // S8 reads one head (block) of EVERY slot, which is then one coalesced line per 32 slots
  float* part_l;
  int n_slots;                   // row length of the transposed arrays
  int slot_row0;                 // first row of this launch's workspace buffer in the partials' tensor map (S8's TMA)
  int2* piece_info;
  unsigned int* arr_ctr;         // arrival counter of this launch's workspace buffer (cumulative over its launches)
  unsigned int arr_target;       // its value once every CTA of this launch has arrived
  int n_mrg;                     // the last n_mrg CTAs of the launch to arrive merge its partials (1 .. n_attn)
  unsigned int* done_ctr;        // merging CTAs that have finished, all launches of the workspace
  unsigned int done_need_buf;    // value it has reached once the launch that used this buffer last has been merged
  unsigned int done_need_prev;   // value it has reached once the previous launch has been merged
  unsigned int done_after;       // its value once this launch's last merger has finished
  unsigned int* host_flag;       // lsa_step_host: PINNED HOST word (mapped) that receives host_flag_val when the launch's
  unsigned int host_flag_val;    // last CTA leaves, i.e. when `out` is complete - the host spins on it instead of
                                 // synchronising the stream; null otherwise
  __nv_bfloat16* out;            // [B][H][D]
  float* lse;                    // [B][H] or null
  unsigned int swap;             // bit b: sequence b's staged table becomes current with this launch (records catch up here)
  int W;                         // ring capacity
  const __nv_bfloat16* k_new;    // [B][D] or null
  const __nv_bfloat16* v_new;
  int grow_wait;                 // 1: an append kernel (lsa_append_compressed) runs beside the previous launch: HCA / page rows
                                 // are read only after SeqDev::grow_epoch has reached seq[b].grow_count
  int wait_inputs;               // 1: griddepcontrol.wait before q / k_new / v_new are read
  const unsigned int* in_ctr;    // lsa_step_host_async: q / k_new / v_new are staged by a gather kernel that runs beside the
  unsigned int in_need;          // previous step; they are complete once this counter (its finished blocks) reaches in_need
  unsigned long long* ktime;     // profiling only, see TcParams
  unsigned long long* tl;        // lsa_timeline_enable: this launch's record [kTlCtas][kTlEvents] of %globaltimer stamps, or null
  unsigned int tl_seq;           // ... and its number among the context's traced launches
};

// Per-CTA timeline (include/lsa.h: lsa_timeline_*, LSA_TL_*): an instantiation of its own (kTl), so that the kernel that runs
// when nothing is stamped carries none of it (eleven `if (p.tl)` in the one kernel cost 0.3 us per step at cfg 3, measured).
constexpr int kTlCtas = 160, kTlEvents = 12;
enum { kTlEntry = 0, kTlSetup, kTlFirstS, kTlLastPV, kTlEpilogue, kTlArrived, kTlAllArrived, kTlMerged, kTlExit, kTlSmid, kTlNCtas, kTlSeq };
#define LSA_TL(ev) do { if constexpr (kTl) p.tl[(size_t)blockIdx.x * kTlEvents + (ev)] = gtime(); } while (0)

// the eight tensor maps of sequence 0 travel with the launch (param space: no descriptor fetch from global memory
// in front of the first TMA); sequences 1.. use SmParams::seq_maps
struct SmMaps0 { CUtensorMap m[8]; };

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
  int pg_page[32], pg_chunk[32];                              // table entries of the pages in this CTA's range
  int pg_off[kSmB], pg_cnt;                                   // entry of (sequence b, table position t) = pg_off[b] + t
  int k0_early;                                               // the setup already requested K of the first sub-tile
  int q_early;                                                // ... and the Q tile of the first piece
  int f0, f1;                                                 // this CTA's half tiles [f0, f1) of the flat list
  int rank;                                                   // this CTA's arrival index among the launch's CTAs (S8)
  uint64_t full[kTcStages], empty[kTcStages];
  uint64_t q_full, q_empty, s_full[2], s_empty[2], p_full, pv_done, o_full[4], o_empty, setup, app_done, mrg_full;
  uint32_t tmem_base;
};

__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ unsigned int ld_relaxed_u32(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void fence_acq_rel_gpu() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
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
  __device__ SubCursor(const SmSmem& sm_, int B_) : sm(sm_), B(B_) {
    f = sm_.f0; f1 = sm_.f1;                   // this CTA's share of the flat list (computed once by the setup)
    b = 0; prev_b = -1;
  }
  // out of line on purpose: four roles walk the list, one copy of the code stays hot in the instruction cache
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

// table entry of a page sub-tile: prefetched into shared memory by the setup, else (more than 32 pages in the range) global
__device__ __forceinline__ int sub_entry(const SmParams& p, const SmSmem& sm, const SubTile& s, const int* tbl, const int* pre) {
  const int i = sm.pg_off[s.b] + s.t;
  if (i >= 0 && i < sm.pg_cnt) return pre[i];
  return tbl[((size_t)s.b * 2 + sm.seq[s.b].cur) * p.k + s.t];
}

// attended rows of a sub-tile (the rest of its rows is masked)
__device__ __forceinline__ int sub_valid(const SmParams& p, const SmSmem& sm, const SubTile& s) {
  const SmSeq& q = sm.seq[s.b];
  if (s.kind == 0) return min(s.rows, q.n_hca - s.row0);
  if (s.kind == 2) return min(s.rows, q.w_len - s.row0);
  const int chunk = sub_entry(p, sm, s, p.tbl_chunk, sm.pg_chunk);
  const int vc = (int)max(0ll, min((long long)kTcC, q.n_csa - (long long)chunk * kTcC));
  return max(0, min(s.rows, vc - s.row0));
}


__device__ __forceinline__ float4 sm_warp_max4(float4 v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    v.x = fmaxf(v.x, __shfl_xor_sync(0xffffffffu, v.x, o)); v.y = fmaxf(v.y, __shfl_xor_sync(0xffffffffu, v.y, o));
    v.z = fmaxf(v.z, __shfl_xor_sync(0xffffffffu, v.z, o)); v.w = fmaxf(v.w, __shfl_xor_sync(0xffffffffu, v.w, o));
  }
  return v;
}
__device__ __forceinline__ float4 sm_warp_sum4(float4 v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    v.x += __shfl_xor_sync(0xffffffffu, v.x, o); v.y += __shfl_xor_sync(0xffffffffu, v.y, o);
    v.z += __shfl_xor_sync(0xffffffffu, v.z, o); v.w += __shfl_xor_sync(0xffffffffu, v.w, o);
  }
  return v;
}
__device__ __forceinline__ float sm_w_of(float m, float M) { return m == -INFINITY ? 0.f : exp2f(m - M); }

// S8 (see the header, item 3).  Called by the 256 softmax threads (t = 0..255) of the launch's MERGING CTAs once all
// partials of the launch are visible.  Unit = (sequence b, 32 consecutive uint2 columns cc of the partial layout) = 4 heads
// x 32 d, 256 per sequence; merger mi of n_mrg takes units [mi * NU / n_mrg, (mi + 1) * NU / n_mrg), one unit per warp and
// round.  The merge runs ONCE per launch, so its cost is its latency chain and its code size as much as its data: one
// thread requests the fp16 columns of all slots by TMA (2-D boxes of 32 slots x 256 B into the shared memory the attention
// phase has left behind); meanwhile every warp fetches m / l / block scale of all slots of its unit in ONE round trip
// (lane l: slots l, l + 32, ...; the rows are contiguous along the slots), parks them in shared memory, turns them into
// weights, and then runs the weighted sum as a short rolled loop over shared memory.  Slots without a partial for the
// sequence get weight 0 and are skipped, never multiplied.
constexpr int kMuLandBytes = 160 * 1024;      // landing area at the start of q + stage (192 KiB contiguous); weights behind it
struct MergePlan {
  int n_box, rows, per;                       // 32-slot boxes per unit, their rows, units per round
  int u0, u1;                                 // this merger's units
};
__device__ __forceinline__ MergePlan merge_plan(const SmParams& p, int mi, int n_mrg) {
  MergePlan mp;
  mp.n_box = (p.n_attn + 31) >> 5; mp.rows = mp.n_box * 32;
  mp.per = mp.rows <= 64 ? 8 : 4;             // per * rows * 256 B <= kMuLandBytes
  const unsigned NU = (unsigned)p.B * 256u;
  mp.u0 = (int)((unsigned)mi * NU / (unsigned)n_mrg); mp.u1 = (int)((unsigned)(mi + 1) * NU / (unsigned)n_mrg);
  return mp;
}
// one thread: request the fp16 columns of units [ub, ub + nu) of every slot of the launch
__device__ __forceinline__ void merge_request(const SmParams& p, SmSmem& sm, const CUtensorMap* map_part, const MergePlan& mp, int ub, int nu) {
  fence_proxy_async_all();                    // the partials were written by generic stores of other CTAs
  mbar_arrive_expect_tx(&sm.mrg_full, (uint32_t)(nu * mp.rows * 256));
#pragma unroll 1
  for (int i = 0; i < nu; ++i) {
    const int u = ub + i, b = u >> 8, cc = u & 255;
#pragma unroll 1
    for (int bx = 0; bx < mp.n_box; ++bx)
      tma_load_2d(sm.q + (size_t)(i * mp.rows + bx * 32) * 256, map_part, cc * 64, p.slot_row0 + b + bx * 32, &sm.mrg_full);
  }
}
// the 256 softmax threads; round 0 has been requested by the thread that saw the last arrival
__device__ __noinline__ void small_merge(const SmParams& p, SmSmem& sm, const CUtensorMap* map_part, int mi, int n_mrg, int t) {
  const int w = t >> 5, lane = t & 31;
  const int n_cta = p.n_attn;
  const MergePlan mp = merge_plan(p, mi, n_mrg);
  const int rows = mp.rows, per = mp.per;
  unsigned char* land = sm.q;                                    // [per][rows][256 B]
  float4* mbuf = reinterpret_cast<float4*>(sm.q + kMuLandBytes); // [per][rows]: m per head, then weight x block scale (<= 10 KiB)
  float4* lbuf = mbuf + per * rows;                              // [per][rows]: l per head
  float* sbuf = reinterpret_cast<float*>(lbuf + per * rows);     // [per][rows]: block scale
  const size_t ns = (size_t)p.n_slots;
  int round = 0;
  for (int ub = mp.u0; ub < mp.u1; ub += per, ++round) {
    const int nu = min(per, mp.u1 - ub);
    if (t == 0 && round > 0) merge_request(p, sm, map_part, mp, ub, nu);
    const bool mine = w < nu;                                    // warp w: unit ub + w, start to finish
    const int u = ub + (mine ? w : 0), b = u >> 8, cc = u & 255;
    const int dq = cc & 3, g = (cc >> 2) & 7, hh = (cc >> 5) & 1, m = cc >> 6, h0 = hh * 32 + g * 4;
    float4 M = make_float4(-INFINITY, -INFINITY, -INFINITY, -INFINITY);
    float4 L = make_float4(0.f, 0.f, 0.f, 0.f);
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    if (mine) {
      float4* mw = mbuf + w * rows;
      float4* lw = lbuf + w * rows;
      float* sw = sbuf + w * rows;
      // two slots per lane and trip (all of them at up to 64 CTAs), every load issued before the first store
#pragma unroll 1
      for (int c = lane; c < n_cta; c += 64) {
        const bool two = c + 32 < n_cta;
        const int c2 = two ? c + 32 : c;
        const size_t sa = (size_t)c + b, sb = (size_t)c2 + b;
        const float* pm = p.part_m + (size_t)h0 * ns;
        const float* pl = p.part_l + (size_t)h0 * ns;
        const float* ps = p.part_s + (size_t)((m * 2 + hh) * 4 + dq) * ns;
        const int2 ia = __ldcg(p.piece_info + c), ib = __ldcg(p.piece_info + c2);
        float4 ma = make_float4(__ldcg(pm + sa), __ldcg(pm + ns + sa), __ldcg(pm + 2 * ns + sa), __ldcg(pm + 3 * ns + sa));
        float4 mb = make_float4(__ldcg(pm + sb), __ldcg(pm + ns + sb), __ldcg(pm + 2 * ns + sb), __ldcg(pm + 3 * ns + sb));
        const float4 la = make_float4(__ldcg(pl + sa), __ldcg(pl + ns + sa), __ldcg(pl + 2 * ns + sa), __ldcg(pl + 3 * ns + sa));
        const float4 lb = make_float4(__ldcg(pl + sb), __ldcg(pl + ns + sb), __ldcg(pl + 2 * ns + sb), __ldcg(pl + 3 * ns + sb));
        const float s1a = __ldcg(ps + sa), s1b = __ldcg(ps + sb);
        // CTA c wrote a partial for sequence b, and the piece had an attended key (else it wrote no O)
        const float4 none = make_float4(-INFINITY, -INFINITY, -INFINITY, -INFINITY);
        if (!(ia.x <= b && b < ia.x + ia.y) || ma.x == -INFINITY) ma = none;
        if (!(ib.x <= b && b < ib.x + ib.y) || mb.x == -INFINITY) mb = none;
        mw[c] = ma; lw[c] = la; sw[c] = s1a;
        M.x = fmaxf(M.x, ma.x); M.y = fmaxf(M.y, ma.y); M.z = fmaxf(M.z, ma.z); M.w = fmaxf(M.w, ma.w);
        if (two) {
          mw[c2] = mb; lw[c2] = lb; sw[c2] = s1b;
          M.x = fmaxf(M.x, mb.x); M.y = fmaxf(M.y, mb.y); M.z = fmaxf(M.z, mb.z); M.w = fmaxf(M.w, mb.w);
        }
      }
      M = sm_warp_max4(M);
#pragma unroll 1
      for (int c = lane; c < n_cta; c += 32) {
        const float4 m4 = mw[c];
        float4 wj = make_float4(0.f, 0.f, 0.f, 0.f);
        if (m4.x != -INFINITY) {
          const float4 l4 = lw[c];
          const float s1 = sw[c];
          const float4 e = make_float4(sm_w_of(m4.x, M.x), sm_w_of(m4.y, M.y), sm_w_of(m4.z, M.z), sm_w_of(m4.w, M.w));
          L.x = fmaf(e.x, l4.x, L.x); L.y = fmaf(e.y, l4.y, L.y); L.z = fmaf(e.z, l4.z, L.z); L.w = fmaf(e.w, l4.w, L.w);
          wj = make_float4(e.x * s1, e.y * s1, e.z * s1, e.w * s1);
        }
        mw[c] = wj;
      }
      L = sm_warp_sum4(L);
      __syncwarp();
      mbar_wait(&sm.mrg_full, round & 1, 57);
      // weighted sum: lane = one uint2 column (4 heads of one d).  A slot of weight 0 (no partial for this sequence: it
      // holds what an earlier launch left there, possibly of another sequence) is selected away, never multiplied - a NaN
      // a caller fed into one sequence must not reach another; a select, not a branch, so the loads of a trip stay batched
      const unsigned char* lp = land + (size_t)w * rows * 256 + lane * 8;
#pragma unroll 8
      for (int sl = 0; sl < n_cta; ++sl) {
        const float4 f = mw[sl];
        uint2 v = *reinterpret_cast<const uint2*>(lp + (size_t)sl * 256);
        if (f.x == 0.f && f.y == 0.f && f.z == 0.f && f.w == 0.f) v = make_uint2(0u, 0u);
        const float2 a01 = unpack_f16x2(v.x), a23 = unpack_f16x2(v.y);
        acc.x = fmaf(f.x, a01.x, acc.x); acc.y = fmaf(f.y, a01.y, acc.y);
        acc.z = fmaf(f.z, a23.x, acc.z); acc.w = fmaf(f.w, a23.y, acc.w);
      }
    }
    if (round == 0) named_bar_sync(4, 288);                      // the previous launch has been merged: `out` may be written
    if (mine) {
      __nv_bfloat16* o = p.out + ((size_t)b * kTcH + h0) * kTcD + m * 128 + dq * 32 + lane;
      o[0] = __float2bfloat16_rn(L.x > 0.f ? acc.x / L.x : 0.f);
      o[kTcD] = __float2bfloat16_rn(L.y > 0.f ? acc.y / L.y : 0.f);
      o[2 * kTcD] = __float2bfloat16_rn(L.z > 0.f ? acc.z / L.z : 0.f);
      o[3 * kTcD] = __float2bfloat16_rn(L.w > 0.f ? acc.w / L.w : 0.f);
      if (p.lse && m == 0 && dq == 0 && lane == 0) {
        float* ls = p.lse + (size_t)b * kTcH + h0;
        ls[0] = L.x > 0.f ? (M.x + log2f(L.x)) * 0.6931471805599453f : -INFINITY;
        ls[1] = L.y > 0.f ? (M.y + log2f(L.y)) * 0.6931471805599453f : -INFINITY;
        ls[2] = L.z > 0.f ? (M.z + log2f(L.z)) * 0.6931471805599453f : -INFINITY;
        ls[3] = L.w > 0.f ? (M.w + log2f(L.w)) * 0.6931471805599453f : -INFINITY;
      }
    }
    if (ub + per < mp.u1) {                                      // the landing buffer and the weights are reused by the next round
      if (!mine) mbar_wait(&sm.mrg_full, round & 1, 58);         // (idle warps keep up with the barrier's phase)
      named_bar_sync(2, 256);
    }
  }
}

template <bool kTl>
__global__ void __launch_bounds__(kTcThreads, 1)
attn_tc_small_kernel(const __grid_constant__ CUtensorMap map_pool, const __grid_constant__ CUtensorMap map_pool64,
                     const __grid_constant__ CUtensorMap map_q, const __grid_constant__ CUtensorMap map_part,
                     const __grid_constant__ SmMaps0 maps0, const __grid_constant__ SmParams p) {
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
    mbar_init(&sm.mrg_full, 1);
    fence_mbar_init();
    prefetch_tmap(&map_pool);
    prefetch_tmap(&map_pool64);
    prefetch_tmap(&map_q);
    prefetch_tmap(&map_part);
  }
  __syncthreads();
  griddep_launch_dependents();    // the combine blocks of this step (and, behind them, the next step's CTAs) may be placed
  if (p.ktime && tid == 0) atomicMin(p.ktime, gtime());
  if (kTl && tid == 0) {
    unsigned long long* r = p.tl + (size_t)cta * kTlEvents;
    unsigned int smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    r[kTlEntry] = gtime(); r[kTlAllArrived] = 0; r[kTlMerged] = 0; r[kTlSmid] = smid; r[kTlNCtas] = (unsigned)n_cta; r[kTlSeq] = p.tl_seq;
  }
  if (warp == 0) {
    // per-sequence shape -> half tiles per segment and their prefix (B <= 4).  Everything this CTA needs from global
    // memory before its first TMA is requested in ONE round trip: the table entries of the pages in its range, the
    // tensor maps of its sequences, and - only if its range holds window rows - the append counter.
    int g = 0, hca = 0, pg = 0;
    SmSeq q{};
    if (lane < p.B) {
      q = p.seq[lane];
      if (q.n_cur < 0) q.n_cur = __ldcg(&p.seqs[lane].n_tbl[q.cur]);       // selection given on the device: its size too
      hca = (q.n_hca + kSmHalf - 1) / kSmHalf; pg = 2 * q.n_cur;
      g = hca + pg + (q.w_len + kSmHalf - 1) / kSmHalf;
      sm.seq[lane] = q; sm.hh_hca[lane] = hca; sm.hh_pg[lane] = pg;
    }
    int incl = g;
#pragma unroll
    for (int o = 1; o < kSmB; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += t;
    }
    if (lane < p.B) sm.gpre[lane + 1] = incl;
    if (lane == 0) sm.gpre[0] = 0;
    const unsigned T = (unsigned)__shfl_sync(0xffffffffu, incl, p.B - 1);
    const int f0 = (int)((unsigned)cta * T / (unsigned)n_cta), f1 = (int)((unsigned)(cta + 1) * T / (unsigned)n_cta);
    if (lane == 0) { sm.f0 = f0; sm.f1 = f1; }
    __syncwarp();
    // A range that starts in HCA rows needs nothing from global memory: its first K sub-tile is requested right here,
    // ahead of the table / counter look-ups below (sm.k0_early tells the producer loop)
    {
      SubCursor c0(sm, p.B);
      SubTile s0;
      const bool any0 = c0.next(s0);
      const bool early = any0 && s0.kind == 0 && !p.grow_wait;
      const bool q_early = any0 && !p.wait_inputs && !p.in_ctr;   // q is ready: nothing to wait for before its tile is requested
      if (lane == 0) { sm.k0_early = early ? 1 : 0; sm.q_early = q_early ? 1 : 0; }
      if (q_early && elect_one()) {
        mbar_arrive_expect_tx(&sm.q_full, 65536);
        tma_load_3d(sm.q, &map_q, 0, s0.b * kTcH, 0, &sm.q_full);
      }
      if (early && elect_one()) {
        const uint64_t pol = l2_policy_evict_first();
        const CUtensorMap* mk = (s0.b == 0 ? maps0.m : p.seq_maps + s0.b * 8) + (s0.rows == kTcTile ? 0 : 4);
#pragma unroll 1
        for (int s4 = 0; s4 < 4; ++s4) {
          mbar_arrive_expect_tx(&sm.full[s4], (uint32_t)s0.rows * 256u);
          tma_load_3d_hint(sm.stage[s4], mk, 0, s0.row0, s4 * 2, &sm.full[s4], pol);
        }
      }
    }
    int cnt = 0;                                       // page slots of this CTA's range, all sequences
    // (rolled, and only over the sequences there are: this code runs once per CTA, instruction-cache cold)
#pragma unroll 1
    for (int b = 0; b < p.B; ++b) {
      const int end_b = __shfl_sync(0xffffffffu, incl, b), g_b = __shfl_sync(0xffffffffu, g, b);
      const int hca_b = __shfl_sync(0xffffffffu, hca, b), pg_b = __shfl_sync(0xffffffffu, pg, b), cur_b = __shfl_sync(0xffffffffu, q.cur, b);
      {
        const int base = end_b - g_b + hca_b;          // first page half tile of sequence b in the flat list
        const int lo = max(f0, base), hi = min(f1, base + pg_b);
        int off = -(1 << 30), vp = 0, vc = 0;
        bool have = false;
        if (lo < hi) {
          const int t_lo = (lo - base) >> 1, n = ((hi - 1 - base) >> 1) - t_lo + 1;
          off = cnt - t_lo;
          if (lane >= cnt && lane < cnt + n) {
            const size_t e = ((size_t)b * 2 + cur_b) * p.k + t_lo + lane - cnt;
            vp = __ldcg(p.tbl_page + e);
            vc = __ldcg(p.tbl_chunk + e);
            have = true;
          }
          cnt += n;
        }
        // window rows in the range: ring rows appended by earlier launches are visible once app_epoch has caught up with
        // the host's count (normally it has); HCA / tail-page rows handed over by an append kernel that runs beside the
        // previous launch: grow_epoch.  Both counters are probed while the table loads are in flight - one round trip.
        const bool need_app = lane == b && f1 > base + pg_b && f0 < end_b;
        const bool need_grow = p.grow_wait && lane == b && f0 < end_b && f1 > end_b - g_b;
        unsigned probe_a = 0, probe_g = 0;
        if (need_app) probe_a = ld_relaxed_u32(&p.seqs[b].app_epoch);
        if (need_grow) probe_g = ld_relaxed_u32(&p.seqs[b].grow_epoch);
        if (have) { sm.pg_page[lane] = vp; sm.pg_chunk[lane] = vc; }
        if (lane == 0) sm.pg_off[b] = off;
        if (need_app && (int)(probe_a - q.app_count) < 0) wait_counter(&p.seqs[b].app_epoch, q.app_count, 50);
        if (need_grow && (int)(probe_g - q.grow_count) < 0) wait_counter(&p.seqs[b].grow_epoch, q.grow_count, 57);
        if (need_app || need_grow) fence_acq_rel_gpu();      // the relaxed probe becomes an acquire
        if (b > 0 && f0 < end_b && f1 > end_b - g_b && lane < 8) prefetch_tmap(p.seq_maps + b * 8 + lane);
      }
    }
    if (lane == 0) sm.pg_cnt = min(cnt, 32);
    if (p.grow_wait) fence_proxy_async_all();          // the rows were written by generic stores, TMA reads them
    __syncwarp();
    if (lane == 0) { LSA_TL(kTlSetup); mbar_arrive(&sm.setup); }
  } else if (warp == 1) {
    tmem_alloc(&sm.tmem_base, 512);
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive(&sm.setup);
  } else {
    for (int i = tid - 64; i < 2048; i += kTcThreads - 64) reinterpret_cast<uint16_t*>(sm.ones)[i] = 0x3f80;   // bf16 1.0
    fence_proxy_async_smem();
    __syncwarp();
    if (lane == 0) mbar_arrive(&sm.setup);
  }

  if (warp == 0) {
    // =========================== TMA producer ===========================
    if (elect_one()) {
      SubCursor cur(sm, p.B);
      SubTile s, nx;
      uint32_t ring = sm.k0_early ? 4u : 0u;
      int item = 0;
      bool app_seen = false, waited = false, k0_pending = sm.k0_early != 0;
      const uint64_t pol_stream = l2_policy_evict_first();   // K/V rows: read once per step
      auto src_of = [&](const SubTile& t, const CUtensorMap*& mk, const CUtensorMap*& mv, int& rk, int& rv) {
        const int big = t.rows == kTcTile ? 0 : 4;
        if (t.kind == 1) {
          const int page = sub_entry(p, sm, t, p.tbl_page, sm.pg_page);
          mk = mv = (t.rows == kTcTile ? &map_pool : &map_pool64);
          rk = page * (2 * kTcC) + t.row0; rv = rk + kTcC;
        } else {
          mk = (t.b == 0 ? maps0.m : p.seq_maps + t.b * 8) + big + (t.kind == 0 ? 0 : 2);
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
          st_release_u32(&p.seqs[t.b].app_epoch, q.app_count + 1u);   // (the writers fenced generic -> async proxy)
        }
      };
      auto issue4 = [&](const CUtensorMap* m, int row, int rows) {
#pragma unroll 1
        for (int s4 = 0; s4 < 4; ++s4) {
          const int st = ring % kTcStages;
          mbar_wait(&sm.empty[st], ((ring / kTcStages) & 1) ^ 1, 11);
          mbar_arrive_expect_tx(&sm.full[st], (uint32_t)rows * 256u);
          tma_load_3d_hint(sm.stage[st], m, 0, row, s4 * 2, &sm.full[st], pol_stream);
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
          if (!k0_pending) issue4(mk, rk, s.rows);         // K of the piece's first sub-tile: in flight before Q is known
          k0_pending = false;
          if (item > 0 || !sm.q_early) {
            if (item > 0) mbar_wait(&sm.q_empty, (item - 1) & 1, 10);
            if (p.wait_inputs && !waited) { griddep_wait(); waited = true; }   // q is the caller's: whatever the stream ran last
            if (p.in_ctr && !waited) { wait_counter(p.in_ctr, p.in_need, 55); fence_proxy_async_all(); waited = true; }
            mbar_arrive_expect_tx(&sm.q_full, 65536);
            tma_load_3d(sm.q, &map_q, 0, s.b * kTcH, 0, &sm.q_full);
          }
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
      SubCursor cur(sm, p.B);
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
          if (item == 0) LSA_TL(kTlFirstS);
        }
        have = cur.next(nx);
        if (!s.last) issue_s(nx.rows, nx.last);
        if (s.rows == kTcTile) issue_pv(std::integral_constant<int, 8>{}, s.first, s.last);
        else issue_pv(std::integral_constant<int, 4>{}, s.first, s.last);
        if (s.last) ++item;
        s = nx;
      }
      LSA_TL(kTlLastPV);
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
    // the launch that used this workspace buffer last (three launches ago) has been merged: normally long ago.  The
    // other softmax warps meet this one at the named barrier of their first sub-tile, before any of them writes a partial.
    if (tid == 64) wait_counter(p.done_ctr, p.done_need_buf, 51);
    if (p.k_new) {
      // window append ("decoded tokens stay resident"; DESIGN R6): the CTA that owns the sub-tile holding
      // ring slot w_head of a sequence writes k_new / v_new there before its producer loads that sub-tile
      SubCursor pc(sm, p.B);
      SubTile a;
      const int t = tid - 64;
      bool waited = false;
      while (pc.next(a)) {
        const SmSeq& q = sm.seq[a.b];
        if (a.kind == 2 && q.app_slot >= a.row0 && q.app_slot < a.row0 + a.rows && t < 128) {
          if (p.wait_inputs && !waited) { griddep_wait(); waited = true; }   // k_new / v_new are the caller's
          if (p.in_ctr && !waited) { wait_counter(p.in_ctr, p.in_need, 56); waited = true; }
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
    SubCursor cur(sm, p.B);
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
          if (tid < 64 + kTcH) { p.part_m[(size_t)(tid - 64) * p.n_slots + cta + e] = -INFINITY; p.part_l[(size_t)(tid - 64) * p.n_slots + cta + e] = 0.f; }
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
        if (lane == 0) p.part_s[(size_t)((m * 2 + hh) * 4 + q4) * p.n_slots + slot] = inv;
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
            p.part_l[(size_t)(hh * 32 + j) * p.n_slots + slot] = __uint_as_float(vreg[j]);
            p.part_m[(size_t)(hh * 32 + j) * p.n_slots + slot] = m_run[j] <= -1e30f ? -INFINITY : m_run[j];   // no attended key: S8 skips the slot
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&sm.o_empty);
      ++piece;
    }
    if (tid == 64) LSA_TL(kTlEpilogue);
    if (tid == 64) p.piece_info[cta] = make_int2(b_first < 0 ? 0 : b_first, b_first < 0 ? 0 : b_last - b_first + 1);
  }
  // ---- S8: publish; the launch's last n_mrg CTAs to arrive merge its partials, the others leave their SM at once ----
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(sm.tmem_base, 512);
  }
  if (tid == 0) {
    __threadfence();                                // cumulative: the partial stores of every thread of this CTA (ordered before
    const unsigned int old = atomicAdd(p.arr_ctr, 1u);   // this thread by the barrier) are visible before the arrival is
    sm.rank = (int)(old - (p.arr_target - (unsigned)n_cta));   // arrival index inside this launch, 0 .. n_cta - 1
    LSA_TL(kTlArrived);
  }
  __syncthreads();
  const int mi = sm.rank - (n_cta - p.n_mrg);       // the last n_mrg arrivals are the mergers 0 .. n_mrg - 1
  if (mi < 0) {
    if (tid == 0) LSA_TL(kTlExit);
    if (p.ktime && tid == 0) atomicMax(p.ktime + 1, gtime());
    return;
  }
  // mergers: warp 0 sees the last arrival, requests the first round of partials and then waits for the previous launch's
  // merge (records, `out`); the softmax warps start on the weights as soon as the partials are visible
  if (warp == 0) {
    if (lane == 0) {
      wait_counter(p.arr_ctr, p.arr_target, 53);    // every partial of the launch is visible from here on
      LSA_TL(kTlAllArrived);
    }
    __syncwarp();
    named_bar_sync(3, 288);                         // the softmax warps start on the weights
    {                                               // round 0 of the partials: one 32-slot box per lane
      const MergePlan mp = merge_plan(p, mi, p.n_mrg);
      const int nu = min(mp.per, mp.u1 - mp.u0);
      if (lane == 0) mbar_arrive_expect_tx(&sm.mrg_full, (uint32_t)(nu * mp.rows * 256));
      __syncwarp();
      if (lane < nu * mp.n_box) {
        const int i = lane / mp.n_box, bx = lane - i * mp.n_box;
        const int u = mp.u0 + i, b = u >> 8, cc = u & 255;
        fence_proxy_async_all();                    // the partials were written by generic stores of other CTAs
        tma_load_2d(sm.q + (size_t)(i * mp.rows + bx * 32) * 256, &map_part, cc * 64, p.slot_row0 + b + bx * 32, &sm.mrg_full);
      }
    }
    if (lane == 0) {
      wait_counter(p.done_ctr, p.done_need_prev, 54);   // the previous launch has been merged
    }
    __syncwarp();
    if (mi == 0 && lane < p.B) {                    // the per-sequence record catches up with the launch's view
      SeqDev& sd = p.seqs[lane];
      if (((p.swap >> lane) & 1u) && sd.pending) { sd.cur_buf = 1 - sd.cur_buf; sd.pending = 0; }
      if (p.k_new) {
        const int slot = sd.w_head;
        sd.w_head = (slot + 1 == p.W) ? 0 : slot + 1;
        sd.w_len = min(p.W, sd.w_len + 1);
      }
    }
    named_bar_sync(4, 288);
  } else if (warp >= 2) {
    named_bar_sync(3, 288);
    small_merge(p, sm, &map_part, mi, p.n_mrg, tid - 64);
  }
  __syncthreads();
  if (tid == 0) LSA_TL(kTlMerged);
  if (tid == 0) {
    if (p.host_flag) {
      // `out` may live in pinned host memory: this CTA's rows are visible system-wide before it is counted, and the
      // merger that completes the count tells the host
      __threadfence_system();
      const unsigned int old = atomicAdd(p.done_ctr, 1u);
      if (old + 1u == p.done_after) {
        __threadfence_system();
        *reinterpret_cast<volatile unsigned int*>(p.host_flag) = p.host_flag_val;
      }
    } else {
      __threadfence();
      red_release_add_u32(p.done_ctr, 1u);
    }
  }
  if (tid == 0) LSA_TL(kTlExit);
  if (p.ktime && tid == 0) atomicMax(p.ktime + 1, gtime());
}

}  // namespace lsa
