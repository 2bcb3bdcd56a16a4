// lsa_l2.cu - Level 2 of LSA (Eq.(6), l.187): every decode step the native
// Lightning Indexer scores the entries of the RESIDENT recalled set only,
//     Score_native(i, s) = sum_h w_{i,h} ReLU(q_{i,h} . K_s^IComp)        (Eq.(4) without the sigmoid, l.75)
// and core attention runs over the Top-k of them (+) HCA (+) window.  DESIGN.md "NEXT-2" lists the readings.
//
// Kernels
//   l2_score_kernel   one 128-entry tile = one page of the current table: S^T[128 entries x 64 heads] =
//                     K_tile[128 x 128] . q^T on tcgen05 (8 MMAs, M=128 N=64 K=16), key tiles by TMA straight from
//                     the sequence's index-K rows [chunk * 128, +128), thread = entry for the gate and the
//                     head-weighted sum.  Per step it reads n_cur * 32 KiB of index keys (2 MiB at 1M / k = 64).
//   l2_topk_kernel    per sequence: the k2 best of the n_cur * 128 scores by (score desc, entry id asc) with the
//                     block-wide select of lsa_select.cuh, written as a row bitmask per page ("mask" of l.187) that
//                     the attention kernel applies to the page tiles - the pages stay where Level 1 put them, no
//                     K/V byte is copied ("remap" is the bitmask), and optionally as a list of entry ids.
#include <cuda.h>
#include <cuda_bf16.h>

#include <string>
#include <vector>

#include "lsa_l2.h"
#include "lsa_select.cuh"
#include "lsa_tc_ptx.cuh"

namespace lsa {
using namespace ptx;

constexpr int kL2H = 64, kL2C = 128, kL2CI = 128;
constexpr int kL2Stages = 4;
constexpr int kL2StageBytes = 32768;                 // [2 d-blocks][128 entries][128 B]
constexpr int kL2Threads = 64 + 128;                 // producer warp, MMA warp, 4 gate warps

struct L2ScoreParams {
  const SeqDev* seqs;
  const int* tbl_chunk;          // [B][2][k]
  const CUtensorMap* k_maps;     // [B]: index keys [n_csa][128] bf16 as (64, rows, 2 d-blocks)
  const float* w_idx;            // [B][64]
  float* score;                  // [B][k * 128]; rows past the chunk's valid entries get -inf
  unsigned* ghist;               // [B][4096] or null: entries per top-12-bit bin of the ordered score (for the mask-only
                                 // Top-k kernel, which zeroes it again); null when the general Top-k kernel follows
  int B, k;
  unsigned swap[8];              // bit b: sequence b's staged table is the one this step attends (S6 folded into the
                                 // attention launch that follows: the records still show it as pending)
};
constexpr int kL2Bins = 4096;

struct L2Swap { unsigned w[8]; };
// which table buffer the attention launch of this step will read
__device__ __forceinline__ int l2_cur_buf(const SeqDev& s, const unsigned* swap, int b) {
  const bool sw = ((swap[b >> 5] >> (b & 31)) & 1u) && s.pending;
  return sw ? 1 - s.cur_buf : s.cur_buf;
}

struct L2Smem {
  alignas(1024) unsigned char q[16384];                          // [2 d-blocks][64 heads][128 B], SW128
  alignas(1024) unsigned char stage[kL2Stages][kL2StageBytes];   // [2 d-blocks][128 entries][128 B], SW128
  uint64_t full[kL2Stages], empty[kL2Stages];
  uint64_t q_full, q_empty, s_full[2], s_empty[2];
  uint32_t tmem_base;
};

// (sequence, slot range) pieces of this CTA's share [f0, f1) of the flat slot list [B][k], clipped to the
// sequence's current table; pieces without a page are skipped by every role alike.
struct L2Cursor {
  const L2ScoreParams& p;
  int f, f1;
  __device__ L2Cursor(const L2ScoreParams& p_, int cta, int n_cta) : p(p_) {
    const unsigned T = (unsigned)p_.B * (unsigned)p_.k;
    f = (int)((unsigned long long)cta * T / (unsigned)n_cta);
    f1 = (int)((unsigned long long)(cta + 1) * T / (unsigned)n_cta);
  }
  __device__ bool next(int& b, int& t0, int& t1, int& cur) {
    while (f < f1) {
      b = f / p.k;
      t0 = f - b * p.k;
      const int end = min(f1, (b + 1) * p.k);
      const SeqDev& s = p.seqs[b];
      cur = l2_cur_buf(s, p.swap, b);
      t1 = min(end - b * p.k, s.n_tbl[cur]);
      f = end;
      if (t0 < t1) return true;
    }
    return false;
  }
};

__global__ void __launch_bounds__(kL2Threads, 1)
l2_score_kernel(const __grid_constant__ CUtensorMap map_q, const __grid_constant__ L2ScoreParams p) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  L2Smem& sm = *reinterpret_cast<L2Smem*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int cta = blockIdx.x, n_cta = gridDim.x;
  if (tid == 0) {
    for (int i = 0; i < kL2Stages; ++i) { mbar_init(&sm.full[i], 1); mbar_init(&sm.empty[i], 1); }
    mbar_init(&sm.q_full, 1); mbar_init(&sm.q_empty, 1);
    for (int i = 0; i < 2; ++i) { mbar_init(&sm.s_full[i], 1); mbar_init(&sm.s_empty[i], 4); }
    fence_mbar_init();
    prefetch_tmap(&map_q);
  }
  if (warp == 1) tmem_alloc(&sm.tmem_base, 128);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  griddep_wait();                 // the tables (S6) and q_idx / w_idx come from work enqueued before this kernel
  griddep_launch_dependents();
  const uint32_t tS = sm.tmem_base;

  if (warp == 0) {
    // =========================== TMA producer ===========================
    if (elect_one()) {
      L2Cursor cur(p, cta, n_cta);
      int b, t0, t1, cb, item = 0;
      uint32_t ring = 0;
      while (cur.next(b, t0, t1, cb)) {
        if (item > 0) mbar_wait(&sm.q_empty, (item - 1) & 1, 50);
        mbar_arrive_expect_tx(&sm.q_full, 16384);
        tma_load_3d(sm.q, &map_q, 0, b * kL2H, 0, &sm.q_full);
        const CUtensorMap* mk = p.k_maps + b;
        const int* chunks = p.tbl_chunk + ((size_t)b * 2 + cb) * p.k;
        for (int t = t0; t < t1; ++t) {
          const int st = ring % kL2Stages;
          mbar_wait(&sm.empty[st], ((ring / kL2Stages) & 1) ^ 1, 51);
          mbar_arrive_expect_tx(&sm.full[st], kL2StageBytes);
          tma_load_3d(sm.stage[st], mk, 0, chunks[t] * kL2C, 0, &sm.full[st]);   // rows past n_csa are zero-filled
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
      L2Cursor cur(p, cta, n_cta);
      int b, t0, t1, cb, item = 0;
      uint32_t ring = 0, n_s = 0;
      while (cur.next(b, t0, t1, cb)) {
        mbar_wait(&sm.q_full, item & 1, 52);
        tc_fence_after();
        for (int t = t0; t < t1; ++t) {
          const int buf = n_s & 1, st = ring % kL2Stages;
          mbar_wait(&sm.s_empty[buf], ((n_s >> 1) & 1) ^ 1, 53);
          mbar_wait(&sm.full[st], (ring / kL2Stages) & 1, 54);
          tc_fence_after();
          const uint64_t a0 = dk0 + (uint64_t)(st * (kL2StageBytes >> 4));
#pragma unroll
          for (int ks = 0; ks < 8; ++ks) {
            const uint64_t off_a = (uint64_t)(((ks >> 2) * 16384 + (ks & 3) * 32) >> 4);
            const uint64_t off_b = (uint64_t)(((ks >> 2) * 8192 + (ks & 3) * 32) >> 4);
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
    // =========================== gate + head-weighted sum (4 warps, thread = entry) ===========================
    const int q4 = warp & 3;
    const uint32_t lane_addr = (uint32_t)(q4 * 32) << 16;
    const int row = q4 * 32 + lane;
    L2Cursor cur(p, cta, n_cta);
    int b, t0, t1, cb;
    uint32_t n_s = 0;
    while (cur.next(b, t0, t1, cb)) {
      float w[kL2H];
      const float4* wp = reinterpret_cast<const float4*>(p.w_idx + (size_t)b * kL2H);
#pragma unroll
      for (int j = 0; j < kL2H / 4; ++j) { const float4 t4 = wp[j]; w[4 * j] = t4.x; w[4 * j + 1] = t4.y; w[4 * j + 2] = t4.z; w[4 * j + 3] = t4.w; }
      const long long n_csa = p.seqs[b].n_csa;
      const int* chunks = p.tbl_chunk + ((size_t)b * 2 + cb) * p.k;
      for (int t = t0; t < t1; ++t) {
        const int buf = n_s & 1;
        const long long first = (long long)chunks[t] * kL2C;
        float x[kL2H];
        mbar_wait(&sm.s_full[buf], (n_s >> 1) & 1, 55);
        tc_fence_after();
        tmem_ld32(tS + buf * 64 + lane_addr, reinterpret_cast<uint32_t*>(x));
        tmem_ld32(tS + buf * 64 + 32 + lane_addr, reinterpret_cast<uint32_t*>(x) + 32);
        tmem_wait_ld();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&sm.s_empty[buf]);
        float pre = 0.f;
#pragma unroll
        for (int h = 0; h < kL2H; ++h) pre = fmaf(w[h], fmaxf(x[h], 0.f), pre);          // Score_native (l.71-75)
        if (first + row >= n_csa) pre = -INFINITY;                                         // not an entry (M1)
        p.score[((size_t)b * p.k + t) * kL2C + row] = pre;
        if (p.ghist) {                                                                     // first radix digit, counted where the scores are
          const bool ok = pre != -INFINITY;
          const unsigned bin = float_to_ordered(pre) >> 20;
          const unsigned am = __ballot_sync(0xffffffffu, ok);
          if (ok) {
            const unsigned peers = __match_any_sync(am, bin);
            if (lane == __ffs(peers) - 1) atomicAdd(p.ghist + (size_t)b * kL2Bins + bin, (unsigned)__popc(peers));
          }
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

// ---- Eq.(6): Top-k2 of the resident entries ----------------------------------------------------------------------
// One block per sequence.  The table is in ascending chunk id, so position i = slot * 128 + row orders the entries
// exactly as their ids s = chunk * 128 + row do: key = (~ordered(score), i) gives (score desc, entry id asc).
__global__ void __launch_bounds__(1024)
l2_topk_kernel(const SeqDev* __restrict__ seqs, L2Swap swap, const int* __restrict__ tbl_chunk, const float* __restrict__ score, int k, int k2,
               uint32_t* __restrict__ mask, int32_t* __restrict__ sel_entries, float* __restrict__ sel_score) {
  __shared__ SelectSmem sm;
  const int b = blockIdx.x;
  pdl_wait();
  pdl_launch_dependents();
  const SeqDev& sq = seqs[b];
  const int cur = l2_cur_buf(sq, swap.w, b), n_cur = sq.n_tbl[cur];
  const float* sc = score + (size_t)b * k * kL2C;
  uint32_t* mk = mask + (size_t)b * k * 4;
  for (int i = threadIdx.x; i < k * 4; i += blockDim.x) mk[i] = 0u;
  auto keyf = [sc](int i) -> unsigned long long {
    const float s = sc[i];
    return s == -INFINITY ? kKeyMax : (((unsigned long long)(~float_to_ordered(s)) << 32) | (unsigned)i);
  };
  const int n = n_cur * kL2C;
  const int m = block_select_smallest(keyf, n, min(k2, n), sm);
  __syncthreads();                                           // the zeroed mask words are visible to the whole block
  const int* chunks = tbl_chunk + ((size_t)b * 2 + cur) * k;
  for (int j = threadIdx.x; j < k2; j += blockDim.x) {
    int entry = -1;
    float val = -INFINITY;
    if (j < m && sm.keys[j] != kKeyMax) {
      const unsigned i = (unsigned)(sm.keys[j] & 0xffffffffull);
      atomicOr(&mk[i >> 5], 1u << (i & 31));
      entry = chunks[i >> 7] * kL2C + (int)(i & 127);
      val = ordered_to_float(~(uint32_t)(sm.keys[j] >> 32));
    }
    if (sel_entries) sel_entries[(size_t)b * k2 + j] = entry;
    if (sel_score) sel_score[(size_t)b * k2 + j] = val;
  }
}


// Mask-only fast path (no entry list asked for, k * 128 <= 16384).  The first radix digit - the top 12 bits of the
// ordered score - is counted by the score kernel's CTAs, which hold the scores in registers (warp-aggregated global
// atomics into ghist[b][4096]); this kernel (one block per sequence, a thread keeps PER consecutive scores in registers:
// position = tid * PER + j, so thread order is entry-id order)
//   1. reads and re-zeroes the histogram, 4 bins per thread; one block scan gives the number of entries and the bin
//      that holds the k2-th largest score,
//   2. collects the keys of that bin (about n / 20 of them) into shared memory and finishes the select on those with
//      3 passes of 8 bits (match.any-aggregated shared-memory histograms, bins scanned by one warp); a bin with more than
//      kL2Cand keys runs the same passes over the register keys instead,
//   3. marks key > cut-off, and resolves ties AT the cut-off by position with one block scan - the same
//      (score desc, entry id asc) rule as the general kernel, without sorting the winners.
// Each mask word is written exactly once.  History: 8-pass radix + sort of the winners 61 us per select at 8192 entries;
// all 4 passes in this block 16.7 us (ncu: ~35 k cycles behind ~560 MATCH.ANY + ATOMS on one SM); see profiles/r01_level2.md.
constexpr int kL2Cand = 2048;

// byte_hi .. 0: 8-bit MSB radix passes over this thread's N keys; keys with (key & pmask) != *s_prefix are out.
// In: *s_prefix / *s_need = digits fixed so far / rank wanted among the matching keys.  Out: the full key / how many
// keys equal to it are taken.  All threads of the block call it.
template <int N>
__device__ __forceinline__ void l2_radix_passes(const uint32_t (&key)[N], uint32_t pmask, int byte_hi, unsigned* hist, unsigned* s_prefix,
                                                unsigned* s_need, int tid, int lane, int warp) {
  for (int byte = byte_hi; byte >= 0; --byte) {
    if (tid < 256) hist[tid] = 0u;
    __syncthreads();
    const uint32_t prefix = *s_prefix;
#pragma unroll
    for (int j = 0; j < N; ++j) {
      const bool act = (key[j] & pmask) == prefix;
      const unsigned bin = (key[j] >> (8 * byte)) & 255u;
      const unsigned amask = __ballot_sync(0xffffffffu, act);
      if (act) {
        const unsigned peers = __match_any_sync(amask, bin);
        if (lane == __ffs(peers) - 1) atomicAdd(&hist[bin], (unsigned)__popc(peers));
      }
    }
    __syncthreads();
    if (warp == 0) {                                        // lane l owns bins 255 - 8l .. 248 - 8l (descending)
      unsigned h[8], mine = 0;
#pragma unroll
      for (int i = 0; i < 8; ++i) { h[i] = hist[255 - 8 * lane - i]; mine += h[i]; }
      unsigned incl = mine;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const unsigned t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
      const unsigned need = *s_need;
      const unsigned before = incl - mine;                  // keys in higher bins than this lane's
      if (before < need && need <= incl) {                  // the cut-off digit is one of this lane's bins
        unsigned cum = before;
        int d = 0;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          if (cum + h[i] >= need) { d = 255 - 8 * lane - i; break; }
          cum += h[i];
        }
        *s_need = need - cum;
        *s_prefix = prefix | ((uint32_t)d << (8 * byte));
      }
    }
    pmask |= 0xffu << (8 * byte);
    __syncthreads();
  }
}

template <int PER>
__global__ void __launch_bounds__(1024)
l2_topk_mask_kernel(const SeqDev* __restrict__ seqs, L2Swap swap, const float* __restrict__ score, unsigned* __restrict__ ghist, int k, int k2,
                    uint32_t* __restrict__ mask) {
  __shared__ unsigned hist[256];
  __shared__ unsigned wsum[33];
  __shared__ uint32_t cand[kL2Cand];
  __shared__ unsigned s_prefix, s_need, s_m, s_cnt;
  const int b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  pdl_wait();
  pdl_launch_dependents();
  const SeqDev& sq = seqs[b];
  const int n = sq.n_tbl[l2_cur_buf(sq, swap.w, b)] * kL2C;  // multiple of 128, PER divides 128
  const float* sc = score + (size_t)b * k * kL2C;
  uint32_t* mk = mask + (size_t)b * k * 4;
  const int base = tid * PER;
  uint4* gh = reinterpret_cast<uint4*>(ghist + (size_t)b * kL2Bins) + tid;     // bins 4 tid .. 4 tid + 3
  const uint4 h4 = *gh;
  *gh = make_uint4(0u, 0u, 0u, 0u);                          // ready for the next step's score kernel
  uint32_t key[PER];                                         // 0 = not an entry (float_to_ordered never returns 0)
#pragma unroll
  for (int j = 0; j < PER; j += 4) {
    float4 v = make_float4(-INFINITY, -INFINITY, -INFINITY, -INFINITY);
    if (base + j < n) v = *reinterpret_cast<const float4*>(sc + base + j);
    key[j] = v.x == -INFINITY ? 0u : float_to_ordered(v.x);
    key[j + 1] = v.y == -INFINITY ? 0u : float_to_ordered(v.y);
    key[j + 2] = v.z == -INFINITY ? 0u : float_to_ordered(v.z);
    key[j + 3] = v.w == -INFINITY ? 0u : float_to_ordered(v.w);
  }
  // block-wide exclusive scan of one value per thread (thread order); returns the prefix, *total = the block sum
  auto block_scan = [&](unsigned v, unsigned* total) -> unsigned {
    unsigned incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const unsigned t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
    __syncthreads();                                         // wsum may still be read from an earlier call
    if (lane == 31) wsum[warp] = incl;
    __syncthreads();
    if (warp == 0) {
      const unsigned w = wsum[lane];
      unsigned wi = w;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const unsigned t = __shfl_up_sync(0xffffffffu, wi, o); if (lane >= o) wi += t; }
      wsum[lane] = wi - w;
      if (lane == 31) wsum[32] = wi;
    }
    __syncthreads();
    *total = wsum[32];
    return wsum[warp] + incl - v;
  };
  // 1. the 12-bit digit of the cut-off: bins ascend with tid, the select wants the LARGEST keys
  const unsigned hs = h4.x + h4.y + h4.z + h4.w;
  unsigned n_valid;
  const unsigned below = block_scan(hs, &n_valid);
  const unsigned want = min((unsigned)k2, n_valid);
  uint32_t thr = 0xffffffffu;                                // want == 0: nothing reaches the cut-off
  unsigned need_eq = 0;
  if (want > 0) {
    if (tid == 0) s_cnt = 0u;
    unsigned cum = n_valid - below - hs;                     // entries in the bins above this thread's four
    const unsigned hb[4] = {h4.w, h4.z, h4.y, h4.x};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      if (cum < want && want <= cum + hb[i]) { s_prefix = (uint32_t)(4 * tid + 3 - i) << 20; s_need = want - cum; s_m = hb[i]; }
      cum += hb[i];
    }
    __syncthreads();
    const uint32_t top = s_prefix;
    if (s_m <= (unsigned)kL2Cand) {
      // 2. the keys of that bin -> shared memory (any order: only their values matter from here on)
#pragma unroll
      for (int j = 0; j < PER; ++j) {
        const bool is = (key[j] & 0xfff00000u) == top && key[j] != 0u;
        const unsigned bal = __ballot_sync(0xffffffffu, is);
        if (is) {
          const int leader = __ffs(bal) - 1;
          unsigned pos0 = 0;
          if (lane == leader) pos0 = atomicAdd(&s_cnt, (unsigned)__popc(bal));
          pos0 = __shfl_sync(bal, pos0, leader);
          const unsigned idx = pos0 + __popc(bal & ((1u << lane) - 1u));
          if (idx < (unsigned)kL2Cand) cand[idx] = key[j];
        }
      }
      __syncthreads();
      const unsigned m = min(s_cnt, (unsigned)kL2Cand);
      uint32_t ck[kL2Cand / 1024];
#pragma unroll
      for (int j = 0; j < kL2Cand / 1024; ++j) ck[j] = (unsigned)(tid + 1024 * j) < m ? cand[tid + 1024 * j] : ~top;   // padding never matches
      l2_radix_passes(ck, 0xfff00000u, 2, hist, &s_prefix, &s_need, tid, lane, warp);
    } else {
      l2_radix_passes(key, 0xfff00000u, 2, hist, &s_prefix, &s_need, tid, lane, warp);
    }
    thr = s_prefix;
    need_eq = s_need;                                         // how many of the keys == thr are taken (lowest positions)
  }
  // 3. mark
  unsigned n_eq_thr = 0;
#pragma unroll
  for (int j = 0; j < PER; ++j) n_eq_thr += (key[j] == thr);
  unsigned dummy;
  unsigned eq_before = block_scan(n_eq_thr, &dummy);
  uint32_t bits = 0u;
#pragma unroll
  for (int j = 0; j < PER; ++j) {
    bool take = want > 0 && key[j] > thr;
    if (want > 0 && key[j] == thr) { take = eq_before < need_eq; ++eq_before; }
    if (take) bits |= 1u << ((base + j) & 31);
  }
#pragma unroll
  for (int o = 1; o < 32 / PER; o <<= 1) bits |= __shfl_xor_sync(0xffffffffu, bits, o);
  const int word = base >> 5;
  if ((lane & (32 / PER - 1)) == 0 && word < k * 4) mk[word] = bits;
  for (int w = 1024 * PER / 32 + tid; w < k * 4; w += 1024) mk[w] = 0u;
}

// ---- host -------------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct L2Plan {
  L2Init init{};
  EncodeTiledFn encode = nullptr;
  CUtensorMap* d_maps = nullptr;       // [B]
  CUtensorMap map_q{};
  const void* q_cached = nullptr;
  float* score = nullptr;              // [B][k * 128]
  uint32_t* mask = nullptr;            // [B][k][4]
  unsigned* ghist = nullptr;           // [B][4096], all zero between steps
  size_t smem = 0;
};

// [rows][128] bf16 seen as (64 columns, rows, 2 d-blocks): a box lands as [2][box_rows][128 B], 128-byte swizzle
static bool l2_encode(EncodeTiledFn enc, CUtensorMap* m, const void* ptr, uint64_t rows, uint32_t box_rows, std::string* msg) {
  cuuint64_t dims[3] = {64, rows, 2};
  cuuint64_t strides[2] = {(cuuint64_t)kL2CI * 2, 128};
  cuuint32_t box[3] = {64, box_rows, 2};
  cuuint32_t es[3] = {1, 1, 1};
  CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(ptr), dims, strides, box, es,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { *msg = "cuTensorMapEncodeTiled failed with CUresult " + std::to_string((int)r); return false; }
  return true;
}

#define L2_CUDA(expr)                                                               \
  do {                                                                              \
    cudaError_t _e = (expr);                                                        \
    if (_e != cudaSuccess) {                                                        \
      *msg = std::string(#expr) + ": " + cudaGetErrorString(_e);                    \
      return -2;                                                                    \
    }                                                                               \
  } while (0)

bool l2_supported(int dtype, int C, int c_I, int n_h) { return dtype == 1 && C == kL2C && c_I == kL2CI && n_h == kL2H; }

int l2_create(const L2Init& init, L2Plan** out, std::string* msg) {
  L2Plan* pl = new L2Plan();
  pl->init = init;
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) {
    *msg = "cuTensorMapEncodeTiled entry point not found"; delete pl; return -2;
  }
  pl->encode = (EncodeTiledFn)fn;
  const int B = init.B;
  L2_CUDA(cudaMalloc(&pl->score, (size_t)B * init.k * kL2C * sizeof(float)));
  L2_CUDA(cudaMalloc(&pl->mask, (size_t)B * init.k * 4 * sizeof(uint32_t)));
  L2_CUDA(cudaMemset(pl->mask, 0, (size_t)B * init.k * 4 * sizeof(uint32_t)));
  L2_CUDA(cudaMalloc(&pl->ghist, (size_t)B * kL2Bins * sizeof(unsigned)));
  L2_CUDA(cudaMemset(pl->ghist, 0, (size_t)B * kL2Bins * sizeof(unsigned)));
  std::vector<CUtensorMap> maps((size_t)B);
  for (int b = 0; b < B; ++b) {
    const void* ptr = init.index_k[b];
    const long long rows = init.seq_host[b].n_csa;
    if (rows > 0 && !ptr) { *msg = "null index_k pointer"; l2_destroy(pl); return -1; }
    if (!l2_encode(pl->encode, &maps[b], rows > 0 ? ptr : (const void*)pl->score, rows > 0 ? (uint64_t)rows : kL2C, kL2C, msg)) {
      l2_destroy(pl); return -2;
    }
  }
  L2_CUDA(cudaMalloc(&pl->d_maps, maps.size() * sizeof(CUtensorMap)));
  L2_CUDA(cudaMemcpy(pl->d_maps, maps.data(), maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice));
  pl->smem = sizeof(L2Smem) + 1024;
  L2_CUDA(cudaFuncSetAttribute(l2_score_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl->smem));
  *out = pl;
  return 0;
}

const uint32_t* l2_mask(const L2Plan* pl) { return pl->mask; }

void l2_destroy(L2Plan* pl) {
  if (!pl) return;
  cudaFree(pl->d_maps); cudaFree(pl->score); cudaFree(pl->mask); cudaFree(pl->ghist);
  delete pl;
}

int l2_select(L2Plan* pl, const SeqDev* d_seqs, const void* q_idx, const float* w_idx, int32_t* sel_entries, float* sel_score,
              const unsigned* swap_words, cudaStream_t st, int* launches, std::string* msg) {
  const L2Init& in = pl->init;
  if (q_idx != pl->q_cached) {
    if (!l2_encode(pl->encode, &pl->map_q, q_idx, (uint64_t)in.B * kL2H, kL2H, msg)) return -2;
    pl->q_cached = q_idx;
  }
  L2ScoreParams sp{};
  sp.seqs = d_seqs; sp.tbl_chunk = in.tbl_chunk; sp.k_maps = pl->d_maps; sp.w_idx = w_idx; sp.score = pl->score;
  sp.B = in.B; sp.k = in.k;
  L2Swap sw{};
  for (int i = 0; i < 8; ++i) sw.w[i] = sp.swap[i] = swap_words ? swap_words[i] : 0u;
  const int n_max = in.k * kL2C;
  const bool mask_only = !sel_entries && !sel_score && n_max <= 16384;     // keys in registers, no sort
  sp.ghist = mask_only ? pl->ghist : nullptr;
  const long long tiles = (long long)in.B * in.k;
  const int grid = (int)std::max(1ll, std::min<long long>(in.n_sms, tiles));
  L2_CUDA(launch_pdl(l2_score_kernel, dim3(grid), dim3(kL2Threads), pl->smem, st, pl->map_q, sp));
  if (mask_only) {
    const float* sc = pl->score;
    if (n_max <= 4096) L2_CUDA(launch_pdl(l2_topk_mask_kernel<4>, dim3(in.B), dim3(1024), 0, st, d_seqs, sw, sc, pl->ghist, in.k, in.k2, pl->mask));
    else if (n_max <= 8192) L2_CUDA(launch_pdl(l2_topk_mask_kernel<8>, dim3(in.B), dim3(1024), 0, st, d_seqs, sw, sc, pl->ghist, in.k, in.k2, pl->mask));
    else L2_CUDA(launch_pdl(l2_topk_mask_kernel<16>, dim3(in.B), dim3(1024), 0, st, d_seqs, sw, sc, pl->ghist, in.k, in.k2, pl->mask));
  } else {
    L2_CUDA(launch_pdl(l2_topk_kernel, dim3(in.B), dim3(1024), 0, st, d_seqs, sw, in.tbl_chunk, (const float*)pl->score, in.k, in.k2, pl->mask,
                       sel_entries, sel_score));
  }
  *launches += 2;
  return 0;
}

}  // namespace lsa
