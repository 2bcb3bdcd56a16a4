// lsa_select.cuh - block-wide "m smallest of n unique 64-bit keys, sorted" used by
//   S3 top-k      (key = ~ordered(score) << 32 | chunk idx  -> score desc, idx asc; BJ north_star)
//   S4 allocation (key = last_used << 20 | page             -> never-used first, then LRU; R12)
// n <= kSortAll: bitonic sort in shared memory.  Larger n: 8-bit MSB radix select of the m-th key,
// compaction of the m winners, bitonic sort of those.  Deterministic: keys are unique.
#pragma once
#include "lsa_common.cuh"

namespace lsa {

constexpr unsigned long long kKeyMax = 0xffffffffffffffffull;
constexpr int kSortAll = kSortCap;         // up to this many keys the whole set is sorted; above, radix select first

struct SelectSmem {
  unsigned long long keys[kSortCap];
  unsigned int hist[256];
  unsigned long long prefix;
  unsigned long long prefix_mask;
  unsigned int need;
  unsigned int count;
};

__device__ __forceinline__ int next_pow2(int n) {
  int p = 2;
  while (p < n) p <<= 1;
  return p;
}

// ascending bitonic sort of keys[0..n_pad), n_pad a power of two; all threads of the block call it.
// One thread per compare-exchange pair: pair t has i = (bits of t above j shifted up by one) | (bits below j),
// partner i | j.  For j <= 32 the 32 pairs of a warp stay inside one 64-key window, so the six lowest strides of
// every phase need only __syncwarp, not a block barrier (51 of the 66 stages at 2048 keys).
__device__ __forceinline__ void bitonic_cas(unsigned long long* keys, int t, int j, int k) {
  const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
  const int ixj = i | j;
  const unsigned long long a = keys[i], b = keys[ixj];
  const bool up = ((i & k) == 0);
  if ((a > b) == up) { keys[i] = b; keys[ixj] = a; }
}

__device__ inline void block_bitonic_sort(unsigned long long* keys, int n_pad) {
  const int pairs = n_pad >> 1;
  const int pairs_up = (pairs + 31) & ~31;                   // whole warps take part in the warp-level stages
  for (int k = 2; k <= n_pad; k <<= 1) {
    int j = k >> 1;
    for (; j > 32; j >>= 1) {
      for (int t = threadIdx.x; t < pairs; t += blockDim.x) bitonic_cas(keys, t, j, k);
      __syncthreads();
    }
    for (int t = threadIdx.x; t < pairs_up; t += blockDim.x) {
      for (int jj = j; jj > 0; jj >>= 1) {
        if (t < pairs) bitonic_cas(keys, t, jj, k);
        __syncwarp();
      }
    }
    __syncthreads();
  }
}

// Writes the min(m, n) smallest keys, ascending, to sm.keys[0..) and returns that count.
// keyf(i) must be pure.  m <= kSortCap.  kKeyMax is a legal "excluded" sentinel (not unique);
// callers check the returned keys for it.
template <class KeyF>
__device__ inline int block_select_smallest(KeyF keyf, int n, int m, SelectSmem& sm) {
  if (m > n) m = n;
  if (m <= 0) return 0;
  if (n <= kSortAll) {
    int n_pad = next_pow2(n);
    for (int i = threadIdx.x; i < n_pad; i += blockDim.x) sm.keys[i] = i < n ? keyf(i) : kKeyMax;
    __syncthreads();
    block_bitonic_sort(sm.keys, n_pad);
    return m;
  }
  if (threadIdx.x == 0) { sm.prefix = 0; sm.prefix_mask = 0; sm.need = (unsigned)m; }
  for (int byte = 7; byte >= 0; --byte) {
    for (int i = threadIdx.x; i < 256; i += blockDim.x) sm.hist[i] = 0;
    __syncthreads();
    const unsigned long long prefix = sm.prefix, pmask = sm.prefix_mask;
    const int n_round = (n + blockDim.x - 1) / blockDim.x * blockDim.x;   // keep warps converged
    for (int i = threadIdx.x; i < n_round; i += blockDim.x) {
      bool act = false;
      unsigned bin = 0;
      if (i < n) {
        unsigned long long key = keyf(i);
        act = (key & pmask) == prefix;
        bin = (unsigned)(key >> (8 * byte)) & 255u;
      }
      unsigned amask = __ballot_sync(0xffffffffu, act);
      if (act) {                                  // warp-aggregated histogram update
        unsigned peers = __match_any_sync(amask, bin);
        if ((threadIdx.x & 31) == (__ffs(peers) - 1)) atomicAdd(&sm.hist[bin], __popc(peers));
      }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      unsigned need = sm.need, cum = 0;
      int d = 0;
      for (; d < 255; ++d) {
        if (cum + sm.hist[d] >= need) break;
        cum += sm.hist[d];
      }
      sm.need = need - cum;
      sm.prefix = prefix | ((unsigned long long)d << (8 * byte));
      sm.prefix_mask = pmask | (0xffull << (8 * byte));
      sm.count = 0;
    }
    __syncthreads();
  }
  const unsigned long long thr = sm.prefix;       // the m-th smallest key
  for (int i = threadIdx.x; i < n; i += blockDim.x) {
    unsigned long long key = keyf(i);
    if (key <= thr) {
      unsigned pos = atomicAdd(&sm.count, 1u);
      if (pos < (unsigned)kSortCap) sm.keys[pos] = key;
    }
  }
  __syncthreads();
  int got = min((int)sm.count, kSortCap);
  int n_pad = next_pow2(got);
  for (int i = got + threadIdx.x; i < n_pad; i += blockDim.x) sm.keys[i] = kKeyMax;
  __syncthreads();
  block_bitonic_sort(sm.keys, n_pad);
  return min(m, got);
}

// ---- S3 for n <= 4096 scores: histogram select + sort of the winners only ------------------------------------------
// The k best of n scores by (score desc, index asc).  Every thread keeps its (up to 4) order-preserving 32-bit scores
// in registers; three radix levels (12 + 12 + 8 bits, most significant first) each count the keys that still match
// the decided prefix into a shared-memory histogram, a block-wide suffix scan finds the bin holding the k-th best and
// how many keys of that bin are still needed.  After the last level the cut-off score is exact: keys above it win,
// keys AT it win by ascending index (one block scan per register slot, only when the tie really straddles the cut).
// The <= k winners are compacted and sorted (bitonic, mostly warp-level at k <= 128) - instead of sorting all n.
// Writes min(k, n) keys (~ordered(score) << 32 | idx, ascending = best first) to sm.keys and returns their count.
// All 1024 threads of the block call it; n <= 4096, k <= 1024.
constexpr int kTopkBins = 4096;

__device__ inline int block_topk_select(const float* __restrict__ sc, int n, int k, SelectSmem& sm) {
  if (k > n) k = n;
  if (k <= 0) return 0;
  unsigned int* hist = reinterpret_cast<unsigned int*>(sm.keys + 1024);      // 16 KiB behind the 1024 output slots
  unsigned int* wsum = sm.hist;                                              // [32] warp totals, [64..] results
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  unsigned int u[4];
  bool have[4];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const int c = tid + 1024 * j;
    have[j] = c < n;
    u[j] = have[j] ? float_to_ordered(sc[c]) : 0u;
  }
  unsigned int prefix = 0, mask = 0, need = (unsigned)k, eq_total = 0;
#pragma unroll 1
  for (int level = 0; level < 3; ++level) {
    const int shift = level == 0 ? 20 : level == 1 ? 8 : 0;
    const unsigned bins = level == 2 ? 256u : (unsigned)kTopkBins;
    for (int i = tid; i < kTopkBins; i += 1024) hist[i] = 0;
    __syncthreads();
#pragma unroll
    for (int j = 0; j < 4; ++j)
      if (have[j] && (u[j] & mask) == prefix) atomicAdd(&hist[(u[j] >> shift) & (bins - 1)], 1u);
    __syncthreads();
    // suffix counts: thread t owns bins [4t, 4t + 4); above(b) = keys in bins > b
    const unsigned h0 = hist[4 * tid], h1 = hist[4 * tid + 1], h2 = hist[4 * tid + 2], h3 = hist[4 * tid + 3];
    const unsigned mine = h0 + h1 + h2 + h3;
    unsigned incl = mine;                                   // inclusive suffix sum over threads (towards higher t)
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned t = __shfl_down_sync(0xffffffffu, incl, o);
      if (lane + o < 32) incl += t;
    }
    if (lane == 0) wsum[warp] = incl;
    __syncthreads();
    unsigned above_w = 0;
    for (int w = warp + 1; w < 32; ++w) above_w += wsum[w];
    const unsigned above_t = above_w + incl - mine;         // keys in bins of higher threads
    const unsigned a3 = above_t, a2 = a3 + h3, a1 = a2 + h2, a0 = a1 + h1;
    // exactly one bin satisfies above(b) < need <= above(b) + hist[b]
    if (a3 < need && need <= a3 + h3) { wsum[64] = 4 * tid + 3; wsum[65] = need - a3; wsum[66] = h3; }
    else if (a2 < need && need <= a2 + h2) { wsum[64] = 4 * tid + 2; wsum[65] = need - a2; wsum[66] = h2; }
    else if (a1 < need && need <= a1 + h1) { wsum[64] = 4 * tid + 1; wsum[65] = need - a1; wsum[66] = h1; }
    else if (a0 < need && need <= a0 + h0) { wsum[64] = 4 * tid; wsum[65] = need - a0; wsum[66] = h0; }
    __syncthreads();
    prefix |= wsum[64] << shift;
    mask |= (bins - 1) << shift;
    need = wsum[65];
    eq_total = wsum[66];
    __syncthreads();                                        // wsum / hist are rewritten by the next level
    if (eq_total == need) break;                            // the whole cut-off bin is taken: nothing left to decide
  }
  // keys whose decided bits exceed the prefix win; keys that match it: all of them (eq_total == need), or - after the
  // last level, where the match is on all 32 bits, i.e. an exact tie - the `need` lowest indices
  const bool tie = eq_total != need;
  if (tid == 0) sm.count = 0;
  __syncthreads();
  unsigned eq_before = 0;                                   // matching keys with a lower index, slots 0..j-1 of all threads
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const bool m = have[j] && (u[j] & mask) == prefix;
    bool win = have[j] && (u[j] & mask) > prefix;
    if (tie) {                                              // block-wide exclusive count of matches in index order
      const unsigned bal = __ballot_sync(0xffffffffu, m);
      if (lane == 0) wsum[warp] = __popc(bal);
      __syncthreads();
      unsigned below = eq_before;
      for (int w = 0; w < warp; ++w) below += wsum[w];
      unsigned tot = 0;
      for (int w = 0; w < 32; ++w) tot += wsum[w];
      below += __popc(bal & ((1u << lane) - 1));
      win = win || (m && below < need);
      eq_before += tot;
      __syncthreads();
    } else {
      win = win || m;
    }
    if (win) {
      const unsigned pos = atomicAdd(&sm.count, 1u);
      sm.keys[pos] = ((unsigned long long)(~u[j]) << 32) | (unsigned)(tid + 1024 * j);
    }
  }
  __syncthreads();
  const int got = (int)sm.count;                            // == k
  const int n_pad = next_pow2(got);
  for (int i = got + tid; i < n_pad; i += 1024) sm.keys[i] = kKeyMax;
  __syncthreads();
  block_bitonic_sort(sm.keys, n_pad);
  return got;
}

// ---- the m smallest of n <= 4096 UNIQUE 64-bit keys (S4: LRU victims), same scheme ---------------------------------
// Keys live in registers (4 per thread); 12-bit radix levels from the highest bit any key has set (kKeyMax =
// "excluded" is ignored) down, until the cut-off bin is taken whole - unique keys always end there.  The winners are
// compacted and sorted.  Returns the number written to sm.keys (< m if fewer than m keys are not excluded).
template <class KeyF>
__device__ inline int block_select_smallest_hist(KeyF keyf, int n, int m, SelectSmem& sm) {
  if (m > n) m = n;
  if (m <= 0) return 0;
  unsigned int* hist = reinterpret_cast<unsigned int*>(sm.keys + 1024);
  unsigned int* wsum = sm.hist;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  unsigned long long u[4];
  bool have[4];
  unsigned long long any = 0;
  unsigned cnt = 0;
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const int c = tid + 1024 * j;
    u[j] = c < n ? keyf(c) : kKeyMax;
    have[j] = u[j] != kKeyMax;
    if (have[j]) { any |= u[j]; ++cnt; }
  }
  // highest set bit over all keys, and how many keys there are
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { any |= __shfl_xor_sync(0xffffffffu, any, o); cnt += __shfl_xor_sync(0xffffffffu, cnt, o); }
  if (lane == 0) { sm.keys[warp] = any; wsum[warp] = cnt; }
  __syncthreads();
  any = 0; cnt = 0;
  for (int w = 0; w < 32; ++w) { any |= sm.keys[w]; cnt += wsum[w]; }
  __syncthreads();
  if ((unsigned)m > cnt) m = (int)cnt;
  if (m == 0) return 0;
  int top = 64 - __clzll((long long)(any | 1ull));           // bits in use
  unsigned long long prefix = 0, mask = 0;
  unsigned need = (unsigned)m, in_bin = 0;
#pragma unroll 1
  for (int shift = ((top + 11) / 12 - 1) * 12; shift >= 0; shift -= 12) {
    for (int i = tid; i < kTopkBins; i += 1024) hist[i] = 0;
    __syncthreads();
#pragma unroll
    for (int j = 0; j < 4; ++j)
      if (have[j] && (u[j] & mask) == prefix) atomicAdd(&hist[(unsigned)(u[j] >> shift) & (kTopkBins - 1)], 1u);
    __syncthreads();
    // prefix counts: thread t owns bins [4t, 4t + 4); below(b) = keys in bins < b
    const unsigned h0 = hist[4 * tid], h1 = hist[4 * tid + 1], h2 = hist[4 * tid + 2], h3 = hist[4 * tid + 3];
    const unsigned mine = h0 + h1 + h2 + h3;
    unsigned incl = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned t = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += t;
    }
    if (lane == 31) wsum[warp] = incl;
    __syncthreads();
    unsigned below_w = 0;
    for (int w = 0; w < warp; ++w) below_w += wsum[w];
    const unsigned b0 = below_w + incl - mine, b1 = b0 + h0, b2 = b1 + h1, b3 = b2 + h2;
    if (b0 < need && need <= b0 + h0) { wsum[64] = 4 * tid; wsum[65] = need - b0; wsum[66] = h0; }
    else if (b1 < need && need <= b1 + h1) { wsum[64] = 4 * tid + 1; wsum[65] = need - b1; wsum[66] = h1; }
    else if (b2 < need && need <= b2 + h2) { wsum[64] = 4 * tid + 2; wsum[65] = need - b2; wsum[66] = h2; }
    else if (b3 < need && need <= b3 + h3) { wsum[64] = 4 * tid + 3; wsum[65] = need - b3; wsum[66] = h3; }
    __syncthreads();
    prefix |= (unsigned long long)wsum[64] << shift;
    mask |= (unsigned long long)(kTopkBins - 1) << shift;
    need = wsum[65];
    in_bin = wsum[66];
    __syncthreads();
    if (in_bin == need) break;
  }
  if (tid == 0) sm.count = 0;
  __syncthreads();
#pragma unroll
  for (int j = 0; j < 4; ++j)
    if (have[j] && (u[j] & mask) <= prefix) sm.keys[atomicAdd(&sm.count, 1u)] = u[j];
  __syncthreads();
  const int got = (int)sm.count;
  const int n_pad = next_pow2(got);
  for (int i = got + tid; i < n_pad; i += 1024) sm.keys[i] = kKeyMax;
  __syncthreads();
  block_bitonic_sort(sm.keys, n_pad);
  return got;
}

}  // namespace lsa
