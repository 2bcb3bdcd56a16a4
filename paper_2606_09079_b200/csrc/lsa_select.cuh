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

}  // namespace lsa
