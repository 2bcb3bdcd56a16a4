// lsa_residency.cu - S4 residency diff + page allocation, S5 chunk fetch, S6 table swap (sm_100a)
//
//   S4  hits = sel & resident, misses = sel \ resident; every miss gets the unpinned page with the
//       smallest (last_used, page) - never-used pages (last_used 0) first, lowest index first - and
//       its previous owner is evicted.  Pages of any current or staged table are pinned.
//       PAPER.md l.185 (recalled subset lands in the "GPU reserve", page granular), l.187
//       (residency bitmap + remap); BASELINE.json cfg 4 (shared pool, LRU); DESIGN R11-R13.
//   S5  copy each missing chunk (one contiguous page image) from the pinned-host cold pool to its
//       hot-pool page.  PAPER.md l.179/l.185 (CPU cold mirror), l.189 (async recall).
//       Device-pull design: the kernel reads the cold pool through its mapped device address with
//       16-byte loads, so the whole trigger path stays on the device - no host round trip, unlike
//       the host-synchronising Level-1 recall the paper describes (l.187).
//   S6  the staged table becomes the attended one ("materialize ... at step t+1").
//
// The residency pass is one 1024-thread block: the pool is shared by all sequences and the oracle
// semantics are sequential in ascending sequence id, so there is no parallelism across sequences;
// inside one sequence every pass (pin marking, hit lookup, victim selection, table write) is
// block-parallel.
#include <cuda_fp16.h>

#include "lsa_kernels.h"
#include "lsa_select.cuh"

namespace lsa {

struct ResSmem {
  SelectSmem sel;
  int sel_up[kMaxK];      // selection sorted by chunk id
  int next_page[kMaxK];
  int miss_rank[kMaxK];   // rank among misses or -1 for a hit
  int warp_cnt[32];
  int n_sel;
  int n_miss;
  unsigned long long tick;
  unsigned int epoch;
  // several sequences firing together on a full pool (P <= kSortCap): the unpinned pages sorted ONCE by (last_used, page)
  int order[kSortCap];    // their page ids in that order
  int victim[kMaxK];      // pages taken by the current sequence's misses, in miss order
  int n_order, cursor, use_order, took, advance;
};

__global__ void __launch_bounds__(1024)
residency_kernel(SeqDev* __restrict__ seqs, PoolDev pool, FireList fire, const int32_t* __restrict__ sel_idx,
                 int B, int k, int P, long long page_bytes, int k_cap, int C) {
  // P = pages the LRU manages, k_cap = recalled chunks per table at most (a growing context keeps 2 B pages and two table
  // slots per sequence for the decode tier, DESIGN R32 / R33)
  extern __shared__ __align__(16) unsigned char smem_raw[];
  ResSmem& sm = *reinterpret_cast<ResSmem*>(smem_raw);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  pdl_wait();
  pdl_launch_dependents();
  if (tid == 0) pool.counters[C_FETCH_COUNT] = 0;
  __syncthreads();

  // ---- several sequences fire together and never-used pages will not cover them: order the unpinned pages ONCE ----
  // A pass only ever touches pages it then lists in its staged table, and staged tables are pinned for every later pass
  // of the launch; untouched pages keep their (last_used, page) key.  So the victims of the whole launch are consumed
  // front to back from ONE sorted list of the pages that are unpinned when the launch starts: sequence b takes the first
  // n_miss(b) entries behind the cursor that have not been pinned since (its own hits, which may sit anywhere in the
  // list).  The per-sequence work shrinks to a hit pass and one scan of a window of the list; the result is the
  // sequential one (DESIGN R12).  Needs: no firing sequence with an unswapped staged table of its own (that table would
  // have to be unpinned for its own pass only - the general path below handles it).
  if (tid == 0) {
    bool ok = fire.n >= 2 && P <= kSortCap && blockDim.x == 1024;
    const long long n_used = (long long)(pool.counters[C_MISSES] - pool.counters[C_EVICTIONS]);
    if (ok && n_used + (long long)fire.n * k_cap <= (long long)P) ok = false;        // index arithmetic will do
    for (int fi = 0; ok && fi < fire.n; ++fi) ok = seqs[fire.ids[fi]].pending == 0;
    sm.use_order = ok ? 1 : 0;
    if (ok) sm.epoch = ++(*pool.epoch);
    sm.cursor = 0;
  }
  __syncthreads();
  const bool use_order = sm.use_order != 0;
  if (use_order) {
    const unsigned int epoch = sm.epoch;
    for (int idx = tid; idx < B * 2 * k; idx += blockDim.x) {
      int bb = idx / (2 * k), r = idx % (2 * k), buf = r / k, j = r % k;
      const SeqDev& o = seqs[bb];
      const bool live = buf == o.cur_buf || o.pending != 0;
      if (live && j < o.n_tbl[buf]) {
        const int pg = pool.tbl_page[((size_t)bb * 2 + buf) * k + j];
        if (pg < P) pool.pin_mark[pg] = epoch;                    // (tier pages of a growing context lie beyond P)
      }
    }
    __syncthreads();
    const int n_pad = next_pow2(P);
    int mine = 0;
    for (int i = tid; i < n_pad; i += blockDim.x) {
      unsigned long long key = kKeyMax;
      if (i < P && pool.pin_mark[i] != epoch) { key = (pool.last_used[i] << kPageBits) | (unsigned long long)i; ++mine; }
      sm.sel.keys[i] = key;
    }
    mine = __reduce_add_sync(0xffffffffu, mine);
    if (lane == 0) sm.warp_cnt[warp] = mine;
    __syncthreads();
    block_bitonic_sort(sm.sel.keys, n_pad);
    if (tid == 0) {
      int n = 0;
      for (int w = 0; w < 32; ++w) n += sm.warp_cnt[w];
      sm.n_order = n;
    }
    for (int i = tid; i < n_pad; i += blockDim.x) sm.order[i] = (int)(sm.sel.keys[i] & ((1ull << kPageBits) - 1));
    __syncthreads();
  }
  // ... and all the selections in one go: key = (position in the fire list, chunk id), invalid ids last in their segment
  const int k_pad = next_pow2(k);
  const bool pre_sorted = use_order && fire.n * k_pad <= kSortCap;
  if (pre_sorted) {
    const int total = fire.n * k_pad, total_pad = next_pow2(total);
    for (int i = tid; i < total_pad; i += blockDim.x) {
      unsigned long long key = kKeyMax;
      if (i < total) {
        const int fi = i / k_pad, j = i - fi * k_pad;
        const int c = j < k ? sel_idx[(size_t)fi * k + j] : -1;
        const bool valid = c >= 0 && c < seqs[fire.ids[fi]].n_chunks;
        key = ((unsigned long long)fi << 32) | (valid ? (unsigned)c : 0xffffffffu);
      }
      sm.sel.keys[i] = key;
    }
    __syncthreads();
    block_bitonic_sort(sm.sel.keys, total_pad);
  }

  for (int fi = 0; fi < fire.n; ++fi) {
    const int b = fire.ids[fi];
    SeqDev& sq = seqs[b];
    const int* my_sel = sel_idx + (size_t)fi * k;

    // ---- selection -> ascending chunk id (R13) ----
    if (pre_sorted) {
      const bool valid = tid < k_pad && (unsigned)sm.sel.keys[fi * k_pad + tid] != 0xffffffffu;
      const int n = __syncthreads_count(valid);            // valid ids sort first inside the segment
      if (valid) sm.sel_up[tid] = (int)(unsigned)sm.sel.keys[fi * k_pad + tid];
      if (tid == 0) {
        sm.n_sel = n;
        sm.tick = pool.counters[C_TICK] + 1;
      }
      __syncthreads();
    } else {
      int n_pad = next_pow2(k);
      for (int i = tid; i < n_pad; i += blockDim.x) {
        int c = (i < k) ? my_sel[i] : -1;
        sm.sel.keys[i] = (c >= 0 && c < sq.n_chunks) ? (unsigned long long)c : kKeyMax;
      }
      __syncthreads();
      block_bitonic_sort(sm.sel.keys, n_pad);
      // valid ids sort first: their number = keys that are not the sentinel (one block-wide count, not a serial scan)
      int mine = 0;
      for (int i = tid; i < k; i += blockDim.x) mine += sm.sel.keys[i] != kKeyMax;
      mine = __reduce_add_sync(0xffffffffu, mine);
      if (lane == 0) sm.warp_cnt[warp] = mine;
      __syncthreads();
      if (tid == 0) {
        int n = 0;
        for (int w = 0; w < 32; ++w) n += sm.warp_cnt[w];
        sm.n_sel = n;
        sm.tick = pool.counters[C_TICK] + 1;     // committed below, once the pass is known to succeed
        if (!use_order) sm.epoch = ++(*pool.epoch);   // scratch stamp of pin_mark: harmless if the pass is abandoned
      }
      __syncthreads();
      for (int i = tid; i < sm.n_sel; i += blockDim.x) sm.sel_up[i] = (int)sm.sel.keys[i];
      __syncthreads();
    }
    const int n_sel = sm.n_sel;
    const unsigned long long tick = sm.tick;
    const unsigned int epoch = sm.epoch;
    if (n_sel > k_cap) {                           // an explicit selection larger than the table's recalled share
      if (tid == 0) pool.counters[C_ERROR] = 2;
      __syncthreads();
      continue;
    }

    // ---- pin every page of a current table and of other sequences' staged tables ----
    for (int idx = tid; !use_order && idx < B * 2 * k; idx += blockDim.x) {
      int bb = idx / (2 * k), r = idx % (2 * k), buf = r / k, j = r % k;
      const SeqDev& o = seqs[bb];
      bool is_cur = (buf == o.cur_buf);
      bool live = is_cur ? true : (o.pending != 0 && bb != b);   // this sequence's own unswapped staged table is superseded
      if (live && j < o.n_tbl[buf]) pool.pin_mark[pool.tbl_page[((size_t)bb * 2 + buf) * k + j]] = epoch;
    }
    __syncthreads();

    // ---- pass 1: hits ----
    int my_miss = 0;
    if (tid < n_sel) {
      int c = sm.sel_up[tid];
      int p = pool.page_of[sq.page_of_off + c];
      if (p >= 0) {
        pool.pin_mark[p] = epoch;
        sm.next_page[tid] = p;
      } else {
        my_miss = 1;
      }
    }
    // block exclusive scan of my_miss over tid < kMaxK (1024 threads = 32 warps)
    unsigned bal = __ballot_sync(0xffffffffu, my_miss);
    int wpre = __popc(bal & ((1u << lane) - 1));
    if (lane == 0) sm.warp_cnt[warp] = __popc(bal);
    __syncthreads();
    if (warp == 0) {
      int v = sm.warp_cnt[lane];
      int incl = v;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
      }
      sm.warp_cnt[lane] = incl - v;
      if (lane == 31) sm.n_miss = incl;
    }
    __syncthreads();
    if (tid < n_sel) sm.miss_rank[tid] = my_miss ? (sm.warp_cnt[warp] + wpre) : -1;
    const int n_miss = sm.n_miss;
    __syncthreads();

    // ---- pass 2: the n_miss smallest (last_used, page) among unpinned pages ----
    // Pages never return to the never-used state and never-used pages (last_used = 0) sort first, lowest index
    // first, so the used pages are always the prefix [0, n_used) with n_used = misses - evictions so far.  While
    // enough never-used pages are left, the victims are simply the next n_miss indices (no scan of the pool).
    bool fast = true;
    long long n_used = 0;
    if (n_miss > 0 && use_order) {
      // the first n_miss entries behind the cursor that are still unpinned, window by window
      int need = n_miss, got = 0;
      bool short_of_pages = false;
      while (need > 0) {
        const int cur = sm.cursor, pos = cur + tid;
        const bool in = pos < sm.n_order;
        const int pg = in ? sm.order[pos] : -1;
        const bool free_pg = in && pool.pin_mark[pg] != epoch;
        const unsigned balf = __ballot_sync(0xffffffffu, free_pg);
        const int wpre_f = __popc(balf & ((1u << lane) - 1));
        __syncthreads();                                   // warp_cnt / took / advance of the previous round are consumed
        if (lane == 0) sm.warp_cnt[warp] = __popc(balf);
        __syncthreads();
        int below = 0;
        for (int w = 0; w < warp; ++w) below += sm.warp_cnt[w];
        const int rank = below + wpre_f;
        if (free_pg && rank < need) sm.victim[got + rank] = pg;
        if (free_pg && rank == need - 1) sm.advance = tid + 1;      // the window is satisfied here
        if (tid == 1023) { sm.took = rank + (free_pg ? 1 : 0); }
        __syncthreads();
        const int took = min(sm.took, need);
        if (sm.took >= need) { if (tid == 0) sm.cursor = cur + sm.advance; need = 0; }
        else {
          if (cur + 1024 >= sm.n_order) { short_of_pages = true; break; }
          if (tid == 0) sm.cursor = cur + 1024;
          need -= took; got += took;
        }
        __syncthreads();
      }
      if (short_of_pages) {
        if (tid == 0) pool.counters[C_ERROR] = 1;
        __syncthreads();
        continue;
      }
      __syncthreads();
      const unsigned long long base = pool.counters[C_FETCH_COUNT];
      if (tid < n_sel && sm.miss_rank[tid] >= 0) {
        const int r = sm.miss_rank[tid];
        const int c = sm.sel_up[tid];
        const int p = sm.victim[r];
        const int ob = pool.owner_seq[p];
        if (ob >= 0) {
          pool.page_of[seqs[ob].page_of_off + pool.owner_chunk[p]] = -1;
          atomicAdd(&pool.counters[C_EVICTIONS], 1ull);
        }
        pool.owner_seq[p] = b;
        pool.owner_chunk[p] = c;
        pool.page_of[sq.page_of_off + c] = p;
        pool.last_used[p] = tick;
        pool.pin_mark[p] = epoch;
        sm.next_page[tid] = p;
        pool.fetch_src[base + r] = reinterpret_cast<const unsigned char*>(sq.cold) + (long long)c * page_bytes;
        pool.fetch_page[base + r] = p;
        if (sq.cold_scale) pool.fetch_scale[base + r] = sq.cold_scale + 2 * (size_t)c;
      }
    } else if (n_miss > 0) {
      n_used = (long long)(pool.counters[C_MISSES] - pool.counters[C_EVICTIONS]);
      fast = n_used + n_miss <= (long long)P;
      if (!fast) {
        const unsigned long long* lu = pool.last_used;
        const unsigned int* pm = pool.pin_mark;
        auto keyf = [lu, pm, epoch](int p) -> unsigned long long {
          return pm[p] == epoch ? kKeyMax : ((lu[p] << kPageBits) | (unsigned long long)p);
        };
        // pools of up to 4096 pages: histogram select + sort of the victims only (the full sort took ~20 us per sequence)
        int got = (P <= 4096 && blockDim.x == 1024) ? block_select_smallest_hist(keyf, P, n_miss, sm.sel)
                                                    : block_select_smallest(keyf, P, n_miss, sm.sel);
        __syncthreads();
        bool bad = (got < n_miss) || (sm.sel.keys[n_miss - 1] == kKeyMax);
        if (bad) {
          // pool exhausted: nothing has been changed yet (pin_mark / epoch are scratch) - tables, residency, LRU
          // stamps and counters stay as they were; lsa_sync / lsa_get_stats report the error
          if (tid == 0) pool.counters[C_ERROR] = 1;
          __syncthreads();
          continue;
        }
      }
      const unsigned long long base = pool.counters[C_FETCH_COUNT];
      if (tid < n_sel && sm.miss_rank[tid] >= 0) {
        const int r = sm.miss_rank[tid];
        const int c = sm.sel_up[tid];
        const int p = fast ? (int)n_used + r : (int)(sm.sel.keys[r] & ((1ull << kPageBits) - 1));
        const int ob = pool.owner_seq[p];
        if (ob >= 0) {
          pool.page_of[seqs[ob].page_of_off + pool.owner_chunk[p]] = -1;
          atomicAdd(&pool.counters[C_EVICTIONS], 1ull);
        }
        pool.owner_seq[p] = b;
        pool.owner_chunk[p] = c;
        pool.page_of[sq.page_of_off + c] = p;
        pool.last_used[p] = tick;
        sm.next_page[tid] = p;
        pool.fetch_src[base + r] = reinterpret_cast<const unsigned char*>(sq.cold) + (long long)c * page_bytes;
        pool.fetch_page[base + r] = p;
        if (sq.cold_scale) pool.fetch_scale[base + r] = sq.cold_scale + 2 * (size_t)c;
      }
    }
    __syncthreads();

    // ---- the pass succeeds: commit the tick, the hits' LRU stamps, and stage the next table (ascending chunk id) ----
    if (tid < n_sel && sm.miss_rank[tid] < 0) pool.last_used[sm.next_page[tid]] = tick;
    if (tid == 0) {
      pool.counters[C_TICK] = tick;
      pool.counters[C_TRIGGERS] += 1;
    }
    const int buf = 1 - sq.cur_buf;
    if (tid < n_sel) {
      pool.tbl_chunk[((size_t)b * 2 + buf) * k + tid] = sm.sel_up[tid];
      pool.tbl_page[((size_t)b * 2 + buf) * k + tid] = sm.next_page[tid];
    }
    if (tid == 0) {
      int n_tbl = n_sel;
      if (sq.tier_page0 >= 0 && sq.n_csa % C != 0) {
        // the tail chunk (being filled by lsa_append_compressed) is always attended: its entry follows the recalled ones.
        // Chunks completed since are not listed: this trigger saw them as candidates (DESIGN R31).
        const int c = (int)(sq.n_csa / C);
        pool.tbl_chunk[((size_t)b * 2 + buf) * k + n_tbl] = c;
        pool.tbl_page[((size_t)b * 2 + buf) * k + n_tbl] = sq.tier_page0 + (c & 1);
        n_tbl += 1;
      }
      sq.n_tbl[buf] = n_tbl;
      sq.pending = 1;
      pool.counters[C_FETCH_COUNT] += n_miss;
      pool.counters[C_MISSES] += n_miss;
      pool.counters[C_HITS] += n_sel - n_miss;
      pool.counters[C_BYTES] += (unsigned long long)n_miss * (unsigned long long)page_bytes;
    }
    __syncthreads();
  }
}

// ---- S5: device-pull fetch ----------------------------------------------------------------
constexpr int kFetchThreads = 256;
constexpr int kFetchUnroll = 4;                                  // 16-byte loads in flight per thread
constexpr int kFetchSlice = kFetchThreads * kFetchUnroll * 16;   // 16 KiB per (page, slice) item

__device__ __forceinline__ uint4 ld_stream16(const uint4* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}

__global__ void __launch_bounds__(kFetchThreads)
fetch_kernel(PoolDev pool, unsigned char* __restrict__ hot_pool, long long page_bytes) {
  pdl_wait();                      // the fetch list of the residency pass is complete
  const int n_fetch = (int)pool.counters[C_FETCH_COUNT];
  const int slices = (int)((page_bytes + kFetchSlice - 1) / kFetchSlice);
  const long long items = (long long)n_fetch * slices;
  for (long long it = blockIdx.x; it < items; it += gridDim.x) {
    const int f = (int)(it / slices), s = (int)(it % slices);
    const unsigned char* src = reinterpret_cast<const unsigned char*>(pool.fetch_src[f]) + (long long)s * kFetchSlice;
    unsigned char* dst = hot_pool + (long long)pool.fetch_page[f] * page_bytes + (long long)s * kFetchSlice;
    const long long left = page_bytes - (long long)s * kFetchSlice;
    uint4 v[kFetchUnroll];
#pragma unroll
    for (int u = 0; u < kFetchUnroll; ++u) {
      long long off = ((long long)u * kFetchThreads + threadIdx.x) * 16;
      if (off < left) v[u] = ld_stream16(reinterpret_cast<const uint4*>(src + off));
    }
#pragma unroll
    for (int u = 0; u < kFetchUnroll; ++u) {
      long long off = ((long long)u * kFetchThreads + threadIdx.x) * 16;
      if (off < left) *reinterpret_cast<uint4*>(dst + off) = v[u];
    }
  }
}

// ---- S5 with FP8 (e4m3) cold pages (DESIGN R34): half the bytes cross the host link, the hot page is bf16 as before ----
// hot element = bf16_rne(fp32(code) * scale): the code is widened exactly (e4m3 -> f16 -> f32), one fp32 multiply, one
// rounding.  16 codes per 16-byte load become two 16-byte stores.
__device__ __forceinline__ uint32_t e4m3x2_to_bf16x2(uint32_t two_codes, float scale) {
  uint32_t h2;
  asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h2) : "h"((unsigned short)two_codes));
  const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&h2));
  const __nv_bfloat162 b = __floats2bfloat162_rn(f.x * scale, f.y * scale);
  return *reinterpret_cast<const uint32_t*>(&b);
}

__global__ void __launch_bounds__(kFetchThreads)
fetch_fp8_kernel(PoolDev pool, unsigned char* __restrict__ hot_pool, long long page_bytes, long long cold_page_bytes) {
  pdl_wait();                      // the fetch list of the residency pass is complete
  const int n_fetch = (int)pool.counters[C_FETCH_COUNT];
  const int slices = (int)((cold_page_bytes + kFetchSlice - 1) / kFetchSlice);
  const long long items = (long long)n_fetch * slices, half = cold_page_bytes / 2;     // K block | V block
  for (long long it = blockIdx.x; it < items; it += gridDim.x) {
    const int f = (int)(it / slices), s = (int)(it % slices);
    const unsigned char* src = reinterpret_cast<const unsigned char*>(pool.fetch_src[f]) + (long long)s * kFetchSlice;
    unsigned char* dst = hot_pool + (long long)pool.fetch_page[f] * page_bytes + 2ll * s * kFetchSlice;
    const long long left = cold_page_bytes - (long long)s * kFetchSlice;
    const float sk = __ldg(pool.fetch_scale[f]), sv = __ldg(pool.fetch_scale[f] + 1);
    uint4 v[kFetchUnroll];
#pragma unroll
    for (int u = 0; u < kFetchUnroll; ++u) {
      long long off = ((long long)u * kFetchThreads + threadIdx.x) * 16;
      if (off < left) v[u] = ld_stream16(reinterpret_cast<const uint4*>(src + off));
    }
#pragma unroll
    for (int u = 0; u < kFetchUnroll; ++u) {
      long long off = ((long long)u * kFetchThreads + threadIdx.x) * 16;
      if (off < left) {
        const float sc = ((long long)s * kFetchSlice + off) < half ? sk : sv;
        const uint32_t w[4] = {v[u].x, v[u].y, v[u].z, v[u].w};
        uint32_t o[8];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          o[2 * j] = e4m3x2_to_bf16x2(w[j] & 0xffffu, sc);
          o[2 * j + 1] = e4m3x2_to_bf16x2(w[j] >> 16, sc);
        }
        uint4* d = reinterpret_cast<uint4*>(dst + 2 * off);
        d[0] = make_uint4(o[0], o[1], o[2], o[3]);
        d[1] = make_uint4(o[4], o[5], o[6], o[7]);
      }
    }
  }
}

// ---- export with FP8 cold pages: quantise (DESIGN R35).  One block per (page, K | V block): the largest magnitude's
// exponent field gives e (max * 2^-e in [128, 256)), scale = 2^e, code = e4m3_rne(x * 2^-e) (the product is exact).
__global__ void __launch_bounds__(256)
export_fp8_kernel(const __nv_bfloat16* __restrict__ src, unsigned char* __restrict__ dst, float* __restrict__ scales, long long block_elems) {
  __shared__ unsigned int wmax[8];
  __shared__ float s_inv, s_scale;
  const long long blk = blockIdx.x;
  const __nv_bfloat16* x = src + blk * block_elems;
  unsigned char* out = dst + blk * block_elems;
  unsigned int mx = 0;                                     // |x| as bf16 bits: integer order = magnitude order
  for (long long i = (long long)threadIdx.x * 8; i < block_elems; i += 256 * 8) {
    const uint4 r = *reinterpret_cast<const uint4*>(x + i);
    const uint32_t w[4] = {r.x, r.y, r.z, r.w};
#pragma unroll
    for (int j = 0; j < 4; ++j) { mx = max(mx, w[j] & 0x7fffu); mx = max(mx, (w[j] >> 16) & 0x7fffu); }
  }
  mx = __reduce_max_sync(0xffffffffu, mx);
  if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = mx;
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned int m = 0;
    for (int w = 0; w < 8; ++w) m = max(m, wmax[w]);
    const int field = (int)(m >> 7) & 0xff;                // bf16: 8 exponent bits above 7 mantissa bits
    int e = field == 0 ? 0 : field - 127 - 7;
    e = max(-120, min(120, e));
    s_scale = __uint_as_float((unsigned)(e + 127) << 23);
    s_inv = __uint_as_float((unsigned)(127 - e) << 23);
    scales[blk] = s_scale;
  }
  __syncthreads();
  const float inv = s_inv;
  for (long long i = (long long)threadIdx.x * 16; i < block_elems; i += 256 * 16) {
    const uint4 r0 = *reinterpret_cast<const uint4*>(x + i), r1 = *reinterpret_cast<const uint4*>(x + i + 8);
    const uint32_t w[8] = {r0.x, r0.y, r0.z, r0.w, r1.x, r1.y, r1.z, r1.w};
    uint32_t o[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      uint32_t acc = 0;
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const uint32_t ww = w[2 * j + h];
        const float lo = __uint_as_float(ww << 16) * inv, hi = __uint_as_float(ww & 0xffff0000u) * inv;
        unsigned short c2;
        asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(c2) : "f"(hi), "f"(lo));   // first operand -> upper byte
        acc |= (uint32_t)c2 << (16 * h);
      }
      o[j] = acc;
    }
    *reinterpret_cast<uint4*>(out + i) = make_uint4(o[0], o[1], o[2], o[3]);
  }
}

cudaError_t launch_export_fp8(const void* src, void* dst_mapped, float* scales, long long n_blocks, long long block_elems, cudaStream_t st) {
  export_fp8_kernel<<<(unsigned)n_blocks, 256, 0, st>>>(reinterpret_cast<const __nv_bfloat16*>(src), reinterpret_cast<unsigned char*>(dst_mapped),
                                                        scales, block_elems);
  return cudaGetLastError();
}

// ---- NEXT-4 (first half): KV export, HBM -> pinned-host cold pool ("P-server streams full KV into D's pinned host
// memory"; P:199 VRAM -> DRAM).  The mirror image of fetch_kernel: 16-byte stores over the mapped pinned pool, the
// loads of a slice all in flight before its stores.
__global__ void __launch_bounds__(kFetchThreads)
export_kernel(const unsigned char* __restrict__ src, unsigned char* __restrict__ dst, long long bytes) {
  const long long slice = (long long)kFetchUnroll * kFetchThreads * 16;
  for (long long base = (long long)blockIdx.x * slice; base < bytes; base += (long long)gridDim.x * slice) {
    uint4 v[kFetchUnroll];
#pragma unroll
    for (int u = 0; u < kFetchUnroll; ++u) {
      const long long off = base + ((long long)u * kFetchThreads + threadIdx.x) * 16;
      if (off < bytes) v[u] = *reinterpret_cast<const uint4*>(src + off);
    }
#pragma unroll
    for (int u = 0; u < kFetchUnroll; ++u) {
      const long long off = base + ((long long)u * kFetchThreads + threadIdx.x) * 16;
      if (off < bytes) *reinterpret_cast<uint4*>(dst + off) = v[u];
    }
  }
}

cudaError_t launch_export(const void* src, void* dst_mapped, long long bytes, int n_ctas, cudaStream_t st) {
  export_kernel<<<n_ctas, kFetchThreads, 0, st>>>(reinterpret_cast<const unsigned char*>(src), reinterpret_cast<unsigned char*>(dst_mapped), bytes);
  return cudaGetLastError();
}

// ---- S6 + window append ---------------------------------------------------------------------
// The swap mask is passed BY VALUE (32 words = up to 1024 sequences): a step needs no extra copy.
struct SwapWords { uint32_t w[32]; };

template <typename T>
__global__ void __launch_bounds__(128)
prestep_kernel_v(SeqDev* __restrict__ seqs, int D, int W, SwapWords sw, int use_swap,
                 const T* __restrict__ k_new, const T* __restrict__ v_new) {
  const int b = blockIdx.x;
  SeqDev& sq = seqs[b];
  const bool swap = use_swap && ((sw.w[(b >> 5) & 31] >> (b & 31)) & 1u);
  if (k_new) {
    const int slot = sq.w_head;
    T* kd = reinterpret_cast<T*>(sq.win_k) + (size_t)slot * D;
    T* vd = reinterpret_cast<T*>(sq.win_v) + (size_t)slot * D;
    constexpr int V = Elem<T>::kVec;
    for (int d = threadIdx.x * V; d < D; d += blockDim.x * V) {
      *reinterpret_cast<uint4*>(kd + d) = *reinterpret_cast<const uint4*>(k_new + (size_t)b * D + d);
      *reinterpret_cast<uint4*>(vd + d) = *reinterpret_cast<const uint4*>(v_new + (size_t)b * D + d);
    }
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    if (swap && sq.pending) {
      sq.cur_buf = 1 - sq.cur_buf;
      sq.pending = 0;
    }
    if (k_new) {
      const int slot = sq.w_head;
      sq.w_head = (slot + 1 == W) ? 0 : slot + 1;
      sq.w_len = min(W, sq.w_len + 1);
      sq.app_epoch += 1;         // visible with the row: this launch is stream-ordered before its readers
    }
  }
}

// ---- NEXT-4 (second half): decoded tokens' compressed entries (P:185 tier 3; DESIGN R29-R33) ------------------
// One block per listed sequence; row = row0 + blockIdx.x of the caller's [n][D] / [n][E] arrays.  The entry becomes row
// n_csa % C of the tail chunk's reserved page; a new tail chunk gets its table entries (current table, and the staged one
// if a swap is pending: the host has made the side band finish first); a completed chunk gets its embedding row and
// becomes a candidate.  The records change after the rows are written; readers are later launches on the same stream.
template <typename T>
__global__ void __launch_bounds__(128)
append_compressed_kernel(SeqDev* __restrict__ seqs, PoolDev pool, unsigned char* __restrict__ hot_pool, AppendList list, int row0,
                         const T* __restrict__ csa_k, const T* __restrict__ csa_v, const T* __restrict__ hca_k,
                         const T* __restrict__ hca_v, const T* __restrict__ emb_rows, int D, int E, int C, int k, int k_sel,
                         long long page_bytes) {
  const int b = list.ids[blockIdx.x], row = row0 + blockIdx.x;
  SeqDev& sq = seqs[b];
  constexpr int V = Elem<T>::kVec;
  const long long n = list.n_csa[blockIdx.x];
  const int n_hca = list.n_hca[blockIdx.x];
  const int c = (int)(n / C), i = (int)(n % C);
  if (hca_k) {
    T* kd = reinterpret_cast<T*>(const_cast<void*>(sq.hca_k)) + (size_t)n_hca * D;
    T* vd = reinterpret_cast<T*>(const_cast<void*>(sq.hca_v)) + (size_t)n_hca * D;
    for (int d = threadIdx.x * V; d < D; d += blockDim.x * V) {
      *reinterpret_cast<uint4*>(kd + d) = *reinterpret_cast<const uint4*>(hca_k + (size_t)row * D + d);
      *reinterpret_cast<uint4*>(vd + d) = *reinterpret_cast<const uint4*>(hca_v + (size_t)row * D + d);
    }
  }
  const int page = sq.tier_page0 + (c & 1);
  if (csa_k) {
    T* pg = reinterpret_cast<T*>(hot_pool + (long long)page * page_bytes);
    T* kd = pg + (size_t)i * D;
    T* vd = pg + (size_t)C * D + (size_t)i * D;
    for (int d = threadIdx.x * V; d < D; d += blockDim.x * V) {
      *reinterpret_cast<uint4*>(kd + d) = *reinterpret_cast<const uint4*>(csa_k + (size_t)row * D + d);
      *reinterpret_cast<uint4*>(vd + d) = *reinterpret_cast<const uint4*>(csa_v + (size_t)row * D + d);
    }
    if (i == C - 1) {                           // the entry completes chunk c: its embedding row
      T* ed = reinterpret_cast<T*>(const_cast<void*>(sq.emb)) + (size_t)c * E;
      for (int e = threadIdx.x * V; e < E; e += blockDim.x * V)
        *reinterpret_cast<uint4*>(ed + e) = *reinterpret_cast<const uint4*>(emb_rows + (size_t)row * E + e);
    }
  }
  asm volatile("fence.proxy.async;" ::: "memory");   // the rows are read by TMA (async proxy) in later launches
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) {
    if (hca_k) sq.n_hca = n_hca + 1;
    if (csa_k) {
      if (i == 0) {                             // a new tail chunk: listed after everything else (its id is the largest)
        const int cur = sq.cur_buf;
        int m = sq.n_tbl[cur];
        pool.tbl_chunk[((size_t)b * 2 + cur) * k + m] = c;
        pool.tbl_page[((size_t)b * 2 + cur) * k + m] = page;
        sq.n_tbl[cur] = m + 1;
        if (sq.pending) {
          m = sq.n_tbl[1 - cur];
          pool.tbl_chunk[((size_t)b * 2 + 1 - cur) * k + m] = c;
          pool.tbl_page[((size_t)b * 2 + 1 - cur) * k + m] = page;
          sq.n_tbl[1 - cur] = m + 1;
        }
      }
      sq.n_csa = n + 1;
      if (i == C - 1) {
        sq.n_chunks = c + 1;
        sq.k_eff = min(k_sel, c + 1);
      }
    }
    // a launch that runs beside this kernel (lsa_attn_tc_small.cuh, grow_wait) reads the rows only after this
    __threadfence();
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(&sq.grow_epoch), "r"(list.epoch[blockIdx.x]) : "memory");
  }
}

cudaError_t launch_append_compressed(int dtype, SeqDev* seqs, PoolDev pool, void* hot_pool, const AppendList& list, int row0,
                                     const void* csa_k, const void* csa_v, const void* hca_k, const void* hca_v, const void* emb_rows,
                                     int D, int E, int C, int k, int k_sel, long long page_bytes, cudaStream_t st, bool beside_previous) {
  unsigned char* hp = reinterpret_cast<unsigned char*>(hot_pool);
  if (beside_previous && dtype != 0)          // no griddepcontrol.wait inside: it touches nothing a launch in flight reads unmasked
    return launch_pdl(append_compressed_kernel<__nv_bfloat16>, dim3(list.n), dim3(128), 0, st, seqs, pool, hp, list, row0,
                      (const __nv_bfloat16*)csa_k, (const __nv_bfloat16*)csa_v, (const __nv_bfloat16*)hca_k, (const __nv_bfloat16*)hca_v,
                      (const __nv_bfloat16*)emb_rows, D, E, C, k, k_sel, page_bytes);
  if (dtype == 0)
    append_compressed_kernel<float><<<list.n, 128, 0, st>>>(seqs, pool, hp, list, row0, (const float*)csa_k, (const float*)csa_v,
                                                            (const float*)hca_k, (const float*)hca_v, (const float*)emb_rows, D, E,
                                                            C, k, k_sel, page_bytes);
  else
    append_compressed_kernel<__nv_bfloat16><<<list.n, 128, 0, st>>>(
        seqs, pool, hp, list, row0, (const __nv_bfloat16*)csa_k, (const __nv_bfloat16*)csa_v, (const __nv_bfloat16*)hca_k,
        (const __nv_bfloat16*)hca_v, (const __nv_bfloat16*)emb_rows, D, E, C, k, k_sel, page_bytes);
  return cudaGetLastError();
}

cudaError_t launch_residency(SeqDev* seqs, PoolDev pool, const FireList& fire, const int32_t* sel_idx, int B, int k,
                             int P, long long page_bytes, cudaStream_t st, int k_cap, int C) {
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(residency_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)sizeof(ResSmem));
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  return launch_pdl(residency_kernel, dim3(1), dim3(1024), sizeof(ResSmem), st, seqs, pool, fire, sel_idx, B, k, P, page_bytes, k_cap > 0 ? k_cap : k,
                    C > 0 ? C : 1);
}

cudaError_t launch_fetch(PoolDev pool, void* hot_pool, long long page_bytes, int n_ctas, cudaStream_t st, long long cold_page_bytes) {
  if (cold_page_bytes != page_bytes)
    return launch_pdl(fetch_fp8_kernel, dim3(n_ctas), dim3(kFetchThreads), 0, st, pool, reinterpret_cast<unsigned char*>(hot_pool), page_bytes,
                      cold_page_bytes);
  return launch_pdl(fetch_kernel, dim3(n_ctas), dim3(kFetchThreads), 0, st, pool, reinterpret_cast<unsigned char*>(hot_pool), page_bytes);
}

cudaError_t launch_prestep(int dtype, SeqDev* seqs, int B, int D, int W, const uint32_t* swap_mask_words,
                           int n_words, const void* k_new, const void* v_new, cudaStream_t st) {
  SwapWords sw;
  for (int i = 0; i < 32; ++i) sw.w[i] = (swap_mask_words && i < n_words) ? swap_mask_words[i] : 0u;
  const int use_swap = swap_mask_words != nullptr;
  if (dtype == 0)
    prestep_kernel_v<float><<<B, 128, 0, st>>>(seqs, D, W, sw, use_swap, (const float*)k_new, (const float*)v_new);
  else
    prestep_kernel_v<__nv_bfloat16><<<B, 128, 0, st>>>(seqs, D, W, sw, use_swap, (const __nv_bfloat16*)k_new,
                                                       (const __nv_bfloat16*)v_new);
  return cudaGetLastError();
}

}  // namespace lsa
