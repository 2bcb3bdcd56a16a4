// lsa_attn_tc_kernel.cuh - the tcgen05 split-K decode attention kernel (see lsa_attn_tc_defs.cuh).
#pragma once
#include "lsa_attn_tc_defs.cuh"

namespace lsa {

__global__ void __launch_bounds__(kTcThreads, 1)
attn_tc_kernel(const __grid_constant__ CUtensorMap map_pool, const __grid_constant__ CUtensorMap map_q, TcParams p) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  TcSmem& sm = *reinterpret_cast<TcSmem*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int cta = blockIdx.x, n_cta = gridDim.x;

  // ---- one-time setup ---------------------------------------------------------------------------
  if (tid == 0) {
    for (int i = 0; i < kTcStages; ++i) { mbar_init(&sm.full[i], 1); mbar_init(&sm.empty[i], 1); }
    mbar_init(&sm.q_full, 1); mbar_init(&sm.q_empty, 1);
    for (int i = 0; i < 2; ++i) { mbar_init(&sm.s_full[i], 1); mbar_init(&sm.s_empty[i], 4); }
    mbar_init(&sm.p_full, 4); mbar_init(&sm.pv_done, 1); mbar_init(&sm.o_empty, 4);
    fence_mbar_init();
    prefetch_tmap(&map_pool);
    prefetch_tmap(&map_q);
  }
  if (warp == 1) tmem_alloc(&sm.tmem_base, 512);
  for (int i = tid; i < 2048; i += kTcThreads) reinterpret_cast<uint16_t*>(sm.ones)[i] = 0x3f80;   // bf16 1.0
  // prefix of groups per sequence (B <= 256): warp 0 scans
  if (warp == 0) {
    int carry = 0;
    for (int base = 0; base < p.B; base += 32) {
      const int b = base + lane;
      int g = b < p.B ? seq_groups(p.seqs[b]) : 0;
      int incl = g;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
      }
      if (b < p.B) sm.gpre[b + 1] = carry + incl;
      carry += __shfl_sync(0xffffffffu, incl, 31);
    }
    if (lane == 0) sm.gpre[0] = 0;
  }
  fence_proxy_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = sm.tmem_base;
  const uint32_t tS = tmem, tO = tmem + 128, tL = tmem + 384;

  if (warp == 0) {
    // =========================== TMA producer ===========================
    if (lane == 0) {
      PieceCursor cur(sm.gpre, p.B, cta, n_cta);
      int b, g0, g1, item = 0;
      uint32_t ring = 0;                                  // stages issued so far
      while (cur.next(b, g0, g1)) {
        if (item > 0) mbar_wait(&sm.q_empty, (item - 1) & 1, 10);
        mbar_arrive_expect_tx(&sm.q_full, 65536);
        for (int db = 0; db < 8; ++db) tma_load_2d(sm.q + db * 8192, &map_q, db * 64, b * kTcH, &sm.q_full);
        const SeqView v = make_view(p, b);
        const int n_tiles = (g1 - g0 + 3) >> 2;
        for (int t = 0; t < n_tiles; ++t) {
          GroupSrc src[4];
#pragma unroll
          for (int gi = 0; gi < 4; ++gi) src[gi] = resolve_group(p, &map_pool, v, g0 + t * 4 + gi, g1);
#pragma unroll 1
          for (int kv = 0; kv < 2; ++kv) {
#pragma unroll 1
            for (int s4 = 0; s4 < 4; ++s4) {
              const int st = ring % kTcStages;
              mbar_wait(&sm.empty[st], ((ring / kTcStages) & 1) ^ 1, 11);
              mbar_arrive_expect_tx(&sm.full[st], kTcStageBytes);
#pragma unroll
              for (int db = 0; db < 2; ++db)
#pragma unroll
                for (int gi = 0; gi < 4; ++gi)
                  tma_load_2d(sm.stage[st] + db * 16384 + gi * 4096, kv ? src[gi].mv : src[gi].mk, (s4 * 2 + db) * 64,
                              kv ? src[gi].row_v : src[gi].row_k, &sm.full[st]);
              ++ring;
            }
          }
        }
        ++item;
      }
    }
  } else if (warp == 1) {
    // =========================== MMA issuer ===========================
    if (lane == 0) {
      constexpr uint32_t id_kk = make_idesc_bf16(128, 64, 0, 0);   // A K-major  (K tile, ones)
      constexpr uint32_t id_mn = make_idesc_bf16(128, 64, 1, 0);   // A MN-major (V tile)
      const uint32_t q_addr = smem_u32(sm.q), p_addr = smem_u32(sm.p);
      const uint64_t ones_desc = make_sdesc(smem_u32(sm.ones), 128, 256, kLayoutNone);
      PieceCursor cur(sm.gpre, p.B, cta, n_cta);
      int b, g0, g1, item = 0;
      uint32_t ring = 0, tcount = 0;
      while (cur.next(b, g0, g1)) {
        mbar_wait(&sm.q_full, item & 1, 20);
        tc_fence_after();
        const int n_tiles = (g1 - g0 + 3) >> 2;
        for (int t = 0; t < n_tiles; ++t) {
          const int buf = tcount & 1;
          // ---- S^T = K Q^T ----
          mbar_wait(&sm.s_empty[buf], ((tcount >> 1) & 1) ^ 1, 21);
          tc_fence_after();
#pragma unroll 1
          for (int s4 = 0; s4 < 4; ++s4) {
            const int st = ring % kTcStages;
            mbar_wait(&sm.full[st], (ring / kTcStages) & 1, 22);
            tc_fence_after();
            const uint32_t st_addr = smem_u32(sm.stage[st]);
#pragma unroll
            for (int ks = 0; ks < 8; ++ks) {
              const uint64_t a = make_sdesc(st_addr + (ks >> 2) * 16384 + (ks & 3) * 32, 16, 1024, kLayoutSw128);
              const uint64_t bq = make_sdesc(q_addr + (s4 * 2 + (ks >> 2)) * 8192 + (ks & 3) * 32, 16, 1024, kLayoutSw128);
              umma_bf16(tS + buf * 64, a, bq, id_kk, (s4 | ks) != 0);
            }
            umma_commit(&sm.empty[st]);
            ++ring;
          }
          umma_commit(&sm.s_full[buf]);
          if (t == n_tiles - 1) umma_commit(&sm.q_empty);
          // ---- O^T += V^T P^T ; L += 1 P^T ----
          mbar_wait(&sm.p_full, tcount & 1, 23);
          tc_fence_after();
          if (t == 0 && item > 0) {
            mbar_wait(&sm.o_empty, (item - 1) & 1, 24);
            tc_fence_after();
          }
#pragma unroll 1
          for (int m = 0; m < 4; ++m) {
            const int st = ring % kTcStages;
            mbar_wait(&sm.full[st], (ring / kTcStages) & 1, 25);
            tc_fence_after();
            const uint32_t st_addr = smem_u32(sm.stage[st]);
#pragma unroll
            for (int ks = 0; ks < 8; ++ks) {
              const uint64_t a = make_sdesc(st_addr + ks * 2048, 16384, 1024, kLayoutSw128);
              const uint64_t bp = make_sdesc(p_addr + (ks >> 2) * 8192 + (ks & 3) * 32, 16, 1024, kLayoutSw128);
              umma_bf16(tO + m * 64, a, bp, id_mn, (t | ks) != 0);
            }
            umma_commit(&sm.empty[st]);
            ++ring;
          }
#pragma unroll
          for (int ks = 0; ks < 8; ++ks) {
            const uint64_t bp = make_sdesc(p_addr + (ks >> 2) * 8192 + (ks & 3) * 32, 16, 1024, kLayoutSw128);
            umma_bf16(tL, ones_desc, bp, id_kk, (t | ks) != 0);
          }
          umma_commit(&sm.pv_done);
          ++tcount;
        }
        ++item;
      }
    }
  } else {
    // =========================== softmax + epilogue (128 threads) ===========================
    const int wq = warp & 3;                              // TMEM sub-partition of this warp
    const uint32_t lane_addr = (uint32_t)(wq * 32) << 16;
    const int key = wq * 32 + lane;                       // key row of the tile owned by this thread
    PieceCursor cur(sm.gpre, p.B, cta, n_cta);
    int b, g0, g1;
    uint32_t tcount = 0;
    while (cur.next(b, g0, g1)) {
      const SeqView v = make_view(p, b);
      const int n_tiles = (g1 - g0 + 3) >> 2;
      float m_run[kTcH];
      for (int t = 0; t < n_tiles; ++t) {
        const int buf = tcount & 1;
        const GroupSrc src = resolve_group(p, &map_pool, v, g0 + t * 4 + wq, g1);
        const bool valid = lane < src.n_valid;
        float x[kTcH];
        mbar_wait(&sm.s_full[buf], (tcount >> 1) & 1, 30);
        tc_fence_after();
        tmem_ld32(tS + buf * 64 + lane_addr, reinterpret_cast<uint32_t*>(x));
        tmem_ld32(tS + buf * 64 + 32 + lane_addr, reinterpret_cast<uint32_t*>(x) + 32);
        tmem_wait_ld();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&sm.s_empty[buf]);
        // masked, scaled logits (log2 domain) and the per-warp maximum of every head
#pragma unroll
        for (int h = 0; h < kTcH; ++h) {
          x[h] = valid ? x[h] * p.scale_log2 : -INFINITY;
          const int r = redux_max_s32(float_ordered_s32(x[h]));
          if ((h & 31) == lane) reinterpret_cast<int*>(sm.wmax[buf][h])[wq] = r;
        }
        named_bar_sync(1, 128);
        // tile maximum of every head (identical in all 128 threads); first tile of a piece adopts it,
        // later tiles keep the stale running maximum unless it is exceeded by more than 2^8
        bool need_rescale = false;
#pragma unroll
        for (int h = 0; h < kTcH; ++h) {
          const int4 w = *reinterpret_cast<const int4*>(sm.wmax[buf][h]);
          const float mt = s32_ordered_float(max(max(w.x, w.y), max(w.z, w.w)));
          if (t == 0) m_run[h] = mt;
          else need_rescale |= (mt > m_run[h] + kRescaleThreshold);
        }
        // P tile buffer (and O) are free once the previous tile's PV MMAs have completed
        if (tcount > 0) {
          mbar_wait(&sm.pv_done, (tcount - 1) & 1, 31);
          tc_fence_after();
        }
        if (need_rescale) {             // rare: O^T and L are rescaled in TMEM, 32 columns at a time
#pragma unroll
          for (int c = 0; c < 10; ++c) {          // 4 x 64 O columns + 64 L columns
            uint32_t vreg[32];
            const uint32_t addr = tO + c * 32 + lane_addr;
            tmem_ld32(addr, vreg);
            tmem_wait_ld();
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              const int h = (c & 1) * 32 + j;
              const int4 w = *reinterpret_cast<const int4*>(sm.wmax[buf][h]);
              const float mn = fmaxf(m_run[h], s32_ordered_float(max(max(w.x, w.y), max(w.z, w.w))));
              const float f = (mn == -INFINITY) ? 1.f : ex2_approx(m_run[h] - mn);
              vreg[j] = __float_as_uint(__uint_as_float(vreg[j]) * f);
            }
            tmem_st32(addr, vreg);
          }
          tmem_wait_st();
#pragma unroll
          for (int h = 0; h < kTcH; ++h) {
            const int4 w = *reinterpret_cast<const int4*>(sm.wmax[buf][h]);
            m_run[h] = fmaxf(m_run[h], s32_ordered_float(max(max(w.x, w.y), max(w.z, w.w))));
          }
        }
        // P^T tile: bf16, K-major (keys contiguous per head), 128-byte swizzle
        {
          const int kb = key >> 6, kk = key & 63;
          unsigned char* pbase = sm.p + kb * 8192 + (kk & 7) * 2;
          const int chunk = kk >> 3;
#pragma unroll
          for (int h = 0; h < kTcH; ++h) {
            const float mu = (m_run[h] == -INFINITY) ? 0.f : m_run[h];
            const float pv = ex2_approx(x[h] - mu);
            *reinterpret_cast<__nv_bfloat16*>(pbase + h * 128 + ((chunk ^ (h & 7)) << 4)) = __float2bfloat16_rn(pv);
          }
        }
        fence_proxy_async_smem();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&sm.p_full);
        ++tcount;
      }
      // ---- epilogue: O^T, L, m -> partial slot (cta + b) ----
      mbar_wait(&sm.pv_done, (tcount - 1) & 1, 32);
      tc_fence_after();
      const size_t slot = (size_t)cta + b;
      float* po = p.part_o + slot * (kTcH * kTcD);
#pragma unroll 1
      for (int c = 0; c < 8; ++c) {               // c>>1 = d-tile, c&1 = head half
        uint32_t vreg[32];
        tmem_ld32(tO + c * 32 + lane_addr, vreg);
        tmem_wait_ld();
        const int d = (c >> 1) * 128 + key;
#pragma unroll
        for (int j = 0; j < 32; ++j) po[(size_t)((c & 1) * 32 + j) * kTcD + d] = __uint_as_float(vreg[j]);
      }
      if (wq == 0) {                              // every lane of L holds the same row sums: lane 0 writes them
#pragma unroll 1
        for (int c = 0; c < 2; ++c) {
          uint32_t vreg[32];
          tmem_ld32(tL + c * 32 + lane_addr, vreg);
          tmem_wait_ld();
          if (lane == 0)
#pragma unroll
            for (int j = 0; j < 32; ++j) p.part_l[slot * kTcH + c * 32 + j] = __uint_as_float(vreg[j]);
        }
      }
      if (wq == 1 && lane == 0) {
#pragma unroll
        for (int h = 0; h < kTcH; ++h) p.part_m[slot * kTcH + h] = m_run[h];
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&sm.o_empty);
    }
  }
  // ---- teardown ----
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem, 512);
}

}  // namespace lsa
