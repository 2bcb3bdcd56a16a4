// lsa_attn_tc_kernel.cuh - the tcgen05 split-K decode attention kernel (see lsa_attn_tc_defs.cuh).
#pragma once
#include "lsa_attn_tc_defs.cuh"
#include "lsa_attn_tc_fused.cuh"

namespace lsa {


// Order of the K/V stage groups of a piece with tiles t0..t1-1, for the producer and the MMA issuer alike:
//   K(t0) | K(t0+1) V(t0) | K(t0+2) V(t0+1) | ... | V(t1-1)
// K runs one tile ahead of V, so S(t+1) is computed (and K(t+2) is in flight) while the softmax of tile t
// runs; with the 4-stage ring a V tile never waits behind the K tile that depends on its completion.

// kMask: the Level-2 row mask (TcParams::l2_mask, lsa_l2.cu) is applied to the page tiles; the unmasked
// instantiation carries none of that code.
template <bool kMask>
__global__ void __launch_bounds__(kTcThreads, 1)
attn_tc_kernel(const __grid_constant__ CUtensorMap map_pool, const __grid_constant__ CUtensorMap map_q, TcParams p) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  TcSmem& sm = *reinterpret_cast<TcSmem*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int cta = blockIdx.x, n_cta = p.n_attn;    // CTAs that own tiles; gridDim.x may be larger (fused S8)

  // ---- setup: mbarriers first (one cheap block barrier), everything slower overlaps behind `setup` ----
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
    prefetch_tmap(&map_q);
  }
  __syncthreads();
  griddep_wait();                 // PDL: everything below may read what the previous kernel wrote
  griddep_launch_dependents();    // the combine kernel may start its prologue; it waits for this grid itself
  if (p.ktime && tid == 0) atomicMin(p.ktime, gtime());
  if (warp == 0) {
    // per-sequence shape and the prefix of tiles per sequence (B <= 256)
    int carry = 0;
    for (int base = 0; base < p.B; base += 32) {
      const int b = base + lane;
      int g = 0;
      if (b < p.B) {
        const SeqView v = make_view(p, b);
        sm.view[b] = v;
        g = v.t_hca + v.n_cur + (v.w_len + kTcTile - 1) / kTcTile;
      }
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
    __syncwarp();
    if (lane == 0) mbar_arrive(&sm.setup);
  }

  if (warp == 0) {
    // =========================== TMA producer (does not wait for `setup`: it wrote gpre itself) ===========
    if (elect_one()) {
      PieceCursor cur(sm.gpre, p.B, cta, n_cta);
      int b, t0, t1, item = 0;
      uint32_t ring = 0;                                  // stages issued so far
      bool app_seen = false;
      // the tile holding this launch's new window row is loaded only after the softmax warps have written it
      auto app_gate = [&](const SeqView& v, int t) {
        if (t == v.app_tile && !app_seen) { mbar_wait(&sm.app_done, 0, 12); app_seen = true; }
      };
      auto issue4 = [&](const CUtensorMap* m, int row) {
#pragma unroll 1
        for (int s4 = 0; s4 < 4; ++s4) {
          const int st = ring % kTcStages;
          mbar_wait(&sm.empty[st], ((ring / kTcStages) & 1) ^ 1, 11);
          mbar_arrive_expect_tx(&sm.full[st], kTcStageBytes);
          tma_load_3d(sm.stage[st], m, 0, row, s4 * 2, &sm.full[st]);
          ++ring;
        }
      };
      while (cur.next(b, t0, t1)) {
        const SeqView v = sm.view[b];
        TileSrc src = tile_src(p, &map_pool, v, t0);      // table look-up overlaps the Q issue
        if (item > 0) mbar_wait(&sm.q_empty, (item - 1) & 1, 10);
        mbar_arrive_expect_tx(&sm.q_full, 65536);
        tma_load_3d(sm.q, &map_q, 0, b * kTcH, 0, &sm.q_full);
        app_gate(v, t0);
        issue4(src.mk, src.row_k);
        for (int t = t0; t < t1; ++t) {
          TileSrc nxt = src;
          if (t + 1 < t1) {
            nxt = tile_src(p, &map_pool, v, t + 1);
            app_gate(v, t + 1);
            issue4(nxt.mk, nxt.row_k);
          }
          issue4(src.mv, src.row_v);
          src = nxt;
        }
        ++item;
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
      // descriptors of stage 0 / the Q tile / the P tile; everything else is a constant added to the address field
      const uint64_t dk0 = make_sdesc(smem_u32(sm.stage[0]), 16, 1024, kLayoutSw128);
      const uint64_t dv0 = make_sdesc(smem_u32(sm.stage[0]), 16384, 1024, kLayoutSw128);
      const uint64_t dq0 = make_sdesc(smem_u32(sm.q), 16, 1024, kLayoutSw128);
      const uint64_t dp0 = make_sdesc(smem_u32(sm.p), 16384, 1024, kLayoutSw128);
      const uint64_t ones_desc = make_sdesc(smem_u32(sm.ones), 128, 256, kLayoutNone);
      PieceCursor cur(sm.gpre, p.B, cta, n_cta);
      int b, t0, t1, item = 0;
      uint32_t ring = 0, n_s = 0, n_pv = 0;               // stages consumed, S tiles issued, PV tiles issued
      // S^T(tile n_s) = K Q^T into S buffer n_s & 1
      auto issue_s = [&](bool last_of_piece) {
        const int buf = n_s & 1;
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
            const uint64_t a = a0 + (uint64_t)(((ks >> 2) * 16384 + (ks & 3) * 32) >> 4);
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
      // O^T (+)= V^T P^T ; L (+)= 1 P^T for tile n_pv.  On the last tile of a piece every 128-row block of O^T
      // is committed on its own, so the epilogue drains block m while blocks m+1.. are still being computed.
      auto issue_pv = [&](bool first_of_piece, bool last_of_piece) {
        mbar_wait(&sm.p_full, n_pv & 1, 23);
        tc_fence_after();
        if (first_of_piece && item > 0) {                 // the previous piece's epilogue has drained O and L
          mbar_wait(&sm.o_empty, (item - 1) & 1, 24);
          tc_fence_after();
        }
        const uint32_t acc = first_of_piece ? 0u : 1u;
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) umma_bf16(tL, ones_desc, dp0 + (uint64_t)((ks * 2048) >> 4), id_l, acc | (ks != 0));
#pragma unroll 1
        for (int m = 0; m < 4; ++m) {
          const int st = ring % kTcStages;
          mbar_wait(&sm.full[st], (ring / kTcStages) & 1, 25);
          tc_fence_after();
          const uint64_t a0 = dv0 + (uint64_t)(st * (kTcStageBytes >> 4));
#pragma unroll
          for (int ks = 0; ks < 8; ++ks)
            umma_bf16(tO + m * 64, a0 + (uint64_t)((ks * 2048) >> 4), dp0 + (uint64_t)((ks * 2048) >> 4), id_pv, acc | (ks != 0));
          umma_commit(&sm.empty[st]);
          if (last_of_piece) umma_commit(&sm.o_full[m]);
          ++ring;
        }
        umma_commit(&sm.pv_done);
        ++n_pv;
      };
      while (cur.next(b, t0, t1)) {
        mbar_wait(&sm.q_full, item & 1, 20);
        tc_fence_after();
        issue_s(t0 + 1 == t1);
        for (int t = t0; t < t1; ++t) {
          if (t + 1 < t1) issue_s(t + 2 == t1);
          issue_pv(t == t0, t + 1 == t1);
        }
        ++item;
      }
    }
  } else {
    // =========================== softmax + epilogue (8 warps) ===========================
    const int q4 = warp & 3;                              // TMEM lane quarter this warp may access
    const int hh = (warp - 2) >> 2;                       // half of the heads owned by this warp
    const uint32_t lane_addr = (uint32_t)(q4 * 32) << 16;
    const int key = q4 * 32 + lane;                       // key row of the tile owned by this thread
    mbar_wait(&sm.setup, 0, 29);
    tc_fence_after();
    const uint32_t tmem = sm.tmem_base;
    const uint32_t tS = tmem, tO = tmem + 128, tL = tmem + 384;
    int b, t0, t1, b_first = -1, b_last = -1;
    if (p.k_new) {
      // window append ("decoded tokens stay resident"; DESIGN R6): the CTA that owns the tile holding ring
      // slot w_head of a sequence writes k_new/v_new there before its producer loads that tile
      PieceCursor pc(sm.gpre, p.B, cta, n_cta);
      const int t = tid - 64;
      while (pc.next(b, t0, t1)) {
        const SeqView v = sm.view[b];
        if (v.app_tile >= t0 && v.app_tile < t1 && t < 128) {
          const SeqDev& s = p.seqs[b];
          const uint4* src = reinterpret_cast<const uint4*>((t < 64 ? p.k_new : p.v_new) + (size_t)b * kTcD) + (t & 63);
          uint4* dst = reinterpret_cast<uint4*>(reinterpret_cast<__nv_bfloat16*>(t < 64 ? s.win_k : s.win_v) + (size_t)v.app_slot * kTcD) + (t & 63);
          *dst = *src;
        }
      }
      fence_proxy_async_all();                            // generic-proxy stores -> later TMA (async proxy) reads
      __syncwarp();
      if (lane == 0) mbar_arrive(&sm.app_done);
    }
    PieceCursor cur(sm.gpre, p.B, cta, n_cta);
    uint32_t tcount = 0, piece = 0;
    float m_run[32];
    // merged maximum of every head of this warp's half over all 128 keys of the tile -> mt[32]
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
    while (cur.next(b, t0, t1)) {
      if (b_first < 0) b_first = b;
      // sequences without keys between two pieces of this CTA get an empty partial (weight 0 in S8)
      for (int e = b_last + 1; b_last >= 0 && e < b; ++e)
        if (tid < 64 + kTcH) { p.part_m[((size_t)cta + e) * kTcH + tid - 64] = -INFINITY; p.part_l[((size_t)cta + e) * kTcH + tid - 64] = 0.f; }
      b_last = b;
      const SeqView v = sm.view[b];
      int nv_next = tile_valid(p, v, t0);
      uint32_t km_next = kMask ? tile_keymask(p, v, t0, q4) : 0xffffffffu;
      for (int t = t0; t < t1; ++t) {
        const int buf = tcount & 1;
        const bool valid = kMask ? (key < nv_next && ((km_next >> lane) & 1u)) : key < nv_next;
        if (t + 1 < t1) {                                         // global look-ups overlap the wait below
          nv_next = tile_valid(p, v, t + 1);
          if (kMask) km_next = tile_keymask(p, v, t + 1, q4);
        }
        float x[32];
        mbar_wait(&sm.s_full[buf], (tcount >> 1) & 1, 30);
        tc_fence_after();
        tmem_ld32(tS + buf * 64 + hh * 32 + lane_addr, reinterpret_cast<uint32_t*>(x));
        tmem_wait_ld();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&sm.s_empty[buf]);
        // masked, scaled logits (log2 domain); inputs are finite, so a tile with >= 1 valid key has a finite maximum
#pragma unroll
        for (int h = 0; h < 32; ++h) x[h] = valid ? x[h] * p.scale_log2 : -INFINITY;
        bool rescale = false;
        float f[32];
        if (t == t0) {
          tile_max(x, m_run);
          // a first tile without any attended key (Level-2 mask) leaves -inf: keep the maximum finite so that
          // 2^(x - m) is 0, not NaN; the first real logit then triggers the rescale path
          if (kMask) {
#pragma unroll
            for (int h = 0; h < 32; ++h) m_run[h] = fmaxf(m_run[h], -1e30f);
          }
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
        // P^T values of this thread: 32 heads of one key, bf16 pairs (computed before waiting for the buffer)
        uint32_t pw[16];
#pragma unroll
        for (int e = 0; e < 16; ++e) pw[e] = pack_bf16x2(ex2_approx(x[2 * e] - m_run[2 * e]), ex2_approx(x[2 * e + 1] - m_run[2 * e + 1]));
        // the P tile buffer (and O) are free once the previous tile's PV MMAs have completed
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
        // P^T tile: bf16 [128 keys][64 heads], 128-byte swizzle; this thread's 32 heads = 4 x 16 B
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
      }
      // ---- epilogue: O^T, L, m -> partial slot (cta + b) ----
      // layout [d-block m][head half][head quad g][d_local][4 heads]: one 16-byte store per (m, g), warp-contiguous
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
            p.part_m[slot * kTcH + hh * 32 + j] = (kMask && m_run[j] <= -1e30f) ? -INFINITY : m_run[j];   // no attended key: S8 skips the slot
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
  if (p.fused) {
    grid_arrive_and_wait(p);                      // every partial of the launch is visible from here on
    if (warp == 1) {
      tc_fence_after();
      tmem_dealloc(sm.tmem_base, 512);
    }
    if (cta == 0 && tid < p.B) commit_state(p, tid);  // every CTA has read the records (they are behind the barrier)
    if (warp >= 2) fused_combine(p, sm.q, cta, gridDim.x, tid - 64);
  } else {
    __syncthreads();
    if (warp == 1) {
      tc_fence_after();
      tmem_dealloc(sm.tmem_base, 512);
    }
  }
  if (p.ktime && tid == 0) atomicMax(p.ktime + 1, gtime());
}

}  // namespace lsa
