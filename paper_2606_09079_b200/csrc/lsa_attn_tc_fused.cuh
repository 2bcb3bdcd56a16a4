// lsa_attn_tc_fused.cuh - S8 inside the attention kernel for small batches (B <= kTcFusedMaxB).
//
// A second kernel costs a launch gap, a cold start and a dependency flush - together several microseconds,
// as much as the whole attention kernel at B = 1.  Instead every CTA of the grid (one per SM, all resident)
// arrives at a global counter once its partials are written, waits until the counter reaches the launch's
// target, and then merges its share of the output:
//   unit = (sequence, 32 consecutive float4 columns of the partial layout) = 4 heads x 32 d;  256 per sequence
//   warp w of the 8 merge warps takes partials w, w+8, ... of the sequence's active list, with its own
//   reference maximum M_w (no exchange needed before the loads are issued); the 8 (M_w, L_w, acc_w) are
//   merged through shared memory by one warp, which writes the bf16 output (and lse).
#pragma once
#include "lsa_attn_tc_defs.cuh"

namespace lsa {

constexpr int kTcFusedMaxB = 4;

__device__ __forceinline__ unsigned int ld_acquire_gpu(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

// All kTcThreads threads call this after their last global store of the launch.
__device__ __noinline__ void grid_arrive_and_wait(const TcParams& p) {
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) {
    atomicAdd(p.grid_ctr, 1u);
    const long long t0 = clock64();
    while ((int)(ld_acquire_gpu(p.grid_ctr) - p.grid_target) < 0) {
      if (clock64() - t0 > 4000000000ll) {
        printf("lsa tc kernel: grid barrier timeout block=%d\n", blockIdx.x);
        __trap();
      }
    }
  }
  __syncthreads();
}

__device__ __forceinline__ float4 warp_max4(float4 v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    v.x = fmaxf(v.x, __shfl_xor_sync(0xffffffffu, v.x, o)); v.y = fmaxf(v.y, __shfl_xor_sync(0xffffffffu, v.y, o));
    v.z = fmaxf(v.z, __shfl_xor_sync(0xffffffffu, v.z, o)); v.w = fmaxf(v.w, __shfl_xor_sync(0xffffffffu, v.w, o));
  }
  return v;
}
__device__ __forceinline__ float4 warp_sum4(float4 v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    v.x += __shfl_xor_sync(0xffffffffu, v.x, o); v.y += __shfl_xor_sync(0xffffffffu, v.y, o);
    v.z += __shfl_xor_sync(0xffffffffu, v.z, o); v.w += __shfl_xor_sync(0xffffffffu, v.w, o);
  }
  return v;
}
__device__ __forceinline__ float w_of(float m, float M) { return m == -INFINITY ? 0.f : exp2f(m - M); }

// Called by the 256 merge threads (t = 0..255) of every CTA after the grid barrier.
// scratch: >= 24 KiB of shared memory no longer used by the attention phase (the Q tile buffer).
__device__ __noinline__ void fused_combine(const TcParams& p, unsigned char* scratch, int cta, int n_cta, int t) {
  const int w = t >> 5, lane = t & 31;
  int* cnt = reinterpret_cast<int*>(scratch);                    // [kTcFusedMaxB]
  int* wcnt = cnt + 8;                                           // [kTcFusedMaxB][8]
  int* list = reinterpret_cast<int*>(scratch + 1024);            // [kTcFusedMaxB][256] partial slots
  float4* mrg = reinterpret_cast<float4*>(scratch + 8192);       // [2][8 warps][34]: acc of 32 lanes, M, L
  // ---- active partials of every sequence: thread t looks at CTA t (n_attn <= 256) ----
  int2 info = make_int2(0, 0);
  if (t < p.n_attn) info = __ldcg(p.piece_info + t);
  unsigned bal[kTcFusedMaxB];
#pragma unroll
  for (int b = 0; b < kTcFusedMaxB; ++b) {
    const bool act = b < p.B && t < p.n_attn && info.x <= b && b < info.x + info.y;
    bal[b] = __ballot_sync(0xffffffffu, act);
    if (lane == 0) wcnt[b * 8 + w] = __popc(bal[b]);
  }
  named_bar_sync(2, 256);
#pragma unroll
  for (int b = 0; b < kTcFusedMaxB; ++b) {
    int base = 0, tot = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) { const int c = wcnt[b * 8 + i]; if (i < w) base += c; tot += c; }
    if ((bal[b] >> lane) & 1u) list[b * 256 + base + __popc(bal[b] & ((1u << lane) - 1))] = t + b;
    if (t == 0) cnt[b] = tot;
  }
  named_bar_sync(2, 256);
  // ---- units ----
  const uint2* part_o4 = p.part_o;                               // 4 heads of one d per element
  constexpr int U = 12;                                          // 16-byte loads in flight per thread
  int it = 0;
  for (int u = cta; u < p.B * 256; u += n_cta, ++it) {
    const int b = u >> 8, cc = u & 255;
    const int dq = cc & 3, g = (cc >> 2) & 7, hh = (cc >> 5) & 1, m = cc >> 6, h0 = hh * 32 + g * 4;
    const int n = cnt[b];
    const int* lst = list + b * 256;
    const int n_w = n > w ? (n - w + 7) >> 3 : 0;                // partials w, w+8, ... of this warp (<= 32)
    const int col = cc * 32 + lane;                              // float4 column inside a partial
    uint2 v[U];
#pragma unroll
    for (int j = 0; j < U; ++j)
      v[j] = j < n_w ? __ldcg(part_o4 + (size_t)lst[w + 8 * j] * (kTcH * kTcD / 4) + col) : make_uint2(0u, 0u);
    float4 mj = make_float4(-INFINITY, -INFINITY, -INFINITY, -INFINITY), lj = make_float4(0.f, 0.f, 0.f, 0.f);
    float sj = 0.f;                                              // scale of the unit's fp16 block in partial `lane`
    if (lane < n_w) {
      const size_t s = (size_t)lst[w + 8 * lane];
      mj = __ldcg(reinterpret_cast<const float4*>(p.part_m + s * kTcH + h0));
      lj = __ldcg(reinterpret_cast<const float4*>(p.part_l + s * kTcH + h0));
      sj = __ldcg(p.part_s + part_scale_idx(s, m, hh, dq));
    }
    const float4 M = warp_max4(mj);
    const float4 wj = make_float4(w_of(mj.x, M.x), w_of(mj.y, M.y), w_of(mj.z, M.z), w_of(mj.w, M.w));
    const float4 L = warp_sum4(make_float4(wj.x * lj.x, wj.y * lj.y, wj.z * lj.z, wj.w * lj.w));
    // a piece without valid keys (m = -inf) wrote no O: its weight is 0 and its data is never multiplied
    const float4 ws = make_float4(wj.x * sj, wj.y * sj, wj.z * sj, wj.w * sj);
    const unsigned live = __ballot_sync(0xffffffffu, mj.x != -INFINITY);
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int j = 0; j < U; ++j) {
      const float2 a01 = unpack_f16x2(v[j].x), a23 = unpack_f16x2(v[j].y);
      const float fx = __shfl_sync(0xffffffffu, ws.x, j), fy = __shfl_sync(0xffffffffu, ws.y, j);
      const float fz = __shfl_sync(0xffffffffu, ws.z, j), fw = __shfl_sync(0xffffffffu, ws.w, j);
      if ((live >> j) & 1u) {
        acc.x = fmaf(fx, a01.x, acc.x); acc.y = fmaf(fy, a01.y, acc.y);
        acc.z = fmaf(fz, a23.x, acc.z); acc.w = fmaf(fw, a23.y, acc.w);
      }
    }
    for (int j = U; j < n_w; ++j) {                              // more than 8*U partials: rare, one at a time
      const uint2 x = __ldcg(part_o4 + (size_t)lst[w + 8 * j] * (kTcH * kTcD / 4) + col);
      const float2 a01 = unpack_f16x2(x.x), a23 = unpack_f16x2(x.y);
      const float fx = __shfl_sync(0xffffffffu, ws.x, j), fy = __shfl_sync(0xffffffffu, ws.y, j);
      const float fz = __shfl_sync(0xffffffffu, ws.z, j), fw = __shfl_sync(0xffffffffu, ws.w, j);
      if ((live >> j) & 1u) {
        acc.x = fmaf(fx, a01.x, acc.x); acc.y = fmaf(fy, a01.y, acc.y);
        acc.z = fmaf(fz, a23.x, acc.z); acc.w = fmaf(fw, a23.y, acc.w);
      }
    }
    float4* mb = mrg + ((it & 1) * 8 + w) * 34;
    mb[lane] = acc;
    if (lane == 0) { mb[32] = M; mb[33] = L; }
    named_bar_sync(2, 256);
    if (w == (it & 7)) {                                         // one warp merges the 8 and writes 4 heads x 32 d
      const float4* base = mrg + (it & 1) * 8 * 34;
      float4 Ms = base[32];
#pragma unroll
      for (int i = 1; i < 8; ++i) {
        const float4 Mi = base[i * 34 + 32];
        Ms.x = fmaxf(Ms.x, Mi.x); Ms.y = fmaxf(Ms.y, Mi.y); Ms.z = fmaxf(Ms.z, Mi.z); Ms.w = fmaxf(Ms.w, Mi.w);
      }
      float4 num = make_float4(0.f, 0.f, 0.f, 0.f), den = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const float4 Mi = base[i * 34 + 32], Li = base[i * 34 + 33], a = base[i * 34 + lane];
        const float4 f = make_float4(w_of(Mi.x, Ms.x), w_of(Mi.y, Ms.y), w_of(Mi.z, Ms.z), w_of(Mi.w, Ms.w));
        num.x = fmaf(f.x, a.x, num.x); num.y = fmaf(f.y, a.y, num.y); num.z = fmaf(f.z, a.z, num.z); num.w = fmaf(f.w, a.w, num.w);
        den.x = fmaf(f.x, Li.x, den.x); den.y = fmaf(f.y, Li.y, den.y); den.z = fmaf(f.z, Li.z, den.z); den.w = fmaf(f.w, Li.w, den.w);
      }
      __nv_bfloat16* o = p.out + ((size_t)b * kTcH + h0) * kTcD + m * 128 + dq * 32 + lane;
      o[0] = __float2bfloat16_rn(den.x > 0.f ? num.x / den.x : 0.f);
      o[kTcD] = __float2bfloat16_rn(den.y > 0.f ? num.y / den.y : 0.f);
      o[2 * kTcD] = __float2bfloat16_rn(den.z > 0.f ? num.z / den.z : 0.f);
      o[3 * kTcD] = __float2bfloat16_rn(den.w > 0.f ? num.w / den.w : 0.f);
      if (p.lse && m == 0 && dq == 0 && lane == 0) {
        float* ls = p.lse + (size_t)b * kTcH + h0;
        ls[0] = den.x > 0.f ? (Ms.x + log2f(den.x)) * 0.6931471805599453f : -INFINITY;
        ls[1] = den.y > 0.f ? (Ms.y + log2f(den.y)) * 0.6931471805599453f : -INFINITY;
        ls[2] = den.z > 0.f ? (Ms.z + log2f(den.z)) * 0.6931471805599453f : -INFINITY;
        ls[3] = den.w > 0.f ? (Ms.w + log2f(den.w)) * 0.6931471805599453f : -INFINITY;
      }
    }
  }
}

}  // namespace lsa
