// lsa_attn_tc.cu - host side of the tcgen05 attention (tensor maps, launch) and the S8 combine kernel.
// Kernel: lsa_attn_tc_kernel.cuh.  Design notes: lsa_attn_tc_defs.cuh.
#include <cstdio>
#include <cstdlib>
#include <mutex>

#include "lsa_attn_tc_kernel.cuh"
#include "lsa_attn_tc_small.cuh"

namespace lsa {

// ---- S8: merge the split partials of one sequence  ----------------------------------------------
//   m* = max m_i ; l* = sum l_i 2^(m_i-m*) ; out = sum o_i 2^(m_i-m*) / l* ; lse = ln2 (m* + log2 l*)
// Partials are stored as [d-block m][head half][head quad g][d_local 128][4 heads] fp16 with one power-of-two
// scale per (m, half, 32 d) block (lsa_attn_tc_defs.cuh, "split-K partial format") - the order the attention
// epilogue drains TMEM in.  grid (128, B): block = (m, half, g, 64 of the 128 d), i.e. 512 contiguous bytes of
// every slot; 512 threads = 64 d x 8 groups, group j accumulates partials j, j+8, ... (4 heads per thread).
// Launched with programmatic stream serialization: the launch and prologue overlap the attention kernel's tail.
constexpr int kCombineThreads = 512;
// The combine grid is launched while attention CTAs still own most SMs (PDL).  Asking for more than half an
// SM's shared memory keeps its blocks at one per SM, so the early ones cannot pile up on the few idle SMs.
constexpr int kCombineSmemPad = 116 * 1024;
constexpr int kCombineSmemMax = 128 * 1024;        // landing buffer of 256 slots x 512 B

// For B <= kCombineSpecMaxB nearly every CTA holds a piece of every sequence: the copies of all n_cta slots are
// issued before anything is known about them, together with the loads of piece_info, m, l and the scales, so the
// kernel is ONE memory round trip deep; slots that turn out to be inactive are discarded (selected away, never
// multiplied).  Larger batches use combine_tc_wide_kernel below.
constexpr int kCombineSpecMaxB = 4;

// The partials themselves come in by TMA: one 2-D box = the block's 512 bytes of kCombRows consecutive slots, so
// the whole read is n_cta / 32 bulk copies issued by one thread of a warp that has nothing else to wait for,
// landing in shared memory behind one mbarrier, instead of 16 loads per thread queued in the LSU.
constexpr int kCombRows = 32;                     // slots per TMA box
constexpr int kCombRowBytes = 512;                // (m, hh, g, half of d): 64 d x 4 heads fp16
constexpr int kCombBoxBytes = kCombRows * kCombRowBytes;

__global__ void __launch_bounds__(kCombineThreads, 1)
combine_tc_kernel(const __grid_constant__ CUtensorMap map_part, TcParams p, int n_cta, __nv_bfloat16* __restrict__ out,
                  float* __restrict__ lse) {
  extern __shared__ __align__(128) unsigned char comb_rows[];   // [slot row][512 B]
  __shared__ __align__(8) uint64_t bar;
  __shared__ float4 w_s[256];
  __shared__ float2 sc_s[256];
  __shared__ int slot_s[256];
  __shared__ float4 red_f[16];
  __shared__ int warp_cnt[16];
  __shared__ float4 acc_s[8][64];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int dh = blockIdx.x & 1, g = (blockIdx.x >> 1) & 7, hh = (blockIdx.x >> 4) & 1, m = blockIdx.x >> 5, b = blockIdx.y;
  const int h0 = hh * 32 + g * 4;
  const int dl = tid & 63, grp = tid >> 6;
  const int n_box = (n_cta + kCombRows - 1) / kCombRows;
  if (tid == 0) {
    mbar_init(&bar, 1);
    fence_mbar_init();
    prefetch_tmap(&map_part);
  }
  __syncthreads();
  griddep_wait();                                 // partials and piece_info are final from here on
  griddep_launch_dependents();                    // the next kernel in the stream may start its own prologue
  if (tid == kCombineThreads - 32) {              // rows b .. b + 32 n_box - 1 of column block (m, hh, g, dh); a warp
                                                  // that has no small loads to wait for issues the copies
    mbar_arrive_expect_tx(&bar, (uint32_t)(n_box * kCombBoxBytes));
    for (int i = 0; i < n_box; ++i)
      tma_load_2d(comb_rows + i * kCombBoxBytes, &map_part, (((m * 2 + hh) * 8 + g) * 2 + dh) * (kCombRowBytes / 4), b + i * kCombRows, &bar);
  }
  if (blockIdx.x == 0 && tid == 0) commit_state(p, b);   // S6 / window append folded into the attention launch
  // thread c < n_cta looks at CTA c: did it write a partial for sequence b?  (n_cta <= 256)
  // These small loads go first so that they are not queued behind the bulk of partial loads below.
  bool active = false;
  float4 mi = make_float4(-INFINITY, -INFINITY, -INFINITY, -INFINITY), li = make_float4(0.f, 0.f, 0.f, 0.f);
  const size_t slot = (size_t)tid + b;
  int2 info = make_int2(0, 0);
  float4 m4 = mi, l4 = li;
  float2 s2 = make_float2(0.f, 0.f);              // scales of this CTA's two lane quarters (d = dh*64 + 0..31 / 32..63)
  if (tid < n_cta) {
    info = __ldcg(p.piece_info + tid);
    m4 = __ldcg(reinterpret_cast<const float4*>(p.part_m + slot * kTcH + h0));
    l4 = __ldcg(reinterpret_cast<const float4*>(p.part_l + slot * kTcH + h0));
    s2 = __ldcg(reinterpret_cast<const float2*>(p.part_s + part_scale_idx(slot, m, hh, dh * 2)));
  }
  if (tid < n_cta) {
    // a piece without valid keys (m = -inf for every head) wrote no O: its slot is skipped like an inactive one
    active = info.x <= b && b < info.x + info.y && m4.x != -INFINITY;
    if (active) { mi = m4; li = l4; }
  }
  float4 mmax = mi;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    mmax.x = fmaxf(mmax.x, __shfl_xor_sync(0xffffffffu, mmax.x, o));
    mmax.y = fmaxf(mmax.y, __shfl_xor_sync(0xffffffffu, mmax.y, o));
    mmax.z = fmaxf(mmax.z, __shfl_xor_sync(0xffffffffu, mmax.z, o));
    mmax.w = fmaxf(mmax.w, __shfl_xor_sync(0xffffffffu, mmax.w, o));
  }
  const unsigned bal = __ballot_sync(0xffffffffu, active);
  if (lane == 0) { red_f[warp] = mmax; warp_cnt[warp] = __popc(bal); }
  __syncthreads();
  float4 m_star = red_f[0];
  int base = 0, n_act = 0;
  for (int w = 0; w < 16; ++w) {
    const float4 r = red_f[w];
    m_star.x = fmaxf(m_star.x, r.x); m_star.y = fmaxf(m_star.y, r.y); m_star.z = fmaxf(m_star.z, r.z); m_star.w = fmaxf(m_star.w, r.w);
    if (w < warp) base += warp_cnt[w];
    n_act += warp_cnt[w];
  }
  float4 wi = make_float4(0.f, 0.f, 0.f, 0.f);
  if (active) {
    wi.x = mi.x == -INFINITY ? 0.f : exp2f(mi.x - m_star.x);
    wi.y = mi.y == -INFINITY ? 0.f : exp2f(mi.y - m_star.y);
    wi.z = mi.z == -INFINITY ? 0.f : exp2f(mi.z - m_star.z);
    wi.w = mi.w == -INFINITY ? 0.f : exp2f(mi.w - m_star.w);
  }
  if (tid < 256) { w_s[tid] = wi; sc_s[tid] = s2; slot_s[tid] = active ? 1 : 0; }   // by CTA index; slot_s marks active slots
  float4 lsum = make_float4(wi.x * li.x, wi.y * li.y, wi.z * li.z, wi.w * li.w);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    lsum.x += __shfl_xor_sync(0xffffffffu, lsum.x, o);
    lsum.y += __shfl_xor_sync(0xffffffffu, lsum.y, o);
    lsum.z += __shfl_xor_sync(0xffffffffu, lsum.z, o);
    lsum.w += __shfl_xor_sync(0xffffffffu, lsum.w, o);
  }
  __syncthreads();                                // red_f is reused; w_s / slot_s are complete
  if (lane == 0) red_f[warp] = lsum;
  __syncthreads();
  float4 l_star = make_float4(0.f, 0.f, 0.f, 0.f);
  for (int w = 0; w < 16; ++w) {
    const float4 r = red_f[w];
    l_star.x += r.x; l_star.y += r.y; l_star.z += r.z; l_star.w += r.w;
  }
  // ---- weighted sum of the partials (row c of the landing buffer = slot b + c = CTA c) ----
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  mbar_wait(&bar, 0, 40);
  {
    const uint2* rows = reinterpret_cast<const uint2*>(comb_rows) + dl;
#pragma unroll 4
    for (int c = grp; c < n_cta; c += 8) {
      if (slot_s[c]) {
        const float4 w = w_s[c];
        const float sc = dl < 32 ? sc_s[c].x : sc_s[c].y;
        const uint2 x = rows[c * (kCombRowBytes / 8)];
        const float2 a01 = unpack_f16x2(x.x), a23 = unpack_f16x2(x.y);
        acc.x = fmaf(w.x * sc, a01.x, acc.x); acc.y = fmaf(w.y * sc, a01.y, acc.y);
        acc.z = fmaf(w.z * sc, a23.x, acc.z); acc.w = fmaf(w.w * sc, a23.y, acc.w);
      }
    }
  }
  acc_s[grp][dl] = acc;
  __syncthreads();
  if (tid < 256) {                                // thread = one output element: head h0 + e, d = m*128 + dh*64 + dl
    const int e = tid >> 6;
    const float* a = reinterpret_cast<const float*>(acc_s);
    float s = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) s += a[(w * 64 + dl) * 4 + e];
    const float ls = e == 0 ? l_star.x : e == 1 ? l_star.y : e == 2 ? l_star.z : l_star.w;
    out[((size_t)b * kTcH + h0 + e) * kTcD + m * 128 + dh * 64 + dl] = __float2bfloat16_rn(ls > 0.f ? s / ls : 0.f);
  }
  if (lse && m == 0 && dh == 0 && tid < 4) {
    const float ls = tid == 0 ? l_star.x : tid == 1 ? l_star.y : tid == 2 ? l_star.z : l_star.w;
    const float ms = tid == 0 ? m_star.x : tid == 1 ? m_star.y : tid == 2 ? m_star.z : m_star.w;
    lse[(size_t)b * kTcH + h0 + tid] = ls > 0.f ? (ms + log2f(ls)) * 0.6931471805599453f : -INFINITY;
  }
}

// S8 for larger batches (B > kCombineSpecMaxB): a sequence is touched by only a few CTAs, so there is nothing to
// split - grid (16, B): block = 4 heads x all 512 d, thread = one float4 column (4 heads of one d) and walks
// the sequence's active partials itself (all loads of a batch of 8 in flight), no cross-thread reduction.
__global__ void __launch_bounds__(512)
combine_tc_wide_kernel(TcParams p, int n_cta, __nv_bfloat16* __restrict__ out, float* __restrict__ lse) {
  __shared__ float4 w_s[256];
  __shared__ int slot_s[256];
  __shared__ float4 red_f[16];
  __shared__ int warp_cnt[16];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = blockIdx.x & 7, hh = blockIdx.x >> 3, b = blockIdx.y;
  const int h0 = hh * 32 + g * 4;
  const int m = tid >> 7, dl = tid & 127;
  griddep_wait();
  griddep_launch_dependents();
  if (blockIdx.x == 0 && tid == 0) commit_state(p, b);
  bool active = false;
  float4 mi = make_float4(-INFINITY, -INFINITY, -INFINITY, -INFINITY), li = make_float4(0.f, 0.f, 0.f, 0.f);
  const size_t slot = (size_t)tid + b;
  if (tid < n_cta) {
    const int2 info = __ldcg(p.piece_info + tid);
    active = info.x <= b && b < info.x + info.y;
    if (active) {
      mi = __ldcg(reinterpret_cast<const float4*>(p.part_m + slot * kTcH + h0));
      li = __ldcg(reinterpret_cast<const float4*>(p.part_l + slot * kTcH + h0));
      active = mi.x != -INFINITY;                 // a piece without valid keys wrote no O: skip its slot
    }
  }
  float4 mmax = mi;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    mmax.x = fmaxf(mmax.x, __shfl_xor_sync(0xffffffffu, mmax.x, o));
    mmax.y = fmaxf(mmax.y, __shfl_xor_sync(0xffffffffu, mmax.y, o));
    mmax.z = fmaxf(mmax.z, __shfl_xor_sync(0xffffffffu, mmax.z, o));
    mmax.w = fmaxf(mmax.w, __shfl_xor_sync(0xffffffffu, mmax.w, o));
  }
  const unsigned bal = __ballot_sync(0xffffffffu, active);
  if (lane == 0) { red_f[warp] = mmax; warp_cnt[warp] = __popc(bal); }
  __syncthreads();
  float4 m_star = red_f[0];
  int base = 0, n_act = 0;
  for (int w = 0; w < 16; ++w) {
    const float4 r = red_f[w];
    m_star.x = fmaxf(m_star.x, r.x); m_star.y = fmaxf(m_star.y, r.y); m_star.z = fmaxf(m_star.z, r.z); m_star.w = fmaxf(m_star.w, r.w);
    if (w < warp) base += warp_cnt[w];
    n_act += warp_cnt[w];
  }
  float4 wi = make_float4(0.f, 0.f, 0.f, 0.f);
  if (active) {
    wi.x = mi.x == -INFINITY ? 0.f : exp2f(mi.x - m_star.x);
    wi.y = mi.y == -INFINITY ? 0.f : exp2f(mi.y - m_star.y);
    wi.z = mi.z == -INFINITY ? 0.f : exp2f(mi.z - m_star.z);
    wi.w = mi.w == -INFINITY ? 0.f : exp2f(mi.w - m_star.w);
    const int pos = base + __popc(bal & ((1u << lane) - 1));
    w_s[pos] = wi;
    slot_s[pos] = (int)slot;
  }
  float4 lsum = make_float4(wi.x * li.x, wi.y * li.y, wi.z * li.z, wi.w * li.w);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    lsum.x += __shfl_xor_sync(0xffffffffu, lsum.x, o);
    lsum.y += __shfl_xor_sync(0xffffffffu, lsum.y, o);
    lsum.z += __shfl_xor_sync(0xffffffffu, lsum.z, o);
    lsum.w += __shfl_xor_sync(0xffffffffu, lsum.w, o);
  }
  __syncthreads();
  if (lane == 0) red_f[warp] = lsum;
  __syncthreads();
  float4 l_star = make_float4(0.f, 0.f, 0.f, 0.f);
  for (int w = 0; w < 16; ++w) {
    const float4 r = red_f[w];
    l_star.x += r.x; l_star.y += r.y; l_star.z += r.z; l_star.w += r.w;
  }
  const uint2* po = p.part_o + (size_t)((m * 2 + hh) * 8 + g) * 128 + dl;
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  constexpr int U = 8;
  for (int i0 = 0; i0 < n_act; i0 += U) {
    uint2 v[U];
    float4 w[U];
    float sc[U];
#pragma unroll
    for (int j = 0; j < U; ++j) {
      const bool ok = i0 + j < n_act;
      const int sl = ok ? slot_s[i0 + j] : 0;
      w[j] = ok ? w_s[i0 + j] : make_float4(0.f, 0.f, 0.f, 0.f);
      v[j] = ok ? __ldcg(po + (size_t)sl * (kTcH * kTcD / 4)) : make_uint2(0u, 0u);
      sc[j] = ok ? __ldcg(p.part_s + part_scale_idx(sl, m, hh, dl >> 5)) : 0.f;   // the same word for a whole warp
    }
#pragma unroll
    for (int j = 0; j < U; ++j) {
      const float2 a01 = unpack_f16x2(v[j].x), a23 = unpack_f16x2(v[j].y);
      acc.x = fmaf(w[j].x * sc[j], a01.x, acc.x); acc.y = fmaf(w[j].y * sc[j], a01.y, acc.y);
      acc.z = fmaf(w[j].z * sc[j], a23.x, acc.z); acc.w = fmaf(w[j].w * sc[j], a23.y, acc.w);
    }
  }
  __nv_bfloat16* o = out + ((size_t)b * kTcH + h0) * kTcD + m * 128 + dl;
  o[0] = __float2bfloat16_rn(l_star.x > 0.f ? acc.x / l_star.x : 0.f);
  o[kTcD] = __float2bfloat16_rn(l_star.y > 0.f ? acc.y / l_star.y : 0.f);
  o[2 * kTcD] = __float2bfloat16_rn(l_star.z > 0.f ? acc.z / l_star.z : 0.f);
  o[3 * kTcD] = __float2bfloat16_rn(l_star.w > 0.f ? acc.w / l_star.w : 0.f);
  if (lse && tid < 4) {
    const float ls = tid == 0 ? l_star.x : tid == 1 ? l_star.y : tid == 2 ? l_star.z : l_star.w;
    const float ms = tid == 0 ? m_star.x : tid == 1 ? m_star.y : tid == 2 ? m_star.z : m_star.w;
    lse[(size_t)b * kTcH + h0 + tid] = ls > 0.f ? (ms + log2f(ls)) * 0.6931471805599453f : -INFINITY;
  }
}

// ---- host ------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct TcWorkspace;

struct TcPlan {
  TcInit init{};
  EncodeTiledFn encode = nullptr;
  CUtensorMap map_pool{}, map_pool64{}, map_q{}, map_part{}, map_part_small{};
  const void* q_cached = nullptr;
  CUtensorMap* d_maps = nullptr;
  CUtensorMap* d_maps8 = nullptr;      // small path: [B][8], 128-row and 64-row boxes
  SmMaps0 maps0{};                     // those of sequence 0, passed by value
  std::vector<std::pair<const void*, CUtensorMap>> q_maps;   // Q tensor maps by buffer address
  bool small_ok = false;
  TcParams params{};
  unsigned long long grid_total = 0;   // host mirror of the fused-S8 arrival counter
  int grid_max = 0;
  int small_mergers = 32;              // small path: merging CTAs of a launch that shares the machine (measured: 16 / 24 / 48 / 64 are slower)
  size_t smem = 0;
  TcWorkspace* ws = nullptr;
};

// ---- split-K workspace, one per compute stream ----
// The partials of one attention launch are consumed by the combine kernel that follows it on the same stream, and
// the next attention launch writes its partials only after griddepcontrol.wait, i.e. after that combine kernel
// has finished.  Contexts that share a compute stream (the layers of a model, the replicas of the benchmark) can
// therefore share one workspace: 12.6 MB at cfg3 that stays in L2 instead of one copy per context that is
// written back to HBM between uses.  A context whose grid or batch does not fit an existing workspace of its
// stream gets a new one.  Slots that a launch does not write are never read with effect (the combine kernels
// skip slots that piece_info does not mark), so nothing is cleared between users.
constexpr int kWsBufs = 3;              // a launch's partials are merged while the next two launches write theirs
struct TcWorkspace {
  int device = 0;
  cudaStream_t stream = nullptr;
  size_t slots = 0, grid_max = 0;
  int refs = 0;
  uint2* part_o = nullptr;              // kWsBufs buffers of `slots` each: the small path rotates, the general path uses the first
  float *part_s = nullptr, *part_m = nullptr, *part_l = nullptr;
  int2* piece_info = nullptr;           // kWsBufs buffers of grid_max
  // small path (lsa_attn_tc_small.cuh): launches so far; the CTAs that arrive per buffer / the mergers that have finished
  // in total, as the host has enqueued them (the kernels wait for these totals)
  unsigned int* ctrs = nullptr;         // DEVICE [kWsBufs + 1]: arrivals per buffer, then the mergers that have finished
  unsigned long long n_small = 0;
  unsigned int arr_total[kWsBufs] = {};
  unsigned int done_total = 0;          // after the last launch
  unsigned int done_hist[kWsBufs] = {}; // after each of the last kWsBufs launches (index: launch number mod kWsBufs)
  bool last_small = false;              // the last launch on this workspace did not wait for its predecessor
};
static std::mutex g_ws_mu;
static std::vector<TcWorkspace*> g_ws;

static void ws_free(TcWorkspace* w) {
  cudaFree(w->part_o); cudaFree(w->part_s); cudaFree(w->part_m); cudaFree(w->part_l); cudaFree(w->piece_info); cudaFree(w->ctrs);
  delete w;
}

static TcWorkspace* ws_acquire(cudaStream_t st, size_t slots, size_t grid_max, std::string* msg) {
  std::lock_guard<std::mutex> lk(g_ws_mu);
  int device = 0;
  cudaGetDevice(&device);
  for (TcWorkspace* w : g_ws)
    if (w->device == device && w->stream == st && w->slots >= slots && w->grid_max >= grid_max) { ++w->refs; return w; }
  TcWorkspace* w = new TcWorkspace();
  w->device = device; w->stream = st; w->slots = slots; w->grid_max = grid_max; w->refs = 1;
  cudaError_t e = cudaMalloc(&w->part_o, kWsBufs * slots * (kTcH * kTcD / 4) * sizeof(uint2));
  if (e == cudaSuccess) e = cudaMalloc(&w->part_s, kWsBufs * slots * kTcPartScales * sizeof(float));
  if (e == cudaSuccess) e = cudaMalloc(&w->part_m, kWsBufs * slots * kTcH * sizeof(float));
  if (e == cudaSuccess) e = cudaMalloc(&w->part_l, kWsBufs * slots * kTcH * sizeof(float));
  if (e == cudaSuccess) e = cudaMalloc(&w->piece_info, kWsBufs * grid_max * sizeof(int2));
  if (e == cudaSuccess) e = cudaMalloc(&w->ctrs, (kWsBufs + 1) * sizeof(unsigned int));
  // (the workspace starts defined: a slot no launch has written yet is still landed by the merge's TMA boxes)
  if (e == cudaSuccess) e = cudaMemset(w->part_o, 0, kWsBufs * slots * (kTcH * kTcD / 4) * sizeof(uint2));
  if (e == cudaSuccess) e = cudaMemset(w->part_s, 0, kWsBufs * slots * kTcPartScales * sizeof(float));
  if (e == cudaSuccess) e = cudaMemset(w->part_m, 0, kWsBufs * slots * kTcH * sizeof(float));
  if (e == cudaSuccess) e = cudaMemset(w->part_l, 0, kWsBufs * slots * kTcH * sizeof(float));
  if (e == cudaSuccess) e = cudaMemset(w->piece_info, 0, kWsBufs * grid_max * sizeof(int2));
  if (e == cudaSuccess) e = cudaMemset(w->ctrs, 0, (kWsBufs + 1) * sizeof(unsigned int));
  if (e != cudaSuccess) {
    *msg = std::string("split-K workspace: ") + cudaGetErrorString(e);
    ws_free(w);
    return nullptr;
  }
  g_ws.push_back(w);
  return w;
}

static void ws_release(TcWorkspace* w) {
  if (!w) return;
  std::lock_guard<std::mutex> lk(g_ws_mu);
  if (--w->refs > 0) return;
  for (size_t i = 0; i < g_ws.size(); ++i)
    if (g_ws[i] == w) { g_ws.erase(g_ws.begin() + i); break; }
  ws_free(w);
}

bool tc_supported(int dtype, int H, int D, int C) { return dtype == 1 && H == kTcH && D == kTcD && C == kTcC; }

// A [rows][512] bf16 matrix seen as (64 columns, rows, 8 d-blocks): one box = [d-blocks][box_rows][128 B],
// which is exactly the K-major / MN-major 128-byte-swizzle operand image tcgen05.mma reads.
static bool encode_rows(EncodeTiledFn enc, CUtensorMap* m, const void* ptr, uint64_t rows, uint32_t box_rows, uint32_t box_dblocks,
                        std::string* msg) {
  cuuint64_t dims[3] = {64, rows, (cuuint64_t)kTcD / 64};
  cuuint64_t strides[2] = {(cuuint64_t)kTcD * 2, 128};
  cuuint32_t box[3] = {64, box_rows, box_dblocks};
  cuuint32_t es[3] = {1, 1, 1};
  CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(ptr), dims, strides, box, es,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    *msg = "cuTensorMapEncodeTiled failed with CUresult " + std::to_string((int)r);
    return false;
  }
  return true;
}

#define TC_CUDA(expr)                                                               \
  do {                                                                              \
    cudaError_t _e = (expr);                                                        \
    if (_e != cudaSuccess) {                                                        \
      *msg = std::string(#expr) + ": " + cudaGetErrorString(_e);                    \
      return -2;                                                                    \
    }                                                                               \
  } while (0)

int tc_create(const TcInit& init, TcPlan** out, std::string* msg) {
  if (init.B > kTcMaxB) { *msg = "tcgen05 attention supports at most 256 sequences per context"; return -6; }
  TcPlan* pl = new TcPlan();
  pl->init = init;
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
  if (e != cudaSuccess || !fn) { *msg = "cuTensorMapEncodeTiled entry point not found"; delete pl; return -2; }
  pl->encode = (EncodeTiledFn)fn;
  pl->grid_max = init.max_ctas > 0 ? std::min(init.max_ctas, init.n_sms) : init.n_sms;
  if (pl->grid_max > 256) pl->grid_max = 256;
  if (!encode_rows(pl->encode, &pl->map_pool, init.hot_pool, (uint64_t)init.P * 2 * kTcC, kTcTile, 2, msg)) { delete pl; return -2; }
  std::vector<CUtensorMap> maps((size_t)init.B * 4);
  for (int b = 0; b < init.B; ++b) {
    const SeqDev& s = init.seq_host[b];
    const void* ptrs[4] = {s.hca_k, s.hca_v, s.win_k, s.win_v};
    const uint64_t rows[4] = {(uint64_t)s.cap_hca, (uint64_t)s.cap_hca, (uint64_t)init.W, (uint64_t)init.W};   // cap_hca = n_hca unless the history grows
    for (int j = 0; j < 4; ++j) {
      const bool none = rows[j] == 0 || ptrs[j] == nullptr;     // never referenced: point at the pool
      if (!encode_rows(pl->encode, &maps[(size_t)b * 4 + j], none ? init.hot_pool : ptrs[j], none ? kTcTile : rows[j], kTcTile, 2, msg)) {
        delete pl;
        return -2;
      }
    }
    // rows of the window ring that are not attended yet must hold finite values (they are multiplied by P = 0)
    if (init.W > s.w_len && s.win_k && s.win_v) {
      const size_t off = (size_t)s.w_len * kTcD * 2, n = (size_t)(init.W - s.w_len) * kTcD * 2;
      TC_CUDA(cudaMemset((char*)s.win_k + off, 0, n));
      TC_CUDA(cudaMemset((char*)s.win_v + off, 0, n));
    }
  }
  TC_CUDA(cudaMalloc(&pl->d_maps, maps.size() * sizeof(CUtensorMap)));
  TC_CUDA(cudaMemcpy(pl->d_maps, maps.data(), maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice));
  if (init.B <= kSmB && !init.fuse_combine) {
    // small path: every source also as 64-row boxes (a lone half tile), lsa_attn_tc_small.cuh
    if (!encode_rows(pl->encode, &pl->map_pool64, init.hot_pool, (uint64_t)init.P * 2 * kTcC, kSmHalf, 2, msg)) { delete pl; return -2; }
    std::vector<CUtensorMap> maps8((size_t)init.B * 8);
    for (int b = 0; b < init.B; ++b) {
      const SeqDev& s = init.seq_host[b];
      const void* ptrs[4] = {s.hca_k, s.hca_v, s.win_k, s.win_v};
      const uint64_t rows[4] = {(uint64_t)s.cap_hca, (uint64_t)s.cap_hca, (uint64_t)init.W, (uint64_t)init.W};   // cap_hca = n_hca unless the history grows
      for (int j = 0; j < 4; ++j) {
        maps8[(size_t)b * 8 + j] = maps[(size_t)b * 4 + j];
        const bool none = rows[j] == 0 || ptrs[j] == nullptr;
        if (!encode_rows(pl->encode, &maps8[(size_t)b * 8 + 4 + j], none ? init.hot_pool : ptrs[j], none ? kTcTile : rows[j], kSmHalf, 2, msg)) {
          delete pl;
          return -2;
        }
      }
    }
    for (int j = 0; j < 8; ++j) pl->maps0.m[j] = maps8[j];
    TC_CUDA(cudaMalloc(&pl->d_maps8, maps8.size() * sizeof(CUtensorMap)));
    TC_CUDA(cudaMemcpy(pl->d_maps8, maps8.data(), maps8.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice));
    TC_CUDA(cudaFuncSetAttribute(attn_tc_small_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(SmSmem) + 1024)));
    TC_CUDA(cudaFuncSetAttribute(attn_tc_small_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(SmSmem) + 1024)));
    pl->small_ok = true;
  }
  const size_t slots = (size_t)pl->grid_max + init.B;
  TcParams& p = pl->params;
  p.seqs = init.d_seqs; p.tbl_chunk = init.pool.tbl_chunk; p.tbl_page = init.pool.tbl_page; p.seq_maps = pl->d_maps;
  p.B = init.B; p.k = init.k; p.W = init.W; p.seqs_mut = init.d_seqs;
  p.scale_log2 = init.sm_scale * 1.4426950408889634f;
  pl->ws = ws_acquire(init.stream, slots, (size_t)pl->grid_max, msg);
  if (!pl->ws) { cudaFree(pl->d_maps); delete pl; return -2; }
  {   // the workspace's O partials as a 2-D u32 tensor [slots][H*D/2]; box = 512 B of kCombRows slots
    cuuint64_t dims[2] = {(cuuint64_t)kTcH * kTcD / 2, (cuuint64_t)pl->ws->slots};
    cuuint64_t strides[1] = {(cuuint64_t)kTcH * kTcD * 2};
    cuuint32_t box[2] = {kCombRowBytes / 4, kCombRows};
    cuuint32_t es[2] = {1, 1};
    CUresult r = pl->encode(&pl->map_part, CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, pl->ws->part_o, dims, strides, box, es,
                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { *msg = "cuTensorMapEncodeTiled (partials) failed"; return -2; }
    // the small-batch path's merge: all workspace buffers as one tensor [kWsBufs * slots][H*D/2]; box = the 256 B of one
    // unit (4 heads x 32 d, fp16) of 32 consecutive slots
    cuuint64_t dims2[2] = {(cuuint64_t)kTcH * kTcD / 2, (cuuint64_t)pl->ws->slots * kWsBufs};
    cuuint32_t box2[2] = {64, 32};
    r = pl->encode(&pl->map_part_small, CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, pl->ws->part_o, dims2, strides, box2, es,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { *msg = "cuTensorMapEncodeTiled (partials, small path) failed"; return -2; }
  }
  p.part_o = pl->ws->part_o; p.part_s = pl->ws->part_s; p.part_m = pl->ws->part_m; p.part_l = pl->ws->part_l; p.piece_info = pl->ws->piece_info;
  TC_CUDA(cudaMalloc(&p.grid_ctr, sizeof(unsigned int)));
  TC_CUDA(cudaMemset(p.grid_ctr, 0, sizeof(unsigned int)));
  p.fused = (init.B <= kTcFusedMaxB && init.fuse_combine) ? 1 : 0;   // opt-in (LSA_MERGE_FUSED)
  pl->smem = sizeof(TcSmem) + 1024;
  TC_CUDA(cudaFuncSetAttribute(attn_tc_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl->smem));
  TC_CUDA(cudaFuncSetAttribute(attn_tc_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl->smem));
  TC_CUDA(cudaFuncSetAttribute(combine_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kCombineSmemMax));
  *out = pl;
  return 0;
}

// One CTA per SM streams at up to ~85 GB/s, twice its fair share of HBM, so the grid is sized to give every
// CTA the same number of whole tiles (e.g. 192 tiles -> 96 CTAs x 2) instead of one CTA per SM with a ragged
// last tile: fewer split partials for S8 to merge, no padded MMA work.
static int pick_grid(const TcPlan* pl, long long tiles_est) {
  const int g = pl->grid_max;
  if (tiles_est <= 0) return 1;
  const long long per = (tiles_est + g - 1) / g;
  return (int)std::max<long long>(1, std::min<long long>(g, (tiles_est + per - 1) / per));
}

int tc_attention(TcPlan* pl, const void* q, void* out, float* lse, long long tiles_est, const TcPrestep* pre, cudaStream_t st,
                 int* launches, int* ctas, std::string* msg, cudaEvent_t ev_mid0, cudaEvent_t ev_mid1, unsigned long long* ktime) {
  if (q != pl->q_cached) {
    if (!encode_rows(pl->encode, &pl->map_q, q, (uint64_t)pl->init.B * kTcH, kTcH, 8, msg)) return -2;
    pl->q_cached = q;
  }
  const int n_attn = pick_grid(pl, tiles_est);
  // fused S8: the whole grid (one CTA per SM, all resident) also merges the partials, so idle SMs help
  const int grid = pl->params.fused ? pl->grid_max : n_attn;
  TcParams prm = pl->params;
  prm.n_attn = n_attn;
  prm.ktime = ktime;
  if (pre) {
    for (int i = 0; i < kTcMaxB / 32; ++i) prm.swap[i] = pre->swap[i];
    prm.k_new = (const __nv_bfloat16*)pre->k_new;
    prm.v_new = (const __nv_bfloat16*)pre->v_new;
  }
  if (prm.fused) {
    pl->grid_total += (unsigned long long)grid;
    prm.grid_target = (unsigned int)pl->grid_total;
    prm.out = (__nv_bfloat16*)out;
    prm.lse = lse;
  }
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t lc{};
  lc.gridDim = dim3(grid); lc.blockDim = dim3(kTcThreads); lc.dynamicSmemBytes = pl->smem; lc.stream = st;
  lc.attrs = attr; lc.numAttrs = 1;
  if (pl->ws->last_small) {       // the small path's launches do not wait for one another: this one waits for all of them
    lc.numAttrs = 0;
    pl->ws->last_small = false;
  }
  if (prm.l2_mask) TC_CUDA(cudaLaunchKernelEx(&lc, attn_tc_kernel<true>, pl->map_pool, pl->map_q, prm));
  else TC_CUDA(cudaLaunchKernelEx(&lc, attn_tc_kernel<false>, pl->map_pool, pl->map_q, prm));
  if (ev_mid0) TC_CUDA(cudaEventRecord(ev_mid0, st));
  if (ev_mid1) TC_CUDA(cudaEventRecord(ev_mid1, st));
  if (prm.fused) {
    *launches = 1;
    *ctas = n_attn;
    return 0;
  }
  cudaLaunchConfig_t lc2{};
  lc2.gridDim = dim3(128, pl->init.B); lc2.blockDim = dim3(kCombineThreads); lc2.dynamicSmemBytes = kCombineSmemPad; lc2.stream = st;
  lc2.attrs = attr; lc2.numAttrs = 1;
  if (pl->init.B <= kCombineSpecMaxB) {
    const int land = (n_attn + kCombRows - 1) / kCombRows * kCombBoxBytes;
    if (land > kCombineSmemPad) lc2.dynamicSmemBytes = land;
    TC_CUDA(cudaLaunchKernelEx(&lc2, combine_tc_kernel, pl->map_part, prm, n_attn, (__nv_bfloat16*)out, lse));
  } else {
    lc2.gridDim = dim3(16, pl->init.B); lc2.dynamicSmemBytes = 0;
    TC_CUDA(cudaLaunchKernelEx(&lc2, combine_tc_wide_kernel, prm, n_attn, (__nv_bfloat16*)out, lse));
  }
  *launches = 2;
  *ctas = n_attn;
  return 0;
}

bool tc_small_supported(const TcPlan* pl) { return pl && pl->small_ok; }

int tc_attention_small(TcPlan* pl, const void* q, void* out, float* lse, const TcSmallStep& step, cudaStream_t st, int* launches,
                       int* ctas, std::string* msg, cudaEvent_t ev_mid0, cudaEvent_t ev_mid1, unsigned long long* ktime) {
  if (q != pl->q_cached) {                          // a few q buffers in rotation (staging images, input rings): keep their maps
    bool hit = false;
    for (auto& e : pl->q_maps)
      if (e.first == q) { pl->map_q = e.second; hit = true; break; }
    if (!hit) {
      if (!encode_rows(pl->encode, &pl->map_q, q, (uint64_t)pl->init.B * kTcH, kTcH, 8, msg)) return -2;
      if (pl->q_maps.size() >= 32) pl->q_maps.clear();
      pl->q_maps.emplace_back(q, pl->map_q);
    }
    pl->q_cached = q;
  }
  TcWorkspace* ws = pl->ws;
  const int B = pl->init.B;
  SmParams prm{};
  long long halves = 0;                              // upper estimate of the flat half-tile list (sizes the grid)
  for (int b = 0; b < B; ++b) {
    const SeqDev& s = pl->init.seq_host[b];
    const TcSmallSeq& h = step.seq[b];
    SmSeq& d = prm.seq[b];
    d.n_hca = s.n_hca; d.cur = h.cur; d.n_cur = h.n_cur; d.w_len = h.w_len; d.app_slot = h.app_slot; d.app_count = h.app_count;
    d.grow_count = h.grow_count;
    d.n_csa = s.n_csa;
    halves += (s.n_hca + kSmHalf - 1) / kSmHalf + 2 * (h.n_cur >= 0 ? h.n_cur : s.k_eff) + (h.w_len + kSmHalf - 1) / kSmHalf;
  }
  // About three launches are in flight at a time (a launch's CTAs start on the SMs its predecessors' CTAs leave), so a
  // launch takes a third of the SMs and every CTA the same, EVEN number of half tiles where the list allows it (an even
  // share keeps the two halves of a 128-row tile together; a lone half is a 64-row box that still costs M = 128 MMAs).
  // Fewer, longer pieces amortise what a CTA pays once - its set-up, the wait for its first rows, the hand-over of the SM
  // (~9 us against ~1.3 us per half tile) - and the step time is SM residence / SM count; measured at cfg 3 (us per
  // step): 32 CTAs 11.2, 48: 10.5, 55: 10.6, 64: 10.85.  A launch the host blocks on has no neighbour to share the
  // machine with and takes every SM; a launch that merely waits for the stream (a swap step: the fetch event) keeps the
  // shared size, because the launches BEHIND it overlap it again (all SMs there: 10.2 us per step, shared size: 10.0).
  const bool alone = step.alone;
  // (the in-launch merge lands at most 160 partial slots per output unit in shared memory: lsa_attn_tc_small.cuh kMuLandBytes)
  const long long g_cap = std::min<long long>(160, (pl->init.max_ctas > 0 || alone) ? pl->grid_max : std::max(1, (pl->init.n_sms - 4) / 3));
  long long per = std::max<long long>(1, (halves + g_cap - 1) / g_cap);
  if (!alone && per > 1 && (per & 1)) ++per;
  const int n_attn = (int)std::max<long long>(1, std::min<long long>(g_cap, (halves + per - 1) / per));
  const int buf = (int)(ws->n_small % kWsBufs);
  // S8: the launch's last n_mrg CTAs to arrive merge its partials (8 units of 4 heads x 32 d each per round), the others
  // leave their SM to the next launch at once; a launch that has the machine to itself lets every CTA merge
  const int n_units = B * 256;
  const int n_mrg = alone ? n_attn : std::min(n_attn, std::max(pl->small_mergers, (n_units + 15) / 16));
  const bool first_after_general = !ws->last_small;  // the general path's combine may still read buffer 0: wait for the stream
  prm.seqs = pl->init.d_seqs; prm.tbl_chunk = pl->init.pool.tbl_chunk; prm.tbl_page = pl->init.pool.tbl_page; prm.seq_maps = pl->d_maps8;
  prm.B = B; prm.k = pl->init.k; prm.n_attn = n_attn; prm.scale_log2 = pl->params.scale_log2;
  prm.part_o = ws->part_o + (size_t)buf * ws->slots * (kTcH * kTcD / 4);
  prm.part_s = ws->part_s + (size_t)buf * ws->slots * kTcPartScales;     // same space, transposed: [32][slots]
  prm.part_m = ws->part_m + (size_t)buf * ws->slots * kTcH;              // [64][slots]
  prm.part_l = ws->part_l + (size_t)buf * ws->slots * kTcH;
  prm.n_slots = (int)ws->slots;
  prm.slot_row0 = buf * (int)ws->slots;
  prm.piece_info = ws->piece_info + (size_t)buf * ws->grid_max;
  prm.arr_ctr = ws->ctrs + buf; prm.arr_target = (ws->arr_total[buf] += (unsigned)n_attn);
  prm.n_mrg = n_mrg;
  prm.done_ctr = ws->ctrs + kWsBufs;
  prm.done_need_buf = ws->done_hist[buf];            // the launch kWsBufs back (same buffer) has been merged
  prm.done_need_prev = ws->done_total;               // the previous launch has been merged
  ws->done_total += (unsigned)n_mrg;
  ws->done_hist[buf] = ws->done_total;
  prm.done_after = ws->done_total;
  prm.host_flag = step.host_flag; prm.host_flag_val = step.host_flag_val;
  prm.out = (__nv_bfloat16*)out; prm.lse = lse; prm.swap = step.swap; prm.W = pl->init.W;
  prm.k_new = (const __nv_bfloat16*)step.k_new; prm.v_new = (const __nv_bfloat16*)step.v_new;
  prm.ktime = ktime;
  prm.tl = n_attn <= kTlCtas ? step.tl : nullptr; prm.tl_seq = step.tl_seq;
  prm.wait_inputs = step.wait_inputs;
  prm.grow_wait = step.grow_wait;
  prm.in_ctr = step.in_ctr; prm.in_need = step.in_need;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t lc{};
  lc.gridDim = dim3(n_attn); lc.blockDim = dim3(kTcThreads); lc.dynamicSmemBytes = sizeof(SmSmem) + 1024; lc.stream = st;
  lc.attrs = attr; lc.numAttrs = (step.serialize || first_after_general) ? 0 : 1;
  if (prm.tl) TC_CUDA(cudaLaunchKernelEx(&lc, attn_tc_small_kernel<true>, pl->map_pool, pl->map_pool64, pl->map_q, pl->map_part_small, pl->maps0, prm));
  else TC_CUDA(cudaLaunchKernelEx(&lc, attn_tc_small_kernel<false>, pl->map_pool, pl->map_pool64, pl->map_q, pl->map_part_small, pl->maps0, prm));
  if (ev_mid0) TC_CUDA(cudaEventRecord(ev_mid0, st));
  if (ev_mid1) TC_CUDA(cudaEventRecord(ev_mid1, st));
  ws->n_small += 1;
  ws->last_small = true;
  *launches = 1;
  *ctas = n_attn;
  return 0;
}

void tc_set_l2_mask(TcPlan* pl, const uint32_t* mask) { pl->params.l2_mask = mask; }

void tc_destroy(TcPlan* pl) {
  if (!pl) return;
  cudaFree(pl->d_maps);
  cudaFree(pl->d_maps8);
  ws_release(pl->ws);
  cudaFree(pl->params.grid_ctr);
  delete pl;
}

}  // namespace lsa
