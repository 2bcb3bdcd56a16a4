// lsa_index_tc.cu - S1 for a batch of firing sequences on tcgen05 tensor cores (sm_100a).
//
//   z[i][e] = sum_d W_q[e][d] * h[i][d]          PAPER.md l.61-65 Eq.(1)-(2) collapsed (DESIGN R1); BASELINE.json
//   north_star: "query-tower projection as a real dense GEMV/GEMM on tensor cores only when batched".
//
// With n >= 8 sequences firing together (BASELINE cfg 5: all 8) the projection is a real [E x Dh] . [Dh x n]
// contraction; the warp-per-row GEMV (lsa_index.cu) reads W_q once per 4 sequences and spends its time on scalar FMAs.
// Here W_q is streamed ONCE: "weights on M" - per CTA a [128 rows of W_q] x [512 columns] block arrives as four 32 KiB
// TMA boxes ([2 d-blocks][128 rows][128 B], 128-byte swizzle = the K-major A operand), the n hidden states (padded to
// N = 16 by the tensor map's zero fill) as four 4 KiB boxes (K-major B operand), 32 MMAs of M=128, N=16, K=16
// accumulate z^T[128 x 16] in TMEM, and the epilogue writes the block's partial sums to z_part[k-split][i][e].
// The E/128 x Dh/512 CTAs (32 at E=512, Dh=4096) split the reduction dimension; the partials are added in a fixed
// order by the scoring kernel (score_kernel's n_part), so the result does not depend on scheduling.
// bf16 only: the fp32 config keeps the fp32 GEMV (TF32 would drop mantissa bits the oracle comparison needs).
#include <cuda.h>
#include <cuda_bf16.h>

#include <string>

#include "lsa_kernels.h"
#include "lsa_tc_ptx.cuh"

namespace lsa {
using namespace ptx;

constexpr int kQtcRows = 128;               // rows of W_q per CTA (M)
constexpr int kQtcCols = 512;               // columns of W_q per CTA: 4 stages of 128
constexpr int kQtcN = 16;                   // sequences per launch, padded (N)
constexpr int kQtcThreads = 128;

struct QtcSmem {
  alignas(1024) unsigned char w[4][32768];  // [2 d-blocks][128 rows][128 B], SW128
  alignas(1024) unsigned char h[4][4096];   // [2 d-blocks][16 rows][128 B], SW128
  uint64_t full[4], done;
  uint32_t tmem_base;
};

__global__ void __launch_bounds__(kQtcThreads, 1)
qtower_tc_kernel(const __grid_constant__ CUtensorMap map_w, const __grid_constant__ CUtensorMap map_h, float* __restrict__ z_part,
                 int n, int E) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  QtcSmem& sm = *reinterpret_cast<QtcSmem*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int e0 = blockIdx.x * kQtcRows, ks = blockIdx.y;
  if (tid == 0) {
    for (int i = 0; i < 4; ++i) mbar_init(&sm.full[i], 1);
    mbar_init(&sm.done, 1);
    fence_mbar_init();
    prefetch_tmap(&map_w);
    prefetch_tmap(&map_h);
  }
  if (warp == 1) tmem_alloc(&sm.tmem_base, 32);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  // W_q never depends on the stream: its four boxes are requested before the launch dependency is waited for
  if (warp == 0 && elect_one()) {
    for (int s = 0; s < 4; ++s) {
      mbar_arrive_expect_tx(&sm.full[s], 32768 + 4096);
      tma_load_3d(sm.w[s], &map_w, 0, e0, (ks * kQtcCols) / 64 + 2 * s, &sm.full[s]);
    }
  }
  griddep_wait();                 // h may come from the kernel before this one
  griddep_launch_dependents();
  if (warp == 0 && elect_one()) {
    for (int s = 0; s < 4; ++s) tma_load_3d(sm.h[s], &map_h, 0, 0, (ks * kQtcCols) / 64 + 2 * s, &sm.full[s]);
    constexpr uint32_t idesc = make_idesc_bf16(kQtcRows, kQtcN, 0, 0);      // A = W rows (K-major), B = h rows (K-major)
    const uint32_t tD = sm.tmem_base;
    for (int s = 0; s < 4; ++s) {
      mbar_wait(&sm.full[s], 0, 60);
      tc_fence_after();
      const uint64_t da = make_sdesc(smem_u32(sm.w[s]), 16, 1024, kLayoutSw128);
      const uint64_t db = make_sdesc(smem_u32(sm.h[s]), 16, 1024, kLayoutSw128);
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        const uint64_t oa = (uint64_t)(((k >> 2) * 16384 + (k & 3) * 32) >> 4);
        const uint64_t ob = (uint64_t)(((k >> 2) * 2048 + (k & 3) * 32) >> 4);
        umma_bf16(tD, da + oa, db + ob, idesc, (s | k) != 0);
      }
    }
    umma_commit(&sm.done);
  }
  __syncwarp();
  // ---- epilogue: thread = row e0 + tid of W_q; 16 accumulator columns = the sequences ----
  mbar_wait(&sm.done, 0, 61);
  tc_fence_after();
  uint32_t v[16];
  const uint32_t taddr = sm.tmem_base + ((uint32_t)(warp * 32) << 16);
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
        "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
      : "r"(taddr) : "memory");
  tmem_wait_ld();
  float* zp = z_part + (size_t)ks * n * E + e0 + tid;
#pragma unroll
  for (int i = 0; i < 16; ++i)
    if (i < n) zp[(size_t)i * E] = __uint_as_float(v[i]);
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(sm.tmem_base, 32);
  }
}

// ---- host ----------------------------------------------------------------------------------------------------------
typedef CUresult (*QtcEncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                CUtensorMapFloatOOBfill);

// [rows][cols] bf16 seen as (64 columns, rows, cols / 64 d-blocks); a box lands as [2 d-blocks][box_rows][128 B]
static bool qtc_encode(QtcEncodeFn enc, CUtensorMap* m, const void* ptr, uint64_t rows, uint64_t cols, uint32_t box_rows) {
  cuuint64_t dims[3] = {64, rows, cols / 64};
  cuuint64_t strides[2] = {cols * 2, 128};
  cuuint32_t box[3] = {64, box_rows, 2};
  cuuint32_t es[3] = {1, 1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(ptr), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

bool qtower_tc_usable(int dtype, int E, int Dh, int n, const int* hrows) {
  if (dtype != 1 || n < 8 || n > kQtcN || E % kQtcRows || Dh % kQtcCols) return false;
  for (int i = 1; i < n; ++i)
    if (hrows[i] != hrows[0] + i) return false;       // the hidden states must be consecutive rows of h (one TMA box)
  return true;
}

int qtower_tc_splits(int Dh) { return Dh / kQtcCols; }

// z_part [Dh / 512][n][E] fp32.  W_q's tensor map is cached by the caller-visible pointer.
cudaError_t launch_qtower_tc(const void* W, const void* h, int h_row0, int n, float* z_part, int E, int Dh, cudaStream_t st) {
  static QtcEncodeFn enc = nullptr;
  static const void* w_cached = nullptr;
  static int e_cached = 0, dh_cached = 0;
  static CUtensorMap map_w;
  static bool attr = false;
  if (!enc) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn) return cudaErrorNotSupported;
    enc = (QtcEncodeFn)fn;
  }
  if (W != w_cached || E != e_cached || Dh != dh_cached) {
    if (!qtc_encode(enc, &map_w, W, (uint64_t)E, (uint64_t)Dh, kQtcRows)) return cudaErrorInvalidValue;
    w_cached = W; e_cached = E; dh_cached = Dh;
  }
  CUtensorMap map_h;
  const __nv_bfloat16* hb = reinterpret_cast<const __nv_bfloat16*>(h) + (size_t)h_row0 * Dh;
  if (!qtc_encode(enc, &map_h, hb, (uint64_t)n, (uint64_t)Dh, kQtcN)) return cudaErrorInvalidValue;   // rows n.. : zero fill
  const size_t smem = sizeof(QtcSmem) + 1024;
  if (!attr) {
    cudaError_t e = cudaFuncSetAttribute(qtower_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    attr = true;
  }
  return launch_pdl(qtower_tc_kernel, dim3(E / kQtcRows, Dh / kQtcCols), dim3(kQtcThreads), smem, st, map_w, map_h, z_part, n, E);
}

}  // namespace lsa
