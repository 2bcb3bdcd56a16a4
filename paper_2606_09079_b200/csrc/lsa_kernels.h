// lsa_kernels.h - host-side launchers of the LSA kernels (internal to liblsa).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "lsa_common.cuh"

namespace lsa {

struct AttnGeom {          // host-computed split geometry of one S7 launch
  int keys_per_cta;        // virtual keys per split (multiple of the tile)
  int s_max;               // gridDim.x : splits of the longest sequence
};

// ---- S1-S3 (lsa_index.cu) ---------------------------------------------------------------
// z[i][e] = sum_d W[e][d] * h[rows.ids[i]][d]           (fp32 out, i < rows.n)
cudaError_t launch_qtower(int dtype, const void* W, const void* h, const FireList& rows, float* z, int E,
                          int Dh, cudaStream_t st);
// scores[i][c] = (z_i . Emb_{b_i}[c]) / max(||z_i||, 1e-12)
// (z may be n_part partial sums [n_part][fire.n][E], added in order)
cudaError_t launch_scores(int dtype, const SeqDev* seqs, const FireList& fire, const float* z,
                          float* scores, int E, int n_chunks_max, cudaStream_t st, int n_part = 1);
// S1 for 8..16 sequences firing together, bf16, on tensor cores (lsa_index_tc.cu): z_part [Dh / 512][n][E]
bool qtower_tc_usable(int dtype, int E, int Dh, int n, const int* hrows);
int qtower_tc_splits(int Dh);
cudaError_t launch_qtower_tc(const void* W, const void* h, int h_row0, int n, float* z_part, int E, int Dh, cudaStream_t st);
// sel_idx[i][0..k) / sel_score: first k_eff by (score desc, chunk idx asc), rest -1 / -inf
cudaError_t launch_topk(const SeqDev* seqs, const FireList& fire, const float* scores,
                        int n_chunks_max, int k, int32_t* sel_idx, float* sel_score, cudaStream_t st);

// S1-S3 with the scratch in a file-scope device array (lsa_index.cu): no allocation.  Limits of that array:
constexpr int kStaticSeqs = 8;         // sequences per call
constexpr int kStaticE = 4096;         // E at most
constexpr int kStaticChunks = 16384;   // chunks per sequence at most
// chunk_emb / n_chunks: HOST arrays [n]; 0 or an lsa_status (text in msg)
int index_select_static(int dtype, const void* W_q, const void* h, const void* const* chunk_emb, const int* n_chunks, int n, int E,
                        int Dh, int k, int32_t* sel_idx, float* sel_score, cudaStream_t st, char* msg, size_t msg_len);

// ---- S4-S6 (lsa_residency.cu) -----------------------------------------------------------
// P = pages managed by the LRU; k_cap = recalled chunks per table at most (0: k); C = entries per chunk (tail entry of a
// growing sequence, 0: static context)
cudaError_t launch_residency(SeqDev* seqs, PoolDev pool, const FireList& fire, const int32_t* sel_idx,
                             int B, int k, int P, long long page_bytes, cudaStream_t st, int k_cap = 0, int C = 0);
// NEXT-4 (second half): one block per listed sequence writes the handed-over CSA / HCA entries and, when a chunk completes
// or a new tail chunk starts, updates the records and page tables (lsa_residency.cu: append_compressed_kernel)
struct AppendList {
  int n;
  int ids[kFireMax];
  long long n_csa[kFireMax];      // host mirrors BEFORE the call: the kernel does not depend on an earlier append having landed
  int n_hca[kFireMax];
  unsigned int epoch[kFireMax];   // value released to SeqDev::grow_epoch once the rows are written
};
cudaError_t launch_append_compressed(int dtype, SeqDev* seqs, PoolDev pool, void* hot_pool, const AppendList& list, int row0,
                                     const void* csa_k, const void* csa_v, const void* hca_k, const void* hca_v, const void* emb_rows,
                                     int D, int E, int C, int k, int k_sel, long long page_bytes, cudaStream_t st, bool beside_previous);
// cold_page_bytes != page_bytes: FP8 cold pages (half the bytes), dequantised while copied
cudaError_t launch_fetch(PoolDev pool, void* hot_pool, long long page_bytes, int n_ctas,
                         cudaStream_t st, long long cold_page_bytes);
// quantise n_blocks blocks of block_elems bf16 elements into e4m3 codes in the mapped cold pool + one scale per block
cudaError_t launch_export_fp8(const void* src, void* dst_mapped, float* scales, long long n_blocks, long long block_elems, cudaStream_t st);
// NEXT-4: copy `bytes` (multiple of 16) from device memory into the mapped pinned cold pool
cudaError_t launch_export(const void* src, void* dst_mapped, long long bytes, int n_ctas, cudaStream_t st);
// swap tables of sequences whose bit is set in swap_mask; append k_new/v_new rows to the ring
cudaError_t launch_prestep(int dtype, SeqDev* seqs, int B, int D, int W, const uint32_t* swap_mask_words,
                           int n_words, const void* k_new, const void* v_new, cudaStream_t st);

// ---- S7-S8, SIMT implementation (lsa_attn_simt.cu) ---------------------------------------
bool simt_supported(int dtype, int H, int D);
int simt_tile_keys();
cudaError_t simt_smem_bytes(int dtype, int H, int D, int k, size_t* bytes);
cudaError_t simt_max_ctas_per_sm(int dtype, int H, int D, int k, int* ctas);
cudaError_t launch_attn_simt(int dtype, int H, int D, int C, int k, const SeqDev* seqs, PoolDev pool,
                             const void* hot_pool, const void* q, float sm_scale, AttnGeom g, int B,
                             float* part_o, float* part_ml, cudaStream_t st);
cudaError_t launch_combine(int dtype, int H, int D, int C, const SeqDev* seqs, AttnGeom g, int B,
                           const float* part_o, const float* part_ml, void* out, float* lse,
                           cudaStream_t st);

}  // namespace lsa
