// lsa_l2.h - host interface of Level 2: the native Lightning Indexer inside the resident set (lsa_l2.cu).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

#include "lsa_common.cuh"

namespace lsa {

struct L2Plan;

struct L2Init {
  int B, k, k2, n_sms;
  const void* const* index_k;   // HOST [B] device pointers, [n_csa_b][c_I] bf16 each (only read during create)
  const SeqDev* seq_host;       // host copy of the per-sequence records
  const int* tbl_chunk;         // DEVICE [B][2][k] page tables (chunk ids)
};

bool l2_supported(int dtype, int C, int c_I, int n_h);
int l2_create(const L2Init& init, L2Plan** out, std::string* msg);     // 0 or an lsa_status
// Scores the valid rows of every page of the sequences' CURRENT tables and marks the Top-k2 of each sequence.
// mask: DEVICE [B][k][4] words (see TcParams::l2_mask) owned by the plan.
// swap_words (HOST [8] or null): bit b = sequence b's staged table becomes current in the attention launch that follows
// (S6 folded into it), so Level 2 must score that table although the records still show it as pending.
int l2_select(L2Plan* plan, const SeqDev* d_seqs, const void* q_idx, const float* w_idx, int32_t* sel_entries, float* sel_score,
              const unsigned* swap_words, cudaStream_t st, int* launches, std::string* msg);
const uint32_t* l2_mask(const L2Plan* plan);
void l2_destroy(L2Plan* plan);

}  // namespace lsa
