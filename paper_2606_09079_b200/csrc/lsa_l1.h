// lsa_l1.h - host interface of the paper-exact Level-1 Memory Indexer (lsa_l1.cu).
#pragma once
#include <cuda_runtime.h>

#include <string>

#include "lsa_common.cuh"

namespace lsa {

struct L1Plan;

struct L1LayerW {
  const void* W_dq;    // DEVICE [d_c][Dh]
  const void* W_iuq;   // DEVICE [n_h * c_I][d_c]
  const void* W_w;     // DEVICE [n_h][Dh]
};

struct L1Init {
  int B, n_layers, Dh, d_c, n_chunks_max, n_sms;
  L1LayerW layers[4];
  const void* const* index_k;   // HOST [B * n_layers] device pointers, [n_csa_b][c_I] each (only read during create)
  const SeqDev* seq_host;       // host copy of the per-sequence records
};

bool l1_supported(int dtype, int C, int c_I, int n_h);
int l1_create(const L1Init& init, L1Plan** out, std::string* msg);     // 0 or an lsa_status
int l1_select(L1Plan* plan, const SeqDev* d_seqs, const void* h, const int* ids, const int* hrows, int n, int k, float threshold,
              int32_t* sel_idx, float* sel_score, cudaStream_t st, int* launches, std::string* msg);
void l1_destroy(L1Plan* plan);

}  // namespace lsa
