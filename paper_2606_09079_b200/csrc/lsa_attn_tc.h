// lsa_attn_tc.h - host interface of the tcgen05/TMA split-K decode attention (lsa_attn_tc.cu).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

#include "lsa_common.cuh"

namespace lsa {

struct TcPlan;

struct TcInit {
  int B, k, W, P, n_sms, max_ctas;
  int fuse_combine;         // 1: merge the split partials inside the attention kernel when B is small
  void* hot_pool;
  const SeqDev* seq_host;   // host copy of the immutable per-sequence fields
  SeqDev* d_seqs;
  PoolDev pool;
  float sm_scale;
  cudaStream_t stream;      // compute stream of the context: contexts of one stream share the split-K workspace
};

// bf16, H = 64 query heads sharing one K/V of D = 512, pages of C = 128 rows (BASELINE cfg 2-5)
bool tc_supported(int dtype, int H, int D, int C);
int tc_create(const TcInit& init, TcPlan** out, std::string* msg);   // 0 or an lsa_status
// S6 + window append folded into the attention launch (steps without a trigger)
struct TcPrestep {
  unsigned int swap[8];     // bit b: the staged table of sequence b becomes current (B <= 256)
  const void* k_new;        // DEVICE [B][D] or null
  const void* v_new;
};

// tiles_est: upper estimate of the batch's 128-key tiles (sizes the grid; the kernel partitions the exact list)
// ev_mid0 / ev_mid1 (optional, profiling): recorded between the attention and the combine kernel
int tc_attention(TcPlan* plan, const void* q, void* out, float* lse, long long tiles_est, const TcPrestep* pre, cudaStream_t st,
                 int* launches, int* ctas, std::string* msg, cudaEvent_t ev_mid0 = nullptr, cudaEvent_t ev_mid1 = nullptr,
                 unsigned long long* ktime = nullptr /* DEVICE [2] = {~0, 0}: kernel working-time stamps */);
// ---- small batches (B <= 4): lsa_attn_tc_small.cuh --------------------------------------------------------------
// The host's mirror of one sequence as the launch will see it (swap and append already applied).
struct TcSmallSeq {
  int cur;                  // table buffer attended
  int n_cur;                // its entries, or -1 when only the device knows (selection given on the device)
  int w_len;                // attended ring rows, this launch's append included
  int app_slot;             // ring slot written by this launch, or -1
  unsigned int app_count;   // appends enqueued before this launch
  unsigned int grow_count;  // lsa_append_compressed calls enqueued for the sequence before this launch
};
struct TcSmallStep {
  TcSmallSeq seq[4];
  unsigned int swap;        // bit b: sequence b's staged table becomes current with this launch (records catch up in S8)
  const void* k_new;        // DEVICE [B][D] or null
  const void* v_new;
  int serialize;            // 1: the launch waits for everything before it in the stream (trigger and swap steps); 0: its
                            // CTAs start as the previous step's leave their SMs, while that step is still being merged
  int wait_inputs;          // 1: q / k_new / v_new may have been produced by the kernel just before this launch
  const unsigned int* in_ctr;   // q / k_new / v_new are complete once *in_ctr has reached in_need (null: see wait_inputs)
  unsigned int in_need;
  int grow_wait;            // 1: an append kernel runs beside the previous launch: wait for grow_count before HCA / page rows
  int alone;                // 1: the caller blocks on this step (no neighbour launch to share the SMs with): use them all
  unsigned int* host_flag;  // PINNED HOST word (device alias) set to host_flag_val when `out` is complete, or null
  unsigned int host_flag_val;
  unsigned long long* tl;   // DEVICE timeline record of this launch ([160 CTAs][12 stamps], include/lsa.h LSA_TL_*) or null
  unsigned int tl_seq;
};
bool tc_small_supported(const TcPlan* plan);
int tc_attention_small(TcPlan* plan, const void* q, void* out, float* lse, const TcSmallStep& step, cudaStream_t st,
                       int* launches, int* ctas, std::string* msg, cudaEvent_t ev_mid0 = nullptr, cudaEvent_t ev_mid1 = nullptr,
                       unsigned long long* ktime = nullptr);

// Level 2: key mask [B][k][4] words used by the launches that follow (null: off); see TcParams::l2_mask
void tc_set_l2_mask(TcPlan* plan, const uint32_t* mask);
void tc_destroy(TcPlan* plan);

}  // namespace lsa
