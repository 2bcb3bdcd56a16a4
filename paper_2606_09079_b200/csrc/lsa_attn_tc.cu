// lsa_attn_tc.cu - tcgen05/TMA split-K decode attention (placeholder until the kernel lands).
#include "lsa_attn_tc.h"

namespace lsa {
struct TcPlan {};
bool tc_supported(int, int, int, int) { return false; }
int tc_create(const TcInit&, TcPlan**, std::string* msg) { *msg = "not built"; return -6; }
int tc_attention(TcPlan*, const void*, void*, float*, cudaStream_t, int*, int*, std::string* msg) { *msg = "not built"; return -6; }
void tc_destroy(TcPlan*) {}
}  // namespace lsa
