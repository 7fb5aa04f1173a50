// Tensor-core backward: not written yet -- the bf16 backward currently runs on the CUDA-core kernels.
#include "cas_internal.h"
namespace cas {
int tc_attn_bwd(const AttnArgs& a) { return simt_attn_bwd(a); }
size_t tc_bwd_workspace(const cas_slot_table*, int, int) { return 0; }
}  // namespace cas
