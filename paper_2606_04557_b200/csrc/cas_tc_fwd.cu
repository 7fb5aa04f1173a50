// placeholder until the tcgen05 kernels land
#include "cas_internal.h"
namespace cas {
bool tc_supported(const cas_pool*, const cas_slot_table*, int) { return false; }
int tc_attn_fwd(const AttnArgs&) { set_error("tc path not built"); return CAS_ERR_SHAPE; }
int tc_attn_bwd(const AttnArgs&) { set_error("tc path not built"); return CAS_ERR_SHAPE; }
size_t tc_bwd_workspace(const cas_slot_table*, int, int) { return 0; }
int tc_make_pool_maps(cas_pool*) { return CAS_OK; }
}
