// placeholder until the tcgen05 K1 lands
#include "common.h"
namespace foldcp {
int launch_k1_project_bf16(const void*, const void*, const foldcp_trimul_params*, int, void*, void*,
                           cudaStream_t) {
  return FOLDCP_ERR_UNSUPPORTED;
}
}  // namespace foldcp
