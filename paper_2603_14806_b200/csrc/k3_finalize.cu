// placeholder until the tcgen05 K3 lands
#include "common.h"
namespace foldcp {
int launch_k3_finalize_bf16(const void*, const void*, const void*, const foldcp_trimul_params*, int,
                            void*, cudaStream_t) {
  return FOLDCP_ERR_UNSUPPORTED;
}
}  // namespace foldcp
