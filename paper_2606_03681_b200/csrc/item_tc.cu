// tcgen05 item-axis kernels (placeholder until the TMA/TMEM pipeline lands): reports "unsupported"
// so that item_dispatch.cu routes every shape to the SIMT kernels.
#include "kernels.h"

namespace tabattn {

bool item_tc_supported(const Shape&) { return false; }

cudaError_t launch_item_fwd_tc(const Shape&, const void*, const void*, const void*, void*, float*, cudaStream_t) {
  return cudaErrorNotSupported;
}

cudaError_t launch_item_bwd_tc(const Shape&, const void*, const void*, const void*, const void*, const void*,
                               const float*, void*, void*, void*, float*, cudaStream_t) {
  return cudaErrorNotSupported;
}

}  // namespace tabattn
