// Item-axis attention backward on tcgen05: placeholder until the
// dQ and dK/dV kernels land; reports "unsupported" so item_dispatch.cu keeps the SIMT kernels.
#include "kernels.h"

namespace tabattn {

bool item_tc_bwd_supported(const Shape&) { return false; }

cudaError_t launch_item_bwd_tc(const Shape&, const void*, const void*, const void*, const void*, const void*,
                               const float*, void*, void*, void*, float*, cudaStream_t) {
  return cudaErrorNotSupported;
}

}  // namespace tabattn
