// Item-axis dispatch: picks the tcgen05 kernels (item_tc_*.cu) or the SIMT bring-up kernels
// (item_simt.cu) for a shape and owns the workspace layout.  SURVEY.md §8(a) rows a3-a5.
//
// Workspace of tabattn_item_bwd: two f32 arrays [B*C*H][Rp] (Rp = R rounded up to 64), written by
// the prep kernel and read by both passes: lse2 = LSE * log2(e) and D = rowsum(dO o O).
// tabattn_item_fwd needs none.
#include <stdlib.h>
#include <string.h>

#include "kernels.h"

namespace tabattn {

// item_simt.cu
cudaError_t launch_item_fwd_simt(const Shape& s, const void* Q, const void* K, const void* V, void* O, float* LSE,
                                 cudaStream_t stream);
cudaError_t launch_item_bwd_simt(const Shape& s, const void* Q, const void* K, const void* V, const void* O,
                                 const void* dO, const float* LSE, void* dQ, void* dK, void* dV, float* Dws,
                                 cudaStream_t stream);
// item_tc_fwd.cu / item_tc_bwd.cu
bool item_tc_supported(const Shape& s);
bool item_tc_bwd_supported(const Shape& s);
int item_bwd_padded_rows(const Shape& s);
cudaError_t launch_item_fwd_tc(const Shape& s, const void* Q, const void* K, const void* V, void* O, float* LSE,
                               cudaStream_t stream);
cudaError_t launch_item_bwd_tc(const Shape& s, const void* Q, const void* K, const void* V, const void* O,
                               const void* dO, const float* LSE, void* dQ, void* dK, void* dV, float* Dws,
                               cudaStream_t stream);

namespace {
// TABATTN_ITEM_IMPL=simt forces the SIMT path (used by the tests to cross-check the two on the GPU).
bool force_simt() {
  const char* e = getenv("TABATTN_ITEM_IMPL");
  return e && strcmp(e, "simt") == 0;
}
}  // namespace

size_t item_fwd_workspace_bytes(const Shape&) { return 0; }

size_t item_bwd_workspace_bytes(const Shape& s) {
  return (size_t)2 * s.B * s.C * s.H * item_bwd_padded_rows(s) * sizeof(float);
}

cudaError_t launch_item_fwd(const Shape& s, const void* Q, const void* K, const void* V, void* O, float* LSE,
                            void* /*ws*/, cudaStream_t stream) {
  if (!force_simt() && item_tc_supported(s)) return launch_item_fwd_tc(s, Q, K, V, O, LSE, stream);
  return launch_item_fwd_simt(s, Q, K, V, O, LSE, stream);
}

cudaError_t launch_item_bwd(const Shape& s, const void* Q, const void* K, const void* V, const void* O,
                            const void* dO, const float* LSE, void* dQ, void* dK, void* dV, void* ws,
                            cudaStream_t stream) {
  float* Dws = static_cast<float*>(ws);
  if (!force_simt() && item_tc_bwd_supported(s))
    return launch_item_bwd_tc(s, Q, K, V, O, dO, LSE, dQ, dK, dV, Dws, stream);
  return launch_item_bwd_simt(s, Q, K, V, O, dO, LSE, dQ, dK, dV, Dws, stream);
}

}  // namespace tabattn
