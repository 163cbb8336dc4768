// Internal launch interface between the C ABI (api.cu) and the kernels.  Not exported.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "common.cuh"
#include "device.h"

namespace tabattn {

// ---- feature axis (feature_tc_fwd.cu, feature_tc_bwd.cu) ---------------------------------------------------------------------
cudaError_t launch_feature_fwd(const Shape& s, const void* Q, const void* K, const void* V, void* O, float* LSE,
                               void* ws, cudaStream_t stream);
cudaError_t launch_feature_bwd(const Shape& s, const void* Q, const void* K, const void* V, const void* O,
                               const void* dO, const float* LSE, void* dQ, void* dK, void* dV, void* ws,
                               cudaStream_t stream);
// forward-only inference: rows [row0, row1) of every table, no LSE
cudaError_t launch_feature_fwd_infer(const Shape& s, const void* Q, const void* K, const void* V, void* O, int row0,
                                     int row1, void* ws, cudaStream_t stream);
bool feature_shape_supported(const Shape& s);
size_t feature_workspace_bytes(const Shape& s);   // masked calls: per-table geometry built by the a0 prep kernel

// ---- item axis (item_tc_fwd.cu, item_tc_bwd.cu) ---------------------------------------------------------
// The backward's workspace holds two f32 arrays [B*C*H][Rp] (Rp = R rounded up to 64): -LSE*log2(e) and
// D = rowsum(dO o O), written by the dQ pass and read by the dK/dV pass.  The forward needs none.
// query rows [q_row0, q_row1) of every sequence; LSE may be NULL (inference)
cudaError_t launch_item_fwd(const Shape& s, const void* Q, const void* K, const void* V, void* O, float* LSE,
                            int q_row0, int q_row1, cudaStream_t stream);
cudaError_t launch_item_bwd(const Shape& s, const void* Q, const void* K, const void* V, const void* O,
                            const void* dO, const float* LSE, void* dQ, void* dK, void* dV, float* ws,
                            cudaStream_t stream);
size_t item_bwd_workspace_bytes(const Shape& s);

}  // namespace tabattn
