// Internal launch interface between the C ABI (api.cu) and the kernels.  Not exported.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "common.cuh"

namespace tabattn {

// ---- feature axis (feature_simt.cu) -------------------------------------------------------------
cudaError_t launch_feature_fwd(const Shape& s, const void* Q, const void* K, const void* V, void* O, float* LSE,
                               cudaStream_t stream);
cudaError_t launch_feature_bwd(const Shape& s, const void* Q, const void* K, const void* V, const void* O,
                               const void* dO, const float* LSE, void* dQ, void* dK, void* dV,
                               cudaStream_t stream);
bool feature_shape_supported(const Shape& s);

// ---- item axis ------------------------------------------------------------------------------------
// D (rowsum(dO o O), [B,C,H,R] f32) lives in the caller's workspace.
cudaError_t launch_item_fwd(const Shape& s, const void* Q, const void* K, const void* V, void* O, float* LSE,
                            void* ws, cudaStream_t stream);
cudaError_t launch_item_bwd(const Shape& s, const void* Q, const void* K, const void* V, const void* O,
                            const void* dO, const float* LSE, void* dQ, void* dK, void* dV, void* ws,
                            cudaStream_t stream);
size_t item_fwd_workspace_bytes(const Shape& s);
int num_sms();  // SM count of the current device (cached)
size_t item_bwd_workspace_bytes(const Shape& s);

}  // namespace tabattn
