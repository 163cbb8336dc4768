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
// The backward's workspace holds, per query row of [B*C*H][Rp] (Rp = R rounded up to 64), -LSE*log2(e) as f32 and
// D = rowsum(dO o O) as f32 (dh = 64) or as a 32-byte MMA operand record (dh <= 32); written by the dQ pass and
// read by the dK/dV pass.  The forward needs none.
// query rows [q_row0, q_row1) of every sequence; LSE may be NULL (inference)
// ws: item_fwd_workspace_bytes(s) bytes, only touched when a column mask is given (the a0 column list)
cudaError_t launch_item_fwd(const Shape& s, const void* Q, const void* K, const void* V, void* O, float* LSE,
                            int q_row0, int q_row1, void* ws, cudaStream_t stream);
size_t item_fwd_workspace_bytes(const Shape& s);
// tabattn_item_fwd_noalloc: the forward over all rows with the column list in the library's own device array
// (item_tc_fwd.cu); a masked call needs item_fwd_workspace_bytes(s) <= item_fwd_noalloc_capacity()
cudaError_t launch_item_fwd_noalloc(const Shape& s, const void* Q, const void* K, const void* V, void* O, float* LSE,
                                    cudaStream_t stream);
size_t item_fwd_noalloc_capacity();
cudaError_t launch_item_bwd(const Shape& s, const void* Q, const void* K, const void* V, const void* O,
                            const void* dO, const float* LSE, void* dQ, void* dK, void* dV, float* ws,
                            cudaStream_t stream);
size_t item_bwd_workspace_bytes(const Shape& s);

// ---- sub-blocks around the attention kernels (block_ops.cu) ------------------------
size_t block_ws_bytes(long long cells, int e, int hidden_or_zero, int num_sms);
cudaError_t launch_mlp_fwd(long long cells, int e, int hidden, float alpha, float eps, const void* x, const void* g,
                           const void* W1, const void* W2, void* y, void* h, float* rstd, void* u, void* a,
                           cudaStream_t stream);
cudaError_t launch_mlp_bwd(long long cells, int e, int hidden, float alpha, const void* x, const void* g,
                           const void* W1, const void* W2, const void* h, const float* rstd, const void* u,
                           const void* a, const void* dy, void* dx, float* dg, float* dW1, float* dW2, void* ws,
                           size_t ws_bytes, cudaStream_t stream);
cudaError_t launch_attn_block_fwd(const Shape& s, int axis, float alpha, float eps, const void* x, const void* g,
                                  const void* Wqkv, const void* Wo, void* y, void* h, float* rstd, void* q, void* k,
                                  void* v, void* o, float* lse, void* ws, cudaStream_t stream);
size_t attn_block_bwd_ws_bytes(const Shape& s, int axis, int num_sms);
cudaError_t launch_attn_block_bwd(const Shape& s, int axis, float alpha, const void* x, const void* g,
                                  const void* Wqkv, const void* Wo, const void* h, const float* rstd, const void* q,
                                  const void* k, const void* v, const void* o, const float* lse, const void* dy,
                                  void* dx, float* dg, float* dWqkv, float* dWo, void* ws, size_t ws_bytes,
                                  cudaStream_t stream);
size_t newton_schulz_ws_bytes(int nb, int m, int n);
cudaError_t launch_newton_schulz(int nb, int m, int n, const void* G, void* X, int steps, float ca, float cb, float cc,
                                 float eps, void* ws, cudaStream_t stream);

}  // namespace tabattn
