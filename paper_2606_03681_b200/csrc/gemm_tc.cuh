// Dense bf16 GEMM core on tcgen05 (the projections, the per-cell MLP and the
// batched Newton-Schulz iteration are plain contractions around the attention kernels).  Internal interface.
//
//   D[b][m][n] = epilogue( sum_k A[b](m, k) * B[b](n, k) )          fp32 accumulation in TMEM
//
// Operand layouts (row-major tensors in global memory):
//   A_MN = 0: A stored [M][K] (K contiguous)        A_MN = 1: A stored [K][M] (M contiguous: A^T of the storage)
//   B_MN = 0: B stored [N][K] (K contiguous)        B_MN = 1: B stored [K][N] (N contiguous)
// so  Y = X W^T (nn.Linear, W [out][in])  is (0,0);  dX = dY W  is (0,1);  dW = dY^T X  is (1,1), reduced over
// the cells with split-K slabs (fp32 partial tiles + a deterministic reduction kernel, no atomics).
//
// Epilogue (per element, in this order): v = alpha * acc;  v *= row_scale[m] (RMSNorm folded into the weights);
// aux_mode 1: v += beta * aux[m][n];  act 1: v = gelu(v);  aux_mode 2: v *= gelu'(aux[m][n]);  aux_mode 3:
// v = beta * aux + v (same as 1, kept for the Newton-Schulz update);  -> bf16, through a swizzled staging tile and
// one TMA store per 64 columns.  The output may be split over up to three tensors of `split_cols` columns each
// (the QKV projection writes Q, K and V).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace tabattn {
namespace gemm {

enum { AUX_NONE = 0, AUX_ADD = 1, AUX_GELU_GRAD = 2 };
enum { ACT_NONE = 0, ACT_GELU = 1 };

struct Operand {
  const void* ptr;          // (A only: first of up to three tensors when a_split_k > 0)
  int mn_major;        // see above
  long long ld;        // leading dimension in elements (row pitch of the stored matrix)
  long long batch_stride;   // elements between batches (0 = shared by all batches)
};

struct Problem {
  int M, N, K, batch;
  Operand A, B;
  // K-major A split along K over up to three tensors of a_split_k columns each (dh = [dq | dk | dv] W):
  // A.ptr, A2, A3, all with A's pitch and batch stride; 0 = one tensor.  a_split_k % 64 == 0.
  const void* A2;
  const void* A3;
  int a_split_k;
  // MN-major A split along M over three tensors of a_split_m rows of the output each (dWqkv = [dq | dk | dv]^T h in
  // one launch): A.ptr, A2, A3 with A's pitch; 0 = one tensor.  a_split_m % 128 == 0, M == 3 a_split_m.
  int a_split_m;
  // output: bf16 [M][ldc] per batch, optionally split over tensors of split_cols columns
  void* C[3];
  long long ldc, c_batch_stride;
  int split_cols;           // 0 = one tensor
  // dual output (MLP up-projection): C[0] receives the value BEFORE the activation, C[1] the value after it
  int dual_out;
  // split-K: partial != nullptr -> fp32 partial tiles [slabs][M][N] instead of C (batch must be 1; slabs >= 1)
  int slabs;
  float* partial;
  // epilogue
  float alpha, beta;
  const float* row_scale;   // [batch * M] or nullptr
  int act, aux_mode;
  const void* aux;          // bf16 [M][ld_aux] per batch
  long long ld_aux, aux_batch_stride;
};

// Split-K slab count for a reduction over K with `tiles` output tiles: about two CTAs per SM, never an empty slab.
// (launch() recomputes the k-blocks per slab from it and rejects a count that leaves a slab empty.)
int slabs_for(long long K, int tiles, int num_sms);

// Enqueue the GEMM on `stream`.  Constraints: K, N multiples of 8; ld* multiples of 8; pointers 16-byte aligned.
cudaError_t launch(const Problem& p, cudaStream_t stream);

// out[m][n] (bf16 or fp32) = sum over slabs of partial[s][m][n] * scale
cudaError_t launch_reduce_slabs(const float* partial, int slabs, long long mn, float scale, void* out, bool out_f32,
                                cudaStream_t stream);

}  // namespace gemm
}  // namespace tabattn
