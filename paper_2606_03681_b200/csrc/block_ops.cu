// The sub-blocks around the attention kernels, built from the tcgen05 GEMM core
// (gemm_tc.cu), the attention kernels and three small memory-bound kernels (RMSNorm forward / backward, Frobenius
// normalisation).  PAPER.md:L69 (block order), L91 (pre-norm), L99 (residual decay), L105/L294 (RMSNorm), L277
// (explicit QKV), L95/L286 (batched Newton-Schulz).  Readings: DESIGN.md §2 (b1-b6).
#include <cuda_runtime.h>
#include <math.h>

#include "common.cuh"
#include "device.h"
#include "gemm_tc.cuh"
#include <algorithm>

#include "kernels.h"

namespace tabattn {

namespace {

constexpr int kNormWarps = 8;        // warps per CTA of the RMSNorm kernels
constexpr int kNormRows = 4;         // rows a warp has in flight (independent 16-byte loads per lane)

// The RMSNorm kernels are pure streams (2-5 passes over [cells][e]); a warp owns whole rows, a lane CPL 16-byte
// chunks of each (CPL = ceil(e / 256): 1 for the model widths 192 and 256), and works on kNormRows rows at once so
// that enough loads are in flight (profiles/r02_blocks.md: one row per warp reached 30 % / 20 % of HBM).

// h = rmsnorm(alpha x) o g (bf16), rstd = 1 / sqrt(mean((alpha x)^2) + eps) (fp32)
template <int CPL>
__global__ void __launch_bounds__(kNormWarps * 32)
rmsnorm_fwd_kernel(const uint4* __restrict__ x, const uint4* __restrict__ g, uint4* __restrict__ h,
                   float* __restrict__ rstd, long long M, int e, float alpha, float eps) {
  const int lane = threadIdx.x & 31, chunks = e >> 3;
  float gv[CPL][8];
#pragma unroll
  for (int q = 0; q < CPL; ++q)
    if (lane + 32 * q < chunks) unpack8(__ldg(g + lane + 32 * q), gv[q]);
  const long long stride = (long long)gridDim.x * kNormWarps * kNormRows;
  for (long long m0 = ((long long)blockIdx.x * kNormWarps + (threadIdx.x >> 5)) * kNormRows; m0 < M; m0 += stride) {
    uint4 raw[kNormRows][CPL];
#pragma unroll
    for (int r = 0; r < kNormRows; ++r)
#pragma unroll
      for (int q = 0; q < CPL; ++q)
        raw[r][q] = (m0 + r < M && lane + 32 * q < chunks) ? ldg_nc_v4(x + (m0 + r) * chunks + lane + 32 * q)
                                                            : make_uint4(0, 0, 0, 0);
#pragma unroll
    for (int r = 0; r < kNormRows; ++r) {
      float v[CPL][8], ss = 0.f;
#pragma unroll
      for (int q = 0; q < CPL; ++q) {
        unpack8(raw[r][q], v[q]);
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          v[q][k] *= alpha;
          ss = fmaf(v[q][k], v[q][k], ss);
        }
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
      const float rs = rsqrtf(ss / (float)e + eps);
      if (m0 + r < M) {
        if (lane == 0) rstd[m0 + r] = rs;
#pragma unroll
        for (int q = 0; q < CPL; ++q)
          if (lane + 32 * q < chunks) {
            float o[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) o[k] = v[q][k] * rs * gv[q][k];
            stg_v4(h + (m0 + r) * chunks + lane + 32 * q, pack8(o));
          }
      }
    }
  }
}

// Backward of  xs = alpha x,  h = xs rstd o g,  out = xs + f(h):  given dh and dy (the gradient of `out`),
//   t = dh o g,  xh = xs rstd,  dxs = dy + rstd (t - xh mean(t o xh)),  dx = alpha dxs,  dg += dh o xh.
// dg: per-warp register sums over the warp's rows, then one partial row per CTA (reduced by colsum_kernel).
template <int CPL>
__global__ void __launch_bounds__(kNormWarps * 32)
rmsnorm_bwd_kernel(const uint4* __restrict__ x, const uint4* __restrict__ g, const float* __restrict__ rstd,
                   const uint4* __restrict__ dh, const uint4* __restrict__ dy, uint4* __restrict__ dx,
                   float* __restrict__ dg_partial, long long M, int e, float alpha) {
  __shared__ float sdg[kNormWarps][CPL * 256];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, chunks = e >> 3;
  constexpr int RB = 2;   // rows in flight (three streams each)
  float gv[CPL][8], acc[CPL][8];
#pragma unroll
  for (int q = 0; q < CPL; ++q) {
#pragma unroll
    for (int k = 0; k < 8; ++k) acc[q][k] = gv[q][k] = 0.f;   // (lanes beyond the row contribute exact zeros)
    if (lane + 32 * q < chunks) unpack8(__ldg(g + lane + 32 * q), gv[q]);
  }
  const long long stride = (long long)gridDim.x * kNormWarps * RB;
  for (long long m0 = ((long long)blockIdx.x * kNormWarps + warp) * RB; m0 < M; m0 += stride) {
    uint4 rx[RB][CPL], rh[RB][CPL], ry[RB][CPL];
    float rr[RB];
#pragma unroll
    for (int r = 0; r < RB; ++r) {
      const bool ok = m0 + r < M;
      rr[r] = ok ? __ldg(rstd + m0 + r) : 0.f;
#pragma unroll
      for (int q = 0; q < CPL; ++q) {
        const bool in = ok && lane + 32 * q < chunks;
        const long long i = (m0 + r) * chunks + lane + 32 * q;
        rx[r][q] = in ? ldg_nc_v4(x + i) : make_uint4(0, 0, 0, 0);
        rh[r][q] = in ? ldg_nc_v4(dh + i) : make_uint4(0, 0, 0, 0);
        ry[r][q] = in ? ldg_nc_v4(dy + i) : make_uint4(0, 0, 0, 0);
      }
    }
#pragma unroll
    for (int r = 0; r < RB; ++r) {
      float xh[CPL][8], t[CPL][8], c = 0.f;
#pragma unroll
      for (int q = 0; q < CPL; ++q) {
        float d[8];
        unpack8(rx[r][q], xh[q]);
        unpack8(rh[r][q], d);
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          xh[q][k] *= alpha * rr[r];
          acc[q][k] = fmaf(d[k], xh[q][k], acc[q][k]);
          t[q][k] = d[k] * gv[q][k];
          c = fmaf(t[q][k], xh[q][k], c);
        }
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
      c /= (float)e;
      if (m0 + r < M) {
#pragma unroll
        for (int q = 0; q < CPL; ++q)
          if (lane + 32 * q < chunks) {
            float d[8], o[8];
            unpack8(ry[r][q], d);
#pragma unroll
            for (int k = 0; k < 8; ++k) o[k] = alpha * (d[k] + rr[r] * (t[q][k] - xh[q][k] * c));
            stg_v4(dx + (m0 + r) * chunks + lane + 32 * q, pack8(o));
          }
      }
    }
  }
#pragma unroll
  for (int q = 0; q < CPL; ++q)
    if (lane + 32 * q < chunks) {
#pragma unroll
      for (int k = 0; k < 8; ++k) sdg[warp][8 * (lane + 32 * q) + k] = acc[q][k];
    }
  __syncthreads();
  for (int j = threadIdx.x; j < e; j += blockDim.x) {
    float s = 0.f;
#pragma unroll
    for (int w = 0; w < kNormWarps; ++w) s += sdg[w][j];
    dg_partial[(size_t)blockIdx.x * e + j] = s;
  }
}

// out[j] = sum_i partial[i][j]   (fixed order: deterministic).  32 columns per CTA, 16 row lanes per column (row i goes
// to lane i % 16, four loads in flight), then a fixed-order sum of the 16 lanes: a single thread per column walking all
// ~1,200 rows was 70 us of dependent loads.
constexpr int kColsumLanes = 16;
__global__ void __launch_bounds__(32 * kColsumLanes) colsum_kernel(const float* __restrict__ partial, int rows, int e,
                                                                    float* __restrict__ out) {
  __shared__ float red[kColsumLanes][33];
  const int jx = threadIdx.x & 31, ly = threadIdx.x >> 5, j = blockIdx.x * 32 + jx;
  float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
  if (j < e) {
    int i = ly;
    for (; i + 3 * kColsumLanes < rows; i += 4 * kColsumLanes) {
      s0 += partial[(size_t)i * e + j];
      s1 += partial[(size_t)(i + kColsumLanes) * e + j];
      s2 += partial[(size_t)(i + 2 * kColsumLanes) * e + j];
      s3 += partial[(size_t)(i + 3 * kColsumLanes) * e + j];
    }
    for (; i < rows; i += kColsumLanes) s0 += partial[(size_t)i * e + j];
  }
  red[ly][jx] = (s0 + s1) + (s2 + s3);
  __syncthreads();
  if (ly == 0 && j < e) {
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < kColsumLanes; ++k) s += red[k][jx];
    out[j] = s;
  }
}

// X0 = G / (||G||_F + eps) per matrix (bf16 in, bf16 out, fp32 sum); one CTA per matrix
__global__ void __launch_bounds__(256) frob_normalize_kernel(const uint16_t* __restrict__ G, uint16_t* __restrict__ X,
                                                             long long elems, float eps) {
  __shared__ float red[8];
  __shared__ float inv_s;
  const uint16_t* g = G + (size_t)blockIdx.x * elems;
  uint16_t* xo = X + (size_t)blockIdx.x * elems;
  float ss = 0.f;
  for (long long i = threadIdx.x; i < elems; i += blockDim.x) {
    const float v = __uint_as_float((uint32_t)g[i] << 16);
    ss = fmaf(v, v, ss);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = ss;
  __syncthreads();
  if (threadIdx.x == 0) {
    float s = 0.f;
    for (int w = 0; w < 8; ++w) s += red[w];
    inv_s = 1.f / (sqrtf(s) + eps);
  }
  __syncthreads();
  const float inv = inv_s;
  for (long long i = threadIdx.x; i < elems; i += blockDim.x) {
    const float v = __uint_as_float((uint32_t)g[i] << 16) * inv;
    xo[i] = (uint16_t)(pack_bf16(v, 0.f) & 0xffffu);
  }
}

int norm_grid(long long M, int num_sms) {
  const long long want = (M + kNormWarps - 1) / kNormWarps;
  const long long cap = (long long)num_sms * 8;
  return (int)(want < cap ? want : cap);
}

void launch_rmsnorm_fwd(const void* x, const void* g, void* h, float* rstd, long long M, int e, float alpha, float eps,
                        int num_sms, cudaStream_t stream) {
  const int grid = norm_grid(M, num_sms), cpl = (e / 8 + 31) / 32;
  auto args = [&](auto kern) {
    kern<<<grid, kNormWarps * 32, 0, stream>>>((const uint4*)x, (const uint4*)g, (uint4*)h, rstd, M, e, alpha, eps);
  };
  if (cpl <= 1) args(rmsnorm_fwd_kernel<1>);
  else if (cpl == 2) args(rmsnorm_fwd_kernel<2>);
  else args(rmsnorm_fwd_kernel<4>);
  count_launch();
}

// returns the number of partial rows written to dg_partial
int launch_rmsnorm_bwd(const void* x, const void* g, const float* rstd, const void* dh, const void* dy, void* dx,
                       float* dg_partial, long long M, int e, float alpha, int num_sms, cudaStream_t stream) {
  const int grid = norm_grid(M, num_sms), cpl = (e / 8 + 31) / 32;
  auto args = [&](auto kern) {
    kern<<<grid, kNormWarps * 32, 0, stream>>>((const uint4*)x, (const uint4*)g, rstd, (const uint4*)dh,
                                                (const uint4*)dy, (uint4*)dx, dg_partial, M, e, alpha);
  };
  if (cpl <= 1) args(rmsnorm_bwd_kernel<1>);
  else if (cpl == 2) args(rmsnorm_bwd_kernel<2>);
  else args(rmsnorm_bwd_kernel<4>);
  count_launch();
  return grid;
}

gemm::Problem linear_problem(long long M, int N, int K) {
  gemm::Problem p{};
  p.M = (int)M; p.N = N; p.K = K; p.batch = 1;
  p.alpha = 1.f; p.beta = 0.f;
  p.slabs = 1;
  return p;
}

// Y[M][N] = A[M][K] W[N][K]^T  (nn.Linear)
gemm::Problem nt(const void* A, long long M, int K, const void* W, int N, void* Y) {
  gemm::Problem p = linear_problem(M, N, K);
  p.A = {A, 0, K, 0};
  p.B = {W, 0, K, 0};
  p.C[0] = Y; p.ldc = N;
  return p;
}
// dA[M][K] = dY[M][N] W[N][K]        (W read as the MN-major B operand)
gemm::Problem nn(const void* dY, long long M, int N, const void* W, int K, void* dA) {
  gemm::Problem p = linear_problem(M, K, N);
  p.A = {dY, 0, N, 0};
  p.B = {W, 1, K, 0};
  p.C[0] = dA; p.ldc = K;
  return p;
}

// dW[N][K] (fp32) = dY[M][N]^T A[M][K], reduced over the M cells in split-K slabs (partials in ws_f32)
// (dY2, dY3 != nullptr: dY is three tensors of N / 3 columns each, stacked along N -- the rows of dW)
cudaError_t weight_grad(const void* dY, long long ldy, const void* A, long long lda, long long M, int N, int K,
                        float* dW, float* ws_f32, size_t ws_floats, const DeviceInfo* di, cudaStream_t stream,
                        const void* dY2 = nullptr, const void* dY3 = nullptr) {
  gemm::Problem p{};
  p.M = N; p.N = K; p.K = (int)M; p.batch = 1;
  p.A = {dY, 1, ldy, 0};
  if (dY2) { p.A2 = dY2; p.A3 = dY3; p.a_split_m = N / 3; }
  p.B = {A, 1, lda, 0};
  p.alpha = 1.f;
  // (256 x 256 tiles when K allows it, else 128 x 128 / 64 -- gemm::launch)
  const int tiles = K % 256 == 0 ? ((N + 255) / 256) * (K / 256) : ((N + 127) / 128) * ((K + 63) / 64);
  if (K % 256 == 0) {
    // one 256 x 256 CTA per SM (192 KB of ring): as many slabs as give one wave
    const long long kb_total = (M + 63) / 64;
    long long want = std::max(1, std::min(128, di->num_sms / tiles));
    if (want > kb_total) want = kb_total;
    const long long per = (kb_total + want - 1) / want;
    p.slabs = (int)((kb_total + per - 1) / per);
  } else {
    p.slabs = gemm::slabs_for(M, tiles, di->num_sms);
  }
  if ((size_t)p.slabs * N * K > ws_floats) return cudaErrorInvalidValue;
  p.partial = ws_f32;
  cudaError_t e = gemm::launch(p, stream);
  if (e != cudaSuccess) return e;
  return gemm::launch_reduce_slabs(ws_f32, p.slabs, (long long)N * K, 1.f, dW, true, stream);
}

}  // namespace

// ---- workspace sizes (bytes) ---------------------------------------------------------------------------------
size_t block_ws_bytes(long long cells, int e, int hidden_or_zero, int num_sms) {
  // bf16 scratch [cells][max(e, hidden)] x 2 + fp32 split-K partials of the largest weight gradient + dg partials
  const size_t wide = (size_t)(hidden_or_zero > e ? hidden_or_zero : e);
  const size_t act = (size_t)cells * wide * 2 * 2;
  const size_t big = (size_t)(hidden_or_zero > 0 ? (size_t)hidden_or_zero * e : (size_t)e * e);
  const size_t partial = (size_t)130 * big * sizeof(float);
  const size_t dg = (size_t)num_sms * 8 * e * sizeof(float);
  return act + partial + dg + 1024;
}

// ---- MLP sub-block --------------------------------------------------------------------------------------------
cudaError_t launch_mlp_fwd(long long cells, int e, int hidden, float alpha, float eps, const void* x, const void* g,
                           const void* W1, const void* W2, void* y, void* h, float* rstd, void* u, void* a,
                           cudaStream_t stream) {
  const DeviceInfo* di = current_device();
  if (!di) return cudaErrorInvalidDevice;
  launch_rmsnorm_fwd(x, g, h, rstd, cells, e, alpha, eps, di->num_sms, stream);
  // u = h W1^T (saved), a = gelu(u) (saved): one GEMM, two outputs
  gemm::Problem p1 = nt(h, cells, e, W1, hidden, u);
  p1.C[1] = a;
  p1.dual_out = 1;
  p1.act = gemm::ACT_GELU;
  cudaError_t er = gemm::launch(p1, stream);
  if (er != cudaSuccess) return er;
  // y = alpha x + a W2^T
  gemm::Problem p2 = nt(a, cells, hidden, W2, e, y);
  p2.aux_mode = gemm::AUX_ADD;
  p2.aux = x; p2.ld_aux = e; p2.beta = alpha;
  return gemm::launch(p2, stream);
}

cudaError_t launch_mlp_bwd(long long cells, int e, int hidden, float alpha, const void* x, const void* g,
                           const void* W1, const void* W2, const void* h, const float* rstd, const void* u,
                           const void* a, const void* dy, void* dx, float* dg, float* dW1, float* dW2, void* ws,
                           size_t ws_bytes, cudaStream_t stream) {
  const DeviceInfo* di = current_device();
  if (!di) return cudaErrorInvalidDevice;
  if (ws_bytes < block_ws_bytes(cells, e, hidden, di->num_sms)) return cudaErrorInvalidValue;
  char* w = static_cast<char*>(ws);
  void* du = w;                                               // [cells][hidden] bf16
  void* dh = w + (size_t)cells * hidden * 2;                  // [cells][e] bf16 (inside the second wide slot)
  float* partial = reinterpret_cast<float*>(w + (size_t)cells * hidden * 2 * 2);
  const size_t partial_floats = (size_t)130 * hidden * e;
  float* dg_partial = partial + partial_floats;
  // du = (dy W2) o gelu'(u)
  gemm::Problem p = nn(dy, cells, e, W2, hidden, du);
  p.aux_mode = gemm::AUX_GELU_GRAD;
  p.aux = u; p.ld_aux = hidden;
  cudaError_t er = gemm::launch(p, stream);
  if (er != cudaSuccess) return er;
  // dW2[e][hidden] = dy^T a ; dW1[hidden][e] = du^T h
  if ((er = weight_grad(dy, e, a, hidden, cells, e, hidden, dW2, partial, partial_floats, di, stream)) != cudaSuccess) return er;
  if ((er = weight_grad(du, hidden, h, e, cells, hidden, e, dW1, partial, partial_floats, di, stream)) != cudaSuccess) return er;
  // dh = du W1
  gemm::Problem q = nn(du, cells, hidden, W1, e, dh);
  if ((er = gemm::launch(q, stream)) != cudaSuccess) return er;
  const int grid = launch_rmsnorm_bwd(x, g, rstd, dh, dy, dx, dg_partial, cells, e, alpha, di->num_sms, stream);
  colsum_kernel<<<(e + 31) / 32, 32 * kColsumLanes, 0, stream>>>(dg_partial, grid, e, dg);
  count_launch();
  return cudaGetLastError();
}

// ---- attention sub-block ---------------------------------------------------------------------------------------
cudaError_t launch_attn_block_fwd(const Shape& s, int axis, float alpha, float eps, const void* x, const void* g,
                                  const void* Wqkv, const void* Wo, void* y, void* h, float* rstd, void* q, void* k,
                                  void* v, void* o, float* lse, void* ws, cudaStream_t stream) {
  const DeviceInfo* di = current_device();
  if (!di) return cudaErrorInvalidDevice;
  const long long cells = (long long)s.B * s.R * s.C;
  const int e = s.H * s.dh;
  launch_rmsnorm_fwd(x, g, h, rstd, cells, e, alpha, eps, di->num_sms, stream);
  // [q | k | v] = h Wqkv^T, written as three [cells][e] tensors (the attention kernels' layout)
  gemm::Problem p = nt(h, cells, e, Wqkv, 3 * e, q);
  p.C[1] = k; p.C[2] = v;
  p.split_cols = e; p.ldc = e;
  cudaError_t er = gemm::launch(p, stream);
  if (er != cudaSuccess) return er;
  er = axis == 0 ? launch_feature_fwd(s, q, k, v, o, lse, ws, stream)
                 : launch_item_fwd(s, q, k, v, o, lse, 0, s.R, ws, stream);
  if (er != cudaSuccess) return er;
  // y = alpha x + o Wo^T
  gemm::Problem p2 = nt(o, cells, e, Wo, e, y);
  p2.aux_mode = gemm::AUX_ADD;
  p2.aux = x; p2.ld_aux = e; p2.beta = alpha;
  return gemm::launch(p2, stream);
}

size_t attn_block_bwd_ws_bytes(const Shape& s, int axis, int num_sms) {
  const long long cells = (long long)s.B * s.R * s.C;
  const int e = s.H * s.dh;
  // do, dq, dk, dv, dh: five [cells][e] bf16 + the attention backward's own workspace + partials
  size_t n = (size_t)cells * e * 2 * 5;
  n += axis == 0 ? feature_workspace_bytes(s) : item_bwd_workspace_bytes(s);
  n = (n + 255) & ~(size_t)255;
  n += (size_t)130 * 3 * e * e * sizeof(float) + (size_t)num_sms * 8 * e * sizeof(float) + 1024;   // (dWqkv partials)
  return n;
}

cudaError_t launch_attn_block_bwd(const Shape& s, int axis, float alpha, const void* x, const void* g,
                                  const void* Wqkv, const void* Wo, const void* h, const float* rstd, const void* q,
                                  const void* k, const void* v, const void* o, const float* lse, const void* dy,
                                  void* dx, float* dg, float* dWqkv, float* dWo, void* ws, size_t ws_bytes,
                                  cudaStream_t stream) {
  const DeviceInfo* di = current_device();
  if (!di) return cudaErrorInvalidDevice;
  if (ws_bytes < attn_block_bwd_ws_bytes(s, axis, di->num_sms)) return cudaErrorInvalidValue;
  const long long cells = (long long)s.B * s.R * s.C;
  const int e = s.H * s.dh;
  const size_t T = (size_t)cells * e * 2;
  char* w = static_cast<char*>(ws);
  void *d_o = w, *dq = w + T, *dk = w + 2 * T, *dv = w + 3 * T, *dh = w + 4 * T;
  size_t off = 5 * T;
  void* attn_ws = w + off;
  off += axis == 0 ? feature_workspace_bytes(s) : item_bwd_workspace_bytes(s);
  off = (off + 255) & ~(size_t)255;
  float* partial = reinterpret_cast<float*>(w + off);
  const size_t partial_floats = (size_t)130 * 3 * e * e;
  float* dg_partial = partial + partial_floats;
  // do = dy Wo ; dWo[e][e] = dy^T o
  gemm::Problem p = nn(dy, cells, e, Wo, e, d_o);
  cudaError_t er = gemm::launch(p, stream);
  if (er != cudaSuccess) return er;
  if ((er = weight_grad(dy, e, o, e, cells, e, e, dWo, partial, partial_floats, di, stream)) != cudaSuccess) return er;
  // attention backward
  er = axis == 0 ? launch_feature_bwd(s, q, k, v, o, d_o, lse, dq, dk, dv, attn_ws, stream)
                 : launch_item_bwd(s, q, k, v, o, d_o, lse, dq, dk, dv, static_cast<float*>(attn_ws), stream);
  if (er != cudaSuccess) return er;
  // dWqkv[3e][e]: three [e][e] blocks  d{q,k,v}^T h
  if (e % 128 == 0) {   // one launch over the three gradients: h is read once
    if ((er = weight_grad(dq, e, h, e, cells, 3 * e, e, dWqkv, partial, partial_floats, di, stream, dk, dv)) != cudaSuccess)
      return er;
  } else {
    const void* grads[3] = {dq, dk, dv};
    for (int t = 0; t < 3; ++t)
      if ((er = weight_grad(grads[t], e, h, e, cells, e, e, dWqkv + (size_t)t * e * e, partial, partial_floats, di,
                            stream)) != cudaSuccess)
        return er;
  }
  // dh = [dq | dk | dv] Wqkv   (A split over the three tensors along K)
  gemm::Problem r = linear_problem(cells, e, 3 * e);
  r.A = {dq, 0, e, 0};
  r.A2 = dk; r.A3 = dv; r.a_split_k = e;
  r.B = {Wqkv, 1, e, 0};
  r.C[0] = dh; r.ldc = e;
  if ((er = gemm::launch(r, stream)) != cudaSuccess) return er;
  const int grid = launch_rmsnorm_bwd(x, g, rstd, dh, dy, dx, dg_partial, cells, e, alpha, di->num_sms, stream);
  colsum_kernel<<<(e + 31) / 32, 32 * kColsumLanes, 0, stream>>>(dg_partial, grid, e, dg);
  count_launch();
  return cudaGetLastError();
}

// ---- batched Newton-Schulz (Muon) -------------------------------------------------------------------------------
size_t newton_schulz_ws_bytes(int nb, int m, int n) {
  return ((size_t)nb * m * n + 2 * (size_t)nb * m * m) * 2 + 1024;
}

cudaError_t launch_newton_schulz(int nb, int m, int n, const void* G, void* X, int steps, float ca, float cb, float cc,
                                 float eps, void* ws, cudaStream_t stream) {
  char* w = static_cast<char*>(ws);
  void* Xt = w;                                        // ping-pong partner of X
  void* A = w + (size_t)nb * m * n * 2;                // [nb][m][m]
  void* Bm = w + (size_t)nb * m * n * 2 + (size_t)nb * m * m * 2;
  // the iterate ends in X after `steps` swaps: start in X if steps is even, else in Xt
  void* cur = (steps & 1) ? Xt : X;
  void* nxt = (steps & 1) ? X : Xt;
  frob_normalize_kernel<<<nb, 256, 0, stream>>>((const uint16_t*)G, (uint16_t*)cur, (long long)m * n, eps);
  count_launch();
  for (int it = 0; it < steps; ++it) {
    // A = X X^T
    gemm::Problem p{};
    p.M = m; p.N = m; p.K = n; p.batch = nb;
    p.A = {cur, 0, n, (long long)m * n};
    p.B = {cur, 0, n, (long long)m * n};
    p.C[0] = A; p.ldc = m; p.c_batch_stride = (long long)m * m;
    p.alpha = 1.f; p.slabs = 1;
    cudaError_t er = gemm::launch(p, stream);
    if (er != cudaSuccess) return er;
    // B = b A + c A A      (A is symmetric: A A = A A^T, both operands K-major)
    gemm::Problem q{};
    q.M = m; q.N = m; q.K = m; q.batch = nb;
    q.A = {A, 0, m, (long long)m * m};
    q.B = {A, 0, m, (long long)m * m};
    q.C[0] = Bm; q.ldc = m; q.c_batch_stride = (long long)m * m;
    q.alpha = cc; q.beta = cb; q.slabs = 1;
    q.aux_mode = gemm::AUX_ADD; q.aux = A; q.ld_aux = m; q.aux_batch_stride = (long long)m * m;
    if ((er = gemm::launch(q, stream)) != cudaSuccess) return er;
    // X' = a X + B X       (X read as the MN-major B operand)
    gemm::Problem r{};
    r.M = m; r.N = n; r.K = m; r.batch = nb;
    r.A = {Bm, 0, m, (long long)m * m};
    r.B = {cur, 1, n, (long long)m * n};
    r.C[0] = nxt; r.ldc = n; r.c_batch_stride = (long long)m * n;
    r.alpha = 1.f; r.beta = ca; r.slabs = 1;
    r.aux_mode = gemm::AUX_ADD; r.aux = cur; r.ld_aux = n; r.aux_batch_stride = (long long)m * n;
    if ((er = gemm::launch(r, stream)) != cudaSuccess) return er;
    void* t = cur; cur = nxt; nxt = t;
  }
  return cudaSuccess;
}

}  // namespace tabattn
