// Item-axis ("sample-axis") attention, SIMT bring-up path.
//
// One CTA = 128 rows of one (table, column, head).  Key/query tiles of 64 rows are staged in
// shared memory as fp32 and every thread walks them with an fp32 online softmax (forward), or
// with P recomputed from LSE (backward: a dQ pass that also emits D, then a dK/dV pass).
// This is the correctness-first path the tcgen05 kernels are validated against on the GPU;
// it computes the same thing as item_tc*.cu and is selected only by TABATTN_ITEM_SIMT=1.
#include "common.cuh"
#include "kernels.h"

namespace tabattn {

namespace {

constexpr int kRowsPerCta = 128;
constexpr int kTile = 64;

__device__ __forceinline__ int clamp_n(const Shape& s, int b) { return max(1, min(s.n_train[b], s.R)); }

// Stage `rows` rows [row0, row0+rows) of one (b, c, h) into smem as fp32 [kTile][DH]; rows >= limit -> 0.
template <int DH>
__device__ __forceinline__ void stage_tile(float* dst, const __nv_bfloat16* src, size_t row_stride, int row0,
                                           int limit) {
  constexpr int VPR = DH / 8;  // 16-byte vectors per row
  for (int v = threadIdx.x; v < kTile * VPR; v += blockDim.x) {
    const int r = v / VPR, k = v % VPR;
    float f[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    if (row0 + r < limit) unpack8(ldg_nc_v4(src + (size_t)(row0 + r) * row_stride + 8 * k), f);
    float4* d4 = reinterpret_cast<float4*>(dst + r * DH + 8 * k);
    d4[0] = make_float4(f[0], f[1], f[2], f[3]);
    d4[1] = make_float4(f[4], f[5], f[6], f[7]);
  }
}

template <int DH>
__global__ void __launch_bounds__(kRowsPerCta) item_fwd_simt(Shape s, const __nv_bfloat16* __restrict__ Q,
                                                             const __nv_bfloat16* __restrict__ K,
                                                             const __nv_bfloat16* __restrict__ V,
                                                             __nv_bfloat16* __restrict__ O,
                                                             float* __restrict__ LSE) {
  __shared__ __align__(16) float sK[kTile * DH];
  __shared__ __align__(16) float sV[kTile * DH];
  const int bc = blockIdx.z, b = bc / s.C, c = bc % s.C, h = blockIdx.y;
  const int i = blockIdx.x * kRowsPerCta + threadIdx.x;
  const int d = s.H * DH;
  const size_t row_stride = (size_t)s.C * d;
  const size_t seq0 = ((size_t)b * s.R * s.C + c) * d + (size_t)h * DH;  // row 0 of this (b,c,h)
  const size_t lse_idx = (((size_t)b * s.C + c) * s.H + h) * s.R + i;
  const bool valid = !s.col_valid || s.col_valid[bc];
  if (!valid) {
    if (i < s.R) {
#pragma unroll
      for (int k = 0; k < DH / 8; ++k) stg_v4(O + seq0 + (size_t)i * row_stride + 8 * k, make_uint4(0, 0, 0, 0));
      LSE[lse_idx] = 0.f;
    }
    return;
  }
  const int n = clamp_n(s, b);
  float q[DH], acc[DH];
#pragma unroll
  for (int k = 0; k < DH; ++k) { q[k] = 0.f; acc[k] = 0.f; }
  if (i < s.R) {
#pragma unroll
    for (int k = 0; k < DH / 8; ++k) unpack8(ldg_nc_v4(Q + seq0 + (size_t)i * row_stride + 8 * k), q + 8 * k);
  }
  const float qscale = s.scale * kLog2e;
#pragma unroll
  for (int k = 0; k < DH; ++k) q[k] *= qscale;
  float m = -INFINITY, l = 0.f;
  for (int j0 = 0; j0 < n; j0 += kTile) {
    __syncthreads();
    stage_tile<DH>(sK, K + seq0, row_stride, j0, n);
    stage_tile<DH>(sV, V + seq0, row_stride, j0, n);
    __syncthreads();
    const int jn = min(kTile, n - j0);
    for (int j = 0; j < jn; ++j) {
      float sc = 0.f;
#pragma unroll
      for (int k = 0; k < DH; ++k) sc = fmaf(q[k], sK[j * DH + k], sc);
      if (sc > m) {
        const float alpha = fast_exp2(m - sc);
        l *= alpha;
#pragma unroll
        for (int k = 0; k < DH; ++k) acc[k] *= alpha;
        m = sc;
      }
      const float p = fast_exp2(sc - m);
      l += p;
#pragma unroll
      for (int k = 0; k < DH; ++k) acc[k] = fmaf(p, sV[j * DH + k], acc[k]);
    }
  }
  if (i < s.R) {
    const float inv = 1.f / l;
#pragma unroll
    for (int k = 0; k < DH / 8; ++k) {
      float o[8];
#pragma unroll
      for (int e = 0; e < 8; ++e) o[e] = acc[8 * k + e] * inv;
      stg_v4(O + seq0 + (size_t)i * row_stride + 8 * k, pack8(o));
    }
    LSE[lse_idx] = (m + log2f(l)) * kLn2;
  }
}

// dQ pass: one thread per query row; also writes D_i = rowsum(dO_i o O_i) to the workspace.
template <int DH>
__global__ void __launch_bounds__(kRowsPerCta) item_bwd_dq_simt(
    Shape s, const __nv_bfloat16* __restrict__ Q, const __nv_bfloat16* __restrict__ K,
    const __nv_bfloat16* __restrict__ V, const __nv_bfloat16* __restrict__ O, const __nv_bfloat16* __restrict__ dO,
    const float* __restrict__ LSE, __nv_bfloat16* __restrict__ dQ, float* __restrict__ Dws) {
  __shared__ __align__(16) float sK[kTile * DH];
  __shared__ __align__(16) float sV[kTile * DH];
  const int bc = blockIdx.z, b = bc / s.C, c = bc % s.C, h = blockIdx.y;
  const int i = blockIdx.x * kRowsPerCta + threadIdx.x;
  const int d = s.H * DH;
  const size_t row_stride = (size_t)s.C * d;
  const size_t seq0 = ((size_t)b * s.R * s.C + c) * d + (size_t)h * DH;
  const size_t lse_idx = (((size_t)b * s.C + c) * s.H + h) * s.R + i;
  const bool valid = !s.col_valid || s.col_valid[bc];
  if (!valid) {
    if (i < s.R) {
#pragma unroll
      for (int k = 0; k < DH / 8; ++k) stg_v4(dQ + seq0 + (size_t)i * row_stride + 8 * k, make_uint4(0, 0, 0, 0));
      Dws[lse_idx] = 0.f;
    }
    return;
  }
  const int n = clamp_n(s, b);
  float q[DH], g[DH], acc[DH];
  float D = 0.f, lse2 = 0.f;
#pragma unroll
  for (int k = 0; k < DH; ++k) { q[k] = 0.f; g[k] = 0.f; acc[k] = 0.f; }
  if (i < s.R) {
    const size_t cell = seq0 + (size_t)i * row_stride;
#pragma unroll
    for (int k = 0; k < DH / 8; ++k) {
      float o[8];
      unpack8(ldg_nc_v4(Q + cell + 8 * k), q + 8 * k);
      unpack8(ldg_nc_v4(dO + cell + 8 * k), g + 8 * k);
      unpack8(ldg_nc_v4(O + cell + 8 * k), o);
#pragma unroll
      for (int e = 0; e < 8; ++e) D = fmaf(o[e], g[8 * k + e], D);
    }
    lse2 = LSE[lse_idx] * kLog2e;
    Dws[lse_idx] = D;
  }
  const float qscale = s.scale * kLog2e;
#pragma unroll
  for (int k = 0; k < DH; ++k) q[k] *= qscale;
  for (int j0 = 0; j0 < n; j0 += kTile) {
    __syncthreads();
    stage_tile<DH>(sK, K + seq0, row_stride, j0, n);
    stage_tile<DH>(sV, V + seq0, row_stride, j0, n);
    __syncthreads();
    const int jn = min(kTile, n - j0);
    for (int j = 0; j < jn; ++j) {
      float sc = 0.f, dp = 0.f;
#pragma unroll
      for (int k = 0; k < DH; ++k) {
        sc = fmaf(q[k], sK[j * DH + k], sc);
        dp = fmaf(g[k], sV[j * DH + k], dp);
      }
      const float ds = fast_exp2(sc - lse2) * (dp - D);
#pragma unroll
      for (int k = 0; k < DH; ++k) acc[k] = fmaf(ds, sK[j * DH + k], acc[k]);
    }
  }
  if (i < s.R) {
#pragma unroll
    for (int k = 0; k < DH / 8; ++k) {
      float o[8];
#pragma unroll
      for (int e = 0; e < 8; ++e) o[e] = acc[8 * k + e] * s.scale;
      stg_v4(dQ + seq0 + (size_t)i * row_stride + 8 * k, pack8(o));
    }
  }
}

// dK/dV pass: one thread per key row j; loops over all R query rows.  Rows j >= n_train: zeros.
template <int DH>
__global__ void __launch_bounds__(kRowsPerCta) item_bwd_dkdv_simt(
    Shape s, const __nv_bfloat16* __restrict__ Q, const __nv_bfloat16* __restrict__ K,
    const __nv_bfloat16* __restrict__ V, const __nv_bfloat16* __restrict__ dO, const float* __restrict__ LSE,
    const float* __restrict__ Dws, __nv_bfloat16* __restrict__ dK, __nv_bfloat16* __restrict__ dV) {
  __shared__ __align__(16) float sQ[kTile * DH];
  __shared__ __align__(16) float sG[kTile * DH];
  __shared__ float sL[kTile], sD[kTile];
  const int bc = blockIdx.z, b = bc / s.C, c = bc % s.C, h = blockIdx.y;
  const int j = blockIdx.x * kRowsPerCta + threadIdx.x;
  const int d = s.H * DH;
  const size_t row_stride = (size_t)s.C * d;
  const size_t seq0 = ((size_t)b * s.R * s.C + c) * d + (size_t)h * DH;
  const size_t lse0 = (((size_t)b * s.C + c) * s.H + h) * s.R;
  const bool valid = !s.col_valid || s.col_valid[bc];
  const int n = valid ? clamp_n(s, b) : 0;
  if (blockIdx.x * kRowsPerCta >= n) {  // whole CTA beyond the train rows (or invalid column): zero-fill
    if (j < s.R) {
#pragma unroll
      for (int k = 0; k < DH / 8; ++k) {
        stg_v4(dK + seq0 + (size_t)j * row_stride + 8 * k, make_uint4(0, 0, 0, 0));
        stg_v4(dV + seq0 + (size_t)j * row_stride + 8 * k, make_uint4(0, 0, 0, 0));
      }
    }
    return;
  }
  float kk[DH], vv[DH], acck[DH], accv[DH];
#pragma unroll
  for (int k = 0; k < DH; ++k) { kk[k] = 0.f; vv[k] = 0.f; acck[k] = 0.f; accv[k] = 0.f; }
  if (j < n) {
#pragma unroll
    for (int k = 0; k < DH / 8; ++k) {
      unpack8(ldg_nc_v4(K + seq0 + (size_t)j * row_stride + 8 * k), kk + 8 * k);
      unpack8(ldg_nc_v4(V + seq0 + (size_t)j * row_stride + 8 * k), vv + 8 * k);
    }
  }
  const float qscale = s.scale * kLog2e;
#pragma unroll
  for (int k = 0; k < DH; ++k) kk[k] *= qscale;
  for (int i0 = 0; i0 < s.R; i0 += kTile) {
    __syncthreads();
    stage_tile<DH>(sQ, Q + seq0, row_stride, i0, s.R);
    stage_tile<DH>(sG, dO + seq0, row_stride, i0, s.R);
    if (threadIdx.x < kTile) {
      const int i = i0 + threadIdx.x;
      sL[threadIdx.x] = i < s.R ? LSE[lse0 + i] * kLog2e : INFINITY;
      sD[threadIdx.x] = i < s.R ? Dws[lse0 + i] : 0.f;
    }
    __syncthreads();
    const int in = min(kTile, s.R - i0);
    for (int i = 0; i < in; ++i) {
      float sc = 0.f, dp = 0.f;
#pragma unroll
      for (int k = 0; k < DH; ++k) {
        sc = fmaf(kk[k], sQ[i * DH + k], sc);
        dp = fmaf(vv[k], sG[i * DH + k], dp);
      }
      const float p = fast_exp2(sc - sL[i]);
      const float ds = p * (dp - sD[i]);
#pragma unroll
      for (int k = 0; k < DH; ++k) {
        accv[k] = fmaf(p, sG[i * DH + k], accv[k]);
        acck[k] = fmaf(ds, sQ[i * DH + k], acck[k]);
      }
    }
  }
  if (j < s.R) {
    const bool live = j < n;
#pragma unroll
    for (int k = 0; k < DH / 8; ++k) {
      float o[8];
#pragma unroll
      for (int e = 0; e < 8; ++e) o[e] = live ? acck[8 * k + e] * s.scale : 0.f;
      stg_v4(dK + seq0 + (size_t)j * row_stride + 8 * k, pack8(o));
#pragma unroll
      for (int e = 0; e < 8; ++e) o[e] = live ? accv[8 * k + e] : 0.f;
      stg_v4(dV + seq0 + (size_t)j * row_stride + 8 * k, pack8(o));
    }
  }
}

}  // namespace

#define TABATTN_DISPATCH_DH(dh, ...)                          \
  switch (dh) {                                               \
    case 16: { constexpr int DH = 16; __VA_ARGS__; } break;   \
    case 32: { constexpr int DH = 32; __VA_ARGS__; } break;   \
    case 64: { constexpr int DH = 64; __VA_ARGS__; } break;   \
    default: return cudaErrorInvalidValue;                    \
  }

cudaError_t launch_item_fwd_simt(const Shape& s, const void* Q, const void* K, const void* V, void* O, float* LSE,
                                 cudaStream_t stream) {
  dim3 grid((s.R + kRowsPerCta - 1) / kRowsPerCta, s.H, s.B * s.C);
  TABATTN_DISPATCH_DH(s.dh, {
    item_fwd_simt<DH><<<grid, kRowsPerCta, 0, stream>>>(s, (const __nv_bfloat16*)Q, (const __nv_bfloat16*)K,
                                                        (const __nv_bfloat16*)V, (__nv_bfloat16*)O, LSE);
  });
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_item_bwd_simt(const Shape& s, const void* Q, const void* K, const void* V, const void* O,
                                 const void* dO, const float* LSE, void* dQ, void* dK, void* dV, float* Dws,
                                 cudaStream_t stream) {
  dim3 grid((s.R + kRowsPerCta - 1) / kRowsPerCta, s.H, s.B * s.C);
  TABATTN_DISPATCH_DH(s.dh, {
    item_bwd_dq_simt<DH><<<grid, kRowsPerCta, 0, stream>>>(
        s, (const __nv_bfloat16*)Q, (const __nv_bfloat16*)K, (const __nv_bfloat16*)V, (const __nv_bfloat16*)O,
        (const __nv_bfloat16*)dO, LSE, (__nv_bfloat16*)dQ, Dws);
    item_bwd_dkdv_simt<DH><<<grid, kRowsPerCta, 0, stream>>>(
        s, (const __nv_bfloat16*)Q, (const __nv_bfloat16*)K, (const __nv_bfloat16*)V, (const __nv_bfloat16*)dO, LSE,
        Dws, (__nv_bfloat16*)dK, (__nv_bfloat16*)dV);
  });
  count_launch(2);
  return cudaGetLastError();
}

}  // namespace tabattn
