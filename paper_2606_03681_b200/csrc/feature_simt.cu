// Feature-axis attention, forward and backward.
//
// Packed many-sequences-per-CTA kernel for the short feature axis: one CTA owns a block of
// consecutive rows of one table (contiguous in HBM), stages the rows' K/V (and Q/dO for the
// backward) in shared memory with 128-bit coalesced loads, and gives every (row, head, column)
// triple to one thread, which walks the row's valid columns with an fp32 online softmax.
// The path is HBM-bound for short rows (intensity 0.58*C flop/B).
#include "common.cuh"
#include "kernels.h"

namespace tabattn {

namespace {

constexpr int kThreads = 256;

__device__ __forceinline__ void copy_block_to_smem(uint4* dst, const uint4* src, int nvec) {
  for (int i = threadIdx.x; i < nvec; i += blockDim.x) dst[i] = ldg_nc_v4(src + i);
}

// Build the list of valid columns of table b in shared memory; returns the count via *cv.
__device__ __forceinline__ void build_valid_cols(const Shape& s, int b, int* vcols, int* cv) {
  if (threadIdx.x == 0) {
    int n = 0;
    for (int c = 0; c < s.C; ++c)
      if (!s.col_valid || s.col_valid[(size_t)b * s.C + c]) vcols[n++] = c;
    *cv = n;
  }
}

template <int DH>
__global__ void __launch_bounds__(kThreads) feature_fwd_kernel(Shape s, const __nv_bfloat16* __restrict__ Q,
                                                               const __nv_bfloat16* __restrict__ K,
                                                               const __nv_bfloat16* __restrict__ V,
                                                               __nv_bfloat16* __restrict__ O,
                                                               float* __restrict__ LSE, int rows_per_cta) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int b = blockIdx.y;
  const int r0 = blockIdx.x * rows_per_cta;
  const int nrows = min(rows_per_cta, s.R - r0);
  const int C = s.C, H = s.H, d = H * DH;
  const size_t row_elems = (size_t)C * d;
  uint4* sK = reinterpret_cast<uint4*>(smem);
  uint4* sV = sK + (size_t)rows_per_cta * row_elems / 8;
  int* vcols = reinterpret_cast<int*>(sV + (size_t)rows_per_cta * row_elems / 8);
  int* cvp = vcols + C;

  const size_t base = ((size_t)b * s.R + r0) * row_elems;
  const int nvec = (int)(nrows * row_elems / 8);
  copy_block_to_smem(sK, reinterpret_cast<const uint4*>(K + base), nvec);
  copy_block_to_smem(sV, reinterpret_cast<const uint4*>(V + base), nvec);
  build_valid_cols(s, b, vcols, cvp);
  __syncthreads();
  const int Cv = *cvp;
  const float qscale = s.scale * kLog2e;

  const int items = nrows * H * C;
  for (int w = threadIdx.x; w < items; w += blockDim.x) {
    const int i = w % C;
    const int h = (w / C) % H;
    const int r = w / (C * H);
    const size_t cell = base + ((size_t)r * C + i) * d + (size_t)h * DH;
    const size_t lse_idx = (((size_t)b * s.R + r0 + r) * H + h) * C + i;
    const bool valid = !s.col_valid || s.col_valid[(size_t)b * C + i];
    if (!valid) {
#pragma unroll
      for (int k = 0; k < DH / 8; ++k) stg_v4(O + cell + 8 * k, make_uint4(0, 0, 0, 0));
      LSE[lse_idx] = 0.f;
      continue;
    }
    float q[DH];
#pragma unroll
    for (int k = 0; k < DH / 8; ++k) {
      uint4 u = ldg_nc_v4(Q + cell + 8 * k);
      unpack8(u, q + 8 * k);
    }
#pragma unroll
    for (int k = 0; k < DH; ++k) q[k] *= qscale;
    float m = -INFINITY, l = 0.f;
    float acc[DH];
#pragma unroll
    for (int k = 0; k < DH; ++k) acc[k] = 0.f;
    for (int jj = 0; jj < Cv; ++jj) {
      const int j = vcols[jj];
      const size_t off = (((size_t)r * C + j) * H + h) * (DH / 8);
      float sc = 0.f;
      float kv[8];
#pragma unroll
      for (int k = 0; k < DH / 8; ++k) {
        unpack8(sK[off + k], kv);
#pragma unroll
        for (int e = 0; e < 8; ++e) sc = fmaf(q[8 * k + e], kv[e], sc);
      }
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
      for (int k = 0; k < DH / 8; ++k) {
        unpack8(sV[off + k], kv);
#pragma unroll
        for (int e = 0; e < 8; ++e) acc[8 * k + e] = fmaf(p, kv[e], acc[8 * k + e]);
      }
    }
    const float inv = 1.f / l;
#pragma unroll
    for (int k = 0; k < DH / 8; ++k) {
      float o[8];
#pragma unroll
      for (int e = 0; e < 8; ++e) o[e] = acc[8 * k + e] * inv;
      stg_v4(O + cell + 8 * k, pack8(o));
    }
    LSE[lse_idx] = (m + log2f(l)) * kLn2;
  }
}

template <int DH>
__global__ void __launch_bounds__(kThreads) feature_bwd_kernel(
    Shape s, const __nv_bfloat16* __restrict__ Q, const __nv_bfloat16* __restrict__ K,
    const __nv_bfloat16* __restrict__ V, const __nv_bfloat16* __restrict__ O, const __nv_bfloat16* __restrict__ dO,
    const float* __restrict__ LSE, __nv_bfloat16* __restrict__ dQ, __nv_bfloat16* __restrict__ dK,
    __nv_bfloat16* __restrict__ dV, int rows_per_cta) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int b = blockIdx.y;
  const int r0 = blockIdx.x * rows_per_cta;
  const int nrows = min(rows_per_cta, s.R - r0);
  const int C = s.C, H = s.H, d = H * DH;
  const size_t row_elems = (size_t)C * d;
  const size_t blk_vec = (size_t)rows_per_cta * row_elems / 8;
  uint4* sQ = reinterpret_cast<uint4*>(smem);
  uint4* sK = sQ + blk_vec;
  uint4* sV = sK + blk_vec;
  uint4* sG = sV + blk_vec;
  float* sL = reinterpret_cast<float*>(sG + blk_vec);   // lse * log2e   [rows][H][C]
  float* sD = sL + (size_t)rows_per_cta * H * C;        // D = rowsum(dO o O)
  int* vcols = reinterpret_cast<int*>(sD + (size_t)rows_per_cta * H * C);
  int* cvp = vcols + C;

  const size_t base = ((size_t)b * s.R + r0) * row_elems;
  const int nvec = (int)(nrows * row_elems / 8);
  copy_block_to_smem(sQ, reinterpret_cast<const uint4*>(Q + base), nvec);
  copy_block_to_smem(sK, reinterpret_cast<const uint4*>(K + base), nvec);
  copy_block_to_smem(sV, reinterpret_cast<const uint4*>(V + base), nvec);
  copy_block_to_smem(sG, reinterpret_cast<const uint4*>(dO + base), nvec);
  build_valid_cols(s, b, vcols, cvp);
  const int items = nrows * H * C;
  // D_i = sum_k dO_i[k] * O_i[k]  (one (row, head, column) per thread; O read once from HBM)
  for (int w = threadIdx.x; w < items; w += blockDim.x) {
    const int i = w % C;
    const int h = (w / C) % H;
    const int r = w / (C * H);
    const size_t cell = base + ((size_t)r * C + i) * d + (size_t)h * DH;
    float D = 0.f;
#pragma unroll
    for (int k = 0; k < DH / 8; ++k) {
      float a[8], g[8];
      unpack8(ldg_nc_v4(O + cell + 8 * k), a);
      unpack8(ldg_nc_v4(dO + cell + 8 * k), g);
#pragma unroll
      for (int e = 0; e < 8; ++e) D = fmaf(a[e], g[e], D);
    }
    sD[w] = D;
    sL[w] = LSE[(((size_t)b * s.R + r0 + r) * H + h) * C + i] * kLog2e;
  }
  __syncthreads();
  const int Cv = *cvp;
  const float qscale = s.scale * kLog2e;

  for (int w = threadIdx.x; w < items; w += blockDim.x) {
    const int i = w % C;
    const int h = (w / C) % H;
    const int r = w / (C * H);
    const size_t cell = base + ((size_t)r * C + i) * d + (size_t)h * DH;
    const bool valid = !s.col_valid || s.col_valid[(size_t)b * C + i];
    if (!valid) {
#pragma unroll
      for (int k = 0; k < DH / 8; ++k) {
        stg_v4(dQ + cell + 8 * k, make_uint4(0, 0, 0, 0));
        stg_v4(dK + cell + 8 * k, make_uint4(0, 0, 0, 0));
        stg_v4(dV + cell + 8 * k, make_uint4(0, 0, 0, 0));
      }
      continue;
    }
    const size_t own = (((size_t)r * C + i) * H + h) * (DH / 8);
    const int rh = (r * H + h) * C;
    float a[DH], g[DH], acc[DH];
    float kv[8];
    // ---- as query i: dQ_i = scale * sum_j dS_ij K_j ------------------------------------------
    {
#pragma unroll
      for (int k = 0; k < DH / 8; ++k) {
        unpack8(sQ[own + k], a + 8 * k);
        unpack8(sG[own + k], g + 8 * k);
      }
#pragma unroll
      for (int k = 0; k < DH; ++k) { a[k] *= qscale; acc[k] = 0.f; }
      const float lse2 = sL[w], D = sD[w];
      for (int jj = 0; jj < Cv; ++jj) {
        const int j = vcols[jj];
        const size_t off = (((size_t)r * C + j) * H + h) * (DH / 8);
        float sc = 0.f, dp = 0.f;
#pragma unroll
        for (int k = 0; k < DH / 8; ++k) {
          unpack8(sK[off + k], kv);
#pragma unroll
          for (int e = 0; e < 8; ++e) sc = fmaf(a[8 * k + e], kv[e], sc);
          unpack8(sV[off + k], kv);
#pragma unroll
          for (int e = 0; e < 8; ++e) dp = fmaf(g[8 * k + e], kv[e], dp);
        }
        const float ds = fast_exp2(sc - lse2) * (dp - D);
#pragma unroll
        for (int k = 0; k < DH / 8; ++k) {
          unpack8(sK[off + k], kv);
#pragma unroll
          for (int e = 0; e < 8; ++e) acc[8 * k + e] = fmaf(ds, kv[e], acc[8 * k + e]);
        }
      }
#pragma unroll
      for (int k = 0; k < DH / 8; ++k) {
        float o[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) o[e] = acc[8 * k + e] * s.scale;
        stg_v4(dQ + cell + 8 * k, pack8(o));
      }
    }
    // ---- as key i: dV_i = sum_j P_ji dO_j ; dK_i = scale * sum_j dS_ji Q_j --------------------
    {
      float accv[DH];
#pragma unroll
      for (int k = 0; k < DH / 8; ++k) {
        unpack8(sK[own + k], a + 8 * k);
        unpack8(sV[own + k], g + 8 * k);
      }
#pragma unroll
      for (int k = 0; k < DH; ++k) { a[k] *= qscale; acc[k] = 0.f; accv[k] = 0.f; }
      for (int jj = 0; jj < Cv; ++jj) {
        const int j = vcols[jj];
        const size_t off = (((size_t)r * C + j) * H + h) * (DH / 8);
        float sc = 0.f, dp = 0.f;
#pragma unroll
        for (int k = 0; k < DH / 8; ++k) {
          unpack8(sQ[off + k], kv);
#pragma unroll
          for (int e = 0; e < 8; ++e) sc = fmaf(a[8 * k + e], kv[e], sc);
          unpack8(sG[off + k], kv);
#pragma unroll
          for (int e = 0; e < 8; ++e) dp = fmaf(g[8 * k + e], kv[e], dp);
        }
        const float p = fast_exp2(sc - sL[rh + j]);
        const float ds = p * (dp - sD[rh + j]);
#pragma unroll
        for (int k = 0; k < DH / 8; ++k) {
          unpack8(sG[off + k], kv);
#pragma unroll
          for (int e = 0; e < 8; ++e) accv[8 * k + e] = fmaf(p, kv[e], accv[8 * k + e]);
          unpack8(sQ[off + k], kv);
#pragma unroll
          for (int e = 0; e < 8; ++e) acc[8 * k + e] = fmaf(ds, kv[e], acc[8 * k + e]);
        }
      }
#pragma unroll
      for (int k = 0; k < DH / 8; ++k) {
        float o[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) o[e] = acc[8 * k + e] * s.scale;
        stg_v4(dK + cell + 8 * k, pack8(o));
        stg_v4(dV + cell + 8 * k, pack8(accv + 8 * k));
      }
    }
  }
}

size_t fwd_smem_bytes(const Shape& s, int rows) {
  return (size_t)2 * rows * s.C * s.H * s.dh * 2 + (size_t)(s.C + 4) * sizeof(int);
}
size_t bwd_smem_bytes(const Shape& s, int rows) {
  return (size_t)4 * rows * s.C * s.H * s.dh * 2 + (size_t)2 * rows * s.H * s.C * sizeof(float) +
         (size_t)(s.C + 4) * sizeof(int);
}

// rows per CTA: as many as fit the shared-memory budget, but keep >= 2 waves of CTAs over 148 SMs
template <typename F>
int pick_rows(const Shape& s, F bytes, size_t budget) {
  int rows = 1;
  while (rows < s.R && rows < 16 && bytes(s, rows + 1) <= budget) ++rows;
  while (rows > 1 && (long long)((s.R + rows - 1) / rows) * s.B < 2 * 148) --rows;
  return rows;
}

}  // namespace

#define TABATTN_DISPATCH_DH(dh, ...)                          \
  switch (dh) {                                               \
    case 16: { constexpr int DH = 16; __VA_ARGS__; } break;   \
    case 32: { constexpr int DH = 32; __VA_ARGS__; } break;   \
    case 64: { constexpr int DH = 64; __VA_ARGS__; } break;   \
    default: return cudaErrorInvalidValue;                    \
  }

bool feature_shape_supported(const Shape& s) {
  return s.C <= 128 && fwd_smem_bytes(s, 1) <= 227 * 1024 && bwd_smem_bytes(s, 1) <= 227 * 1024;
}

cudaError_t launch_feature_fwd(const Shape& s, const void* Q, const void* K, const void* V, void* O, float* LSE,
                               cudaStream_t stream) {
  const int rows = pick_rows(s, fwd_smem_bytes, 64 * 1024);
  const size_t smem = fwd_smem_bytes(s, rows);
  if (smem > 227 * 1024) return cudaErrorInvalidValue;
  dim3 grid((s.R + rows - 1) / rows, s.B);
  TABATTN_DISPATCH_DH(s.dh, {
    auto kern = feature_fwd_kernel<DH>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<grid, kThreads, smem, stream>>>(s, (const __nv_bfloat16*)Q, (const __nv_bfloat16*)K,
                                           (const __nv_bfloat16*)V, (__nv_bfloat16*)O, LSE, rows);
  });
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_feature_bwd(const Shape& s, const void* Q, const void* K, const void* V, const void* O,
                               const void* dO, const float* LSE, void* dQ, void* dK, void* dV,
                               cudaStream_t stream) {
  const int rows = pick_rows(s, bwd_smem_bytes, 100 * 1024);
  const size_t smem = bwd_smem_bytes(s, rows);
  if (smem > 227 * 1024) return cudaErrorInvalidValue;
  dim3 grid((s.R + rows - 1) / rows, s.B);
  TABATTN_DISPATCH_DH(s.dh, {
    auto kern = feature_bwd_kernel<DH>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<grid, kThreads, smem, stream>>>(s, (const __nv_bfloat16*)Q, (const __nv_bfloat16*)K,
                                           (const __nv_bfloat16*)V, (const __nv_bfloat16*)O,
                                           (const __nv_bfloat16*)dO, LSE, (__nv_bfloat16*)dQ, (__nv_bfloat16*)dK,
                                           (__nv_bfloat16*)dV, rows);
  });
  count_launch();
  return cudaGetLastError();
}

}  // namespace tabattn
