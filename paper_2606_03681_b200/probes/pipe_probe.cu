// Developer probe, not part of libtabattn.so: what the softmax arithmetic of the item kernels costs on one SM
// sub-partition.  Built and run by `python -m paper_2606_03681_b200.pipe_probe` (needs a B200); the table it printed
// is in profiles/r02_attention.md ("Issue cost of the softmax arithmetic").
//
// Part 1: clocks per warp instruction of independent MUFU.EX2 / FFMA / FFMA2 / FADD2 / FMNMX streams and of
//         two mixes, with 1, 2 and 4 warps per sub-partition (one CTA per SM, clock64 of CTA 0).
// Part 2: the forward kernel's row step (common.cuh: fma2, exp2_pair, add2, pack) on 128 scores per thread, read from
//         and written to shared memory in place of TMEM, with 1 and 2 warps per sub-partition.
#include <cstdint>
#include <cstdio>
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include "../csrc/common.cuh"

using namespace tabattn;

namespace {

enum { MUFU, FFMA, FFMA2, FADD2, FMNMX, MIX_FMA2_MNMX, MIX_SOFTMAX };

template <int WHAT>
__global__ void __launch_bounds__(512, 1) stream_kernel(float* out, long long* clk, int iters) {
  float a[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) a[i] = threadIdx.x * 1e-3f + i * 0.01f;
  const float f0 = 1.0001f, f1 = 0.5f;
  const uint64_t c = f2pack(f0, f1);
  uint64_t x[8];
  uint32_t d[4] = {0, 0, 0, 0};
#pragma unroll
  for (int i = 0; i < 8; ++i) x[i] = f2pack(a[2 * i], a[2 * i + 1]);
  __syncthreads();
  const long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 64; ++i) {
      if (WHAT == MUFU) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(a[i & 15]));
      if (WHAT == FFMA) asm volatile("fma.rn.ftz.f32 %0, %0, %1, %1;" : "+f"(a[i & 15]) : "f"(f0));
      if (WHAT == FFMA2) asm volatile("fma.rn.ftz.f32x2 %0, %0, %1, %1;" : "+l"(x[i & 7]) : "l"(c));
      if (WHAT == FADD2) asm volatile("add.rn.ftz.f32x2 %0, %0, %1;" : "+l"(x[i & 7]) : "l"(c));
      if (WHAT == FMNMX) asm volatile("max.ftz.f32 %0, %0, %1;" : "+f"(a[i & 15]) : "f"(f1));
      if (WHAT == MIX_FMA2_MNMX) {   // two pipes, 32 + 32: 64 clk if they issue side by side, 128 if not
        if (i & 1) asm volatile("max.ftz.f32 %0, %0, %1;" : "+f"(a[i & 15]) : "f"(f1));
        else asm volatile("fma.rn.ftz.f32x2 %0, %0, %1, %1;" : "+l"(x[(i >> 1) & 7]) : "l"(c));
      }
      if (WHAT == MIX_SOFTMAX) {     // per 12 MUFU: 14 FFMA2, 14 FADD2, 4 FMNMX, 8 F2FP (the forward's proportions)
        if (i < 12) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(a[i & 15]));
        else if (i < 26) asm volatile("fma.rn.ftz.f32x2 %0, %0, %1, %1;" : "+l"(x[i & 7]) : "l"(c));
        else if (i < 40) asm volatile("add.rn.ftz.f32x2 %0, %0, %1;" : "+l"(x[i & 7]) : "l"(c));
        else if (i < 44) asm volatile("max.ftz.f32 %0, %0, %1;" : "+f"(a[12 + (i & 3)]) : "f"(f1));
        else if (i < 52) asm volatile("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(d[i & 3]) : "f"(f0), "f"(f1));
      }
    }
  }
  const long long t1 = clock64();
  float s = 0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += a[i];
#pragma unroll
  for (int i = 0; i < 8; ++i) s += (float)(x[i] & 0xff);
  out[blockIdx.x * blockDim.x + threadIdx.x] = s + (float)(d[0] + d[1] + d[2] + d[3]);
  if (threadIdx.x == 0 && blockIdx.x == 0) clk[0] = t1 - t0;
}

template <int WHAT>
void run_stream(const char* name, int ninstr, float* out, long long* clk) {
  printf("| %-44s |", name);
  for (int wps = 1; wps <= 4; wps *= 2) {
    const int iters = 2000;
    for (int rep = 0; rep < 2; ++rep) stream_kernel<WHAT><<<148, wps * 128>>>(out, clk, iters);
    long long h = 0;
    cudaMemcpy(&h, clk, 8, cudaMemcpyDeviceToHost);
    printf(" %6.2f |", (double)h / iters / ninstr / wps);
  }
  printf("\n");
}

// ---- part 2: the forward's row step ------------------------------------------------------------------------------
template <int POLY, bool MAX, bool SUM = true>
__global__ void __launch_bounds__(256, 1) row_kernel(const float* in, float* out, long long* clk, int iters) {
  extern __shared__ uint4 sm[];   // [32 chunks of S + 16 of P][256 threads] x 16 B: conflict-free per-thread rows
  for (int i = threadIdx.x; i < 32 * 256; i += blockDim.x) {
    const float f = in[i & 4095];
    sm[i] = make_uint4(__float_as_uint(f), __float_as_uint(f * 0.5f), __float_as_uint(f * 0.25f), __float_as_uint(-f));
  }
  __syncthreads();
  const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(sm);
  uint32_t sr[128];
  float* sf = reinterpret_cast<float*>(sr);
  float m = 3.f, l = 0.f;
  const float c2 = 0.18f;
  __syncthreads();
  const long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 32; ++i)
      asm volatile("ld.shared.v4.b32 {%0,%1,%2,%3}, [%4];"
                   : "=r"(sr[4 * i]), "=r"(sr[4 * i + 1]), "=r"(sr[4 * i + 2]), "=r"(sr[4 * i + 3])
                   : "r"(sbase + (i * 256 + threadIdx.x) * 16)
                   : "memory");
    if (MAX) {
      float mx0 = sf[0], mx1 = sf[1], mx2 = sf[2], mx3 = sf[3];
#pragma unroll
      for (int k = 4; k < 124; k += 8) {
        mx0 = fmax3(mx0, sf[k], sf[k + 1]);
        mx1 = fmax3(mx1, sf[k + 2], sf[k + 3]);
        mx2 = fmax3(mx2, sf[k + 4], sf[k + 5]);
        mx3 = fmax3(mx3, sf[k + 6], sf[k + 7]);
      }
      mx0 = fmax3(mx0, sf[124], sf[125]);
      mx1 = fmax3(mx1, sf[126], sf[127]);
      m = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * c2;
    }
    const uint64_t cc = f2pack(c2, c2), nm = f2pack(-m, -m);
    uint64_t la = 0, lb = 0;
    uint32_t p[64];
#pragma unroll
    for (int k = 0; k < 64; ++k) {
      const uint64_t x = fma2(f2pack(sf[2 * k], sf[2 * k + 1]), cc, nm);
      float e0, e1;
      exp2_pair(pair_is_poly<POLY>(k), x, e0, e1);
      if (SUM) { if (k & 1) lb = add2(lb, f2pack(e0, e1)); else la = add2(la, f2pack(e0, e1)); }
      p[k] = pack_bf16(e0, e1);
    }
    float s0, s1;
    f2unpack(add2(la, lb), s0, s1);
    l += s0 + s1;
#pragma unroll
    for (int i = 0; i < 16; ++i)
      asm volatile("st.shared.v4.b32 [%4], {%0,%1,%2,%3};" ::"r"(p[4 * i]), "r"(p[4 * i + 1]), "r"(p[4 * i + 2]),
                   "r"(p[4 * i + 3]), "r"(sbase + ((32 + i) * 256 + threadIdx.x) * 16)
                   : "memory");
  }
  const long long t1 = clock64();
  out[blockIdx.x * blockDim.x + threadIdx.x] = l + m;
  if (threadIdx.x == 0 && blockIdx.x == 0) clk[0] = t1 - t0;
}

// The same row step in three phases (all scaled scores, then all exponentials in place, then sums and packs), the
// phases kept apart by warp barriers: does a longer distance between a MUFU and its consumer help?
template <int POLY>
__global__ void __launch_bounds__(256, 1) row_phased_kernel(const float* in, float* out, long long* clk, int iters) {
  extern __shared__ uint4 sm[];
  for (int i = threadIdx.x; i < 32 * 256; i += blockDim.x) {
    const float f = in[i & 4095];
    sm[i] = make_uint4(__float_as_uint(f), __float_as_uint(f * 0.5f), __float_as_uint(f * 0.25f), __float_as_uint(-f));
  }
  __syncthreads();
  const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(sm);
  uint32_t sr[128];
  float* sf = reinterpret_cast<float*>(sr);
  float m = 3.f, l = 0.f;
  const float c2 = 0.18f;
  __syncthreads();
  const long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 32; ++i)
      asm volatile("ld.shared.v4.b32 {%0,%1,%2,%3}, [%4];"
                   : "=r"(sr[4 * i]), "=r"(sr[4 * i + 1]), "=r"(sr[4 * i + 2]), "=r"(sr[4 * i + 3])
                   : "r"(sbase + (i * 256 + threadIdx.x) * 16)
                   : "memory");
    float mx0 = sf[0], mx1 = sf[1], mx2 = sf[2], mx3 = sf[3];
#pragma unroll
    for (int k = 4; k < 124; k += 8) {
      mx0 = fmax3(mx0, sf[k], sf[k + 1]);
      mx1 = fmax3(mx1, sf[k + 2], sf[k + 3]);
      mx2 = fmax3(mx2, sf[k + 4], sf[k + 5]);
      mx3 = fmax3(mx3, sf[k + 6], sf[k + 7]);
    }
    mx0 = fmax3(mx0, sf[124], sf[125]);
    mx1 = fmax3(mx1, sf[126], sf[127]);
    m = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * c2;
    const uint64_t cc = f2pack(c2, c2), nm = f2pack(-m, -m);
#pragma unroll
    for (int k = 0; k < 64; ++k) f2unpack(fma2(f2pack(sf[2 * k], sf[2 * k + 1]), cc, nm), sf[2 * k], sf[2 * k + 1]);
    asm volatile("bar.warp.sync 0xffffffff;" ::: "memory");
#pragma unroll
    for (int k = 0; k < 64; ++k) exp2_pair(pair_is_poly<POLY>(k), f2pack(sf[2 * k], sf[2 * k + 1]), sf[2 * k], sf[2 * k + 1]);
    asm volatile("bar.warp.sync 0xffffffff;" ::: "memory");
    uint64_t la = 0, lb = 0;
    uint32_t p[64];
#pragma unroll
    for (int k = 0; k < 64; ++k) {
      if (k & 1) lb = add2(lb, f2pack(sf[2 * k], sf[2 * k + 1])); else la = add2(la, f2pack(sf[2 * k], sf[2 * k + 1]));
      p[k] = pack_bf16(sf[2 * k], sf[2 * k + 1]);
    }
    float s0, s1;
    f2unpack(add2(la, lb), s0, s1);
    l += s0 + s1;
#pragma unroll
    for (int i = 0; i < 16; ++i)
      asm volatile("st.shared.v4.b32 [%4], {%0,%1,%2,%3};" ::"r"(p[4 * i]), "r"(p[4 * i + 1]), "r"(p[4 * i + 2]),
                   "r"(p[4 * i + 3]), "r"(sbase + ((32 + i) * 256 + threadIdx.x) * 16)
                   : "memory");
  }
  const long long t1 = clock64();
  out[blockIdx.x * blockDim.x + threadIdx.x] = l + m;
  if (threadIdx.x == 0 && blockIdx.x == 0) clk[0] = t1 - t0;
}

template <int POLY>
void run_row_phased(const float* in, float* out, long long* clk) {
  constexpr int SMEM = 48 * 256 * 16;
  cudaFuncSetAttribute(row_phased_kernel<POLY>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
  printf("| %d of 8 pairs polynomial, row maximum yes, phased |", POLY);
  for (int wps = 1; wps <= 2; ++wps) {
    const int iters = 500;
    for (int rep = 0; rep < 2; ++rep) row_phased_kernel<POLY><<<148, wps * 128, SMEM>>>(in, out, clk, iters);
    long long h = 0;
    cudaMemcpy(&h, clk, 8, cudaMemcpyDeviceToHost);
    printf(" %6.0f |", (double)h / iters);
  }
  printf(" %5d |\n", 128 * 8 * (8 - POLY) / 8);
}

template <int POLY, bool MAX, bool SUM = true>
void run_row(const float* in, float* out, long long* clk) {
  constexpr int SMEM = 48 * 256 * 16;
  cudaFuncSetAttribute(row_kernel<POLY, MAX, SUM>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
  printf("| %d of 8 pairs polynomial, row maximum %-3s%s |", POLY, MAX ? "yes" : "no", SUM ? "        " : ", no sum");
  for (int wps = 1; wps <= 2; ++wps) {
    const int iters = 500;
    for (int rep = 0; rep < 2; ++rep) row_kernel<POLY, MAX, SUM><<<148, wps * 128, SMEM>>>(in, out, clk, iters);
    long long h = 0;
    cudaMemcpy(&h, clk, 8, cudaMemcpyDeviceToHost);
    printf(" %6.0f |", (double)h / iters);
  }
  printf(" %5d |\n", 128 * 8 * (8 - POLY) / 8);
}

}  // namespace

int main() {
  float *out, *in;
  long long* clk;
  cudaMalloc(&out, 148 * 512 * 4);
  cudaMalloc(&clk, 8);
  cudaMalloc(&in, 4096 * 4);
  static float h[4096];
  for (int i = 0; i < 4096; ++i) h[i] = (float)((i * 37) % 101) * 0.1f - 5.f;
  cudaMemcpy(in, h, sizeof(h), cudaMemcpyHostToDevice);
  printf("clocks between two instructions of one SM sub-partition (independent streams)\n");
  printf("| stream                                       | 1 warp | 2 warps | 4 warps |\n|---|---|---|---|\n");
  run_stream<MUFU>("MUFU.EX2", 64, out, clk);
  run_stream<FFMA>("FFMA", 64, out, clk);
  run_stream<FFMA2>("FFMA2 (fp32x2)", 64, out, clk);
  run_stream<FADD2>("FADD2 (fp32x2)", 64, out, clk);
  run_stream<FMNMX>("FMNMX", 64, out, clk);
  run_stream<MIX_FMA2_MNMX>("FFMA2 and FMNMX alternating", 64, out, clk);
  run_stream<MIX_SOFTMAX>("12 MUFU + 14 FFMA2 + 14 FADD2 + 4 FMNMX + 8 F2FP", 52, out, clk);
  printf("\nclocks per row step (128 scores per thread: load, [maximum,] exponentials, sum, pack, store)\n");
  printf("| variant                                      | 1 warp / sub-partition | 2 warps | MUFU clocks of one warp |\n|---|---|---|---|\n");
  run_row<0, false>(in, out, clk);
  run_row<2, false>(in, out, clk);
  run_row<3, false>(in, out, clk);
  run_row<4, false>(in, out, clk);
  run_row<2, true>(in, out, clk);
  run_row<3, true>(in, out, clk);
  run_row<2, true, false>(in, out, clk);   // (row sum left to the tensor core: a 16-column MMA against ones)
  run_row<3, true, false>(in, out, clk);
  run_row<4, true, false>(in, out, clk);
  run_row_phased<0>(in, out, clk);
  run_row_phased<2>(in, out, clk);
  run_row_phased<3>(in, out, clk);
  const cudaError_t e = cudaDeviceSynchronize();
  if (e != cudaSuccess) printf("CUDA error: %s\n", cudaGetErrorString(e));
  return e != cudaSuccess;
}
