// Shared device helpers for libtabattn kernels (sm_100a only).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace tabattn {

constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

// Every kernel launch of the library goes through this counter (tabattn_launch_count()).
void count_launch(int n = 1);

struct Shape {
  int B, R, C, H, dh;
  const int32_t* n_train;   // device [B] (item only)
  const uint8_t* col_valid; // device [B*C] or nullptr
  float scale;              // softmax scale (already defaulted to 1/sqrt(dh))
};

__device__ __forceinline__ float bf16lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf16hi(uint32_t u) { return __uint_as_float(u & 0xffff0000u); }

// two fp32 -> packed bf16x2 (lo = a, hi = b), round-to-nearest-even
__device__ __forceinline__ uint32_t pack_bf16(float a, float b) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(b), "f"(a));
  return r;
}

__device__ __forceinline__ uint4 ldg_nc_v4(const void* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}

__device__ __forceinline__ void stg_v4(void* p, uint4 v) {
  asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z),
               "r"(v.w)
               : "memory");
}

// unpack 8 bf16 (one 16-byte vector) into 8 floats
__device__ __forceinline__ void unpack8(const uint4& u, float* f) {
  f[0] = bf16lo(u.x); f[1] = bf16hi(u.x);
  f[2] = bf16lo(u.y); f[3] = bf16hi(u.y);
  f[4] = bf16lo(u.z); f[5] = bf16hi(u.z);
  f[6] = bf16lo(u.w); f[7] = bf16hi(u.w);
}

__device__ __forceinline__ uint4 pack8(const float* f) {
  uint4 u;
  u.x = pack_bf16(f[0], f[1]);
  u.y = pack_bf16(f[2], f[3]);
  u.z = pack_bf16(f[4], f[5]);
  u.w = pack_bf16(f[6], f[7]);
  return u;
}

// max of three (sm_100: FMNMX3, one instruction)
__device__ __forceinline__ float fmax3(float a, float b, float c) {
  float r;
  asm("max.ftz.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
  return r;
}

__device__ __forceinline__ float fast_exp2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}


// ---- packed fp32x2 arithmetic (sm_100: FFMA2 / FADD2 / FMUL2, two fp32 lanes per issue slot) ---------
__device__ __forceinline__ uint64_t f2pack(float lo, float hi) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void f2unpack(uint64_t v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t d;
  asm("fma.rn.ftz.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b) {
  uint64_t d;
  asm("add.rn.ftz.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}
__device__ __forceinline__ uint64_t sub2(uint64_t a, uint64_t b) {
  uint64_t d;
  asm("sub.rn.ftz.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}
__device__ __forceinline__ uint64_t mul2(uint64_t a, uint64_t b) {
  uint64_t d;
  asm("mul.rn.ftz.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}

// 2^x for two values on the FMA pipe instead of the MUFU (16 ex2/clk/SM is the ceiling of the item
// kernels at dh <= 64): x is clamped to >= -126, split as n + f with n = round(x)
// (magic-number add) and f in [-0.5, 0.5]; 2^f by a cubic (max relative error 2.0e-4, an eighth of
// the bf16 rounding step the result is rounded to); 2^n by adding n to the exponent field.
// x = -inf (masked score) gives 2^-126 instead of 0: callers multiply it by zeroed operands or mask it.
__device__ __forceinline__ void exp2_poly2(uint64_t x, float& e0, float& e1) {
  float a, b;
  f2unpack(x, a, b);
  const uint64_t v = f2pack(fmaxf(a, -126.f), fmaxf(b, -126.f));
  const uint64_t magic = f2pack(12582912.f, 12582912.f);  // 1.5 * 2^23
  const uint64_t t = add2(v, magic);
  const uint64_t f = sub2(v, sub2(t, magic));
  uint64_t p = fma2(f2pack(0.053027521818876266f, 0.053027521818876266f), f,
                    f2pack(0.24221394956111908f, 0.24221394956111908f));
  p = fma2(p, f, f2pack(0.6935725808143616f, 0.6935725808143616f));
  p = fma2(p, f, f2pack(0.9999590516090393f, 0.9999590516090393f));
  float pl, ph, tl, th;
  f2unpack(p, pl, ph);
  f2unpack(t, tl, th);
  e0 = __int_as_float(__float_as_int(pl) + (__float_as_int(tl) << 23));
  e1 = __int_as_float(__float_as_int(ph) + (__float_as_int(th) << 23));
}
// 2^x for a pair: the polynomial when POLY, else two MUFU ex2
// (`poly` is a compile-time constant after unrolling the caller's loop)
__device__ __forceinline__ void exp2_pair(bool poly, uint64_t x, float& e0, float& e1) {
  if (poly) {
    exp2_poly2(x, e0, e1);
  } else {
    float a, b;
    f2unpack(x, a, b);
    e0 = fast_exp2(a);
    e1 = fast_exp2(b);
  }
}
// which pairs of an unrolled loop take the polynomial: kPolyOf8 of every 8 consecutive pairs, spread out
template <int POLY_OF_8>
__host__ __device__ constexpr bool pair_is_poly(int k) {
  return ((k % 8) * POLY_OF_8) / 8 != (((k % 8) + 1) * POLY_OF_8) / 8;
}

// Timeline instrumentation (only with -DTABATTN_TRACE, `TABATTN_TRACE=1 python -m paper_2606_03681_b200.build`; the
// shipped library has none of it): clock64() stamps of CTA 0's first 64 steps, event e of step n at trace[16 n + e].
// A kernel file that traces says TABATTN_TRACE_DEFINE(setter) once at namespace scope (its own buffer pointer and
// exported setter); paper_2606_03681_b200/trace_feature_bwd.py prints a trace; profiles/r02_attention.md has the
// reading that found the LSU jam of the per-thread row stores.
#ifdef TABATTN_TRACE
#define TABATTN_TRACE_DEFINE(setter)                                                                      \
  static __device__ long long* g_trace = nullptr;                                                         \
  extern "C" __attribute__((visibility("default"))) void setter(long long* p) {                            \
    cudaMemcpyToSymbol(g_trace, &p, sizeof(p));                                                            \
  }
// TR_INIT() once per kernel (reads the buffer pointer into a register: a stamp must not wait for a global load;
// measured ~200 clk per stamp with the load, which distorted what it timed)
#define TR_INIT() long long* const tr_buf_ = (blockIdx.x | blockIdx.y | blockIdx.z) == 0 ? g_trace : nullptr
#define TR(ev, tile) \
  do { if (tr_buf_ && (tile) < 64) tr_buf_[(tile) * 16 + (ev)] = clock64(); } while (0)
#else
#define TABATTN_TRACE_DEFINE(setter)
#define TR_INIT() do { } while (0)
#define TR(ev, tile) do { } while (0)
#endif

// 4 x 4 transpose of 16-byte chunks among the four lanes of a quad: on return lane i of the quad holds in a[k] the
// chunk i that lane k of the quad passed in.  It turns "every lane stores its own 64-byte row in four instructions"
// (32 different lines per instruction) into "a quad stores one row per instruction" (8 lines per instruction): the
// per-thread row stores of the backward were 1,536 line requests per tile and kept the LSU busy for the whole tile
// period, which also delayed the shared-memory stores of the serial P/dS section (timeline in profiles/r02_attention.md).
__device__ __forceinline__ void quad_transpose(uint4 (&a)[4], int lane) {
#pragma unroll
  for (int st = 0; st < 2; ++st) {
    const int m = 1 << st;
    const bool up = (lane & m) != 0;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      if (c & m) continue;
      uint4 send = up ? a[c] : a[c | m];
      send.x = __shfl_xor_sync(0xffffffffu, send.x, m);
      send.y = __shfl_xor_sync(0xffffffffu, send.y, m);
      send.z = __shfl_xor_sync(0xffffffffu, send.z, m);
      send.w = __shfl_xor_sync(0xffffffffu, send.w, m);
      if (up) a[c] = send; else a[c | m] = send;
    }
  }
}

// Offsets and liveness of the four rows of this lane's quad, as seen by the lane that stores chunk (lane & 3) of them.
struct QuadRows {
  size_t off[4];
  bool live[4];
  __device__ __forceinline__ void init(size_t my_off, bool my_live, int lane) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int src = (lane & ~3) + k;
      const unsigned long long o = __shfl_sync(0xffffffffu, (unsigned long long)my_off, src);
      off[k] = (size_t)o + (size_t)(lane & 3) * 16;
      live[k] = __shfl_sync(0xffffffffu, (int)my_live, src) != 0;
    }
  }
};

}  // namespace tabattn
