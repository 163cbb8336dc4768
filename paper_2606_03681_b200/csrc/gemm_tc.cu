// tcgen05 GEMM core (gemm_tc.cuh): 128 x BN output tiles, a 2-3 stage TMA ring over 64-wide k-blocks, fp32 accumulators
// in TMEM, fused epilogue, TMA store.  Warp 0 = TMA producer (one lane), warp 1 = MMA issuer (owns the TMEM
// allocation), warps 2-9 = epilogue (one thread per accumulator row and column half).  A CTA is persistent over the
// row tiles of its column tile and alternates TWO accumulators, so that tile i's epilogue runs under tile i+1's loads
// and MMAs; two such CTAs fit an SM (96 KB of shared memory and 256 TMEM columns each at BN = 128).  Two epilogues:
// with an auxiliary tile (residual, gelu') the tile is prefetched by TMA into a staging tile, overwritten in place and
// stored by TMA, behind a two-stage ring; without one the epilogue stores straight from registers (quad-transposed
// rows) and the staging tile's shared memory is a third ring stage.  These contractions have K = 192..768 only: a tile is 4-12 k-blocks of work and the
// kernels are bound by HBM and the epilogue, not by the tensor pipe (profiles/r02_blocks.md).
#include "gemm_tc.cuh"

#include <cudaTypedefs.h>

#include <algorithm>

#include "common.cuh"
#include "device.h"
#include "tc_common.cuh"

namespace tabattn {
namespace gemm {

TABATTN_TRACE_DEFINE(tabattn_debug_set_trace_gemm)

namespace {

using namespace tc;

constexpr int BM = 128, BK = 64;
constexpr int kEpiWarps = 8;                     // two per TMEM lane quadrant, each half of the tile's columns
constexpr int kThreads = (2 + kEpiWarps) * 32;
constexpr int A_BYTES = BM * BK * 2;   // 16 KB, either layout

struct KParams {
  int M, N, K;
  int kb_total, kb_per_slab, slabs;
  float alpha, beta;
  const float* row_scale;
  int act, aux_mode;
  float* partial;
  int split_cols;
  int a_batched, b_batched;   // 0: operand shared by all batches (TMA batch coordinate 0)
  int a_split_k;              // > 0: A is three tensors of this many columns
  int a_split_m;              // > 0: (MN-major A) three tensors of this many output rows
  int dual_out;
  // direct epilogue (no auxiliary tile, not split-K): the outputs as raw pointers
  unsigned char* c_ptr[3];
  long long ldc, c_bstride;   // elements
};

__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* m, uint32_t bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(m)), "r"(bar), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}
__device__ __forceinline__ void tma_store_3d(const CUtensorMap* m, uint32_t src, int c0, int c1, int c2) {
  asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.tile.bulk_group [%0, {%2, %3, %4}], [%1];" ::"l"(
                   reinterpret_cast<uint64_t>(m)),
               "r"(src), "r"(c0), "r"(c1), "r"(c2)
               : "memory");
}

// GELU (exact, erf form) in the epilogues.  The MLP up-projection's epilogue was bound by this arithmetic: the timeline
// (profiles/r02_blocks.md) shows 9,800 of a tile's 16,000 clocks in the GELU pass, ~39 issue slots per element with
// erf by Abramowitz & Stegun (a reciprocal, an ex2 and ten scalar FMAs per element).  Now erf(x / sqrt 2) is evaluated
// for two values at a time on the FMA pipe alone: z = x / sqrt 2 clamped to [-3, 3] (erf(3) = 1 - 2.2e-5), then
// z P(z^2) with a degree-8 polynomial fitted at Chebyshev nodes of z^2 in [0, 9].  |erf error| <= 4.2e-5 in fp32,
// |gelu error| <= 8.8e-5 (x in [-6, 6], checked on 200,001 points against math.erf): 1/20 of the bf16 rounding step of
// an activation of size 1, absolute -- the far negative tail, where gelu itself is below 4e-3, is only that accurate.
__device__ __forceinline__ uint64_t pk2(float c) { return f2pack(c, c); }
__device__ __forceinline__ uint64_t erf_half2(uint64_t x) {
  float a, b;
  f2unpack(mul2(x, pk2(0.70710678118654752f)), a, b);
  a = fminf(fmaxf(a, -3.f), 3.f);
  b = fminf(fmaxf(b, -3.f), 3.f);
  const uint64_t z = f2pack(a, b), s = mul2(z, z);
  uint64_t p = fma2(pk2(4.918276073e-08f), s, pk2(-2.267730623e-06f));
  p = fma2(p, s, pk2(4.614729186e-05f));
  p = fma2(p, s, pk2(-5.535572417e-04f));
  p = fma2(p, s, pk2(4.437862287e-03f));
  p = fma2(p, s, pk2(-2.564961361e-02f));
  p = fma2(p, s, pk2(1.118625027e-01f));
  p = fma2(p, s, pk2(-3.758186012e-01f));
  p = fma2(p, s, pk2(1.128362939e+00f));
  return mul2(z, p);
}
// gelu(x) = x/2 + x/2 erf(x / sqrt 2) for a pair
__device__ __forceinline__ void gelu_pair(float& x0, float& x1) {
  const uint64_t x = f2pack(x0, x1), h = mul2(x, pk2(0.5f));
  f2unpack(fma2(h, erf_half2(x), h), x0, x1);
}
// gelu'(x) = 1/2 + 1/2 erf(x / sqrt 2) + x exp(-x^2 / 2) / sqrt(2 pi) for a pair (the Gaussian on the MUFU)
__device__ __forceinline__ void gelu_grad_pair(float x0, float x1, float& g0, float& g1) {
  const uint64_t x = f2pack(x0, x1);
  float e0, e1;
  f2unpack(mul2(mul2(x, x), pk2(-0.5f * kLog2e)), e0, e1);
  const uint64_t gauss = mul2(mul2(x, pk2(0.3989422804014327f)), f2pack(fast_exp2(e0), fast_exp2(e1)));
  f2unpack(add2(fma2(erf_half2(x), pk2(0.5f), pk2(0.5f)), gauss), g0, g1);
}

template <int BN>
struct Cfg {
  // BN = 256 (split-K weight gradients only): a CTA computes TWO row tiles, 256 x 256, from one B stage -- these
  // kernels are bound by operand traffic from L2 (~8.5 TB/s) and this fetches every operand byte the fewest times
  static constexpr bool PAIR = BN == 256;
  static constexpr int A_STAGE = (PAIR ? 2 : 1) * A_BYTES;
  static constexpr int ST = BN == 128 ? 2 : 3;
  // ring depth when the epilogue needs no staging tile (it stores straight from registers): the freed shared memory
  // holds one more stage -- the plain projections are bound by the latency of their operand loads (timeline,
  // profiles/r02_blocks.md: a round trip is ~2,400 clk and a K = 768 tile was six of them)
  static constexpr int ST_DIRECT = ST + 1, ST_MAX = ST_DIRECT;
  static constexpr int B_BYTES = BN * BK * 2;
  static constexpr int STAGE = A_STAGE + B_BYTES;
  static constexpr int STAGING = (BN / 64) * (BM * 128);
  // the epilogue's staging tile is a buffer of its own (an auxiliary tile is prefetched into it when there is one):
  // the ring keeps loading the next tile while the epilogue of the current one writes it
  static constexpr int SMEM_AUX = ST * STAGE + STAGING + 1024;
  static constexpr int SMEM_SPLITK = ST * STAGE + 1024;
  static constexpr int SMEM_DIRECT = ST_DIRECT * STAGE + 1024;   // (fp32 partial tiles go straight to global memory)
};

template <int BN, int A_MN, int B_MN>
__global__ void __launch_bounds__(kThreads, 2)
gemm_tc_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapA2,
               const __grid_constant__ CUtensorMap mapA3, const __grid_constant__ CUtensorMap mapB,
               const __grid_constant__ CUtensorMap mapAux, const __grid_constant__ CUtensorMap mapC0,
               const __grid_constant__ CUtensorMap mapC1, const __grid_constant__ CUtensorMap mapC2,
               const __grid_constant__ KParams p) {
  TR_INIT();
  using C = Cfg<BN>;
  constexpr int ST = C::ST;
  // (trace builds: only the QKV projection, the MLP up-projection and the gelu' product are stamped)
  [[maybe_unused]] const bool traced = p.split_cols > 0 || p.dual_out || p.aux_mode == AUX_GELU_GRAD;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const bool direct = BN <= 128 && p.aux_mode == AUX_NONE && p.partial == nullptr;
  const uint32_t st_n = direct ? C::ST_DIRECT : ST;          // ring depth
  const uint32_t sA = sbase, sB = sA + st_n * C::A_STAGE;
  const uint32_t sOut = sB + st_n * C::B_BYTES;   // the epilogue's staging tile (the auxiliary tile lands in it first)
  __shared__ uint64_t bar_full[C::ST_MAX], bar_empty[C::ST_MAX], bar_acc[2], bar_aux, bar_acc_free[2], bar_out_free;
  __shared__ uint32_t tmem_slot;

  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;
  // A CTA walks the row tiles my = blockIdx.y, blockIdx.y + gridDim.y, ... of its column tile (the host sizes
  // gridDim.y so that all CTAs are resident at once): TMEM allocation, barrier set-up and the CTA launch are paid once
  // per CTA instead of once per 128 x BN tile -- with K = 256..768 a tile is only 4-12 k-blocks of work.
  constexpr int BMT = C::PAIR ? 2 * BM : BM;   // rows per CTA step
  const int n0 = blockIdx.x * BN, tiles_m = (p.M + BMT - 1) / BMT;
  const bool splitk = p.partial != nullptr;   // fp32 partial tiles instead of the bf16 output
  const int bz = splitk ? 0 : blockIdx.z, slab = splitk ? blockIdx.z : 0;
  const int kb0 = slab * p.kb_per_slab, kb1 = min(p.kb_total, kb0 + p.kb_per_slab);

  // two accumulators (tile i's epilogue under tile i+1's MMAs); a split-K CTA computes one tile and needs one
  // Programmatic dependent launch: the next GEMM of the stream may bring its CTAs up (TMEM allocation, barrier set-up)
  // while this one runs, and this one did the same under its predecessor; nothing below the griddepcontrol.wait
  // touches global memory before the predecessor has completed and flushed.  (Chains of small GEMMs -- the 16
  // launches of Newton-Schulz -- are latency-bound: ~7 us per kernel.)
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  if (warp == 1) tmem_alloc(smem_u32(&tmem_slot), (splitk && !C::PAIR) ? BN : 2 * BN);
  if (threadIdx.x == 0) {
    for (int i = 0; i < C::ST_MAX; ++i) {
      mbar_init(smem_u32(&bar_full[i]), 1);
      mbar_init(smem_u32(&bar_empty[i]), 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(smem_u32(&bar_acc[i]), 1);
      mbar_init(smem_u32(&bar_acc_free[i]), kEpiWarps);   // the epilogue warps have read the accumulator
    }
    mbar_init(smem_u32(&bar_aux), 1);
    mbar_init(smem_u32(&bar_out_free), 1);           // the tile's store has read the staging tile
    fence_barrier_init();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  asm volatile("griddepcontrol.wait;" ::: "memory");

  if (warp == 0) {
    if (lane == 0) {
      tma_prefetch_desc(&mapA);
      tma_prefetch_desc(&mapB);
      const int ba = p.a_batched ? bz : 0, bb = p.b_batched ? bz : 0;
      uint32_t st = 0, ph = 0, it = 0;
      for (int my = blockIdx.y; my < tiles_m; my += gridDim.y, ++it) {
      const int m0 = my * BMT;
      // (the A / B loads of a tile run ahead under the previous tile's epilogue; the auxiliary load, below, waits for
      // the staging tile)
      for (int kb = kb0; kb < kb1; ++kb) {
        const uint32_t full = smem_u32(&bar_full[st]);
        mbar_wait<true>(smem_u32(&bar_empty[st]), ph ^ 1);
        if (traced && kb == kb0) TR(0, it);                 // first stage of the tile free, loads start
        mbar_arrive_expect_tx(full, C::STAGE);
        const uint32_t a = sA + st * C::A_STAGE, b = sB + st * C::B_BYTES;
        if (A_MN) {
#pragma unroll
          for (int mt = 0; mt < (C::PAIR ? 2 : 1); ++mt) {
            const CUtensorMap* ma = &mapA;
            int ml = m0 + BM * mt;
            if (p.a_split_m > 0) {
              const int seg = min(ml / p.a_split_m, 2);
              ml -= seg * p.a_split_m;
              ma = seg == 0 ? &mapA : (seg == 1 ? &mapA2 : &mapA3);
            }
            tma_load_3d(a + mt * A_BYTES, ma, full, ml, kb * BK, ba);
            tma_load_3d(a + mt * A_BYTES + 64 * 128, ma, full, ml + 64, kb * BK, ba);
          }
        } else if (p.a_split_k > 0) {
          const int seg = (kb * BK) / p.a_split_k, kin = kb * BK - seg * p.a_split_k;
          tma_load_3d(a, seg == 0 ? &mapA : (seg == 1 ? &mapA2 : &mapA3), full, kin, m0, ba);
        } else {
          tma_load_3d(a, &mapA, full, kb * BK, m0, ba);
        }
        if (B_MN) {
#pragma unroll
          for (int h = 0; h < BN / 64; ++h) tma_load_3d(b + h * (64 * 128), &mapB, full, n0 + 64 * h, kb * BK, bb);
        } else {
          tma_load_3d(b, &mapB, full, kb * BK, n0, bb);
        }
        if (++st == st_n) { st = 0; ph ^= 1; }
      }
      if (traced) TR(1, it);                                // last load of the tile issued
      if (p.aux_mode != AUX_NONE) {
        // the tile of the auxiliary operand lands in the staging tile the epilogue later overwrites in place
        if (it > 0) mbar_wait<true>(smem_u32(&bar_out_free), (it - 1) & 1);
        mbar_arrive_expect_tx(smem_u32(&bar_aux), C::STAGING);
#pragma unroll
        for (int h = 0; h < BN / 64; ++h) tma_load_3d(sOut + h * (BM * 128), &mapAux, smem_u32(&bar_aux), n0 + 64 * h, m0, bz);
      }
      }
    }
  } else if (warp == 1) {
    constexpr uint32_t idesc = make_idesc_bf16(BM, BN, A_MN != 0, B_MN != 0);
    // K-major: rows of 128 bytes, 8-row groups 1024 bytes apart, 32 bytes per k-step.
    // MN-major: [64 k-rows][128 bytes] atoms of 64 M/N elements, 8192 bytes apart; 16 k-rows = 2048 bytes per k-step.
    const uint64_t dA = A_MN ? make_smem_desc<128>(sA, 64 * 128, 1024) : make_smem_desc<128>(sA, 16, 1024);
    const uint64_t dB = B_MN ? make_smem_desc<128>(sB, 64 * 128, 1024) : make_smem_desc<128>(sB, 16, 1024);
    uint32_t st = 0, ph = 0, it = 0;
    for (int my = blockIdx.y; my < tiles_m; my += gridDim.y, ++it) {
      const uint32_t ab = it & 1, acc = tmem + ab * BN;
      if (it > 1) {   // the epilogue has read this accumulator's previous tile out of TMEM
        mbar_wait(smem_u32(&bar_acc_free[ab]), ((it >> 1) - 1) & 1);
        tc_fence_after();
      }
      for (int kb = kb0; kb < kb1; ++kb) {
        mbar_wait(smem_u32(&bar_full[st]), ph);
        if (traced && lane == 0 && kb == kb0) TR(2, it);    // first k-block landed
        tc_fence_after();
        const uint64_t a = dA + (uint64_t)((st * C::A_STAGE) >> 4), b = dB + (uint64_t)((st * C::B_BYTES) >> 4);
#pragma unroll
        for (int kk = 0; kk < BK / 16; ++kk) {
          mma_ss_e(acc, a + (A_MN ? kk * 128 : 2 * kk), b + (B_MN ? kk * 128 : 2 * kk), idesc,
                   (kb > kb0 || kk > 0) ? 1u : 0u);
          if constexpr (C::PAIR)   // the second row tile of the pair, same B stage, second accumulator
            mma_ss_e(acc + BN, a + (A_BYTES >> 4) + (A_MN ? kk * 128 : 2 * kk), b + (B_MN ? kk * 128 : 2 * kk), idesc,
                     (kb > kb0 || kk > 0) ? 1u : 0u);
        }
        tc_commit_e(smem_u32(&bar_empty[st]));
        if (++st == st_n) { st = 0; ph ^= 1; }
      }
      tc_commit_e(smem_u32(&bar_acc[ab]));
      if (traced && lane == 0) TR(3, it);                   // MMAs of the tile issued
    }
  } else {
    // ------------------------------------------------------------------------------ epilogue
    const int q = warp & 3, r = 32 * q + lane;
    const int c_lo = ((warp - 2) >> 2) * (BN / 64), c_hi = c_lo + BN / 64;   // this warp's 32-column groups
    const uint32_t tacc0 = tmem + ((uint32_t)(32 * q) << 16);
    const bool has_k = kb1 > kb0;
    const int passes = p.dual_out ? 2 : 1;
    uint32_t it = 0;
    for (int my = blockIdx.y; my < tiles_m; my += gridDim.y, ++it) {
    const int m0 = my * BMT, m = m0 + r;
    float rs = p.alpha;
    if (p.row_scale && m < p.M) rs *= __ldg(p.row_scale + (size_t)bz * p.M + m);
    const uint32_t ab = it & 1, tacc = tacc0 + ab * BN;
    mbar_wait(smem_u32(&bar_acc[ab]), (it >> 1) & 1);
    if (traced && threadIdx.x == 64) TR(4, it);             // accumulator complete
    tc_fence_after();
    if (direct) {
      // no staging tile: a quad of lanes transposes its four rows' 64-byte groups in registers and stores one row per
      // instruction (quad_transpose, common.cuh); no fence, CTA barrier or store wait in the tile's path
      if constexpr (BN <= 128) {
        QuadRows qr;
        qr.init((size_t)m * (size_t)p.ldc * 2, m < p.M, lane);
        for (int pass = 0; pass < passes; ++pass) {
          const bool do_act = p.act == ACT_GELU && (!p.dual_out || pass == 1);
#pragma unroll 1
          for (int c = c_lo; c < c_hi; ++c) {
            uint32_t v[32];
            tmem_ld32(tacc + 32 * c, v);
            tmem_wait_ld();
            uint4 u[4];
#pragma unroll
            for (int ch = 0; ch < 4; ++ch) {
              float f[8];
#pragma unroll
              for (int e = 0; e < 8; ++e) f[e] = has_k ? __uint_as_float(v[8 * ch + e]) * rs : 0.f;
              if (do_act) {
#pragma unroll
                for (int e = 0; e < 8; e += 2) gelu_pair(f[e], f[e + 1]);
              }
              u[ch] = pack8(f);
            }
            const int col = n0 + 32 * c;
            int t = p.split_cols > 0 ? col / p.split_cols : 0;
            const int cin = col - t * p.split_cols;
            if (p.dual_out) t = pass;
            unsigned char* base = p.c_ptr[t] + ((size_t)bz * (size_t)p.c_bstride + (size_t)cin) * 2;
            quad_transpose(u, lane);
            const bool col_ok = col + 8 * (lane & 3) < p.N;
#pragma unroll
            for (int k4 = 0; k4 < 4; ++k4)
              if (qr.live[k4] && col_ok) stg_v4(base + qr.off[k4], u[k4]);
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&bar_acc_free[ab]));
        if (traced && threadIdx.x == 64) TR(5, it);           // tile stored
      }
      continue;
    }
    // the staging tile: free once the previous tile's store has read it (with an auxiliary tile the producer waited
    // for that before loading it)
    if (p.aux_mode != AUX_NONE) mbar_wait(smem_u32(&bar_aux), it & 1);
    else if (it > 0 && !splitk) mbar_wait(smem_u32(&bar_out_free), (it - 1) & 1);
    for (int pass = 0; pass < passes; ++pass) {
      // dual output: pass 0 stores the value before the activation (C0), pass 1 the value after it (C1)
      const bool do_act = p.act == ACT_GELU && (!p.dual_out || pass == 1);
#pragma unroll 1
      for (int c = c_lo; c < c_hi; ++c) {
        uint32_t v[32];
        tmem_ld32(tacc + 32 * c, v);
        tmem_wait_ld();
        if (!has_k) {
#pragma unroll
          for (int j = 0; j < 32; ++j) v[j] = 0u;
        }
        if (splitk) {
#pragma unroll
          for (int mt = 0; mt < (C::PAIR ? 2 : 1); ++mt) {
            if (mt == 1) {   // the pair's second row tile (second accumulator)
              tmem_ld32(tacc + BN + 32 * c, v);
              tmem_wait_ld();
              if (!has_k) {
#pragma unroll
                for (int j = 0; j < 32; ++j) v[j] = 0u;
              }
            }
            const int mm = m + BM * mt;
            if (mm < p.M) {
              float* dst = p.partial + ((size_t)slab * p.M + mm) * p.N + n0 + 32 * c;
#pragma unroll
              for (int j = 0; j < 8; ++j)
                if (n0 + 32 * c + 4 * j < p.N)
                  *reinterpret_cast<float4*>(dst + 4 * j) =
                      make_float4(__uint_as_float(v[4 * j]), __uint_as_float(v[4 * j + 1]),
                                  __uint_as_float(v[4 * j + 2]), __uint_as_float(v[4 * j + 3]));
            }
          }
          continue;
        }
#pragma unroll
        for (int ch = 0; ch < 4; ++ch) {
          const int col = 32 * c + 8 * ch;                       // first of 8 columns inside the tile
          const uint32_t off = sOut + (uint32_t)(col >> 6) * (BM * 128) + (uint32_t)r * 128 +
                               (uint32_t)((((col & 63) >> 3) ^ (r & 7)) << 4);
          float f[8], a[8];
#pragma unroll
          for (int e = 0; e < 8; ++e) f[e] = __uint_as_float(v[8 * ch + e]) * rs;
          if (p.aux_mode != AUX_NONE) {
            const uint4 u = lds_v4(off);
            unpack8(u, a);
          }
          if (p.aux_mode == AUX_ADD) {
#pragma unroll
            for (int e = 0; e < 8; ++e) f[e] = fmaf(p.beta, a[e], f[e]);
          }
          if (do_act) {
#pragma unroll
            for (int e = 0; e < 8; e += 2) gelu_pair(f[e], f[e + 1]);
          }
          if (p.aux_mode == AUX_GELU_GRAD) {
#pragma unroll
            for (int e = 0; e < 8; e += 2) {
              float g0, g1;
              gelu_grad_pair(a[e], a[e + 1], g0, g1);
              f[e] *= g0;
              f[e + 1] *= g1;
            }
          }
          const uint4 o = pack8(f);
          sts_v4(off, o.x, o.y, o.z, o.w);
        }
      }
      if (pass == passes - 1 || splitk) {   // the accumulator has been read for the last time
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&bar_acc_free[ab]));
      }
      if (splitk) break;
      if (traced && threadIdx.x == 64) TR(5 + 4 * pass, it);  // this warp's part of the staging tile written
      fence_proxy_async_smem();
      named_bar_sync(1, kEpiWarps * 32);
      if (traced && threadIdx.x == 64) TR(6 + 4 * pass, it);  // all epilogue warps done
      if (warp == 2 && lane == 0) {
#pragma unroll
        for (int h = 0; h < BN / 64; ++h) {
          const int col = n0 + 64 * h;
          if (col >= p.N) continue;
          int t = p.split_cols > 0 ? col / p.split_cols : 0;
          const int cin = col - t * p.split_cols;
          if (p.dual_out) t = pass;
          const CUtensorMap* mc = t == 0 ? &mapC0 : (t == 1 ? &mapC1 : &mapC2);
          tma_store_3d(mc, sOut + h * (BM * 128), cin, m0, bz);
        }
        bulk_commit();
        if (traced) TR(7 + 4 * pass, it);                   // store issued
        bulk_wait_read<0>();   // (the staging tile has been read; the writes themselves complete in the background)
        if (traced) TR(8 + 4 * pass, it);                   // staging tile read by the store
      }
      // (dual output: the staging tile is rewritten by the next pass only after the store has read it)
      if (passes > 1) named_bar_sync(1, kEpiWarps * 32);
    }
    // next tile: the producer may overwrite the staging tile (the store above has completed), and through it -- its
    // loads precede the MMAs that precede bar_acc -- so may the other epilogue warps
    if (warp == 2 && lane == 0) mbar_arrive(smem_u32(&bar_out_free));
    }
    if (warp == 2 && lane == 0) bulk_wait<0>();   // the CTA's stores are complete before it exits
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem, (splitk && !C::PAIR) ? BN : 2 * BN);
}

__global__ void reduce_slabs_kernel(const float* __restrict__ partial, int slabs, long long mn, float scale,
                                    void* __restrict__ out, int out_f32) {
  const long long i = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * 4;
  if (i >= mn) return;
  float4 a = make_float4(0.f, 0.f, 0.f, 0.f);
  for (int s = 0; s < slabs; ++s) {
    const float4 v = *reinterpret_cast<const float4*>(partial + (long long)s * mn + i);
    a.x += v.x; a.y += v.y; a.z += v.z; a.w += v.w;
  }
  a.x *= scale; a.y *= scale; a.z *= scale; a.w *= scale;
  if (out_f32) {
    *reinterpret_cast<float4*>(static_cast<float*>(out) + i) = a;
  } else {
    uint2 o;
    o.x = pack_bf16(a.x, a.y);
    o.y = pack_bf16(a.z, a.w);
    *reinterpret_cast<uint2*>(static_cast<uint16_t*>(out) + i) = o;
  }
}

PFN_cuTensorMapEncodeTiled_v12000 encode_fn() {
  static PFN_cuTensorMapEncodeTiled_v12000 fn = []() -> PFN_cuTensorMapEncodeTiled_v12000 {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      return nullptr;
    return reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(p);
  }();
  return fn;
}

// bf16 matrix [rows][inner] (pitch ld elements) x batch -> 3-D map, box (64 inner, box_rows, 1), 128-byte swizzle
bool make_map(CUtensorMap* m, const void* ptr, long long inner, long long rows, long long ld, int batch,
              long long batch_stride, int box_rows) {
  auto fn = encode_fn();
  if (!fn || !ptr) return false;
  const bool shared = batch_stride == 0 || batch <= 1;
  cuuint64_t dims[3] = {(cuuint64_t)inner, (cuuint64_t)rows, (cuuint64_t)(shared ? 1 : batch)};
  cuuint64_t strides[2] = {(cuuint64_t)ld * 2, (cuuint64_t)(shared ? rows * ld : batch_stride) * 2};
  cuuint32_t box[3] = {64, (cuuint32_t)box_rows, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(ptr), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int BN, int A_MN, int B_MN>
cudaError_t launch_t(const Problem& p, const KParams& kp, cudaStream_t stream) {
  const DeviceInfo* di = current_device();
  if (!di) return cudaErrorInvalidDevice;
  CUtensorMap ma, ma2, ma3, mb, maux, mc[3];
  // A: K-major -> stored [M][K]: inner K, box rows 128; MN-major -> stored [K][M]: inner M, box 64 k-rows
  bool ok = p.A.mn_major ? make_map(&ma, p.A.ptr, p.M, p.K, p.A.ld, p.batch, p.A.batch_stride, 64)
                         : make_map(&ma, p.A.ptr, p.K, p.M, p.A.ld, p.batch, p.A.batch_stride, BM);
  ma2 = ma; ma3 = ma;
  if (p.a_split_m > 0) {
    ok = ok && p.A.mn_major && make_map(&ma, p.A.ptr, p.a_split_m, p.K, p.A.ld, p.batch, p.A.batch_stride, 64) &&
         make_map(&ma2, p.A2, p.a_split_m, p.K, p.A.ld, p.batch, p.A.batch_stride, 64) &&
         make_map(&ma3, p.A3, p.a_split_m, p.K, p.A.ld, p.batch, p.A.batch_stride, 64);
  }
  if (p.a_split_k > 0) {
    ok = ok && !p.A.mn_major && make_map(&ma, p.A.ptr, p.a_split_k, p.M, p.A.ld, p.batch, p.A.batch_stride, BM) &&
         make_map(&ma2, p.A2, p.a_split_k, p.M, p.A.ld, p.batch, p.A.batch_stride, BM) &&
         make_map(&ma3, p.A3, p.a_split_k, p.M, p.A.ld, p.batch, p.A.batch_stride, BM);
  }
  ok = ok && (p.B.mn_major ? make_map(&mb, p.B.ptr, p.N, p.K, p.B.ld, p.batch, p.B.batch_stride, 64)
                           : make_map(&mb, p.B.ptr, p.K, p.N, p.B.ld, p.batch, p.B.batch_stride, BN));
  const int nout = p.partial ? 0 : (p.dual_out ? 2 : (p.split_cols > 0 ? (p.N + p.split_cols - 1) / p.split_cols : 1));
  const long long out_cols = p.split_cols > 0 ? p.split_cols : p.N;
  for (int t = 0; t < 3; ++t) {
    if (t < nout) ok = ok && make_map(&mc[t], p.C[t], out_cols, p.M, p.ldc, p.batch, p.c_batch_stride, BM);
    else mc[t] = t > 0 && nout > 0 ? mc[0] : ma;
  }
  if (p.aux_mode != AUX_NONE) ok = ok && make_map(&maux, p.aux, p.N, p.M, p.ld_aux, p.batch, p.aux_batch_stride, BM);
  else maux = ma;
  if (!ok) return cudaErrorInvalidValue;
  auto kern = gemm_tc_kernel<BN, A_MN, B_MN>;
  static SmemAttr attr;
  constexpr int kSmemMax = BN > 128 ? Cfg<BN>::SMEM_SPLITK
                                    : (Cfg<BN>::SMEM_AUX > Cfg<BN>::SMEM_DIRECT ? Cfg<BN>::SMEM_AUX : Cfg<BN>::SMEM_DIRECT);
  cudaError_t e = attr.ensure(kern, kSmemMax, di->ordinal);
  if (e != cudaSuccess) return e;
  if (BN > 128 && !p.partial) return cudaErrorInvalidValue;   // (256-wide tiles: split-K only)
  const int smem = p.partial ? Cfg<BN>::SMEM_SPLITK : (p.aux_mode == AUX_NONE ? Cfg<BN>::SMEM_DIRECT : Cfg<BN>::SMEM_AUX);
  // row tiles per launch: all of them (split-K, batched and small problems), else as many as keep every CTA resident
  // (three per SM); each CTA then walks its column of row tiles (see the kernel)
  constexpr int kRowsPerCta = BN == 256 ? 2 * BM : BM;   // (256-wide tiles come in pairs of row tiles)
  const int tiles_n = (p.N + BN - 1) / BN, tiles_m = (p.M + kRowsPerCta - 1) / kRowsPerCta, gz = p.partial ? kp.slabs : p.batch;
  int gy = tiles_m;
  if (!p.partial) gy = std::min(tiles_m, std::max(1, (2 * di->num_sms) / (tiles_n * gz)));
  dim3 grid(tiles_n, gy, gz);
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid;
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = stream;
  cudaLaunchAttribute attr_pdl{};
  attr_pdl.id = cudaLaunchAttributeProgrammaticStreamSerialization;   // (see griddepcontrol in the kernel)
  attr_pdl.val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = &attr_pdl;
  cfg.numAttrs = 1;
  e = cudaLaunchKernelEx(&cfg, kern, ma, ma2, ma3, mb, maux, mc[0], mc[1], mc[2], kp);
  count_launch();
  return e != cudaSuccess ? e : cudaGetLastError();
}

template <int BN>
cudaError_t launch_bn(const Problem& p, const KParams& kp, cudaStream_t stream) {
  if (!p.A.mn_major && !p.B.mn_major) return launch_t<BN, 0, 0>(p, kp, stream);
  if (!p.A.mn_major && p.B.mn_major) return launch_t<BN, 0, 1>(p, kp, stream);
  if (p.A.mn_major && p.B.mn_major) return launch_t<BN, 1, 1>(p, kp, stream);
  return cudaErrorInvalidValue;   // (A MN-major with B K-major is not needed by any caller)
}

}  // namespace

int slabs_for(long long K, int tiles, int num_sms) {
  const long long kb_total = (K + BK - 1) / BK;
  long long want = (2LL * num_sms + tiles - 1) / tiles;
  want = want < 1 ? 1 : (want > 128 ? 128 : want);
  if (want > kb_total) want = kb_total;
  const long long per = (kb_total + want - 1) / want;
  return (int)((kb_total + per - 1) / per);
}

cudaError_t launch(const Problem& p, cudaStream_t stream) {
  if (p.M < 1 || p.N < 1 || p.K < 1 || p.batch < 1) return cudaErrorInvalidValue;
  // TMA: row pitches are multiples of 16 bytes; the extents themselves are free (out-of-range box parts read 0)
  if ((p.A.ld & 7) || (p.B.ld & 7) || (!p.partial && (p.ldc & 7)) || (p.aux_mode != AUX_NONE && (p.ld_aux & 7)))
    return cudaErrorInvalidValue;
  if (p.slabs > 1 && !p.partial) return cudaErrorInvalidValue;
  if (p.partial && (p.batch != 1 || (p.N & 3))) return cudaErrorInvalidValue;
  if (p.split_cols > 0 && (p.split_cols % 64 != 0)) return cudaErrorInvalidValue;
  KParams kp{};
  kp.M = p.M; kp.N = p.N; kp.K = p.K;
  kp.kb_total = (p.K + BK - 1) / BK;
  const int want = p.slabs > 1 ? p.slabs : 1;
  kp.kb_per_slab = (kp.kb_total + want - 1) / want;
  kp.slabs = (kp.kb_total + kp.kb_per_slab - 1) / kp.kb_per_slab;
  if (kp.slabs != want) return cudaErrorInvalidValue;   // (callers size slabs with gemm::slabs_for)
  kp.alpha = p.alpha; kp.beta = p.beta; kp.row_scale = p.row_scale; kp.act = p.act; kp.aux_mode = p.aux_mode;
  kp.partial = p.partial; kp.split_cols = p.split_cols;
  kp.a_batched = p.A.batch_stride != 0; kp.b_batched = p.B.batch_stride != 0;
  kp.a_split_k = p.a_split_k; kp.a_split_m = p.a_split_m; kp.dual_out = p.dual_out;
  for (int t = 0; t < 3; ++t) kp.c_ptr[t] = static_cast<unsigned char*>(p.C[t] ? p.C[t] : p.C[0]);
  kp.ldc = p.ldc; kp.c_bstride = p.c_batch_stride;
  if (p.a_split_m > 0 && (p.a_split_m % 128 != 0 || p.M != 3 * p.a_split_m || !p.A2 || !p.A3 || !p.A.mn_major || p.a_split_k > 0))
    return cudaErrorInvalidValue;
  if (p.a_split_k > 0 && (p.a_split_k % 64 != 0 || p.K != 3 * p.a_split_k || !p.A2 || !p.A3)) return cudaErrorInvalidValue;
  if (p.dual_out && (p.split_cols > 0 || p.partial)) return cudaErrorInvalidValue;
  // 128-wide tiles when N allows it (fewer re-reads of A), else 64; split outputs need 64-column granularity
  // Split-K weight gradients (both operands MN-major, K = all cells): these are bound by the operand traffic from L2
  // (~8 TB/s measured with 128 x 128 tiles, each operand byte fetched by two to six CTAs), so the tile is as wide as
  // the MMA allows
  if (p.partial && p.A.mn_major && p.B.mn_major && p.N % 256 == 0) return launch_t<256, 1, 1>(p, kp, stream);
  const bool bn128 = (p.N % 128 == 0) && (p.split_cols == 0 || p.split_cols % 128 == 0);
  return bn128 ? launch_bn<128>(p, kp, stream) : launch_bn<64>(p, kp, stream);
}

cudaError_t launch_reduce_slabs(const float* partial, int slabs, long long mn, float scale, void* out, bool out_f32,
                                cudaStream_t stream) {
  if (mn & 3) return cudaErrorInvalidValue;
  const int threads = 256;
  const long long blocks = (mn / 4 + threads - 1) / threads;
  reduce_slabs_kernel<<<(unsigned)blocks, threads, 0, stream>>>(partial, slabs, mn, scale, out, out_f32 ? 1 : 0);
  count_launch();
  return cudaGetLastError();
}

}  // namespace gemm
}  // namespace tabattn
