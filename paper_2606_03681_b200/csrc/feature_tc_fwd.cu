// Feature-axis attention forward on tcgen05.  Packing, masking and
// the tile walk are described in feature_tc.cuh.
//
// Persistent, warp-specialised kernel, one CTA per SM (448 threads):
//   warps 0-3 / 4-7  softmax warpgroup of TMEM set 0 / 1 (tiles alternate between the sets): one thread per
//                    slot reads its W = max(Cp, 32) score columns from TMEM, base-2 softmax (no running
//                    maximum: a tile holds whole rows), writes P (bf16) back to TMEM; epilogue O / l -> bf16
//                    through a staging tile and one TMA store (unmasked) or 16-byte stores to the gathered
//                    columns (masked), LSE (natural log)
//   warps 8-11       producer: unmasked -> one lane issues three TMA boxes per tile (Q, K, V);
//                    masked -> all 128 lanes gather the valid cells with cp.async
//   warp 12          issuer of S = Q K^T + mask bias (SS MMAs, fp32 in TMEM); owns the TMEM allocation and
//                    rewrites the mask operands when the table geometry changes
//   warp 13          issuer of O = P V (A = P from TMEM, B = the V tile MN-major)
//   warps 14, 15     masked tables: zero-fill of the invalid columns (a6), whole cells, concurrently with the rest
// (warp numbers for dh <= 32, three softmax warpgroups; dh = 64 has two)
// TMEM: S0, S1 (128 columns each), P0, P1 (64 each: 128 bf16), O0, O1 (dh each).
#include <cuda.h>

#include <algorithm>

#include "feature_tc.cuh"
#include "kernels.h"

namespace tabattn {

namespace {

using namespace tc;
using namespace ftc;

// Warp roles.  NSETS softmax warpgroups (one per TMEM set), then four producer warps, the two MMA-issuing
// warps, padded to whole warpgroups (setmaxnreg is a warpgroup-wide instruction).
template <int DH>
struct FwdCfg {
  static constexpr int ROWB = DH * 2;
  static constexpr int TILE = kSlots * ROWB;          // bytes of one operand tile
  // TMEM set = S (128 columns; P, 128 bf16 = 64 columns, is written over it) + O (dh columns)
  static constexpr int NSETS = DH >= 64 ? 2 : 3;
  static constexpr int SET = 128 + DH, COLS = 512;
  static_assert(NSETS * SET <= COLS, "TMEM budget");
  static constexpr int SM_WARPS = 4 * NSETS;          // softmax warps
  static constexpr int PROD0 = SM_WARPS, SWARP = SM_WARPS + 4, PVWARP = SM_WARPS + 5;
  static constexpr int WARPS = (SM_WARPS + 7 + 3) / 4 * 4;   // (+ the zero-fill warp)
  static constexpr int THREADS = WARPS * 32;
  static constexpr int REG_OTHER = DH >= 64 ? 72 : 56;
  // register pool = THREADS x (launch allocation, 65536 / THREADS rounded down to 8); what the other warps
  // give up goes to the softmax warps
  static constexpr int REG_LAUNCH = (65536 / THREADS) / 8 * 8;
  static constexpr int REG_SOFTMAX =
      ((THREADS * REG_LAUNCH - (WARPS - SM_WARPS) * 32 * REG_OTHER) / (SM_WARPS * 32)) / 8 * 8;
  static constexpr int ST = DH >= 64 ? 3 : (DH == 32 ? 5 : 8);   // stage ring (Q, K, V per stage)
  static constexpr int STAGE = 3 * TILE;
  static constexpr int SMEM = ST * STAGE + 2 * NSETS * TILE + 2 * kMaskTile + 1024;   // + O staging (2 per set)
};

// ---- a0 prep (masked tables): per-table geometry, tile ranges, valid-column lists -------------------------
__global__ void __launch_bounds__(256) feature_prep_kernel(Shape s, FeatTab* __restrict__ tabs,
                                                           uint8_t* __restrict__ vcol, int32_t* __restrict__ total) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
  for (int b = warp; b < s.B; b += nw) {
    uint32_t m[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int c = 32 * k + lane;
      const bool v = c < s.C && __ldg(s.col_valid + (size_t)b * s.C + c) != 0;
      m[k] = __ballot_sync(0xffffffffu, v);
    }
    const int Cv = __popc(m[0]) + __popc(m[1]) + __popc(m[2]) + __popc(m[3]);
    int below = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int c = 32 * k + lane;
      if (c < s.C) {
        const uint32_t lt = m[k] & ((1u << lane) - 1u);
        const int vr = below + __popc(lt);           // valid columns before c
        const bool v = (m[k] >> lane) & 1u;
        vcol[(size_t)b * 128 + (v ? vr : Cv + (c - vr))] = (uint8_t)c;
      }
      below += __popc(m[k]);
    }
    if (lane == 0) {
      int lg = 4;
      while ((1 << lg) < Cv) ++lg;
      const int rpt = kSlots >> lg;
      tabs[b].Cv = Cv;
      tabs[b].lgCp = lg;
      tabs[b].tile0 = 0;
      // tile count, turned into a range below; a table without a valid column has none (its outputs are
      // zero-filled in the kernels' prologue)
      tabs[b].tile1 = Cv == 0 ? 0 : ((s.R + rpt - 1) / rpt) * s.H;
    }
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    int t = 0;
    for (int b = 0; b < s.B; ++b) {
      const int n = tabs[b].tile1;
      tabs[b].tile0 = t;
      t += n;
      tabs[b].tile1 = t;
    }
    *total = t;
  }
}

// Softmax of one slot over its W-column window, in 32-column chunks (two passes over TMEM at W > 32: maximum,
// then exponentials -- TMEM reads are cheap and the thread stays under ~100 registers).  P (bf16) is written
// over the set's own S columns: the thread's whole 64-column P row, zeros outside its window (the S MMA left
// scores there).  Before the first P store the thread drains the accumulator of the set's PREVIOUS tile
// (`drain`): that tile's P V MMA finished long ago (the S MMA of this tile was issued behind it), so its
// round trip is never waited for.
// `nlive`: chunks of the window that hold live keys, ceil(Cv / 32).  A W = 128 window of a table with Cv <= 96 has a
// whole chunk of masked keys, whose P is exactly zero: it is neither read nor exponentiated (feature_heavy: 65 % of
// the tiles are one-row Cp = 128 tiles and 8 of 9 of those have Cv <= 96).
template <int W, int DH>
__device__ __forceinline__ void softmax_window(uint32_t tSwin, uint32_t tProw, int pgrp0, int nlive, float c2,
                                               float& m_out, float& l_out, bool drain, uint32_t tO, uint32_t (&o)[DH]) {
  constexpr int NCH = W / 32;
  uint32_t sr[32];
  float mx0 = -INFINITY, mx1 = -INFINITY, mx2 = -INFINITY, mx3 = -INFINITY;
#pragma unroll
  for (int c = 0; c < NCH; ++c) {
    if (NCH > 2 && c >= nlive) continue;
    tmem_ld32(tSwin + 32 * c, sr);
    tmem_wait_ld();
    const float* sf = reinterpret_cast<const float*>(sr);
#pragma unroll
    for (int k = 0; k < 32; k += 8) {
      mx0 = fmax3(mx0, sf[k], sf[k + 1]);
      mx1 = fmax3(mx1, sf[k + 2], sf[k + 3]);
      mx2 = fmax3(mx2, sf[k + 4], sf[k + 5]);
      mx3 = fmax3(mx3, sf[k + 6], sf[k + 7]);
    }
  }
  // every slot sees at least one live key of its own block (bias 0), so the maximum is a real score
  const float m = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * c2;
  const uint64_t cc = f2pack(c2, c2), nm = f2pack(-m, -m);
  uint64_t la = 0, lb = 0;
  if (drain) {
    tmem_ld_cols<DH>(tO, o);   // (waits for the load)
  }
#pragma unroll
  for (int c = 0; c < NCH; ++c) {
    if (NCH > 2 && c >= nlive) {
      uint32_t z[16];
#pragma unroll
      for (int k = 0; k < 16; ++k) z[k] = 0u;
      tmem_st16(tProw + 16 * (pgrp0 + c), z);
      continue;
    }
    if (NCH > 1) {
      tmem_ld32(tSwin + 32 * c, sr);
      tmem_wait_ld();
    }
    const float* sf = reinterpret_cast<const float*>(sr);
    uint32_t p[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const uint64_t x = fma2(f2pack(sf[2 * k], sf[2 * k + 1]), cc, nm);
      float a, b;
      f2unpack(x, a, b);
      const float e0 = fast_exp2(a), e1 = fast_exp2(b);   // masked: 2^(-2^100 c2 - m) = 0
      if (k & 1) lb = add2(lb, f2pack(e0, e1)); else la = add2(la, f2pack(e0, e1));
      p[k] = pack_bf16(e0, e1);
    }
    // P chunk c -> columns [16 (pgrp0 + c), +16) of the P row: always at or below the S columns already read
    tmem_st16(tProw + 16 * (pgrp0 + c), p);
  }
  // zeros in the 16-column groups of the P row outside the window
  {
    uint32_t z[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) z[k] = 0u;
#pragma unroll
    for (int gq = 0; gq < 4; ++gq)
      if (gq < pgrp0 || gq >= pgrp0 + NCH) tmem_st16(tProw + 16 * gq, z);
  }
  float s0, s1;
  f2unpack(add2(la, lb), s0, s1);
  m_out = m;
  l_out = s0 + s1;
  tmem_wait_st();
  tc_fence_before();
}

template <int DH>
__global__ void __launch_bounds__(FwdCfg<DH>::THREADS, 1)
feature_fwd_tc_kernel(const __grid_constant__ CUtensorMap mapQ, const __grid_constant__ CUtensorMap mapK,
                      const __grid_constant__ CUtensorMap mapV, const __grid_constant__ CUtensorMap mapO,
                      const __grid_constant__ FeatParams p, const unsigned char* __restrict__ Q,
                      const unsigned char* __restrict__ K, const unsigned char* __restrict__ V,
                      unsigned char* __restrict__ O, float* __restrict__ LSE) {
  using Cfg = FwdCfg<DH>;
  constexpr int ST = Cfg::ST, TILE = Cfg::TILE, ROWB = Cfg::ROWB, STAGE = Cfg::STAGE, NSETS = Cfg::NSETS;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sStage = sbase;                         // [ST][Q, K, V][TILE]
  const uint32_t sOut = sStage + ST * STAGE;             // [NSETS][2][TILE]  O staging (unmasked)
  const uint32_t sMQ = sOut + 2 * NSETS * TILE, sMK = sMQ + kMaskTile;
  __shared__ uint64_t bar_full[ST], bar_empty[ST];
  __shared__ uint64_t bar_s_full[NSETS], bar_p_full[NSETS], bar_pv_done[NSETS];
  __shared__ uint32_t tmem_slot;
  const Shape& s = p.s;

  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;
  if (warp == Cfg::SWARP) tmem_alloc(smem_u32(&tmem_slot), Cfg::COLS);
  if (threadIdx.x == 0) {
    for (int i = 0; i < ST; ++i) {
      mbar_init(smem_u32(&bar_full[i]), p.masked ? 128 : 1);
      mbar_init(smem_u32(&bar_empty[i]), 1);
    }
    for (int i = 0; i < NSETS; ++i) {
      mbar_init(smem_u32(&bar_s_full[i]), 1);
      mbar_init(smem_u32(&bar_p_full[i]), 4);
      mbar_init(smem_u32(&bar_pv_done[i]), 1);
    }
    fence_barrier_init();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  const uint32_t d2 = (uint32_t)s.H * DH * 2;            // bytes per cell

  // Tile n of the CTA's walk (all tiles, also the zero-fill-only ones of tables without a valid column) belongs
  // to set n % NSETS; `use[g]` counts the compute tiles a set has seen (its mbarrier phases), `ns` the compute
  // tiles of the CTA (the stage ring).
  if (warp >= Cfg::SM_WARPS) {
    setmaxnreg_dec<Cfg::REG_OTHER>();
    if (warp < Cfg::SWARP) {
      // ---------------------------------------------------------------------------- producer
      TileWalk wk;
      Tile x;
      uint32_t ns = 0;
      if (!p.masked) {
        if (warp == Cfg::PROD0 && lane == 0) {
          tma_prefetch_desc(&mapQ);
          tma_prefetch_desc(&mapK);
          tma_prefetch_desc(&mapV);
          for (wk.init(p); wk.get(p, x); wk.next(p), ++ns) {
            const uint32_t st = ns % ST, full = smem_u32(&bar_full[st]), dst = sStage + st * STAGE;
            mbar_wait<true>(smem_u32(&bar_empty[st]), ((ns / ST) & 1) ^ 1);
            mbar_arrive_expect_tx(full, STAGE);
            tma_load_4d(dst, &mapQ, full, 0, x.h, 0, x.row0);
            tma_load_4d(dst + TILE, &mapK, full, 0, x.h, 0, x.row0);
            tma_load_4d(dst + 2 * TILE, &mapV, full, 0, x.h, 0, x.row0);
          }
        }
      } else {
        // gather: every lane issues its chunks of the three tiles, commits, and completes the PREVIOUS
        // stage (wait for its copies, make them visible to the tensor core, arrive)
        Gather<ROWB> ga;
        int cur_b = -1, pend = -1;
        for (wk.init(p); wk.get(p, x); wk.next(p)) {
          if (x.Cv == 0) continue;
          if (x.b != cur_b) {
            cur_b = x.b;
            ga.setup(p, x.b, x.Cv, x.lgCp, warp - Cfg::PROD0, lane);
          }
          const uint32_t st = ns % ST, dst = sStage + st * STAGE;
          mbar_wait<true>(smem_u32(&bar_empty[st]), ((ns / ST) & 1) ^ 1);
          const size_t g0 = ((size_t)x.b * s.R + x.row0) * s.C * d2 + (size_t)x.h * ROWB;
          ga.issue(dst, Q + g0, x.nrows);
          ga.issue(dst + TILE, K + g0, x.nrows);
          ga.issue(dst + 2 * TILE, V + g0, x.nrows);
          cp_async_commit();
          if (pend >= 0) {
            cp_async_wait<1>();
            fence_proxy_async_smem();
            mbar_arrive(smem_u32(&bar_full[pend]));
          }
          pend = (int)st;
          ++ns;
        }
        if (pend >= 0) {
          cp_async_wait<0>();
          fence_proxy_async_smem();
          mbar_arrive(smem_u32(&bar_full[pend]));
        }
      }
    } else if (warp == Cfg::SWARP) {
      // ---------------------------------------------------------------------------- S = Q K^T + bias
      constexpr uint32_t idS = make_idesc_bf16(128, 128, false, false);
      const uint64_t dQ = make_smem_desc<ROWB>(sStage, 16, 8 * ROWB);
      const uint64_t dK = make_smem_desc<ROWB>(sStage + TILE, 16, 8 * ROWB);
      const uint64_t dMQ = make_smem_desc<32>(sMQ, 16, 256), dMK = make_smem_desc<32>(sMK, 16, 256);
      TileWalk wk;
      Tile x;
      uint32_t ns = 0, g = 0, use[NSETS];
#pragma unroll
      for (int i = 0; i < NSETS; ++i) use[i] = 0;
      int geo = -1;
      uint32_t last_bar = 0, last_par = 0;
      for (wk.init(p); wk.get(p, x); wk.next(p), g = g + 1 == NSETS ? 0 : g + 1) {
        if (x.Cv == 0) continue;
        uint32_t k = 0;
#pragma unroll
        for (int i = 0; i < NSETS; ++i)
          if (g == (uint32_t)i) k = use[i]++;
        const uint32_t st = ns % ST;
        if (geo != (x.Cv << 4 | x.lgCp)) {
          // the mask operands change with the table geometry: wait until every MMA issued so far has
          // completed (they complete in order), then rewrite them
          if (ns > 0) mbar_wait(last_bar, last_par);
          write_mask_tiles(sMQ, sMK, x.lgCp, x.Cv, lane);
          geo = x.Cv << 4 | x.lgCp;
        }
        mbar_wait(smem_u32(&bar_full[st]), (ns / ST) & 1);
        // the set's previous P V MMA has read P (which lives in the S columns)
        if (k > 0) mbar_wait(smem_u32(&bar_pv_done[g]), (k - 1) & 1);
        tc_fence_after();
        const uint64_t qd = dQ + (uint64_t)((st * STAGE) >> 4), kd = dK + (uint64_t)((st * STAGE) >> 4);
        const uint32_t tS = tmem + Cfg::SET * g;
#pragma unroll
        for (int kk = 0; kk < DH / 16; ++kk) mma_ss_e(tS, qd + 2 * kk, kd + 2 * kk, idS, kk > 0);
        mma_ss_e(tS, dMQ, dMK, idS, 1u);
        last_bar = smem_u32(&bar_s_full[g]);
        last_par = k & 1;
        tc_commit_e(last_bar);
        ++ns;
      }
    } else if (warp > Cfg::PVWARP) {
      // ---------------------------------------------------------------------------- zero-fill of invalid columns (a6)
      unsigned char* const outs[1] = {O};
      zero_invalid_cells<1>(p, outs, LSE, lane, warp - Cfg::PVWARP - 1, Cfg::WARPS - Cfg::PVWARP - 1);
    } else if (warp == Cfg::PVWARP) {
      // ---------------------------------------------------------------------------- O = P V
      constexpr uint32_t idO = make_idesc_bf16(128, DH, false, true);
      const uint64_t dV = make_smem_desc<ROWB>(sStage + 2 * TILE, 16, 8 * ROWB);
      TileWalk wk;
      Tile x;
      uint32_t ns = 0, g = 0, use[NSETS];
#pragma unroll
      for (int i = 0; i < NSETS; ++i) use[i] = 0;
      for (wk.init(p); wk.get(p, x); wk.next(p), g = g + 1 == NSETS ? 0 : g + 1) {
        if (x.Cv == 0) continue;
        uint32_t k = 0;
#pragma unroll
        for (int i = 0; i < NSETS; ++i)
          if (g == (uint32_t)i) k = use[i]++;
        const uint32_t st = ns % ST;
        mbar_wait(smem_u32(&bar_full[st]), (ns / ST) & 1);
        mbar_wait(smem_u32(&bar_p_full[g]), k & 1);
        tc_fence_after();
        const uint64_t vd = dV + (uint64_t)((st * STAGE) >> 4);
        const uint32_t tP = tmem + Cfg::SET * g, tO = tP + 128;
#pragma unroll
        for (int kk = 0; kk < kSlots / 16; ++kk) mma_ts_e(tO, tP + 8 * kk, vd + kk * ROWB, idO, kk > 0);
        tc_commit_e(smem_u32(&bar_pv_done[g]));
        tc_commit_e(smem_u32(&bar_empty[st]));
        ++ns;
      }
    }
  } else {
    // ------------------------------------------------------------------------------ softmax warpgroups
    setmaxnreg_inc<Cfg::REG_SOFTMAX>();
    const int g = warp >> 2, wq = warp & 3;
    const int slot = threadIdx.x & 127;                    // = TMEM lane
    const uint32_t lane_base = tmem + ((uint32_t)(32 * wq) << 16) + Cfg::SET * g;
    const uint32_t tS = lane_base, tO = lane_base + 128;
    const uint32_t b_s_full = smem_u32(&bar_s_full[g]), b_p_full = smem_u32(&bar_p_full[g]),
                   b_pv_done = smem_u32(&bar_pv_done[g]);
    const float c2 = s.scale * kLog2e;
    {
      unsigned char* const outs[1] = {O};
      zero_dead_tables<1>(p, outs, LSE, threadIdx.x, Cfg::SM_WARPS * 32);
    }
    // per-thread constants of the staging path
    uint32_t st_off[DH / 8];
#pragma unroll
    for (int q = 0; q < DH / 8; ++q) st_off[q] = swz_off<ROWB>(slot, q);
    // the epilogue of a tile (accumulator -> O) is deferred: its accumulator is drained inside the NEXT tile's
    // softmax and stored after that tile's P has been handed to the tensor core
    bool pd_on = false, pd_live = false;
    float pd_inv = 0.f;
    int pd_h = 0, pd_col = 0;
    uint32_t pd_row = 0;                                   // global table row of the thread's slot / of the tile
    uint32_t o[DH];
    uint32_t n_store = 0;                                  // TMA stores issued by this warpgroup (staging parity)
    auto store_prev = [&]() {
      const uint64_t iv = f2pack(pd_inv, pd_inv);
      if (!p.masked) {
        // staging tile (double-buffered) -> one TMA store; columns >= C and rows beyond the tensor are clipped
        const uint32_t sO = sOut + (2 * g + (n_store & 1)) * TILE;
#pragma unroll
        for (int q = 0; q < DH / 8; ++q) {
          uint32_t u[4];
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            float a, b;
            f2unpack(mul2(f2pack(__uint_as_float(o[8 * q + 2 * e]), __uint_as_float(o[8 * q + 2 * e + 1])), iv), a, b);
            u[e] = pack_bf16(a, b);
          }
          sts_v4(sO + st_off[q], u[0], u[1], u[2], u[3]);
        }
        fence_proxy_async_smem();
        // the previous store (issued a tile ago) has read ITS staging tile, which the next tile reuses: waited
        // for BEFORE the barrier, so that every thread's next writes are ordered after it
        if (slot == 0) bulk_wait_read<0>();
        named_bar_sync(1 + g, 128);
        if (slot == 0) {
          tma_store_4d(&mapO, sO, 0, pd_h, 0, (int)pd_row);
          bulk_commit();
        }
        ++n_store;
      } else {
        // gathered columns: a quad of lanes stores one 64-byte group of a row per instruction (quad_transpose)
        const size_t off = ((size_t)pd_row * s.C + pd_col) * d2 + (size_t)pd_h * ROWB;
        uint4 u[DH / 8];
#pragma unroll
        for (int q = 0; q < DH / 8; ++q) {
          uint32_t* up = &u[q].x;
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            float a, b;
            f2unpack(mul2(f2pack(__uint_as_float(o[8 * q + 2 * e]), __uint_as_float(o[8 * q + 2 * e + 1])), iv), a, b);
            up[e] = pack_bf16(a, b);
          }
        }
        if constexpr (DH >= 32) {
          QuadRows qr;
          qr.init(off, pd_live, lane);
#pragma unroll
          for (int gq = 0; gq < DH / 32; ++gq) {
            uint4 t4[4] = {u[4 * gq], u[4 * gq + 1], u[4 * gq + 2], u[4 * gq + 3]};
            quad_transpose(t4, lane);
#pragma unroll
            for (int k4 = 0; k4 < 4; ++k4)
              if (qr.live[k4]) stg_v4(O + qr.off[k4] + 64 * gq, t4[k4]);
          }
        } else if (pd_live) {
#pragma unroll
          for (int q = 0; q < DH / 8; ++q) stg_v4(O + off + 16 * q, u[q]);
        }
      }
    };
    TileWalk wk;
    Tile x;
    uint32_t k = 0;                                        // compute tiles of this set so far
    int cur_b = -1, my_col = 0;
    for (wk.init(p, g, NSETS); wk.get(p, x); wk.next(p)) {
      const int Cp = 1 << x.lgCp;
      const int rl = slot >> x.lgCp, v = slot & (Cp - 1);
      const uint32_t grow0 = (uint32_t)x.b * p.Rt + x.row0;   // first table row of the tile, global (< 2^31)
      if (p.masked) {
        if (x.Cv == 0) continue;
        if (x.b != cur_b) {
          cur_b = x.b;
          my_col = v < x.Cv ? __ldg(p.vcol + (size_t)x.b * 128 + v) : 0;
        }
      } else {
        my_col = v;
      }
      // the thread's window: its own block, or (Cp = 16) the two blocks of its warp
      const int colbase = x.lgCp >= 5 ? (((32 * wq) >> x.lgCp) << x.lgCp) : 32 * wq;
      mbar_wait(b_s_full, k & 1);
      // the S MMA of this tile was issued behind the previous tile's P V MMA: the accumulator is ready
      tc_fence_after();
      float m, l;
      const int nlive = (x.Cv + 31) >> 5;
      if (x.lgCp <= 5) softmax_window<32, DH>(tS + colbase, tS, colbase >> 5, nlive, c2, m, l, pd_on, tO, o);
      else if (x.lgCp == 6) softmax_window<64, DH>(tS + colbase, tS, colbase >> 5, nlive, c2, m, l, pd_on, tO, o);
      else softmax_window<128, DH>(tS + colbase, tS, colbase >> 5, nlive, c2, m, l, pd_on, tO, o);
      __syncwarp();
      if (lane == 0) mbar_arrive(b_p_full);
      if (pd_on) store_prev();
      // ---- this tile: LSE = (m + log2 l) ln 2 now, O = acc / l deferred
      const bool live = rl < x.nrows && v < x.Cv;
      if (live && LSE) LSE[((size_t)(grow0 + rl) * s.H + x.h) * s.C + my_col] = (m + log2f(l)) * kLn2;
      pd_on = true; pd_live = live; pd_inv = 1.f / l; pd_h = x.h; pd_col = my_col;
      pd_row = p.masked ? grow0 + rl : grow0;
      ++k;
    }
    if (pd_on) {
      mbar_wait(b_pv_done, (k - 1) & 1);
      tc_fence_after();
      tmem_ld_cols<DH>(tO, o);
      tc_fence_before();
      store_prev();
    }
    if (!p.masked && slot == 0) bulk_wait_read<0>();
  }
  tc_fence_before();
  __syncthreads();
  if (warp == Cfg::SWARP) tmem_dealloc(tmem, Cfg::COLS);
}

int ceil_log2_min16(int c) {
  int lg = 4;
  while ((1 << lg) < c) ++lg;
  return lg;
}

}  // namespace

// Geometry of one feature call.  Unmasked: one virtual table of B*R rows.  Masked: the a0 prep kernel builds the
// per-table records in the workspace.  `lg` = log2 of the slots per row the TMA boxes are built for (unmasked).
void feature_fill_params(const Shape& s, void* ws, cudaStream_t stream, ftc::FeatParams* pp, long long* max_tiles,
                         int* lg_out) {
  ftc::FeatParams& p = *pp;
  p = ftc::FeatParams{};
  p.s = s;
  p.masked = s.col_valid != nullptr;
  int lg = ceil_log2_min16(s.C);
  if (p.masked) {
    p.nTab = s.B;
    p.Rt = s.R;
    ftc::FeatTab* tabs = static_cast<ftc::FeatTab*>(ws);
    uint8_t* vcol = reinterpret_cast<uint8_t*>(tabs + s.B);
    int32_t* total = reinterpret_cast<int32_t*>(vcol + (size_t)s.B * 128);
    p.tabs = tabs; p.vcol = vcol; p.total = total;
    feature_prep_kernel<<<1, 256, 0, stream>>>(s, tabs, vcol, total);
    count_launch();
    *max_tiles = (long long)s.B * s.R * s.H;    // upper bound (Cp = 128: one row per tile)
    lg = 7;                                     // (tensor maps unused)
  } else {
    const int rpt = ftc::kSlots >> lg;
    const long long rows = (long long)s.B * s.R;
    p.nTab = 1;
    p.Rt = (int)rows;
    p.n_tiles = (int)(((rows + rpt - 1) / rpt) * s.H);
    p.uni.Cv = s.C; p.uni.lgCp = lg; p.uni.tile0 = 0; p.uni.tile1 = p.n_tiles;
    *max_tiles = p.n_tiles;
  }
  *lg_out = lg;
}

namespace {

template <int DH>
cudaError_t launch_fwd(const Shape& s, const void* Q, const void* K, const void* V, void* O, float* LSE, void* ws,
                       cudaStream_t stream) {
  using Cfg = FwdCfg<DH>;
  const DeviceInfo* di = current_device();
  if (!di) return cudaErrorInvalidDevice;
  FeatParams p{};
  long long max_tiles;
  int lg;
  feature_fill_params(s, ws, stream, &p, &max_tiles, &lg);
  CUtensorMap mq, mk, mv, mo;
  const int rpt = kSlots >> lg;
  if (!get_tensor_map(&mq, 1, Q, s.B, s.R, s.C, s.H, DH, rpt, 1 << lg) ||
      !get_tensor_map(&mk, 1, K, s.B, s.R, s.C, s.H, DH, rpt, 1 << lg) ||
      !get_tensor_map(&mv, 1, V, s.B, s.R, s.C, s.H, DH, rpt, 1 << lg) ||
      !get_tensor_map(&mo, 1, O, s.B, s.R, s.C, s.H, DH, rpt, 1 << lg))
    return cudaErrorInvalidValue;
  auto kern = feature_fwd_tc_kernel<DH>;
  static SmemAttr attr;
  cudaError_t e = attr.ensure(kern, Cfg::SMEM, di->ordinal);
  if (e != cudaSuccess) return e;
  const int grid = (int)std::min<long long>(max_tiles, di->num_sms);
  kern<<<grid, Cfg::THREADS, Cfg::SMEM, stream>>>(mq, mk, mv, mo, p, (const unsigned char*)Q, (const unsigned char*)K,
                                                 (const unsigned char*)V, (unsigned char*)O, LSE);
  count_launch();
  return cudaGetLastError();
}

}  // namespace

// bytes per table: FeatTab + vcol[128] + the tile total, so that a call on ONE table (the row-range inference path
// launches per table) can use its own aligned slice of the same workspace
constexpr size_t kFeatureWsPerTable = sizeof(ftc::FeatTab) + 128 + 16;

size_t feature_workspace_bytes(const Shape& s) {
  // FeatTab[B] + vcol[B][128] + total, for masked calls (sized without looking at col_valid, so that one
  // workspace serves both)
  return (size_t)s.B * kFeatureWsPerTable;
}

bool feature_shape_supported(const Shape& s) { return s.C <= 128; }

// Forward-only inference on the table rows [row0, row1): feature attention treats every row
// alone, so a row range is the same kernel on a sub-tensor -- one launch per table (the range of table b starts
// (b R + row0) C d elements into the tensors); the whole range is one launch.  No LSE.
cudaError_t launch_feature_fwd_infer(const Shape& s, const void* Q, const void* K, const void* V, void* O, int row0,
                                     int row1, void* ws, cudaStream_t stream) {
  if (row0 == 0 && row1 == s.R) return launch_feature_fwd(s, Q, K, V, O, nullptr, ws, stream);
  const size_t cell = (size_t)s.C * s.H * s.dh * 2;
  for (int b = 0; b < s.B; ++b) {
    Shape t = s;
    t.B = 1;
    t.R = row1 - row0;
    if (s.col_valid) t.col_valid = s.col_valid + (size_t)b * s.C;
    const size_t off = ((size_t)b * s.R + row0) * cell;
    cudaError_t e = launch_feature_fwd(t, (const char*)Q + off, (const char*)K + off, (const char*)V + off,
                                       (char*)O + off, nullptr, ws ? (char*)ws + b * kFeatureWsPerTable : nullptr,
                                       stream);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

cudaError_t launch_feature_fwd(const Shape& s, const void* Q, const void* K, const void* V, void* O, float* LSE,
                               void* ws, cudaStream_t stream) {
  switch (s.dh) {
    case 16: return launch_fwd<16>(s, Q, K, V, O, LSE, ws, stream);
    case 32: return launch_fwd<32>(s, Q, K, V, O, LSE, ws, stream);
    case 64: return launch_fwd<64>(s, Q, K, V, O, LSE, ws, stream);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace tabattn
