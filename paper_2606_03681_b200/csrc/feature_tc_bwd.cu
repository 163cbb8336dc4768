// Feature-axis attention backward on tcgen05.  Packing, masking and the
// tile walk are described in feature_tc.cuh; a tile is 128 slots = RPT whole table rows of one head.
//
// Per tile, with P recomputed from the saved LSE (whole rows sit in one tile, so no pass is split):
//   S  = Q K^T + mask bias           SS MMA, fp32 in TMEM
//   P  = 2^(S c2 - LSE log2e)        softmax thread i (one slot = one TMEM lane), W-column window
//   dP = dO V^T                      SS MMA into the SAME TMEM columns once every thread has read S
//   D  = sum_j P_ij dP_ij            the definition itself -- O is not read at all
//   dS = P o (dP - D)
//   P, dS -> shared memory as bf16 [128 i][128 j] (two 64-column halves of 128-byte swizzled rows): the same
//            bytes are the K-major A operand of dQ = dS K and the MN-major A operand of dV = P^T dO, dK = dS^T Q
//   dQ, dK, dV accumulate in the set's TMEM columns (S / dP are dead by then), are drained by the softmax
//   threads, scaled, rounded to bf16 and stored.
// One P/dS buffer serves all sets: tiles take it in order (a tile waits for the accumulation MMAs of the
// compute tile before it, on that tile's set).
//
// Warp roles (one persistent CTA per SM): NSETS softmax warpgroups (3 at dh <= 32, 2 at dh = 64), four producer
// warps (unmasked: one lane issues four TMA boxes per tile; masked: cp.async gather of the valid cells), and
// three MMA-issuing warps (S, dP, accumulation).  No atomics: every output element has one writer.
#include <cuda.h>

#include <algorithm>
#include <type_traits>

#include "feature_tc.cuh"
#include "kernels.h"

namespace tabattn {

TABATTN_TRACE_DEFINE(tabattn_debug_set_trace)

namespace {

using namespace tc;
using namespace ftc;

template <int DH>
struct BwdCfg {
  static constexpr int ROWB = DH * 2;
  static constexpr int TILE = kSlots * ROWB;
  static constexpr int NSETS = DH >= 64 ? 2 : 3;
  static constexpr int SET = DH >= 64 ? 192 : 128;     // S / dP (128 columns), then dQ | dK | dV (3 dh columns)
  static constexpr int COLS = 512;
  static_assert(NSETS * SET <= COLS && 3 * DH <= SET, "TMEM budget");
  static constexpr int SM_WARPS = 4 * NSETS;
  static constexpr int PROD0 = SM_WARPS, SWARP = SM_WARPS + 4, DPWARP = SM_WARPS + 5, ACCWARP = SM_WARPS + 6;
  static constexpr int ZWARP = SM_WARPS + 7;                 // zero-fill of invalid columns (masked tables)
  static constexpr int WARPS = (SM_WARPS + 8 + 3) / 4 * 4;
  static constexpr int THREADS = WARPS * 32;
  static constexpr int REG_OTHER = DH >= 64 ? 72 : 48;
  static constexpr int REG_LAUNCH = (65536 / THREADS) / 8 * 8;
  static constexpr int REG_SOFTMAX =
      ((THREADS * REG_LAUNCH - (WARPS - SM_WARPS) * 32 * REG_OTHER) / (SM_WARPS * 32)) / 8 * 8;
  static constexpr int NIN = 4;                        // Q, K, V, dO
  static constexpr int STAGE = NIN * TILE;
  static constexpr int ST = DH >= 64 ? 2 : (DH == 32 ? 4 : 6);
  static constexpr int NLW = ST < 3 ? ST : 3;          // LSE-staging warps (unmasked tables)
  static constexpr int PDS = 2 * kSlots * 256;         // P and dS: [128][128] bf16 each
  static constexpr int SMEM = ST * STAGE + PDS + 2 * kMaskTile + 1024;
};

// shared-memory byte offset of the 16-byte chunk holding columns [8 cj, 8 cj + 8) of row i in a [128][128] bf16
// matrix stored as two halves of [128][64] with 128-byte swizzled rows
__device__ __forceinline__ uint32_t pds_off(int i, int cj) {
  return (uint32_t)(cj >> 3) * (kSlots * 128) + (uint32_t)i * 128 + (uint32_t)(((cj & 7) ^ (i & 7)) << 4);
}

template <int DH>
__global__ void __launch_bounds__(BwdCfg<DH>::THREADS, 1)
feature_bwd_tc_kernel(const __grid_constant__ CUtensorMap mapQ, const __grid_constant__ CUtensorMap mapK,
                      const __grid_constant__ CUtensorMap mapV, const __grid_constant__ CUtensorMap mapG,
                      const __grid_constant__ FeatParams p, const unsigned char* __restrict__ Q,
                      const unsigned char* __restrict__ K, const unsigned char* __restrict__ V,
                      const unsigned char* __restrict__ dO, const float* __restrict__ LSE,
                      unsigned char* __restrict__ dQ, unsigned char* __restrict__ dK, unsigned char* __restrict__ dV) {
  TR_INIT();
  using Cfg = BwdCfg<DH>;
  constexpr int ST = Cfg::ST, TILE = Cfg::TILE, ROWB = Cfg::ROWB, STAGE = Cfg::STAGE, NSETS = Cfg::NSETS;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sStage = sbase;                         // [ST][Q, K, V, dO][TILE]
  const uint32_t sP = sStage + ST * STAGE;               // [2 halves][128][128 B]
  const uint32_t sDS = sP + kSlots * 256;
  const uint32_t sMQ = sDS + kSlots * 256, sMK = sMQ + kMaskTile;
  __shared__ uint64_t bar_full[ST], bar_empty[ST];
  __shared__ uint64_t bar_s_full[NSETS], bar_s_taken[NSETS], bar_dp_full[NSETS], bar_pds_full[NSETS],
      bar_acc_full[NSETS], bar_acc_free[NSETS];
  __shared__ uint32_t tmem_slot;
  // -LSE log2(e) of every slot of a staged tile (+inf -> P = 0 for dead slots), written by the producer warps with
  // the tile: the softmax threads used to fetch it themselves one tile ahead, which cost them a register they
  // did not have (the value was spilled right behind the load: 19 % of their time, profiles/r02_attention.md)
  __shared__ float sNL2[ST][kSlots];
  const Shape& s = p.s;

  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;
  if (warp == Cfg::SWARP) tmem_alloc(smem_u32(&tmem_slot), Cfg::COLS);
  if (threadIdx.x == 0) {
    for (int i = 0; i < ST; ++i) {
      mbar_init(smem_u32(&bar_full[i]), p.masked ? 128 : 2);   // unmasked: the TMA lane + the tile's LSE warp
      mbar_init(smem_u32(&bar_empty[i]), 1);
    }
    for (int i = 0; i < NSETS; ++i) {
      mbar_init(smem_u32(&bar_s_full[i]), 1);
      mbar_init(smem_u32(&bar_s_taken[i]), 4);
      mbar_init(smem_u32(&bar_dp_full[i]), 1);
      mbar_init(smem_u32(&bar_pds_full[i]), 4);
      mbar_init(smem_u32(&bar_acc_full[i]), 1);
      mbar_init(smem_u32(&bar_acc_free[i]), 4);
    }
    fence_barrier_init();
  }
  // the P / dS matrices start as zeros (threads only ever write their windows, see below)
  for (uint32_t a = sP + 16 * threadIdx.x; a < sP + Cfg::PDS; a += 16 * blockDim.x) sts_v4(a, 0u, 0u, 0u, 0u);
  fence_proxy_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  const uint32_t d2 = (uint32_t)s.H * DH * 2;            // bytes per cell

  // Tile n of the CTA's walk (compute tiles only: dead tables have none) belongs to set n % NSETS and is that
  // set's use n / NSETS (the mbarrier phases); stage = n % ST.
  if (warp >= Cfg::SM_WARPS) {
    setmaxnreg_dec<Cfg::REG_OTHER>();
    if (warp < Cfg::SWARP) {
      // ---------------------------------------------------------------------------- producer
      TileWalk wk;
      Tile x;
      uint32_t n = 0;
      if (!p.masked) {
        if (warp == Cfg::PROD0 && lane == 0) {
          tma_prefetch_desc(&mapQ);
          tma_prefetch_desc(&mapK);
          tma_prefetch_desc(&mapV);
          tma_prefetch_desc(&mapG);
          for (wk.init(p); wk.get(p, x); wk.next(p), ++n) {
            const uint32_t st = n % ST, full = smem_u32(&bar_full[st]), dst = sStage + st * STAGE;
            mbar_wait<true>(smem_u32(&bar_empty[st]), ((n / ST) & 1) ^ 1);
            mbar_arrive_expect_tx(full, STAGE);
            TR(0, n);                                     // TMA issued
            tma_load_4d(dst, &mapQ, full, 0, x.h, 0, x.row0);
            tma_load_4d(dst + TILE, &mapK, full, 0, x.h, 0, x.row0);
            tma_load_4d(dst + 2 * TILE, &mapV, full, 0, x.h, 0, x.row0);
            tma_load_4d(dst + 3 * TILE, &mapG, full, 0, x.h, 0, x.row0);
          }
        } else if (warp > Cfg::PROD0 && warp <= Cfg::PROD0 + Cfg::NLW) {
          // LSE of the tiles n = j, j + NLW, ... (one of the other producer warps each), four slots per lane, fetched
          // one own tile ahead of the stage wait.  NLW <= ST: a warp that strides further than the ring is deep
          // could be two phases ahead of a stage's mbarrier, which a parity wait cannot tell from none.
          constexpr int NLW = Cfg::NLW;
          const int j = warp - Cfg::PROD0 - 1;
          const int lg = p.uni.lgCp, Cv = p.uni.Cv, cm = (1 << lg) - 1;
          float cur[4];
          auto fetch = [&](const Tile& y, float (&v)[4]) {
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              const int slot = lane + 32 * q, rl = slot >> lg, c = slot & cm;
              v[q] = (rl < y.nrows && c < Cv)
                         ? __ldg(LSE + ((size_t)(y.row0 + rl) * s.H + y.h) * s.C + c) : INFINITY;
            }
          };
          wk.init(p, j, NLW);
          bool have = wk.get(p, x);
          if (have) fetch(x, cur);
          for (n = j; have; n += NLW) {
            float nxt[4] = {INFINITY, INFINITY, INFINITY, INFINITY};
            wk.next(p);
            Tile y;
            have = wk.get(p, y);
            if (have) fetch(y, nxt);
            const uint32_t st = n % ST;
            mbar_wait<true>(smem_u32(&bar_empty[st]), ((n / ST) & 1) ^ 1);
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              sNL2[st][lane + 32 * q] = -cur[q] * kLog2e;
              cur[q] = nxt[q];
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&bar_full[st]));
          }
        }
      } else {
        Gather<ROWB> ga;
        int cur_b = -1, pend = -1;
        float pend_lse = INFINITY;
        for (wk.init(p); wk.get(p, x); wk.next(p), ++n) {
          if (x.b != cur_b) {
            cur_b = x.b;
            ga.setup(p, x.b, x.Cv, x.lgCp, warp - Cfg::PROD0, lane);
          }
          const uint32_t st = n % ST, dst = sStage + st * STAGE;
          mbar_wait<true>(smem_u32(&bar_empty[st]), ((n / ST) & 1) ^ 1);
          const size_t g0 = ((size_t)x.b * s.R + x.row0) * s.C * d2 + (size_t)x.h * ROWB;
          ga.issue(dst, Q + g0, x.nrows);
          ga.issue(dst + TILE, K + g0, x.nrows);
          ga.issue(dst + 2 * TILE, V + g0, x.nrows);
          ga.issue(dst + 3 * TILE, dO + g0, x.nrows);
          cp_async_commit();
          // the LSE of this lane's slot of the tile (stored when the stage is completed, an iteration later)
          const int slot = (warp - Cfg::PROD0) * 32 + lane, rl = slot >> x.lgCp, v = slot & ((1 << x.lgCp) - 1);
          float lse = INFINITY;
          if (rl < x.nrows && v < x.Cv)
            lse = __ldg(LSE + ((size_t)((size_t)x.b * s.R + x.row0 + rl) * s.H + x.h) * s.C +
                        __ldg(p.vcol + (size_t)x.b * 128 + v));
          if (pend >= 0) {
            sNL2[pend][slot] = -pend_lse * kLog2e;
            cp_async_wait<1>();
            fence_proxy_async_smem();
            mbar_arrive(smem_u32(&bar_full[pend]));
          }
          pend = (int)st;
          pend_lse = lse;
        }
        if (pend >= 0) {
          sNL2[pend][(warp - Cfg::PROD0) * 32 + lane] = -pend_lse * kLog2e;
          cp_async_wait<0>();
          fence_proxy_async_smem();
          mbar_arrive(smem_u32(&bar_full[pend]));
        }
      }
    } else if (warp == Cfg::SWARP || warp == Cfg::DPWARP) {
      // ---------------------------------------------------------------------------- S = Q K^T + bias | dP = dO V^T
      const bool is_s = warp == Cfg::SWARP;
      constexpr uint32_t idS = make_idesc_bf16(128, 128, false, false);
      // A: Q (tile 0) or dO (tile 3); B: K (tile 1) or V (tile 2)
      const uint64_t dA = make_smem_desc<ROWB>(sStage + (is_s ? 0 : 3 * TILE), 16, 8 * ROWB);
      const uint64_t dB = make_smem_desc<ROWB>(sStage + (is_s ? TILE : 2 * TILE), 16, 8 * ROWB);
      const uint64_t dMQ = make_smem_desc<32>(sMQ, 16, 256), dMK = make_smem_desc<32>(sMK, 16, 256);
      TileWalk wk;
      Tile x;
      uint32_t n = 0, g = 0, k = 0;
      int geo = -1;
      uint32_t last_bar = 0, last_par = 0;
      for (wk.init(p); wk.get(p, x); wk.next(p), ++n) {
        const uint32_t st = n % ST;
        const uint64_t ad = dA + (uint64_t)((st * STAGE) >> 4), bd = dB + (uint64_t)((st * STAGE) >> 4);
        const uint32_t tS = tmem + Cfg::SET * g;
        if (is_s) {
          if (geo != (x.Cv << 4 | x.lgCp)) {
            // new table geometry: every MMA issued so far has completed (in order) before the mask operands change
            if (n > 0) mbar_wait(last_bar, last_par);
            write_mask_tiles(sMQ, sMK, x.lgCp, x.Cv, lane);
            geo = x.Cv << 4 | x.lgCp;
          }
          mbar_wait(smem_u32(&bar_full[st]), (n / ST) & 1);
          if (k > 0) mbar_wait(smem_u32(&bar_acc_free[g]), (k - 1) & 1);   // the set's accumulators were drained
          tc_fence_after();
#pragma unroll
          for (int kk = 0; kk < DH / 16; ++kk) mma_ss_e(tS, ad + 2 * kk, bd + 2 * kk, idS, kk > 0);
          mma_ss_e(tS, dMQ, dMK, idS, 1u);
          last_bar = smem_u32(&bar_s_full[g]);
          last_par = k & 1;
          tc_commit_e(last_bar);
          if (lane == 0) TR(1, n);                      // S MMAs issued
        } else {
          mbar_wait(smem_u32(&bar_full[st]), (n / ST) & 1);
          mbar_wait(smem_u32(&bar_s_taken[g]), k & 1);                     // every thread has read its S window
          tc_fence_after();
#pragma unroll
          for (int kk = 0; kk < DH / 16; ++kk) mma_ss_e(tS, ad + 2 * kk, bd + 2 * kk, idS, kk > 0);
          tc_commit_e(smem_u32(&bar_dp_full[g]));
          if (lane == 0) TR(2, n);                      // dP MMAs issued
        }
        if (++g == NSETS) { g = 0; ++k; }
      }
    } else if (warp >= Cfg::ZWARP) {
      // ---------------------------------------------------------------------------- zero-fill of invalid columns (a6)
      unsigned char* const outs[3] = {dQ, dK, dV};
      zero_invalid_cells<3>(p, outs, nullptr, lane, warp - Cfg::ZWARP, Cfg::WARPS - Cfg::ZWARP);
    } else if (warp == Cfg::ACCWARP) {
      // ---------------------------------------------------------------------------- dQ = dS K, dK = dS^T Q, dV = P^T dO
      constexpr uint32_t idQ = make_idesc_bf16(128, DH, false, true);   // A K-major, B MN-major
      constexpr uint32_t idT = make_idesc_bf16(128, DH, true, true);    // A MN-major (transposed), B MN-major
      // B operands: the K, Q, dO tiles read as [k = slot][n = dh]
      const uint64_t bK = make_smem_desc<ROWB>(sStage + TILE, 16, 8 * ROWB);
      const uint64_t bQ = make_smem_desc<ROWB>(sStage, 16, 8 * ROWB);
      const uint64_t bG = make_smem_desc<ROWB>(sStage + 3 * TILE, 16, 8 * ROWB);
      // A operands.  K-major dS: k-steps 0-3 in half 0, 4-7 in half 1, 32 bytes per step inside the 128-byte rows.
      const uint64_t aDS = make_smem_desc<128>(sDS, 16, 1024);
      // MN-major P / dS (M = key j across the two halves: LBO = one half; K = query i, 8 rows = 1024 bytes)
      const uint64_t aPT = make_smem_desc<128>(sP, kSlots * 128, 1024);
      const uint64_t aDST = make_smem_desc<128>(sDS, kSlots * 128, 1024);
      TileWalk wk;
      Tile x;
      uint32_t n = 0, g = 0, k = 0;
      for (wk.init(p); wk.get(p, x); wk.next(p), ++n) {
        const uint32_t st = n % ST;
        mbar_wait(smem_u32(&bar_pds_full[g]), k & 1);
        if (lane == 0) TR(3, n);                        // accumulation warp has P/dS
        tc_fence_after();
        const uint64_t so = (uint64_t)((st * STAGE) >> 4);
        const uint32_t tA = tmem + Cfg::SET * g;
#pragma unroll
        for (int kk = 0; kk < 8; ++kk)
          mma_ss_e(tA, aDS + (uint64_t)((kk >> 2) * (kSlots * 128 >> 4) + 2 * (kk & 3)), bK + so + kk * ROWB, idQ, kk > 0);
#pragma unroll
        for (int kk = 0; kk < 8; ++kk)
          mma_ss_e(tA + DH, aDST + (uint64_t)(kk * (16 * 128 >> 4)), bQ + so + kk * ROWB, idT, kk > 0);
#pragma unroll
        for (int kk = 0; kk < 8; ++kk)
          mma_ss_e(tA + 2 * DH, aPT + (uint64_t)(kk * (16 * 128 >> 4)), bG + so + kk * ROWB, idT, kk > 0);
        tc_commit_e(smem_u32(&bar_acc_full[g]));
        if (lane == 0) TR(4, n);                        // accumulation MMAs issued
        tc_commit_e(smem_u32(&bar_empty[st]));
        if (++g == NSETS) { g = 0; ++k; }
      }
    }
  } else {
    // ------------------------------------------------------------------------------ softmax warpgroups
    setmaxnreg_inc<Cfg::REG_SOFTMAX>();
    const int g = warp >> 2, wq = warp & 3;
    const int slot = threadIdx.x & 127;                    // = TMEM lane
    const uint32_t lane_off = (uint32_t)(32 * wq) << 16;
    const uint32_t tS = tmem + lane_off + Cfg::SET * g;
    // W = 128 parks the upper half of its packed P (32 columns) in spare TMEM columns behind the sets
    const uint32_t tScr = tmem + lane_off + NSETS * Cfg::SET + 32 * g;
    static_assert(NSETS * Cfg::SET + 32 * NSETS <= Cfg::COLS, "TMEM scratch");
    const uint32_t b_s_full = smem_u32(&bar_s_full[g]), b_s_taken = smem_u32(&bar_s_taken[g]),
                   b_dp_full = smem_u32(&bar_dp_full[g]), b_pds_full = smem_u32(&bar_pds_full[g]),
                   b_acc_full = smem_u32(&bar_acc_full[g]), b_acc_free = smem_u32(&bar_acc_free[g]);
    // P/dS turn: the tile before this set's tile n is in set g - 1 (same use) or, for set 0, in the last set
    // (previous use); the buffer is free once THAT tile's accumulation MMAs have completed
    const uint32_t b_turn = smem_u32(&bar_acc_full[g == 0 ? NSETS - 1 : g - 1]);
    const float c2 = s.scale * kLog2e;
    {
      unsigned char* const outs[3] = {dQ, dK, dV};
      zero_dead_tables<3>(p, outs, nullptr, threadIdx.x, Cfg::SM_WARPS * 32);
    }
    TileWalk wk;
    Tile x;
    uint32_t k = 0;            // this set's tiles so far (= use index)
    int cur_b = -1, my_col = 0;
    for (wk.init(p, g, NSETS); wk.get(p, x); wk.next(p), ++k) {
      const int Cp = 1 << x.lgCp;
      const int rl = slot >> x.lgCp, v = slot & (Cp - 1);
      const uint32_t grow0 = (uint32_t)x.b * p.Rt + x.row0;
      const uint32_t n = k * NSETS + g, st = n % ST;        // the tile's place in the CTA's walk, its stage
      int old_lg = x.lgCp;    // geometry the P/dS rows were last written with (the CTA's previous tile)
      if (p.masked) {
        if (x.b != cur_b) {
          cur_b = x.b;
          my_col = v < x.Cv ? __ldg(p.vcol + (size_t)x.b * 128 + v) : 0;
        }
        old_lg = lgcp_of_earlier_tile(p, wk.tb, wk.b, wk.t, (int)gridDim.x);
      } else {
        my_col = v;
      }
      const bool live = rl < x.nrows && v < x.Cv;
      // the thread's window: its own block, or (Cp = 16) the two blocks of its warp
      const int colbase = x.lgCp >= 5 ? (((32 * wq) >> x.lgCp) << x.lgCp) : 32 * wq;
      const uint64_t cc = f2pack(c2, c2);
      const bool first_tile = g == 0 && k == 0;

      auto body = [&](auto WC) {
        // W = 96: a Cp = 128 window whose last 32 columns are masked keys only (Cv <= 96; P = dS = 0 there exactly):
        // three chunks are computed and the fourth is stored as zeros.  Its own instantiation, so that the loops keep
        // compile-time bounds (a run-time chunk count in the W = 128 body spilled 104 bytes and lost 5-8 %).
        constexpr int W = decltype(WC)::value, NCH = W / 32;
        constexpr int NREG = NCH > 2 ? 2 : NCH;            // chunks of packed P kept in registers
        uint32_t pp[16 * NREG];
        // ---- pass A: P = 2^(S c2 - LSE log2e), packed bf16 pairs
        mbar_wait(b_s_full, k & 1);
        if (wq == 0 && lane == 0) TR(5, k * NSETS + g);   // softmax: S ready
        tc_fence_after();
        // -LSE log2(e) of the slot, staged with the tile (the stage's barrier completed before the S MMA was issued;
        // waiting on it here is what makes the producers' stores visible to this thread)
        mbar_wait(smem_u32(&bar_full[st]), (n / ST) & 1);
        const float nl2 = sNL2[st][slot];
        const uint64_t nl = f2pack(nl2, nl2);
#pragma unroll
        for (int c = 0; c < NCH; ++c) {
          uint32_t sr[32], pk[16];
          tmem_ld32(tS + colbase + 32 * c, sr);
          tmem_wait_ld();
#pragma unroll
          for (int q = 0; q < 16; ++q) {
            const uint64_t xx = fma2(f2pack(__uint_as_float(sr[2 * q]), __uint_as_float(sr[2 * q + 1])), cc, nl);
            float a, b;
            f2unpack(xx, a, b);
            pk[q] = pack_bf16(fast_exp2(a), fast_exp2(b));
          }
          if (c < NREG) {
#pragma unroll
            for (int q = 0; q < 16; ++q) pp[16 * c + q] = pk[q];
          } else {
            tmem_st16(tScr + 16 * (c - NREG), pk);
          }
        }
        if (NCH > NREG) tmem_wait_st();
        tc_fence_before();
        __syncwarp();
        if (wq == 0 && lane == 0) TR(6, k * NSETS + g);   // pass A done
        if (lane == 0) mbar_arrive(b_s_taken);
        // packed P of chunk c (registers or the TMEM scratch)
        auto p_chunk = [&](int c, uint32_t (&pk)[16]) {
          if (c < NREG) {
#pragma unroll
            for (int q = 0; q < 16; ++q) pk[q] = pp[16 * c + q];
          } else {
            tmem_ld16(tScr + 16 * (c - NREG), pk);
            tmem_wait_ld();
          }
        };
        // ---- pass B: D = sum P dP, then dS = P (dP - D), from the bf16-rounded P (the value the dV MMA uses)
        mbar_wait(b_dp_full, k & 1);
        if (wq == 0 && lane == 0) TR(7, k * NSETS + g);   // dP ready
        tc_fence_after();
        uint64_t dacc = 0;
        uint32_t dr[32];
#pragma unroll
        for (int c = 0; c < NCH; ++c) {
          uint32_t pk[16];
          p_chunk(c, pk);
          tmem_ld32(tS + colbase + 32 * c, dr);
          tmem_wait_ld();
#pragma unroll
          for (int q = 0; q < 16; ++q)
            dacc = fma2(f2pack(bf16lo(pk[q]), bf16hi(pk[q])),
                        f2pack(__uint_as_float(dr[2 * q]), __uint_as_float(dr[2 * q + 1])), dacc);
        }
        float d0, d1;
        f2unpack(dacc, d0, d1);
        const float D = d0 + d1;
        const uint64_t dd = f2pack(D, D);
        // dS = P (dP - D) of one chunk (dr = the chunk's dP)
        auto ds_chunk = [&](const uint32_t (&pk)[16], uint32_t (&ds)[16]) {
#pragma unroll
          for (int q = 0; q < 16; ++q) {
            const uint64_t t = mul2(f2pack(bf16lo(pk[q]), bf16hi(pk[q])),
                                    sub2(f2pack(__uint_as_float(dr[2 * q]), __uint_as_float(dr[2 * q + 1])), dd));
            float a, b;
            f2unpack(t, a, b);
            ds[q] = pack_bf16(a, b);
          }
        };
        auto store_chunk = [&](int c, const uint32_t (&pk)[16], const uint32_t (&ds)[16]) {
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const int cj = colbase / 8 + 4 * c + q;
            sts_v4(sP + pds_off(slot, cj), pk[4 * q], pk[4 * q + 1], pk[4 * q + 2], pk[4 * q + 3]);
            sts_v4(sDS + pds_off(slot, cj), ds[4 * q], ds[4 * q + 1], ds[4 * q + 2], ds[4 * q + 3]);
          }
        };
        // The single P/dS buffer is the serial section of the kernel (a tile holds it from its first store to
        // the completion of its accumulation MMAs), so everything that can be computed before the tile's turn
        // is: the dS chunks wait in registers (W <= 64) or in TMEM (W = 128) and the turn only covers the stores
        // (profiles/r02_attention.md: the turn wait was 20 % of the softmax warps' samples at base).
        constexpr bool PRE = NCH <= 2;
        uint32_t dsr[PRE ? 16 * NCH : 16];
        if constexpr (PRE) {
#pragma unroll
          for (int c = 0; c < NCH; ++c) {
            uint32_t pk[16], ds[16];
            p_chunk(c, pk);
            if (NCH > 1) {
              tmem_ld32(tS + colbase + 32 * c, dr);
              tmem_wait_ld();
            }
            ds_chunk(pk, ds);
#pragma unroll
            for (int q = 0; q < 16; ++q) dsr[16 * c + q] = ds[q];
          }
        } else {
          // W = 128: the packed dS chunks are parked in TMEM, over the first half of the dP chunk they came from
#pragma unroll
          for (int c = 0; c < NCH; ++c) {
            uint32_t pk[16], ds[16];
            p_chunk(c, pk);
            tmem_ld32(tS + colbase + 32 * c, dr);
            tmem_wait_ld();
            ds_chunk(pk, ds);
            tmem_st16(tS + colbase + 32 * c, ds);
          }
          tmem_wait_st();
        }
        // this tile's turn on the P/dS buffer
        if (wq == 0 && lane == 0) TR(8, k * NSETS + g);   // pass B done, waiting for the turn
        if (!first_tile) mbar_wait(b_turn, (g == 0 ? k - 1 : k) & 1);
        if (wq == 0 && lane == 0) TR(9, k * NSETS + g);   // turn acquired
        if (old_lg >= 0 && old_lg != x.lgCp) {
          // the rows were last written with another geometry: clear that window
          const int ocb = old_lg >= 5 ? (((32 * wq) >> old_lg) << old_lg) : 32 * wq;
          const int oW = (1 << old_lg) < 32 ? 32 : (1 << old_lg);
          for (int q = 0; q < oW / 8; ++q) {
            sts_v4(sP + pds_off(slot, ocb / 8 + q), 0u, 0u, 0u, 0u);
            sts_v4(sDS + pds_off(slot, ocb / 8 + q), 0u, 0u, 0u, 0u);
          }
        }
#pragma unroll
        for (int c = 0; c < NCH; ++c) {
          uint32_t pk[16], ds[16];
          p_chunk(c, pk);
          if constexpr (PRE) {
#pragma unroll
            for (int q = 0; q < 16; ++q) ds[q] = dsr[16 * c + q];
          } else {
            tmem_ld16(tS + colbase + 32 * c, ds);
            tmem_wait_ld();
          }
          store_chunk(c, pk, ds);
        }
        if constexpr (W == 96) {
          uint32_t z[16];
#pragma unroll
          for (int q = 0; q < 16; ++q) z[q] = 0u;
          store_chunk(3, z, z);
        }
      };
      if (x.lgCp <= 5) body(std::integral_constant<int, 32>{});
      else if (x.lgCp == 6) body(std::integral_constant<int, 64>{});
      else if (x.Cv <= 96) body(std::integral_constant<int, 96>{});
      else body(std::integral_constant<int, 128>{});
      tc_fence_before();
      fence_proxy_async_smem();
      __syncwarp();
      if (wq == 0 && lane == 0) TR(10, k * NSETS + g);    // P/dS stored and fenced
      if (lane == 0) mbar_arrive(b_pds_full);

      // ---- drain dQ | dK | dV
      mbar_wait(b_acc_full, k & 1);
      if (wq == 0 && lane == 0) TR(11, k * NSETS + g);    // accumulators ready
      tc_fence_after();
      const size_t off = ((size_t)(grow0 + rl) * s.C + my_col) * d2 + (size_t)x.h * ROWB;
      const uint64_t sc = f2pack(s.scale, s.scale);
      QuadRows qr;
      if constexpr (DH >= 32) qr.init(off, live, lane);
#pragma unroll
      for (int w = 0; w < 3; ++w) {
        uint32_t acc[DH];
        tmem_ld_cols<DH>(tS + w * DH, acc);
        if (w == 2) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(b_acc_free);
          if (wq == 0 && lane == 0) TR(12, k * NSETS + g);  // accumulators drained
        }
        unsigned char* dst = w == 0 ? dQ : (w == 1 ? dK : dV);
        uint4 u[DH / 8];
#pragma unroll
        for (int q = 0; q < DH / 8; ++q) {
          uint32_t* up = &u[q].x;
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            float a = __uint_as_float(acc[8 * q + 2 * e]), b = __uint_as_float(acc[8 * q + 2 * e + 1]);
            if (w < 2) f2unpack(mul2(f2pack(a, b), sc), a, b);
            up[e] = pack_bf16(a, b);
          }
        }
        if constexpr (DH >= 32) {
          // a quad of lanes stores one 64-byte group of a row per instruction (quad_transpose, feature_tc.cuh)
#pragma unroll
          for (int gq = 0; gq < DH / 32; ++gq) {
            uint4 t4[4] = {u[4 * gq], u[4 * gq + 1], u[4 * gq + 2], u[4 * gq + 3]};
            quad_transpose(t4, lane);
#pragma unroll
            for (int k4 = 0; k4 < 4; ++k4)
              if (qr.live[k4]) stg_v4(dst + qr.off[k4] + 64 * gq, t4[k4]);
          }
        } else if (live) {
#pragma unroll
          for (int q = 0; q < DH / 8; ++q) stg_v4(dst + off + 16 * q, u[q]);
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == Cfg::SWARP) tmem_dealloc(tmem, Cfg::COLS);
}

}  // namespace

// (feature_tc_fwd.cu) fills the geometry of a call and, for masked tables, launches the a0 prep kernel
void feature_fill_params(const Shape& s, void* ws, cudaStream_t stream, ftc::FeatParams* p, long long* max_tiles, int* lg);

namespace {

template <int DH>
cudaError_t launch_bwd(const Shape& s, const void* Q, const void* K, const void* V, const void* dO, const float* LSE,
                       void* dQ, void* dK, void* dV, void* ws, cudaStream_t stream) {
  using Cfg = BwdCfg<DH>;
  const DeviceInfo* di = current_device();
  if (!di) return cudaErrorInvalidDevice;
  FeatParams p{};
  long long max_tiles;
  int lg;
  feature_fill_params(s, ws, stream, &p, &max_tiles, &lg);
  CUtensorMap mq, mk, mv, mg;
  const int rpt = kSlots >> lg;
  if (!get_tensor_map(&mq, 1, Q, s.B, s.R, s.C, s.H, DH, rpt, 1 << lg) ||
      !get_tensor_map(&mk, 1, K, s.B, s.R, s.C, s.H, DH, rpt, 1 << lg) ||
      !get_tensor_map(&mv, 1, V, s.B, s.R, s.C, s.H, DH, rpt, 1 << lg) ||
      !get_tensor_map(&mg, 1, dO, s.B, s.R, s.C, s.H, DH, rpt, 1 << lg))
    return cudaErrorInvalidValue;
  auto kern = feature_bwd_tc_kernel<DH>;
  static SmemAttr attr;
  cudaError_t e = attr.ensure(kern, Cfg::SMEM, di->ordinal);
  if (e != cudaSuccess) return e;
  const int grid = (int)std::min<long long>(max_tiles, di->num_sms);
  kern<<<grid, Cfg::THREADS, Cfg::SMEM, stream>>>(mq, mk, mv, mg, p, (const unsigned char*)Q, (const unsigned char*)K,
                                                  (const unsigned char*)V, (const unsigned char*)dO, LSE,
                                                  (unsigned char*)dQ, (unsigned char*)dK, (unsigned char*)dV);
  count_launch();
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_feature_bwd(const Shape& s, const void* Q, const void* K, const void* V, const void* O,
                               const void* dO, const float* LSE, void* dQ, void* dK, void* dV, void* ws,
                               cudaStream_t stream) {
  (void)O;   // D = sum_j P_ij dP_ij is computed from P and dP (whole rows sit in one tile): O is not read
  switch (s.dh) {
    case 16: return launch_bwd<16>(s, Q, K, V, dO, LSE, dQ, dK, dV, ws, stream);
    case 32: return launch_bwd<32>(s, Q, K, V, dO, LSE, dQ, dK, dV, ws, stream);
    case 64: return launch_bwd<64>(s, Q, K, V, dO, LSE, dQ, dK, dV, ws, stream);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace tabattn
