// Item-axis attention forward on tcgen05.
//
// Persistent, warp-specialised kernel; one CTA per SM walks work items (b, c, h, 256 query rows):
//   warp 8        TMA producer: Q tiles (2 x 128 rows, double-buffered over items) and a ring of K/V
//                 tiles of the train rows [0, n_train[b]) only
//   warp 9        issuer of S_t = Q_t K_j^T (SS, fp32 in TMEM) for both query tiles; also zeroes the
//                 V rows >= n_train of a partially valid last key tile
//   warp 10 / 11  issuer of O_t += P_t V_j (A = P in TMEM as bf16) for query tile 0 / 1
//   warps 0-3/4-7 softmax warpgroup of query tile t = 0 / 1: one thread per query row reads its S row
//                 from TMEM, online softmax in base 2 with lazy rescaling of O, writes P (bf16) back
//                 to TMEM; epilogue O / l -> bf16, LSE (natural log)
// S for the next key tile is issued before the PV of the current one, across item boundaries, so
// the softmax warps (the exp-bound critical path at dh <= 64) never wait for the tensor core.
// Keys >= n_train[b] never reach an output: their S columns are masked to -inf (whatever K holds) and
// their V rows are zeroed in shared memory after the TMA load (0 x NaN would still be NaN).
#include <cuda.h>

#include <algorithm>
#include <atomic>

#include "../../include/tabattn.h"
#include "item_tc_common.cuh"
#include "kernels.h"

namespace tabattn {

TABATTN_TRACE_DEFINE(tabattn_debug_set_trace_item_fwd)

namespace {

using namespace tc;
using namespace itc;

template <int DH>
struct FwdCfg {
  static constexpr int ROWB = DH * 2;
  static constexpr int TILE = kTileRows * ROWB;  // bytes of one 128-row operand tile
  static constexpr int ST = 3;                   // K/V ring depth
  static constexpr int QBUF = 2;                 // Q double buffer (over items), 2 tiles each
  static constexpr int SMEM = (2 * QBUF + 2 * ST) * TILE + 1024;
  // TMEM columns
  static constexpr int S0 = 0, P0 = 256, O0 = 384, COLS = 512;
  static_assert(O0 + 2 * DH <= COLS, "TMEM budget");
  // pairs of every 8 whose exponential runs on the FMA pipe (exp2_poly2) instead of the MUFU.  Measured on B200
  // (profiles/r01_s14_item.md, r01_s46_final.md): 2 of 8 gives +8 % at dh = 32 and +2 % at dh = 64 (after the issue
  // and item-decode overheads were removed; it was -1.5 % before), larger shares lose at both.
  static constexpr int POLY_OF_8 = 2;
};

constexpr int kFwdThreads = 384;

template <int DH, bool MASKED>
__global__ void __launch_bounds__(kFwdThreads, 1)
item_fwd_tc_kernel(const __grid_constant__ CUtensorMap mapQ, const __grid_constant__ CUtensorMap mapK,
                   const __grid_constant__ CUtensorMap mapV, Shape s, __nv_bfloat16* __restrict__ O,
                   float* __restrict__ LSE, const uint32_t* __restrict__ col_list, int n_items_all,
                   int blocks_per_seq, int q_row0, int q_row1) {
  TR_INIT();
  using Cfg = FwdCfg<DH>;
  constexpr int ST = Cfg::ST, TILE = Cfg::TILE, ROWB = Cfg::ROWB;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sQ = sbase;                               // [QBUF][2][TILE]
  const uint32_t sK = sQ + 2 * Cfg::QBUF * TILE;           // [ST][TILE]
  const uint32_t sV = sK + ST * TILE;                      // [ST][TILE]
  __shared__ uint64_t bar_q_full[2], bar_q_empty[2], bar_k_full[ST], bar_v_full[ST], bar_v_land[ST], bar_k_empty[ST], bar_v_empty[ST];
  __shared__ uint64_t bar_s_full[2], bar_s_empty[2], bar_p_full[2], bar_pv_done[2];
  __shared__ uint32_t tmem_slot;

  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;  // provably warp-uniform
  ColList<MASKED> cl;
  cl.init(s, col_list);
  // (unmasked: the host's count, a kernel parameter, keeps the issuing warps' loop bounds in uniform registers)
  const int n_items = MASKED ? cl.nv * s.H * blocks_per_seq : n_items_all;
  if (warp == 10) tmem_alloc(smem_u32(&tmem_slot), Cfg::COLS);
  if (threadIdx.x == 0) {
    for (int i = 0; i < 2; ++i) {
      mbar_init(smem_u32(&bar_q_full[i]), 1);
      mbar_init(smem_u32(&bar_q_empty[i]), 1);
      mbar_init(smem_u32(&bar_s_full[i]), 1);
      mbar_init(smem_u32(&bar_s_empty[i]), 128);
      mbar_init(smem_u32(&bar_p_full[i]), 128);
      mbar_init(smem_u32(&bar_pv_done[i]), 1);
    }
    for (int i = 0; i < ST; ++i) {
      mbar_init(smem_u32(&bar_k_full[i]), 1);
      mbar_init(smem_u32(&bar_v_full[i]), 1);
      mbar_init(smem_u32(&bar_v_land[i]), 1);
      mbar_init(smem_u32(&bar_k_empty[i]), 1);
      mbar_init(smem_u32(&bar_v_empty[i]), 2);   // both PV issuers
    }
    fence_barrier_init();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;

  if (warp >= 8) {
    setmaxnreg_dec<64>();
    if (warp == 8) {
      // ------------------------------------------------------------------ TMA producer
      if (lane == 0) {
        tma_prefetch_desc(&mapQ);
        tma_prefetch_desc(&mapK);
        tma_prefetch_desc(&mapV);
        Walker<MASKED> wk;
        for (wk.init(s, cl, blocks_per_seq, kTileRows, true); wk.ok; wk.next(s)) {
          if (wk.j == 0) {
            const int qb = wk.k & 1;
            mbar_wait<true>(smem_u32(&bar_q_empty[qb]), ((wk.k >> 1) & 1) ^ 1);
            mbar_arrive_expect_tx(smem_u32(&bar_q_full[qb]), 2 * TILE);
            const int q0 = q_row0 + wk.blk * 2 * kTileRows;
            tma_load_5d(sQ + (2 * qb) * TILE, &mapQ, smem_u32(&bar_q_full[qb]), 0, wk.h, wk.c, q0, wk.b);
            tma_load_5d(sQ + (2 * qb + 1) * TILE, &mapQ, smem_u32(&bar_q_full[qb]), 0, wk.h, wk.c, q0 + kTileRows,
                        wk.b);
          }
          const int st = wk.t % ST;
          mbar_wait<true>(smem_u32(&bar_k_empty[st]), ((wk.t / ST) & 1) ^ 1);
          mbar_arrive_expect_tx(smem_u32(&bar_k_full[st]), TILE);
          tma_load_5d(sK + st * TILE, &mapK, smem_u32(&bar_k_full[st]), 0, wk.h, wk.c, wk.j * kTileRows, wk.b);
          mbar_wait<true>(smem_u32(&bar_v_empty[st]), ((wk.t / ST) & 1) ^ 1);
          // a partially valid last tile goes through the tail fix (warp 9) before the PV MMAs see it
          const bool tail = wk.j == wk.tiles - 1 && wk.n % kTileRows != 0;
          const uint32_t vbar = tail ? smem_u32(&bar_v_land[st]) : smem_u32(&bar_v_full[st]);
          mbar_arrive_expect_tx(vbar, TILE);
          tma_load_5d(sV + st * TILE, &mapV, vbar, 0, wk.h, wk.c, wk.j * kTileRows, wk.b);
        }
      }
    } else {
      // ------------------------------------------------------------------ MMA issuers
      // warp 9: S_t = Q_t K_j^T for both query tiles (runs ahead as far as the S buffers allow) and the
      // V tail fix; warp 10 / 11: O_t += P_t V_j for query tile t = 0 / 1.  Each warp runs its loop
      // convergently (elect.sync inside every issue) on precomputed descriptors.  One issuing warp costs
      // ~65 clk per tcgen05.mma (a dependent chain of ~10 SASS instructions), which bound the first two
      // builds of this kernel (profiles/r01_s14_item.md); three warps in parallel do not.
      constexpr uint32_t TILE16 = TILE >> 4;
      uint32_t st = 0, ph = 0, par = 0, j = 0, tiles = 0, k = 0;
      int n = 0;
      ItemCoord ic;
      ic.init(s, blocks_per_seq, cl.masked() ? max(cl.nv, 1) : 0);
      auto seek = [&]() {
        if (ic.w >= n_items) return false;
        int rb = ic.b, rc = ic.c;
        if (cl.masked()) cl.pair(ic.c, rb, rc);
        n = clamp_n(s, rb);
        tiles = (uint32_t)(n + kTileRows - 1) / kTileRows;
        return true;
      };
      bool ok = seek();
      if (warp == 9) {
        constexpr uint32_t idS = make_idesc_bf16(128, 128, false, false);
        const uint64_t dQ = make_smem_desc<ROWB>(sQ, 16, 8 * ROWB);
        const uint64_t dK = make_smem_desc<ROWB>(sK, 16, 8 * ROWB);
        const uint32_t b_k_full = smem_u32(&bar_k_full[0]), b_k_empty = smem_u32(&bar_k_empty[0]),
                       b_q_full = smem_u32(&bar_q_full[0]), b_q_empty = smem_u32(&bar_q_empty[0]),
                       b_s_full = smem_u32(&bar_s_full[0]), b_s_empty = smem_u32(&bar_s_empty[0]);
        uint32_t tph = 0;  // per-slot phase bits of bar_v_land
        while (ok) {
          const uint32_t qb = k & 1;
          if (j == 0) mbar_wait(b_q_full + 8 * qb, (k >> 1) & 1);
          mbar_wait(b_k_full + 8 * st, ph);
          const uint64_t kd = dK + st * TILE16;
#pragma unroll
          for (int t = 0; t < 2; ++t) {
            const uint64_t qd = dQ + (2 * qb + t) * TILE16;
            mbar_wait(b_s_empty + 8 * t, par ^ 1);
            tc_fence_after();
#pragma unroll
            for (int kk = 0; kk < DH / 16; ++kk)
              mma_ss_e(tmem + Cfg::S0 + 128 * t, qd + 2 * kk, kd + 2 * kk, idS, kk > 0);
            tc_commit_e(b_s_full + 8 * t);
          }
          tc_commit_e(b_k_empty + 8 * st);
          if (j == tiles - 1) {
            tc_commit_e(b_q_empty + 8 * qb);
            // The last key tile of an item with n % 128 != 0 holds rows >= n_train (test rows).  Their S
            // columns are masked to -inf by the softmax threads (P = 0), but 0 x (Inf/NaN) would still
            // poison O, so those V rows are zeroed in shared memory: the producer lands such a tile on
            // bar_v_land and this warp completes bar_v_full in the TMA's place.
            const int rem = n - (int)(tiles - 1) * kTileRows;
            if (rem != kTileRows) {
              mbar_wait(smem_u32(&bar_v_land[0]) + 8 * st, (tph >> st) & 1);
              tph ^= 1u << st;
              zero_tail_rows<ROWB>(sV + st * TILE, rem, lane);
              if (lane == 0) mbar_arrive(smem_u32(&bar_v_full[0]) + 8 * st);
            }
          }
          par ^= 1;
          if (++st == ST) { st = 0; ph ^= 1; }
          if (++j == tiles) {
            j = 0;
            ++k;
            ic.next();
            ok = seek();
          }
        }
      } else if (warp <= 11) {
        const uint32_t t = warp - 10;
        constexpr uint32_t idO = make_idesc_bf16(128, DH, false, true);
        const uint64_t dV = make_smem_desc<ROWB>(sV, 16, 8 * ROWB);
        const uint32_t b_v_full = smem_u32(&bar_v_full[0]), b_v_empty = smem_u32(&bar_v_empty[0]),
                       b_p_full = smem_u32(&bar_p_full[t]), b_pv_done = smem_u32(&bar_pv_done[t]);
        const uint32_t tO = tmem + Cfg::O0 + DH * t, tP = tmem + Cfg::P0 + 64 * t;
        while (ok) {
          mbar_wait(b_v_full + 8 * st, ph);
          const uint64_t vd = dV + st * TILE16;
          mbar_wait(b_p_full, par);
          tc_fence_after();
#pragma unroll
          for (int kk = 0; kk < kTileRows / 16; ++kk)
            mma_ts_e(tO, tP + 8 * kk, vd + kk * ROWB, idO, (j > 0 || kk > 0) ? 1u : 0u);
          tc_commit_e(b_pv_done);
          tc_commit_e(b_v_empty + 8 * st);
          par ^= 1;
          if (++st == ST) { st = 0; ph ^= 1; }
          if (++j == tiles) {
            j = 0;
            ic.next();
            ok = seek();
          }
        }
      }
    }
  } else {
    // -------------------------------------------------------------------- softmax warpgroups
    setmaxnreg_inc<216>();
    const int t = warp >> 2;                  // query tile of this warpgroup
    const int r = threadIdx.x & 127;          // row inside the tile = TMEM lane
    const uint32_t lane_base = tmem + ((uint32_t)(32 * (warp & 3)) << 16);
    const uint32_t tS = lane_base + Cfg::S0 + 128 * t, tP = lane_base + Cfg::P0 + 64 * t,
                   tO = lane_base + Cfg::O0 + DH * t;
    const uint32_t b_s_full = smem_u32(&bar_s_full[t]), b_s_empty = smem_u32(&bar_s_empty[t]),
                   b_p_full = smem_u32(&bar_p_full[t]), b_pv_done = smem_u32(&bar_pv_done[t]);
    const float c2 = s.scale * kLog2e;
    const int d = s.H * DH;
    uint32_t g = 0;  // tiles processed by this CTA so far
    // a6: the invalid columns (masked tables) are dealt to the CTAs like the items (O := +0, LSE := 0); a CTA clears
    // one invalid item after every item it computes, so the stores spread over the kernel instead of forming a tail
    const int n_zero = MASKED ? cl.ni * s.H * blocks_per_seq : 0;
    int wz = blockIdx.x;
    auto zero_one = [&]() {
      const int blk = wz % blocks_per_seq, seq = wz / blocks_per_seq, h = seq % s.H;
      int b, c;
      cl.pair(cl.nv + seq / s.H, b, c);
      const int row = q_row0 + blk * 2 * kTileRows + t * kTileRows + r;
      if (row < q_row1) {
        __nv_bfloat16* oz = O + (((size_t)b * s.R + row) * s.C + c) * d + (size_t)h * DH;
#pragma unroll
        for (int k = 0; k < DH / 8; ++k) stg_v4(oz + 8 * k, make_uint4(0, 0, 0, 0));
        if (LSE) LSE[(((size_t)b * s.C + c) * s.H + h) * s.R + row] = 0.f;
      }
      wz += gridDim.x;
    };
    Walker<MASKED> it;
    it.cl = cl; it.n_items = n_items; it.chunk = kTileRows; it.over_keys = true;
    it.ic.init(s, blocks_per_seq, cl.masked() ? max(cl.nv, 1) : 0);
    for (; it.ic.w < n_items; it.ic.next()) {
      bool valid;
      it.decode(s, valid);
      const int row = q_row0 + it.blk * 2 * kTileRows + t * kTileRows + r;
      __nv_bfloat16* orow = O + (((size_t)it.b * s.R + row) * s.C + it.c) * d + (size_t)it.h * DH;
      float* lse = LSE + (((size_t)it.b * s.C + it.c) * s.H + it.h) * s.R + row;
      if (!valid) {   // (never taken: see Walker::decode)
        if (row < q_row1) {
#pragma unroll
          for (int k = 0; k < DH / 8; ++k) stg_v4(orow + 8 * k, make_uint4(0, 0, 0, 0));
          if (LSE) *lse = 0.f;
        }
        continue;
      }
      const int tiles = (it.n + kTileRows - 1) / kTileRows;
      float m = -INFINITY, l = 0.f;
      for (int j = 0; j < tiles; ++j, ++g) {
        mbar_wait(b_s_full, g & 1);
        if (r == 0) TR(0 + 7 * t, g);                      // S ready
        tc_fence_after();
        uint32_t sr[128];
        tmem_ld32(tS, sr);
        tmem_ld32(tS + 32, sr + 32);
        tmem_ld32(tS + 64, sr + 64);
        tmem_ld32(tS + 96, sr + 96);
        tmem_wait_ld();
        tc_fence_before();
        mbar_arrive(b_s_empty);
        if (r == 0) TR(1 + 7 * t, g);                      // S loaded, buffer released
        float* sf = reinterpret_cast<float*>(sr);
        const int rem = it.n - j * kTileRows;
        if (rem < kTileRows) {
#pragma unroll
          for (int k = 0; k < 128; ++k)
            if (k >= rem) sf[k] = -INFINITY;
        }
        // row maximum with three-input max (FMNMX3): 64 instead of 127 instructions, four independent chains
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
        const float mxs = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * c2;
        if (j == 0) {
          m = mxs;
        } else if (__any_sync(0xffffffffu, mxs > m + kRescaleLog2)) {
          // rare after the first tiles: bring the accumulated O and l to the new reference maximum
          const float mn = fmaxf(m, mxs);
          const float alpha = fast_exp2(m - mn);
          l *= alpha;
          m = mn;
          mbar_wait(b_pv_done, (g - 1) & 1);
          tc_fence_after();
          uint32_t o[DH];
          tmem_ld_cols<DH>(tO, o);
#pragma unroll
          for (int k = 0; k < DH; ++k) o[k] = __float_as_uint(__uint_as_float(o[k]) * alpha);
          tmem_st_cols<DH>(tO, o);
          tmem_wait_st();
        }
        // P = 2^(S*c2 - m) on packed pairs; Cfg::POLY_OF_8 of every 8 pairs take the FMA-pipe polynomial, the
        // rest the MUFU, so that the two pipes finish together
        if (r == 0) TR(2 + 7 * t, g);                      // maximum done
        const uint64_t cc = f2pack(c2, c2), nm = f2pack(-m, -m);
        uint64_t la = 0, lb = 0;  // two packed partial row sums (+0.f, +0.f)
        uint32_t p[64];
#pragma unroll
        for (int k = 0; k < 64; ++k) {
          const uint64_t x = fma2(f2pack(sf[2 * k], sf[2 * k + 1]), cc, nm);
          float e0, e1;
          exp2_pair(pair_is_poly<Cfg::POLY_OF_8>(k), x, e0, e1);
          if (k & 1) lb = add2(lb, f2pack(e0, e1)); else la = add2(la, f2pack(e0, e1));
          p[k] = pack_bf16(e0, e1);
        }
        {
          float s0, s1;
          f2unpack(add2(la, lb), s0, s1);
          l += s0 + s1;
        }
        if (r == 0) TR(3 + 7 * t, g);                      // exponentials done
        if (g > 0) mbar_wait(b_pv_done, (g - 1) & 1);  // previous PV has finished reading the P buffer
        if (r == 0) TR(4 + 7 * t, g);                      // P buffer free
        tmem_st32(tP, p);
        tmem_st32(tP + 32, p + 32);
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(b_p_full);
        if (r == 0) TR(5 + 7 * t, g);                      // P stored
      }
      // ---- epilogue: O = acc / l, LSE = ln(sum exp) ---------------------------------------------
      mbar_wait(b_pv_done, (g - 1) & 1);
      if (threadIdx.x == 0) TR(14, g - 1);                 // last PV of the item done
      tc_fence_after();
      uint32_t o[DH];
      tmem_ld_cols<DH>(tO, o);
      tc_fence_before();
      if constexpr (DH >= 64) {
        // a quad of lanes stores one 64-byte group of a row per instruction (four times fewer line requests than
        // every lane storing its own row in DH / 8 instructions; measured +2 % at dh = 64, -2 % at dh = 32)
        const float inv = 1.f / l;
        uint4 u[DH / 8];
#pragma unroll
        for (int k = 0; k < DH / 8; ++k) {
          float f[8];
#pragma unroll
          for (int e = 0; e < 8; ++e) f[e] = __uint_as_float(o[8 * k + e]) * inv;
          u[k] = pack8(f);
        }
        const bool live = row < q_row1;
        QuadRows qr;
        qr.init(reinterpret_cast<size_t>(orow), live, lane);
#pragma unroll
        for (int gq = 0; gq < DH / 32; ++gq) {
          uint4 t4[4] = {u[4 * gq], u[4 * gq + 1], u[4 * gq + 2], u[4 * gq + 3]};
          quad_transpose(t4, lane);
#pragma unroll
          for (int k4 = 0; k4 < 4; ++k4)
            if (qr.live[k4]) stg_v4(reinterpret_cast<void*>(qr.off[k4] + 64 * gq), t4[k4]);
        }
        if (live && LSE) *lse = (m + log2f(l)) * kLn2;
      } else if (row < q_row1) {
        const float inv = 1.f / l;
#pragma unroll
        for (int k = 0; k < DH / 8; ++k) {
          float f[8];
#pragma unroll
          for (int e = 0; e < 8; ++e) f[e] = __uint_as_float(o[8 * k + e]) * inv;
          stg_v4(orow + 8 * k, pack8(f));
        }
        if (LSE) *lse = (m + log2f(l)) * kLn2;
      }
      if (threadIdx.x == 0) TR(15, g - 1);                 // O and LSE stored
      if (MASKED && wz < n_zero) zero_one();
    }
    while (MASKED && wz < n_zero) zero_one();   // (what is left of the invalid columns)
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 10) tmem_dealloc(tmem, Cfg::COLS);
}

template <int DH>
cudaError_t launch_fwd(const Shape& s, const void* Q, const void* K, const void* V, void* O, float* LSE,
                       int q_row0, int q_row1, void* ws, cudaStream_t stream) {
  using Cfg = FwdCfg<DH>;
  const DeviceInfo* di = current_device();
  if (!di) return cudaErrorInvalidDevice;
  CUtensorMap mq, mk, mv;
  if (!get_tensor_map(&mq, 0, Q, s.B, s.R, s.C, s.H, DH, kTileRows, 1) ||
      !get_tensor_map(&mk, 0, K, s.B, s.R, s.C, s.H, DH, kTileRows, 1) ||
      !get_tensor_map(&mv, 0, V, s.B, s.R, s.C, s.H, DH, kTileRows, 1))
    return cudaErrorInvalidValue;
  const uint32_t* list = item_build_list(s, ws, stream);   // (a0 prep kernel for masked tables)
  auto kern = list ? item_fwd_tc_kernel<DH, true> : item_fwd_tc_kernel<DH, false>;
  static SmemAttr attr_m, attr_u;
  cudaError_t e = (list ? attr_m : attr_u).ensure(kern, Cfg::SMEM, di->ordinal);
  if (e != cudaSuccess) return e;
  // query rows [q_row0, q_row1) of every sequence (the training forward passes [0, R)); keys are always [0, n_train)
  const int bps = (q_row1 - q_row0 + 2 * kTileRows - 1) / (2 * kTileRows);
  const long long n_items = (long long)s.B * s.C * s.H * bps;
  const int grid = (int)std::min<long long>(n_items, di->num_sms);
  kern<<<grid, kFwdThreads, Cfg::SMEM, stream>>>(mq, mk, mv, s, (__nv_bfloat16*)O, LSE, list, (int)n_items, bps, q_row0, q_row1);
  count_launch();
  return cudaGetLastError();
}

}  // namespace

// ---- a0 prep (masked tables): the compacted (b, c) list of item_tc_common.cuh ---------------------------------
__global__ void __launch_bounds__(256) item_prep_kernel(Shape s, uint32_t* __restrict__ out) {
  __shared__ int warp_cnt[8];
  __shared__ int base_s, nv_s;
  const int cells = s.B * s.C, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t* list = out + 4;
  // pass 1: NV
  int cnt = 0;
  for (int i = threadIdx.x; i < cells; i += 256) cnt += __ldg(s.col_valid + i) != 0;
  for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
  if (lane == 0) warp_cnt[warp] = cnt;
  __syncthreads();
  if (threadIdx.x == 0) {
    int t = 0;
    for (int w = 0; w < 8; ++w) t += warp_cnt[w];
    nv_s = t;
    base_s = 0;
    out[0] = (uint32_t)t;
  }
  __syncthreads();
  const int nv = nv_s;
  // pass 2: valid pairs ascending into [0, NV), invalid ones ascending into [NV, cells)
  for (int i0 = 0; i0 < cells; i0 += 256) {
    const int i = i0 + threadIdx.x;
    const bool in = i < cells, v = in && __ldg(s.col_valid + i) != 0;
    const uint32_t m = __ballot_sync(0xffffffffu, v);
    if (lane == 0) warp_cnt[warp] = __popc(m);
    __syncthreads();
    int before = base_s;                       // valid pairs before this 256-chunk
    for (int w = 0; w < warp; ++w) before += warp_cnt[w];
    before += __popc(m & ((1u << lane) - 1u));
    if (in) {
      const int b = i / s.C, c = i - b * s.C;
      list[v ? before : nv + (i - before)] = ((uint32_t)b << 16) | (uint32_t)c;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      int t = 0;
      for (int w = 0; w < 8; ++w) t += warp_cnt[w];
      base_s += t;
    }
    __syncthreads();
  }
}

size_t item_list_bytes(const Shape& s) { return ((size_t)s.B * s.C + 4) * sizeof(uint32_t); }
size_t item_fwd_workspace_bytes(const Shape& s) { return item_list_bytes(s); }

const uint32_t* item_build_list(const Shape& s, void* list_ws, cudaStream_t stream) {
  if (!s.col_valid || !list_ws) return nullptr;
  item_prep_kernel<<<1, 256, 0, stream>>>(s, static_cast<uint32_t*>(list_ws));
  count_launch();
  return static_cast<const uint32_t*>(list_ws);
}

cudaError_t launch_item_fwd(const Shape& s, const void* Q, const void* K, const void* V, void* O, float* LSE,
                            int q_row0, int q_row1, void* ws, cudaStream_t stream) {
  switch (s.dh) {
    case 16: return launch_fwd<16>(s, Q, K, V, O, LSE, q_row0, q_row1, ws, stream);
    case 32: return launch_fwd<32>(s, Q, K, V, O, LSE, q_row0, q_row1, ws, stream);
    case 64: return launch_fwd<64>(s, Q, K, V, O, LSE, q_row0, q_row1, ws, stream);
    default: return cudaErrorInvalidValue;
  }
}

// ---- tabattn_item_fwd_noalloc: the same forward with its scratch inside the library -----------------------------
// For callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): the a0
// column list of a masked call lives in a file-scope device array instead of a caller workspace.  Every GPU that
// loads the library holds the array (256 KiB + 256 B) until the process exits.  Nothing in it has to start at zero:
// item_prep_kernel rewrites the count and every list entry the main kernel reads, on the call's stream, before the
// main kernel runs.  All calls share the array, so two calls that overlap on the GPU (different streams) race.
constexpr size_t kNoAllocScratchBytes = ((size_t)TABATTN_NOALLOC_MAX_BC + 4) * sizeof(uint32_t) + 240;
static __device__ __align__(256) unsigned char g_item_fwd_scratch[kNoAllocScratchBytes];

size_t item_fwd_noalloc_capacity() { return kNoAllocScratchBytes; }

namespace {
// In host code `g_item_fwd_scratch` is only the symbol's host-side stand-in: the device address comes from
// cudaGetSymbolAddress, asked once per device with that device current.
struct ScratchAddr {
  std::atomic<void*> ptr[kMaxDevices];
  ScratchAddr() { for (auto& p : ptr) p.store(nullptr, std::memory_order_relaxed); }
  cudaError_t get(int ordinal, void** out) {
    void* p = ptr[ordinal].load(std::memory_order_acquire);
    if (!p) {
      const cudaError_t e = cudaGetSymbolAddress(&p, g_item_fwd_scratch);   // (the calling thread's current device)
      if (e != cudaSuccess) return e;
      if (!p) return cudaErrorInvalidSymbol;
      ptr[ordinal].store(p, std::memory_order_release);   // (a lost race stores the same address twice)
    }
    *out = p;
    return cudaSuccess;
  }
};
ScratchAddr g_scratch_addr;
}  // namespace

cudaError_t launch_item_fwd_noalloc(const Shape& s, const void* Q, const void* K, const void* V, void* O, float* LSE,
                                    cudaStream_t stream) {
  void* scratch = nullptr;
  if (s.col_valid) {   // (an unmasked call has no scratch)
    if (item_fwd_workspace_bytes(s) > kNoAllocScratchBytes) return cudaErrorInvalidValue;   // (the ABI checks first)
    const DeviceInfo* di = current_device();
    if (!di) return cudaErrorInvalidDevice;
    const cudaError_t e = g_scratch_addr.get(di->ordinal, &scratch);
    if (e != cudaSuccess) return e;
  }
  return launch_item_fwd(s, Q, K, V, O, LSE, 0, s.R, scratch, stream);
}

}  // namespace tabattn
