// Item-axis attention backward on tcgen05: the dQ pass (which
// also emits D = rowsum(dO o O)) and the separate dK/dV pass, one kernel template with two modes.
// Deterministic: no atomics, every output element has exactly one writer.
//
// Both passes have the same shape: a STATIONARY 128-row tile pair (A1, A2) against a STREAM of
// 64-row chunk pairs (B1, B2):
//   MODE_DQ   A = (Q, dO) rows of one query block; B = (K, V) chunks of the train rows [0, n)
//             S  = Q K^T, dP = dO V^T (rows = queries), dS = P o (dP - D), acc0 (dQ) += dS K
//   MODE_DKV  A = (K, V) rows of one key block (< n); B = (Q, dO) chunks of all R query rows
//             S^T = K Q^T, dP^T = V dO^T (rows = keys), acc0 (dV) += P^T dO, acc1 (dK) += dS^T Q
// with P = exp2(S * scale*log2e - LSE*log2e) recomputed from the saved LSE.  S/dP accumulate in
// TMEM (fp32); P and dS go back to TMEM as bf16 and are the A operands of the second-stage MMAs.
//
// Warp roles (384 threads, one persistent CTA per SM): warp 8 TMA producer (+ LSE/D chunk staging in
// MODE_DKV), warp 9 MMA issuer, warpgroups 0/1 = "set" 0/1: each owns one TMEM set (S, dP, dS, P) and
// takes every other chunk, one thread per tile row; the score MMAs run up to three chunks ahead of the
// accumulation MMAs, across item boundaries.
#include <cuda.h>

#include <algorithm>

#include "item_tc_common.cuh"
#include "kernels.h"

namespace tabattn {

namespace {

using namespace tc;
using namespace itc;

constexpr int MODE_DQ = 0, MODE_DKV = 1;
constexpr int kChunk = 64;
constexpr int kBwdThreads = 384;

template <int DH>
struct BwdCfg {
  static constexpr int ROWB = DH * 2;
  static constexpr int TILE_A = kTileRows * ROWB;  // stationary tile
  static constexpr int TILE_B = kChunk * ROWB;     // streamed chunk
  static constexpr int ST = 4;                     // chunk ring depth
  static constexpr int LD_BYTES = 2 * kChunk * 4;  // per stage: lse2[64], D[64] (MODE_DKV)
  static constexpr int SMEM = 4 * TILE_A + ST * (2 * TILE_B + LD_BYTES) + 1024;
  // TMEM columns: set g at g*SET: S [0,64) dP [64,128) dS [128,160) P [160,192); accumulators after
  static constexpr int SET = 192, S_OFF = 0, DP_OFF = 64, DS_OFF = 128, P_OFF = 160;
  static constexpr int ACC0 = 384, ACC1 = 384 + DH, COLS = 512;
  static_assert(ACC1 + DH <= COLS, "TMEM budget");
};

template <int DH, int MODE>
__global__ void __launch_bounds__(kBwdThreads, 1)
item_bwd_tc_kernel(const __grid_constant__ CUtensorMap mapA1, const __grid_constant__ CUtensorMap mapA2,
                   const __grid_constant__ CUtensorMap mapB1, const __grid_constant__ CUtensorMap mapB2, Shape s,
                   const __nv_bfloat16* __restrict__ O, const __nv_bfloat16* __restrict__ dO,
                   const float* __restrict__ LSE, float* __restrict__ Dws, __nv_bfloat16* __restrict__ out0,
                   __nv_bfloat16* __restrict__ out1, int n_items, int blocks_per_seq) {
  using Cfg = BwdCfg<DH>;
  constexpr int ST = Cfg::ST, TILE_A = Cfg::TILE_A, TILE_B = Cfg::TILE_B, ROWB = Cfg::ROWB;
  constexpr bool kOverKeys = MODE == MODE_DQ;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sA = sbase;                         // [2 item buffers][A1, A2][TILE_A]
  const uint32_t sB = sA + 4 * TILE_A;               // [ST][B1, B2][TILE_B]
  const uint32_t sLD = sB + ST * 2 * TILE_B;         // [ST][lse2[64], D[64]]
  float* sLD_ptr = reinterpret_cast<float*>(smem_raw + (sLD - smem_u32(smem_raw)));
  __shared__ uint64_t bar_a_full[2], bar_a_empty[2], bar_b_full[ST], bar_b_empty[ST];
  __shared__ uint64_t bar_s_full[2], bar_s_empty[2], bar_p_full[2], bar_p_empty[2], bar_acc_full, bar_acc_free;
  __shared__ uint32_t tmem_slot;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (warp == 10) tmem_alloc(smem_u32(&tmem_slot), Cfg::COLS);
  if (threadIdx.x == 0) {
    for (int i = 0; i < 2; ++i) {
      mbar_init(smem_u32(&bar_a_full[i]), 1);
      mbar_init(smem_u32(&bar_a_empty[i]), 1);
      mbar_init(smem_u32(&bar_s_full[i]), 1);
      mbar_init(smem_u32(&bar_s_empty[i]), 128);
      mbar_init(smem_u32(&bar_p_full[i]), 128);
      mbar_init(smem_u32(&bar_p_empty[i]), 1);
    }
    for (int i = 0; i < ST; ++i) {
      mbar_init(smem_u32(&bar_b_full[i]), MODE == MODE_DKV ? 2 : 1);
      mbar_init(smem_u32(&bar_b_empty[i]), 1);
    }
    mbar_init(smem_u32(&bar_acc_full), 1);
    mbar_init(smem_u32(&bar_acc_free), 256);
    fence_barrier_init();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  const int d = s.H * DH;

  if (warp >= 8) {
    setmaxnreg_dec<56>();
    if (warp == 8) {
      // ------------------------------------------------------------------ producer
      if (lane == 0) {
        tma_prefetch_desc(&mapA1);
        tma_prefetch_desc(&mapA2);
        tma_prefetch_desc(&mapB1);
        tma_prefetch_desc(&mapB2);
      }
      Walker wk;
      for (wk.init(s, n_items, blocks_per_seq, kChunk, kOverKeys); wk.ok; wk.next(s)) {
        const int st = wk.t % ST;
        if (lane == 0) {
          if (wk.j == 0) {
            const int ab = wk.k & 1;
            mbar_wait(smem_u32(&bar_a_empty[ab]), ((wk.k >> 1) & 1) ^ 1);
            mbar_arrive_expect_tx(smem_u32(&bar_a_full[ab]), 2 * TILE_A);
            tma_load_5d(sA + (2 * ab) * TILE_A, &mapA1, smem_u32(&bar_a_full[ab]), 0, wk.h, wk.c,
                        wk.blk * kTileRows, wk.b);
            tma_load_5d(sA + (2 * ab + 1) * TILE_A, &mapA2, smem_u32(&bar_a_full[ab]), 0, wk.h, wk.c,
                        wk.blk * kTileRows, wk.b);
          }
          mbar_wait(smem_u32(&bar_b_empty[st]), ((wk.t / ST) & 1) ^ 1);
          mbar_arrive_expect_tx(smem_u32(&bar_b_full[st]), 2 * TILE_B);
          tma_load_5d(sB + (2 * st) * TILE_B, &mapB1, smem_u32(&bar_b_full[st]), 0, wk.h, wk.c, wk.j * kChunk, wk.b);
          tma_load_5d(sB + (2 * st + 1) * TILE_B, &mapB2, smem_u32(&bar_b_full[st]), 0, wk.h, wk.c, wk.j * kChunk,
                      wk.b);
        }
        if (MODE == MODE_DKV) {
          __syncwarp();  // lane 0 has seen the stage free
          const size_t seq = (((size_t)wk.b * s.C + wk.c) * s.H + wk.h) * s.R;
          float* ld = sLD_ptr + st * (2 * kChunk);
#pragma unroll
          for (int e = 0; e < kChunk / 32; ++e) {
            const int i = wk.j * kChunk + 32 * e + lane;
            const bool in = i < s.R;
            ld[32 * e + lane] = in ? __ldg(LSE + seq + i) * kLog2e : INFINITY;
            ld[kChunk + 32 * e + lane] = in ? __ldg(Dws + seq + i) : 0.f;
          }
          __syncwarp();
          if (lane == 0) mbar_arrive(smem_u32(&bar_b_full[st]));
        }
      }
    } else if (warp == 9) {
      // ------------------------------------------------------------------ MMA issuer
      // a: score MMAs (up to three chunks ahead), p: accumulation MMAs.  Chunk t of the CTA's
      // lifetime uses TMEM set t & 1 (global alternation: consecutive chunks never share a set, also
      // across items, so a score issue never waits on a warpgroup that is itself waiting for an
      // accumulation MMA that is issued later); it is that set's (t >> 1)-th chunk.
      Walker a, p;
      a.init(s, n_items, blocks_per_seq, kChunk, kOverKeys);
      p = a;
      auto issue_scores = [&]() {
        const int ab = a.k & 1, st = a.t % ST, g = a.t & 1;
        if (a.j == 0) mbar_wait(smem_u32(&bar_a_full[ab]), (a.k >> 1) & 1);
        mbar_wait(smem_u32(&bar_b_full[st]), (a.t / ST) & 1);
        if (MODE == MODE_DQ) {
          const int rem = a.n - a.j * kChunk;  // keys >= n must not reach dQ through dS K
          if (rem < kChunk) zero_tail_rows<ROWB, kChunk>(sB + (2 * st) * TILE_B, rem, lane);
        }
        if (lane == 0) {
          mbar_wait(smem_u32(&bar_s_empty[g]), ((a.t >> 1) & 1) ^ 1);
          tc_fence_after();
          const uint32_t set = tmem + g * Cfg::SET;
          issue_qk<DH, kChunk>(set + Cfg::S_OFF, sA + (2 * ab) * TILE_A, sB + (2 * st) * TILE_B);
          issue_qk<DH, kChunk>(set + Cfg::DP_OFF, sA + (2 * ab + 1) * TILE_A, sB + (2 * st + 1) * TILE_B);
          tc_commit(smem_u32(&bar_s_full[g]));
          if (a.j == a.tiles - 1) tc_commit(smem_u32(&bar_a_empty[ab]));
        }
        __syncwarp();
        a.next(s);
      };
      auto issue_acc = [&]() {
        const int st = p.t % ST, g = p.t & 1;
        if (lane == 0) {
          if (p.j == 0) mbar_wait(smem_u32(&bar_acc_free), (p.k & 1) ^ 1);
          mbar_wait(smem_u32(&bar_p_full[g]), (p.t >> 1) & 1);
          tc_fence_after();
          const uint32_t set = tmem + g * Cfg::SET;
          if (MODE == MODE_DQ) {
            issue_pv<DH, kChunk>(tmem + Cfg::ACC0, set + Cfg::DS_OFF, sB + (2 * st) * TILE_B, p.j > 0);
          } else {
            issue_pv<DH, kChunk>(tmem + Cfg::ACC0, set + Cfg::P_OFF, sB + (2 * st + 1) * TILE_B, p.j > 0);
            issue_pv<DH, kChunk>(tmem + Cfg::ACC1, set + Cfg::DS_OFF, sB + (2 * st) * TILE_B, p.j > 0);
          }
          tc_commit(smem_u32(&bar_p_empty[g]));
          tc_commit(smem_u32(&bar_b_empty[st]));
          if (p.j == p.tiles - 1) tc_commit(smem_u32(&bar_acc_full));
        }
        __syncwarp();
        p.next(s);
      };
      if (a.ok) issue_scores();
      if (a.ok) issue_scores();
      while (p.ok) {
        if (a.ok) issue_scores();
        issue_acc();
      }
    }
  } else {
    // -------------------------------------------------------------------- score warpgroups (sets)
    setmaxnreg_inc<224>();
    const int g = warp >> 2;                 // TMEM set / chunk parity of this warpgroup
    const int r = threadIdx.x & 127;         // tile row = TMEM lane
    const uint32_t lane_base = tmem + ((uint32_t)(32 * (warp & 3)) << 16);
    const uint32_t set = lane_base + g * Cfg::SET;
    const uint32_t b_s_full = smem_u32(&bar_s_full[g]), b_s_empty = smem_u32(&bar_s_empty[g]),
                   b_p_full = smem_u32(&bar_p_full[g]), b_p_empty = smem_u32(&bar_p_empty[g]);
    const float c2 = s.scale * kLog2e;
    uint32_t kitem = 0;   // valid items seen
    uint32_t tbase = 0;   // chunks of all previous valid items (ring position)
    Walker it;
    it.n_items = n_items; it.bps = blocks_per_seq; it.chunk = kChunk; it.over_keys = kOverKeys;
    for (int w = blockIdx.x; w < n_items; w += gridDim.x) {
      it.w = w;
      bool valid;
      it.decode(s, valid);
      const int row = it.blk * kTileRows + r;
      const size_t cell = (((size_t)it.b * s.R + row) * s.C + it.c) * d + (size_t)it.h * DH;
      const size_t seq = (((size_t)it.b * s.C + it.c) * s.H + it.h) * s.R;
      if (!valid) {
        // invalid column, or (MODE_DKV) a key block entirely beyond the train rows: zeros
        if (row < s.R) {
          if (MODE == MODE_DQ) {
#pragma unroll
            for (int k = 0; k < DH / 16; ++k) stg_v4(out0 + cell + g * (DH / 2) + 8 * k, make_uint4(0, 0, 0, 0));
            if (g == 0) Dws[seq + row] = 0.f;
          } else {
            __nv_bfloat16* dst = (g == 0 ? out0 : out1) + cell;
#pragma unroll
            for (int k = 0; k < DH / 8; ++k) stg_v4(dst + 8 * k, make_uint4(0, 0, 0, 0));
          }
        }
        continue;
      }
      // per-row constants of the dQ pass: LSE_i and D_i = sum_k dO_ik O_ik (also saved for the dK/dV pass)
      float lse2 = INFINITY, Drow = 0.f;
      if (MODE == MODE_DQ && row < s.R) {
        lse2 = __ldg(LSE + seq + row) * kLog2e;
#pragma unroll
        for (int k = 0; k < DH / 8; ++k) {
          float fo[8], fg[8];
          unpack8(ldg_nc_v4(O + cell + 8 * k), fo);
          unpack8(ldg_nc_v4(dO + cell + 8 * k), fg);
#pragma unroll
          for (int e = 0; e < 8; ++e) Drow = fmaf(fo[e], fg[e], Drow);
        }
        if (g == 0) Dws[seq + row] = Drow;
      }
      const int chunks = it.tiles;
      for (int j = (g ^ tbase) & 1; j < chunks; j += 2) {
        const uint32_t u = (tbase + j) >> 1;  // this set's chunk counter
        mbar_wait(b_s_full, u & 1);
        tc_fence_after();
        uint32_t sr[64], dr[64];
        tmem_ld32(set + Cfg::S_OFF, sr);
        tmem_ld32(set + Cfg::S_OFF + 32, sr + 32);
        tmem_ld32(set + Cfg::DP_OFF, dr);
        tmem_ld32(set + Cfg::DP_OFF + 32, dr + 32);
        tmem_wait_ld();
        tc_fence_before();
        mbar_arrive(b_s_empty);
        uint32_t pds[32], pp[32];
        if (MODE == MODE_DQ) {
          const int rem = it.n - j * kChunk;
#pragma unroll
          for (int k = 0; k < 64; k += 2) {
            const float p0 = fast_exp2(fmaf(__uint_as_float(sr[k]), c2, -lse2));
            const float p1 = fast_exp2(fmaf(__uint_as_float(sr[k + 1]), c2, -lse2));
            float d0 = p0 * (__uint_as_float(dr[k]) - Drow);
            float d1 = p1 * (__uint_as_float(dr[k + 1]) - Drow);
            if (rem < kChunk) {  // keys >= n_train: dS = 0 exactly, whatever the masked K/V hold
              d0 = k < rem ? d0 : 0.f;
              d1 = k + 1 < rem ? d1 : 0.f;
            }
            pds[k >> 1] = pack_bf16(d0, d1);
          }
        } else {
          const uint32_t st = (tbase + j) % ST;
          mbar_wait(smem_u32(&bar_b_full[st]), ((tbase + j) / ST) & 1);  // LSE/D chunk is visible
          const float4* l4 = reinterpret_cast<const float4*>(sLD_ptr + st * (2 * kChunk));
          const float4* d4 = l4 + kChunk / 4;
#pragma unroll
          for (int k = 0; k < 64; k += 4) {
            const float4 L = l4[k >> 2], Dv = d4[k >> 2];
            const float p0 = fast_exp2(fmaf(__uint_as_float(sr[k]), c2, -L.x));
            const float p1 = fast_exp2(fmaf(__uint_as_float(sr[k + 1]), c2, -L.y));
            const float p2 = fast_exp2(fmaf(__uint_as_float(sr[k + 2]), c2, -L.z));
            const float p3 = fast_exp2(fmaf(__uint_as_float(sr[k + 3]), c2, -L.w));
            pp[k >> 1] = pack_bf16(p0, p1);
            pp[(k >> 1) + 1] = pack_bf16(p2, p3);
            pds[k >> 1] = pack_bf16(p0 * (__uint_as_float(dr[k]) - Dv.x), p1 * (__uint_as_float(dr[k + 1]) - Dv.y));
            pds[(k >> 1) + 1] =
                pack_bf16(p2 * (__uint_as_float(dr[k + 2]) - Dv.z), p3 * (__uint_as_float(dr[k + 3]) - Dv.w));
          }
        }
        mbar_wait(b_p_empty, (u & 1) ^ 1);  // the MMAs that read this set's previous P/dS are done
        tmem_st32(set + Cfg::DS_OFF, pds);
        if (MODE == MODE_DKV) tmem_st32(set + Cfg::P_OFF, pp);
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(b_p_full);
      }
      // ---- epilogue ---------------------------------------------------------------------------------
      mbar_wait(smem_u32(&bar_acc_full), kitem & 1);
      tc_fence_after();
      if (MODE == MODE_DQ) {
        constexpr int HALF = DH / 2;  // each warpgroup stores half of the dQ columns of its row
        uint32_t acc[HALF];
        tmem_ld_cols<HALF>(lane_base + Cfg::ACC0 + g * HALF, acc);
        tc_fence_before();
        mbar_arrive(smem_u32(&bar_acc_free));
        if (row < s.R) {
#pragma unroll
          for (int k = 0; k < HALF / 8; ++k) {
            float f[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) f[e] = __uint_as_float(acc[8 * k + e]) * s.scale;
            stg_v4(out0 + cell + g * HALF + 8 * k, pack8(f));
          }
        }
      } else {
        uint32_t acc[DH];  // warpgroup 0: dV = acc0; warpgroup 1: dK = scale * acc1
        tmem_ld_cols<DH>(lane_base + (g == 0 ? Cfg::ACC0 : Cfg::ACC1), acc);
        tc_fence_before();
        mbar_arrive(smem_u32(&bar_acc_free));
        if (row < s.R) {
          const float mul = row < it.n ? (g == 0 ? 1.f : s.scale) : 0.f;
          __nv_bfloat16* dst = (g == 0 ? out0 : out1) + cell;
#pragma unroll
          for (int k = 0; k < DH / 8; ++k) {
            float f[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) f[e] = row < it.n ? __uint_as_float(acc[8 * k + e]) * mul : 0.f;
            stg_v4(dst + 8 * k, pack8(f));
          }
        }
      }
      ++kitem;
      tbase += chunks;
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 10) tmem_dealloc(tmem, Cfg::COLS);
}

template <int DH>
cudaError_t launch_bwd(const Shape& s, const void* Q, const void* K, const void* V, const void* O, const void* dO,
                       const float* LSE, void* dQ, void* dK, void* dV, float* Dws, cudaStream_t stream) {
  using Cfg = BwdCfg<DH>;
  CUtensorMap q128, g128, k128, v128, q64, g64, k64, v64;
  bool ok = make_cell_tensor_map(&q128, Q, s.B, s.R, s.C, s.H, DH, kTileRows) &&
            make_cell_tensor_map(&g128, dO, s.B, s.R, s.C, s.H, DH, kTileRows) &&
            make_cell_tensor_map(&k128, K, s.B, s.R, s.C, s.H, DH, kTileRows) &&
            make_cell_tensor_map(&v128, V, s.B, s.R, s.C, s.H, DH, kTileRows) &&
            make_cell_tensor_map(&q64, Q, s.B, s.R, s.C, s.H, DH, kChunk) &&
            make_cell_tensor_map(&g64, dO, s.B, s.R, s.C, s.H, DH, kChunk) &&
            make_cell_tensor_map(&k64, K, s.B, s.R, s.C, s.H, DH, kChunk) &&
            make_cell_tensor_map(&v64, V, s.B, s.R, s.C, s.H, DH, kChunk);
  if (!ok) return cudaErrorInvalidValue;
  auto kq = item_bwd_tc_kernel<DH, MODE_DQ>;
  auto kkv = item_bwd_tc_kernel<DH, MODE_DKV>;
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(kq, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(kkv, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  const int bps = (s.R + kTileRows - 1) / kTileRows;
  const long long n_items = (long long)s.B * s.C * s.H * bps;
  const int grid = (int)std::min<long long>(n_items, num_sms());
  const __nv_bfloat16* Ob = (const __nv_bfloat16*)O;
  const __nv_bfloat16* dOb = (const __nv_bfloat16*)dO;
  kq<<<grid, kBwdThreads, Cfg::SMEM, stream>>>(q128, g128, k64, v64, s, Ob, dOb, LSE, Dws, (__nv_bfloat16*)dQ,
                                               nullptr, (int)n_items, bps);
  kkv<<<grid, kBwdThreads, Cfg::SMEM, stream>>>(k128, v128, q64, g64, s, Ob, dOb, LSE, Dws, (__nv_bfloat16*)dV,
                                                (__nv_bfloat16*)dK, (int)n_items, bps);
  count_launch(2);
  return cudaGetLastError();
}

}  // namespace

bool item_tc_bwd_supported(const Shape& s) { return s.dh == 16 || s.dh == 32 || s.dh == 64; }

cudaError_t launch_item_bwd_tc(const Shape& s, const void* Q, const void* K, const void* V, const void* O,
                               const void* dO, const float* LSE, void* dQ, void* dK, void* dV, float* Dws,
                               cudaStream_t stream) {
  switch (s.dh) {
    case 16: return launch_bwd<16>(s, Q, K, V, O, dO, LSE, dQ, dK, dV, Dws, stream);
    case 32: return launch_bwd<32>(s, Q, K, V, O, dO, LSE, dQ, dK, dV, Dws, stream);
    case 64: return launch_bwd<64>(s, Q, K, V, O, dO, LSE, dQ, dK, dV, Dws, stream);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace tabattn
