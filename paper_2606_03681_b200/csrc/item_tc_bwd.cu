// Item-axis attention backward on tcgen05: the dQ pass (which also
// computes D = rowsum(dO o O) and -LSE*log2(e) per query row and leaves them in the workspace) and
// the separate dK/dV pass -- one kernel template with two modes.  Deterministic: no atomics, every output
// element has exactly one writer.  (The split costs one extra exp and two extra tile-matmuls per
// (query, key) pair over a fused pass, but a fused pass must reduce dQ across key tiles with fp32
// atomics: at dh = 32/64 that is 8-16 B of L2 atomic traffic per 10*dh flops -- see DESIGN.md.)
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
// Warp roles (640 threads, one persistent CTA per SM; setmaxnreg gives the score warpgroups 104
// registers and leaves the issuing warps 64):
//   warps 0-15  four score warpgroups: wg & 1 = TMEM set (S, dP, dS, P) = chunk parity, wg >> 1 = which 32
//               of the chunk's 64 columns; one thread per (tile row, 32 columns).  Four score warps per
//               SM sub-partition instead of two: base bwd 1.92 -> 1.79 ms, ragged 8.26 -> 7.77 ms
//   warp 16     TMA producer (one lane): stationary tiles (double-buffered over items), ring of chunk
//               pairs (+ the chunk's LSE/D vectors by 1-D bulk copy in MODE_DKV)
//   warp 17     issuer of the score MMAs (S, dP), runs ahead of the accumulation as far as the two TMEM
//               sets allow; owns the TMEM allocation
//   warp 18     issuer of the acc0 MMAs (dQ or dV)
//   warp 19     MODE_DKV: issuer of the acc1 MMAs (dK).  MODE_DQ: row statistics -- D_i = sum_k dO_ik O_ik
//               from the item's dO tile and a TMA-staged O tile, -LSE_i*log2(e); handed to the score
//               warpgroups through shared memory one item ahead, and written to the workspace for the
//               dK/dV pass (this replaces a separate prep kernel: one pass less over O and dO)
// Every role walks the same item list with its own counters.  The issuing warps run convergently with a
// provably warp-uniform warp index, so ptxas keeps descriptors in uniform registers (~3 SASS instructions
// per tcgen05.mma; the earlier builds needed ~10-20 and were bound by the issue chain,
// profiles/r01_s14_item.md).
#include <cuda.h>

#include <algorithm>

#include "item_tc_common.cuh"
#include "kernels.h"

namespace tabattn {

TABATTN_TRACE_DEFINE(tabattn_debug_set_trace_item_bwd)

namespace {

int item_bwd_padded_rows(const Shape& s);

using namespace tc;
using namespace itc;

constexpr int MODE_DQ = 0, MODE_DKV = 1;
constexpr int kChunk = 64;
constexpr int kScoreWarps = 16;                       // four score warpgroups
constexpr int kBwdThreads = (kScoreWarps + 4) * 32;   // + producer, score issuer, two accumulation issuers
__host__ __device__ constexpr int kAccWarps(int mode) { return mode == 0 ? 1 : 2; }

template <int DH>
struct BwdCfg {
  static constexpr int ROWB = DH * 2;
  static constexpr int TILE_A = kTileRows * ROWB;  // stationary tile
  static constexpr int TILE_B = kChunk * ROWB;     // streamed chunk
  // chunk ring depth: as deep as shared memory allows at dh = 64 (8 stages, 196 KB); 16 at dh <= 32 (B200 sweep:
  // base bwd 1.451 / 1.436 / 1.414 / 1.404 / 1.418 ms at 6 / 8 / 12 / 16 / 20 stages, 1.586 at 4)
  // FOLD: `dP - D` is computed by the dP MMA itself (one extra k-step, see `D records` below) instead of a
  // subtraction per score element in the issue-bound score loops of dh <= 32 (profiles/r02_attention.md: issue
  // 76 % / 70 %, XU 56 % / 43 %).  At dh = 64 the tensor pipe is as busy as the MUFU and the loop is not issue-bound.
  static constexpr bool FOLD = DH <= 32;
  static constexpr int ST = DH >= 64 ? 8 : 12;
  static constexpr int LD_BYTES = 2 * kChunk * 4;  // per stage: lse2[64], D[64] (MODE_DKV; D unused with FOLD)
  static constexpr int STAGE = 2 * TILE_B;         // bytes of one ring stage (B1, B2)
  static constexpr int STAT_BYTES = 2 * 2 * kTileRows * 4;   // MODE_DQ: [2 item buffers][nlse2[128], D[128]]
  // D records (FOLD): one 32-byte row per query, (-D_hi, -D_lo, 0 x 14) bf16 in the 32-byte-swizzle K-major layout,
  // so that a [rows][16] tile of them is an MMA operand: against a tile of (1, 1, 0 x 14) rows the product is -D.
  static constexpr int REC = 32;
  static constexpr int ONES_BYTES = kTileRows * REC;                 // the (1, 1, 0...) operand
  static constexpr int DA_BYTES = 2 * kTileRows * REC;               // MODE_DQ: [2 item buffers][128 query rows]
  static constexpr int DB_BYTES = kChunk * REC;                      // MODE_DKV: per stage, the chunk's 64 queries
  static constexpr int FOLD_BYTES = FOLD ? ONES_BYTES + DA_BYTES + ST * DB_BYTES : 0;
  // (+ one O tile in MODE_DQ; sized for the larger of the two modes)
  static constexpr int SMEM = 4 * TILE_A + ST * (STAGE + LD_BYTES) + TILE_A + STAT_BYTES + FOLD_BYTES + 1024;
  // TMEM columns: set g at g*SET: S [0,64) dP [64,128) dS [128,160) P [160,192); accumulators after
  static constexpr int SET = 192, S_OFF = 0, DP_OFF = 64, DS_OFF = 128, P_OFF = 160;
  static constexpr int ACC0 = 384, ACC1 = 384 + DH, COLS = 512;
  static_assert(ACC1 + DH <= COLS, "TMEM budget");
  // pairs of every 8 whose exponential runs on the FMA pipe (exp2_poly2, common.cuh) instead of the MUFU
  static constexpr int POLY_OF_8 = DH >= 64 ? 0 : 1;
};

// One work item = (table b, column c, head h, 128-row block blk) of the stationary axis.
struct Item {
  int b, c, h, blk, n, chunks;
  bool valid;
};

template <int MODE, bool MASKED>
__device__ __forceinline__ Item decode_item(const Shape& s, const Meta& meta, const ColList<MASKED>& cl, int w, int bps) {
  Item it;
  const int rest = w / bps;
  // MODE_DKV: key blocks >= n_train are invalid (skipped).  With blk = w % bps a CTA (w = x + 148 k) would see
  // only a few residues of blk -- at bps = 8, n = 768 half of the CTAs get 50 % invalid items and the others
  // none (1.33x imbalance, base) -- so the block index is rotated by the sequence index.
  it.blk = MODE == MODE_DKV ? (w % bps + rest) % bps : w % bps;
  it.h = rest % s.H;
  const int bc = rest / s.H;          // (masked: the virtual column, an index into the list of valid pairs)
  if (cl.masked()) {
    cl.pair(bc, it.b, it.c);
  } else {
    it.b = bc / s.C;
    it.c = bc - it.b * s.C;
  }
  it.n = meta.n(s, it.b);
  it.valid = MODE == MODE_DQ || it.blk * kTileRows < it.n;
  it.chunks = ((MODE == MODE_DQ ? it.n : s.R) + kChunk - 1) / kChunk;
  return it;
}

// 1-D bulk copy global -> shared, completion on an mbarrier (bytes multiple of 16, both 16 B aligned)
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}

template <int DH, int MODE, bool MASKED>
__global__ void __launch_bounds__(kBwdThreads, 1)
item_bwd_tc_kernel(const __grid_constant__ CUtensorMap mapA1, const __grid_constant__ CUtensorMap mapA2,
                   const __grid_constant__ CUtensorMap mapB1, const __grid_constant__ CUtensorMap mapB2,
                   const __grid_constant__ CUtensorMap mapO, Shape s, const float* __restrict__ LSE,
                   float* lse2_ws, float* D_ws, uint4* Drec_ws, __nv_bfloat16* __restrict__ out0,
                   __nv_bfloat16* __restrict__ out1, const uint32_t* __restrict__ col_list, int n_items_all,
                   int blocks_per_seq, int Rp) {
  TR_INIT();
  using Cfg = BwdCfg<DH>;
  constexpr int ST = Cfg::ST, TILE_A = Cfg::TILE_A, TILE_B = Cfg::TILE_B, ROWB = Cfg::ROWB;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sA = sbase;                         // [2 item buffers][A1, A2][TILE_A]
  const uint32_t sB = sA + 4 * TILE_A;               // [ST][B1, B2][TILE_B]
  const uint32_t sLD = sB + ST * Cfg::STAGE;         // [ST][lse2[64], D[64]]
  const uint32_t sO = sLD + ST * Cfg::LD_BYTES;      // MODE_DQ: the item's O tile (single buffer)
  const uint32_t sStat = sO + TILE_A;                // MODE_DQ: [2][nlse2[128], D[128]]
  constexpr bool FOLD = Cfg::FOLD;
  const uint32_t sOnes = (sStat + Cfg::STAT_BYTES + 1023u) & ~1023u;   // FOLD: [128][32 B] rows (1, 1, 0...)
  const uint32_t sDA = sOnes + Cfg::ONES_BYTES;      // FOLD, MODE_DQ: [2][128][32 B] D records of the item's queries
  const uint32_t sDB = sDA + Cfg::DA_BYTES;          // FOLD, MODE_DKV: [ST][64][32 B] D records of the chunk's queries
  const float* sLD_ptr = reinterpret_cast<const float*>(smem_raw + (sLD - smem_u32(smem_raw)));
  float* sStat_ptr = reinterpret_cast<float*>(smem_raw + (sStat - smem_u32(smem_raw)));
  __shared__ uint64_t bar_a_full[2], bar_a_empty[2], bar_b_full[ST], bar_b_empty[ST];
  __shared__ uint64_t bar_o_full, bar_o_empty, bar_d_full[2], bar_d_empty[2];
  __shared__ uint64_t bar_s_full[2], bar_s_empty[2], bar_p_full[2], bar_p_empty[2], bar_acc_full, bar_acc_free;
  __shared__ uint32_t tmem_slot;
  __shared__ int32_t s_ntrain[kMetaTabs];
  __shared__ uint8_t s_colvalid[kMetaCells];
  Meta meta;
  meta.fill(s, s_ntrain, s_colvalid);
  ColList<MASKED> cl;
  cl.init(s, col_list);
  const int n_items = MASKED ? cl.nv * s.H * blocks_per_seq : n_items_all;   // (unmasked: a kernel parameter, uniform)

  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;  // provably warp-uniform
  if (warp == kScoreWarps + 1) tmem_alloc(smem_u32(&tmem_slot), Cfg::COLS);
  if (threadIdx.x == 0) {
    for (int i = 0; i < 2; ++i) {
      mbar_init(smem_u32(&bar_a_full[i]), 1);
      mbar_init(smem_u32(&bar_a_empty[i]), 1);
      mbar_init(smem_u32(&bar_s_full[i]), 1);
      mbar_init(smem_u32(&bar_s_empty[i]), 8);   // one arrive per warp of the set's two warpgroups
      mbar_init(smem_u32(&bar_p_full[i]), 8);
      mbar_init(smem_u32(&bar_p_empty[i]), kAccWarps(MODE));
      mbar_init(smem_u32(&bar_d_full[i]), 1);
      mbar_init(smem_u32(&bar_d_empty[i]), kScoreWarps);
    }
    mbar_init(smem_u32(&bar_o_full), 1);
    mbar_init(smem_u32(&bar_o_empty), 1);
    for (int i = 0; i < ST; ++i) {
      mbar_init(smem_u32(&bar_b_full[i]), 1);
      mbar_init(smem_u32(&bar_b_empty[i]), kAccWarps(MODE));
    }
    mbar_init(smem_u32(&bar_acc_full), kAccWarps(MODE));
    mbar_init(smem_u32(&bar_acc_free), (MODE == MODE_DQ && DH < 32) ? 8 : 16);   // warps that read the accumulators
    fence_barrier_init();
  }
  if (FOLD) {
    // the (1, 1, 0 x 14) rows: k = 0..7 sit in the 16-byte half selected by the 32-byte swizzle (bit 2 of the row)
    for (int r = threadIdx.x; r < kTileRows; r += blockDim.x) {
      const uint32_t sw = (r >> 2) & 1;
      sts_v4(sOnes + r * Cfg::REC + (sw << 4), 0x3F803F80u, 0u, 0u, 0u);
      sts_v4(sOnes + r * Cfg::REC + ((sw ^ 1) << 4), 0u, 0u, 0u, 0u);
    }
    fence_proxy_async_smem();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_slot;
  const int d = s.H * DH;
  // 640 threads start with 96 registers each; the score warpgroups take 104, the issuing warps keep 64
  // (setmaxnreg can only redistribute the 640 x 96 registers the CTA was launched with)
  if (warp >= kScoreWarps) {
  setmaxnreg_dec<64>();
  if (warp == kScoreWarps) {
    // ------------------------------------------------------------------ producer (one lane)
    if (lane == 0) {
      tma_prefetch_desc(&mapA1);
      tma_prefetch_desc(&mapA2);
      tma_prefetch_desc(&mapB1);
      tma_prefetch_desc(&mapB2);
      if (MODE == MODE_DQ) tma_prefetch_desc(&mapO);
      uint32_t t = 0, k = 0;
      for (int w = blockIdx.x; w < n_items; w += gridDim.x) {
        const Item it = decode_item<MODE, MASKED>(s, meta, cl, w, blocks_per_seq);
        if (!it.valid) continue;
        const uint32_t ab = k & 1, a_full = smem_u32(&bar_a_full[ab]);
        mbar_wait<true>(smem_u32(&bar_a_empty[ab]), ((k >> 1) & 1) ^ 1);
        mbar_arrive_expect_tx(a_full, 2 * TILE_A);
        tma_load_5d(sA + (2 * ab) * TILE_A, &mapA1, a_full, 0, it.h, it.c, it.blk * kTileRows, it.b);
        tma_load_5d(sA + (2 * ab + 1) * TILE_A, &mapA2, a_full, 0, it.h, it.c, it.blk * kTileRows, it.b);
        if (MODE == MODE_DQ) {
          // the item's O rows, for the stats warp (single buffer: it is read out right after it lands)
          mbar_wait<true>(smem_u32(&bar_o_empty), (k & 1) ^ 1);
          mbar_arrive_expect_tx(smem_u32(&bar_o_full), TILE_A);
          tma_load_5d(sO, &mapO, smem_u32(&bar_o_full), 0, it.h, it.c, it.blk * kTileRows, it.b);
        }
        const size_t seq = (((size_t)it.b * s.C + it.c) * s.H + it.h) * Rp;
        for (int j = 0; j < it.chunks; ++j, ++t) {
          const uint32_t st = t % ST, b_full = smem_u32(&bar_b_full[st]);
          mbar_wait<true>(smem_u32(&bar_b_empty[st]), ((t / ST) & 1) ^ 1);
          mbar_arrive_expect_tx(b_full, Cfg::STAGE + (MODE == MODE_DKV ? (FOLD ? kChunk * 4 + Cfg::DB_BYTES : Cfg::LD_BYTES) : 0));
          tma_load_5d(sB + st * Cfg::STAGE, &mapB1, b_full, 0, it.h, it.c, j * kChunk, it.b);
          tma_load_5d(sB + st * Cfg::STAGE + TILE_B, &mapB2, b_full, 0, it.h, it.c, j * kChunk, it.b);
          if (MODE == MODE_DKV) {
            bulk_load(sLD + st * Cfg::LD_BYTES, lse2_ws + seq + j * kChunk, kChunk * 4, b_full);
            if (FOLD) bulk_load(sDB + st * Cfg::DB_BYTES, Drec_ws + 2 * (seq + j * kChunk), Cfg::DB_BYTES, b_full);
            else bulk_load(sLD + st * Cfg::LD_BYTES + kChunk * 4, D_ws + seq + j * kChunk, kChunk * 4, b_full);
          }
        }
        ++k;
      }
    }
  } else if (warp == kScoreWarps + 1) {
    // ------------------------------------------------------------------ score MMAs (S, dP)
    // Chunk t of the CTA's lifetime uses TMEM set t & 1 and ring stage t % ST.  The warp walks its loop
    // convergently (elect.sync inside every issue; `warp` is provably uniform, so ptxas keeps the
    // descriptors in uniform registers: ~3 SASS instructions per tcgen05.mma, profiles/r01_s14_item.md).
    constexpr uint32_t idesc = make_idesc_bf16(128, kChunk, false, false);
    const uint64_t dA = make_smem_desc<ROWB>(sA, 16, 8 * ROWB);
    const uint64_t dB = make_smem_desc<ROWB>(sB, 16, 8 * ROWB);
    const uint64_t dOnes = make_smem_desc<32>(sOnes, 16, 256), dRecA = make_smem_desc<32>(sDA, 16, 256),
                   dRecB = make_smem_desc<32>(sDB, 16, 256);
    const uint32_t b_a_full = smem_u32(&bar_a_full[0]), b_a_empty = smem_u32(&bar_a_empty[0]),
                   b_b_full = smem_u32(&bar_b_full[0]), b_s_full = smem_u32(&bar_s_full[0]),
                   b_s_empty = smem_u32(&bar_s_empty[0]);
    uint32_t t = 0, k = 0, st = 0, ph = 0;
    for (int w = blockIdx.x; w < n_items; w += gridDim.x) {
      const Item it = decode_item<MODE, MASKED>(s, meta, cl, w, blocks_per_seq);
      if (!it.valid) continue;
      const uint32_t ab = k & 1;
      mbar_wait(b_a_full + 8 * ab, (k >> 1) & 1);
      // FOLD, dQ pass: the item's D records (written by the statistics warp) are the A operand of the extra k-step
      if (FOLD && MODE == MODE_DQ) mbar_wait(smem_u32(&bar_d_full[ab]), (k >> 1) & 1);
      const uint64_t a1 = dA + ((2 * ab) * TILE_A >> 4), a2 = a1 + (TILE_A >> 4);
      for (int j = 0; j < it.chunks; ++j, ++t) {
        const uint32_t g = t & 1;
        mbar_wait(b_b_full + 8 * st, ph);
        if (lane == 0 && g == 0 && (t >> 1) < 32) TR(10, (int)(t >> 1) + 32 * MODE);   // chunk landed
        if (MODE == MODE_DQ) {
          // keys >= n must not reach dQ through dS K: zero the K rows beyond n (dS is forced to 0 there,
          // but 0 x NaN would still be NaN).  Ordered before the accumulation MMAs of this chunk through
          // S MMA -> bar_s_full -> score warpgroups -> bar_p_full.
          const int rem = it.n - j * kChunk;
          if (rem < kChunk) zero_tail_rows<ROWB, kChunk>(sB + st * Cfg::STAGE, rem, lane);
        }
        mbar_wait(b_s_empty + 8 * g, ((t >> 1) & 1) ^ 1);
        if (lane == 0 && g == 0 && (t >> 1) < 32) TR(11, (int)(t >> 1) + 32 * MODE);   // set free
        tc_fence_after();
        const uint32_t set = tmem + g * Cfg::SET;
        const uint64_t b1 = dB + (st * Cfg::STAGE >> 4), b2 = b1 + (TILE_B >> 4);
#pragma unroll
        for (int kk = 0; kk < DH / 16; ++kk) mma_ss_e(set + Cfg::S_OFF, a1 + 2 * kk, b1 + 2 * kk, idesc, kk > 0);
#pragma unroll
        for (int kk = 0; kk < DH / 16; ++kk) mma_ss_e(set + Cfg::DP_OFF, a2 + 2 * kk, b2 + 2 * kk, idesc, kk > 0);
        if (FOLD) {
          // dP -= D: (-D_hi, -D_lo) of the row (dQ pass: queries are rows) or of the column (dK/dV pass) times (1, 1)
          if (MODE == MODE_DQ) mma_ss_e(set + Cfg::DP_OFF, dRecA + (ab * (kTileRows * Cfg::REC) >> 4), dOnes, idesc, 1u);
          else mma_ss_e(set + Cfg::DP_OFF, dOnes, dRecB + (st * Cfg::DB_BYTES >> 4), idesc, 1u);
        }
        tc_commit_e(b_s_full + 8 * g);
        if (lane == 0 && g == 0 && (t >> 1) < 32) TR(12, (int)(t >> 1) + 32 * MODE);   // S / dP issued
        if (j == it.chunks - 1) tc_commit_e(b_a_empty + 8 * ab);
        if (++st == ST) { st = 0; ph ^= 1; }
      }
      ++k;
    }
  } else if (warp == kScoreWarps + 2 || (warp == kScoreWarps + 3 && MODE == MODE_DKV)) {
    // ------------------------------------------------------------------ accumulation MMAs
    // first warp: acc0 (dQ += dS K, or dV += P^T dO); second warp (MODE_DKV): acc1 (dK += dS^T Q)
    constexpr uint32_t idesc = make_idesc_bf16(128, DH, false, true);
    const bool first = warp == kScoreWarps + 2;
    // A = 128 x 64 bf16 in TMEM (8 columns per 16-wide k step); B = 16 chunk rows per k step
    const uint32_t acol = (MODE == MODE_DQ || !first) ? Cfg::DS_OFF : Cfg::P_OFF;
    const uint32_t acc = tmem + (first ? Cfg::ACC0 : Cfg::ACC1);
    // B operand: dQ <- K chunk (B1); dV <- dO chunk (B2); dK <- Q chunk (B1)
    const uint64_t dB = make_smem_desc<ROWB>(sB + ((MODE == MODE_DKV && first) ? TILE_B : 0), 16, 8 * ROWB);
    const uint32_t b_p_full = smem_u32(&bar_p_full[0]), b_p_empty = smem_u32(&bar_p_empty[0]),
                   b_b_empty = smem_u32(&bar_b_empty[0]);
    uint32_t t = 0, k = 0, st = 0;
    for (int w = blockIdx.x; w < n_items; w += gridDim.x) {
      const Item it = decode_item<MODE, MASKED>(s, meta, cl, w, blocks_per_seq);
      if (!it.valid) continue;
      mbar_wait(smem_u32(&bar_acc_free), (k & 1) ^ 1);
      for (int j = 0; j < it.chunks; ++j, ++t) {
        const uint32_t g = t & 1;
        mbar_wait(b_p_full + 8 * g, (t >> 1) & 1);
        tc_fence_after();
        const uint32_t a = tmem + g * Cfg::SET + acol;
        const uint64_t b = dB + (st * Cfg::STAGE >> 4);
#pragma unroll
        for (int kk = 0; kk < kChunk / 16; ++kk)
          mma_ts_e(acc, a + 8 * kk, b + kk * ROWB, idesc, (j > 0 || kk > 0) ? 1u : 0u);
        tc_commit_e(b_p_empty + 8 * g);
        tc_commit_e(b_b_empty + 8 * st);
        if (j == it.chunks - 1) tc_commit_e(smem_u32(&bar_acc_full));
        if (++st == ST) st = 0;
      }
      ++k;
    }
  } else if (MODE == MODE_DQ && warp == kScoreWarps + 3) {
    // ------------------------------------------------------------------ row statistics (MODE_DQ)
    // D_i = sum_k dO_ik O_ik over the item's 128 query rows, from the dO tile (A2) and the O tile in shared
    // memory: both tiles carry the same swizzle, so equal physical 16-byte chunks hold equal logical ones and
    // the dot product needs no address arithmetic.  CH lanes share a row; rows >= R were zero-filled by the
    // TMA (D = 0) and get nlse2 = -inf (P = 0).  Runs one item ahead of the score warpgroups.
    constexpr int CH = DH / 8, RPI = 32 / CH;   // 16-byte chunks per row, rows per warp iteration
    const int sub = lane / CH, ch = lane % CH;
    uint32_t k = 0;
    for (int w = blockIdx.x; w < n_items; w += gridDim.x) {
      const Item it = decode_item<MODE, MASKED>(s, meta, cl, w, blocks_per_seq);
      if (!it.valid) continue;
      const uint32_t ab = k & 1;
      const size_t seq = ((size_t)it.b * s.C + it.c) * s.H + it.h;
      float l[4];
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int row = it.blk * kTileRows + lane + 32 * q;
        l[q] = row < s.R ? __ldg(LSE + seq * s.R + row) : INFINITY;
      }
      mbar_wait(smem_u32(&bar_a_full[ab]), (k >> 1) & 1);
      mbar_wait(smem_u32(&bar_o_full), k & 1);
      mbar_wait(smem_u32(&bar_d_empty[ab]), ((k >> 1) & 1) ^ 1);
      float* st = sStat_ptr + ab * (2 * kTileRows);
      const uint32_t tG = sA + (2 * ab + 1) * TILE_A + ch * 16, tO = sO + ch * 16;
#pragma unroll 4
      for (int r0 = 0; r0 < kTileRows; r0 += RPI) {
        const int row = r0 + sub;
        float fo[8], fg[8];
        unpack8(lds_v4(tO + row * ROWB), fo);
        unpack8(lds_v4(tG + row * ROWB), fg);
        float a = 0.f;
#pragma unroll
        for (int e = 0; e < 8; ++e) a = fmaf(fo[e], fg[e], a);
#pragma unroll
        for (int o = 1; o < CH; o <<= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
        if (ch == 0) st[kTileRows + row] = a;
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&bar_o_empty));
#pragma unroll
      for (int q = 0; q < 4; ++q) st[lane + 32 * q] = -l[q] * kLog2e;
      __syncwarp();
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int rr = lane + 32 * q, row = it.blk * kTileRows + rr;
        const float Dv = st[kTileRows + rr];
        if (FOLD) {
          // -D as two bf16 (hi + lo carries 16 mantissa bits), in the half of the 32-byte row the swizzle selects
          const uint32_t hi = pack_bf16(-Dv, 0.f) & 0xffffu;
          const uint32_t lo = pack_bf16(-Dv - bf16lo(hi), 0.f) & 0xffffu;
          const uint32_t sw = (rr >> 2) & 1;
          sts_v4(sDA + ab * (kTileRows * Cfg::REC) + rr * Cfg::REC + (sw << 4), hi | (lo << 16), 0u, 0u, 0u);
          sts_v4(sDA + ab * (kTileRows * Cfg::REC) + rr * Cfg::REC + ((sw ^ 1) << 4), 0u, 0u, 0u, 0u);
          if (row < Rp) {
            uint4* rec = Drec_ws + 2 * (seq * Rp + row);
            rec[sw] = make_uint4(hi | (lo << 16), 0u, 0u, 0u);
            rec[sw ^ 1] = make_uint4(0u, 0u, 0u, 0u);
          }
        }
        if (row < Rp) {
          lse2_ws[seq * Rp + row] = st[rr];
          if (!FOLD) D_ws[seq * Rp + row] = Dv;
        }
      }
      if (FOLD) fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&bar_d_full[ab]));
      ++k;
    }
  }
  } else {
    // -------------------------------------------------------------------- score warpgroups
    // Four warpgroups: wg = warp >> 2; set g = wg & 1 (TMEM set / chunk parity), column half c = wg >> 1:
    // the two warpgroups of a set split the chunk's 64 columns, one thread per (tile row, 32 columns).
    // Four instead of two score warps per SM sub-partition hide each other's MUFU / FMA latencies.
    setmaxnreg_inc<104>();
    const int g = (warp >> 2) & 1, c = warp >> 3;
    const int r = threadIdx.x & 127;         // tile row = TMEM lane
    const uint32_t lane_base = tmem + ((uint32_t)(32 * (warp & 3)) << 16);
    const uint32_t set = lane_base + g * Cfg::SET;
    const uint32_t b_s_full = smem_u32(&bar_s_full[g]), b_s_empty = smem_u32(&bar_s_empty[g]),
                   b_p_full = smem_u32(&bar_p_full[g]), b_p_empty = smem_u32(&bar_p_empty[g]);
    const float c2 = s.scale * kLog2e;
    uint32_t kitem = 0;   // valid items seen
    uint32_t tbase = 0;   // chunks of all previous valid items (ring position)
    // ---- epilogue of one item (accumulators -> global), as a deferred step: it runs after the warpgroup's first
    // chunk of the NEXT item, so that the wait for the item's last accumulation MMAs (bar_acc_full) is covered
    // by that chunk's arithmetic instead of idling at every item boundary.
    auto epilogue = [&](size_t e_cell, int e_row, int e_n, uint32_t e_par) {
        if (MODE == MODE_DQ) {
          // the dQ columns of a row are split over the four warpgroups (two at dh = 16: 16-byte stores)
          constexpr int EPW = DH >= 32 ? 4 : 2, PART = DH / EPW;
          const int q = g + 2 * c;
          if (q < EPW) {
            mbar_wait(smem_u32(&bar_acc_full), e_par);
            tc_fence_after();
            uint32_t acc[PART];
            tmem_ld_cols<PART>(lane_base + Cfg::ACC0 + q * PART, acc);
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&bar_acc_free));
            if (e_row < s.R) {
  #pragma unroll
              for (int k = 0; k < PART / 8; ++k) {
                float f[8];
  #pragma unroll
                for (int e = 0; e < 8; ++e) f[e] = __uint_as_float(acc[8 * k + e]) * s.scale;
                stg_v4(out0 + e_cell + q * PART + 8 * k, pack8(f));
              }
            }
          }
        } else {
          // set 0 warpgroups: dV = acc0; set 1 warpgroups: dK = scale * acc1; column half c each
          constexpr int HALF = DH / 2;
          mbar_wait(smem_u32(&bar_acc_full), e_par);
          tc_fence_after();
          uint32_t acc[HALF];
          tmem_ld_cols<HALF>(lane_base + (g == 0 ? Cfg::ACC0 : Cfg::ACC1) + c * HALF, acc);
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(smem_u32(&bar_acc_free));
          if (e_row < s.R) {
            const float mul = g == 0 ? 1.f : s.scale;
            __nv_bfloat16* dst = (g == 0 ? out0 : out1) + e_cell + c * HALF;
  #pragma unroll
            for (int k = 0; k < HALF / 8; ++k) {
              float f[8];
  #pragma unroll
              for (int e = 0; e < 8; ++e) f[e] = e_row < e_n ? __uint_as_float(acc[8 * k + e]) * mul : 0.f;
              stg_v4(dst + 8 * k, pack8(f));
            }
          }
        }
    };
    // a6: the invalid columns (masked tables) are dealt to the CTAs like the items (dQ, or dK and dV, := +0); a CTA
    // clears one invalid item after every item it walks, so the stores spread over the kernel
    const int n_zero = MASKED ? cl.ni * s.H * blocks_per_seq : 0;
    int wz = blockIdx.x;
    auto zero_one = [&]() {
      const int blk = wz % blocks_per_seq, seq = wz / blocks_per_seq, h = seq % s.H;
      int b, cc;
      cl.pair(cl.nv + seq / s.H, b, cc);
      const int row = blk * kTileRows + r;
      if (row < s.R && c == 0) {
        const size_t cell = (((size_t)b * s.R + row) * s.C + cc) * d + (size_t)h * DH;
        if (MODE == MODE_DQ) {
#pragma unroll
          for (int k = 0; k < DH / 16; ++k) stg_v4(out0 + cell + g * (DH / 2) + 8 * k, make_uint4(0, 0, 0, 0));
        } else {
          __nv_bfloat16* dst = (g == 0 ? out0 : out1) + cell;
#pragma unroll
          for (int k = 0; k < DH / 8; ++k) stg_v4(dst + 8 * k, make_uint4(0, 0, 0, 0));
        }
      }
      wz += gridDim.x;
    };
    bool pend = false;
    size_t p_cell = 0;
    int p_row = 0, p_n = 0;
    uint32_t p_par = 0;
    for (int w = blockIdx.x; w < n_items; w += gridDim.x) {
      const Item it = decode_item<MODE, MASKED>(s, meta, cl, w, blocks_per_seq);
      const int row = it.blk * kTileRows + r;
      const size_t cell = (((size_t)it.b * s.R + row) * s.C + it.c) * d + (size_t)it.h * DH;
      if (MASKED && wz < n_zero) zero_one();
      if (!it.valid) {
        // invalid column, or (MODE_DKV) a key block entirely beyond the train rows: zeros
        if (row < s.R && c == 0) {
          if (MODE == MODE_DQ) {
#pragma unroll
            for (int k = 0; k < DH / 16; ++k) stg_v4(out0 + cell + g * (DH / 2) + 8 * k, make_uint4(0, 0, 0, 0));
          } else {
            __nv_bfloat16* dst = (g == 0 ? out0 : out1) + cell;
#pragma unroll
            for (int k = 0; k < DH / 8; ++k) stg_v4(dst + 8 * k, make_uint4(0, 0, 0, 0));
          }
        }
        continue;
      }
      const int tfirst = (int)((tbase + ((g ^ tbase) & 1)) >> 1) + 32 * MODE;   // (trace slot of the item's first chunk)
      if (threadIdx.x == 0 && tfirst - 32 * MODE < 32) TR(13, tfirst);   // item decoded
      // per-row constants of the dQ pass, from the stats warp (rows >= R: nlse2 = -inf -> P = 0)
      float nlse2 = -INFINITY, Drow = 0.f;
      if (MODE == MODE_DQ) {
        const uint32_t db = kitem & 1;
        mbar_wait(smem_u32(&bar_d_full[db]), (kitem >> 1) & 1);
        nlse2 = sStat_ptr[db * (2 * kTileRows) + r];
        Drow = sStat_ptr[db * (2 * kTileRows) + kTileRows + r];
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&bar_d_empty[db]));
      }
      if (threadIdx.x == 0 && tfirst - 32 * MODE < 32) TR(14, tfirst);   // row statistics read
      const uint64_t nl = f2pack(nlse2, nlse2), dd = f2pack(Drow, Drow);
      const int chunks = it.chunks;
      for (int j = (g ^ tbase) & 1; j < chunks; j += 2) {
        const uint32_t u = (tbase + j) >> 1;  // this set's chunk counter
        mbar_wait(b_s_full, u & 1);
        const int tbv = 5 * (g + 2 * c), tst = (int)u + 32 * MODE;   // (trace slots)
        if (r == 0 && u < 32 && tbv < 10) TR(tbv + 0, tst);     // S / dP ready
        if (r == 0 && u < 32 && tbv == 0) TR(15, tst);          // (calibration: cost of one stamp)
        tc_fence_after();
        uint32_t sr[32], dr[32];
        tmem_ld32(set + Cfg::S_OFF + 32 * c, sr);
        tmem_ld32(set + Cfg::DP_OFF + 32 * c, dr);
        tmem_wait_ld();
        tc_fence_before();
        __syncwarp();
        // Release the set's S/dP columns.  At dh = 64 the next S/dP MMAs (256 tensor clk) are on the critical
        // chain, so the arithmetic is made to depend on the arrive (mbar_arrive_then: long_item bwd 7.52 ->
        // 7.28 ms); at dh <= 32 they are not, and letting ptxas overlap the arithmetic on S with the dP load
        // is worth more (base bwd 1.56 against 1.63 ms).
        float c2d = c2;
        if constexpr (DH >= 64) c2d = mbar_arrive_then(b_s_empty, lane == 0, c2);
        else if (lane == 0) mbar_arrive(b_s_empty);
        if (r == 0 && u < 32 && tbv < 10) TR(tbv + 1, tst);     // S / dP loaded, set released
        const uint64_t cc = f2pack(c2d, c2d);
        uint32_t pds[16], pp[16];
        if (MODE == MODE_DQ) {
          // P = 2^(S*c2 - lse2), dS = P o (dP - D) on packed fp32 pairs
#pragma unroll
          for (int k = 0; k < 16; ++k) {
            const uint64_t x = fma2(f2pack(__uint_as_float(sr[2 * k]), __uint_as_float(sr[2 * k + 1])), cc, nl);
            float p0, p1, d0, d1;
            exp2_pair(pair_is_poly<Cfg::POLY_OF_8>(k), x, p0, p1);
            uint64_t dpd = f2pack(__uint_as_float(dr[2 * k]), __uint_as_float(dr[2 * k + 1]));
            if (!FOLD) dpd = sub2(dpd, dd);
            f2unpack(mul2(f2pack(p0, p1), dpd), d0, d1);
            pds[k] = pack_bf16(d0, d1);
          }
          const int rem = it.n - j * kChunk - 32 * c;
          if (rem < 32) {  // last chunk only: keys >= n_train get dS = 0 exactly, whatever the masked K/V hold
#pragma unroll
            for (int k = 0; k < 16; ++k) {
              const uint32_t keep = (2 * k < rem ? 0x0000ffffu : 0u) | (2 * k + 1 < rem ? 0xffff0000u : 0u);
              pds[k] &= keep;
            }
          }
        } else {
          const uint32_t st = (tbase + j) % ST;
          // the chunk's LSE/D vectors landed with the chunk (same mbarrier as the score MMAs waited on)
          mbar_wait(smem_u32(&bar_b_full[st]), ((tbase + j) / ST) & 1);
          const ulonglong2* l4 = reinterpret_cast<const ulonglong2*>(sLD_ptr + st * (2 * kChunk)) + 8 * c;
          const ulonglong2* d4 = l4 + kChunk / 4;
#pragma unroll
          for (int k = 0; k < 32; k += 4) {
            const ulonglong2 L = l4[k >> 2];  // (nlse2, D) of query columns 32c + k .. k+3
            ulonglong2 Dv = make_ulonglong2(0ull, 0ull);
            if (!FOLD) Dv = d4[k >> 2];
            float p0, p1, p2, p3, d0, d1, d2, d3;
            const uint64_t xa = fma2(f2pack(__uint_as_float(sr[k]), __uint_as_float(sr[k + 1])), cc, L.x);
            const uint64_t xb = fma2(f2pack(__uint_as_float(sr[k + 2]), __uint_as_float(sr[k + 3])), cc, L.y);
            exp2_pair(pair_is_poly<Cfg::POLY_OF_8>(k >> 1), xa, p0, p1);
            exp2_pair(pair_is_poly<Cfg::POLY_OF_8>((k >> 1) + 1), xb, p2, p3);
            pp[k >> 1] = pack_bf16(p0, p1);
            pp[(k >> 1) + 1] = pack_bf16(p2, p3);
            uint64_t da = f2pack(__uint_as_float(dr[k]), __uint_as_float(dr[k + 1]));
            uint64_t db = f2pack(__uint_as_float(dr[k + 2]), __uint_as_float(dr[k + 3]));
            if (!FOLD) {
              da = sub2(da, Dv.x);
              db = sub2(db, Dv.y);
            }
            f2unpack(mul2(f2pack(p0, p1), da), d0, d1);
            f2unpack(mul2(f2pack(p2, p3), db), d2, d3);
            pds[k >> 1] = pack_bf16(d0, d1);
            pds[(k >> 1) + 1] = pack_bf16(d2, d3);
          }
        }
        if (r == 0 && u < 32 && tbv < 10) TR(tbv + 2, tst);     // arithmetic done
        mbar_wait(b_p_empty, (u & 1) ^ 1);  // the MMAs that read this set's previous P/dS are done
        if (r == 0 && u < 32 && tbv < 10) TR(tbv + 3, tst);     // P / dS columns free
        tmem_st16(set + Cfg::DS_OFF + 16 * c, pds);
        if (MODE == MODE_DKV) tmem_st16(set + Cfg::P_OFF + 16 * c, pp);
        tmem_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(b_p_full);
        if (r == 0 && u < 32 && tbv < 10) TR(tbv + 4, tst);     // P / dS stored
        if (pend) {
          epilogue(p_cell, p_row, p_n, p_par);
          pend = false;
        }
      }
      // the epilogue of this item is deferred (see `epilogue` above)
      if (pend) epilogue(p_cell, p_row, p_n, p_par);   // (no chunk of the item was ours)
      pend = true; p_cell = cell; p_row = row; p_n = it.n; p_par = kitem & 1;
      ++kitem;
      tbase += chunks;
    }
    if (pend) epilogue(p_cell, p_row, p_n, p_par);
    while (MASKED && wz < n_zero) zero_one();   // (what is left of the invalid columns)
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kScoreWarps + 1) tmem_dealloc(tmem, Cfg::COLS);
}

template <int DH>
cudaError_t launch_bwd(const Shape& s, const void* Q, const void* K, const void* V, const void* O, const void* dO,
                       const float* LSE, void* dQ, void* dK, void* dV, float* ws, cudaStream_t stream) {
  using Cfg = BwdCfg<DH>;
  const DeviceInfo* di = current_device();
  if (!di) return cudaErrorInvalidDevice;
  CUtensorMap q128, g128, o128, k128, v128, q64, g64, k64, v64;
  auto map = [&](CUtensorMap* m, const void* base, int rows) {
    return get_tensor_map(m, 0, base, s.B, s.R, s.C, s.H, DH, rows, 1);
  };
  const bool ok = map(&q128, Q, kTileRows) && map(&g128, dO, kTileRows) && map(&o128, O, kTileRows) &&
                  map(&k128, K, kTileRows) && map(&v128, V, kTileRows) && map(&q64, Q, kChunk) &&
                  map(&g64, dO, kChunk) && map(&k64, K, kChunk) && map(&v64, V, kChunk);
  if (!ok) return cudaErrorInvalidValue;
  const bool masked = s.col_valid != nullptr;
  auto kq = masked ? item_bwd_tc_kernel<DH, MODE_DQ, true> : item_bwd_tc_kernel<DH, MODE_DQ, false>;
  auto kkv = masked ? item_bwd_tc_kernel<DH, MODE_DKV, true> : item_bwd_tc_kernel<DH, MODE_DKV, false>;
  static SmemAttr attr_q[2], attr_kv[2];
  cudaError_t e = attr_q[masked].ensure(kq, Cfg::SMEM, di->ordinal);
  if (e == cudaSuccess) e = attr_kv[masked].ensure(kkv, Cfg::SMEM, di->ordinal);
  if (e != cudaSuccess) return e;
  const int Rp = item_bwd_padded_rows(s);
  float* lse2_ws = ws;
  float* D_ws = ws + (size_t)s.B * s.C * s.H * Rp;            // fp32 D per row (dh = 64) ...
  uint4* Drec_ws = reinterpret_cast<uint4*>(D_ws);            // ... or one 32-byte D record per row (dh <= 32)
  const int bps = (s.R + kTileRows - 1) / kTileRows;
  const long long n_items = (long long)s.B * s.C * s.H * bps;   // (upper bound: masked tables walk the valid pairs only)
  const int grid = (int)std::min<long long>(n_items, di->num_sms);
  // a0: the column list sits behind the row statistics in the workspace
  const size_t stat_bytes = (size_t)s.B * s.C * s.H * Rp * (sizeof(float) + (s.dh <= 32 ? 32 : sizeof(float)));
  const uint32_t* list = item_build_list(s, reinterpret_cast<char*>(ws) + stat_bytes, stream);
  kq<<<grid, kBwdThreads, Cfg::SMEM, stream>>>(q128, g128, k64, v64, o128, s, LSE, lse2_ws, D_ws, Drec_ws,
                                               (__nv_bfloat16*)dQ, nullptr, list, (int)n_items, bps, Rp);
  kkv<<<grid, kBwdThreads, Cfg::SMEM, stream>>>(k128, v128, q64, g64, o128, s, LSE, lse2_ws, D_ws, Drec_ws,
                                                (__nv_bfloat16*)dV, (__nv_bfloat16*)dK, list, (int)n_items, bps, Rp);
  count_launch(2);
  return cudaGetLastError();
}

// rows of the per-sequence LSE/D workspace vectors: R rounded up to the 64-row chunk, so that every
// chunk's vectors are one aligned 256-byte bulk copy
int item_bwd_padded_rows(const Shape& s) { return (s.R + kChunk - 1) / kChunk * kChunk; }

}  // namespace

size_t item_bwd_workspace_bytes(const Shape& s) {
  // per query row: -LSE log2(e) as f32, and D as f32 (dh = 64) or as a 32-byte operand record (dh <= 32, BwdCfg::FOLD)
  const size_t per_row = sizeof(float) + (s.dh <= 32 ? 32 : sizeof(float));
  return (size_t)s.B * s.C * s.H * item_bwd_padded_rows(s) * per_row + item_list_bytes(s);
}

cudaError_t launch_item_bwd(const Shape& s, const void* Q, const void* K, const void* V, const void* O,
                            const void* dO, const float* LSE, void* dQ, void* dK, void* dV, float* ws,
                            cudaStream_t stream) {
  switch (s.dh) {
    case 16: return launch_bwd<16>(s, Q, K, V, O, dO, LSE, dQ, dK, dV, ws, stream);
    case 32: return launch_bwd<32>(s, Q, K, V, O, dO, LSE, dQ, dK, dV, ws, stream);
    case 64: return launch_bwd<64>(s, Q, K, V, O, dO, LSE, dQ, dK, dV, ws, stream);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace tabattn
