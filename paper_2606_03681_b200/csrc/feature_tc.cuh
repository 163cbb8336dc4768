// Shared pieces of the tcgen05 feature-axis kernels (feature_tc_fwd.cu, feature_tc_bwd.cu).
//
// Packing.  The feature axis is short (Cv <= 128 valid columns), so one
// 128-row tcgen05 tile holds SEVERAL table rows of one head: every table row takes Cp slots, Cp = the
// power of two >= max(Cv, 16), and a tile = RPT = 128 / Cp consecutive table rows:
//     slot = rl * Cp + v          rl = row inside the tile, v = rank of the column among the valid ones
// S = Q K^T of the whole tile is one 128 x 128 x dh MMA; only its RPT diagonal Cp x Cp blocks mean
// anything.  The off-diagonal blocks and the pad slots (v >= Cv) are pushed to -2^100 INSIDE the MMA by
// one extra k-step against two small "mask" operands (Q'[i][blk_i] = 1, K'[j][k] = 0 if k = blk_j and
// v_j < Cv, else -2^100), so the softmax threads spend no instruction on masking and exp2 gives exactly 0
// there.  A softmax thread owns one slot (one TMEM lane) and reads only the W = max(Cp, 32) score columns
// around its own block.  The tensor pipe is < 5 % busy on this axis, so the wasted off-diagonal flops are
// free; what the packing buys is ~100 instead of ~460-930 warp instructions per (row, head) and bulk
// TMA traffic, i.e. a kernel that is HBM-bound instead of issue-bound (profiles/r02_attention.md).
//
// Unmasked tables are one "virtual table" of B*R rows (every row has the same columns), fetched and
// stored by 4-D TMA boxes (dh, 1 head, Cp columns, RPT rows): columns >= C are zero-filled on load and
// clipped on store.  Masked tables (col_valid != NULL) are compacted: a small prep kernel (a0) builds,
// per table, Cv, Cp, the table's tile range and the list of valid columns; producer warps gather only
// the valid cells with 16-byte cp.async, so invalid columns cost no DRAM read and NaNs there cannot leak.
#pragma once
#include "common.cuh"
#include "tc_common.cuh"

namespace tabattn {
namespace ftc {

using namespace tc;

constexpr int kSlots = 128;           // rows of every operand tile (UMMA M and N of the score tile)
constexpr uint32_t kNegBig = 0xF180u; // bf16 -2^100: the mask bias (finite: 0 * it = -0, it + s = it)
constexpr uint32_t kOne = 0x3F80u;    // bf16 1.0
constexpr int kMaskTile = kSlots * 32; // bytes of one mask operand: [128][16] bf16, 32-byte rows

// Per-table geometry.  Unmasked: one virtual table; masked: written by feature_prep_kernel.
struct __align__(16) FeatTab {
  int32_t Cv;     // valid columns
  int32_t lgCp;   // log2 of the slots per table row (4..7)
  int32_t tile0;  // first tile of the table (tiles = row groups x heads, head fastest)
  int32_t tile1;  // one past the last tile
};

struct FeatParams {
  Shape s;
  int masked;           // 0: one virtual table of B*R rows with all C columns valid
  int nTab, Rt;         // tables and rows per table as the kernel sees them
  FeatTab uni;          // unmasked geometry
  int n_tiles;          // unmasked tile count
  const FeatTab* tabs;  // masked: [B]                       (workspace)
  const uint8_t* vcol;  // masked: [B][128] valid columns ascending, then the invalid ones ascending
  const int32_t* total; // masked: total tile count
};

struct Tile {
  int b, h, row0, nrows, Cv, lgCp;   // row0 is table-local; nrows <= RPT real rows in the tile
};

// Every role walks the same tile list t = blockIdx.x, += gridDim.x.  Tables ascend with t, so the table
// record is advanced incrementally, and (row group, head) of the tile inside its table are kept by
// carries instead of a division per tile (eight softmax warps walk every tile).
struct TileWalk {
  int t, b, total;
  int rg, h;        // tile inside the current table: local = rg * H + h
  int step, d_rg, d_h;   // tiles per step = d_rg * H + d_h
  FeatTab tb;
  // first tile = blockIdx.x + first * gridDim.x, step = every * gridDim.x tiles
  __device__ __forceinline__ void init(const FeatParams& p, int first = 0, int every = 1) {
    const int G = every * (int)gridDim.x;
    t = blockIdx.x + first * (int)gridDim.x;
    b = 0;
    if (p.masked) {
      total = __ldg(p.total);
      tb = *reinterpret_cast<const FeatTab*>(p.tabs);
    } else {
      total = p.n_tiles;
      tb = p.uni;
    }
    step = G;
    d_rg = G / p.s.H;
    d_h = G - d_rg * p.s.H;
    rg = t / p.s.H;
    h = t - rg * p.s.H;
  }
  __device__ __forceinline__ bool get(const FeatParams& p, Tile& x) {
    if (t >= total) return false;
    if (t >= tb.tile1) {      // masked only (the virtual table spans all tiles)
      do {
        ++b;
        const int4 v = __ldg(reinterpret_cast<const int4*>(p.tabs + b));
        tb.Cv = v.x; tb.lgCp = v.y; tb.tile0 = v.z; tb.tile1 = v.w;
      } while (t >= tb.tile1);
      const int local = t - tb.tile0;
      rg = local / p.s.H;
      h = local - rg * p.s.H;
    }
    const int rpt = kSlots >> tb.lgCp;
    x.h = h;
    x.row0 = rg * rpt;
    x.nrows = min(rpt, p.Rt - x.row0);
    x.b = b; x.Cv = tb.Cv; x.lgCp = tb.lgCp;
    return true;
  }
  __device__ __forceinline__ void next(const FeatParams& p) {
    t += step;
    h += d_h;
    rg += d_rg;
    if (h >= p.s.H) { h -= p.s.H; ++rg; }
  }
};

// Tables without a valid column have no tiles; their outputs are defined as +0 (LSE 0).  Called in the kernel
// prologue by `nthr` threads of every CTA (grid-strided over the launch).
template <int NOUT>
__device__ __forceinline__ void zero_dead_tables(const FeatParams& p, unsigned char* const (&out)[NOUT], float* lse,
                                                 int tid, int nthr) {
  if (!p.masked) return;
  const size_t tab_bytes = (size_t)p.s.R * p.s.C * p.s.H * p.s.dh * 2;
  const size_t tab_lse = (size_t)p.s.R * p.s.H * p.s.C;
  const size_t first = (size_t)blockIdx.x * nthr + tid, stride = (size_t)gridDim.x * nthr;
  for (int b = 0; b < p.s.B; ++b) {
    if (__ldg(&p.tabs[b].Cv) != 0) continue;
    for (size_t i = first * 16; i < tab_bytes; i += stride * 16)
#pragma unroll
      for (int k = 0; k < NOUT; ++k) stg_v4(out[k] + (size_t)b * tab_bytes + i, make_uint4(0, 0, 0, 0));
    if (lse)
      for (size_t i = first; i < tab_lse; i += stride) lse[(size_t)b * tab_lse + i] = 0.f;
  }
}

// Zero-fill (a6) of the INVALID columns of masked tables, by spare warps of every CTA while the other warps
// compute: a cell's H heads are d2 contiguous bytes, so a warp clears whole cells with coalesced 16-byte stores
// (the softmax warps used to clear 2 dh bytes per (cell, head) with an integer division per store).  The CTA's
// `nzw` zero-fill warps (this one is `zw`) share the rows r = blockIdx.x, += gridDim.x of every table; four
// independent (column lookup, store) groups per lane and iteration keep several stores in flight.
// lse (forward): 0.0f at [b][r][h][invalid c].  Tables without a valid column are left to zero_dead_tables.
template <int NOUT>
__device__ __forceinline__ void zero_invalid_cells(const FeatParams& p, unsigned char* const (&out)[NOUT], float* lse,
                                                   int lane, int zw, int nzw) {
  if (!p.masked) return;
  const Shape& s = p.s;
  const uint32_t d2 = (uint32_t)s.H * s.dh * 2;
  const uint32_t chunks = d2 >> 4;                                     // 16-byte chunks per cell (<= 512)
  const uint32_t m_ch = (uint32_t)((0x100000000ull + chunks - 1) / chunks);   // i / chunks = umulhi(i, m_ch), i < 2^16
  for (int b = 0; b < s.B; ++b) {
    const int Cv = __ldg(&p.tabs[b].Cv), ninv = s.C - Cv;
    if (Cv == 0 || ninv == 0) continue;
    const uint8_t* inv = p.vcol + (size_t)b * 128 + Cv;
    const uint32_t total = (uint32_t)ninv * chunks;                    // <= 128 * 512
    const uint32_t m_ni = (uint32_t)((0x100000000ull + ninv - 1) / ninv);
    for (int r = blockIdx.x + zw * (int)gridDim.x; r < s.R; r += nzw * (int)gridDim.x) {
      const size_t row = (size_t)b * s.R + r;
      unsigned char* base[NOUT];
#pragma unroll
      for (int o = 0; o < NOUT; ++o) base[o] = out[o] + row * s.C * d2;
      for (uint32_t i0 = lane; i0 < total; i0 += 128) {
        uint32_t off[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const uint32_t i = i0 + 32 * u, k = __umulhi(i, m_ch), ch = i - k * chunks;
          off[u] = i < total ? (uint32_t)__ldg(inv + k) * d2 + ch * 16 : 0xffffffffu;
        }
#pragma unroll
        for (int u = 0; u < 4; ++u)
          if (off[u] != 0xffffffffu) {
#pragma unroll
            for (int o = 0; o < NOUT; ++o) stg_v4(base[o] + off[u], make_uint4(0, 0, 0, 0));
          }
      }
      if (lse)
        for (uint32_t i = lane; i < (uint32_t)ninv * s.H; i += 32) {
          const uint32_t h = ninv == 1 ? i : __umulhi(i, m_ni), kk = i - h * ninv;   // (the magic number is 2^32 at ninv = 1)
          lse[(row * s.H + h) * s.C + __ldg(inv + kk)] = 0.f;
        }
    }
  }
}

// log2(Cp) of the tile `back` tiles before tile t of table b (masked tables; -1 if there is none): the
// same table almost always, else the nearest earlier table that has tiles.
__device__ __forceinline__ int lgcp_of_earlier_tile(const FeatParams& p, const FeatTab& tb, int b, int t, int back) {
  const int tp = t - back;
  if (tp < 0) return -1;
  if (tp >= tb.tile0) return tb.lgCp;
  for (int bb = b - 1; bb >= 0; --bb) {
    const int4 v = __ldg(reinterpret_cast<const int4*>(p.tabs + bb));
    if (tp >= v.z && tp < v.w) return v.y;
  }
  return -1;
}

// 16-byte-chunk swizzle of a [rows][ROWB] tile whose swizzle span is one row (the TMA / UMMA layout):
// chunk index XOR bits [7, 7+log2(CH)) of the byte offset.
template <int ROWB>
__device__ __forceinline__ uint32_t swz_off(int slot, int ch) {
  constexpr int CH = ROWB / 16;
  return (uint32_t)slot * ROWB + ((uint32_t)(ch ^ (((slot * ROWB) >> 7) & (CH - 1))) << 4);
}

// The two mask operands of a (Cp, Cv) geometry, written by one full warp: [128][16] bf16 each, rows of
// 32 bytes in the 32-byte-swizzle K-major layout (the dh = 16 operand format).  Generic-proxy stores:
// made visible to the tensor core before returning.
__device__ __forceinline__ void write_mask_tiles(uint32_t sMQ, uint32_t sMK, int lgCp, int Cv, int lane) {
  const int Cp = 1 << lgCp;
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const int r = lane + 32 * q;
    const int blk = r >> lgCp, v = r & (Cp - 1);          // blk in [0, 8)
    const bool live = v < Cv;
    uint32_t qa[4], ka[4];                                  // k = 0..7 as four bf16 pairs
#pragma unroll
    for (int k2 = 0; k2 < 4; ++k2) {
      const uint32_t q_lo = (2 * k2 == blk) ? kOne : 0u, q_hi = (2 * k2 + 1 == blk) ? kOne : 0u;
      const uint32_t k_lo = (2 * k2 == blk && live) ? 0u : kNegBig, k_hi = (2 * k2 + 1 == blk && live) ? 0u : kNegBig;
      qa[k2] = q_lo | (q_hi << 16);
      ka[k2] = k_lo | (k_hi << 16);
    }
    const uint32_t sw = (r >> 2) & 1;                       // 32-byte swizzle: chunk ^= bit 7 of the offset
    sts_v4(sMQ + r * 32 + ((0 ^ sw) << 4), qa[0], qa[1], qa[2], qa[3]);
    sts_v4(sMQ + r * 32 + ((1 ^ sw) << 4), 0u, 0u, 0u, 0u);   // k = 8..15 unused
    sts_v4(sMK + r * 32 + ((0 ^ sw) << 4), ka[0], ka[1], ka[2], ka[3]);
    sts_v4(sMK + r * 32 + ((1 ^ sw) << 4), 0u, 0u, 0u, 0u);
  }
  fence_proxy_async_smem();
  __syncwarp();
}

// ---- gather producer (masked tables): 4 warps, every lane owns CH 16-byte chunks of every operand tile
template <int ROWB>
struct Gather {
  static constexpr int CH = ROWB / 16;
  uint32_t src[CH];   // byte offset of the chunk relative to (first row of the tile, column 0, head h)
  uint32_t dst[CH];   // byte offset inside the operand tile
  int rl[CH];         // row inside the tile; >= 128 marks a pad slot (always zero-filled)
  // per-table precompute; pw = producer warp 0..3
  __device__ __forceinline__ void setup(const FeatParams& p, int b, int Cv, int lgCp, int pw, int lane) {
    const int Cp = 1 << lgCp;
    const uint32_t d2 = (uint32_t)p.s.H * p.s.dh * 2;
#pragma unroll
    for (int q = 0; q < CH; ++q) {
      const int g = q * 128 + pw * 32 + lane;
      const int slot = g / CH, ch = g % CH;
      const int r = slot >> lgCp, v = slot & (Cp - 1);
      dst[q] = swz_off<ROWB>(slot, ch);
      if (v < Cv) {
        const int col = __ldg(p.vcol + (size_t)b * 128 + v);
        src[q] = ((uint32_t)r * p.s.C + col) * d2 + ch * 16;
        rl[q] = r;
      } else {
        src[q] = 0;
        rl[q] = 1 << 20;
      }
    }
  }
  // one operand tile: valid chunks by cp.async, the rest zero-filled (K/V pad rows must be finite)
  __device__ __forceinline__ void issue(uint32_t tile, const unsigned char* base, int nrows) const {
#pragma unroll
    for (int q = 0; q < CH; ++q) {
      if (rl[q] < nrows) cp_async16(tile + dst[q], base + src[q]);
      else sts_v4(tile + dst[q], 0u, 0u, 0u, 0u);
    }
  }
};

using ::tabattn::quad_transpose;
using ::tabattn::QuadRows;

template <int N>
__device__ __forceinline__ void setmaxnreg_inc() {
  asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N));
}
template <int N>
__device__ __forceinline__ void setmaxnreg_dec() {
  asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N));
}

}  // namespace ftc

// host side (feature_tc_fwd.cu): per-call geometry, the prep launch for masked tables
size_t feature_workspace_bytes(const Shape& s);

}  // namespace tabattn
