// Shared pieces of the tcgen05 item-axis kernels (item_tc_fwd.cu, item_tc_bwd.cu): the persistent
// work walker, the shared-memory tail zeroing that enforces the train-only key rule on partially
// filled tiles, and the setmaxnreg wrappers.
#pragma once
#include "common.cuh"
#include "tc_common.cuh"

namespace tabattn {
namespace itc {

constexpr int kTileRows = 128;       // rows of every operand tile (UMMA M, and N of the score tiles)
constexpr float kRescaleLog2 = 8.f;  // lazy-rescale threshold of the online softmax (log2 units)

__device__ __forceinline__ int clamp_n(const Shape& s, int b) { return max(1, min(__ldg(s.n_train + b), s.R)); }

// One CTA walks the work items w = blockIdx.x, blockIdx.x + gridDim.x, ...; an item is one
// (table b, column c, head h, block of `rows_per_item` rows).  Consecutive items of one (b,c,h) are
// adjacent in w, so CTAs that run at the same time share K/V (or Q/dO) tiles in L2.  Items of
// invalid columns are skipped here (the zero-fill of their outputs is done by the epilogue warps).
// `tiles` = number of 128-row tiles of the looped axis; `t` counts tiles over the CTA's lifetime
// and `k` counts valid items: they index the mbarrier ring phases.
struct Walker {
  int w, j, tiles, n, b, c, h, blk;
  uint32_t k, t;
  bool ok;
  int n_items, bps, chunk;   // items in the launch, 128/256-row blocks per sequence, rows per inner tile
  bool over_keys;            // inner axis = key rows [0, n) (fwd, dQ); else query rows [0, R) (dK/dV)

  __device__ __forceinline__ void decode(const Shape& s, bool& valid) {
    blk = w % bps;
    const int rest = w / bps;
    h = rest % s.H;
    const int bc = rest / s.H;
    b = bc / s.C;
    c = bc - b * s.C;
    n = clamp_n(s, b);
    valid = (!s.col_valid || __ldg(s.col_valid + bc) != 0) && (over_keys || blk * kTileRows < n);
    tiles = ((over_keys ? n : s.R) + chunk - 1) / chunk;
  }
  __device__ __forceinline__ void seek(const Shape& s) {
    ok = false;
    while (w < n_items) {
      bool valid;
      decode(s, valid);
      if (valid) {
        j = 0;
        ok = true;
        return;
      }
      w += gridDim.x;
    }
  }
  __device__ __forceinline__ void init(const Shape& s, int n_items_, int bps_, int chunk_, bool over_keys_) {
    n_items = n_items_; bps = bps_; chunk = chunk_; over_keys = over_keys_;
    w = blockIdx.x; k = 0; t = 0;
    seek(s);
  }
  __device__ __forceinline__ void next(const Shape& s) {
    ++t;
    if (++j == tiles) {
      w += gridDim.x;
      ++k;
      seek(s);
    }
  }
};

// Zero rows [first_row, ROWS) of a [ROWS][ROWB bytes] tile (whole rows: the 16-byte-chunk swizzle only
// permutes bytes inside a row).  Called by one full warp after the TMA load has landed; makes the
// generic-proxy stores visible to the tensor core (async proxy) before returning.
template <int ROWB, int ROWS = kTileRows>
__device__ __forceinline__ void zero_tail_rows(uint32_t tile_saddr, int first_row, int lane) {
  const uint32_t begin = tile_saddr + first_row * ROWB, end = tile_saddr + ROWS * ROWB;
  for (uint32_t a = begin + 16 * lane; a < end; a += 16 * 32)
    asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(a), "r"(0u) : "memory");
  tc::fence_proxy_async_smem();
  __syncwarp();
}

template <int N>
__device__ __forceinline__ void setmaxnreg_inc() {
  asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N));
}
template <int N>
__device__ __forceinline__ void setmaxnreg_dec() {
  asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N));
}

}  // namespace itc
}  // namespace tabattn
