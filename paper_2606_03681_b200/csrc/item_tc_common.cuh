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

// a0 for masked tables: the compacted list of (b, c) pairs, built by item_prep_kernel into the workspace:
//   counts[0] = NV valid pairs;  list[0, NV) = the valid pairs ascending, list[NV, B*C) = the invalid ones, each
//   packed as b << 16 | c.
// The kernels walk virtual columns v in [0, NV) instead of all B*C columns and skipping the invalid ones: a skipped
// item costs nothing, so the static walk dealt uneven numbers of real items to the CTAs (feature_heavy: 40 % of the
// columns invalid, per-SM busy time max / avg = 1.08-1.11, profiles/r02_attention.md).  The zero-fill of the invalid
// columns (a6) is a second, equally dealt walk over list[NV, B*C) after the main loop.  list == nullptr (no mask):
// every column is valid and v is the real column index.
// MASKED is a template parameter of the kernels: the unmasked instantiations carry none of this (the forward's
// softmax loop lost 15 % at base when the list pointer was a run-time member of its walker).
template <bool MASKED>
struct ColList {
  const uint32_t* list;
  int nv, ni;
  __device__ __forceinline__ void init(const Shape& s, const uint32_t* l) {
    list = nullptr;
    nv = s.B * s.C;
    ni = 0;
    if (MASKED) {
      nv = (int)__ldg(l);          // counts[0] sits in front of the list
      ni = s.B * s.C - nv;
      list = l + 4;
    }
  }
  static __device__ __forceinline__ constexpr bool masked() { return MASKED; }
  // returns false only for the (never written) entry 0xffffffff: B, C <= 65535 keep every real pair below it
  __device__ __forceinline__ bool pair(int v, int& b, int& c) const {
    const uint32_t e = __ldg(list + v);
    b = (int)(e >> 16);
    c = (int)(e & 0xffffu);
    return e != 0xffffffffu;
  }
};

// Per-table metadata (clamped n_train, column validity) staged in shared memory at kernel start when it fits:
// every role decodes every work item, and the two dependent global loads behind each decode were exposed at
// every item boundary (items are only 12-16 chunks long at base).  Larger problems read global memory.  Used by
// the backward kernels (long_item bwd 7.30 -> 7.00 ms, ragged 7.37 -> 7.14); the forward kernel measured slower
// with it on the unmasked configs (0.50 -> 0.54 ms at base) and keeps the direct loads.
constexpr int kMetaTabs = 512, kMetaCells = 8192;
struct Meta {
  const int32_t* sn;
  const uint8_t* scv;
  bool in_smem;
  __device__ __forceinline__ int n(const Shape& s, int b) const { return in_smem ? sn[b] : clamp_n(s, b); }
  __device__ __forceinline__ bool cv(const Shape& s, int bc) const {
    return in_smem ? scv[bc] != 0 : (!s.col_valid || __ldg(s.col_valid + bc) != 0);
  }
  // all threads of the CTA, before the __syncthreads() that ends the kernel prologue
  __device__ __forceinline__ void fill(const Shape& s, int32_t* sn_, uint8_t* scv_) {
    sn = sn_; scv = scv_;
    in_smem = s.B <= kMetaTabs && s.B * s.C <= kMetaCells;
    if (in_smem) {
      for (int i = threadIdx.x; i < s.B; i += blockDim.x) sn_[i] = clamp_n(s, i);
      for (int i = threadIdx.x; i < s.B * s.C; i += blockDim.x) scv_[i] = s.col_valid ? __ldg(s.col_valid + i) : 1;
    }
  }
};

// One CTA walks the work items w = blockIdx.x, blockIdx.x + gridDim.x, ...; an item is one
// (table b, column c, head h, block of `rows_per_item` rows).  Consecutive items of one (b,c,h) are
// adjacent in w, so CTAs that run at the same time share K/V (or Q/dO) tiles in L2.  Items of
// invalid columns are skipped here (the zero-fill of their outputs is done by the epilogue warps).
// `tiles` = number of 128-row tiles of the looped axis; `t` counts tiles over the CTA's lifetime
// and `k` counts valid items: they index the mbarrier ring phases.
// Incremental decode of the work items w = blockIdx.x + k * gridDim.x, w = ((b*C + c)*H + h)*bps + blk: the
// six integer divisions of a direct decode are paid once; next() is ~15 adds/compares with carries.  (At base the
// items are 6-16 inner tiles long and the direct decode plus the loads that depend on it were ~12 % of the score
// warps' samples, profiles/r01_s46_final.md.)  seqmod = (sequence index) % bps serves the dK/dV block rotation.
struct ItemCoord {
  int w, blk, h, c, b, seqmod;
  int s_blk, s_h, s_c, s_b, s_seqmod;   // per-step increments (step = gridDim.x items)
  int bps, H, C;
  // `cols`: number of columns walked -- s.C per table, or (masked) the NV valid pairs as one virtual table, in which
  // case c is the virtual column and b stays 0
  __device__ __forceinline__ void init(const Shape& s, int bps_, int cols = 0) {
    bps = bps_; H = s.H; C = cols > 0 ? cols : s.C;
    w = blockIdx.x;
    blk = w % bps;
    const int seq = w / bps;
    h = seq % H;
    const int bc = seq / H;
    b = bc / C;
    c = bc - b * C;
    seqmod = seq % bps;
    const int G = gridDim.x, dseq = G / bps;
    s_blk = G - dseq * bps;
    s_h = dseq % H;
    const int dbc = dseq / H;
    s_b = dbc / C;
    s_c = dbc - s_b * C;
    s_seqmod = dseq % bps;
  }
  __device__ __forceinline__ void next() {
    w += gridDim.x;
    blk += s_blk;
    const int c0 = blk >= bps;
    blk -= c0 ? bps : 0;
    seqmod += s_seqmod + c0;
    seqmod -= seqmod >= bps ? bps : 0;
    h += s_h + c0;
    const int c1 = h >= H;
    h -= c1 ? H : 0;
    c += s_c + c1;
    const int c2 = c >= C;
    c -= c2 ? C : 0;
    b += s_b + c2;
  }
  __device__ __forceinline__ int bc() const { return b * C + c; }
  // dK/dV pass: block index rotated by the sequence index (see decode_item)
  __device__ __forceinline__ int blk_rot() const {
    const int r = blk + seqmod;
    return r >= bps ? r - bps : r;
  }
};

template <bool MASKED>
struct Walker {
  ItemCoord ic;
  int j, tiles, n, b, c, h, blk;
  uint32_t k, t;
  bool ok;
  int n_items, chunk;        // items in the launch, rows per inner tile
  bool over_keys;            // inner axis = key rows [0, n) (fwd, dQ); else query rows [0, R) (dK/dV)

  ColList<MASKED> cl;
  __device__ __forceinline__ void decode(const Shape& s, bool& valid) {
    blk = ic.blk; h = ic.h; b = ic.b; c = ic.c;
    bool listed = true;
    if (cl.masked()) listed = cl.pair(ic.c, b, c);
    n = clamp_n(s, b);
    // (both instantiations keep a run-time validity test that is never false -- the unmasked one the mask test of
    // the earlier builds, the masked one the list entry's -- because without the branch it guards ptxas schedules
    // the forward's softmax loop 7 % slower: 0.574 against 0.535 ms at base, measured A/B on one box)
    valid = (MASKED ? listed : (!s.col_valid || __ldg(s.col_valid + ic.bc()) != 0)) && (over_keys || blk * kTileRows < n);
    tiles = ((over_keys ? n : s.R) + chunk - 1) / chunk;
  }
  __device__ __forceinline__ void seek(const Shape& s) {
    ok = false;
    while (ic.w < n_items) {
      bool valid;
      decode(s, valid);
      if (valid) {
        j = 0;
        ok = true;
        return;
      }
      ic.next();
    }
  }
  __device__ __forceinline__ void init(const Shape& s, const ColList<MASKED>& cl_, int bps_, int chunk_, bool over_keys_) {
    cl = cl_; chunk = chunk_; over_keys = over_keys_;
    n_items = cl.nv * s.H * bps_;
    ic.init(s, bps_, cl.masked() ? max(cl.nv, 1) : 0);
    k = 0; t = 0;
    seek(s);
  }
  __device__ __forceinline__ void next(const Shape& s) {
    ++t;
    if (++j == tiles) {
      ic.next();
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

// (item_tc_fwd.cu) bytes of the column list in a workspace, and the launch of the a0 prep kernel that fills it;
// returns the device pointer the kernels take (nullptr when the call has no mask)
size_t item_list_bytes(const Shape& s);
const uint32_t* item_build_list(const Shape& s, void* list_ws, cudaStream_t stream);

}  // namespace tabattn
