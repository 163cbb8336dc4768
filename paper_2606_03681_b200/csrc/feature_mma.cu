// Feature-axis attention, forward and backward.
//
// The feature axis is short (C <= 128 columns) and the path is HBM-bound (0.58*C flop/B), so the
// kernels are built around the memory stream, not around the contraction:
//   * persistent CTAs of 3-8 warps, several per SM; every CTA walks "stage units" = (table b, block of
//     `rows` table rows, group of `hg` heads) and keeps a ring of NSTAGE stages in flight with
//     16-byte cp.async (LDGSTS) copies -- one stage is being computed while the next ones land.
//     (One 1-D bulk copy per cell was measured first: the TMA unit retires one cp.async.bulk per
//     ~68 clk per SM whatever its size, 3x too slow for 384-byte cells: profiles/r01_feature_mma.md);
//   * only VALID columns are loaded (gathered): the cells of a row are compacted to slots
//     v = 0..Cv-1 in shared memory, so DRAM traffic equals the algorithmic bytes even under a mask;
//     each cell slot is padded by 16 B, which makes every ldmatrix phase hit 8 distinct 16-byte
//     bank groups (an unpadded 384/512-byte cell stride is an 8-way conflict: profiles/r01_feature_mma.md);
//   * the C x C problems of one (row, head) run on the legacy tensor path, mma.sync m16n8k16 bf16
//     with fp32 accumulators (555 TFLOP/s measured on B200 -- far above what this path needs; a
//     128-row tcgen05 tile would be mostly padding at C = 11..21); a warp owns one 16-row tile of one
//     (row, head): FlashAttention-2 style register pipeline, quad-shuffle softmax in base 2;
//   * backward = two independent task kinds per (row, head, 16-row tile), both recomputing P from the
//     saved LSE: key-stationary (S^T = K Q^T, dP^T = V dO^T -> dV, dK) and query-stationary
//     (S = Q K^T, dP = dO V^T -> dQ).  No atomics, no cross-warp reduction: deterministic.
//     D = rowsum(dO o O) is computed once per stage from the staged dO and O;
//   * results leave through a 16-row per-warp staging tile as full 16-byte vectors; cells of invalid
//     columns are zero-filled by the loader threads (a6).
// Stale data in padded slots is always finite (shared memory is zeroed once, then only valid cells
// land in it) and every masked probability is forced to 0 by a select, so nothing at an invalid
// column or in a padded slot can reach an output.
#include "common.cuh"
#include "kernels.h"

#include <stdio.h>
#include <stdlib.h>

namespace tabattn {

namespace {

constexpr int kMaxWarps = 8;
constexpr int kMaxStages = 4;

struct FeatParams {
  Shape s;
  int hg, nhg;          // heads per stage unit, units per (table, row block)
  int rows;             // table rows per stage unit
  int Cp;               // C rounded up to 16: pitch of the per-(row, head) statistics vectors
  int slot_stride;      // bytes per cell slot: hg*dh*2 + 16
  int chunks;           // 16-byte chunks per cell slot payload: hg*dh/8
  int rb_per_table;     // ceil(R / rows)
  int n_su;             // B * rb_per_table
  uint32_t div_chunks;  // ceil(2^32 / chunks)
  uint32_t div_C;       // ceil(2^32 / C)
  uint32_t div_hgC;     // ceil(2^32 / (hg*C))
  uint32_t slot_bytes;  // rows * Cp * slot_stride
  uint32_t off_lse, off_D, off_vcol, off_cv, stage_bytes;  // layout of one stage
  uint32_t stage0;      // offset of stage 0 (after the per-warp staging tiles)
  int nstage;
  int ld_dcell, ld_dch; // loader step of one CTA-wide stride: nthreads / chunks, nthreads % chunks
};

// x / d for x < 2^32 / d with magic = floor(2^32 / d) + 1 (0 stands for d == 1)
__device__ __forceinline__ uint32_t fdiv(uint32_t x, uint32_t magic) { return magic ? __umulhi(x, magic) : x; }

__device__ __forceinline__ uint32_t smem_addr(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global.L2::128B [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async4(uint32_t dst, const void* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ void ldsm4(uint32_t addr, uint32_t (&r)[4]) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
               : "r"(addr));
}
__device__ __forceinline__ void ldsm4t(uint32_t addr, uint32_t (&r)[4]) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
               : "r"(addr));
}
// C[16x8] += A[16x16] * B[16x8], bf16 inputs, fp32 accumulate
__device__ __forceinline__ void mma_bf16(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void sts32(uint32_t addr, uint32_t v) {
  asm volatile("st.shared.b32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
  uint4 r;
  asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(addr));
  return r;
}
__device__ __forceinline__ float quad_max(float v) {
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 1));
  return fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 2));
}
__device__ __forceinline__ float quad_sum(float v) {
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  return v + __shfl_xor_sync(0xffffffffu, v, 2);
}

// ---- the unit walker: which (table, row block, head group) is the q-th stage of this CTA ---------------
struct Unit {
  int su, hgi;   // super unit (table, row block) and head group
  int b, r0, nrows;
  __device__ __forceinline__ void set(const FeatParams& p) {
    b = su / p.rb_per_table;
    r0 = (su - b * p.rb_per_table) * p.rows;
    nrows = min(p.rows, p.s.R - r0);
  }
  __device__ __forceinline__ void init(const FeatParams& p) {
    su = blockIdx.x; hgi = 0;
    if (su < p.n_su) set(p);
  }
  __device__ __forceinline__ bool ok(const FeatParams& p) const { return su < p.n_su; }
  __device__ __forceinline__ void next(const FeatParams& p) {
    if (++hgi == p.nhg) {
      hgi = 0;
      su += gridDim.x;
      if (su < p.n_su) set(p);
    }
  }
};

// Validity bit mask of table b (C <= 128 -> 4 words), identical in every lane; cnt[k] = valid columns
// below word k.  All 32 lanes of the warp must call this.
struct ColMask {
  uint32_t m[4];
  int below[4];
  int Cv;
  int b = -1;   // table the mask was built for (the walker revisits a table for many stages)
  __device__ __forceinline__ void build(const Shape& s, int b_) {
    if (b_ == b) return;
    b = b_;
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int c = 32 * k + lane;
      bool v = c < s.C;
      if (v && s.col_valid) v = __ldg(s.col_valid + (size_t)b * s.C + c) != 0;
      m[k] = __ballot_sync(0xffffffffu, v);
    }
    below[0] = 0;
    below[1] = __popc(m[0]);
    below[2] = below[1] + __popc(m[1]);
    below[3] = below[2] + __popc(m[2]);
    Cv = below[3] + __popc(m[3]);
  }
  // selects instead of dynamic indexing: the arrays stay in registers
  __device__ __forceinline__ uint32_t word(int c) const {
    return c < 64 ? (c < 32 ? m[0] : m[1]) : (c < 96 ? m[2] : m[3]);
  }
  __device__ __forceinline__ bool valid(int c) const { return (word(c) >> (c & 31)) & 1u; }
  __device__ __forceinline__ int rank(int c) const {
    const int bl = c < 64 ? (c < 32 ? below[0] : below[1]) : (c < 96 ? below[2] : below[3]);
    return bl + __popc(word(c) & ((1u << (c & 31)) - 1u));
  }
};


// Per-lane byte offsets of the three ldmatrix address patterns (slot stride `str`), computed once.
struct LaneOff {
  uint32_t a;    // A fragment, 16 rows x 16 k:      row = lane & 15,                 col = (lane >> 4) * 16 B
  uint32_t nb;   // B fragment from an [n][k] tile:  row = (lane & 7) + 8*(lane >> 4), col = ((lane >> 3) & 1) * 16 B
  uint32_t tb;   // B fragment from a [k][n] tile (.trans): row = (lane & 7) + 8*((lane >> 3) & 1), col = (lane >> 4) * 16 B
  __device__ __forceinline__ void init(int str) {
    const int lane = threadIdx.x & 31;
    a = (lane & 15) * str + (lane >> 4) * 16;
    nb = ((lane & 7) + ((lane >> 4) << 3)) * str + ((lane >> 3) & 1) * 16;
    tb = ((lane & 7) + (((lane >> 3) & 1) << 3)) * str + (lane >> 4) * 16;
  }
};

// ---- stage loader ------------------------------------------------------------------------------------
// Issues the 16-byte cp.async copies of one stage unit into ring buffer `stage` (shared byte address):
// valid cell (r, c) -> compacted, padded slot (r*Cv + rank(c)); zero-fills the outputs of invalid cells
// (a6); (backward) fetches the saved LSE of the valid triples.  All threads of the CTA call it,
// uniformly; the caller commits the group.
template <int NIN, int NOUT, bool BWD>
__device__ __forceinline__ void issue_stage(const FeatParams& p, const Unit& u, ColMask& cm, uint32_t stage,
                                            unsigned char* stage_ptr, const unsigned char* const (&in)[NIN],
                                            unsigned char* const (&out)[NOUT], float* __restrict__ LSE_out,
                                            const float* __restrict__ LSE_in) {
  const Shape& s = p.s;
  cm.build(s, u.b);
  const uint32_t d2 = s.H * s.dh * 2;                    // bytes per cell
  const uint32_t hoff = u.hgi * p.hg * s.dh * 2;         // byte offset of the head group inside a cell
  const size_t row0 = (size_t)u.b * s.R + u.r0;
  const size_t gbase = row0 * s.C * (size_t)d2 + hoff;
  const uint32_t ncell = (uint32_t)u.nrows * s.C;
  uint32_t cell = fdiv(threadIdx.x, p.div_chunks);
  uint32_t ch = threadIdx.x - cell * p.chunks;
  if (cm.Cv == s.C) {
    // all columns valid: slot index = cell index
    uint32_t soff = cell * p.slot_stride + ch * 16;
    uint32_t goff = cell * d2 + ch * 16;
    const uint32_t ds_lo = p.ld_dcell * p.slot_stride + p.ld_dch * 16, dg_lo = p.ld_dcell * d2 + p.ld_dch * 16;
    const uint32_t ds_wrap = p.slot_stride - p.chunks * 16, dg_wrap = d2 - p.chunks * 16;
    while (cell < ncell) {
#pragma unroll
      for (int k = 0; k < NIN; ++k) cp_async16(stage + k * p.slot_bytes + soff, in[k] + gbase + goff);
      cell += p.ld_dcell; ch += p.ld_dch; soff += ds_lo; goff += dg_lo;
      if (ch >= (uint32_t)p.chunks) { ch -= p.chunks; ++cell; soff += ds_wrap; goff += dg_wrap; }
    }
    if (threadIdx.x < (uint32_t)s.C) stage_ptr[p.off_vcol + threadIdx.x] = (unsigned char)threadIdx.x;
  } else {
    while (cell < ncell) {
      const uint32_t r = fdiv(cell, p.div_C);
      const int c = (int)(cell - r * s.C);
      const size_t g = gbase + (size_t)cell * d2 + ch * 16;
      if (cm.valid(c)) {
        const int v = cm.rank(c);
        const uint32_t soff = (r * cm.Cv + v) * p.slot_stride + ch * 16;
#pragma unroll
        for (int k = 0; k < NIN; ++k) cp_async16(stage + k * p.slot_bytes + soff, in[k] + g);
        if (r == 0 && ch == 0) stage_ptr[p.off_vcol + v] = (unsigned char)c;
      } else {
#pragma unroll
        for (int k = 0; k < NOUT; ++k) stg_v4(out[k] + g, make_uint4(0, 0, 0, 0));
        if (!BWD && ch == 0) {
          for (int hl = 0; hl < p.hg; ++hl) LSE_out[((row0 + r) * s.H + u.hgi * p.hg + hl) * s.C + c] = 0.f;
        }
      }
      cell += p.ld_dcell; ch += p.ld_dch;
      if (ch >= (uint32_t)p.chunks) { ch -= p.chunks; ++cell; }
    }
  }
  if (BWD) {
    // saved LSE of the unit's valid (row, head, column) triples -> sL[(r*hg + hl)*Cp + v]
    const uint32_t total2 = (uint32_t)u.nrows * p.hg * s.C;
    for (uint32_t idx = threadIdx.x; idx < total2; idx += blockDim.x) {
      const uint32_t r = fdiv(idx, p.div_hgC);
      const uint32_t rem = idx - r * p.hg * s.C;
      const uint32_t hl = fdiv(rem, p.div_C);
      const int c = (int)(rem - hl * s.C);
      if (cm.valid(c))
        cp_async4(stage + p.off_lse + ((r * p.hg + hl) * p.Cp + cm.rank(c)) * 4,
                  LSE_in + ((row0 + r) * s.H + u.hgi * p.hg + hl) * s.C + c);
    }
  }
  if (threadIdx.x == 0) *reinterpret_cast<int*>(stage_ptr + p.off_cv) = cm.Cv;
}

__device__ __forceinline__ void stsm4(uint32_t addr, uint32_t r0, uint32_t r1, uint32_t r2, uint32_t r3) {
  asm volatile("stmatrix.sync.aligned.m8n8.x4.shared.b16 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(r0), "r"(r1), "r"(r2),
               "r"(r3)
               : "memory");
}

// Output path of one 16 x DH accumulator tile (C fragments: DH/8 n-tiles, rows g and g+8): scale per
// row, round to bf16, transpose through the warp's staging tile (stmatrix), and write full 16-byte
// vectors to the cells (row r of the unit, compacted columns v0..v0+15, head h) of a [B,R,C,H,dh] tensor.
// `dst_row` points at (table row, column 0, head h); cells of one row are d2 bytes apart.
__device__ __forceinline__ uint32_t lds_u8(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}

// IDENT: all columns of the table are valid, slot v is column v (no vcol lookup).
template <int DH, bool IDENT>
__device__ __forceinline__ void write_tile(uint32_t stg, const float (&acc)[DH / 8][4], float mul0, float mul1,
                                           unsigned char* dst_row, uint32_t d2, int v0, int Cv, uint32_t vcol_s) {
  constexpr int SSTR = DH * 2 + 16, CH = DH / 8;
  const int lane = threadIdx.x & 31;
  {
    const uint32_t a = stg + ((lane & 7) + ((lane >> 3) & 1) * 8) * SSTR + (lane >> 4) * 16;
#pragma unroll
    for (int np = 0; np < DH / 16; ++np)
      stsm4(a + np * 32, pack_bf16(acc[2 * np][0] * mul0, acc[2 * np][1] * mul0),
            pack_bf16(acc[2 * np][2] * mul1, acc[2 * np][3] * mul1),
            pack_bf16(acc[2 * np + 1][0] * mul0, acc[2 * np + 1][1] * mul0),
            pack_bf16(acc[2 * np + 1][2] * mul1, acc[2 * np + 1][3] * mul1));
  }
  __syncwarp();
#pragma unroll
  for (int it = 0; it < (16 * CH + 31) / 32; ++it) {
    const int idx = it * 32 + lane;
    const int row = idx / CH, ch = idx % CH;
    if (v0 + row < Cv) {
      const uint32_t c = IDENT ? (uint32_t)(v0 + row) : lds_u8(vcol_s + v0 + row);
      stg_v4(dst_row + (c * d2 + ch * 16), lds128(stg + row * SSTR + ch * 16));
    }
  }
  __syncwarp();
}

// What a task needs to know about its stage, its warp and its lane.
struct TaskCtx {
  uint32_t stg;              // the warp's staging tile
  LaneOff lo;
  uint32_t str, d2;          // slot stride, bytes per cell
  float c2, scale;           // scale * log2(e), scale
  int Cv;
  uint32_t vcol_s;           // shared address of the slot -> column table of the stage
};

// ---- forward task, one pass (online softmax): one warp, 16 query cells (slots v0..v0+15) of one (row, head) ------------------------
// sQ/sK/sV: shared byte addresses of the slots at (row r of the unit, slot 0, this head).
template <int DH, bool IDENT>
__device__ __forceinline__ void fwd_task_1p(const TaskCtx& x, uint32_t sQ, uint32_t sK, uint32_t sV, int v0,
                                         unsigned char* O_row, float* __restrict__ LSE_row) {
  constexpr int KS = DH / 16, NT = DH / 8;
  const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int Cv = x.Cv;
  uint32_t qa[KS][4];
#pragma unroll
  for (int ks = 0; ks < KS; ++ks) ldsm4(sQ + v0 * x.str + x.lo.a + ks * 32, qa[ks]);
  float o[NT][4];
#pragma unroll
  for (int nt = 0; nt < NT; ++nt) o[nt][0] = o[nt][1] = o[nt][2] = o[nt][3] = 0.f;
  float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;
  for (int k0 = 0; k0 < Cv; k0 += 16) {
    float sc[2][4];
    sc[0][0] = sc[0][1] = sc[0][2] = sc[0][3] = 0.f;
    sc[1][0] = sc[1][1] = sc[1][2] = sc[1][3] = 0.f;
    {
      const uint32_t a = sK + k0 * x.str + x.lo.nb;
#pragma unroll
      for (int ks = 0; ks < KS; ++ks) {
        uint32_t kb[4];
        ldsm4(a + ks * 32, kb);
        mma_bf16(sc[0], qa[ks], kb[0], kb[1]);
        mma_bf16(sc[1], qa[ks], kb[2], kb[3]);
      }
    }
    // scale to log2 units; keys >= Cv (padded slots) -> -inf
#pragma unroll
    for (int nt = 0; nt < 2; ++nt)
#pragma unroll
      for (int e = 0; e < 4; ++e) sc[nt][e] *= x.c2;
    if (k0 + 16 > Cv) {
      const int lim = Cv - k0 - 2 * t;   // key offset nt*8 + (e&1) must be < lim
#pragma unroll
      for (int nt = 0; nt < 2; ++nt)
#pragma unroll
        for (int e = 0; e < 4; ++e)
          if (nt * 8 + (e & 1) >= lim) sc[nt][e] = -INFINITY;
    }
    float mx0 = fmaxf(fmaxf(sc[0][0], sc[0][1]), fmaxf(sc[1][0], sc[1][1]));
    float mx1 = fmaxf(fmaxf(sc[0][2], sc[0][3]), fmaxf(sc[1][2], sc[1][3]));
    mx0 = quad_max(mx0);
    mx1 = quad_max(mx1);
    const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);   // finite: the chunk holds >= 1 valid key
    if (k0 > 0) {
      const float al0 = fast_exp2(m0 - mn0), al1 = fast_exp2(m1 - mn1);
      l0 *= al0;
      l1 *= al1;
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) {
        o[nt][0] *= al0; o[nt][1] *= al0;
        o[nt][2] *= al1; o[nt][3] *= al1;
      }
    }
    m0 = mn0;
    m1 = mn1;
    uint32_t pa[4];
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) {
      const float p0 = fast_exp2(sc[nt][0] - m0), p1 = fast_exp2(sc[nt][1] - m0);
      const float p2 = fast_exp2(sc[nt][2] - m1), p3 = fast_exp2(sc[nt][3] - m1);
      l0 += p0 + p1;
      l1 += p2 + p3;
      pa[nt * 2] = pack_bf16(p0, p1);
      pa[nt * 2 + 1] = pack_bf16(p2, p3);
    }
    {
      const uint32_t a = sV + k0 * x.str + x.lo.tb;
#pragma unroll
      for (int np = 0; np < NT / 2; ++np) {
        uint32_t vb[4];
        ldsm4t(a + np * 32, vb);
        mma_bf16(o[2 * np], pa, vb[0], vb[1]);
        mma_bf16(o[2 * np + 1], pa, vb[2], vb[3]);
      }
    }
  }
  l0 = quad_sum(l0);
  l1 = quad_sum(l1);
  if (t < 2) {   // lane t = 0 stores row g, lane t = 1 row g + 8 (every lane of the quad holds both sums)
    const int rr = v0 + g + 8 * t;
    if (rr < Cv) {
      const float lsel = t ? l1 : l0, msel = t ? m1 : m0;
      LSE_row[IDENT ? (uint32_t)rr : lds_u8(x.vcol_s + rr)] = (msel + log2f(lsel)) * kLn2;
    }
  }
  write_tile<DH, IDENT>(x.stg, o, 1.f / l0, 1.f / l1, O_row, x.d2, v0, Cv, x.vcol_s);
}

// ---- forward task, two passes: one warp, 16 query cells (slots v0..v0+15) of one (row, head) ------------
// Two passes over the (at most KB = ceil(C/16)) key blocks: all score tiles first (they fit in registers at
// C <= 128), one row maximum, then exp and P V -- no running maximum and no rescaling of the accumulator, which
// cost ~40 of the ~100 instructions per key block of the one-pass form.  Measured on B200 against the one-pass
// form: C = 21 (KB = 2) 0.343 -> 0.306 ms, C = 51 masked (KB = 4) 0.655 -> 0.626 ms, but C = 101 masked (KB = 8:
// 64 score registers, spills) 0.412 -> 0.447 ms and C = 11 (KB = 1) 0.121 -> 0.133 ms: used for KB = 2, 4 only.
template <int DH, bool IDENT, int KB>
__device__ __forceinline__ void fwd_task_2p(const TaskCtx& x, uint32_t sQ, uint32_t sK, uint32_t sV, int v0,
                                         unsigned char* O_row, float* __restrict__ LSE_row) {
  constexpr int KS = DH / 16, NT = DH / 8;
  const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int Cv = x.Cv;
  uint32_t qa[KS][4];
#pragma unroll
  for (int ks = 0; ks < KS; ++ks) ldsm4(sQ + v0 * x.str + x.lo.a + ks * 32, qa[ks]);
  // ---- pass 1: S = Q K^T for every key block (raw scores; blocks beyond Cv stay at -inf) -----------------
  float sc[KB][2][4];
#pragma unroll
  for (int kb = 0; kb < KB; ++kb) {
    if (kb * 16 < Cv) {
#pragma unroll
      for (int e = 0; e < 4; ++e) sc[kb][0][e] = sc[kb][1][e] = 0.f;
      const uint32_t a = sK + kb * 16 * x.str + x.lo.nb;
#pragma unroll
      for (int ks = 0; ks < KS; ++ks) {
        uint32_t kbf[4];
        ldsm4(a + ks * 32, kbf);
        mma_bf16(sc[kb][0], qa[ks], kbf[0], kbf[1]);
        mma_bf16(sc[kb][1], qa[ks], kbf[2], kbf[3]);
      }
      if (kb * 16 + 16 > Cv) {           // keys >= Cv (padded slots) -> -inf
        const int lim = Cv - kb * 16 - 2 * t;   // key offset nt*8 + (e&1) must be < lim
#pragma unroll
        for (int nt = 0; nt < 2; ++nt)
#pragma unroll
          for (int e = 0; e < 4; ++e)
            if (nt * 8 + (e & 1) >= lim) sc[kb][nt][e] = -INFINITY;
      }
    } else {
#pragma unroll
      for (int e = 0; e < 4; ++e) sc[kb][0][e] = sc[kb][1][e] = -INFINITY;
    }
  }
  // ---- row maxima (rows g and g+8 of the tile): finite, every row sees >= 1 valid key ------------------
  float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
  for (int kb = 0; kb < KB; ++kb) {
    mx0 = fmaxf(mx0, fmaxf(fmaxf(sc[kb][0][0], sc[kb][0][1]), fmaxf(sc[kb][1][0], sc[kb][1][1])));
    mx1 = fmaxf(mx1, fmaxf(fmaxf(sc[kb][0][2], sc[kb][0][3]), fmaxf(sc[kb][1][2], sc[kb][1][3])));
  }
  mx0 = quad_max(mx0);
  mx1 = quad_max(mx1);
  const float m0 = mx0 * x.c2, m1 = mx1 * x.c2;   // c2 = scale * log2(e) > 0
  // ---- pass 2: P = 2^(S c2 - m), l = rowsum(P), O = P V -----------------------------------------------------
  float o[NT][4];
#pragma unroll
  for (int nt = 0; nt < NT; ++nt) o[nt][0] = o[nt][1] = o[nt][2] = o[nt][3] = 0.f;
  float l0 = 0.f, l1 = 0.f;
#pragma unroll
  for (int kb = 0; kb < KB; ++kb) {
    if (kb * 16 < Cv) {
      uint32_t pa[4];
#pragma unroll
      for (int nt = 0; nt < 2; ++nt) {
        const float p0 = fast_exp2(fmaf(sc[kb][nt][0], x.c2, -m0)), p1 = fast_exp2(fmaf(sc[kb][nt][1], x.c2, -m0));
        const float p2 = fast_exp2(fmaf(sc[kb][nt][2], x.c2, -m1)), p3 = fast_exp2(fmaf(sc[kb][nt][3], x.c2, -m1));
        l0 += p0 + p1;
        l1 += p2 + p3;
        pa[nt * 2] = pack_bf16(p0, p1);
        pa[nt * 2 + 1] = pack_bf16(p2, p3);
      }
      const uint32_t a = sV + kb * 16 * x.str + x.lo.tb;
#pragma unroll
      for (int np = 0; np < NT / 2; ++np) {
        uint32_t vb[4];
        ldsm4t(a + np * 32, vb);
        mma_bf16(o[2 * np], pa, vb[0], vb[1]);
        mma_bf16(o[2 * np + 1], pa, vb[2], vb[3]);
      }
    }
  }
  l0 = quad_sum(l0);
  l1 = quad_sum(l1);
  if (t < 2) {   // lane t = 0 stores row g, lane t = 1 row g + 8 (every lane of the quad holds both sums)
    const int rr = v0 + g + 8 * t;
    if (rr < Cv) {
      const float lsel = t ? l1 : l0, msel = t ? m1 : m0;
      LSE_row[IDENT ? (uint32_t)rr : lds_u8(x.vcol_s + rr)] = (msel + log2f(lsel)) * kLn2;
    }
  }
  write_tile<DH, IDENT>(x.stg, o, 1.f / l0, 1.f / l1, O_row, x.d2, v0, Cv, x.vcol_s);
}

// ---- backward, key-stationary task: 16 key cells (slots j0..j0+15) of one (row, head) -> dV, dK -----------
// sL / sD: this (row, head)'s lse*log2e and D vectors, indexed by column slot.
template <int DH, bool IDENT>
__device__ __forceinline__ void bwd_key_task(const TaskCtx& x, uint32_t sQ, uint32_t sK, uint32_t sV, uint32_t sG,
                                             const float* sL, const float* sD, int j0, unsigned char* dK_row,
                                             unsigned char* dV_row) {
  constexpr int KS = DH / 16, NT = DH / 8;
  const int lane = threadIdx.x & 31, t = lane & 3;
  const int Cv = x.Cv;
  uint32_t ka[KS][4], va[KS][4];
#pragma unroll
  for (int ks = 0; ks < KS; ++ks) {
    ldsm4(sK + j0 * x.str + x.lo.a + ks * 32, ka[ks]);
    ldsm4(sV + j0 * x.str + x.lo.a + ks * 32, va[ks]);
  }
  float dv[NT][4], dk[NT][4];
#pragma unroll
  for (int nt = 0; nt < NT; ++nt) {
    dv[nt][0] = dv[nt][1] = dv[nt][2] = dv[nt][3] = 0.f;
    dk[nt][0] = dk[nt][1] = dk[nt][2] = dk[nt][3] = 0.f;
  }
  for (int i0 = 0; i0 < Cv; i0 += 16) {
    float st[2][4], dp[2][4];
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) {
      st[nt][0] = st[nt][1] = st[nt][2] = st[nt][3] = 0.f;
      dp[nt][0] = dp[nt][1] = dp[nt][2] = dp[nt][3] = 0.f;
    }
    {
      const uint32_t off = i0 * x.str + x.lo.nb;
#pragma unroll
      for (int ks = 0; ks < KS; ++ks) {
        uint32_t b[4];
        ldsm4(sQ + off + ks * 32, b);
        mma_bf16(st[0], ka[ks], b[0], b[1]);
        mma_bf16(st[1], ka[ks], b[2], b[3]);
        ldsm4(sG + off + ks * 32, b);
        mma_bf16(dp[0], va[ks], b[0], b[1]);
        mma_bf16(dp[1], va[ks], b[2], b[3]);
      }
    }
    // P^T[j][i] = exp2(S^T c2 - lse2_i), dS^T = P^T (dP^T - D_i); queries i >= Cv (padded slots) -> 0
    uint32_t pa[4], da[4];
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) {
      const int i = i0 + nt * 8 + 2 * t;
      const float2 L = *reinterpret_cast<const float2*>(sL + i);
      const float2 D = *reinterpret_cast<const float2*>(sD + i);
      const bool ok0 = i < Cv, ok1 = i + 1 < Cv;
      const float p0 = ok0 ? fast_exp2(fmaf(st[nt][0], x.c2, -L.x)) : 0.f;
      const float p1 = ok1 ? fast_exp2(fmaf(st[nt][1], x.c2, -L.y)) : 0.f;
      const float p2 = ok0 ? fast_exp2(fmaf(st[nt][2], x.c2, -L.x)) : 0.f;
      const float p3 = ok1 ? fast_exp2(fmaf(st[nt][3], x.c2, -L.y)) : 0.f;
      pa[nt * 2] = pack_bf16(p0, p1);
      pa[nt * 2 + 1] = pack_bf16(p2, p3);
      da[nt * 2] = pack_bf16(p0 * (dp[nt][0] - D.x), p1 * (dp[nt][1] - D.y));
      da[nt * 2 + 1] = pack_bf16(p2 * (dp[nt][2] - D.x), p3 * (dp[nt][3] - D.y));
    }
    {
      const uint32_t off = i0 * x.str + x.lo.tb;
#pragma unroll
      for (int np = 0; np < NT / 2; ++np) {
        uint32_t b[4];
        ldsm4t(sG + off + np * 32, b);
        mma_bf16(dv[2 * np], pa, b[0], b[1]);
        mma_bf16(dv[2 * np + 1], pa, b[2], b[3]);
        ldsm4t(sQ + off + np * 32, b);
        mma_bf16(dk[2 * np], da, b[0], b[1]);
        mma_bf16(dk[2 * np + 1], da, b[2], b[3]);
      }
    }
  }
  write_tile<DH, IDENT>(x.stg, dv, 1.f, 1.f, dV_row, x.d2, j0, Cv, x.vcol_s);
  write_tile<DH, IDENT>(x.stg, dk, x.scale, x.scale, dK_row, x.d2, j0, Cv, x.vcol_s);
}

// ---- backward, query-stationary task: 16 query cells (slots i0..i0+15) of one (row, head) -> dQ -----------
template <int DH, bool IDENT>
__device__ __forceinline__ void bwd_query_task(const TaskCtx& x, uint32_t sQ, uint32_t sK, uint32_t sV, uint32_t sG,
                                               const float* sL, const float* sD, int i0, unsigned char* dQ_row) {
  constexpr int KS = DH / 16, NT = DH / 8;
  const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int Cv = x.Cv;
  uint32_t qa[KS][4], ga[KS][4];
#pragma unroll
  for (int ks = 0; ks < KS; ++ks) {
    ldsm4(sQ + i0 * x.str + x.lo.a + ks * 32, qa[ks]);
    ldsm4(sG + i0 * x.str + x.lo.a + ks * 32, ga[ks]);
  }
  // rows g and g+8 of the tile; padded rows read stale (finite) statistics and are never stored
  const float L0 = sL[i0 + g], L1 = sL[i0 + g + 8], D0 = sD[i0 + g], D1 = sD[i0 + g + 8];
  float dq[NT][4];
#pragma unroll
  for (int nt = 0; nt < NT; ++nt) dq[nt][0] = dq[nt][1] = dq[nt][2] = dq[nt][3] = 0.f;
  for (int k0 = 0; k0 < Cv; k0 += 16) {
    float sc[2][4], dp[2][4];
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) {
      sc[nt][0] = sc[nt][1] = sc[nt][2] = sc[nt][3] = 0.f;
      dp[nt][0] = dp[nt][1] = dp[nt][2] = dp[nt][3] = 0.f;
    }
    {
      const uint32_t off = k0 * x.str + x.lo.nb;
#pragma unroll
      for (int ks = 0; ks < KS; ++ks) {
        uint32_t b[4];
        ldsm4(sK + off + ks * 32, b);
        mma_bf16(sc[0], qa[ks], b[0], b[1]);
        mma_bf16(sc[1], qa[ks], b[2], b[3]);
        ldsm4(sV + off + ks * 32, b);
        mma_bf16(dp[0], ga[ks], b[0], b[1]);
        mma_bf16(dp[1], ga[ks], b[2], b[3]);
      }
    }
    uint32_t da[4];
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) {
      const int key = k0 + nt * 8 + 2 * t;
      const bool ok0 = key < Cv, ok1 = key + 1 < Cv;   // keys in padded slots: P = 0 exactly
      const float p0 = ok0 ? fast_exp2(fmaf(sc[nt][0], x.c2, -L0)) : 0.f;
      const float p1 = ok1 ? fast_exp2(fmaf(sc[nt][1], x.c2, -L0)) : 0.f;
      const float p2 = ok0 ? fast_exp2(fmaf(sc[nt][2], x.c2, -L1)) : 0.f;
      const float p3 = ok1 ? fast_exp2(fmaf(sc[nt][3], x.c2, -L1)) : 0.f;
      da[nt * 2] = pack_bf16(p0 * (dp[nt][0] - D0), p1 * (dp[nt][1] - D0));
      da[nt * 2 + 1] = pack_bf16(p2 * (dp[nt][2] - D1), p3 * (dp[nt][3] - D1));
    }
    {
      const uint32_t off = k0 * x.str + x.lo.tb;
#pragma unroll
      for (int np = 0; np < NT / 2; ++np) {
        uint32_t b[4];
        ldsm4t(sK + off + np * 32, b);
        mma_bf16(dq[2 * np], da, b[0], b[1]);
        mma_bf16(dq[2 * np + 1], da, b[2], b[3]);
      }
    }
  }
  write_tile<DH, IDENT>(x.stg, dq, x.scale, x.scale, dQ_row, x.d2, i0, Cv, x.vcol_s);
}

// ---- kernels -------------------------------------------------------------------------------------------------
// Task walker of one warp inside a stage: tasks (tile mt, head hl, row r), mt fastest, strided by the
// warp count; advanced with carries instead of divisions.
struct TaskIt {
  int mt, hl, r;
  __device__ __forceinline__ void carry(int MT, int hg) {
    while (mt >= MT) { mt -= MT; ++hl; }
    while (hl >= hg) { hl -= hg; ++r; }
  }
};

__device__ __forceinline__ void zero_smem(unsigned char* smem, uint32_t smem_total) {
  for (uint32_t i = threadIdx.x * 16; i < smem_total; i += blockDim.x * 16)
    *reinterpret_cast<uint4*>(smem + i) = make_uint4(0, 0, 0, 0);
  __syncthreads();
}

// (minBlocks = 2 -> an explicit 128-register budget: without it ptxas caps some instantiations at 80 registers and spills)
template <int DH, int NSTAGE, int KB>
__global__ void __launch_bounds__(kMaxWarps * 32, 2) feature_fwd_mma_kernel(const __grid_constant__ FeatParams p,
                                                                         const unsigned char* __restrict__ Q,
                                                                         const unsigned char* __restrict__ K,
                                                                         const unsigned char* __restrict__ V,
                                                                         unsigned char* __restrict__ O,
                                                                         float* __restrict__ LSE, uint32_t smem_total) {
  extern __shared__ __align__(16) unsigned char smem[];
  zero_smem(smem, smem_total);
  const uint32_t sbase = smem_addr(smem);
  const int warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  const unsigned char* const in[3] = {Q, K, V};
  unsigned char* const out[1] = {O};
  const Shape& s = p.s;
  TaskCtx x;
  x.stg = sbase + warp * 16 * (DH * 2 + 16);
  x.lo.init(p.slot_stride);
  x.str = p.slot_stride;
  x.d2 = s.H * DH * 2;
  x.c2 = s.scale * kLog2e;
  x.scale = s.scale;

  Unit ld, cu;
  ColMask cm;
  ld.init(p);
  cu = ld;
#pragma unroll
  for (int q = 0; q < NSTAGE - 1; ++q) {
    if (ld.ok(p)) {
      issue_stage<3, 1, false>(p, ld, cm, sbase + p.stage0 + q * p.stage_bytes, smem + p.stage0 + q * p.stage_bytes, in,
                               out, LSE, nullptr);
      ld.next(p);
    }
    cp_async_commit();
  }
  uint32_t buf = 0;
  for (; cu.ok(p); cu.next(p)) {
    cp_async_wait<NSTAGE - 2>();
    __syncthreads();   // stage `buf` has landed for everyone; everyone is done with the previous stage
    {
      const uint32_t nb = buf == 0 ? NSTAGE - 1 : buf - 1;
      if (ld.ok(p)) {
        issue_stage<3, 1, false>(p, ld, cm, sbase + p.stage0 + nb * p.stage_bytes, smem + p.stage0 + nb * p.stage_bytes,
                                 in, out, LSE, nullptr);
        ld.next(p);
      }
      cp_async_commit();
    }
    const uint32_t stage = sbase + p.stage0 + buf * p.stage_bytes;
    const unsigned char* sp = smem + p.stage0 + buf * p.stage_bytes;
    x.Cv = *reinterpret_cast<const int*>(sp + p.off_cv);
    x.vcol_s = stage + p.off_vcol;
    const bool identity = x.Cv == s.C;
    const int MT = (x.Cv + 15) >> 4;
    // 64-bit bases once per stage, 32-bit offsets per task
    const size_t row0 = (size_t)cu.b * s.R + cu.r0;
    unsigned char* O_st = O + row0 * s.C * x.d2 + (size_t)cu.hgi * p.hg * DH * 2;
    float* LSE_st = LSE + (row0 * s.H + (size_t)cu.hgi * p.hg) * s.C;
    const uint32_t o_row = s.C * x.d2, l_row = s.H * s.C;
    TaskIt it{warp, 0, 0};
    if (MT > 0) {
      for (it.carry(MT, p.hg); it.r < cu.nrows; it.mt += nwarps, it.carry(MT, p.hg)) {
        const uint32_t off = (uint32_t)(it.r * x.Cv) * p.slot_stride + it.hl * DH * 2;
        unsigned char* O_row = O_st + (it.r * o_row + it.hl * DH * 2);
        float* LSE_row = LSE_st + (it.r * l_row + it.hl * s.C);
        if constexpr (KB == 0) {   // one-pass online softmax
          if (identity)
            fwd_task_1p<DH, true>(x, stage + off, stage + p.slot_bytes + off, stage + 2 * p.slot_bytes + off, it.mt * 16,
                               O_row, LSE_row);
          else
            fwd_task_1p<DH, false>(x, stage + off, stage + p.slot_bytes + off, stage + 2 * p.slot_bytes + off, it.mt * 16,
                                O_row, LSE_row);
        } else {                   // two passes over at most KB key blocks
          // (operands spelled out: with `sk = sq + slot_bytes` temporaries ptxas caps these kernels at 80 registers)
          if (identity)
            fwd_task_2p<DH, true, KB>(x, stage + off, stage + p.slot_bytes + off, stage + 2 * p.slot_bytes + off,
                                      it.mt * 16, O_row, LSE_row);
          else
            fwd_task_2p<DH, false, KB>(x, stage + off, stage + p.slot_bytes + off, stage + 2 * p.slot_bytes + off,
                                       it.mt * 16, O_row, LSE_row);
        }
      }
    }
    buf = buf + 1 == NSTAGE ? 0 : buf + 1;
  }
  cp_async_wait<0>();
}

template <int DH, int NSTAGE>
__global__ void __launch_bounds__(kMaxWarps * 32) feature_bwd_mma_kernel(
    const __grid_constant__ FeatParams p, const unsigned char* __restrict__ Q, const unsigned char* __restrict__ K,
    const unsigned char* __restrict__ V, const unsigned char* __restrict__ O, const unsigned char* __restrict__ dO,
    const float* __restrict__ LSE, unsigned char* __restrict__ dQ, unsigned char* __restrict__ dK,
    unsigned char* __restrict__ dV, uint32_t smem_total) {
  extern __shared__ __align__(16) unsigned char smem[];
  zero_smem(smem, smem_total);
  const uint32_t sbase = smem_addr(smem);
  const int warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  // slot order: Q, K, V, dO, O
  const unsigned char* const in[5] = {Q, K, V, dO, O};
  unsigned char* const out[3] = {dQ, dK, dV};
  const Shape& s = p.s;
  TaskCtx x;
  x.stg = sbase + warp * 16 * (DH * 2 + 16);
  x.lo.init(p.slot_stride);
  x.str = p.slot_stride;
  x.d2 = s.H * DH * 2;
  x.c2 = s.scale * kLog2e;
  x.scale = s.scale;

  Unit ld, cu;
  ColMask cm;
  ld.init(p);
  cu = ld;
#pragma unroll
  for (int q = 0; q < NSTAGE - 1; ++q) {
    if (ld.ok(p)) {
      issue_stage<5, 3, true>(p, ld, cm, sbase + p.stage0 + q * p.stage_bytes, smem + p.stage0 + q * p.stage_bytes, in,
                              out, nullptr, LSE);
      ld.next(p);
    }
    cp_async_commit();
  }
  uint32_t buf = 0;
  for (; cu.ok(p); cu.next(p)) {
    cp_async_wait<NSTAGE - 2>();
    __syncthreads();
    {
      const uint32_t nb = buf == 0 ? NSTAGE - 1 : buf - 1;
      if (ld.ok(p)) {
        issue_stage<5, 3, true>(p, ld, cm, sbase + p.stage0 + nb * p.stage_bytes, smem + p.stage0 + nb * p.stage_bytes,
                                in, out, nullptr, LSE);
        ld.next(p);
      }
      cp_async_commit();
    }
    const uint32_t stage = sbase + p.stage0 + buf * p.stage_bytes;
    unsigned char* sp = smem + p.stage0 + buf * p.stage_bytes;
    x.Cv = *reinterpret_cast<const int*>(sp + p.off_cv);
    x.vcol_s = stage + p.off_vcol;
    const bool identity = x.Cv == s.C;
    const int Cv = x.Cv;
    float* sL = reinterpret_cast<float*>(sp + p.off_lse);
    float* sD = reinterpret_cast<float*>(sp + p.off_D);
    // D[r][hl][v] = sum_k dO O over the head's dh elements; LSE -> log2 units.  Thread <-> (r, hl, v).
    if (Cv > 0) {
      int v = threadIdx.x, rh = 0;
      const int nrh = cu.nrows * p.hg;
      while (true) {
        while (v >= Cv) { v -= Cv; ++rh; }
        if (rh >= nrh) break;
        int r = 0, hl = rh;
        while (hl >= p.hg) { hl -= p.hg; ++r; }
        const uint32_t off = (uint32_t)(r * Cv + v) * p.slot_stride + hl * DH * 2;
        float acc = 0.f;
#pragma unroll
        for (int k = 0; k < DH / 8; ++k) {
          float a[8], g[8];
          unpack8(lds128(stage + 3 * p.slot_bytes + off + 16 * k), g);
          unpack8(lds128(stage + 4 * p.slot_bytes + off + 16 * k), a);
#pragma unroll
          for (int e = 0; e < 8; ++e) acc = fmaf(a[e], g[e], acc);
        }
        const int si = rh * p.Cp + v;
        sD[si] = acc;
        sL[si] *= kLog2e;
        v += blockDim.x;
      }
    }
    __syncthreads();
    const int MT = (Cv + 15) >> 4;
    const size_t rowcell0 = ((size_t)cu.b * s.R + cu.r0) * s.C;
    // tasks 0 .. nrows*hg*MT-1: key-stationary; the same count again: query-stationary
    TaskIt it{warp, 0, 0};
    bool key_task = true;
    while (MT > 0) {
      it.carry(MT, p.hg);
      if (it.r >= cu.nrows) {
        if (!key_task) break;
        key_task = false;
        it.r -= cu.nrows;
        continue;
      }
      const uint32_t off = (uint32_t)(it.r * Cv) * p.slot_stride + it.hl * DH * 2;
      const float* L = sL + (it.r * p.hg + it.hl) * p.Cp;
      const float* D = sD + (it.r * p.hg + it.hl) * p.Cp;
      const size_t goff = (rowcell0 + (size_t)it.r * s.C) * x.d2 + (cu.hgi * p.hg + it.hl) * DH * 2;
      const uint32_t sq = stage + off, sk = sq + p.slot_bytes, sv = sk + p.slot_bytes, sg = sv + p.slot_bytes;
      if (key_task) {
        if (identity) bwd_key_task<DH, true>(x, sq, sk, sv, sg, L, D, it.mt * 16, dK + goff, dV + goff);
        else bwd_key_task<DH, false>(x, sq, sk, sv, sg, L, D, it.mt * 16, dK + goff, dV + goff);
      } else {
        if (identity) bwd_query_task<DH, true>(x, sq, sk, sv, sg, L, D, it.mt * 16, dQ + goff);
        else bwd_query_task<DH, false>(x, sq, sk, sv, sg, L, D, it.mt * 16, dQ + goff);
      }
      it.mt += nwarps;
    }
    buf = buf + 1 == NSTAGE ? 0 : buf + 1;
  }
  cp_async_wait<0>();
}

// ---- host side: stage geometry ---------------------------------------------------------------------------
uint32_t magic(uint32_t d) { return d <= 1 ? 0u : (uint32_t)((1ull << 32) / d) + 1u; }
int env_int(const char* name, int dflt) {
  const char* e = getenv(name);
  return e && *e ? atoi(e) : dflt;
}

constexpr size_t kSmemPerSM = 227 * 1024;

struct Plan {
  FeatParams p;
  size_t smem;
  int warps, ctas_per_sm;
};

// Picks heads-per-unit, rows-per-unit, warps per CTA and ring depth.
Plan make_plan(const Shape& s, bool bwd) {
  Plan pl{};
  FeatParams& p = pl.p;
  p.s = s;
  const int nslot = bwd ? 5 : 3;
  p.Cp = (s.C + 15) / 16 * 16;
  auto stage_bytes = [&](int hg, int rows) {
    const size_t stride = (size_t)hg * s.dh * 2 + 16;
    size_t b = nslot * (size_t)rows * s.C * stride + 16 * stride;   // slots + read slack after the last one
    if (bwd) b += (size_t)2 * rows * hg * p.Cp * 4;
    return b + 256 + 128 /* vcol */ + 16 /* Cv */;
  };
  // Measured on B200 (profiles/r01_feature_mma.md): small CTAs with small stages win -- many CTAs per SM
  // hide each other's barrier and latency bubbles.  Head groups of 128 contiguous bytes per cell
  // (one L2 line), 1-2 table rows per stage, 2 warps (C <= 16) or 4 warps per CTA.
  const size_t target = (size_t)env_int("TABATTN_FEAT_STAGE_KB", 40) * 1024;
  int hg = 128 / (s.dh * 2);
  if (hg < 1) hg = 1;
  while (hg > 1 && s.H % hg != 0) --hg;
  while (hg > 1 && stage_bytes(hg, 1) > target) {
    --hg;
    while (hg > 1 && s.H % hg != 0) --hg;
  }
  int warps = s.C <= 16 ? 2 : 4;
  int nstage = env_int("TABATTN_FEAT_NSTAGE", 2);
  if (bwd) {
    // The backward needs >= 12 resident warps per SM to cover its latencies (B200 sweep,
    // profiles/r01_s23_feature_sweep.md): ragged (C = 51) 1.63 -> 1.41 ms with one head per stage (4 CTAs per SM
    // instead of 2), feature_heavy (C = 101, already one head per stage) 0.94 -> 0.84 ms with 6 warps per CTA.
    auto ctas = [&](int hg_, int warps_) {
      const size_t smem = (size_t)warps_ * 16 * (s.dh * 2 + 16) + (size_t)nstage * stage_bytes(hg_, 1);
      int c = (int)(kSmemPerSM / (smem + 1024));
      const int by_regs = 65536 / (warps_ * 32 * (s.dh >= 64 ? 168 : 128));
      c = c < by_regs ? c : by_regs;
      return c < 1 ? 1 : (c > 8 ? 8 : c);
    };
    if (ctas(hg, warps) * warps < 12 && hg > 1 && ctas(1, warps) > ctas(hg, warps)) hg = 1;
    const int c = ctas(hg, warps);
    if (c * warps < 12) warps = (12 + c - 1) / c;
  }
  hg = env_int("TABATTN_FEAT_HG", hg);
  warps = env_int("TABATTN_FEAT_WARPS", warps);
  if (warps > kMaxWarps) warps = kMaxWarps;
  if (warps < 1) warps = 1;
  int rows = (!bwd && s.C <= 32 && s.R >= 2 && stage_bytes(hg, 2) <= target) ? 2 : 1;
  // backward: a stage should hold at least two tasks per warp (key- and query-stationary tasks of every
  // (row, head, 16-column tile)), else the per-stage barriers dominate: long_item (C = 21, one head per
  // stage, 4 warps) 1.15 -> 0.92 ms with two rows per stage (B200 sweep, profiles/r01_s23_feature_sweep.md)
  if (bwd && rows == 1 && s.R >= 2 && 2 * hg * ((s.C + 15) / 16) < 2 * warps && stage_bytes(hg, 2) <= target) rows = 2;
  rows = env_int("TABATTN_FEAT_ROWS", rows);
  const size_t stg_bytes = (size_t)warps * 16 * (s.dh * 2 + 16);
  p.hg = hg;
  p.nhg = s.H / hg;
  p.rows = rows;
  p.slot_stride = hg * s.dh * 2 + 16;
  p.chunks = hg * s.dh / 8;
  p.rb_per_table = (s.R + rows - 1) / rows;
  p.n_su = s.B * p.rb_per_table;
  p.div_chunks = magic(p.chunks);
  p.div_C = magic(s.C);
  p.div_hgC = magic(hg * s.C);
  p.slot_bytes = (uint32_t)((size_t)rows * s.C * p.slot_stride);
  uint32_t o = nslot * p.slot_bytes + 16 * p.slot_stride;
  p.off_lse = o;
  if (bwd) o += rows * hg * p.Cp * 4;
  p.off_D = o;
  if (bwd) o += rows * hg * p.Cp * 4;
  o += 256;
  p.off_vcol = o;
  o += 128;
  p.off_cv = o;
  o += 16;
  p.stage_bytes = o;
  p.stage0 = (uint32_t)stg_bytes;
  p.nstage = nstage;
  p.ld_dcell = warps * 32 / p.chunks;
  p.ld_dch = warps * 32 % p.chunks;
  pl.smem = stg_bytes + (size_t)nstage * p.stage_bytes;
  pl.warps = warps;
  int per_sm = (int)(kSmemPerSM / (pl.smem + 1024));
  per_sm = per_sm < 1 ? 1 : (per_sm > 8 ? 8 : per_sm);
  pl.ctas_per_sm = env_int("TABATTN_FEAT_CTAS", per_sm);
  return pl;
}

}  // namespace


namespace {

template <typename Kern, typename... Args>
cudaError_t launch_persistent(Kern kern, const Plan& pl, cudaStream_t stream, Args... args) {
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem);
  if (e != cudaSuccess) return e;
  int occ = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, pl.warps * 32, pl.smem);
  if (e != cudaSuccess) return e;
  if (occ < 1) return cudaErrorInvalidValue;
  const int per_sm = occ < pl.ctas_per_sm ? occ : pl.ctas_per_sm;
  const long long want = (long long)current_device()->num_sms * per_sm;
  const int grid = (int)(pl.p.n_su < want ? pl.p.n_su : want);
  if (env_int("TABATTN_FEAT_DEBUG", 0))
    fprintf(stderr, "feature plan: hg=%d rows=%d warps=%d nstage=%d stage=%u B smem=%zu B occ=%d ctas/sm=%d grid=%d\n",
            pl.p.hg, pl.p.rows, pl.warps, pl.p.nstage, pl.p.stage_bytes, pl.smem, occ, per_sm, grid);
  kern<<<grid, pl.warps * 32, pl.smem, stream>>>(pl.p, args..., (uint32_t)pl.smem);
  count_launch();
  return cudaGetLastError();
}

#define TABATTN_FEAT_DISPATCH(NAME, ...)                                              \
  switch (s.dh * 10 + pl.p.nstage) {                                                  \
    case 162: return launch_persistent(NAME<16, 2>, pl, stream, __VA_ARGS__);         \
    case 163: return launch_persistent(NAME<16, 3>, pl, stream, __VA_ARGS__);         \
    case 322: return launch_persistent(NAME<32, 2>, pl, stream, __VA_ARGS__);         \
    case 323: return launch_persistent(NAME<32, 3>, pl, stream, __VA_ARGS__);         \
    case 642: return launch_persistent(NAME<64, 2>, pl, stream, __VA_ARGS__);         \
    case 643: return launch_persistent(NAME<64, 3>, pl, stream, __VA_ARGS__);         \
    default: return cudaErrorInvalidValue;                                            \
  }

bool plan_ok(const Shape& s, const Plan& pl) {
  return pl.smem <= kSmemPerSM && pl.p.nstage >= 2 && pl.p.nstage <= 3 && pl.p.hg >= 1 && s.H % pl.p.hg == 0 &&
         pl.p.rows >= 1;
}

}  // namespace

cudaError_t launch_feature_bwd(const Shape& s, const void* Q, const void* K, const void* V, const void* O,
                               const void* dO, const float* LSE, void* dQ, void* dK, void* dV,
                               cudaStream_t stream) {
  const Plan pl = make_plan(s, true);
  if (!plan_ok(s, pl)) return cudaErrorInvalidValue;
  TABATTN_FEAT_DISPATCH(feature_bwd_mma_kernel, (const unsigned char*)Q, (const unsigned char*)K,
                        (const unsigned char*)V, (const unsigned char*)O, (const unsigned char*)dO, LSE,
                        (unsigned char*)dQ, (unsigned char*)dK, (unsigned char*)dV);
}

}  // namespace tabattn
