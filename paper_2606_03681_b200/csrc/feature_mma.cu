// Feature-axis attention, forward and backward.
//
// The feature axis is short (C <= 128 columns) and the path is HBM-bound (0.58*C flop/B), so the
// kernels are built around the memory stream, not around the contraction:
//   * persistent CTAs of 4 warps, several per SM; every CTA walks "stage units" = (table b, block of
//     `rows` table rows, group of `hg` heads) and keeps a ring of NSTAGE stages in flight with
//     16-byte cp.async (LDGSTS) copies -- one stage is being computed while the next ones land;
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

#include <stdlib.h>

namespace tabattn {

namespace {

constexpr int kWarps = 4;
constexpr int kThreads = kWarps * 32;
constexpr int kMaxStages = 4;

struct FeatParams {
  Shape s;
  int hg, nhg;          // heads per stage unit, units per (table, row block)
  int rows;             // table rows per stage unit
  int Cp;               // cell slots per table row: C rounded up to 16
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
  __device__ __forceinline__ void build(const Shape& s, int b) {
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

// ---- stage loader ------------------------------------------------------------------------------------
// Issues the cp.async copies of one stage unit into ring buffer `stage` (shared-memory byte address)
// and zero-fills the outputs of the unit's invalid cells.  NIN input tensors share one offset map.
// Called by all threads of the CTA (uniformly); the caller commits the group.
template <int NIN, int NOUT, bool BWD>
__device__ __forceinline__ void issue_stage(const FeatParams& p, const Unit& u, uint32_t stage, unsigned char* stage_ptr,
                                            const unsigned char* const (&in)[NIN], unsigned char* const (&out)[NOUT],
                                            float* __restrict__ LSE_out, const float* __restrict__ LSE_in) {
  const Shape& s = p.s;
  ColMask cm;
  cm.build(s, u.b);
  const int d2 = s.H * s.dh * 2;                    // bytes per cell
  const int hoff = u.hgi * p.hg * s.dh * 2;         // byte offset of the head group inside a cell
  const size_t row0 = (size_t)u.b * s.R + u.r0;
  const uint32_t total = (uint32_t)u.nrows * s.C * p.chunks;
  for (uint32_t idx = threadIdx.x; idx < total; idx += kThreads) {
    const uint32_t cellidx = fdiv(idx, p.div_chunks);
    const uint32_t ch = idx - cellidx * p.chunks;
    const uint32_t r = fdiv(cellidx, p.div_C);
    const int c = (int)(cellidx - r * s.C);
    const size_t goff = ((row0 + r) * s.C + c) * (size_t)d2 + hoff + ch * 16;
    if (cm.valid(c)) {
      const int v = cm.rank(c);
      const uint32_t soff = (r * p.Cp + v) * p.slot_stride + ch * 16;
#pragma unroll
      for (int k = 0; k < NIN; ++k) cp_async16(stage + k * p.slot_bytes + soff, in[k] + goff);
      if (r == 0 && ch == 0) stage_ptr[p.off_vcol + v] = (unsigned char)c;
    } else {
#pragma unroll
      for (int k = 0; k < NOUT; ++k) stg_v4(out[k] + goff, make_uint4(0, 0, 0, 0));
      if (!BWD && ch == 0) {
        for (int hl = 0; hl < p.hg; ++hl) LSE_out[((row0 + r) * s.H + u.hgi * p.hg + hl) * s.C + c] = 0.f;
      }
    }
  }
  if (BWD) {
    // saved LSE of the unit's valid (row, head, column) triples -> sL[(r*hg + hl)*Cp + v]
    const uint32_t total2 = (uint32_t)u.nrows * p.hg * s.C;
    for (uint32_t idx = threadIdx.x; idx < total2; idx += kThreads) {
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

// Store a 16 x DH bf16 tile that sits in the warp's staging area to the cells (row r of the unit,
// compacted columns v0 .. v0+15, head h) of a [B,R,C,H,dh] tensor, as full 16-byte vectors.
template <int DH>
__device__ __forceinline__ void store_tile(uint32_t stg, unsigned char* dst, const FeatParams& p, const Unit& u, int r,
                                           int h, int v0, int Cv, const unsigned char* vcol) {
  constexpr int SSTR = DH * 2 + 16, CH = DH / 8;
  const int lane = threadIdx.x & 31;
  const Shape& s = p.s;
  const size_t rowcell = ((size_t)u.b * s.R + u.r0 + r) * s.C;
#pragma unroll
  for (int idx = lane; idx < 16 * CH; idx += 32) {
    const int row = idx / CH, ch = idx - row * CH;
    if (v0 + row < Cv) {
      const int c = vcol[v0 + row];
      const uint4 val = lds128(stg + row * SSTR + ch * 16);
      stg_v4(dst + ((rowcell + c) * s.H + h) * (size_t)(DH * 2) + ch * 16, val);
    }
  }
}

// Write an accumulator tile (C fragments of DH/8 n-tiles, rows g and g+8) to the staging area as bf16,
// scaled per row.
template <int DH>
__device__ __forceinline__ void stage_tile(uint32_t stg, const float (&acc)[DH / 8][4], float mul0, float mul1) {
  constexpr int SSTR = DH * 2 + 16;
  const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
#pragma unroll
  for (int nt = 0; nt < DH / 8; ++nt) {
    sts32(stg + g * SSTR + nt * 16 + t * 4, pack_bf16(acc[nt][0] * mul0, acc[nt][1] * mul0));
    sts32(stg + (g + 8) * SSTR + nt * 16 + t * 4, pack_bf16(acc[nt][2] * mul1, acc[nt][3] * mul1));
  }
}

// ---- forward task: one warp, 16 query cells (compacted columns v0..v0+15) of one (row, head) -----------
// sQ/sK/sV: shared byte addresses of the slots at (row r of the unit, column slot 0, this head).
template <int DH>
__device__ __forceinline__ void fwd_task(const FeatParams& p, const Unit& u, uint32_t sQ, uint32_t sK, uint32_t sV,
                                         int r, int h, int v0, int Cv, const unsigned char* vcol, uint32_t stg,
                                         unsigned char* O, float* __restrict__ LSE) {
  constexpr int KS = DH / 16, NT = DH / 8;
  const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int str = p.slot_stride;
  const float c2 = p.s.scale * kLog2e;
  uint32_t qa[KS][4];
  {
    const uint32_t a = sQ + (v0 + (lane & 15)) * str + (lane >> 4) * 16;
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) ldsm4(a + ks * 32, qa[ks]);
  }
  float o[NT][4];
#pragma unroll
  for (int nt = 0; nt < NT; ++nt) o[nt][0] = o[nt][1] = o[nt][2] = o[nt][3] = 0.f;
  float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;
  // lane address patterns of the B-fragment loads
  const uint32_t kb_lane = ((lane & 7) + ((lane >> 4) << 3)) * str + ((lane >> 3) & 1) * 16;  // [n][k] operand
  const uint32_t vb_lane = ((lane & 7) + (((lane >> 3) & 1) << 3)) * str + (lane >> 4) * 16;  // [k][n] operand
  for (int k0 = 0; k0 < Cv; k0 += 32) {
    float sc[4][4];
#pragma unroll
    for (int nt = 0; nt < 4; ++nt) sc[nt][0] = sc[nt][1] = sc[nt][2] = sc[nt][3] = 0.f;
#pragma unroll
    for (int pr = 0; pr < 2; ++pr) {
      if (k0 + pr * 16 < Cv) {
        const uint32_t a = sK + (k0 + pr * 16) * str + kb_lane;
#pragma unroll
        for (int ks = 0; ks < KS; ++ks) {
          uint32_t kb[4];
          ldsm4(a + ks * 32, kb);
          mma_bf16(sc[2 * pr], qa[ks], kb[0], kb[1]);
          mma_bf16(sc[2 * pr + 1], qa[ks], kb[2], kb[3]);
        }
      }
    }
    // scale to log2 units, mask keys >= Cv (padded slots), row maxima of rows g and g+8
    float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
    for (int nt = 0; nt < 4; ++nt) {
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int key = k0 + nt * 8 + 2 * t + (e & 1);
        sc[nt][e] = key < Cv ? sc[nt][e] * c2 : -INFINITY;
      }
      mx0 = fmaxf(mx0, fmaxf(sc[nt][0], sc[nt][1]));
      mx1 = fmaxf(mx1, fmaxf(sc[nt][2], sc[nt][3]));
    }
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
    uint32_t pa[2][4];
#pragma unroll
    for (int nt = 0; nt < 4; ++nt) {
      const float p0 = fast_exp2(sc[nt][0] - m0), p1 = fast_exp2(sc[nt][1] - m0);
      const float p2 = fast_exp2(sc[nt][2] - m1), p3 = fast_exp2(sc[nt][3] - m1);
      l0 += p0 + p1;
      l1 += p2 + p3;
      pa[nt >> 1][(nt & 1) * 2] = pack_bf16(p0, p1);
      pa[nt >> 1][(nt & 1) * 2 + 1] = pack_bf16(p2, p3);
    }
#pragma unroll
    for (int pr = 0; pr < 2; ++pr) {
      if (k0 + pr * 16 < Cv) {
        const uint32_t a = sV + (k0 + pr * 16) * str + vb_lane;
#pragma unroll
        for (int np = 0; np < NT / 2; ++np) {
          uint32_t vb[4];
          ldsm4t(a + np * 32, vb);
          mma_bf16(o[2 * np], pa[pr], vb[0], vb[1]);
          mma_bf16(o[2 * np + 1], pa[pr], vb[2], vb[3]);
        }
      }
    }
  }
  l0 = quad_sum(l0);
  l1 = quad_sum(l1);
  stage_tile<DH>(stg, o, 1.f / l0, 1.f / l1);
  __syncwarp();
  store_tile<DH>(stg, O, p, u, r, h, v0, Cv, vcol);
  if (t == 0) {
    const Shape& s = p.s;
    float* lrow = LSE + (((size_t)u.b * s.R + u.r0 + r) * s.H + h) * s.C;
    if (v0 + g < Cv) lrow[vcol[v0 + g]] = (m0 + log2f(l0)) * kLn2;
    if (v0 + g + 8 < Cv) lrow[vcol[v0 + g + 8]] = (m1 + log2f(l1)) * kLn2;
  }
  __syncwarp();
}

template <int DH, int NSTAGE>
__global__ void __launch_bounds__(kThreads) feature_fwd_mma_kernel(const __grid_constant__ FeatParams p,
                                                                   const unsigned char* __restrict__ Q,
                                                                   const unsigned char* __restrict__ K,
                                                                   const unsigned char* __restrict__ V,
                                                                   unsigned char* __restrict__ O,
                                                                   float* __restrict__ LSE, uint32_t smem_total) {
  extern __shared__ __align__(16) unsigned char smem[];
  for (uint32_t i = threadIdx.x * 16; i < smem_total; i += kThreads * 16)
    *reinterpret_cast<uint4*>(smem + i) = make_uint4(0, 0, 0, 0);
  __syncthreads();
  const uint32_t sbase = smem_addr(smem);
  const int warp = threadIdx.x >> 5;
  const uint32_t stg = sbase + warp * 16 * (DH * 2 + 16);
  const unsigned char* const in[3] = {Q, K, V};
  unsigned char* const out[1] = {O};

  Unit ld, cu;
  ld.init(p);
  cu = ld;
#pragma unroll
  for (int q = 0; q < NSTAGE - 1; ++q) {
    if (ld.ok(p)) {
      issue_stage<3, 1, false>(p, ld, sbase + p.stage0 + q * p.stage_bytes, smem + p.stage0 + q * p.stage_bytes, in, out,
                               LSE, nullptr);
      ld.next(p);
    }
    cp_async_commit();
  }
  for (uint32_t q = 0; cu.ok(p); ++q, cu.next(p)) {
    cp_async_wait<NSTAGE - 2>();
    __syncthreads();   // stage q has landed for everyone; everyone is done with stage q-1
    {
      const uint32_t nb = (q + NSTAGE - 1) % NSTAGE;
      if (ld.ok(p)) {
        issue_stage<3, 1, false>(p, ld, sbase + p.stage0 + nb * p.stage_bytes, smem + p.stage0 + nb * p.stage_bytes, in,
                                 out, LSE, nullptr);
        ld.next(p);
      }
      cp_async_commit();
    }
    const uint32_t buf = q % NSTAGE;
    const uint32_t stage = sbase + p.stage0 + buf * p.stage_bytes;
    const unsigned char* sp = smem + p.stage0 + buf * p.stage_bytes;
    const int Cv = *reinterpret_cast<const int*>(sp + p.off_cv);
    const unsigned char* vcol = sp + p.off_vcol;
    const int MT = (Cv + 15) >> 4;
    const int ntask = cu.nrows * p.hg * MT;
    for (int task = warp; task < ntask; task += kWarps) {
      const int mt = task % MT, rest = task / MT;
      const int hl = rest % p.hg, r = rest / p.hg;
      const uint32_t off = (uint32_t)(r * p.Cp) * p.slot_stride + hl * DH * 2;
      fwd_task<DH>(p, cu, stage + off, stage + p.slot_bytes + off, stage + 2 * p.slot_bytes + off, r,
                   cu.hgi * p.hg + hl, mt * 16, Cv, vcol, stg, O, LSE);
    }
  }
  cp_async_wait<0>();
}

// ---- backward, key-stationary task: 16 key cells (slots j0..j0+15) of one (row, head) -> dV, dK -----------
// sL / sD: this (row, head)'s lse*log2e and D vectors, indexed by column slot.
template <int DH>
__device__ __forceinline__ void bwd_key_task(const FeatParams& p, const Unit& u, uint32_t sQ, uint32_t sK, uint32_t sV,
                                             uint32_t sG, const float* sL, const float* sD, int r, int h, int j0,
                                             int Cv, const unsigned char* vcol, uint32_t stg, unsigned char* dK,
                                             unsigned char* dV) {
  constexpr int KS = DH / 16, NT = DH / 8;
  const int lane = threadIdx.x & 31, t = lane & 3;
  const int str = p.slot_stride;
  const float c2 = p.s.scale * kLog2e;
  uint32_t ka[KS][4], va[KS][4];
  {
    const uint32_t off = (j0 + (lane & 15)) * str + (lane >> 4) * 16;
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
      ldsm4(sK + off + ks * 32, ka[ks]);
      ldsm4(sV + off + ks * 32, va[ks]);
    }
  }
  float dv[NT][4], dk[NT][4];
#pragma unroll
  for (int nt = 0; nt < NT; ++nt) {
    dv[nt][0] = dv[nt][1] = dv[nt][2] = dv[nt][3] = 0.f;
    dk[nt][0] = dk[nt][1] = dk[nt][2] = dk[nt][3] = 0.f;
  }
  const uint32_t nb_lane = ((lane & 7) + ((lane >> 4) << 3)) * str + ((lane >> 3) & 1) * 16;  // [n][k] operand
  const uint32_t tb_lane = ((lane & 7) + (((lane >> 3) & 1) << 3)) * str + (lane >> 4) * 16;  // [k][n] operand
  for (int i0 = 0; i0 < Cv; i0 += 32) {
    float st[4][4], dp[4][4];
#pragma unroll
    for (int nt = 0; nt < 4; ++nt) {
      st[nt][0] = st[nt][1] = st[nt][2] = st[nt][3] = 0.f;
      dp[nt][0] = dp[nt][1] = dp[nt][2] = dp[nt][3] = 0.f;
    }
#pragma unroll
    for (int pr = 0; pr < 2; ++pr) {
      if (i0 + pr * 16 < Cv) {
        const uint32_t off = (i0 + pr * 16) * str + nb_lane;
#pragma unroll
        for (int ks = 0; ks < KS; ++ks) {
          uint32_t b[4];
          ldsm4(sQ + off + ks * 32, b);
          mma_bf16(st[2 * pr], ka[ks], b[0], b[1]);
          mma_bf16(st[2 * pr + 1], ka[ks], b[2], b[3]);
          ldsm4(sG + off + ks * 32, b);
          mma_bf16(dp[2 * pr], va[ks], b[0], b[1]);
          mma_bf16(dp[2 * pr + 1], va[ks], b[2], b[3]);
        }
      }
    }
    // P^T[j][i] = exp2(S^T c2 - lse2_i), dS^T = P^T (dP^T - D_i); queries i >= Cv (padded slots) -> 0
    uint32_t pa[2][4], da[2][4];
#pragma unroll
    for (int nt = 0; nt < 4; ++nt) {
      const int i = i0 + nt * 8 + 2 * t;
      const float2 L = *reinterpret_cast<const float2*>(sL + i);
      const float2 D = *reinterpret_cast<const float2*>(sD + i);
      const bool ok0 = i < Cv, ok1 = i + 1 < Cv;
      const float p0 = ok0 ? fast_exp2(fmaf(st[nt][0], c2, -L.x)) : 0.f;
      const float p1 = ok1 ? fast_exp2(fmaf(st[nt][1], c2, -L.y)) : 0.f;
      const float p2 = ok0 ? fast_exp2(fmaf(st[nt][2], c2, -L.x)) : 0.f;
      const float p3 = ok1 ? fast_exp2(fmaf(st[nt][3], c2, -L.y)) : 0.f;
      pa[nt >> 1][(nt & 1) * 2] = pack_bf16(p0, p1);
      pa[nt >> 1][(nt & 1) * 2 + 1] = pack_bf16(p2, p3);
      da[nt >> 1][(nt & 1) * 2] = pack_bf16(p0 * (dp[nt][0] - D.x), p1 * (dp[nt][1] - D.y));
      da[nt >> 1][(nt & 1) * 2 + 1] = pack_bf16(p2 * (dp[nt][2] - D.x), p3 * (dp[nt][3] - D.y));
    }
#pragma unroll
    for (int pr = 0; pr < 2; ++pr) {
      if (i0 + pr * 16 < Cv) {
        const uint32_t off = (i0 + pr * 16) * str + tb_lane;
#pragma unroll
        for (int np = 0; np < NT / 2; ++np) {
          uint32_t b[4];
          ldsm4t(sG + off + np * 32, b);
          mma_bf16(dv[2 * np], pa[pr], b[0], b[1]);
          mma_bf16(dv[2 * np + 1], pa[pr], b[2], b[3]);
          ldsm4t(sQ + off + np * 32, b);
          mma_bf16(dk[2 * np], da[pr], b[0], b[1]);
          mma_bf16(dk[2 * np + 1], da[pr], b[2], b[3]);
        }
      }
    }
  }
  stage_tile<DH>(stg, dv, 1.f, 1.f);
  __syncwarp();
  store_tile<DH>(stg, dV, p, u, r, h, j0, Cv, vcol);
  __syncwarp();
  stage_tile<DH>(stg, dk, p.s.scale, p.s.scale);
  __syncwarp();
  store_tile<DH>(stg, dK, p, u, r, h, j0, Cv, vcol);
  __syncwarp();
}

// ---- backward, query-stationary task: 16 query cells (slots i0..i0+15) of one (row, head) -> dQ -----------
template <int DH>
__device__ __forceinline__ void bwd_query_task(const FeatParams& p, const Unit& u, uint32_t sQ, uint32_t sK,
                                               uint32_t sV, uint32_t sG, const float* sL, const float* sD, int r, int h,
                                               int i0, int Cv, const unsigned char* vcol, uint32_t stg,
                                               unsigned char* dQ) {
  constexpr int KS = DH / 16, NT = DH / 8;
  const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int str = p.slot_stride;
  const float c2 = p.s.scale * kLog2e;
  uint32_t qa[KS][4], ga[KS][4];
  {
    const uint32_t off = (i0 + (lane & 15)) * str + (lane >> 4) * 16;
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
      ldsm4(sQ + off + ks * 32, qa[ks]);
      ldsm4(sG + off + ks * 32, ga[ks]);
    }
  }
  // rows g and g+8 of the tile; padded rows read stale (finite) statistics and are never stored
  const float L0 = sL[i0 + g], L1 = sL[i0 + g + 8], D0 = sD[i0 + g], D1 = sD[i0 + g + 8];
  float dq[NT][4];
#pragma unroll
  for (int nt = 0; nt < NT; ++nt) dq[nt][0] = dq[nt][1] = dq[nt][2] = dq[nt][3] = 0.f;
  const uint32_t nb_lane = ((lane & 7) + ((lane >> 4) << 3)) * str + ((lane >> 3) & 1) * 16;
  const uint32_t tb_lane = ((lane & 7) + (((lane >> 3) & 1) << 3)) * str + (lane >> 4) * 16;
  for (int k0 = 0; k0 < Cv; k0 += 32) {
    float sc[4][4], dp[4][4];
#pragma unroll
    for (int nt = 0; nt < 4; ++nt) {
      sc[nt][0] = sc[nt][1] = sc[nt][2] = sc[nt][3] = 0.f;
      dp[nt][0] = dp[nt][1] = dp[nt][2] = dp[nt][3] = 0.f;
    }
#pragma unroll
    for (int pr = 0; pr < 2; ++pr) {
      if (k0 + pr * 16 < Cv) {
        const uint32_t off = (k0 + pr * 16) * str + nb_lane;
#pragma unroll
        for (int ks = 0; ks < KS; ++ks) {
          uint32_t b[4];
          ldsm4(sK + off + ks * 32, b);
          mma_bf16(sc[2 * pr], qa[ks], b[0], b[1]);
          mma_bf16(sc[2 * pr + 1], qa[ks], b[2], b[3]);
          ldsm4(sV + off + ks * 32, b);
          mma_bf16(dp[2 * pr], ga[ks], b[0], b[1]);
          mma_bf16(dp[2 * pr + 1], ga[ks], b[2], b[3]);
        }
      }
    }
    uint32_t da[2][4];
#pragma unroll
    for (int nt = 0; nt < 4; ++nt) {
      const int key = k0 + nt * 8 + 2 * t;
      const bool ok0 = key < Cv, ok1 = key + 1 < Cv;   // keys in padded slots: P = 0 exactly
      const float p0 = ok0 ? fast_exp2(fmaf(sc[nt][0], c2, -L0)) : 0.f;
      const float p1 = ok1 ? fast_exp2(fmaf(sc[nt][1], c2, -L0)) : 0.f;
      const float p2 = ok0 ? fast_exp2(fmaf(sc[nt][2], c2, -L1)) : 0.f;
      const float p3 = ok1 ? fast_exp2(fmaf(sc[nt][3], c2, -L1)) : 0.f;
      da[nt >> 1][(nt & 1) * 2] = pack_bf16(p0 * (dp[nt][0] - D0), p1 * (dp[nt][1] - D0));
      da[nt >> 1][(nt & 1) * 2 + 1] = pack_bf16(p2 * (dp[nt][2] - D1), p3 * (dp[nt][3] - D1));
    }
#pragma unroll
    for (int pr = 0; pr < 2; ++pr) {
      if (k0 + pr * 16 < Cv) {
        const uint32_t off = (k0 + pr * 16) * str + tb_lane;
#pragma unroll
        for (int np = 0; np < NT / 2; ++np) {
          uint32_t b[4];
          ldsm4t(sK + off + np * 32, b);
          mma_bf16(dq[2 * np], da[pr], b[0], b[1]);
          mma_bf16(dq[2 * np + 1], da[pr], b[2], b[3]);
        }
      }
    }
  }
  stage_tile<DH>(stg, dq, p.s.scale, p.s.scale);
  __syncwarp();
  store_tile<DH>(stg, dQ, p, u, r, h, i0, Cv, vcol);
  __syncwarp();
}

template <int DH, int NSTAGE>
__global__ void __launch_bounds__(kThreads) feature_bwd_mma_kernel(
    const __grid_constant__ FeatParams p, const unsigned char* __restrict__ Q, const unsigned char* __restrict__ K,
    const unsigned char* __restrict__ V, const unsigned char* __restrict__ O, const unsigned char* __restrict__ dO,
    const float* __restrict__ LSE, unsigned char* __restrict__ dQ, unsigned char* __restrict__ dK,
    unsigned char* __restrict__ dV, uint32_t smem_total) {
  extern __shared__ __align__(16) unsigned char smem[];
  for (uint32_t i = threadIdx.x * 16; i < smem_total; i += kThreads * 16)
    *reinterpret_cast<uint4*>(smem + i) = make_uint4(0, 0, 0, 0);
  __syncthreads();
  const uint32_t sbase = smem_addr(smem);
  const int warp = threadIdx.x >> 5;
  const uint32_t stg = sbase + warp * 16 * (DH * 2 + 16);
  // slot order: Q, K, V, dO, O
  const unsigned char* const in[5] = {Q, K, V, dO, O};
  unsigned char* const out[3] = {dQ, dK, dV};

  Unit ld, cu;
  ld.init(p);
  cu = ld;
#pragma unroll
  for (int q = 0; q < NSTAGE - 1; ++q) {
    if (ld.ok(p)) {
      issue_stage<5, 3, true>(p, ld, sbase + p.stage0 + q * p.stage_bytes, smem + p.stage0 + q * p.stage_bytes, in, out,
                              nullptr, LSE);
      ld.next(p);
    }
    cp_async_commit();
  }
  for (uint32_t q = 0; cu.ok(p); ++q, cu.next(p)) {
    cp_async_wait<NSTAGE - 2>();
    __syncthreads();
    {
      const uint32_t nb = (q + NSTAGE - 1) % NSTAGE;
      if (ld.ok(p)) {
        issue_stage<5, 3, true>(p, ld, sbase + p.stage0 + nb * p.stage_bytes, smem + p.stage0 + nb * p.stage_bytes, in,
                                out, nullptr, LSE);
        ld.next(p);
      }
      cp_async_commit();
    }
    const uint32_t buf = q % NSTAGE;
    const uint32_t stage = sbase + p.stage0 + buf * p.stage_bytes;
    unsigned char* sp = smem + p.stage0 + buf * p.stage_bytes;
    const int Cv = *reinterpret_cast<const int*>(sp + p.off_cv);
    const unsigned char* vcol = sp + p.off_vcol;
    float* sL = reinterpret_cast<float*>(sp + p.off_lse);
    float* sD = reinterpret_cast<float*>(sp + p.off_D);
    // D[r][hl][v] = sum_k dO O over the head's dh elements; LSE -> log2 units
    {
      const int n = cu.nrows * p.hg * Cv;
      for (int idx = threadIdx.x; idx < n; idx += kThreads) {
        const int v = idx % Cv, rest = idx / Cv;
        const int hl = rest % p.hg, r = rest / p.hg;
        const uint32_t off = (uint32_t)(r * p.Cp + v) * p.slot_stride + hl * DH * 2;
        float acc = 0.f;
#pragma unroll
        for (int k = 0; k < DH / 8; ++k) {
          float a[8], g[8];
          unpack8(lds128(stage + 3 * p.slot_bytes + off + 16 * k), g);
          unpack8(lds128(stage + 4 * p.slot_bytes + off + 16 * k), a);
#pragma unroll
          for (int e = 0; e < 8; ++e) acc = fmaf(a[e], g[e], acc);
        }
        const int si = (r * p.hg + hl) * p.Cp + v;
        sD[si] = acc;
        sL[si] *= kLog2e;
      }
    }
    __syncthreads();
    const int MT = (Cv + 15) >> 4;
    const int nhalf = cu.nrows * p.hg * MT;
    for (int task = warp; task < 2 * nhalf; task += kWarps) {
      const bool key_task = task < nhalf;
      const int tk = key_task ? task : task - nhalf;
      const int mt = tk % MT, rest = tk / MT;
      const int hl = rest % p.hg, r = rest / p.hg;
      const uint32_t off = (uint32_t)(r * p.Cp) * p.slot_stride + hl * DH * 2;
      const float* L = sL + (r * p.hg + hl) * p.Cp;
      const float* D = sD + (r * p.hg + hl) * p.Cp;
      const int h = cu.hgi * p.hg + hl;
      if (key_task)
        bwd_key_task<DH>(p, cu, stage + off, stage + p.slot_bytes + off, stage + 2 * p.slot_bytes + off,
                         stage + 3 * p.slot_bytes + off, L, D, r, h, mt * 16, Cv, vcol, stg, dK, dV);
      else
        bwd_query_task<DH>(p, cu, stage + off, stage + p.slot_bytes + off, stage + 2 * p.slot_bytes + off,
                           stage + 3 * p.slot_bytes + off, L, D, r, h, mt * 16, Cv, vcol, stg, dQ);
    }
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

// Picks heads-per-unit, rows-per-unit and ring depth: a stage of roughly 16-48 KB (enough bytes in
// flight per SM to cover HBM latency with 2-3 CTAs per SM), at least ~3 tasks per warp per stage.
FeatParams make_plan(const Shape& s, bool bwd, size_t* smem_total, int* ctas_per_sm) {
  FeatParams p{};
  p.s = s;
  const int nslot = bwd ? 5 : 3;
  p.Cp = (s.C + 15) / 16 * 16;
  auto stage_bytes = [&](int hg, int rows) {
    size_t slot = (size_t)rows * p.Cp * (hg * s.dh * 2 + 16);
    size_t b = nslot * slot;
    if (bwd) b += (size_t)2 * rows * hg * p.Cp * 4;
    return b + 128 /* vcol */ + 16 /* Cv */ + 256 /* slack for reads of padded statistics */;
  };
  const size_t target = 40 * 1024;
  int hg = s.H;
  while (hg > 1 && stage_bytes(hg, 1) > target) {
    int nh = hg - 1;
    while (nh > 1 && (s.H % nh != 0)) --nh;
    hg = nh;
  }
  const int MT = (s.C + 15) / 16;
  const int per_row_tasks = hg * MT * (bwd ? 2 : 1);
  int rows = 1;
  while (rows < s.R && rows * per_row_tasks < 3 * kWarps && stage_bytes(hg, rows + 1) <= target) ++rows;
  hg = env_int("TABATTN_FEAT_HG", hg);
  rows = env_int("TABATTN_FEAT_ROWS", rows);
  const size_t stg_bytes = (size_t)kWarps * 16 * (s.dh * 2 + 16);
  const size_t sb = stage_bytes(hg, rows);
  int nstage = 3;
  if (stg_bytes + 3 * sb > 76 * 1024 && stg_bytes + 2 * sb <= kSmemPerSM) nstage = 2;
  if (stg_bytes + 3 * sb <= 56 * 1024) nstage = 4;
  nstage = env_int("TABATTN_FEAT_NSTAGE", nstage);
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
  p.slot_bytes = (uint32_t)((size_t)rows * p.Cp * p.slot_stride);
  uint32_t o = nslot * p.slot_bytes;
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
  *smem_total = stg_bytes + (size_t)nstage * p.stage_bytes;
  int per_sm = (int)(kSmemPerSM / (*smem_total + 1024));
  *ctas_per_sm = per_sm < 1 ? 1 : (per_sm > 4 ? 4 : per_sm);
  return p;
}

}  // namespace

bool feature_shape_supported(const Shape& s) { return s.C <= 128; }

namespace {

template <typename Kern, typename... Args>
cudaError_t launch_persistent(Kern kern, const FeatParams& p, size_t smem, int ctas_per_sm, cudaStream_t stream,
                              Args... args) {
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  int occ = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, kThreads, smem);
  if (e != cudaSuccess) return e;
  if (occ < 1) return cudaErrorInvalidValue;
  const int per_sm = occ < ctas_per_sm ? occ : ctas_per_sm;
  const long long want = (long long)num_sms() * per_sm;
  const int grid = (int)(p.n_su < want ? p.n_su : want);
  kern<<<grid, kThreads, smem, stream>>>(p, args..., (uint32_t)smem);
  count_launch();
  return cudaGetLastError();
}

#define TABATTN_FEAT_DISPATCH(NAME, ...)                                              \
  switch (s.dh * 10 + p.nstage) {                                                     \
    case 162: return launch_persistent(NAME<16, 2>, p, smem, per_sm, stream, __VA_ARGS__); \
    case 163: return launch_persistent(NAME<16, 3>, p, smem, per_sm, stream, __VA_ARGS__); \
    case 164: return launch_persistent(NAME<16, 4>, p, smem, per_sm, stream, __VA_ARGS__); \
    case 322: return launch_persistent(NAME<32, 2>, p, smem, per_sm, stream, __VA_ARGS__); \
    case 323: return launch_persistent(NAME<32, 3>, p, smem, per_sm, stream, __VA_ARGS__); \
    case 324: return launch_persistent(NAME<32, 4>, p, smem, per_sm, stream, __VA_ARGS__); \
    case 642: return launch_persistent(NAME<64, 2>, p, smem, per_sm, stream, __VA_ARGS__); \
    case 643: return launch_persistent(NAME<64, 3>, p, smem, per_sm, stream, __VA_ARGS__); \
    case 644: return launch_persistent(NAME<64, 4>, p, smem, per_sm, stream, __VA_ARGS__); \
    default: return cudaErrorInvalidValue;                                            \
  }

}  // namespace

cudaError_t launch_feature_fwd(const Shape& s, const void* Q, const void* K, const void* V, void* O, float* LSE,
                               cudaStream_t stream) {
  size_t smem;
  int per_sm;
  const FeatParams p = make_plan(s, false, &smem, &per_sm);
  if (smem > kSmemPerSM || p.nstage < 2 || p.nstage > kMaxStages || s.H % p.hg != 0) return cudaErrorInvalidValue;
  TABATTN_FEAT_DISPATCH(feature_fwd_mma_kernel, (const unsigned char*)Q, (const unsigned char*)K,
                        (const unsigned char*)V, (unsigned char*)O, LSE);
}

cudaError_t launch_feature_bwd(const Shape& s, const void* Q, const void* K, const void* V, const void* O,
                               const void* dO, const float* LSE, void* dQ, void* dK, void* dV,
                               cudaStream_t stream) {
  size_t smem;
  int per_sm;
  const FeatParams p = make_plan(s, true, &smem, &per_sm);
  if (smem > kSmemPerSM || p.nstage < 2 || p.nstage > kMaxStages || s.H % p.hg != 0) return cudaErrorInvalidValue;
  TABATTN_FEAT_DISPATCH(feature_bwd_mma_kernel, (const unsigned char*)Q, (const unsigned char*)K,
                        (const unsigned char*)V, (const unsigned char*)O, (const unsigned char*)dO, LSE,
                        (unsigned char*)dQ, (unsigned char*)dK, (unsigned char*)dV);
}

}  // namespace tabattn
