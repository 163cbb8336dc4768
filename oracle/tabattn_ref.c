/* oracle/tabattn_ref.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU statement of what libtabattn computes: the dual-axis
 * attention of a TabPFN-v2-style block (Fig. 3: "feature-axis
 * attention ... sample-axis attention"; "scaled dot-product
 * attention ... Explicit-QKV"), forward and analytic backward.  The method
 * reaches exactly the textbook result, so this file is that definition written
 * out: no tiling, no online softmax, no LSE reuse,
 * no blocking or reordering.  It shares no code with the CUDA path under
 * paper_2606_03681_b200/csrc/ and is only ever called from tests/, from
 * __graft_entry__.smoke() and from bench.py's cpu_baseline / --impl reference.
 *
 * Parity pins (tests/test_oracle_*.py): closed forms (identical keys, Q = 0,
 * single key, dominant key, key shift), the train-only-key invariances,
 * mask == physical compaction, NaN poisoning, an independent numpy fp64
 * softmax(QK^T)V, scalar-loop brute force (oracle/brute.py) and central finite
 * differences for every gradient.  The paper prints no worked attention value,
 * so no paper-printed fixture exists.
 *
 * Layout of every tensor: [B, R, C, H, dh] row-major, dh fastest
 * (SURVEY.md §8(a)).  Inputs are either bf16 bit patterns (uint16_t, widened
 * exactly to double) or doubles (in_f64 != 0; used by the finite-difference
 * tests, which need perturbations bf16 cannot hold).
 *
 * Readings of the paper adopted here: c1 keys of item
 * attention are rows [0, n_train[b]) for every query row; c2 scale = 1/sqrt(dh)
 * unless given; c3 no bias / dropout / causal mask; c7 invalid columns are
 * excluded as keys and produce zeros as queries, item attention skips them;
 * c11 LSE is the natural log of the scaled scores.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- exact widening of the input element type ---------------------------------- */
static double load_elem(const void *base, int in_f64, size_t idx) {
    if (in_f64) return ((const double *)base)[idx];
    uint32_t u = (uint32_t)((const uint16_t *)base)[idx] << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

/* Copy one head's sequence (L positions x dh) out of a [B,R,C,H,dh] tensor into a
 * dense double array.  pos[t] is the element offset of position t's vector. */
static void gather_seq(const void *base, int in_f64, const size_t *pos, int L, int dh, double *out) {
    for (int t = 0; t < L; ++t)
        for (int k = 0; k < dh; ++k) out[(size_t)t * dh + k] = load_elem(base, in_f64, pos[t] + k);
}

/* ---- the definition: one head, one sequence, dense arrays ------------------------
 * q [Lq,dh], k [Lk,dh], v [Lk,dh].  SURVEY.md §8(c) steps 1-3:
 *   s_ij = scale * <q_i, k_j>;  m_i = max_j s_ij;  l_i = sum_j exp(s_ij - m_i);
 *   p_ij = exp(s_ij - m_i) / l_i;  LSE_i = m_i + ln l_i;  o_i = sum_j p_ij v_j.  */
static void attn_fwd_dense(int Lq, int Lk, int dh, const double *q, const double *k, const double *v,
                           double scale, double *o, double *lse) {
    double *s = (double *)malloc(sizeof(double) * (size_t)Lk);
    for (int i = 0; i < Lq; ++i) {
        double m = -INFINITY;
        for (int j = 0; j < Lk; ++j) {
            double acc = 0.0;
            for (int t = 0; t < dh; ++t) acc += q[(size_t)i * dh + t] * k[(size_t)j * dh + t];
            s[j] = scale * acc;
            if (s[j] > m) m = s[j];
        }
        double l = 0.0;
        for (int j = 0; j < Lk; ++j) l += exp(s[j] - m);
        for (int t = 0; t < dh; ++t) o[(size_t)i * dh + t] = 0.0;
        for (int j = 0; j < Lk; ++j) {
            double p = exp(s[j] - m) / l;
            for (int t = 0; t < dh; ++t) o[(size_t)i * dh + t] += p * v[(size_t)j * dh + t];
        }
        lse[i] = m + log(l);
    }
    free(s);
}

/* SURVEY.md §8(c) steps 5-7, given the upstream gradient g = dO [Lq,dh]:
 *   dP_ij = <g_i, v_j>;  D_i = sum_j p_ij dP_ij;  dS_ij = p_ij (dP_ij - D_i);
 *   dv_j = sum_i p_ij g_i;  dq_i = scale sum_j dS_ij k_j;  dk_j = scale sum_i dS_ij q_i.
 * Recomputes p from q,k (takes neither O nor LSE). */
static void attn_bwd_dense(int Lq, int Lk, int dh, const double *q, const double *k, const double *v,
                           const double *g, double scale, double *dq, double *dk, double *dv) {
    double *p = (double *)malloc(sizeof(double) * (size_t)Lk);
    double *dp = (double *)malloc(sizeof(double) * (size_t)Lk);
    for (size_t x = 0; x < (size_t)Lk * dh; ++x) { dk[x] = 0.0; dv[x] = 0.0; }
    for (int i = 0; i < Lq; ++i) {
        double m = -INFINITY;
        for (int j = 0; j < Lk; ++j) {
            double acc = 0.0;
            for (int t = 0; t < dh; ++t) acc += q[(size_t)i * dh + t] * k[(size_t)j * dh + t];
            p[j] = scale * acc;
            if (p[j] > m) m = p[j];
        }
        double l = 0.0;
        for (int j = 0; j < Lk; ++j) l += exp(p[j] - m);
        for (int j = 0; j < Lk; ++j) p[j] = exp(p[j] - m) / l;
        double D = 0.0;
        for (int j = 0; j < Lk; ++j) {
            double acc = 0.0;
            for (int t = 0; t < dh; ++t) acc += g[(size_t)i * dh + t] * v[(size_t)j * dh + t];
            dp[j] = acc;
            D += p[j] * acc;
        }
        for (int t = 0; t < dh; ++t) dq[(size_t)i * dh + t] = 0.0;
        for (int j = 0; j < Lk; ++j) {
            double ds = p[j] * (dp[j] - D);
            for (int t = 0; t < dh; ++t) {
                dv[(size_t)j * dh + t] += p[j] * g[(size_t)i * dh + t];
                dk[(size_t)j * dh + t] += scale * ds * q[(size_t)i * dh + t];
                dq[(size_t)i * dh + t] += scale * ds * k[(size_t)j * dh + t];
            }
        }
    }
    free(p);
    free(dp);
}

static double pick_scale(double scale, int dh) { return scale > 0.0 ? scale : 1.0 / sqrt((double)dh); }

static void set_threads(int nthreads) {
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
}

int ref_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ================================================================================
 * Feature attention ("feature-axis attention"): for each selected
 * (b, r) and each head, the sequence runs over the VALID columns of that row.
 * Outputs are compact per selection: O/dQ/dK/dV [n_sel, C, H, dh], LSE [n_sel, H, C];
 * invalid columns hold 0.
 * mode 0 = forward (writes O, LSE), mode 1 = backward (writes dQ, dK, dV).
 * ================================================================================ */
static int feature_run(int mode, const void *Q, const void *K, const void *V, const void *dO, int in_f64,
                       int B, int R, int C, int H, int dh, const uint8_t *col_valid, double scale,
                       int n_sel, const int32_t *sel_b, const int32_t *sel_r,
                       double *out0, double *out1, double *out2, int nthreads) {
    if (B < 1 || R < 1 || C < 1 || H < 1 || dh < 1 || n_sel < 0) return 1;
    scale = pick_scale(scale, dh);
    const size_t d = (size_t)H * dh;
    set_threads(nthreads);
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < n_sel; ++s) {
        const int b = sel_b[s], r = sel_r[s];
        if (b < 0 || b >= B || r < 0 || r >= R) { bad = 1; continue; }
        int *cols = (int *)malloc(sizeof(int) * (size_t)C);
        size_t *pos = (size_t *)malloc(sizeof(size_t) * (size_t)C);
        int L = 0;
        for (int c = 0; c < C; ++c)
            if (!col_valid || col_valid[(size_t)b * C + c]) cols[L++] = c;
        double *q = (double *)malloc(sizeof(double) * (size_t)(L + 1) * dh * 8);
        double *k = q + (size_t)(L + 1) * dh, *v = k + (size_t)(L + 1) * dh, *g = v + (size_t)(L + 1) * dh;
        double *r0 = g + (size_t)(L + 1) * dh, *r1 = r0 + (size_t)(L + 1) * dh, *r2 = r1 + (size_t)(L + 1) * dh;
        double *lse = r2 + (size_t)(L + 1) * dh;
        const size_t cell0 = ((size_t)b * R + r) * C;
        /* zero the whole compact output row block first (invalid columns stay 0) */
        for (size_t x = 0; x < (size_t)C * d; ++x) {
            out0[(size_t)s * C * d + x] = 0.0;
            if (mode == 1) { out1[(size_t)s * C * d + x] = 0.0; out2[(size_t)s * C * d + x] = 0.0; }
        }
        if (mode == 0) for (size_t x = 0; x < (size_t)H * C; ++x) out1[(size_t)s * H * C + x] = 0.0;
        for (int h = 0; h < H && L > 0; ++h) {
            for (int t = 0; t < L; ++t) pos[t] = (cell0 + cols[t]) * d + (size_t)h * dh;
            gather_seq(Q, in_f64, pos, L, dh, q);
            gather_seq(K, in_f64, pos, L, dh, k);
            gather_seq(V, in_f64, pos, L, dh, v);
            if (mode == 0) {
                attn_fwd_dense(L, L, dh, q, k, v, scale, r0, lse);
                for (int t = 0; t < L; ++t) {
                    for (int e = 0; e < dh; ++e)
                        out0[((size_t)s * C + cols[t]) * d + (size_t)h * dh + e] = r0[(size_t)t * dh + e];
                    out1[((size_t)s * H + h) * C + cols[t]] = lse[t];
                }
            } else {
                gather_seq(dO, in_f64, pos, L, dh, g);
                attn_bwd_dense(L, L, dh, q, k, v, g, scale, r0, r1, r2);
                for (int t = 0; t < L; ++t)
                    for (int e = 0; e < dh; ++e) {
                        const size_t o = ((size_t)s * C + cols[t]) * d + (size_t)h * dh + e;
                        out0[o] = r0[(size_t)t * dh + e];
                        out1[o] = r1[(size_t)t * dh + e];
                        out2[o] = r2[(size_t)t * dh + e];
                    }
            }
        }
        free(q); free(pos); free(cols);
    }
    return bad;
}

int ref_feature_fwd(const void *Q, const void *K, const void *V, int in_f64, int B, int R, int C, int H, int dh,
                    const uint8_t *col_valid, double scale, int n_sel, const int32_t *sel_b, const int32_t *sel_r,
                    double *O, double *LSE, int nthreads) {
    return feature_run(0, Q, K, V, NULL, in_f64, B, R, C, H, dh, col_valid, scale, n_sel, sel_b, sel_r, O, LSE, NULL, nthreads);
}

int ref_feature_bwd(const void *Q, const void *K, const void *V, const void *dO, int in_f64, int B, int R, int C,
                    int H, int dh, const uint8_t *col_valid, double scale, int n_sel, const int32_t *sel_b,
                    const int32_t *sel_r, double *dQ, double *dK, double *dV, int nthreads) {
    return feature_run(1, Q, K, V, dO, in_f64, B, R, C, H, dh, col_valid, scale, n_sel, sel_b, sel_r, dQ, dK, dV, nthreads);
}

/* ================================================================================
 * Item ("sample-axis", "row-axis") attention:
 * for each selected (b, c) and each head, queries are ALL R rows, keys/values are
 * rows [0, n_train[b]) only -- train and test queries alike (reading c1).
 * Outputs compact per selection: O/dQ/dK/dV [n_sel, R, H, dh], LSE [n_sel, H, R].
 * dK, dV at rows >= n_train[b] are 0; an invalid column gives all zeros.
 * ================================================================================ */
static int item_run(int mode, const void *Q, const void *K, const void *V, const void *dO, int in_f64,
                    int B, int R, int C, int H, int dh, const int32_t *n_train, const uint8_t *col_valid,
                    double scale, int n_sel, const int32_t *sel_b, const int32_t *sel_c,
                    double *out0, double *out1, double *out2, int nthreads) {
    if (B < 1 || R < 1 || C < 1 || H < 1 || dh < 1 || n_sel < 0 || !n_train) return 1;
    for (int b = 0; b < B; ++b) if (n_train[b] < 1 || n_train[b] > R) return 2;
    scale = pick_scale(scale, dh);
    const size_t d = (size_t)H * dh;
    set_threads(nthreads);
    int bad = 0;
    const int n_work = n_sel * H;
#pragma omp parallel for schedule(dynamic, 1)
    for (int w = 0; w < n_work; ++w) {
        const int s = w / H, h = w % H;
        const int b = sel_b[s], c = sel_c[s];
        if (b < 0 || b >= B || c < 0 || c >= C) { bad = 1; continue; }
        const int n = n_train[b];
        const int valid = !col_valid || col_valid[(size_t)b * C + c];
        /* zero this (selection, head) slice of the outputs */
        for (int i = 0; i < R; ++i)
            for (int e = 0; e < dh; ++e) {
                const size_t o = ((size_t)s * R + i) * d + (size_t)h * dh + e;
                out0[o] = 0.0;
                if (mode == 1) { out1[o] = 0.0; out2[o] = 0.0; }
            }
        if (mode == 0) for (int i = 0; i < R; ++i) out1[((size_t)s * H + h) * R + i] = 0.0;
        if (!valid) continue;
        size_t *pos = (size_t *)malloc(sizeof(size_t) * (size_t)R);
        for (int i = 0; i < R; ++i) pos[i] = ((((size_t)b * R + i) * C + c) * d) + (size_t)h * dh;
        double *q = (double *)malloc(sizeof(double) * ((size_t)R * dh * 5 + (size_t)n * dh * 4 + R));
        double *g = q + (size_t)R * dh, *r0 = g + (size_t)R * dh, *k = r0 + (size_t)R * dh;
        double *v = k + (size_t)n * dh, *r1 = v + (size_t)n * dh, *r2 = r1 + (size_t)n * dh;
        double *lse = r2 + (size_t)n * dh;
        gather_seq(Q, in_f64, pos, R, dh, q);
        gather_seq(K, in_f64, pos, n, dh, k);   /* keys: train rows only */
        gather_seq(V, in_f64, pos, n, dh, v);
        if (mode == 0) {
            attn_fwd_dense(R, n, dh, q, k, v, scale, r0, lse);
            for (int i = 0; i < R; ++i) {
                for (int e = 0; e < dh; ++e) out0[((size_t)s * R + i) * d + (size_t)h * dh + e] = r0[(size_t)i * dh + e];
                out1[((size_t)s * H + h) * R + i] = lse[i];
            }
        } else {
            gather_seq(dO, in_f64, pos, R, dh, g);
            attn_bwd_dense(R, n, dh, q, k, v, g, scale, r0, r1, r2);
            for (int i = 0; i < R; ++i)
                for (int e = 0; e < dh; ++e) out0[((size_t)s * R + i) * d + (size_t)h * dh + e] = r0[(size_t)i * dh + e];
            for (int j = 0; j < n; ++j)
                for (int e = 0; e < dh; ++e) {
                    const size_t o = ((size_t)s * R + j) * d + (size_t)h * dh + e;
                    out1[o] = r1[(size_t)j * dh + e];
                    out2[o] = r2[(size_t)j * dh + e];
                }
        }
        free(q); free(pos);
    }
    return bad;
}

int ref_item_fwd(const void *Q, const void *K, const void *V, int in_f64, int B, int R, int C, int H, int dh,
                 const int32_t *n_train, const uint8_t *col_valid, double scale, int n_sel, const int32_t *sel_b,
                 const int32_t *sel_c, double *O, double *LSE, int nthreads) {
    return item_run(0, Q, K, V, NULL, in_f64, B, R, C, H, dh, n_train, col_valid, scale, n_sel, sel_b, sel_c, O, LSE, NULL, nthreads);
}

int ref_item_bwd(const void *Q, const void *K, const void *V, const void *dO, int in_f64, int B, int R, int C, int H,
                 int dh, const int32_t *n_train, const uint8_t *col_valid, double scale, int n_sel,
                 const int32_t *sel_b, const int32_t *sel_c, double *dQ, double *dK, double *dV, int nthreads) {
    return item_run(1, Q, K, V, dO, in_f64, B, R, C, H, dh, n_train, col_valid, scale, n_sel, sel_b, sel_c, dQ, dK, dV, nthreads);
}
