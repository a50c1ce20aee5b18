/*
 * fp64 CPU ORACLE for the fused graph-attention hot path of arxiv/paper_2605_31500.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  It shares no
 * code, header, table or helper with the CUDA path (paper_2605_31500_b200/csrc), and the
 * product path never routes through it.
 *
 * What it is: the plain textbook definition of the two layers, two-pass softmax per
 * (destination row i, head h), all arithmetic in double.  The paper's fused kernels compute
 * exactly this result (online softmax is an exact rewrite), so
 * the oracle is the definition written out, with no blocking, fusion or reordering.
 *
 * Layouts (same as include/gnn_attn.h): features [N, H, d] row-major, node-major
 * (PAPER.md:492 indexes O[i,h,:], logsumexp[i,h]); CSR int32, ROW = DESTINATION i, entries
 * colidx[e] = source j.  Inputs are the STORED fp32 / bf16 values up-cast
 * exactly to float by the caller; every product and sum below is done in double.
 *
 * Definitions followed (section 2.2, lines 68-76):
 *   h_i = sum_{j in N(i) u {i}} alpha_ij v_j,  alpha_ij = softmax_j(e_ij)
 *   Graph Transformer: e_ij = q_i^T k_j / sqrt(D)             (D = per-head dim)
 *   GATv2:             e_ij = a^T LeakyReLU(W_l h_i + W_r h_j), v_j = W_r h_j
 *                      = a^T sigma(xl_i + xr_j),  value = xr_j
 *   L[i,h] = logsumexp_j e_ij (natural log; reading A7).
 * The self-loop is whatever the caller stored in the CSR (reading A3); duplicate entries
 * are separate softmax terms (A4); an empty row gives O = 0, L = -inf (A5).
 *
 * Backward identities (PAPER.md:494; GATv2 PAPER.md:496, :539):
 *   alpha_ij = exp(e_ij - L_i);  Delta_i = <O_i, dO_i>;  dP_ij = <dO_i, v_j>
 *   dS_ij = alpha_ij (dP_ij - Delta_i)
 *   GT:    dQ_i += dS_ij k_j / sqrt(D);  dK_j += dS_ij q_i / sqrt(D);  dV_j += alpha_ij dO_i
 *   GATv2: G_i = <O_i, dO_i> (= sum_j alpha_ij <dO_i, xr_j>);  de_ij = alpha_ij (dP_ij - G_i)
 *          da += de_ij sigma(z_ij);  dz_ij = de_ij a . sigma'(z_ij)
 *          dxl_i += dz_ij;  dxr_j += dz_ij + alpha_ij dO_i;   sigma'(0) = slope (A8)
 * Pins: tests/test_oracle_pins.py (dense brute force, library SDPA, autograd on the dense
 * formulation, central finite differences, closed forms, invariants, golden fixtures).
 *
 * Row subsets: every function takes `rows` (NULL = all n rows in order) and `nrows`; output
 * slot t belongs to row rows[t].  This lets full-size parity tests evaluate sampled outputs.
 * Source-side gradients (dK, dV, dxr) are evaluated per SOURCE row of the oracle's own
 * transposed CSR (built in oracle/plan_ref.py by a stable argsort), which is the same sum
 * dK_j = sum_{i : j in N(i)} ... grouped by j; L and Delta/G are read from full [N,H] arrays.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* Input scalar type: float (the stored fp32 / up-cast bf16 values; default) or double (second
 * build, -DORACLE_IN_T=double, used only by the finite-difference pins which need eps ~ 1e-6). */
#ifndef ORACLE_IN_T
#define ORACLE_IN_T float
#endif
typedef ORACLE_IN_T in_t;

#define IDX3(i, h, c, H, d) ((((int64_t)(i)) * (H) + (h)) * (d) + (c))

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int t) {
#ifdef _OPENMP
    if (t > 0) omp_set_num_threads(t);
#else
    (void)t;
#endif
}

static inline double lrelu(double z, double slope) { return z > 0.0 ? z : slope * z; }
static inline double dlrelu(double z, double slope) { return z > 0.0 ? 1.0 : slope; }

/* e_ij for Graph Transformer */
static inline double gt_score(const in_t* q, const in_t* k, int64_t i, int64_t j, int h, int H, int d) {
    double s = 0.0;
    for (int c = 0; c < d; ++c) s += (double)q[IDX3(i, h, c, H, d)] * (double)k[IDX3(j, h, c, H, d)];
    return s / sqrt((double)d);
}

/* e_ij for GATv2, PAPER.md:74 / :488 */
static inline double gat_score(const in_t* xl, const in_t* xr, const in_t* a, double slope, int64_t i, int64_t j,
                               int h, int H, int d) {
    double s = 0.0;
    for (int c = 0; c < d; ++c) {
        double z = (double)xl[IDX3(i, h, c, H, d)] + (double)xr[IDX3(j, h, c, H, d)];
        s += (double)a[h * d + c] * lrelu(z, slope);
    }
    return s;
}

/* ------------------------------------------------------------------ forward (both layers)
 * kind 0: GT (p0 = q, p1 = k, p2 = v);  kind 1: GATv2 (p0 = xl, p1 = xr, p2 = xr, a, slope).
 * O [nrows, H, d], L [nrows, H].                                                          */
static void fwd_generic(int kind, int n, const int32_t* rowptr, const int32_t* colidx, const in_t* p0,
                        const in_t* p1, const in_t* p2, const in_t* a, double slope, int H, int d,
                        const int32_t* rows, int nrows, double* O, double* L) {
    (void)n;
#pragma omp parallel for schedule(dynamic, 64)
    for (int t = 0; t < nrows; ++t) {
        const int64_t i = rows ? rows[t] : t;
        const int32_t b = rowptr[i], e = rowptr[i + 1];
        for (int h = 0; h < H; ++h) {
            double* o = O + IDX3(t, h, 0, H, d);
            for (int c = 0; c < d; ++c) o[c] = 0.0;
            if (b == e) { L[(int64_t)t * H + h] = -INFINITY; continue; }
            /* pass 1: max */
            double m = -INFINITY;
            for (int32_t x = b; x < e; ++x) {
                const int64_t j = colidx[x];
                double s = kind == 0 ? gt_score(p0, p1, i, j, h, H, d) : gat_score(p0, p1, a, slope, i, j, h, H, d);
                if (s > m) m = s;
            }
            /* pass 2: denominator */
            double z = 0.0;
            for (int32_t x = b; x < e; ++x) {
                const int64_t j = colidx[x];
                double s = kind == 0 ? gt_score(p0, p1, i, j, h, H, d) : gat_score(p0, p1, a, slope, i, j, h, H, d);
                z += exp(s - m);
            }
            const double lse = m + log(z);
            L[(int64_t)t * H + h] = lse;
            /* pass 3: O = sum alpha v */
            for (int32_t x = b; x < e; ++x) {
                const int64_t j = colidx[x];
                double s = kind == 0 ? gt_score(p0, p1, i, j, h, H, d) : gat_score(p0, p1, a, slope, i, j, h, H, d);
                const double alpha = exp(s - lse);
                for (int c = 0; c < d; ++c) o[c] += alpha * (double)p2[IDX3(j, h, c, H, d)];
            }
        }
    }
}

void oracle_gt_fwd(int n, const int32_t* rowptr, const int32_t* colidx, const in_t* q, const in_t* k,
                   const in_t* v, int H, int d, const int32_t* rows, int nrows, double* O, double* L) {
    fwd_generic(0, n, rowptr, colidx, q, k, v, NULL, 0.0, H, d, rows, nrows, O, L);
}

void oracle_gatv2_fwd(int n, const int32_t* rowptr, const int32_t* colidx, const in_t* xl, const in_t* xr,
                      const in_t* a, double slope, int H, int d, const int32_t* rows, int nrows, double* O,
                      double* L) {
    fwd_generic(1, n, rowptr, colidx, xl, xr, xr, a, slope, H, d, rows, nrows, O, L);
}

/* Delta[t,h] = <O[t,h,:], dO[rows[t],h,:]>   (same formula gives GATv2's G) */
void oracle_rowdot(const double* O, const in_t* dO, int H, int d, const int32_t* rows, int nrows, double* out) {
#pragma omp parallel for schedule(static)
    for (int t = 0; t < nrows; ++t) {
        const int64_t i = rows ? rows[t] : t;
        for (int h = 0; h < H; ++h) {
            double s = 0.0;
            for (int c = 0; c < d; ++c) s += O[IDX3(t, h, c, H, d)] * (double)dO[IDX3(i, h, c, H, d)];
            out[(int64_t)t * H + h] = s;
        }
    }
}

/* ------------------------------------------------------------------ GT backward, dst side
 * dQ[t,h,:] = sum_j dS_ij k_j / sqrt(d) for i = rows[t].  L, Delta: full [n,H] arrays.      */
void oracle_gt_bwd_dst(int n, const int32_t* rowptr, const int32_t* colidx, const in_t* q, const in_t* k,
                       const in_t* v, const in_t* dO, const double* L, const double* Delta, int H, int d,
                       const int32_t* rows, int nrows, double* dQ) {
    (void)n;
    const double inv = 1.0 / sqrt((double)d);
#pragma omp parallel for schedule(dynamic, 64)
    for (int t = 0; t < nrows; ++t) {
        const int64_t i = rows ? rows[t] : t;
        for (int h = 0; h < H; ++h) {
            double* g = dQ + IDX3(t, h, 0, H, d);
            for (int c = 0; c < d; ++c) g[c] = 0.0;
            for (int32_t x = rowptr[i]; x < rowptr[i + 1]; ++x) {
                const int64_t j = colidx[x];
                const double alpha = exp(gt_score(q, k, i, j, h, H, d) - L[i * H + h]);
                double dP = 0.0;
                for (int c = 0; c < d; ++c) dP += (double)dO[IDX3(i, h, c, H, d)] * (double)v[IDX3(j, h, c, H, d)];
                const double dS = alpha * (dP - Delta[i * H + h]);
                for (int c = 0; c < d; ++c) g[c] += dS * (double)k[IDX3(j, h, c, H, d)] * inv;
            }
        }
    }
}

/* ------------------------------------------------------------------ GT backward, src side
 * For source j = srcs[t]: the destinations it feeds are colidx_t[rowptr_t[j] .. rowptr_t[j+1])
 * (the oracle's own transposed CSR).  dK[t,h,:] = sum_i dS_ij q_i / sqrt(d); dV = sum_i alpha_ij dO_i. */
void oracle_gt_bwd_src(int n, const int32_t* rowptr_t, const int32_t* colidx_t, const in_t* q, const in_t* k,
                       const in_t* v, const in_t* dO, const double* L, const double* Delta, int H, int d,
                       const int32_t* srcs, int nsrcs, double* dK, double* dV) {
    (void)n;
    const double inv = 1.0 / sqrt((double)d);
#pragma omp parallel for schedule(dynamic, 64)
    for (int t = 0; t < nsrcs; ++t) {
        const int64_t j = srcs ? srcs[t] : t;
        for (int h = 0; h < H; ++h) {
            double* gk = dK + IDX3(t, h, 0, H, d);
            double* gv = dV + IDX3(t, h, 0, H, d);
            for (int c = 0; c < d; ++c) { gk[c] = 0.0; gv[c] = 0.0; }
            for (int32_t x = rowptr_t[j]; x < rowptr_t[j + 1]; ++x) {
                const int64_t i = colidx_t[x];
                const double alpha = exp(gt_score(q, k, i, j, h, H, d) - L[i * H + h]);
                double dP = 0.0;
                for (int c = 0; c < d; ++c) dP += (double)dO[IDX3(i, h, c, H, d)] * (double)v[IDX3(j, h, c, H, d)];
                const double dS = alpha * (dP - Delta[i * H + h]);
                for (int c = 0; c < d; ++c) {
                    gk[c] += dS * (double)q[IDX3(i, h, c, H, d)] * inv;
                    gv[c] += alpha * (double)dO[IDX3(i, h, c, H, d)];
                }
            }
        }
    }
}

/* ------------------------------------------------------------------ GATv2 backward, dst side
 * dxl[t,h,:] = sum_j de_ij a . sigma'(z_ij);  da_rows[t,h,:] = sum_j de_ij sigma(z_ij)
 * (this row's contribution to da; da = sum over all rows, done by the caller in fp64).     */
void oracle_gatv2_bwd_dst(int n, const int32_t* rowptr, const int32_t* colidx, const in_t* xl, const in_t* xr,
                          const in_t* a, double slope, const in_t* dO, const double* L, const double* G, int H,
                          int d, const int32_t* rows, int nrows, double* dxl, double* da_rows) {
    (void)n;
#pragma omp parallel for schedule(dynamic, 64)
    for (int t = 0; t < nrows; ++t) {
        const int64_t i = rows ? rows[t] : t;
        for (int h = 0; h < H; ++h) {
            double* gl = dxl + IDX3(t, h, 0, H, d);
            double* ga = da_rows + IDX3(t, h, 0, H, d);
            for (int c = 0; c < d; ++c) { gl[c] = 0.0; ga[c] = 0.0; }
            for (int32_t x = rowptr[i]; x < rowptr[i + 1]; ++x) {
                const int64_t j = colidx[x];
                const double alpha = exp(gat_score(xl, xr, a, slope, i, j, h, H, d) - L[i * H + h]);
                double dP = 0.0;
                for (int c = 0; c < d; ++c) dP += (double)dO[IDX3(i, h, c, H, d)] * (double)xr[IDX3(j, h, c, H, d)];
                const double de = alpha * (dP - G[i * H + h]);
                for (int c = 0; c < d; ++c) {
                    const double z = (double)xl[IDX3(i, h, c, H, d)] + (double)xr[IDX3(j, h, c, H, d)];
                    ga[c] += de * lrelu(z, slope);
                    gl[c] += de * (double)a[h * d + c] * dlrelu(z, slope);
                }
            }
        }
    }
}

/* ------------------------------------------------------------------ GATv2 backward, src side
 * dxr[t,h,:] = sum_i ( de_ij a . sigma'(z_ij) + alpha_ij dO_i ) for source j = srcs[t].     */
void oracle_gatv2_bwd_src(int n, const int32_t* rowptr_t, const int32_t* colidx_t, const in_t* xl,
                          const in_t* xr, const in_t* a, double slope, const in_t* dO, const double* L,
                          const double* G, int H, int d, const int32_t* srcs, int nsrcs, double* dxr) {
    (void)n;
#pragma omp parallel for schedule(dynamic, 64)
    for (int t = 0; t < nsrcs; ++t) {
        const int64_t j = srcs ? srcs[t] : t;
        for (int h = 0; h < H; ++h) {
            double* g = dxr + IDX3(t, h, 0, H, d);
            for (int c = 0; c < d; ++c) g[c] = 0.0;
            for (int32_t x = rowptr_t[j]; x < rowptr_t[j + 1]; ++x) {
                const int64_t i = colidx_t[x];
                const double alpha = exp(gat_score(xl, xr, a, slope, i, j, h, H, d) - L[i * H + h]);
                double dP = 0.0;
                for (int c = 0; c < d; ++c) dP += (double)dO[IDX3(i, h, c, H, d)] * (double)xr[IDX3(j, h, c, H, d)];
                const double de = alpha * (dP - G[i * H + h]);
                for (int c = 0; c < d; ++c) {
                    const double z = (double)xl[IDX3(i, h, c, H, d)] + (double)xr[IDX3(j, h, c, H, d)];
                    g[c] += de * (double)a[h * d + c] * dlrelu(z, slope) + alpha * (double)dO[IDX3(i, h, c, H, d)];
                }
            }
        }
    }
}
