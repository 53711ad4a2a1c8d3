/*
 * cc_oracle.c -- plain fp64 CPU oracle for the proximal distance (MM) algorithm for convex
 * clustering, written from PAPER.md (arXiv 1409.2065, Chen, Chi, Ranola, Lange), section 3.
 *
 * THIS IS TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.  It shares no code, header, table or helper
 * with the CUDA path (paper_1409_2065_b200/csrc) and neither side includes the other.
 *
 * It follows the algorithm step by step, in the paper's order and notation, with the matrix V
 * stored explicitly (one p-vector per pair i<j with w_ij>0) exactly as the paper has it:
 *
 *   projection onto C by sequential block descent ...... PAPER.md L90-L103
 *   d_m .................................................. PAPER.md L76 (eq. 5)
 *   approximate objective Phi_m ......................... PAPER.md L64-L66 with the loss of eq. 6 (L109)
 *   U update ............................................. PAPER.md L82, missing data y_ij L116
 *   V update (block soft-threshold) ...................... PAPER.md L86-L88
 *   k nearest neighbours for the weights of eq. 8 ........ PAPER.md L127-L129
 *
 * Where the paper is silent (rho, eps, start, stop rule, garbled L94-L101) the readings S1-S22 of
 * DESIGN.md apply; each is marked [reading Sx] below.
 *
 * Pins: tests/test_oracle_pins.py (P1-P13 of DESIGN.md).  No function here is "parity unpinned"
 * except orc_knn's masked-distance rule (reading S11, a definition, not a result of the paper).
 *
 * Parallelism: OpenMP over independent rows / pairs / column slabs only; every floating-point sum
 * is formed in a fixed order (per-item partial results are stored and then added sequentially), so
 * results do not depend on the thread count.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_threads(int t) {
#ifdef _OPENMP
    if (t > 0) omp_set_num_threads(t);
#else
    (void)t;
#endif
}

/* ------------------------------------------------------------------------------------------
 * Distances for the weights (d_ij = ||x_i - x_j||).  With missing entries the paper
 * uses multiple imputation (L160, third-party); [reading S11]: squared distance over co-observed
 * coordinates, scaled by p / #co-observed; no co-observed coordinate => +inf.
 * ------------------------------------------------------------------------------------------ */
static double pair_dist2(int64_t p, const double *xi, const double *xj, const uint8_t *mi,
                         const uint8_t *mj) {
    double s = 0.0;
    if (!mi) {
        for (int64_t c = 0; c < p; ++c) {
            double t = xi[c] - xj[c];
            s += t * t;
        }
        return s;
    }
    int64_t co = 0;
    for (int64_t c = 0; c < p; ++c) {
        if (mi[c] && mj[c]) {
            double t = xi[c] - xj[c];
            s += t * t;
            ++co;
        }
    }
    if (co == 0) return INFINITY;
    return s * (double)p / (double)co;
}

/* squared distances from row i to every row (out[i] = +inf so that i is never its own neighbour) */
void orc_row_dist2(int64_t n, int64_t p, const double *X, const uint8_t *mask, int64_t i, double *out) {
    for (int64_t j = 0; j < n; ++j) {
        if (j == i) { out[j] = INFINITY; continue; }
        out[j] = pair_dist2(p, X + i * p, X + j * p, mask ? mask + i * p : NULL, mask ? mask + j * p : NULL);
    }
}

/* k nearest neighbours of the listed rows by brute force.  [reading S9]: self excluded, ties broken
 * by the smaller index.  nbr/d2 are nrows*k, sorted by increasing distance. */
int orc_knn(int64_t n, int64_t p, const double *X, const uint8_t *mask, int k, int64_t nrows,
            const int64_t *rows, int32_t *nbr, double *d2) {
    if (k < 1 || k > n - 1) return -1;
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t r = 0; r < nrows; ++r) {
        int64_t i = rows ? rows[r] : r;
        int32_t *nb = nbr + r * k;
        double *dd = d2 + r * k;
        int cnt = 0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double d = pair_dist2(p, X + i * p, X + j * p, mask ? mask + i * p : NULL,
                                  mask ? mask + j * p : NULL);
            /* insertion into the sorted list; strict '<' keeps the earlier (smaller) index on ties */
            if (cnt < k || d < dd[cnt - 1]) {
                int pos = cnt < k ? cnt : k - 1;
                while (pos > 0 && d < dd[pos - 1]) {
                    dd[pos] = dd[pos - 1];
                    nb[pos] = nb[pos - 1];
                    --pos;
                }
                dd[pos] = d;
                nb[pos] = (int32_t)j;
                if (cnt < k) ++cnt;
            }
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Neighbourhoods N_i = L_i u R_i of PAPER.md L90, from the pair list (ei[e] < ej[e]).
 * ------------------------------------------------------------------------------------------ */
typedef struct {
    int64_t *ptr;  /* n+1 */
    int32_t *nbr;  /* 2m */
} nbr_t;

static int build_nbr(int64_t n, int64_t m, const int32_t *ei, const int32_t *ej, nbr_t *g) {
    g->ptr = (int64_t *)calloc((size_t)n + 1, sizeof(int64_t));
    g->nbr = (int32_t *)malloc((size_t)(2 * m + 1) * sizeof(int32_t));
    if (!g->ptr || !g->nbr) return -1;
    for (int64_t e = 0; e < m; ++e) {
        g->ptr[ei[e] + 1]++;
        g->ptr[ej[e] + 1]++;
    }
    for (int64_t i = 0; i < n; ++i) g->ptr[i + 1] += g->ptr[i];
    int64_t *fill = (int64_t *)malloc((size_t)n * sizeof(int64_t));
    if (!fill) return -1;
    memcpy(fill, g->ptr, (size_t)n * sizeof(int64_t));
    for (int64_t e = 0; e < m; ++e) {
        g->nbr[fill[ei[e]]++] = ej[e];
        g->nbr[fill[ej[e]]++] = ei[e];
    }
    free(fill);
    return 0;
}

static void free_nbr(nbr_t *g) {
    free(g->ptr);
    free(g->nbr);
}

/* right-hand side of the block update, PAPER.md L100 [reading S13 of the garbled line]:
 *   r_i = u~_i + sum_{j in R_i} v~_ij - sum_{j in L_i} v~_ji                                   */
static void build_rhs(int64_t n, int64_t p, int64_t m, const int32_t *ei, const int32_t *ej,
                      const double *U, const double *V, double *R) {
    memcpy(R, U, (size_t)(n * p) * sizeof(double));
    for (int64_t e = 0; e < m; ++e) {
        double *ri = R + (int64_t)ei[e] * p, *rj = R + (int64_t)ej[e] * p;
        const double *v = V + e * p;
        for (int64_t c = 0; c < p; ++c) {
            ri[c] += v[c];
            rj[c] -= v[c];
        }
    }
}

/* Projection by the paper's block descent: one cycle updates u_1..u_n
 * sequentially, u_i = (r_i + sum_{j in N_i} u_j) / (1 + |N_i|); cycles repeat "until all of the
 * vectors u_i stabilize" -- [reading S5]: start from A = U~, stop when the largest change of any
 * entry in a cycle is <= tol * (1 + max|a|).  The p coordinates are independent systems with the
 * same matrix, so column slabs run in parallel without changing any arithmetic.
 * Returns the number of cycles, or -1 if maxcycles was hit. */
static int64_t project_block_descent(int64_t n, int64_t p, const nbr_t *g, const double *R, double *A,
                                     double tol, int64_t maxcycles) {
    int nth = orc_num_threads();
    if (nth > p) nth = (int)p;
    if (n * p <= 32768) nth = 1; /* thread start-up would dominate; arithmetic is identical */
    if (nth < 1) nth = 1;
    double *tdelta = (double *)malloc(sizeof(double) * (size_t)nth * 2);
    int64_t cycles = 0;
    int done = 0;
    while (!done && cycles < maxcycles) {
#pragma omp parallel num_threads(nth)
        {
#ifdef _OPENMP
            int t = omp_get_thread_num();
#else
            int t = 0;
#endif
            int64_t c0 = p * t / nth, c1 = p * (t + 1) / nth;
            double md = 0.0, ma = 0.0;
            for (int64_t i = 0; i < n; ++i) {
                double *ai = A + i * p;
                const double *ri = R + i * p;
                int64_t b = g->ptr[i], e = g->ptr[i + 1];
                double inv = 1.0 / (1.0 + (double)(e - b));
                for (int64_t c = c0; c < c1; ++c) {
                    double s = ri[c];
                    for (int64_t q = b; q < e; ++q) s += A[(int64_t)g->nbr[q] * p + c];
                    double nv = s * inv;
                    double dl = fabs(nv - ai[c]);
                    if (dl > md) md = dl;
                    if (fabs(nv) > ma) ma = fabs(nv);
                    ai[c] = nv;
                }
            }
            tdelta[2 * t] = md;
            tdelta[2 * t + 1] = ma;
        }
        double md = 0.0, ma = 0.0;
        for (int t = 0; t < nth; ++t) {
            if (tdelta[2 * t] > md) md = tdelta[2 * t];
            if (tdelta[2 * t + 1] > ma) ma = tdelta[2 * t + 1];
        }
        ++cycles;
        if (md <= tol * (1.0 + ma)) done = 1;
    }
    free(tdelta);
    return done ? cycles : -1;
}

/* (I+L) applied to all p columns:  out_i = (1+|N_i|) z_i - sum_{j in N_i} z_j  (Appendix of DESIGN.md:
 * collecting terms in the stationarity equation PAPER.md). */
static void apply_IL(int64_t n, int64_t p, const nbr_t *g, const double *Z, double *out) {
#pragma omp parallel for schedule(static) if (n * p > 32768)
    for (int64_t i = 0; i < n; ++i) {
        int64_t b = g->ptr[i], e = g->ptr[i + 1];
        double dg = 1.0 + (double)(e - b);
        const double *zi = Z + i * p;
        double *oi = out + i * p;
        for (int64_t c = 0; c < p; ++c) oi[c] = dg * zi[c];
        for (int64_t q = b; q < e; ++q) {
            const double *zj = Z + (int64_t)g->nbr[q] * p;
            for (int64_t c = 0; c < p; ++c) oi[c] -= zj[c];
        }
    }
}

static double dot_seq(int64_t len, const double *a, const double *b) {
    double s = 0.0;
    for (int64_t k = 0; k < len; ++k) s += a[k] * b[k];
    return s;
}

/* Second back-end for the same projection: conjugate gradients on (I+L)A = R (SPD, spectrum in
 * [1, 1+2 maxdeg]) -- the unique solution the block descent converges to [reading S5].  Used where
 * the sequential sweep is too slow (large sparse); accepted because tests pin it to the block
 * descent and to a dense solve (P4).  Stops at ||residual||_F <= tol * ||R||_F. */
static int64_t project_cg(int64_t n, int64_t p, const nbr_t *g, const double *R, double *A, double tol,
                          int64_t maxit) {
    int64_t len = n * p;
    double *r = (double *)malloc(sizeof(double) * (size_t)len);
    double *d = (double *)malloc(sizeof(double) * (size_t)len);
    double *q = (double *)malloc(sizeof(double) * (size_t)len);
    if (!r || !d || !q) return -1;
    apply_IL(n, p, g, A, q);
    for (int64_t k = 0; k < len; ++k) r[k] = R[k] - q[k];
    memcpy(d, r, sizeof(double) * (size_t)len);
    double rr = dot_seq(len, r, r);
    double stop = tol * tol * dot_seq(len, R, R);
    int64_t it = 0;
    while (rr > stop && it < maxit) {
        apply_IL(n, p, g, d, q);
        double alpha = rr / dot_seq(len, d, q);
        for (int64_t k = 0; k < len; ++k) {
            A[k] += alpha * d[k];
            r[k] -= alpha * q[k];
        }
        double rr2 = dot_seq(len, r, r);
        double beta = rr2 / rr;
        for (int64_t k = 0; k < len; ++k) d[k] = r[k] + beta * d[k];
        rr = rr2;
        ++it;
    }
    free(r);
    free(d);
    free(q);
    return rr <= stop ? it : -1;
}

/* Exposed for the pins: project (U~, V~) onto C = {v_ij = u_i - u_j}; returns A (B = DA is implied,
 * PAPER.md L103 "one sets v_ij = u_i - u_j"). method 0 = block descent, 1 = CG. */
int64_t orc_project(int64_t n, int64_t p, int64_t m, const int32_t *ei, const int32_t *ej, const double *U,
                    const double *V, int method, double tol, int64_t maxcycles, double *A) {
    nbr_t g;
    if (build_nbr(n, m, ei, ej, &g)) return -2;
    double *R = (double *)malloc(sizeof(double) * (size_t)(n * p));
    if (!R) return -2;
    build_rhs(n, p, m, ei, ej, U, V, R);
    memcpy(A, U, sizeof(double) * (size_t)(n * p));
    int64_t cyc = method == 0 ? project_block_descent(n, p, &g, R, A, tol, maxcycles)
                              : project_cg(n, p, &g, R, A, tol, maxcycles);
    free(R);
    free_nbr(&g);
    return cyc;
}

/* ------------------------------------------------------------------------------------------
 * The MM iteration.  State (U, V) in / out.  Iteration m = 0,1,...:
 *   1. (A,B) = P_C(U_m, V_m)                                         L90-L103
 *   2. d_m = sqrt(||U_m - A||^2 + sum_E ||v_m,ij - b_ij||^2 + eps)   L76
 *   3. Phi_m = 1/2 sum_Gamma (x-u_m)^2 + gamma sum_E w ||v_m|| + rho d_m   L64-L66, L109
 *   4. y = x where observed else u_m (L116);  u_{m+1} = (d_m y + rho a)/(d_m + rho)   L82
 *   5. v_{m+1} = max(1 - gamma w d_m / (rho ||b||), 0) b;  ||b|| <= thr (incl. b = 0) => 0   L86-L88, [S6]
 *   6. [reading S3] stop after update m if m+1 >= min_it, m >= 1 and
 *      Phi_{m-1} - Phi_m <= tol (1 + |Phi_{m-1}|); tol = 0 runs exactly maxit iterations.
 * phi_hist[m], d_hist[m] are recorded for every iteration performed.
 * Returns 0, or a negative code (-1 projection did not converge, -2 out of memory,
 * -3 Phi increased beyond rounding: the MM descent property PAPER.md L64-L68 failed).
 * ------------------------------------------------------------------------------------------ */
int orc_mm(int64_t n, int64_t p, const double *X, const uint8_t *mask, int64_t m, const int32_t *ei,
           const int32_t *ej, const double *w, double gamma, double rho, double eps, int maxit, double tol,
           int min_it, int proj_method, double proj_tol, int64_t proj_maxcycles, double *U, double *V,
           double *phi_hist, double *d_hist, int *iters_done, int64_t *proj_cycles) {
    nbr_t g;
    if (build_nbr(n, m, ei, ej, &g)) return -2;
    int64_t len = n * p;
    double *R = (double *)malloc(sizeof(double) * (size_t)len);
    double *A = (double *)malloc(sizeof(double) * (size_t)len);
    double *part = (double *)malloc(sizeof(double) * (size_t)((m > n ? m : n) + 1));
    if (!R || !A || !part) return -2;
    int rc = 0;
    int it = 0;
    *proj_cycles = 0;
    for (it = 0; it < maxit; ++it) {
        /* 1. projection */
        build_rhs(n, p, m, ei, ej, U, V, R);
        memcpy(A, U, sizeof(double) * (size_t)len); /* [S5] start from U_m */
        int64_t cyc = proj_method == 0 ? project_block_descent(n, p, &g, R, A, proj_tol, proj_maxcycles)
                                       : project_cg(n, p, &g, R, A, proj_tol, proj_maxcycles);
        if (cyc < 0) { rc = -1; break; }
        *proj_cycles += cyc;

        /* 2. distance to C */
        double dist2 = 0.0;
#pragma omp parallel for schedule(static) if (n * p > 32768)
        for (int64_t i = 0; i < n; ++i) {
            double s = 0.0;
            for (int64_t c = 0; c < p; ++c) {
                double t = U[i * p + c] - A[i * p + c];
                s += t * t;
            }
            part[i] = s;
        }
        for (int64_t i = 0; i < n; ++i) dist2 += part[i];
#pragma omp parallel for schedule(static) if (n * p > 32768)
        for (int64_t e = 0; e < m; ++e) {
            const double *ai = A + (int64_t)ei[e] * p, *aj = A + (int64_t)ej[e] * p, *v = V + e * p;
            double s = 0.0;
            for (int64_t c = 0; c < p; ++c) {
                double t = v[c] - (ai[c] - aj[c]);
                s += t * t;
            }
            part[e] = s;
        }
        for (int64_t e = 0; e < m; ++e) dist2 += part[e];
        double d = sqrt(dist2 + eps);

        /* 3. approximate objective */
        double loss = 0.0, pen = 0.0;
#pragma omp parallel for schedule(static) if (n * p > 32768)
        for (int64_t i = 0; i < n; ++i) {
            double s = 0.0;
            for (int64_t c = 0; c < p; ++c) {
                if (!mask || mask[i * p + c]) {
                    double t = X[i * p + c] - U[i * p + c];
                    s += t * t;
                }
            }
            part[i] = s;
        }
        for (int64_t i = 0; i < n; ++i) loss += part[i];
#pragma omp parallel for schedule(static) if (n * p > 32768)
        for (int64_t e = 0; e < m; ++e) {
            const double *v = V + e * p;
            double s = 0.0;
            for (int64_t c = 0; c < p; ++c) s += v[c] * v[c];
            part[e] = w[e] * sqrt(s);
        }
        for (int64_t e = 0; e < m; ++e) pen += part[e];
        double phi = 0.5 * loss + gamma * pen + rho * d;
        phi_hist[it] = phi;
        d_hist[it] = d;
        if (it > 0 && phi > phi_hist[it - 1] * (1.0 + 1e-12) + 1e-300) { rc = -3; ++it; break; }

        /* 4. U update */
        double cu = d / (d + rho), ca = rho / (d + rho);
#pragma omp parallel for schedule(static) if (n * p > 32768)
        for (int64_t i = 0; i < n; ++i) {
            for (int64_t c = 0; c < p; ++c) {
                int64_t k = i * p + c;
                double y = (!mask || mask[k]) ? X[k] : U[k];
                U[k] = cu * y + ca * A[k];
            }
        }
        /* 5. V update */
#pragma omp parallel for schedule(static) if (n * p > 32768)
        for (int64_t e = 0; e < m; ++e) {
            const double *ai = A + (int64_t)ei[e] * p, *aj = A + (int64_t)ej[e] * p;
            double *v = V + e * p;
            double s = 0.0;
            for (int64_t c = 0; c < p; ++c) {
                double b = ai[c] - aj[c];
                s += b * b;
            }
            double nb = sqrt(s);
            double thr = gamma * w[e] * d / rho;
            if (nb <= thr) {
                for (int64_t c = 0; c < p; ++c) v[c] = 0.0;
            } else {
                double f = 1.0 - thr / nb;
                for (int64_t c = 0; c < p; ++c) v[c] = f * (ai[c] - aj[c]);
            }
        }
        /* 6. stop rule */
        if (tol > 0.0 && it + 1 >= min_it && it >= 1 &&
            phi_hist[it - 1] - phi <= tol * (1.0 + fabs(phi_hist[it - 1]))) {
            ++it;
            break;
        }
    }
    *iters_done = it;
    free(R);
    free(A);
    free(part);
    free_nbr(&g);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * Cluster read-out [reading S16; the paper never defines it, L154, L206]: connected components of
 * the graph whose edges are the pairs with v_ij = 0 exactly, numbered in increasing order of each
 * component's smallest member.  Returns the number of clusters.
 * ------------------------------------------------------------------------------------------ */
static int64_t uf_find(int64_t *par, int64_t x) {
    while (par[x] != x) {
        par[x] = par[par[x]];
        x = par[x];
    }
    return x;
}

int64_t orc_labels(int64_t n, int64_t p, int64_t m, const int32_t *ei, const int32_t *ej, const double *V,
                   int32_t *labels) {
    int64_t *par = (int64_t *)malloc(sizeof(int64_t) * (size_t)n);
    if (!par) return -2;
    for (int64_t i = 0; i < n; ++i) par[i] = i;
    for (int64_t e = 0; e < m; ++e) {
        const double *v = V + e * p;
        int zero = 1;
        for (int64_t c = 0; c < p; ++c)
            if (v[c] != 0.0) { zero = 0; break; }
        if (zero) {
            int64_t a = uf_find(par, ei[e]), b = uf_find(par, ej[e]);
            if (a != b) {
                if (a < b) par[b] = a; else par[a] = b; /* root = smallest member */
            }
        }
    }
    int64_t k = 0;
    for (int64_t i = 0; i < n; ++i) {
        int64_t r = uf_find(par, i);
        if (r == i) labels[i] = (int32_t)k++; /* roots are smallest members, met in increasing order */
        else labels[i] = labels[r];
    }
    free(par);
    return k;
}
