/*
 * cc_b200.h -- C ABI of libcc_b200.so: the data-parallel hot path of the proximal distance (MM)
 * algorithm for convex clustering (Chen, Chi, Ranola, Lange, arXiv 1409.2065; cited below as
 * PAPER.md:L<line>), hand-written CUDA for NVIDIA B200 (sm_100a).
 *
 * Problem (eq. 1; missing data L107-L110 eq. 6):
 *     minimise_U  1/2 sum_{(i,c) observed} (x_ic - u_ic)^2  +  gamma sum_{(i,j) in E} w_ij ||u_i - u_j||_2
 * The paper writes the penalty constant as mu; this library (like BASELINE.json) calls it gamma.
 *
 * Conventions
 *   - X, U are n x p row-major fp32 (one contiguous row per case -- the same memory as the paper's
 *     column-per-case p x n matrix, L38).  mask is n x p uint8, 1 = observed (the set Gamma, L107).
 *   - The graph is a SYMMETRIC CSR over the n cases: both (i,j) and (j,i) are stored, no self
 *     loops, w_ij = w_ji > 0 (L90, L125; zero-weight pairs are simply absent, L40).  rowptr is
 *     int64[n+1], col is int32[nnz] sorted increasingly inside a row, w is fp32[nnz].
 *   - Every array argument says HOST or DEVICE.  DEVICE pointers must belong to the current CUDA
 *     device.  The caller owns every pointer it passes; cc_create copies what it needs into
 *     library-owned device buffers, so inputs may be freed after it returns.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  All device work
 *     of a handle is enqueued on the stream given to cc_create.  Calls that return scalars to the
 *     host synchronise that stream; cc_get_U / cc_clusters with DEVICE outputs do not.
 *   - Return value: CC_OK (0) or a negative CC_E* code; cc_last_error() gives a message.  The library
 *     never aborts, throws or prints.  There is no CPU fallback: without a CUDA device every compute
 *     entry point fails with CC_ECUDA.
 *   - Determinism: no floating-point atomics anywhere; all reductions run in a fixed order, so the
 *     same inputs give bit-identical outputs on the same GPU model.
 */
#ifndef CC_B200_H
#define CC_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CC_OK 0
#define CC_EINVAL (-1) /* bad size / NULL pointer / negative gamma / NaN or Inf in observed X or in w  */
#define CC_EGRAPH (-2) /* CSR not symmetric, w_ij != w_ji, self loop, w <= 0, col out of range/unsorted */
#define CC_EMASK (-3)  /* a column has no observed entry at all (its fused value is undetermined)       */
#define CC_ENOMEM (-4) /* host or device allocation failed                                              */
#define CC_ECUDA (-5)  /* CUDA runtime error (message in cc_last_error)                                 */
#define CC_ESTATE (-6) /* bad gamma_index, or the call needs state that does not exist yet              */
#define CC_ENOCONV (-7)/* the inner projection solve hit proj_maxit (state is still consistent)         */

typedef struct cc_handle cc_handle; /* opaque; owns all device buffers */

/* Constants the paper leaves open ("rho large enough", L57 "epsilon > 0 small"; no
 * stopping rule anywhere in L57-L103).  DESIGN.md readings S1-S5 define them; oracle and GPU take
 * the same numbers. */
typedef struct {
    double rho_scale; /* S1: rho = rho_scale * sqrt(sum_obs (x - colmean)^2 + gamma^2 sum_E w^2); used when rho_abs <= 0 */
    double rho_abs;   /*     > 0: use this rho for every gamma                                           */
    double kappa;     /* S2: eps = (kappa * rho)^2; used when eps_abs <= 0                               */
    double eps_abs;   /*     > 0: use this eps for every gamma                                           */
    double proj_tol;  /* S5: the projection's linear solve (I+L) A = R stops when its
                             residual r has sqrt(r' D^-1 r) <= proj_tol * (d_prev / rho) * sqrt(sum_obs (x-colmean)^2),
                             D = diag(1 + |N_i|).  Default 1e-5.      */
    int32_t proj_maxit; /*   cap on inner iterations per MM iteration (default 500); hitting it => CC_ENOCONV */
    int32_t min_it;   /* S3: never stop before this many MM iterations (default 10)                      */
    int32_t dense;    /* 0: graph given as CSR.  1: complete graph; `w` is an n x n row-major symmetric
                             fp32 matrix (diagonal ignored, off-diagonal >= 0), rowptr/col ignored.  The
                             constraint set stays the complete graph: a zero entry is a pair of E that
                             carries no penalty (its threshold is 0), not an absent pair                 */
    int32_t use_graph;/* 1 (default): one CUDA-graph launch per solve with device-side WHILE loops;
                         0: plain stream launches with a host loop (debugging)                           */
    int32_t hist_cap; /* capacity of the per-solve Phi_m / d_m history kept on the device (default 4096;
                         iterations beyond it are not recorded)                                          */
    int32_t max_snapshots; /* how many per-gamma snapshots of U cc_path may keep (default 64)            */
    int32_t reserved; /* must be 0 */
} cc_params;

/* Fill *prm with the defaults above.  HOST pointer. */
int cc_default_params(cc_params* prm);

/* ---- a0: one-time k-NN + Gaussian weights, PAPER.md L127-L133 (eq. 8) -------------------------------
 * w_ij = 1{i ~_k j} exp(-phi ||x_i - x_j||^2), i ~_k j iff j is among the k nearest of i OR vice versa
 * (L127); self excluded, ties to the smaller index (S9).  With a mask, the squared distance is taken
 * over co-observed coordinates and scaled by p / #co-observed (S11); rows without a common observed
 * coordinate are at infinite distance and are never neighbours.  Which points are the k nearest is
 * decided on fp64 distances of the fp32 inputs (an fp32 pass only shortlists), so the graph is the one
 * the definition gives, ties included.  A pair whose weight underflows to 0 in fp32 is absent from the
 * result (L40: a zero weight is no pair), in both directions, so the result always passes cc_create.
 * normalize != 0 divides the weights by their sum over pairs i<j (L133, S8).
 * X (DEVICE, n*p fp32), mask (DEVICE n*p uint8 or NULL).  Outputs: *rowptr (int64[n+1]), *col
 * (int32[nnz]), *w (fp32[nnz]) are DEVICE arrays allocated by the library (cudaMalloc) and owned by
 * the caller, to be released with cc_free_graph; *nnz (HOST) receives the directed entry count.
 * Needs 1 <= k <= n-1.  Synchronises `stream`. */
int cc_knn_weights(int64_t n, int64_t p, const float* X, const uint8_t* mask, int32_t k, float phi,
                   int32_t normalize, int64_t** rowptr, int32_t** col, float** w, int64_t* nnz,
                   void* stream);

/* ---- f4: the same build on the composite distance of eq. 9, PAPER.md L135-L137 -------------------------
 *   d_ij = alpha ||x_i - x_j|| + (1 - alpha) ||y_i - y_j||,  0 <= alpha <= 1,
 * y_i the caller's side coordinates (e.g. GPS): Y (DEVICE, n*q fp32 row-major, 1 <= q <= 4).  "The components
 * of the difference y_i - y_j must be computed in modulo arithmetic" (L137): period (HOST, q floats, or NULL)
 * gives each coordinate's period (360 for a longitude in degrees), 0 = plain difference; a periodic difference
 * is wrapped to [-period/2, period/2] (S27).  ||x_i - x_j|| is the square root of the (masked, S11) squared
 * distance of cc_knn_weights.  Neighbours are the k smallest d_ij, w_ij = exp(-phi d_ij^2); everything else
 * (OR rule, ties, normalisation, outputs, ownership, errors) as cc_knn_weights. */
int cc_knn_weights_composite(int64_t n, int64_t p, const float* X, const uint8_t* mask, int32_t q, const float* Y,
                             const float* period, float alpha, int32_t k, float phi, int32_t normalize,
                             int64_t** rowptr, int32_t** col, float** w, int64_t* nnz, void* stream);

/* ---- f4: eq. 9 with the geodesic alternative, PAPER.md L137 ("an even better alternative replaces ||y_i - y_j||
 * by the geodesic distance between i and j"; reading S28 in DESIGN.md) ------------------------------------
 *   d_ij = alpha ||x_i - x_j|| + (1 - alpha) radius * theta_ij,
 * theta_ij the great-circle angle between the two positions (haversine formula).  lonlat: DEVICE, n*2 fp32
 * row-major, (longitude, latitude) in degrees (any longitude branch: the formula wraps by itself).  radius
 * (> 0, finite) sets the unit of the geodesic term: 6371 for km, 57.29578 for degrees of arc.  Everything else
 * as cc_knn_weights_composite.  CC_EINVAL: lonlat NULL, radius <= 0 or not finite, alpha outside [0, 1]. */
int cc_knn_weights_geodesic(int64_t n, int64_t p, const float* X, const uint8_t* mask, const float* lonlat, float radius,
                            float alpha, int32_t k, float phi, int32_t normalize,
                            int64_t** rowptr, int32_t** col, float** w, int64_t* nnz, void* stream);

/* a0 for complete graphs (k = n-1): W_out (DEVICE, caller-owned, n*n fp32 row-major) receives
 * w_ij = exp(-phi ||x_i - x_j||^2) for i != j and 0 on the diagonal, symmetric bit for bit; same distance
 * rules and normalisation as cc_knn_weights.  The result feeds cc_create with prm.dense = 1.  X, mask:
 * DEVICE.  Synchronises `stream`. */
int cc_dense_weights(int64_t n, int64_t p, const float* X, const uint8_t* mask, float phi, int32_t normalize,
                     float* W_out, void* stream);

/* The same weights for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): this entry point calls no cudaMalloc / cudaFree or any allocating routine.  The column slices'
 * partial sums, which cc_dense_weights keeps in a temporary buffer, live in a static device array of 2 Mi floats (8 MB) that
 * every GPU loading the library holds until the process exits.  A problem whose slices need more (n * n * slices floats,
 * twice that with a mask; e.g. 52 x 200,000 fits with or without a mask, 64 x 200,000 with a mask does not) is rejected with CC_EINVAL and a message;
 * problems with enough pair tiles to fill the GPU (n >= ~1100) use no scratch and are never rejected.  No normalisation
 * (S8): scale the result yourself.  Results are bit-identical to cc_dense_weights with normalize = 0.
 * ALL calls share the one array: calls that overlap on the GPU (other streams, threads) race -- serialise them.
 * X, mask, W_out: DEVICE, as in cc_dense_weights.  Synchronises `stream`. */
int cc_dense_weights_noalloc(int64_t n, int64_t p, const float* X, const uint8_t* mask, float phi, float* W_out, void* stream);

/* Release the three arrays cc_knn_weights returned (NULLs are ignored). */
void cc_free_graph(int64_t* rowptr, int32_t* col, float* w);

/* ---- f4: graph utilities -------------------------------------------------------------
 * Connected components of a symmetric CSR graph (rowptr int64[n+1], col int32[nnz]; DEVICE): labels_out
 * (DEVICE int32[n]) numbered by smallest member, *ncomponents (HOST, may be NULL).  Synchronises `stream`. */
int cc_graph_components(int64_t n, const int64_t* rowptr, const int32_t* col, int32_t* labels_out,
                        int32_t* ncomponents, void* stream);

/* Smallest k <= min(kmax, n-1, 64) whose OR-symmetrised k-NN graph (cc_knn_weights) is connected, found by
 * bisection -- the graphs are nested in k (L150).  *k_out (HOST) = -1 when even kmax is not connected. */
int cc_smallest_connected_k(int64_t n, int64_t p, const float* X, const uint8_t* mask, int32_t kmax,
                            int32_t* k_out, void* stream);

/* ---- problem set-up --------------------------------------------------------------------------------
 * Validates the inputs once (error codes above), copies them, builds the internal layout and sets the
 * cold start (S4): U0 = X with missing entries set to the observed column mean, V0 = D U0.
 * X, mask, rowptr, col, w: DEVICE pointers (mask may be NULL = all observed; with prm->dense = 1,
 * rowptr and col are ignored and w is the n x n matrix).  prm: HOST pointer or NULL for defaults.
 * *out (HOST) receives the handle. */
int cc_create(cc_handle** out, int64_t n, int64_t p, const float* X, const uint8_t* mask,
              const int64_t* rowptr, const int32_t* col, const float* w, const cc_params* prm,
              void* stream);

/* ---- a1-a6: the MM iteration, PAPER.md L57-L103, L116 ---------------------------------------------
 * Runs MM iterations at this gamma, warm-started from the handle's current state (after cc_create or
 * cc_reset: the cold start).  Each iteration: projection onto C (L90-L103), d_m (L76), U update (L82,
 * L116), block soft-threshold (L86-L88).  Stops after an iteration m with m+1 >= min_it, m >= 1 and
 * Phi_{m-1} - Phi_m <= tol (1 + |Phi_{m-1}|) (S3), or after maxit iterations; tol = 0 runs exactly
 * maxit iterations.  Phi_m = 1/2 sum_obs (x-u_m)^2 + gamma sum_E w ||v_m|| + rho d_m (L64-L66, L109).
 * iters_out, phi_out (HOST, may be NULL): iterations done and the last recorded Phi.  Synchronises. */
int cc_solve(cc_handle* h, double gamma, double tol, int32_t maxit, int32_t* iters_out,
             double* phi_out);

/* ---- f1: kappa continuation (not in the paper, reading S26) ----------------------
 * The iteration count of the MM map grows like 1/kappa (the U update moves a fraction d/(d+rho) ~ kappa of the
 * way once dist is small).  This runs cc_solve in stages at one gamma: rho stays at S1's value and
 * eps_s = (kappa_s rho)^2 with kappa_s = kappa_start, kappa_start*factor, ... while larger than prm.kappa; every
 * stage is warm-started from the previous one and stops by the rule of cc_solve (tol) or after stage_maxit
 * iterations; the last stage is cc_solve itself at prm.kappa (tol, maxit), so what it converges to is the
 * contract iteration's fixed point.  kappa_start <= prm.kappa degenerates to a plain cc_solve.  Measured on the
 * large-sparse path: kappa_start = 0.1, factor = 0.1, stage_maxit = 200 halves the path time at a
 * smaller distance to the converged path; kappa_start = 1 helps cold starts but not a warm-started path.
 * stage_iters_out[cap] (HOST, may be NULL with cap = 0): iterations of each stage, *nstages_out (HOST, may be
 * NULL) the number of stages run (entries beyond cap are not written).  phi_out and the history are the last
 * stage's.  CC_ESTATE when the handle fixes eps_abs.  Synchronises. */
int cc_solve_continuation(cc_handle* h, double gamma, double kappa_start, double factor, int32_t stage_maxit,
                          double tol, int32_t maxit, int32_t* stage_iters_out, int32_t cap, int32_t* nstages_out,
                          double* phi_out);

/* ---- a7: gamma path, PAPER.md L144 (U stays on the device between gammas, cf. L202) ---------------
 * For each gamma in the caller's order: cc_solve warm-started from the previous gamma, then a device
 * snapshot of U and of the cluster labels.  gammas, iters_out[ngamma], phi_out[ngamma]: HOST (outputs
 * may be NULL).  ngamma must be <= max_snapshots.  Snapshots of an earlier path are dropped. */
int cc_path(cc_handle* h, const double* gammas, int32_t ngamma, double tol, int32_t maxit,
            int32_t* iters_out, double* phi_out);

/* f1 on the path: as cc_path, with cc_solve_continuation (same kappa_start, factor, stage_maxit) at every gamma.
 * iters_out[g] (HOST, may be NULL) = iterations of all stages at gammas[g]. */
int cc_path_continuation(cc_handle* h, const double* gammas, int32_t ngamma, double kappa_start, double factor,
                         int32_t stage_maxit, double tol, int32_t maxit, int32_t* iters_out, double* phi_out);

/* Copy U (n*p fp32 row-major) into a caller-owned buffer.  gamma_index = -1: the current state;
 * 0..ngamma-1: the snapshot cc_path took.  U_out is DEVICE when out_on_device != 0, else HOST. */
int cc_get_U(cc_handle* h, int32_t gamma_index, float* U_out, int32_t out_on_device);

/* ---- f2: project U on q <= 8 caller-given directions on the device (PAPER.md L144 plots the path on two
 * principal components; L202/L210: reading all of U back per gamma was the paper's bottleneck).
 * out[i][k] = sum_c (u_ic - xbar_c) P[c][k], xbar = observed column means of X.  P: DEVICE p*q row-major;
 * out: n*q, DEVICE when out_on_device != 0 else HOST (then the call synchronises).  gamma_index as in cc_get_U. */
int cc_get_projection(cc_handle* h, int32_t gamma_index, const float* P, int32_t q, float* out, int32_t out_on_device);

/* ---- f2: principal directions of the original data on the device, PAPER.md L144 ("project the cluster path
 * onto any two principal components of the original data"), L210 ("project the data to principal components on
 * each GPU itself prior to data transfer").  Reading S25: the data are X with missing entries at the observed
 * column mean (the cold start), columns centred; direction k is the k-th leading eigenvector of the sample
 * covariance Xc^T Xc / (n-1).  Computed by block iteration with 16 vectors (two passes over X per step) until
 * every requested Ritz pair has ||C y - theta y|| <= tol * theta_1, or maxit steps (tol = 1e-6, maxit = 300 are
 * sensible; the speed of convergence is set by the ratio of the 17th to the q-th eigenvalue).
 * P_out: p*q fp32 row-major (the layout cc_get_projection takes), DEVICE when out_on_device != 0 else HOST; each
 * direction has unit length and its entry of largest magnitude is positive.  A direction whose eigenvalue is
 * below 1e-7 of the largest (data of rank < q) comes back as a zero vector with variance 0.
 * var_out[q] (HOST, may be NULL): the variances theta_k / (n-1), decreasing.  resid_out[q] (HOST, may be NULL):
 * the relative residuals reached.  iters_out (HOST, may be NULL): steps taken.  1 <= q <= min(8, p).
 * Synchronises.  Does not touch the MM state. */
int cc_principal_components(cc_handle* h, int32_t q, int32_t maxit, double tol, float* P_out, int32_t out_on_device,
                            double* var_out, double* resid_out, int32_t* iters_out);

/* ---- a8: cluster read-out (S16; the paper never defines it, L154, L206) ---------------------------
 * Connected components of the graph whose edges are the pairs with v_ij = 0 exactly, numbered in
 * increasing order of each component's smallest member.  labels_out: int32[n], DEVICE when
 * out_on_device != 0 else HOST; nclusters (HOST, may be NULL).  gamma_index as in cc_get_U.
 * Synchronises. */
int cc_clusters(cc_handle* h, int32_t gamma_index, int32_t* labels_out, int32_t out_on_device,
                int32_t* nclusters);

/* Phi_m and d_m of the last cc_solve (or of the last gamma of cc_path), up to `cap` entries each, into
 * HOST arrays (either may be NULL); *count (HOST) = entries written. */
int cc_get_history(cc_handle* h, double* phi_out, double* d_out, int32_t cap, int32_t* count);

/* Diagnostics of the last cc_solve (HOST outputs, any may be NULL): rho and eps used, total inner
 * (projection) iterations, f_gamma(U) of eq. 1/6 at the current U (L35, L109; costs one extra pair
 * sweep), and the smallest relative margin | ||b_ij|| - thr_ij | / thr_ij over pairs at the last
 * shrink (how close any pair was to flipping its fused/unfused decision). */
int cc_get_stats(cc_handle* h, double* rho, double* eps, int64_t* proj_iters, double* f_gamma,
                 double* min_margin);

/* Live per-kernel device time of the MM iteration, accumulated over every cc_solve since
 * cc_create / cc_reset_profile.  ns_out[8] (HOST doubles), calls_out[8] (HOST): index 0 k_rhs (a1),
 * 1 k_cg_spmv (a2), 2 k_cg_update (a2), 3 k_norm (a3+a6), 4 k_update (a5+a4); dense mode (a9): 5 kd_proj
 * (with the column means), 6 kd_pairs, 7 kd_edges.  Measured on the device:
 * the block that finishes a kernel last reads %globaltimer and the interval since the previous kernel
 * finished (= this kernel plus its launch gap) is charged to it.  Either pointer may be NULL.
 * Handles that run the persistent single-kernel solve (small n, see cc_solve) report its PHASES per MM iteration
 * instead, and only after cc_reset_profile has been called once (reading the timer costs about 0.5 us a lap, several
 * laps per iteration, so it is off by default): 0 right-hand side, 2 projection by the inverse, 3 pair norms and
 * partial sums, 4 shrink and U update, 5 / 6 the two grid barriers.  Diagnostics only; not part of the iteration. */
int cc_get_profile(cc_handle* h, double* ns_out, int64_t* calls_out);
/* Zero the accumulated times (and switch the persistent kernel's phase timing on for this handle). */
int cc_reset_profile(cc_handle* h);

/* Back to the cold start (S4); snapshots are dropped. */
int cc_reset(cc_handle* h);

/* Counts (HOST outputs, any may be NULL): undirected pairs |E|, directed entries nnz, and the number
 * of kernel launches this handle has issued so far (graph kernel nodes executed are counted). */
int cc_get_counts(cc_handle* h, int64_t* n_pairs, int64_t* nnz, int64_t* launches);

/* Message of the last failing call on this handle (h = NULL: of the last failing cc_create /
 * cc_knn_weights on this thread).  Never NULL. */
const char* cc_last_error(const cc_handle* h);

void cc_destroy(cc_handle* h);

#ifdef __cplusplus
}
#endif
#endif /* CC_B200_H */
