// cc_internal.h -- internal layout shared by the .cu files of libcc_b200.so (never installed, never
// seen by the oracle).  Notation follows PAPER.md section 3: U (cases), A = projection of U onto the
// constraint set C (L90-L103), b_ij = a_i - a_j (L84), v_ij (L48-L53), d_m (L76), rho, eps.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/cc_b200.h"

// ---------------------------------------------------------------------------------------------
// Device-resident scalars of one solve.  Written by the "last block" of the reducing kernels and by
// single-thread control kernels; read by every kernel of the iteration.  doubles first.
// ---------------------------------------------------------------------------------------------
struct cc_scal {
    // problem constants for this gamma
    double gamma, rho, eps, tol;
    double xscale;      // sqrt(sum_obs (x - colmean)^2): the data scale of the projection stop rule
    double proj_tol;
    // MM iteration
    double d, d_prev;   // d_m of L76; d_prev seeds the projection stop rule (sqrt(eps) at m = 0)
    double dist2, loss, pen;
    double phi, phi_prev;
    double min_margin;  // smallest | ||b|| - thr | / thr at the last shrink
    double pen_next;    // dense mode: sum_{i<j} w ||v|| of the state kd_edges just wrote (the next iteration's penalty)
    float cu, ca;       // d/(d+rho), rho/(d+rho)          (U update, L82)
    float cthr;         // gamma d / rho                   (threshold = cthr * w_ij, L86)
    float pad0;
    // inner conjugate-gradient solve of (I+L) delta = r0
    double cg_gamma, cg_gamma_old, cg_delta, cg_alpha, cg_beta, cg_thresh;
    // control
    int32_t mm_iter;      // iterations completed in this solve
    int32_t mm_maxit;
    int32_t mm_min_it;
    int32_t mm_active;    // 1 while the outer loop runs
    int32_t stop_pending; // the stop rule fired in k_norm: finish this iteration's updates, then stop
    int32_t cg_iter;      // inner iterations of the current projection
    int32_t cg_active;
    int32_t cg_maxit;
    int32_t cg_failed;    // some projection hit cg_maxit
    int32_t hist_cap;
    long long cg_total;   // inner iterations over the whole solve
    // last-block tickets (one per reducing kernel)
    unsigned int ticket[8];
    // live per-kernel timing: the block that finishes a kernel last reads %globaltimer; the interval
    // since the previous kernel's end (kernel + launch gap) is charged to this kernel
    unsigned long long t_last;
    unsigned long long prof_ns[8];
    unsigned long long prof_calls[8];
    unsigned long long nlaunch;   // kernels of this solve that executed (each counts itself on the device)
    int32_t prof_phases;          // persistent kernel: time its phases (reading %globaltimer costs ~0.5 us a lap; off by default)
    int32_t pad1;
};

// Per-block partial sums: up to CC_NPART doubles per block, CC_MAXBLK blocks.
#define CC_INV_NMAX 384     // largest n whose projection uses the precomputed inverse (n x 128 floats of shared memory)
#define CC_INVW_NMAX 4096   // ... and with at most 32 columns (all of uc in one CTA's shared memory): the inverse applied from L2
#define CC_NPART 4
#define CC_MAXBLK 16384

struct cc_handle {
    // sizes
    int64_t n, p, ld;        // ld = p rounded up to a multiple of 4 (padding columns stay 0)
    int64_t nnz, npairs;
    int dense;
    int G;                   // lanes per row group (power of two <= 32); a group covers 4*G columns
    int nchunk;              // ceil(ld / (4G)) column chunks
    cc_params prm;
    cudaStream_t stream;
    // node arrays (n x ld fp32)
    float *X, *U, *A, *Ap, *Z;        // Z = warm start of the projection (u + previous correction)
    float *R, *Pv, *Sv, *Uc;          // CG: (R unused: r = D uc), search dir, (I+L) search dir, D^-1 r
    float* Dl;                        // previous correction a - u (warm-start extrapolation)
    uint8_t* mask;                    // n x ld or NULL
    float* colmean;                   // ld
    // graph (symmetric CSR)
    int32_t* rowptr;                  // n+1 (nnz < 2^31 enforced)
    int32_t* rowup;                   // n: first entry of row i with col > i (rows are sorted)
    int32_t* order;                   // n: rows by decreasing degree (processing order of the gather kernels)
    int4* rowdesc;                    // n: (row, rowup, row end, row begin) in that order: one independent 16-byte load per walked row
    int32_t* col;                     // nnz
    int32_t* peer;                    // nnz: index of the reverse entry
    float* w;                         // nnz
    float* s;                         // nnz: shrink factor of v_ij = s_ij (a'_i - a'_j)   (L86)
    float* vn;                        // nnz: ||v_ij||
    float* nb2;                       // nchunk x nnz partial squared norms of b_ij
    float* tmpE;                      // nnz scratch (diagnostics)
    float* dinv;                      // n: 1 / (1 + |N_i|)
    float* Minv;                      // n x n: (D^-1 (I+L))^-1 for n <= CC_INV_NMAX, else NULL (CG solver)
    int inv_wide;                     // 1: Minv is applied by k_apply_inv_wide (n > CC_INV_NMAX, few columns)
    // dense mode (complete graph): n x n matrices instead of the CSR arrays
    float *Wd, *Sd, *VNd, *NB2d;      // weights, shrink factors, ||v||, ||b||^2 (dn_ksplit column-range slices); tensor-core path: Wd, NB2d =
                                      // ||b|| (pairs i < j) and Rd only (S and ||v|| are recomputed where they are used)
    float *ubar, *abar;               // column means of U and A'
    float* dbar;                      // column means of A - U (dense mode; subtracted by k_update)
    double* colps;                    // partial column sums
    uint8_t* pre_pairs;               // kd_prep_pairs: TF32 hi/lo operand tiles in the tensor core's smem layout
    float* nrm_part;                  // per-K-block partial row norms
    uint8_t* pre_B;                   // kd_proj_tc3's B operand (A' - abar)^T, TF32 hi/lo tiles in the operand layout (by kd_prep_proj)
    float* Rd;                        // tensor-core path: R = w / ||b|| (n x n, both triangles): all the contraction needs to form S
    int dn_ksplit, dn_big, dn_tc, dn_small, dn_small_cs, dn_small_grid, dn_small_tc;
    unsigned long long dn_small_tm[4][16];          // kd_small_tc: the tensor maps of U, A', X, A (CUtensorMap, 128 bytes each)
    float dn_cthr;                    // tensor-core path: the threshold factor gamma d / rho that defines the current implicit S
    // scalars
    cc_scal* sc;                      // device
    cc_scal* sc_host;                 // pinned mirror
    double* part;                     // CC_MAXBLK * CC_NPART doubles per reducing kernel (x8)
    double *hist_phi, *hist_d;        // hist_cap each
    double* dout;                     // 4 doubles: results of the one-off reductions
    int* dflag;                       // validation flags
    int sms;                          // multiprocessor count
    double sumw2, xss;                // sum_E w^2, sum_obs (x-colmean)^2
    double kappa_stage;               // > 0 inside cc_solve_continuation: the kappa of the running stage (f1, S26)
    // snapshots
    float* snapU;                     // max_snapshots x n x ld
    int32_t* snapLab;                 // max_snapshots x n
    int32_t* snapK;                   // host
    int nsnap;
    int32_t* lab;                     // n (scratch for cc_clusters)
    int32_t* lab_flag;                // device int
    int32_t* lab_rank;                // n, allocated on first cc_clusters
    // graph execution
    cudaGraphExec_t gexec;
    cudaGraphConditionalHandle cond_outer, cond_inner;   // 0 while launching eagerly
    cudaGraph_t graph;
    long long launches;
    unsigned long long prof_ns[8], prof_calls[8];   // accumulated over solves (cc_get_profile)
    int grid_nodes, grid_rows, grid_edges;   // launch sizes, fixed per handle (determinism)
    // persistent single-kernel solve (cc_persist.cu): 0 slabs = not used by this handle
    int pt_slabs, pt_sw, pt_minv_smem, pt_prof;     // pt_minv_smem: the projection mode of k_mm_persist (0, 1, 2)
    size_t pt_smem;
    float* pt_nbpart;                 // pt_slabs x nnz partial squared norms
    double* pt_spart;                 // pt_slabs x 4 partial scalars
    char err[256];
};

// ---- launchers implemented in cc_sparse.cu (all enqueue on h->stream) -----------------------------
void ccs_begin_iter(cc_handle* h);   // resets per-iteration control
void ccs_rhs(cc_handle* h);          // a1: r0 and CG start
void ccs_cg_spmv(cc_handle* h);      // a2: Wv = (I+L) Uc, delta = (Wv, Uc)
void ccs_cg_update(cc_handle* h);    // a2: CG vector updates, gamma' = (r, D^-1 r)
void ccs_norm(cc_handle* h);         // a3 + a6: pair norms, dist^2, loss, penalty -> d, Phi, stop rule
void ccs_update(cc_handle* h);       // a5 + a4: U update, shrink
void ccs_init_state(cc_handle* h);   // cold start of (Ap, Z, s, vn)
void ccs_pair_norms(cc_handle* h, const float* V, float* out, float* s_out);
int ccs_solve_eager(cc_handle* h, int maxit);
int ccs_build_graph(cc_handle* h);
int ccs_setup_inverse(cc_handle* h);

// ---- cc_persist.cu: one persistent kernel per solve for small-n problems (n <= CC_INV_NMAX, state in shared memory)
int ccp_setup(cc_handle* h);
int ccp_solve(cc_handle* h);

// ---- cc_dense.cu (a9) ------------------------------------------------------------------------------
int ccd_setup(cc_handle* h, const float* W);
void ccd_sumw2(cc_handle* h);
void ccd_init_state(cc_handle* h);
void ccd_lab_hook(cc_handle* h, int* changed);
int ccd_solve_eager(cc_handle* h, int maxit);
int ccd_build_graph(cc_handle* h);
void ccs_update_nodes(cc_handle* h, int with_edges, int store_ap);  // k_update, node part (dense mode) [+ the block soft-threshold of the stored-S paths]
// ---- cc_small.cu (a9, n <= 64): the fused kernel with the contraction on the tensor cores
int ccd_small_tc_setup(cc_handle* h);     // 1: use it (sets dn_small_cs, dn_small_grid); 0: not available
int ccd_small_tc_maps(cc_handle* h);      // after the node arrays exist
void ccd_small_tc_launch(cc_handle* h);

// ---- cc_setup.cu ------------------------------------------------------------------------------------
int ccu_validate_and_build(cc_handle* h, const float* X, const uint8_t* mask, const int64_t* rowptr,
                           const int32_t* col, const float* w);
int ccu_cold_start(cc_handle* h);                       // U0 = X, missing -> observed column mean (S4)
int ccu_fgamma(cc_handle* h, double* f_out);            // eq. 1/6 at the current U
int ccu_min_margin(cc_handle* h, double* margin_out);   // min | ||b|| - thr | / thr at the last shrink
void ccu_free(cc_handle* h);
// ---- cc_clusters.cu -----------------------------------------------------------------------------------
int ccl_labels(cc_handle* h, int32_t* labels_dev, int32_t* nclusters_host);

// Device memory comes from the stream-ordered allocator: the default pool keeps freed blocks (release
// threshold raised once), so creating and destroying handles repeatedly does not pay cudaMalloc/cudaFree.
cudaError_t cc_dev_alloc(void** p, size_t bytes, cudaStream_t st);
void cc_dev_free(void* p, cudaStream_t st);

// message of the last failing handle-less call on this thread (cc_create, cc_knn_weights)
extern thread_local char cc_g_err[256];

#define CC_CUDA(h, call)                                                                  \
    do {                                                                                  \
        cudaError_t e_ = (call);                                                          \
        if (e_ != cudaSuccess) {                                                          \
            snprintf((h)->err, sizeof((h)->err), "%s: %s", #call, cudaGetErrorString(e_)); \
            return CC_ECUDA;                                                              \
        }                                                                                 \
    } while (0)
