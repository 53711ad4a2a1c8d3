// cc_api.cu -- the extern "C" entry points of include/cc_b200.h: argument checks, the per-gamma
// constants (S1, S2), launching the solve graph, snapshots along the gamma path.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "cc_internal.h"

thread_local char cc_g_err[256] = "";
#define g_err cc_g_err

cudaError_t cc_dev_alloc(void** p, size_t bytes, cudaStream_t st) {
    static bool pool_ready = false;
    if (!pool_ready) {
        int dev = 0;
        cudaMemPool_t pool;
        if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
            unsigned long long thr = ~0ULL;
            cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
        }
        cudaGetLastError();
        pool_ready = true;
    }
    return cudaMallocAsync(p, bytes ? bytes : 1, st);
}

void cc_dev_free(void* p, cudaStream_t st) {
    if (p) cudaFreeAsync(p, st);
}

extern "C" {

int cc_default_params(cc_params* prm) {
    if (!prm) return CC_EINVAL;
    memset(prm, 0, sizeof(*prm));
    prm->rho_scale = 1.1;
    prm->rho_abs = 0.0;
    prm->kappa = 1e-2;
    prm->eps_abs = 0.0;
    prm->proj_tol = 1e-5;
    prm->proj_maxit = 500;
    prm->min_it = 10;
    prm->dense = 0;
    prm->use_graph = 1;
    prm->hist_cap = 4096;
    prm->max_snapshots = 64;
    return CC_OK;
}

int cc_create(cc_handle** out, int64_t n, int64_t p, const float* X, const uint8_t* mask, const int64_t* rowptr,
              const int32_t* col, const float* w, const cc_params* prm, void* stream) {
    if (!out) { snprintf(g_err, sizeof(g_err), "out is NULL"); return CC_EINVAL; }
    *out = nullptr;
    cc_params P;
    cc_default_params(&P);
    if (prm) P = *prm;
    const bool dense = P.dense != 0;
    if (n < 1 || p < 1 || !X || (dense && !w) || (!dense && !rowptr) || n > 2147483647LL / 2 || p > (1LL << 28)) {
        snprintf(g_err, sizeof(g_err), "cc_create: bad size or NULL pointer (n=%lld p=%lld)", (long long)n, (long long)p);
        return CC_EINVAL;
    }
    if (P.reserved != 0 || P.proj_maxit < 1 || P.hist_cap < 0 || P.max_snapshots < 0 || !(P.proj_tol > 0.0) ||
        (P.rho_abs <= 0.0 && !(P.rho_scale > 0.0)) || (P.eps_abs <= 0.0 && !(P.kappa > 0.0))) {
        snprintf(g_err, sizeof(g_err), "cc_create: bad cc_params");
        return CC_EINVAL;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        snprintf(g_err, sizeof(g_err), "no CUDA device: libcc_b200 has no CPU fallback");
        return CC_ECUDA;
    }
    cc_handle* h = (cc_handle*)calloc(1, sizeof(cc_handle));
    if (!h) { snprintf(g_err, sizeof(g_err), "out of host memory"); return CC_ENOMEM; }
    h->n = n;
    h->p = p;
    h->prm = P;
    h->dense = dense ? 1 : 0;
    h->stream = (cudaStream_t)stream;
    int rc = ccu_validate_and_build(h, X, mask, rowptr, col, w);
    if (rc == CC_OK && P.max_snapshots > 0) {
        h->snapK = (int32_t*)calloc((size_t)P.max_snapshots, sizeof(int32_t));
        if (!h->snapK) rc = CC_ENOMEM;
    }
    if (rc == CC_OK) {
        cudaError_t e = cudaStreamSynchronize(h->stream);
        if (e != cudaSuccess) { snprintf(h->err, sizeof(h->err), "cc_create: %s", cudaGetErrorString(e)); rc = CC_ECUDA; }
    }
    if (rc != CC_OK) {
        snprintf(g_err, sizeof(g_err), "%s", h->err[0] ? h->err : "cc_create failed");
        cudaStreamSynchronize(h->stream);
        ccu_free(h);
        free(h);
        return rc;
    }
    *out = h;
    return CC_OK;
}

static void rho_eps(const cc_handle* h, double gamma, double* rho, double* eps) {
    // S1: rho = rho_scale * G_bound(gamma), G_bound = sqrt(sum_obs (x - colmean)^2 + gamma^2 sum_E w^2)
    // S2: eps = (kappa rho)^2
    double r = h->prm.rho_abs > 0.0 ? h->prm.rho_abs
                                    : h->prm.rho_scale * sqrt(h->xss + gamma * gamma * h->sumw2);
    if (!(r > 0.0)) r = 1.0;  // constant data and gamma = 0: any rho works (U = X at once)
    *rho = r;
    const double kappa = h->kappa_stage > 0.0 ? h->kappa_stage : h->prm.kappa;
    *eps = (h->prm.eps_abs > 0.0 && !(h->kappa_stage > 0.0)) ? h->prm.eps_abs : (kappa * r) * (kappa * r);
}

int cc_solve(cc_handle* h, double gamma, double tol, int32_t maxit, int32_t* iters_out, double* phi_out) {
    if (!h) return CC_EINVAL;
    if (!(gamma >= 0.0) || std::isinf(gamma) || !(tol >= 0.0) || maxit < 0) {
        snprintf(h->err, sizeof(h->err), "cc_solve: need gamma >= 0 finite, tol >= 0, maxit >= 0");
        return CC_EINVAL;
    }
    cc_scal* S = h->sc_host;
    const double pen_keep = S->pen_next;   // dense mode: penalty of the current state, written by the last kd_edges
    memset(S, 0, sizeof(*S));
    S->pen_next = pen_keep;
    S->gamma = gamma;
    rho_eps(h, gamma, &S->rho, &S->eps);
    S->tol = tol;
    S->xscale = sqrt(h->xss);
    S->proj_tol = h->prm.proj_tol;
    S->d = S->d_prev = sqrt(S->eps);
    S->cthr = h->dense && h->dn_tc ? h->dn_cthr : (float)(gamma * S->d / S->rho);   // tensor-core dense path: the factor that made the current (implicit) S
    S->mm_maxit = maxit;
    S->mm_min_it = h->prm.min_it;
    S->mm_active = 1;
    S->cg_maxit = h->prm.proj_maxit;
    S->hist_cap = h->prm.hist_cap;
    S->prof_phases = h->pt_prof;
    if (maxit == 0) {
        if (iters_out) *iters_out = 0;
        if (phi_out) *phi_out = NAN;
        return CC_OK;
    }
    CC_CUDA(h, cudaMemcpyAsync(h->sc, S, sizeof(cc_scal), cudaMemcpyHostToDevice, h->stream));
    if (h->pt_slabs) {
        // small n: the whole MM loop is one persistent kernel (cc_persist.cu)
        int rc = ccp_solve(h);
        if (rc != CC_OK) return rc;
        CC_CUDA(h, cudaMemcpyAsync(S, h->sc, sizeof(cc_scal), cudaMemcpyDeviceToHost, h->stream));
        CC_CUDA(h, cudaStreamSynchronize(h->stream));
    } else if (h->prm.use_graph) {
        int rc = h->dense ? ccd_build_graph(h) : ccs_build_graph(h);
        if (rc != CC_OK) return rc;
        CC_CUDA(h, cudaGraphLaunch(h->gexec, h->stream));
        CC_CUDA(h, cudaMemcpyAsync(S, h->sc, sizeof(cc_scal), cudaMemcpyDeviceToHost, h->stream));
        CC_CUDA(h, cudaStreamSynchronize(h->stream));
    } else {
        int rc = h->dense ? ccd_solve_eager(h, maxit) : ccs_solve_eager(h, maxit);
        if (rc != CC_OK) return rc;
    }
    h->launches += (long long)S->nlaunch;      // counted on the device: every kernel of the iteration that executed
    if (h->dense && h->dn_tc) h->dn_cthr = S->cthr;
    for (int k = 0; k < 8; ++k) { h->prof_ns[k] += S->prof_ns[k]; h->prof_calls[k] += S->prof_calls[k]; }
    if (iters_out) *iters_out = S->mm_iter;
    if (phi_out) *phi_out = S->phi;
    if (S->cg_failed) {
        snprintf(h->err, sizeof(h->err), "projection solve hit proj_maxit=%d", h->prm.proj_maxit);
        return CC_ENOCONV;
    }
    return CC_OK;
}

int cc_solve_continuation(cc_handle* h, double gamma, double kappa_start, double factor, int32_t stage_maxit,
                          double tol, int32_t maxit, int32_t* stage_iters_out, int32_t cap, int32_t* nstages_out,
                          double* phi_out) {
    if (!h) return CC_EINVAL;
    if (!(kappa_start > 0.0) || std::isinf(kappa_start) || !(factor > 0.0 && factor < 1.0) || stage_maxit < 1 ||
        cap < 0 || (cap > 0 && !stage_iters_out)) {
        snprintf(h->err, sizeof(h->err), "cc_solve_continuation: need kappa_start > 0 finite, 0 < factor < 1, stage_maxit >= 1");
        return CC_EINVAL;
    }
    if (h->prm.eps_abs > 0.0) {
        snprintf(h->err, sizeof(h->err), "cc_solve_continuation: the handle fixes eps_abs; stages need eps = (kappa rho)^2");
        return CC_ESTATE;
    }
    int stage = 0, worst = CC_OK;
    for (double kappa = kappa_start; kappa > h->prm.kappa * (1.0 + 1e-12); kappa *= factor, ++stage) {
        int it = 0;
        h->kappa_stage = kappa;
        const int rc = cc_solve(h, gamma, tol, stage_maxit, &it, nullptr);
        h->kappa_stage = 0.0;
        if (rc != CC_OK && rc != CC_ENOCONV) return rc;
        if (rc == CC_ENOCONV) worst = rc;
        if (stage < cap) stage_iters_out[stage] = it;
    }
    int it = 0;
    const int rc = cc_solve(h, gamma, tol, maxit, &it, phi_out);   // the contract iteration, warm-started
    if (rc != CC_OK && rc != CC_ENOCONV) return rc;
    if (stage < cap) stage_iters_out[stage] = it;
    if (nstages_out) *nstages_out = stage + 1;
    return rc == CC_ENOCONV ? rc : worst;
}

// kappa_start <= 0: the plain path (cc_solve per gamma); else staged solves (f1).  iters_out[g] = all iterations at gamma g.
static int path_impl(cc_handle* h, const double* gammas, int32_t ngamma, double kappa_start, double factor,
                     int32_t stage_maxit, double tol, int32_t maxit, int32_t* iters_out, double* phi_out) {
    if (!h) return CC_EINVAL;
    if (!gammas || ngamma < 0) { snprintf(h->err, sizeof(h->err), "cc_path: bad arguments"); return CC_EINVAL; }
    if (ngamma > h->prm.max_snapshots) {
        snprintf(h->err, sizeof(h->err), "cc_path: ngamma=%d exceeds max_snapshots=%d", ngamma, h->prm.max_snapshots);
        return CC_ESTATE;
    }
    const size_t nl = (size_t)h->n * h->ld;
    if (!h->snapU && ngamma > 0) {
        cudaError_t e1 = cc_dev_alloc((void**)&h->snapU, nl * sizeof(float) * (size_t)h->prm.max_snapshots, h->stream);
        cudaError_t e2 = cc_dev_alloc((void**)&h->snapLab, (size_t)h->n * sizeof(int32_t) * (size_t)h->prm.max_snapshots, h->stream);
        if (e1 != cudaSuccess || e2 != cudaSuccess) {
            cudaGetLastError();
            snprintf(h->err, sizeof(h->err), "cc_path: cannot allocate %d snapshots", h->prm.max_snapshots);
            return CC_ENOMEM;
        }
    }
    h->nsnap = 0;
    int worst = CC_OK;
    for (int g = 0; g < ngamma; ++g) {
        int it = 0;
        double phi = 0.0;
        int rc;
        if (kappa_start > 0.0) {
            int32_t st[64], ns = 0;
            rc = cc_solve_continuation(h, gammas[g], kappa_start, factor, stage_maxit, tol, maxit, st, 64, &ns, &phi);
            for (int k = 0; k < ns && k < 64; ++k) it += st[k];
        } else {
            rc = cc_solve(h, gammas[g], tol, maxit, &it, &phi);
        }
        if (rc != CC_OK && rc != CC_ENOCONV) return rc;
        if (rc == CC_ENOCONV) worst = rc;
        if (iters_out) iters_out[g] = it;
        if (phi_out) phi_out[g] = phi;
        CC_CUDA(h, cudaMemcpyAsync(h->snapU + (size_t)g * nl, h->U, nl * sizeof(float), cudaMemcpyDeviceToDevice, h->stream));
        rc = ccl_labels(h, h->snapLab + (size_t)g * h->n, &h->snapK[g]);
        if (rc != CC_OK) return rc;
        h->nsnap = g + 1;
    }
    return worst;
}

int cc_path(cc_handle* h, const double* gammas, int32_t ngamma, double tol, int32_t maxit, int32_t* iters_out,
            double* phi_out) {
    return path_impl(h, gammas, ngamma, 0.0, 0.0, 0, tol, maxit, iters_out, phi_out);
}

int cc_path_continuation(cc_handle* h, const double* gammas, int32_t ngamma, double kappa_start, double factor,
                         int32_t stage_maxit, double tol, int32_t maxit, int32_t* iters_out, double* phi_out) {
    if (!h) return CC_EINVAL;
    if (!(kappa_start > 0.0)) {
        snprintf(h->err, sizeof(h->err), "cc_path_continuation: need kappa_start > 0");
        return CC_EINVAL;
    }
    return path_impl(h, gammas, ngamma, kappa_start, factor, stage_maxit, tol, maxit, iters_out, phi_out);
}

// strided (ld -> p) copy out of the padded layout
static int copy_out_U(cc_handle* h, const float* src, float* dst, int on_device) {
    CC_CUDA(h, cudaMemcpy2DAsync(dst, (size_t)h->p * sizeof(float), src, (size_t)h->ld * sizeof(float),
                                 (size_t)h->p * sizeof(float), (size_t)h->n,
                                 on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h->stream));
    if (!on_device) CC_CUDA(h, cudaStreamSynchronize(h->stream));
    return CC_OK;
}

int cc_get_U(cc_handle* h, int32_t gamma_index, float* U_out, int32_t out_on_device) {
    if (!h) return CC_EINVAL;
    if (!U_out) { snprintf(h->err, sizeof(h->err), "cc_get_U: U_out is NULL"); return CC_EINVAL; }
    if (gamma_index < -1 || gamma_index >= h->nsnap) {
        snprintf(h->err, sizeof(h->err), "cc_get_U: gamma_index %d outside [-1, %d)", gamma_index, h->nsnap);
        return CC_ESTATE;
    }
    const float* src = gamma_index < 0 ? h->U : h->snapU + (size_t)gamma_index * h->n * h->ld;
    return copy_out_U(h, src, U_out, out_on_device);
}

int cc_clusters(cc_handle* h, int32_t gamma_index, int32_t* labels_out, int32_t out_on_device, int32_t* nclusters) {
    if (!h) return CC_EINVAL;
    if (!labels_out) { snprintf(h->err, sizeof(h->err), "cc_clusters: labels_out is NULL"); return CC_EINVAL; }
    if (gamma_index < -1 || gamma_index >= h->nsnap) {
        snprintf(h->err, sizeof(h->err), "cc_clusters: gamma_index %d outside [-1, %d)", gamma_index, h->nsnap);
        return CC_ESTATE;
    }
    const size_t bytes = (size_t)h->n * sizeof(int32_t);
    if (gamma_index < 0) {
        if (out_on_device) return ccl_labels(h, labels_out, nclusters);
        int32_t* tmp = nullptr;
        CC_CUDA(h, cc_dev_alloc((void**)&tmp, bytes, h->stream));
        int rc = ccl_labels(h, tmp, nclusters);
        if (rc == CC_OK) {
            cudaError_t e = cudaMemcpyAsync(labels_out, tmp, bytes, cudaMemcpyDeviceToHost, h->stream);
            if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
            if (e != cudaSuccess) { snprintf(h->err, sizeof(h->err), "cc_clusters: %s", cudaGetErrorString(e)); rc = CC_ECUDA; }
        }
        cc_dev_free(tmp, h->stream);
        return rc;
    }
    CC_CUDA(h, cudaMemcpyAsync(labels_out, h->snapLab + (size_t)gamma_index * h->n, bytes,
                               out_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h->stream));
    CC_CUDA(h, cudaStreamSynchronize(h->stream));
    if (nclusters) *nclusters = h->snapK[gamma_index];
    return CC_OK;
}

int cc_get_history(cc_handle* h, double* phi_out, double* d_out, int32_t cap, int32_t* count) {
    if (!h) return CC_EINVAL;
    int k = h->sc_host ? h->sc_host->mm_iter : 0;
    if (k > h->prm.hist_cap) k = h->prm.hist_cap;
    if (k > cap) k = cap;
    if (k < 0) k = 0;
    if (phi_out && k) CC_CUDA(h, cudaMemcpyAsync(phi_out, h->hist_phi, (size_t)k * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    if (d_out && k) CC_CUDA(h, cudaMemcpyAsync(d_out, h->hist_d, (size_t)k * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CC_CUDA(h, cudaStreamSynchronize(h->stream));
    if (count) *count = k;
    return CC_OK;
}

int cc_get_stats(cc_handle* h, double* rho, double* eps, int64_t* proj_iters, double* f_gamma, double* min_margin) {
    if (!h) return CC_EINVAL;
    if (rho) *rho = h->sc_host->rho;
    if (eps) *eps = h->sc_host->eps;
    if (proj_iters) *proj_iters = h->sc_host->cg_total;
    if ((f_gamma || min_margin) && h->dense) {
        snprintf(h->err, sizeof(h->err), "cc_get_stats: f_gamma / min_margin are not available in dense mode yet");
        return CC_ESTATE;
    }
    if (f_gamma) { int rc = ccu_fgamma(h, f_gamma); if (rc != CC_OK) return rc; }
    if (min_margin) { int rc = ccu_min_margin(h, min_margin); if (rc != CC_OK) return rc; }
    return CC_OK;
}

int cc_get_profile(cc_handle* h, double* ns_out, int64_t* calls_out) {
    if (!h) return CC_EINVAL;
    for (int k = 0; k < 8; ++k) {
        if (ns_out) ns_out[k] = (double)h->prof_ns[k];
        if (calls_out) calls_out[k] = (int64_t)h->prof_calls[k];
    }
    return CC_OK;
}

int cc_reset_profile(cc_handle* h) {
    if (!h) return CC_EINVAL;
    memset(h->prof_ns, 0, sizeof(h->prof_ns));
    memset(h->prof_calls, 0, sizeof(h->prof_calls));
    h->pt_prof = 1;      // from now on the persistent kernel times its phases too (see cc_b200.h)
    return CC_OK;
}

int cc_reset(cc_handle* h) {
    if (!h) return CC_EINVAL;
    h->nsnap = 0;
    int rc = ccu_cold_start(h);
    if (rc != CC_OK) return rc;
    CC_CUDA(h, cudaStreamSynchronize(h->stream));
    return CC_OK;
}

int cc_get_counts(cc_handle* h, int64_t* n_pairs, int64_t* nnz, int64_t* launches) {
    if (!h) return CC_EINVAL;
    if (n_pairs) *n_pairs = h->npairs;
    if (nnz) *nnz = h->nnz;
    if (launches) *launches = h->launches;
    return CC_OK;
}

const char* cc_last_error(const cc_handle* h) { return h ? h->err : g_err; }

void cc_destroy(cc_handle* h) {
    if (!h) return;
    cudaStreamSynchronize(h->stream);
    ccu_free(h);
    free(h);
}

}  // extern "C"
