// cc_clusters.cu -- a8, cluster read-out (S16; the paper never defines it, PAPER.md L154,
// L206): connected components of the graph whose edges are the pairs with v_ij = 0 exactly (s_ij = 0
// after the block soft-threshold, L86-L88), numbered in increasing order of each component's smallest
// member.  Integer work only: min-label hooking + pointer jumping, then a scan over the roots.
#include <cstdio>

#include "cc_internal.h"

namespace {

__global__ void k_lab_init(int n, int* __restrict__ lab) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) lab[i] = i;
}

// One thread per row: smallest label among the row and its fused neighbours; hook the old root to it.
template <typename RP>
__global__ void k_lab_hook(int n, const RP* __restrict__ rowptr, const int* __restrict__ col,
                           const float* __restrict__ s, int* lab, int* changed) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int li = lab[i];
    int m = li;
    for (long long e = rowptr[i]; e < rowptr[i + 1]; ++e)
        if (!s || s[e] == 0.f) m = min(m, lab[col[e]]);   // s == NULL: every edge joins (plain graph components)
    if (m < li) {
        atomicMin(&lab[li], m);
        atomicMin(&lab[i], m);
        *changed = 1;
    }
}

__global__ void k_lab_jump(int n, int* lab) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int l = lab[i];
    while (true) {
        const int ll = lab[l];
        if (ll == l) break;
        l = ll;
    }
    lab[i] = l;
}

// Roots are the smallest members; canonical label = number of roots before this root.  One block.
__global__ void k_lab_rank(int n, const int* __restrict__ lab, int* __restrict__ rank, int* nclusters) {
    __shared__ int sm[1024];
    __shared__ int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < n; base += 1024) {
        const int i = base + threadIdx.x;
        const int isroot = (i < n && lab[i] == i) ? 1 : 0;
        sm[threadIdx.x] = isroot;
        __syncthreads();
        for (int o = 1; o < 1024; o <<= 1) {
            int v = threadIdx.x >= o ? sm[threadIdx.x - o] : 0;
            __syncthreads();
            sm[threadIdx.x] += v;
            __syncthreads();
        }
        if (i < n) rank[i] = carry + sm[threadIdx.x] - isroot;  // exclusive
        __syncthreads();
        if (threadIdx.x == 0) carry += sm[1023];
        __syncthreads();
    }
    if (threadIdx.x == 0) *nclusters = carry;
}

__global__ void k_lab_final(int n, const int* __restrict__ lab, const int* __restrict__ rank, int* __restrict__ out) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = rank[lab[i]];
}

}  // namespace

// labels_dev: int32[n] device output.  Uses h->lab (roots), h->tmpE reinterpret is avoided: rank lives
// in a scratch allocation made on first use.
int ccl_labels(cc_handle* h, int32_t* labels_dev, int32_t* nclusters_host) {
    const int n = (int)h->n;
    const int grid = (n + 255) / 256;
    cudaStream_t st = h->stream;
    if (!h->lab_rank) {
        cudaError_t e = cc_dev_alloc((void**)&h->lab_rank, (size_t)n * sizeof(int), st);
        if (e != cudaSuccess) { snprintf(h->err, sizeof(h->err), "cudaMalloc labels scratch: %s", cudaGetErrorString(e)); return CC_ENOMEM; }
    }
    k_lab_init<<<grid, 256, 0, st>>>(n, h->lab);
    h->launches += 1;
    for (int round = 0; round < 100000; ++round) {
        CC_CUDA(h, cudaMemsetAsync(h->lab_flag, 0, sizeof(int), st));
        if (h->dense) ccd_lab_hook(h, h->lab_flag);
        else k_lab_hook<int><<<grid, 256, 0, st>>>(n, h->rowptr, h->col, h->s, h->lab, h->lab_flag);
        k_lab_jump<<<grid, 256, 0, st>>>(n, h->lab);
        h->launches += 2;
        int changed = 0;
        CC_CUDA(h, cudaMemcpyAsync(&changed, h->lab_flag, sizeof(int), cudaMemcpyDeviceToHost, st));
        CC_CUDA(h, cudaStreamSynchronize(st));
        if (!changed) break;
    }
    k_lab_rank<<<1, 1024, 0, st>>>(n, h->lab, h->lab_rank, h->lab_flag);
    k_lab_final<<<grid, 256, 0, st>>>(n, h->lab, h->lab_rank, labels_dev);
    h->launches += 2;
    int k = 0;
    CC_CUDA(h, cudaMemcpyAsync(&k, h->lab_flag, sizeof(int), cudaMemcpyDeviceToHost, st));
    CC_CUDA(h, cudaStreamSynchronize(st));
    if (nclusters_host) *nclusters_host = k;
    return CC_OK;
}


// ---- f4: graph utilities ("the smallest k giving a connected graph") -------------------------
extern "C" int cc_graph_components(int64_t n, const int64_t* rowptr, const int32_t* col, int32_t* labels_out,
                                   int32_t* ncomponents, void* stream) {
    if (n < 1 || n > 2147483647LL || !rowptr || !labels_out) {
        snprintf(cc_g_err, sizeof(cc_g_err), "cc_graph_components: bad arguments");
        return CC_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    int *lab = nullptr, *rank = nullptr, *flag = nullptr;
    cudaError_t e = cc_dev_alloc((void**)&lab, (size_t)n * sizeof(int), st);
    if (e == cudaSuccess) e = cc_dev_alloc((void**)&rank, (size_t)n * sizeof(int), st);
    if (e == cudaSuccess) e = cc_dev_alloc((void**)&flag, sizeof(int), st);
    int k = 0;
    const int grid = (int)((n + 255) / 256);
    if (e == cudaSuccess) {
        k_lab_init<<<grid, 256, 0, st>>>((int)n, lab);
        for (int round = 0; round < 100000 && e == cudaSuccess; ++round) {
            cudaMemsetAsync(flag, 0, sizeof(int), st);
            k_lab_hook<int64_t><<<grid, 256, 0, st>>>((int)n, rowptr, col, (const float*)nullptr, lab, flag);
            k_lab_jump<<<grid, 256, 0, st>>>((int)n, lab);
            int changed = 0;
            e = cudaMemcpyAsync(&changed, flag, sizeof(int), cudaMemcpyDeviceToHost, st);
            if (e == cudaSuccess) e = cudaStreamSynchronize(st);
            if (!changed) break;
        }
        k_lab_rank<<<1, 1024, 0, st>>>((int)n, lab, rank, flag);
        k_lab_final<<<grid, 256, 0, st>>>((int)n, lab, rank, labels_out);
        if (e == cudaSuccess) e = cudaMemcpyAsync(&k, flag, sizeof(int), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    }
    cc_dev_free(lab, st); cc_dev_free(rank, st); cc_dev_free(flag, st);
    if (e != cudaSuccess) {
        cudaGetLastError();
        snprintf(cc_g_err, sizeof(cc_g_err), "cc_graph_components: %s", cudaGetErrorString(e));
        return e == cudaErrorMemoryAllocation ? CC_ENOMEM : CC_ECUDA;
    }
    if (ncomponents) *ncomponents = k;
    return CC_OK;
}

extern "C" int cc_smallest_connected_k(int64_t n, int64_t p, const float* X, const uint8_t* mask, int32_t kmax,
                                       int32_t* k_out, void* stream) {
    if (!k_out || kmax < 1) { snprintf(cc_g_err, sizeof(cc_g_err), "cc_smallest_connected_k: bad arguments"); return CC_EINVAL; }
    if (kmax > n - 1) kmax = (int32_t)(n - 1);
    if (kmax > 64) kmax = 64;
    cudaStream_t st = (cudaStream_t)stream;
    int32_t* lab = nullptr;
    cudaError_t e = cc_dev_alloc((void**)&lab, (size_t)n * sizeof(int32_t), st);
    if (e != cudaSuccess) { cudaGetLastError(); snprintf(cc_g_err, sizeof(cc_g_err), "cc_smallest_connected_k: out of device memory"); return CC_ENOMEM; }
    // the symmetrised k-NN graphs are nested in k, so connectivity is monotone: bisection (L150)
    int lo = 1, hi = kmax, best = -1, rc = CC_OK;
    while (lo <= hi && rc == CC_OK) {
        const int mid = (lo + hi) / 2;
        int64_t *rp = nullptr, nnz = 0;
        int32_t* cl = nullptr;
        float* w = nullptr;
        rc = cc_knn_weights(n, p, X, mask, mid, 0.f, 0, &rp, &cl, &w, &nnz, stream);
        int32_t nc = 0;
        if (rc == CC_OK) rc = cc_graph_components(n, rp, cl, lab, &nc, stream);
        cc_free_graph(rp, cl, w);
        if (rc != CC_OK) break;
        if (nc == 1) { best = mid; hi = mid - 1; } else lo = mid + 1;
    }
    cc_dev_free(lab, st);
    if (rc != CC_OK) return rc;
    *k_out = best;   // -1: not connected even at kmax
    return CC_OK;
}


// ---- f2 (part): project U(gamma) on q given directions before any read-back ---------------
// out[i][k] = sum_c (u_ic - xbar_c) P[c][k], xbar = observed column means of X.  One warp per row, fixed reduction order.
namespace {
constexpr int PQMAX = 8;
__global__ void __launch_bounds__(256) k_project(int n, int p, int ld, int q, const float* __restrict__ U,
                                                 const float* __restrict__ xbar, const float* __restrict__ P,
                                                 float* __restrict__ out) {
    const int lane = threadIdx.x & 31;
    const long long nw = (long long)gridDim.x * (blockDim.x >> 5);
    for (long long i = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); i < n; i += nw) {
        float acc[PQMAX];
#pragma unroll
        for (int k = 0; k < PQMAX; ++k) acc[k] = 0.f;
        for (int c = lane; c < p; c += 32) {
            const float v = U[(size_t)i * ld + c] - xbar[c];
#pragma unroll
            for (int k = 0; k < PQMAX; ++k)
                if (k < q) acc[k] = fmaf(v, __ldg(P + (size_t)c * q + k), acc[k]);
        }
#pragma unroll
        for (int k = 0; k < PQMAX; ++k) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) acc[k] += __shfl_xor_sync(0xffffffffu, acc[k], o);
            if (lane == 0 && k < q) out[(size_t)i * q + k] = acc[k];
        }
    }
}
}  // namespace

extern "C" int cc_get_projection(cc_handle* h, int32_t gamma_index, const float* P, int32_t q, float* out,
                                 int32_t out_on_device) {
    if (!h) return CC_EINVAL;
    if (!P || !out || q < 1 || q > PQMAX) {
        snprintf(h->err, sizeof(h->err), "cc_get_projection: need P, out and 1 <= q <= %d", PQMAX);
        return CC_EINVAL;
    }
    if (gamma_index < -1 || gamma_index >= h->nsnap) {
        snprintf(h->err, sizeof(h->err), "cc_get_projection: gamma_index %d outside [-1, %d)", gamma_index, h->nsnap);
        return CC_ESTATE;
    }
    const float* src = gamma_index < 0 ? h->U : h->snapU + (size_t)gamma_index * h->n * h->ld;
    float* dst = out;
    const size_t bytes = (size_t)h->n * q * sizeof(float);
    if (!out_on_device) CC_CUDA(h, cc_dev_alloc((void**)&dst, bytes, h->stream));
    const long long g = (h->n + 7) / 8;
    k_project<<<(unsigned)(g < h->grid_nodes ? g : h->grid_nodes), 256, 0, h->stream>>>((int)h->n, (int)h->p, (int)h->ld, q, src,
                                                                                      h->colmean, P, dst);
    h->launches += 1;
    if (!out_on_device) {
        cudaError_t e = cudaMemcpyAsync(out, dst, bytes, cudaMemcpyDeviceToHost, h->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
        cc_dev_free(dst, h->stream);
        if (e != cudaSuccess) { snprintf(h->err, sizeof(h->err), "cc_get_projection: %s", cudaGetErrorString(e)); return CC_ECUDA; }
    }
    return CC_OK;
}
