// cc_setup.cu -- one-time work of cc_create: input validation (cc_b200.h error codes), the padded
// internal layout, the symmetric-CSR helpers (reverse-entry index, first upper entry, 1/(1+|N_i|)),
// the cold start (S4) and the constants of the default rho rule (S1).  Also the two
// diagnostic sweeps of cc_get_stats.  All arithmetic runs in kernels; the host only reads flags.
#include <cstdio>

#include "cc_device.cuh"
#include "cc_internal.h"

namespace {

enum { F_ROWPTR = 1, F_COLRANGE = 2, F_SELF = 4, F_UNSORTED = 8, F_NOPEER = 16, F_WASYM = 32, F_WBAD = 64,
       F_XBAD = 128, F_DEADCOL = 256 };

__global__ void k_rowptr32(int n, const int64_t* __restrict__ rp64, int* __restrict__ rp32, int* flag) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i > n) return;
    int64_t v = rp64[i];
    if (i == 0 && v != 0) atomicOr(flag, F_ROWPTR);
    if (i < n && rp64[i + 1] < v) atomicOr(flag, F_ROWPTR);
    if (v < 0 || v > 2147483647LL) { atomicOr(flag, F_ROWPTR); v = 0; }
    rp32[i] = (int)v;
}

// One warp per row: checks col / w, finds the reverse entry of every (i,j) by binary search in row j,
// and the first upper entry of the row.
__global__ void k_check_graph(int n, const int* __restrict__ rowptr, const int* __restrict__ col,
                              const float* __restrict__ w, int* __restrict__ peer, int* __restrict__ rowup,
                              float* __restrict__ dinv, int* flag) {
    const int lane = threadIdx.x & 31;
    const long long nw = (long long)gridDim.x * (blockDim.x >> 5);
    for (long long i = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); i < n; i += nw) {
        const int rs = rowptr[i], re = rowptr[i + 1];
        int up = re;
        int bad = 0;
        for (int e = rs + lane; e < re; e += 32) {
            const int j = col[e];
            const float we = w[e];
            if (!(we > 0.f) || isinf(we)) bad |= F_WBAD;
            if (j < 0 || j >= n) { bad |= F_COLRANGE; peer[e] = e; continue; }
            if (j == (int)i) bad |= F_SELF;
            if (e > rs && col[e - 1] >= j) bad |= F_UNSORTED;
            if (j > (int)i) up = min(up, e);
            int lo = rowptr[j], hi = rowptr[j + 1] - 1, f = -1;
            while (lo <= hi) {
                const int mid = (lo + hi) >> 1;
                const int c = col[mid];
                if (c == (int)i) { f = mid; break; }
                if (c < (int)i) lo = mid + 1; else hi = mid - 1;
            }
            if (f < 0) { bad |= F_NOPEER; peer[e] = e; }
            else {
                peer[e] = f;
                if (w[f] != we) bad |= F_WASYM;
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) up = min(up, __shfl_xor_sync(0xffffffffu, up, o));
        if (lane == 0) {
            rowup[i] = up;
            dinv[i] = 1.f / (1.f + (float)(re - rs));
        }
        if (bad) atomicOr(flag, bad);
    }
}


// Processing order for the row-gather kernels: rows sorted by decreasing degree (stable in the row
// index, hence deterministic).  A grid-stride walk over this order hands every row group the same mix
// of heavy and light rows (longest-processing-time-first), which removes the end-of-kernel wait on the
// hub rows of a k-NN graph.  One block: histogram, scan, then a stable scatter chunk by chunk.
#define CC_DEGBINS 4096
__global__ void __launch_bounds__(1024) k_degree_order(int n, const int* __restrict__ rowptr, int* __restrict__ order) {
    __shared__ int cursor[CC_DEGBINS];
    __shared__ int wsum[32];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    for (int b = tid; b < CC_DEGBINS; b += 1024) cursor[b] = 0;
    __syncthreads();
    for (int i = tid; i < n; i += 1024) atomicAdd(&cursor[min(rowptr[i + 1] - rowptr[i], CC_DEGBINS - 1)], 1);
    __syncthreads();
    // exclusive scan over bins taken from the highest degree down: thread t owns bins 4t .. 4t+3 of the reversed axis
    int loc[4], tot = 0;
#pragma unroll
    for (int q = 0; q < 4; ++q) { loc[q] = cursor[CC_DEGBINS - 1 - (tid * 4 + q)]; tot += loc[q]; }
    int inc = tot;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += v; }
    if (lane == 31) wsum[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        int v = wsum[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int u = __shfl_up_sync(0xffffffffu, v, o); if (lane >= o) v += u; }
        wsum[lane] = v;
    }
    __syncthreads();
    int run = inc - tot + (wid ? wsum[wid - 1] : 0);
#pragma unroll
    for (int q = 0; q < 4; ++q) { cursor[CC_DEGBINS - 1 - (tid * 4 + q)] = run; run += loc[q]; }
    __syncthreads();
    // stable scatter: chunks of 1024 rows in index order, warps of a chunk one after the other
    for (int base = 0; base < n; base += 1024) {
        const int i = base + tid;
        const int b = i < n ? min(rowptr[i + 1] - rowptr[i], CC_DEGBINS - 1) : -1 - lane;  // unique dummy keys
        const unsigned same = __match_any_sync(0xffffffffu, b);
        const int rank = __popc(same & ((1u << lane) - 1u));
        for (int w2 = 0; w2 < 32; ++w2) {
            if (wid == w2 && i < n) {
                order[cursor[b] + rank] = i;
            }
            __syncthreads();
            if (wid == w2 && i < n && rank == 0) cursor[b] += __popc(same);
            __syncthreads();
        }
    }
}

// The walk order as a table of row descriptors: (row, first entry with col > row, row end, row begin).  A kernel that
// walks the rows in `order` would need three dependent loads (order -> rowptr/rowup -> col) before its first gather;
// with the table the first two are one 16-byte load that depends on nothing and can be issued an iteration ahead.
__global__ void k_row_desc(int n, const int* __restrict__ order, const int* __restrict__ rowptr, const int* __restrict__ rowup,
                           int4* __restrict__ desc) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n) {
        const int i = order[t];
        desc[t] = make_int4(i, rowup[i], rowptr[i + 1], rowptr[i]);
    }
}

// X (n x p) -> padded n x ld copy; mask likewise (padding = observed zeros); NaN/Inf check on observed.
__global__ void k_pad_copy(long long n, int p, int ld, const float* __restrict__ X, const uint8_t* __restrict__ mask,
                           float* __restrict__ Xo, uint8_t* __restrict__ Mo, int* flag) {
    const long long tot = n * ld;
    const long long nt = (long long)gridDim.x * blockDim.x;
    int bad = 0;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < tot; q += nt) {
        const long long i = q / ld;
        const int c = (int)(q % ld);
        float x = 0.f;
        uint8_t m = 1;
        if (c < p) {
            m = mask ? (mask[i * p + c] ? 1 : 0) : 1;
            x = X[i * p + c];
            if (m && !isfinite(x)) bad = F_XBAD;
            if (!m) x = 0.f;  // values at missing entries are ignored (cc_b200.h)
        }
        Xo[q] = x;
        if (Mo) Mo[q] = m;
    }
    if (bad) atomicOr(flag, bad);
}

// Observed column sums / counts, stage 1: slice s of the rows, one thread per column.
__global__ void k_colsum1(long long n, int ld, int nslice, const float* __restrict__ X, const uint8_t* __restrict__ mask,
                          double* __restrict__ psum, int* __restrict__ pcnt) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    const int sl = blockIdx.y;
    if (c >= ld) return;
    const long long r0 = n * sl / nslice, r1 = n * (sl + 1) / nslice;
    double s = 0.0;
    int cnt = 0;
    for (long long i = r0; i < r1; ++i) {
        const bool m = mask ? mask[i * ld + c] != 0 : true;
        if (m) { s += (double)X[i * ld + c]; ++cnt; }
    }
    psum[(size_t)sl * ld + c] = s;
    pcnt[(size_t)sl * ld + c] = cnt;
}

__global__ void k_colsum2(int p, int ld, int nslice, const double* __restrict__ psum, const int* __restrict__ pcnt,
                          float* __restrict__ colmean, int* flag) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ld) return;
    double s = 0.0;
    long long cnt = 0;
    for (int sl = 0; sl < nslice; ++sl) { s += psum[(size_t)sl * ld + c]; cnt += pcnt[(size_t)sl * ld + c]; }
    if (cnt == 0 && c < p) atomicOr(flag, F_DEADCOL);
    colmean[c] = cnt > 0 ? (float)(s / (double)cnt) : 0.f;
}

// U0 = x where observed, else the observed column mean (S4).
__global__ void k_cold_start(long long n, int ld, const float* __restrict__ X, const uint8_t* __restrict__ mask,
                             const float* __restrict__ colmean, float* __restrict__ U) {
    const long long tot = n * ld;
    const long long nt = (long long)gridDim.x * blockDim.x;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < tot; q += nt) {
        const bool m = mask ? mask[q] != 0 : true;
        U[q] = m ? X[q] : colmean[q % ld];
    }
}

// out[0] = sum_obs (x - ref)^2 with ref = colmean (mode 0) or U (mode 1);  out[1] = sum_{i<j} w^2 (mode 0)
// or sum_{i<j} w_ij * val_ij (mode 1, val = pair norms).
__global__ void __launch_bounds__(CC_THREADS) k_sums(long long n, int ld, long long nnz, int mode,
                                                      const float* __restrict__ X, const uint8_t* __restrict__ mask,
                                                      const float* __restrict__ ref, const int* __restrict__ peer,
                                                      const float* __restrict__ w, const float* __restrict__ val,
                                                      double* part, unsigned int* ticket, double* out) {
    const long long nt = (long long)gridDim.x * blockDim.x;
    double acc[2] = {0.0, 0.0};
    const long long tot = n * ld;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < tot; q += nt) {
        const bool m = mask ? mask[q] != 0 : true;
        if (m) {
            const float t = X[q] - (mode == 0 ? ref[q % ld] : ref[q]);
            acc[0] += (double)t * (double)t;
        }
    }
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < nnz; e += nt) {
        if (peer[e] > e) {  // each undirected pair once
            const double we = (double)w[e];
            acc[1] += mode == 0 ? we * we : we * (double)val[e];
        }
    }
    double tot2[2];
    if (grid_reduce<2>(acc, part, ticket, tot2)) { out[0] = tot2[0]; out[1] = tot2[1]; }
}

// min over entries of | ||b|| - thr | / thr  (how close a pair was to switching between fused and not).
__global__ void __launch_bounds__(CC_THREADS) k_margin(long long nnz, int nchunk, const float* __restrict__ nb2,
                                                        const float* __restrict__ w, const cc_scal* sc, double* part,
                                                        unsigned int* ticket, double* out) {
    const long long nt = (long long)gridDim.x * blockDim.x;
    const float cthr = sc->cthr;
    float mn = 3.0e38f;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < nnz; e += nt) {
        float q = nb2[e];
        for (int c = 1; c < nchunk; ++c) q += nb2[(size_t)c * nnz + e];
        const float thr = cthr * w[e];
        if (thr > 0.f) mn = fminf(mn, fabsf(sqrtf(q) - thr) / thr);
    }
    // min-reduce through the sum machinery: exact, order-independent
    __shared__ float smn[CC_THREADS];
    smn[threadIdx.x] = mn;
    __syncthreads();
    for (int o = CC_THREADS / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) smn[threadIdx.x] = fminf(smn[threadIdx.x], smn[threadIdx.x + o]);
        __syncthreads();
    }
    __shared__ bool last;
    if (threadIdx.x == 0) {
        part[blockIdx.x] = (double)smn[0];
        __threadfence();
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (last && threadIdx.x == 0) {
        __threadfence();
        double m2 = 3.0e38;
        for (unsigned b = 0; b < gridDim.x; ++b) m2 = fmin(m2, __ldcg(&part[b]));
        out[0] = m2;
        *ticket = 0u;
    }
}

}  // namespace

// =============================================================================================
// Host side
// =============================================================================================
template <typename T>
static int dmalloc(cc_handle* h, T** p, size_t count) {
    *p = nullptr;
    if (count == 0) count = 1;
    cudaError_t e = cc_dev_alloc((void**)p, count * sizeof(T), h->stream);
    if (e != cudaSuccess) {
        cudaGetLastError();
        snprintf(h->err, sizeof(h->err), "cudaMalloc of %zu bytes failed: %s", count * sizeof(T), cudaGetErrorString(e));
        return CC_ENOMEM;
    }
    return CC_OK;
}
#define CC_TRY(x) do { int rc_ = (x); if (rc_ != CC_OK) return rc_; } while (0)

static int read_flag(cc_handle* h, int* out) {
    CC_CUDA(h, cudaMemcpyAsync(out, h->dflag, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    CC_CUDA(h, cudaStreamSynchronize(h->stream));
    return CC_OK;
}

static int flag_to_error(cc_handle* h, int f) {
    if (!f) return CC_OK;
    if (f & F_XBAD) { snprintf(h->err, sizeof(h->err), "X has a NaN or Inf at an observed entry"); return CC_EINVAL; }
    if (f & F_WBAD) { snprintf(h->err, sizeof(h->err), "a weight is <= 0, NaN or Inf"); return CC_EGRAPH; }
    if (f & F_DEADCOL) { snprintf(h->err, sizeof(h->err), "a column has no observed entry"); return CC_EMASK; }
    const char* what = (f & F_ROWPTR) ? "rowptr is not a non-decreasing int32-range prefix sum starting at 0"
                     : (f & F_COLRANGE) ? "a column index is out of range"
                     : (f & F_SELF) ? "self loop"
                     : (f & F_UNSORTED) ? "column indices of a row are not strictly increasing"
                     : (f & F_NOPEER) ? "the CSR is not symmetric (an entry has no reverse entry)"
                     : "w_ij != w_ji";
    snprintf(h->err, sizeof(h->err), "bad graph: %s", what);
    return CC_EGRAPH;
}

int ccu_validate_and_build(cc_handle* h, const float* X, const uint8_t* mask, const int64_t* rowptr,
                           const int32_t* col, const float* w) {
    const int64_t n = h->n, p = h->p;
    h->ld = (p + 3) / 4 * 4;
    int G = 2;
    while (G < 32 && (int64_t)G * 4 < h->ld) G *= 2;
    h->G = G;
    h->nchunk = (int)((h->ld + 4 * G - 1) / (4 * G));
    int dev = 0;
    CC_CUDA(h, cudaGetDevice(&dev));
    CC_CUDA(h, cudaDeviceGetAttribute(&h->sms, cudaDevAttrMultiProcessorCount, dev));
    const int64_t items = n * h->nchunk, gpb = CC_THREADS / G;
    int64_t grid = (items + gpb - 1) / gpb;
    const int64_t cap = (int64_t)h->sms * 8 < CC_MAXBLK ? (int64_t)h->sms * 8 : CC_MAXBLK;
    if (grid > cap) grid = cap;
    if (grid < 1) grid = 1;
    h->grid_rows = (int)grid;
    h->grid_nodes = (int)cap;
    cudaStream_t st = h->stream;

    CC_TRY(dmalloc(h, &h->dflag, 1));
    CC_TRY(dmalloc(h, &h->dout, 4));
    CC_TRY(dmalloc(h, &h->sc, 1));
    CC_TRY(dmalloc(h, &h->part, (size_t)8 * CC_MAXBLK * CC_NPART));
    CC_CUDA(h, cudaMallocHost((void**)&h->sc_host, sizeof(cc_scal)));
    CC_CUDA(h, cudaMemsetAsync(h->dflag, 0, sizeof(int), st));
    CC_CUDA(h, cudaMemsetAsync(h->sc, 0, sizeof(cc_scal), st));

    // ---- graph ----
    CC_TRY(dmalloc(h, &h->rowptr, (size_t)n + 1));
    if (h->dense) {
        if (n < 2) { snprintf(h->err, sizeof(h->err), "dense mode needs n >= 2"); return CC_EINVAL; }
        CC_TRY(ccd_setup(h, w));
        CC_TRY(dmalloc(h, &h->col, 1));
        CC_TRY(dmalloc(h, &h->w, 1));
        CC_CUDA(h, cudaMemsetAsync(h->rowptr, 0, (size_t)(n + 1) * sizeof(int), st));
    } else {
        k_rowptr32<<<(int)((n + 256) / 256), 256, 0, st>>>((int)n, rowptr, h->rowptr, h->dflag);
        int64_t nnz64 = 0;
        CC_CUDA(h, cudaMemcpyAsync(&nnz64, rowptr + n, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
        int f = 0;
        CC_TRY(read_flag(h, &f));
        if (f || nnz64 < 0 || nnz64 > 2147483647LL) return flag_to_error(h, f | F_ROWPTR);
        h->nnz = nnz64;
        if (nnz64 > 0 && (!col || !w)) { snprintf(h->err, sizeof(h->err), "col or w is NULL but rowptr[n] > 0"); return CC_EINVAL; }
        CC_TRY(dmalloc(h, &h->col, (size_t)h->nnz));
        CC_TRY(dmalloc(h, &h->w, (size_t)h->nnz));
        if (h->nnz > 0) {
            CC_CUDA(h, cudaMemcpyAsync(h->col, col, (size_t)h->nnz * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
            CC_CUDA(h, cudaMemcpyAsync(h->w, w, (size_t)h->nnz * sizeof(float), cudaMemcpyDeviceToDevice, st));
        }
    }
    h->npairs = h->nnz / 2;
    const int64_t nnz_csr = h->dense ? 0 : h->nnz;   // the CSR arrays are empty in dense mode
    CC_TRY(dmalloc(h, &h->peer, (size_t)nnz_csr));
    CC_TRY(dmalloc(h, &h->rowup, (size_t)n));
    CC_TRY(dmalloc(h, &h->dinv, (size_t)n));
    {
        int64_t g2 = (n + 7) / 8;
        if (g2 > cap) g2 = cap;
        k_check_graph<<<(int)g2, 256, 0, st>>>((int)n, h->rowptr, h->col, h->w, h->peer, h->rowup, h->dinv, h->dflag);
    }
    CC_TRY(dmalloc(h, &h->order, (size_t)n));
    k_degree_order<<<1, 1024, 0, st>>>((int)n, h->rowptr, h->order);
    CC_TRY(dmalloc(h, &h->rowdesc, (size_t)n));
    k_row_desc<<<(int)((n + 255) / 256), 256, 0, st>>>((int)n, h->order, h->rowptr, h->rowup, h->rowdesc);
    // ---- data ----
    const size_t nl = (size_t)n * h->ld;
    CC_TRY(dmalloc(h, &h->X, nl));
    if (mask) CC_TRY(dmalloc(h, &h->mask, nl));
    k_pad_copy<<<(int)cap, 256, 0, st>>>(n, (int)p, (int)h->ld, X, mask, h->X, h->mask, h->dflag);
    CC_TRY(dmalloc(h, &h->colmean, (size_t)h->ld));
    {
        const int nslice = n >= 4096 ? 64 : (n >= 64 ? 8 : 1);
        double* psum = nullptr;
        int* pcnt = nullptr;
        CC_TRY(dmalloc(h, &psum, (size_t)nslice * h->ld));
        CC_TRY(dmalloc(h, &pcnt, (size_t)nslice * h->ld));
        dim3 g1((unsigned)((h->ld + 127) / 128), (unsigned)nslice);
        k_colsum1<<<g1, 128, 0, st>>>(n, (int)h->ld, nslice, h->X, h->mask, psum, pcnt);
        k_colsum2<<<(unsigned)((h->ld + 127) / 128), 128, 0, st>>>((int)p, (int)h->ld, nslice, psum, pcnt, h->colmean, h->dflag);
        CC_CUDA(h, cudaStreamSynchronize(st));
        cc_dev_free(psum, st);
        cc_dev_free(pcnt, st);
    }
    int f = 0;
    CC_TRY(read_flag(h, &f));
    if (f) return flag_to_error(h, f);
    // constants of the rho rule (S1): sum_obs (x - colmean)^2 and sum_E w^2
    k_sums<<<(int)cap, CC_THREADS, 0, st>>>(n, (int)h->ld, (long long)nnz_csr, 0, h->X, h->mask, h->colmean, h->peer,
                                           h->w, nullptr, h->part + 4 * CC_MAXBLK * CC_NPART, &h->sc->ticket[4], h->dout);
    if (h->dense) ccd_sumw2(h);
    double two[2];
    CC_CUDA(h, cudaMemcpyAsync(two, h->dout, sizeof(two), cudaMemcpyDeviceToHost, st));
    CC_CUDA(h, cudaStreamSynchronize(st));
    h->xss = two[0];
    h->sumw2 = two[1];

    // ---- state ----
    float** node_arrays[] = {&h->U, &h->A, &h->Ap, &h->Z, &h->Pv, &h->Sv, &h->Uc, &h->Dl};
    for (float** a : node_arrays) {
        CC_TRY(dmalloc(h, a, nl));
        CC_CUDA(h, cudaMemsetAsync(*a, 0, nl * sizeof(float), st));
    }
    if (h->dense && h->dn_small_tc) CC_TRY(ccd_small_tc_maps(h));     // the TMA tensor maps of U, A', X, A
    CC_TRY(dmalloc(h, &h->s, (size_t)nnz_csr));
    CC_TRY(dmalloc(h, &h->vn, (size_t)nnz_csr));
    CC_TRY(dmalloc(h, &h->tmpE, (size_t)nnz_csr));
    CC_TRY(dmalloc(h, &h->nb2, (size_t)nnz_csr * h->nchunk + 1));
    CC_CUDA(h, cudaMemsetAsync(h->nb2, 0, ((size_t)nnz_csr * h->nchunk + 1) * sizeof(float), st));
    const int hc = h->prm.hist_cap > 0 ? h->prm.hist_cap : 1;
    CC_TRY(dmalloc(h, &h->hist_phi, (size_t)hc));
    CC_TRY(dmalloc(h, &h->hist_d, (size_t)hc));
    CC_TRY(dmalloc(h, &h->lab, (size_t)n));
    CC_TRY(dmalloc(h, &h->lab_flag, 1));
    h->launches += 7;
    CC_TRY(ccs_setup_inverse(h));
    CC_TRY(ccp_setup(h));
    return ccu_cold_start(h);
}

int ccu_cold_start(cc_handle* h) {
    k_cold_start<<<h->grid_nodes, 256, 0, h->stream>>>(h->n, (int)h->ld, h->X, h->mask, h->colmean, h->U);
    if (h->dense) {
        ccd_init_state(h);
        CC_CUDA(h, cudaMemcpyAsync(h->sc_host, h->sc, sizeof(cc_scal), cudaMemcpyDeviceToHost, h->stream));   // pen_next
        CC_CUDA(h, cudaStreamSynchronize(h->stream));
    } else {
        ccs_init_state(h);
    }
    h->launches += 1;
    CC_CUDA(h, cudaGetLastError());
    return CC_OK;
}

int ccu_fgamma(cc_handle* h, double* f_out) {
    ccs_pair_norms(h, h->U, h->tmpE, nullptr);
    k_sums<<<h->grid_nodes, CC_THREADS, 0, h->stream>>>(h->n, (int)h->ld, (long long)h->nnz, 1, h->X, h->mask, h->U, h->peer,
                                                       h->w, h->tmpE, h->part + 4 * CC_MAXBLK * CC_NPART,
                                                       &h->sc->ticket[4], h->dout);
    double two[2];
    CC_CUDA(h, cudaMemcpyAsync(two, h->dout, sizeof(two), cudaMemcpyDeviceToHost, h->stream));
    CC_CUDA(h, cudaStreamSynchronize(h->stream));
    h->launches += 2;
    *f_out = 0.5 * two[0] + h->sc_host->gamma * two[1];
    return CC_OK;
}

int ccu_min_margin(cc_handle* h, double* margin_out) {
    k_margin<<<h->grid_nodes, CC_THREADS, 0, h->stream>>>((long long)h->nnz, h->nchunk, h->nb2, h->w, h->sc,
                                                         h->part + 5 * CC_MAXBLK * CC_NPART, &h->sc->ticket[5], h->dout + 2);
    CC_CUDA(h, cudaMemcpyAsync(margin_out, h->dout + 2, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CC_CUDA(h, cudaStreamSynchronize(h->stream));
    h->launches += 1;
    return CC_OK;
}

void ccu_free(cc_handle* h) {
    void* ptrs[] = {h->X, h->U, h->A, h->Ap, h->Z, h->R, h->Pv, h->Sv, h->Dl, h->Uc, h->mask, h->colmean, h->rowptr,
                    h->rowup, h->col, h->peer, h->w, h->s, h->vn, h->nb2, h->tmpE, h->dinv, h->Minv, h->Wd, h->Sd, h->VNd, h->NB2d, h->ubar, h->abar, h->dbar, h->colps, h->pre_pairs, h->nrm_part, h->pre_B, h->Rd, h->sc, h->part,
                    h->hist_phi, h->hist_d, h->dout, h->dflag, h->pt_nbpart, h->pt_spart, h->snapU, h->snapLab, h->lab, h->lab_flag, h->lab_rank, h->order, h->rowdesc};
    for (void* q : ptrs)
        cc_dev_free(q, h->stream);
    if (h->sc_host) cudaFreeHost(h->sc_host);
    if (h->gexec) cudaGraphExecDestroy(h->gexec);
    if (h->graph) cudaGraphDestroy(h->graph);
    free(h->snapK);
}
