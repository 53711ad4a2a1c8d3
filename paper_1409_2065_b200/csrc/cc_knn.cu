// cc_knn.cu -- a0, the one-time weight build of PAPER.md L127-L133 (eq. 8):
//     w_ij = 1{i ~_k j} exp(-phi ||x_i - x_j||^2),  i ~_k j iff j is among i's k nearest OR vice versa.
// Readings: S9 self excluded, ties to the smaller index; S11 with a mask the squared
// distance runs over co-observed coordinates and is scaled by p / #co-observed; S8 normalisation over
// pairs i<j is optional.
//
// f4 (eq. 9): with side coordinates Y (q <= 4 columns, e.g. GPS) the distance is the composite
//     d_ij = alpha ||x_i - x_j|| + (1 - alpha) ||y_i - y_j||,   y-differences wrapped modulo a per-coordinate period (S27),
//     or ||y_i - y_j|| replaced by the great-circle distance of (longitude, latitude) pairs (L137's alternative, S28),
// and eq. 8 is applied to this d (kernels instantiated with SIDE = true).
//
// Three steps, all on the device, no sort library and no floating-point atomics:
//   1. k_knn_tile: brute-force distances in 64 x 64 register tiles (direct differences, fp32), a sorted
//      k-list per query in shared memory, filtered insertion (a candidate is looked at only if it beats
//      the current k-th distance).  The n x n distance matrix never exists.
//   2. symmetrise by OR: count reverse-only entries (integer atomics), scan, fill, sort each row by column.
//   3. weights from recomputed distances (so w_ij == w_ji bitwise), optional normalisation.
#include <cfloat>
#include <cmath>
#include <cstdio>

#include "cc_device.cuh"
#include "cc_internal.h"

namespace {

constexpr int TQ = 64, TC = 64, PC = 16, KMAX = 64, QSIDE = 4;

struct side_t {
    const float* Y;   // n x q row-major, or NULL
    int q;
    float period[QSIDE];   // 0: plain difference
    float alpha;
    float radius;          // > 0: Y = (longitude, latitude) in degrees, side distance = great circle on this sphere (S28)
};

// ||y_i - y_j|| with modulo differences (L137, S27), or the geodesic alternative of L137 (S28): the great-circle
// distance radius * theta, hav(theta) = sin^2(dlat/2) + cos(lat_i) cos(lat_j) sin^2(dlon/2), theta =
// 2 atan2(sqrt(hav), sqrt(1 - hav)).  The half differences are formed in degrees first (exact for nearby points).
__device__ __forceinline__ float side_dist(const side_t& sd, int i, int j) {
    if (sd.radius > 0.f) {
        constexpr float RAD = 0.017453292519943295f;
        const float2 yi = *reinterpret_cast<const float2*>(sd.Y + (size_t)i * 2), yj = *reinterpret_cast<const float2*>(sd.Y + (size_t)j * 2);
        const float so = sinf(0.5f * RAD * (yi.x - yj.x)), sl = sinf(0.5f * RAD * (yi.y - yj.y));
        const float hav = fminf(fmaf(cosf(RAD * yi.y) * cosf(RAD * yj.y), so * so, sl * sl), 1.f);
        return sd.radius * 2.f * atan2f(sqrtf(hav), sqrtf(1.f - hav));
    }
    float s = 0.f;
    for (int c = 0; c < sd.q; ++c) {
        float df = sd.Y[(size_t)i * sd.q + c] - sd.Y[(size_t)j * sd.q + c];
        if (sd.period[c] > 0.f) df -= sd.period[c] * rintf(df / sd.period[c]);
        s = fmaf(df, df, s);
    }
    return sqrtf(s);
}

template <bool MASKED, bool SIDE>
__global__ void __launch_bounds__(256) k_knn_tile(int n, int p, int k, const float* __restrict__ X,
                                                   const uint8_t* __restrict__ mask, const side_t sd, int* __restrict__ nbr) {
    extern __shared__ float smem[];
    float* Xq = smem;                        // TQ x (PC+1)
    float* Xc = Xq + TQ * (PC + 1);          // TC x (PC+1)
    float* Mq = Xc + TC * (PC + 1);          // masks as 0/1 floats (MASKED only)
    float* Mc = Mq + (MASKED ? TQ * (PC + 1) : 0);
    float* Dt = Mc + (MASKED ? TC * (PC + 1) : 0);   // TQ x (TC+1)
    float* Ld = Dt + TQ * (TC + 1);          // TQ x k  list distances (ascending)
    int* Li = reinterpret_cast<int*>(Ld + TQ * k);   // TQ x k  list indices

    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    const int q0 = blockIdx.x * TQ;
    for (int t = tid; t < TQ * k; t += 256) { Ld[t] = FLT_MAX; Li[t] = -1; }
    __syncthreads();

    for (int c0 = 0; c0 < n; c0 += TC) {
        float acc[4][4], cnt[4][4];
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) { acc[a][b] = 0.f; cnt[a][b] = 0.f; }
        for (int pc = 0; pc < p; pc += PC) {
            // stage PC columns of the query tile and of the candidate tile
            for (int t = tid; t < TQ * PC; t += 256) {
                const int r = t / PC, c = t % PC;
                const int gi = q0 + r, gj = c0 + r, gc = pc + c;
                const bool vi = gi < n && gc < p, vj = gj < n && gc < p;
                Xq[r * (PC + 1) + c] = vi ? X[(size_t)gi * p + gc] : 0.f;
                Xc[r * (PC + 1) + c] = vj ? X[(size_t)gj * p + gc] : 0.f;
                if (MASKED) {
                    Mq[r * (PC + 1) + c] = vi && mask[(size_t)gi * p + gc] ? 1.f : 0.f;
                    Mc[r * (PC + 1) + c] = vj && mask[(size_t)gj * p + gc] ? 1.f : 0.f;
                }
            }
            __syncthreads();
#pragma unroll
            for (int c = 0; c < PC; ++c) {
                float xq[4], xc[4], mq[4], mc[4];
#pragma unroll
                for (int a = 0; a < 4; ++a) {
                    xq[a] = Xq[(ty * 4 + a) * (PC + 1) + c];
                    xc[a] = Xc[(tx + 16 * a) * (PC + 1) + c];
                    if (MASKED) { mq[a] = Mq[(ty * 4 + a) * (PC + 1) + c]; mc[a] = Mc[(tx + 16 * a) * (PC + 1) + c]; }
                }
#pragma unroll
                for (int a = 0; a < 4; ++a)
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        const float df = xq[a] - xc[b];
                        if (MASKED) {
                            const float m = mq[a] * mc[b];
                            acc[a][b] = fmaf(m * df, df, acc[a][b]);
                            cnt[a][b] += m;
                        } else {
                            acc[a][b] = fmaf(df, df, acc[a][b]);
                        }
                    }
            }
            __syncthreads();
        }
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                float d = acc[a][b];
                if (MASKED) d = cnt[a][b] > 0.f ? d * (float)p / cnt[a][b] : FLT_MAX;
                if (SIDE) {
                    const int gi = q0 + ty * 4 + a, gj = c0 + tx + 16 * b;
                    if (gi < n && gj < n && d < FLT_MAX) d = sd.alpha * sqrtf(d) + (1.f - sd.alpha) * side_dist(sd, gi, gj);
                }
                Dt[(ty * 4 + a) * (TC + 1) + tx + 16 * b] = d;
            }
        __syncthreads();
        // selection: warp wq handles queries wq*8 .. wq*8+7; lanes look at candidates lane, lane+32
        const int lane = tid & 31, wq = tid >> 5;
        for (int qq = 0; qq < 8; ++qq) {
            const int q = wq * 8 + qq, gi = q0 + q;
            if (gi >= n) break;
            float* ld = Ld + q * k;
            int* li = Li + q * k;
            for (int half = 0; half < 2; ++half) {
                const int cj = lane + 32 * half, gj = c0 + cj;
                const float d = Dt[q * (TC + 1) + cj];
                const float kth = ld[k - 1];
                unsigned bal = __ballot_sync(0xffffffffu, gj < n && gj != gi && d < kth);
                while (bal) {   // ascending candidate index: equal distances keep the smaller index ahead
                    const int src = __ffs(bal) - 1;
                    bal &= bal - 1;
                    const float dc = __shfl_sync(0xffffffffu, d, src);
                    if (lane == 0 && dc < ld[k - 1]) {
                        int pos = k - 1;
                        while (pos > 0 && dc < ld[pos - 1]) { ld[pos] = ld[pos - 1]; li[pos] = li[pos - 1]; --pos; }
                        ld[pos] = dc;
                        li[pos] = c0 + 32 * half + src;
                    }
                    __syncwarp();
                }
            }
        }
        __syncthreads();
    }
    for (int t = tid; t < TQ * k; t += 256) {
        const int gi = q0 + t / k;
        if (gi < n) nbr[(size_t)gi * k + t % k] = Li[t];
    }
}

// sort each k-list by neighbour index (needed for the membership tests and the CSR fill)
__global__ void k_sort_lists(int n, int k, int* __restrict__ nbr) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int* a = nbr + (size_t)i * k;
    for (int x = 1; x < k; ++x) {
        const int v = a[x];
        int y = x;
        while (y > 0 && a[y - 1] > v) { a[y] = a[y - 1]; --y; }
        a[y] = v;
    }
}

__device__ __forceinline__ bool in_list(const int* a, int k, int v) {
    int lo = 0, hi = k - 1;
    while (lo <= hi) {
        const int mid = (lo + hi) >> 1;
        if (a[mid] == v) return true;
        if (a[mid] < v) lo = mid + 1; else hi = mid - 1;
    }
    return false;
}

// i ~ j "or vice versa": j gets a reverse-only entry when i lists j but j does not list i
__global__ void k_count_reverse(int n, int k, const int* __restrict__ nbr, int* __restrict__ extra) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)n * k) return;
    const int i = (int)(t / k), j = nbr[t];
    if (j >= 0 && !in_list(nbr + (size_t)j * k, k, i)) atomicAdd(&extra[j], 1);
}

// exclusive scan of (k_i + extra_i) -> rowptr (int64).  One block; n is at most ~1e6.
__global__ void k_scan_rows(int n, int k, const int* __restrict__ nbr, const int* __restrict__ extra,
                            int64_t* __restrict__ rowptr) {
    __shared__ long long sm[1024];
    __shared__ long long carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < n; base += 1024) {
        const int i = base + threadIdx.x;
        long long v = 0;
        if (i < n) {
            int own = 0;
            for (int q = 0; q < k; ++q) own += nbr[(size_t)i * k + q] >= 0 ? 1 : 0;
            v = own + extra[i];
        }
        sm[threadIdx.x] = v;
        __syncthreads();
        for (int o = 1; o < 1024; o <<= 1) {
            const long long u = threadIdx.x >= o ? sm[threadIdx.x - o] : 0;
            __syncthreads();
            sm[threadIdx.x] += u;
            __syncthreads();
        }
        if (i < n) rowptr[i] = carry + sm[threadIdx.x] - v;
        __syncthreads();
        if (threadIdx.x == 0) carry += sm[1023];
        __syncthreads();
    }
    if (threadIdx.x == 0) rowptr[n] = carry;
}

__global__ void k_fill_rows(int n, int k, const int* __restrict__ nbr, const int64_t* __restrict__ rowptr,
                            int* __restrict__ cursor, int* __restrict__ col) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)n * k) return;
    const int i = (int)(t / k), q = (int)(t % k), j = nbr[t];
    if (j < 0) return;
    col[rowptr[i] + q] = j;   // own list occupies the first slots of the row (k valid entries when n > k)
    if (!in_list(nbr + (size_t)j * k, k, i)) {
        const int slot = atomicAdd(&cursor[j], 1);
        int own = 0;
        for (int r = 0; r < k; ++r) own += nbr[(size_t)j * k + r] >= 0 ? 1 : 0;
        col[rowptr[j] + own + slot] = i;
    }
}

// sort each row by column (the set is unique, so the result does not depend on the fill order) and
// compute the weight of every entry from the ordered pair (min, max) so that w_ij == w_ji bitwise.
template <bool MASKED, bool SIDE>
__global__ void k_rows_finish(int n, int p, float phi, const float* __restrict__ X, const uint8_t* __restrict__ mask,
                              const side_t sd, const int64_t* __restrict__ rowptr, int* __restrict__ col, float* __restrict__ w) {
    const int lane = threadIdx.x & 31;
    const long long nw = (long long)gridDim.x * (blockDim.x >> 5);
    for (long long i = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); i < n; i += nw) {
        const long long rs = rowptr[i], re = rowptr[i + 1];
        if (lane == 0) {
            for (long long x = rs + 1; x < re; ++x) {
                const int v = col[x];
                long long y = x;
                while (y > rs && col[y - 1] > v) { col[y] = col[y - 1]; --y; }
                col[y] = v;
            }
        }
        __syncwarp();
        for (long long e = rs; e < re; ++e) {
            const int j = col[e];
            const int lo = min((int)i, j), hi = max((int)i, j);
            float s = 0.f, c = 0.f;
            for (int q = lane; q < p; q += 32) {
                const float df = X[(size_t)lo * p + q] - X[(size_t)hi * p + q];
                if (MASKED) {
                    const float m = (mask[(size_t)lo * p + q] && mask[(size_t)hi * p + q]) ? 1.f : 0.f;
                    s = fmaf(m * df, df, s);
                    c += m;
                } else {
                    s = fmaf(df, df, s);
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) { s += __shfl_xor_sync(0xffffffffu, s, o); c += __shfl_xor_sync(0xffffffffu, c, o); }
            if (MASKED) s = c > 0.f ? s * (float)p / c : FLT_MAX;
            if (SIDE && s < FLT_MAX) {   // eq. 9, then eq. 8 on d^2
                const float d = sd.alpha * sqrtf(s) + (1.f - sd.alpha) * side_dist(sd, lo, hi);
                s = d * d;
            }
            if (lane == 0) w[e] = expf(-phi * s);
        }
    }
}

// sum of w over entries with col > row (each pair once), deterministic
__global__ void __launch_bounds__(CC_THREADS) k_wsum(int n, const int64_t* __restrict__ rowptr, const int* __restrict__ col,
                                                      const float* __restrict__ w, double* part, unsigned int* ticket,
                                                      double* out) {
    double acc[1] = {0.0};
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x)
        for (long long e = rowptr[i]; e < rowptr[i + 1]; ++e)
            if (col[e] > i) acc[0] += (double)w[e];
    double tot[1];
    if (grid_reduce<1>(acc, part, ticket, tot)) out[0] = tot[0];
}

__global__ void k_wscale(long long nnz, float* __restrict__ w, const double* __restrict__ total) {
    const double t = total[0];
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < nnz; e += (long long)gridDim.x * blockDim.x)
        w[e] = (float)((double)w[e] / t);
}

}  // namespace

#define g_knn_err cc_g_err

#define KCUDA(call)                                                                          \
    do {                                                                                     \
        cudaError_t e_ = (call);                                                             \
        if (e_ != cudaSuccess) {                                                             \
            snprintf(g_knn_err, sizeof(g_knn_err), "%s: %s", #call, cudaGetErrorString(e_)); \
            rc = e_ == cudaErrorMemoryAllocation ? CC_ENOMEM : CC_ECUDA;                     \
            goto done;                                                                       \
        }                                                                                    \
    } while (0)

static int knn_impl(int64_t n, int64_t p, const float* X, const uint8_t* mask, const side_t sd, int32_t k, float phi,
                    int32_t normalize, int64_t** rowptr_out, int32_t** col_out, float** w_out, int64_t* nnz_out, void* stream) {
    if (!X || !rowptr_out || !col_out || !w_out || !nnz_out || n < 2 || p < 1 || k < 1 || k > n - 1 || k > KMAX ||
        n > 1000000000LL || !(phi >= 0.f)) {
        snprintf(g_knn_err, sizeof(g_knn_err), "cc_knn_weights: need n >= 2, p >= 1, 1 <= k <= min(n-1, %d), phi >= 0", KMAX);
        return CC_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    int rc = CC_OK;
    int *nbr = nullptr, *extra = nullptr, *cursor = nullptr, *col = nullptr;
    int64_t* rowptr = nullptr;
    float* w = nullptr;
    double* red = nullptr;   // [0] total, then partials, then ticket
    int64_t nnz = 0;
    const long long nk = (long long)n * k;
    const size_t smem = (size_t)((mask ? 4 : 2) * TQ * (PC + 1) + TQ * (TC + 1) + 2 * TQ * k) * sizeof(float);
    *rowptr_out = nullptr; *col_out = nullptr; *w_out = nullptr; *nnz_out = 0;
    KCUDA(cudaMalloc((void**)&nbr, (size_t)nk * sizeof(int)));
    KCUDA(cudaMalloc((void**)&extra, (size_t)n * sizeof(int)));
    KCUDA(cudaMalloc((void**)&cursor, (size_t)n * sizeof(int)));
    KCUDA(cudaMalloc((void**)&rowptr, (size_t)(n + 1) * sizeof(int64_t)));
    KCUDA(cudaMalloc((void**)&red, (size_t)(2 + CC_MAXBLK) * sizeof(double)));
    KCUDA(cudaMemsetAsync(extra, 0, (size_t)n * sizeof(int), st));
    KCUDA(cudaMemsetAsync(cursor, 0, (size_t)n * sizeof(int), st));
    KCUDA(cudaMemsetAsync(red, 0, (size_t)(2 + CC_MAXBLK) * sizeof(double), st));
    {
        const unsigned g = (unsigned)((n + TQ - 1) / TQ);
#define KNN_TILE(M, S)                                                                                               \
    do {                                                                                                             \
        KCUDA(cudaFuncSetAttribute(k_knn_tile<M, S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));       \
        k_knn_tile<M, S><<<g, 256, smem, st>>>((int)n, (int)p, k, X, mask, sd, nbr);                                 \
    } while (0)
        if (mask && sd.Y) KNN_TILE(true, true);
        else if (mask) KNN_TILE(true, false);
        else if (sd.Y) KNN_TILE(false, true);
        else KNN_TILE(false, false);
#undef KNN_TILE
    }
    k_sort_lists<<<(unsigned)((n + 255) / 256), 256, 0, st>>>((int)n, k, nbr);
    k_count_reverse<<<(unsigned)((nk + 255) / 256), 256, 0, st>>>((int)n, k, nbr, extra);
    k_scan_rows<<<1, 1024, 0, st>>>((int)n, k, nbr, extra, rowptr);
    KCUDA(cudaMemcpyAsync(&nnz, rowptr + n, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    KCUDA(cudaStreamSynchronize(st));
    KCUDA(cudaMalloc((void**)&col, (size_t)(nnz ? nnz : 1) * sizeof(int)));
    KCUDA(cudaMalloc((void**)&w, (size_t)(nnz ? nnz : 1) * sizeof(float)));
    k_fill_rows<<<(unsigned)((nk + 255) / 256), 256, 0, st>>>((int)n, k, nbr, rowptr, cursor, col);
    {
        const unsigned g = (unsigned)((n + 7) / 8 < 148 * 16 ? (n + 7) / 8 : 148 * 16);
        if (mask && sd.Y) k_rows_finish<true, true><<<g, 256, 0, st>>>((int)n, (int)p, phi, X, mask, sd, rowptr, col, w);
        else if (mask) k_rows_finish<true, false><<<g, 256, 0, st>>>((int)n, (int)p, phi, X, mask, sd, rowptr, col, w);
        else if (sd.Y) k_rows_finish<false, true><<<g, 256, 0, st>>>((int)n, (int)p, phi, X, mask, sd, rowptr, col, w);
        else k_rows_finish<false, false><<<g, 256, 0, st>>>((int)n, (int)p, phi, X, mask, sd, rowptr, col, w);
    }
    if (normalize) {
        k_wsum<<<1024, CC_THREADS, 0, st>>>((int)n, rowptr, col, w, red + 2, reinterpret_cast<unsigned int*>(red + 1), red);
        k_wscale<<<1024, 256, 0, st>>>((long long)nnz, w, red);
    }
    KCUDA(cudaStreamSynchronize(st));
    KCUDA(cudaGetLastError());
    *rowptr_out = rowptr; *col_out = col; *w_out = w; *nnz_out = nnz;
    rowptr = nullptr; col = nullptr; w = nullptr;
done:
    cudaFree(nbr); cudaFree(extra); cudaFree(cursor); cudaFree(red);
    if (rowptr) cudaFree(rowptr);
    if (col) cudaFree(col);
    if (w) cudaFree(w);
    return rc;
}

extern "C" {

int cc_knn_weights(int64_t n, int64_t p, const float* X, const uint8_t* mask, int32_t k, float phi, int32_t normalize,
                   int64_t** rowptr_out, int32_t** col_out, float** w_out, int64_t* nnz_out, void* stream) {
    side_t sd = {};
    return knn_impl(n, p, X, mask, sd, k, phi, normalize, rowptr_out, col_out, w_out, nnz_out, stream);
}

int cc_knn_weights_composite(int64_t n, int64_t p, const float* X, const uint8_t* mask, int32_t q, const float* Y,
                             const float* period, float alpha, int32_t k, float phi, int32_t normalize,
                             int64_t** rowptr_out, int32_t** col_out, float** w_out, int64_t* nnz_out, void* stream) {
    if (!Y || q < 1 || q > QSIDE || !(alpha >= 0.f && alpha <= 1.f)) {
        snprintf(g_knn_err, sizeof(g_knn_err), "cc_knn_weights_composite: need Y, 1 <= q <= %d, 0 <= alpha <= 1", QSIDE);
        return CC_EINVAL;
    }
    side_t sd = {};
    sd.Y = Y;
    sd.q = q;
    sd.alpha = alpha;
    for (int c = 0; c < q; ++c) {
        sd.period[c] = period ? period[c] : 0.f;
        if (!(sd.period[c] >= 0.f) || std::isinf(sd.period[c])) {
            snprintf(g_knn_err, sizeof(g_knn_err), "cc_knn_weights_composite: period[%d] must be finite and >= 0", c);
            return CC_EINVAL;
        }
    }
    return knn_impl(n, p, X, mask, sd, k, phi, normalize, rowptr_out, col_out, w_out, nnz_out, stream);
}

int cc_knn_weights_geodesic(int64_t n, int64_t p, const float* X, const uint8_t* mask, const float* lonlat, float radius,
                            float alpha, int32_t k, float phi, int32_t normalize, int64_t** rowptr_out, int32_t** col_out,
                            float** w_out, int64_t* nnz_out, void* stream) {
    if (!lonlat || !(radius > 0.f) || std::isinf(radius) || !(alpha >= 0.f && alpha <= 1.f)) {
        snprintf(g_knn_err, sizeof(g_knn_err), "cc_knn_weights_geodesic: need lonlat, finite radius > 0, 0 <= alpha <= 1");
        return CC_EINVAL;
    }
    side_t sd = {};
    sd.Y = lonlat;
    sd.q = 2;
    sd.alpha = alpha;
    sd.radius = radius;
    return knn_impl(n, p, X, mask, sd, k, phi, normalize, rowptr_out, col_out, w_out, nnz_out, stream);
}

void cc_free_graph(int64_t* rowptr, int32_t* col, float* w) {
    if (rowptr) cudaFree(rowptr);
    if (col) cudaFree(col);
    if (w) cudaFree(w);
}

}  // extern "C"
