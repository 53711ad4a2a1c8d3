// cc_pca.cu -- f2: the leading principal directions of the original data, computed on the device so that a
// gamma path can be read back as n x q coordinates (cc_get_projection) instead of n x p centres
// (the path is drawn on two principal components; L202/L210: moving U to the host for
// plotting was the paper's bottleneck, "one could easily project the data to principal components on
// each GPU itself prior to data transfer").  Reading S25: the data are X with missing entries at the
// observed column mean (the cold start), columns centred; the directions are the leading eigenvectors of
// Xc^T Xc.
//
// Method: block (subspace) iteration with PB = 16 vectors.  One step applies C = Xc^T Xc to the
// orthonormal block Q in two HBM-bound passes over X (Y = Xc Q, warp per 4 rows; Z = Xc^T Y, thread per
// column over row chunks, fp32 inside a chunk, fp64 across chunks), forms the 16 x 16 matrices
// G = Z^T Z and T = Q^T Z in fp64, diagonalises both with a cyclic Jacobi sweep in one block, and sets
// Q <- Z W_G Lambda_G^{-1/2} (orthonormal by construction, rank-deficient directions dropped).  The
// Ritz pairs (theta_j, Q w_j) of T give the residuals ||C y - theta y||^2 = w^T G w - theta^2 without
// another pass; the host reads 16 numbers every few steps to decide when to stop.
#include <math.h>

#include "cc_internal.h"

namespace {
constexpr int PB = 16;      // vectors in the iterated block
constexpr int PQ = 8;       // directions a caller may ask for
constexpr int XQ_ROWS = 4;  // rows per warp in kp_xq
constexpr int XT_COLS = 128;
constexpr int XT_BATCH = 32;
constexpr int GR_COLS = 16;

__device__ __forceinline__ double unit_hash(unsigned long long x) {
    x += 0x9E3779B97F4A7C15ull;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    x ^= x >> 31;
    return (double)(x >> 11) * (2.0 / 9007199254740992.0) - 1.0;
}

// Start block: fixed pseudo-random entries in (-1,1); columns >= b stay zero (b = min(PB, p)).
__global__ void kp_init(int p, int b, double* __restrict__ Z) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)p * PB) return;
    const int k = (int)(t % PB);
    Z[t] = k < b ? unit_hash((unsigned long long)t) : 0.0;
}

// Y[i][k] = sum_c xc_ic Q[c][k],  xc = x - xbar on observed entries, 0 on missing ones.
__global__ void __launch_bounds__(256) kp_xq(int n, int p, int ld, const float* __restrict__ X,
                                             const uint8_t* __restrict__ mask, const float* __restrict__ xbar,
                                             const float* __restrict__ Qf, float* __restrict__ Y) {
    const int lane = threadIdx.x & 31;
    const long long nwarp = (long long)gridDim.x * (blockDim.x >> 5);
    const long long ngroup = ((long long)n + XQ_ROWS - 1) / XQ_ROWS;
    for (long long g = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); g < ngroup; g += nwarp) {
        const long long base = g * XQ_ROWS;
        float v[XQ_ROWS * PB];
#pragma unroll
        for (int j = 0; j < XQ_ROWS * PB; ++j) v[j] = 0.f;
        for (int c = lane; c < p; c += 32) {
            const float4* qp = reinterpret_cast<const float4*>(Qf + (size_t)c * PB);
            const float4 q0 = __ldg(qp), q1 = __ldg(qp + 1), q2 = __ldg(qp + 2), q3 = __ldg(qp + 3);
            const float qq[PB] = {q0.x, q0.y, q0.z, q0.w, q1.x, q1.y, q1.z, q1.w,
                                  q2.x, q2.y, q2.z, q2.w, q3.x, q3.y, q3.z, q3.w};
            const float mu = __ldg(xbar + c);
#pragma unroll
            for (int r = 0; r < XQ_ROWS; ++r) {
                const long long i = base + r;
                float x = 0.f;
                if (i < n) {
                    const size_t o = (size_t)i * ld + c;
                    if (!mask || mask[o]) x = X[o] - mu;
                }
#pragma unroll
                for (int k = 0; k < PB; ++k) v[r * PB + k] = fmaf(x, qq[k], v[r * PB + k]);
            }
        }
        // transpose-reduce: every stage halves the values a lane keeps; lane l ends with entries 2l, 2l+1
#pragma unroll
        for (int off = 16, cnt = XQ_ROWS * PB / 2; off >= 1; off >>= 1, cnt >>= 1) {
            const bool up = (lane & off) != 0;
#pragma unroll
            for (int j = 0; j < cnt; ++j) {
                const float send = up ? v[j] : v[j + cnt];
                const float keep = up ? v[j + cnt] : v[j];
                v[j] = keep + __shfl_xor_sync(0xffffffffu, send, off);
            }
        }
        const long long i = base + (lane >> 3);
        if (i < n) *reinterpret_cast<float2*>(Y + (size_t)i * PB + 2 * (lane & 7)) = make_float2(v[0], v[1]);
    }
}

// Same product for few rows and many columns: the eight warps of a block share one group of four rows and the
// column slice blockIdx.y, each warp striding the slice; partial results of the slices go to
// Y + slice * n * PB and are added when kp_xty stages them.
__global__ void __launch_bounds__(256) kp_xq_wide(int n, int p, int ld, int cols_per_slice, const float* __restrict__ X,
                                                  const uint8_t* __restrict__ mask, const float* __restrict__ xbar,
                                                  const float* __restrict__ Qf, float* __restrict__ Y) {
    __shared__ float red[8][XQ_ROWS * PB];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long base = (long long)blockIdx.x * XQ_ROWS;
    const int c0 = blockIdx.y * cols_per_slice;
    const int c1 = c0 + cols_per_slice < p ? c0 + cols_per_slice : p;
    float v[XQ_ROWS * PB];
#pragma unroll
    for (int j = 0; j < XQ_ROWS * PB; ++j) v[j] = 0.f;
    for (int c = c0 + warp * 32 + lane; c < c1; c += 256) {
        const float4* qp = reinterpret_cast<const float4*>(Qf + (size_t)c * PB);
        const float4 q0 = __ldg(qp), q1 = __ldg(qp + 1), q2 = __ldg(qp + 2), q3 = __ldg(qp + 3);
        const float qq[PB] = {q0.x, q0.y, q0.z, q0.w, q1.x, q1.y, q1.z, q1.w,
                              q2.x, q2.y, q2.z, q2.w, q3.x, q3.y, q3.z, q3.w};
        const float mu = __ldg(xbar + c);
#pragma unroll
        for (int r = 0; r < XQ_ROWS; ++r) {
            const long long i = base + r;
            float x = 0.f;
            if (i < n) {
                const size_t o = (size_t)i * ld + c;
                if (!mask || mask[o]) x = X[o] - mu;
            }
#pragma unroll
            for (int k = 0; k < PB; ++k) v[r * PB + k] = fmaf(x, qq[k], v[r * PB + k]);
        }
    }
#pragma unroll
    for (int off = 16, cnt = XQ_ROWS * PB / 2; off >= 1; off >>= 1, cnt >>= 1) {
        const bool up = (lane & off) != 0;
#pragma unroll
        for (int j = 0; j < cnt; ++j) {
            const float send = up ? v[j] : v[j + cnt];
            const float keep = up ? v[j + cnt] : v[j];
            v[j] = keep + __shfl_xor_sync(0xffffffffu, send, off);
        }
    }
    red[warp][2 * lane] = v[0];
    red[warp][2 * lane + 1] = v[1];
    __syncthreads();
    if (threadIdx.x < XQ_ROWS * PB) {
        float s = 0.f;
#pragma unroll
        for (int w = 0; w < 8; ++w) s += red[w][threadIdx.x];
        const long long i = base + (threadIdx.x >> 4);
        if (i < n) Y[(size_t)blockIdx.y * n * PB + (size_t)i * PB + (threadIdx.x & 15)] = s;
    }
}

// part[chunk][c][k] = sum_{i in chunk} xc_ic Y[i][k]   (fp32 inside a chunk)
__global__ void __launch_bounds__(XT_COLS) kp_xty(int n, int p, int ld, int rows_per_chunk, int nslices, const float* __restrict__ X,
                                                  const uint8_t* __restrict__ mask, const float* __restrict__ xbar,
                                                  const float* __restrict__ Y, float* __restrict__ part) {
    __shared__ float4 Ys[XT_BATCH][PB / 4];
    const int c = blockIdx.x * XT_COLS + threadIdx.x;
    const long long r0 = (long long)blockIdx.y * rows_per_chunk;
    const long long r1 = r0 + rows_per_chunk < n ? r0 + rows_per_chunk : n;
    const float mu = c < p ? __ldg(xbar + c) : 0.f;
    float acc[PB];
#pragma unroll
    for (int k = 0; k < PB; ++k) acc[k] = 0.f;
    for (long long i0 = r0; i0 < r1; i0 += XT_BATCH) {
        const int nb = (int)(r1 - i0 < XT_BATCH ? r1 - i0 : XT_BATCH);
        __syncthreads();
        {
            const int r = threadIdx.x >> 2, f = threadIdx.x & 3;  // 128 threads = 32 rows x 4 float4
            float4 y = make_float4(0.f, 0.f, 0.f, 0.f);
            if (r < nb)
                for (int sl = 0; sl < nslices; ++sl) {
                    const float4 a = __ldg(reinterpret_cast<const float4*>(Y + ((size_t)sl * n + (size_t)(i0 + r)) * PB) + f);
                    y.x += a.x; y.y += a.y; y.z += a.z; y.w += a.w;
                }
            Ys[r][f] = y;
        }
        __syncthreads();
        if (c < p) {
#pragma unroll 8
            for (int r = 0; r < nb; ++r) {
                const size_t o = (size_t)(i0 + r) * ld + c;
                float x = 0.f;
                if (!mask || mask[o]) x = X[o] - mu;
#pragma unroll
                for (int f = 0; f < PB / 4; ++f) {
                    const float4 y = Ys[r][f];
                    acc[4 * f + 0] = fmaf(x, y.x, acc[4 * f + 0]);
                    acc[4 * f + 1] = fmaf(x, y.y, acc[4 * f + 1]);
                    acc[4 * f + 2] = fmaf(x, y.z, acc[4 * f + 2]);
                    acc[4 * f + 3] = fmaf(x, y.w, acc[4 * f + 3]);
                }
            }
        }
    }
    if (c < p) {
        float4* o = reinterpret_cast<float4*>(part + ((size_t)blockIdx.y * p + c) * PB);
#pragma unroll
        for (int f = 0; f < PB / 4; ++f) o[f] = make_float4(acc[4 * f], acc[4 * f + 1], acc[4 * f + 2], acc[4 * f + 3]);
    }
}

// Z = sum over chunks of part (fp64, fixed order; skipped when nchunks == 0: Z is already there), then this
// block's share of G = Z^T Z and T = Q^T Z.  gpart[block][0..255] = G, [256..511] = T.
__global__ void __launch_bounds__(256) kp_gram(int p, int nchunks, const float* __restrict__ part, double* __restrict__ Z,
                                               const double* __restrict__ Q, double* __restrict__ gpart) {
    __shared__ double zs[GR_COLS][PB + 1], qs[GR_COLS][PB + 1];
    const int t = threadIdx.x, cl = t >> 4, k = t & 15;
    const int ngroups = (p + GR_COLS - 1) / GR_COLS;
    double g = 0.0, tt = 0.0;
    for (int grp = blockIdx.x; grp < ngroups; grp += gridDim.x) {
        const int c = grp * GR_COLS + cl;
        double z = 0.0, q = 0.0;
        if (c < p) {
            if (nchunks > 0) {
                const float* src = part + (size_t)c * PB + k;
                const size_t stride = (size_t)p * PB;
                double z0 = 0.0, z1 = 0.0, z2 = 0.0, z3 = 0.0;
                int ch = 0;
                for (; ch + 4 <= nchunks; ch += 4) {
                    z0 += (double)src[(size_t)ch * stride];
                    z1 += (double)src[(size_t)(ch + 1) * stride];
                    z2 += (double)src[(size_t)(ch + 2) * stride];
                    z3 += (double)src[(size_t)(ch + 3) * stride];
                }
                for (; ch < nchunks; ++ch) z0 += (double)src[(size_t)ch * stride];
                z = (z0 + z1) + (z2 + z3);
                Z[(size_t)c * PB + k] = z;
            } else {
                z = Z[(size_t)c * PB + k];
            }
            q = Q[(size_t)c * PB + k];
        }
        __syncthreads();
        zs[cl][k] = z;
        qs[cl][k] = q;
        __syncthreads();
        // thread (a, b) = (t >> 4, t & 15)
#pragma unroll
        for (int cc = 0; cc < GR_COLS; ++cc) {
            g += zs[cc][cl] * zs[cc][k];
            tt += qs[cc][cl] * zs[cc][k];
        }
    }
    gpart[(size_t)blockIdx.x * 512 + t] = g;
    gpart[(size_t)blockIdx.x * 512 + 256 + t] = tt;
}

// Cyclic Jacobi on a symmetric 16 x 16 matrix in shared memory, run by one warp (lanes 0..15 own one
// row/column each).  On return diag(A) holds the eigenvalues, the columns of V the eigenvectors.
__device__ void jacobi16(double (*A)[PB + 1], double (*V)[PB + 1], int lane) {
    if (lane < PB)
        for (int j = 0; j < PB; ++j) V[lane][j] = lane == j ? 1.0 : 0.0;
    __syncwarp();
    for (int sweep = 0; sweep < 30; ++sweep) {
        double off = 0.0, dg = 0.0;
        for (int i = 0; i < PB; ++i) {
            dg += A[i][i] * A[i][i];
            for (int j = i + 1; j < PB; ++j) off += A[i][j] * A[i][j];
        }
        if (off <= 1e-34 * dg || off == 0.0) break;
        for (int a = 0; a < PB - 1; ++a)
            for (int b = a + 1; b < PB; ++b) {
                const double apq = A[a][b];
                if (apq == 0.0) continue;  // uniform across the warp: every lane reads the same entry
                const double tau = (A[b][b] - A[a][a]) / (2.0 * apq);
                const double tn = (tau >= 0.0 ? 1.0 : -1.0) / (fabs(tau) + sqrt(1.0 + tau * tau));
                const double cs = 1.0 / sqrt(1.0 + tn * tn), sn = tn * cs;
                __syncwarp();
                if (lane < PB) {  // A <- A J : row `lane`, columns a and b
                    const double x = A[lane][a], y = A[lane][b];
                    A[lane][a] = cs * x - sn * y;
                    A[lane][b] = sn * x + cs * y;
                }
                __syncwarp();
                if (lane < PB) {  // A <- J^T A : column `lane`, rows a and b;  V <- V J
                    const double x = A[a][lane], y = A[b][lane];
                    A[a][lane] = cs * x - sn * y;
                    A[b][lane] = sn * x + cs * y;
                    const double vx = V[lane][a], vy = V[lane][b];
                    V[lane][a] = cs * vx - sn * vy;
                    V[lane][b] = sn * vx + cs * vy;
                }
                __syncwarp();
                if (lane == 0) A[a][b] = A[b][a] = 0.0;
                __syncwarp();
            }
    }
    __syncwarp();
}

// out: M[16][16] (Q <- Z M), W[16][16] (Ritz vectors of T, decreasing theta), theta[16], res[16]
__global__ void __launch_bounds__(256) kp_small(int nblk, const double* __restrict__ gpart, double* __restrict__ out) {
    __shared__ double G[PB][PB + 1], T[PB][PB + 1], G0[PB][PB + 1], VG[PB][PB + 1], VT[PB][PB + 1];
    __shared__ int permG[PB], permT[PB];
    const int t = threadIdx.x, a = t >> 4, b = t & 15;
    double g = 0.0, tt = 0.0;
    for (int i = 0; i < nblk; ++i) {
        g += gpart[(size_t)i * 512 + t];
        tt += gpart[(size_t)i * 512 + 256 + t];
    }
    G[a][b] = g;
    T[a][b] = tt;
    __syncthreads();
    const double gs = 0.5 * (G[a][b] + G[b][a]), ts = 0.5 * (T[a][b] + T[b][a]);
    __syncthreads();
    G[a][b] = gs;
    G0[a][b] = gs;
    T[a][b] = ts;
    __syncthreads();
    if (t < 32) jacobi16(G, VG, t);
    else if (t < 64) jacobi16(T, VT, t - 32);
    __syncthreads();
    if (t == 0 || t == 32) {  // decreasing order, stable
        double (*A)[PB + 1] = t == 0 ? G : T;
        int* perm = t == 0 ? permG : permT;
        for (int i = 0; i < PB; ++i) perm[i] = i;
        for (int i = 1; i < PB; ++i) {
            const int pi = perm[i];
            int j = i - 1;
            while (j >= 0 && A[perm[j]][perm[j]] < A[pi][pi]) { perm[j + 1] = perm[j]; --j; }
            perm[j + 1] = pi;
        }
    }
    __syncthreads();
    const double lg = G[permG[b]][permG[b]], lg0 = G[permG[0]][permG[0]];
    out[t] = (lg > 1e-14 * lg0 && lg > 0.0) ? VG[a][permG[b]] / sqrt(lg) : 0.0;
    out[256 + t] = VT[a][permT[b]];
    if (t < PB) {
        const int j = permT[t];
        const double th = T[j][j], th0 = T[permT[0]][permT[0]];
        double q = 0.0;
        for (int x = 0; x < PB; ++x) {
            double s = 0.0;
            for (int y = 0; y < PB; ++y) s += G0[x][y] * VT[y][j];
            q += VT[x][j] * s;
        }
        const double r2 = q - th * th;
        out[512 + t] = th;
        out[528 + t] = th0 > 0.0 ? sqrt(r2 > 0.0 ? r2 : 0.0) / th0 : 0.0;
    }
}

// dst[c][j] = sum_k src[c][k] M[k][j]  (fp64), optional fp32 copy; optional per-block signed entry of
// largest magnitude per column (first on ties) for the sign convention.
__global__ void __launch_bounds__(256) kp_mul(int p, const double* __restrict__ src, const double* __restrict__ M,
                                              double* __restrict__ dst, float* __restrict__ dstf, double* __restrict__ bmax) {
    __shared__ double Ms[PB][PB + 1], vs[GR_COLS][PB + 1];
    const int t = threadIdx.x, cl = t >> 4, j = t & 15;
    Ms[cl][j] = M[t];
    __syncthreads();
    const int c = blockIdx.x * GR_COLS + cl;
    double v = 0.0;
    if (c < p) {
        const double* s = src + (size_t)c * PB;
#pragma unroll
        for (int k = 0; k < PB; ++k) v += s[k] * Ms[k][j];
        dst[(size_t)c * PB + j] = v;
        if (dstf) dstf[(size_t)c * PB + j] = (float)v;
    }
    if (bmax) {
        vs[cl][j] = v;
        __syncthreads();
        if (t < PB) {
            double best = vs[0][t];
            for (int r = 1; r < GR_COLS; ++r)
                if (fabs(vs[r][t]) > fabs(best)) best = vs[r][t];
            bmax[(size_t)blockIdx.x * PB + t] = best;
        }
    }
}

__global__ void kp_sign(int nblk, const double* __restrict__ bmax, double* __restrict__ sgn) {
    const int j = threadIdx.x;
    if (j >= PB) return;
    double best = 0.0;
    for (int i = 0; i < nblk; ++i) {
        const double v = bmax[(size_t)i * PB + j];
        if (fabs(v) > fabs(best)) best = v;
    }
    sgn[j] = best < 0.0 ? -1.0 : 1.0;
}

__global__ void kp_write(int p, int q, const double* __restrict__ Pd, const double* __restrict__ sgn, float* __restrict__ out) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)p * q) return;
    const int j = (int)(t % q);
    const long long c = t / q;
    out[t] = (float)(sgn[j] * Pd[(size_t)c * PB + j]);
}
}  // namespace

extern "C" int cc_principal_components(cc_handle* h, int32_t q, int32_t maxit, double tol, float* P_out,
                                       int32_t out_on_device, double* var_out, double* resid_out, int32_t* iters_out) {
    if (!h) return CC_EINVAL;
    if (!P_out || q < 1 || q > PQ || q > h->p || maxit < 1 || !(tol >= 0.0)) {
        snprintf(h->err, sizeof(h->err), "cc_principal_components: need P_out, 1 <= q <= min(%d, p), maxit >= 1, tol >= 0", PQ);
        return CC_EINVAL;
    }
    const int n = (int)h->n, p = (int)h->p, ld = (int)h->ld;
    const int b = p < PB ? p : PB;
    cudaStream_t st = h->stream;
    // row chunks of kp_xty: about four blocks per SM in all, whole batches of rows per chunk
    const int colblocks = (p + XT_COLS - 1) / XT_COLS;
    int nchunks = (4 * h->sms + colblocks - 1) / colblocks;
    if (nchunks > (n + 63) / 64) nchunks = (n + 63) / 64;
    if (nchunks < 1) nchunks = 1;
    int rows_per_chunk = ((n + nchunks - 1) / nchunks + XT_BATCH - 1) / XT_BATCH * XT_BATCH;
    nchunks = (n + rows_per_chunk - 1) / rows_per_chunk;
    const int ngroups = (p + GR_COLS - 1) / GR_COLS;
    const int gram_blocks = ngroups < 2 * h->sms ? ngroups : 2 * h->sms;
    const size_t pv = (size_t)p * PB;

    float *Y = nullptr, *part = nullptr, *Qf = nullptr, *Pdev = nullptr;
    double *Zd = nullptr, *Qd = nullptr, *gpart = nullptr, *small = nullptr, *bmax = nullptr, *sgn = nullptr;
    int rc = CC_OK;
    double host[2 * PB];
    int iters = 0;
    auto fail = [&](cudaError_t e, const char* what) {
        snprintf(h->err, sizeof(h->err), "cc_principal_components: %s: %s", what, cudaGetErrorString(e));
        rc = CC_ECUDA;
    };
#define PCA_TRY(call, what) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { fail(e_, what); goto done; } } while (0)
    // Y = Xc Q: a warp per four rows when there are rows enough to fill the machine, else a block per four rows
    // and column slices
    const long long rowgroups = ((long long)n + XQ_ROWS - 1) / XQ_ROWS;
    const bool wide = rowgroups < 32LL * h->sms;
    int nslices = 1, cols_per_slice = p;
    if (wide) {
        nslices = (int)((4LL * h->sms + rowgroups - 1) / rowgroups);
        if (nslices > (p + 255) / 256) nslices = (p + 255) / 256;
        if (nslices > 64) nslices = 64;
        cols_per_slice = ((p + nslices - 1) / nslices + 31) / 32 * 32;
        nslices = (p + cols_per_slice - 1) / cols_per_slice;
    }
    PCA_TRY(cc_dev_alloc((void**)&Y, (size_t)nslices * n * PB * sizeof(float), st), "alloc Y");
    PCA_TRY(cc_dev_alloc((void**)&part, (size_t)nchunks * pv * sizeof(float), st), "alloc partial sums");
    PCA_TRY(cc_dev_alloc((void**)&Qf, pv * sizeof(float), st), "alloc Q");
    PCA_TRY(cc_dev_alloc((void**)&Zd, pv * sizeof(double), st), "alloc Z");
    PCA_TRY(cc_dev_alloc((void**)&Qd, pv * sizeof(double), st), "alloc Q");
    PCA_TRY(cc_dev_alloc((void**)&gpart, (size_t)gram_blocks * 512 * sizeof(double), st), "alloc Gram partials");
    PCA_TRY(cc_dev_alloc((void**)&small, 1024 * sizeof(double), st), "alloc small");
    PCA_TRY(cc_dev_alloc((void**)&bmax, (size_t)ngroups * PB * sizeof(double), st), "alloc sign partials");
    PCA_TRY(cc_dev_alloc((void**)&sgn, PB * sizeof(double), st), "alloc signs");
    PCA_TRY(cudaMemsetAsync(Qd, 0, pv * sizeof(double), st), "memset");

    // orthonormal start: Z = fixed pseudo-random block, Q = Z W Lambda^{-1/2}
    kp_init<<<(unsigned)((pv + 255) / 256), 256, 0, st>>>(p, b, Zd);
    kp_gram<<<gram_blocks, 256, 0, st>>>(p, 0, part, Zd, Qd, gpart);
    kp_small<<<1, 256, 0, st>>>(gram_blocks, gpart, small);
    kp_mul<<<ngroups, 256, 0, st>>>(p, Zd, small, Qd, Qf, nullptr);
    h->launches += 4;
    {
        long long xq_blocks = (((long long)n + XQ_ROWS - 1) / XQ_ROWS + 7) / 8;
        if (xq_blocks > 8LL * h->sms) xq_blocks = 8LL * h->sms;
        if (xq_blocks < 1) xq_blocks = 1;
        for (int it = 0; it < maxit; ++it) {
            if (wide)
                kp_xq_wide<<<dim3((unsigned)rowgroups, nslices), 256, 0, st>>>(n, p, ld, cols_per_slice, h->X, h->mask, h->colmean, Qf, Y);
            else
                kp_xq<<<(unsigned)xq_blocks, 256, 0, st>>>(n, p, ld, h->X, h->mask, h->colmean, Qf, Y);
            kp_xty<<<dim3(colblocks, nchunks), XT_COLS, 0, st>>>(n, p, ld, rows_per_chunk, nslices, h->X, h->mask, h->colmean, Y, part);
            kp_gram<<<gram_blocks, 256, 0, st>>>(p, nchunks, part, Zd, Qd, gpart);
            kp_small<<<1, 256, 0, st>>>(gram_blocks, gpart, small);
            h->launches += 4;
            iters = it + 1;
            const bool last = it + 1 == maxit;
            if (last || (it >= 1 && (it & 1))) {  // the Ritz residuals of the block that was just multiplied
                PCA_TRY(cudaMemcpyAsync(host, small + 512, 2 * PB * sizeof(double), cudaMemcpyDeviceToHost, st), "read residuals");
                PCA_TRY(cudaStreamSynchronize(st), "sync");
                double worst = 0.0;
                for (int j = 0; j < q; ++j) worst = host[PB + j] > worst ? host[PB + j] : worst;
                if (worst <= tol || last) break;
            }
            kp_mul<<<ngroups, 256, 0, st>>>(p, Zd, small, Qd, Qf, nullptr);
            h->launches += 1;
        }
    }
    // Ritz rotation of the last multiplied block, sign convention, write-out
    kp_mul<<<ngroups, 256, 0, st>>>(p, Qd, small + 256, Zd, nullptr, bmax);
    kp_sign<<<1, 32, 0, st>>>(ngroups, bmax, sgn);
    Pdev = P_out;
    if (!out_on_device) PCA_TRY(cc_dev_alloc((void**)&Pdev, (size_t)p * q * sizeof(float), st), "alloc P");
    kp_write<<<(unsigned)(((size_t)p * q + 255) / 256), 256, 0, st>>>(p, q, Zd, sgn, Pdev);
    h->launches += 3;
    if (!out_on_device) PCA_TRY(cudaMemcpyAsync(P_out, Pdev, (size_t)p * q * sizeof(float), cudaMemcpyDeviceToHost, st), "copy P");
    PCA_TRY(cudaStreamSynchronize(st), "sync");
    PCA_TRY(cudaGetLastError(), "kernels");
    for (int j = 0; j < q; ++j) {
        if (var_out) var_out[j] = (host[j] > 0.0 ? host[j] : 0.0) / (double)(n > 1 ? n - 1 : 1);
        if (resid_out) resid_out[j] = host[PB + j];
    }
    if (iters_out) *iters_out = iters;
done:
#undef PCA_TRY
    if (Pdev && Pdev != P_out) cc_dev_free(Pdev, st);
    cc_dev_free(Y, st); cc_dev_free(part, st); cc_dev_free(Qf, st); cc_dev_free(Zd, st); cc_dev_free(Qd, st);
    cc_dev_free(gpart, st); cc_dev_free(small, st); cc_dev_free(bmax, st); cc_dev_free(sgn, st);
    return rc;
}
