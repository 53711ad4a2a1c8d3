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
// Steps, all on the device, no sort library and no floating-point atomics:
//   1. k_knn_tile<float>: brute-force distances in 64 x 64 register tiles (direct differences, fp32), a sorted
//      list per query in shared memory, filtered insertion (a candidate is looked at only if it beats the
//      current last distance).  The n x n distance matrix never exists.  The list holds k + CC_KNN_SLACK
//      candidates: a SHORTLIST, because which neighbours are the k nearest is index output and is decided in
//      the arithmetic the definition is stated in, not in fp32:
//   2. k_rerank: the shortlist's distances recomputed in fp64 from the fp32 inputs -- differences of fp32 numbers
//      are exact in fp64, the squares are added one coordinate after the other with separate multiply and add
//      (no FMA contraction) -- then ordered by (distance, index): ties go to the smaller index (S9).  A row is
//      SAFE when its k-th fp64 distance lies below the shortlist's last fp32 distance by more than the fp32
//      rounding bound (p + 8) 2^-23: then no candidate outside the shortlist can belong to the k nearest.
//   3. rows that are not safe (near-ties wider than the slack, lattice data or duplicated points with many exact
//      ties) go through k_knn_tile<double>: the same tiles with the fp64 arithmetic of step 2 over all candidates.
//   4. symmetrise by OR: count reverse-only entries (integer atomics), scan, fill, sort each row by column.
//   5. weights w = exp(-phi d^2) from the fp64 distance of the ordered pair (so w_ij == w_ji bitwise), entries whose
//      weight underflows to 0 in fp32 are removed in both directions (a zero weight is an absent pair, L40 / S24),
//      optional normalisation.
// With side coordinates (eq. 9) the composite distance involves square roots and trigonometric functions whose fp64
// values are library-dependent; that path ranks in fp32 as before (k candidates, no re-rank).
#include <cfloat>
#include <cmath>
#include <cstdio>

#include "cc_device.cuh"
#include "cc_internal.h"

namespace {

constexpr int TQ = 64, TC = 64, PC = 16, KMAX = 64, QSIDE = 4;

// Packed fp32 pairs (FADD2 / FFMA2 on sm_100: one issue slot for two lanes' worth; each half is the same IEEE operation as
// the scalar instruction, so the distances are bit-identical).  The fp32 shortlist pass is 32 FP instructions per 8 shared
// loads and was issue-bound at 40 % of the FP32 peak.
typedef unsigned long long knn_f2;
__device__ __forceinline__ knn_f2 knn_pk(float lo, float hi) { knn_f2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ knn_f2 knn_sub2(knn_f2 a, knn_f2 b) { knn_f2 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ knn_f2 knn_fma2(knn_f2 a, knn_f2 b, knn_f2 c) { knn_f2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ void knn_unpk(knn_f2 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
constexpr int CC_KNN_SLACK = 4;          // extra shortlist candidates per row for the fp64 re-rank
constexpr int KLMAX = KMAX + CC_KNN_SLACK;

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


// The distance of a pair in the arithmetic of the definition (see the header): fp64, one coordinate after the other,
// separate multiply and add.  With a mask: over co-observed coordinates, scaled by p / #co-observed (S11); no
// co-observed coordinate: +inf.
template <bool MASKED>
__device__ __forceinline__ double exact_dist2(int p, const float* __restrict__ xi, const float* __restrict__ xj,
                                              const uint8_t* __restrict__ mi, const uint8_t* __restrict__ mj) {
    double s = 0.0;
    int co = 0;
    for (int c = 0; c < p; ++c) {
        if (MASKED && !(mi[c] && mj[c])) continue;
        const double t = (double)xi[c] - (double)xj[c];
        s = __dadd_rn(s, __dmul_rn(t, t));
        ++co;
    }
    if (MASKED) return co ? __ddiv_rn(__dmul_rn(s, (double)p), (double)co) : (double)INFINITY;
    return s;
}

template <typename T> __device__ __forceinline__ T knn_big();
template <> __device__ __forceinline__ float knn_big<float>() { return FLT_MAX; }
template <> __device__ __forceinline__ double knn_big<double>() { return (double)INFINITY; }

// T = float: the fast pass over all rows (a shortlist of kk candidates per row).  T = double: the exact pass over the
// listed rows only, distances bit-identical to exact_dist2 (same order of the additions).  rows == NULL: query r is row r.
template <typename T, bool MASKED, bool SIDE>
__global__ void __launch_bounds__(256) k_knn_tile(int n, int p, int kk, const float* __restrict__ X,
                                                   const uint8_t* __restrict__ mask, const side_t sd,
                                                   const int* __restrict__ rows, int nrows, int* __restrict__ nbr,
                                                   float* __restrict__ dlast) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* Dt = reinterpret_cast<T*>(smem_raw);            // TQ x (TC+1)
    T* Ld = Dt + TQ * (TC + 1);                        // TQ x kk  list distances (ascending)
    int* Li = reinterpret_cast<int*>(Ld + TQ * kk);    // TQ x kk  list indices
    float* Xq = reinterpret_cast<float*>(Li + TQ * kk);   // TQ x (PC+1)
    float* Xc = Xq + TQ * (PC + 1);                    // TC x (PC+1)
    float* Mq = Xc + TC * (PC + 1);                    // masks as 0/1 floats (MASKED only)
    float* Mc = Mq + (MASKED ? TQ * (PC + 1) : 0);
    __shared__ int qrow[TQ];

    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    // The fp32 shortlist pass without a mask: packed arithmetic, and the two staged tiles TRANSPOSED ([column][row], row
    // stride TQ + 4) with four CONSECUTIVE candidate rows per thread, so that a column costs two 16-byte shared loads
    // instead of eight scalar ones (same footprint: PC x (TQ + 4) = TQ x (PC + 1) floats).
    constexpr bool PACKED = sizeof(T) == 4 && !MASKED;
    const int q0 = blockIdx.x * TQ;
    const T big = knn_big<T>();
    for (int t = tid; t < TQ * kk; t += 256) { Ld[t] = big; Li[t] = -1; }
    if (tid < TQ) qrow[tid] = q0 + tid < nrows ? (rows ? rows[q0 + tid] : q0 + tid) : -1;
    __syncthreads();

    for (int c0 = 0; c0 < n; c0 += TC) {
        T acc[4][4];
        float cnt[4][4];
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) { acc[a][b] = (T)0; cnt[a][b] = 0.f; }
        knn_f2 accp[4][2] = {{0ull, 0ull}, {0ull, 0ull}, {0ull, 0ull}, {0ull, 0ull}};
        for (int pc = 0; pc < p; pc += PC) {
            // stage PC columns of the query tile and of the candidate tile; values at missing entries are never read
            for (int t = tid; t < TQ * PC; t += 256) {
                const int r = t / PC, c = t % PC;
                const int gi = qrow[r], gj = c0 + r, gc = pc + c;
                bool vi = gi >= 0 && gc < p, vj = gj < n && gc < p;
                if (MASKED) {
                    vi = vi && mask[(size_t)gi * p + gc];
                    vj = vj && mask[(size_t)gj * p + gc];
                    Mq[r * (PC + 1) + c] = vi ? 1.f : 0.f;
                    Mc[r * (PC + 1) + c] = vj ? 1.f : 0.f;
                }
                if constexpr (PACKED) {
                    Xq[c * (TQ + 4) + r] = vi ? X[(size_t)gi * p + gc] : 0.f;
                    Xc[c * (TC + 4) + r] = vj ? X[(size_t)gj * p + gc] : 0.f;
                } else {
                    Xq[r * (PC + 1) + c] = vi ? X[(size_t)gi * p + gc] : 0.f;
                    Xc[r * (PC + 1) + c] = vj ? X[(size_t)gj * p + gc] : 0.f;
                }
            }
            __syncthreads();
#pragma unroll
            for (int c = 0; c < PC; ++c) {
                float xq[4], xc[4], mq[4], mc[4];
                if constexpr (PACKED) {
                    const float4 q4 = *reinterpret_cast<const float4*>(Xq + c * (TQ + 4) + ty * 4);
                    const float4 c4 = *reinterpret_cast<const float4*>(Xc + c * (TC + 4) + tx * 4);
                    xq[0] = q4.x; xq[1] = q4.y; xq[2] = q4.z; xq[3] = q4.w;
                    xc[0] = c4.x; xc[1] = c4.y; xc[2] = c4.z; xc[3] = c4.w;
                } else
#pragma unroll
                for (int a = 0; a < 4; ++a) {
                    xq[a] = Xq[(ty * 4 + a) * (PC + 1) + c];
                    xc[a] = Xc[(tx + 16 * a) * (PC + 1) + c];
                    if (MASKED) { mq[a] = Mq[(ty * 4 + a) * (PC + 1) + c]; mc[a] = Mc[(tx + 16 * a) * (PC + 1) + c]; }
                }
                if constexpr (PACKED) {
                    const knn_f2 xc01 = knn_pk(xc[0], xc[1]), xc23 = knn_pk(xc[2], xc[3]);
#pragma unroll
                    for (int a = 0; a < 4; ++a) {
                        const knn_f2 qq = knn_pk(xq[a], xq[a]);
                        const knn_f2 d01 = knn_sub2(qq, xc01), d23 = knn_sub2(qq, xc23);
                        accp[a][0] = knn_fma2(d01, d01, accp[a][0]);
                        accp[a][1] = knn_fma2(d23, d23, accp[a][1]);
                    }
                } else {
#pragma unroll
                for (int a = 0; a < 4; ++a)
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        if constexpr (sizeof(T) == 8) {
                            // masked-out coordinates were staged as 0 on both sides only when BOTH are missing; a term
                            // is added only where both are observed (adding an exact 0 otherwise would be harmless too)
                            const double df = (double)xq[a] - (double)xc[b];
                            const double sq = __dmul_rn(df, df);
                            if (MASKED) {
                                const float m = mq[a] * mc[b];
                                if (m != 0.f) { acc[a][b] = __dadd_rn(acc[a][b], sq); cnt[a][b] += 1.f; }
                            } else {
                                acc[a][b] = __dadd_rn(acc[a][b], sq);
                            }
                        } else {
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
            }
            }
            __syncthreads();
        }
        if constexpr (PACKED) {
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                float v0, v1, v2, v3;
                knn_unpk(accp[a][0], v0, v1);
                knn_unpk(accp[a][1], v2, v3);
                acc[a][0] = (T)v0; acc[a][1] = (T)v1; acc[a][2] = (T)v2; acc[a][3] = (T)v3;
            }
        }
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                T d = acc[a][b];
                if (MASKED) {
                    if constexpr (sizeof(T) == 8) d = cnt[a][b] > 0.f ? __ddiv_rn(__dmul_rn(d, (double)p), (double)cnt[a][b]) : big;
                    else d = cnt[a][b] > 0.f ? d * (float)p / cnt[a][b] : big;
                }
                if (SIDE) {
                    const int gi = qrow[ty * 4 + a], gj = c0 + (PACKED ? tx * 4 + b : tx + 16 * b);
                    if (gi >= 0 && gj < n && d < big) d = sd.alpha * sqrtf((float)d) + (1.f - sd.alpha) * side_dist(sd, gi, gj);
                }
                Dt[(ty * 4 + a) * (TC + 1) + (PACKED ? tx * 4 + b : tx + 16 * b)] = d;
            }
        __syncthreads();
        // selection: warp wq handles queries wq*8 .. wq*8+7; lanes look at candidates lane, lane+32
        const int lane = tid & 31, wq = tid >> 5;
        for (int qq = 0; qq < 8; ++qq) {
            const int q = wq * 8 + qq, gi = qrow[q];
            if (gi < 0) break;
            T* ld = Ld + q * kk;
            int* li = Li + q * kk;
            for (int half = 0; half < 2; ++half) {
                const int cj = lane + 32 * half, gj = c0 + cj;
                const T d = Dt[q * (TC + 1) + cj];
                const T kth = ld[kk - 1];
                unsigned bal = __ballot_sync(0xffffffffu, gj < n && gj != gi && d < kth);
                while (bal) {   // ascending candidate index: equal distances keep the smaller index ahead (S9)
                    const int src = __ffs(bal) - 1;
                    bal &= bal - 1;
                    const T dc = __shfl_sync(0xffffffffu, d, src);
                    if (lane == 0 && dc < ld[kk - 1]) {
                        int pos = kk - 1;
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
    for (int t = tid; t < TQ * kk; t += 256) {
        const int r = q0 + t / kk;
        if (r < nrows) nbr[(size_t)r * kk + t % kk] = Li[t];
    }
    if (dlast && tid < TQ && q0 + tid < nrows)     // last shortlist distance, or -1 when the list is not full
        dlast[q0 + tid] = Li[tid * kk + kk - 1] >= 0 ? (float)Ld[tid * kk + kk - 1] : -1.f;
}

// Step 2 of the header.  One warp per row: the shortlist's exact distances (a lane per candidate), ordered by
// (distance, index); the first k are the row's neighbours when the row is safe, else the row joins `flagged`.
template <bool MASKED>
__global__ void __launch_bounds__(256) k_rerank(int n, int p, int k, int kk, const float* __restrict__ X,
                                                const uint8_t* __restrict__ mask, const int* __restrict__ cand,
                                                const float* __restrict__ dlast, int* __restrict__ fin,
                                                int* __restrict__ flagged, int* __restrict__ nflag) {
    __shared__ double sdist[8][KLMAX];
    __shared__ int sidx[8][KLMAX];
    const int lane = threadIdx.x & 31, wl = threadIdx.x >> 5;
    const long long nw = (long long)gridDim.x * 8;
    const double beta = (double)(p + 8) * 1.1920928955078125e-7;     // (p + 8) 2^-23
    for (long long i = (long long)blockIdx.x * 8 + wl; i < n; i += nw) {
        for (int q = lane; q < kk; q += 32) {
            const int j = cand[(size_t)i * kk + q];
            sidx[wl][q] = j;
            sdist[wl][q] = j >= 0 ? exact_dist2<MASKED>(p, X + (size_t)i * p, X + (size_t)j * p,
                                                        MASKED ? mask + (size_t)i * p : nullptr,
                                                        MASKED ? mask + (size_t)j * p : nullptr)
                                  : (double)INFINITY;
        }
        __syncwarp();
        if (lane == 0) {
            for (int x = 1; x < kk; ++x) {
                const double dv = sdist[wl][x];
                const int jv = sidx[wl][x];
                int y = x;
                while (y > 0 && (sdist[wl][y - 1] > dv || (sdist[wl][y - 1] == dv && (unsigned)sidx[wl][y - 1] > (unsigned)jv))) {
                    sdist[wl][y] = sdist[wl][y - 1]; sidx[wl][y] = sidx[wl][y - 1]; --y;
                }
                sdist[wl][y] = dv; sidx[wl][y] = jv;
            }
            const float dl = dlast[i];
            const bool safe = dl < 0.f || sdist[wl][k - 1] < (double)dl * (1.0 - beta);
            if (!safe) flagged[atomicAdd(nflag, 1)] = (int)i;
        }
        __syncwarp();
        for (int q = lane; q < k; q += 32) fin[(size_t)i * k + q] = sdist[wl][q] < (double)INFINITY ? sidx[wl][q] : -1;
        __syncwarp();
    }
}

// lists of the flagged rows (exact pass) into their rows of `fin`
__global__ void k_scatter_lists(int nrows, int k, const int* __restrict__ rows, const int* __restrict__ src, int* __restrict__ fin) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)nrows * k) return;
    fin[(size_t)rows[t / k] * k + t % k] = src[t];
}

// order of the list entries: valid neighbour indices ascending, the empty slots (-1) last
__device__ __forceinline__ unsigned list_key(int v) { return v < 0 ? 0xffffffffu : (unsigned)v; }

// sort each k-list by neighbour index (needed for the membership tests and the CSR fill); own[i] = valid entries
__global__ void k_sort_lists(int n, int k, int* __restrict__ nbr, int* __restrict__ own) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int* a = nbr + (size_t)i * k;
    int cnt = a[0] >= 0 ? 1 : 0;
    for (int x = 1; x < k; ++x) {
        const int v = a[x];
        cnt += v >= 0 ? 1 : 0;
        int y = x;
        while (y > 0 && list_key(a[y - 1]) > list_key(v)) { a[y] = a[y - 1]; --y; }
        a[y] = v;
    }
    own[i] = cnt;
}

__device__ __forceinline__ bool in_list(const int* a, int cnt, int v) {
    int lo = 0, hi = cnt - 1;
    while (lo <= hi) {
        const int mid = (lo + hi) >> 1;
        if (a[mid] == v) return true;
        if (a[mid] < v) lo = mid + 1; else hi = mid - 1;
    }
    return false;
}

// i ~ j "or vice versa": j gets a reverse-only entry when i lists j but j does not list i
__global__ void k_count_reverse(int n, int k, const int* __restrict__ nbr, const int* __restrict__ own, int* __restrict__ extra) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)n * k) return;
    const int i = (int)(t / k), j = nbr[t];
    if (j >= 0 && !in_list(nbr + (size_t)j * k, own[j], i)) atomicAdd(&extra[j], 1);
}

// exclusive scan of a[i] + b[i] (b may be NULL) -> rowptr (int64).  One block; n is at most ~1e6.
__global__ void k_scan_rows(int n, const int* __restrict__ a, const int* __restrict__ b, int64_t* __restrict__ rowptr) {
    __shared__ long long sm[1024];
    __shared__ long long carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < n; base += 1024) {
        const int i = base + threadIdx.x;
        const long long v = i < n ? (long long)a[i] + (b ? b[i] : 0) : 0;
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

// Row i = its own list (the first own[i] slots, in list order) followed by the reverse-only entries.
__global__ void k_fill_rows(int n, int k, const int* __restrict__ nbr, const int* __restrict__ own,
                            const int64_t* __restrict__ rowptr, int* __restrict__ cursor, int* __restrict__ col) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)n * k) return;
    const int i = (int)(t / k), q = (int)(t % k), j = nbr[t];
    if (j < 0) return;          // the valid entries are the first own[i] of the sorted list: q < own[i] here
    col[rowptr[i] + q] = j;
    if (!in_list(nbr + (size_t)j * k, own[j], i)) {
        const int slot = atomicAdd(&cursor[j], 1);
        col[rowptr[j] + own[j] + slot] = i;
    }
}

// sort each row by column (the set is unique, so the result does not depend on the fill order) and compute the
// weight of every entry from the ordered pair (min, max) so that w_ij == w_ji bitwise.  Without side coordinates:
// a lane per entry, the exact fp64 distance (the oracle's d_ij^2), w = (float) exp(-phi d^2) in fp64.  With side
// coordinates (eq. 9): the fp32 composite distance, a warp per entry.
template <bool MASKED, bool SIDE>
__global__ void k_rows_finish(int n, int p, float phi, const float* __restrict__ X, const uint8_t* __restrict__ mask,
                              const side_t sd, const int64_t* __restrict__ rowptr, int* __restrict__ col, float* __restrict__ w,
                              int* __restrict__ nzero) {
    const int lane = threadIdx.x & 31;
    const long long nw = (long long)gridDim.x * (blockDim.x >> 5);
    int zeros = 0;
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
        if constexpr (!SIDE) {
            for (long long e = rs + lane; e < re; e += 32) {
                const int j = col[e];
                const int lo = min((int)i, j), hi = max((int)i, j);
                const double d2 = exact_dist2<MASKED>(p, X + (size_t)lo * p, X + (size_t)hi * p,
                                                      MASKED ? mask + (size_t)lo * p : nullptr, MASKED ? mask + (size_t)hi * p : nullptr);
                const float we = d2 < (double)INFINITY ? (float)exp(-(double)phi * d2) : 0.f;
                w[e] = we;
                zeros += we == 0.f ? 1 : 0;
            }
        } else {
        for (long long e = rs; e < re; ++e) {
            const int j = col[e];
            const int lo = min((int)i, j), hi = max((int)i, j);
            float s = 0.f, c = 0.f;
            for (int q = lane; q < p; q += 32) {
                if (MASKED) {
                    const bool m = mask[(size_t)lo * p + q] && mask[(size_t)hi * p + q];
                    const float df = m ? X[(size_t)lo * p + q] - X[(size_t)hi * p + q] : 0.f;
                    s = fmaf(df, df, s);
                    c += m ? 1.f : 0.f;
                } else {
                    const float df = X[(size_t)lo * p + q] - X[(size_t)hi * p + q];
                    s = fmaf(df, df, s);
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) { s += __shfl_xor_sync(0xffffffffu, s, o); c += __shfl_xor_sync(0xffffffffu, c, o); }
            if (MASKED) s = c > 0.f ? s * (float)p / c : FLT_MAX;
            float we = 0.f;
            if (s < FLT_MAX) {   // eq. 9, then eq. 8 on d^2
                const float d = sd.alpha * sqrtf(s) + (1.f - sd.alpha) * side_dist(sd, lo, hi);
                we = expf(-phi * d * d);
            }
            if (lane == 0) { w[e] = we; zeros += we == 0.f ? 1 : 0; }
        }
        }
    }
    if (zeros) atomicAdd(nzero, zeros);
}

// A weight that is 0 in fp32 is an absent pair: since w_ij == w_ji bitwise, dropping the zero
// entries row by row keeps the CSR symmetric.  cnt[i] = entries of row i that stay.
__global__ void k_count_pos(int n, const int64_t* __restrict__ rowptr, const float* __restrict__ w, int* __restrict__ cnt) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int c = 0;
    for (long long e = rowptr[i]; e < rowptr[i + 1]; ++e) c += w[e] != 0.f ? 1 : 0;
    cnt[i] = c;
}

__global__ void k_compact_rows(int n, const int64_t* __restrict__ rowptr, const int* __restrict__ col, const float* __restrict__ w,
                               const int64_t* __restrict__ rowptr2, int* __restrict__ col2, float* __restrict__ w2) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    long long o = rowptr2[i];
    for (long long e = rowptr[i]; e < rowptr[i + 1]; ++e)
        if (w[e] != 0.f) { col2[o] = col[e]; w2[o] = w[e]; ++o; }
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

template <typename T>
size_t knn_smem(int kk, bool masked) {
    return (size_t)TQ * (TC + 1) * sizeof(T) + (size_t)TQ * kk * (sizeof(T) + sizeof(int)) +
           (size_t)(masked ? 4 : 2) * TQ * (PC + 1) * sizeof(float);
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
    const bool side = sd.Y != nullptr;
    // shortlist length of the fp32 pass (the re-rank needs the slack; the eq.-9 path ranks in fp32 and needs none)
    const int kk = side ? k : (int)((int64_t)k + CC_KNN_SLACK < n - 1 ? k + CC_KNN_SLACK : n - 1);
    int *cand = nullptr, *nbr = nullptr, *own = nullptr, *extra = nullptr, *cursor = nullptr, *col = nullptr, *flagged = nullptr,
        *counters = nullptr, *nbr2 = nullptr, *col2 = nullptr;
    float *dlast = nullptr, *w = nullptr, *w2 = nullptr;
    int64_t *rowptr = nullptr, *rowptr2 = nullptr;
    double* red = nullptr;   // [0] total, then partials, then ticket
    int64_t nnz = 0;
    int hcount[2] = {0, 0};  // flagged rows, zero weights
    const long long nk = (long long)n * k;
    *rowptr_out = nullptr; *col_out = nullptr; *w_out = nullptr; *nnz_out = 0;
    KCUDA(cudaMalloc((void**)&nbr, (size_t)nk * sizeof(int)));
    KCUDA(cudaMalloc((void**)&own, (size_t)n * sizeof(int)));
    KCUDA(cudaMalloc((void**)&extra, (size_t)n * sizeof(int)));
    KCUDA(cudaMalloc((void**)&cursor, (size_t)n * sizeof(int)));
    KCUDA(cudaMalloc((void**)&counters, 2 * sizeof(int)));
    KCUDA(cudaMalloc((void**)&rowptr, (size_t)(n + 1) * sizeof(int64_t)));
    KCUDA(cudaMalloc((void**)&red, (size_t)(2 + CC_MAXBLK) * sizeof(double)));
    KCUDA(cudaMemsetAsync(extra, 0, (size_t)n * sizeof(int), st));
    KCUDA(cudaMemsetAsync(cursor, 0, (size_t)n * sizeof(int), st));
    KCUDA(cudaMemsetAsync(counters, 0, 2 * sizeof(int), st));
    KCUDA(cudaMemsetAsync(red, 0, (size_t)(2 + CC_MAXBLK) * sizeof(double), st));
#define KNN_TILE(T, M, S, ROWS, NROWS, KK, OUT, DLAST)                                                                      \
    do {                                                                                                                    \
        const size_t smem_ = knn_smem<T>(KK, M);                                                                            \
        KCUDA(cudaFuncSetAttribute(k_knn_tile<T, M, S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_));          \
        k_knn_tile<T, M, S><<<(unsigned)(((NROWS) + TQ - 1) / TQ), 256, smem_, st>>>((int)n, (int)p, KK, X, mask, sd, ROWS, \
                                                                                    (int)(NROWS), OUT, DLAST);              \
    } while (0)
    if (side) {
        if (mask) KNN_TILE(float, true, true, nullptr, n, k, nbr, nullptr);
        else KNN_TILE(float, false, true, nullptr, n, k, nbr, nullptr);
    } else {
        KCUDA(cudaMalloc((void**)&cand, (size_t)n * kk * sizeof(int)));
        KCUDA(cudaMalloc((void**)&dlast, (size_t)n * sizeof(float)));
        KCUDA(cudaMalloc((void**)&flagged, (size_t)n * sizeof(int)));
        if (mask) KNN_TILE(float, true, false, nullptr, n, kk, cand, dlast);
        else KNN_TILE(float, false, false, nullptr, n, kk, cand, dlast);
        const unsigned gr = (unsigned)((n + 7) / 8 < 148 * 32 ? (n + 7) / 8 : 148 * 32);
        if (mask) k_rerank<true><<<gr, 256, 0, st>>>((int)n, (int)p, k, kk, X, mask, cand, dlast, nbr, flagged, counters);
        else k_rerank<false><<<gr, 256, 0, st>>>((int)n, (int)p, k, kk, X, mask, cand, dlast, nbr, flagged, counters);
        KCUDA(cudaMemcpyAsync(hcount, counters, sizeof(int), cudaMemcpyDeviceToHost, st));
        KCUDA(cudaStreamSynchronize(st));
        if (hcount[0] > 0) {      // rows the shortlist could not decide: the exact pass over all candidates
            const int nf = hcount[0];
            KCUDA(cudaMalloc((void**)&nbr2, (size_t)nf * k * sizeof(int)));
            if (mask) KNN_TILE(double, true, false, flagged, nf, k, nbr2, nullptr);
            else KNN_TILE(double, false, false, flagged, nf, k, nbr2, nullptr);
            k_scatter_lists<<<(unsigned)(((long long)nf * k + 255) / 256), 256, 0, st>>>(nf, k, flagged, nbr2, nbr);
        }
    }
#undef KNN_TILE
    k_sort_lists<<<(unsigned)((n + 255) / 256), 256, 0, st>>>((int)n, k, nbr, own);
    k_count_reverse<<<(unsigned)((nk + 255) / 256), 256, 0, st>>>((int)n, k, nbr, own, extra);
    k_scan_rows<<<1, 1024, 0, st>>>((int)n, own, extra, rowptr);
    KCUDA(cudaMemcpyAsync(&nnz, rowptr + n, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    KCUDA(cudaStreamSynchronize(st));
    KCUDA(cudaMalloc((void**)&col, (size_t)(nnz ? nnz : 1) * sizeof(int)));
    KCUDA(cudaMalloc((void**)&w, (size_t)(nnz ? nnz : 1) * sizeof(float)));
    k_fill_rows<<<(unsigned)((nk + 255) / 256), 256, 0, st>>>((int)n, k, nbr, own, rowptr, cursor, col);
    {
        const unsigned g = (unsigned)((n + 7) / 8 < 148 * 16 ? (n + 7) / 8 : 148 * 16);
        int* nz = counters + 1;
        if (mask && side) k_rows_finish<true, true><<<g, 256, 0, st>>>((int)n, (int)p, phi, X, mask, sd, rowptr, col, w, nz);
        else if (mask) k_rows_finish<true, false><<<g, 256, 0, st>>>((int)n, (int)p, phi, X, mask, sd, rowptr, col, w, nz);
        else if (side) k_rows_finish<false, true><<<g, 256, 0, st>>>((int)n, (int)p, phi, X, mask, sd, rowptr, col, w, nz);
        else k_rows_finish<false, false><<<g, 256, 0, st>>>((int)n, (int)p, phi, X, mask, sd, rowptr, col, w, nz);
    }
    KCUDA(cudaMemcpyAsync(hcount + 1, counters + 1, sizeof(int), cudaMemcpyDeviceToHost, st));
    KCUDA(cudaStreamSynchronize(st));
    if (hcount[1] > 0) {          // drop the pairs whose weight underflowed (both directions go: w_ij == w_ji bitwise)
        KCUDA(cudaMalloc((void**)&rowptr2, (size_t)(n + 1) * sizeof(int64_t)));
        k_count_pos<<<(unsigned)((n + 255) / 256), 256, 0, st>>>((int)n, rowptr, w, own);
        k_scan_rows<<<1, 1024, 0, st>>>((int)n, own, nullptr, rowptr2);
        int64_t nnz2 = 0;
        KCUDA(cudaMemcpyAsync(&nnz2, rowptr2 + n, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
        KCUDA(cudaStreamSynchronize(st));
        KCUDA(cudaMalloc((void**)&col2, (size_t)(nnz2 ? nnz2 : 1) * sizeof(int)));
        KCUDA(cudaMalloc((void**)&w2, (size_t)(nnz2 ? nnz2 : 1) * sizeof(float)));
        k_compact_rows<<<(unsigned)((n + 255) / 256), 256, 0, st>>>((int)n, rowptr, col, w, rowptr2, col2, w2);
        KCUDA(cudaStreamSynchronize(st));
        cudaFree(rowptr); cudaFree(col); cudaFree(w);
        rowptr = rowptr2; col = col2; w = w2; nnz = nnz2;
        rowptr2 = nullptr; col2 = nullptr; w2 = nullptr;
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
    cudaFree(cand); cudaFree(nbr); cudaFree(own); cudaFree(extra); cudaFree(cursor); cudaFree(red); cudaFree(flagged);
    cudaFree(counters); cudaFree(nbr2); cudaFree(dlast); cudaFree(rowptr2); cudaFree(col2); cudaFree(w2);
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
