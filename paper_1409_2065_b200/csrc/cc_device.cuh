// cc_device.cuh -- device helpers shared by the kernels of libcc_b200.so: float4 arithmetic, row-group
// shuffles, and the deterministic grid reduction (no floating-point atomics anywhere).
#pragma once
#include <cuda_runtime.h>

#define CC_THREADS 256

namespace {

__device__ __forceinline__ float4 ld4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ float4 ld4s(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ void st4(float* p, float4 v) { *reinterpret_cast<float4*>(p) = v; }
__device__ __forceinline__ float4 f4(float a) { return make_float4(a, a, a, a); }
__device__ __forceinline__ float4 operator+(float4 a, float4 b) { return make_float4(a.x + b.x, a.y + b.y, a.z + b.z, a.w + b.w); }
__device__ __forceinline__ float4 operator-(float4 a, float4 b) { return make_float4(a.x - b.x, a.y - b.y, a.z - b.z, a.w - b.w); }
__device__ __forceinline__ float4 operator*(float a, float4 b) { return make_float4(a * b.x, a * b.y, a * b.z, a * b.w); }
__device__ __forceinline__ float dot4(float4 a, float4 b) { return a.x * b.x + a.y * b.y + a.z * b.z + a.w * b.w; }
__device__ __forceinline__ float4 fma4(float a, float4 b, float4 c) {
    return make_float4(fmaf(a, b.x, c.x), fmaf(a, b.y, c.y), fmaf(a, b.z, c.z), fmaf(a, b.w, c.w));
}

template <int G>
__device__ __forceinline__ unsigned group_mask() {
    if constexpr (G == 32) {
        return 0xffffffffu;
    } else {
        const unsigned lane = threadIdx.x & 31u;
        return ((1u << G) - 1u) << (lane & ~(unsigned)(G - 1));
    }
}

// Sum over the G lanes of a row group (xor butterfly: every lane gets the total, in the same order).
template <int G>
__device__ __forceinline__ float group_sum(float v, unsigned m) {
#pragma unroll
    for (int o = G / 2; o > 0; o >>= 1) v += __shfl_xor_sync(m, v, o, G);
    return v;
}

// Deterministic grid reduction of NV doubles per thread.  Every block writes its partial sums; the
// block that takes the last ticket adds all partials in a fixed order.  Returns true in thread 0 of
// that last block, with the totals in out[].  All other blocks have finished their work by then.
template <int NV, int NT = CC_THREADS>
__device__ bool grid_reduce(double (&v)[NV], double* part, unsigned int* ticket, double (&out)[NV]) {
    __shared__ double sm[NV][NT / 32];
    __shared__ bool last;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const unsigned bid = blockIdx.y * gridDim.x + blockIdx.x, nblk = gridDim.x * gridDim.y;   // 1-D or 2-D grids
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        double x = v[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
        if (lane == 0) sm[k][wid] = x;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < NV; ++k) {
            double x = 0.0;
            for (int w2 = 0; w2 < NT / 32; ++w2) x += sm[k][w2];
            part[(size_t)bid * NV + k] = x;
        }
        __threadfence();
        unsigned t = atomicAdd(ticket, 1u);
        last = (t == nblk - 1);
    }
    __syncthreads();
    if (!last) return false;
    __threadfence();
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        double x = 0.0;
        for (unsigned b = threadIdx.x; b < nblk; b += NT) x += __ldcg(&part[(size_t)b * NV + k]);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
        __syncthreads();
        if (lane == 0) sm[k][wid] = x;
        __syncthreads();
        if (threadIdx.x == 0) {
            double y = 0.0;
            for (int w2 = 0; w2 < NT / 32; ++w2) y += sm[k][w2];
            out[k] = y;
        }
    }
    if (threadIdx.x == 0) *ticket = 0u;
    return threadIdx.x == 0;
}


__device__ __forceinline__ unsigned long long global_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// Called by one thread when kernel `id` has finished all its work (see cc_scal::t_last).
template <typename S>
__device__ __forceinline__ void prof_mark(S* sc, int id) {
    const unsigned long long now = global_ns();
    if (sc->t_last) { sc->prof_ns[id] += now - sc->t_last; sc->prof_calls[id] += 1; }
    sc->t_last = now;
    atomicAdd(&sc->nlaunch, 1ULL);
}

// The kernels that carry no timer count themselves here (one thread of the grid calls it).
template <typename S>
__device__ __forceinline__ void count_launch(S* sc) {
    if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) atomicAdd(&sc->nlaunch, 1ULL);
}


// End of the reductions of one MM iteration (called by one thread): d_m = sqrt(dist^2 + eps) (PAPER.md
// L76), Phi_m = 1/2 loss + gamma pen + rho d_m (L64-L66, L109), the stop rule (reading S3), and the
// coefficients of the U update (L82) and of the shrink (L86).  `outer` = the MM WHILE node's handle in
// graph mode, else 0.
template <typename S>
__device__ __forceinline__ void finish_iteration(S* sc, double dist2, double loss, double pen, double* hist_phi,
                                                 double* hist_d, cudaGraphConditionalHandle outer) {
    const double d = sqrt(dist2 + sc->eps);
    const double phi = 0.5 * loss + sc->gamma * pen + sc->rho * d;
    const int m = sc->mm_iter;
    if (m < sc->hist_cap) { hist_phi[m] = phi; hist_d[m] = d; }
    int stop = (m + 1 >= sc->mm_maxit) ? 1 : 0;
    if (sc->tol > 0.0 && m + 1 >= sc->mm_min_it && m >= 1 &&
        sc->phi_prev - phi <= sc->tol * (1.0 + fabs(sc->phi_prev)))
        stop = 1;
    sc->dist2 = dist2; sc->loss = loss; sc->pen = pen;
    sc->d = d; sc->d_prev = d;
    sc->phi_prev = phi; sc->phi = phi;
    sc->cu = (float)(d / (d + sc->rho));
    sc->ca = (float)(sc->rho / (d + sc->rho));
    sc->cthr = (float)(sc->gamma * d / sc->rho);
    sc->mm_iter = m + 1;
    sc->stop_pending = stop;
    if (outer) cudaGraphSetConditional(outer, stop ? 0 : 1);
}

}  // namespace
