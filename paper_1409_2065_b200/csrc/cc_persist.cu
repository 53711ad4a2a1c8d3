// cc_persist.cu -- the whole MM loop of one cc_solve as ONE persistent kernel, for problems whose projection uses
// the precomputed inverse (n <= CC_INV_NMAX) and whose state fits in shared memory: `tiny`, `expression`, and the
// small instances of every test.  PAPER.md L202 is this regime: the paper's own GPU code lost to its CPU code on
// POPRES because of per-step overheads; here a kernel node inside the CUDA graph's WHILE loops costs ~5 us and an
// MM iteration was four of them (30 us on `tiny`, 57 us on `expression`).
//
// Decomposition: the columns are cut into slabs of `sw` columns, one CTA per slab, all CTAs co-resident (cooperative
// launch).  Every step of the iteration is separable over columns -- the right-hand side (L100), the projection
// A = U + Minv (D^-1 r0) (L90-L103), the U update (L82, L116) -- except the pair norms ||b_ij||^2 (a sum over the
// columns, L84/L86) and the scalars dist^2, loss, penalty (L76, L64-L66).  So a CTA keeps its slab of X, U, A', A in
// shared memory for the whole solve and one MM iteration needs two grid-wide barriers:
//   phase 1 (local)  r0, A, the slab's share of every ||b_ij||^2 and of dist^2 / loss / penalty  -> global partials
//   ---- barrier A ----
//   phase 2          every CTA adds the scalar partials in the same fixed order -> d_m, Phi_m, stop rule (S3), the
//                    update coefficients; each CTA adds the norm partials of ITS share of the pairs, shrinks them
//                    (L86-L88) and writes s, ||v||; U update of the slab, A' <- A
//   ---- barrier B ----   (the new shrink factors are visible to everybody)
// No atomics on data, every sum in a fixed order: results are reproducible run to run.  With one slab (`tiny`) the
// barriers are plain __syncthreads.
#include <cstdio>

#include "cc_device.cuh"
#include "cc_internal.h"
#include "cc_tc.cuh"

namespace {

constexpr int PT_THREADS = 512;

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// Grid-wide barrier over co-resident CTAs: a monotone arrival counter (zeroed by the host with the control block).
__device__ __forceinline__ void grid_barrier(unsigned* ctr, unsigned& target, unsigned nblk) {
    __syncthreads();
    if (nblk > 1) {
        if (threadIdx.x == 0) {
            target += nblk;
            __threadfence();                    // release the CTA's writes (cumulative over the __syncthreads above)
            atomicAdd(ctr, 1u);
            while (ld_acquire_u32(ctr) < target) { }
            __threadfence();
        }
        __syncthreads();
    }
}

// block-wide sums of NV doubles, fixed order; the totals are valid in thread 0
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double (*sm)[PT_THREADS / 32]) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
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
            for (int w2 = 0; w2 < PT_THREADS / 32; ++w2) x += sm[k][w2];
            v[k] = x;
        }
    }
}

struct pt_ctl {
    float cu, ca, cthr;
    int stop, fail;
};

// MODE 0: the inverse stays in global memory; 1: transposed copy in shared memory, 4 x 8 register tiles (FFMA);
// 2 (n <= 128): the inverse lives in TENSOR MEMORY for the whole solve (lane = row i, column = j, TF32 hi and lo) and the
// projection of a slab is one tcgen05.mma tile per iteration: M = 128 rows, N = slab columns (padded to 16), K = n, 3xTF32;
// phase 1a writes D^-1 r0 straight into the shared-memory operand (K-major, SWIZZLE_128B, hi and lo), the four warps that
// own the TMEM lanes read the products back and add z.  (`expression`: 5.1 us of the 18.9 us iteration were the FFMA tiles.)
constexpr int PT_KP = 128;                         // TMEM columns per plane of the inverse; the accumulator starts at 2 * PT_KP
__device__ __forceinline__ void pt_mma_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}\n"
        :: "r"(tmem_d), "r"(tmem_a), "l"(db), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void pt_tmem_st8(uint32_t taddr, const float (&v)[8]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                 :: "r"(taddr), "r"(__float_as_uint(v[0])), "r"(__float_as_uint(v[1])), "r"(__float_as_uint(v[2])),
                    "r"(__float_as_uint(v[3])), "r"(__float_as_uint(v[4])), "r"(__float_as_uint(v[5])),
                    "r"(__float_as_uint(v[6])), "r"(__float_as_uint(v[7])) : "memory");
}

template <int MODE>
__global__ void __launch_bounds__(PT_THREADS, 1)
k_mm_persist(int n, int ld, int sw, int rs_, int nnz, const int* __restrict__ rowptr, const int* __restrict__ rowup,
             const int* __restrict__ col, const int* __restrict__ peer, const float* __restrict__ w, float* s, float* vn,
             float* nb2, const float* __restrict__ dinv, const float* __restrict__ Minv, const float* __restrict__ X,
             const uint8_t* __restrict__ mask, float* U, float* A, float* Ap, cc_scal* sc, float* nbpart, double* spart,
             double* hist_phi, double* hist_d) {
    constexpr bool MINV_SMEM = MODE == 1, PROJ_TC = MODE == 2;
    extern __shared__ __align__(16) unsigned char pt_smem_raw[];
    __shared__ double red_s[3][PT_THREADS / 32];
    __shared__ pt_ctl ctl;
    __shared__ __align__(8) uint64_t mma_done;
    __shared__ uint32_t tmem_base_s;
    // MODE 2: the operand of D^-1 r0 comes first (1024-byte aligned): {hi, lo} x ceil(n / 32) K chunks x NP rows x 128 bytes
    const int NP = (sw + 15) & ~15, KCH = (n + 31) >> 5;
    const uint32_t opb = PROJ_TC ? ((smem_u32(pt_smem_raw) + 1023u) & ~1023u) : 0u;
    const uint32_t opsz = PROJ_TC ? (uint32_t)(2 * KCH * NP * 128) : 0u;
    unsigned char* pt_smem = PROJ_TC ? pt_smem_raw + (opb - smem_u32(pt_smem_raw)) + opsz : pt_smem_raw;
    const int tid = threadIdx.x, c = blockIdx.x, nslab = gridDim.x;
    const int c0 = c * sw;
    const int wq = (min(sw, ld - c0)) >> 2;              // float4 quads of this slab (ld and sw are multiples of 4)
    const int npairs = nnz >> 1;
    // ---- carve shared memory
    // rows of a slab are `rs_` floats apart: sw, or sw + 4 when sw / 4 is even, so that rs_ / 4 is odd and rows r .. r+7 at
    // the same quad fall into 8 different 16-byte bank groups (the pair loop reads rows scattered over the slab)
    float* Xs = reinterpret_cast<float*>(pt_smem);
    float* Us = Xs + (size_t)n * rs_;
    float* Ps = Us + (size_t)n * rs_;                    // A' (the previous projection)
    float* As = Ps + (size_t)n * rs_;
    float* Cs = As + (size_t)n * rs_;                    // D^-1 r0 (MODE 2: not there, the operand takes its place)
    float* ss = Cs + (PROJ_TC ? 0 : (size_t)n * rs_);    // shrink factors, all directed entries
    const int n4 = (n + 3) & ~3;
    float* Mv = ss + ((nnz + 3) & ~3);                   // Minv TRANSPOSED, n rows of n4 floats (rows i >= n of a column: 0), when it fits
    int* plist = reinterpret_cast<int*>(Mv + (MINV_SMEM ? (size_t)n * n4 : 0));   // upper entries (col > row), in order
    unsigned short* cols = reinterpret_cast<unsigned short*>(plist + npairs);
    unsigned short* rows = cols + nnz;
    uint8_t* Ms = reinterpret_cast<uint8_t*>(rows + nnz);    // mask slab, if any (nnz is even: 4-byte aligned)
    // one slab (the whole problem in this CTA): per-pair ||b||^2, ||v|| and w live in shared memory too and the loop never
    // touches global memory; s, ||v||, ||b||^2 go back once, after the last iteration
    const bool single = gridDim.x == 1;
    float* nbs = reinterpret_cast<float*>(Ms + (mask ? (size_t)n * rs_ : 0));
    float* vns = nbs + npairs;
    float* wps = vns + npairs;

    // ---- one-time loads
    if (tid == 0) ctl.fail = 0;
    if constexpr (PROJ_TC) {
        if (tid == 0) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(smem_u32(&mma_done)));
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        if (tid < 32) {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(smem_u32(&tmem_base_s)), "n"(512));
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
        }
        for (uint32_t t = tid; t < opsz / 4; t += PT_THREADS)      // rows >= the slab's columns and K >= n stay zero for good
            asm volatile("st.shared.f32 [%0], %1;" :: "r"(opb + 4u * t), "f"(0.f) : "memory");
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        if (tid < 128) {                                           // lane i of tensor memory = row i of the inverse
            const uint32_t tl = tmem_base_s + ((uint32_t)((tid >> 5) * 32) << 16);
            for (int j0 = 0; j0 < KCH * 32; j0 += 8) {
                float hi[8], lo[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    const float v = (tid < n && j0 + q < n) ? Minv[(size_t)tid * n + j0 + q] : 0.f;
                    split_tf32(v, hi[q], lo[q]);
                }
                pt_tmem_st8(tl + j0, hi);
                pt_tmem_st8(tl + PT_KP + j0, lo);
            }
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        }
    }
    for (int it = tid; it < n * wq; it += PT_THREADS) {
        const int i = it / wq, q = it - i * wq;
        const size_t g = (size_t)i * ld + c0 + 4 * q;
        const int o = i * rs_ + 4 * q;
        st4(Xs + o, ld4s(X + g));
        st4(Us + o, ld4s(U + g));
        st4(Ps + o, ld4s(Ap + g));
        if (mask) *reinterpret_cast<uchar4*>(Ms + o) = *reinterpret_cast<const uchar4*>(mask + g);
    }
    if (MINV_SMEM)
        for (int t = tid; t < n * n4; t += PT_THREADS) {
            const int j = t / n4, i = t - j * n4;
            Mv[t] = i < n ? Minv[(size_t)i * n + j] : 0.f;
        }
    for (int i = tid; i < n; i += PT_THREADS) {
        const int rs = rowptr[i], re = rowptr[i + 1];
        for (int e = rs; e < re; ++e) {
            cols[e] = (unsigned short)col[e];
            rows[e] = (unsigned short)i;
        }
    }
    __syncthreads();
    // upper entries in entry order: entry e is upper iff cols[e] > rows[e]; its slot = number of upper entries before it.
    // One thread per row counts its lower entries; a serial prefix over n <= 384 rows by thread 0 is cheap and runs once.
    __shared__ int pbase[CC_INV_NMAX + 1], rp_s[CC_INV_NMAX + 1];
    __shared__ float dinv_s[CC_INV_NMAX];
    for (int i = tid; i <= n; i += PT_THREADS) rp_s[i] = rowptr[i];
    for (int i = tid; i < n; i += PT_THREADS) dinv_s[i] = dinv[i];
    if (tid == 0) {
        int acc = 0;
        for (int i = 0; i < n; ++i) { pbase[i] = acc; acc += rowptr[i + 1] - rowup[i]; }
        pbase[n] = acc;
    }
    __syncthreads();
    for (int i = tid; i < n; i += PT_THREADS) {
        const int ru = rowup[i], re = rowptr[i + 1];
        for (int e = ru; e < re; ++e) plist[pbase[i] + (e - ru)] = e;
    }
    for (int e = tid; e < nnz; e += PT_THREADS) ss[e] = s[e];
    __syncthreads();
    if (single) {
        for (int k = tid; k < npairs; k += PT_THREADS) { vns[k] = vn[plist[k]]; wps[k] = w[plist[k]]; nbs[k] = nb2[plist[k]]; }
        __syncthreads();
    }

    // ---- control (identical in every CTA)
    const double gamma = sc->gamma, rho = sc->rho, eps = sc->eps, tol = sc->tol;
    const int maxit = sc->mm_maxit, min_it = sc->mm_min_it, hist_cap = sc->hist_cap;
    unsigned* bar = &sc->ticket[7];
    unsigned target = 0;
    double phi_prev = 0.0, phi = 0.0, d = sqrt(eps), dist2_t = 0.0, loss_t = 0.0, pen_t = 0.0;
    // this CTA's share of the pairs (phase 2): a contiguous range of plist
    const int k0 = (int)((long long)npairs * c / nslab), k1 = (int)((long long)npairs * (c + 1) / nslab);
    // per-phase device time of this solve, read by CTA 0 (it waits for the slowest CTA at the barriers), into the
    // control block's timer slots: 0 right-hand side, 2 projection, 3 norms + scalars, 4 shrink + update, 5 / 6 the two barriers
    const bool timing = c == 0 && tid == 0 && sc->prof_phases;
    unsigned long long tph[6] = {0, 0, 0, 0, 0, 0}, tlast = timing ? global_ns() : 0ULL;
    auto lap = [&](int k) {
        if (timing) { const unsigned long long now = global_ns(); tph[k] += now - tlast; tlast = now; }
    };
    int JS = 1;                                           // j-split of the projection (power of two <= 8)
    while (JS < 8 && ((n4 >> 2) * ((wq + 1) >> 1)) * JS * 2 <= PT_THREADS) JS *= 2;      // 32 / JS tiles per warp
    int m = 0;
    for (; m < maxit; ++m) {
        // ===== phase 1a: D^-1 r0 with the warm start z = a' (any z gives the same projection, S5):
        //   r0_i = sum_j s_ij (a'_i - a'_j) - sum_j (z_i - z_j) - (z_i - u_i) = sum_j (s_ij - 1)(a'_i - a'_j) - (a'_i - u_i)
        // (L100's right-hand side minus (I+L) z).  One row gather per entry; z = u would need a'_j and u_j.
        for (int it = tid; it < n * wq; it += PT_THREADS) {
            const int i = it / wq, q = it - i * wq;
            const int o = i * rs_ + 4 * q;
            const float4 api = ld4s(Ps + o);
            float4 acc = f4(0.f);
            const int rs = rp_s[i], re = rp_s[i + 1];
            for (int e = rs; e < re; e += 4) {        // batches of 4 entries: the four 16-byte loads before the arithmetic
                int oj[4];
                float sv[4];
                float4 pj[4];
#pragma unroll
                for (int b = 0; b < 4; ++b) {          // past the row's end: the row itself contributes exact zeros
                    oj[b] = (e + b < re ? (int)cols[e + b] : i) * rs_ + 4 * q;
                    sv[b] = e + b < re ? ss[e + b] - 1.f : 0.f;
                }
#pragma unroll
                for (int b = 0; b < 4; ++b) pj[b] = ld4s(Ps + oj[b]);
#pragma unroll
                for (int b = 0; b < 4; ++b) acc = fma4(sv[b], api - pj[b], acc);
            }
            acc = acc - (api - ld4s(Us + o));
            const float4 cv4 = dinv_s[i] * acc;
            if constexpr (PROJ_TC) {
                // element (column, j = i) of the operand: K chunk i / 32, row = column, 16-byte piece (i % 32) / 4 at position
                // piece ^ (column % 8), word i % 4
                const float cv[4] = {cv4.x, cv4.y, cv4.z, cv4.w};
                const uint32_t kb = opb + (uint32_t)((i >> 5) * NP * 128 + (i & 3) * 4), pc = (uint32_t)((i & 31) >> 2);
#pragma unroll
                for (int e2 = 0; e2 < 4; ++e2) {
                    const int colm = 4 * q + e2;
                    float h2, l2;
                    split_tf32(cv[e2], h2, l2);
                    const uint32_t ad = kb + (uint32_t)(colm * 128) + ((pc ^ (uint32_t)(colm & 7)) << 4);
                    asm volatile("st.shared.f32 [%0], %1;" :: "r"(ad), "f"(h2) : "memory");
                    asm volatile("st.shared.f32 [%0], %1;" :: "r"(ad + (uint32_t)(KCH * NP * 128)), "f"(l2) : "memory");
                }
            } else {
                st4(Cs + o, cv4);
            }
        }
        if constexpr (PROJ_TC) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        }
        __syncthreads();
        lap(0);
        // ===== phase 1b: A = z + Minv (D^-1 r0), z = a'   (the projection, L90-L103, by the inverse formed once in cc_create)
        if constexpr (PROJ_TC) {
            if (tid == 0) {
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t td = tmem_base_s + 2 * PT_KP;
                const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(NP >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
                const uint64_t d0 = ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) | ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
                const uint64_t dbh = d0 | (uint64_t)(opb >> 4), dbl = d0 | (uint64_t)((opb + (uint32_t)(KCH * NP * 128)) >> 4);
                const int nks = (n + 7) >> 3;
                for (int ks = 0; ks < nks; ++ks) {
                    const uint64_t kb = (uint64_t)((ks >> 2) * ((NP * 128) >> 4) + (ks & 3) * 2);       // K chunk, then 32 bytes per step
                    pt_mma_ts(td, tmem_base_s + 8 * ks, dbh + kb, idesc, ks > 0 ? 1u : 0u);
                    pt_mma_ts(td, tmem_base_s + 8 * ks, dbl + kb, idesc, 1u);
                    pt_mma_ts(td, tmem_base_s + PT_KP + 8 * ks, dbh + kb, idesc, 1u);
                }
                asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(smem_u32(&mma_done)) : "memory");
            }
            if (tid < 128) {
                if (!mbar_wait(smem_u32(&mma_done), (uint32_t)(m & 1))) ctl.fail = 1;
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t tl = tmem_base_s + ((uint32_t)((tid >> 5) * 32) << 16) + 2 * PT_KP;
                for (int cb = 0; cb < 4 * wq; cb += 16) {
                    uint32_t v[16];
                    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                                   "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                                 : "r"(tl + (uint32_t)cb));
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    if (tid < n) {
#pragma unroll
                        for (int q4 = 0; q4 < 4; ++q4) {
                            if (cb + 4 * q4 < 4 * wq) {
                                const int o = tid * rs_ + cb + 4 * q4;
                                st4(As + o, ld4s(Ps + o) + make_float4(__uint_as_float(v[4 * q4]), __uint_as_float(v[4 * q4 + 1]),
                                                                      __uint_as_float(v[4 * q4 + 2]), __uint_as_float(v[4 * q4 + 3])));
                            }
                        }
                    }
                }
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            }
        } else if constexpr (MINV_SMEM) {
            // register tile of 4 rows x 4 columns per thread; the sum over j is split over JS adjacent lanes (j = jp, jp + JS, ...)
            // and combined by a fixed shuffle tree, so that small problems still occupy the CTA.  Per j step: one 16-byte
            // load of D^-1 r0 and one of the transposed inverse for 16 FFMA (the one-row form was bound by shared-memory
            // wavefronts: 12.7 us of a 27.7 us iteration on `expression`).
            const int nrg = n4 >> 2, nqp = (wq + 1) >> 1, ntile = nrg * nqp;
            // lanes of a warp: jp = lane / (32 / JS) (so the 8 lanes that share a shared-memory wavefront read the same row j
            // of D^-1 r0 and of the inverse), tile = warp-slot * (32 / JS) + lane % (32 / JS); the partial sums of a tile sit
            // in lanes 32 / JS apart and are combined by xor-shuffles over those strides
            const int lpt = 32 / JS, lane = tid & 31, wid = tid >> 5;
            const int tiles_per_pass = (PT_THREADS / 32) * lpt;
            for (int base = 0; base < ntile; base += tiles_per_pass) {
                const int tile_ = base + wid * lpt + (lane % lpt);
                const bool valid = tile_ < ntile;
                const int jp = lane / lpt, tile = valid ? tile_ : 0;
                const int rg = tile / nqp, q = 2 * (tile - rg * nqp);
                const bool two = q + 1 < wq;                     // the last quad of an odd slab stands alone
                const int q1 = two ? q + 1 : q;
                float4 a0 = f4(0.f), a1 = f4(0.f), a2 = f4(0.f), a3 = f4(0.f), b0 = f4(0.f), b1 = f4(0.f), b2 = f4(0.f), b3 = f4(0.f);
                if (valid) {
#pragma unroll 2
                    for (int j = jp; j < n; j += JS) {
                        const float4 cv = ld4s(Cs + j * rs_ + 4 * q), dv4 = ld4s(Cs + j * rs_ + 4 * q1);
                        const float4 mv = ld4s(Mv + j * n4 + 4 * rg);
                        a0 = fma4(mv.x, cv, a0); a1 = fma4(mv.y, cv, a1); a2 = fma4(mv.z, cv, a2); a3 = fma4(mv.w, cv, a3);
                        b0 = fma4(mv.x, dv4, b0); b1 = fma4(mv.y, dv4, b1); b2 = fma4(mv.z, dv4, b2); b3 = fma4(mv.w, dv4, b3);
                    }
                }
                float4* acc[8] = {&a0, &a1, &a2, &a3, &b0, &b1, &b2, &b3};
                for (int o = 16; o >= lpt; o >>= 1) {
#pragma unroll
                    for (int r = 0; r < 8; ++r) {
                        acc[r]->x += __shfl_xor_sync(0xffffffffu, acc[r]->x, o); acc[r]->y += __shfl_xor_sync(0xffffffffu, acc[r]->y, o);
                        acc[r]->z += __shfl_xor_sync(0xffffffffu, acc[r]->z, o); acc[r]->w += __shfl_xor_sync(0xffffffffu, acc[r]->w, o);
                    }
                }
                if (valid && jp == 0) {
                    const int i0 = 4 * rg;
#pragma unroll
                    for (int r = 0; r < 4; ++r) {
                        if (i0 + r < n) {
                            const int o = (i0 + r) * rs_ + 4 * q;
                            st4(As + o, ld4s(Ps + o) + *acc[r]);
                            if (two) st4(As + o + 4, ld4s(Ps + o + 4) + *acc[4 + r]);
                        }
                    }
                }
            }
        } else {
            for (int it = tid; it < n * wq; it += PT_THREADS) {
                const int i = it / wq, q = it - i * wq;
                float4 acc0 = f4(0.f), acc1 = f4(0.f);
                int j = 0;
                for (; j + 1 < n; j += 2) {
                    acc0 = fma4(__ldg(Minv + (size_t)i * n + j), ld4s(Cs + j * rs_ + 4 * q), acc0);
                    acc1 = fma4(__ldg(Minv + (size_t)i * n + j + 1), ld4s(Cs + (j + 1) * rs_ + 4 * q), acc1);
                }
                if (j < n) acc0 = fma4(__ldg(Minv + (size_t)i * n + j), ld4s(Cs + j * rs_ + 4 * q), acc0);
                const int o = i * rs_ + 4 * q;
                st4(As + o, ld4s(Ps + o) + (acc0 + acc1));
            }
        }
        __syncthreads();
        lap(1);
        // ===== phase 1c: the slab's share of ||u - a||^2, the loss, every ||b_ij||^2 and ||v_ij - b_ij||^2, the penalty
        double red[3] = {0.0, 0.0, 0.0};      // dist^2, loss, penalty
        {
            float dl = 0.f, ls = 0.f;
            for (int it = tid; it < n * wq; it += PT_THREADS) {
                const int i = it / wq, q = it - i * wq;
                const int o = i * rs_ + 4 * q;
                const float4 u = ld4s(Us + o);
                const float4 t = u - ld4s(As + o);
                float4 qx = ld4s(Xs + o) - u;
                if (mask) {
                    const uchar4 mk = *reinterpret_cast<const uchar4*>(Ms + o);
                    qx.x = mk.x ? qx.x : 0.f; qx.y = mk.y ? qx.y : 0.f; qx.z = mk.z ? qx.z : 0.f; qx.w = mk.w ? qx.w : 0.f;
                }
                dl += dot4(t, t);
                ls += dot4(qx, qx);
            }
            red[0] += (double)dl;
            red[1] += (double)ls;
        }
        for (int k = tid; k < npairs; k += PT_THREADS) {
            const int e = plist[k];
            const int oi = (int)rows[e] * rs_, oj = (int)cols[e] * rs_;
            const float se = ss[e];
            float nbp = 0.f, dv = 0.f;
#pragma unroll 3
            for (int q = 0; q < wq; ++q) {
                const float4 b = ld4s(As + oi + 4 * q) - ld4s(As + oj + 4 * q);
                const float4 bp = ld4s(Ps + oi + 4 * q) - ld4s(Ps + oj + 4 * q);
                const float4 vb = fma4(se, bp, f4(0.f)) - b;
                nbp += dot4(b, b);
                dv += dot4(vb, vb);
            }
            if (single) { nbs[k] = nbp; red[2] += (double)(wps[k] * vns[k]); }
            else __stcg(nbpart + (size_t)c * nnz + e, nbp);
            red[0] += (double)dv;
        }
        if (!single)
            for (int k = k0 + tid; k < k1; k += PT_THREADS) {
                const int e = plist[k];
                red[2] += (double)(__ldg(w + e) * __ldcg(vn + e));
            }
        block_sum<3>(red, red_s);
        if (tid == 0 && !single) {
            __stcg(spart + (size_t)c * 4 + 0, red[0]);
            __stcg(spart + (size_t)c * 4 + 1, red[1]);
            __stcg(spart + (size_t)c * 4 + 2, red[2]);
        }
        lap(2);
        grid_barrier(bar, target, nslab);
        lap(4);
        // ===== phase 2: scalars (every CTA, same order), stop rule S3, coefficients
        if (tid < 32) {
            double a0 = red[0], a1 = red[1], a2 = red[2];        // one slab: thread 0 holds the totals already
            if (!single) {
                a0 = a1 = a2 = 0.0;
                for (int b = tid; b < nslab; b += 32) {
                    a0 += __ldcg(spart + (size_t)b * 4 + 0);
                    a1 += __ldcg(spart + (size_t)b * 4 + 1);
                    a2 += __ldcg(spart + (size_t)b * 4 + 2);
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    a0 += __shfl_xor_sync(0xffffffffu, a0, o);
                    a1 += __shfl_xor_sync(0xffffffffu, a1, o);
                    a2 += __shfl_xor_sync(0xffffffffu, a2, o);
                }
            }
            if (tid == 0) {
                dist2_t = a0; loss_t = a1; pen_t = a2;
                d = sqrt(a0 + eps);                                  // L76
                phi = 0.5 * a1 + gamma * a2 + rho * d;               // L64-L66, L109
                int stop = (m + 1 >= maxit) ? 1 : 0;
                if (tol > 0.0 && m + 1 >= min_it && m >= 1 && phi_prev - phi <= tol * (1.0 + fabs(phi_prev))) stop = 1;
                phi_prev = phi;
                ctl.cu = (float)(d / (d + rho));
                ctl.ca = (float)(rho / (d + rho));
                ctl.cthr = (float)(gamma * d / rho);
                ctl.stop = stop;
                if (c == 0 && m < hist_cap) { hist_phi[m] = phi; hist_d[m] = d; }
            }
        }
        __syncthreads();
        const float cu = ctl.cu, ca = ctl.ca, cthr = ctl.cthr;
        const int stop = ctl.stop;
        // ===== phase 2: this CTA's pairs -- add the slabs' partial norms in order, block soft-threshold (L86-L88, S6)
        if (nslab > 1) {
            // a warp per pair: the lanes add the slabs' partials b = lane, lane + 32, ... then combine in a fixed tree
            const int lane = tid & 31, wid = tid >> 5;
            for (int k = k0 + wid; k < k1; k += PT_THREADS / 32) {
                const int e = plist[k];
                float q = 0.f;
                for (int b = lane; b < nslab; b += 32) q += __ldcg(nbpart + (size_t)b * nnz + e);
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) q += __shfl_xor_sync(0xffffffffu, q, o);
                if (lane == 0) {
                    const int pe = __ldg(peer + e);
                    const float nb = sqrtf(q);
                    const float thr = cthr * __ldg(w + e);
                    const float sn = nb <= thr ? 0.f : 1.f - thr / nb;
                    s[e] = sn; s[pe] = sn;
                    vn[e] = sn * nb; vn[pe] = sn * nb;
                    nb2[e] = q; nb2[pe] = q;
                }
            }
        } else {
            for (int k = tid; k < npairs; k += PT_THREADS) {
                const int e = plist[k], pe = __ldg(peer + e);
                const float nb = sqrtf(nbs[k]);
                const float thr = cthr * wps[k];
                const float sn = nb <= thr ? 0.f : 1.f - thr / nb;
                ss[e] = sn; ss[pe] = sn;
                vns[k] = sn * nb;
            }
        }
        // ===== phase 2: U update (L82, L116), A' <- A
        for (int it = tid; it < n * wq; it += PT_THREADS) {
            const int i = it / wq, q = it - i * wq;
            const int o = i * rs_ + 4 * q;
            const float4 a = ld4s(As + o), u = ld4s(Us + o);
            float4 y = ld4s(Xs + o);
            if (mask) {
                const uchar4 mk = *reinterpret_cast<const uchar4*>(Ms + o);
                y.x = mk.x ? y.x : u.x; y.y = mk.y ? y.y : u.y; y.z = mk.z ? y.z : u.z; y.w = mk.w ? y.w : u.w;
            }
            st4(Us + o, fma4(cu, y, ca * a));
            st4(Ps + o, a);
        }
        lap(3);
        grid_barrier(bar, target, nslab);
        lap(5);
        if (stop) { ++m; break; }
        if (!single) {
            for (int e = tid; e < nnz; e += PT_THREADS) ss[e] = __ldcg(s + e);
            __syncthreads();
        }
    }
    if (single && m > 0) {
        for (int k = tid; k < npairs; k += PT_THREADS) {
            const int e = plist[k], pe = peer[e];
            s[e] = ss[e]; s[pe] = ss[e];
            vn[e] = vns[k]; vn[pe] = vns[k];
            nb2[e] = nbs[k]; nb2[pe] = nbs[k];
        }
    }
    // ---- state back to global memory (what cc_get_U, cc_clusters and the next solve read)
    for (int it = tid; it < n * wq; it += PT_THREADS) {
        const int i = it / wq, q = it - i * wq;
        const size_t g = (size_t)i * ld + c0 + 4 * q;
        const int o = i * rs_ + 4 * q;
        st4(U + g, ld4s(Us + o));
        st4(Ap + g, ld4s(Ps + o));
        if (m > 0) st4(A + g, ld4s(As + o));
    }
    if constexpr (PROJ_TC) {
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (tid < 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem_base_s), "n"(512));
        if (tid == 0 && ctl.fail) sc->cg_failed = 2;
    }
    if (c == 0 && tid == 0) {
        sc->mm_iter = m;
        sc->dist2 = dist2_t; sc->loss = loss_t; sc->pen = pen_t;
        sc->d = d; sc->d_prev = d;
        sc->phi = phi; sc->phi_prev = phi_prev;
        sc->cu = ctl.cu; sc->ca = ctl.ca; sc->cthr = ctl.cthr;
        sc->stop_pending = 1;
        sc->mm_active = 0;
        atomicAdd(&sc->nlaunch, 1ULL);
        const int slot[6] = {0, 2, 3, 4, 5, 6};
        for (int k = 0; k < 6; ++k) { sc->prof_ns[slot[k]] += tph[k]; sc->prof_calls[slot[k]] += (unsigned long long)m; }
    }
}

}  // namespace

// ---- host side -----------------------------------------------------------------------------------------------------
static int persist_stride(int sw) { return ((sw >> 2) & 1) ? sw : sw + 4; }

// mode: 0 inverse in global memory, 1 transposed copy in shared memory, 2 inverse in tensor memory (n <= 128)
static size_t persist_smem(const cc_handle* h, int sw, int mode) {
    const size_t n = (size_t)h->n, nnz = (size_t)h->nnz, rs = (size_t)persist_stride(sw);
    size_t b = (mode == 2 ? 4 : 5) * n * rs * sizeof(float) + ((nnz + 3) & ~(size_t)3) * sizeof(float);
    if (mode == 1) b += n * ((n + 3) & ~(size_t)3) * sizeof(float);
    if (mode == 2) b += 1024 + 2 * ((n + 31) / 32) * (size_t)((sw + 15) & ~15) * 128;     // alignment + the operand of D^-1 r0
    b += (nnz / 2) * sizeof(int) + 2 * nnz * sizeof(unsigned short);
    if (h->mask) b += n * rs;
    if ((h->ld + sw - 1) / sw == 1) b += 3 * (nnz / 2) * sizeof(float);      // one slab: per-pair arrays
    return b + 16;
}
static const void* persist_fn(int mode) {
    return mode == 2 ? (const void*)k_mm_persist<2> : mode == 1 ? (const void*)k_mm_persist<1> : (const void*)k_mm_persist<0>;
}

// Decide whether this handle runs the persistent kernel, and with which slab width.  Called once from cc_create after
// the inverse exists.  Leaves h->pt_slabs = 0 when the handle stays on the CUDA-graph path.
int ccp_setup(cc_handle* h) {
    h->pt_slabs = 0;
    if (h->dense || !h->Minv || h->inv_wide || !h->prm.use_graph || h->n > CC_INV_NMAX) return CC_OK;
    int dev = 0, coop = 0, maxsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) != cudaSuccess || !coop) {
        cudaGetLastError();
        return CC_OK;
    }
    cudaDeviceGetAttribute(&maxsm, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    // slab width: enough columns that the n x n x sw products of the projection outweigh a barrier (~64k FMA), and at
    // least ld / #SM so that the slabs fit the GPU in one co-resident wave
    const long long n = h->n, ld = h->ld;
    long long sw = (65536 + n * n - 1) / (n * n);
    const long long per_sm = (ld + h->sms - 1) / h->sms;
    if (sw < per_sm) sw = per_sm;
    sw = (sw + 3) / 4 * 4;
    if (sw > ld) sw = ld;
    for (;; sw += 4) {            // shrink nothing: a wider slab only lowers the CTA count; stop when it cannot fit
        const int nslab = (int)((ld + sw - 1) / sw);
        int mode = (n <= 128 && sw <= 256) ? 2 : 1;
        size_t need = persist_smem(h, (int)sw, mode);
        if (need > (size_t)maxsm && mode == 2) { mode = 1; need = persist_smem(h, (int)sw, 1); }
        if (need > (size_t)maxsm) { mode = 0; need = persist_smem(h, (int)sw, 0); }
        if (need > (size_t)maxsm) return CC_OK;            // does not fit at the narrowest admissible slab: graph path
        if (nslab > h->sms) { if (sw >= ld) return CC_OK; continue; }
        const void* fn = persist_fn(mode);
        if (cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)need) != cudaSuccess) {
            cudaGetLastError();
            return CC_OK;
        }
        int occ = 0;
        cudaError_t eo = mode == 2 ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_mm_persist<2>, PT_THREADS, need)
                       : mode == 1 ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_mm_persist<1>, PT_THREADS, need)
                                   : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_mm_persist<0>, PT_THREADS, need);
        if (eo != cudaSuccess || occ < 1) {
            cudaGetLastError();
            return CC_OK;
        }
        h->pt_slabs = nslab;
        h->pt_sw = (int)sw;
        h->pt_minv_smem = mode;
        h->pt_smem = need;
        break;
    }
    cudaError_t e = cc_dev_alloc((void**)&h->pt_nbpart, (size_t)h->pt_slabs * (h->nnz ? h->nnz : 1) * sizeof(float), h->stream);
    if (e == cudaSuccess) e = cc_dev_alloc((void**)&h->pt_spart, (size_t)h->pt_slabs * 4 * sizeof(double), h->stream);
    if (e != cudaSuccess) { cudaGetLastError(); h->pt_slabs = 0; }
    return CC_OK;
}

int ccp_solve(cc_handle* h) {
    int n = (int)h->n, ld = (int)h->ld, sw = h->pt_sw, rs = persist_stride(h->pt_sw), nnz = (int)h->nnz;
    void* args[] = {&n, &ld, &sw, &rs, &nnz, &h->rowptr, &h->rowup, &h->col, &h->peer, &h->w, &h->s, &h->vn, &h->nb2,
                    &h->dinv, &h->Minv, &h->X, &h->mask, &h->U, &h->A, &h->Ap, &h->sc, &h->pt_nbpart, &h->pt_spart,
                    &h->hist_phi, &h->hist_d};
    CC_CUDA(h, cudaLaunchCooperativeKernel(persist_fn(h->pt_minv_smem), dim3((unsigned)h->pt_slabs), dim3(PT_THREADS), args,
                                           h->pt_smem, h->stream));
    return CC_OK;
}
