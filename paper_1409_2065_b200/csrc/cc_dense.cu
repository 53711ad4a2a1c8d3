// cc_dense.cu -- a9, the complete-graph ("dense weight") form of the MM iteration, sm_100a.
//
// With E = all pairs, L = n I - 1 1^T and the projection is closed form
// (DESIGN.md / SURVEY P3):   A = U + g / (n+1),   g_i = sum_j s_ij (a'_i - a'_j) - sum_j (u_i - u_j)
//                                                   = rowsum(S)_i a'_i - (S A')_i - n (u_i - ubar),
// because 1^T g = 0.  So one iteration is two passes over pairs plus two streaming passes:
//   kd_colmeans  column means of U and A' (centring: every formula below is translation invariant)
//   kd_proj      a1+a2  the contraction S (A' - abar') tile by tile (S from HBM, n x n), A, ||U-A||^2, loss
//   kd_pairs     a3+a6  ||b_ij||^2 and ||s_ij b'_ij - b_ij||^2 by direct differences over 64 x 64 pair tiles
//                (optionally split over column ranges), d_m, Phi_m, stop rule
//   k_update     a5     (the sparse file's kernel, node part only)
//   kd_edges     a4     S, ||v|| from ||b||^2 and W, elementwise over the n x n matrices
// The contraction runs on tcgen05 (kd_proj_tc: kind::tf32, 3xTF32 split, TMEM accumulator) when n >= 128, on
// FP32 FFMA register tiles (kd_proj) for small n.  V (|E| x p: 34 GB at n=8192, p=256) is never formed.
#include <cstdio>

#include "cc_device.cuh"
#include "cc_internal.h"
#include "cc_tc.cuh"

namespace {

// ---- column means of two node arrays, deterministic two-stage ------------------------------------
// Stage 1: slice sl of the rows, a thread per column (coalesced rows), up to 256 slices so that the two passes over the
// node arrays fill the GPU (with 32 slices the grid was 64 CTAs and kd_colsum1 took 73 us per iteration at n = 8192,
// p = 256, kd_dsum1 41 us).  Stage 2: a warp per column adds the slices -- lanes stride over them, then a fixed shuffle tree.
__global__ void kd_colsum1(int n, int ld, int nslice, const float* __restrict__ U, const float* __restrict__ Ap,
                           double* __restrict__ ps, cc_scal* sc) {
    if (!sc->mm_active) return;
    count_launch(sc);
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    const int sl = blockIdx.y;
    if (c >= ld) return;
    const int r0 = (int)((long long)n * sl / nslice), r1 = (int)((long long)n * (sl + 1) / nslice);
    double su = 0.0, sa = 0.0;
    int i = r0;
    for (; i + 4 <= r1; i += 4) {          // four rows in flight
        const float u0 = U[(size_t)i * ld + c], u1 = U[(size_t)(i + 1) * ld + c], u2 = U[(size_t)(i + 2) * ld + c], u3 = U[(size_t)(i + 3) * ld + c];
        const float a0 = Ap[(size_t)i * ld + c], a1 = Ap[(size_t)(i + 1) * ld + c], a2 = Ap[(size_t)(i + 2) * ld + c], a3 = Ap[(size_t)(i + 3) * ld + c];
        su += (double)u0; su += (double)u1; su += (double)u2; su += (double)u3;
        sa += (double)a0; sa += (double)a1; sa += (double)a2; sa += (double)a3;
    }
    for (; i < r1; ++i) {
        su += (double)U[(size_t)i * ld + c];
        sa += (double)Ap[(size_t)i * ld + c];
    }
    ps[((size_t)sl * 2 + 0) * ld + c] = su;
    ps[((size_t)sl * 2 + 1) * ld + c] = sa;
}

__device__ __forceinline__ double warp_sum_slices(const double* __restrict__ p, size_t stride, int nslice, int lane) {
    double v = 0.0;
    for (int sl = lane; sl < nslice; sl += 32) v += p[(size_t)sl * stride];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__global__ void kd_colsum2(int n, int ld, int nslice, const double* __restrict__ ps, float* __restrict__ ubar,
                           float* __restrict__ abar, cc_scal* sc) {
    if (!sc->mm_active) return;
    count_launch(sc);
    const int c = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;    // a warp per column
    if (c >= ld) return;
    const double su = warp_sum_slices(ps + c, (size_t)2 * ld, nslice, lane);
    const double sa = warp_sum_slices(ps + ld + c, (size_t)2 * ld, nslice, lane);
    if (lane == 0) {
        ubar[c] = (float)(su / n);
        abar[c] = (float)(sa / n);
    }
}

// ---- kd_dsum: dbar_c = mean_i (a_ic - u_ic).  The projection satisfies 1'(A - U) = 0 exactly (1'L = 0); in fp32 the
// contraction leaves a residual of ~5e-7 (relative) per iteration in the column sums, which would add up along a
// path of thousands of iterations.  k_update subtracts dbar from A, restoring the invariant every iteration.
__global__ void kd_dsum1(int n, int ld, int nslice, const float* __restrict__ A, const float* __restrict__ U,
                         double* __restrict__ ps, cc_scal* sc) {
    if (!sc->mm_active) return;
    count_launch(sc);
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    const int sl = blockIdx.y;
    if (c >= ld) return;
    const int r0 = (int)((long long)n * sl / nslice), r1 = (int)((long long)n * (sl + 1) / nslice);
    double s = 0.0;
    int i = r0;
    for (; i + 4 <= r1; i += 4) {
        const float d0 = A[(size_t)i * ld + c] - U[(size_t)i * ld + c], d1 = A[(size_t)(i + 1) * ld + c] - U[(size_t)(i + 1) * ld + c];
        const float d2 = A[(size_t)(i + 2) * ld + c] - U[(size_t)(i + 2) * ld + c], d3 = A[(size_t)(i + 3) * ld + c] - U[(size_t)(i + 3) * ld + c];
        s += (double)d0; s += (double)d1; s += (double)d2; s += (double)d3;
    }
    for (; i < r1; ++i) s += (double)(A[(size_t)i * ld + c] - U[(size_t)i * ld + c]);
    ps[(size_t)sl * ld + c] = s;
}

__global__ void kd_dsum2(int n, int ld, int nslice, const double* __restrict__ ps, float* __restrict__ dbar, cc_scal* sc) {
    if (!sc->mm_active) return;
    count_launch(sc);
    const int c = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (c >= ld) return;
    const double s = warp_sum_slices(ps + c, (size_t)ld, nslice, lane);
    if (lane == 0) dbar[c] = (float)(s / n);
}

// ---- kd_proj ---------------------------------------------------------------------------------------
// CTA tile: BI = 16 TM rows x C = 16 TN columns, 256 threads as 16 (rows) x 16 (columns), thread tile
// TM x TN.  Loop over j in blocks of BJ = 32: stage S[I, J] (transposed) and A'[J, C] - abar in shared
// memory, rank-1 updates in registers.  Rows / columns of a thread are interleaved in groups of 4 so that
// every shared-memory read is a conflict-free 128-bit load.
constexpr int BJ = 32;

template <int TM, int TN>
__global__ void __launch_bounds__(256) kd_proj(int n, int ld, const float* __restrict__ S, const float* __restrict__ Ap,
                                               const float* __restrict__ U, const float* __restrict__ X,
                                               const uint8_t* __restrict__ mask, const float* __restrict__ ubar,
                                               const float* __restrict__ abar, float* __restrict__ A, cc_scal* sc,
                                               double* part) {
    if (!sc->mm_active) return;
    constexpr int BI = 16 * TM, C = 16 * TN;
    __shared__ __align__(16) float St[BJ][BI];
    __shared__ __align__(16) float At[BJ][C];
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    const int i0 = blockIdx.y * BI, c0 = blockIdx.x * C;
    // fp32 partial sums over one block of BJ terms, totals in fp64: at n = 8192 a single fp32 running sum of
    // s_ij (magnitude ~n) costs 1e-4 of accuracy on U after a dozen iterations (measured against the oracle)
    float acc[TM][TN], rs[TM];
    double accd[TM][TN], rsd[TM];
#pragma unroll
    for (int a = 0; a < TM; ++a) {
        rsd[a] = 0.0;
#pragma unroll
        for (int b = 0; b < TN; ++b) accd[a][b] = 0.0;
    }
    for (int j0 = 0; j0 < n; j0 += BJ) {
#pragma unroll
        for (int a = 0; a < TM; ++a) {
            rs[a] = 0.f;
#pragma unroll
            for (int b = 0; b < TN; ++b) acc[a][b] = 0.f;
        }
        for (int t = tid; t < BI * BJ; t += 256) {      // S[i0+ii][j0+jj], jj fastest: 128-byte segments
            const int jj = t % BJ, ii = t / BJ;
            const int gi = i0 + ii, gj = j0 + jj;
            St[jj][ii] = (gi < n && gj < n) ? __ldg(S + (size_t)gi * n + gj) : 0.f;
        }
        for (int t = tid; t < BJ * (C / 4); t += 256) {
            const int c4 = t % (C / 4), jj = t / (C / 4);
            const int gj = j0 + jj, gc = c0 + c4 * 4;
            float4 v = f4(0.f);
            if (gj < n && gc < ld) v = ld4s(Ap + (size_t)gj * ld + gc) - ld4s(abar + gc);
            *reinterpret_cast<float4*>(&At[jj][c4 * 4]) = v;
        }
        __syncthreads();
#pragma unroll 4
        for (int jj = 0; jj < BJ; ++jj) {
            float sv[TM], av[TN];
#pragma unroll
            for (int a4 = 0; a4 < TM / 4; ++a4) {
                const float4 v = *reinterpret_cast<const float4*>(&St[jj][a4 * 64 + ty * 4]);
                sv[a4 * 4 + 0] = v.x; sv[a4 * 4 + 1] = v.y; sv[a4 * 4 + 2] = v.z; sv[a4 * 4 + 3] = v.w;
            }
#pragma unroll
            for (int b4 = 0; b4 < TN / 4; ++b4) {
                const float4 v = *reinterpret_cast<const float4*>(&At[jj][b4 * 64 + tx * 4]);
                av[b4 * 4 + 0] = v.x; av[b4 * 4 + 1] = v.y; av[b4 * 4 + 2] = v.z; av[b4 * 4 + 3] = v.w;
            }
#pragma unroll
            for (int a = 0; a < TM; ++a) {
                rs[a] += sv[a];
#pragma unroll
                for (int b = 0; b < TN; ++b) acc[a][b] = fmaf(sv[a], av[b], acc[a][b]);
            }
        }
#pragma unroll
        for (int a = 0; a < TM; ++a) {
            rsd[a] += (double)rs[a];
#pragma unroll
            for (int b = 0; b < TN; ++b) accd[a][b] += (double)acc[a][b];
        }
        __syncthreads();
    }
    // epilogue: a = u + [rowsum(S) (a' - abar) - S(A' - abar) - n (u - ubar)] / (n+1)
    const float inv = 1.f / (float)(n + 1), fn = (float)n;
    double red[2] = {0.0, 0.0};   // ||U - A||^2, observed loss
#pragma unroll
    for (int a = 0; a < TM; ++a) {
        const int gi = i0 + (a / 4) * 64 + ty * 4 + (a % 4);
        if (gi >= n) continue;
#pragma unroll
        for (int b4 = 0; b4 < TN / 4; ++b4) {
            const int gc = c0 + b4 * 64 + tx * 4;
            if (gc >= ld) continue;
            const size_t o = (size_t)gi * ld + gc;
            const float4 ap = ld4s(Ap + o) - ld4s(abar + gc), u = ld4s(U + o), ub = ld4s(ubar + gc);
            // the two large terms are combined in fp64
            const float4 sg = make_float4((float)(rsd[a] * (double)ap.x - accd[a][b4 * 4 + 0]), (float)(rsd[a] * (double)ap.y - accd[a][b4 * 4 + 1]),
                                          (float)(rsd[a] * (double)ap.z - accd[a][b4 * 4 + 2]), (float)(rsd[a] * (double)ap.w - accd[a][b4 * 4 + 3]));
            const float4 g = sg - fn * (u - ub);
            const float4 dl = inv * g;
            st4(A + o, u + dl);
            float4 q = ld4s(X + o) - u;
            if (mask) {
                const uchar4 mk = *reinterpret_cast<const uchar4*>(mask + o);
                q.x = mk.x ? q.x : 0.f; q.y = mk.y ? q.y : 0.f; q.z = mk.z ? q.z : 0.f; q.w = mk.w ? q.w : 0.f;
            }
            red[0] += (double)dot4(dl, dl);
            red[1] += (double)dot4(q, q);
        }
    }
    double tot[2];
    if (grid_reduce<2>(red, part, &sc->ticket[0], tot)) {
        sc->dist2 = tot[0];
        sc->loss = tot[1];
        prof_mark(sc, 5);
    }
}

// ---- the contraction S (A' - abar) on the 5th-generation tensor cores: common pieces ---------------------------
// tcgen05.mma kind::tf32, M = 128 rows x N = 128 columns per CTA, fp32 accumulators in TMEM, K walked in blocks
// of 16.  fp32 accuracy is kept with the 3xTF32 split: x = hi + lo with hi = x rounded to TF32 (10 mantissa bits)
// and lo = x - hi rounded to TF32;  S A' ~= S_hi B_hi + S_hi B_lo + S_lo B_hi, three MMAs per K step into the same
// accumulator (the dropped lo*lo term is 2^-22 relative).  Operands sit in shared memory in the canonical K-major
// no-swizzle layout -- core matrices of 8 rows x 16 bytes, SBO between 8-row groups, LBO between K cores.
// The tensor core's fp32 accumulation truncates; over K = n terms that is a systematic bias (measured: U drifts 5e-8
// per MM iteration at n = 4096 against 2e-9 for FFMA, and the U update accumulates a bias by 1/kappa).  So the K blocks
// rotate over FOUR TMEM accumulators (all 512 columns) and every F_CH K blocks they are drained with tcgen05.ld into
// fp32 registers (round-to-nearest adds) and restarted: no accumulator ever sums more than F_CH / 4 K blocks (128 terms).
constexpr int TC_M = 128, TC_N = 128;
constexpr int TC_THREADS = 512, TC_WARPS = TC_THREADS / 32;
constexpr int TC_SBO = 128;                         // bytes between 8-row groups (one core matrix)
constexpr int TC_LBO = (TC_M / 8) * 128 + 16;       // bytes between K cores; +16 spreads the staging stores over banks

__device__ __forceinline__ uint64_t tc_desc(uint32_t saddr) {
    // UMMA shared-memory descriptor (cute::UMMA::SmemDescriptor): start address, LBO, SBO in 16-byte units,
    // version 1 (Blackwell), no swizzle, base offset 0
    uint64_t d = 0;
    d |= (uint64_t)((saddr >> 4) & 0x3fff);
    d |= (uint64_t)((TC_LBO >> 4) & 0x3fff) << 16;
    d |= (uint64_t)((TC_SBO >> 4) & 0x3fff) << 32;
    d |= (uint64_t)1 << 46;
    return d;
}

// ---- kd_prep_proj: the B operand (A' - abar)^T, split hi/lo ONCE per iteration, already in the tile layout (one
// contiguous F_SIDE block per column tile and K block), so that kd_proj_tc3 fetches it with one TMA bulk copy per K block

// kd_proj_tc3's operands use the SWIZZLE_128B K-major layout (what a TMA tensor map with 128-byte swizzle writes): a K
// block is 32 TF32 values = one 128-byte row per operand row; rows are stacked in 8-row atoms of 1024 bytes; inside an atom
// the 16-byte chunk c of row r sits at chunk position c ^ (r % 8).  Descriptor: layout type 2, SBO = 1024 bytes between
// 8-row groups, start address advanced by 32 bytes per K step of 8; tiles are 1024-byte aligned.  (The no-swizzle
// core-matrix layout of the other tensor kernels fed the MMAs at ~190 cycles each in this kernel, operands resident:
// measured with the staging and the TMA stubbed out.)
constexpr int FK = 32;                               // K block of kd_proj_tc3: 32 columns of S = 4 MMA K steps
constexpr int F_TILE = TC_M * FK * 4;                // bytes of one 128 x 32 operand tile (16 KB)
constexpr int F_SIDE = 2 * F_TILE;                   // hi + lo
constexpr int F_RAWT = TC_M * FK * 4;                // bytes of one raw fp32 tile of R, 128 rows x 32 columns, row-major
__device__ __forceinline__ uint32_t sw128_off(int row, int chunk) { return (uint32_t)(row * 128 + ((chunk ^ (row & 7)) << 4)); }

__global__ void __launch_bounds__(TC_THREADS) kd_prep_proj(int n, int ld, int nkb, const float* __restrict__ Ap,
                                                           const float* __restrict__ abar, uint8_t* __restrict__ Bpre,
                                                           cc_scal* sc) {
    if (!sc->mm_active) return;
    count_launch(sc);
    const int kb = blockIdx.x, ct = blockIdx.y, tid = threadIdx.x;
    const int nl = tid & 127, gc = ct * TC_N + nl;       // column of A' = a row of the N x K operand
    const bool ok = gc < ld;
    const float mean = ok ? __ldg(abar + gc) : 0.f;
    uint8_t* base = Bpre + ((size_t)ct * nkb + kb) * F_SIDE;
#pragma unroll
    for (int pass = 0; pass < 2; ++pass) {
        const int kc = (tid >> 7) + 4 * pass;            // 16-byte chunk of the row: K indices 4 kc .. 4 kc + 3
        float v[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int gk = kb * FK + kc * 4 + q;
            v[q] = (ok && gk < n) ? __ldg(Ap + (size_t)gk * ld + gc) - mean : 0.f;
        }
        float4 h, l;
        split_tf32(v[0], h.x, l.x); split_tf32(v[1], h.y, l.y); split_tf32(v[2], h.z, l.z); split_tf32(v[3], h.w, l.w);
        const uint32_t off = sw128_off(nl, kc);
        *reinterpret_cast<float4*>(base + off) = h;
        *reinterpret_cast<float4*>(base + F_TILE + off) = l;
    }
}

// The block soft-threshold factor depends on a pair only through the ratio R = w / ||b||:
//   s = max(0, 1 - thr / ||b||),  thr = (gamma d / rho) w  =>  s = max(0, 1 - cthr R),   ||b|| <= thr  <=>  cthr R >= 1.
// On the tensor-core path the pair state is ||b|| (for the penalty and the next ||v||) and R; S is never stored: the
// contraction (kd_proj_tc3), the pair epilogue (kd_pairs_tc2) and the cluster read-out recompute s_ij from R_ij and the
// threshold factor with THESE functions, so they see bit-identical factors.  ||b|| = 0 gives R = FLT_MAX: fused for every
// cthr > 0 (L88: b = 0 => v = 0), and s = 1 at the cold start's factor 0, where v = b = 0 anyway.
__device__ __forceinline__ float pair_ratio(float w, float nb) { return nb > 0.f ? fminf(__fdividef(w, nb), 3.402823466e38f) : 3.402823466e38f; }
__device__ __forceinline__ float shrink_ratio(float cthr, float R) {
    const float x = cthr * R;
    return x >= 1.f ? 0.f : 1.f - x;
}

// ---- kd_proj_tc3: shrink -> S tile -> S (A' - abar) in one kernel; S never reaches HBM ---------------
// One CTA = 128 rows x 128 columns of S (A' - abar), K = all n columns of S walked in blocks of FK = 32.  18 warps:
//   warps 0-15 (staging)  thread = (row 32 (w % 4) + lane, 8 consecutive K indices w / 4).  Per K block its 32 bytes of
//              R = w / ||b|| come in by cp.async, F_RAW K blocks deep; a thread fetches exactly what it will consume, so the
//              ring needs no barrier, only cp.async.wait_group.  The thread clamps (Rc = min(R, 1 / cthr): S = 1 - cthr Rc),
//              adds to the row sum (the flash-attention style running `l`), splits into TF32 hi + lo and writes both with
//              tcgen05.st into TENSOR MEMORY: the A operand of the MMA lives in TMEM (lane = row, column = K index), in
//              F_AST stages of 64 columns.  Each warp then arrives on the stage's `fullA` mbarrier.  A chunk of F_CH K blocks
//              accumulates in one of two accumulators; a few K blocks into the next chunk (which runs in the other
//              accumulator) the warps add the finished one to fp32 registers and arrive on its `drained` barrier.
//   warp 16, one lane     waits fullA and the B operand's fullB, issues the 12 tcgen05.mma of the K block (3xTF32, A from
//              TMEM, B from shared memory), commits freeA / freeB.
//   warp 17, one lane     keeps the B ring filled: (A' - abar)^T, pre-split once per iteration by kd_prep_proj in the
//              SWIZZLE_128B operand layout, one TMA bulk copy per K block.
// Why A in TMEM: with both operands in shared memory a kind::tf32 MMA (M128 N128 K8) reads 4 + 4 KB of shared memory for 64
// cycles of math -- all of the SM's 128 B/cycle -- and ran at ~190 cycles in this kernel whatever the layout (stub
// experiments: no staging, no TMA, operands resident: still 190).  S is produced by threads anyway, so writing it to TMEM
// costs nothing extra and halves the tensor core's shared-memory reads.
// History (n = 8192, p = 256, us for the kernel): register prefetch of ||b|| and W one block ahead 454; TMA for B two blocks
// ahead 657; cp.async for both operands, both TF32 splits in the loop 618 (194 instructions per thread and block: ptxas
// emulates cvt.rna.tf32); integer rounding, B by TMA, MMA lane also a staging thread behind __syncthreads 482; dedicated
// MMA warp, mbarrier hand-off 500; lean MMA lane (descriptor = base + constant) and separate TMA warp 400; K block 32 with
// SWIZZLE_128B operands 295; accumulators ping-pong per chunk, drains pipelined 281 -> 266 (the tensor core used to idle at
// every chunk boundary).  Stub with every wait removed (pure MMA issue): 115 us = 73 cycles per MMA; the rest is operand
// feeding: the barrier hand-shake per K block, the B ring from L2 (2 GB per launch through L2), the staging arithmetic.
constexpr int F_AST = 3, F_BST = 4, F_RAW = 4, F_CH = 16;
constexpr int F_THREADS = TC_THREADS + 64;          // 16 staging warps + the MMA warp + the TMA warp
constexpr int F_ACOL = 2 * TC_N;                     // TMEM columns 0 .. 255: two accumulators; from 256: the A stages
constexpr int F_SMEM = F_BST * F_SIDE + F_RAW * F_RAWT + 1024;

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" :: "r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const float (&v)[8]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                 :: "r"(taddr), "r"(__float_as_uint(v[0])), "r"(__float_as_uint(v[1])), "r"(__float_as_uint(v[2])),
                    "r"(__float_as_uint(v[3])), "r"(__float_as_uint(v[4])), "r"(__float_as_uint(v[5])),
                    "r"(__float_as_uint(v[6])), "r"(__float_as_uint(v[7])) : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem descriptor]
__device__ __forceinline__ void tc_mma_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}\n"
        :: "r"(tmem_d), "r"(tmem_a), "l"(db), "r"(idesc), "r"(accumulate) : "memory");
}

__global__ void __launch_bounds__(F_THREADS, 1) kd_proj_tc3(int n, int ld, int nkb, const float* __restrict__ Rm,
                                                     const uint8_t* __restrict__ Bpre,
                                                     const float* __restrict__ Ap, const float* __restrict__ U,
                                                     const float* __restrict__ X, const uint8_t* __restrict__ mask,
                                                     const float* __restrict__ ubar, const float* __restrict__ abar,
                                                     float* __restrict__ A, cc_scal* sc, double* part) {
    if (!sc->mm_active) return;
    extern __shared__ uint8_t tc_smem_raw[];
    __shared__ __align__(8) uint64_t fullA[F_AST], freeA[F_AST], fullB[F_BST], freeB[F_BST], mbar_acc, drained[2];
    __shared__ uint32_t tmem_base_s;
    __shared__ float rs_part[4][TC_M];
    __shared__ int fail_s;
    const uint32_t smB = (smem_u32(tc_smem_raw) + 1023u) & ~1023u;       // shared-space byte addresses from here on
    const uint32_t smR = smB + F_BST * F_SIDE;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int It = blockIdx.y, Ct = blockIdx.x, i0 = It * TC_M, c0 = Ct * TC_N;
    const float cthr = sc->cthr;
    if (tid == 0) {
        fail_s = 0;
        for (int b = 0; b < F_AST; ++b) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(&fullA[b])), "r"(TC_WARPS));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(smem_u32(&freeA[b])));
        }
        for (int b = 0; b < F_BST; ++b) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(smem_u32(&fullB[b])));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(smem_u32(&freeB[b])));
        }
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(smem_u32(&mbar_acc)));
        for (int b = 0; b < 2; ++b) asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(&drained[b])), "r"(TC_WARPS));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(smem_u32(&tmem_base_s)), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_d = tmem_base_s;
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(TC_N >> 3) << 17) | ((uint32_t)(TC_M >> 4) << 24);
    constexpr int TC_CPW = TC_N / (TC_WARPS / 4);
    float accr[TC_CPW];
#pragma unroll
    for (int q = 0; q < TC_CPW; ++q) accr[q] = 0.f;
    if (warp == TC_WARPS + 1) {
        // ===== TMA warp (one lane): keeps the B ring filled, up to F_BST K blocks ahead of the tensor core =====
        if (lane == 0) {
            const uint8_t* srcB = Bpre + (size_t)Ct * nkb * F_SIDE;
            for (int kb = 0; kb < nkb; ++kb) {
                const int st = kb % F_BST;
                // the stage held block kb - F_BST: its MMAs must be complete
                if (kb >= F_BST && !mbar_wait_idle(smem_u32(&freeB[st]), (uint32_t)((kb / F_BST - 1) & 1))) fail_s = 1;
                const uint32_t bar = smem_u32(&fullB[st]);
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(F_SIDE) : "memory");
                asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                             :: "r"(smB + (uint32_t)st * F_SIDE), "l"(srcB + (size_t)kb * F_SIDE), "r"(F_SIDE), "r"(bar) : "memory");
            }
        }
    } else if (warp == TC_WARPS) {
        // ===== MMA warp (one lane).  A single thread issues about one instruction every few cycles, so this loop is kept
        // lean: descriptors by adding constants to a per-stage base =====
        if (lane == 0) {
            // SWIZZLE_128B K-major descriptor: LBO unused (1), SBO = 1024 bytes, version 1, layout type 2
            const uint64_t dconst = ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) | ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
            constexpr uint64_t LO = F_TILE >> 4;                 // hi -> lo tile, in descriptor units (16 bytes)
            for (int kb = 0; kb < nkb; ++kb) {
                const int stA = kb % F_AST, stB = kb % F_BST, ch = kb / F_CH;
                // Chunk ch (F_CH K blocks) accumulates in accumulator ch % 2 while the staging warps drain the other one, so
                // the tensor core does not idle at a chunk boundary (it did, ~3.7 us each, when both accumulators restarted
                // together).  Before chunk ch >= 2 starts, the drain of chunk ch - 2 must be complete: one barrier per
                // accumulator, one phase per two chunks -- a barrier cannot run ahead of this wait.
                if (kb % F_CH == 0 && ch >= 2 && !mbar_wait(smem_u32(&drained[ch & 1]), (uint32_t)(((ch >> 1) - 1) & 1))) fail_s = 1;
                if (!mbar_wait(smem_u32(&fullA[stA]), (uint32_t)((kb / F_AST) & 1))) fail_s = 1;
                if (!mbar_wait(smem_u32(&fullB[stB]), (uint32_t)((kb / F_BST) & 1))) fail_s = 1;
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t ta = tmem_d + (uint32_t)(F_ACOL + stA * 2 * FK);      // hi at ta, lo at ta + FK columns
                const uint64_t db = dconst | (uint64_t)((smB + (uint32_t)stB * F_SIDE) >> 4);
                const uint32_t td = tmem_d + (uint32_t)((ch & 1) * TC_N);
#pragma unroll
                for (int ks = 0; ks < FK / 8; ++ks) {                        // 8 K indices: 8 TMEM columns of A, 32 bytes of B's row
                    const uint64_t ko = (uint64_t)(2 * ks);
                    tc_mma_ts(td, ta + 8 * ks, db + ko, idesc, ((kb % F_CH) > 0 || ks > 0) ? 1u : 0u);
                    tc_mma_ts(td, ta + 8 * ks, db + ko + LO, idesc, 1u);
                    tc_mma_ts(td, ta + FK + 8 * ks, db + ko, idesc, 1u);
                }
                asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(smem_u32(&freeA[stA])) : "memory");
                asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(smem_u32(&freeB[stB])) : "memory");
                if ((kb + 1) % F_CH == 0 || kb + 1 == nkb)
                    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(smem_u32(&mbar_acc)) : "memory");
            }
        }
    } else {
        // ===== staging warps =====
        const int row = (warp & 3) * 32 + lane, kq = warp >> 2, gir = i0 + row;     // TMEM lane quadrant of the warp, K octet
        const uint32_t raw_off = (uint32_t)tid * 32u;
        auto fetch = [&](int kb) {        // cp.async of this thread's 32 bytes of R for K block kb into ring slot kb % F_RAW
            if (kb < nkb) {
                const uint32_t dst = smR + (uint32_t)(kb % F_RAW) * F_RAWT + raw_off;
#pragma unroll
                for (int h2 = 0; h2 < 2; ++h2) {
                    const int gk = kb * FK + kq * 8 + 4 * h2;
                    const bool ok = gir < n && gk < n;       // n is a multiple of 4 on this path; outside: zero fill
                    cp_async16(dst + 16 * h2, Rm + (ok ? (size_t)gir * n + gk : 0), ok ? 16 : 0);
                }
            }
            asm volatile("cp.async.commit_group;" ::: "memory");     // one group per K block, empty past the end
        };
#pragma unroll
        for (int k = 0; k < F_RAW - 1; ++k) fetch(k);
        const float rcap = cthr > 0.f ? 1.f / cthr : 0.f;
        const uint32_t tlane = tmem_d + ((uint32_t)((warp & 3) * 32) << 16);
        float rsum = 0.f;
        int next_drain = 0;
        const int last_chunk = (nkb - 1) / F_CH;
        auto drain = [&](int ch) {      // chunk ch is complete in accumulator ch % 2: add it to the fp32 registers, free the accumulator
            if (!mbar_wait_idle(smem_u32(&mbar_acc), (uint32_t)(ch & 1))) fail_s = 1;
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
            for (int h2 = 0; h2 < TC_CPW / 16; ++h2) {
                uint32_t v[16];
                const uint32_t taddr = tlane + (uint32_t)((ch & 1) * TC_N + (warp >> 2) * TC_CPW + h2 * 16);
                asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                             : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                               "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                             : "r"(taddr));
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                for (int q = 0; q < 16; ++q) accr[h2 * 16 + q] += __uint_as_float(v[q]);
            }
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&drained[ch & 1]));
        };
        for (int kb = 0; kb < nkb; ++kb) {
            const int st = kb % F_AST;
            fetch(kb + F_RAW - 1);                                   // its slot held block kb - 1, which this thread has consumed
            asm volatile("cp.async.wait_group %0;" :: "n"(F_RAW - 1) : "memory");   // block kb's chunks have landed
            const uint32_t rp = smR + (uint32_t)(kb % F_RAW) * F_RAWT + raw_off;
            const float4 r4 = lds128(rp), q4 = lds128(rp + 16);
            // s = 1 - cthr min(R, 1 / cthr), and the rows of the B operand sum to zero over j (A' is centred by its column
            // mean), so  S (A' - abar) = -cthr Rc (A' - abar)  with Rc = min(R, 1 / cthr):  the operand is Rc, one FMNMX per
            // entry.  rowsum(S) = n - cthr rowsum(Rc).  Zero-filled entries (columns k >= n) contribute nothing; the diagonal
            // (R = FLT_MAX) is clamped like a fused pair, and whatever factor it gets multiplies a'_i - a'_i = 0 in the sum
            // the epilogue forms.  cthr = 0 (cold start): Rc = 0, S = 1.
            float hi[8], lo[8];
            const float rc[8] = {fminf(r4.x, rcap), fminf(r4.y, rcap), fminf(r4.z, rcap), fminf(r4.w, rcap),
                                 fminf(q4.x, rcap), fminf(q4.y, rcap), fminf(q4.z, rcap), fminf(q4.w, rcap)};
            rsum += ((rc[0] + rc[1]) + (rc[2] + rc[3])) + ((rc[4] + rc[5]) + (rc[6] + rc[7]));
#pragma unroll
            for (int q = 0; q < 8; ++q) split_tf32(rc[q], hi[q], lo[q]);
            // the MMAs of K block kb - F_AST are done: this TMEM stage is free
            if (kb >= F_AST && !mbar_wait_idle(smem_u32(&freeA[st]), (uint32_t)((kb / F_AST - 1) & 1))) fail_s = 1;
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t ta = tlane + (uint32_t)(F_ACOL + st * 2 * FK + kq * 8);
            tmem_st8(ta, hi);
            tmem_st8(ta + FK, lo);
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&fullA[st]));
            // the previous chunk's MMAs were issued F_AST K blocks ago at the latest: drain it now, a few blocks into this
            // chunk, while the tensor core works on the other accumulator
            if (kb % F_CH == F_AST + 1 && kb >= F_CH) drain(next_drain++);
        }
        while (next_drain <= last_chunk) drain(next_drain++);
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        rs_part[kq][row] = rsum;       // four K octets per row, added in a fixed order below
    }
    __syncthreads();
    // epilogue: warp w reads its rows (TMEM lanes 32 (w % 4) ..) and the column group w / 4:
    // a = u + [rowsum(S) (a' - abar) - S(A' - abar) - n (u - ubar)] / (n+1)      (closed-form projection, pin P3)
    const float inv = 1.f / (float)(n + 1), fn = (float)n;
    double red[2] = {0.0, 0.0};
    const int row = (warp & 3) * 32 + lane, gi = warp < TC_WARPS ? i0 + row : n;     // the MMA and TMA warps have no rows
    const float rs = (float)n - cthr * ((rs_part[0][row] + rs_part[1][row]) + (rs_part[2][row] + rs_part[3][row]));
#pragma unroll
    for (int cb = (warp >> 2) * TC_CPW, h2 = 0; h2 < TC_CPW / 16; cb += 16, ++h2) {
        if (gi < n) {
#pragma unroll
            for (int q4 = 0; q4 < 4; ++q4) {
                const int gc = c0 + cb + q4 * 4;
                if (gc >= ld) continue;
                const size_t o = (size_t)gi * ld + gc;
                const float4 ap = ld4s(Ap + o) - ld4s(abar + gc), u = ld4s(U + o), ub = ld4s(ubar + gc);
                const float4 sa = make_float4(-cthr * accr[h2 * 16 + q4 * 4 + 0], -cthr * accr[h2 * 16 + q4 * 4 + 1],
                                              -cthr * accr[h2 * 16 + q4 * 4 + 2], -cthr * accr[h2 * 16 + q4 * 4 + 3]);
                // the two large terms (magnitude ~n) are combined in fp64
                const float4 sg = make_float4((float)((double)rs * ap.x - sa.x), (float)((double)rs * ap.y - sa.y),
                                              (float)((double)rs * ap.z - sa.z), (float)((double)rs * ap.w - sa.w));
                const float4 g = sg - fn * (u - ub);
                const float4 dl = inv * g;
                st4(A + o, u + dl);
                float4 q = ld4s(X + o) - u;
                if (mask) {
                    const uchar4 mk = *reinterpret_cast<const uchar4*>(mask + o);
                    q.x = mk.x ? q.x : 0.f; q.y = mk.y ? q.y : 0.f; q.z = mk.z ? q.z : 0.f; q.w = mk.w ? q.w : 0.f;
                }
                red[0] += (double)dot4(dl, dl);
                red[1] += (double)dot4(q, q);
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem_d), "n"(512));
    if (tid == 0 && fail_s) sc->cg_failed = 2;
    double tot[2];
    if (grid_reduce<2, F_THREADS>(red, part, &sc->ticket[0], tot)) {
        sc->dist2 = tot[0];
        sc->loss = tot[1];
        prof_mark(sc, 5);
    }
}


// ---- kd_pairs_tc: pair norms on the tensor cores, with a direct fp32 recompute where a Gram block is not enough ---
// For a 128 x 128 tile of pairs (I <= J), with alpha = a - abar (any common shift cancels) and e = a' - a:
//   ||b||^2        = |alpha_i|^2 + |alpha_j|^2 - 2 G1,           G1 = alpha_I alpha_J^T
//   b . delta      = alpha_i.e_i - G2 - G3 + alpha_j.e_j,        G2 = alpha_I e_J^T,  G3 = e_I alpha_J^T
//   ||delta||^2    = |e_i|^2 + |e_j|^2 - 2 G4,                   G4 = e_I e_J^T          (delta = b' - b = e_i - e_j)
//   ||s b' - b||^2 = (1-s)^2 ||b||^2 - 2 s (1-s) b.delta + s^2 ||delta||^2
// -- the last line has no cancellation (each term is O(kappa^2) small), unlike an expansion around ||b||^2.
// G1..G3 use the 3xTF32 split, G4 (tiny numbers) one TF32 product: 10 tcgen05.mma per K step, four fp32
// accumulators = all 512 TMEM columns.  ||b||^2 from a Gram block carries an ABSOLUTE error ~ 3e-7 (|alpha_i|^2 +
// |alpha_j|^2); a pair whose ||b||^2 is below CC_RECOMP_REL times that scale -- every pair that is fused, about to
// fuse, or close inside a cluster -- is flagged in a shared-memory bit mask and recomputed by direct differences
// in fp32 (one warp per pair), so the fused / not-fused decision never sees Gram rounding.
constexpr int PK = 16;                               // K block: 16 columns = 4 K cores = 2 MMA K steps
constexpr int PK_TILE = (PK / 4) * TC_LBO;           // bytes of one 128 x 16 operand tile
#define CC_RECOMP_REL 1.0e-2f

// Epilogue shared by the two staging variants of kd_pairs_tc: combine the four Gram accumulators, flag and recompute.
__device__ __forceinline__ void pairs_tc_epilogue(int n, int ld, int I, int J, int i0, int j0, uint32_t tmem_d,
                                                  float (*nrm)[3][TC_M], unsigned int (*flag_s)[4], float* svbuf,
                                                  const int* fail_p, const float* __restrict__ A,
                                                  const float* __restrict__ Ap, const float* __restrict__ W,
                                                  float* NB, float* __restrict__ Rm, float cthr, cc_scal* sc, double* part,
                                                  double* hist_phi, double* hist_d, cudaGraphConditionalHandle outer) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // epilogue: warp w owns TMEM lanes 32 (w % 4) .. (its rows) and the 32-column group w / 4 of all four accumulators
    const int row = (warp & 3) * 32 + lane, gi = i0 + row, grp = warp >> 2;
    const float naI = nrm[0][0][row], aeI = nrm[0][1][row], neI = nrm[0][2][row];
    double red[2] = {0.0, 0.0};      // sum_{i<j} ||v - b||^2,  sum_{i<j} w ||v||
    unsigned int myflags = 0u;
    // this thread's places: row gi of ||b|| and R (columns j0 ..), and column gi of R (rows j0 ..: the other triangle)
    const size_t orow = (size_t)min(gi, n - 1) * n + j0;
    float* const NBr = NB + orow;
    float* const Rmr = Rm + orow;
    float* const RmT = Rm + (size_t)j0 * n + gi;
    const float* const Wr = W + orow;
    const bool diag = I == J;
#pragma unroll 1
    for (int half = 0; half < 2; ++half) {
        const int cb = grp * 32 + half * 16;
        uint32_t g[4][16];
        // this row's 16 previous ||b|| (the pairs' state: v = s b', ||v|| = s ||b'||) and weights: eight float4 loads issued
        // before the accumulators are read.  Afterwards nbp[] / wq[] are reused for the new ||b|| and the new ratios R, which
        // go to the same places (in-place: only this tile reads them; ||b|| is kept for pairs i < j only, R on both sides)
        float nbp[16], wq[16];
#pragma unroll
        for (int q4 = 0; q4 < 4; ++q4) {
            const bool ok = gi < n && j0 + cb + q4 * 4 < n;
            const float4 v = ok ? *reinterpret_cast<const float4*>(NBr + cb + q4 * 4) : f4(0.f);
            const float4 u = ok ? __ldg(reinterpret_cast<const float4*>(Wr + cb + q4 * 4)) : f4(0.f);
            nbp[q4 * 4 + 0] = v.x; nbp[q4 * 4 + 1] = v.y; nbp[q4 * 4 + 2] = v.z; nbp[q4 * 4 + 3] = v.w;
            wq[q4 * 4 + 0] = u.x; wq[q4 * 4 + 1] = u.y; wq[q4 * 4 + 2] = u.z; wq[q4 * 4 + 3] = u.w;
        }
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            const uint32_t taddr = tmem_d + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)(a * TC_N + cb);
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                         : "=r"(g[a][0]), "=r"(g[a][1]), "=r"(g[a][2]), "=r"(g[a][3]), "=r"(g[a][4]), "=r"(g[a][5]), "=r"(g[a][6]),
                           "=r"(g[a][7]), "=r"(g[a][8]), "=r"(g[a][9]), "=r"(g[a][10]), "=r"(g[a][11]), "=r"(g[a][12]),
                           "=r"(g[a][13]), "=r"(g[a][14]), "=r"(g[a][15])
                         : "r"(taddr));
        }
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        if (gi < n) {
            // the 16 pairs' sums stay in fp32 here (16 terms) and join the fp64 totals once per half
            float dvs = 0.f, pens = 0.f;
#pragma unroll
            for (int q = 0; q < 16; ++q) {
                const int cl = cb + q;
                // pairs of the tile that exist: column inside the matrix; diagonal tiles: i < j only
                const bool live = j0 + cl < n && (!diag || row < cl);
                const float naJ = nrm[1][0][cl], aeJ = nrm[1][1][cl], neJ = nrm[1][2][cl];
                // the factor of v_m = s b' (L86), recomputed as kd_proj_tc3 did, and this pair's share of the penalty of Phi_m
                const float sv = shrink_ratio(cthr, pair_ratio(wq[q], nbp[q]));
                const float pen = wq[q] * (sv * nbp[q]);
                const float nb2 = naI + naJ - 2.f * __uint_as_float(g[0][q]);
                // unflagged pairs have relative error <= 3e-7 / CC_RECOMP_REL = 3e-5 in ||b||^2, whatever the threshold.
                // ||b|| = nb2 rsqrt(nb2): 2 ulp, one MUFU (the IEEE square root was a call on the slow path); the ratio R is
                // formed from the stored ||b||, here and by every later reader, so the factors stay bit-identical
                const float nb2c = fmaxf(nb2, 0.f);
                const float nbn = nb2c > 0.f ? nb2c * rsqrtf(nb2c) : 0.f;
                const float rn = pair_ratio(wq[q], nbn);
                const bool flagged = nb2 < CC_RECOMP_REL * (naI + naJ);
                const float bd = (aeI + aeJ) - (__uint_as_float(g[1][q]) + __uint_as_float(g[2][q]));
                const float dd = fmaxf(neI + neJ - 2.f * __uint_as_float(g[3][q]), 0.f);
                const float om = 1.f - sv;
                const float dv = fmaxf(om * om * nb2 - 2.f * sv * om * bd + sv * sv * dd, 0.f);
                if (live) {
                    pens += pen;
                    nbp[q] = nbn;
                    wq[q] = rn;
                    if (flagged) {
                        myflags |= 1u << (half * 16 + q);               // recomputed directly below, with this factor
                        svbuf[row * (TC_N + 1) + cl] = sv;              // stride 129: the 32 rows of a warp fall into 32 banks
                    } else {
                        dvs += dv;
                        if (diag) { NBr[cl] = nbn; Rmr[cl] = rn; }      // diagonal tiles: guarded scalar stores (i < j only)
                        RmT[(size_t)cl * n] = rn;
                    }
                }
            }
            red[0] += (double)dvs;
            red[1] += (double)pens;
            if (!diag) {
                // off-diagonal tiles: this row's 16 values as four 16-byte stores per array (flagged entries are rewritten by
                // the recompute phase, which runs after the barrier below)
#pragma unroll
                for (int q4 = 0; q4 < 4; ++q4) {
                    if (j0 + cb + q4 * 4 < n) {
                        st4(NBr + cb + q4 * 4, make_float4(nbp[q4 * 4 + 0], nbp[q4 * 4 + 1], nbp[q4 * 4 + 2], nbp[q4 * 4 + 3]));
                        st4(Rmr + cb + q4 * 4, make_float4(wq[q4 * 4 + 0], wq[q4 * 4 + 1], wq[q4 * 4 + 2], wq[q4 * 4 + 3]));
                    }
                }
            }
        }
    }
    flag_s[row][grp] = myflags;
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem_d), "n"(512));
    // flagged pairs: direct differences in fp32, one warp per pair, rows dealt to warps round-robin (fixed order)
    for (int rr = warp; rr < TC_M; rr += TC_WARPS) {
        const int gi2 = i0 + rr;
        for (int gq = 0; gq < 4; ++gq) {
            unsigned int m = flag_s[rr][gq];
            while (m) {
                const int b = __ffs(m) - 1;
                m &= m - 1;
                const int gj2 = j0 + gq * 32 + b;
                const size_t o = (size_t)gi2 * n + gj2;
                const float sv = svbuf[rr * (TC_N + 1) + gq * 32 + b];
                float nbv = 0.f, dvv = 0.f;
                for (int c = lane * 4; c < ld; c += 128) {
                    const float4 bb = ld4s(A + (size_t)gi2 * ld + c) - ld4s(A + (size_t)gj2 * ld + c);
                    const float4 bp = ld4s(Ap + (size_t)gi2 * ld + c) - ld4s(Ap + (size_t)gj2 * ld + c);
                    const float4 tt = fma4(sv, bp, f4(0.f)) - bb;
                    nbv += dot4(bb, bb);
                    dvv += dot4(tt, tt);
                }
#pragma unroll
                for (int of = 16; of > 0; of >>= 1) {
                    nbv += __shfl_xor_sync(0xffffffffu, nbv, of);
                    dvv += __shfl_xor_sync(0xffffffffu, dvv, of);
                }
                if (lane == 0) {
                    const float nbn = sqrtf(nbv), rn = pair_ratio(__ldg(W + o), nbn);
                    NB[o] = nbn;
                    Rm[o] = rn;
                    Rm[(size_t)gj2 * n + gi2] = rn;
                    red[0] += (double)dvv;
                }
            }
        }
    }
    if (tid == 0 && *fail_p) sc->cg_failed = 2;
    double tot[2];
    if (grid_reduce<2, TC_THREADS>(red, part, &sc->ticket[3], tot)) {
        finish_iteration(sc, sc->dist2 + tot[0], sc->loss, tot[1], hist_phi, hist_d, outer);
        prof_mark(sc, 6);
    }
}

// ---- kd_pairs_tc, bulk-copy variant ------------------------------------------------------------------------------
// kd_prep_pairs splits alpha = a - abar and e = a' - a into TF32 hi/lo ONCE per iteration and writes them already in
// the tensor core's shared-memory layout: for row tile T and K block kb one contiguous 4 x PK_TILE block
// {alpha_hi, alpha_lo, e_hi, e_lo}.  kd_pairs_tc2 then needs no staging threads: one thread issues two
// cp.async.bulk (TMA 1-D) per K block -- tile I and tile J -- completing on an mbarrier, one thread issues the MMAs,
// three stages in flight.  (In kd_pairs_tc every CTA re-split both tiles: 65 times per tile at n = 8192.)
constexpr int PK_SIDE = 4 * PK_TILE;                 // bytes of one tile's four operands for one K block
constexpr int PK_NST = 3;
constexpr int PK2_SMEM = PK_NST * 2 * PK_SIDE + 1024;

__global__ void __launch_bounds__(TC_THREADS) kd_prep_pairs(int n, int ld, int nkb, const float* __restrict__ A,
                                                            const float* __restrict__ Ap, const float* __restrict__ abar,
                                                            uint8_t* __restrict__ pre, float* __restrict__ nrm_part,
                                                            int npad, cc_scal* sc) {
    if (!sc->mm_active) return;
    count_launch(sc);
    const int T = blockIdx.y, kb = blockIdx.x;
    const int tid = threadIdx.x, r = tid >> 2, kc = tid & 3;
    const int gi = T * TC_M + r, gc = kb * PK + kc * 4;
    const bool okc = gc < ld;
    const float4 mb = okc ? ld4s(abar + gc) : f4(0.f);
    const float4 a = (okc && gi < n) ? ld4s(A + (size_t)gi * ld + gc) : mb;
    const float4 pp = (okc && gi < n) ? ld4s(Ap + (size_t)gi * ld + gc) : mb;
    const float4 al = a - mb, e = pp - a;
    uint8_t* base = pre + ((size_t)T * nkb + kb) * PK_SIDE;
    const int off = kc * TC_LBO + (r >> 3) * TC_SBO + (r & 7) * 16;
    float4 h, l;
    split_tf32(al.x, h.x, l.x); split_tf32(al.y, h.y, l.y); split_tf32(al.z, h.z, l.z); split_tf32(al.w, h.w, l.w);
    *reinterpret_cast<float4*>(base + 0 * PK_TILE + off) = h;
    *reinterpret_cast<float4*>(base + 1 * PK_TILE + off) = l;
    split_tf32(e.x, h.x, l.x); split_tf32(e.y, h.y, l.y); split_tf32(e.z, h.z, l.z); split_tf32(e.w, h.w, l.w);
    *reinterpret_cast<float4*>(base + 2 * PK_TILE + off) = h;
    *reinterpret_cast<float4*>(base + 3 * PK_TILE + off) = l;
    // partial row norms of this K block (summed over kb, in order, by the consumer)
    float v0 = dot4(al, al), v1 = dot4(al, e), v2 = dot4(e, e);
    v0 += __shfl_xor_sync(0xffffffffu, v0, 1); v0 += __shfl_xor_sync(0xffffffffu, v0, 2);
    v1 += __shfl_xor_sync(0xffffffffu, v1, 1); v1 += __shfl_xor_sync(0xffffffffu, v1, 2);
    v2 += __shfl_xor_sync(0xffffffffu, v2, 1); v2 += __shfl_xor_sync(0xffffffffu, v2, 2);
    if (kc == 0) {
        float* q = nrm_part + (size_t)kb * 3 * npad + T * TC_M + r;
        q[0] = v0; q[npad] = v1; q[2 * (size_t)npad] = v2;
    }
}

__global__ void __launch_bounds__(TC_THREADS, 1) kd_pairs_tc2(int n, int ld, int ntile, int nkb, const uint8_t* __restrict__ pre,
                                                       const float* __restrict__ nrm_part, int npad,
                                                       const float* __restrict__ A, const float* __restrict__ Ap,
                                                       const float* __restrict__ W, float* NB, float* __restrict__ Rm, cc_scal* sc,
                                                       double* part, double* hist_phi, double* hist_d,
                                                       cudaGraphConditionalHandle outer) {
    if (!sc->mm_active) return;
    const float cthr = sc->cthr;     // the factor that made the current S; the last block replaces it after every block is done
    extern __shared__ uint8_t tc_smem_raw[];
    __shared__ __align__(8) uint64_t full[PK_NST], empty[PK_NST], done;
    __shared__ uint32_t tmem_base_s;
    __shared__ float nrm[2][3][TC_M];
    __shared__ unsigned int flag_s[TC_M][4];
    __shared__ int fail_s;
    uint8_t* sm = reinterpret_cast<uint8_t*>(((uintptr_t)tc_smem_raw + 1023) & ~(uintptr_t)1023);
    const int tid = threadIdx.x, warp = tid >> 5;
    int I = 0, rem = blockIdx.x;
    while (rem >= ntile - I) { rem -= ntile - I; ++I; }
    const int J = I + rem, i0 = I * TC_M, j0 = J * TC_M;
    if (tid == 0) {
        fail_s = 0;
        for (int b = 0; b < PK_NST; ++b) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(smem_u32(&full[b])));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(smem_u32(&empty[b])));
        }
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(smem_u32(&done)));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(smem_u32(&tmem_base_s)), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    if (tid < TC_M * 4) flag_s[tid >> 2][tid & 3] = 0u;
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_d = tmem_base_s;
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(TC_N >> 3) << 17) | ((uint32_t)(TC_M >> 4) << 24);

    // The epilogue reads this tile of ||b|| and W (and writes ||b|| and R) once the MMAs are done; it was bound by the
    // latency of those loads from DRAM (ncu: long-scoreboard stalls 10.8 per issue, issue slots 18 % busy).  The threads
    // have nothing to do while the tensor core works, so they pull the tile's lines into L2 now: 128 rows x 512 bytes
    // per array = 512 lines, one per thread and array.
    {
        const int pr = tid >> 2, pc = (tid & 3) * 32;
        if (i0 + pr < n && j0 + pc < n) {
            const size_t o = (size_t)(i0 + pr) * n + j0 + pc;
            asm volatile("prefetch.global.L2 [%0];" :: "l"(NB + o));
            asm volatile("prefetch.global.L2 [%0];" :: "l"(W + o));
            asm volatile("prefetch.global.L2 [%0];" :: "l"(Rm + o));
        }
    }
    if (tid == 32) {
        // ===== producer: TMA bulk copies =====
        const uint8_t* srcI = pre + (size_t)I * nkb * PK_SIDE;
        const uint8_t* srcJ = pre + (size_t)J * nkb * PK_SIDE;
        for (int kb = 0; kb < nkb; ++kb) {
            const int st = kb % PK_NST;
            if (kb >= PK_NST && !mbar_wait(smem_u32(&empty[st]), (uint32_t)((kb / PK_NST - 1) & 1))) fail_s = 1;
            const uint32_t bar = smem_u32(&full[st]);
            const uint32_t dI = smem_u32(sm + (size_t)st * 2 * PK_SIDE), dJ = dI + PK_SIDE;
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(2 * PK_SIDE) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         :: "r"(dI), "l"(srcI + (size_t)kb * PK_SIDE), "r"(PK_SIDE), "r"(bar) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         :: "r"(dJ), "l"(srcJ + (size_t)kb * PK_SIDE), "r"(PK_SIDE), "r"(bar) : "memory");
        }
    } else if (tid == 0) {
        // ===== MMA issuer =====
        for (int kb = 0; kb < nkb; ++kb) {
            const int st = kb % PK_NST;
            if (!mbar_wait(smem_u32(&full[st]), (uint32_t)((kb / PK_NST) & 1))) fail_s = 1;
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t sI = smem_u32(sm + (size_t)st * 2 * PK_SIDE), sJ = sI + PK_SIDE;
#pragma unroll
            for (int ks = 0; ks < PK / 8; ++ks) {
                const uint32_t koff = (uint32_t)(2 * ks * TC_LBO);
                const uint32_t bI = sI + koff, bJ = sJ + koff;
                const uint64_t Iah = tc_desc(bI), Ial = tc_desc(bI + PK_TILE), Ieh = tc_desc(bI + 2 * PK_TILE), Iel = tc_desc(bI + 3 * PK_TILE);
                const uint64_t Jah = tc_desc(bJ), Jal = tc_desc(bJ + PK_TILE), Jeh = tc_desc(bJ + 2 * PK_TILE), Jel = tc_desc(bJ + 3 * PK_TILE);
                const uint32_t acc = (kb > 0 || ks > 0) ? 1u : 0u;
                tc_mma(tmem_d + 0 * TC_N, Iah, Jah, idesc, acc); tc_mma(tmem_d + 0 * TC_N, Iah, Jal, idesc, 1u); tc_mma(tmem_d + 0 * TC_N, Ial, Jah, idesc, 1u);
                tc_mma(tmem_d + 1 * TC_N, Iah, Jeh, idesc, acc); tc_mma(tmem_d + 1 * TC_N, Iah, Jel, idesc, 1u); tc_mma(tmem_d + 1 * TC_N, Ial, Jeh, idesc, 1u);
                tc_mma(tmem_d + 2 * TC_N, Ieh, Jah, idesc, acc); tc_mma(tmem_d + 2 * TC_N, Ieh, Jal, idesc, 1u); tc_mma(tmem_d + 2 * TC_N, Iel, Jah, idesc, 1u);
                tc_mma(tmem_d + 3 * TC_N, Ieh, Jeh, idesc, acc);
            }
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(smem_u32(&empty[st])) : "memory");
        }
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(smem_u32(&done)) : "memory");
    } else if (tid >= 64 && tid < 64 + 2 * TC_M) {
        // ===== meanwhile: row norms = the K-block partials summed in order (same arithmetic for tile I and tile J rows)
        const int t2 = tid - 64, side = t2 / TC_M, rr = t2 % TC_M;
        const int g = (side ? j0 : i0) + rr;
        float v0 = 0.f, v1 = 0.f, v2 = 0.f;
#pragma unroll 4
        for (int kb = 0; kb < nkb; ++kb) {
            const float* q = nrm_part + (size_t)kb * 3 * npad + g;
            v0 += __ldg(q); v1 += __ldg(q + npad); v2 += __ldg(q + 2 * (size_t)npad);
        }
        nrm[side][0][rr] = v0; nrm[side][1][rr] = v1; nrm[side][2][rr] = v2;
    }
    __syncwarp();
    if (nkb > 0 && !mbar_wait(smem_u32(&done), 0u)) fail_s = 1;
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    __syncthreads();
    // every MMA is complete: the operand stages are free and serve as the 128 x 128 buffer of shrink factors
    pairs_tc_epilogue(n, ld, I, J, i0, j0, tmem_d, nrm, flag_s, reinterpret_cast<float*>(sm), &fail_s, A, Ap, W, NB, Rm, cthr, sc, part,
                      hist_phi, hist_d, outer);
}

// ---- kd_pairs --------------------------------------------------------------------------------------
// One CTA = one 64 x 64 tile of pairs (I <= J) x one range of columns (blockIdx.y of `ksplit`).  Direct
// differences (no Gram trick: a pair about to fuse has ||b|| far below ||a||, and the fused / not fused
// decision is taken on ||b||):  nb2 += b^2,  dv += (s b' - b)^2  with b = a_i - a_j, b' = a'_i - a'_j.
// Partial ||b||^2 go to NB2[ks][i][j] and [j][i]; kd_edges adds the ks slices in order.
constexpr int PT = 64, PCK = 16;

__global__ void __launch_bounds__(256) kd_pairs(int n, int ld, int ntile, int ksplit, const float* __restrict__ A,
                                                const float* __restrict__ Ap, const float* __restrict__ S,
                                                const float* __restrict__ W, const float* __restrict__ VN,
                                                float* __restrict__ NB2, cc_scal* sc, double* part, double* hist_phi,
                                                double* hist_d, cudaGraphConditionalHandle outer, int init_only) {
    if (!init_only && !sc->mm_active) return;
    __shared__ float Ai[PT][PCK + 1], Aj[PT][PCK + 1], Pi[PT][PCK + 1], Pj[PT][PCK + 1];
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    // tile index -> (I, J), I <= J, row-major over the upper triangle
    int I = 0, rem = blockIdx.x;
    while (rem >= ntile - I) { rem -= ntile - I; ++I; }
    const int J = I + rem;
    const int i0 = I * PT, j0 = J * PT;
    const int ks = blockIdx.y;
    const int cper = ((ld + ksplit - 1) / ksplit + PCK - 1) / PCK * PCK;
    const int cb = ks * cper, ce = min(ld, cb + cper);
    float sv[4][4], nb[4][4], dv[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const int gi = i0 + ty * 4 + a, gj = j0 + tx + 16 * b;
            sv[a][b] = (gi < n && gj < n && !init_only) ? __ldg(S + (size_t)gi * n + gj) : 0.f;
            nb[a][b] = 0.f;
            dv[a][b] = 0.f;
        }
    for (int c0 = cb; c0 < ce; c0 += PCK) {
        for (int t = tid; t < PT * PCK; t += 256) {
            const int r = t / PCK, c = t % PCK;
            const int gc = c0 + c;
            const bool vi = i0 + r < n && gc < ce, vj = j0 + r < n && gc < ce;
            Ai[r][c] = vi ? A[(size_t)(i0 + r) * ld + gc] : 0.f;
            Pi[r][c] = vi ? Ap[(size_t)(i0 + r) * ld + gc] : 0.f;
            Aj[r][c] = vj ? A[(size_t)(j0 + r) * ld + gc] : 0.f;
            Pj[r][c] = vj ? Ap[(size_t)(j0 + r) * ld + gc] : 0.f;
        }
        __syncthreads();
#pragma unroll
        for (int c = 0; c < PCK; ++c) {
            float ai[4], aj[4], pi[4], pj[4];
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                ai[a] = Ai[ty * 4 + a][c]; pi[a] = Pi[ty * 4 + a][c];
                aj[a] = Aj[tx + 16 * a][c]; pj[a] = Pj[tx + 16 * a][c];
            }
#pragma unroll
            for (int a = 0; a < 4; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    const float bb = ai[a] - aj[b];
                    const float tt = fmaf(sv[a][b], pi[a] - pj[b], -bb);
                    nb[a][b] = fmaf(bb, bb, nb[a][b]);
                    dv[a][b] = fmaf(tt, tt, dv[a][b]);
                }
        }
        __syncthreads();
    }
    double red[2] = {0.0, 0.0};   // sum_{i<j} ||v - b||^2,  sum_{i<j} w ||v||
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const int gi = i0 + ty * 4 + a, gj = j0 + tx + 16 * b;
            if (gi < n && gj < n && gi != gj) {
                float* out = NB2 + (size_t)ks * n * n;
                if (I != J) { out[(size_t)gi * n + gj] = nb[a][b]; out[(size_t)gj * n + gi] = nb[a][b]; }
                else out[(size_t)gi * n + gj] = nb[a][b];   // a diagonal tile holds both (i,j) and (j,i)
                if (gi < gj) {
                    red[0] += (double)dv[a][b];
                    if (ks == 0 && !init_only)
                        red[1] += (double)(__ldg(W + (size_t)gi * n + gj) * __ldg(VN + (size_t)gi * n + gj));
                }
            }
        }
    double tot[2];
    if (grid_reduce<2>(red, part, &sc->ticket[3], tot)) {
        if (!init_only) {
            finish_iteration(sc, sc->dist2 + tot[0], sc->loss, tot[1], hist_phi, hist_d, outer);
            prof_mark(sc, 6);
        }
    }
}

// ---- kd_edges: block soft-threshold over the n x n matrices; the FFMA / n <= 64 paths only, and
// since late round 2 only their cold start (inside the iteration the same arithmetic rides in k_update's launch)
// (the tensor-core path never stores S: see shrink_ratio)
__global__ void __launch_bounds__(256, 4) kd_edges(int n, int ksplit, const float* __restrict__ NB2, const float* __restrict__ W,
                                                float* __restrict__ S, float* __restrict__ VN, cc_scal* sc, double* part,
                                                int init_only) {
    if (!init_only && !sc->mm_active) return;
    const size_t nn = (size_t)n * n;
    const float cthr = sc->cthr;
    double pen[1] = {0.0};     // sum_{i<j} w ||v|| of the state written here = the penalty term of the next Phi
    // few slices: one thread per entry; many slices (small n, long rows): one warp per entry, lanes stride
    // over the slices and combine with a fixed shuffle tree (deterministic either way)
    const bool warp_per = ksplit >= 32;
    const int lane = threadIdx.x & 31;
    const long long nwork = (long long)gridDim.x * (warp_per ? blockDim.x / 32 : blockDim.x);
    for (long long e = warp_per ? (long long)blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32
                                : (long long)blockIdx.x * blockDim.x + threadIdx.x;
         e < nn; e += nwork) {
        const int i = (int)(e / n), j = (int)(e % n);
        float q = 0.f;
        if (warp_per) {
            for (int k = lane; k < ksplit; k += 32) q += NB2[(size_t)k * nn + e];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) q += __shfl_xor_sync(0xffffffffu, q, o);
            if (lane) continue;
        } else {
            q = NB2[e];
            for (int k = 1; k < ksplit; ++k) q += NB2[(size_t)k * nn + e];
        }
        float sn = 0.f, vn = 0.f;
        if (i != j) {
            const float nb = sqrtf(q);
            if (init_only) { sn = 1.f; vn = nb; }
            else {
                const float thr = cthr * W[e];
                sn = nb <= thr ? 0.f : 1.f - thr / nb;
                vn = sn * nb;
            }
        }
        S[e] = sn;
        VN[e] = vn;
        if (j > i) pen[0] += (double)(W[e] * vn);
    }
    double ptot[1];
    if (grid_reduce<1>(pen, part, &sc->ticket[7], ptot)) sc->pen_next = ptot[0];
    __syncthreads();
    if (!init_only && threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(&sc->ticket[6], 1u) == gridDim.x - 1) {
            sc->ticket[6] = 0u;
            prof_mark(sc, 7);
        }
    }
}

// tensor-core path, cold start: the pair state is ||b|| and R = w / ||b|| (S4: V0 = D U0, so ||v|| = ||b|| and s = 1,
// which the threshold factor 0 reproduces); kd_pairs wrote ||u0_i - u0_j||^2
__global__ void kd_nb_init(long long nn, float* __restrict__ NB, const float* __restrict__ W, float* __restrict__ Rm) {
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < nn; e += (long long)gridDim.x * blockDim.x) {
        const float nb = sqrtf(NB[e]);
        NB[e] = nb;
        Rm[e] = pair_ratio(W[e], nb);
    }
}

// dense-mode validation of W: symmetric, finite, > 0 off the diagonal
__global__ void kd_check_w(int n, const float* __restrict__ W, int* flag) {
    const long long nn = (long long)n * n, nt = (long long)gridDim.x * blockDim.x;
    int bad = 0;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < nn; e += nt) {
        const int i = (int)(e / n), j = (int)(e % n);
        if (i == j) continue;
        const float a = W[e];
        if (!(a >= 0.f) || isinf(a)) bad |= 64;                // F_WBAD (a zero weight is allowed here: see cc_b200.h, prm.dense)
        if (a != W[(size_t)j * n + i]) bad |= 32;              // F_WASYM
    }
    if (bad) atomicOr(flag, bad);
}

// cluster read-out on the dense S matrix: same hooking as cc_clusters.cu, neighbours = all j with s_ij = 0
__global__ void kd_lab_hook(int n, const float* __restrict__ S, int* lab, int* changed) {
    const int i = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);   // one warp per row
    const int lane = threadIdx.x & 31;
    if (i >= n) return;
    const int li = lab[i];
    int m = li;
    for (int j = lane; j < n; j += 32)
        if (j != i && S[(size_t)i * n + j] == 0.f) m = min(m, lab[j]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = min(m, __shfl_xor_sync(0xffffffffu, m, o));
    if (lane == 0 && m < li) {
        atomicMin(&lab[li], m);
        atomicMin(&lab[i], m);
        *changed = 1;
    }
}

// the same on the tensor-core path, where S is implicit: s_ij = 0 iff cthr R_ij >= 1 (shrink_ratio's own test)
__global__ void kd_lab_hook_r(int n, const float* __restrict__ Rm, float cthr, int* lab, int* changed) {
    const int i = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);   // one warp per row
    const int lane = threadIdx.x & 31;
    if (i >= n) return;
    const int li = lab[i];
    int m = li;
    for (int j = lane; j < n; j += 32)
        if (j != i && shrink_ratio(cthr, Rm[(size_t)i * n + j]) == 0.f) m = min(m, lab[j]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = min(m, __shfl_xor_sync(0xffffffffu, m, o));
    if (lane == 0 && m < li) {
        atomicMin(&lab[li], m);
        atomicMin(&lab[i], m);
        *changed = 1;
    }
}

// ---- a0 for complete graphs: W_ij = exp(-phi ||x_i - x_j||^2), all pairs (PAPER.md L127-L133 with k = n-1;
// masked distances by reading S11), optional normalisation by the sum over i<j (S8).  64 x 64 pair tiles.
template <bool MASKED>
__global__ void __launch_bounds__(256) kd_weights(int n, int p, int ntile, float phi, const float* __restrict__ X,
                                                  const uint8_t* __restrict__ mask, float* __restrict__ W,
                                                  int cols_per_slice, float* __restrict__ part) {
    __shared__ float Xi[PT][PCK + 1], Xj[PT][PCK + 1], Mi[MASKED ? PT : 1][PCK + 1], Mj[MASKED ? PT : 1][PCK + 1];
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    int I = 0, rem = blockIdx.x;
    while (rem >= ntile - I) { rem -= ntile - I; ++I; }
    const int J = I + rem, i0 = I * PT, j0 = J * PT;
    float acc[4][4], cnt[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) { acc[a][b] = 0.f; cnt[a][b] = 0.f; }
    // few tiles and many columns (52 x 200,000: one tile): blockIdx.y slices the columns, the slices' partial sums go to
    // `part` and kd_weights_fin adds them in slice order (one CTA walking all columns alone took 29 ms there)
    const int cbeg = blockIdx.y * cols_per_slice, cend = min(p, cbeg + cols_per_slice);
    for (int c0 = cbeg; c0 < cend; c0 += PCK) {
        for (int t = tid; t < PT * PCK; t += 256) {
            const int r = t / PCK, c = t % PCK, gc = c0 + c;
            const bool vi = i0 + r < n && gc < cend, vj = j0 + r < n && gc < cend;
            Xi[r][c] = vi ? X[(size_t)(i0 + r) * p + gc] : 0.f;
            Xj[r][c] = vj ? X[(size_t)(j0 + r) * p + gc] : 0.f;
            if (MASKED) {
                Mi[r][c] = vi && mask[(size_t)(i0 + r) * p + gc] ? 1.f : 0.f;
                Mj[r][c] = vj && mask[(size_t)(j0 + r) * p + gc] ? 1.f : 0.f;
            }
        }
        __syncthreads();
#pragma unroll
        for (int c = 0; c < PCK; ++c) {
#pragma unroll
            for (int a = 0; a < 4; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    const float df = Xi[ty * 4 + a][c] - Xj[tx + 16 * b][c];
                    if (MASKED) {
                        const float m = Mi[ty * 4 + a][c] * Mj[tx + 16 * b][c];
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
            const int gi = i0 + ty * 4 + a, gj = j0 + tx + 16 * b;
            if (gi < n && gj < n) {
                if (part) {
                    const size_t nn = (size_t)n * n, o = (size_t)blockIdx.y * nn * (MASKED ? 2 : 1);
                    part[o + (size_t)gi * n + gj] = acc[a][b];
                    if (I != J) part[o + (size_t)gj * n + gi] = acc[a][b];
                    if (MASKED) {
                        part[o + nn + (size_t)gi * n + gj] = cnt[a][b];
                        if (I != J) part[o + nn + (size_t)gj * n + gi] = cnt[a][b];
                    }
                    continue;
                }
                float d = acc[a][b];
                if (MASKED) d = cnt[a][b] > 0.f ? d * (float)p / cnt[a][b] : 3.0e38f;
                const float w = gi == gj ? 0.f : expf(-phi * d);
                W[(size_t)gi * n + gj] = w;
                if (I != J) W[(size_t)gj * n + gi] = w;
            }
        }
}

// Sum of the column slices of kd_weights in slice order, then the same last step: masked rescaling (S11), exp.
template <bool MASKED>
__global__ void __launch_bounds__(256) kd_weights_fin(int n, int p, int ksplit, float phi, const float* __restrict__ part,
                                                      float* __restrict__ W) {
    const size_t nn = (size_t)n * n, e = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (e >= nn) return;
    float d = 0.f, c = 0.f;
    for (int k = 0; k < ksplit; ++k) {
        d += part[(size_t)k * nn * (MASKED ? 2 : 1) + e];
        if (MASKED) c += part[(size_t)k * nn * 2 + nn + e];
    }
    if (MASKED) d = c > 0.f ? d * (float)p / c : 3.0e38f;
    W[e] = (e / n == e % n) ? 0.f : expf(-phi * d);
}

__global__ void __launch_bounds__(CC_THREADS) kd_wsum(int n, const float* __restrict__ W, double* part, unsigned int* ticket,
                                                       double* out) {
    const long long nn = (long long)n * n, nt = (long long)gridDim.x * blockDim.x;
    double acc[1] = {0.0};
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < nn; e += nt)
        if (e / n < e % n) acc[0] += (double)W[e];
    double tot[1];
    if (grid_reduce<1>(acc, part, ticket, tot)) out[0] = tot[0];
}

__global__ void kd_wscale(long long nn, float* __restrict__ W, const double* __restrict__ total) {
    const double t = total[0];
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < nn; e += (long long)gridDim.x * blockDim.x)
        W[e] = (float)((double)W[e] / t);
}

}  // namespace

// =============================================================================================
// Host side
// =============================================================================================
static const int kSliceDense = 256;      // most row slices of the column-sum kernels
static int dense_slices(const cc_handle* h) {       // about 32 rows per slice
    long long s = h->n / 32;
    return (int)(s < 1 ? 1 : (s > kSliceDense ? kSliceDense : s));
}

void ccd_colmeans(cc_handle* h) {
    const int ns = dense_slices(h);
    dim3 g1((unsigned)((h->ld + 127) / 128), (unsigned)ns);
    kd_colsum1<<<g1, 128, 0, h->stream>>>((int)h->n, (int)h->ld, ns, h->U, h->Ap, h->colps, h->sc);
    kd_colsum2<<<(unsigned)((h->ld + 7) / 8), 256, 0, h->stream>>>((int)h->n, (int)h->ld, ns, h->colps,
                                                                      h->ubar, h->abar, h->sc);
}

template <int TM, int TN>
static void launch_proj(cc_handle* h) {
    dim3 g((unsigned)((h->ld + 16 * TN - 1) / (16 * TN)), (unsigned)((h->n + 16 * TM - 1) / (16 * TM)));
    kd_proj<TM, TN><<<g, 256, 0, h->stream>>>((int)h->n, (int)h->ld, h->Sd, h->Ap, h->U, h->X, h->mask, h->ubar, h->abar,
                                              h->A, h->sc, h->part + 0 * CC_MAXBLK * CC_NPART);
}

void ccd_proj(cc_handle* h) {
    if (h->dn_tc) {
        const int nkb = (int)((h->n + FK - 1) / FK);
        dim3 g((unsigned)((h->ld + TC_N - 1) / TC_N), (unsigned)((h->n + TC_M - 1) / TC_M));
        dim3 gp((unsigned)nkb, g.x);
        kd_prep_proj<<<gp, TC_THREADS, 0, h->stream>>>((int)h->n, (int)h->ld, nkb, h->Ap, h->abar, h->pre_B, h->sc);
        kd_proj_tc3<<<g, F_THREADS, F_SMEM, h->stream>>>((int)h->n, (int)h->ld, nkb, h->Rd, h->pre_B, h->Ap, h->U, h->X,
                                                          h->mask, h->ubar, h->abar, h->A, h->sc,
                                                          h->part + 0 * CC_MAXBLK * CC_NPART);
        return;
    }
    if (!h->dn_big) launch_proj<4, 4>(h);
    else launch_proj<4, 8>(h);
}

static void launch_pairs(cc_handle* h, const float* A, const float* Ap, int init_only) {
    const int ntile = (int)((h->n + PT - 1) / PT);
    dim3 g((unsigned)(ntile * (ntile + 1) / 2), (unsigned)h->dn_ksplit);
    kd_pairs<<<g, 256, 0, h->stream>>>((int)h->n, (int)h->ld, ntile, h->dn_ksplit, A, Ap, h->Sd, h->Wd, h->VNd, h->NB2d,
                                       h->sc, h->part + 3 * CC_MAXBLK * CC_NPART, h->hist_phi, h->hist_d,
                                       init_only ? 0 : h->cond_outer, init_only);
}

void ccd_pairs(cc_handle* h) {
    if (h->dn_tc) {
        const int ntile = (int)((h->n + TC_M - 1) / TC_M), nkb = (int)((h->ld + PK - 1) / PK), npad = ntile * TC_M;
        dim3 gp((unsigned)nkb, (unsigned)ntile);
        kd_prep_pairs<<<gp, TC_THREADS, 0, h->stream>>>((int)h->n, (int)h->ld, nkb, h->A, h->Ap, h->abar, h->pre_pairs,
                                                       h->nrm_part, npad, h->sc);
        kd_pairs_tc2<<<(unsigned)(ntile * (ntile + 1) / 2), TC_THREADS, PK2_SMEM, h->stream>>>(
            (int)h->n, (int)h->ld, ntile, nkb, h->pre_pairs, h->nrm_part, npad, h->A, h->Ap, h->Wd, h->NB2d, h->Rd,
            h->sc, h->part + 3 * CC_MAXBLK * CC_NPART, h->hist_phi, h->hist_d, h->cond_outer);
        return;
    }
    launch_pairs(h, h->A, h->Ap, 0);
}

static void launch_small(cc_handle* h) { ccd_small_tc_launch(h); }      // cc_small.cu

void ccd_edges(cc_handle* h, int init_only) {
    kd_edges<<<h->grid_nodes, 256, 0, h->stream>>>((int)h->n, h->dn_ksplit, h->NB2d, h->Wd, h->Sd, h->VNd, h->sc,
                                                   h->part + 6 * CC_MAXBLK * CC_NPART, init_only);
}

void ccd_lab_hook(cc_handle* h, int* changed) {
    if (h->dn_tc)
        kd_lab_hook_r<<<(unsigned)((h->n + 7) / 8), 256, 0, h->stream>>>((int)h->n, h->Rd, h->dn_cthr, h->lab, changed);
    else
        kd_lab_hook<<<(unsigned)((h->n + 7) / 8), 256, 0, h->stream>>>((int)h->n, h->Sd, h->lab, changed);
}

// sizes, allocations and validation of the dense mode; W is copied.  Returns CC_* codes.
int ccd_setup(cc_handle* h, const float* W) {
    const int64_t n = h->n, nn = n * n;
    const int ntile = (int)((n + PT - 1) / PT);
    const long long ntp = (long long)ntile * (ntile + 1) / 2;
    h->dn_big = (n > 64 && h->ld >= 128) ? 1 : 0;
    // tensor-core path when the tile shape pays (M = 128 rows) and rows of the n x n matrices are float4-aligned; there the
    // pair state is ||b|| alone (NB2d holds ||b||, S is implicit), elsewhere S and ||v|| are stored and kd_edges makes them
    h->dn_tc = (n >= 128 && (n & 3) == 0) ? 1 : 0;
    if (h->dn_tc) {
        cudaError_t ea = cudaFuncSetAttribute(kd_pairs_tc2, cudaFuncAttributeMaxDynamicSharedMemorySize, PK2_SMEM);
        if (ea == cudaSuccess) ea = cudaFuncSetAttribute(kd_proj_tc3, cudaFuncAttributeMaxDynamicSharedMemorySize, F_SMEM);
        if (ea != cudaSuccess) { cudaGetLastError(); h->dn_tc = 0; }
    }
    long long ks = (4LL * h->sms + ntp - 1) / ntp;
    const long long ksmax = (h->ld + 63) / 64;
    if (ks > ksmax) ks = ksmax;
    if (ks < 1) ks = 1;
    if (h->dn_tc) ks = 1;                      // kd_pairs_tc2 walks all columns itself
    h->dn_ksplit = (int)ks;
    // n <= 64: the fused kernel kd_small_tc (cc_small.cu), which sets its own launch shape; its slices are (CTA, column
    // phase).  Where it cannot run (no tensor-map encoder in the driver) the FFMA tiles above serve these shapes too.
    h->dn_small = (n <= 64 && ccd_small_tc_setup(h)) ? 1 : 0;
    h->dn_small_tc = h->dn_small;
    if (h->dn_small) {
        h->dn_ksplit = h->dn_small_grid * h->dn_small_cs;
        ks = h->dn_ksplit;
    }
    const long long bproj = ((h->ld + 63) / 64) * ((n + 63) / 64);   // upper bound over the tile shapes used
    if (ntp * ks > CC_MAXBLK || bproj > CC_MAXBLK) {
        snprintf(h->err, sizeof(h->err), "dense mode: problem too large for this build (n=%lld, p=%lld)", (long long)n, (long long)h->p);
        return CC_EINVAL;
    }
    cudaError_t e = cc_dev_alloc((void**)&h->Wd, (size_t)nn * sizeof(float), h->stream);
    if (e == cudaSuccess && !h->dn_tc) e = cc_dev_alloc((void**)&h->Sd, (size_t)nn * sizeof(float), h->stream);
    if (e == cudaSuccess && !h->dn_tc) e = cc_dev_alloc((void**)&h->VNd, (size_t)nn * sizeof(float), h->stream);
    if (e != cudaSuccess) { cudaGetLastError(); snprintf(h->err, sizeof(h->err), "dense mode: cudaMalloc n*n failed"); return CC_ENOMEM; }
    e = cc_dev_alloc((void**)&h->NB2d, (size_t)nn * ks * sizeof(float), h->stream);
    if (e == cudaSuccess) e = cc_dev_alloc((void**)&h->ubar, (size_t)h->ld * sizeof(float), h->stream);
    if (e == cudaSuccess) e = cc_dev_alloc((void**)&h->abar, (size_t)h->ld * sizeof(float), h->stream);
    if (e == cudaSuccess && (!h->dn_small || h->dn_small_tc)) e = cc_dev_alloc((void**)&h->dbar, (size_t)h->ld * sizeof(float), h->stream);
    if (e == cudaSuccess && h->dbar) e = cudaMemsetAsync(h->dbar, 0, (size_t)h->ld * sizeof(float), h->stream);
    if (e == cudaSuccess) e = cc_dev_alloc((void**)&h->colps, (size_t)kSliceDense * 2 * h->ld * sizeof(double), h->stream);
    if (e != cudaSuccess) { cudaGetLastError(); snprintf(h->err, sizeof(h->err), "dense mode: cudaMalloc failed"); return CC_ENOMEM; }
    if (h->dn_tc) {
        const size_t ntile = (size_t)((n + TC_M - 1) / TC_M), nkb = (size_t)((h->ld + PK - 1) / PK);
        e = cc_dev_alloc((void**)&h->pre_pairs, ntile * nkb * PK_SIDE, h->stream);
        const size_t nkb16 = (size_t)((n + FK - 1) / FK), nct = (size_t)((h->ld + TC_N - 1) / TC_N);
        if (e == cudaSuccess) e = cc_dev_alloc((void**)&h->pre_B, nct * nkb16 * F_SIDE, h->stream);
        if (e == cudaSuccess) e = cc_dev_alloc((void**)&h->Rd, (size_t)nn * sizeof(float), h->stream);
        if (e == cudaSuccess) e = cc_dev_alloc((void**)&h->nrm_part, nkb * 3 * ntile * TC_M * sizeof(float), h->stream);
        if (e != cudaSuccess) { cudaGetLastError(); snprintf(h->err, sizeof(h->err), "dense mode: cudaMalloc failed"); return CC_ENOMEM; }
    }
    CC_CUDA(h, cudaMemcpyAsync(h->Wd, W, (size_t)nn * sizeof(float), cudaMemcpyDeviceToDevice, h->stream));
    CC_CUDA(h, cudaMemsetAsync(h->NB2d, 0, (size_t)nn * ks * sizeof(float), h->stream));
    if (h->Sd) CC_CUDA(h, cudaMemsetAsync(h->Sd, 0, (size_t)nn * sizeof(float), h->stream));
    if (h->VNd) CC_CUDA(h, cudaMemsetAsync(h->VNd, 0, (size_t)nn * sizeof(float), h->stream));
    kd_check_w<<<h->grid_nodes, 256, 0, h->stream>>>((int)n, h->Wd, h->dflag);
    h->nnz = n * (n - 1);
    h->npairs = h->nnz / 2;
    h->launches += 1;
    return CC_OK;
}

// sum_{i<j} w_ij^2 for the rho rule (S1): reuse kd_pairs' reduction machinery would be overkill; a plain
// deterministic kernel over the upper triangle.
namespace {
__global__ void __launch_bounds__(CC_THREADS) kd_sumw2(int n, const float* __restrict__ W, double* part, unsigned int* ticket,
                                                        double* out) {
    const long long nn = (long long)n * n, nt = (long long)gridDim.x * blockDim.x;
    double acc[1] = {0.0};
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < nn; e += nt) {
        const int i = (int)(e / n), j = (int)(e % n);
        if (i < j) { const double w = (double)W[e]; acc[0] += w * w; }
    }
    double tot[1];
    if (grid_reduce<1>(acc, part, ticket, tot)) out[1] = tot[0];
}
}  // namespace

void ccd_sumw2(cc_handle* h) {
    kd_sumw2<<<h->grid_nodes, CC_THREADS, 0, h->stream>>>((int)h->n, h->Wd, h->part + 5 * CC_MAXBLK * CC_NPART,
                                                         &h->sc->ticket[5], h->dout);
}

// cold start of the pair state (S4: V0 = D U0): s = 1, ||v_ij|| = ||u0_i - u0_j||
void ccd_init_state(cc_handle* h) {
    const size_t bytes = (size_t)h->n * h->ld * sizeof(float);
    cudaMemcpyAsync(h->Ap, h->U, bytes, cudaMemcpyDeviceToDevice, h->stream);
    if (h->dn_small) {                         // this path keeps the previous projection as (A, dbar): A = U0, dbar = 0
        cudaMemcpyAsync(h->A, h->U, bytes, cudaMemcpyDeviceToDevice, h->stream);
        cudaMemsetAsync(h->dbar, 0, (size_t)h->ld * sizeof(float), h->stream);
    }
    launch_pairs(h, h->U, h->U, 1);            // ||u0_i - u0_j||^2 by direct differences (every dense path starts here)
    if (h->dn_tc) {
        kd_nb_init<<<h->grid_nodes, 256, 0, h->stream>>>((long long)h->n * h->n, h->NB2d, h->Wd, h->Rd);
        h->dn_cthr = 0.f;                      // threshold factor 0: s = 1 wherever ||b|| > 0
    } else {
        ccd_edges(h, 1);
    }
    h->launches += 2;
}

void ccd_iteration(cc_handle* h) {
    if (h->dn_small) {
        launch_small(h);
        ccs_update_nodes(h, 1, 0);             // the block soft-threshold over the n x n matrices rides along (kd_edges' work);
                                               // no A' = A - dbar is stored: kd_small_tc reads A and dbar
        return;
    }
    ccd_colmeans(h);
    ccd_proj(h);
    {
        const int ns = dense_slices(h);
        dim3 g1((unsigned)((h->ld + 127) / 128), (unsigned)ns);
        kd_dsum1<<<g1, 128, 0, h->stream>>>((int)h->n, (int)h->ld, ns, h->A, h->U, h->colps, h->sc);
        kd_dsum2<<<(unsigned)((h->ld + 7) / 8), 256, 0, h->stream>>>((int)h->n, (int)h->ld, ns, h->colps, h->dbar, h->sc);
    }
    ccd_pairs(h);
    ccs_update_nodes(h, h->dn_tc ? 0 : 1, 1);  // the tensor-core path keeps ||b|| only: no pass over the n x n matrices
}

int ccd_solve_eager(cc_handle* h, int maxit) {
    h->cond_inner = 0;
    h->cond_outer = 0;
    for (int it = 0; it < maxit; ++it) {
        ccs_begin_iter(h);
        ccd_iteration(h);
        CC_CUDA(h, cudaMemcpyAsync(h->sc_host, h->sc, sizeof(cc_scal), cudaMemcpyDeviceToHost, h->stream));
        CC_CUDA(h, cudaStreamSynchronize(h->stream));
        if (!h->sc_host->mm_active || h->sc_host->stop_pending) break;
    }
    CC_CUDA(h, cudaGetLastError());
    return CC_OK;
}

// graph:  WHILE(outer){ kd_colsum1; kd_colsum2; [kd_prep_proj;] kd_proj*; kd_dsum1; kd_dsum2; [kd_prep_pairs;] kd_pairs*; k_update }   or   WHILE(outer){ kd_small_tc; k_update }
int ccd_build_graph(cc_handle* h) {
    if (h->gexec) return CC_OK;
    cudaStream_t cap;
    CC_CUDA(h, cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
    cudaStream_t user = h->stream;
    CC_CUDA(h, cudaGraphCreate(&h->graph, 0));
    CC_CUDA(h, cudaGraphConditionalHandleCreate(&h->cond_outer, h->graph, 1, cudaGraphCondAssignDefault));
    cudaGraphNodeParams op = {};
    op.type = cudaGraphNodeTypeConditional;
    op.conditional.handle = h->cond_outer;
    op.conditional.type = cudaGraphCondTypeWhile;
    op.conditional.size = 1;
    cudaGraphNode_t onode;
    CC_CUDA(h, cudaGraphAddNode(&onode, h->graph, nullptr, 0, &op));
    cudaGraph_t og = op.conditional.phGraph_out[0];
    h->stream = cap;
    cudaError_t e = cudaStreamBeginCaptureToGraph(cap, og, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed);
    if (e == cudaSuccess) {
        ccd_iteration(h);
        e = cudaStreamEndCapture(cap, nullptr);
    }
    h->stream = user;
    cudaStreamDestroy(cap);
    if (e != cudaSuccess) {
        snprintf(h->err, sizeof(h->err), "building the dense solve graph: %s", cudaGetErrorString(e));
        return CC_ECUDA;
    }
    CC_CUDA(h, cudaGraphInstantiate(&h->gexec, h->graph, 0));
    return CC_OK;
}


extern "C" int cc_dense_weights(int64_t n, int64_t p, const float* X, const uint8_t* mask, float phi, int32_t normalize,
                                float* W_out, void* stream) {
    if (!X || !W_out || n < 2 || p < 1 || !(phi >= 0.f) || n > 46340) {
        snprintf(cc_g_err, sizeof(cc_g_err), "cc_dense_weights: need n in [2, 46340], p >= 1, phi >= 0, non-NULL pointers");
        return CC_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const int ntile = (int)((n + PT - 1) / PT);
    const unsigned grid = (unsigned)(ntile * (ntile + 1) / 2);
    cudaError_t e = cudaSuccess;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    // column slices when the pair tiles alone cannot fill the GPU: about two CTAs per SM, at least 8 column blocks per slice
    long long ksplit = grid >= (unsigned)sms ? 1 : (2LL * sms + grid - 1) / grid;
    const long long kmax = (p + 8LL * PCK - 1) / (8LL * PCK);
    if (ksplit > kmax) ksplit = kmax;
    if (ksplit <= 1) {
        if (mask) kd_weights<true><<<grid, 256, 0, st>>>((int)n, (int)p, ntile, phi, X, mask, W_out, (int)p, nullptr);
        else kd_weights<false><<<grid, 256, 0, st>>>((int)n, (int)p, ntile, phi, X, mask, W_out, (int)p, nullptr);
    } else {
        const long long cols = ((p + ksplit - 1) / ksplit + PCK - 1) / PCK * PCK;
        ksplit = (p + cols - 1) / cols;
        float* part = nullptr;
        e = cc_dev_alloc((void**)&part, (size_t)ksplit * n * n * (mask ? 2 : 1) * sizeof(float), st);
        if (e == cudaSuccess) {
            const dim3 g2(grid, (unsigned)ksplit);
            const unsigned gf = (unsigned)(((size_t)n * n + 255) / 256);
            if (mask) {
                kd_weights<true><<<g2, 256, 0, st>>>((int)n, (int)p, ntile, phi, X, mask, W_out, (int)cols, part);
                kd_weights_fin<true><<<gf, 256, 0, st>>>((int)n, (int)p, (int)ksplit, phi, part, W_out);
            } else {
                kd_weights<false><<<g2, 256, 0, st>>>((int)n, (int)p, ntile, phi, X, mask, W_out, (int)cols, part);
                kd_weights_fin<false><<<gf, 256, 0, st>>>((int)n, (int)p, (int)ksplit, phi, part, W_out);
            }
            cc_dev_free(part, st);
        }
    }
    if (normalize && e == cudaSuccess) {
        double* red = nullptr;
        e = cc_dev_alloc((void**)&red, (size_t)(2 + 1024) * sizeof(double), st);
        if (e == cudaSuccess) {
            cudaMemsetAsync(red, 0, (size_t)(2 + 1024) * sizeof(double), st);
            kd_wsum<<<1024, CC_THREADS, 0, st>>>((int)n, W_out, red + 2, reinterpret_cast<unsigned int*>(red + 1), red);
            kd_wscale<<<1024, 256, 0, st>>>((long long)n * n, W_out, red);
            e = cudaStreamSynchronize(st);
            cc_dev_free(red, st);
        }
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(cc_g_err, sizeof(cc_g_err), "cc_dense_weights: %s", cudaGetErrorString(e));
        return e == cudaErrorMemoryAllocation ? CC_ENOMEM : CC_ECUDA;
    }
    return CC_OK;
}

// ---- cc_dense_weights_noalloc: the same weights with no allocation at all ----------------------------------------------
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
// cc_dense_weights takes the column slices' partial sums from a cudaMalloc'ed buffer; here they live in a file-scope device
// array of CC_NOALLOC_FLOATS floats (8 MB; every GPU that loads the library holds it until the process exits).
// In host code the array's NAME is only a host-side stand-in, not a device address: its address is taken once per device
// with cudaGetSymbolAddress (that device current) and the pointer is what the kernels get.
// Every call shares the array (it keeps the last call's contents; nothing in it has to start at zero, because kd_weights
// writes every entry kd_weights_fin reads), so calls that overlap on the GPU -- different streams, threads or processes of
// one context -- RACE: serialise them.
#define CC_NOALLOC_FLOATS (2u << 20)
static __device__ __align__(256) float cc_noalloc_scratch[CC_NOALLOC_FLOATS];
static float* cc_noalloc_ptr[64];     // per device: the array's device address (NULL = not looked up yet)

extern "C" int cc_dense_weights_noalloc(int64_t n, int64_t p, const float* X, const uint8_t* mask, float phi, float* W_out,
                                        void* stream) {
    if (!X || !W_out || n < 2 || p < 1 || !(phi >= 0.f) || n > 46340) {
        snprintf(cc_g_err, sizeof(cc_g_err), "cc_dense_weights_noalloc: need n in [2, 46340], p >= 1, phi >= 0, non-NULL pointers");
        return CC_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 148;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess || dev < 0 || dev >= 64) {
        cudaGetLastError();
        snprintf(cc_g_err, sizeof(cc_g_err), "cc_dense_weights_noalloc: %s", e != cudaSuccess ? cudaGetErrorString(e) : "device ordinal >= 64");
        return CC_ECUDA;
    }
    if (!cc_noalloc_ptr[dev]) {       // set-up, once per device, with that device current
        float* ptr = nullptr;
        e = cudaGetSymbolAddress((void**)&ptr, cc_noalloc_scratch);
        if (e != cudaSuccess || !ptr) {
            cudaGetLastError();
            snprintf(cc_g_err, sizeof(cc_g_err), "cc_dense_weights_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
            return CC_ECUDA;
        }
        cc_noalloc_ptr[dev] = ptr;
    }
    float* part = cc_noalloc_ptr[dev];
    // the slicing rule of cc_dense_weights, so that both entry points add the same partial sums in the same order
    const int ntile = (int)((n + PT - 1) / PT);
    const unsigned grid = (unsigned)(ntile * (ntile + 1) / 2);
    long long ksplit = grid >= (unsigned)sms ? 1 : (2LL * sms + grid - 1) / grid;
    const long long kmax = (p + 8LL * PCK - 1) / (8LL * PCK);
    if (ksplit > kmax) ksplit = kmax;
    if (ksplit <= 1) {                // enough pair tiles to fill the GPU: no scratch is used at all
        if (mask) kd_weights<true><<<grid, 256, 0, st>>>((int)n, (int)p, ntile, phi, X, mask, W_out, (int)p, nullptr);
        else kd_weights<false><<<grid, 256, 0, st>>>((int)n, (int)p, ntile, phi, X, mask, W_out, (int)p, nullptr);
    } else {
        const long long cols = ((p + ksplit - 1) / ksplit + PCK - 1) / PCK * PCK;
        ksplit = (p + cols - 1) / cols;
        const unsigned long long need = (unsigned long long)ksplit * n * n * (mask ? 2 : 1);
        if (need > CC_NOALLOC_FLOATS) {
            snprintf(cc_g_err, sizeof(cc_g_err), "cc_dense_weights_noalloc: n=%lld, p=%lld%s needs %llu floats of scratch, the static "
                     "array holds %u (8 MB): use cc_dense_weights", (long long)n, (long long)p, mask ? " with a mask" : "", need,
                     (unsigned)CC_NOALLOC_FLOATS);
            return CC_EINVAL;
        }
        const dim3 g2(grid, (unsigned)ksplit);
        const unsigned gf = (unsigned)(((size_t)n * n + 255) / 256);
        if (mask) {
            kd_weights<true><<<g2, 256, 0, st>>>((int)n, (int)p, ntile, phi, X, mask, W_out, (int)cols, part);
            kd_weights_fin<true><<<gf, 256, 0, st>>>((int)n, (int)p, (int)ksplit, phi, part, W_out);
        } else {
            kd_weights<false><<<g2, 256, 0, st>>>((int)n, (int)p, ntile, phi, X, mask, W_out, (int)cols, part);
            kd_weights_fin<false><<<gf, 256, 0, st>>>((int)n, (int)p, (int)ksplit, phi, part, W_out);
        }
    }
    e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(cc_g_err, sizeof(cc_g_err), "cc_dense_weights_noalloc: %s", cudaGetErrorString(e));
        return CC_ECUDA;
    }
    return CC_OK;
}
