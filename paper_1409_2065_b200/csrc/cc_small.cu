// cc_small.cu -- a9 for n <= 64 (the genotype shape: 52 rows x 200,000 columns): one fused kernel per MM iteration with
// the projection's contraction on the tensor cores.
//
// Complete graph, closed-form projection (PAPER.md L90-L103 with L = nI - 11', pin P3):
//     a_i = u_i + [ rowsum(S)_i p~_i - sum_j s_ij p~_j - n (u_i - ubar) ] / (n+1),   p~ = a' - ubar,
// then ||b_ij||^2 and ||s_ij b'_ij - b_ij||^2 for all pairs by direct differences (the fused / not-fused decision is taken on
// ||b||, far below ||a|| for a pair about to fuse: no Gram trick).  U, the previous projection and X are read once, A is
// written once.  The previous projection a' arrives as the array A of one iteration ago plus its residual column mean dbar
// (a' = A - dbar: k_update removes dbar in its own arithmetic and stores no A' for this path).
//
// One 512-thread CTA per SM walks chunks of 128 columns; two roles work on different chunks at the same time:
//   projection role, warps 0-3: thread = one column c of the chunk, so the column mean of U, the mean of A - U (the exact
//     invariant 1'(A-U) = 0) and the loss are thread-local sums over shared memory.  The contraction
//     D[c][i] = sum_j p~[j][c] S[j][i]  is one tcgen05.mma tile: M = 128 columns, N = 64 rows i, K = rows j, kind::tf32 with
//     the 3xTF32 split (hi.hi + hi.lo + lo.hi).  Both the accumulator and the chunk operand live in TENSOR MEMORY, whose
//     lane is the thread's column: the thread writes its own p~ (hi and lo) with tcgen05.st and reads its own results with
//     tcgen05.ld -- no transposition, no shared-memory operand.  S (N x K, K-major, SWIZZLE_128B) is staged once per launch.
//   pair role, warps 4-15: register tiles of 4 x 2 pairs on or above the diagonal blocks, interleaved column quads, packed
//     fp32 arithmetic (FADD2 / FFMA2).
// Data movement is the copy engine's: a chunk of U, A or X is four TMA tensor copies (32 columns x n rows each,
// cp.async.bulk.tensor.2d, SWIZZLE_128B) completing on an mbarrier, and A leaves by four tensor stores -- 16 instructions
// per chunk, issued by one lane.  A shared-memory array is [4 column groups][64 rows][128 bytes] with the 16-byte pieces of
// row r at position piece ^ (r % 8): the projection role's column walks and the pair role's 16-byte reads of eight rows at
// once are both conflict-free.  Columns beyond the matrix arrive as zeros (TMA's out-of-bounds fill) and are clipped on the
// way out.  Chunks alternate between two {U -> A, A (previous)} buffers: a pair warp refills a buffer as soon as its role
// has left it.
// (History, 52 x 200,000: FFMA kernel kd_small_ws 182 us; tensor-core contraction with thread-issued loads 194-250 us --
// the 26 cp.async + 13 LDG.128 per thread took 7 us per chunk to ISSUE next to twelve warps of LDS.128 traffic; one
// cp.async.bulk per 512-byte row segment: 180 us, every bulk copy costs ~25 ns of its issuing warp, 208 of them per chunk.)
// Per-(CTA, column phase) partial ||b||^2 go to NB2 slices; the edge section of k_update adds them in order.
#include <cstdio>
#include <cstring>

#include <cuda.h>

#include "cc_device.cuh"
#include "cc_internal.h"
#include "cc_tc.cuh"

namespace {

constexpr int ST_THREADS = 512, ST_PROJ = 128, ST_PAIR = ST_THREADS - ST_PROJ;
constexpr int ST_CN = 128;                      // columns per chunk = M of the MMA
constexpr int ST_K = 64;                        // rows padded to 64 = N (and the largest K) of the MMA
constexpr int ST_GRP = ST_K * 32;               // floats of one column group of an array: 64 rows x 32 columns
constexpr int ST_ARR = 4 * ST_GRP;              // floats of one array of a chunk (32 KB)
constexpr int ST_NBUF = 2;                      // {UA, P} buffers
constexpr int ST_BOP = 2 * 2 * ST_K * 128;      // S operand: {hi, lo} x 2 K-halves x 64 rows x 128 bytes
constexpr int ST_TMEM = 256;                    // tensor-memory columns: D at 0..63, p~ hi at 64..127, p~ lo at 128..191

__device__ __forceinline__ float lds32(uint32_t addr) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void sts32(uint32_t addr, float v) { asm volatile("st.shared.f32 [%0], %1;" :: "r"(addr), "f"(v) : "memory"); }

// D[tmem] (+)= A[tmem] * B[smem descriptor], kind::tf32
__device__ __forceinline__ void st_mma_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}\n"
        :: "r"(tmem_d), "r"(tmem_a), "l"(db), "r"(idesc), "r"(accumulate) : "memory");
}

__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16]) {
    uint32_t r[16];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                   "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                 : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int q = 0; q < 16; ++q) v[q] = __uint_as_float(r[q]);
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const float (&v)[8]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                 :: "r"(taddr), "r"(__float_as_uint(v[0])), "r"(__float_as_uint(v[1])), "r"(__float_as_uint(v[2])),
                    "r"(__float_as_uint(v[3])), "r"(__float_as_uint(v[4])), "r"(__float_as_uint(v[5])),
                    "r"(__float_as_uint(v[6])), "r"(__float_as_uint(v[7])) : "memory");
}

// Packed fp32 pairs (sm_100: FADD2 / FFMA2, one issue slot for two lanes' worth of arithmetic; the FP32 pipe's rate is
// unchanged -- measured 71 TFLOP/s either way -- but the pair loop, 84 % FP instructions, stops being issue-bound and the
// projection warps on the same schedulers get their slots).  A pair is a 64-bit register, low word = first element.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 f2sub(f32x2 a, f32x2 b) { f32x2 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 f2fma(f32x2 a, f32x2 b, f32x2 c) { f32x2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ f32x2 f2fma_s(f32x2 a, float s, f32x2 c) {       // a * (s, s) + c: ptxas folds the pair into a scalar operand
    f32x2 ss, r;
    asm("mov.b64 %0, {%1, %1};" : "=l"(ss) : "f"(s));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(ss), "l"(c));
    return r;
}
__device__ __forceinline__ float f2sum(f32x2 a) { float lo, hi; asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a)); return lo + hi; }
__device__ __forceinline__ void lds2x64(uint32_t addr, f32x2& lo, f32x2& hi) {
    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(lo), "=l"(hi) : "r"(addr) : "memory");
}

// global -> shared and shared -> global copies of a 32-column x n-row box by the copy engine (TMA, 2-D tensor map)
__device__ __forceinline__ void tma_load(uint32_t dst, const CUtensorMap* tm, int col, uint32_t bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 :: "r"(dst), "l"(tm), "r"(col), "r"(0), "r"(bar) : "memory");
}
__device__ __forceinline__ void tma_store(const CUtensorMap* tm, int col, uint32_t src) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.tile.bulk_group [%0, {%1, %2}], [%3];"
                 :: "l"(tm), "r"(col), "r"(0), "r"(src) : "memory");
}
__device__ __forceinline__ void expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
// (float offset of element (row r, column c of the chunk) in a shared-memory array:
//  (c / 32) * ST_GRP + r * 32 + ((((c % 32) / 4) ^ (r % 8)) << 2) + c % 4)

// One lane hands a chunk (first column c0) of one array to the copy engine
__device__ __forceinline__ void small_issue_array(uint32_t dst, const CUtensorMap* tm, int c0, uint32_t bar) {
#pragma unroll
    for (int g = 0; g < 4; ++g) tma_load(dst + (uint32_t)(g * ST_GRP * 4), tm, c0 + 32 * g, bar);
}

__global__ void __launch_bounds__(ST_THREADS, 1) kd_small_tc(int n, int ld, int cs_per_tile, const float* __restrict__ S,
                                                             const __grid_constant__ CUtensorMap tmU,
                                                             const __grid_constant__ CUtensorMap tmX, const __grid_constant__ CUtensorMap tmA,
                                                             const uint8_t* __restrict__ mask,
                                                             const float* __restrict__ W, const float* __restrict__ VN,
                                                             float* __restrict__ dbar, float* __restrict__ NB2, cc_scal* sc,
                                                             double* part, double* hist_phi, double* hist_d,
                                                             cudaGraphConditionalHandle outer) {
    if (!sc->mm_active) return;
    constexpr int BAR_PROJ = 1, BAR_PAIR = 2, BAR_FULL = 3;      // named barriers (FULL: one per buffer); 0 is __syncthreads
    constexpr int nbuf = ST_NBUF;
    extern __shared__ uint8_t st_smem_raw[];
    __shared__ __align__(8) uint64_t mma_done, xfull, full[ST_NBUF];
    __shared__ uint32_t tmem_base_s;
    __shared__ __align__(16) float rsS[ST_K];
    __shared__ int fail_s;
    const int tid = threadIdx.x, warp = tid >> 5;
    const int n4 = (n + 3) & ~3;
    // shared memory: [S operand | 2 data buffers {UA, P} | X buffer], every array 32 KB
    const uint32_t smb = (smem_u32(st_smem_raw) + 1023u) & ~1023u;
    uint8_t* smg = st_smem_raw + (smb - smem_u32(st_smem_raw));       // the same place as a generic pointer
    const uint32_t bop = smb;
    float* dbuf = reinterpret_cast<float*>(smg + ST_BOP);
    constexpr int bufsz = ST_ARR;                                       // floats of one array of one buffer
    float* xbuf = dbuf + (size_t)nbuf * 2 * bufsz;
    const uint32_t tx_bytes = (uint32_t)n * 4u * 128u;                  // one array of one chunk as the copy engine counts it

    const int nchunks = (ld + ST_CN - 1) / ST_CN;
    const int nmine = blockIdx.x < nchunks ? (nchunks - 1 - blockIdx.x) / gridDim.x + 1 : 0;   // chunks this CTA walks
    if (tid == 0) {
        fail_s = 0;
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(smem_u32(&mma_done)));
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(smem_u32(&xfull)));
        for (int b = 0; b < ST_NBUF; ++b) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(smem_u32(&full[b])));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        // the first chunks go to the copy engine at once (it writes rows < n only; the rest of this prologue touches other rows)
        for (int kk = 0; kk < nbuf && kk < nmine; ++kk) {
            const int c0 = (blockIdx.x + kk * gridDim.x) * ST_CN;
            const uint32_t bar = smem_u32(&full[kk]), dst = smem_u32(dbuf + (size_t)kk * 2 * bufsz);
            expect_tx(bar, 2u * tx_bytes);
            small_issue_array(dst, &tmU, c0, bar);
            small_issue_array(dst + bufsz * 4, &tmA, c0, bar);
        }
        if (nmine > 0) {
            expect_tx(smem_u32(&xfull), tx_bytes);
            small_issue_array(smem_u32(xbuf), &tmX, blockIdx.x * ST_CN, smem_u32(&xfull));
        }
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(smem_u32(&tmem_base_s)), "n"(ST_TMEM));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    // S as the B operand (N = i, K = j; K-major, SWIZZLE_128B): element (i, j) in K-half j / 32, row i, 16-byte chunk
    // (j % 32) / 4 at position chunk ^ (i % 8); rows and columns >= n are zero.  hi at 0, lo at 16 KB.
    if (tid < ST_K) {            // row sums of S, fixed order
        float r = 0.f;
        if (tid < n)
            for (int j = 0; j < n; ++j) r += S[(size_t)tid * n + j];
        rsS[tid] = r;
    }
    for (int t = tid; t < ST_K * ST_K; t += ST_THREADS) {
        const int i = t >> 6, j = t & 63;
        const float v = (i < n && j < n) ? S[(size_t)i * n + j] : 0.f;
        float h, l;
        split_tf32(v, h, l);
        const uint32_t off = (uint32_t)((j >> 5) * (ST_K * 128) + i * 128 + ((((j & 31) >> 2) ^ (i & 7)) << 4) + (j & 3) * 4);
        sts32(bop + off, h);
        sts32(bop + ST_BOP / 2 + off, l);
    }
    // the copy engine never writes rows >= n: zero once (the pair tiles read whole 4-row tiles, the column walks whole
    // 8-row blocks); the X buffer follows the data buffers
    {
        const int padf = (ST_K - n) * 32;                               // floats to clear per column group
        for (int t = tid; t < (nbuf * 2 + 1) * 4 * padf; t += ST_THREADS) dbuf[(t / padf) * ST_GRP + n * 32 + t % padf] = 0.f;
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_d = tmem_base_s;
    double red[4] = {0.0, 0.0, 0.0, 0.0};   // ||U-A||^2, loss, sum ||v-b||^2, sum w ||v||
    if (tid < ST_PROJ) {
        // ================= projection role: thread = column c of the chunk = lane c of tensor memory =================
        const int c = tid;
        uint32_t xa[8], xq[8];        // byte offset of this column in row i of an array: xa[i % 8] + 128 i;  xq: the same in the X buffer
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            xa[q] = (uint32_t)((c >> 5) * ST_GRP * 4 + (((((c & 31) >> 2) ^ q)) << 4) + (c & 3) * 4);
            xq[q] = smem_u32(xbuf) + xa[q];
        }
        const float inv = 1.f / (float)(n + 1), fn = (float)n, rfn = 1.f / (float)n;
        const int nks = (n + 7) >> 3;                                   // K steps of 8 rows
        // instruction descriptor: D = F32, A = B = TF32, both K-major (A: tensor memory), N = 64, M = 128
        const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(ST_K >> 3) << 17) | ((uint32_t)(ST_CN >> 4) << 24);
        const uint64_t db0 = ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) | ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
        const uint32_t tl = tmem_d + ((uint32_t)(warp * 32) << 16);     // this warp's 32 lanes
        const uint32_t rs_addr = smem_u32(rsS);
        for (int k = 0; k < nmine; ++k) {
            const int c0 = (blockIdx.x + k * gridDim.x) * ST_CN, gc = c0 + c;
            const bool inside = gc < ld;
            const int b = k % nbuf;
            float* UA = dbuf + (size_t)b * 2 * bufsz;           // A' is bufsz floats further
            if (!mbar_wait(smem_u32(&full[b]), (uint32_t)((k / nbuf) & 1))) fail_s = 1;
            if (!mbar_wait(smem_u32(&xfull), (uint32_t)(k & 1))) fail_s = 1;
            // Shared-memory addresses of this thread's column: row i of array X sits at X + xa[i % 8] + 128 i, so with the row
            // loops unrolled every load below is [register + immediate] (computing the swizzled offset per element cost three
            // integer instructions per load and made this role the slower one).
            uint32_t uq[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) uq[q] = smem_u32(UA) + xa[q];
            // (1) this thread's column: the sum of U and the loss.  Rows n .. 63 are zeros in both arrays: no predicates,
            // eight independent loads per array in flight.
            float su = 0.f, los = 0.f;
            if (mask == nullptr) {
#pragma unroll
                for (int i0 = 0; i0 < ST_K; i0 += 8)
                    if (i0 < n) {
                        float u8[8], x8[8];
#pragma unroll
                        for (int q = 0; q < 8; ++q) {
                            u8[q] = lds32(uq[q] + (i0 + q) * 128);
                            x8[q] = lds32(xq[q] + (i0 + q) * 128);
                        }
#pragma unroll
                        for (int q = 0; q < 8; ++q) {
                            const float d = x8[q] - u8[q];
                            su += u8[q];
                            los = fmaf(d, d, los);
                        }
                    }
            } else {
                for (int i = 0; i < n; ++i) {       // (masked problems of this size are rare: plain addressing, mask from global memory)
                    const uint32_t o = (uint32_t)((c >> 5) * ST_GRP * 4 + i * 128 + (((((c & 31) >> 2) ^ (i & 7))) << 4) + (c & 3) * 4);
                    const float u = lds32(smem_u32(UA) + o);
                    const bool obs = inside && mask[(size_t)i * ld + gc] != 0;
                    const float d = obs ? lds32(smem_u32(xbuf) + o) - u : 0.f;
                    su += u;
                    los = fmaf(d, d, los);
                }
            }
            if (!inside) los = 0.f;
            const float ub = su * rfn;
            // The previous projection arrives as the array A this kernel wrote one iteration ago, whose residual column mean
            // dbar k_update removed only in its own arithmetic (it no longer stores A' = A - dbar for this path: 41.6 MB per
            // iteration at 52 x 200,000): a' - ubar = A - (ubar + dbar).  The pair role needs no correction at all -- a shift of
            // a whole column cancels in a'_i - a'_j.
            const float ubp = ub + (inside ? dbar[gc] : 0.f);
            // (2) p~ = a' - ubar split into TF32 hi + lo -> this thread's lane of tensor memory, 8 rows j per store
#pragma unroll
            for (int ks = 0; ks < ST_K / 8; ++ks)
                if (ks * 8 < n) {
                    float hi[8], lo[8], pv[8];
#pragma unroll
                    for (int q = 0; q < 8; ++q) pv[q] = lds32(uq[q] + ST_ARR * 4 + (ks * 8 + q) * 128);
#pragma unroll
                    for (int q = 0; q < 8; ++q) split_tf32((inside && ks * 8 + q < n) ? pv[q] - ubp : 0.f, hi[q], lo[q]);
                    tmem_st8(tl + ST_K + ks * 8, hi);
                    tmem_st8(tl + 2 * ST_K + ks * 8, lo);
                }
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");   // (orders the previous chunk's TMEM reads too)
            named_sync(BAR_PROJ, ST_PROJ);
            if (tid == 0) {
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint64_t dbh = db0 | (uint64_t)(bop >> 4), dbl = db0 | (uint64_t)((bop + ST_BOP / 2) >> 4);
#pragma unroll
                for (int ks = 0; ks < ST_K / 8; ++ks)
                    if (ks < nks) {
                        const uint64_t kb = (uint64_t)((ks >> 2) * ((ST_K * 128) >> 4) + (ks & 3) * 2);   // K-half, then 32 bytes per step
                        st_mma_ts(tmem_d, tmem_d + ST_K + ks * 8, dbh + kb, idesc, ks > 0 ? 1u : 0u);
                        st_mma_ts(tmem_d, tmem_d + ST_K + ks * 8, dbl + kb, idesc, 1u);
                        st_mma_ts(tmem_d, tmem_d + 2 * ST_K + ks * 8, dbh + kb, idesc, 1u);
                    }
                asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(smem_u32(&mma_done)) : "memory");
            }
            // every thread of the role is past its reads of the X buffer: the next chunk's X may land
            if (tid == 32 && k + 1 < nmine) {
                expect_tx(smem_u32(&xfull), tx_bytes);
                small_issue_array(smem_u32(xbuf), &tmX, c0 + gridDim.x * ST_CN, smem_u32(&xfull));
            }
            if (!mbar_wait(smem_u32(&mma_done), (uint32_t)(k & 1))) fail_s = 1;
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            // (3) epilogue: a = u + [rowsum(S)_i p~ - sum_j s_ij p~_j - n (u - ubar)] / (n+1); the accumulator's lane is this
            // column.  (The diagonal term stays an fp32 product: folded into the tensor-core operand, L_S = diag(rowsum S) - S,
            // its 3xTF32 rounding -- n times a single term's -- took the error on U from 3e-7 to 3e-5.)
            float dua = 0.f, dsl = 0.f;
#pragma unroll
            for (int i0 = 0; i0 < ST_K; i0 += 16) {
                if (i0 < n) {
                    float sa[16], u16[16], p16[16], rs16[16];
#pragma unroll
                    for (int q = 0; q < 16; ++q) {
                        u16[q] = lds32(uq[q & 7] + (i0 + q) * 128);
                        p16[q] = lds32(uq[q & 7] + ST_ARR * 4 + (i0 + q) * 128);
                    }
#pragma unroll
                    for (int m = 0; m < 4; ++m) {        // (loaded outside the conditional below: a load inside it becomes a branch per row)
                        const float4 r4 = lds128(rs_addr + (uint32_t)(i0 + 4 * m) * 4u);
                        rs16[4 * m] = r4.x; rs16[4 * m + 1] = r4.y; rs16[4 * m + 2] = r4.z; rs16[4 * m + 3] = r4.w;
                    }
                    tmem_ld16(tl + (uint32_t)i0, sa);
#pragma unroll
                    for (int q = 0; q < 16; ++q) {
                        const float u = u16[q];
                        const float dlr = inv * fmaf(-fn, u - ub, fmaf(rs16[q], p16[q] - ubp, -sa[q]));
                        const float dl = (i0 + q < n && inside) ? dlr : 0.f;
                        const float a = u + dl;
                        u16[q] = a;
                        dsl += a - u;              // the stored difference, not dl: this is what must sum to zero
                        dua = fmaf(dl, dl, dua);
                    }
#pragma unroll
                    for (int q = 0; q < 16; ++q)
                        if (i0 + q < n) sts32(uq[q & 7] + (i0 + q) * 128, u16[q]);
                }
            }
            // 1'(A - U) = 0 holds exactly for the projection; the fp32 residual of this column goes to dbar and k_update removes
            // it from A (as on the large dense path: kd_dsum).  The pair role needs no correction: a shift of the whole column
            // cancels in a_i - a_j.
            if (inside) dbar[gc] = dsl * rfn;
            red[0] += (double)dua;
            red[1] += (double)los;
            // (4) A -> global memory: four tensor stores, issued by one lane once every thread's writes are visible to the
            // copy engine; the pair role may start as soon as the engine has READ the rows (it only reads them too)
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            named_sync(BAR_PROJ, ST_PROJ);
            if (tid == 0) {
#pragma unroll
                for (int g = 0; g < 4; ++g)
                    if (c0 + 32 * g < ld) tma_store(&tmA, c0 + 32 * g, smem_u32(UA + g * ST_GRP));
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
                asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
            }
            __syncwarp();
            named_arrive(BAR_FULL + b, ST_THREADS);
        }
        if (tid == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    }

    // ================= pair role (and, after the loop, everybody): tiles of 4 x 2 pairs, packed fp32 arithmetic =================
    const int nt2 = n4 >> 1, ntiles = (n4 >> 2) * ((n4 >> 2) + 1);      // row block ty owns the 2-row blocks tx = 2 ty .. nt2 - 1
    const bool pair_role = tid >= ST_PROJ;
    const int rt = tid - ST_PROJ;
    const bool pair_thread = pair_role && rt < ntiles * cs_per_tile;
    const int tile = pair_thread ? rt / cs_per_tile : 0, cph = pair_thread ? rt % cs_per_tile : 0;
    int ty = 0, tx = tile;                                // rows 4 ty + a (a < 4) against rows 2 tx + b (b < 2)
    while (tx >= nt2 - 2 * ty) { tx -= nt2 - 2 * ty; ++ty; }
    tx += 2 * ty;
    f32x2 nb[4][2], dv[4][2];                             // (even columns, odd columns) partial sums
    if (pair_role) {
        float sv[4][2];
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 2; ++b) {
                const int gi = ty * 4 + a, gj = tx * 2 + b;
                sv[a][b] = (pair_thread && gi < n && gj < n) ? __ldg(S + (size_t)gi * n + gj) : 0.f;
                nb[a][b] = 0ull;
                dv[a][b] = 0ull;
            }
        for (int k = 0; k < nmine; ++k) {
            const int b = k % nbuf;
            const float* As = dbuf + (size_t)b * 2 * bufsz;          // A; A' is bufsz floats further
            named_sync(BAR_FULL + b, ST_THREADS);
            if (pair_thread) {
                const uint32_t ay = smem_u32(As) + (uint32_t)(ty * 4 * 128), ax = smem_u32(As) + (uint32_t)(tx * 2 * 128);
                const int my = (ty & 1) << 2, mx = (tx & 3) << 1;             // (row % 8) of the tiles' first rows
                for (int cq = cph; cq < ST_CN / 4; cq += cs_per_tile) {
                    const uint32_t go = (uint32_t)((cq >> 3) * ST_GRP * 4);
                    const uint32_t qy = (uint32_t)(((cq & 7) ^ my) << 4), qx = (uint32_t)(((cq & 7) ^ mx) << 4);
                    f32x2 ai[4][2], pi[4][2], aj[2][2], pj[2][2];
#pragma unroll
                    for (int a = 0; a < 4; ++a) {
                        const uint32_t oy = ay + go + a * 128 + (qy ^ (a << 4));
                        lds2x64(oy, ai[a][0], ai[a][1]);
                        lds2x64(oy + ST_ARR * 4, pi[a][0], pi[a][1]);
                    }
#pragma unroll
                    for (int b2 = 0; b2 < 2; ++b2) {
                        const uint32_t ox = ax + go + b2 * 128 + (qx ^ (b2 << 4));
                        lds2x64(ox, aj[b2][0], aj[b2][1]);
                        lds2x64(ox + ST_ARR * 4, pj[b2][0], pj[b2][1]);
                    }
#pragma unroll
                    for (int a = 0; a < 4; ++a)
#pragma unroll
                        for (int b2 = 0; b2 < 2; ++b2) {
                            const f32x2 bl = f2sub(aj[b2][0], ai[a][0]), bh = f2sub(aj[b2][1], ai[a][1]);      // -b_ij
                            const f32x2 dl = f2sub(pi[a][0], pj[b2][0]), dh = f2sub(pi[a][1], pj[b2][1]);      // b'_ij
                            const f32x2 tl2 = f2fma_s(dl, sv[a][b2], bl), th2 = f2fma_s(dh, sv[a][b2], bh);    // s b' - b
                            nb[a][b2] = f2fma(bh, bh, f2fma(bl, bl, nb[a][b2]));
                            dv[a][b2] = f2fma(th2, th2, f2fma(tl2, tl2, dv[a][b2]));
                        }
                }
            }
            // the role has left buffer b: its next tenant goes to the copy engine
            if (k + nbuf < nmine) {
                named_sync(BAR_PAIR, ST_PAIR);
                if (tid == ST_PROJ) {
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    const int c0 = (blockIdx.x + (k + nbuf) * gridDim.x) * ST_CN;
                    const uint32_t bar = smem_u32(&full[b]), dst = smem_u32(As);
                    expect_tx(bar, 2u * tx_bytes);
                    small_issue_array(dst, &tmU, c0, bar);
                    small_issue_array(dst + bufsz * 4, &tmA, c0, bar);
                }
            }
        }
    }
    if (pair_thread) {
        float* out = NB2 + (size_t)(blockIdx.x * cs_per_tile + cph) * n * n;
        const bool diag = (tx >> 1) == ty;               // the two tiles on the diagonal block hold (i, j) and (j, i) themselves
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 2; ++b) {
                const int gi = ty * 4 + a, gj = tx * 2 + b;
                if (gi < n && gj < n && gi != gj) {
                    const float nbv = f2sum(nb[a][b]);
                    out[(size_t)gi * n + gj] = nbv;
                    if (!diag) out[(size_t)gj * n + gi] = nbv;
                    if (gi < gj) {
                        red[2] += (double)f2sum(dv[a][b]);
                        if (blockIdx.x == 0 && cph == 0) red[3] += (double)(W[(size_t)gi * n + gj] * VN[(size_t)gi * n + gj]);
                    }
                }
            }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem_d), "n"(ST_TMEM));
    if (tid == 0 && fail_s) sc->cg_failed = 2;
    double tot[4];
    if (grid_reduce<4, ST_THREADS>(red, part, &sc->ticket[3], tot)) {
        finish_iteration(sc, tot[0] + tot[2], tot[1], tot[3], hist_phi, hist_d, outer);
        prof_mark(sc, 5);
    }
}

}  // namespace

// Shared memory of one launch: S operand + 2 buffers x {A (over U), A'} + the X buffer, 32 KB each (+ alignment slack).
static constexpr size_t kSmallTcSmem = (size_t)ST_BOP + (size_t)(2 * ST_NBUF + 1) * ST_ARR * sizeof(float) + 1024;

typedef CUresult (*cc_encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                       const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                       CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// The driver's cuTensorMapEncodeTiled, through the runtime (the library does not link libcuda).
static cc_encode_tiled_fn small_tc_encoder() {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return nullptr;
    }
    return reinterpret_cast<cc_encode_tiled_fn>(fn);
}

// Tensor map of an n x ld row-major fp32 matrix, box = 32 columns x n rows, SWIZZLE_128B, zeros out of bounds.
static bool small_tc_map(cc_encode_tiled_fn enc, CUtensorMap* tm, const float* base, int64_t n, int64_t ld) {
    const cuuint64_t dims[2] = {(cuuint64_t)ld, (cuuint64_t)n};
    const cuuint64_t strides[1] = {(cuuint64_t)ld * sizeof(float)};
    const cuuint32_t box[2] = {32u, (cuuint32_t)n};
    const cuuint32_t estr[2] = {1u, 1u};
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Decide the launch shape (called by ccd_setup when n <= 64).  Returns 0 when the kernel cannot run here.
int ccd_small_tc_setup(cc_handle* h) {
    const int nt4 = (int)((h->n + 3) / 4), ntiles = nt4 * (nt4 + 1);      // 4 x 2 tiles on or above the diagonal blocks
    int cs = ST_PAIR / ntiles;
    if (cs > 4) cs = 4;
    if (cs < 1 || small_tc_encoder() == nullptr) return 0;
    if (cudaFuncSetAttribute(kd_small_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmallTcSmem) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    long long g = (h->ld + ST_CN - 1) / ST_CN;
    if (g > h->sms) g = h->sms;             // one 512-thread CTA per SM
    h->dn_small_cs = cs;
    h->dn_small_grid = (int)g;
    return 1;
}

int ccd_small_tc_maps(cc_handle* h) {
    static_assert(sizeof(CUtensorMap) == sizeof(h->dn_small_tm[0]), "tensor map storage");
    cc_encode_tiled_fn enc = small_tc_encoder();
    const float* base[4] = {h->U, h->A, h->X, h->A};      // (slot 1 unused: the previous projection is read from A)
    for (int k = 0; k < 4; ++k) {
        CUtensorMap tm;
        if (enc == nullptr || !small_tc_map(enc, &tm, base[k], h->n, h->ld)) {
            snprintf(h->err, sizeof(h->err), "dense mode: cuTensorMapEncodeTiled failed (n=%lld, ld=%lld)", (long long)h->n, (long long)h->ld);
            return CC_ECUDA;
        }
        memcpy(h->dn_small_tm[k], &tm, sizeof(tm));
    }
    return CC_OK;
}

void ccd_small_tc_launch(cc_handle* h) {
    CUtensorMap tm[4];
    memcpy(tm, h->dn_small_tm, sizeof(tm));
    kd_small_tc<<<h->dn_small_grid, ST_THREADS, kSmallTcSmem, h->stream>>>(
        (int)h->n, (int)h->ld, h->dn_small_cs, h->Sd, tm[0], tm[2], tm[3], h->mask, h->Wd, h->VNd, h->dbar, h->NB2d, h->sc,
        h->part + 3 * CC_MAXBLK * CC_NPART, h->hist_phi, h->hist_d, h->cond_outer);
}
