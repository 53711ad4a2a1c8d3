// cc_tc.cuh -- small device helpers shared by the tensor-core kernels (cc_dense.cu, cc_small.cu): shared-space addresses,
// mbarrier waits, tcgen05.mma issue, TF32 rounding, named barriers.  sm_100a only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }


__device__ __forceinline__ void tc_mma(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}\n"
        :: "r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate) : "memory");
}


// try_wait suspends the waiting thread (up to a system-dependent time) instead of spinning: the warps that wait do not
// take issue slots from the one lane that feeds the tensor core.
__device__ __forceinline__ bool mbar_wait(uint32_t bar, uint32_t parity) {
    for (int spin = 0; spin < (1 << 24); ++spin) {
        uint32_t ok;
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (ok) return true;
    }
    return false;   // never hang the GPU: the caller raises cg_failed
}
// the same for warps with slack (staging): back off between polls, so that a warp that waits leaves its scheduler to the
// MMA-issuing lane (a single lane issuing ~10 instructions per MMA next to four spinning warps ran at ~190 cycles per MMA
// where the tensor core takes 64)
__device__ __forceinline__ bool mbar_wait_idle(uint32_t bar, uint32_t parity) {
    for (int spin = 0; spin < (1 << 22); ++spin) {
        uint32_t ok;
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (ok) return true;
        __nanosleep(100);
    }
    return false;
}

// Round to the nearest TF32 value (10 mantissa bits), ties away from zero -- what cvt.rna.tf32.f32 does.  ptxas emulates
// that instruction on sm_100a with ~6 instructions (Inf / NaN handling included); for the finite numbers of this path the
// integer form below is the same rounding in 2 (ncu: the staging loop of kd_proj_tc3 ran 194 instructions per thread and
// K block, half of them these conversions, and was issue-bound with the tensor pipe 19 % busy).
__device__ __forceinline__ float rna_tf32(float x) { return __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xffffe000u); }

// x = hi + lo + O(2^-23 |x|), both parts exactly representable in TF32 and ROUNDED to nearest: truncating instead
// (masking the low mantissa bits) biases every product the same way and the bias accumulates over the MM iterations
// (measured: 1.6e-4 relative error on U after 480 iterations against 8e-6 for the FFMA kernel).
__device__ __forceinline__ void split_tf32(float x, float& hi, float& lo) {
    hi = rna_tf32(x);
    lo = rna_tf32(x - hi);
}

__device__ __forceinline__ float4 lds128(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
    return v;
}


__device__ __forceinline__ void named_sync(int id, int count) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }
__device__ __forceinline__ void named_arrive(int id, int count) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory"); }


}  // namespace
