// device_utils.cuh -- device-side helpers shared by the hot kernels (theta_kernels.cu, theta_mma.cu): mbarrier / 1-D bulk-TMA
// wrappers, power-of-two helpers and the packed window counters of the renormalisation scheme (internal.h; Sec. 3.4,
// PAPER.md:250-266).  Internal; not part of the public ABI.
#pragma once
#include "internal.h"

#include <cuda_runtime.h>
#include <stdint.h>

namespace shtdev {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// 1-D bulk copy global -> shared (SASS UBLKCP), completion counted on `bar`
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile(
            "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
            : "=r"(ok)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!ok);
}
// the same for a warp with slack (the reducers waiting for the compute warps): back off between polls instead of spinning, so that the
// polling loop does not compete with the compute warps of the same scheduler for issue slots
__device__ __forceinline__ void mbar_wait_relaxed(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    for (;;) {
        asm volatile(
            "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
            : "=r"(ok)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
        if (ok) break;
        __nanosleep(100);
    }
}
// fire-and-forget fp64 add to GLOBAL memory (SASS RED.E.ADD.F64)
__device__ __forceinline__ void red_add_f64(double* gptr, double v) {
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(gptr), "d"(v) : "memory");
}
// global[dst .. dst+bytes) += shared[src .. src+bytes) as doubles, asynchronously (SASS UBLKRED; bulk async-group completion)
__device__ __forceinline__ void bulk_reduce_add_f64(double* gdst, const void* ssrc, uint32_t bytes) {
    asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f64 [%0], [%1], %2;" ::"l"(gdst), "r"(smem_u32(ssrc)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// 2^e as a double, e in [-1022, 1023]
__device__ __forceinline__ double pow2i(int e) { return __hiloint2double((1023 + e) << 20, 0); }
__device__ __forceinline__ int hi_abs(double v) { return __double2hiint(v) & 0x7fffffff; }

#define SHT_HI_TWIN ((1023 + SHT_TWIN) << 20)
#define SHT_HI_DEAD ((1023 + 500) << 20)

// Register budgets re-split with setmaxnreg.  The kernels launch 12 warps (8 compute + 4 auxiliary, 3 per SM sub-partition) at 168
// registers per thread, so each sub-partition's pool is 3 * 32 * 168 = 16128 registers, and a split must satisfy
// 2 * 32 * RC + 32 * RA <= 16128 EXACTLY within that pool -- a compute warp asking for more than the auxiliary warps released waits
// forever.  RA = 40 -> RC = 232 (default); RA = 56 -> RC = 224 (kernels whose auxiliary warps carry more state).
template <int RA>
struct RegSplit {
    static constexpr int RC = (3 * 32 * 168 - 32 * RA) / 64;
    static_assert(RA % 8 == 0 && RC % 8 == 0 && 64 * RC + 32 * RA <= 3 * 32 * 168, "register split exceeds the CTA's pool");
};
template <int RA = 40>
__device__ __forceinline__ void reg_dealloc_aux() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(RA)); }
template <int RA = 40>
__device__ __forceinline__ void reg_alloc_compute() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(RegSplit<RA>::RC)); }

// Window counters k (internal.h) of the NI items of a thread, one byte each.  0xff = item not started yet.
template <int NI>
struct KPack {
    uint32_t w[(NI + 3) / 4];
    __device__ __forceinline__ void fill(uint32_t v) {
#pragma unroll
        for (int i = 0; i < (NI + 3) / 4; ++i) w[i] = v;
    }
    __device__ __forceinline__ void set(int idx, uint32_t k) {
        const int sh = (idx & 3) * 8;
        w[idx >> 2] = (w[idx >> 2] & ~(0xffu << sh)) | (k << sh);
    }
    __device__ __forceinline__ uint32_t get(int idx) const { return (w[idx >> 2] >> ((idx & 3) * 8)) & 0xffu; }
    __device__ __forceinline__ void dec(int idx) { w[idx >> 2] -= 1u << ((idx & 3) * 8); }
    __device__ __forceinline__ bool any_nonzero() const {
        uint32_t o = 0;
#pragma unroll
        for (int i = 0; i < (NI + 3) / 4; ++i) o |= w[i];
        return o != 0;
    }
    __device__ __forceinline__ bool any_zero_byte() const {
        bool z = false;
#pragma unroll
        for (int i = 0; i < (NI + 3) / 4; ++i) z = z || (((w[i] - 0x01010101u) & ~w[i] & 0x80808080u) != 0);
        return z;
    }
};
// Window maintenance (Sec. 3.4 renormalisation; internal.h): a stored value above 2^TWIN with k > 0 shifts its window.
template <int NI>
__device__ __forceinline__ void window_check(double (&cur)[NI], double (&prev)[NI], KPack<NI>& kp) {
    const double s = pow2i(-SHT_SWIN);
#pragma unroll
    for (int q = 0; q < NI; ++q) {
        if (hi_abs(cur[q]) > SHT_HI_TWIN && kp.get(q) != 0u && kp.get(q) != 0xffu) {
            cur[q] *= s; prev[q] *= s; kp.dec(q);
        }
    }
}
// On rings a pass no longer serves (m < m_lo, R5) the iterate leaves its stable range; it is zeroed before it
// can overflow.  Legitimate stored values never exceed ~2^250.
template <int NI>
__device__ __forceinline__ void dead_check(double (&cur)[NI], double (&prev)[NI]) {
#pragma unroll
    for (int q = 0; q < NI; ++q)
        if (hi_abs(cur[q]) > SHT_HI_DEAD) { cur[q] = 0.0; prev[q] = 0.0; }
}

}  // namespace shtdev
