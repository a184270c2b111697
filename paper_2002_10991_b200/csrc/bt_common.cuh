// bt_common.cuh -- device helpers shared by the back-transformation kernels (sm_100a only).
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace elpa2bt {

// ---- reflector slot layout (include/elpa2_bt.h; R3) --------------------------------
// F(x) = sum_{y=1..x} ceil(y / nbw) = nbw t (t+1) / 2 + r (t+1) with x = t nbw + r;  off(s) = F(N-1) - F(N-1-s).
// Any nbw >= 1 (the kernels pass a compile-time constant, so the division is a multiply-shift).
__host__ __device__ __forceinline__ int64_t hh_F(int64_t x, int nbw)
{
    const int64_t t = x / nbw, r = x - t * nbw;
    return ((t * (t + 1)) >> 1) * nbw + r * (t + 1);
}
__host__ __device__ __forceinline__ int64_t hh_off(int64_t N, int nbw, int64_t s)
{
    return hh_F(N - 1, nbw) - hh_F(N - 1 - s, nbw);
}

// Opt-in to more than 48 KB of dynamic shared memory.  The attribute belongs to the (function, device)
// pair, so it is set on every launch path call (a host-side table lookup in the runtime, no device
// work) instead of once per process: a second device in the same process gets it too.
inline cudaError_t set_max_smem(const void *func, int bytes)
{
    return cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}

// ---- kernel arguments of the window kernels ------------------------------------------------------
struct WinArgs {
    int64_t N, nev, ldq;
    const double *hh_v;    // G * nbw elements
    const double *hh_tau;  // G elements
    double *q;
    int nw;                // consumer warps per CTA
    int align16;           // q base and ldq*ESZ are 16-byte aligned (always 1 for complex)
};

// ---- shared-memory / mbarrier / bulk-copy PTX wrappers ---------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_inval(uint32_t bar)
{
    asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
// polling wait with back-off for a warp that has nothing else to do (the producer): keeps its
// spin from taking issue slots away from the consumer warps of the same scheduler
__device__ __forceinline__ void mbar_wait_backoff(uint32_t bar, uint32_t parity)
{
    uint32_t done;
    for (;;) {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(done)
            : "r"(bar), "r"(parity)
            : "memory");
        if (done) break;
        __nanosleep(256);
    }
}
// 1-D bulk copy global -> shared (TMA engine, SASS UBLKCP), completion on an mbarrier.
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
        "l"(src), "r"(bytes), "r"(bar)
        : "memory");
}
// Ampere-style async copy with zero fill (src_bytes <= CP bytes are read, the rest is zeroed).
__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src, uint32_t src_bytes)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes)
                 : "memory");
}
__device__ __forceinline__ void cp_async8(uint32_t dst, const void *src, uint32_t src_bytes)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "r"(src_bytes)
                 : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

__device__ __forceinline__ double shfl_xor_f64(double v, int mask)
{
    return __shfl_xor_sync(0xffffffffu, v, mask);
}

}  // namespace elpa2bt
