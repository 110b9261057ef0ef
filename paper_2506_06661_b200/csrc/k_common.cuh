/*
 * k_common.cuh -- device helpers of the exchange (K) kernels: FP64 tensor-core
 * MMA (SASS DMMA.8x8x4, the only FP64 tensor shape sm_100a has), cp.async staging.
 *
 * Fragment layout of mma.sync.m8n8k4.f64 (PTX ISA; checked by tests/test_gpu_parity.py
 * through the K results):  lane l holds
 *     A[row = l/4][k = l%4]        (row-major 8x4)
 *     B[k = l%4][col = l/4]        (col-major 4x8)
 *     C[row = l/4][col = 2*(l%4) + {0,1}]
 *
 * Shared-memory tiles are stored with a leading dimension == 4 (mod 16) doubles,
 * which makes the 16 lanes of each 64-bit half-warp phase hit 16 distinct
 * 8-byte bank pairs for both access patterns above.
 */
#ifndef DFJK_K_COMMON_CUH
#define DFJK_K_COMMON_CUH

#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

namespace dfjk {

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c0), "+d"(c1)
        : "d"(a), "d"(b));
}

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}

/* 8-byte async copy global -> shared; ok == false writes zeros (src-size 0). */
__device__ __forceinline__ void cp_async8(uint32_t dst, const void *src, bool ok)
{
    const int n = ok ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "r"(n) : "memory");
}

/* 16-byte async copy, L2 only (.cg); both addresses 16-B aligned. */
__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src, bool ok)
{
    const int n = ok ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(n) : "memory");
}

__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }

template <int N>
__device__ __forceinline__ void cp_async_wait()
{
    asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

/* ------------------------------------------------------------------ mbarrier pipeline */
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
/* arrive on `bar` once all cp.async issued so far by this thread have landed
 * (does not change the pending count: the barrier's init count includes this thread) */
__device__ __forceinline__ void cp_async_mbar_arrive_noinc(uint32_t bar)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    while (!mbar_try_wait(bar, parity)) { }
}
/* try_wait that gives up after about `ns` nanoseconds (suspend-time hint) */
__device__ __forceinline__ bool mbar_try_wait_for(uint32_t bar, uint32_t parity, uint32_t ns)
{
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(bar), "r"(parity), "r"(ns) : "memory");
    return ok != 0;
}
/* non-blocking phase check */
__device__ __forceinline__ bool mbar_test_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
/* 1-D bulk copy (TMA engine, SASS UBLKCP) global -> shared; completes tx bytes on `bar`.
 * dst, src 16-B aligned, bytes a multiple of 16. */
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
template <int N>
__device__ __forceinline__ void reg_dealloc() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N>
__device__ __forceinline__ void reg_alloc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }

/* Host side: the opt-in to more than 48 KB of dynamic shared memory is per function AND per device;
 * `done` (one static atomic word per call site) remembers the devices that already have it.  Two
 * host threads may race here: the attribute call is idempotent, the flag is set only AFTER it has
 * returned (so nobody launches before the opt-in exists) and with an atomic OR (so no bit is lost). */
template <class F>
inline cudaError_t ensure_dynamic_smem(F func, int bytes, std::atomic<unsigned long long> &done)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const unsigned long long bit = 1ull << (dev & 63);
    if (!(done.load(std::memory_order_acquire) & bit)) {
        e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
        if (e != cudaSuccess) return e;
        done.fetch_or(bit, std::memory_order_release);
    }
    return cudaSuccess;
}

}  // namespace dfjk
#endif
