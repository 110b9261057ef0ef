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

}  // namespace dfjk
#endif
