/*
 * k1_half_transform.cu -- K1 of the exchange build (include/dfjk.h), sm_100a:
 *
 *     X_P[mu][i] = sum_nu B_P(mu,nu) Ccat[nu][i],   B_P(mu,nu) = Bp[P][max(max+1)/2 + min]
 *
 * One CTA computes a 128 x NW tile of X_P for one auxiliary index P (NW = 8*NT8 <= 136
 * columns of the concatenated, zero-padded orbital block), marching over nu in chunks
 * of 16.  The packed triangle is unpacked on the fly while staging to shared memory:
 *   - nu-chunk left of the row block   : rows of the packed triangle, tile stored [m][k]
 *   - nu-chunk right of the row block  : B_P(mu,nu) = packed(nu,mu): rows nu of the packed
 *                                        triangle, contiguous in mu, tile stored [k][m]
 *   - chunk crossing the diagonal      : element-wise max/min gather, tile stored [m][k]
 * so every packed element is read twice per call (K1 is compute-bound: ~65 flop/B).
 * Math: FP64 tensor-core DMMA.8x8x4; each of the 8 warps owns 16 rows x NW columns
 * (2 x NT8 accumulator tiles), so one k4 step costs 2+NT8 shared loads for 2*NT8 MMAs.
 * Staging: 4-stage cp.async ring (8-byte copies for B: packed rows are only 8-B aligned;
 * 16-byte copies for C).
 */
#include "dfjk_internal.h"
#include "k_common.cuh"

namespace dfjk {
namespace {

constexpr int K1_M = 128;
constexpr int K1_KC = 16;
constexpr int K1_LDA = 20;                 /* [m][k] tile pitch, == 4 mod 16 */
constexpr int K1_LDT = 132;                /* [k][m] tile pitch, == 4 mod 16 */
constexpr int K1_STAGES = 4;
constexpr int K1_A_DOUBLES = K1_M * K1_LDA;   /* 2560 >= 16*132 */
constexpr int K1_THREADS = 256;

template <int NT8>
struct K1Cfg {
    static constexpr int NW = 8 * NT8;
    static constexpr int LDCS = NW + ((NT8 & 1) ? 12 : 4);   /* == 4 mod 16 */
    static constexpr int C_DOUBLES = K1_KC * LDCS;
    static constexpr int STAGE = K1_A_DOUBLES + C_DOUBLES;
    static constexpr int SMEM_BYTES = K1_STAGES * STAGE * 8;
};

enum { MODE_DIRECT = 0, MODE_TRANSPOSED = 1, MODE_DIAG = 2 };

__device__ __forceinline__ int k1_mode(int64_t mu0, int64_t nu0)
{
    if (nu0 + K1_KC - 1 <= mu0) return MODE_DIRECT;
    if (nu0 >= mu0 + K1_M - 1) return MODE_TRANSPOSED;
    return MODE_DIAG;
}

template <int NT8>
__global__ void __launch_bounds__(K1_THREADS, 1)
k1_half_transform_kernel(const double *__restrict__ B, int64_t nao, int64_t npair, int64_t P0,
                         const double *__restrict__ Ccat, int64_t ldc, int ntiles_n,
                         double *__restrict__ X, int64_t xpitch)
{
    using Cfg = K1Cfg<NT8>;
    extern __shared__ __align__(16) double smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nt_idx = blockIdx.x % ntiles_n;
    const int ib = blockIdx.x / ntiles_n;
    const int64_t p = blockIdx.y;
    const double *__restrict__ Bp = B + (P0 + p) * npair;
    const int64_t mu0 = (int64_t)ib * K1_M;
    const int64_t n0 = (int64_t)nt_idx * Cfg::NW;
    const int nk = (int)((nao + K1_KC - 1) / K1_KC);

    auto issue = [&](int kc, int slot) {
        double *As = smem + slot * Cfg::STAGE;
        double *Cs = As + K1_A_DOUBLES;
        const int64_t nu0 = (int64_t)kc * K1_KC;
        /* C tile: 16 rows x NW columns in 16-byte pieces */
        for (int e = tid; e < K1_KC * (Cfg::NW / 2); e += K1_THREADS) {
            const int k = e / (Cfg::NW / 2), c2 = e % (Cfg::NW / 2);
            const int64_t nu = nu0 + k, col = n0 + 2 * c2;
            const bool ok = nu < nao && col < ldc;
            cp_async16(smem_u32(Cs + k * Cfg::LDCS + 2 * c2), ok ? Ccat + nu * ldc + col : Ccat, ok);
        }
        const int mode = k1_mode(mu0, nu0);
        if (mode == MODE_TRANSPOSED) {
#pragma unroll
            for (int r = 0; r < (K1_M * K1_KC) / K1_THREADS; ++r) {
                const int e = tid + K1_THREADS * r;
                const int k = e >> 7, m = e & 127;
                const int64_t nu = nu0 + k, mu = mu0 + m;
                const bool ok = nu < nao && mu < nao;
                cp_async8(smem_u32(As + k * K1_LDT + m), ok ? Bp + nu * (nu + 1) / 2 + mu : Bp, ok);
            }
        } else {
#pragma unroll
            for (int r = 0; r < (K1_M * K1_KC) / K1_THREADS; ++r) {
                const int e = tid + K1_THREADS * r;
                const int m = e >> 4, k = e & 15;
                const int64_t mu = mu0 + m, nu = nu0 + k;
                const bool ok = mu < nao && nu < nao;
                const int64_t a = mu > nu ? mu : nu, b = mu > nu ? nu : mu;
                cp_async8(smem_u32(As + m * K1_LDA + k), ok ? Bp + a * (a + 1) / 2 + b : Bp, ok);
            }
        }
    };

    double acc[2][NT8][2];
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
        for (int nt = 0; nt < NT8; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;

    const bool warp_active = mu0 + 16 * warp < nao;
    const int lq = lane >> 2, lr = lane & 3;

#pragma unroll
    for (int s = 0; s < K1_STAGES - 1; ++s) {
        if (s < nk) issue(s, s);
        cp_async_commit();
    }
    for (int kc = 0; kc < nk; ++kc) {
        cp_async_wait<K1_STAGES - 2>();
        __syncthreads();
        {
            const int nxt = kc + K1_STAGES - 1;
            if (nxt < nk) issue(nxt, nxt % K1_STAGES);
            cp_async_commit();
        }
        if (warp_active) {
            const double *As = smem + (kc % K1_STAGES) * Cfg::STAGE;
            const double *Cs = As + K1_A_DOUBLES;
            const bool tr = k1_mode(mu0, (int64_t)kc * K1_KC) == MODE_TRANSPOSED;
            const double *a_base = tr ? As + lr * K1_LDT + 16 * warp + lq
                                      : As + (16 * warp + lq) * K1_LDA + lr;
            const int a_kstep = tr ? 4 * K1_LDT : 4;
            const int a_mstep = tr ? 8 : 8 * K1_LDA;
            const double *b_base = Cs + lr * Cfg::LDCS + lq;
#pragma unroll
            for (int k4 = 0; k4 < K1_KC / 4; ++k4) {
                const double a0 = a_base[k4 * a_kstep];
                const double a1 = a_base[k4 * a_kstep + a_mstep];
#pragma unroll
                for (int nt = 0; nt < NT8; ++nt) {
                    const double b = b_base[k4 * 4 * Cfg::LDCS + 8 * nt];
                    dmma884(acc[0][nt][0], acc[0][nt][1], a0, b);
                    dmma884(acc[1][nt][0], acc[1][nt][1], a1, b);
                }
            }
        }
    }
    cp_async_wait<0>();

    if (warp_active) {
#pragma unroll
        for (int mt = 0; mt < 2; ++mt) {
            const int64_t mu = mu0 + 16 * warp + 8 * mt + lq;
            if (mu >= nao) continue;
            double *xrow = X + mu * xpitch + p * ldc + n0;
#pragma unroll
            for (int nt = 0; nt < NT8; ++nt) {
                const int64_t col = 8 * nt + 2 * lr;
                if (n0 + col < ldc)
                    *reinterpret_cast<double2 *>(xrow + col) = make_double2(acc[mt][nt][0], acc[mt][nt][1]);
            }
        }
    }
}

template <int NT8>
void k1_launch_t(const double *B, int64_t nao, int64_t npair, int64_t P0, int64_t np,
                 const double *Ccat, int64_t ldc, int ntiles_n, double *X, int64_t xpitch,
                 cudaStream_t st)
{
    static bool configured = false;   /* attribute is per function, set once per process */
    if (!configured) {
        cudaFuncSetAttribute(k1_half_transform_kernel<NT8>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             K1Cfg<NT8>::SMEM_BYTES);
        configured = true;
    }
    const unsigned nib = (unsigned)((nao + K1_M - 1) / K1_M);
    dim3 grid(nib * ntiles_n, (unsigned)np);
    k1_half_transform_kernel<NT8><<<grid, K1_THREADS, K1Cfg<NT8>::SMEM_BYTES, st>>>(
        B, nao, npair, P0, Ccat, ldc, ntiles_n, X, xpitch);
}

}  // namespace

void launch_k1_half_transform(const double *B, int64_t nao, int64_t npair, int64_t P0, int64_t np,
                              const double *Ccat, int64_t ldc, double *X, int64_t xpitch,
                              cudaStream_t st)
{
    const int n8 = (int)(ldc / 8);
    const int ntiles_n = (n8 + 16) / 17;
    const int nt8 = (n8 + ntiles_n - 1) / ntiles_n;
    /* grid.y <= 65535: chunks are far smaller than that */
#define DFJK_K1_CASE(N) \
    case N: k1_launch_t<N>(B, nao, npair, P0, np, Ccat, ldc, ntiles_n, X, xpitch, st); break;
    switch (nt8) {
        DFJK_K1_CASE(1) DFJK_K1_CASE(2) DFJK_K1_CASE(3) DFJK_K1_CASE(4) DFJK_K1_CASE(5)
        DFJK_K1_CASE(6) DFJK_K1_CASE(7) DFJK_K1_CASE(8) DFJK_K1_CASE(9) DFJK_K1_CASE(10)
        DFJK_K1_CASE(11) DFJK_K1_CASE(12) DFJK_K1_CASE(13) DFJK_K1_CASE(14) DFJK_K1_CASE(15)
        DFJK_K1_CASE(16) DFJK_K1_CASE(17)
    default: break;
    }
#undef DFJK_K1_CASE
}

}  // namespace dfjk
