/*
 * k1_half_transform.cu -- K1 of the exchange build (include/dfjk.h), sm_100a:
 *
 *     X_P[mu][i] = sum_nu B_P(mu,nu) Ccat[nu][i],   B_P(mu,nu) = Bp[P][max(max+1)/2 + min]
 *
 * One CTA computes a 128 x NW tile of X_P for one auxiliary index P (NW = 8*NT8 <= 136
 * columns of the concatenated, zero-padded orbital block), marching over nu in stages of
 * 32.  Warp-specialised, mbarrier-pipelined (no __syncthreads in the main loop):
 *
 *   producer warpgroup (4 warps, 40 registers after setmaxnreg.dec)
 *     - A tile: the packed triangle is unpacked while staging.  Every element (mu,nu) is
 *       fetched from Bp[max(max+1)/2+min] by an 8-byte cp.async (packed rows are only
 *       8-byte aligned), so tiles left of the diagonal read packed rows, tiles right of
 *       it read the transposed packed tile, and the diagonal tile mixes both; each
 *       thread's copies signal the stage's "full" mbarrier on completion
 *       (cp.async.mbarrier.arrive.noinc).  Every packed element is read twice per call
 *       (K1 is compute-bound: ~65 flop per byte of B).
 *     - C tile: Ccat is kept k-group-major ([nu/4][ldc][4]), so the 4 x NW x 4 tile of a
 *       stage is four contiguous 1-D bulk copies (TMA engine, cp.async.bulk -> UBLKCP)
 *       completing on the same mbarrier.
 *   two consumer warpgroups (8 warps, 232 registers after setmaxnreg.inc)
 *     - each warp owns 16 rows x NW columns = 2 x NT8 DMMA.8x8x4 accumulator tiles;
 *       one k4 step costs 2+NT8 shared loads for 2*NT8 MMAs.  Tiles are stored dense as
 *       [k/4][row][4] doubles: the 16 lanes of each 64-bit half-warp phase read 16
 *       consecutive doubles => conflict-free with no padding.
 *
 * Output: X in k-group-major layout X4[(p*ldc + i)/4][mu][(p*ldc + i)%4], which makes
 * every K2 operand tile a contiguous 4 KB bulk copy.
 */
#include "dfjk_internal.h"
#include "k_common.cuh"

namespace dfjk {
namespace {

constexpr int K1_M = 128;
constexpr int K1_KG = 8;                          /* k-groups (of 4) per stage */
constexpr int K1_KC = 4 * K1_KG;
constexpr int K1_PRODUCERS = 128;                 /* one warpgroup */
constexpr int K1_CONSUMERS = 256;                 /* two warpgroups */
constexpr int K1_THREADS = K1_PRODUCERS + K1_CONSUMERS;
constexpr int K1_A_BYTES = K1_M * K1_KC * 8;      /* 16384 */
constexpr int K1_SMEM_BUDGET = 220 * 1024;

template <int NT8>
struct K1Cfg {
    static constexpr int NW = 8 * NT8;
    static constexpr int C_BYTES = K1_KC * NW * 8;
    static constexpr int STAGE_BYTES = K1_A_BYTES + C_BYTES;
    static constexpr int STAGES_RAW = K1_SMEM_BUDGET / STAGE_BYTES;
    static constexpr int STAGES = STAGES_RAW > 8 ? 8 : STAGES_RAW;
    static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 2 * STAGES * 8 + 16;
};

template <int NT8>
__global__ void __launch_bounds__(K1_THREADS, 1)
k1_half_transform_kernel(const double *__restrict__ B, int64_t nao, int64_t npair, int64_t P0,
                         const double *__restrict__ Ccat4, int64_t ldc, int ntiles_n,
                         double *__restrict__ X4)
{
    using Cfg = K1Cfg<NT8>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nt_idx = blockIdx.x % ntiles_n;
    const int ib = blockIdx.x / ntiles_n;
    const int64_t p = blockIdx.y;
    const int64_t mu0 = (int64_t)ib * K1_M;
    const int64_t n0 = (int64_t)nt_idx * Cfg::NW;
    const int nk = (int)((nao + K1_KC - 1) / K1_KC);

    const uint32_t smem_base = smem_u32(smem_raw);
    const uint32_t bar_base = smem_base + Cfg::STAGES * Cfg::STAGE_BYTES;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (Cfg::STAGES + s); };

    if (tid == 0) {
        for (int s = 0; s < Cfg::STAGES; ++s) {
            mbar_init(full_bar(s), K1_PRODUCERS + 1);
            mbar_init(empty_bar(s), K1_CONSUMERS / 32);
        }
        mbar_fence_init();
    }
    __syncthreads();

    if (warp < K1_PRODUCERS / 32) {
        /* ------------------------------------------------------------ producers */
        reg_dealloc<40>();
        const double *__restrict__ Bp = B + (P0 + p) * npair;
        const int pw = warp;                               /* k-groups pw, pw+4, .. of the stage */
        const int mrow = lane >> 2;
        int64_t ncols = ldc - n0;                          /* valid columns of this N tile */
        if (ncols > Cfg::NW) ncols = Cfg::NW;
        const uint32_t c_bytes_g = (uint32_t)ncols * 32u;  /* per k-group */
        int slot = 0;
        uint32_t phase = 1;                                /* parity of the "empty" phase to wait for */
        for (int kc = 0; kc < nk; ++kc) {
            if (kc >= Cfg::STAGES) mbar_wait(empty_bar(slot), phase);
            if (tid == 0) {
                const uint32_t c_dst = smem_base + slot * Cfg::STAGE_BYTES + K1_A_BYTES;
                mbar_arrive_expect_tx(full_bar(slot), K1_KG * c_bytes_g);
#pragma unroll
                for (int g = 0; g < K1_KG; ++g)
                    bulk_g2s(c_dst + g * Cfg::NW * 32, Ccat4 + (((int64_t)kc * K1_KG + g) * ldc + n0) * 4,
                             c_bytes_g, full_bar(slot));
            }
#pragma unroll
            for (int gg = 0; gg < K1_KG / 4; ++gg) {
                const int g = pw + 4 * gg;
                const uint32_t a_dst = smem_base + slot * Cfg::STAGE_BYTES + g * 4096 + lane * 8;
                const int64_t nu = (int64_t)kc * K1_KC + 4 * g + (lane & 3);
                const bool nu_ok = nu < nao;
                const int64_t tri_nu = nu * (nu + 1) / 2;
#pragma unroll 4
                for (int r = 0; r < 16; ++r) {
                    const int64_t mu = mu0 + 8 * r + mrow;
                    const bool ok = nu_ok && mu < nao;
                    const int64_t off = mu >= nu ? mu * (mu + 1) / 2 + nu : tri_nu + mu;
                    cp_async8(a_dst + r * 256, ok ? Bp + off : Bp, ok);
                }
            }
            cp_async_mbar_arrive_noinc(full_bar(slot));
            if (++slot == Cfg::STAGES) { slot = 0; phase ^= 1; }
        }
    } else {
        /* ------------------------------------------------------------ consumers */
        reg_alloc<232>();
        const int cw = warp - K1_PRODUCERS / 32;           /* 0..7: rows 16*cw .. 16*cw+15 */
        const int lq = lane >> 2, lr = lane & 3;
        const bool warp_active = mu0 + 16 * cw < nao;
        double acc[2][NT8][2];
#pragma unroll
        for (int mt = 0; mt < 2; ++mt)
#pragma unroll
            for (int nt = 0; nt < NT8; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;

        int slot = 0;
        uint32_t phase = 0;
        for (int kc = 0; kc < nk; ++kc) {
            mbar_wait(full_bar(slot), phase);
            if (warp_active) {
                const double *As = reinterpret_cast<const double *>(smem_raw + slot * Cfg::STAGE_BYTES);
                const double *Cs = As + K1_A_BYTES / 8;
                const double *a_base = As + (16 * cw + lq) * 4 + lr;
                const double *b_base = Cs + lq * 4 + lr;
#pragma unroll
                for (int g = 0; g < K1_KG; ++g) {
                    const double a0 = a_base[g * (K1_M * 4)];
                    const double a1 = a_base[g * (K1_M * 4) + 32];
#pragma unroll
                    for (int nt = 0; nt < NT8; ++nt) {
                        const double b = b_base[g * (Cfg::NW * 4) + nt * 32];
                        dmma884(acc[0][nt][0], acc[0][nt][1], a0, b);
                        dmma884(acc[1][nt][0], acc[1][nt][1], a1, b);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty_bar(slot));
            if (++slot == Cfg::STAGES) { slot = 0; phase ^= 1; }
        }

        if (warp_active) {
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) {
                const int64_t mu = mu0 + 16 * cw + 8 * mt + lq;
                if (mu >= nao) continue;
#pragma unroll
                for (int nt = 0; nt < NT8; ++nt) {
                    const int64_t col = n0 + 8 * nt + 2 * lr;          /* even */
                    if (col < ldc) {
                        const int64_t k = p * ldc + col;
                        double *dst = X4 + ((k >> 2) * nao + mu) * 4 + (k & 3);
                        *reinterpret_cast<double2 *>(dst) = make_double2(acc[mt][nt][0], acc[mt][nt][1]);
                    }
                }
            }
        }
    }
}

template <int NT8>
void k1_launch_t(const double *B, int64_t nao, int64_t npair, int64_t P0, int64_t np,
                 const double *Ccat4, int64_t ldc, int ntiles_n, double *X4, cudaStream_t st)
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
        B, nao, npair, P0, Ccat4, ldc, ntiles_n, X4);
}

}  // namespace

void launch_k1_half_transform(const double *B, int64_t nao, int64_t npair, int64_t P0, int64_t np,
                              const double *Ccat4, int64_t ldc, double *X4, cudaStream_t st)
{
    const int n8 = (int)(ldc / 8);
    const int ntiles_n = (n8 + 16) / 17;
    const int nt8 = (n8 + ntiles_n - 1) / ntiles_n;
    /* grid.y <= 65535: chunks are far smaller than that */
#define DFJK_K1_CASE(N) \
    case N: k1_launch_t<N>(B, nao, npair, P0, np, Ccat4, ldc, ntiles_n, X4, st); break;
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
