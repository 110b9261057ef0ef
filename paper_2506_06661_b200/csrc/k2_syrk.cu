/*
 * k2_syrk.cu -- K0 (orbital packing), K2 (lower-triangle SYRK) and K3 (finish) of the
 * exchange build (include/dfjk.h), sm_100a:
 *
 *     K_s[mu][nu] += sum_{P in chunk} sum_{i in set s} X_P[mu][i] X_P[nu][i]     mu-tile >= nu-tile
 *
 * X chunk layout (written by K1): X[mu][p*ldc + i], row pitch xpitch, so the contraction
 * index k = (p, i) is contiguous per row apart from the jump between sets/P.  The k axis
 * is walked in groups of 8 columns (every set is zero-padded to a multiple of 8, so each
 * group is 64 contiguous, 16-B aligned bytes); a stage holds two groups (k = 16).
 * One CTA owns a 128 x 128 tile of K for one k-split: 8 warps as 2 (M) x 4 (N), warp tile
 * 64 x 32 = 8 x 4 DMMA.8x8x4 accumulators, 12 shared loads per 32 MMAs.  Both operands are
 * k-contiguous row tiles of X, so A (row-major) and B (col-major) fragments are read with
 * the same pattern; diagonal tiles load the panel once.
 * Splits: work item = (lower tile, split) with its own partial accumulator Kpart[split],
 * read-modify-written by exactly one CTA per launch => deterministic, no atomics.
 */
#include "dfjk_internal.h"
#include "k_common.cuh"

namespace dfjk {
namespace {

/* ------------------------------------------------------------------ K0 */
struct PackDesc {
    int nset;
    const double *C[4];
    int nocc[4];
    int col0[4];
};

__global__ void k0_pack_c_kernel(PackDesc pd, int64_t nao, int64_t ldc, double *__restrict__ Ccat)
{
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= nao * ldc) return;
    const int64_t mu = idx / ldc;
    const int c = (int)(idx % ldc);
    double v = 0.0;
    for (int s = 0; s < pd.nset; ++s)
        if (c >= pd.col0[s] && c < pd.col0[s] + pd.nocc[s])
            v = pd.C[s][mu * pd.nocc[s] + (c - pd.col0[s])];
    Ccat[idx] = v;
}

/* ------------------------------------------------------------------ K2 */
constexpr int K2_T = 128;
constexpr int K2_KC = 16;
constexpr int K2_LD = 20;                   /* == 4 mod 16 */
constexpr int K2_STAGES = 4;
constexpr int K2_PANEL = K2_T * K2_LD;      /* doubles per operand per stage */
constexpr int K2_THREADS = 256;
constexpr int K2_SMEM_BYTES = K2_STAGES * 2 * K2_PANEL * 8;   /* 163840 */

__global__ void __launch_bounds__(K2_THREADS, 1)
k2_syrk_lower_kernel(const double *__restrict__ X, int64_t xpitch, int64_t nao, int64_t np,
                     int64_t ldc, int64_t col0, int n8s, double *__restrict__ Kpart, int nsplit,
                     int accumulate)
{
    extern __shared__ __align__(16) double smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    /* lower-triangle tile index -> (bi, bj), bi >= bj */
    const int t = blockIdx.x;
    int bi = (int)((sqrtf(8.0f * (float)t + 1.0f) - 1.0f) * 0.5f);
    while (bi * (bi + 1) / 2 > t) --bi;
    while ((bi + 1) * (bi + 2) / 2 <= t) ++bi;
    const int bj = t - bi * (bi + 1) / 2;
    const bool diag = bi == bj;
    const int split = blockIdx.y;
    const int64_t mu0 = (int64_t)bi * K2_T, nu0 = (int64_t)bj * K2_T;

    /* this split's share of the k groups (8 columns each) */
    const int64_t ng = np * n8s;
    const int64_t gbeg = ng * split / nsplit, gend = ng * (split + 1) / nsplit;
    const int nk = (int)((gend - gbeg + 1) / 2);

    auto issue = [&](int kc, int slot) {
        double *Xa = smem + slot * 2 * K2_PANEL;
        double *Xb = Xa + K2_PANEL;
        /* per operand: 128 rows x 2 groups x 4 pieces of 16 B = 1024 pieces */
        const int npieces = diag ? 1024 : 2048;
        for (int e = tid; e < npieces; e += K2_THREADS) {
            const int op = e >> 10;
            const int r = (e >> 3) & 127, q = e & 7;      /* q: piece within the 16-double row */
            const int64_t g = gbeg + 2 * (int64_t)kc + (q >> 2);
            const int64_t row = (op ? nu0 : mu0) + r;
            const bool ok = g < gend && row < nao;
            const int64_t pp = g / n8s, j = g % n8s;
            const double *src = X + row * xpitch + pp * ldc + col0 + 8 * j + 2 * (q & 3);
            cp_async16(smem_u32((op ? Xb : Xa) + r * K2_LD + 2 * q), ok ? src : X, ok);
        }
    };

    double acc[8][4][2];
#pragma unroll
    for (int mt = 0; mt < 8; ++mt)
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;

    const int wm = warp >> 2, wn = warp & 3;     /* warp tile: rows 64*wm.., cols 32*wn.. */
    const int lq = lane >> 2, lr = lane & 3;

#pragma unroll
    for (int s = 0; s < K2_STAGES - 1; ++s) {
        if (s < nk) issue(s, s);
        cp_async_commit();
    }
    for (int kc = 0; kc < nk; ++kc) {
        cp_async_wait<K2_STAGES - 2>();
        __syncthreads();
        {
            const int nxt = kc + K2_STAGES - 1;
            if (nxt < nk) issue(nxt, nxt % K2_STAGES);
            cp_async_commit();
        }
        const double *Xa = smem + (kc % K2_STAGES) * 2 * K2_PANEL;
        const double *Xb = diag ? Xa : Xa + K2_PANEL;
        const double *a_base = Xa + (64 * wm + lq) * K2_LD + lr;
        const double *b_base = Xb + (32 * wn + lq) * K2_LD + lr;
#pragma unroll
        for (int k4 = 0; k4 < K2_KC / 4; ++k4) {
            double a[8], b[4];
#pragma unroll
            for (int mt = 0; mt < 8; ++mt) a[mt] = a_base[mt * 8 * K2_LD + 4 * k4];
#pragma unroll
            for (int nt = 0; nt < 4; ++nt) b[nt] = b_base[nt * 8 * K2_LD + 4 * k4];
#pragma unroll
            for (int mt = 0; mt < 8; ++mt)
#pragma unroll
                for (int nt = 0; nt < 4; ++nt) dmma884(acc[mt][nt][0], acc[mt][nt][1], a[mt], b[nt]);
        }
    }
    cp_async_wait<0>();

    double *Kp = Kpart + (int64_t)split * nao * nao;
#pragma unroll
    for (int mt = 0; mt < 8; ++mt) {
        const int64_t mu = mu0 + 64 * wm + 8 * mt + lq;
        if (mu >= nao) continue;
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) {
            const int64_t nu = nu0 + 32 * wn + 8 * nt + 2 * lr;
            double *dst = Kp + mu * nao + nu;
            if (nu < nao) dst[0] = accumulate ? dst[0] + acc[mt][nt][0] : acc[mt][nt][0];
            if (nu + 1 < nao) dst[1] = accumulate ? dst[1] + acc[mt][nt][1] : acc[mt][nt][1];
        }
    }
}

/* ------------------------------------------------------------------ K3 */
constexpr int K3_T = 32;

__global__ void __launch_bounds__(256)
k3_finish_kernel(const double *__restrict__ Kpart, int nsplit, int64_t nao, double *__restrict__ K)
{
    const int bi = blockIdx.y, bj = blockIdx.x;
    if (bj > bi) return;
    __shared__ double t[K3_T][K3_T + 1];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int64_t mu0 = (int64_t)bi * K3_T, nu0 = (int64_t)bj * K3_T;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int row = ty + 8 * r;
        const int64_t mu = mu0 + row, nu = nu0 + tx;
        double v = 0.0;
        if (mu < nao && nu <= mu)
            for (int s = 0; s < nsplit; ++s) v += Kpart[(int64_t)s * nao * nao + mu * nao + nu];
        t[row][tx] = v;
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int row = ty + 8 * r;
        const int64_t mu = mu0 + row, nu = nu0 + tx;
        if (mu < nao && nu < nao) K[mu * nao + nu] = (bi == bj && tx > row) ? t[tx][row] : t[row][tx];
        if (bi != bj) {
            const int64_t a = nu0 + row, b = mu0 + tx;
            if (a < nao && b < nao) K[a * nao + b] = t[tx][row];
        }
    }
}

}  // namespace

void launch_k0_pack_c(const double *const *C, const int *nocc, const int *col0, int nset, int64_t nao,
                      int64_t ldc, double *Ccat, cudaStream_t st)
{
    PackDesc pd;
    pd.nset = nset;
    for (int s = 0; s < 4; ++s) {
        pd.C[s] = s < nset ? C[s] : nullptr;
        pd.nocc[s] = s < nset ? nocc[s] : 0;
        pd.col0[s] = s < nset ? col0[s] : 0;
    }
    const int64_t n = nao * ldc;
    k0_pack_c_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(pd, nao, ldc, Ccat);
}

void launch_k2_syrk_lower(const double *X, int64_t xpitch, int64_t nao, int64_t np, int64_t ldc,
                          int64_t col0, int64_t ncol, double *Kpart, int nsplit, int accumulate,
                          cudaStream_t st)
{
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(k2_syrk_lower_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             K2_SMEM_BYTES);
        configured = true;
    }
    const int nb = (int)((nao + K2_T - 1) / K2_T);
    const int ntile = nb * (nb + 1) / 2;
    const int n8s = (int)((ncol + 7) / 8);
    k2_syrk_lower_kernel<<<dim3((unsigned)ntile, (unsigned)nsplit), K2_THREADS, K2_SMEM_BYTES, st>>>(
        X, xpitch, nao, np, ldc, col0, n8s, Kpart, nsplit, accumulate);
}

void launch_k3_finish(const double *Kpart, int nsplit, int64_t nao, double *K, cudaStream_t st)
{
    const unsigned nb = (unsigned)((nao + K3_T - 1) / K3_T);
    k3_finish_kernel<<<dim3(nb, nb), 256, 0, st>>>(Kpart, nsplit, nao, K);
}

}  // namespace dfjk
