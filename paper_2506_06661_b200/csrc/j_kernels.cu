/*
 * j_kernels.cu -- the Coulomb half of DF get_jk (include/dfjk.h), sm_100a.
 *
 *     Dt[pair]  = (2 - delta) * D[mu][nu]              J0   (tiny)
 *     d_P       = sum_pair B[P][pair] Dt[pair]         J1   streams |B| bytes   HBM-bound
 *     Jp[pair]  = sum_P d_P B[P][pair]                 J2   streams |B| bytes   HBM-bound
 *     J         = unpack(Jp), both triangles           J3   (tiny)
 *
 * J1/J2 are pure streaming kernels (0.25 flop/byte): what matters is bytes in
 * flight per SM (>= ~40 KB by Little's law), 128-bit coalesced loads that bypass
 * L1 and are marked evict-first in L2, Dt/d/Jp staying on chip, and reductions
 * that never serialise.  Packed rows start at P*npair doubles, which is only
 * 8-byte aligned when npair is odd: all vector loads are issued on the 16-byte
 * grid of the FLAT array and the (at most two) straddling elements per row
 * segment are handled by scalar loads.
 */
#include "dfjk_internal.h"

namespace dfjk {

namespace {

__device__ __forceinline__ double2 ldg_stream2(const double *p)
{
    /* read-once data: non-coherent path, streaming (evict-first) policy */
    return __ldcs(reinterpret_cast<const double2 *>(p));
}
__device__ __forceinline__ double ldg_stream1(const double *p) { return __ldcs(p); }

/* ------------------------------------------------------------------ J0 */
struct SetDesc {
    int nset;
    int col0[4];
    int nocc[4];
    double w[4];
};

constexpr int J0_T = 32;

__global__ void __launch_bounds__(256)
j0_build_dt_kernel(const double *__restrict__ Ccat, int64_t ldc, int64_t nao, SetDesc sd,
                   double *__restrict__ Dt)
{
    const int bi = blockIdx.y, bj = blockIdx.x;
    if (bj > bi) return;
    __shared__ double Cm[J0_T][J0_T + 1];
    __shared__ double Cn[J0_T][J0_T + 1];
    __shared__ double wcol[J0_T];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;   /* ty 0..7 */
    const int64_t mu0 = (int64_t)bi * J0_T, nu0 = (int64_t)bj * J0_T;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    for (int64_t c0 = 0; c0 < ldc; c0 += J0_T) {
        if (threadIdx.x < J0_T) {
            const int64_t c = c0 + threadIdx.x;
            double wv = 0.0;
            for (int s = 0; s < sd.nset; ++s)
                if (c >= sd.col0[s] && c < sd.col0[s] + sd.nocc[s]) wv = sd.w[s];
            wcol[threadIdx.x] = wv;
        }
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int row = ty + 8 * r;
            const int64_t c = c0 + tx;
            const int64_t mu = mu0 + row, nu = nu0 + row;
            /* k-group-major Ccat4[(mu/4)][c][mu%4] */
            Cm[row][tx] = (mu < nao && c < ldc) ? Ccat[((mu >> 2) * ldc + c) * 4 + (mu & 3)] : 0.0;
            Cn[row][tx] = (nu < nao && c < ldc) ? Ccat[((nu >> 2) * ldc + c) * 4 + (nu & 3)] : 0.0;
        }
        __syncthreads();
#pragma unroll 8
        for (int c = 0; c < J0_T; ++c) {
            const double wn = wcol[c] * Cn[tx][c];
#pragma unroll
            for (int r = 0; r < 4; ++r) acc[r] += Cm[ty + 8 * r][c] * wn;
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int64_t mu = mu0 + ty + 8 * r, nu = nu0 + tx;
        if (mu < nao && nu <= mu)
            Dt[mu * (mu + 1) / 2 + nu] = (mu == nu ? 1.0 : 2.0) * acc[r];
    }
}

/* J0 for a general (non-symmetric, non-idempotent) density, 32 x 32 lower tiles:
 *   C2 == NULL:  dm = C1 (nao x nao);   else dm = C1 C2^T (nao x ncol factors)
 *   Dt[mu(mu+1)/2 + nu] = dm[mu][nu] + (mu != nu) * dm[nu][mu]       (J sees only dm + dm^T) */
__global__ void __launch_bounds__(256)
j0_general_dt_kernel(const double *__restrict__ C1, const double *__restrict__ C2, int64_t ncol,
                     int64_t nao, double *__restrict__ Dt)
{
    const int bi = blockIdx.y, bj = blockIdx.x;
    if (bj > bi) return;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int64_t mu0 = (int64_t)bi * J0_T, nu0 = (int64_t)bj * J0_T;
    __shared__ double A1[J0_T][J0_T + 1];      /* C1 rows mu0.. (or dm tile [mu][nu]) */
    __shared__ double A2[J0_T][J0_T + 1];      /* C2 rows mu0.. (or dm tile [nu][mu]) */
    __shared__ double B1[J0_T][J0_T + 1];      /* C1 rows nu0.. */
    __shared__ double B2[J0_T][J0_T + 1];      /* C2 rows nu0.. */
    if (C2 == nullptr) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int row = ty + 8 * r;
            const int64_t mu = mu0 + row, nu = nu0 + tx;
            A1[row][tx] = (mu < nao && nu < nao) ? C1[mu * nao + nu] : 0.0;
            const int64_t a = nu0 + row, b = mu0 + tx;
            A2[row][tx] = (a < nao && b < nao) ? C1[a * nao + b] : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int row = ty + 8 * r;
            const int64_t mu = mu0 + row, nu = nu0 + tx;
            if (mu < nao && nu <= mu)
                Dt[mu * (mu + 1) / 2 + nu] = A1[row][tx] + (mu == nu ? 0.0 : A2[tx][row]);
        }
        return;
    }
    double acc[4] = {0.0, 0.0, 0.0, 0.0};      /* dm[mu][nu] */
    double acct[4] = {0.0, 0.0, 0.0, 0.0};     /* dm[nu][mu] */
    for (int64_t c0 = 0; c0 < ncol; c0 += J0_T) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int row = ty + 8 * r;
            const int64_t c = c0 + tx;
            const int64_t mu = mu0 + row, nu = nu0 + row;
            const bool okm = mu < nao && c < ncol, okn = nu < nao && c < ncol;
            A1[row][tx] = okm ? C1[mu * ncol + c] : 0.0;
            A2[row][tx] = okm ? C2[mu * ncol + c] : 0.0;
            B1[row][tx] = okn ? C1[nu * ncol + c] : 0.0;
            B2[row][tx] = okn ? C2[nu * ncol + c] : 0.0;
        }
        __syncthreads();
#pragma unroll 8
        for (int c = 0; c < J0_T; ++c) {
            const double b1 = B1[tx][c], b2 = B2[tx][c];
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                acc[r] += A1[ty + 8 * r][c] * b2;
                acct[r] += A2[ty + 8 * r][c] * b1;
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int64_t mu = mu0 + ty + 8 * r, nu = nu0 + tx;
        if (mu < nao && nu <= mu)
            Dt[mu * (mu + 1) / 2 + nu] = acc[r] + (mu == nu ? 0.0 : acct[r]);
    }
}

/* ------------------------------------------------------------------ J1 */
constexpr int J1_CH = 4096;          /* columns (pairs) per chunk; Dt chunk = 32 KB of smem */
#ifndef DFJK_J1_WARPS
#define DFJK_J1_WARPS 16   /* swept on B200 at cfg 4 (warps x unroll): 8x8 7.51 ms, 16x8 7.12, 16x6 7.07, 32x8 7.10, 16x16 7.62 */
#endif
#ifndef DFJK_J1_UNROLL
#define DFJK_J1_UNROLL 8
#endif
constexpr int J1_WARPS = DFJK_J1_WARPS;
constexpr int J1_UNROLL = DFJK_J1_UNROLL;         /* 128-bit loads in flight per lane */

__global__ void __launch_bounds__(J1_WARPS * 32)
j1_dot_kernel(const double *__restrict__ B, int64_t naux, int64_t npair,
              const double *__restrict__ Dt, double *__restrict__ d_part)
{
    /* sDt[k] = Dt[c0 - 2 + k], k = 0 .. CH+3 (zero outside [c0, c1)): column c0 sits at the 16-B
     * aligned index 2, so a row segment that starts on the 16-B grid of B (always, when npair is
     * even) reads its Dt pairs with one conflict-free 128-bit shared load per 128-bit global load;
     * two 64-bit loads at a 16-B lane stride would cost twice the shared-memory wavefronts
     * (profiles/r01b: mio_throttle was J1's top stall). */
    __shared__ __align__(16) double sDt[J1_CH + 4];
    const int64_t chunk = blockIdx.x;
    const int64_t c0 = chunk * J1_CH;
    const int64_t c1 = (c0 + J1_CH < npair) ? c0 + J1_CH : npair;
    for (int k = threadIdx.x; k < J1_CH + 4; k += blockDim.x) {
        const int64_t col = c0 - 2 + k;
        sDt[k] = (col >= c0 && col < c1) ? Dt[col] : 0.0;
    }
    __syncthreads();

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t row_stride = (int64_t)gridDim.y * J1_WARPS;
    for (int64_t P = (int64_t)blockIdx.y * J1_WARPS + warp; P < naux; P += row_stride) {
        const int64_t base = P * npair;
        const int64_t f0 = base + c0, f1 = base + c1;       /* flat range of this segment */
        const int64_t fa = (f0 + 1) & ~(int64_t)1;          /* first 16-B aligned element */
        const int64_t fb = f1 & ~(int64_t)1;                /* end of aligned body */
        double acc0 = 0.0, acc1 = 0.0;
        if (fa <= fb) {
            /* head / tail scalars */
            if (lane == 0 && f0 < fa) acc0 += ldg_stream1(B + f0) * sDt[2];
            if (lane == 1 && fb < f1) acc1 += ldg_stream1(B + fb) * sDt[fb - f0 + 2];
            const int64_t nvec = (fb - fa) >> 1;
            const double *bp = B + fa;
            const double *sp = sDt + (fa - f0 + 2);
            int64_t v = lane;
            if (fa == f0) {
                /* aligned segment: 128-bit shared loads */
                const double2 *sp2 = reinterpret_cast<const double2 *>(sp);
                for (; v + 32 * (J1_UNROLL - 1) < nvec; v += 32 * J1_UNROLL) {
                    double2 b[J1_UNROLL];
#pragma unroll
                    for (int u = 0; u < J1_UNROLL; ++u) b[u] = ldg_stream2(bp + 2 * (v + 32 * u));
#pragma unroll
                    for (int u = 0; u < J1_UNROLL; ++u) {
                        const double2 t = sp2[v + 32 * u];
                        acc0 += b[u].x * t.x;
                        acc1 += b[u].y * t.y;
                    }
                }
                for (; v < nvec; v += 32) {
                    const double2 b = ldg_stream2(bp + 2 * v);
                    const double2 t = sp2[v];
                    acc0 += b.x * t.x;
                    acc1 += b.y * t.y;
                }
            } else {
                for (; v + 32 * (J1_UNROLL - 1) < nvec; v += 32 * J1_UNROLL) {
                    double2 b[J1_UNROLL];
#pragma unroll
                    for (int u = 0; u < J1_UNROLL; ++u) b[u] = ldg_stream2(bp + 2 * (v + 32 * u));
#pragma unroll
                    for (int u = 0; u < J1_UNROLL; ++u) {
                        const int64_t k = 2 * (v + 32 * u);
                        acc0 += b[u].x * sp[k];
                        acc1 += b[u].y * sp[k + 1];
                    }
                }
                for (; v < nvec; v += 32) {
                    const double2 b = ldg_stream2(bp + 2 * v);
                    acc0 += b.x * sp[2 * v];
                    acc1 += b.y * sp[2 * v + 1];
                }
            }
        } else {
            /* segment of a single element straddling the 16-B grid */
            if (lane == 0) acc0 += ldg_stream1(B + f0) * sDt[2];
        }
        double acc = acc0 + acc1;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (lane == 0) d_part[chunk * naux + P] = acc;
    }
}

/* ------------------------------------------------------------------ J1X */
/* d_P without a pass over B, for calls that also build K:  <B_P, C C^T> = <B_P C, C> = <X_P, C>, and
 * X_P = B_P C is what K1 has just written.  So
 *     d_P = sum_s w_s sum_{mu,i} X_P^s[mu][i] C_s[mu][i]
 * is one pass over the X chunk (8.7 GB per call at cfg 4 instead of the 51 GB of B that J1 streams).
 * For one P, X4[(p*ldx4 + cg)][mu][4] is a contiguous array of nao*ldx doubles; "unit" u is its
 * u-th 16-byte piece = X_P[mu][col], X_P[mu][col+1] with col = 4 cg + 2 h, u = (cg*nao + mu)*2 + h.
 * A thread takes one unit per tile of 256, keeps the two matching C values (times w) in registers
 * and walks J1X_PB consecutive P with them: every warp load is 512 contiguous bytes.  A CTA covers
 * `tiles` tiles; its 256 x PB shares are reduced through shared memory in a fixed order into
 * d_part[blockIdx.x][P] (deterministic; J1R adds the blocks). */
constexpr int J1X_PB = 16;            /* P per CTA */
constexpr int J1X_PARTS = 256 / J1X_PB;
/* tiles of 256 units per CTA: swept on B200 at cfg 4, PB x tiles = 16 x 8: 2.10 ms, 16 x 2: 1.50, 8 x 1: 1.41,
 * 16 x 1: 1.29 ms (6.7 TB/s) -- short CTAs, many in flight; J1R then adds 425 instead of 53 partials per P.
 * One tile per CTA up to J1X_MAX_BLOCKS blocks (occupied-orbital widths: cfg 4 has 425, cfg 5 1313); wider
 * column blocks (pair / raw-dm calls up to ldc = 2 nao) give each CTA more tiles, so that d_part -- one
 * row of naux doubles per block -- stays below J1X_MAX_BLOCKS * naux doubles (82 MB at cfg 4) instead of
 * nao^2/256 * naux (0.8 GB). */
constexpr int64_t J1X_MAX_BLOCKS = 2048;

__global__ void __launch_bounds__(256)
j1x_dot_kernel(const double *__restrict__ X4, const double *__restrict__ Ccat4, int64_t nao, int64_t np,
               int64_t ldx4, int64_t ldc, int64_t c_shift, SetDesc sd, int64_t P0, int64_t naux,
               int tiles, double *__restrict__ d_part)
{
    __shared__ double ts[J1X_PB][264];                     /* this thread's share of d_P, P in the CTA's range */
    const int64_t nunit = (ldc / 4) * nao * 2;             /* units that face columns of Ccat */
    const int64_t p0 = (int64_t)blockIdx.y * J1X_PB;
    const int64_t pstride = ldx4 * nao * 4;                /* doubles between consecutive P */
    double t[J1X_PB];
#pragma unroll
    for (int pp = 0; pp < J1X_PB; ++pp) t[pp] = 0.0;
    for (int tile = 0; tile < tiles; ++tile) {
        const int64_t u = ((int64_t)blockIdx.x * tiles + tile) * 256 + threadIdx.x;
        if (u >= nunit) break;
        const int64_t row = u >> 1;                        /* cg*nao + mu */
        const int64_t cg = row / nao, mu = row - cg * nao;
        const int64_t col = 4 * cg + 2 * (u & 1);
        double w = 0.0;
        for (int s = 0; s < sd.nset; ++s)
            if (col >= sd.col0[s] && col < sd.col0[s] + sd.nocc[s]) w = sd.w[s];
        if (w == 0.0) continue;                            /* padding columns: C is zero there */
        /* c_shift: the C columns are taken c_shift to the right of the X columns (pair form:
         * d_P = <B_P C1, C2> with Ccat = [C1 | C2]) */
        const double *cp = Ccat4 + ((mu >> 2) * ldc + col + c_shift) * 4 + (mu & 3);
        const double c0 = w * cp[0], c1 = w * cp[4];
        const double2 *x = reinterpret_cast<const double2 *>(X4) + u + p0 * (pstride / 2);
#pragma unroll
        for (int pp = 0; pp < J1X_PB; ++pp) {
            if (p0 + pp < np) {
                const double2 v = __ldcs(x + pp * (pstride / 2));
                t[pp] += v.x * c0 + v.y * c1;
            }
        }
    }
#pragma unroll
    for (int pp = 0; pp < J1X_PB; ++pp) ts[pp][threadIdx.x] = t[pp];
    __syncthreads();
    /* thread (pp, part) adds 256 / PARTS of the 256 shares of P = p0 + pp, then the parts are added
     * across lanes: a fixed order */
    {
        const int pp = threadIdx.x / J1X_PARTS, part = threadIdx.x % J1X_PARTS;
        double acc = 0.0;
#pragma unroll 8
        for (int j = 0; j < 256 / J1X_PARTS; ++j) acc += ts[pp][part + J1X_PARTS * j];
#pragma unroll
        for (int o = 1; o < J1X_PARTS; o <<= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (part == 0 && p0 + pp < np) d_part[(int64_t)blockIdx.x * naux + P0 + p0 + pp] = acc;
    }
}

/* d[P] = sum_c d_part[c][P]: 32 P x 8 groups per CTA, group g adds the chunks c = g, g + 8, ... (loads
 * pipelined), the eight group sums are added in order: a fixed order, as everywhere */
__global__ void __launch_bounds__(256)
j1_reduce_kernel(const double *__restrict__ d_part, int64_t nchunk, int64_t naux, double *__restrict__ d)
{
    __shared__ double gs[8][33];
    const int pl = threadIdx.x & 31, g = threadIdx.x >> 5;
    const int64_t P = (int64_t)blockIdx.x * 32 + pl;
    double acc = 0.0;
    if (P < naux) {
#pragma unroll 8
        for (int c = g; c < (int)nchunk; c += 8) acc += d_part[(int64_t)c * naux + P];
    }
    gs[g][pl] = acc;
    __syncthreads();
    if (g == 0 && P < naux) {
        double v = gs[0][pl];
#pragma unroll
        for (int q = 1; q < 8; ++q) v += gs[q][pl];
        d[P] = v;
    }
}

/* the same sum for the np rows [P0, P0 + np) only, written to d_out[P0 ..]: the batched build
 * (dfjk_get_jk_pairs) reduces every X chunk's partials at once, into the d vector of one density */
__global__ void __launch_bounds__(256)
j1_reduce_rows_kernel(const double *__restrict__ d_part, int64_t nchunk, int64_t naux, int64_t P0, int64_t np,
                      double *__restrict__ d_out)
{
    __shared__ double gs[8][33];
    const int pl = threadIdx.x & 31, g = threadIdx.x >> 5;
    const int64_t p = (int64_t)blockIdx.x * 32 + pl;
    double acc = 0.0;
    if (p < np) {
#pragma unroll 8
        for (int c = g; c < (int)nchunk; c += 8) acc += d_part[(int64_t)c * naux + P0 + p];
    }
    gs[g][pl] = acc;
    __syncthreads();
    if (g == 0 && p < np) {
        double v = gs[0][pl];
#pragma unroll
        for (int q = 1; q < 8; ++q) v += gs[q][pl];
        d_out[P0 + p] = v;
    }
}

/* ------------------------------------------------------------------ J2 */
#ifndef DFJK_J2_THREADS
#define DFJK_J2_THREADS 256
#endif
#ifndef DFJK_J2_UNROLL
#define DFJK_J2_UNROLL 12  /* swept on B200 at cfg 4: 8 -> 8.13 ms, 12 -> 7.18, 16 -> 7.22, 32 -> 7.43 */
#endif
constexpr int J2_THREADS = DFJK_J2_THREADS;
constexpr int J2_UNROLL = DFJK_J2_UNROLL;

/* SQ == false: J2 proper, Jp_part[g][pair] = sum_{P in group g} d[P] B[P][pair].
 * SQ == true : the DF diagonal of Eq. 7, sum_P B[P][pair]^2 -- the same stream
 *              with each element weighted by itself (d is not read). */
template <bool SQ>
__global__ void __launch_bounds__(J2_THREADS)
j2_axpy_kernel(const double *__restrict__ B, int64_t naux, int64_t npair,
               const double *__restrict__ d, double *__restrict__ Jp_part, int64_t ngroup)
{
    const int64_t g = blockIdx.y;
    /* all rows of group g (P = g + t*ngroup, ngroup even) share the parity of P*npair */
    const int64_t s = (g * npair) & 1;
    const int64_t vv = (int64_t)blockIdx.x * J2_THREADS + threadIdx.x;
    const int64_t colx = 2 * vv - s, coly = colx + 1;       /* columns this thread owns */
    const bool okx = colx >= 0 && colx < npair;
    const bool oky = coly < npair;                          /* coly >= 0 always */
    if (!okx && !oky) return;
    double ax = 0.0, ay = 0.0;
    if (okx && oky) {
        const double *bp = B + colx;                        /* + P*npair is 16-B aligned */
        int64_t P = g;
        for (; P + (J2_UNROLL - 1) * ngroup < naux; P += J2_UNROLL * ngroup) {
            double2 b[J2_UNROLL];
            double dv[J2_UNROLL];
#pragma unroll
            for (int u = 0; u < J2_UNROLL; ++u) {
                b[u] = ldg_stream2(bp + (P + u * ngroup) * npair);
                dv[u] = SQ ? 0.0 : __ldg(d + P + u * ngroup);
            }
#pragma unroll
            for (int u = 0; u < J2_UNROLL; ++u) {
                ax += (SQ ? b[u].x : dv[u]) * b[u].x;
                ay += (SQ ? b[u].y : dv[u]) * b[u].y;
            }
        }
        for (; P < naux; P += ngroup) {
            const double2 b = ldg_stream2(bp + P * npair);
            const double dv = SQ ? 0.0 : __ldg(d + P);
            ax += (SQ ? b.x : dv) * b.x;
            ay += (SQ ? b.y : dv) * b.y;
        }
    } else {
        const int64_t col = okx ? colx : coly;
        double a = 0.0;
        for (int64_t P = g; P < naux; P += ngroup) {
            const double b = ldg_stream1(B + P * npair + col);
            a += (SQ ? b : __ldg(d + P)) * b;
        }
        if (okx) ax = a; else ay = a;
    }
    double *out = Jp_part + g * npair;
    if (okx) out[colx] = ax;
    if (oky) out[coly] = ay;
}

/* J2 for NB densities in ONE pass over B (dfjk_get_jk_pairs / _dms: "an arbitrary number of density
 * matrices"):  Jp_part[(k*ngroup + g)][pair] = sum_{P in group g} d[k][P] B[P][pair], k < NB.
 * The stream is J2's (same column ownership, same 128-bit evict-first loads, same row groups); every
 * loaded element feeds NB FMAs instead of one, so B is read once for the whole batch.  Per density the
 * additions happen in J2's order: the result is bitwise that of NB single-density passes. */
template <int NB, int UNROLL>
__global__ void __launch_bounds__(J2_THREADS)
j2_axpy_multi_kernel(const double *__restrict__ B, int64_t naux, int64_t npair, const double *__restrict__ d,
                     double *__restrict__ Jp_part, int64_t ngroup)
{
    const int64_t g = blockIdx.y;
    const int64_t s = (g * npair) & 1;
    const int64_t vv = (int64_t)blockIdx.x * J2_THREADS + threadIdx.x;
    const int64_t colx = 2 * vv - s, coly = colx + 1;
    const bool okx = colx >= 0 && colx < npair;
    const bool oky = coly < npair;
    if (!okx && !oky) return;
    double ax[NB], ay[NB];
#pragma unroll
    for (int k = 0; k < NB; ++k) ax[k] = ay[k] = 0.0;
    if (okx && oky) {
        const double *bp = B + colx;
        int64_t P = g;
        for (; P + (UNROLL - 1) * ngroup < naux; P += UNROLL * ngroup) {
            double2 b[UNROLL];
#pragma unroll
            for (int u = 0; u < UNROLL; ++u) b[u] = ldg_stream2(bp + (P + u * ngroup) * npair);
#pragma unroll
            for (int u = 0; u < UNROLL; ++u) {
#pragma unroll
                for (int k = 0; k < NB; ++k) {
                    const double dv = __ldg(d + k * naux + P + u * ngroup);
                    ax[k] += dv * b[u].x;
                    ay[k] += dv * b[u].y;
                }
            }
        }
        for (; P < naux; P += ngroup) {
            const double2 b = ldg_stream2(bp + P * npair);
#pragma unroll
            for (int k = 0; k < NB; ++k) {
                const double dv = __ldg(d + k * naux + P);
                ax[k] += dv * b.x;
                ay[k] += dv * b.y;
            }
        }
    } else {
        const int64_t col = okx ? colx : coly;
        for (int64_t P = g; P < naux; P += ngroup) {
            const double b = ldg_stream1(B + P * npair + col);
#pragma unroll
            for (int k = 0; k < NB; ++k) {
                const double t = __ldg(d + k * naux + P) * b;
                if (okx) ax[k] += t; else ay[k] += t;
            }
        }
    }
#pragma unroll
    for (int k = 0; k < NB; ++k) {
        double *out = Jp_part + (k * ngroup + g) * npair;
        if (okx) out[colx] = ax[k];
        if (oky) out[coly] = ay[k];
    }
}

/* ------------------------------------------------------------------ J3 */
constexpr int J3_T = 32;

__global__ void __launch_bounds__(256)
j3_unpack_kernel(const double *__restrict__ Jp_part, int64_t ngroup, int64_t npair, int64_t nao,
                 double *__restrict__ Jdirect, double *const *__restrict__ Jslot)
{
    const int bi = blockIdx.y, bj = blockIdx.x;
    if (bj > bi) return;
    /* Jslot != NULL: the output pointer of THIS call sits in device memory (written by K0), so that
     * one captured launch sequence serves every call (dfjk_api.cu, "graph") */
    double *__restrict__ J = Jslot ? *Jslot : Jdirect;
    __shared__ double t[J3_T][J3_T + 1];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int64_t mu0 = (int64_t)bi * J3_T, nu0 = (int64_t)bj * J3_T;
    /* the four rows of a thread are summed side by side, eight groups per round, so that 32 loads are
     * in flight at once (one row after the other was a chain of L2 round trips: 29 us at nao = 290);
     * each element still adds its groups in ascending order */
    const double *src[4];
    double v[4];
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int64_t mu = mu0 + ty + 8 * r, nu = nu0 + tx;
        src[r] = (mu < nao && nu <= mu) ? Jp_part + mu * (mu + 1) / 2 + nu : nullptr;
        v[r] = 0.0;
    }
#pragma unroll 8
    for (int g = 0; g < (int)ngroup; ++g)
#pragma unroll
        for (int r = 0; r < 4; ++r)
            if (src[r]) v[r] += src[r][(int64_t)g * npair];
#pragma unroll
    for (int r = 0; r < 4; ++r) t[ty + 8 * r][tx] = v[r];
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int row = ty + 8 * r;
        const int64_t mu = mu0 + row, nu = nu0 + tx;
        if (mu < nao && nu < nao) {
            const double v = (bi == bj && tx > row) ? t[tx][row] : t[row][tx];
            J[mu * nao + nu] = v;
        }
        if (bi != bj) {
            /* mirrored tile: J[nu0+row][mu0+tx] = t[tx][row] */
            const int64_t a = nu0 + row, b = mu0 + tx;
            if (a < nao && b < nao) J[a * nao + b] = t[tx][row];
        }
    }
}

}  // namespace

/* ------------------------------------------------------------------ launchers */
void launch_j0_build_dt(const double *Ccat, int64_t ldc, int64_t nao, int nset, const int *col0,
                        const int *nocc, const double *w, double *Dt, cudaStream_t st)
{
    SetDesc sd;
    sd.nset = nset;
    for (int s = 0; s < 4; ++s) {
        sd.col0[s] = s < nset ? col0[s] : 0;
        sd.nocc[s] = s < nset ? nocc[s] : 0;
        sd.w[s] = s < nset ? w[s] : 0.0;
    }
    const unsigned nb = (unsigned)((nao + J0_T - 1) / J0_T);
    j0_build_dt_kernel<<<dim3(nb, nb), 256, 0, st>>>(Ccat, ldc, nao, sd, Dt);
}

void launch_j0_general_dt(const double *C1, const double *C2, int64_t ncol, int64_t nao, double *Dt,
                          cudaStream_t st)
{
    const unsigned nb = (unsigned)((nao + J0_T - 1) / J0_T);
    j0_general_dt_kernel<<<dim3(nb, nb), 256, 0, st>>>(C1, C2, ncol, nao, Dt);
}

int64_t j1_num_chunks(int64_t npair) { return (npair + J1_CH - 1) / J1_CH; }

void launch_j1_dot(const double *B, int64_t naux, int64_t npair, const double *Dt, double *d_part,
                   int sm_count, cudaStream_t st)
{
    const int64_t nchunk = j1_num_chunks(npair);
    int64_t rg = (16LL * sm_count + nchunk - 1) / nchunk;   /* aim at >= 16 CTAs per SM in total */
    const int64_t rg_max = (naux + J1_WARPS - 1) / J1_WARPS;
    if (rg > rg_max) rg = rg_max;
    if (rg < 1) rg = 1;
    if (rg > 65535) rg = 65535;
    j1_dot_kernel<<<dim3((unsigned)nchunk, (unsigned)rg), J1_WARPS * 32, 0, st>>>(B, naux, npair, Dt,
                                                                                  d_part);
}

static int64_t j1x_tiles_per_cta(int64_t nao, int64_t ldc)
{
    const int64_t ntile = ((ldc / 4) * nao * 2 + 255) / 256;
    return ntile <= J1X_MAX_BLOCKS ? 1 : (ntile + J1X_MAX_BLOCKS - 1) / J1X_MAX_BLOCKS;
}

/* upper bound of j1x_num_blocks over every ldc <= ldc_max (the block count is not monotonic in ldc
 * once CTAs take several tiles): what dfjk_create sizes d_part for */
int64_t j1x_max_blocks(int64_t nao, int64_t ldc_max)
{
    const int64_t ntile = ((ldc_max / 4) * nao * 2 + 255) / 256;
    return ntile < J1X_MAX_BLOCKS ? ntile : J1X_MAX_BLOCKS;
}

int64_t j1x_num_blocks(int64_t nao, int64_t ldc)
{
    const int64_t per_cta = 256LL * j1x_tiles_per_cta(nao, ldc);
    return ((ldc / 4) * nao * 2 + per_cta - 1) / per_cta;
}

void launch_j1x_dot(const double *X4, const double *Ccat4, int64_t nao, int64_t np, int64_t ldx, int64_t ldc,
                    int64_t c_shift, int nset, const int *col0, const int *nocc, const double *w, int64_t P0,
                    int64_t naux, double *d_part, cudaStream_t st)
{
    SetDesc sd;
    sd.nset = nset;
    for (int s = 0; s < 4; ++s) {
        sd.col0[s] = s < nset ? col0[s] : 0;
        sd.nocc[s] = s < nset ? nocc[s] : 0;
        sd.w[s] = s < nset ? w[s] : 0.0;
    }
    dim3 grid((unsigned)j1x_num_blocks(nao, ldc), (unsigned)((np + J1X_PB - 1) / J1X_PB));
    j1x_dot_kernel<<<grid, 256, 0, st>>>(X4, Ccat4, nao, np, ldx / 4, ldc, c_shift, sd, P0, naux,
                                         (int)j1x_tiles_per_cta(nao, ldc), d_part);
}

void launch_j1_reduce(const double *d_part, int64_t nchunk, int64_t naux, double *d, cudaStream_t st)
{
    j1_reduce_kernel<<<(unsigned)((naux + 31) / 32), 256, 0, st>>>(d_part, nchunk, naux, d);
}

int64_t j2_num_groups(int64_t naux, int64_t npair, int sm_count)
{
    const int64_t nbx = (npair + 1) / 2 / J2_THREADS + 1;
    int64_t g = (16LL * sm_count + nbx - 1) / nbx;
    if (g < 2) g = 2;
    g += g & 1;                               /* even: one 16-B alignment class per group */
    int64_t gmax = naux / 8;                  /* keep >= 8 rows per group when possible */
    gmax -= gmax & 1;
    if (gmax < 2) gmax = 2;
    if (g > gmax) g = gmax;
    return g;
}

void launch_j2_axpy(const double *B, int64_t naux, int64_t npair, const double *d, double *Jp_part,
                    int64_t ngroup, cudaStream_t st)
{
    const int64_t nvec = (npair + 1) / 2 + 1;               /* one spare vector for shifted rows */
    const unsigned nbx = (unsigned)((nvec + J2_THREADS - 1) / J2_THREADS);
    if (d)
        j2_axpy_kernel<false><<<dim3(nbx, (unsigned)ngroup), J2_THREADS, 0, st>>>(B, naux, npair, d,
                                                                                  Jp_part, ngroup);
    else    /* d == NULL: Eq. 7's DF diagonal, sum_P B[P][pair]^2 */
        j2_axpy_kernel<true><<<dim3(nbx, (unsigned)ngroup), J2_THREADS, 0, st>>>(B, naux, npair, nullptr,
                                                                                 Jp_part, ngroup);
}

void launch_j1_reduce_rows(const double *d_part, int64_t nchunk, int64_t naux, int64_t P0, int64_t np,
                           double *d_out, cudaStream_t st)
{
    j1_reduce_rows_kernel<<<(unsigned)((np + 31) / 32), 256, 0, st>>>(d_part, nchunk, naux, P0, np, d_out);
}

void launch_j2_axpy_multi(const double *B, int64_t naux, int64_t npair, const double *d, int nbatch,
                          double *Jp_part, int64_t ngroup, cudaStream_t st)
{
    const int64_t nvec = (npair + 1) / 2 + 1;
    const dim3 grid((unsigned)((nvec + J2_THREADS - 1) / J2_THREADS), (unsigned)ngroup);
#define DFJK_J2M(NB, U) j2_axpy_multi_kernel<NB, U><<<grid, J2_THREADS, 0, st>>>(B, naux, npair, d, Jp_part, ngroup)
    switch (nbatch) {
    case 1: DFJK_J2M(1, 12); break;
    case 2: DFJK_J2M(2, 12); break;
    case 3: DFJK_J2M(3, 12); break;
    case 4: DFJK_J2M(4, 12); break;
    case 5: DFJK_J2M(5, 8); break;
    case 6: DFJK_J2M(6, 8); break;
    case 7: DFJK_J2M(7, 8); break;
    default: DFJK_J2M(8, 8); break;     /* nbatch <= DFJK_MAX_BATCH = 8, checked by the caller */
    }
#undef DFJK_J2M
}

void launch_j3_unpack(const double *Jp_part, int64_t ngroup, int64_t npair, int64_t nao, double *J,
                      double *const *Jslot, cudaStream_t st)
{
    const unsigned nb = (unsigned)((nao + J3_T - 1) / J3_T);
    j3_unpack_kernel<<<dim3(nb, nb), 256, 0, st>>>(Jp_part, ngroup, npair, nao, J, Jslot);
}

}  // namespace dfjk
