/*
 * k2_syrk.cu -- K0 (orbital packing), K2 (lower-triangle SYRK) and K3 (finish) of the
 * exchange build (include/dfjk.h), sm_100a:
 *
 *     K_s[mu][nu] += sum_{P in chunk} sum_{i in set s} X_P[mu][i] X_P[nu][i]     mu-tile >= nu-tile
 *
 * X chunk layout (written by K1): k-group-major X4[k/4][mu][k%4], k = p*ldc + i, so the
 * 128-row operand panel of one k-group (4 columns) is 4 KB of contiguous memory and lands
 * in shared memory, by one 1-D bulk copy (TMA engine, UBLKCP), already in the dense
 * [row][4] form whose DMMA fragment loads are bank-conflict-free.  A stage holds eight
 * k-groups (k = 32) of both operands; 3 stages, full/empty mbarriers, one producer lane.
 * One CTA owns a 128 x 128 tile of K for one k-split: 8 consumer warps as 2 (M) x 4 (N),
 * warp tile 64 x 32 = 8 x 4 DMMA.8x8x4 accumulators, 12 shared loads per 32 MMAs.  Both
 * operands are row panels of X, so A (row-major) and B (col-major) fragments are read with
 * the same pattern; diagonal tiles load the panel once and use a triangular warp layout (the
 * 36 units of 16 x 16 that touch the lower triangle, five or four per warp: tri_unit); block rows with
 * <= 64 valid rows use a 1 x 8 layout of 64 x 16 warp tiles (and, in the full product, block columns
 * with <= 64 valid columns a 4 x 2 layout of 32 x 32), so no warp idles on ragged tiles; the number
 * of valid 8-row MMA rows of a ragged warp tile is a template parameter (rect_stage).
 * The same kernel with FULL = true covers all nb x nb tiles with operands from two column
 * ranges of X (the non-symmetric product of the general-density entry points).
 * Splits: work item = (lower tile, split) with its own partial accumulator Kpart[split],
 * read-modify-written by exactly one CTA per launch => deterministic, no atomics; small problems
 * cut each tile in proportion to its cost (k2_tile_splits).
 * Larger problems (>= 21 lower tiles, X chunk beyond L2) run the panel-synchronous K2P kernel below.
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
    double *out[DFJK_OUT_SLOTS];        /* this call's output pointers (J, K_0, K_1, ...) */
    double **out_slots;                 /* device array they are published to, or NULL */
};

/* Ccat4[(mu/4)][c][mu%4], mu < nao16 (rows >= nao and padding columns are zero).  Thread 0 also
 * publishes the call's output pointers to out_slots: the finishing kernels (K3, J3) of a captured
 * launch sequence read them from there (stream order makes K0's write visible to them). */
__global__ void k0_pack_c_kernel(PackDesc pd, int64_t nao, int64_t nao16, int64_t ldc,
                                 double *__restrict__ Ccat4)
{
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx == 0 && pd.out_slots)
        for (int i = 0; i < DFJK_OUT_SLOTS; ++i) pd.out_slots[i] = pd.out[i];
    if (idx >= nao16 * ldc) return;
    const int64_t mu = idx / ldc;
    const int c = (int)(idx % ldc);
    double v = 0.0;
    if (mu < nao)
        for (int s = 0; s < pd.nset; ++s)
            if (c >= pd.col0[s] && c < pd.col0[s] + pd.nocc[s])
                v = pd.C[s][mu * pd.nocc[s] + (c - pd.col0[s])];
    Ccat4[((mu >> 2) * ldc + c) * 4 + (mu & 3)] = v;
}

/* One factor into a column range of Ccat4: columns [col0, col0 + width) = C (nao x ncol, zero beyond
 * ncol and for rows >= nao).  The batched build packs its 2 x nbatch factors one by one. */
__global__ void k0_pack_cols_kernel(const double *__restrict__ C, int64_t ncol, int64_t col0, int64_t width,
                                    int64_t nao, int64_t nao16, int64_t ldc, double *__restrict__ Ccat4)
{
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= nao16 * width) return;
    const int64_t mu = idx / width;
    const int64_t j = idx % width;
    const double v = (mu < nao && j < ncol) ? C[mu * ncol + j] : 0.0;
    Ccat4[((mu >> 2) * ldc + col0 + j) * 4 + (mu & 3)] = v;
}

/* ------------------------------------------------------------------ K2 */
constexpr int K2_T = 128;
constexpr int K2_KG = 8;                              /* k-groups (of 4) per stage: k = 32 */
constexpr int K2_STAGES = 3;
constexpr int K2_OP_BYTES = K2_KG * K2_T * 32;        /* one operand, one stage: [kg][128][4] */
constexpr int K2_STAGE_BYTES = 2 * K2_OP_BYTES;       /* 65536 */
constexpr int K2_CONSUMER_WARPS = 8;
constexpr int K2_THREADS = 32 * (1 + K2_CONSUMER_WARPS);
constexpr int K2_SMEM_BYTES = K2_STAGES * K2_STAGE_BYTES + 2 * K2_STAGES * 8 + 16;

/* Lower tiles are not equally expensive: a full-height diagonal tile issues 9/16 of the MMAs of an
 * off-diagonal one, a ragged last block row its share of valid MMA rows (rect_stage_full / _narrow), its
 * diagonal tile half of that when it has <= 64 rows.  The split kernel therefore cuts the k range of a tile into a number of splits
 * PROPORTIONAL to its cost -- nsplit is the count of a full off-diagonal tile -- so that all CTAs of
 * the single wave runs about equally long; with the same count for every tile a launch took as long
 * as its off-diagonal CTAs while the others idled (44 % of the SM-time at nao = 290).  Used while
 * there are fewer lower tiles than SMs ("weighted"): with many waves the equal split does better
 * (the cheap last block row runs last and shortens the tail: nao = 4000, 61.7 vs 63.1 ms). */
__host__ __device__ inline int k2_tile_splits(int bi, int bj, int64_t nao, int nsplit)
{
    const int64_t rows = nao - (int64_t)bi * K2_T;
    int c16 = bi == bj ? 9 : 16;                             /* cost in sixteenths of a full tile */
    if (rows <= 64) c16 = (rows <= 16 ? 2 : (rows <= 32 ? 4 : 8)) / (bi == bj ? 2 : 1);   /* 1 x 8 layout */
    else if (rows < K2_T && bi != bj) c16 = 8 + 2 * (int)((rows - 64 + 15) / 16);      /* 2 x 4: ragged lower warp row */
    if (c16 < 1) c16 = 1;
    const int s = (nsplit * c16 + 8) / 16;
    return s < 1 ? 1 : s;
}

/* Triangular layout of a full-height DIAGONAL tile: the lower triangle in units of 16 x 16 (2 x 2
 * MMA tiles), strip r (rows 16r .. 16r+15) holding the units c = 0 .. r -- 36 units = 144 MMA tiles
 * where the square has 256 (an earlier 32 x 16 unit layout issued 192).  Warps 0-3 take five units
 * each, all in one strip (strip 7 - cw, c = 0 .. 4: a 16 x 80 warp tile); warps 4-7 take the other
 * sixteen, four each, as listed below.  The two warps of a sub-partition (cw, cw + 4) hold 5 + 4. */
__device__ __forceinline__ void tri_unit(int j, int u, int &r, int &c)      /* j = cw - 4, u < 4 */
{
    /* j = 0: (7,5) (7,6) (7,7) (0,0);  1: (6,5) (6,6) (1,0) (1,1);  2: (5,5) (2,0) (2,1) (2,2);  3: (3,0..3) */
    const unsigned rows = j == 0 ? 0x0777u : (j == 1 ? 0x1166u : (j == 2 ? 0x2225u : 0x3333u));
    const unsigned cols = j == 0 ? 0x0765u : (j == 1 ? 0x1065u : (j == 2 ? 0x2105u : 0x3210u));
    r = (int)((rows >> (4 * u)) & 15u);
    c = (int)((cols >> (4 * u)) & 15u);
}

/* one stage (n <= 8 k-groups) of a diagonal tile for a warp of the wide kind (cw < 4): acc[mt * 10 + nt] */
__device__ __forceinline__ void tri_stage_wide(double (*acc)[2], const double *a_base, const double *b_base, int n)
{
#pragma unroll
    for (int q = 0; q < K2_KG; ++q) {
        if (q < n) {
            double a[2], b[10];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) a[mt] = a_base[q * (K2_T * 4) + mt * 32];
#pragma unroll
            for (int nt = 0; nt < 10; ++nt) b[nt] = b_base[q * (K2_T * 4) + nt * 32];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int nt = 0; nt < 10; ++nt)
                    dmma884(acc[mt * 10 + nt][0], acc[mt * 10 + nt][1], a[mt], b[nt]);
        }
    }
}

/* ... and of the unit kind (cw >= 4): four 16 x 16 units at ua[u] / ub[u] (offsets in doubles into the
 * panel, lane part included): acc[4 u + 2 mt + nt] */
__device__ __forceinline__ void tri_stage_units(double (*acc)[2], const double *X, const int (&ua)[4],
                                                const int (&ub)[4], int n)
{
#pragma unroll
    for (int q = 0; q < K2_KG; ++q) {
        if (q < n) {
            double a[4][2], b[4][2];
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    a[u][t] = X[ua[u] + q * (K2_T * 4) + t * 32];
                    b[u][t] = X[ub[u] + q * (K2_T * 4) + t * 32];
                }
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                    for (int nt = 0; nt < 2; ++nt)
                        dmma884(acc[4 * u + 2 * mt + nt][0], acc[4 * u + 2 * mt + nt][1], a[u][mt], b[u][nt]);
        }
    }
}

/* one stage (n <= 8 k-groups) of a rectangular warp tile of NMT x NNT MMA tiles: acc[mt * 4 + nt].
 * The tile shape is a TEMPLATE parameter, never a runtime bound: with `if (mt < nmt)` around the
 * (non-volatile) MMA the compiler is free to issue it anyway and select the result, and did (7.5 % more
 * DMMAs at nao = 800, visible only in ncu's op count). */
template <int NMT, int NNT>
__device__ __forceinline__ void rect_stage(double (*acc)[2], const double *a_base, const double *b_base, int n)
{
#pragma unroll
    for (int q = 0; q < K2_KG; ++q) {
        if (q < n) {
            double a[NMT], b[NNT];
#pragma unroll
            for (int mt = 0; mt < NMT; ++mt) a[mt] = a_base[q * (K2_T * 4) + mt * 32];
#pragma unroll
            for (int nt = 0; nt < NNT; ++nt) b[nt] = b_base[q * (K2_T * 4) + nt * 32];
#pragma unroll
            for (int mt = 0; mt < NMT; ++mt)
#pragma unroll
                for (int nt = 0; nt < NNT; ++nt)
                    dmma884(acc[mt * 4 + nt][0], acc[mt * 4 + nt][1], a[mt], b[nt]);
        }
    }
}

/* ... with the number of valid 8-row MMA rows of the warp tile chosen at run time (warp-uniform), from
 * a SHORT list: ragged block rows cost what they hold in steps of 16 rows (2 x 4 layout: 2, 4, 6 or 8 MMA
 * rows in the lower warp row) or 16 / 32 / 64 rows (1 x 8 layout).  One instantiation per MMA row count
 * (8 + 8 unrolled loops) cost more in instruction fetch than it saved: cfg 4 K2 +1.5 %, cfg 2 +21 %. */
__device__ __forceinline__ void rect_stage_full(int nmt, double (*acc)[2], const double *a_base,
                                                const double *b_base, int n)
{
    if (nmt > 6) rect_stage<8, 4>(acc, a_base, b_base, n);
    else if (nmt > 4) rect_stage<6, 4>(acc, a_base, b_base, n);
    else if (nmt > 2) rect_stage<4, 4>(acc, a_base, b_base, n);
    else rect_stage<2, 4>(acc, a_base, b_base, n);
}
__device__ __forceinline__ void rect_stage_narrow(int nmt, double (*acc)[2], const double *a_base,
                                                  const double *b_base, int n)
{
    if (nmt > 4) rect_stage<8, 2>(acc, a_base, b_base, n);
    else if (nmt > 2) rect_stage<4, 2>(acc, a_base, b_base, n);
    else rect_stage<2, 2>(acc, a_base, b_base, n);
}

/* FULL == false: the SYRK above (one column range, lower tiles only).
 * FULL == true : the general product  Kpart += X[:, range a] X[:, range b]^T  over ALL nb x nb
 *                tiles (K[C1 C2^T] = sum_P (B_P C1)(B_P C2)^T is not symmetric); blockIdx.y is the
 *                row-major tile index and the operands come from two column ranges of X. */
template <bool FULL>
__global__ void __launch_bounds__(K2_THREADS, 1)
k2_syrk_lower_kernel(const double *__restrict__ X4, int64_t nao, int64_t np, int64_t ldc4,
                     int64_t col04, int64_t col04b, int n4s, double *__restrict__ Kpart, int nsplit,
                     int weighted, int accumulate)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    /* lower-triangle tile index -> (bi, bj), bi >= bj */
    /* blockIdx.x = split (fastest), blockIdx.y = tile: the hardware dispatches CTAs in linear
     * order, so the last block row -- the ragged, cheaper tiles -- runs last and the launch's
     * tail is made of short CTAs.  (Tile-fastest order shares k ranges between co-resident CTAs --
     * X from HBM 3.5 instead of 8.3 times -- but was 5.7 % slower; the panel-synchronous kernel
     * below is the real answer to the re-reads.) */
    const int t = blockIdx.y;
    int bi, bj;
    if (FULL) {
        const int nb = (int)((nao + K2_T - 1) / K2_T);
        bi = t / nb;
        bj = t - bi * nb;
    } else {
        bi = (int)((sqrtf(8.0f * (float)t + 1.0f) - 1.0f) * 0.5f);
        while (bi * (bi + 1) / 2 > t) --bi;
        while ((bi + 1) * (bi + 2) / 2 <= t) ++bi;
        bj = t - bi * (bi + 1) / 2;
    }
    const bool diag = !FULL && bi == bj;         /* both operands are the same panel */
    const int split = blockIdx.x;
    if (!FULL && weighted) {                     /* this tile's own split count (k2_tile_splits) */
        nsplit = k2_tile_splits(bi, bj, nao, nsplit);
        if (split >= nsplit) return;
    }
    const int64_t mu0 = (int64_t)bi * K2_T, nu0 = (int64_t)bj * K2_T;

    /* this split's share of the k groups (4 columns each) of the set */
    const int64_t ng = np * n4s;
    const int64_t gbeg = ng * split / nsplit, gend = ng * (split + 1) / nsplit;
    const int nk = (int)((gend - gbeg + K2_KG - 1) / K2_KG);

    const uint32_t smem_base = smem_u32(smem_raw);
    const uint32_t bar_base = smem_base + K2_STAGES * K2_STAGE_BYTES;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (K2_STAGES + s); };
    if (tid == 0) {
        for (int s = 0; s < K2_STAGES; ++s) {
            mbar_init(full_bar(s), 1);
            mbar_init(empty_bar(s), K2_CONSUMER_WARPS);
        }
        mbar_fence_init();
    }
    __syncthreads();

    if (warp == 0) {
        /* ------------------------------------------------------------ producer (one lane) */
        if (lane == 0) {
            const int64_t rows_a = (nao - mu0 < K2_T) ? nao - mu0 : K2_T;
            const int64_t rows_b = (nao - nu0 < K2_T) ? nao - nu0 : K2_T;
            int64_t gp = gbeg / n4s;                      /* (g / n4s, g % n4s), kept incrementally */
            int gi = (int)(gbeg - gp * n4s);
            for (int kc = 0; kc < nk; ++kc) {
                const int slot = kc % K2_STAGES;
                const int round = kc / K2_STAGES;
                if (round > 0) mbar_wait(empty_bar(slot), (round - 1) & 1);
                const int64_t g0 = gbeg + K2_KG * (int64_t)kc;
                const int n = (int)((gend - g0 < K2_KG) ? gend - g0 : K2_KG);
                const uint32_t bytes = (uint32_t)(n * 32 * (rows_a + (diag ? 0 : rows_b)));
                mbar_arrive_expect_tx(full_bar(slot), bytes);
                const uint32_t dst = smem_base + slot * K2_STAGE_BYTES;
                for (int q = 0; q < n; ++q) {
                    const int64_t kg = gp * ldc4 + col04 + gi;                 /* k-group in X4 */
                    if (++gi == n4s) { gi = 0; ++gp; }
                    const double *src = X4 + kg * nao * 4;
                    bulk_g2s(dst + q * (K2_T * 32), src + mu0 * 4, (uint32_t)(rows_a * 32), full_bar(slot));
                    if (!diag) {
                        const double *srcb = FULL ? src + (col04b - col04) * nao * 4 : src;
                        bulk_g2s(dst + K2_OP_BYTES + q * (K2_T * 32), srcb + nu0 * 4,
                                 (uint32_t)(rows_b * 32), full_bar(slot));
                    }
                }
            }
        }
        return;
    }

    /* ---------------------------------------------------------------- consumers */
    const int cw = warp - 1;
    /* warp tiles: 2 (M) x 4 (N) of 64 x 32.  A tile of the ragged last block row with <= 64 valid
     * rows would leave the lower four warps idle: it is covered 1 (M) x 8 (N) with 64 x 16 warp
     * tiles instead, so all eight warps share the work ("narrow"; CTA-uniform). */
    const bool narrow = nao - mu0 <= 64;

    /* A full-height diagonal tile needs only its lower triangle: see tri_unit() ("tri"; the 2 x 4
     * layout would leave two warps idle and the CTA would take as long as an off-diagonal one). */
    const bool tri = diag && !narrow;
    /* full product only: a tile of the ragged last block COLUMN (<= 64 valid columns) would idle the
     * warps of the right half: 4 (M) x 2 (N) warp tiles of 32 x 32 instead ("tall") */
    const bool tall = FULL && !narrow && nao - nu0 <= 64;
    const int wm = narrow ? 0 : cw >> 2, wn = narrow ? cw : cw & 3;
    const int wcols = narrow ? 16 : 32;          /* columns per warp tile (2 x 4 and 1 x 8 layouts) */
    const int lq = lane >> 2, lr = lane & 3;
    const int row_w = tri ? 16 * (7 - (cw & 3)) : (tall ? 32 * (cw >> 1) : 64 * wm);   /* first row / column of this warp's tile */
    /* valid 8-row MMA rows of a rectangular (2 x 4 or 1 x 8) warp tile: ragged block rows in steps of 8 */
    const int nmt_w = (int)((nao - mu0 - row_w + 7) / 8 < 8 ? (nao - mu0 - row_w + 7) / 8 : 8);
    const int col_w = tri ? 0 : (tall ? 32 * (cw & 1) : wcols * wn);
    int ua[4] = {0, 0, 0, 0}, ub[4] = {0, 0, 0, 0};       /* tri, cw >= 4: the four units' panel offsets */
    if (tri && cw >= 4) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            int r, c;
            tri_unit(cw - 4, u, r, c);
            ua[u] = (16 * r + lq) * 4 + lr;
            ub[u] = (16 * c + lq) * 4 + lr;
        }
    }
    /* skip warp tiles that lie outside the matrix or strictly above the diagonal */
    const bool warp_active = tri || ((mu0 + row_w < nao) && (nu0 + col_w < nao) &&
                                     !(diag && col_w > row_w + 63));   /* diag is false when FULL */
    double acc[32][2];                           /* [mt*4+nt] (8 x 4, or 8 x 2 narrow); tri: see tri_stage_* */
#pragma unroll
    for (int t = 0; t < 32; ++t) acc[t][0] = acc[t][1] = 0.0;

    for (int kc = 0; kc < nk; ++kc) {
        const int slot = kc % K2_STAGES;
        mbar_wait(full_bar(slot), (kc / K2_STAGES) & 1);
        if (warp_active) {
            const int64_t g0 = gbeg + K2_KG * (int64_t)kc;
            const int n = (int)((gend - g0 < K2_KG) ? gend - g0 : K2_KG);
            const double *Xa = reinterpret_cast<const double *>(smem_raw + slot * K2_STAGE_BYTES);
            const double *Xb = diag ? Xa : Xa + K2_OP_BYTES / 8;
            const double *a_base = Xa + (row_w + lq) * 4 + lr;
            const double *b_base = Xb + (col_w + lq) * 4 + lr;
            if (tall) {
                rect_stage<4, 4>(acc, a_base, b_base, n);
            } else if (tri) {
                if (cw < 4) tri_stage_wide(acc, a_base, b_base, n);
                else tri_stage_units(acc, Xa, ua, ub, n);
            } else if (!narrow) {
                rect_stage_full(nmt_w, acc, a_base, b_base, n);
            } else {
                rect_stage_narrow(nmt_w, acc, a_base, b_base, n);
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(empty_bar(slot));
    }

    if (!warp_active) return;
    double *Kp = Kpart + (int64_t)split * nao * nao;
    if (tri) {
        if (cw < 4) {
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) {
                const int64_t mu = mu0 + row_w + 8 * mt + lq;
                if (mu >= nao) continue;
#pragma unroll
                for (int nt = 0; nt < 10; ++nt) {
                    const int64_t nu = nu0 + 8 * nt + 2 * lr;
                    double *dst = Kp + mu * nao + nu;
                    if (nu < nao) dst[0] = accumulate ? dst[0] + acc[mt * 10 + nt][0] : acc[mt * 10 + nt][0];
                    if (nu + 1 < nao) dst[1] = accumulate ? dst[1] + acc[mt * 10 + nt][1] : acc[mt * 10 + nt][1];
                }
            }
        } else {
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                int r, c;
                tri_unit(cw - 4, u, r, c);
#pragma unroll
                for (int mt = 0; mt < 2; ++mt) {
                    const int64_t mu = mu0 + 16 * r + 8 * mt + lq;
                    if (mu >= nao) continue;
#pragma unroll
                    for (int nt = 0; nt < 2; ++nt) {
                        const int64_t nu = nu0 + 16 * c + 8 * nt + 2 * lr;
                        double *dst = Kp + mu * nao + nu;
                        const int t = 4 * u + 2 * mt + nt;
                        if (nu < nao) dst[0] = accumulate ? dst[0] + acc[t][0] : acc[t][0];
                        if (nu + 1 < nao) dst[1] = accumulate ? dst[1] + acc[t][1] : acc[t][1];
                    }
                }
            }
        }
        return;
    }
#pragma unroll
    for (int mt = 0; mt < 8; ++mt) {
        const int64_t mu = mu0 + row_w + 8 * mt + lq;
        if (mu >= nao || (tall && mt >= 4)) continue;
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) {
            if (narrow && nt >= 2) continue;
            const int64_t nu = nu0 + col_w + 8 * nt + 2 * lr;
            double *dst = Kp + mu * nao + nu;
            if (nu < nao) dst[0] = accumulate ? dst[0] + acc[mt * 4 + nt][0] : acc[mt * 4 + nt][0];
            if (nu + 1 < nao) dst[1] = accumulate ? dst[1] + acc[mt * 4 + nt][1] : acc[mt * 4 + nt][1];
        }
    }
}

/* ------------------------------------------------------------------ K2P: panel-synchronous K2 */
/* The same product with the k range cut into short PANELS and the work dealt out dynamically:
 * item = (panel p, tile t), tile fastest, claimed in order from a global counter by persistent
 * CTAs (one per SM).  The CTAs working at any moment therefore sit on one or two neighbouring
 * panels -- a k window of X a few MB wide that stays in L2 while every tile of the block row /
 * column that needs it comes by (k2_syrk_lower_kernel hands each CTA a long contiguous k range:
 * co-resident CTAs read 13 different ranges and X comes from HBM 8.3 times, ncu r01e).  The price
 * is that a tile's accumulator no longer lives in one CTA's registers for the whole range: item
 * (p, t) adds its 128 x 128 partial into slab p % S of Kpart, after item (p - S, t) has (a per
 * (slab, tile) counter in global memory, release/acquire; items are claimed in order and never
 * wait on later ones, so the wait cannot deadlock and in practice never spins).  The slabs are
 * L2-resident (S x nao^2 doubles) and summed in the fixed order K3 uses => deterministic.
 * The adds are `red.add.f64` at L2, ordered by that counter (each address receives them in panel
 * order), so no consumer waits for a slab line.  Four producer lanes, one per sub-partition, run
 * ahead through item boundaries (the stage ring never drains); warp layouts per tile are those of
 * k2_syrk_lower_kernel. */
struct K2PArgs {
    const double *X4;
    int64_t nao, np, ldc4, col04, col04b;
    int n4s;
    double *Kpart;            /* S slabs of nao x nao */
    int nslab, accumulate, npanel, ntile, nb;
    int *work;                /* [0]: item counter; [1 + slab * ntile + tile]: items completed */
};

constexpr int K2P_THREADS = 128 + 32 * K2_CONSUMER_WARPS;     /* producer warpgroup + 8 consumer warps */
constexpr int K2P_SMEM_BYTES = K2_STAGES * K2_STAGE_BYTES + 2 * K2_STAGES * 8 + 6 * 8 + 2 * 8 + 16;

__device__ __forceinline__ int ld_acquire_gpu(const int *p)
{
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_gpu(int *p, int v)
{
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

template <bool FULL>
__device__ __forceinline__ void k2p_decode(int t, int nb, int &bi, int &bj)
{
    if (FULL) {
        bi = t / nb;
        bj = t - bi * nb;
    } else {
        bi = (int)((sqrtf(8.0f * (float)t + 1.0f) - 1.0f) * 0.5f);
        while (bi * (bi + 1) / 2 > t) --bi;
        while ((bi + 1) * (bi + 2) / 2 <= t) ++bi;
        bj = t - bi * (bi + 1) / 2;
    }
}

/* fire-and-forget FP64 add at L2 (SASS RED.E.ADD.F64): no load, no round trip */
__device__ __forceinline__ void red_add_f64(double *p, double v)
{
    asm volatile("red.relaxed.gpu.global.add.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory");
}

/* NR rows (8 apart) of the warp tile at once:  row_r[8 nt + {0,1}] (+)= acc[r * AST + nt][{0,1}],
 * nt < NNT, for the rows r with mu_first + 8 r < nao and the columns nu_first + 8 nt + {0,1} < nao.
 * The first item of a (slab, tile) stores, every later one adds with `red` at L2: the consumers
 * never wait for a slab line to come back, and since the items of one (slab, tile) are chained by
 * its release/acquire counter each address still receives its adds in panel order => the sum is
 * the same on every run.  (The load-add-store version idled the FP64 pipe ~3 us per item.) */
template <int NNT, int NR, int AST>
__device__ __forceinline__ void k2p_add_rows(const double (*acc)[2], double *row, int64_t mu_first,
                                             int64_t nu_first, int64_t nao, bool overwrite, bool vec)
{
#pragma unroll
    for (int r = 0; r < NR; ++r) {
        if (mu_first + 8 * r >= nao) continue;
        double *rp = row + (int64_t)8 * r * nao;
#pragma unroll
        for (int nt = 0; nt < NNT; ++nt) {
            const double r0 = acc[r * AST + nt][0], r1 = acc[r * AST + nt][1];
            if (overwrite) {
                if (vec) {
                    if (nu_first + 8 * nt < nao)              /* nao and nu even: the pair is inside */
                        *reinterpret_cast<double2 *>(rp + 8 * nt) = make_double2(r0, r1);
                } else {
                    if (nu_first + 8 * nt < nao) rp[8 * nt] = r0;
                    if (nu_first + 8 * nt + 1 < nao) rp[8 * nt + 1] = r1;
                }
            } else {
                if (nu_first + 8 * nt < nao) red_add_f64(rp + 8 * nt, r0);
                if (nu_first + 8 * nt + 1 < nao) red_add_f64(rp + 8 * nt + 1, r1);
            }
        }
    }
}


template <bool FULL>
__global__ void __launch_bounds__(K2P_THREADS, 1)
k2p_kernel(const K2PArgs a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t nao = a.nao;
    const int64_t ng = a.np * a.n4s;                      /* k groups (4 columns each) of the set */
    const int nitems = a.npanel * a.ntile;

    const uint32_t smem_base = smem_u32(smem_raw);
    const uint32_t bar_base = smem_base + K2_STAGES * K2_STAGE_BYTES;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (K2_STAGES + s); };
    auto item_full = [&](int s) { return bar_base + 8u * (2 * K2_STAGES + s); };
    auto item_empty = [&](int s) { return bar_base + 8u * (2 * K2_STAGES + 2 + s); };
    auto item_done = [&](int s) { return bar_base + 8u * (2 * K2_STAGES + 4 + s); };
    volatile int *item_id = reinterpret_cast<volatile int *>(smem_raw + K2_STAGES * K2_STAGE_BYTES + 8 * (2 * K2_STAGES + 6));
    if (tid == 0) {
        for (int s = 0; s < K2_STAGES; ++s) {
            mbar_init(full_bar(s), 4);                            /* the four producer lanes */
            mbar_init(empty_bar(s), K2_CONSUMER_WARPS);
        }
        for (int s = 0; s < 2; ++s) {
            mbar_init(item_full(s), 1);
            mbar_init(item_empty(s), K2_CONSUMER_WARPS + 3);       /* consumers + producers 1-3 */
            mbar_init(item_done(s), K2_CONSUMER_WARPS);
        }
        mbar_fence_init();
    }
    __syncthreads();

    if (warp < 4) {
        /* ------------------------------------------------------------ producers: lane 0 of each warp
         * of the first warpgroup (which gives its registers to the consumers).  Producer w issues the
         * k-groups q = w and w + 4 of every stage, so each of the four sub-partitions carries a quarter
         * of the copy-issuing instructions: with ONE producer lane its ~640 instructions per stage took
         * issue slots from the two consumer warps of its sub-partition exactly when their DMMAs were due,
         * that sub-partition ran 270 cycles per stage behind and the other three waited for it at the
         * full barrier.  Producer 0 also claims the items; producer 1 also publishes finished ones. */
        reg_dealloc<40>();
        if (lane == 0) {
            const int w = warp;
            int st = 0;                                   /* stages issued so far (ring position) */
            bool pending = false;                         /* producer 1: an item waits to be published */
            int pend_is = 0, pend_val = 0;
            uint32_t pend_phase = 0;
            int *pend_flag = nullptr;
            for (int ir = 0;; ++ir) {
                const int is = ir & 1;
                int item;
                if (w == 0) {
                    item = atomicAdd(a.work, 1);
                    if (item >= nitems) item = -1;
                    if (ir >= 2) mbar_wait(item_empty(is), ((ir >> 1) - 1) & 1);
                    item_id[is] = item;
                    mbar_arrive(item_full(is));
                } else {
                    mbar_wait(item_full(is), (ir >> 1) & 1);
                    item = item_id[is];
                    mbar_arrive(item_empty(is));
                }
                if (item < 0) break;
                const int p = item / a.ntile, t = item - p * a.ntile;
                int bi, bj;
                k2p_decode<FULL>(t, a.nb, bi, bj);
                const bool diag = !FULL && bi == bj;
                const int64_t mu0 = (int64_t)bi * K2_T, nu0 = (int64_t)bj * K2_T;
                const uint32_t bytes_a = (uint32_t)(((nao - mu0 < K2_T) ? nao - mu0 : K2_T) * 32);
                const uint32_t bytes_b = (uint32_t)(((nao - nu0 < K2_T) ? nao - nu0 : K2_T) * 32);
                const int64_t gbeg = ng * p / a.npanel, gend = ng * (p + 1) / a.npanel;
                const int nk = (int)((gend - gbeg + K2_KG - 1) / K2_KG);
                /* this lane's k-groups are gbeg + w, + 4, + 8, ...: the index inside its P (gi) and the
                 * source pointers are kept incrementally, no division in the stage loop */
                int64_t g = gbeg + w;
                const int64_t gp = g / a.n4s;
                int gi = (int)(g - gp * a.n4s);
                const int64_t gstride = nao * 4;                              /* doubles per k-group */
                const double *src_a = a.X4 + (gp * a.ldc4 + a.col04 + gi) * gstride + mu0 * 4;
                const double *src_b = a.X4 + (gp * a.ldc4 + (FULL ? a.col04b : a.col04) + gi) * gstride + nu0 * 4;
                const int64_t wrap_skip = (a.ldc4 - a.n4s) * gstride;         /* past the other columns of a P */
                for (int kc = 0; kc < nk; ++kc, ++st) {
                    const int slot = st % K2_STAGES;
                    const int round = st / K2_STAGES;
                    if (w == 1 && pending) {
                        /* keep an eye on item_done while waiting for the slot: a finished item must be
                         * published at once, the next item of its (slab, tile) chain may be waiting for
                         * it in another CTA (published only between stages, the chains of a 21-tile
                         * problem cost 13 % of K2 in flag waits) */
                        while (true) {
                            if (mbar_test_wait(item_done(pend_is), pend_phase)) {
                                st_release_gpu(pend_flag, pend_val);
                                pending = false;
                                break;
                            }
                            if (round == 0 || mbar_try_wait_for(empty_bar(slot), (round - 1) & 1, 200)) break;
                        }
                    }
                    if (round > 0) mbar_wait(empty_bar(slot), (round - 1) & 1);
                    const uint32_t dst = smem_base + slot * K2_STAGE_BYTES;
                    const int mine = (g < gend ? 1 : 0) + (g + 4 < gend ? 1 : 0);     /* my groups in this stage */
                    if (mine) mbar_arrive_expect_tx(full_bar(slot), (uint32_t)mine * (bytes_a + (diag ? 0u : bytes_b)));
                    else mbar_arrive(full_bar(slot));
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        if (g < gend) {
                            const int q = w + 4 * h;
                            bulk_g2s(dst + q * (K2_T * 32), src_a, bytes_a, full_bar(slot));
                            if (!diag) bulk_g2s(dst + K2_OP_BYTES + q * (K2_T * 32), src_b, bytes_b, full_bar(slot));
                        }
                        g += 4; gi += 4;
                        src_a += 4 * gstride; src_b += 4 * gstride;
                        while (gi >= a.n4s) { gi -= a.n4s; src_a += wrap_skip; src_b += wrap_skip; }
                    }
                }
                if (w == 1) {
                    /* the item just issued is published once its consumers report their adds issued
                     * (item_done): polled from the stage loop of the NEXT item, never waited for while
                     * stages remain to be issued; the gpu-scope release is cumulative over what the
                     * mbarrier made visible to this thread, i.e. it orders the adds, not the consumers */
                    if (pending) {
                        mbar_wait(item_done(pend_is), pend_phase);
                        st_release_gpu(pend_flag, pend_val);
                    }
                    pending = true;
                    pend_is = is;
                    pend_phase = (uint32_t)((ir >> 1) & 1);
                    pend_flag = a.work + 1 + (p % a.nslab) * a.ntile + t;
                    pend_val = p / a.nslab + 1;
                }
            }
            if (w == 1 && pending) {
                mbar_wait(item_done(pend_is), pend_phase);
                st_release_gpu(pend_flag, pend_val);
            }
        }
        return;
    }

    /* ---------------------------------------------------------------- consumers (two warpgroups) */
    reg_alloc<232>();
    const int cw = warp - 4;
    const int lq = lane >> 2, lr = lane & 3;
    /* this warp's units of the triangular layout (tri_unit) */
    int ua[4] = {0, 0, 0, 0}, ub[4] = {0, 0, 0, 0}, ur[4] = {0, 0, 0, 0}, uc[4] = {0, 0, 0, 0};
    if (cw >= 4) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            tri_unit(cw - 4, u, ur[u], uc[u]);
            ua[u] = (16 * ur[u] + lq) * 4 + lr;
            ub[u] = (16 * uc[u] + lq) * 4 + lr;
        }
    }
    int st = 0;
    for (int ir = 0;; ++ir) {
        const int is = ir & 1;
        mbar_wait(item_full(is), (ir >> 1) & 1);
        const int item = item_id[is];
        __syncwarp();
        if (lane == 0) mbar_arrive(item_empty(is));
        if (item < 0) break;
        const int p = item / a.ntile, t = item - p * a.ntile;
        int bi, bj;
        k2p_decode<FULL>(t, a.nb, bi, bj);
        const bool diag = !FULL && bi == bj;
        const int64_t mu0 = (int64_t)bi * K2_T, nu0 = (int64_t)bj * K2_T;
        const int64_t gbeg = ng * p / a.npanel, gend = ng * (p + 1) / a.npanel;
        const int nk = (int)((gend - gbeg + K2_KG - 1) / K2_KG);
        const bool narrow = nao - mu0 <= 64;
    
        const bool tri = diag && !narrow;
        const bool tall = FULL && !narrow && nao - nu0 <= 64;
        const int wm = narrow ? 0 : cw >> 2, wn = narrow ? cw : cw & 3;
        const int wcols = narrow ? 16 : 32;
        const int row_w = tri ? 16 * (7 - (cw & 3)) : (tall ? 32 * (cw >> 1) : 64 * wm);
        const int nmt_w = (int)((nao - mu0 - row_w + 7) / 8 < 8 ? (nao - mu0 - row_w + 7) / 8 : 8);   /* valid MMA rows */
        const int col_w = tri ? 0 : (tall ? 32 * (cw & 1) : wcols * wn);
        const bool warp_active = tri || ((mu0 + row_w < nao) && (nu0 + col_w < nao) &&
                                         !(diag && col_w > row_w + 63));
        double acc[32][2];
#pragma unroll
        for (int q = 0; q < 32; ++q) acc[q][0] = acc[q][1] = 0.0;

        for (int kc = 0; kc < nk; ++kc, ++st) {
            const int slot = st % K2_STAGES;
            mbar_wait(full_bar(slot), (st / K2_STAGES) & 1);
            if (warp_active) {
                const int64_t g0 = gbeg + K2_KG * (int64_t)kc;
                const int n = (int)((gend - g0 < K2_KG) ? gend - g0 : K2_KG);
                const double *Xa = reinterpret_cast<const double *>(smem_raw + slot * K2_STAGE_BYTES);
                const double *Xb = diag ? Xa : Xa + K2_OP_BYTES / 8;
                const double *a_base = Xa + (row_w + lq) * 4 + lr;
                const double *b_base = Xb + (col_w + lq) * 4 + lr;
                if (tall) {
                    rect_stage<4, 4>(acc, a_base, b_base, n);
                } else if (tri) {
                    if (cw < 4) tri_stage_wide(acc, a_base, b_base, n);
                    else tri_stage_units(acc, Xa, ua, ub, n);
                } else if (!narrow) {
                    rect_stage_full(nmt_w, acc, a_base, b_base, n);
                } else {
                    rect_stage_narrow(nmt_w, acc, a_base, b_base, n);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty_bar(slot));
        }

        /* ---- add the partial into slab p % S, after item (p - S, t) has */
        const int slab = p % a.nslab, seq = p / a.nslab;
        int *flag = a.work + 1 + slab * a.ntile + t;
        const bool overwrite = seq == 0 && !a.accumulate;
        if (warp_active) {
            if (seq > 0) {
                if (lane == 0) while (ld_acquire_gpu(flag) < seq) { }
                __syncwarp();
                (void)ld_acquire_gpu(flag);              /* every lane orders its adds after the flag */
            }
            double *Kp = a.Kpart + (int64_t)slab * nao * nao;
            /* first item of the (slab, tile): 16-byte stores when the row pitch allows (nao even);
             * later ones: `red` adds, ordered behind the previous item by the flag (k2p_add_rows) */
            const bool vec = (nao & 1) == 0;
            const int64_t nu_first = nu0 + col_w + 2 * lr;
            double *row0 = Kp + (mu0 + row_w + lq) * nao + nu_first;
            const int64_t mu_first = mu0 + row_w + lq;
            if (tri) {
                if (cw < 4) {
                    k2p_add_rows<10, 2, 10>(&acc[0], row0, mu_first, nu_first, nao, overwrite, vec);
                } else {
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int64_t mu_u = mu0 + 16 * ur[u] + lq, nu_u = nu0 + 16 * uc[u] + 2 * lr;
                        k2p_add_rows<2, 2, 2>(&acc[4 * u], Kp + mu_u * nao + nu_u, mu_u, nu_u, nao, overwrite, vec);
                    }
                }
            } else if (narrow) {
                k2p_add_rows<2, 8, 4>(&acc[0], row0, mu_first, nu_first, nao, overwrite, vec);
            } else if (tall) {
                k2p_add_rows<4, 4, 4>(&acc[0], row0, mu_first, nu_first, nao, overwrite, vec);
            } else {
                k2p_add_rows<4, 4, 4>(&acc[0], row0, mu_first, nu_first, nao, overwrite, vec);
                k2p_add_rows<4, 4, 4>(&acc[16], row0 + 32 * nao, mu_first + 32, nu_first, nao, overwrite, vec);
            }
        }
        /* every consumer warp (the idle ones too) reports its adds issued and moves on; producer 1
         * publishes the item (no CTA-wide barrier, no consumer waits for the adds to land) */
        __syncwarp();
        if (lane == 0) mbar_arrive(item_done(is));
    }
}

/* ------------------------------------------------------------------ K3 */
constexpr int K3_T = 32;

__global__ void __launch_bounds__(256)
k3_finish_kernel(const double *__restrict__ Kpart, int nsplit, int weighted, int64_t nao,
                 double *__restrict__ Kdirect, double *const *__restrict__ Kslot)
{
    const int bi = blockIdx.y, bj = blockIdx.x;
    if (bj > bi) return;
    /* partials of the split kernel: as many as the 128 x 128 tile around this block was cut into */
    if (weighted) nsplit = k2_tile_splits(bi / (K2_T / K3_T), bj / (K2_T / K3_T), nao, nsplit);
    double *__restrict__ K = Kslot ? *Kslot : Kdirect;        /* see j3_unpack_kernel */
    __shared__ double t[K3_T][K3_T + 1];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int64_t mu0 = (int64_t)bi * K3_T, nu0 = (int64_t)bj * K3_T;
    /* four rows side by side, eight splits per round: 32 loads in flight (see j3_unpack_kernel) */
    const double *src[4];
    double v[4];
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int64_t mu = mu0 + ty + 8 * r, nu = nu0 + tx;
        src[r] = (mu < nao && nu <= mu) ? Kpart + mu * nao + nu : nullptr;
        v[r] = 0.0;
    }
#pragma unroll 8
    for (int s = 0; s < nsplit; ++s)
#pragma unroll
        for (int r = 0; r < 4; ++r)
            if (src[r]) v[r] += src[r][(int64_t)s * nao * nao];
#pragma unroll
    for (int r = 0; r < 4; ++r) t[ty + 8 * r][tx] = v[r];
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

/* ------------------------------------------------------------------ FP64 pipe probe */
/* Register-only DMMA loop: 8 warps per CTA, 16 independent accumulator tiles per warp.  Measures
 * what the FP64 pipe sustains with nothing else in the way -- the denominator of K's roofline. */
__global__ void __launch_bounds__(256)
fp64_peak_probe_kernel(int iters, double *__restrict__ sink)
{
    double acc[16][2];
#pragma unroll
    for (int t = 0; t < 16; ++t) { acc[t][0] = 0.0; acc[t][1] = 0.0; }
    double a = 1.0 + 1e-9 * threadIdx.x, b = 1.0 - 1e-9 * threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int t = 0; t < 16; ++t) dmma884(acc[t][0], acc[t][1], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int t = 0; t < 16; ++t) s += acc[t][0] + acc[t][1];
    if (s == 123.456) sink[0] = s;                       /* keeps the loop alive */
}

/* general (non-symmetric) finish: K[mu][nu] = sum_split Kpart[split][mu][nu], every entry */
__global__ void __launch_bounds__(256)
k3_sum_kernel(const double *__restrict__ Kpart, int nsplit, int64_t n2, double *__restrict__ K, int accumulate)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n2) return;
    double v = accumulate ? K[i] : 0.0;    /* batched build: K collects one X chunk after the other */
#pragma unroll 8
    for (int s = 0; s < nsplit; ++s) v += Kpart[(int64_t)s * n2 + i];
    K[i] = v;
}

}  // namespace


void launch_k0_pack_c(const double *const *C, const int *nocc, const int *col0, int nset, int64_t nao,
                      int64_t ldc, double *Ccat, double *const *outs, double **out_slots, cudaStream_t st)
{
    PackDesc pd;
    pd.nset = nset;
    for (int i = 0; i < DFJK_OUT_SLOTS; ++i) pd.out[i] = outs ? outs[i] : nullptr;
    pd.out_slots = outs ? out_slots : nullptr;
    for (int s = 0; s < 4; ++s) {
        pd.C[s] = s < nset ? C[s] : nullptr;
        pd.nocc[s] = s < nset ? nocc[s] : 0;
        pd.col0[s] = s < nset ? col0[s] : 0;
    }
    const int64_t nao16 = (nao + 31) / 32 * 32;   /* K1 stages cover 32 rows of C */
    const int64_t n = nao16 * ldc;
    k0_pack_c_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(pd, nao, nao16, ldc, Ccat);
}

cudaError_t launch_k2_syrk_lower(const double *X4, int64_t nao, int64_t np, int64_t ldc, int64_t col0,
                                 int64_t ncol, double *Kpart, int nsplit, int weighted, int accumulate,
                                 cudaStream_t st)
{
    static std::atomic<unsigned long long> smem_ok{0};
    const cudaError_t e = ensure_dynamic_smem(k2_syrk_lower_kernel<false>, K2_SMEM_BYTES, smem_ok);
    if (e != cudaSuccess) return e;
    const int nb = (int)((nao + K2_T - 1) / K2_T);
    const int ntile = nb * (nb + 1) / 2;
    const int n4s = (int)((ncol + 3) / 4);              /* k step 4: Ccat's padding to 8 is not read */
    k2_syrk_lower_kernel<false><<<dim3((unsigned)nsplit, (unsigned)ntile), K2_THREADS, K2_SMEM_BYTES, st>>>(
        X4, nao, np, ldc / 4, col0 / 4, col0 / 4, n4s, Kpart, nsplit, weighted, accumulate);
    return cudaPeekAtLastError();
}

cudaError_t launch_k2_gemm_full(const double *X4, int64_t nao, int64_t np, int64_t ldc, int64_t col0a,
                                int64_t col0b, int64_t ncol, double *Kpart, int nsplit, int accumulate,
                                cudaStream_t st)
{
    static std::atomic<unsigned long long> smem_ok{0};
    const cudaError_t e = ensure_dynamic_smem(k2_syrk_lower_kernel<true>, K2_SMEM_BYTES, smem_ok);
    if (e != cudaSuccess) return e;
    const int nb = (int)((nao + K2_T - 1) / K2_T);
    const int n4s = (int)((ncol + 3) / 4);
    k2_syrk_lower_kernel<true><<<dim3((unsigned)nsplit, (unsigned)(nb * nb)), K2_THREADS, K2_SMEM_BYTES, st>>>(
        X4, nao, np, ldc / 4, col0a / 4, col0b / 4, n4s, Kpart, nsplit, 0, accumulate);
    return cudaPeekAtLastError();
}

/* panel length (stages of k = 32) and slab count of the panel-synchronous K2, see k2p_kernel;
 * planned once per build from its first (largest) chunk */
void k2p_plan(int64_t nao, int64_t ng, int ntile, int sm_count, int max_slabs, int64_t panel_bytes,
              int *panel_stages, int *nslab)
{
    const int64_t stages_total = (ng + K2_KG - 1) / K2_KG;
    /* L2: one panel of X (all nao rows) is about panel_bytes */
    int64_t len = panel_bytes / (nao * 32 * K2_KG);
    /* balance: at least ~30 items per SM when the problem is big enough for that (15 .. 45 measure
     * the same within 1 %) */
    const int64_t len_bal = stages_total * ntile / (30LL * sm_count);
    if (len > len_bal) len = len_bal;
    if (len < 8) len = 8;                                 /* the 128 KB read-modify-write must amortise */
    if (len > stages_total) len = stages_total > 0 ? stages_total : 1;
    const int64_t np_ = (stages_total + len - 1) / len;
    /* slabs: the chain of read-modify-writes of one (slab, tile) must be short beside an item;
     * ~3 us per add, items of len x 4.2 us, sm_count / ntile items of a tile in flight at once */
    int64_t s_ = (2LL * sm_count * 3 * 10 + (int64_t)ntile * len * 42 - 1) / ((int64_t)ntile * len * 42);
    if (s_ < 1) s_ = 1;
    if (s_ > max_slabs) s_ = max_slabs;
    if (s_ > np_) s_ = np_ > 0 ? np_ : 1;
    *panel_stages = (int)len;
    *nslab = (int)s_;
}

template <bool FULL>
cudaError_t k2p_launch(const double *X4, int64_t nao, int64_t np, int64_t ldc, int64_t col0a, int64_t col0b,
                       int64_t ncol, double *Kpart, int panel_stages, int nslab, int accumulate, int *work,
                       int sm_count, cudaStream_t st)
{
    static std::atomic<unsigned long long> smem_ok{0};
    cudaError_t e = ensure_dynamic_smem(k2p_kernel<FULL>, K2P_SMEM_BYTES, smem_ok);
    if (e != cudaSuccess) return e;
    K2PArgs a;
    a.X4 = X4; a.nao = nao; a.np = np; a.ldc4 = ldc / 4; a.col04 = col0a / 4; a.col04b = col0b / 4;
    a.n4s = (int)((ncol + 3) / 4);
    const int64_t stages_total = (np * a.n4s + K2_KG - 1) / K2_KG;
    const int npanel = (int)((stages_total + panel_stages - 1) / panel_stages);
    a.Kpart = Kpart; a.nslab = nslab; a.accumulate = accumulate; a.npanel = npanel;
    a.nb = (int)((nao + K2_T - 1) / K2_T);
    a.ntile = FULL ? a.nb * a.nb : a.nb * (a.nb + 1) / 2;
    a.work = work;
    e = cudaMemsetAsync(work, 0, sizeof(int) * (size_t)(1 + nslab * a.ntile), st);
    if (e != cudaSuccess) return e;
    const int64_t nitems = (int64_t)npanel * a.ntile;
    const unsigned grid = (unsigned)(nitems < sm_count ? nitems : sm_count);
    k2p_kernel<FULL><<<grid, K2P_THREADS, K2P_SMEM_BYTES, st>>>(a);
    return cudaPeekAtLastError();
}

cudaError_t launch_k2p_syrk_lower(const double *X4, int64_t nao, int64_t np, int64_t ldc, int64_t col0,
                                  int64_t ncol, double *Kpart, int panel_stages, int nslab, int accumulate,
                                  int *work, int sm_count, cudaStream_t st)
{
    return k2p_launch<false>(X4, nao, np, ldc, col0, col0, ncol, Kpart, panel_stages, nslab, accumulate, work,
                             sm_count, st);
}

cudaError_t launch_k2p_gemm_full(const double *X4, int64_t nao, int64_t np, int64_t ldc, int64_t col0a,
                                 int64_t col0b, int64_t ncol, double *Kpart, int panel_stages, int nslab,
                                 int accumulate, int *work, int sm_count, cudaStream_t st)
{
    return k2p_launch<true>(X4, nao, np, ldc, col0a, col0b, ncol, Kpart, panel_stages, nslab, accumulate, work,
                            sm_count, st);
}

int64_t k2_lower_items(int64_t nao, int nsplit)
{
    const int nb = (int)((nao + K2_T - 1) / K2_T);
    /* rows 0 .. nb-2 are full height: bi off-diagonal tiles and one diagonal tile each */
    int64_t items = 0;
    for (int bi = 0; bi < nb; ++bi)
        items += (int64_t)bi * k2_tile_splits(bi, 0, nao, nsplit) + k2_tile_splits(bi, bi, nao, nsplit);
    return items;
}

void launch_k3_finish(const double *Kpart, int nsplit, int weighted, int64_t nao, double *K, double *const *Kslot,
                      cudaStream_t st)
{
    const unsigned nb = (unsigned)((nao + K3_T - 1) / K3_T);
    k3_finish_kernel<<<dim3(nb, nb), 256, 0, st>>>(Kpart, nsplit, weighted, nao, K, Kslot);
}

double fp64_peak_probe_flops(int ctas, int iters) { return (double)ctas * 8.0 * iters * 16.0 * 512.0; }

void launch_fp64_peak_probe(int ctas, int iters, double *sink, cudaStream_t st)
{
    fp64_peak_probe_kernel<<<ctas, 256, 0, st>>>(iters, sink);
}

void launch_k3_sum(const double *Kpart, int nsplit, int64_t nao, double *K, cudaStream_t st, int accumulate)
{
    const int64_t n2 = nao * nao;
    k3_sum_kernel<<<(unsigned)((n2 + 255) / 256), 256, 0, st>>>(Kpart, nsplit, n2, K, accumulate);
}

void launch_k0_pack_cols(const double *C, int64_t ncol, int64_t col0, int64_t width, int64_t nao, int64_t ldc,
                         double *Ccat, cudaStream_t st)
{
    const int64_t nao16 = (nao + 31) / 32 * 32;
    const int64_t n = nao16 * width;
    k0_pack_cols_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(C, ncol, col0, width, nao, nao16, ldc, Ccat);
}

}  // namespace dfjk
