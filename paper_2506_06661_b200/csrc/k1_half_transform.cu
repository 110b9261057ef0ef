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
 *     - A tile: the packed triangle is unpacked while staging, by the TMA engine.  A stage
 *       left of the diagonal is 128 row copies of 32 doubles (packed rows mu, "row" form);
 *       a stage right of it is 32 row copies of 128 doubles (packed rows nu, i.e. the
 *       transposed tile, "col" form); each is one 1-D bulk copy (cp.async.bulk -> UBLKCP)
 *       issued by one producer thread.  Packed rows are only 8-byte aligned: a copy whose
 *       source index is odd starts one element early and the consumer reads that row with
 *       a +1 column shift, which is a per-lane constant (see K1_LDD/K1_LDT).  The four
 *       stages inside the diagonal block mix the two forms band by band and gather only the
 *       32 x 32 block that sits on the diagonal element-wise (8-byte cp.async, max/min
 *       addressing, zero fill; see K1_MODE_DIAG).  An earlier version gathered every stage
 *       with cp.async: the 4096 LDGSTS per stage cost 7 % of K1 through the LSU.
 *       Every packed element is read twice per call (K1 is compute-bound: ~65 flop/B).
 *     - a ragged last row block (<= 64 rows) is batched over 2/4/8 auxiliary indices into one
 *       full 128-row item (see K1Item).
 *     - C tile: Ccat is kept k-group-major ([nu/4][ldc][4]), so the 8 x NW x 4 tile of a
 *       stage is eight contiguous bulk copies completing on the same mbarrier.
 *   two consumer warpgroups (8 warps, 232 registers after setmaxnreg.inc)
 *     - each warp owns 16 rows x NW columns = 2 x NT8 DMMA.8x8x4 accumulator tiles;
 *       one k4 step costs 2+NT8 shared loads for 2*NT8 MMAs.  The C tile and X are stored
 *       dense as [k/4][row][4] doubles: the 16 lanes of each 64-bit half-warp phase read
 *       16 consecutive doubles => conflict-free with no padding; the A tile pitches (36,
 *       132 doubles) are == 4 mod 16 for the same reason (one 2-way conflict per phase
 *       remains from the alignment shift).
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
/* A tile of a stage, one of two shapes (both reached by plain row copies of the packed triangle):
 *   "row" form   [m][K1_LDD]: row m holds B_P(mu0+m, nu0 .. nu0+31) at column k + sd(m)
 *   "col" form   [k][K1_LDT]: row k holds B_P(mu0 .. mu0+127, nu0+k) = packed(nu0+k, mu0 ..) at column m + st(k)
 * sd/st in {0,1} is the parity of the source element's index in B: a packed row starts on an
 * 8-byte, not a 16-byte boundary, so the bulk copy starts one element early when that index is
 * odd and the data lands shifted by one.  mu0 is a multiple of 128 and nu0 of 32, so the shift
 * pattern is (0,1,1,0) in (row mod 4) xor the parity of P*npair: a per-lane constant. */
constexpr int K1_LDD = 36;                        /* 32 + shift + pad, 16-B multiple */
constexpr int K1_LDT = 132;                       /* 128 + shift + pad, 16-B multiple */
constexpr int K1_A_BYTES = K1_M * K1_LDD * 8;     /* 36864 >= 32 * K1_LDT * 8 = 33792 */
constexpr int K1_SMEM_BUDGET = 220 * 1024;
/* Every off-diagonal packed element is staged twice: in "row" form by the item of its row block and
 * in "col" form by the item of its column block.  The nib items of one P run at the same time on
 * neighbouring CTAs, so the two reads can be made to COINCIDE: item i does not walk nu from 0 up but
 * visits the 128-wide column blocks j in the round-robin tournament order j = (s - i) mod nib,
 * s = 0 .. nib-1.  At step s the pair (i, j) with i + j == s (mod nib) work on each other's block:
 * i stages B_P[block i, block j] while j stages B_P[block j, block i] -- the same packed elements, at
 * (nearly) the same time, so whichever read arrives second is an L2 hit.  B comes from HBM 1.22
 * times per build at nao = 1600 and 1.01 times at nao = 800 instead of 1.44 (ncu r01e / r02).
 * L2 eviction hints on top of this made it worse. */

enum { K1_MODE_ROW = 0, K1_MODE_COL = 1, K1_MODE_GATHER = 2, K1_MODE_DIAG = 3 };

/* which form stage kc of row block mu0 takes; identical on producer and consumer side */
__device__ __forceinline__ int k1_mode(int mu0, int nu0, int nao, bool last_p, bool multi)
{
    if (nu0 < mu0) return K1_MODE_ROW;                         /* every nu <= every mu (32 | 128 aligned) */
    if (nu0 < mu0 + K1_M)                                      /* inside the diagonal block */
        return (nu0 + K1_KC <= nao && !multi) ? K1_MODE_DIAG : K1_MODE_GATHER;   /* (ragged last stage: zero
                                                                  fill; a ragged item stacks several P) */
    if (!(last_p && nu0 + K1_KC >= nao)) return K1_MODE_COL;   /* every nu >= every mu */
    return K1_MODE_GATHER;                                     /* a bulk copy would read past the end of B */
}

__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}


template <int NT8>
struct K1Cfg {
    static constexpr int NW = 8 * NT8;
    static constexpr int C_BYTES = K1_KC * NW * 8;
    static constexpr int STAGE_BYTES = K1_A_BYTES + C_BYTES;
    static constexpr int STAGES_RAW = K1_SMEM_BUDGET / STAGE_BYTES;
    static constexpr int STAGES = STAGES_RAW > 8 ? 8 : STAGES_RAW;
    static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 2 * STAGES * 8 + 16;
};

/* Work items.  A plain item is (p, row block, column tile): 128 rows of one B_P.  A ragged last row
 * block with r <= 64 valid rows would be a low-intensity item (the whole C tile staged for a quarter
 * of the MMAs: its stages outrun the 3-4 stage ring, 4.5 % of K1 at nao = 800), so its rows are
 * batched over G = 2, 4 or 8 consecutive P (r <= 64, 32, 16): a RAGGED item stacks the r rows of G
 * different B_P into one 128-row tile -- slot pp = m >> rshift of the tile holds P = p + pp, its row
 * m & (rpad - 1) is mu0 + that -- against the one C tile they all share.  Items are numbered per group
 * of G auxiliary indices: the G (nib - 1) ntiles_n plain items first (p-major, so the items of one P
 * still run side by side for the tournament order), then the group's ntiles_n ragged items. */
struct K1Item {
    int64_t p, mu0, n0;      /* first (or only) auxiliary index relative to P0, first row, first column */
    int np_item, rshift;     /* P slots in use (1 for a plain item), log2(rows per slot) (7: plain) */
};

__device__ __forceinline__ K1Item k1_decode(int64_t item, int nib, int ntiles_n, int rag_g, int64_t np, int nw)
{
    K1Item it;
    if (rag_g == 0) {
        const int per_p = nib * ntiles_n;
        it.p = item / per_p;
        const int rem = (int)(item - it.p * per_p);
        it.mu0 = (int64_t)(rem / ntiles_n) * K1_M;
        it.n0 = (int64_t)(rem % ntiles_n) * nw;
        it.np_item = 1;
        it.rshift = 7;
        return it;
    }
    const int nfull = nib - 1;
    const int per_group = (rag_g * nfull + 1) * ntiles_n;
    const int64_t grp = item / per_group;
    const int w = (int)(item - grp * per_group);
    const int64_t left = np - grp * rag_g;                    /* auxiliary indices from this group on */
    const int gg = left < rag_g ? (int)left : rag_g;
    const int nf = gg * nfull * ntiles_n;
    if (w < nf) {
        const int pl = w / (nfull * ntiles_n), rem = w - pl * (nfull * ntiles_n);
        it.p = grp * rag_g + pl;
        it.mu0 = (int64_t)(rem / ntiles_n) * K1_M;
        it.n0 = (int64_t)(rem % ntiles_n) * nw;
        it.np_item = 1;
        it.rshift = 7;
    } else {
        it.p = grp * rag_g;
        it.mu0 = (int64_t)nfull * K1_M;
        it.n0 = (int64_t)(w - nf) * nw;
        it.np_item = gg;
        it.rshift = rag_g == 2 ? 6 : (rag_g == 4 ? 5 : 4);
    }
    return it;
}

/* PERSISTENT: the grid is one CTA per SM; CTA b processes the work items b, b + gridDim.x, ...
 * with the mbarrier ring running THROUGH item boundaries: while the consumers write one item's X
 * tile, the producers are already filling the stages of the next one.  Producers and consumers walk
 * the same item sequence independently.
 * (One CTA per item cost a pipeline fill + drain per 25-50 stages: 16 % of K1 at nao = 290.) */
template <int NT8>
__global__ void __launch_bounds__(K1_THREADS, 1)
k1_half_transform_kernel(const double *__restrict__ B, int64_t naux, int64_t nao, int64_t npair, int64_t P0,
                         int64_t np, const double *__restrict__ Ccat4, int64_t ldc, int64_t ldx, int ntiles_n,
                         int rag_g, int64_t nitems, double *__restrict__ X4)
{
    using Cfg = K1Cfg<NT8>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nk = (int)((nao + K1_KC - 1) / K1_KC);
    const int nib = (int)((nao + K1_M - 1) / K1_M);

    const uint32_t smem_base = smem_u32(smem_raw);
    const uint32_t bar_base = smem_base + Cfg::STAGES * Cfg::STAGE_BYTES;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (Cfg::STAGES + s); };

    if (tid == 0) {
        for (int s = 0; s < Cfg::STAGES; ++s) {
            mbar_init(full_bar(s), K1_PRODUCERS);
            mbar_init(empty_bar(s), K1_CONSUMERS / 32);
        }
        mbar_fence_init();
    }
    __syncthreads();

    if (warp < K1_PRODUCERS / 32) {
        /* ------------------------------------------------------------ producers */
        reg_dealloc<40>();
        int slot = 0;
        uint32_t phase = 1;                                /* parity of the "empty" phase to wait for */
        bool ring_full = false;                            /* all STAGES slots have been used once */
        for (int64_t item = blockIdx.x; item < nitems; item += gridDim.x) {
        const K1Item it = k1_decode(item, nib, ntiles_n, rag_g, np, Cfg::NW);
        const int64_t mu0 = it.mu0, n0 = it.n0;
        const bool multi = it.rshift != 7;
        const int64_t pb = (P0 + it.p) * npair;            /* index of B_P's first element in B */
        const bool last_p = P0 + it.p == naux - 1;
        int64_t ncols = ldc - n0;                          /* valid columns of this N tile */
        if (ncols > Cfg::NW) ncols = Cfg::NW;
        const uint32_t c_bytes = K1_KG * (uint32_t)ncols * 32u;
        int64_t rows_valid = nao - mu0;
        if (rows_valid > K1_M) rows_valid = K1_M;
        /* "row" form: thread t stages tile row t = packed row mu_t of slot t >> rshift */
        const int pp_t = tid >> it.rshift;
        const int64_t mu_t = mu0 + (tid & ((1 << it.rshift) - 1));
        const bool ok_t = mu_t < nao && pp_t < it.np_item;
        const int64_t erow = pb + pp_t * npair + mu_t * (mu_t + 1) / 2;      /* element (mu_t, 0) of that P */
        const int rbi = (int)(mu0 / K1_M);
        for (int sstep = 0; sstep < nib; ++sstep) {
        /* column block of this step: the tournament partner */
        const int jb = sstep >= rbi ? sstep - rbi : sstep - rbi + nib;
        const int kc_end = (jb + 1) * (K1_M / K1_KC) < nk ? (jb + 1) * (K1_M / K1_KC) : nk;
        for (int kc = jb * (K1_M / K1_KC); kc < kc_end; ++kc) {
            if (ring_full) mbar_wait(empty_bar(slot), phase);
            const int64_t nu0 = (int64_t)kc * K1_KC;
            const uint32_t a_dst = smem_base + slot * Cfg::STAGE_BYTES;
            const uint32_t bar = full_bar(slot);
            const int mode = k1_mode((int)mu0, kc * K1_KC, (int)nao, last_p, multi);
            uint32_t my_bytes = tid == 0 ? c_bytes : 0u;
            if (mode == K1_MODE_ROW) {
                /* columns nu0 .. nu0+31 of the thread's packed row (+ alignment slack) */
                const int64_t e = erow + nu0;
                const int sft = (int)(e & 1);
                const uint32_t nb = ok_t ? (uint32_t)(K1_KC + 2 * sft) * 8u : 0u;
                my_bytes += nb;
                if (my_bytes) mbar_arrive_expect_tx(bar, my_bytes); else mbar_arrive(bar);
                if (ok_t) bulk_g2s(a_dst + tid * (K1_LDD * 8), B + (e - sft), nb, bar);
            } else if (mode == K1_MODE_COL) {
                /* thread t < 32 copies packed row nu0+t, columns mu0 .. mu0+rows_valid-1 */
                const int64_t nu = nu0 + tid;
                const bool ok = tid < K1_KC && nu < nao;
                const int64_t e = pb + nu * (nu + 1) / 2 + mu0;
                const int sft = (int)(e & 1);
                const uint32_t nb = ok ? (uint32_t)((rows_valid + sft + 1) & ~(int64_t)1) * 8u : 0u;
                my_bytes += nb;
                /* rows nu >= nao of the tile multiply zero rows of C: they must not hold NaNs */
                for (int k = (int)(nao - nu0); k < K1_KC; ++k)
                    for (int c = tid; c < K1_LDT; c += K1_PRODUCERS)
                        reinterpret_cast<double *>(smem_raw + slot * Cfg::STAGE_BYTES)[k * K1_LDT + c] = 0.0;
                if (my_bytes) mbar_arrive_expect_tx(bar, my_bytes); else mbar_arrive(bar);
                if (ok) bulk_g2s(a_dst + tid * (K1_LDT * 8), B + (e - sft), nb, bar);
            } else if (mode == K1_MODE_DIAG) {
                /* A stage inside the diagonal block of a plain item, R0 = nu0 - mu0 in {0, 32, 64, 96}:
                 * three bands of rows.
                 *   m <  R0      : every nu > mu -> "col" form, 32 copies of R0 doubles (packed rows nu0+k),
                 *                  pitch R0 + 4, at the start of the stage buffer (it ends below row R0 of
                 *                  the "row" form: 32 (R0 + 4) 8 <= R0 36 8)
                 *   m >= R0 + 32 : every nu < mu -> "row" form, one copy of 32 doubles per row
                 *   the 32 x 32 block on the diagonal: element-wise (8-byte cp.async, zero fill outside)
                 * so 1024 instead of 4096 gathered elements per stage (they cost 16 % of K1 at nao = 290). */
                const int R0 = (int)(nu0 - mu0);
                if (tid >= R0 + K1_KC) {
                    if (ok_t) {
                        const int64_t e = erow + nu0;
                        const int sft = (int)(e & 1);
                        const uint32_t nb = (uint32_t)(K1_KC + 2 * sft) * 8u;
                        mbar_expect_tx(bar, my_bytes + nb);
                        bulk_g2s(a_dst + tid * (K1_LDD * 8), B + (e - sft), nb, bar);
                        my_bytes = 0;
                    }
                } else if (tid < K1_KC && R0 > 0) {           /* nu0 + 31 < nao in this mode */
                    const int64_t nu = nu0 + tid;
                    const int64_t e = pb + nu * (nu + 1) / 2 + mu0;
                    const int sft = (int)(e & 1);
                    const uint32_t nb = (uint32_t)((R0 + sft + 1) & ~1) * 8u;
                    mbar_expect_tx(bar, my_bytes + nb);
                    bulk_g2s(a_dst + tid * ((R0 + 4) * 8), B + (e - sft), nb, bar);
                    my_bytes = 0;
                }
                if (my_bytes) mbar_expect_tx(bar, my_bytes);   /* thread 0 without a copy of its own */
                {
                    const int pbpar = (int)(pb & 1);
                    const int k = tid & 31;
                    const int64_t nu = nu0 + k;
                    const int64_t tri_nu = nu * (nu + 1) / 2;
#pragma unroll
                    for (int r = 0; r < K1_KC / 4; ++r) {
                        const int m = R0 + 4 * r + (tid >> 5);
                        const int64_t mu = mu0 + m;
                        const bool ok = nu < nao && mu < nao;
                        const int64_t off = mu >= nu ? mu * (mu + 1) / 2 + nu : tri_nu + mu;
                        const int sd = (((m & 3) == 1 || (m & 3) == 2) ? 1 : 0) ^ pbpar;
                        cp_async8(a_dst + (m * K1_LDD + k + sd) * 8, ok ? B + pb + off : B, ok);
                    }
                }
                cp_async_mbar_arrive_noinc(bar);
            } else {
                /* element-wise gather into the "row" form (8-byte cp.async, zero fill outside); tile row
                 * m belongs to slot m >> rshift (a plain item has one slot) */
                if (tid == 0) mbar_expect_tx(bar, c_bytes);
                const int k = tid & 31;
                const int64_t nu = nu0 + k;
                const int64_t tri_nu = nu * (nu + 1) / 2;
#pragma unroll 4
                for (int r = 0; r < K1_M / 4; ++r) {
                    const int m = 4 * r + (tid >> 5);
                    const int pp = m >> it.rshift;
                    const int64_t mu = mu0 + (m & ((1 << it.rshift) - 1));
                    const bool ok = nu < nao && mu < nao && pp < it.np_item;
                    const int64_t pbm = pb + pp * npair;
                    const int64_t off = mu >= nu ? mu * (mu + 1) / 2 + nu : tri_nu + mu;
                    const int sd = (((m & 3) == 1 || (m & 3) == 2) ? 1 : 0) ^ (int)(pbm & 1);
                    cp_async8(a_dst + (m * K1_LDD + k + sd) * 8, ok ? B + pbm + off : B, ok);
                }
                cp_async_mbar_arrive_noinc(bar);
            }
            if (tid == 0) {
                const uint32_t c_dst = a_dst + K1_A_BYTES;
#pragma unroll
                for (int g = 0; g < K1_KG; ++g)
                    bulk_g2s(c_dst + g * Cfg::NW * 32, Ccat4 + (((int64_t)kc * K1_KG + g) * ldc + n0) * 4,
                             (uint32_t)ncols * 32u, bar);
            }
            if (++slot == Cfg::STAGES) { slot = 0; phase ^= 1; ring_full = true; }
        }
        }   /* column blocks */
        }   /* items */
    } else {
        /* ------------------------------------------------------------ consumers */
        reg_alloc<232>();
        const int cw = warp - K1_PRODUCERS / 32;           /* 0..7: tile rows 16*cw .. 16*cw+15 */
        const int row_w = 16 * cw;
        const int lq = lane >> 2, lr = lane & 3;
        int slot = 0;
        uint32_t phase = 0;
        for (int64_t item = blockIdx.x; item < nitems; item += gridDim.x) {
        const K1Item it = k1_decode(item, nib, ntiles_n, rag_g, np, Cfg::NW);
        const int64_t mu0 = it.mu0, n0 = it.n0;
        const bool multi = it.rshift != 7;
        /* this warp's 16 tile rows lie in one slot: auxiliary index pw, rows mu_w .. mu_w + 15 */
        const int pp_w = row_w >> it.rshift;
        const int64_t pw = it.p + pp_w;
        const int64_t mu_w = mu0 + (row_w & ((1 << it.rshift) - 1));
        const bool warp_active = mu_w < nao && pp_w < it.np_item;
        const int pbpar = (int)(((P0 + pw) * npair) & 1);
        const bool last_p = P0 + it.p == naux - 1;
        /* per-lane alignment shifts of the two tile forms (see K1_LDD / K1_LDT) */
        const int sd_shift = (((lq & 3) == 1 || (lq & 3) == 2) ? 1 : 0) ^ pbpar;
        const int st_shift = ((lr == 1 || lr == 2) ? 1 : 0) ^ pbpar;
        double acc[2][NT8][2];
#pragma unroll
        for (int mt = 0; mt < 2; ++mt)
#pragma unroll
            for (int nt = 0; nt < NT8; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;

        const int rbi = (int)(mu0 / K1_M);
        for (int sstep = 0; sstep < nib; ++sstep) {
        const int jb = sstep >= rbi ? sstep - rbi : sstep - rbi + nib;
        const int kc_end = (jb + 1) * (K1_M / K1_KC) < nk ? (jb + 1) * (K1_M / K1_KC) : nk;
        for (int kc = jb * (K1_M / K1_KC); kc < kc_end; ++kc) {
            mbar_wait(full_bar(slot), phase);
            if (warp_active) {
                const double *As = reinterpret_cast<const double *>(smem_raw + slot * Cfg::STAGE_BYTES);
                const double *Cs = As + K1_A_BYTES / 8;
                /* "col" form: COL stages, and the rows above the diagonal of a DIAG stage (pitch R0 + 4) */
                const int mode = k1_mode((int)mu0, kc * K1_KC, (int)nao, last_p, multi);
                const int R0 = kc * K1_KC - (int)mu0;
                const bool colform = mode == K1_MODE_COL || (mode == K1_MODE_DIAG && row_w < R0);
                const int ldt = mode == K1_MODE_COL ? K1_LDT : R0 + 4;
                const double *a_base = colform ? As + lr * ldt + row_w + lq + st_shift
                                               : As + (row_w + lq) * K1_LDD + lr + sd_shift;
                const int a_gstep = colform ? 4 * ldt : 4;           /* next k-group */
                const int a_mstep = colform ? 8 : 8 * K1_LDD;        /* next 8 rows */
                const double *b_base = Cs + lq * 4 + lr;
#pragma unroll
                for (int g = 0; g < K1_KG; ++g) {
                    const double a0 = a_base[g * a_gstep];
                    const double a1 = a_base[g * a_gstep + a_mstep];
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
        }   /* column blocks */

        if (warp_active) {
            /* X4[(k >> 2)][mu][k & 3], k = pw ldx + n0 + 8 nt + 2 lr: ldx and n0 are multiples of 8, so the
             * k-group is kb + 2 nt + (lr >> 1) and the store of column tile nt sits 8 nao doubles after
             * the one of nt - 1 (per-store 64-bit index arithmetic cost 1.6 % of K1 at nao = 800) */
            const int64_t kb = (pw * ldx + n0) >> 2;
            const int nt_valid = (int)((ldc - n0) >> 3);           /* column tiles inside ldc */
            double *dst0 = X4 + ((kb + (lr >> 1)) * nao + mu_w + lq) * 4 + 2 * (lr & 1);
            const int64_t nt_step = 8 * nao;
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) {
                if (mu_w + 8 * mt + lq >= nao) continue;
                double *dst = dst0 + 32 * mt;
#pragma unroll
                for (int nt = 0; nt < NT8; ++nt) {
                    if (nt < nt_valid)
                        *reinterpret_cast<double2 *>(dst) = make_double2(acc[mt][nt][0], acc[mt][nt][1]);
                    dst += nt_step;
                }
            }
        }
        }   /* items */
    }
}

/* K1U: the identity half of the raw-dm build, X_P = B_P . I = B_P unpacked, written straight
 * into X's k-group-major layout without touching the FP64 pipe:
 *     X4[(k/4)][mu][k%4] = B_P(mu, i),   k = p*ldx + col0 + i,   i < round_up(nao, 4) (0 for i >= nao)
 * One thread per (mu, group of four i): four packed loads (max/min addressing), one 32-byte store;
 * consecutive threads own consecutive mu, so the stores are contiguous. */
__global__ void __launch_bounds__(128)
k1u_unpack_kernel(const double *__restrict__ B, int64_t nao, int64_t npair, int64_t P0, int64_t ldx,
                  int64_t col0, double *__restrict__ X4)
{
    const int64_t mu = (int64_t)blockIdx.x * 128 + threadIdx.x;
    if (mu >= nao) return;
    const int64_t i0 = 4 * (int64_t)blockIdx.y, p = blockIdx.z;
    const double *Bp = B + (P0 + p) * npair;
    double v[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const int64_t i = i0 + q;
        const int64_t a = mu > i ? mu : i, b = mu > i ? i : mu;
        v[q] = i < nao ? Bp[a * (a + 1) / 2 + b] : 0.0;
    }
    const int64_t k = p * ldx + col0 + i0;                 /* multiple of 4 */
    double2 *dst = reinterpret_cast<double2 *>(X4 + ((k >> 2) * nao + mu) * 4);
    dst[0] = make_double2(v[0], v[1]);
    dst[1] = make_double2(v[2], v[3]);
}

template <int NT8>
cudaError_t k1_launch_t(const double *B, int64_t naux, int64_t nao, int64_t npair, int64_t P0, int64_t np,
                        const double *Ccat4, int64_t ldc, int64_t ldx, int ntiles_n, double *X4, cudaStream_t st)
{
    static std::atomic<unsigned long long> smem_ok{0};
    cudaError_t e = ensure_dynamic_smem(k1_half_transform_kernel<NT8>, K1Cfg<NT8>::SMEM_BYTES, smem_ok);
    if (e != cudaSuccess) return e;
    int dev = 0, sm_count = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev);
    if (sm_count <= 0) sm_count = 148;
    const int64_t nib = (nao + K1_M - 1) / K1_M;
    /* a ragged last row block with <= 64 rows is batched over G auxiliary indices (see K1Item) */
    const int64_t rlast = nao - (nib - 1) * K1_M;
    const int rag_g = rlast <= 16 ? 8 : (rlast <= 32 ? 4 : (rlast <= 64 ? 2 : 0));
    int64_t nitems;
    if (rag_g == 0) {
        nitems = nib * ntiles_n * np;
    } else {
        const int64_t ngroups = (np + rag_g - 1) / rag_g, gl = np - (ngroups - 1) * rag_g;
        nitems = (ngroups - 1) * (rag_g * (nib - 1) + 1) * ntiles_n + (gl * (nib - 1) + 1) * ntiles_n;
    }
    const unsigned grid = (unsigned)(nitems < sm_count ? nitems : sm_count);   /* persistent: 1 CTA / SM */
    k1_half_transform_kernel<NT8><<<grid, K1_THREADS, K1Cfg<NT8>::SMEM_BYTES, st>>>(
        B, naux, nao, npair, P0, np, Ccat4, ldc, ldx, ntiles_n, rag_g, nitems, X4);
    return cudaPeekAtLastError();
}

}  // namespace


cudaError_t launch_k1_half_transform(const double *B, int64_t naux, int64_t nao, int64_t npair, int64_t P0,
                                     int64_t np, const double *Ccat4, int64_t ldc, int64_t ldx, double *X4,
                                     cudaStream_t st)
{
    if (ldc % 8 != 0 || ldx % 8 != 0) return cudaErrorInvalidValue;   /* the kernel's X addressing relies on it */
    const int n8 = (int)(ldc / 8);
    const int ntiles_n = (n8 + 16) / 17;
    const int nt8 = (n8 + ntiles_n - 1) / ntiles_n;
    /* grid.y <= 65535: chunks are far smaller than that */
#define DFJK_K1_CASE(N) \
    case N: return k1_launch_t<N>(B, naux, nao, npair, P0, np, Ccat4, ldc, ldx, ntiles_n, X4, st);
    switch (nt8) {
        DFJK_K1_CASE(1) DFJK_K1_CASE(2) DFJK_K1_CASE(3) DFJK_K1_CASE(4) DFJK_K1_CASE(5)
        DFJK_K1_CASE(6) DFJK_K1_CASE(7) DFJK_K1_CASE(8) DFJK_K1_CASE(9) DFJK_K1_CASE(10)
        DFJK_K1_CASE(11) DFJK_K1_CASE(12) DFJK_K1_CASE(13) DFJK_K1_CASE(14) DFJK_K1_CASE(15)
        DFJK_K1_CASE(16) DFJK_K1_CASE(17)
    default: return cudaErrorInvalidValue;      /* no tile shape for this width: never launch nothing silently */
    }
#undef DFJK_K1_CASE
}

void launch_k1u_unpack(const double *B, int64_t nao, int64_t npair, int64_t P0, int64_t np, int64_t ldx,
                       int64_t col0, double *X4, cudaStream_t st)
{
    dim3 grid((unsigned)((nao + 127) / 128), (unsigned)((nao + 3) / 4), (unsigned)np);
    k1u_unpack_kernel<<<grid, 128, 0, st>>>(B, nao, npair, P0, ldx, col0, X4);
}

}  // namespace dfjk
