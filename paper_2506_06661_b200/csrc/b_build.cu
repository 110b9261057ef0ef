/*
 * b_build.cu -- building the whitened DF tensor on the device (include/dfjk.h, dfjk_build_b),
 * PAPER.md:353-356, Eq. 2-3:
 *
 *     M_PQ = (chi_P|chi_Q) = L L^T                       Eq. 2   (FP64 Cholesky, naux x naux)
 *     B[P][pair] = sum_Q (L^-1)[P][Q] R[Q][pair]          Eq. 3   (triangular solve over npair columns)
 *
 * Phase 1 (tiny: naux^3/3 flop, latency-bound): right-looking blocked Cholesky, block 128.
 *   per block column j:  W1 factor the 128 x 128 diagonal block in shared memory
 *                        W2 invert it (one thread per column, forward substitution)
 *                        W3 panel   L_ij = M_ij Linv_jj^T            (plain FP64 FMA tiles)
 *                        W4 trailing M_ik -= L_ij L_kj^T, i >= k > j  (plain FP64 FMA tiles)
 *   and the row block of the "solve operator"
 *                        Aw[i] = Linv_ii [ -L_{i,<i} | I ]  =  [ -Linv_ii L_{i,<i} | Linv_ii ]
 * Phase 2 (the work: naux^2 npair flop = 3.2e13 at cfg 4; FP64 pipe bound, DMMA.8x8x4):
 *   per block row i, ONE product over the array being overwritten in place,
 *       B_i = Aw[i] . [ B_0 ; ... ; B_{i-1} ; R_i ]         (128 x (128 i + 128)) . ((128 i + 128) x npair)
 *   i.e. B_i = Linv_ii (R_i - sum_{j<i} L_ij B_j): rows < 128 i are already final, rows of block
 *   i still hold R.  A CTA owns a 128-column tile and all 128 rows of the block, reads its
 *   columns of rows 128 i .. in the last k stages and overwrites them only in the epilogue, so
 *   the update is in place without a second copy of the 51-96 GB tensor.
 *   Kernel W5 has K1's structure: 4 producer warps (TMA 1-D bulk copies into a 3-stage
 *   mbarrier ring; packed rows are only 8-byte aligned, handled by K1's one-element shift),
 *   8 consumer warps with 16 x 128 accumulators each.
 *
 * Using the inverse of the 128 x 128 diagonal blocks (not of L) is the standard blocked TRSM;
 * its extra rounding error is bounded by cond(L_ii) * eps per block.
 */
#include "dfjk_internal.h"
#include "k_common.cuh"

namespace dfjk {
namespace {

constexpr int NB = 128;                       /* block size of both phases */

/* ------------------------------------------------------------------ W1: diagonal block */
/* In-place Cholesky of the n x n (n <= 128) block at M[r0][r0] (leading dimension ld), lower
 * triangle; the strict upper triangle of the block is set to zero.  info (may be NULL): set to
 * r0 + k + 1 at the first non-positive pivot k (LAPACK convention), left unchanged otherwise. */
__global__ void __launch_bounds__(256, 1)
chol_diag_kernel(double *__restrict__ M, int64_t ld, int64_t r0, int n, long long *info)
{
    extern __shared__ __align__(16) double sA[];          /* [NB][NB + 1] */
    constexpr int P = NB + 1;
    const int tid = threadIdx.x;
    double *blk = M + r0 * ld + r0;
    for (int idx = tid; idx < n * n; idx += 256) {
        const int i = idx / n, j = idx - i * n;
        sA[i * P + j] = (j <= i) ? blk[(int64_t)i * ld + j] : 0.0;
    }
    __syncthreads();
    for (int k = 0; k < n; ++k) {
        if (tid == 0) {
            const double piv = sA[k * P + k];
            if (!(piv > 0.0) && info && *info == 0) *info = (long long)(r0 + k + 1);
            sA[k * P + k] = sqrt(piv);
        }
        __syncthreads();
        const double dinv = 1.0 / sA[k * P + k];
        for (int i = k + 1 + tid; i < n; i += 256) sA[i * P + k] *= dinv;
        __syncthreads();
        const int m = n - k - 1;
        for (int idx = tid; idx < m * m; idx += 256) {
            const int i = k + 1 + idx / m, j = k + 1 + idx % m;
            if (j <= i) sA[i * P + j] -= sA[i * P + k] * sA[j * P + k];
        }
        __syncthreads();
    }
    for (int idx = tid; idx < n * n; idx += 256) {
        const int i = idx / n, j = idx - i * n;
        blk[(int64_t)i * ld + j] = sA[i * P + j];
    }
}

/* ------------------------------------------------------------------ W2: invert the block */
/* Linv = L_jj^-1 (lower triangular), thread c owns column c:
 *     Linv[r][c] = ( delta_rc - sum_{c <= k < r} L[r][k] Linv[k][c] ) / L[r][r],   r >= c
 * written, zero-padded to 128 x 128, into Aw[r0 + r][r0 + c] (leading dimension ldw). */
__global__ void __launch_bounds__(NB, 1)
tri_inv_kernel(const double *__restrict__ M, int64_t ld, int64_t r0, int n,
               double *__restrict__ Aw, int64_t ldw)
{
    extern __shared__ __align__(16) double sS[];          /* [NB][NB]: column c is private to thread c */
    const int c = threadIdx.x;
    const double *L = M + r0 * ld + r0;
    if (c < n) {
        for (int r = c; r < n; ++r) {
            double s = (r == c) ? 1.0 : 0.0;
            const double *Lr = L + (int64_t)r * ld;
            for (int k = c; k < r; ++k) s -= Lr[k] * sS[k * NB + c];
            sS[r * NB + c] = s / Lr[r];
        }
    }
    double *out = Aw + r0 * ldw + r0;
    for (int r = 0; r < NB; ++r)
        out[(int64_t)r * ldw + c] = (c < n && r < n && r >= c) ? sS[r * NB + c] : 0.0;
}

/* ------------------------------------------------------------------ W3/W4: small FP64 tiles */
/* C[m][n] = beta C[m][n] + alpha sum_k A[m*lda + k] * Bop[k*sbk + n*sbn],  m < Mr, n < Nc, k < Kd.
 * (sbk, sbn) = (ldb, 1) is A.B, (1, ldb) is A.B^T.  64 x 64 tiles, 256 threads, 4 x 4 per thread.
 * lower_only: only entries n <= m are computed and written (C is a diagonal sub-block of M).
 * Phase 1 is ~0.1 % of the flops of dfjk_build_b: plain FMAs, no tensor pipe. */
constexpr int SG_T = 64, SG_K = 16;

__global__ void __launch_bounds__(256)
small_gemm_kernel(const double *__restrict__ A, int64_t lda, const double *__restrict__ Bop,
                  int64_t sbk, int64_t sbn, double *__restrict__ C, int64_t ldc, int64_t Mr,
                  int64_t Nc, int64_t Kd, double alpha, double beta, int lower_only)
{
    const int64_t m0 = (int64_t)blockIdx.y * SG_T, n0 = (int64_t)blockIdx.x * SG_T;
    if (lower_only && n0 > m0 + SG_T - 1) return;
    __shared__ double sA[SG_K][SG_T + 1];                 /* [k][m] */
    __shared__ double sB[SG_K][SG_T + 1];                 /* [k][n] */
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    double acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = 0.0;
    for (int64_t k0 = 0; k0 < Kd; k0 += SG_K) {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int idx = tid + 256 * q;                /* 0 .. 1023 */
            {   /* A: consecutive threads walk k (contiguous in memory) */
                const int k = idx & 15, m = idx >> 4;
                const int64_t gm = m0 + m, gk = k0 + k;
                sA[k][m] = (gm < Mr && gk < Kd) ? A[gm * lda + gk] : 0.0;
            }
            {   /* Bop: walk whichever index is contiguous */
                int k, n;
                if (sbk == 1) { k = idx & 15; n = idx >> 4; } else { n = idx & 63; k = idx >> 6; }
                const int64_t gn = n0 + n, gk = k0 + k;
                sB[k][n] = (gn < Nc && gk < Kd) ? Bop[gk * sbk + gn * sbn] : 0.0;
            }
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < SG_K; ++k) {
            double a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = sA[k][ty + 16 * i];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = sB[k][tx + 16 * j];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] += a[i] * b[j];
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int64_t gm = m0 + ty + 16 * i;
        if (gm >= Mr) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int64_t gn = n0 + tx + 16 * j;
            if (gn >= Nc || (lower_only && gn > gm)) continue;
            double *c = C + gm * ldc + gn;
            *c = (beta == 0.0 ? 0.0 : beta * *c) + alpha * acc[i][j];
        }
    }
}

void small_gemm(const double *A, int64_t lda, const double *Bop, int64_t sbk, int64_t sbn, double *C,
                int64_t ldc, int64_t Mr, int64_t Nc, int64_t Kd, double alpha, double beta,
                int lower_only, cudaStream_t st)
{
    if (Mr <= 0 || Nc <= 0) return;
    dim3 grid((unsigned)((Nc + SG_T - 1) / SG_T), (unsigned)((Mr + SG_T - 1) / SG_T));
    small_gemm_kernel<<<grid, 256, 0, st>>>(A, lda, Bop, sbk, sbn, C, ldc, Mr, Nc, Kd, alpha, beta,
                                            lower_only);
}

/* ------------------------------------------------------------------ W5: the DMMA product */
constexpr int W_KG = 8;                              /* k-groups (of 4) per stage */
constexpr int W_KC = 4 * W_KG;                       /* 32 */
constexpr int W_PRODUCERS = 128, W_CONSUMERS = 256, W_THREADS = W_PRODUCERS + W_CONSUMERS;
constexpr int W_LDA = 36;                            /* A stage [128 m][36]: 32 k + pad, == 4 mod 16 */
constexpr int W_LDB = 132;                           /* B stage [32 k][132]: 128 n + shift + pad     */
constexpr int W_A_BYTES = NB * W_LDA * 8;            /* 36864 */
constexpr int W_B_BYTES = W_KC * W_LDB * 8;          /* 33792 */
constexpr int W_STAGE_BYTES = W_A_BYTES + W_B_BYTES; /* 70656 */
constexpr int W_STAGES = 3;
constexpr int W_SMEM_BYTES = W_STAGES * W_STAGE_BYTES + 2 * W_STAGES * 8 + 16;

__device__ __forceinline__ void w_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}

/* T[r0 + m][n] = sum_{k < kend} Aw[r0 + m][k] * T[k][n]   for m < 128 (rows < naux), n in this
 * CTA's 128-column tile; T = the packed tensor, R on entry / B on exit for rows >= r0.
 * kend = r0 + (rows of this block); Aw's columns >= kend are zero (workspace zero-padded to
 * multiples of 128), rows k >= naux of T are replaced by zeros in shared memory. */
__global__ void __launch_bounds__(W_THREADS, 1)
whiten_gemm_kernel(double *__restrict__ T, int64_t naux, int64_t npair,
                   const double *__restrict__ Aw, int64_t ldw, int64_t r0, int64_t kend)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t n0 = (int64_t)blockIdx.x * NB;
    const int nk = (int)((kend + W_KC - 1) / W_KC);
    const int podd = (int)(npair & 1);
    /* the last column tile gathers element-wise: its bulk copies could read past the end of T */
    const bool edge = n0 + NB >= npair;
    int64_t cols_valid = npair - n0;
    if (cols_valid > NB) cols_valid = NB;

    const uint32_t smem_base = smem_u32(smem_raw);
    const uint32_t bar_base = smem_base + W_STAGES * W_STAGE_BYTES;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (W_STAGES + s); };
    if (tid == 0) {
        for (int s = 0; s < W_STAGES; ++s) {
            mbar_init(full_bar(s), W_PRODUCERS);
            mbar_init(empty_bar(s), W_CONSUMERS / 32);
        }
        mbar_fence_init();
    }
    __syncthreads();

    if (warp < W_PRODUCERS / 32) {
        /* ------------------------------------------------------------ producers */
        reg_dealloc<40>();
        int slot = 0;
        uint32_t phase = 1;
        for (int kc = 0; kc < nk; ++kc) {
            if (kc >= W_STAGES) mbar_wait(empty_bar(slot), phase);
            const int64_t k0 = (int64_t)kc * W_KC;
            const uint32_t a_dst = smem_base + slot * W_STAGE_BYTES;
            const uint32_t b_dst = a_dst + W_A_BYTES;
            const uint32_t bar = full_bar(slot);
            double *bs = reinterpret_cast<double *>(smem_raw + slot * W_STAGE_BYTES + W_A_BYTES);
            /* A: thread t copies row r0+t of the operator, columns k0 .. k0+31 (16-B aligned) */
            const double *a_src = Aw + (r0 + tid) * ldw + k0;
            if (!edge) {
                uint32_t my_bytes = W_KC * 8;
                /* B: thread t < 32 copies row k0+t of T, columns n0 .. n0+127 (+ alignment slack) */
                const int64_t k = k0 + tid;
                const bool ok = tid < W_KC && k < naux;
                const int64_t e = k * npair + n0;
                const int sft = (int)(e & 1);
                const uint32_t nb = ok ? (uint32_t)((NB + sft + 1) & ~1) * 8u : 0u;
                my_bytes += nb;
                /* rows k >= naux multiply zero columns of the operator: they must not hold NaNs */
                for (int kk = (int)(naux - k0); kk < W_KC; ++kk)
                    for (int c = tid; c < W_LDB; c += W_PRODUCERS) bs[kk * W_LDB + c] = 0.0;
                mbar_arrive_expect_tx(bar, my_bytes);
                bulk_g2s(a_dst + tid * (W_LDA * 8), a_src, W_KC * 8, bar);
                if (ok) bulk_g2s(b_dst + tid * (W_LDB * 8), T + (e - sft), nb, bar);
            } else {
                w_expect_tx(bar, W_KC * 8);
                bulk_g2s(a_dst + tid * (W_LDA * 8), a_src, W_KC * 8, bar);
                const int kk = tid & 31;
                const int64_t k = k0 + kk;
                const int sk = (kk & 1) & podd;            /* parity of k*npair + n0 (n0 even) */
#pragma unroll 4
                for (int r = 0; r < NB / 4; ++r) {
                    const int c = 4 * r + (tid >> 5);
                    const bool ok = k < naux && c < cols_valid;
                    cp_async8(b_dst + (kk * W_LDB + c + sk) * 8, ok ? T + k * npair + n0 + c : T, ok);
                }
                cp_async_mbar_arrive_noinc(bar);
            }
            if (++slot == W_STAGES) { slot = 0; phase ^= 1; }
        }
    } else {
        /* ------------------------------------------------------------ consumers */
        reg_alloc<232>();
        const int cw = warp - W_PRODUCERS / 32;            /* rows 16*cw .. 16*cw+15 of the block */
        const int lq = lane >> 2, lr = lane & 3;
        const int sb = (lr & 1) & podd;                    /* alignment shift of row k = 4g + lr */
        double acc[2][16][2];
#pragma unroll
        for (int mt = 0; mt < 2; ++mt)
#pragma unroll
            for (int nt = 0; nt < 16; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;
        const bool warp_active = r0 + 16 * cw < naux;
        int slot = 0;
        uint32_t phase = 0;
        for (int kc = 0; kc < nk; ++kc) {
            mbar_wait(full_bar(slot), phase);
            if (warp_active) {
                const double *As = reinterpret_cast<const double *>(smem_raw + slot * W_STAGE_BYTES);
                const double *Bs = As + W_A_BYTES / 8;
                const double *a_base = As + (16 * cw + lq) * W_LDA + lr;
                const double *b_base = Bs + lr * W_LDB + lq + sb;
#pragma unroll
                for (int g = 0; g < W_KG; ++g) {
                    const double a0 = a_base[4 * g];
                    const double a1 = a_base[4 * g + 8 * W_LDA];
#pragma unroll
                    for (int nt = 0; nt < 16; ++nt) {
                        const double b = b_base[g * (4 * W_LDB) + 8 * nt];
                        dmma884(acc[0][nt][0], acc[0][nt][1], a0, b);
                        dmma884(acc[1][nt][0], acc[1][nt][1], a1, b);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty_bar(slot));
            if (++slot == W_STAGES) { slot = 0; phase ^= 1; }
        }
        /* epilogue: overwrite rows r0.. of this column tile (every read of them is complete: the
         * last full barrier was waited on by this warp, and other warps own other rows) */
        if (warp_active) {
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) {
                const int64_t row = r0 + 16 * cw + 8 * mt + lq;
                if (row >= naux) continue;
#pragma unroll
                for (int nt = 0; nt < 16; ++nt) {
                    const int64_t col = n0 + 8 * nt + 2 * lr;
                    const int64_t e = row * npair + col;
                    if (col + 1 < npair && !(e & 1)) {
                        *reinterpret_cast<double2 *>(T + e) = make_double2(acc[mt][nt][0], acc[mt][nt][1]);
                    } else {
                        if (col < npair) T[e] = acc[mt][nt][0];
                        if (col + 1 < npair) T[e + 1] = acc[mt][nt][1];
                    }
                }
            }
        }
    }
}

}  // namespace

void launch_fp64_tile_gemm(const double *A, int64_t lda, const double *Bop, int64_t sbk, int64_t sbn,
                           double *C, int64_t ldc, int64_t Mr, int64_t Nc, int64_t Kd, double alpha,
                           double beta, int lower_only, cudaStream_t st)
{
    small_gemm(A, lda, Bop, sbk, sbn, C, ldc, Mr, Nc, Kd, alpha, beta, lower_only, st);
}

int64_t build_b_workspace_doubles(int64_t naux)
{
    const int64_t ldw = (naux + NB - 1) / NB * NB;
    return ldw * ldw + ldw * NB;                       /* Aw + panel scratch */
}

/* Enqueue Eq. 2-3 on `st`.  M: naux x naux (lower triangle read, overwritten by L); T: packed
 * R in, B out; ws: build_b_workspace_doubles(naux) doubles; info: device flag or NULL. */
cudaError_t launch_build_b(int64_t naux, int64_t npair, double *M, double *T, double *ws,
                           long long *info, cudaStream_t st)
{
    static std::atomic<unsigned long long> ok1{0}, ok2{0}, ok3{0};
    cudaError_t e = ensure_dynamic_smem(chol_diag_kernel, NB * (NB + 1) * 8, ok1);
    if (e == cudaSuccess) e = ensure_dynamic_smem(tri_inv_kernel, NB * NB * 8, ok2);
    if (e == cudaSuccess) e = ensure_dynamic_smem(whiten_gemm_kernel, W_SMEM_BYTES, ok3);
    if (e != cudaSuccess) return e;
    const int64_t ldw = (naux + NB - 1) / NB * NB;
    double *Aw = ws, *panel = ws + ldw * ldw;
    e = cudaMemsetAsync(Aw, 0, (size_t)(ldw * ldw) * sizeof(double), st);
    if (e != cudaSuccess) return e;
    if (info) {
        e = cudaMemsetAsync(info, 0, sizeof(long long), st);
        if (e != cudaSuccess) return e;
    }
    /* ---- phase 1: Cholesky of M, diagonal-block inverses, the operator Aw */
    for (int64_t r0 = 0; r0 < naux; r0 += NB) {
        const int n = (int)((naux - r0 < NB) ? naux - r0 : NB);
        const int64_t r1 = r0 + n, below = naux - r1;
        chol_diag_kernel<<<1, 256, NB * (NB + 1) * 8, st>>>(M, naux, r0, n, info);
        tri_inv_kernel<<<1, NB, NB * NB * 8, st>>>(M, naux, r0, n, Aw, ldw);
        double *Linv = Aw + r0 * ldw + r0;
        /* Aw[r0.., 0..r0) = -Linv . L[r0.., 0..r0) */
        small_gemm(Linv, ldw, M + r0 * naux, naux, 1, Aw + r0 * ldw, ldw, n, r0, n, -1.0, 0.0, 0, st);
        if (below > 0) {
            /* panel: L[r1.., r0..r1) = M[r1.., r0..r1) . Linv^T  (through scratch: not in place) */
            small_gemm(M + r1 * naux + r0, naux, Linv, 1, ldw, panel, NB, below, n, n, 1.0, 0.0, 0, st);
            e = cudaMemcpy2DAsync(M + r1 * naux + r0, (size_t)naux * 8, panel, (size_t)NB * 8,
                                  (size_t)n * 8, (size_t)below, cudaMemcpyDeviceToDevice, st);
            if (e != cudaSuccess) return e;
            /* trailing: M[r1.., r1..) -= L[r1.., r0..r1) . L[r1.., r0..r1)^T, lower triangle */
            small_gemm(M + r1 * naux + r0, naux, M + r1 * naux + r0, 1, naux, M + r1 * naux + r1, naux,
                       below, below, n, -1.0, 1.0, 1, st);
        }
    }
    /* ---- phase 2: B_i = Aw[i] . [B_<i ; R_i], block row by block row, in place */
    const unsigned ntile = (unsigned)((npair + NB - 1) / NB);
    for (int64_t r0 = 0; r0 < naux; r0 += NB) {
        const int64_t n = (naux - r0 < NB) ? naux - r0 : NB;
        whiten_gemm_kernel<<<ntile, W_THREADS, W_SMEM_BYTES, st>>>(T, naux, npair, Aw, ldw, r0, r0 + n);
    }
    return cudaGetLastError();
}

}  // namespace dfjk
