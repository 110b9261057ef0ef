/*
 * dfjk_internal.h -- launcher prototypes shared by the translation units of
 * libdfjk.so (CUDA path only; nothing here is used by, or uses, oracle/).
 *
 * Notation follows include/dfjk.h: B packed [naux][npair], C [nao][nocc],
 * Dt = D-tilde (packed density with doubled off-diagonals), d[naux],
 * X = half-transformed tensor, K lower tiles.
 */
#ifndef DFJK_INTERNAL_H
#define DFJK_INTERNAL_H

#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

namespace dfjk {

/* ---------------------------------------------------------------- J path */

/* J0: Dt[mu(mu+1)/2+nu] = (2 - delta_mu,nu) * sum_s w_s sum_i C_s[mu,i] C_s[nu,i].
 * Ccat4 is the zero-padded, k-group-major concatenation built by k0_pack_c (see K0), set s
 * occupying columns [col0[s], col0[s]+nocc[s]). */
void launch_j0_build_dt(const double *Ccat, int64_t ldc, int64_t nao,
                        int nset, const int *col0, const int *nocc, const double *w,
                        double *Dt, cudaStream_t st);

/* J0 for a general density: Dt[mu(mu+1)/2+nu] = dm[mu][nu] + (mu != nu) dm[nu][mu] where dm is either
 * given (C2 == NULL, C1 = dm, nao x nao row-major) or the product C1 C2^T of two nao x ncol factors. */
void launch_j0_general_dt(const double *C1, const double *C2, int64_t ncol, int64_t nao, double *Dt,
                          cudaStream_t st);

/* J1: d_part[c][P] = sum_{pair in chunk c} B[P][pair] Dt[pair];  nchunk = j1_num_chunks(npair). */
int64_t j1_num_chunks(int64_t npair);
void launch_j1_dot(const double *B, int64_t naux, int64_t npair, const double *Dt,
                   double *d_part, int sm_count, cudaStream_t st);
/* J1X: d_part[b][P0 + p] = block b's share of sum_s w_s <X_P^s, C_s> for the np rows of the X chunk
 * K1 has just written (= <B_P, sum_s w_s C_s C_s^T>: d_P without streaming B; used when K is built in
 * the same call).  b < j1x_num_blocks(nao, ldc); J1R adds the blocks.  c_shift (columns, multiple of
 * 4): the C block of X column c is Ccat column c + c_shift -- 0 for C C^T densities, the width of C1
 * for the pair form, where d_P = <B_P C1, C2>. */
int64_t j1x_num_blocks(int64_t nao, int64_t ldc);
int64_t j1x_max_blocks(int64_t nao, int64_t ldc_max);   /* >= j1x_num_blocks(nao, ldc) for every ldc <= ldc_max */
void launch_j1x_dot(const double *X4, const double *Ccat4, int64_t nao, int64_t np, int64_t ldx, int64_t ldc,
                    int64_t c_shift, int nset, const int *col0, const int *nocc, const double *w, int64_t P0,
                    int64_t naux, double *d_part, cudaStream_t st);
/* J1b: d[P] = sum_c d_part[c][P] (fixed order: deterministic). */
void launch_j1_reduce(const double *d_part, int64_t nchunk, int64_t naux, double *d,
                      cudaStream_t st);

/* J2: Jp_part[g][pair] = sum_{P in row group g} d[P] B[P][pair];  ngroup = j2_num_groups(...).
 * d == NULL: the same stream with every element weighted by itself, sum_P B[P][pair]^2 (Eq. 7). */
int64_t j2_num_groups(int64_t naux, int64_t npair, int sm_count);
void launch_j2_axpy(const double *B, int64_t naux, int64_t npair, const double *d,
                    double *Jp_part, int64_t ngroup, cudaStream_t st);

/* J3: J[mu][nu] = J[nu][mu] = sum_g Jp_part[g][mu(mu+1)/2+nu]. */
/* Jslot != NULL: the kernel writes to *Jslot (a device-resident pointer published by K0) instead of J */
void launch_j3_unpack(const double *Jp_part, int64_t ngroup, int64_t npair, int64_t nao,
                      double *J, double *const *Jslot, cudaStream_t st);

/* ---------------------------------------------------------------- K path */

/* K0: the zero-padded concatenation [C_0 | C_1 | ...] (every set padded to a multiple of 8
 * columns, ldc columns in total) in k-group-major layout
 *   Ccat4[(mu/4)*ldc*4 + c*4 + mu%4],  mu < round_up(nao, 32) (rows >= nao are zero). */
#define DFJK_OUT_SLOTS 4
/* outs != NULL: the kernel also copies the DFJK_OUT_SLOTS output pointers outs[] (J, K_0, K_1, ...) of
 * this call to the device array out_slots, where K3 / J3 of a captured launch sequence find them. */
void launch_k0_pack_c(const double *const *C, const int *nocc, const int *col0, int nset,
                      int64_t nao, int64_t ldc, double *Ccat, double *const *outs, double **out_slots,
                      cudaStream_t st);

/* K1: for P in [P0, P0+np), k = (P-P0)*ldc + i:
 *   X4[(k/4)*nao*4 + mu*4 + k%4] = sum_nu B_P(mu,nu) Ccat[nu][i]      (k-group-major X)
 * with k = (P-P0)*ldx + i: ldx >= ldc is X's row pitch (ldx > ldc leaves room for K1U's columns). */
cudaError_t launch_k1_half_transform(const double *B, int64_t naux, int64_t nao, int64_t npair,
                                     int64_t P0, int64_t np, const double *Ccat4, int64_t ldc, int64_t ldx,
                                     double *X4, cudaStream_t st);

/* K1U: X4 columns [col0, col0 + round_up(nao,4)) of the chunk = B_P unpacked (X_P = B_P . I). */
void launch_k1u_unpack(const double *B, int64_t nao, int64_t npair, int64_t P0, int64_t np, int64_t ldx,
                       int64_t col0, double *X4, cudaStream_t st);

/* K2: Kpart[split][mu][nu] (+)= sum_{k in split's share} X[mu][k] X[nu][k]
 * for mu-tile >= nu-tile (lower 128x128 tiles).  The set uses k = p*ldc + [col0, col0+round_up(ncol,4)),
 * p < np: K2's MMA k step is 4, so the 8-padding columns of Ccat beyond that are never read.  accumulate = 0 overwrites. */
cudaError_t launch_k2_syrk_lower(const double *X4, int64_t nao, int64_t np, int64_t ldc, int64_t col0,
                                 int64_t ncol, double *Kpart, int nsplit, int weighted, int accumulate,
                                 cudaStream_t st);

/* K2 general: Kpart[split][mu][nu] (+)= sum_k X[mu][k_a] X[nu][k_b] over ALL tiles, with
 * k_a = p*ldc + col0a + j, k_b = p*ldc + col0b + j, j < round_up(ncol,4): the product
 * sum_P (B_P C1)(B_P C2)^T of two column ranges of the same X chunk (not symmetric). */
cudaError_t launch_k2_gemm_full(const double *X4, int64_t nao, int64_t np, int64_t ldc, int64_t col0a,
                                int64_t col0b, int64_t ncol, double *Kpart, int nsplit, int accumulate,
                                cudaStream_t st);

/* K2P: the same two products, panel-synchronous (k2_syrk.cu, k2p_kernel): the k range of the chunk is
 * cut into npanel panels, items (panel, tile) are dealt dynamically to one persistent CTA per SM and
 * added into slab (panel % nslab) of Kpart in panel order.  k2p_plan picks npanel / nslab from the
 * shape of the build's FIRST chunk (ng = np * ceil(ncol / 4) k-groups, ntile tiles, panel_bytes of X
 * per panel) as a panel length in stages of k = 32; every chunk is then cut at that length.  `work` is a
 * device array of 1 + nslab * ntile ints (zeroed by the launcher).  The slab count must be the same
 * for every chunk of a build (accumulate != 0 continues the slabs of the previous chunk). */
void k2p_plan(int64_t nao, int64_t ng, int ntile, int sm_count, int max_slabs, int64_t panel_bytes,
              int *panel_stages, int *nslab);
cudaError_t launch_k2p_syrk_lower(const double *X4, int64_t nao, int64_t np, int64_t ldc, int64_t col0,
                                  int64_t ncol, double *Kpart, int panel_stages, int nslab, int accumulate,
                                  int *work, int sm_count, cudaStream_t st);
cudaError_t launch_k2p_gemm_full(const double *X4, int64_t nao, int64_t np, int64_t ldc, int64_t col0a,
                                 int64_t col0b, int64_t ncol, double *Kpart, int panel_stages, int nslab,
                                 int accumulate, int *work, int sm_count, cudaStream_t st);

/* K3 general: K[mu][nu] = sum_split Kpart[split][mu][nu] for every (mu, nu). */
/* accumulate != 0: K[mu][nu] += the sum (the batched build adds one X chunk after the other) */
void launch_k3_sum(const double *Kpart, int nsplit, int64_t nao, double *K, cudaStream_t st, int accumulate = 0);

/* ---------------------------------------------------------------- batched densities (dfjk_get_jk_pairs) */
#define DFJK_MAX_BATCH 8   /* densities per multi-right-hand-side J2 pass / per d_batch workspace */
/* one factor C (nao x ncol) into columns [col0, col0 + width) of Ccat4 (zero beyond ncol) */
void launch_k0_pack_cols(const double *C, int64_t ncol, int64_t col0, int64_t width, int64_t nao, int64_t ldc,
                         double *Ccat, cudaStream_t st);
/* d_out[P0 + p] = sum_c d_part[c][P0 + p], p < np (J1R for the rows of one X chunk) */
void launch_j1_reduce_rows(const double *d_part, int64_t nchunk, int64_t naux, int64_t P0, int64_t np,
                           double *d_out, cudaStream_t st);
/* J2 for nbatch <= DFJK_MAX_BATCH densities in one pass over B: d[k][P] (pitch naux),
 * Jp_part[(k*ngroup + g)][pair]; per density bitwise equal to launch_j2_axpy */
void launch_j2_axpy_multi(const double *B, int64_t naux, int64_t npair, const double *d, int nbatch,
                          double *Jp_part, int64_t ngroup, cudaStream_t st);

/* K3: K[mu][nu] = K[nu][mu] = sum_split Kpart[split][mu][nu], mu >= nu. */
void launch_k3_finish(const double *Kpart, int nsplit, int weighted, int64_t nao, double *K, double *const *Kslot,
                      cudaStream_t st);

/* ---------------------------------------------------------------- building B (Eq. 2-3) */

/* Workspace (doubles) and launch sequence of dfjk_build_b: M = L L^T in place (lower triangle),
 * T (packed R, naux x npair) overwritten by B = L^-1 R.  info: device flag (0 ok, j+1 = first
 * non-positive pivot) or NULL. */
int64_t build_b_workspace_doubles(int64_t naux);
cudaError_t launch_build_b(int64_t naux, int64_t npair, double *M, double *T, double *ws,
                           long long *info, cudaStream_t st);

/* FP64-pipe probe (register-only DMMA.8x8x4 loop): flops of one launch, and the launch. */
double fp64_peak_probe_flops(int ctas, int iters);
void launch_fp64_peak_probe(int ctas, int iters, double *sink, cudaStream_t st);

/* Plain FP64 FMA tile product for the small dense steps around the hot kernels (Cholesky panels,
 * SCF driver):  C[m][n] = beta C[m][n] + alpha sum_k A[m*lda + k] * Bop[k*sbk + n*sbn],
 * m < Mr, n < Nc, k < Kd; (sbk, sbn) = (ldb, 1) is A.B, (1, ldb) is A.B^T. */
void launch_fp64_tile_gemm(const double *A, int64_t lda, const double *Bop, int64_t sbk, int64_t sbn,
                           double *C, int64_t ldc, int64_t Mr, int64_t Nc, int64_t Kd, double alpha,
                           double beta, int lower_only, cudaStream_t st);

}  // namespace dfjk

/* ---------------------------------------------------------------- error text */
namespace dfjk {
/* printf-style: stores the calling thread's dfjk_last_error() text and returns `code` */
int set_last_error(int code, const char *fmt, ...);
}  // namespace dfjk

/* ---------------------------------------------------------------- SCF driver (scf_rhf.cu) */
struct dfjk_handle;
namespace dfjk {
/* what the SCF driver borrows from the handle (dfjk_api.cu): the X workspace and the partial-K slots
 * (idle between two get_jk calls) for its own DMMA products, and where it leaves its timing */
struct ScfWorkspace { double *X; int64_t x_doubles; double *Kpart; int nsplit_alloc; int sm_count; };
ScfWorkspace scf_workspace(dfjk_handle *h);
void scf_store_timing(dfjk_handle *h, int64_t iters, double get_jk_ms, double eig_ms, double total_ms);
/* split count that fills sm_count SMs best with ntile * s equal work items (dfjk_api.cu) */
int choose_splits(int ntile, int sm_count, int max_splits);
/* split count (of a full off-diagonal tile) of the lower-triangle split kernel, whose tiles get
 * splits in proportion to their cost (k2_tile_splits); k2_lower_items counts the CTAs that do work */
int choose_splits_lower(int64_t nao, int sm_count, int max_splits);
int64_t k2_lower_items(int64_t nao, int nsplit);
/* nspin = 1: restricted (get_jk), nspin = 2: unrestricted (get_jk_u); per-spin arguments are arrays */
int scf_run(dfjk_handle *h, int64_t nao, int nspin, const double *hcore, const double *S,
            const int64_t *nocc, int64_t max_iter, double conv_tol, int64_t diis_space,
            double *const *C_out, double *const *mo_energy_out, double *const *D_out,
            double *const *F_out, double *e_hist, int64_t *n_iter, int *converged, cudaStream_t st,
            char *err, size_t errlen);
}  // namespace dfjk
#endif
