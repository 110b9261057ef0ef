/*
 * dfjk.h -- C ABI of the B200-native density-fitted Coulomb/exchange build.
 *
 * The operation (what the paper calls  jmat, kmat = get_jk(mol, dm),
 * PAPER.md:96 and PAPER.md:126-131, Sec. II.C / III) with the two-electron
 * integrals density-fitted (Sec. IV.C.2, Eq. 1-3):
 *
 *     (mu nu|kappa lambda) ~= sum_P T_{P,mu nu} T_{P,kappa lambda}            Eq. 1
 *
 * T is the Cholesky-whitened 3-centre tensor (Eq. 2-3); it is called B here and
 * is symmetric in (mu,nu), stored as a packed lower triangle (aosym='s2',
 * PAPER.md:669; tril order PAPER.md:726).  Inserting Eq. 1 into the textbook
 * J_mn = sum_ls (mn|ls) D_ls and K_mn = sum_ls (ml|ns) D_ls gives what this
 * library computes (BASELINE.json north_star):
 *
 *     D     = sum_s w_s C_s C_s^T         restricted: one set, w = 2  (D = 2 C C^T)
 *                                         unrestricted: two sets, w = 1 each
 *     d_P   = sum_{mu,nu} B_P[mu,nu] D[mu,nu]
 *     J     = sum_P d_P B_P
 *     X_P   = B_P C_s
 *     K_s   = sum_P X_P X_P^T             NO factor 2  (reading R1)
 *
 * Conventions common to every entry point
 *   - All arithmetic is IEEE binary64.  All arrays are C order (row-major),
 *     contiguous, with 64-bit element offsets.
 *   - "DEVICE" pointers live on the CUDA device that was current when
 *     dfjk_create() ran; "HOST" pointers are ordinary host memory (pinned memory
 *     makes the copies asynchronous, pageable memory is accepted).
 *   - Return value: 0 (DFJK_OK) on success, a negative DFJK_E* code on failure;
 *     dfjk_last_error() then returns a thread-local message.  No exception and
 *     no signal crosses this boundary.  There is NO CPU fallback: without a
 *     CUDA device every compute entry point fails with DFJK_ECUDA.
 *   - The device entry points only ENQUEUE work on `stream` (a cudaStream_t
 *     passed as void*; NULL = the legacy default stream).  They never
 *     synchronise the host and never allocate.  Outputs are valid once the
 *     stream reaches that point.  Calls on one handle share its workspace and
 *     must therefore be stream-ordered with respect to each other.
 */
#ifndef DFJK_H
#define DFJK_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DFJK_OK       0
#define DFJK_EINVAL  -1   /* bad argument: null pointer, size out of range, misaligned B */
#define DFJK_ENOMEM  -2   /* device or host allocation failed */
#define DFJK_ECUDA   -3   /* CUDA runtime / launch error (text in dfjk_last_error) */

typedef struct dfjk_handle dfjk_handle;

/*
 * dfjk_create -- bind a resident DF tensor and allocate the fixed workspace.
 *
 *   naux      number of auxiliary functions P (rows of B), >= 1
 *   nao       number of orbital basis functions, 1 <= nao <= 32640;  npair = nao*(nao+1)/2
 *   B_packed  DEVICE, naux*npair doubles:  B_packed[P*npair + mu*(mu+1)/2 + nu], mu >= nu
 *             (Eq. 1's T_{P,mu nu}; row-major lower triangle, R3/R4).
 *             BORROWED: never copied, never written, must stay valid and unchanged
 *             until dfjk_destroy (it is up to 96 GB).  Must be 16-byte aligned.
 *
 * Returns the handle, or NULL on failure (dfjk_last_error says why).
 * Workspace (at most ~3 GB: a 2 GB chunk of the half-transformed tensor plus the partial-K
 * slots; independent of naux*npair) is allocated
 * here with cudaMalloc and freed by dfjk_destroy; get_jk never allocates.
 */
dfjk_handle *dfjk_create(int64_t naux, int64_t nao, const double *B_packed);

/*
 * dfjk_get_jk -- restricted build, D = 2 C_occ C_occ^T  (north_star).
 *
 *   C_occ   DEVICE, nao x nocc, C_occ[mu*nocc + i];  1 <= nocc <= nao.  Need not be
 *           orthonormal (R8).  Read only.
 *   J       DEVICE, nao x nao, OVERWRITTEN, both triangles written.  NULL skips J.
 *   K       DEVICE, nao x nao, OVERWRITTEN, both triangles written.  NULL skips K.
 *           J == NULL and K == NULL together is DFJK_EINVAL.
 *   stream  cudaStream_t
 */
int dfjk_get_jk(dfjk_handle *h, const double *C_occ, int64_t nocc,
                double *J, double *K, void *stream);

/*
 * dfjk_get_jk_u -- unrestricted (two-spin) build (UKS usage PAPER.md:172-180;
 * BASELINE.json config 5; R7):  D_s = C_s C_s^T (weight 1),
 *     J   = J[D_a + D_b]     formed in ONE pair of passes over B
 *     K_s = sum_P (B_P C_s)(B_P C_s)^T,  s = a, b   (B is unpacked once for both)
 *   C_a (nao x nocc_a), C_b (nao x nocc_b): DEVICE, as C_occ above.
 *   J, K_a, K_b: DEVICE nao x nao, overwritten; any may be NULL, not all three.
 */
int dfjk_get_jk_u(dfjk_handle *h, const double *C_a, int64_t nocc_a,
                  const double *C_b, int64_t nocc_b,
                  double *J, double *K_a, double *K_b, void *stream);

/*
 * General densities.  PAPER.md:96: get_jk "supports an
 * arbitrary number of density matrices"; the DF-approximated
 * orbital Hessian of SOSCF contracts Eq. 1's integrals with response densities that are
 * neither idempotent nor symmetric.  For ANY real nao x nao matrix dm, with Eq. 1:
 *
 *     J[dm] = sum_P B_P <B_P, dm>          (only dm + dm^T matters; J is symmetric)
 *     K[dm] = sum_P B_P dm B_P             (K[dm^T] = K[dm]^T; not symmetric in general)
 *
 * Both are LINEAR in dm (PySCF's vj, vk).  Relation to dfjk_get_jk: its J is J[2 C C^T]
 * and its K is K[C C^T] (no factor 2, R1).
 *
 * dfjk_get_jk_pair -- dm = C1 C2^T given by its factors (the usual form of a response
 * density, e.g. C_occ and the rotated orbitals C_vir kappa):
 *     K = sum_P (B_P C1)(B_P C2)^T        one half transform over [C1|C2], then a
 *                                          full (non-symmetric) DMMA product
 *   C1, C2  DEVICE, nao x ncol row-major, 1 <= ncol <= nao (any dm has such a factorisation).
 *   J, K    DEVICE, nao x nao, OVERWRITTEN; either may be NULL, not both.
 */
int dfjk_get_jk_pair(dfjk_handle *h, const double *C1, const double *C2, int64_t ncol,
                     double *J, double *K, void *stream);

/*
 * dfjk_get_jk_dm -- the same for a raw density matrix (no factorisation needed):
 *   dm      DEVICE, nao x nao row-major, any real matrix.
 * K is built as the pair (dm, I): X_P = B_P dm by the half transform, B_P itself unpacked
 * beside it, then K = sum_P X_P B_P^T as a full DMMA product.  Cost 4 naux nao^3 flop: prefer
 * dfjk_get_jk / dfjk_get_jk_pair whenever factors with few columns are known.
 */
int dfjk_get_jk_dm(dfjk_handle *h, const double *dm, double *J, double *K, void *stream);

/*
 * dfjk_get_jk_pairs -- several factored densities dm_i = C1_i C2_i^T, i < nbatch, from ONE sweep over B
 * ("an arbitrary number of density matrices"; the batches of Hessian x trial-vector
 * products of SOSCF).  Per density the results are those of dfjk_get_jk_pair:
 *     J_i = sum_P B_P <B_P, C1_i C2_i^T>        K_i = sum_P (B_P C1_i)(B_P C2_i)^T
 * How B is shared: the factors of as many pairs as fit 2 round_up(nao, 8) columns are packed side by side
 * and half-transformed by ONE K1 launch per X chunk (the packed triangle is read and unpacked once for
 * all of them -- with few columns per pair K1 is bound by exactly that); each pair's d_P is read off its
 * columns of X and its product added to K_i chunk by chunk; all J_i of up to 8 densities come out of ONE
 * axpy pass over B (every loaded element feeds 8 FMAs).  Larger batches are cut into sub-batches of 8.
 *   C1s, C2s  HOST arrays of nbatch DEVICE pointers, factor i is nao x ncols[i] row-major
 *   ncols     HOST array of nbatch column counts, 1 <= ncols[i] <= nao (they may differ)
 *   Js, Ks    HOST arrays of nbatch DEVICE pointers to nao x nao outputs (OVERWRITTEN); either ARRAY may
 *             be NULL (skip all J / all K), not both; an array that is given has no NULL entry.
 *             With Ks == NULL (or option "j_fused" = 0) every d_i costs its own dot pass over B; the
 *             axpy pass is still shared.
 * With d from the dot pass J_i is bitwise what dfjk_get_jk_pair gives (the shared axpy pass adds in the
 * same order per density); read off X, d_P is summed over other column blocks than in a single-pair call,
 * and K_i adds its X chunks in another order: deterministic, a different rounding.  dfjk_get_d is not
 * updated by batched calls.
 */
int dfjk_get_jk_pairs(dfjk_handle *h, int64_t nbatch, const double *const *C1s,
                      const double *const *C2s, const int64_t *ncols, double *const *Js,
                      double *const *Ks, void *stream);

/*
 * dfjk_get_jk_dms -- the same for raw density matrices:
 *   dms     DEVICE, ndm x nao x nao;  Js, Ks  DEVICE, ndm x nao x nao (either may be NULL, not both).
 * Results per density as dfjk_get_jk_dm.  The J_i of up to 8 densities share ONE axpy pass over B
 * (ndm + 1 streaming passes instead of 2 ndm); K_i is built per density as the pair (dm_i, I), which is
 * bound by its 4 naux nao^3 flop, not by B.
 */
int dfjk_get_jk_dms(dfjk_handle *h, int64_t ndm, const double *dms, double *Js, double *Ks,
                    void *stream);

/*
 * dfjk_get_jk_host -- the same restricted build for a caller whose orbitals and
 * results live in HOST memory (the end-to-end call bench.py times):
 * copies C_occ host->device, runs dfjk_get_jk on an internal stream, copies J and
 * K device->host and SYNCHRONISES before returning.  B stays resident on the device.
 *   C_occ_host  HOST nao x nocc;  J_host, K_host  HOST nao x nao (either may be NULL).
 */
int dfjk_get_jk_host(dfjk_handle *h, const double *C_occ_host, int64_t nocc,
                     double *J_host, double *K_host);

/*
 * dfjk_scf_rhf -- a closed-shell DF-SCF driver around dfjk_get_jk.
 * The paper gives the loop in words (Fock build -> diagonalisation -> new density, DIIS by
 * default: PAPER.md:258-262; mf.kernel(dm0): PAPER.md:154-159); written out (Roothaan-Hall + Pulay
 * DIIS):
 *     core guess  hcore C = S C eps;   then per iteration k = 0, 1, ...
 *     C_occ = nocc lowest orbitals;  J, K = get_jk(C_occ);  F = hcore + J - K
 *     E_k = 1/2 sum D o (hcore + F), D = 2 C_occ C_occ^T;   e = F D S - S D F
 *     stop when k > 0, |E_k - E_{k-1}| <= conv_tol max(1, |E_k|) and max|e| <= sqrt(conv_tol)
 *     DIIS over the last diis_space (F, e) pairs;  F_ext C = S C eps
 *   hcore, S   DEVICE nao x nao, symmetric (S positive definite); read only
 *   nocc       doubly occupied orbitals, 1 <= nocc <= nao;  max_iter >= 1;  1 <= diis_space <= 16
 *   C          DEVICE nao x nao OUT, C[mu*nao + i], orbitals of the last diagonalisation (C^T S C = 1)
 *   mo_energy  DEVICE nao OUT or NULL;  D, F  DEVICE nao x nao OUT or NULL (density and Fock matrix of
 *              the last energy evaluation)
 *   e_hist     HOST max_iter doubles OUT (E_k);  n_iter, converged  HOST OUT
 * SYNCHRONOUS: the host reads E and max|e| back every iteration.  Allocates its workspace
 * (about (9 + 2 diis_space) nao^2 doubles) for the duration of the call.  Every step runs in this
 * library's kernels except the generalised symmetric eigenproblem, which is cuSOLVER's Dsygvd
 * (loaded with dlopen at the first call; DFJK_ECUDA if libcusolver is not available).
 */
int dfjk_scf_rhf(dfjk_handle *h, const double *hcore, const double *S, int64_t nocc,
                 int64_t max_iter, double conv_tol, int64_t diis_space, double *C,
                 double *mo_energy, double *D, double *F, double *e_hist, int64_t *n_iter,
                 int *converged, void *stream);

/*
 * dfjk_scf_uhf -- the unrestricted (two-spin) counterpart of dfjk_scf_rhf around dfjk_get_jk_u (the
 * paper's UKS/UHF objects): Pople-Nesbet equations,
 *     D_s = C_s,occ C_s,occ^T;  J = J[D_a + D_b];  K_s = K[D_s];  F_s = hcore + J - K_s
 *     E = 1/2 sum_s sum D_s o (hcore + F_s);  e_s = F_s D_s S - S D_s F_s
 * one DIIS over both spin blocks (B_ij = <e_a^i, e_a^j> + <e_b^i, e_b^j>), both spins started from the
 * core guess, the same stopping rule (max over both spins of max|e_s|).
 *   C_a, C_b             DEVICE nao x nao OUT;  mo_energy_a/b  DEVICE nao OUT or NULL
 *   D_a, D_b             DEVICE nao x nao OUT or NULL (weight-1 spin densities)
 *   other arguments as in dfjk_scf_rhf.  SYNCHRONOUS.
 */
int dfjk_scf_uhf(dfjk_handle *h, const double *hcore, const double *S, int64_t nocc_a,
                 int64_t nocc_b, int64_t max_iter, double conv_tol, int64_t diis_space,
                 double *C_a, double *C_b, double *mo_energy_a, double *mo_energy_b,
                 double *D_a, double *D_b, double *e_hist, int64_t *n_iter, int *converged,
                 void *stream);

/*
 * dfjk_build_b -- build the whitened tensor on the device,
 * PAPER.md:353-356, Eq. 2-3:
 *     M_PQ = (chi_P|chi_Q) = L L^T                              Eq. 2
 *     T_{P,mu nu} = sum_Q (L^-1)_{PQ} (chi_Q|mu nu)             Eq. 3      (T is this library's B)
 *
 *   naux, nao  as in dfjk_create;  npair = nao*(nao+1)/2
 *   M          DEVICE, naux x naux row-major, symmetric positive definite.  Only the lower
 *              triangle is read.  OVERWRITTEN: on exit the lower triangle holds L; the strict
 *              upper triangle is left as it was, except inside the 128 x 128 diagonal blocks,
 *              where it is zeroed.  16-byte aligned.
 *   R_packed   DEVICE, naux x npair, the raw 3-centre tensor (Q|mu nu), packed like B_packed.
 *              OVERWRITTEN IN PLACE by B = L^-1 R (the tensor is up to 96 GB: no second copy).
 *              16-byte aligned.  Pass the result to dfjk_create.
 *   info       DEVICE int64 flag or NULL: 0 on success, j+1 if pivot j of the Cholesky
 *              factorisation was not positive (LAPACK's convention; B is then garbage).
 *   stream     cudaStream_t; the call only enqueues (workspace of ~naux^2 doubles comes from
 *              the stream-ordered allocator, cudaMallocAsync / cudaFreeAsync).
 *
 * Cost: naux^2 npair flop for the solve (3.2e13 at naux=5000, nao=1600; FP64 DMMA, in place,
 * block row by block row) + naux^3/3 for the factorisation.  The integrals (chi_P|chi_Q) and
 * (chi_Q|mu nu) themselves need an integral engine and are inputs here.
 */
int dfjk_build_b(int64_t naux, int64_t nao, double *M, double *R_packed, int64_t *info,
                 void *stream);

/*
 * dfjk_get_df_diag -- the DF term of the diagonal-error diagnostic, Eq. 7:
 *     diag[mu][nu] = (mu nu|mu nu)_DF = sum_P T_{P,mu nu}^2
 * (Delta of Eq. 7 is sum_{mu nu} [(mu nu|mu nu)_exact - diag[mu][nu]]; the exact integrals
 * need an integral engine and are outside this library).  One streaming pass over B
 * (HBM-bound, |B| bytes), same kernel as J2 with each element weighted by itself.
 *   diag    DEVICE, nao x nao, OVERWRITTEN, both triangles written.
 */
int dfjk_get_df_diag(dfjk_handle *h, double *diag, void *stream);

/*
 * dfjk_df_diag_noalloc -- the same Eq. 7 diagonal as dfjk_get_df_diag,
 *     diag[mu][nu] = sum_P T_{P,mu nu}^2,
 * WITHOUT a handle and without a single device allocation, for callers that cannot allocate:
 * code running inside a framework whose caching allocator already owns the device (a stray
 * cudaMalloc there fails or fragments the pool), code bound by a "no allocation after start-up"
 * rule (cudaMalloc / cudaFree synchronise the whole device and would stall a serving or
 * real-time loop), and processes that have given every free byte of HBM to B itself.  Such
 * callers cannot use dfjk_create, whose workspace comes from cudaMalloc.
 *
 *   naux, nao  as in dfjk_create, with nao <= DFJK_NOALLOC_MAX_NAO (= dfjk_noalloc_max_nao());
 *              naux is not limited.  A larger nao is DFJK_EINVAL with a message naming the limit.
 *   B_packed   DEVICE, naux*npair doubles, packed as in dfjk_create, 16-byte aligned, read only.
 *   diag       DEVICE, nao x nao, OVERWRITTEN, both triangles written.
 *   stream     cudaStream_t; the call only enqueues two kernels (the J2 stream with every element
 *              weighted by itself, then the J3 unpack) and returns.
 *
 * Scratch: the per-row-group partial triangles that the handle keeps in its workspace live here in
 * a fixed array of DFJK_NOALLOC_SCRATCH_BYTES inside the library image; every GPU that loads
 * libdfjk.so holds it until the process exits.  The call uses cudaMalloc, cudaFree or an
 * allocating library routine nowhere.  Consequences the caller has to know:
 *   - The FIRST call on each device looks up the array's device address (cudaGetSymbolAddress)
 *     and the SM count, with that device current; make that first call during start-up, before
 *     any stream capture begins.  Later calls on the device reuse the cached values.
 *   - All calls on a device share the one array, which simply keeps what the last call wrote.
 *     Nothing in it needs to be zero at entry (each call overwrites every partial it later
 *     reads), so calls of different sizes may follow each other freely -- but two calls whose
 *     kernels can run at the same time on the GPU (different streams without an event between
 *     them, or two host threads) RACE on it and give garbage.  Order them on one stream or with
 *     events.  Handle-based calls are unaffected: they never touch this array.
 *   - With fewer row groups than the handle path would choose when the array is the limit
 *     (nao > ~500), the additions happen in another order: results agree with dfjk_get_df_diag to
 *     rounding (the library's 1e-11 relative Frobenius bar), not necessarily bit for bit.
 */
#define DFJK_NOALLOC_SCRATCH_BYTES 8388608   /* 8 MiB = 1048576 doubles */
#define DFJK_NOALLOC_MAX_NAO       1023      /* 2 * npair = nao (nao + 1) <= 1048576 */
int dfjk_df_diag_noalloc(int64_t naux, int64_t nao, const double *B_packed, double *diag,
                         void *stream);
/* the largest nao dfjk_df_diag_noalloc accepts (DFJK_NOALLOC_MAX_NAO of the loaded library) */
int64_t dfjk_noalloc_max_nao(void);

/*
 * dfjk_get_jk_u_host -- the unrestricted build (dfjk_get_jk_u) for HOST orbitals and results, with the
 * same copy-in / run / copy-out / synchronise sequence as dfjk_get_jk_host.
 *   C_a_host (nao x nocc_a), C_b_host (nao x nocc_b): HOST;  J_host, K_a_host, K_b_host: HOST nao x nao,
 *   any may be NULL, not all three.
 */
int dfjk_get_jk_u_host(dfjk_handle *h, const double *C_a_host, int64_t nocc_a,
                       const double *C_b_host, int64_t nocc_b,
                       double *J_host, double *K_a_host, double *K_b_host);

/*
 * dfjk_get_d -- debug/inspection getter: copies the naux fitting coefficients
 * d_P of the most recent J build on this handle into d_out (DEVICE, naux doubles),
 * enqueued on `stream`.  DFJK_EINVAL if no J has been built yet.
 */
int dfjk_get_d(dfjk_handle *h, double *d_out, void *stream);

/*
 * dfjk_set_option -- tuning knobs, for benchmarks and tests only.  Unknown names
 * return DFJK_EINVAL.  Known names:
 *   "k_chunk"   number of auxiliary rows whose half-transformed X stays in the
 *               L2-sized workspace between the K1 and K2 kernels (0 = automatic)
 *   "k_splits"  number of partial-K accumulators the SYRK is split over / the largest number of
 *               slabs the panel-synchronous kernel may use (0 = automatic)
 *   "time_kernels"  1 = bracket every kernel launch with CUDA events on the call's stream
 *               (read back with dfjk_kernel_time); setting it (to 0 or 1) clears the record
 *   "j_fused"   1 (default) = in a call that builds J and K together, the fitting coefficients
 *               d_P = <B_P, D> are read off the half-transformed tensor the K build produces
 *               anyway (<B_P, C C^T> = <B_P C, C>), so B is streamed ONCE for J (the axpy pass)
 *               instead of twice; 0 = always the two plain streaming passes over B (dot, then
 *               axpy).  Applies to dfjk_get_jk, dfjk_get_jk_u and dfjk_get_jk_pair (there
 *               <B_P, C1 C2^T> = <B_P C1, C2>); J-only calls and raw-dm calls always use two passes.
 *   "k2_panel"  which K2 kernel forms K += X X^T: 0 = one CTA per (tile, contiguous k range) with a
 *               partial K per range; 1 = panel-synchronous (the k range is cut into short panels,
 *               items (panel, tile) are dealt dynamically to persistent CTAs and added in panel
 *               order into L2-resident slabs, so that X is read from HBM once instead of ~8 times);
 *               2 (default) = 1 when the X chunk is larger than L2 and there are at least 21
 *               lower tiles (nao > 640), else 0.  The full (non-symmetric) product of
 *               dfjk_get_jk_pair / _dm has nb^2 tiles instead of nb(nb+1)/2 and switches one block
 *               row earlier: at nb >= 5 (nao > 512, 25 tiles).
 *   "k2_panel_kb"  target size in KB of one k panel of X for "k2_panel" (default 32768; accepted
 *               range 64 .. 4194304)
 *   "k2_weighted"  split counts of the "k2_panel" = 0 kernel: 0 = the same for every lower tile; 1 = in
 *               proportion to the tile's cost (diagonal and ragged tiles are cheaper), so that the
 *               CTAs of a single wave run equally long; 2 (default) = 1 when there are no more lower
 *               tiles than SMs and the X chunk stays in L2 (small problems), else 0.  Ignored
 *               while "k_splits" is set.  K is deterministic either way (different roundings).
 *   "graph"     1 (default) = dfjk_get_jk / dfjk_get_jk_u replay a CUDA graph of their own launch
 *               sequence: the first call of a shape (orbital counts, requested outputs, options)
 *               launches kernel by kernel, the second captures the sequence after the orbital
 *               packing into a graph kept in the handle, later ones launch that graph (the call's
 *               output pointers reach the finishing kernels through device memory).  Small problems
 *               are bound by launch count, not by work.  0 = always launch kernel by kernel.  Not
 *               used while "time_kernels" is on or while `stream` is itself being captured.
 *   "poison_workspace"  test aid, not a setting: value 1 waits for the device and fills the handle's
 *               whole workspace with 0xFF bytes (NaN as doubles) once, so that a later call that reads
 *               workspace it has not written itself produces NaN instead of a plausible number.
 */
int dfjk_set_option(dfjk_handle *h, const char *name, int64_t value);

/* kernel ids for dfjk_kernel_time (one per step of the path) */
#define DFJK_KERNEL_K0   0   /* pack / zero-pad C_occ */
#define DFJK_KERNEL_J0   1   /* build D-tilde */
#define DFJK_KERNEL_J1   2   /* d_P = <B_P, D-tilde> (streams B), or <X_P, C> (streams X) when fused */
#define DFJK_KERNEL_J1R  3   /* reduce d partials */
#define DFJK_KERNEL_J2   4   /* Jp = sum_P d_P B_P         (streams B) */
#define DFJK_KERNEL_J3   5   /* unpack Jp -> J */
#define DFJK_KERNEL_K1   6   /* X_P = B_P C                (DMMA) */
#define DFJK_KERNEL_K2   7   /* K_lower += X X^T           (DMMA) */
#define DFJK_KERNEL_K3   8   /* reduce splits, mirror */
#define DFJK_KERNEL_COUNT 9

/*
 * dfjk_launch_count -- number of kernels this handle has launched since dfjk_create.
 */
int64_t dfjk_launch_count(const dfjk_handle *h);

/*
 * dfjk_kernel_time -- with option "time_kernels" = 1: total device time (ms, CUDA events
 * on the launching stream) and number of launches of kernel `kernel` (DFJK_KERNEL_*)
 * recorded since the option was last set.  Waits for the recorded events (HOST pointers
 * ms_total, count).  The event ring grows as needed (1024 launches at first, doubling); if it
 * cannot grow, later launches go unrecorded and this call reports DFJK_ENOMEM.
 */
int dfjk_kernel_time(dfjk_handle *h, int kernel, double *ms_total, int64_t *count);

/*
 * dfjk_workspace_bytes -- bytes of device workspace owned by the handle.
 */
int64_t dfjk_workspace_bytes(const dfjk_handle *h);

/*
 * dfjk_destroy -- frees the workspace; never frees B.  NULL is a no-op.  Returns 0.
 * The caller must make sure no enqueued work still uses the handle.
 */
int dfjk_destroy(dfjk_handle *h);

/*
 * dfjk_probe_dmma_peak -- measurement aid: runs a register-only DMMA.8x8x4 loop on every SM of the
 * current device (default stream, synchronous, ~0.2 s) and returns the sustained FP64 rate in
 * TFLOP/s (HOST pointer).  This is the measured counterpart of the derived FP64 peak
 * (SMs x 64 FMA/clk x 2 x clock) that K's roofline fraction is quoted against.
 */
int dfjk_probe_dmma_peak(double *tflops);

/*
 * dfjk_scf_timing -- where the time of the LAST dfjk_scf_rhf / dfjk_scf_uhf run on this handle went
 * (HOST pointers, any may be NULL), measured with CUDA events on the run's stream: iterations done,
 * total ms inside get_jk / get_jk_u, total ms inside the eigensolver (cuSOLVER Dsygvd, core guess
 * included) and everything else (Fock, density, energy, DIIS error and extrapolation, host solves
 * and read-backs).  DFJK_EINVAL if there is nothing valid to report: no SCF has run, or the last run
 * failed or could not create / record one of its events (a run never reports an earlier run's
 * figures).  PAPER.md:258-262 (the SCF loop).
 */
int dfjk_scf_timing(const dfjk_handle *h, int64_t *iters, double *get_jk_ms, double *eig_ms, double *other_ms);

/*
 * dfjk_device_info -- measurement aid: what the roofline denominators are derived from, read from
 * the CURRENT device (HOST pointers, any may be NULL): number of SMs, the peak SM clock in kHz
 * (cudaDevAttrClockRate) and the L2 size in bytes.  Derived FP64 peak = sm_count x 64 FMA/clk x 2 x
 * clock (DMMA.8x8x4 runs on the FP64 pipe).  Returns 0 or DFJK_ECUDA.
 */
int dfjk_device_info(int *sm_count, int *sm_clock_khz, int64_t *l2_bytes);

/* dfjk_last_error -- thread-local text of the last failure ("" if none). */
const char *dfjk_last_error(void);

/* dfjk_version -- "major.minor.patch" of the library. */
const char *dfjk_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DFJK_H */
