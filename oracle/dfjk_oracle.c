/*
 * dfjk_oracle.c -- CPU ORACLE for the density-fitted Coulomb/exchange build.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load this library.
 * It shares no code, header, table or helper with the CUDA path under
 * paper_2506_06661_b200/ and neither side includes the other.
 *
 * What it computes (the plain definition, nothing clever):
 *
 *   PAPER.md:346-351 (Sec. IV.C.2, Eq. 1):  (mu nu|kappa lambda) ~= sum_P T_{P,mu nu} T_{P,kappa lambda}
 *   PAPER.md:353-356 (Eq. 2-3): T is the Cholesky-whitened 3-centre tensor; it is
 *       symmetric in (mu,nu) and stored packed (aosym='s2'; lower
 *       triangle via tril_indices).  T is called B here.
 *   PAPER.md:96, 126-131 (Sec. II.C / III):  jmat, kmat = get_jk(mol, dm)
 *
 *   With Eq. 1 inserted into the textbook J_mn = sum_ls (mn|ls) D_ls and
 *   K_mn = sum_ls (ml|ns) D_ls (BASELINE.json north_star states them in this form):
 *
 *       D        = sum_s w_s C_s C_s^T                (restricted: one set, w = 2)
 *       d_P      = sum_mu sum_nu B(P,mu,nu) D[mu][nu]             FULL square
 *       J[mu][nu]= sum_P d_P B(P,mu,nu)                           FULL square
 *       X_P[mu][i] = sum_nu B(P,mu,nu) C_s[nu][i]
 *       K_s[mu][nu]= sum_P sum_i X_P[mu][i] X_P[nu][i]            FULL square, NO factor 2
 *                                                       (reading R1)
 *   B(P,mu,nu) := Bp[P][a(a+1)/2 + b],  a = max(mu,nu), b = min(mu,nu)
 *                                                       (readings R3, R4)
 *
 * Deliberately NOT done here (the CUDA path does all of these, so a shared slip
 * cannot cancel): off-diagonal doubling of D, packed dot products, lower-triangle
 * only updates, tiling, chunking of X, mirrored output.
 *
 * P is the outermost loop and every output is ACCUMULATED, so B may be fed in
 * slabs of rows (51 GB / 96 GB tensors never have to fit in host memory): the
 * caller zeroes J, K_s once and calls oracle_jk_slab() per slab.
 *
 * d_P is summed two-level (row sums, then the sum of row sums) in binary64; a
 * single running total over 1e6 terms drifts to ~1e-13 (reading R9).
 *
 * Parity pins (tests/test_oracle_pins.py): brute force over the explicit 4-index
 * tensor built by oracle_bruteforce_jk() below (itself a different formula:
 * Eq. 1 materialised, then the textbook J/K contractions), closed forms,
 * invariants, single-element probes, numpy library reductions; the general-density
 * functions at the end of the file (oracle_jk_dm_slab, oracle_jk_pair_slab) are pinned
 * the same way in tests/test_oracle_general_pins.py.  No function in this file is
 * "parity unpinned".
 *
 * Build: gcc -O3 -march=x86-64-v3 -ffp-contract=off -fopenmp -shared -fPIC (no -ffast-math, no
 * reassociation, no FMA contraction: bit-for-bit the results of a plain -O2 build).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK      0
#define ORACLE_EINVAL -1
#define ORACLE_ENOMEM -2

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* B(P,mu,nu) of one packed row: Bp_row[a(a+1)/2+b], a=max, b=min (reading R3). */
static inline double b_elem(const double *Bp_row, int64_t mu, int64_t nu)
{
    int64_t a = mu > nu ? mu : nu;
    int64_t b = mu > nu ? nu : mu;
    return Bp_row[a * (a + 1) / 2 + b];
}

/*
 * oracle_jk_slab: accumulate the contribution of `nrows` rows of packed B
 * (Bp_slab[r][npair], r = 0..nrows-1) into J and K_s.
 *
 *   nao            number of orbital basis functions
 *   nset           number of orbital sets (1 restricted, 2 unrestricted, any >= 1)
 *   C[s]           nao x nocc[s], row-major (C[s][mu*nocc[s]+i])
 *   w[s]           density weight of set s (D = sum_s w_s C_s C_s^T)
 *   J              nao x nao row-major, accumulated (may be NULL)
 *   K[s]           nao x nao row-major, accumulated (K may be NULL, or K[s] NULL)
 *   d_out          nrows doubles, d_P of each slab row (may be NULL)
 */
int oracle_jk_slab(int64_t nrows, int64_t nao, const double *Bp_slab,
                   int nset, const double *const *C, const int64_t *nocc,
                   const double *w, double *J, double *const *K, double *d_out)
{
    if (nrows < 0 || nao < 1 || nset < 1 || !Bp_slab || !C || !nocc || !w)
        return ORACLE_EINVAL;
    for (int s = 0; s < nset; ++s)
        if (!C[s] || nocc[s] < 1)
            return ORACLE_EINVAL;
    const int64_t npair = nao * (nao + 1) / 2;
    int64_t nocc_max = 0;
    for (int s = 0; s < nset; ++s)
        if (nocc[s] > nocc_max) nocc_max = nocc[s];

    double *D = (double *)malloc(sizeof(double) * nao * nao);
    double *Bf = (double *)malloc(sizeof(double) * nao * nao);
    double *Xt = (double *)malloc(sizeof(double) * nocc_max * nao);
    double *X = (double *)malloc(sizeof(double) * nocc_max * nao);
    double *rowsum = (double *)malloc(sizeof(double) * nao);
    if (!D || !Bf || !Xt || !X || !rowsum) {
        free(D); free(Bf); free(Xt); free(X); free(rowsum);
        return ORACLE_ENOMEM;
    }

    /* D[mu][nu] = sum_s w_s sum_i C_s[mu][i] C_s[nu][i] */
#pragma omp parallel for schedule(static)
    for (int64_t mu = 0; mu < nao; ++mu)
        for (int64_t nu = 0; nu < nao; ++nu) {
            double acc = 0.0;
            for (int s = 0; s < nset; ++s) {
                const double *Cs = C[s];
                const int64_t no = nocc[s];
                double t = 0.0;
                for (int64_t i = 0; i < no; ++i)
                    t += Cs[mu * no + i] * Cs[nu * no + i];
                acc += w[s] * t;
            }
            D[mu * nao + nu] = acc;
        }

    for (int64_t r = 0; r < nrows; ++r) {
        const double *Bp_row = Bp_slab + r * npair;

        /* unpack B_P to the full square by max/min */
#pragma omp parallel for schedule(static)
        for (int64_t mu = 0; mu < nao; ++mu)
            for (int64_t nu = 0; nu < nao; ++nu)
                Bf[mu * nao + nu] = b_elem(Bp_row, mu, nu);

        /* d_P = sum_mu ( sum_nu B(P,mu,nu) D[mu][nu] ) */
#pragma omp parallel for schedule(static)
        for (int64_t mu = 0; mu < nao; ++mu) {
            double t = 0.0;
            for (int64_t nu = 0; nu < nao; ++nu)
                t += Bf[mu * nao + nu] * D[mu * nao + nu];
            rowsum[mu] = t;
        }
        double dP = 0.0;
        for (int64_t mu = 0; mu < nao; ++mu)
            dP += rowsum[mu];
        if (d_out) d_out[r] = dP;

        /* J += d_P * B_P */
        if (J) {
#pragma omp parallel for schedule(static)
            for (int64_t mu = 0; mu < nao; ++mu)
                for (int64_t nu = 0; nu < nao; ++nu)
                    J[mu * nao + nu] += dP * Bf[mu * nao + nu];
        }

        if (K) {
            for (int s = 0; s < nset; ++s) {
                if (!K[s]) continue;
                const double *Cs = C[s];
                const int64_t no = nocc[s];
                double *Ks = K[s];
                /* X_P[mu][i] = sum_nu B(P,mu,nu) C_s[nu][i]  (i innermost: axpy
                 * form, so the compiler vectorises without reassociation);
                 * kept transposed, Xt[i][mu], for the update below */
#pragma omp parallel for schedule(static)
                for (int64_t mu = 0; mu < nao; ++mu) {
                    double *xrow = X + mu * no;
                    for (int64_t i = 0; i < no; ++i) xrow[i] = 0.0;
                    for (int64_t nu = 0; nu < nao; ++nu) {
                        const double b = Bf[mu * nao + nu];
                        const double *crow = Cs + nu * no;
                        for (int64_t i = 0; i < no; ++i)
                            xrow[i] += b * crow[i];
                    }
                    for (int64_t i = 0; i < no; ++i)
                        Xt[i * nao + mu] = xrow[i];
                }
                /* K_s[mu][nu] += sum_i Xt[i][mu] Xt[i][nu], all mu, nu */
#pragma omp parallel for schedule(static)
                for (int64_t mu = 0; mu < nao; ++mu) {
                    double *Krow = Ks + mu * nao;
                    for (int64_t i = 0; i < no; ++i) {
                        const double xm = Xt[i * nao + mu];
                        const double *Xi = Xt + i * nao;
                        for (int64_t nu = 0; nu < nao; ++nu)
                            Krow[nu] += xm * Xi[nu];
                    }
                }
            }
        }
    }
    free(D); free(Bf); free(Xt); free(X); free(rowsum);
    return ORACLE_OK;
}

/*
 * oracle_bruteforce_jk: the definition with Eq. 1 MATERIALISED.
 * Tiny inputs only (nao^4 doubles are allocated).
 *
 *   eri[m][n][l][s] = sum_P B(P,m,n) B(P,l,s)                     (Eq. 1)
 *   D               = sum_s w_s C_s C_s^T
 *   J[m][n]         = sum_{l,s} eri[m][n][l][s] D[l][s]            (textbook Coulomb)
 *   K_s[m][n]       = sum_{l,s} eri[m][l][n][s] (C_s C_s^T)[l][s]  (textbook exchange,
 *                     per-set density WITHOUT weight: reading R1/R7)
 *   diag[m][n]      = eri[m][n][m][n]  (Eq. 7's DF diagonal), optional
 *
 * Outputs are OVERWRITTEN.  This is the pin for oracle_jk_slab, never the other
 * way round; the two share only b_elem().
 */
int oracle_bruteforce_jk(int64_t naux, int64_t nao, const double *Bp,
                         int nset, const double *const *C, const int64_t *nocc,
                         const double *w, double *J, double *const *K, double *diag)
{
    if (naux < 1 || nao < 1 || nao > 40 || nset < 1 || !Bp || !C || !nocc || !w)
        return ORACLE_EINVAL;
    const int64_t npair = nao * (nao + 1) / 2;
    const int64_t n2 = nao * nao, n3 = n2 * nao, n4 = n3 * nao;
    double *eri = (double *)calloc((size_t)n4, sizeof(double));
    double *Ds = (double *)malloc(sizeof(double) * n2);
    if (!eri || !Ds) { free(eri); free(Ds); return ORACLE_ENOMEM; }

    for (int64_t m = 0; m < nao; ++m)
        for (int64_t n = 0; n < nao; ++n)
            for (int64_t l = 0; l < nao; ++l)
                for (int64_t s = 0; s < nao; ++s) {
                    double acc = 0.0;
                    for (int64_t P = 0; P < naux; ++P)
                        acc += b_elem(Bp + P * npair, m, n) * b_elem(Bp + P * npair, l, s);
                    eri[m * n3 + n * n2 + l * nao + s] = acc;
                }

    if (diag)
        for (int64_t m = 0; m < nao; ++m)
            for (int64_t n = 0; n < nao; ++n)
                diag[m * nao + n] = eri[m * n3 + n * n2 + m * nao + n];

    if (J)
        for (int64_t i = 0; i < n2; ++i) J[i] = 0.0;

    for (int set = 0; set < nset; ++set) {
        const double *Cs = C[set];
        const int64_t no = nocc[set];
        for (int64_t l = 0; l < nao; ++l)
            for (int64_t s = 0; s < nao; ++s) {
                double t = 0.0;
                for (int64_t i = 0; i < no; ++i)
                    t += Cs[l * no + i] * Cs[s * no + i];
                Ds[l * nao + s] = t;
            }
        if (J)
            for (int64_t m = 0; m < nao; ++m)
                for (int64_t n = 0; n < nao; ++n) {
                    double acc = 0.0;
                    for (int64_t l = 0; l < nao; ++l)
                        for (int64_t s = 0; s < nao; ++s)
                            acc += eri[m * n3 + n * n2 + l * nao + s] * Ds[l * nao + s];
                    J[m * nao + n] += w[set] * acc;
                }
        if (K && K[set])
            for (int64_t m = 0; m < nao; ++m)
                for (int64_t n = 0; n < nao; ++n) {
                    double acc = 0.0;
                    for (int64_t l = 0; l < nao; ++l)
                        for (int64_t s = 0; s < nao; ++s)
                            acc += eri[m * n3 + l * n2 + n * nao + s] * Ds[l * nao + s];
                    K[set][m * nao + n] = acc;
                }
    }
    free(eri); free(Ds);
    return ORACLE_OK;
}

/*
 * oracle_kv_slab: matrix-vector form of the K definition, for sizes where the
 * full-square K update is too slow on a CPU (cfg 4-5).
 *
 *   (K_s v)[mu] = sum_P sum_nu B(P,mu,nu) u_P[nu],
 *        u_P    = C_s ( C_s^T ( B_P v ) )          with  (B_P v)[l] = sum_s' B(P,l,s') v[s']
 *
 * which is K_s = sum_P B_P C_s C_s^T B_P (the K of the header, X_P X_P^T expanded)
 * applied to v, evaluated right-to-left so no nao x nao product is formed.
 * V holds nvec vectors, V[k*nao + mu]; KV[s][k*nao + mu] is ACCUMULATED over slabs.
 */
int oracle_kv_slab(int64_t nrows, int64_t nao, const double *Bp_slab,
                   int nset, const double *const *C, const int64_t *nocc,
                   int64_t nvec, const double *V, double *const *KV)
{
    if (nrows < 0 || nao < 1 || nset < 1 || nvec < 1 || !Bp_slab || !C || !nocc || !V || !KV)
        return ORACLE_EINVAL;
    const int64_t npair = nao * (nao + 1) / 2;
    int64_t nocc_max = 0;
    for (int s = 0; s < nset; ++s)
        if (nocc[s] > nocc_max) nocc_max = nocc[s];
    int rc = ORACLE_OK;

#pragma omp parallel
    {
        double *t = (double *)malloc(sizeof(double) * nao);
        double *u = (double *)malloc(sizeof(double) * nao);
        double *y = (double *)malloc(sizeof(double) * nocc_max);
        double *acc = (double *)calloc((size_t)(nset * nvec * nao), sizeof(double));
        if (!t || !u || !y || !acc) {
#pragma omp critical
            rc = ORACLE_ENOMEM;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (int64_t r = 0; r < nrows; ++r) {
                const double *Bp_row = Bp_slab + r * npair;
                for (int64_t k = 0; k < nvec; ++k) {
                    const double *v = V + k * nao;
                    /* t = B_P v */
                    for (int64_t l = 0; l < nao; ++l) {
                        double a = 0.0;
                        for (int64_t s2 = 0; s2 < nao; ++s2)
                            a += b_elem(Bp_row, l, s2) * v[s2];
                        t[l] = a;
                    }
                    for (int s = 0; s < nset; ++s) {
                        const double *Cs = C[s];
                        const int64_t no = nocc[s];
                        /* y = C_s^T t ; u = C_s y */
                        for (int64_t i = 0; i < no; ++i) {
                            double a = 0.0;
                            for (int64_t l = 0; l < nao; ++l)
                                a += Cs[l * no + i] * t[l];
                            y[i] = a;
                        }
                        for (int64_t l = 0; l < nao; ++l) {
                            double a = 0.0;
                            for (int64_t i = 0; i < no; ++i)
                                a += Cs[l * no + i] * y[i];
                            u[l] = a;
                        }
                        /* acc += B_P u */
                        double *out = acc + (s * nvec + k) * nao;
                        for (int64_t m = 0; m < nao; ++m) {
                            double a = 0.0;
                            for (int64_t n = 0; n < nao; ++n)
                                a += b_elem(Bp_row, m, n) * u[n];
                            out[m] += a;
                        }
                    }
                }
            }
#pragma omp critical
            {
                for (int s = 0; s < nset; ++s)
                    if (KV[s])
                        for (int64_t i = 0; i < nvec * nao; ++i)
                            KV[s][i] += acc[s * nvec * nao + i];
            }
        }
        free(t); free(u); free(y); free(acc);
    }
    return rc;
}

/* ======================================================================================
 * General densities.  PAPER.md:96: get_jk "supports an
 * arbitrary number of density matrices"; the DF-approximated orbital
 * Hessian of SOSCF contracts the same integrals with NON-idempotent, in general
 * non-symmetric, response densities.  With Eq. 1 in the textbook
 * contractions, for ANY real nao x nao matrix dm:
 *
 *     J[dm][m][n] = sum_{l,s} (mn|ls) dm[l][s] = sum_P B(P,m,n) * ( sum_{l,s} B(P,l,s) dm[l][s] )
 *     K[dm][m][n] = sum_{l,s} (ml|ns) dm[l][s] = sum_P sum_{l,s} B(P,m,l) dm[l][s] B(P,n,s)
 *
 * Both are LINEAR in dm (this is PySCF's vj, vk).  The occupied-orbital build above is the
 * special case  K_s = K[C_s C_s^T]  (no weight: reading R1) and  J = J[sum_s w_s C_s C_s^T].
 * ====================================================================================== */

/*
 * oracle_jk_dm_slab: accumulate J[dm] and K[dm] of `nrows` packed rows, straight from the
 * two formulas above: plain triple loops, full squares, nothing factorised.
 *   dm  nao x nao row-major, ANY real matrix;  J, K accumulated (either may be NULL);
 *   d_out[r] = sum_{l,s} B(P,l,s) dm[l][s]  (may be NULL).
 */
int oracle_jk_dm_slab(int64_t nrows, int64_t nao, const double *Bp_slab, const double *dm,
                      double *J, double *K, double *d_out)
{
    if (nrows < 0 || nao < 1 || !Bp_slab || !dm) return ORACLE_EINVAL;
    const int64_t npair = nao * (nao + 1) / 2;
    double *Bf = (double *)malloc(sizeof(double) * nao * nao);
    double *T = (double *)malloc(sizeof(double) * nao * nao);
    double *rowsum = (double *)malloc(sizeof(double) * nao);
    if (!Bf || !T || !rowsum) { free(Bf); free(T); free(rowsum); return ORACLE_ENOMEM; }

    for (int64_t r = 0; r < nrows; ++r) {
        const double *Bp_row = Bp_slab + r * npair;
#pragma omp parallel for schedule(static)
        for (int64_t m = 0; m < nao; ++m)
            for (int64_t n = 0; n < nao; ++n)
                Bf[m * nao + n] = b_elem(Bp_row, m, n);

        /* d_P = sum_l ( sum_s B(P,l,s) dm[l][s] )  -- two-level, reading R9 */
#pragma omp parallel for schedule(static)
        for (int64_t l = 0; l < nao; ++l) {
            double t = 0.0;
            for (int64_t s = 0; s < nao; ++s)
                t += Bf[l * nao + s] * dm[l * nao + s];
            rowsum[l] = t;
        }
        double dP = 0.0;
        for (int64_t l = 0; l < nao; ++l) dP += rowsum[l];
        if (d_out) d_out[r] = dP;

        if (J) {
#pragma omp parallel for schedule(static)
            for (int64_t m = 0; m < nao; ++m)
                for (int64_t n = 0; n < nao; ++n)
                    J[m * nao + n] += dP * Bf[m * nao + n];
        }
        if (K) {
            /* T[m][s] = sum_l B(P,m,l) dm[l][s]   (s innermost: axpy form) */
#pragma omp parallel for schedule(static)
            for (int64_t m = 0; m < nao; ++m) {
                double *Trow = T + m * nao;
                for (int64_t s = 0; s < nao; ++s) Trow[s] = 0.0;
                for (int64_t l = 0; l < nao; ++l) {
                    const double b = Bf[m * nao + l];
                    const double *drow = dm + l * nao;
                    for (int64_t s = 0; s < nao; ++s) Trow[s] += b * drow[s];
                }
            }
            /* K[m][n] += sum_s T[m][s] B(P,n,s)  =  sum_s T[m][s] Bf[s][n]  (B_P symmetric
             * BY CONSTRUCTION of Bf: Bf[s][n] and Bf[n][s] are the same packed element) */
#pragma omp parallel for schedule(static)
            for (int64_t m = 0; m < nao; ++m) {
                double *Krow = K + m * nao;
                for (int64_t s = 0; s < nao; ++s) {
                    const double t = T[m * nao + s];
                    const double *brow = Bf + s * nao;
                    for (int64_t n = 0; n < nao; ++n) Krow[n] += t * brow[n];
                }
            }
        }
    }
    free(Bf); free(T); free(rowsum);
    return ORACLE_OK;
}

/*
 * oracle_jk_pair_slab: the factorised form used when dm = C1 C2^T is given by its factors
 * (response densities of SOSCF / TDDFT):
 *
 *     X1_P = B_P C1,  X2_P = B_P C2   (nao x ncol each)
 *     K[m][n] += sum_i X1_P[m][i] X2_P[n][i]                 (= K[C1 C2^T], not symmetric)
 *     d_P = sum_{l,s} B(P,l,s) (C1 C2^T)[l][s],   J += d_P B_P
 *
 * Pinned against oracle_jk_dm_slab (a different formula) and the brute force below.
 */
int oracle_jk_pair_slab(int64_t nrows, int64_t nao, const double *Bp_slab, int64_t ncol,
                        const double *C1, const double *C2, double *J, double *K, double *d_out)
{
    if (nrows < 0 || nao < 1 || ncol < 1 || !Bp_slab || !C1 || !C2) return ORACLE_EINVAL;
    const int64_t npair = nao * (nao + 1) / 2;
    double *D = (double *)malloc(sizeof(double) * nao * nao);
    double *Bf = (double *)malloc(sizeof(double) * nao * nao);
    double *X1 = (double *)malloc(sizeof(double) * nao * ncol);
    double *X2t = (double *)malloc(sizeof(double) * nao * ncol);
    double *rowsum = (double *)malloc(sizeof(double) * nao);
    if (!D || !Bf || !X1 || !X2t || !rowsum) {
        free(D); free(Bf); free(X1); free(X2t); free(rowsum);
        return ORACLE_ENOMEM;
    }
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < nao; ++l)
        for (int64_t s = 0; s < nao; ++s) {
            double t = 0.0;
            for (int64_t i = 0; i < ncol; ++i) t += C1[l * ncol + i] * C2[s * ncol + i];
            D[l * nao + s] = t;
        }
    for (int64_t r = 0; r < nrows; ++r) {
        const double *Bp_row = Bp_slab + r * npair;
#pragma omp parallel for schedule(static)
        for (int64_t m = 0; m < nao; ++m)
            for (int64_t n = 0; n < nao; ++n)
                Bf[m * nao + n] = b_elem(Bp_row, m, n);
#pragma omp parallel for schedule(static)
        for (int64_t l = 0; l < nao; ++l) {
            double t = 0.0;
            for (int64_t s = 0; s < nao; ++s) t += Bf[l * nao + s] * D[l * nao + s];
            rowsum[l] = t;
        }
        double dP = 0.0;
        for (int64_t l = 0; l < nao; ++l) dP += rowsum[l];
        if (d_out) d_out[r] = dP;
        if (J) {
#pragma omp parallel for schedule(static)
            for (int64_t m = 0; m < nao; ++m)
                for (int64_t n = 0; n < nao; ++n)
                    J[m * nao + n] += dP * Bf[m * nao + n];
        }
        if (K) {
            /* X1[m][i] = sum_l B(P,m,l) C1[l][i];  X2t[i][n] = sum_l B(P,n,l) C2[l][i] */
#pragma omp parallel for schedule(static)
            for (int64_t m = 0; m < nao; ++m) {
                for (int64_t i = 0; i < ncol; ++i) {
                    double a = 0.0, b = 0.0;
                    for (int64_t l = 0; l < nao; ++l) {
                        a += Bf[m * nao + l] * C1[l * ncol + i];
                        b += Bf[m * nao + l] * C2[l * ncol + i];
                    }
                    X1[m * ncol + i] = a;
                    X2t[i * nao + m] = b;
                }
            }
#pragma omp parallel for schedule(static)
            for (int64_t m = 0; m < nao; ++m) {
                double *Krow = K + m * nao;
                for (int64_t i = 0; i < ncol; ++i) {
                    const double x = X1[m * ncol + i];
                    const double *x2 = X2t + i * nao;
                    for (int64_t n = 0; n < nao; ++n) Krow[n] += x * x2[n];
                }
            }
        }
    }
    free(D); free(Bf); free(X1); free(X2t); free(rowsum);
    return ORACLE_OK;
}

/*
 * oracle_bruteforce_jk_dm: Eq. 1 materialised, then the textbook contractions with an
 * arbitrary dm (tiny inputs only).  J, K OVERWRITTEN.
 *     eri[m][n][l][s] = sum_P B(P,m,n) B(P,l,s)
 *     J[m][n] = sum_{l,s} eri[m][n][l][s] dm[l][s];   K[m][n] = sum_{l,s} eri[m][l][n][s] dm[l][s]
 */
int oracle_bruteforce_jk_dm(int64_t naux, int64_t nao, const double *Bp, const double *dm,
                            double *J, double *K)
{
    if (naux < 1 || nao < 1 || nao > 40 || !Bp || !dm) return ORACLE_EINVAL;
    const int64_t npair = nao * (nao + 1) / 2;
    const int64_t n2 = nao * nao, n3 = n2 * nao, n4 = n3 * nao;
    double *eri = (double *)calloc((size_t)n4, sizeof(double));
    if (!eri) return ORACLE_ENOMEM;
    for (int64_t m = 0; m < nao; ++m)
        for (int64_t n = 0; n < nao; ++n)
            for (int64_t l = 0; l < nao; ++l)
                for (int64_t s = 0; s < nao; ++s) {
                    double acc = 0.0;
                    for (int64_t P = 0; P < naux; ++P)
                        acc += b_elem(Bp + P * npair, m, n) * b_elem(Bp + P * npair, l, s);
                    eri[m * n3 + n * n2 + l * nao + s] = acc;
                }
    for (int64_t m = 0; m < nao; ++m)
        for (int64_t n = 0; n < nao; ++n) {
            double aj = 0.0, ak = 0.0;
            for (int64_t l = 0; l < nao; ++l)
                for (int64_t s = 0; s < nao; ++s) {
                    aj += eri[m * n3 + n * n2 + l * nao + s] * dm[l * nao + s];
                    ak += eri[m * n3 + l * n2 + n * nao + s] * dm[l * nao + s];
                }
            if (J) J[m * nao + n] = aj;
            if (K) K[m * nao + n] = ak;
        }
    free(eri);
    return ORACLE_OK;
}

/*
 * oracle_df_diag_slab: the DF term of Eq. 7,
 *     diag[m][n] += sum_{P in slab} B(P,m,n)^2        = (mn|mn) of Eq. 1 with kappa lambda = mu nu
 * full square, accumulated over slabs.  Pinned (tests/test_oracle_general_pins.py) against the
 * materialised eri[m][n][m][n] of oracle_bruteforce_jk, numpy, and the identity
 * sum_n diag[m][n] = K[m][m] for C = I (K = sum_P B_P^2).
 */
int oracle_df_diag_slab(int64_t nrows, int64_t nao, const double *Bp_slab, double *diag)
{
    if (nrows < 0 || nao < 1 || !Bp_slab || !diag) return ORACLE_EINVAL;
    const int64_t npair = nao * (nao + 1) / 2;
    for (int64_t r = 0; r < nrows; ++r) {
        const double *Bp_row = Bp_slab + r * npair;
#pragma omp parallel for schedule(static)
        for (int64_t m = 0; m < nao; ++m)
            for (int64_t n = 0; n < nao; ++n) {
                const double b = b_elem(Bp_row, m, n);
                diag[m * nao + n] += b * b;
            }
    }
    return ORACLE_OK;
}

/* ======================================================================================
 * Building the whitened tensor -- PAPER.md:353-356, Eq. 2-3:
 *
 *     M_PQ = (chi_P|chi_Q) = L L^T                                            (Eq. 2)
 *     T_{P,mu nu} = sum_Q (L^-1)_{PQ} (chi_Q|mu nu)                            (Eq. 3)
 *
 * T is this library's B.  The oracle follows the two equations literally: the textbook
 * Cholesky-Banachiewicz recurrence for L (row by row), then, for every packed column, the
 * forward substitution that applies L^-1 (no explicit inverse, no blocking).
 * ====================================================================================== */
#include <math.h>

/*
 * oracle_cholesky_lower: L (n x n row-major, lower triangle; the strict upper triangle is set
 * to 0) with M = L L^T, M symmetric positive definite (only its lower triangle is read):
 *     L[i][j] = ( M[i][j] - sum_{k<j} L[i][k] L[j][k] ) / L[j][j]      j < i
 *     L[i][i] = sqrt( M[i][i] - sum_{k<i} L[i][k]^2 )
 * Returns ORACLE_EINVAL and stops at the first non-positive pivot.
 */
int oracle_cholesky_lower(int64_t n, const double *M, double *L)
{
    if (n < 1 || !M || !L) return ORACLE_EINVAL;
    for (int64_t i = 0; i < n * n; ++i) L[i] = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        for (int64_t j = 0; j <= i; ++j) {
            double s = M[i * n + j];
            for (int64_t k = 0; k < j; ++k) s -= L[i * n + k] * L[j * n + k];
            if (i == j) {
                if (!(s > 0.0)) return ORACLE_EINVAL;
                L[i * n + i] = sqrt(s);
            } else {
                L[i * n + j] = s / L[j * n + j];
            }
        }
    }
    return ORACLE_OK;
}

/*
 * oracle_whiten: B[P][c] = sum_Q (L^-1)[P][Q] R[Q][c] for every column c < ncols (Eq. 3), by
 * forward substitution  B[P][c] = ( R[P][c] - sum_{Q<P} L[P][Q] B[Q][c] ) / L[P][P].
 * R and B are naux x ncols row-major (ncols = npair for the packed tensor); B may alias R.
 */
int oracle_whiten(int64_t naux, int64_t ncols, const double *L, const double *R, double *B)
{
    if (naux < 1 || ncols < 1 || !L || !R || !B) return ORACLE_EINVAL;
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < ncols; ++c) {
        for (int64_t P = 0; P < naux; ++P) {
            double s = R[P * ncols + c];
            for (int64_t Q = 0; Q < P; ++Q) s -= L[P * naux + Q] * B[Q * ncols + c];
            B[P * ncols + c] = s / L[P * naux + P];
        }
    }
    return ORACLE_OK;
}
