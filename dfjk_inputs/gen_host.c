/* gen_host.c -- host side of the synthetic input generator (see gen_core.h). */
#include "gen_core.h"
#include <stdlib.h>

void gen_uniform(uint64_t seed, uint64_t stream, int64_t n, double *out)
{
    const uint64_t key = gen_key(seed, stream);
    for (int64_t i = 0; i < n; ++i) out[i] = gen_u01(key, (uint64_t)i);
}

void gen_normals(uint64_t seed, uint64_t stream, int64_t n, double *out)
{
    const uint64_t key = gen_key(seed, stream);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) out[i] = gen_normal(key, (uint64_t)i);
}

void gen_bits_host(uint64_t seed, uint64_t stream, int64_t n, uint64_t *out)
{
    const uint64_t key = gen_key(seed, stream);
    for (int64_t i = 0; i < n; ++i) out[i] = gen_bits(key, (uint64_t)i);
}

/* rows P0 .. P0+nrows-1 of packed B into out[nrows][npair]; x[nao], a[naux] given */
int gen_fill_B_rows_host(uint64_t seed, int64_t nao, const double *x, const double *a,
                         int64_t P0, int64_t nrows, double *out)
{
    const int64_t npair = nao * (nao + 1) / 2;
    const uint64_t zkey = gen_key(seed, GEN_STREAM_Z);
    double *g = (double *)malloc(sizeof(double) * npair);
    if (!g) return -2;
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t mu = 0; mu < nao; ++mu)
        for (int64_t nu = 0; nu <= mu; ++nu)
            g[mu * (mu + 1) / 2 + nu] = gen_locality(x[mu], x[nu]);
#pragma omp parallel for schedule(static) collapse(2)
    for (int64_t r = 0; r < nrows; ++r)
        for (int64_t pair = 0; pair < npair; ++pair) {
            const int64_t P = P0 + r;
            out[r * npair + pair] =
                gen_b_elem(zkey, a[P], g[pair], (uint64_t)(P * npair + pair));
        }
    free(g);
    return 0;
}
