/* gen_device.cu -- device side of the synthetic input generator (see gen_core.h).
 * Fills the 51 GB / 96 GB tensors in place; no DF-JK arithmetic in here. */
#include "gen_core.h"
#include <cuda_runtime.h>

__global__ void gen_fill_B_kernel(uint64_t zkey, int64_t nao, int64_t npair,
                                  const double *__restrict__ x, const double *__restrict__ a,
                                  int64_t P0, int64_t nrows, int rows_per_block,
                                  double *__restrict__ out)
{
    const int64_t pair = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (pair >= npair) return;
    /* invert pair = mu(mu+1)/2 + nu; never trust the bare sqrt */
    int64_t mu = (int64_t)((sqrt(8.0 * (double)pair + 1.0) - 1.0) * 0.5);
    while (mu * (mu + 1) / 2 > pair) --mu;
    while ((mu + 1) * (mu + 2) / 2 <= pair) ++mu;
    const int64_t nu = pair - mu * (mu + 1) / 2;
    const double g = gen_locality(x[mu], x[nu]);
    const int64_t r0 = (int64_t)blockIdx.y * rows_per_block;
    int64_t r1 = r0 + rows_per_block;
    if (r1 > nrows) r1 = nrows;
    for (int64_t r = r0; r < r1; ++r) {
        const int64_t P = P0 + r;
        out[r * npair + pair] = gen_b_elem(zkey, a[P], g, (uint64_t)(P * npair + pair));
    }
}

extern "C" int gen_fill_B_rows_device(uint64_t seed, int64_t nao, const double *x_dev,
                                      const double *a_dev, int64_t P0, int64_t nrows,
                                      double *out_dev, void *stream)
{
    const int64_t npair = nao * (nao + 1) / 2;
    const int threads = 256;
    const int rows_per_block = 16;
    int64_t done = 0;
    while (done < nrows) {           /* grid.y <= 65535 */
        int64_t n = nrows - done;
        if (n > 65535LL * rows_per_block) n = 65535LL * rows_per_block;
        dim3 grid((unsigned)((npair + threads - 1) / threads),
                  (unsigned)((n + rows_per_block - 1) / rows_per_block));
        gen_fill_B_kernel<<<grid, threads, 0, (cudaStream_t)stream>>>(
            gen_key(seed, GEN_STREAM_Z), nao, npair, x_dev, a_dev, P0 + done, n,
            rows_per_block, out_dev + done * npair);
        done += n;
    }
    return (int)cudaGetLastError();
}
