/*
 * scf_rhf.cu -- the DF-SCF drivers around the get_jk kernels (include/dfjk.h: dfjk_scf_rhf,
 * closed shell, and dfjk_scf_uhf, two spins -- one loop, scf_run, for both; SURVEY.md section 8f
 * rank 4).  The paper describes the loop in words only: the
 * mean-field object iterates Fock build -> diagonalisation -> new density, DIIS being the default
 * accelerator (mf.kernel(dm0)), with get_jk(dm) -> (vj, vk)
 * as the expensive step.  Per iteration, all on the device:
 *
 *     J, K = get_jk(C_occ)                       this library's hot path (J0-J3, K0-K3)
 *     F    = hcore + J - K                        S1 (elementwise)
 *     D    = 2 C_occ C_occ^T                      FP64 tile product
 *     E    = 1/2 sum D o (hcore + F)              S2 (two-stage deterministic reduction)
 *     e    = F D S - (F D S)^T                    two DMMA products (S6 packs the operands into the
 *                                                 k-group-major layout of the X workspace, then the
 *                                                 full-product kernel of k2_syrk.cu and K3's sum) + S3
 *     DIIS: B_im = <e_i, e_m> for all i in ONE launch pair (S2b), read back together with E and
 *           max|e| in ONE host sync; the (m+1) x (m+1) system on the host, F_ext = sum c_i F_i (S4)
 *     F_ext C = S C eps                           cuSOLVER Dsygvd -- the one library step, loaded
 *                                                 with dlopen so libdfjk.so itself has no
 *                                                 dependency on it
 *     C (row-major), C_occ                        S5 (transpose of the column-major eigenvectors)
 *
 * Unrestricted: the same per spin block with D_s = C_s,occ C_s,occ^T, get_jk_u, F_s = hcore + J - K_s,
 * E = sum_s 1/2 sum D_s o (hcore + F_s) and ONE DIIS over both blocks (B_ij = sum_s <e_s^i, e_s^j>).
 * The host reads back a few scalars per iteration (E, max|e|, the new DIIS dots) to decide convergence.
 */
#include "../../include/dfjk.h"
#include "dfjk_internal.h"

#include <cusolverDn.h>
#include <dlfcn.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

namespace dfjk {
namespace {

/* ------------------------------------------------------------------ cuSOLVER through dlopen */
struct Cusolver {
    void *lib = nullptr;
    cusolverStatus_t (*create)(cusolverDnHandle_t *) = nullptr;
    cusolverStatus_t (*destroy)(cusolverDnHandle_t) = nullptr;
    cusolverStatus_t (*set_stream)(cusolverDnHandle_t, cudaStream_t) = nullptr;
    cusolverStatus_t (*sygvd_bufsize)(cusolverDnHandle_t, cusolverEigType_t, cusolverEigMode_t,
                                      cublasFillMode_t, int, const double *, int, const double *, int,
                                      const double *, int *) = nullptr;
    cusolverStatus_t (*sygvd)(cusolverDnHandle_t, cusolverEigType_t, cusolverEigMode_t, cublasFillMode_t,
                              int, double *, int, double *, int, double *, double *, int, int *) = nullptr;
    char why[256] = "";                 /* why loading failed (dlerror of the first name tried) */
    bool ok() const { return lib && create && destroy && set_stream && sygvd_bufsize && sygvd; }
};

Cusolver &cusolver()
{
    static Cusolver cs;
    static std::once_flag once;
    std::call_once(once, [] {
        const char *names[] = {"libcusolver.so.11", "libcusolver.so",
                               "/usr/local/cuda/lib64/libcusolver.so.11", "libcusolver.so.12"};
        for (const char *n : names) {
            cs.lib = dlopen(n, RTLD_NOW | RTLD_LOCAL);
            if (cs.lib) break;
            const char *e = dlerror();          /* dlerror() clears itself: read it exactly once */
            if (e && !cs.why[0]) snprintf(cs.why, sizeof cs.why, "%s", e);
        }
        if (cs.lib) {
            cs.create = (decltype(cs.create))dlsym(cs.lib, "cusolverDnCreate");
            cs.destroy = (decltype(cs.destroy))dlsym(cs.lib, "cusolverDnDestroy");
            cs.set_stream = (decltype(cs.set_stream))dlsym(cs.lib, "cusolverDnSetStream");
            cs.sygvd_bufsize = (decltype(cs.sygvd_bufsize))dlsym(cs.lib, "cusolverDnDsygvd_bufferSize");
            cs.sygvd = (decltype(cs.sygvd))dlsym(cs.lib, "cusolverDnDsygvd");
            if (!cs.ok()) snprintf(cs.why, sizeof cs.why, "a cusolverDn symbol is missing");
        }
    });
    return cs;
}

/* ------------------------------------------------------------------ S1-S5: small kernels */
__global__ void fock_kernel(const double *__restrict__ h, const double *__restrict__ J,
                            const double *__restrict__ K, int64_t n2, double *__restrict__ F)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n2) F[i] = h[i] + J[i] - K[i];
}

/* partial[b] = reduction over this block's grid-stride share; mode 0: sum a*b, 1: sum a*(b+c),
 * 2: max |a|.  Fixed grid + fixed-order second stage => deterministic. */
constexpr int RED_BLOCKS = 256, RED_THREADS = 256;

__global__ void __launch_bounds__(RED_THREADS)
reduce_partial_kernel(int mode, const double *__restrict__ a, const double *__restrict__ b,
                      const double *__restrict__ c, int64_t n, double *__restrict__ partial)
{
    __shared__ double sh[RED_THREADS];
    double acc = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += (int64_t)RED_BLOCKS * RED_THREADS) {
        if (mode == 0) acc += a[i] * b[i];
        else if (mode == 1) acc += a[i] * (b[i] + c[i]);
        else acc = fmax(acc, fabs(a[i]));
    }
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int s = RED_THREADS / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s)
            sh[threadIdx.x] = mode == 2 ? fmax(sh[threadIdx.x], sh[threadIdx.x + s])
                                        : sh[threadIdx.x] + sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}

__global__ void reduce_final_kernel(int mode, const double *__restrict__ partial, double scale,
                                    double *__restrict__ out)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    double acc = 0.0;
    for (int i = 0; i < RED_BLOCKS; ++i) acc = mode == 2 ? fmax(acc, partial[i]) : acc + partial[i];
    *out = scale * acc;
}

/* e = T - T^T (T = F D S, so e = F D S - S D F) */
__global__ void antisym_kernel(const double *__restrict__ T, int64_t n, double *__restrict__ e)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n * n) return;
    const int64_t r = i / n, c = i - r * n;
    e[i] = T[i] - T[c * n + r];
}

struct Coefs { double c[16]; const double *F[16]; int m; };

__global__ void lincomb_kernel(Coefs cf, int64_t n2, double *__restrict__ out)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n2) return;
    double acc = 0.0;
    for (int k = 0; k < cf.m; ++k) acc += cf.c[k] * cf.F[k][i];
    out[i] = acc;
}

/* S6: operand packing for the DMMA product kernel of k2_syrk.cu, which reads both operands from one
 * k-group-major array X4[(k/4)][row][k%4]:  X4 column c0 + k of row r = M[r][k], k < n (zero for the
 * padding columns up to round_up(n, 4)).  One thread per (row, group of 4 columns): 32-byte store,
 * consecutive threads own consecutive rows => contiguous stores. */
__global__ void __launch_bounds__(256)
pack_x4_kernel(const double *__restrict__ M, int64_t n, int64_t c0, double *__restrict__ X4)
{
    const int64_t r = (int64_t)blockIdx.x * 256 + threadIdx.x;
    const int64_t g = blockIdx.y;
    if (r >= n) return;
    double v[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) v[q] = 4 * g + q < n ? M[r * n + 4 * g + q] : 0.0;
    double2 *dst = reinterpret_cast<double2 *>(X4 + (((c0 >> 2) + g) * n + r) * 4);
    dst[0] = make_double2(v[0], v[1]);
    dst[1] = make_double2(v[2], v[3]);
}

/* S2b: all DIIS dots of one iteration at once: partial[(i*nspin + s)*RED_BLOCKS + b] = block b's
 * share of <Ering_s[slot_i], Er_s>; dots_final sums blocks and spins in a fixed order. */
struct DotArgs { const double *a[32]; const double *b[32]; int npairs; };

__global__ void __launch_bounds__(RED_THREADS)
dots_partial_kernel(DotArgs da, int64_t n, double *__restrict__ partial)
{
    __shared__ double sh[RED_THREADS];
    const double *__restrict__ a = da.a[blockIdx.y];
    const double *__restrict__ b = da.b[blockIdx.y];
    double acc = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += (int64_t)RED_BLOCKS * RED_THREADS)
        acc += a[i] * b[i];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int s = RED_THREADS / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[(int64_t)blockIdx.y * RED_BLOCKS + blockIdx.x] = sh[0];
}

/* out[i] = sum_s sum_b partial[(i*nspin + s)][b], i < m */
__global__ void dots_final_kernel(const double *__restrict__ partial, int m, int nspin, double *__restrict__ out)
{
    const int i = threadIdx.x;
    if (i >= m) return;
    double acc = 0.0;
    for (int s = 0; s < nspin; ++s)
        for (int b = 0; b < RED_BLOCKS; ++b) acc += partial[(int64_t)(i * nspin + s) * RED_BLOCKS + b];
    out[i] = acc;
}

/* V holds the eigenvectors as columns of a column-major matrix: V[mu + i*n] = C[mu][i].
 * Writes C row-major (C[mu*n + i]) and the occupied block C_occ[mu*nocc + i], i < nocc. */
__global__ void __launch_bounds__(256)
unpack_vectors_kernel(const double *__restrict__ V, int64_t n, int64_t nocc, double *__restrict__ C,
                      double *__restrict__ C_occ)
{
    __shared__ double t[32][33];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int64_t i0 = (int64_t)blockIdx.y * 32, m0 = (int64_t)blockIdx.x * 32;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int64_t i = i0 + ty + 8 * r, mu = m0 + tx;
        t[ty + 8 * r][tx] = (i < n && mu < n) ? V[i * n + mu] : 0.0;
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int64_t mu = m0 + ty + 8 * r, i = i0 + tx;
        if (mu < n && i < n) {
            const double v = t[tx][ty + 8 * r];
            C[mu * n + i] = v;
            if (i < nocc) C_occ[mu * nocc + i] = v;
        }
    }
}

/* (m+1) x (m+1) DIIS system on the host: Gaussian elimination with partial pivoting */
bool solve_dense(std::vector<double> &A, std::vector<double> &b, int n)
{
    for (int k = 0; k < n; ++k) {
        int p = k;
        for (int i = k + 1; i < n; ++i)
            if (std::fabs(A[i * n + k]) > std::fabs(A[p * n + k])) p = i;
        if (A[p * n + k] == 0.0) return false;
        if (p != k) {
            for (int j = 0; j < n; ++j) std::swap(A[k * n + j], A[p * n + j]);
            std::swap(b[k], b[p]);
        }
        for (int i = k + 1; i < n; ++i) {
            const double f = A[i * n + k] / A[k * n + k];
            for (int j = k; j < n; ++j) A[i * n + j] -= f * A[k * n + j];
            b[i] -= f * b[k];
        }
    }
    for (int k = n - 1; k >= 0; --k) {
        double s = b[k];
        for (int j = k + 1; j < n; ++j) s -= A[k * n + j] * b[j];
        b[k] = s / A[k * n + k];
    }
    return true;
}

}  // namespace

namespace {
/* one timing mark: an event created and recorded on the run's stream.  A mark that cannot be made
 * clears *ok -- the (begin, end) pairing of its vector is then broken, and the run's timing is
 * reported as invalid instead of as a wrong sum. */
void mark_event(std::vector<cudaEvent_t> &v, cudaStream_t st, bool *ok)
{
    cudaEvent_t e = nullptr;
    if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); *ok = false; return; }
    if (cudaEventRecord(e, st) != cudaSuccess) { cudaGetLastError(); cudaEventDestroy(e); *ok = false; return; }
    v.push_back(e);
}
}  // namespace

#define SCF_TRY(expr)                                                                      \
    do {                                                                                   \
        cudaError_t e_ = (expr);                                                           \
        if (e_ != cudaSuccess) {                                                           \
            snprintf(err, errlen, "dfjk_scf: %s: %s", #expr, cudaGetErrorString(e_));      \
            rc = DFJK_ECUDA;                                                               \
            goto done;                                                                     \
        }                                                                                  \
    } while (0)

/* The loop of the file header for nspin = 1 (restricted: D = 2 C_occ C_occ^T, get_jk) or nspin = 2
 * (unrestricted: D_s = C_s,occ C_s,occ^T, get_jk_u; Pople-Nesbet with one DIIS over both spin
 * blocks).  Per-spin arrays are indexed [s].  All pointers except e_hist / n_iter / converged are
 * DEVICE.  Returns a DFJK_* code; on failure `err` holds the message. */
int scf_run(dfjk_handle *h, int64_t nao, int nspin, const double *hcore, const double *S,
            const int64_t *nocc, int64_t max_iter, double conv_tol, int64_t diis_space,
            double *const *C_out, double *const *mo_energy_out, double *const *D_out,
            double *const *F_out, double *e_hist, int64_t *n_iter, int *converged, cudaStream_t st,
            char *err, size_t errlen)
{
    Cusolver &cs = cusolver();
    if (!cs.ok()) {
        snprintf(err, errlen, "dfjk_scf: libcusolver could not be loaded (%s)", cs.why[0] ? cs.why : "unknown reason");
        return DFJK_ECUDA;
    }
    const int64_t n2 = nao * nao;
    const int m_max = (int)diis_space;
    const double dw = nspin == 1 ? 2.0 : 1.0;           /* density weight of one spin block */
    int rc = DFJK_OK;
    cusolverDnHandle_t sol = nullptr;
    double *ws = nullptr, *work = nullptr;
    int *dev_info = nullptr;
    int lwork = 0;
    std::vector<double> Bmat((size_t)m_max * m_max, 0.0);
    std::vector<int> slot_of;                        /* history, oldest first: ring slot ids */
    std::vector<cudaEvent_t> ev_jk, ev_eig, ev_total; /* timing: pairs (begin, end) */
    bool timing_ok = true;
    scf_store_timing(h, 0, 0.0, 0.0, 0.0);             /* a failed run must not report the previous run's timing */
    double e_prev = 0.0;
    *n_iter = 0;
    *converged = 0;

    /* workspace (doubles): per spin F, D, E(rr), C, K, C_occ, W and the DIIS rings; shared T1, T2, Va
     * (eigenvector / A copy), Sb (B copy), J, partials, scalars */
    const int64_t per_spin = 5 * n2 + nao * nao + nao + 2 * (int64_t)m_max * n2;
    const int64_t total = nspin * per_spin + 5 * n2 + 33 * RED_BLOCKS + 32;
    double *F[2], *D[2], *Er[2], *C[2], *K[2], *Cocc[2], *W[2], *Fring[2], *Ering[2];
    double *T1, *T2, *Va, *Sb, *J, *part, *scal;
    const unsigned eb = (unsigned)((n2 + 255) / 256);
    const dim3 tgrid((unsigned)((nao + 31) / 32), (unsigned)((nao + 31) / 32));

    if (cs.create(&sol) != CUSOLVER_STATUS_SUCCESS || cs.set_stream(sol, st) != CUSOLVER_STATUS_SUCCESS) {
        snprintf(err, errlen, "dfjk_scf: cusolverDnCreate / SetStream failed");
        rc = DFJK_ECUDA;
        goto done;
    }
    SCF_TRY(cudaMalloc((void **)&ws, (size_t)total * sizeof(double)));
    {
        double *q = ws;
        for (int s = 0; s < nspin; ++s) {
            F[s] = q; q += n2; D[s] = q; q += n2; Er[s] = q; q += n2; C[s] = q; q += n2; K[s] = q; q += n2;
            Cocc[s] = q; q += nao * nao; W[s] = q; q += nao;
            Fring[s] = q; q += (int64_t)m_max * n2; Ering[s] = q; q += (int64_t)m_max * n2;
        }
        T1 = q; q += n2; T2 = q; q += n2; Va = q; q += n2; Sb = q; q += n2; J = q; q += n2;
        part = q; q += 33 * RED_BLOCKS; scal = q;          /* scal[0..3] E, max|e| per spin; scal[4..] DIIS dots */
    }
    if (cs.sygvd_bufsize(sol, CUSOLVER_EIG_TYPE_1, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER,
                         (int)nao, Va, (int)nao, Sb, (int)nao, W[0], &lwork) != CUSOLVER_STATUS_SUCCESS) {
        snprintf(err, errlen, "dfjk_scf: cusolverDnDsygvd_bufferSize failed");
        rc = DFJK_ECUDA;
        goto done;
    }
    SCF_TRY(cudaMalloc((void **)&work, (size_t)lwork * sizeof(double)));
    SCF_TRY(cudaMalloc((void **)&dev_info, sizeof(int)));

    /* generalised symmetric eigenproblem A C = S C eps; a symmetric row-major matrix is its own
     * column-major image, the eigenvectors come back as columns of the column-major Va */
    {
        auto mark_eig = [&]() { mark_event(ev_eig, st, &timing_ok); };
        auto diagonalise = [&](const double *A, int s) -> int {
            if (cudaMemcpyAsync(Va, A, (size_t)n2 * 8, cudaMemcpyDeviceToDevice, st) != cudaSuccess) return 1;
            if (cudaMemcpyAsync(Sb, S, (size_t)n2 * 8, cudaMemcpyDeviceToDevice, st) != cudaSuccess) return 1;
            mark_eig();
            const cusolverStatus_t es = cs.sygvd(sol, CUSOLVER_EIG_TYPE_1, CUSOLVER_EIG_MODE_VECTOR,
                                                 CUBLAS_FILL_MODE_LOWER, (int)nao, Va, (int)nao, Sb, (int)nao,
                                                 W[s], work, lwork, dev_info);
            mark_eig();
            if (es != CUSOLVER_STATUS_SUCCESS) return 2;
            unpack_vectors_kernel<<<tgrid, 256, 0, st>>>(Va, nao, nocc[s], C[s], Cocc[s]);
            int info = 0;
            if (cudaMemcpyAsync(&info, dev_info, sizeof(int), cudaMemcpyDeviceToHost, st) != cudaSuccess) return 1;
            if (cudaStreamSynchronize(st) != cudaSuccess) return 1;
            return info == 0 ? 0 : 3;
        };
        auto reduce = [&](int mode, const double *a, const double *b, const double *c, double scale, double *out) {
            reduce_partial_kernel<<<RED_BLOCKS, RED_THREADS, 0, st>>>(mode, a, b, c, n2, part);
            reduce_final_kernel<<<1, 32, 0, st>>>(mode, part, scale, out);
        };
        auto read_scalars = [&](double *dst, int n) -> cudaError_t {
            cudaError_t e = cudaMemcpyAsync(dst, scal, n * sizeof(double), cudaMemcpyDeviceToHost, st);
            return e != cudaSuccess ? e : cudaStreamSynchronize(st);
        };

        /* T = A Bs for a SYMMETRIC Bs (A Bs = A Bs^T): both operands packed side by side into the X
         * workspace, one full DMMA product over all tiles with k = nao, splits summed by K3's kernel */
        const ScfWorkspace wsx = scf_workspace(h);
        const int64_t w4 = (nao + 3) / 4 * 4;
        const int nbt = (int)((nao + 127) / 128);
        const int psplit = choose_splits(nbt * nbt, wsx.sm_count, wsx.nsplit_alloc < 8 ? wsx.nsplit_alloc : 8);
        const dim3 pgrid((unsigned)((nao + 255) / 256), (unsigned)(w4 / 4));
        auto product_sym = [&](const double *A, const double *Bs, double *T) -> cudaError_t {
            pack_x4_kernel<<<pgrid, 256, 0, st>>>(A, nao, 0, wsx.X);
            pack_x4_kernel<<<pgrid, 256, 0, st>>>(Bs, nao, w4, wsx.X);
            const cudaError_t e = launch_k2_gemm_full(wsx.X, nao, 1, 2 * w4, 0, w4, nao, wsx.Kpart, psplit, 0, st);
            if (e != cudaSuccess) return e;
            launch_k3_sum(wsx.Kpart, psplit, nao, T, st);
            return cudaSuccess;
        };
        if (wsx.x_doubles < 2 * w4 * nao) {
            snprintf(err, errlen, "dfjk_scf: X workspace too small for the DIIS products");
            rc = DFJK_ENOMEM;
            goto done;
        }
        /* timing (dfjk_scf_timing): event pairs around every get_jk and every Dsygvd */
        auto mark = [&](std::vector<cudaEvent_t> &v) { mark_event(v, st, &timing_ok); };
        mark(ev_total);

        for (int s = 0; s < nspin; ++s) {                               /* 0. core guess, both spins */
            const int dr = diagonalise(hcore, s);
            if (dr != 0) {
                snprintf(err, errlen, "dfjk_scf: Dsygvd failed on the core guess (%d; S not positive definite?)", dr);
                rc = DFJK_ECUDA;
                goto done;
            }
        }
        for (int64_t k = 0; k < max_iter; ++k) {
            mark(ev_jk);
            rc = nspin == 1 ? dfjk_get_jk(h, Cocc[0], nocc[0], J, K[0], (void *)st)
                            : dfjk_get_jk_u(h, Cocc[0], nocc[0], Cocc[1], nocc[1], J, K[0], K[1], (void *)st);
            if (rc != DFJK_OK) { snprintf(err, errlen, "%s", dfjk_last_error()); goto done; }
            mark(ev_jk);
            /* the new (F, e) pair goes into the ring slot of the entry it evicts (or a fresh one) */
            int slot;
            if ((int)slot_of.size() < m_max) slot = (int)slot_of.size();
            else slot = slot_of.front();
            for (int s = 0; s < nspin; ++s) {
                fock_kernel<<<eb, 256, 0, st>>>(hcore, J, K[s], n2, F[s]);
                launch_fp64_tile_gemm(Cocc[s], nocc[s], Cocc[s], 1, nocc[s], D[s], nao, nao, nao, nocc[s], dw, 0.0, 0, st);
                reduce(1, D[s], hcore, F[s], 0.5, scal + s);            /* E_s = 1/2 sum D_s o (h + F_s) */
                SCF_TRY(product_sym(F[s], D[s], T1));                   /* F D   (D symmetric) */
                SCF_TRY(product_sym(T1, S, T2));                        /* F D S (S symmetric) */
                antisym_kernel<<<eb, 256, 0, st>>>(T2, nao, Er[s]);     /* e_s = F D S - S D F */
                reduce(2, Er[s], nullptr, nullptr, 1.0, scal + 2 + s);  /* max |e_s| */
            }
            /* the DIIS dots of this iteration against the history it WOULD have (oldest entry dropped
             * when the ring is full, the new error last), all in one launch pair, so that E, max|e| and
             * the dots come back in ONE host sync */
            std::vector<int> hist(slot_of);
            if ((int)hist.size() == m_max) hist.erase(hist.begin());
            const int m = (int)hist.size() + 1;
            {
                DotArgs da;
                da.npairs = m * nspin;
                for (int i = 0; i < m; ++i)
                    for (int s = 0; s < nspin; ++s) {
                        da.a[i * nspin + s] = i + 1 < m ? Ering[s] + (int64_t)hist[i] * n2 : Er[s];
                        da.b[i * nspin + s] = Er[s];
                    }
                dots_partial_kernel<<<dim3(RED_BLOCKS, (unsigned)da.npairs), RED_THREADS, 0, st>>>(da, n2, part);
                dots_final_kernel<<<1, 32, 0, st>>>(part, m, nspin, scal + 4);
            }
            double hs[4 + 16] = {0.0};
            SCF_TRY(read_scalars(hs, 4 + m));
            const double E = nspin == 1 ? hs[0] : hs[0] + hs[1];
            const double emax = nspin == 1 ? hs[2] : std::fmax(hs[2], hs[3]);
            e_hist[k] = E;
            *n_iter = k + 1;
            if (k > 0 && std::fabs(E - e_prev) <= conv_tol * std::fmax(1.0, std::fabs(E)) &&
                emax <= std::sqrt(conv_tol)) {
                *converged = 1;
                break;
            }
            e_prev = E;
            if (k + 1 == max_iter) break;
            /* DIIS history (oldest first) */
            if ((int)slot_of.size() == m_max) {
                slot_of.erase(slot_of.begin());
                for (int i = 0; i + 1 < m_max; ++i)
                    for (int j = 0; j + 1 < m_max; ++j) Bmat[i * m_max + j] = Bmat[(i + 1) * m_max + j + 1];
            }
            slot_of.push_back(slot);
            for (int s = 0; s < nspin; ++s) {
                SCF_TRY(cudaMemcpyAsync(Ering[s] + (int64_t)slot * n2, Er[s], (size_t)n2 * 8, cudaMemcpyDeviceToDevice, st));
                SCF_TRY(cudaMemcpyAsync(Fring[s] + (int64_t)slot * n2, F[s], (size_t)n2 * 8, cudaMemcpyDeviceToDevice, st));
            }
            for (int i = 0; i < m; ++i) Bmat[i * m_max + (m - 1)] = Bmat[(m - 1) * m_max + i] = hs[4 + i];
            std::vector<double> A((size_t)(m + 1) * (m + 1), 0.0), rhs(m + 1, 0.0);
            for (int i = 0; i < m; ++i) {
                for (int j = 0; j < m; ++j) A[i * (m + 1) + j] = Bmat[i * m_max + j];
                A[i * (m + 1) + m] = A[m * (m + 1) + i] = -1.0;
            }
            rhs[m] = -1.0;
            if (!solve_dense(A, rhs, m + 1)) {
                snprintf(err, errlen, "dfjk_scf: singular DIIS system at iteration %lld", (long long)k);
                rc = DFJK_ECUDA;
                goto done;
            }
            for (int s = 0; s < nspin; ++s) {
                Coefs cf;
                cf.m = m;
                for (int i = 0; i < m; ++i) { cf.c[i] = rhs[i]; cf.F[i] = Fring[s] + (int64_t)slot_of[i] * n2; }
                lincomb_kernel<<<eb, 256, 0, st>>>(cf, n2, T2);         /* T2 = F_s,ext */
                const int dr = diagonalise(T2, s);
                if (dr != 0) {
                    snprintf(err, errlen, "dfjk_scf: Dsygvd failed at iteration %lld (%d)", (long long)k, dr);
                    rc = DFJK_ECUDA;
                    goto done;
                }
            }
        }
        for (int s = 0; s < nspin; ++s) {
            SCF_TRY(cudaMemcpyAsync(C_out[s], C[s], (size_t)n2 * 8, cudaMemcpyDeviceToDevice, st));
            if (mo_energy_out && mo_energy_out[s])
                SCF_TRY(cudaMemcpyAsync(mo_energy_out[s], W[s], (size_t)nao * 8, cudaMemcpyDeviceToDevice, st));
            if (D_out && D_out[s]) SCF_TRY(cudaMemcpyAsync(D_out[s], D[s], (size_t)n2 * 8, cudaMemcpyDeviceToDevice, st));
            if (F_out && F_out[s]) SCF_TRY(cudaMemcpyAsync(F_out[s], F[s], (size_t)n2 * 8, cudaMemcpyDeviceToDevice, st));
        }
        SCF_TRY(cudaStreamSynchronize(st));
        SCF_TRY(cudaGetLastError());
    }
done:
    {
        /* where the time went: sums over the (begin, end) event pairs; the run has synchronised */
        if (ev_total.size() == 1) mark_event(ev_total, st, &timing_ok);
        cudaStreamSynchronize(st);
        auto total = [&timing_ok](std::vector<cudaEvent_t> &v) {
            double t = 0.0;
            if (v.size() & 1) timing_ok = false;          /* an unmatched begin */
            for (size_t i = 0; i + 1 < v.size(); i += 2) {
                float ms = 0.f;
                if (cudaEventElapsedTime(&ms, v[i], v[i + 1]) == cudaSuccess) t += ms;
                else timing_ok = false;
            }
            for (cudaEvent_t e : v) cudaEventDestroy(e);
            v.clear();
            return t;
        };
        const double t_jk = total(ev_jk), t_eig = total(ev_eig), t_all = total(ev_total);
        cudaGetLastError();
        if (rc == DFJK_OK && timing_ok) scf_store_timing(h, *n_iter, t_jk, t_eig, t_all);
    }
    if (sol) cs.destroy(sol);
    cudaFree(ws);
    cudaFree(work);
    cudaFree(dev_info);
    return rc;
}

}  // namespace dfjk
