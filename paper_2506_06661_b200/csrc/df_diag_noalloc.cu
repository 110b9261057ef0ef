/*
 * df_diag_noalloc.cu -- dfjk_df_diag_noalloc (include/dfjk.h): Eq. 7's DF diagonal
 *     diag[mu][nu] = sum_P B[P][mu nu]^2
 * for callers that must not allocate device memory.
 *
 * Who cannot allocate?  Code that runs where cudaMalloc is forbidden or would hurt: inside a
 * framework's memory pool that owns the whole device (a second allocator fragments it or fails
 * outright), under a no-allocation policy after start-up (real-time / serving loops, where
 * cudaMalloc's implicit device synchronisation stalls every other stream), or in a process that
 * has already handed all free HBM to the resident tensor B.  dfjk_create() gives the handle a
 * workspace with cudaMalloc, so the handle-based dfjk_get_df_diag is out of reach for them.
 *
 * The handle path's only scratch for this operation is Jp_part: `ngroup` partial packed
 * triangles (row group g sums the rows P = g, g + ngroup, ...), which J3 then adds in order and
 * unpacks.  Here those partials live in a file-scope device array of fixed size that is part of
 * the library image: every GPU that loads libdfjk.so carries these 8 MiB until the process
 * exits, whether or not this entry point is ever called.  The kernels are the ones of the
 * handle path (j2_axpy<SQ>, j3_unpack in j_kernels.cu), given the array's device address.
 *
 * `noalloc_scratch` below is, in HOST code, only a stand-in symbol: its host-side address is not
 * a device address (a kernel handed `noalloc_scratch` directly would fault, or scribble on host
 * memory where the GPU can reach it).  The device address comes from cudaGetSymbolAddress, asked
 * once per device with that device current, in first_use_setup().
 */
#include "../../include/dfjk.h"
#include "dfjk_internal.h"

#include <initializer_list>
#include <mutex>

namespace {

constexpr int64_t SCRATCH_DOUBLES = DFJK_NOALLOC_SCRATCH_BYTES / 8;
static_assert(DFJK_NOALLOC_SCRATCH_BYTES % 256 == 0, "whole 256-byte lines");
/* two partial triangles (the fewest j2_axpy works with) of the largest nao must fit */
static_assert((int64_t)DFJK_NOALLOC_MAX_NAO * (DFJK_NOALLOC_MAX_NAO + 1) <= SCRATCH_DOUBLES,
              "DFJK_NOALLOC_MAX_NAO does not fit DFJK_NOALLOC_SCRATCH_BYTES");

static __device__ __align__(256) double noalloc_scratch[SCRATCH_DOUBLES];

constexpr int MAX_DEVICES = 64;

struct PerDevice {
    double *scratch = nullptr;   /* device address of noalloc_scratch ON THIS device */
    int sm_count = 0;
};
PerDevice g_dev[MAX_DEVICES];
std::mutex g_dev_mutex;

/* First use on the current device: resolve the array's device address and read the SM count.
 * Neither call allocates.  The result is cached per device ordinal, so later calls on that device
 * touch no CUDA API besides cudaGetDevice and the launches. */
int first_use_setup(int dev, PerDevice *out)
{
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    if (!g_dev[dev].scratch) {
        double *p = nullptr;
        cudaError_t e = cudaGetSymbolAddress((void **)&p, noalloc_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return dfjk::set_last_error(DFJK_ECUDA, "dfjk_df_diag_noalloc: cudaGetSymbolAddress(scratch) on device %d: %s",
                                        dev, cudaGetErrorString(e));
        }
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess || sms < 1) {
            cudaGetLastError();
            return dfjk::set_last_error(DFJK_ECUDA, "dfjk_df_diag_noalloc: SM count of device %d: %s", dev,
                                        cudaGetErrorString(e));
        }
        g_dev[dev].sm_count = sms;
        g_dev[dev].scratch = p;
    }
    *out = g_dev[dev];
    return DFJK_OK;
}

}  // namespace

extern "C" int64_t dfjk_noalloc_max_nao(void) { return DFJK_NOALLOC_MAX_NAO; }

extern "C" int dfjk_df_diag_noalloc(int64_t naux, int64_t nao, const double *B_packed, double *diag,
                                    void *stream)
{
    dfjk::set_last_error(DFJK_OK, "%s", "");
    if (naux < 1 || nao < 1)
        return dfjk::set_last_error(DFJK_EINVAL, "dfjk_df_diag_noalloc: naux and nao must be >= 1");
    if (nao > DFJK_NOALLOC_MAX_NAO)
        return dfjk::set_last_error(DFJK_EINVAL,
                                    "dfjk_df_diag_noalloc: nao = %lld is beyond the built-in scratch (nao <= %d: two packed "
                                    "triangles must fit %d bytes); use dfjk_create + dfjk_get_df_diag, which allocate",
                                    (long long)nao, DFJK_NOALLOC_MAX_NAO, DFJK_NOALLOC_SCRATCH_BYTES);
    if (!B_packed || !diag) return dfjk::set_last_error(DFJK_EINVAL, "dfjk_df_diag_noalloc: NULL pointer");
    if (((uintptr_t)B_packed & 15) != 0 || ((uintptr_t)diag & 7) != 0)
        return dfjk::set_last_error(DFJK_EINVAL, "dfjk_df_diag_noalloc: B_packed must be 16-byte aligned (diag 8)");
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return dfjk::set_last_error(DFJK_ECUDA, "dfjk_df_diag_noalloc: cudaGetDevice: %s", cudaGetErrorString(e));
    }
    if (dev < 0 || dev >= MAX_DEVICES)
        return dfjk::set_last_error(DFJK_EINVAL, "dfjk_df_diag_noalloc: device ordinal %d (at most %d devices)", dev,
                                    MAX_DEVICES);
    for (const void *p : {(const void *)B_packed, (const void *)diag}) {
        cudaPointerAttributes pa;
        e = cudaPointerGetAttributes(&pa, p);
        if (e != cudaSuccess || (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged)) {
            cudaGetLastError();
            return dfjk::set_last_error(DFJK_EINVAL,
                                        "dfjk_df_diag_noalloc: B_packed / diag is not a device pointer (no CPU fallback)");
        }
        if (pa.type == cudaMemoryTypeDevice && pa.device != dev)
            return dfjk::set_last_error(DFJK_EINVAL, "dfjk_df_diag_noalloc: pointer lives on device %d, current is %d",
                                        pa.device, dev);
    }
    PerDevice pd;
    const int rc = first_use_setup(dev, &pd);
    if (rc != DFJK_OK) return rc;

    const int64_t npair = nao * (nao + 1) / 2;
    /* as many row groups as the handle path would take, cut down to what the array holds; the
     * count stays even (all rows of a group then share one 16-byte alignment class) and >= 2 */
    int64_t ngroup = dfjk::j2_num_groups(naux, npair, pd.sm_count);
    int64_t fit = SCRATCH_DOUBLES / npair;
    fit -= fit & 1;
    if (ngroup > fit) ngroup = fit;
    if (ngroup < 2)   /* unreachable while the static_assert above holds */
        return dfjk::set_last_error(DFJK_EINVAL, "dfjk_df_diag_noalloc: scratch too small for nao = %lld", (long long)nao);

    cudaStream_t st = (cudaStream_t)stream;
    /* j2_axpy<SQ> writes every element [g][0, npair) of the ngroup partials it is given, and
     * j3_unpack reads exactly those: nothing in the array has to start at zero, and whatever the
     * previous call (of any size) left behind is never read. */
    dfjk::launch_j2_axpy(B_packed, naux, npair, nullptr, pd.scratch, ngroup, st);
    dfjk::launch_j3_unpack(pd.scratch, ngroup, npair, nao, diag, nullptr, st);
    e = cudaGetLastError();
    if (e != cudaSuccess)
        return dfjk::set_last_error(DFJK_ECUDA, "dfjk_df_diag_noalloc: launch: %s", cudaGetErrorString(e));
    return DFJK_OK;
}
