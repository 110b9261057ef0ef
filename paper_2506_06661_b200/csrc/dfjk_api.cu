/*
 * dfjk_api.cu -- the C ABI of include/dfjk.h: handle, argument checks, workspace,
 * and the launch sequence of one get_jk call.  Every step of the path runs in the
 * kernels of j_kernels.cu / k1_half_transform.cu / k2_syrk.cu; there is no CPU
 * fallback (a missing device is DFJK_ECUDA).
 *
 *   J and K together (default, "j_fused"):
 *     K0 pack C -> for P-chunks: [K1 half transform -> J1X d_P from X -> K2 SYRK (per set)]
 *               -> K3 finish -> J1R reduce -> J2 axpy (the one pass over B for J) -> J3 unpack
 *   J only, or j_fused = 0:
 *     K0 -> J0 Dt -> J1 dot -> J1R -> J2 axpy -> J3  (two streaming passes over B), then the K chain
 *   general densities (get_jk_pair / _dm), building B (build_b) and the SCF driver live below.
 */
#include "../../include/dfjk.h"
#include "dfjk_internal.h"

#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <initializer_list>
#include <new>

#ifndef DFJK_X_MB
#define DFJK_X_MB 2048   /* 512 -> 2048 MB: 17 -> 5 K1/K2 launch pairs at cfg 4, -1.1 % step time */
#endif

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}

#define DFJK_CUDA_TRY(expr)                                                              \
    do {                                                                                 \
        cudaError_t e_ = (expr);                                                         \
        if (e_ != cudaSuccess)                                                           \
            return fail(DFJK_ECUDA, "%s: %s", #expr, cudaGetErrorString(e_));            \
    } while (0)

/* a launcher that reports failure (no tile shape, no shared-memory opt-in, bad launch) */
#define DFJK_LAUNCH_TRY(expr)                                                            \
    do {                                                                                 \
        cudaError_t e_ = (expr);                                                         \
        if (e_ != cudaSuccess)                                                           \
            return fail(DFJK_ECUDA, "%s: %s", who, cudaGetErrorString(e_));              \
    } while (0)

int64_t round_up(int64_t x, int64_t m) { return (x + m - 1) / m * m; }

}  // namespace

/* for the entry points that live in other translation units (df_diag_noalloc.cu): the same
 * thread-local text dfjk_last_error() returns */
int dfjk::set_last_error(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}

#define DFJK_GRAPH_SLOTS 4
#ifndef DFJK_K2P_MIN_NB
#define DFJK_K2P_MIN_NB 6   /* K2P needs enough tiles per panel: below 21 lower tiles the split kernel wins */
#endif

namespace dfjk {
/* split count that fills the SMs best: work items = ntile * s on sm_count SMs (one CTA each).
 * Whole waves matter because a CTA's duration is fixed by its k range; a small penalty per
 * split accounts for the read-modify-write of the partial tile. */
int choose_splits(int ntile, int sm_count, int max_splits)
{
    int best = 1;
    double best_score = -1.0;
    for (int s = 1; s <= max_splits; ++s) {
        const int items = ntile * s;
        const int waves = (items + sm_count - 1) / sm_count;
        const double score = (double)items / ((double)waves * sm_count) - 0.002 * s;
        if (score > best_score) { best_score = score; best = s; }
    }
    return best;
}

/* The lower-triangle split kernel: tiles are cut in proportion to their cost, s is the count of a
 * full off-diagonal tile and a CTA then lasts ~1/s of a tile; minimise waves / s (small penalty per
 * split for the partials K3 has to add). */
int choose_splits_lower(int64_t nao, int sm_count, int max_splits)
{
    int best = 1;
    double best_time = 1e300;
    for (int s = 1; s <= max_splits; ++s) {
        const int64_t items = k2_lower_items(nao, s);
        const int64_t waves = (items + sm_count - 1) / sm_count;
        const double t = (double)waves / s * (1.0 + 0.002 * s);
        if (t < best_time) { best_time = t; best = s; }
    }
    return best;
}

}  // namespace dfjk
using dfjk::choose_splits;
using dfjk::choose_splits_lower;

struct dfjk_handle {
    int64_t naux, nao, npair;
    const double *B;
    int device, sm_count;
    int64_t l2_bytes;
    /* workspace (device) */
    double *Ccat;        /* round_up(nao,32) x ldc_max, k-group-major */
    int64_t ldc_max;
    double *Dt;          /* npair */
    double *d_part;      /* nchunk x naux */
    double *d;           /* naux */
    double *d_batch;     /* DFJK_MAX_BATCH x naux: d of every density of a batched call */
    double *Jp_part;     /* j2_groups x npair */
    double *X;           /* x_doubles */
    double *Kpart;       /* 2 x nsplit_alloc x nao x nao */
    int64_t nchunk, j2_groups, x_doubles;
    int nsplit_alloc, nsplit_default;
    int nsplit_weighted; /* split kernel with per-tile split counts in proportion to tile cost (k2_tile_splits):
                            the count of a full tile, 0 if there are more lower tiles than SMs */
    int64_t opt_k2_weighted;
    int64_t ws_bytes;
    /* options */
    int64_t opt_k_chunk, opt_k_splits, opt_j_fused, opt_k2_panel, opt_k2_panel_kb;
    int *k2work;         /* 1 + nsplit_alloc * nb^2 ints: item counter and per-(slab, tile) counters of K2P */
    struct WsBuf { void *p; size_t bytes; } ws_list[12];   /* every alloc_ws buffer, for "poison_workspace" */
    int ws_count;
    bool have_d;
    /* instrumentation: launch counter and optional per-kernel CUDA-event timing */
    int64_t launches;
    int64_t opt_time_kernels;
    cudaEvent_t *ev;     /* pairs: ev[2*i], ev[2*i+1] */
    int *ev_kind;        /* which kernel pair i brackets (DFJK_KERNEL_*) */
    int ev_cap, ev_used;
    bool ev_overflow;    /* a launch went unrecorded (the ring could not grow): kernel_time reports it */
    /* replayed launch sequences of get_jk / get_jk_u (see get_jk_impl) */
    /* key: the bytes of a GraphKey (defined with get_jk_impl below), copied in and out with memcpy */
    struct GraphSlot { bool seen; alignas(8) unsigned char key[64]; cudaGraphExec_t exec; int64_t launches; };
    GraphSlot graphs[DFJK_GRAPH_SLOTS];
    int graph_next;
    int64_t opt_graph;
    cudaStream_t cap_stream;
    double **out_slots;  /* device: this call's output pointers (J, K_0, K_1), written by K0 */
    /* the last SCF run's timing (dfjk_scf_timing) */
    int64_t scf_iters;
    double scf_get_jk_ms, scf_eig_ms, scf_total_ms;
    /* host-call resources (lazy) */
    cudaStream_t host_stream;
    double *hostC, *hostJ, *hostK, *hostC2, *hostK2;
};

namespace {

void free_all(dfjk_handle *h)
{
    cudaFree(h->Ccat); cudaFree(h->Dt); cudaFree(h->d_part); cudaFree(h->d); cudaFree(h->d_batch);
    cudaFree(h->Jp_part); cudaFree(h->X); cudaFree(h->Kpart); cudaFree(h->k2work);
    cudaFree(h->hostC); cudaFree(h->hostJ); cudaFree(h->hostK); cudaFree(h->hostC2); cudaFree(h->hostK2);
    if (h->host_stream) cudaStreamDestroy(h->host_stream);
    for (auto &g : h->graphs) if (g.exec) cudaGraphExecDestroy(g.exec);
    if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
    cudaFree(h->out_slots);
    for (int i = 0; i < 2 * h->ev_cap; ++i) cudaEventDestroy(h->ev[i]);
    delete[] h->ev;
    delete[] h->ev_kind;
}

/* the event ring of "time_kernels": (re)allocate to `cap` pairs, keeping the recorded ones */
bool grow_events(dfjk_handle *h, int cap)
{
    cudaEvent_t *ev = new (std::nothrow) cudaEvent_t[2 * (size_t)cap];
    int *kind = new (std::nothrow) int[cap];
    if (!ev || !kind) { delete[] ev; delete[] kind; return false; }
    for (int i = 0; i < 2 * h->ev_cap; ++i) ev[i] = h->ev[i];
    for (int i = 0; i < h->ev_cap; ++i) kind[i] = h->ev_kind[i];
    for (int i = 2 * h->ev_cap; i < 2 * cap; ++i)
        if (cudaEventCreate(&ev[i]) != cudaSuccess) {
            cudaGetLastError();
            for (int j = 2 * h->ev_cap; j < i; ++j) cudaEventDestroy(ev[j]);
            delete[] ev; delete[] kind;
            return false;
        }
    delete[] h->ev; delete[] h->ev_kind;
    h->ev = ev; h->ev_kind = kind; h->ev_cap = cap;
    return true;
}

/* bracket one kernel launch with events when "time_kernels" is on; the ring grows on demand and a
 * launch that could not be recorded raises ev_overflow (dfjk_kernel_time then fails loudly) */
struct Timed {
    dfjk_handle *h; cudaStream_t st; int slot;
    Timed(dfjk_handle *h_, int kind, cudaStream_t st_) : h(h_), st(st_), slot(-1)
    {
        ++h->launches;
        if (!h->opt_time_kernels) return;
        if (h->ev_used == h->ev_cap && !grow_events(h, h->ev_cap > 0 ? 2 * h->ev_cap : 1024)) {
            h->ev_overflow = true;
            return;
        }
        slot = h->ev_used++;
        h->ev_kind[slot] = kind;
        cudaEventRecord(h->ev[2 * slot], st);
    }
    ~Timed() { if (slot >= 0) cudaEventRecord(h->ev[2 * slot + 1], st); }
};

int alloc_ws(dfjk_handle *h, double **p, int64_t ndoubles)
{
    const cudaError_t e = cudaMalloc((void **)p, (size_t)ndoubles * sizeof(double));
    if (e != cudaSuccess) {
        *p = nullptr;
        return fail(DFJK_ENOMEM, "cudaMalloc of %lld bytes: %s", (long long)(ndoubles * 8),
                    cudaGetErrorString(e));
    }
    h->ws_bytes += ndoubles * 8;
    if (h->ws_count < (int)(sizeof h->ws_list / sizeof h->ws_list[0]))
        h->ws_list[h->ws_count++] = {(void *)*p, (size_t)ndoubles * sizeof(double)};
    return DFJK_OK;
}

}  // namespace

extern "C" const char *dfjk_last_error(void) { return g_err; }
extern "C" const char *dfjk_version(void) { return "0.1.0"; }

extern "C" dfjk_handle *dfjk_create(int64_t naux, int64_t nao, const double *B_packed)
{
    g_err[0] = 0;
    if (naux < 1 || nao < 1) { fail(DFJK_EINVAL, "dfjk_create: naux and nao must be >= 1"); return nullptr; }
    /* 255 x 255 tiles of 128 keep every grid dimension below 65536 (one packed row is 4.3 GB there) */
    if (nao > 32640) { fail(DFJK_EINVAL, "dfjk_create: nao > 32640 is not supported"); return nullptr; }
    if (!B_packed) { fail(DFJK_EINVAL, "dfjk_create: B_packed is NULL"); return nullptr; }
    if (((uintptr_t)B_packed & 15) != 0) { fail(DFJK_EINVAL, "dfjk_create: B_packed must be 16-byte aligned"); return nullptr; }
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { fail(DFJK_ECUDA, "cudaGetDevice: %s (no CUDA device, no CPU fallback)", cudaGetErrorString(e)); return nullptr; }
    cudaPointerAttributes pa;
    e = cudaPointerGetAttributes(&pa, B_packed);
    if (e != cudaSuccess || (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged)) {
        cudaGetLastError();
        fail(DFJK_EINVAL, "dfjk_create: B_packed is not a device pointer");
        return nullptr;
    }
    dfjk_handle *h = new (std::nothrow) dfjk_handle();
    if (!h) { fail(DFJK_ENOMEM, "dfjk_create: host allocation failed"); return nullptr; }
    memset(h, 0, sizeof *h);
    h->naux = naux; h->nao = nao; h->npair = nao * (nao + 1) / 2; h->B = B_packed; h->device = dev;
    h->opt_j_fused = 1;
    h->opt_graph = 1;
    h->opt_k2_panel = 2;             /* automatic */
    h->opt_k2_weighted = 2;          /* automatic */
    h->opt_k2_panel_kb = 32768;
    int v = 0;
    cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev); h->sm_count = v > 0 ? v : 148;
    cudaDeviceGetAttribute(&v, cudaDevAttrL2CacheSize, dev); h->l2_bytes = v;

    h->ldc_max = 2 * round_up(nao, 8);
    h->nchunk = dfjk::j1_num_chunks(h->npair);
    h->j2_groups = dfjk::j2_num_groups(naux, h->npair, h->sm_count);
    /* X chunk (the half-transformed rows that live between K1 and K2), at least two rows at the
     * widest ldc */
    int64_t xd = ((int64_t)DFJK_X_MB << 20) / 8;
    if (xd < 2 * nao * h->ldc_max) xd = 2 * nao * h->ldc_max;
    if (xd > naux * nao * h->ldc_max) xd = naux * nao * h->ldc_max;
    h->x_doubles = xd;
    const int nb = (int)((nao + 127) / 128);
    h->nsplit_default = choose_splits(nb * (nb + 1) / 2, h->sm_count, 32);
    /* small problems (fewer lower tiles than SMs, X chunk L2-resident): ONE wave, balanced tile by tile;
     * up to 64 splits of a full tile while the 2 x nsplit_alloc partial-K slots stay below 512 MB */
    h->nsplit_weighted = 0;
    if (nb * (nb + 1) / 2 <= h->sm_count) {
        int max_s = (int)((512LL << 20) / (2 * nao * nao * 8));
        if (max_s > 64) max_s = 64;
        if (max_s < 8) max_s = 8;
        h->nsplit_weighted = choose_splits_lower(nao, h->sm_count, max_s);
    }
    /* partial-K slots: what the two automatic choices (lower tiles; all tiles for the general
     * product) need, at least 8 for the "k_splits" option -- 2*32 slots would be 8 GB at nao=4000 */
    h->nsplit_alloc = h->nsplit_default;
    if (h->nsplit_weighted > h->nsplit_alloc) h->nsplit_alloc = h->nsplit_weighted;
    if (choose_splits(nb * nb, h->sm_count, 32) > h->nsplit_alloc)
        h->nsplit_alloc = choose_splits(nb * nb, h->sm_count, 32);
    if (h->nsplit_alloc < 8) h->nsplit_alloc = 8;

    int rc = DFJK_OK;
    if (rc == DFJK_OK) rc = alloc_ws(h, &h->Ccat, round_up(nao, 32) * h->ldc_max);
    if (rc == DFJK_OK) rc = alloc_ws(h, &h->Dt, h->npair);
    /* d partials: J1's column chunks, or J1X's blocks at the widest ldc */
    int64_t dparts = dfjk::j1x_max_blocks(nao, h->ldc_max);
    if (dparts < h->nchunk) dparts = h->nchunk;
    if (rc == DFJK_OK) rc = alloc_ws(h, &h->d_part, dparts * naux);
    if (rc == DFJK_OK) rc = alloc_ws(h, &h->d, naux);
    if (rc == DFJK_OK) rc = alloc_ws(h, &h->d_batch, DFJK_MAX_BATCH * naux);
    if (rc == DFJK_OK) rc = alloc_ws(h, &h->Jp_part, h->j2_groups * h->npair);
    if (rc == DFJK_OK) rc = alloc_ws(h, &h->X, h->x_doubles);
    if (rc == DFJK_OK) rc = alloc_ws(h, &h->Kpart, 2LL * h->nsplit_alloc * nao * nao);
    if (rc == DFJK_OK && cudaMalloc((void **)&h->k2work, sizeof(int) * (size_t)(1 + h->nsplit_alloc * nb * nb)) != cudaSuccess) {
        h->k2work = nullptr;
        rc = fail(DFJK_ENOMEM, "dfjk_create: cudaMalloc of the K2 work counters failed");
    }
    if (rc == DFJK_OK && cudaMalloc((void **)&h->out_slots, DFJK_OUT_SLOTS * sizeof(double *)) != cudaSuccess) {
        h->out_slots = nullptr;
        rc = fail(DFJK_ENOMEM, "dfjk_create: cudaMalloc of the output-pointer slots failed");
    }
    if (rc == DFJK_OK) {   /* "poison_workspace" covers these two as well */
        h->ws_list[h->ws_count++] = {(void *)h->k2work, sizeof(int) * (size_t)(1 + h->nsplit_alloc * nb * nb)};
        h->ws_list[h->ws_count++] = {(void *)h->out_slots, DFJK_OUT_SLOTS * sizeof(double *)};
    }
    if (rc != DFJK_OK) { free_all(h); delete h; return nullptr; }
    return h;
}

extern "C" int dfjk_destroy(dfjk_handle *h)
{
    if (!h) return DFJK_OK;
    free_all(h);
    delete h;
    return DFJK_OK;
}

extern "C" int64_t dfjk_workspace_bytes(const dfjk_handle *h) { return h ? h->ws_bytes : 0; }

extern "C" int dfjk_set_option(dfjk_handle *h, const char *name, int64_t value)
{
    if (!h || !name) return fail(DFJK_EINVAL, "dfjk_set_option: NULL argument");
    if (value < 0) return fail(DFJK_EINVAL, "dfjk_set_option: negative value");
    if (!strcmp(name, "k_chunk")) { h->opt_k_chunk = value; return DFJK_OK; }
    if (!strcmp(name, "k_splits")) {
        if (value > h->nsplit_alloc) return fail(DFJK_EINVAL, "k_splits > %d allocated", h->nsplit_alloc);
        h->opt_k_splits = value; return DFJK_OK;
    }
    if (!strcmp(name, "time_kernels")) {
        if (value && !h->ev && !grow_events(h, 1024))
            return fail(DFJK_ENOMEM, "time_kernels: could not create the event ring");
        h->opt_time_kernels = value; h->ev_used = 0; h->ev_overflow = false; return DFJK_OK;
    }
    if (!strcmp(name, "j_fused")) { h->opt_j_fused = value != 0; return DFJK_OK; }
    if (!strcmp(name, "graph")) { h->opt_graph = value != 0; return DFJK_OK; }
    if (!strcmp(name, "k2_panel")) {
        if (value > 2) return fail(DFJK_EINVAL, "k2_panel must be 0, 1 or 2");
        h->opt_k2_panel = value; return DFJK_OK;
    }
    if (!strcmp(name, "k2_weighted")) {
        if (value > 2) return fail(DFJK_EINVAL, "k2_weighted must be 0, 1 or 2");
        h->opt_k2_weighted = value; return DFJK_OK;
    }
    if (!strcmp(name, "k2_panel_kb")) {
        if (value < 64 || value > (1 << 22)) return fail(DFJK_EINVAL, "k2_panel_kb must be in [64, 4194304] (KB)");
        h->opt_k2_panel_kb = value; return DFJK_OK;
    }
    if (!strcmp(name, "poison_workspace")) {
        /* test aid (tests/test_gpu_guard.py): waits for the device, then fills every workspace buffer
         * with 0xFF bytes -- NaN as doubles -- so that a kernel that reads workspace no earlier kernel
         * of the same call has written shows up as NaN in J / K instead of passing by luck */
        if (value == 0) return DFJK_OK;
        DFJK_CUDA_TRY(cudaDeviceSynchronize());
        for (int i = 0; i < h->ws_count; ++i) DFJK_CUDA_TRY(cudaMemset(h->ws_list[i].p, 0xFF, h->ws_list[i].bytes));
        DFJK_CUDA_TRY(cudaDeviceSynchronize());
        h->have_d = false;
        return DFJK_OK;
    }
    return fail(DFJK_EINVAL, "dfjk_set_option: unknown option '%s'", name);
}

/* ------------------------------------------------------------------ one build */
namespace {

/* Everything of one get_jk after K0 (the orbital packing), enqueued on `st`.  With slots != NULL
 * the finishing kernels take their output pointers from the device array K0 published them to
 * (slot 0 = J, slot 1 + s = K_s) instead of from J / K[]: the sequence then depends on the CALL only
 * through (nset, nocc, which outputs, options) and can be captured once and replayed. */
int enqueue_jk_body(dfjk_handle *h, int nset, const int *nocc, const int *col0, int64_t ldc,
                    const double *w, double *J, double *const *K, bool want_j, const bool *want_k,
                    double *const *slots, cudaStream_t st, const char *who)
{
    const int64_t nao = h->nao, naux = h->naux, npair = h->npair;
    bool any_k = false;
    for (int s = 0; s < nset; ++s) any_k = any_k || want_k[s];
    /* J and K in one call: d_P = <B_P, D> = sum_s w_s <X_P^s, C_s> is read off the half-transformed
     * X that K1 writes anyway (J1X), so B is streamed once for J (J2) instead of twice */
    const bool fused = want_j && any_k && h->opt_j_fused != 0;
    if (want_j && !fused) {
        { Timed t_(h, DFJK_KERNEL_J0, st); dfjk::launch_j0_build_dt(h->Ccat, ldc, nao, nset, col0, nocc, w, h->Dt, st); }
        { Timed t_(h, DFJK_KERNEL_J1, st); dfjk::launch_j1_dot(h->B, naux, npair, h->Dt, h->d_part, h->sm_count, st); }
        { Timed t_(h, DFJK_KERNEL_J1R, st); dfjk::launch_j1_reduce(h->d_part, h->nchunk, naux, h->d, st); }
        { Timed t_(h, DFJK_KERNEL_J2, st); dfjk::launch_j2_axpy(h->B, naux, npair, h->d, h->Jp_part, h->j2_groups, st); }
        { Timed t_(h, DFJK_KERNEL_J3, st); dfjk::launch_j3_unpack(h->Jp_part, h->j2_groups, npair, nao, J, slots ? slots + 0 : nullptr, st); }
    }

    if (any_k) {
        int64_t pc = h->x_doubles / (nao * ldc);
        if (h->opt_k_chunk > 0 && h->opt_k_chunk < pc) pc = h->opt_k_chunk;
        if (pc > naux) pc = naux;
        if (pc < 1) return fail(DFJK_ENOMEM, "%s: X workspace too small", who);
        /* K2P pays an add per item to keep the k window of X inside L2; an X chunk that fits in L2
         * whole has nothing to gain from it, and small problems are all overhead.  The slab it adds
         * into need NOT stay in L2 since the adds are `red` operations (nobody waits for the line):
         * nao = 4000, a 128 MB slab: 61.0 ms against the split kernel's 62.5 */
        const int nbk = (int)((nao + 127) / 128);
        const bool panel = h->opt_k2_panel == 1 ||
                           (h->opt_k2_panel == 2 && pc * nao * ldc * 8 > h->l2_bytes && nbk >= DFJK_K2P_MIN_NB);
        /* the split kernel balances a single wave tile by tile when the chunk of X it re-reads stays in
         * L2 (tiles then cut the k range at different places: no two CTAs stream the same lines together) */
        const bool weighted = !panel && h->nsplit_weighted > 0 && h->opt_k_splits == 0 &&
                              (h->opt_k2_weighted == 1 ||
                               (h->opt_k2_weighted == 2 && pc * nao * ldc * 8 * 10 <= h->l2_bytes * 7));
        /* K2P: panel length and slab count per set, planned from the first (largest) chunk; the old
         * split kernel: one partial per k-split */
        int nsplit[2] = {0, 0}, pstages[2] = {0, 0};
        for (int s = 0; s < nset; ++s) {
            if (panel)
                dfjk::k2p_plan(nao, pc * ((nocc[s] + 3) / 4), nbk * (nbk + 1) / 2, h->sm_count,
                               h->opt_k_splits > 0 ? (int)h->opt_k_splits : h->nsplit_alloc,
                               h->opt_k2_panel_kb << 10, &pstages[s], &nsplit[s]);
            else
                nsplit[s] = h->opt_k_splits > 0 ? (int)h->opt_k_splits : (weighted ? h->nsplit_weighted : h->nsplit_default);
        }
        int chunk = 0;
        for (int64_t P0 = 0; P0 < naux; P0 += pc, ++chunk) {
            const int64_t np = (P0 + pc <= naux) ? pc : naux - P0;
            { Timed t_(h, DFJK_KERNEL_K1, st); DFJK_LAUNCH_TRY(dfjk::launch_k1_half_transform(h->B, naux, nao, npair, P0, np, h->Ccat, ldc, ldc, h->X, st)); }
            if (fused) {
                Timed t_(h, DFJK_KERNEL_J1, st);
                dfjk::launch_j1x_dot(h->X, h->Ccat, nao, np, ldc, ldc, 0, nset, col0, nocc, w, P0, naux, h->d_part, st);
            }
            for (int s = 0; s < nset; ++s)
                if (want_k[s]) {
                    Timed t_(h, DFJK_KERNEL_K2, st);
                    double *Kp = h->Kpart + (int64_t)s * h->nsplit_alloc * nao * nao;
                    if (panel)
                        DFJK_LAUNCH_TRY(dfjk::launch_k2p_syrk_lower(h->X, nao, np, ldc, col0[s], nocc[s], Kp, pstages[s],
                                                                    nsplit[s], chunk > 0, h->k2work, h->sm_count, st));
                    else
                        DFJK_LAUNCH_TRY(dfjk::launch_k2_syrk_lower(h->X, nao, np, ldc, col0[s], nocc[s], Kp,
                                                                   nsplit[s], weighted ? 1 : 0, chunk > 0, st));
                }
        }
        for (int s = 0; s < nset; ++s)
            if (want_k[s]) {
                Timed t_(h, DFJK_KERNEL_K3, st);
                dfjk::launch_k3_finish(h->Kpart + (int64_t)s * h->nsplit_alloc * nao * nao, nsplit[s], weighted ? 1 : 0,
                                       nao, K[s], slots ? slots + 1 + s : nullptr, st);
            }
    }
    if (fused) {
        { Timed t_(h, DFJK_KERNEL_J1R, st); dfjk::launch_j1_reduce(h->d_part, dfjk::j1x_num_blocks(nao, ldc), naux, h->d, st); }
        { Timed t_(h, DFJK_KERNEL_J2, st); dfjk::launch_j2_axpy(h->B, naux, npair, h->d, h->Jp_part, h->j2_groups, st); }
        { Timed t_(h, DFJK_KERNEL_J3, st); dfjk::launch_j3_unpack(h->Jp_part, h->j2_groups, npair, nao, J, slots ? slots + 0 : nullptr, st); }
    }
    return DFJK_OK;
}

/* The launch sequence of a get_jk depends on the call only through its shape (sets, nocc, outputs,
 * options): the second call with a shape already seen captures the body into a CUDA graph, later
 * ones replay it -- one graph launch instead of 8-20 kernel launches, which is what bounds the small
 * configs (cfg 1: 17 launches = 0.15 ms for 0.03 ms of work).  K0 stays a plain launch in front: it
 * takes the call's C pointers and publishes the call's output pointers for the replayed K3 / J3. */
struct GraphKey {
    int nset, nocc[2];
    bool want_j, want_k[2];
    int64_t k_chunk, k_splits, j_fused, k2_panel, k2_panel_kb, k2_weighted;
    bool operator==(const GraphKey &o) const
    {
        if (k2_panel != o.k2_panel || k2_panel_kb != o.k2_panel_kb || k2_weighted != o.k2_weighted) return false;
        return nset == o.nset && nocc[0] == o.nocc[0] && nocc[1] == o.nocc[1] && want_j == o.want_j &&
               want_k[0] == o.want_k[0] && want_k[1] == o.want_k[1] && k_chunk == o.k_chunk &&
               k_splits == o.k_splits && j_fused == o.j_fused;
    }
};

int get_jk_impl(dfjk_handle *h, int nset, const double *const *C, const int64_t *nocc64,
                const double *w, double *J, double *const *K, cudaStream_t st, const char *who)
{
    g_err[0] = 0;
    if (!h) return fail(DFJK_EINVAL, "%s: NULL handle", who);
    bool any_k = false;
    for (int s = 0; s < nset; ++s) {
        if (!C[s]) return fail(DFJK_EINVAL, "%s: orbital pointer %d is NULL", who, s);
        if (nocc64[s] < 1 || nocc64[s] > h->nao)
            return fail(DFJK_EINVAL, "%s: nocc[%d]=%lld outside [1, nao=%lld]", who, s,
                        (long long)nocc64[s], (long long)h->nao);
        any_k = any_k || K[s] != nullptr;
    }
    if (!J && !any_k) return fail(DFJK_EINVAL, "%s: no output requested", who);
    int dev = -1;
    DFJK_CUDA_TRY(cudaGetDevice(&dev));
    if (dev != h->device) return fail(DFJK_EINVAL, "%s: handle belongs to device %d, current is %d", who, h->device, dev);

    const int64_t nao = h->nao;
    int nocc[4], col0[4];
    int64_t ldc = 0;
    for (int s = 0; s < nset; ++s) {
        nocc[s] = (int)nocc64[s];
        col0[s] = (int)ldc;
        ldc += round_up(nocc64[s], 8);
    }
    GraphKey key = {};
    key.nset = nset; key.want_j = J != nullptr;
    key.k_chunk = h->opt_k_chunk; key.k_splits = h->opt_k_splits; key.j_fused = h->opt_j_fused;
    key.k2_panel = h->opt_k2_panel; key.k2_panel_kb = h->opt_k2_panel_kb; key.k2_weighted = h->opt_k2_weighted;
    bool want_k[2] = {false, false};
    for (int s = 0; s < nset; ++s) { key.nocc[s] = nocc[s]; key.want_k[s] = want_k[s] = K[s] != nullptr; }

    /* graph replay is for plain calls only: not while the per-kernel event brackets are on, and not
     * inside someone else's capture (there the launches simply join the caller's graph) */
    bool use_graph = h->opt_graph != 0 && h->opt_time_kernels == 0;
    if (use_graph) {
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(st, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) {
            cudaGetLastError();
            use_graph = false;
        }
    }
    dfjk_handle::GraphSlot *slot = nullptr;
    bool first_of_shape = false;
    if (use_graph) {
        for (auto &g : h->graphs) {
            if (!g.seen) continue;
            GraphKey k;
            static_assert(sizeof(GraphKey) <= sizeof(g.key), "GraphSlot::key too small");
            memcpy(&k, g.key, sizeof k);
            if (k == key) { slot = &g; break; }
        }
        first_of_shape = slot == nullptr;   /* launched plainly; remembered below once it has succeeded */
    }

    /* K0: zero-padded concatenation [C_0 | C_1], each set padded to a multiple of 8 columns; it also
     * publishes this call's output pointers (slot 0 = J, 1 + s = K_s) */
    double *outs[DFJK_OUT_SLOTS] = {J, nset > 0 ? K[0] : nullptr, nset > 1 ? K[1] : nullptr, nullptr};
    { Timed t_(h, DFJK_KERNEL_K0, st); dfjk::launch_k0_pack_c(C, nocc, col0, nset, nao, ldc, h->Ccat, outs, h->out_slots, st); }

    if (slot && !slot->exec) {
        /* second call of this shape: capture the body on the handle's own stream */
        if (!h->cap_stream) DFJK_CUDA_TRY(cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking));
        const int64_t launches0 = h->launches;
        cudaGraph_t graph = nullptr;
        DFJK_CUDA_TRY(cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal));
        const int rc = enqueue_jk_body(h, nset, nocc, col0, ldc, w, nullptr, K, J != nullptr, want_k,
                                       h->out_slots, h->cap_stream, who);
        const cudaError_t ec = cudaStreamEndCapture(h->cap_stream, &graph);
        slot->launches = h->launches - launches0;
        h->launches = launches0;
        if (rc != DFJK_OK) { if (graph) cudaGraphDestroy(graph); cudaGetLastError(); return rc; }
        if (ec != cudaSuccess) { cudaGetLastError(); return fail(DFJK_ECUDA, "%s: stream capture: %s", who, cudaGetErrorString(ec)); }
        const cudaError_t ei = cudaGraphInstantiate(&slot->exec, graph, 0);
        cudaGraphDestroy(graph);
        if (ei != cudaSuccess) { slot->exec = nullptr; cudaGetLastError(); return fail(DFJK_ECUDA, "%s: cudaGraphInstantiate: %s", who, cudaGetErrorString(ei)); }
    }
    if (slot) {
        DFJK_CUDA_TRY(cudaGraphLaunch(slot->exec, st));
        h->launches += slot->launches;
    } else {
        const int rc = enqueue_jk_body(h, nset, nocc, col0, ldc, w, J, K, J != nullptr, want_k, nullptr, st, who);
        if (rc != DFJK_OK) return rc;
    }
    if (J) h->have_d = true;
    DFJK_CUDA_TRY(cudaGetLastError());
    if (first_of_shape) {
        /* first successful call of this shape: remember it (round-robin over the slots) */
        dfjk_handle::GraphSlot *ns = &h->graphs[h->graph_next];
        h->graph_next = (h->graph_next + 1) % DFJK_GRAPH_SLOTS;
        if (ns->exec) { cudaGraphExecDestroy(ns->exec); ns->exec = nullptr; }
        memcpy(ns->key, &key, sizeof key);
        ns->seen = true;
    }
    return DFJK_OK;
}


/* general density: dm = C1 C2^T (pair form) or dm = C1 with C2 == NULL (raw nao x nao matrix,
 * built as the pair (dm, I)).  J = J[dm], K = K[dm] = sum_P (B_P C1)(B_P C2)^T, both linear. */
int get_jk_general_impl(dfjk_handle *h, const double *C1, const double *C2, int64_t ncol,
                        double *J, double *K, cudaStream_t st, const char *who)
{
    g_err[0] = 0;
    if (!h) return fail(DFJK_EINVAL, "%s: NULL handle", who);
    if (!C1) return fail(DFJK_EINVAL, "%s: density / factor pointer is NULL", who);
    if (ncol < 1 || ncol > h->nao)
        return fail(DFJK_EINVAL, "%s: ncol=%lld outside [1, nao=%lld]", who, (long long)ncol, (long long)h->nao);
    if (!J && !K) return fail(DFJK_EINVAL, "%s: no output requested", who);
    int dev = -1;
    DFJK_CUDA_TRY(cudaGetDevice(&dev));
    if (dev != h->device) return fail(DFJK_EINVAL, "%s: handle belongs to device %d, current is %d", who, h->device, dev);

    const int64_t nao = h->nao, naux = h->naux, npair = h->npair;
    /* pair form with J and K in one call: d_P = <B_P, C1 C2^T> = <B_P C1, C2> is read off X (J1X) */
    const bool fused = J && K && C2 != nullptr && h->opt_j_fused != 0;
    if (J && !fused) {
        { Timed t_(h, DFJK_KERNEL_J0, st); dfjk::launch_j0_general_dt(C1, C2, ncol, nao, h->Dt, st); }
        { Timed t_(h, DFJK_KERNEL_J1, st); dfjk::launch_j1_dot(h->B, naux, npair, h->Dt, h->d_part, h->sm_count, st); }
        { Timed t_(h, DFJK_KERNEL_J1R, st); dfjk::launch_j1_reduce(h->d_part, h->nchunk, naux, h->d, st); }
        { Timed t_(h, DFJK_KERNEL_J2, st); dfjk::launch_j2_axpy(h->B, naux, npair, h->d, h->Jp_part, h->j2_groups, st); }
        { Timed t_(h, DFJK_KERNEL_J3, st); dfjk::launch_j3_unpack(h->Jp_part, h->j2_groups, npair, nao, J, nullptr, st); }
        h->have_d = true;
    }
    if (K) {
        /* X chunk columns [0, w8) = B_P C1 and [w8, 2 w8) = B_P C2.  Pair form: one half transform
         * over Ccat = [C1 | C2].  Raw dm (C2 == NULL, the pair (dm, I)): the half transform runs over
         * Ccat = [dm] only and the identity half, B_P itself, is unpacked straight into X (K1U). */
        const bool raw = C2 == nullptr;
        const double *Cp[2] = {C1, C2};
        const int nocc[2] = {(int)ncol, (int)ncol};
        const int64_t w8 = round_up(ncol, 8);
        const int col0[2] = {0, (int)w8};
        const int64_t ldx = 2 * w8, ldc = raw ? w8 : ldx;
        { Timed t_(h, DFJK_KERNEL_K0, st); dfjk::launch_k0_pack_c(Cp, nocc, col0, raw ? 1 : 2, nao, ldc, h->Ccat, nullptr, nullptr, st); }
        int64_t pc = h->x_doubles / (nao * ldx);
        if (h->opt_k_chunk > 0 && h->opt_k_chunk < pc) pc = h->opt_k_chunk;
        if (pc > naux) pc = naux;
        if (pc > 65535) pc = 65535;                /* K1U's grid.z */
        if (pc < 1) return fail(DFJK_ENOMEM, "%s: X workspace too small", who);
        const int nb = (int)((nao + 127) / 128);
        const bool panel = h->opt_k2_panel == 1 ||
                           (h->opt_k2_panel == 2 && pc * nao * ldx * 8 > h->l2_bytes && nb >= DFJK_K2P_MIN_NB - 1);
        int nsplit = h->opt_k_splits > 0 ? (int)h->opt_k_splits
                                         : choose_splits(nb * nb, h->sm_count, h->nsplit_alloc);
        int pstages = 0;
        if (panel)
            dfjk::k2p_plan(nao, pc * ((ncol + 3) / 4), nb * nb, h->sm_count,
                           h->opt_k_splits > 0 ? (int)h->opt_k_splits : h->nsplit_alloc,
                           h->opt_k2_panel_kb << 10, &pstages, &nsplit);
        int chunk = 0;
        for (int64_t P0 = 0; P0 < naux; P0 += pc, ++chunk) {
            const int64_t np = (P0 + pc <= naux) ? pc : naux - P0;
            { Timed t_(h, DFJK_KERNEL_K1, st); DFJK_LAUNCH_TRY(dfjk::launch_k1_half_transform(h->B, naux, nao, npair, P0, np, h->Ccat, ldc, ldx, h->X, st)); }
            if (raw) { Timed t_(h, DFJK_KERNEL_K1, st); dfjk::launch_k1u_unpack(h->B, nao, npair, P0, np, ldx, w8, h->X, st); }
            if (fused) {
                const double one = 1.0;
                Timed t_(h, DFJK_KERNEL_J1, st);
                dfjk::launch_j1x_dot(h->X, h->Ccat, nao, np, ldx, ldc, w8, 1, col0, nocc, &one, P0, naux, h->d_part, st);
            }
            { Timed t_(h, DFJK_KERNEL_K2, st);
              if (panel)
                  DFJK_LAUNCH_TRY(dfjk::launch_k2p_gemm_full(h->X, nao, np, ldx, col0[0], col0[1], ncol, h->Kpart, pstages,
                                                             nsplit, chunk > 0, h->k2work, h->sm_count, st));
              else
                  DFJK_LAUNCH_TRY(dfjk::launch_k2_gemm_full(h->X, nao, np, ldx, col0[0], col0[1], ncol, h->Kpart, nsplit, chunk > 0, st)); }
        }
        { Timed t_(h, DFJK_KERNEL_K3, st); dfjk::launch_k3_sum(h->Kpart, nsplit, nao, K, st); }
        if (fused) {
            { Timed t_(h, DFJK_KERNEL_J1R, st); dfjk::launch_j1_reduce(h->d_part, dfjk::j1x_num_blocks(nao, ldc), naux, h->d, st); }
            { Timed t_(h, DFJK_KERNEL_J2, st); dfjk::launch_j2_axpy(h->B, naux, npair, h->d, h->Jp_part, h->j2_groups, st); }
            { Timed t_(h, DFJK_KERNEL_J3, st); dfjk::launch_j3_unpack(h->Jp_part, h->j2_groups, npair, nao, J, nullptr, st); }
            h->have_d = true;
        }
    }
    DFJK_CUDA_TRY(cudaGetLastError());
    return DFJK_OK;
}

}  // namespace

extern "C" int dfjk_get_jk_pair(dfjk_handle *h, const double *C1, const double *C2, int64_t ncol,
                                double *J, double *K, void *stream)
{
    if (!C2) { g_err[0] = 0; return fail(DFJK_EINVAL, "dfjk_get_jk_pair: C2 is NULL"); }
    return get_jk_general_impl(h, C1, C2, ncol, J, K, (cudaStream_t)stream, "dfjk_get_jk_pair");
}

extern "C" int dfjk_get_jk_dm(dfjk_handle *h, const double *dm, double *J, double *K, void *stream)
{
    return get_jk_general_impl(h, dm, nullptr, h ? h->nao : 1, J, K, (cudaStream_t)stream, "dfjk_get_jk_dm");
}

namespace {

/* The Coulomb matrices of nb <= DFJK_MAX_BATCH densities whose fitting coefficients d_k[P] already sit in
 * h->d_batch: ONE pass over B carries all of them (launch_j2_axpy_multi), the partial triangles live in the
 * X workspace, which is idle at this point of a call.  Falls back to one pass per density only when the X
 * workspace cannot hold nb x j2_groups partial triangles. */
int batched_j_from_d(dfjk_handle *h, int nb, double *const *Js, cudaStream_t st)
{
    const int64_t nao = h->nao, naux = h->naux, npair = h->npair;
    const int64_t per = h->j2_groups * npair;
    if ((int64_t)nb * per <= h->x_doubles) {
        { Timed t_(h, DFJK_KERNEL_J2, st); dfjk::launch_j2_axpy_multi(h->B, naux, npair, h->d_batch, nb, h->X, h->j2_groups, st); }
        for (int i = 0; i < nb; ++i) {
            Timed t_(h, DFJK_KERNEL_J3, st);
            dfjk::launch_j3_unpack(h->X + i * per, h->j2_groups, npair, nao, Js[i], nullptr, st);
        }
    } else {
        for (int i = 0; i < nb; ++i) {
            { Timed t_(h, DFJK_KERNEL_J2, st); dfjk::launch_j2_axpy(h->B, naux, npair, h->d_batch + i * naux, h->Jp_part, h->j2_groups, st); }
            { Timed t_(h, DFJK_KERNEL_J3, st); dfjk::launch_j3_unpack(h->Jp_part, h->j2_groups, npair, nao, Js[i], nullptr, st); }
        }
    }
    return DFJK_OK;
}

/* d_k = <B_P, dm_k> by a streaming pass over B per density (J0 general -> J1 -> J1R into d_batch[k]) */
void d_by_pass_over_b(dfjk_handle *h, int k, const double *C1, const double *C2, int64_t ncol, cudaStream_t st)
{
    { Timed t_(h, DFJK_KERNEL_J0, st); dfjk::launch_j0_general_dt(C1, C2, ncol, h->nao, h->Dt, st); }
    { Timed t_(h, DFJK_KERNEL_J1, st); dfjk::launch_j1_dot(h->B, h->naux, h->npair, h->Dt, h->d_part, h->sm_count, st); }
    { Timed t_(h, DFJK_KERNEL_J1R, st); dfjk::launch_j1_reduce(h->d_part, h->nchunk, h->naux, h->d_batch + (int64_t)k * h->naux, st); }
}

/* One sub-batch (nb <= DFJK_MAX_BATCH) of dfjk_get_jk_pairs.  K: the factors of as many pairs as fit
 * ldc_max columns are packed side by side, ONE half transform (K1) per X chunk serves them all; per pair
 * d_P is read off its columns of X (J1X) and its full product (K2) is added to K_i chunk by chunk.
 * J: one multi-right-hand-side pass over B for the whole sub-batch. */
int pairs_subbatch(dfjk_handle *h, int nb, const double *const *C1s, const double *const *C2s,
                   const int64_t *ncols, double *const *Js, double *const *Ks, cudaStream_t st, const char *who)
{
    const int64_t nao = h->nao, naux = h->naux, npair = h->npair;
    const bool want_j = Js != nullptr, want_k = Ks != nullptr;
    const bool fused = want_j && want_k && h->opt_j_fused != 0;
    if (want_j && !fused)
        for (int i = 0; i < nb; ++i) d_by_pass_over_b(h, i, C1s[i], C2s[i], ncols[i], st);
    if (want_k) {
        const int nbk = (int)((nao + 127) / 128);
        int i0 = 0;
        while (i0 < nb) {
            int i1 = i0;
            int64_t ldc = 0, col1[DFJK_MAX_BATCH], w8[DFJK_MAX_BATCH];
            while (i1 < nb && ldc + 2 * round_up(ncols[i1], 8) <= h->ldc_max) {
                w8[i1] = round_up(ncols[i1], 8);
                col1[i1] = ldc;
                ldc += 2 * w8[i1];
                ++i1;
            }
            for (int i = i0; i < i1; ++i) {
                { Timed t_(h, DFJK_KERNEL_K0, st); dfjk::launch_k0_pack_cols(C1s[i], ncols[i], col1[i], w8[i], nao, ldc, h->Ccat, st); }
                { Timed t_(h, DFJK_KERNEL_K0, st); dfjk::launch_k0_pack_cols(C2s[i], ncols[i], col1[i] + w8[i], w8[i], nao, ldc, h->Ccat, st); }
            }
            int64_t pc = h->x_doubles / (nao * ldc);
            if (h->opt_k_chunk > 0 && h->opt_k_chunk < pc) pc = h->opt_k_chunk;
            if (pc > naux) pc = naux;
            if (pc < 1) return fail(DFJK_ENOMEM, "%s: X workspace too small", who);
            bool panel[DFJK_MAX_BATCH];
            int nsplit[DFJK_MAX_BATCH], pstages[DFJK_MAX_BATCH];
            for (int i = i0; i < i1; ++i) {
                panel[i] = h->opt_k2_panel == 1 ||
                           (h->opt_k2_panel == 2 && pc * nao * ldc * 8 > h->l2_bytes && nbk >= DFJK_K2P_MIN_NB - 1);
                nsplit[i] = h->opt_k_splits > 0 ? (int)h->opt_k_splits : choose_splits(nbk * nbk, h->sm_count, h->nsplit_alloc);
                pstages[i] = 0;
            }
            const int64_t nblk = dfjk::j1x_num_blocks(nao, ldc);
            int chunk = 0;
            for (int64_t P0 = 0; P0 < naux; P0 += pc, ++chunk) {
                const int64_t np = (P0 + pc <= naux) ? pc : naux - P0;
                { Timed t_(h, DFJK_KERNEL_K1, st); DFJK_LAUNCH_TRY(dfjk::launch_k1_half_transform(h->B, naux, nao, npair, P0, np, h->Ccat, ldc, ldc, h->X, st)); }
                for (int i = i0; i < i1; ++i) {
                    const int c1 = (int)col1[i], c2 = (int)(col1[i] + w8[i]), nc = (int)ncols[i];
                    if (fused) {
                        const double one = 1.0;
                        { Timed t_(h, DFJK_KERNEL_J1, st);
                          dfjk::launch_j1x_dot(h->X, h->Ccat, nao, np, ldc, ldc, w8[i], 1, &c1, &nc, &one, P0, naux, h->d_part, st); }
                        { Timed t_(h, DFJK_KERNEL_J1R, st);
                          dfjk::launch_j1_reduce_rows(h->d_part, nblk, naux, P0, np, h->d_batch + (int64_t)i * naux, st); }
                    }
                    /* every (chunk, pair) product starts its slabs afresh (accumulate = 0) and is summed into
                     * K_i right away, so the panel plan is made for THIS chunk's row count: a short last
                     * chunk must not leave slabs unwritten that K3 would then add */
                    if (panel[i])
                        dfjk::k2p_plan(nao, np * ((ncols[i] + 3) / 4), nbk * nbk, h->sm_count,
                                       h->opt_k_splits > 0 ? (int)h->opt_k_splits : h->nsplit_alloc,
                                       h->opt_k2_panel_kb << 10, &pstages[i], &nsplit[i]);
                    { Timed t_(h, DFJK_KERNEL_K2, st);
                      if (panel[i])
                          DFJK_LAUNCH_TRY(dfjk::launch_k2p_gemm_full(h->X, nao, np, ldc, c1, c2, nc, h->Kpart, pstages[i],
                                                                     nsplit[i], 0, h->k2work, h->sm_count, st));
                      else
                          DFJK_LAUNCH_TRY(dfjk::launch_k2_gemm_full(h->X, nao, np, ldc, c1, c2, nc, h->Kpart, nsplit[i], 0, st)); }
                    { Timed t_(h, DFJK_KERNEL_K3, st); dfjk::launch_k3_sum(h->Kpart, nsplit[i], nao, Ks[i], st, chunk > 0); }
                }
            }
            i0 = i1;
        }
    }
    if (want_j) {
        const int rc = batched_j_from_d(h, nb, Js, st);
        if (rc != DFJK_OK) return rc;
    }
    DFJK_CUDA_TRY(cudaGetLastError());
    return DFJK_OK;
}

}  // namespace

extern "C" int dfjk_get_jk_pairs(dfjk_handle *h, int64_t nbatch, const double *const *C1s,
                                 const double *const *C2s, const int64_t *ncols, double *const *Js,
                                 double *const *Ks, void *stream)
{
    const char *who = "dfjk_get_jk_pairs";
    g_err[0] = 0;
    if (!h) return fail(DFJK_EINVAL, "%s: NULL handle", who);
    if (nbatch < 1) return fail(DFJK_EINVAL, "%s: nbatch must be >= 1", who);
    if (!C1s || !C2s || !ncols) return fail(DFJK_EINVAL, "%s: NULL factor / ncols array", who);
    if (!Js && !Ks) return fail(DFJK_EINVAL, "%s: no output requested", who);
    for (int64_t i = 0; i < nbatch; ++i) {
        if (!C1s[i] || !C2s[i]) return fail(DFJK_EINVAL, "%s: factor pointer %lld is NULL", who, (long long)i);
        if (ncols[i] < 1 || ncols[i] > h->nao)
            return fail(DFJK_EINVAL, "%s: ncols[%lld]=%lld outside [1, nao=%lld]", who, (long long)i,
                        (long long)ncols[i], (long long)h->nao);
        if ((Js && !Js[i]) || (Ks && !Ks[i]))
            return fail(DFJK_EINVAL, "%s: output pointer %lld is NULL (pass a NULL array to skip J or K)", who, (long long)i);
    }
    int dev = -1;
    DFJK_CUDA_TRY(cudaGetDevice(&dev));
    if (dev != h->device) return fail(DFJK_EINVAL, "%s: handle belongs to device %d, current is %d", who, h->device, dev);
    for (int64_t b0 = 0; b0 < nbatch; b0 += DFJK_MAX_BATCH) {
        const int nb = (int)(nbatch - b0 < DFJK_MAX_BATCH ? nbatch - b0 : DFJK_MAX_BATCH);
        const int rc = pairs_subbatch(h, nb, C1s + b0, C2s + b0, ncols + b0, Js ? Js + b0 : nullptr,
                                      Ks ? Ks + b0 : nullptr, (cudaStream_t)stream, who);
        if (rc != DFJK_OK) return rc;
    }
    return DFJK_OK;
}

extern "C" int dfjk_get_jk_dms(dfjk_handle *h, int64_t ndm, const double *dms, double *Js, double *Ks,
                               void *stream)
{
    const char *who = "dfjk_get_jk_dms";
    g_err[0] = 0;
    if (!h) return fail(DFJK_EINVAL, "%s: NULL handle", who);
    if (ndm < 1) return fail(DFJK_EINVAL, "%s: ndm must be >= 1", who);
    if (!dms) return fail(DFJK_EINVAL, "%s: density / factor pointer is NULL", who);
    if (!Js && !Ks) return fail(DFJK_EINVAL, "%s: no output requested", who);
    int dev = -1;
    DFJK_CUDA_TRY(cudaGetDevice(&dev));
    if (dev != h->device) return fail(DFJK_EINVAL, "%s: handle belongs to device %d, current is %d", who, h->device, dev);
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t n2 = h->nao * h->nao;
    for (int64_t b0 = 0; b0 < ndm; b0 += DFJK_MAX_BATCH) {
        const int nb = (int)(ndm - b0 < DFJK_MAX_BATCH ? ndm - b0 : DFJK_MAX_BATCH);
        if (Js) {
            /* J of the whole sub-batch: a dot pass per density, then ONE axpy pass over B for all of them
             * (nb + 1 passes instead of 2 nb) */
            double *Jp[DFJK_MAX_BATCH];
            for (int i = 0; i < nb; ++i) {
                d_by_pass_over_b(h, i, dms + (b0 + i) * n2, nullptr, h->nao, st);
                Jp[i] = Js + (b0 + i) * n2;
            }
            const int rc = batched_j_from_d(h, nb, Jp, st);
            if (rc != DFJK_OK) return rc;
            DFJK_CUDA_TRY(cudaGetLastError());
        }
        if (Ks)   /* K[dm] as the pair (dm, I): 4 naux nao^3 flop each, FP64-bound -- nothing to share but B's unpack */
            for (int i = 0; i < nb; ++i) {
                const int rc = get_jk_general_impl(h, dms + (b0 + i) * n2, nullptr, h->nao, nullptr, Ks + (b0 + i) * n2, st, who);
                if (rc != DFJK_OK) return rc;
            }
    }
    return DFJK_OK;
}

extern "C" int dfjk_get_jk(dfjk_handle *h, const double *C_occ, int64_t nocc, double *J, double *K,
                           void *stream)
{
    const double *C[1] = {C_occ};
    const int64_t no[1] = {nocc};
    const double w[1] = {2.0};
    double *Ks[1] = {K};
    return get_jk_impl(h, 1, C, no, w, J, Ks, (cudaStream_t)stream, "dfjk_get_jk");
}

extern "C" int dfjk_get_jk_u(dfjk_handle *h, const double *C_a, int64_t nocc_a, const double *C_b,
                             int64_t nocc_b, double *J, double *K_a, double *K_b, void *stream)
{
    const double *C[2] = {C_a, C_b};
    const int64_t no[2] = {nocc_a, nocc_b};
    const double w[2] = {1.0, 1.0};
    double *Ks[2] = {K_a, K_b};
    return get_jk_impl(h, 2, C, no, w, J, Ks, (cudaStream_t)stream, "dfjk_get_jk_u");
}

extern "C" int dfjk_probe_dmma_peak(double *tflops)
{
    g_err[0] = 0;
    if (!tflops) return fail(DFJK_EINVAL, "dfjk_probe_dmma_peak: NULL pointer");
    int dev = 0, sms = 0;
    DFJK_CUDA_TRY(cudaGetDevice(&dev));
    DFJK_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double *sink = nullptr;
    DFJK_CUDA_TRY(cudaMalloc((void **)&sink, sizeof(double)));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int ctas = 8 * sms, iters = 20000;
    dfjk::launch_fp64_peak_probe(ctas, 2000, sink, 0);            /* warm-up */
    double best = 0.0;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(e0, 0);
        dfjk::launch_fp64_peak_probe(ctas, iters, sink, 0);
        cudaEventRecord(e1, 0);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double tf = dfjk::fp64_peak_probe_flops(ctas, iters) / (ms * 1e-3) / 1e12;
        if (tf > best) best = tf;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(sink);
    DFJK_CUDA_TRY(cudaGetLastError());
    *tflops = best;
    return DFJK_OK;
}

namespace dfjk {
ScfWorkspace scf_workspace(dfjk_handle *h)
{
    return ScfWorkspace{h->X, h->x_doubles, h->Kpart, h->nsplit_alloc, h->sm_count};
}
void scf_store_timing(dfjk_handle *h, int64_t iters, double get_jk_ms, double eig_ms, double total_ms)
{
    h->scf_iters = iters; h->scf_get_jk_ms = get_jk_ms; h->scf_eig_ms = eig_ms; h->scf_total_ms = total_ms;
}
}  // namespace dfjk

extern "C" int dfjk_scf_timing(const dfjk_handle *h, int64_t *iters, double *get_jk_ms, double *eig_ms,
                               double *other_ms)
{
    g_err[0] = 0;
    if (!h) return fail(DFJK_EINVAL, "dfjk_scf_timing: NULL handle");
    if (h->scf_iters <= 0) return fail(DFJK_EINVAL, "dfjk_scf_timing: no timing on record (no SCF has run on this handle, or the last run failed or could not record its events)");
    if (iters) *iters = h->scf_iters;
    if (get_jk_ms) *get_jk_ms = h->scf_get_jk_ms;
    if (eig_ms) *eig_ms = h->scf_eig_ms;
    if (other_ms) *other_ms = h->scf_total_ms - h->scf_get_jk_ms - h->scf_eig_ms;
    return DFJK_OK;
}

extern "C" int dfjk_device_info(int *sm_count, int *sm_clock_khz, int64_t *l2_bytes)
{
    g_err[0] = 0;
    int dev = 0, v = 0;
    DFJK_CUDA_TRY(cudaGetDevice(&dev));
    if (sm_count) { DFJK_CUDA_TRY(cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev)); *sm_count = v; }
    if (sm_clock_khz) { DFJK_CUDA_TRY(cudaDeviceGetAttribute(&v, cudaDevAttrClockRate, dev)); *sm_clock_khz = v; }
    if (l2_bytes) { DFJK_CUDA_TRY(cudaDeviceGetAttribute(&v, cudaDevAttrL2CacheSize, dev)); *l2_bytes = v; }
    return DFJK_OK;
}

extern "C" int dfjk_scf_rhf(dfjk_handle *h, const double *hcore, const double *S, int64_t nocc,
                            int64_t max_iter, double conv_tol, int64_t diis_space, double *C,
                            double *mo_energy, double *D, double *F, double *e_hist, int64_t *n_iter,
                            int *converged, void *stream)
{
    g_err[0] = 0;
    if (!h) return fail(DFJK_EINVAL, "dfjk_scf_rhf: NULL handle");
    if (!hcore || !S || !C || !e_hist || !n_iter || !converged)
        return fail(DFJK_EINVAL, "dfjk_scf_rhf: NULL pointer");
    if (nocc < 1 || nocc > h->nao) return fail(DFJK_EINVAL, "dfjk_scf_rhf: nocc outside [1, nao]");
    if (max_iter < 1) return fail(DFJK_EINVAL, "dfjk_scf_rhf: max_iter must be >= 1");
    if (diis_space < 1 || diis_space > 16) return fail(DFJK_EINVAL, "dfjk_scf_rhf: diis_space outside [1, 16]");
    if (!(conv_tol > 0.0)) return fail(DFJK_EINVAL, "dfjk_scf_rhf: conv_tol must be positive");
    if (h->nao > 32768) return fail(DFJK_EINVAL, "dfjk_scf_rhf: nao too large for the dense eigensolver");
    int dev = -1;
    DFJK_CUDA_TRY(cudaGetDevice(&dev));
    if (dev != h->device) return fail(DFJK_EINVAL, "dfjk_scf_rhf: handle belongs to device %d, current is %d", h->device, dev);
    const int64_t no[1] = {nocc};
    double *Cs[1] = {C}, *Ws[1] = {mo_energy}, *Ds[1] = {D}, *Fs[1] = {F};
    return dfjk::scf_run(h, h->nao, 1, hcore, S, no, max_iter, conv_tol, diis_space, Cs, Ws, Ds, Fs,
                         e_hist, n_iter, converged, (cudaStream_t)stream, g_err, sizeof g_err);
}

extern "C" int dfjk_scf_uhf(dfjk_handle *h, const double *hcore, const double *S, int64_t nocc_a,
                            int64_t nocc_b, int64_t max_iter, double conv_tol, int64_t diis_space,
                            double *C_a, double *C_b, double *mo_energy_a, double *mo_energy_b,
                            double *D_a, double *D_b, double *e_hist, int64_t *n_iter, int *converged,
                            void *stream)
{
    g_err[0] = 0;
    if (!h) return fail(DFJK_EINVAL, "dfjk_scf_uhf: NULL handle");
    if (!hcore || !S || !C_a || !C_b || !e_hist || !n_iter || !converged)
        return fail(DFJK_EINVAL, "dfjk_scf_uhf: NULL pointer");
    if (nocc_a < 1 || nocc_a > h->nao || nocc_b < 1 || nocc_b > h->nao)
        return fail(DFJK_EINVAL, "dfjk_scf_uhf: nocc outside [1, nao]");
    if (max_iter < 1) return fail(DFJK_EINVAL, "dfjk_scf_uhf: max_iter must be >= 1");
    if (diis_space < 1 || diis_space > 16) return fail(DFJK_EINVAL, "dfjk_scf_uhf: diis_space outside [1, 16]");
    if (!(conv_tol > 0.0)) return fail(DFJK_EINVAL, "dfjk_scf_uhf: conv_tol must be positive");
    if (h->nao > 32768) return fail(DFJK_EINVAL, "dfjk_scf_uhf: nao too large for the dense eigensolver");
    int dev = -1;
    DFJK_CUDA_TRY(cudaGetDevice(&dev));
    if (dev != h->device) return fail(DFJK_EINVAL, "dfjk_scf_uhf: handle belongs to device %d, current is %d", h->device, dev);
    const int64_t no[2] = {nocc_a, nocc_b};
    double *Cs[2] = {C_a, C_b}, *Ws[2] = {mo_energy_a, mo_energy_b}, *Ds[2] = {D_a, D_b}, *Fs[2] = {nullptr, nullptr};
    return dfjk::scf_run(h, h->nao, 2, hcore, S, no, max_iter, conv_tol, diis_space, Cs, Ws, Ds, Fs,
                         e_hist, n_iter, converged, (cudaStream_t)stream, g_err, sizeof g_err);
}

extern "C" int dfjk_build_b(int64_t naux, int64_t nao, double *M, double *R_packed, int64_t *info,
                            void *stream)
{
    g_err[0] = 0;
    if (naux < 1 || nao < 1 || nao > 46340) return fail(DFJK_EINVAL, "dfjk_build_b: naux and nao must be >= 1");
    if (!M || !R_packed) return fail(DFJK_EINVAL, "dfjk_build_b: NULL pointer");
    if (((uintptr_t)R_packed & 15) != 0 || ((uintptr_t)M & 15) != 0)
        return fail(DFJK_EINVAL, "dfjk_build_b: M and R_packed must be 16-byte aligned");
    for (const void *p : {(const void *)M, (const void *)R_packed}) {
        cudaPointerAttributes pa;
        const cudaError_t e = cudaPointerGetAttributes(&pa, p);
        if (e != cudaSuccess || (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged)) {
            cudaGetLastError();
            return fail(DFJK_EINVAL, "dfjk_build_b: M / R_packed is not a device pointer (no CPU fallback)");
        }
    }
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t npair = nao * (nao + 1) / 2;
    double *ws = nullptr;
    const size_t bytes = (size_t)dfjk::build_b_workspace_doubles(naux) * sizeof(double);
    cudaError_t e = cudaMallocAsync((void **)&ws, bytes, st);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(DFJK_ENOMEM, "dfjk_build_b: cudaMallocAsync of %zu bytes: %s", bytes, cudaGetErrorString(e));
    }
    static_assert(sizeof(long long) == sizeof(int64_t), "info is a 64-bit flag");
    e = dfjk::launch_build_b(naux, npair, M, R_packed, ws, (long long *)info, st);
    cudaFreeAsync(ws, st);
    if (e != cudaSuccess) return fail(DFJK_ECUDA, "dfjk_build_b: %s", cudaGetErrorString(e));
    return DFJK_OK;
}

extern "C" int dfjk_get_df_diag(dfjk_handle *h, double *diag, void *stream)
{
    g_err[0] = 0;
    if (!h || !diag) return fail(DFJK_EINVAL, "dfjk_get_df_diag: NULL argument");
    int dev = -1;
    DFJK_CUDA_TRY(cudaGetDevice(&dev));
    if (dev != h->device) return fail(DFJK_EINVAL, "dfjk_get_df_diag: handle belongs to device %d, current is %d", h->device, dev);
    cudaStream_t st = (cudaStream_t)stream;
    { Timed t_(h, DFJK_KERNEL_J2, st); dfjk::launch_j2_axpy(h->B, h->naux, h->npair, nullptr, h->Jp_part, h->j2_groups, st); }
    { Timed t_(h, DFJK_KERNEL_J3, st); dfjk::launch_j3_unpack(h->Jp_part, h->j2_groups, h->npair, h->nao, diag, nullptr, st); }
    DFJK_CUDA_TRY(cudaGetLastError());
    return DFJK_OK;
}

extern "C" int dfjk_get_d(dfjk_handle *h, double *d_out, void *stream)
{
    g_err[0] = 0;
    if (!h || !d_out) return fail(DFJK_EINVAL, "dfjk_get_d: NULL argument");
    if (!h->have_d) return fail(DFJK_EINVAL, "dfjk_get_d: no J has been built on this handle");
    DFJK_CUDA_TRY(cudaMemcpyAsync(d_out, h->d, (size_t)h->naux * 8, cudaMemcpyDeviceToDevice,
                                  (cudaStream_t)stream));
    return DFJK_OK;
}

namespace {

/* Lazy resources of the host entry points: a stream and device staging buffers for C, J, K (and a
 * second C, K for the unrestricted call), kept until destroy.  Nothing is published in the handle
 * unless everything was obtained: a failed first call leaves the handle exactly as it was, and
 * the device check comes first so the resources can never be bound to a foreign device. */
int host_resources(dfjk_handle *h, bool second_set, const char *who)
{
    int dev = -1;
    DFJK_CUDA_TRY(cudaGetDevice(&dev));
    if (dev != h->device) return fail(DFJK_EINVAL, "%s: handle belongs to device %d, current is %d", who, h->device, dev);
    const size_t bytes = (size_t)h->nao * h->nao * sizeof(double);
    if (!h->host_stream) {
        cudaStream_t s = nullptr;
        double *p[3] = {nullptr, nullptr, nullptr};
        cudaError_t e = cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking);
        for (int i = 0; i < 3 && e == cudaSuccess; ++i) e = cudaMalloc((void **)&p[i], bytes);
        if (e != cudaSuccess) {
            cudaGetLastError();
            for (double *q : p) cudaFree(q);
            if (s) cudaStreamDestroy(s);
            return fail(DFJK_ENOMEM, "%s: staging resources (3 x %zu bytes): %s", who, bytes, cudaGetErrorString(e));
        }
        h->hostC = p[0]; h->hostJ = p[1]; h->hostK = p[2];
        h->ws_bytes += 3 * (int64_t)bytes;
        h->host_stream = s;                       /* published last */
    }
    if (second_set && !h->hostC2) {
        double *p[2] = {nullptr, nullptr};
        cudaError_t e = cudaSuccess;
        for (int i = 0; i < 2 && e == cudaSuccess; ++i) e = cudaMalloc((void **)&p[i], bytes);
        if (e != cudaSuccess) {
            cudaGetLastError();
            for (double *q : p) cudaFree(q);
            return fail(DFJK_ENOMEM, "%s: staging resources (2 x %zu bytes): %s", who, bytes, cudaGetErrorString(e));
        }
        h->hostK2 = p[1];
        h->ws_bytes += 2 * (int64_t)bytes;
        h->hostC2 = p[0];                         /* published last */
    }
    return DFJK_OK;
}

}  // namespace

extern "C" int dfjk_get_jk_host(dfjk_handle *h, const double *C_occ_host, int64_t nocc,
                                double *J_host, double *K_host)
{
    g_err[0] = 0;
    if (!h) return fail(DFJK_EINVAL, "dfjk_get_jk_host: NULL handle");
    if (!C_occ_host) return fail(DFJK_EINVAL, "dfjk_get_jk_host: C_occ_host is NULL");
    if (nocc < 1 || nocc > h->nao) return fail(DFJK_EINVAL, "dfjk_get_jk_host: nocc outside [1, nao]");
    if (!J_host && !K_host) return fail(DFJK_EINVAL, "dfjk_get_jk_host: no output requested");
    const int64_t n2 = h->nao * h->nao;
    { const int rc0 = host_resources(h, false, "dfjk_get_jk_host"); if (rc0 != DFJK_OK) return rc0; }
    cudaStream_t st = h->host_stream;
    DFJK_CUDA_TRY(cudaMemcpyAsync(h->hostC, C_occ_host, (size_t)h->nao * nocc * 8, cudaMemcpyHostToDevice, st));
    const int rc = dfjk_get_jk(h, h->hostC, nocc, J_host ? h->hostJ : nullptr,
                               K_host ? h->hostK : nullptr, st);
    if (rc != DFJK_OK) return rc;
    if (J_host) DFJK_CUDA_TRY(cudaMemcpyAsync(J_host, h->hostJ, (size_t)n2 * 8, cudaMemcpyDeviceToHost, st));
    if (K_host) DFJK_CUDA_TRY(cudaMemcpyAsync(K_host, h->hostK, (size_t)n2 * 8, cudaMemcpyDeviceToHost, st));
    DFJK_CUDA_TRY(cudaStreamSynchronize(st));
    return DFJK_OK;
}

extern "C" int dfjk_get_jk_u_host(dfjk_handle *h, const double *C_a_host, int64_t nocc_a,
                                  const double *C_b_host, int64_t nocc_b, double *J_host,
                                  double *K_a_host, double *K_b_host)
{
    g_err[0] = 0;
    if (!h) return fail(DFJK_EINVAL, "dfjk_get_jk_u_host: NULL handle");
    if (!C_a_host || !C_b_host) return fail(DFJK_EINVAL, "dfjk_get_jk_u_host: orbital pointer is NULL");
    if (nocc_a < 1 || nocc_a > h->nao || nocc_b < 1 || nocc_b > h->nao)
        return fail(DFJK_EINVAL, "dfjk_get_jk_u_host: nocc outside [1, nao]");
    if (!J_host && !K_a_host && !K_b_host) return fail(DFJK_EINVAL, "dfjk_get_jk_u_host: no output requested");
    const int64_t n2 = h->nao * h->nao;
    { const int rc0 = host_resources(h, true, "dfjk_get_jk_u_host"); if (rc0 != DFJK_OK) return rc0; }
    cudaStream_t st = h->host_stream;
    DFJK_CUDA_TRY(cudaMemcpyAsync(h->hostC, C_a_host, (size_t)h->nao * nocc_a * 8, cudaMemcpyHostToDevice, st));
    DFJK_CUDA_TRY(cudaMemcpyAsync(h->hostC2, C_b_host, (size_t)h->nao * nocc_b * 8, cudaMemcpyHostToDevice, st));
    const int rc = dfjk_get_jk_u(h, h->hostC, nocc_a, h->hostC2, nocc_b, J_host ? h->hostJ : nullptr,
                                 K_a_host ? h->hostK : nullptr, K_b_host ? h->hostK2 : nullptr, st);
    if (rc != DFJK_OK) return rc;
    if (J_host) DFJK_CUDA_TRY(cudaMemcpyAsync(J_host, h->hostJ, (size_t)n2 * 8, cudaMemcpyDeviceToHost, st));
    if (K_a_host) DFJK_CUDA_TRY(cudaMemcpyAsync(K_a_host, h->hostK, (size_t)n2 * 8, cudaMemcpyDeviceToHost, st));
    if (K_b_host) DFJK_CUDA_TRY(cudaMemcpyAsync(K_b_host, h->hostK2, (size_t)n2 * 8, cudaMemcpyDeviceToHost, st));
    DFJK_CUDA_TRY(cudaStreamSynchronize(st));
    return DFJK_OK;
}

extern "C" int64_t dfjk_launch_count(const dfjk_handle *h) { return h ? h->launches : 0; }

extern "C" int dfjk_kernel_time(dfjk_handle *h, int kernel, double *ms_total, int64_t *count)
{
    g_err[0] = 0;
    if (!h || !ms_total || !count) return fail(DFJK_EINVAL, "dfjk_kernel_time: NULL argument");
    if (kernel < 0 || kernel >= DFJK_KERNEL_COUNT) return fail(DFJK_EINVAL, "dfjk_kernel_time: bad kernel id");
    if (h->ev_overflow)
        return fail(DFJK_ENOMEM, "dfjk_kernel_time: the event ring could not grow, some launches since the last "
                                 "set_option(time_kernels) were not recorded");
    double tot = 0.0;
    int64_t n = 0;
    for (int i = 0; i < h->ev_used; ++i) {
        if (h->ev_kind[i] != kernel) continue;
        DFJK_CUDA_TRY(cudaEventSynchronize(h->ev[2 * i + 1]));
        float ms = 0.f;
        DFJK_CUDA_TRY(cudaEventElapsedTime(&ms, h->ev[2 * i], h->ev[2 * i + 1]));
        tot += ms;
        ++n;
    }
    *ms_total = tot;
    *count = n;
    return DFJK_OK;
}
