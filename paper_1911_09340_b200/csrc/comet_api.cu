// comet_api.cu -- C ABI of include/comet.h on top of the sm_100a kernels (argument checks,
// workspace, launches).  No torch types, no exceptions, no host synchronisation in the
// device-buffer entry points.
#include "../../include/comet.h"

#include <cuda_runtime.h>
#include <math.h>
#include <mutex>
#include <new>
#include <stdio.h>
#include <string.h>

#include "common.cuh"
#include "dca.cuh"
#include "extrapolate.cuh"
#include "select.cuh"
#include "scan_fused.cuh"
#include "scan_zgroup.cuh"
#include "scan_zrun.cuh"
#include "scan_small.cuh"
#include "refine.cuh"
#include "turns.cuh"
#include "hough.cuh"
#include "half.cuh"
#include "seedgrid.cuh"

static_assert(COMET_SEL_CK == COMET_FUSED_CK, "select.cuh steps the states between the checkpoints of scan_fused.cuh");

#ifndef COMET_PRUNED_WT
#define COMET_PRUNED_WT 3
#endif
#define COMET_TEV_RING 64
#define COMET_MAX_LANES 8
#ifndef COMET_DEFAULT_LANES
#define COMET_DEFAULT_LANES 6
#endif
#ifndef COMET_ZG_MIN_CHUNKS
#define COMET_ZG_MIN_CHUNKS 1024
#endif
#define COMET_PR_CAP_S 96      // sub-block samples staged in shared memory per chunk (72 KB)

using namespace comet;

struct comet_ctx {
    int device;
    int last_cuda;
    int opt_coarse;
    int opt_stats;
    int opt_timing;
    int n_sm;
    cudaEvent_t tev[COMET_TEV_RING][5];   // COMET_OPT_TIMING: around (k_gen_unique,) the coarse / scan kernel, the fine kernel, k_rss_sum
    long long tev_count;         // timed comet_dca_rss slabs since the option was set / last read
    unsigned long long* stats;   // device [ST_N] work counters of the pruned kernels
    // pair workspace of the pruned path: shortlisted state and e^2 per (wire, seed)
    int32_t* kb;
    double* e2;
    unsigned long long* items;   // [pair_cap / 32] work list of k_fine
    unsigned int* n_items;       // [COMET_MAX_LANES][4] per internal stream lane: items listed, items handed out by k_fine_ck
    // comet_scan_rss runs the sub-slabs of a slab concurrently: scan kernels on ls[], the fine stage on
    // the high-priority lf[] so that its CTAs take the slots retiring scan CTAs free
    int opt_lanes;
    int opt_zgroup;              // 1 (default): seeds in z-runs go through the ZG kernels (scan_zgroup.cuh)
    int lanes_set;               // COMET_OPT_LANES was set by the caller
    int* ref_fb;                 // [COMET_MAX_PARTITIONS] k_select_refs_short: the partition needs the full rule
    unsigned int* zg_flag;       // [COMET_MAX_LANES] run length found by k_zgroup_check
    double* ub;                  // distinct transverse tracks of a slab (k_gen_unique)
    size_t ub_bytes;
    int32_t* npu;
    size_t npu_bytes;
    cudaStream_t ls[COMET_MAX_LANES], lf[COMET_MAX_LANES];
    cudaEvent_t ev_fork, ev_scan[COMET_MAX_LANES], ev_join[COMET_MAX_LANES];
    int fine_blocks;             // persistent grid of k_fine
    size_t pair_cap;             // pairs e2 / items hold
    size_t kb_cap;               // pairs kb holds (allocated on the first pruned comet_dca_rss)
    size_t pair_max;             // growth limit (larger problems are processed in seed slabs)
    // fused path: checkpoints [chunks][n_ck][6][32] and n_pts when the caller does not want them
    double* ck;
    size_t ck_bytes;
    size_t ck_max;               // growth limit of the checkpoint workspace
    int32_t* npw;
    size_t npw_cap;
    double* cw;                  // [slab seeds] curvature constant c of every seed (fused path)
    size_t cw_bytes;
    double* tw;                  // T_z per seed of a slab (ZG variants)
    size_t tw_bytes;
    unsigned int* tmk;           // [chunks][ceil(W / 32)] rows of the pair workspace that exist (scan_zrun.cuh)
    size_t tm_bytes;
    int fused_smem;
    FieldMap field;              // field.B == nullptr: uniform field (the bz_tesla arguments)
    double* bmax;                // device scalar: largest |B| of the map
    // device workspace
    double* wt;            // wire table [15][wt_cap]
    float* wtf;            // single-precision shortlist fields [11][wt_cap]
    int32_t wt_cap;
    double* pv;            // argmin partials [MAX_PART][SPLIT]
    int64_t* pi;
    // host-buffer entry point workspace (grown on demand)
    void* hbuf;            // one device slab for the event's inputs and outputs
    size_t hbuf_bytes;
    void* tbuf;            // track slab
    size_t tbuf_bytes;
    // the comet_scan_rss call whose distinct transverse tracks are still in `ub`, one slab, run length promised: the
    // classification of the winners copies their rows instead of stepping them again (select.cuh)
    // (valid = 2: uniform field, plain kernels: the (x, T) checkpoints of every 4th recorded state are still in `ck`)
    struct {
        const double* seeds;
        int64_t stride, n_seeds;
        double qkb, step, r_stop;
        int32_t n_steps, zshift, u_rows, n_ck, valid;
    } last;
    // events in flight through comet_scan_event_grid_submit / _collect: per slot one device slab (inputs, seeds, rss,
    // results), one pinned host staging buffer of the same input / result layout (one copy in, one copy out per event)
    // and the event that marks the results' arrival
    struct EventSlot {
        void* dbuf; size_t dbuf_bytes;
        void* hstage; size_t hstage_bytes;
        cudaEvent_t done;
        int pending;
        size_t in_bytes, o_out, out_bytes, o_bs, o_br, o_bd, o_cls, o_rss;
        int32_t n_part, n_fired, n_hits;
        int64_t n_seeds;
    } slot[COMET_EVENT_SLOTS];
    // detector geometry kept on the device for the host-buffer entry points (comet_set_geometry)
    double* geom_a;
    double* geom_b;
    int32_t geom_n;
};

#define CU(ctx, call)                                  \
    do {                                               \
        cudaError_t e__ = (call);                      \
        if (e__ != cudaSuccess) {                      \
            (ctx)->last_cuda = (int)e__;               \
            return COMET_ECUDA;                        \
        }                                              \
    } while (0)

static int set_device(comet_ctx* ctx)
{
    CU(ctx, cudaSetDevice(ctx->device));
    return COMET_OK;
}

extern "C" const char* comet_status_string(int status)
{
    switch (status) {
        case COMET_OK: return "ok";
        case COMET_EINVAL: return "invalid argument";
        case COMET_ENOMEM: return "out of memory";
        case COMET_ECUDA: return "CUDA runtime error";
        case COMET_ELIMIT: return "size beyond the limit of the statically allocated scratch";
        default: return "unknown status";
    }
}

extern "C" int comet_last_cuda_error(const comet_ctx* ctx) { return ctx ? ctx->last_cuda : 0; }

extern "C" int comet_create(comet_ctx** out, int cuda_device)
{
    if (!out || cuda_device < 0) return COMET_EINVAL;
    *out = nullptr;
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || cuda_device >= n_dev) return COMET_ECUDA;
    comet_ctx* ctx = new (std::nothrow) comet_ctx();
    if (!ctx) return COMET_ENOMEM;
    memset(ctx, 0, sizeof(*ctx));
    ctx->device = cuda_device;
    ctx->opt_coarse = COMET_COARSE_PRUNED;
    cudaError_t e = cudaSetDevice(cuda_device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->n_sm, cudaDevAttrMultiProcessorCount, cuda_device);
    ctx->wt_cap = 8192;
    if (e == cudaSuccess) e = cudaMalloc(&ctx->wt, sizeof(double) * COMET_WT_FIELDS * (size_t)ctx->wt_cap);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->wtf, sizeof(float) * 11 * (size_t)ctx->wt_cap);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->pv, sizeof(double) * COMET_MAX_PARTITIONS * COMET_ARGMIN_SPLIT);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->pi, sizeof(int64_t) * COMET_MAX_PARTITIONS * COMET_ARGMIN_SPLIT);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->stats, sizeof(unsigned long long) * ST_N);
    if (e == cudaSuccess) e = cudaMemset(ctx->stats, 0, sizeof(unsigned long long) * ST_N);
    ctx->pair_max = (size_t)1 << 29;                        // 4 GiB of pair keys: configs[3] (4.2e8 pairs) is one slab
    ctx->ck_max = (size_t)8 << 30;
    ctx->fused_smem = ((COMET_FUSED_WFIELDS + 1) * COMET_FUSED_WCAP + COMET_FUSED_WARPS * COMET_FUSED_TR * 3 * COMET_LANES) * (int)sizeof(double);
    {
        const void* fk[6] = {(const void*)k_scan_fused<false, false>, (const void*)k_scan_fused<true, false>,
                             (const void*)k_scan_fused<false, true>, (const void*)k_scan_fused<true, true>,
                             (const void*)k_scan_fused<false, true, true>, (const void*)k_scan_fused<true, true, true>};
        for (int j = 0; j < 6 && e == cudaSuccess; ++j) {
            e = cudaFuncSetAttribute(fk[j], cudaFuncAttributeMaxDynamicSharedMemorySize, ctx->fused_smem);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(fk[j], cudaFuncAttributePreferredSharedMemoryCarveout, 100);
        }
    }
    if (e == cudaSuccess) e = cudaMalloc(&ctx->bmax, sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->n_items, sizeof(unsigned int) * 4 * COMET_MAX_LANES);
    ctx->opt_lanes = COMET_DEFAULT_LANES;
    ctx->opt_zgroup = 1;
    if (e == cudaSuccess) e = cudaMalloc(&ctx->zg_flag, sizeof(unsigned int) * (COMET_MAX_LANES + 1));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->ref_fb, sizeof(int) * COMET_MAX_PARTITIONS);
    {
        int prio_lo = 0, prio_hi = 0;
        if (e == cudaSuccess) e = cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);
        for (int l = 0; l < COMET_MAX_LANES && e == cudaSuccess; ++l) {
            e = cudaStreamCreateWithPriority(&ctx->ls[l], cudaStreamNonBlocking, prio_lo);
            if (e == cudaSuccess) e = cudaStreamCreateWithPriority(&ctx->lf[l], cudaStreamNonBlocking, prio_hi);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_scan[l], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_join[l], cudaEventDisableTiming);
        }
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming);
    }
    if (e == cudaSuccess) {
        int per_sm = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_fine<false>, COMET_FINE_THREADS, 0);
        ctx->fine_blocks = ctx->n_sm * (per_sm > 0 ? per_sm : 1);
    }
    const int pr_smem = COMET_PR_CAP_S * 3 * COMET_LANES * (int)sizeof(double);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_coarse_pruned<COMET_PRUNED_WT, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, pr_smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_coarse_pruned<COMET_PRUNED_WT, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, pr_smem);
    for (int j = 0; j < COMET_TEV_RING * 5 && e == cudaSuccess; ++j) e = cudaEventCreate(&ctx->tev[j / 5][j % 5]);
    // shared-memory opt-ins (done once here, never on the hot path)
#define COMET_ZRUN_OPTIN(NU)                                                                                                   \
    do {                                                                                                                       \
        const int zs = COMET_ZR_SMEM(NU, COMET_ZR_WCAP, false), zb = COMET_ZR_SMEM(NU, ctx->wt_cap, true);                     \
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_scan_zrun<false, NU, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, zs); \
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_scan_zrun<false, NU, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, zb);  \
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_scan_zrun<true, NU, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, zs);  \
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_scan_zrun<true, NU, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, zb);   \
    } while (0)
    COMET_ZRUN_OPTIN(1);
    COMET_ZRUN_OPTIN(2);
    COMET_ZRUN_OPTIN(4);
#undef COMET_ZRUN_OPTIN
    const int dca_smem = (2 * COMET_KT * 3 * COMET_LANES + COMET_DCA_WARPS * 4 * 32) * (int)sizeof(double);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_dca_rss<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, dca_smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_dca_rss<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, dca_smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_dca_rss<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, dca_smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_dca_rss<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, dca_smem);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_select_classify<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (COMET_MAX_STEPS + 1) * 6 * (int)sizeof(double));
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_select_classify<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (COMET_MAX_STEPS_FIELD + 1) * 7 * (int)sizeof(double));
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_classify_seeds<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (COMET_MAX_STEPS_FIELD + 1) * 7 * (int)sizeof(double));
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_select_refs_cluster<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 COMET_REF_SMEM_MAX * (int)sizeof(double));
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_classify_seeds<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (COMET_MAX_STEPS + 1) * 6 * (int)sizeof(double));
    if (e != cudaSuccess) {
        cudaFree(ctx->wt); cudaFree(ctx->wtf); cudaFree(ctx->pv); cudaFree(ctx->pi); cudaFree(ctx->stats); cudaFree(ctx->n_items);
        delete ctx;
        return e == cudaErrorMemoryAllocation ? COMET_ENOMEM : COMET_ECUDA;
    }
    *out = ctx;
    return COMET_OK;
}

extern "C" int comet_destroy(comet_ctx* ctx)
{
    if (!ctx) return COMET_EINVAL;
    cudaSetDevice(ctx->device);
    cudaFree(ctx->wt); cudaFree(ctx->wtf); cudaFree(ctx->pv); cudaFree(ctx->pi); cudaFree(ctx->stats);
    cudaFree(ctx->kb); cudaFree(ctx->e2); cudaFree(ctx->items); cudaFree(ctx->n_items); cudaFree(ctx->zg_flag); cudaFree(ctx->ref_fb); cudaFree(ctx->ub); cudaFree(ctx->npu);
    for (int j = 0; j < COMET_TEV_RING * 5; ++j) if (ctx->tev[j / 5][j % 5]) cudaEventDestroy(ctx->tev[j / 5][j % 5]);
    cudaFree(ctx->geom_a); cudaFree(ctx->geom_b);
    for (int q = 0; q < COMET_EVENT_SLOTS; ++q) {
        if (ctx->slot[q].hstage) cudaFreeHost(ctx->slot[q].hstage);
        cudaFree(ctx->slot[q].dbuf);
        if (ctx->slot[q].done) cudaEventDestroy(ctx->slot[q].done);
    }
    cudaFree(ctx->hbuf); cudaFree(ctx->tbuf); cudaFree(ctx->ck); cudaFree(ctx->npw); cudaFree(ctx->cw); cudaFree(ctx->tw); cudaFree(ctx->tmk); cudaFree(ctx->bmax);
    for (int l = 0; l < COMET_MAX_LANES; ++l) {
        if (ctx->ls[l]) cudaStreamDestroy(ctx->ls[l]);
        if (ctx->lf[l]) cudaStreamDestroy(ctx->lf[l]);
        if (ctx->ev_scan[l]) cudaEventDestroy(ctx->ev_scan[l]);
        if (ctx->ev_join[l]) cudaEventDestroy(ctx->ev_join[l]);
    }
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    delete ctx;
    return COMET_OK;
}

extern "C" int comet_set_option(comet_ctx* ctx, int option, int value)
{
    if (!ctx) return COMET_EINVAL;
    if (option == COMET_OPT_COARSE_SEARCH && (value == COMET_COARSE_EXHAUSTIVE || value == COMET_COARSE_PRUNED)) {
        ctx->opt_coarse = value;
        return COMET_OK;
    }
    if (option == COMET_OPT_STATS && (value == 0 || value == 1)) {
        ctx->opt_stats = value;
        return COMET_OK;
    }
    if (option == COMET_OPT_ZGROUP && value >= 0 && value <= 2) {
        ctx->opt_zgroup = value;
        return COMET_OK;
    }
    if (option == COMET_OPT_LANES && value >= 1 && value <= COMET_MAX_LANES) {
        ctx->opt_lanes = value;
        ctx->lanes_set = 1;
        return COMET_OK;
    }
    if (option == COMET_OPT_TIMING && (value == 0 || value == 1)) {
        ctx->opt_timing = value;
        ctx->tev_count = 0;
        return COMET_OK;
    }
    return COMET_EINVAL;
}

extern "C" int comet_get_option(const comet_ctx* ctx, int option, int* value)
{
    if (!ctx || !value) return COMET_EINVAL;
    if (option == COMET_OPT_COARSE_SEARCH) { *value = ctx->opt_coarse; return COMET_OK; }
    if (option == COMET_OPT_STATS) { *value = ctx->opt_stats; return COMET_OK; }
    if (option == COMET_OPT_LANES) { *value = ctx->opt_lanes; return COMET_OK; }
    if (option == COMET_OPT_ZGROUP) { *value = ctx->opt_zgroup; return COMET_OK; }
    if (option == COMET_OPT_TIMING) { *value = ctx->opt_timing; return COMET_OK; }
    return COMET_EINVAL;
}

extern "C" int comet_read_timing(comet_ctx* ctx, float* ms_host, int32_t n, int32_t* n_calls)
{
    if (!ctx || !ms_host || n < 0 || n > 4) return COMET_EINVAL;
    if (ctx->tev_count <= 0) return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    const long long have = ctx->tev_count < COMET_TEV_RING ? ctx->tev_count : COMET_TEV_RING;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    for (long long r = ctx->tev_count - have; r < ctx->tev_count; ++r) {
        cudaEvent_t* ev = ctx->tev[r % COMET_TEV_RING];
        CU(ctx, cudaEventSynchronize(ev[4]));
        // slots: coarse / scan kernel, fine kernel, k_rss_sum, then k_gen_unique (0 when it did not run)
        const int a0[4] = {1, 2, 3, 0};
        for (int j = 0; j < n; ++j) {
            float ms = 0.f;
            CU(ctx, cudaEventElapsedTime(&ms, ev[a0[j]], ev[a0[j] + 1]));
            acc[j] += ms;
        }
    }
    for (int j = 0; j < n; ++j) ms_host[j] = (float)(acc[j] / (double)have);
    if (n_calls) *n_calls = (int32_t)have;
    ctx->tev_count = 0;
    return COMET_OK;
}

extern "C" int comet_read_stats(comet_ctx* ctx, uint64_t* out_host, int32_t n, int32_t reset, void* cuda_stream)
{
    if (!ctx || !out_host || n < 0 || n > ST_N) return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CU(ctx, cudaMemcpyAsync(out_host, ctx->stats, sizeof(uint64_t) * (size_t)n, cudaMemcpyDeviceToHost, st));
    if (reset) CU(ctx, cudaMemsetAsync(ctx->stats, 0, sizeof(unsigned long long) * ST_N, st));
    CU(ctx, cudaStreamSynchronize(st));
    return COMET_OK;
}

static inline int64_t n_chunks_of(int64_t n_seeds) { return (n_seeds + COMET_LANES - 1) / COMET_LANES; }

// grows the pair workspace to hold `pairs` (seed, wire) pairs (synchronises when it reallocates)
static int ensure_pairs(comet_ctx* ctx, size_t pairs, bool need_kb)
{
    if (pairs > ctx->pair_cap) {
        CU(ctx, cudaDeviceSynchronize());
        cudaFree(ctx->kb); cudaFree(ctx->e2); cudaFree(ctx->items);
        ctx->kb = nullptr; ctx->e2 = nullptr; ctx->items = nullptr; ctx->pair_cap = 0; ctx->kb_cap = 0;
        cudaError_t e = cudaMalloc(&ctx->e2, sizeof(double) * pairs);
        if (e == cudaSuccess) e = cudaMalloc(&ctx->items, sizeof(unsigned long long) * (pairs / COMET_LANES + 1));
        if (e != cudaSuccess) {
            ctx->last_cuda = (int)e;
            cudaFree(ctx->e2); ctx->e2 = nullptr;
            cudaFree(ctx->items); ctx->items = nullptr;
            cudaGetLastError();
            return COMET_ENOMEM;
        }
        ctx->pair_cap = pairs;
    }
    // the shortlisted-state buffer is used by the materialised pruned path only
    if (need_kb && ctx->kb_cap < ctx->pair_cap) {
        CU(ctx, cudaDeviceSynchronize());
        cudaFree(ctx->kb);
        ctx->kb = nullptr; ctx->kb_cap = 0;
        cudaError_t e = cudaMalloc(&ctx->kb, sizeof(int32_t) * ctx->pair_cap);
        if (e != cudaSuccess) { ctx->last_cuda = (int)e; cudaGetLastError(); return COMET_ENOMEM; }
        ctx->kb_cap = ctx->pair_cap;
    }
    return COMET_OK;
}

extern "C" int comet_reserve(comet_ctx* ctx, int64_t max_pairs_per_launch)
{
    if (!ctx || max_pairs_per_launch < COMET_LANES) return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    ctx->pair_max = (size_t)max_pairs_per_launch;
    return ensure_pairs(ctx, ctx->pair_max, false);
}

extern "C" size_t comet_track_bytes(int64_t n_seeds, int32_t n_steps)
{
    if (n_seeds < 0 || n_steps < 1 || n_steps > COMET_MAX_STEPS) return 0;
    return 2 * sizeof(double) * track_row(n_chunks_of(n_seeds), track_rows(n_steps), 0);
}

static inline double* plane_X(void* track) { return (double*)track; }
static inline double* plane_T(void* track, int64_t n_seeds, int32_t n_steps)
{
    return (double*)track + track_row(n_chunks_of(n_seeds), track_rows(n_steps), 0);
}

// COMET_MAX_STEPS_FIELD (comet.h): the classification kernels hold 7 doubles per state in shared memory

// |B| maximum of a field map -> *out (one CTA; runs once per comet_set_field)
__global__ void __launch_bounds__(1024) k_field_bmax(const double* __restrict__ B, int64_t n_nodes, double* out)
{
    __shared__ double sm[32];
    double m = 0.0;
    for (int64_t i = threadIdx.x; i < n_nodes; i += blockDim.x) {
        const double b0 = B[3 * i], b1 = B[3 * i + 1], b2 = B[3 * i + 2];
        m = fmax(m, sqrt(b0 * b0 + b1 * b1 + b2 * b2));
    }
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_down_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 32; ++w) m = fmax(m, sm[w]);
        *out = m * 1.000001;
    }
}

extern "C" int comet_set_field(comet_ctx* ctx, const double* field_dev, const int32_t* n_nodes, const double* origin_cm,
                               const double* spacing_cm, double rkn_tol_cm, void* cuda_stream)
{
    if (!ctx) return COMET_EINVAL;
    if (!field_dev) { ctx->field.B = nullptr; return COMET_OK; }
    if (!n_nodes || !origin_cm || !spacing_cm || !(rkn_tol_cm > 0.0)) return COMET_EINVAL;
    int64_t nodes = 1;
    for (int a = 0; a < 3; ++a) {
        if (n_nodes[a] < 2 || n_nodes[a] > 4096 || !(spacing_cm[a] > 0.0) || !isfinite(spacing_cm[a]) || !isfinite(origin_cm[a]))
            return COMET_EINVAL;
        nodes *= n_nodes[a];
    }
    int rc = set_device(ctx);
    if (rc) return rc;
    FieldMap F;
    F.B = field_dev;
    for (int a = 0; a < 3; ++a) { F.n[a] = n_nodes[a]; F.o[a] = origin_cm[a]; F.d[a] = spacing_cm[a]; }
    F.tol = rkn_tol_cm;
    F.tol32 = rkn_tol_cm / 32.0;
    F.pow2 = 1;
    for (int a = 0; a < 3; ++a) {
        int ex = 0;
        if (frexp(spacing_cm[a], &ex) != 0.5 || ex < -500 || ex > 500) F.pow2 = 0;
        F.inv[a] = 1.0 / spacing_cm[a];
    }
    F.bmax = ctx->bmax;
    k_field_bmax<<<1, 1024, 0, (cudaStream_t)cuda_stream>>>(field_dev, nodes, ctx->bmax);
    CU(ctx, cudaGetLastError());
    ctx->field = F;
    return COMET_OK;
}

static bool bad_physics(int32_t charge, double bz, double step, int32_t n_steps)
{
    return (charge != 1 && charge != -1) || !isfinite(bz) || !(step > 0.0) || !isfinite(step) ||
           n_steps < 1 || n_steps > COMET_MAX_STEPS;
}

extern "C" int comet_seed_extrapolate(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds,
                                      int32_t charge, double bz_tesla, double step_cm, int32_t n_steps,
                                      double r_stop_cm, void* track, int32_t* n_pts, void* cuda_stream)
{
    if (!ctx || n_seeds < 0 || seed_stride < n_seeds || bad_physics(charge, bz_tesla, step_cm, n_steps) ||
        !(r_stop_cm >= 0.0))
        return COMET_EINVAL;
    if (ctx->field.B) return COMET_EINVAL;      // the materialised track is a uniform-field path (comet_set_field)
    if (n_seeds == 0) return COMET_OK;
    if (!seeds || !track || !n_pts) return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    const double qkb = COMET_KAPPA * (double)charge * bz_tesla;
    const StepK hk = make_stepk_host(step_cm);
    const int threads = 128;
    const int64_t n_thr = n_chunks_of(n_seeds) * COMET_LANES;
    const unsigned blocks = (unsigned)((n_thr + threads - 1) / threads);
    k_extrapolate<<<blocks, threads, 0, (cudaStream_t)cuda_stream>>>(
        seeds, seed_stride, n_seeds, qkb, hk, n_steps, r_stop_cm * r_stop_cm, plane_X(track),
        plane_T(track, n_seeds, n_steps), n_pts);
    CU(ctx, cudaGetLastError());
    return COMET_OK;
}

extern "C" int comet_track_export(comet_ctx* ctx, const void* track, const int32_t* n_pts, int64_t n_seeds,
                                  int32_t n_steps, int64_t seed_begin, int64_t seed_end, double* out,
                                  void* cuda_stream)
{
    if (!ctx || n_seeds < 0 || n_steps < 1 || n_steps > COMET_MAX_STEPS || seed_begin < 0 ||
        seed_end < seed_begin || seed_end > n_seeds)
        return COMET_EINVAL;
    if (seed_end == seed_begin) return COMET_OK;
    if (!track || !n_pts || !out) return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    const int64_t total = (seed_end - seed_begin) * (int64_t)(n_steps + 1);
    const unsigned blocks = (unsigned)min((int64_t)(ctx->n_sm * 16), (total + 255) / 256);
    k_track_export<<<blocks, 256, 0, (cudaStream_t)cuda_stream>>>(
        plane_X((void*)track), plane_T((void*)track, n_seeds, n_steps), n_pts, n_steps, seed_begin, seed_end, out);
    CU(ctx, cudaGetLastError());
    return COMET_OK;
}

static int launch_wire_prep(comet_ctx* ctx, const double* wire_a, const double* wire_b, int32_t n_wires,
                            const int32_t* fired_wire, const int32_t* hit_off, const double* rho, int32_t n_fired,
                            double cutoff_cm, double step_cm, cudaStream_t st)
{
    if (n_fired > ctx->wt_cap) return COMET_EINVAL;
    if (n_fired == 0) return COMET_OK;
    const int32_t uniform = ctx->field.B == nullptr ? 1 : 0;
    k_wire_prep<<<(n_fired + 127) / 128, 128, 0, st>>>(wire_a, wire_b, n_wires, fired_wire, n_fired, hit_off, rho,
                                                       cutoff_cm, step_cm, uniform, ctx->wt, ctx->wtf);
    CU(ctx, cudaGetLastError());
    return COMET_OK;
}

static bool bad_hits(const double* wire_a, const double* wire_b, int32_t n_wires, const int32_t* fired_wire,
                     const int32_t* hit_off, const double* rho, int32_t n_fired, int32_t n_hits, double cutoff)
{
    if (n_wires < 0 || n_fired < 0 || n_hits < 0 || n_fired > n_wires || !(cutoff >= 0.0) || !isfinite(cutoff))
        return true;
    if (n_fired > 0 && (!wire_a || !wire_b || !fired_wire || !hit_off)) return true;
    if (n_hits > 0 && !rho) return true;
    return false;
}

extern "C" int comet_dca_rss(comet_ctx* ctx, const void* track, const int32_t* n_pts, int64_t n_seeds,
                             int32_t n_steps, int32_t charge, double bz_tesla, double step_cm,
                             const double* seeds, int64_t seed_stride,
                             const double* wire_a, const double* wire_b, int32_t n_wires,
                             const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                             int32_t n_fired, int32_t n_hits, double cutoff_cm,
                             double* rss, double* dca, int32_t* kstar, void* cuda_stream)
{
    if (!ctx || n_seeds < 0 || seed_stride < n_seeds || bad_physics(charge, bz_tesla, step_cm, n_steps) ||
        bad_hits(wire_a, wire_b, n_wires, fired_wire, hit_off, rho, n_fired, n_hits, cutoff_cm))
        return COMET_EINVAL;
    if (n_seeds == 0) return COMET_OK;
    if (ctx->field.B) return COMET_EINVAL;      // uniform-field path only (comet_set_field)
    if (!track || !n_pts || !seeds || !rss) return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    rc = launch_wire_prep(ctx, wire_a, wire_b, n_wires, fired_wire, hit_off, rho, n_fired, cutoff_cm, step_cm, st);
    if (rc) return rc;
    DcaArgs a;
    a.X = plane_X((void*)track);
    a.T = plane_T((void*)track, n_seeds, n_steps);
    a.n_pts = n_pts;
    a.n_seeds = n_seeds;
    a.n_steps = n_steps;
    a.qkb = COMET_KAPPA * (double)charge * bz_tesla;
    a.h = step_cm;
    a.seeds = seeds;
    a.stride = seed_stride;
    a.wt = ctx->wt;
    a.W = n_fired;
    a.hit_off = hit_off;
    a.rho = rho;
    a.lambda = cutoff_cm;
    a.rss = rss;
    a.dca = dca;
    a.kstar = kstar;
    a.stats = ctx->opt_stats ? ctx->stats : nullptr;
    const unsigned blocks = (unsigned)n_chunks_of(n_seeds);
    const int threads = COMET_DCA_WARPS * 32;
    (void)threads;
    if (ctx->opt_coarse == COMET_COARSE_PRUNED) {
        if (n_fired == 0) {
            CU(ctx, cudaMemsetAsync(rss, 0, sizeof(double) * (size_t)n_seeds, st));
            return COMET_OK;
        }
        // seed slabs so that (wires x padded seeds) fits the pair workspace
        const int64_t total_chunks = n_chunks_of(n_seeds);
        int64_t slab_chunks = (int64_t)(ctx->pair_max / ((size_t)COMET_LANES * (size_t)n_fired));
        if (slab_chunks < 1) slab_chunks = 1;
        if (slab_chunks > total_chunks) slab_chunks = total_chunks;
        rc = ensure_pairs(ctx, (size_t)slab_chunks * COMET_LANES * (size_t)n_fired, true);
        if (rc) return rc;
        const int32_t n_rows = track_rows(n_steps);
        for (int64_t c0 = 0; c0 < total_chunks; c0 += slab_chunks) {
            const int64_t nc = (total_chunks - c0 < slab_chunks) ? (total_chunks - c0) : slab_chunks;
            const int64_t s0 = c0 * COMET_LANES;
            PrunedArgs pa;
            pa.d = a;
            pa.d.X = a.X + track_row(c0, n_rows, 0);
            pa.d.T = a.T + track_row(c0, n_rows, 0);
            pa.d.n_pts = n_pts + s0;
            pa.d.seeds = seeds + s0;
            pa.d.n_seeds = (n_seeds - s0 < nc * COMET_LANES) ? (n_seeds - s0) : nc * COMET_LANES;
            pa.d.rss = rss + s0;
            pa.d.dca = dca ? dca + (size_t)s0 * n_fired : nullptr;
            pa.d.kstar = kstar ? kstar + (size_t)s0 * n_fired : nullptr;
            pa.n_chunks = nc;
            pa.SP = nc * COMET_LANES;
            pa.n_groups = (n_fired + COMET_PRUNED_WT - 1) / COMET_PRUNED_WT;
            pa.full = (dca || kstar) ? 1 : 0;
            pa.kb = ctx->kb;
            pa.e2 = ctx->e2;
            pa.items = ctx->items;
            pa.n_items = ctx->n_items;
            CU(ctx, cudaMemsetAsync(ctx->n_items, 0, sizeof(unsigned int), st));
            pa.cap_s = track_rows(n_steps) / COMET_M1;
            if (pa.cap_s > COMET_PR_CAP_S) pa.cap_s = COMET_PR_CAP_S;
            const size_t sm1 = (size_t)pa.cap_s * 3 * COMET_LANES * sizeof(double);
            const int64_t w2 = nc * (int64_t)n_fired;          // upper bound on the work list
            const unsigned b1 = (unsigned)nc;
            const int64_t b2_all = (w2 + COMET_FINE_THREADS / 32 - 1) / (COMET_FINE_THREADS / 32);
            const unsigned b2 = (unsigned)(b2_all < ctx->fine_blocks ? b2_all : ctx->fine_blocks);
            const bool tm = ctx->opt_timing != 0;
            cudaEvent_t* tev = ctx->tev[ctx->tev_count % COMET_TEV_RING];
            if (tm) { CU(ctx, cudaEventRecord(tev[0], st)); CU(ctx, cudaEventRecord(tev[1], st)); }
            if (ctx->opt_stats) k_coarse_pruned<COMET_PRUNED_WT, true><<<b1, COMET_PR_WARPS * 32, sm1, st>>>(pa);
            else k_coarse_pruned<COMET_PRUNED_WT, false><<<b1, COMET_PR_WARPS * 32, sm1, st>>>(pa);
            if (tm) CU(ctx, cudaEventRecord(tev[2], st));
            if (ctx->opt_stats) k_fine<true><<<b2, COMET_FINE_THREADS, 0, st>>>(pa);
            else k_fine<false><<<b2, COMET_FINE_THREADS, 0, st>>>(pa);
            if (tm) CU(ctx, cudaEventRecord(tev[3], st));
            k_rss_sum<<<(unsigned)((pa.d.n_seeds + 255) / 256), 256, 0, st>>>(pa.e2, pa.SP, n_fired, pa.d.n_seeds, pa.d.rss, nullptr, 0.0, nullptr);
            if (tm) { CU(ctx, cudaEventRecord(tev[4], st)); ctx->tev_count += 1; }
            CU(ctx, cudaGetLastError());
        }
        return COMET_OK;
    } else {
        // wires per warp per pass: spread n_fired evenly over ceil(n_fired/32) passes of 8 warps
        const int n_pass = (n_fired + COMET_DCA_WARPS * 4 - 1) / (COMET_DCA_WARPS * 4);
        int wt = n_pass > 0 ? (n_fired + COMET_DCA_WARPS * n_pass - 1) / (COMET_DCA_WARPS * n_pass) : 1;
        if (wt < 1) wt = 1;
        const size_t smem = (2 * COMET_KT * 3 * COMET_LANES + (size_t)COMET_DCA_WARPS * wt * 32) * sizeof(double);
        switch (wt) {
            case 1: k_dca_rss<1><<<blocks, threads, smem, st>>>(a); break;
            case 2: k_dca_rss<2><<<blocks, threads, smem, st>>>(a); break;
            case 3: k_dca_rss<3><<<blocks, threads, smem, st>>>(a); break;
            default: k_dca_rss<4><<<blocks, threads, smem, st>>>(a); break;
        }
    }
    CU(ctx, cudaGetLastError());
    return COMET_OK;
}

// ---------------------------------------------------------------------------------------------
// kernels A + B fused (scan_fused.cuh)
// ---------------------------------------------------------------------------------------------
// Workspace of comet_scan_rss for a call of `total_chunks` track chunks (sizes in bytes; slab_chunks = chunks a
// slab holds: bounded by the pair workspace limit and by 8 GiB of checkpoints).
struct ScanWs {
    int64_t slab_chunks;
    int32_t n_ck;
    size_t ck_chunk, pairs, ck, cw, ub, npu, tw, npw, tm;
    int32_t tpc, u_rows;      // distinct tracks per chunk the workspace is sized for, rows per track
    bool zgroup;
};
static ScanWs scan_ws(const comet_ctx* ctx, int64_t total_chunks, int32_t n_steps, int32_t n_fired, int32_t z_run)
{
    ScanWs w;
    const bool field = ctx->field.B != nullptr;
    // (small calls are launch- and latency-bound: the run-length check and the chain of k_gen_unique in front of the
    // scan cost more than they save below about a thousand chunks -- configs[0], the refined sets of a stage)
    w.zgroup = !field && ctx->opt_zgroup != 0 && z_run != 1 &&
               (ctx->opt_zgroup == 2 || total_chunks >= COMET_ZG_MIN_CHUNKS);
    // checkpoints per chunk: (x, T) every 4th state for the plain kernels; with the run length promised only the
    // z-run kernels run, which keep one z per seed every COMET_ZR_CK states
    w.n_ck = n_steps / COMET_CK_ROWS(field) + 1;
    w.ck_chunk = (size_t)w.n_ck * COMET_CK_FIELDS(field) * COMET_LANES * sizeof(double);
    if (w.zgroup && z_run >= COMET_ZG_MIN) w.ck_chunk = (size_t)(n_steps / COMET_ZR_CK + 1) * COMET_LANES * sizeof(double);
    int64_t slab_chunks = total_chunks;
    if (n_fired > 0) {
        const int64_t by_pairs = (int64_t)(ctx->pair_max / ((size_t)COMET_LANES * (size_t)n_fired));
        if (by_pairs < slab_chunks) slab_chunks = by_pairs;
    }
    const int64_t by_ck = (int64_t)(ctx->ck_max / w.ck_chunk);
    if (by_ck < slab_chunks) slab_chunks = by_ck;
    if (slab_chunks < 1) slab_chunks = 1;
    w.slab_chunks = slab_chunks;
    w.pairs = (size_t)slab_chunks * COMET_LANES * (size_t)(n_fired > 0 ? n_fired : 1);
    w.ck = (size_t)slab_chunks * w.ck_chunk;
    w.cw = (size_t)slab_chunks * COMET_LANES * sizeof(double);
    w.npw = (size_t)slab_chunks * COMET_LANES * sizeof(int32_t);
    // distinct transverse tracks (scan_zgroup.cuh): 32 / run length per chunk (at most 4: runs of >= 8 seeds), each
    // u_rows = n_steps + 1 rounded up to whole 64-row blocks, 32 bytes per row
    w.tpc = (z_run >= COMET_ZG_MIN) ? (z_run >= 32 ? 1 : 32 / z_run) : 4;
    w.u_rows = (n_steps + 64) & ~63;
    const size_t tracks = (size_t)slab_chunks * w.tpc + 64;
    w.ub = w.zgroup ? tracks * (size_t)w.u_rows * 4 * sizeof(double) : 0;
    w.npu = w.zgroup ? tracks * sizeof(int32_t) : 0;
    w.tw = w.zgroup ? w.cw : 0;
    w.tm = w.zgroup ? (size_t)slab_chunks * (size_t)((n_fired + 31) / 32 + 1) * sizeof(unsigned int) : 0;
    return w;
}

static bool scan_ws_fits(const comet_ctx* ctx, const ScanWs& w)
{
    return w.pairs <= ctx->pair_cap && w.ck <= ctx->ck_bytes && w.cw <= ctx->cw_bytes && w.ub <= ctx->ub_bytes &&
           w.npu <= ctx->npu_bytes && w.tw <= ctx->tw_bytes && w.tm <= ctx->tm_bytes && w.npw <= ctx->npw_cap * sizeof(int32_t);
}

static int grow_dev(comet_ctx* ctx, void** buf, size_t* have, size_t need)
{
    if (need <= *have) return COMET_OK;
    CU(ctx, cudaDeviceSynchronize());
    if (*buf) { CU(ctx, cudaFree(*buf)); *buf = nullptr; *have = 0; }
    cudaError_t e = cudaMalloc(buf, need);
    if (e != cudaSuccess) { ctx->last_cuda = (int)e; *buf = nullptr; cudaGetLastError(); return COMET_ENOMEM; }
    *have = need;
    return COMET_OK;
}

// grows the ctx's workspace to `w` (synchronises the device when anything is reallocated)
static int scan_ws_grow(comet_ctx* ctx, const ScanWs& w)
{
    ctx->last.valid = 0;                                    // (the distinct-track rows may move)
    int rc = ensure_pairs(ctx, w.pairs, false);
    if (rc) return rc;
    if ((rc = grow_dev(ctx, (void**)&ctx->ck, &ctx->ck_bytes, w.ck))) return rc;
    if ((rc = grow_dev(ctx, (void**)&ctx->cw, &ctx->cw_bytes, w.cw))) return rc;
    if ((rc = grow_dev(ctx, (void**)&ctx->ub, &ctx->ub_bytes, w.ub))) return rc;
    if ((rc = grow_dev(ctx, (void**)&ctx->npu, &ctx->npu_bytes, w.npu))) return rc;
    if ((rc = grow_dev(ctx, (void**)&ctx->tw, &ctx->tw_bytes, w.tw))) return rc;
    if ((rc = grow_dev(ctx, (void**)&ctx->tmk, &ctx->tm_bytes, w.tm))) return rc;
    size_t have = ctx->npw_cap * sizeof(int32_t);
    if ((rc = grow_dev(ctx, (void**)&ctx->npw, &have, w.npw))) return rc;
    ctx->npw_cap = have / sizeof(int32_t);
    return COMET_OK;
}

static bool bad_zrun(int32_t z_run) { return z_run < 0 || (z_run > 1 && (z_run < 8 || (z_run & (z_run - 1)) != 0)); }

extern "C" int comet_reserve_scan(comet_ctx* ctx, int64_t n_seeds, int32_t z_run, int32_t n_steps, int32_t n_fired)
{
    if (!ctx || n_seeds < 1 || n_steps < 1 || n_steps > COMET_MAX_STEPS || n_fired < 0 || n_fired > ctx->wt_cap || bad_zrun(z_run))
        return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    // a workspace that serves the promised run length and the call without a promise (whichever is larger, buffer by buffer)
    ScanWs w = scan_ws(ctx, n_chunks_of(n_seeds), n_steps, n_fired, z_run);
    if (z_run != 0) {
        const ScanWs w0 = scan_ws(ctx, n_chunks_of(n_seeds), n_steps, n_fired, 0);
        auto mx = [](size_t a, size_t b) { return a > b ? a : b; };
        w.pairs = mx(w.pairs, w0.pairs); w.ck = mx(w.ck, w0.ck); w.cw = mx(w.cw, w0.cw); w.ub = mx(w.ub, w0.ub);
        w.npu = mx(w.npu, w0.npu); w.tw = mx(w.tw, w0.tw); w.tm = mx(w.tm, w0.tm); w.npw = mx(w.npw, w0.npw);
    }
    return scan_ws_grow(ctx, w);
}

// comet_scan_rss; with seeds_host != NULL (HOST SoA [6][n_seeds]) every sub-slab first copies its seeds to
// `seeds` on its own stream, so the upload of one sub-slab overlaps the kernels of the others
static int scan_rss_impl(comet_ctx* ctx, double* seeds_w, const double* seeds_host,
                         const double* seeds, int64_t seed_stride, int64_t n_seeds, int32_t z_run,
                         int32_t charge, double bz_tesla, double step_cm, int32_t n_steps, double r_stop_cm,
                         const double* wire_a, const double* wire_b, int32_t n_wires,
                         const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                         int32_t n_fired, int32_t n_hits, double cutoff_cm,
                         double* rss, int32_t* n_pts, void* cuda_stream, const int32_t* dyn = nullptr,
                         bool wire_table_ready = false)
{
    if (!ctx || n_seeds < 0 || seed_stride < n_seeds || bad_physics(charge, bz_tesla, step_cm, n_steps) ||
        !(r_stop_cm >= 0.0) || bad_zrun(z_run) ||
        bad_hits(wire_a, wire_b, n_wires, fired_wire, hit_off, rho, n_fired, n_hits, cutoff_cm))
        return COMET_EINVAL;
    if (ctx->field.B && n_steps > COMET_MAX_STEPS_FIELD) return COMET_EINVAL;
    if (n_fired > ctx->wt_cap) return COMET_EINVAL;
    if (n_seeds == 0) return COMET_OK;
    if (!seeds || !rss) return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int64_t total_chunks = n_chunks_of(n_seeds);
    const bool field = ctx->field.B != nullptr;
    // workspace: sized by comet_reserve_scan, else grown here -- never while the stream is being captured
    const ScanWs ws = scan_ws(ctx, total_chunks, n_steps, n_fired, z_run);
    if (!scan_ws_fits(ctx, ws)) {
        cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
        CU(ctx, cudaStreamIsCapturing(st, &cap));
        if (cap != cudaStreamCaptureStatusNone) return COMET_ENOMEM;
        rc = scan_ws_grow(ctx, ws);
        if (rc) return rc;
    }
    // (the later iterations of a stage scan against the same hit list: the table of the first one stands)
    if (!wire_table_ready) {
        rc = launch_wire_prep(ctx, wire_a, wire_b, n_wires, fired_wire, hit_off, rho, n_fired, cutoff_cm, step_cm, st);
        if (rc) return rc;
    }
    const int32_t n_ck = ws.n_ck;
    const size_t ck_chunk = ws.ck_chunk;
    const int64_t slab_chunks = ws.slab_chunks;
    const bool zgroup = ws.zgroup;
    const int32_t zrun_host = (zgroup && z_run >= COMET_ZG_MIN) ? (z_run > 32 ? 32 : z_run) : 0;
    // A slab (what the workspace holds) is cut into up to opt_lanes sub-slabs that run concurrently on the
    // ctx's internal streams: k_scan_fused of sub-slab l on ls[l], its fine stage on the high-priority
    // lf[l], so that k_fine_ck of one sub-slab shares the SMs with k_scan_fused of the next ones (the two
    // kernels leave different parts of the FP64 pipe idle).  The caller's stream forks into the lanes and
    // joins them again with events: the call stays asynchronous and capturable.  Per-kernel timing
    // (COMET_OPT_TIMING) and the work counters run one lane on the caller's stream.
    const bool tm = ctx->opt_timing != 0;
    // (in a field map the sub-slab kernels gain nothing from sharing the SMs: one lane)
    // (measured on configs[1]: 6 lanes suit the plain kernels, 4 the z-run kernels, whose sub-slabs start with a
    // latency-bound k_gen_unique; a value set with COMET_OPT_LANES is taken as it is)
    // (with seeds coming from the host the sub-slabs also pipeline the upload: finer sub-slabs)
    const int lanes_auto = ctx->lanes_set ? ctx->opt_lanes : (seeds_host ? COMET_MAX_LANES : (zgroup ? 4 : ctx->opt_lanes));
    const int lanes_opt = (tm || ctx->opt_stats || field) ? 1 : lanes_auto;
    for (int64_t c0 = 0; c0 < total_chunks; c0 += slab_chunks) {
        const int64_t nc_slab = (total_chunks - c0 < slab_chunks) ? (total_chunks - c0) : slab_chunks;
        // sub-slabs of whole CTAs, at least two CTAs per SM each
        const int64_t min_sub = (int64_t)COMET_FUSED_WARPS * ctx->n_sm * 2;
        int lanes = lanes_opt;
        while (lanes > 1 && nc_slab / lanes < min_sub) --lanes;
        int64_t sub = (nc_slab + lanes - 1) / lanes;
        sub = (sub + COMET_FUSED_WARPS - 1) / COMET_FUSED_WARPS * COMET_FUSED_WARPS;
        if (lanes > 1) CU(ctx, cudaEventRecord(ctx->ev_fork, st));
        int used = 0;
        for (int l = 0; l < lanes; ++l) {
            const int64_t cl = (int64_t)l * sub;             // first chunk of the sub-slab within the slab
            if (cl >= nc_slab) break;
            const int64_t nc = (nc_slab - cl < sub) ? (nc_slab - cl) : sub;
            const int64_t s0 = (c0 + cl) * COMET_LANES;
            cudaStream_t s_scan = lanes > 1 ? ctx->ls[l] : st, s_fine = lanes > 1 ? ctx->lf[l] : st;
            FusedArgs a;
            a.seeds = seeds + s0;
            a.stride = seed_stride;
            a.n_seeds = (n_seeds - s0 < nc * COMET_LANES) ? (n_seeds - s0) : nc * COMET_LANES;
            a.qkb = field ? COMET_KAPPA * (double)charge : COMET_KAPPA * (double)charge * bz_tesla;
            a.F = ctx->field;
            a.h_min = step_cm / 64.0;
            a.hk = make_stepk_host(step_cm);
            a.n_steps = n_steps;
            a.r_stop2 = r_stop_cm * r_stop_cm;
            a.wt = ctx->wt;
            a.wtf = ctx->wtf;
            a.W = n_fired;
            a.hit_off = hit_off;
            a.rho = rho;
            a.lambda = cutoff_cm;
            a.SP = nc * COMET_LANES;
            a.n_ck = n_ck;
            a.ck = ctx->ck + (size_t)cl * (ck_chunk / sizeof(double));
            a.bd = ctx->e2 + (size_t)cl * COMET_LANES * (size_t)n_fired;
            a.n_pts = n_pts ? n_pts + s0 : ctx->npw + cl * COMET_LANES;
            a.cw = ctx->cw + cl * COMET_LANES;
            a.tw = zgroup ? ctx->tw + cl * COMET_LANES : nullptr;
            a.items = ctx->items + (size_t)cl * (size_t)n_fired;
            a.n_items = ctx->n_items + 4 * l;
            a.stats = ctx->opt_stats ? ctx->stats : nullptr;
            a.dyn = dyn;
            if (lanes > 1) CU(ctx, cudaStreamWaitEvent(s_scan, ctx->ev_fork, 0));
            if (seeds_host)
                for (int j = 0; j < 6; ++j)
                    CU(ctx, cudaMemcpyAsync(seeds_w + (size_t)j * seed_stride + s0, seeds_host + (size_t)j * n_seeds + s0,
                                            sizeof(double) * (size_t)a.n_seeds, cudaMemcpyHostToDevice, s_scan));
            CU(ctx, cudaMemsetAsync(a.n_items, 0, 4 * sizeof(unsigned int), s_scan));
            const unsigned b1_packed = (unsigned)((nc + COMET_FUSED_WARPS - 1) / COMET_FUSED_WARPS);
            const int64_t w2 = nc * (int64_t)n_fired;
            const int64_t b2_all = (w2 + COMET_FINE_THREADS / 32 - 1) / (COMET_FINE_THREADS / 32);
            unsigned b2 = (unsigned)(b2_all < ctx->fine_blocks ? b2_all : ctx->fine_blocks);
            if (b2 < 1) b2 = 1;
            cudaEvent_t* tev = ctx->tev[ctx->tev_count % COMET_TEV_RING];
            if (tm) CU(ctx, cudaEventRecord(tev[0], st));
            if (tm && !zgroup) CU(ctx, cudaEventRecord(tev[1], st));    // (no k_gen_unique: an empty slot)
            const int thr = 32 * COMET_FUSED_WARPS;
            // a launch that cannot give every SM two CTAs of four chunks: the CTA's warps share one chunk's wires
            const bool small = !zgroup && nc < (int64_t)COMET_FUSED_WARPS * ctx->n_sm * 2;
            const bool split = small && field && n_fired > 32;   // (field map: the warps of a CTA repeat the chunk's chain)
            const bool overlap = small && !field;                // uniform field: one generator warp, three search warps (scan_small.cuh)
            const unsigned b1 = (split || overlap) ? (unsigned)nc : b1_packed;
            a.zg = nullptr;
            a.zrun = zrun_host;
            a.ub = nullptr;
            a.np_u = nullptr;
            a.tm = nullptr;
            a.u_rows = ws.u_rows;
            FusedArgs az = a;                                   // the arguments of the z-run kernels
            if (zgroup) {
                // seeds in runs that differ only in z: every distinct transverse track is stepped once (k_gen_unique) and
                // k_scan_zrun works from those tracks (scan_zrun.cuh); the run length is the caller's promise, else it is
                // found on the device and the kernels that are not needed exit at once
                az.ub = ctx->ub + (size_t)cl * ws.tpc * (size_t)ws.u_rows * 4;
                az.np_u = ctx->npu + (size_t)cl * ws.tpc;
                az.tm = ctx->tmk + (size_t)cl * (size_t)((n_fired + 31) / 32);
                az.n_ck = n_steps / COMET_ZR_CK + 1;             // z checkpoints only, inside the sub-slab's checkpoint region
                if (!zrun_host) {
                    az.zg = ctx->zg_flag + l;
                    a.zg = az.zg;
                    CU(ctx, cudaMemsetAsync(ctx->zg_flag + l, 0xff, sizeof(unsigned int), s_scan));
                    k_zgroup_check<<<(unsigned)((a.n_seeds + 255) / 256), 256, 0, s_scan>>>(a.seeds, a.stride, a.n_seeds, ctx->zg_flag + l);
                }
                const int64_t zr_min = zrun_host ? zrun_host : COMET_ZG_MIN;
                const unsigned bu = (unsigned)(((a.n_seeds + zr_min - 1) / zr_min + 31) / 32);  // one warp per CTA: a latency-bound chain
                if (a.stats) k_gen_unique<true><<<bu, 32, 0, s_scan>>>(az);
                else k_gen_unique<false><<<bu, 32, 0, s_scan>>>(az);
                if (tm) CU(ctx, cudaEventRecord(tev[1], st));
                const bool bigw = n_fired > COMET_ZR_WCAP;
                const int wpc = COMET_ZR_WPC(bigw);              // (many wires: CTAs of one warp, no wire table)
                const unsigned bz = (unsigned)((nc + wpc - 1) / wpc);
                const int zthr = 32 * wpc;
#define COMET_LAUNCH_ZRUN(NU)                                                                                         \
                do {                                                                                                  \
                    if (a.stats) { if (bigw) k_scan_zrun<true, NU, true><<<bz, zthr, COMET_ZR_SMEM(NU, n_fired, true), s_scan>>>(az);     \
                                   else k_scan_zrun<true, NU, false><<<bz, zthr, COMET_ZR_SMEM(NU, n_fired, false), s_scan>>>(az); }      \
                    else { if (bigw) k_scan_zrun<false, NU, true><<<bz, zthr, COMET_ZR_SMEM(NU, n_fired, true), s_scan>>>(az);            \
                           else k_scan_zrun<false, NU, false><<<bz, zthr, COMET_ZR_SMEM(NU, n_fired, false), s_scan>>>(az); }             \
                } while (0)
                if (!zrun_host || zrun_host == 32) COMET_LAUNCH_ZRUN(1);
                if (!zrun_host || zrun_host == 16) COMET_LAUNCH_ZRUN(2);
                if (!zrun_host || zrun_host == 8) COMET_LAUNCH_ZRUN(4);
#undef COMET_LAUNCH_ZRUN
            }
            if (zrun_host) {
                // (the ZG kernels serve the launch: the plain variants are not enqueued)
            } else if (overlap) {
                if (a.stats) k_scan_small<true><<<b1, 128, COMET_SMALL_SMEM, s_scan>>>(a);
                else k_scan_small<false><<<b1, 128, COMET_SMALL_SMEM, s_scan>>>(a);
            } else if (split) {
                if (a.stats) k_scan_fused<true, true, true><<<b1, thr, ctx->fused_smem, s_scan>>>(a);
                else k_scan_fused<false, true, true><<<b1, thr, ctx->fused_smem, s_scan>>>(a);
            } else if (field) {
                if (a.stats) k_scan_fused<true, true><<<b1, thr, ctx->fused_smem, s_scan>>>(a);
                else k_scan_fused<false, true><<<b1, thr, ctx->fused_smem, s_scan>>>(a);
            } else {
                if (a.stats) k_scan_fused<true, false><<<b1, thr, ctx->fused_smem, s_scan>>>(a);
                else k_scan_fused<false, false><<<b1, thr, ctx->fused_smem, s_scan>>>(a);
            }
            if (tm) CU(ctx, cudaEventRecord(tev[2], st));
            if (lanes > 1) {
                CU(ctx, cudaEventRecord(ctx->ev_scan[l], s_scan));
                CU(ctx, cudaStreamWaitEvent(s_fine, ctx->ev_scan[l], 0));
            }
            if (n_fired > 0) {
                if (field) k_fine_ck<true><<<b2, COMET_FINE_THREADS, 0, s_fine>>>(a);
                else {
                    if (zgroup) k_fine_ck<false, true><<<b2, COMET_FINE_THREADS, 0, s_fine>>>(az);
                    if (!zrun_host) k_fine_ck<false><<<b2, COMET_FINE_THREADS, 0, s_fine>>>(a);
                }
            }
            if (tm) CU(ctx, cudaEventRecord(tev[3], st));
            k_rss_sum<<<(unsigned)((a.n_seeds + 255) / 256), 256, 0, s_fine>>>(a.bd, a.SP, n_fired, a.n_seeds, rss + s0,
                                                                              zgroup ? az.tm : nullptr, cutoff_cm * cutoff_cm, az.zg, dyn);
            if (tm) { CU(ctx, cudaEventRecord(tev[4], st)); ctx->tev_count += 1; }
            if (lanes > 1) CU(ctx, cudaEventRecord(ctx->ev_join[l], s_fine));
            CU(ctx, cudaGetLastError());
            used = l + 1;
        }
        if (lanes > 1)
            for (int l = 0; l < used; ++l) CU(ctx, cudaStreamWaitEvent(st, ctx->ev_join[l], 0));
    }
    ctx->last.valid = 0;
    if (!zgroup && !field && slab_chunks >= total_chunks && !seeds_host) {
        // plain kernels, uniform field: the checkpoints of the whole seed set are in `ck`, chunk after chunk
        ctx->last.seeds = seeds; ctx->last.stride = seed_stride; ctx->last.n_seeds = n_seeds;
        ctx->last.qkb = COMET_KAPPA * (double)charge * bz_tesla; ctx->last.step = step_cm; ctx->last.r_stop = r_stop_cm;
        ctx->last.n_steps = n_steps; ctx->last.n_ck = n_ck;
        ctx->last.valid = 2;
    }
    if (zrun_host && slab_chunks >= total_chunks && !seeds_host) {
        ctx->last.seeds = seeds; ctx->last.stride = seed_stride; ctx->last.n_seeds = n_seeds;
        ctx->last.qkb = COMET_KAPPA * (double)charge * bz_tesla; ctx->last.step = step_cm; ctx->last.r_stop = r_stop_cm;
        ctx->last.n_steps = n_steps; ctx->last.u_rows = ws.u_rows;
        ctx->last.zshift = zrun_host == 32 ? 5 : (zrun_host == 16 ? 4 : 3);
        ctx->last.valid = 1;
    }
    return COMET_OK;
}

extern "C" int comet_scan_rss(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds, int32_t z_run,
                              int32_t charge, double bz_tesla, double step_cm, int32_t n_steps, double r_stop_cm,
                              const double* wire_a, const double* wire_b, int32_t n_wires,
                              const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                              int32_t n_fired, int32_t n_hits, double cutoff_cm,
                              double* rss, int32_t* n_pts, void* cuda_stream)
{
    return scan_rss_impl(ctx, nullptr, nullptr, seeds, seed_stride, n_seeds, z_run, charge, bz_tesla, step_cm, n_steps, r_stop_cm,
                         wire_a, wire_b, n_wires, fired_wire, hit_off, rho, n_fired, n_hits, cutoff_cm, rss, n_pts,
                         cuda_stream);
}

extern "C" int comet_select_and_classify(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds,
                                         int32_t charge, double bz_tesla, double step_cm, int32_t n_steps,
                                         double r_stop_cm,
                                         const double* wire_a, const double* wire_b, int32_t n_wires,
                                         const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                                         int32_t n_fired, int32_t n_hits, double cutoff_cm,
                                         const double* rss, const int64_t* part_off, int32_t n_part,
                                         int64_t* best_seed, double* best_rss, double* best_dca, uint8_t* cls,
                                         void* cuda_stream)
{
    if (!ctx || n_seeds < 0 || seed_stride < n_seeds || bad_physics(charge, bz_tesla, step_cm, n_steps) ||
        !(r_stop_cm >= 0.0) ||
        bad_hits(wire_a, wire_b, n_wires, fired_wire, hit_off, rho, n_fired, n_hits, cutoff_cm) ||
        n_part < 0 || n_part > COMET_MAX_PARTITIONS)
        return COMET_EINVAL;
    if (ctx->field.B && n_steps > COMET_MAX_STEPS_FIELD) return COMET_EINVAL;
    if (n_part == 0) return COMET_OK;
    if (!part_off || !best_seed || !best_rss || (n_fired > 0 && !best_dca) || (n_hits > 0 && !cls)) return COMET_EINVAL;
    PartOff po;
    memset(&po, 0, sizeof(po));
    for (int p = 0; p <= n_part; ++p) {
        po.off[p] = part_off[p];
        if (part_off[p] < 0 || part_off[p] > n_seeds || (p > 0 && part_off[p] < part_off[p - 1])) return COMET_EINVAL;
    }
    if (po.off[n_part] > 0 && (!seeds || !rss)) return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // what the comet_scan_rss call that produced rss left in the ctx, if this is that seed set (same buffer, same physics)
    const bool field = ctx->field.B != nullptr;
    const double qkb_u = COMET_KAPPA * (double)charge * bz_tesla;
    const bool same_scan = !field && ctx->last.valid && ctx->last.seeds == seeds && ctx->last.stride == seed_stride &&
                           ctx->last.n_seeds == n_seeds && ctx->last.qkb == qkb_u && ctx->last.step == step_cm &&
                           ctx->last.r_stop == r_stop_cm && ctx->last.n_steps == n_steps;
    int64_t part_max = 0;
    for (int p = 0; p < n_part; ++p)
        if (po.off[p + 1] - po.off[p] > part_max) part_max = po.off[p + 1] - po.off[p];
    const bool fused_argmin = part_max <= COMET_ARGMIN_FUSED;
    if (!fused_argmin) {
        k_argmin_stage1<<<dim3(COMET_ARGMIN_SPLIT, n_part), COMET_ARGMIN_THREADS, 0, st>>>(rss, po, ctx->pv, ctx->pi);
        CU(ctx, cudaGetLastError());
    }
    ClassifyArgs a;
    a.rss = fused_argmin ? rss : nullptr;
    a.po = po;
    a.seeds = seeds;
    a.stride = seed_stride;
    a.qkb = COMET_KAPPA * (double)charge * bz_tesla;
    a.hk = make_stepk_host(step_cm);
    a.n_steps = n_steps;
    a.r_stop2 = r_stop_cm * r_stop_cm;
    a.wire_a = wire_a; a.wire_b = wire_b; a.n_wires = n_wires; a.fired_wire = fired_wire;
    a.W = n_fired;
    a.hit_off = hit_off;
    a.rho = rho;
    a.n_hits = n_hits;
    a.lambda = cutoff_cm;
    a.pv = ctx->pv;
    a.pi = ctx->pi;
    a.best_seed = best_seed;
    a.best_rss = best_rss;
    a.best_dca = best_dca;
    a.cls = cls;
    if (field) a.qkb = COMET_KAPPA * (double)charge;
    a.F = ctx->field;
    a.h_min = step_cm / 64.0;
    // the winners' tracks: the rows of their distinct transverse tracks, or the checkpoints of the plain kernels
    a.ub = nullptr; a.np_u = nullptr; a.zshift = 0; a.u_rows = 0; a.dyn = nullptr; a.ck = nullptr; a.n_ck = 0;
    if (same_scan && ctx->last.valid == 1) { a.ub = ctx->ub; a.np_u = ctx->npu; a.zshift = ctx->last.zshift; a.u_rows = ctx->last.u_rows; }
    if (same_scan && ctx->last.valid == 2) { a.ck = ctx->ck; a.n_ck = ctx->last.n_ck; }
    const size_t smem = (size_t)(n_steps + 1) * (field ? 7 : 6) * sizeof(double);
    // (the search over the winner's states is most of the kernel and a CTA is one SM: groups of about 8 wires per CTA)
    int n_grp = (n_fired + 7) / 8;
    if (n_grp > 16) n_grp = 16;
    if (n_grp < 1) n_grp = 1;
    if (field) k_select_classify<true><<<dim3(n_part, n_grp), 256, smem, st>>>(a);
    else k_select_classify<false><<<dim3(n_part, n_grp), 256, smem, st>>>(a);
    CU(ctx, cudaGetLastError());
    return COMET_OK;
}

// ---------------------------------------------------------------------------------------------
// iterative seed refinement (readings R24-R28)
// ---------------------------------------------------------------------------------------------
static int fill_partoff(PartOff* po, const int64_t* part_off, int32_t n_part, int64_t n_seeds, bool non_empty)
{
    memset(po, 0, sizeof(*po));
    for (int p = 0; p <= n_part; ++p) {
        po->off[p] = part_off[p];
        if (part_off[p] < 0 || part_off[p] > n_seeds || (p > 0 && part_off[p] < part_off[p - 1])) return COMET_EINVAL;
        if (non_empty && p > 0 && part_off[p] == part_off[p - 1]) return COMET_EINVAL;
    }
    return COMET_OK;
}

static bool bad_box(const double* half_width)
{
    if (!half_width) return true;
    for (int d = 0; d < 4; ++d)
        if (!(half_width[d] >= 0.0) || !isfinite(half_width[d])) return true;
    return false;
}

extern "C" int comet_select_references(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds,
                                       const double* rss, const int64_t* part_off, int32_t n_part,
                                       const double* half_width, int32_t k_ref, int64_t* ref_seed,
                                       void* cuda_stream)
{
    if (!ctx || n_seeds < 0 || seed_stride < n_seeds || n_part < 0 || n_part > COMET_MAX_PARTITIONS ||
        k_ref < 1 || k_ref > COMET_MAX_REFS || bad_box(half_width))
        return COMET_EINVAL;
    if (n_part == 0) return COMET_OK;
    if (!part_off || !ref_seed) return COMET_EINVAL;
    PartOff po;
    if (fill_partoff(&po, part_off, n_part, n_seeds, false)) return COMET_EINVAL;
    if (po.off[n_part] > 0 && (!seeds || !rss)) return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    RefBox box;
    for (int d = 0; d < 4; ++d) box.two_hw[d] = 2.0 * half_width[d];
    // small partitions: one CTA each; large ones: a cluster of CTAs each (RSS staged in shared memory when it fits)
    int64_t n_max = 0;
    for (int p = 0; p < n_part; ++p)
        if (po.off[p + 1] - po.off[p] > n_max) n_max = po.off[p + 1] - po.off[p];
    const int64_t per = (n_max + COMET_REF_CLUSTER - 1) / COMET_REF_CLUSTER;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (n_max <= 16 * COMET_REF_THREADS) {
        k_select_refs<<<n_part, COMET_REF_THREADS, 0, st>>>(seeds, seed_stride, rss, po, box, k_ref, ref_seed);
    } else {
        // the seeds of lowest RSS first (k_select_refs_short); the cluster kernel redoes a partition only if they ran out
        k_select_refs_short<<<n_part, COMET_REF_THREADS, 0, st>>>(seeds, seed_stride, rss, po, box, k_ref, ref_seed, ctx->ref_fb);
        if (per <= COMET_REF_SMEM_MAX)
            k_select_refs_cluster<true><<<dim3(COMET_REF_CLUSTER, n_part), COMET_REF_THREADS, (size_t)per * sizeof(double), st>>>(
                seeds, seed_stride, rss, po, box, k_ref, ref_seed, ctx->ref_fb);
        else
            k_select_refs_cluster<false><<<dim3(COMET_REF_CLUSTER, n_part), COMET_REF_THREADS, 0, st>>>(
                seeds, seed_stride, rss, po, box, k_ref, ref_seed, ctx->ref_fb);
    }
    CU(ctx, cudaGetLastError());
    return COMET_OK;
}

static int make_grid(RefineGrid* g, int64_t* G, const double* half_width, const int32_t* n_grid)
{
    if (bad_box(half_width) || !n_grid) return COMET_EINVAL;
    *G = 1;
    for (int d = 0; d < 4; ++d) {
        if (n_grid[d] < 1 || n_grid[d] > 4096) return COMET_EINVAL;
        g->n[d] = n_grid[d];
        g->hw[d] = half_width[d];
        g->step[d] = n_grid[d] > 1 ? (2.0 * half_width[d]) / (double)(n_grid[d] - 1) : 0.0;
        *G *= n_grid[d];
        if (*G > ((int64_t)1 << 31)) return COMET_EINVAL;
    }
    return COMET_OK;
}

extern "C" int comet_refine_seeds(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds,
                                  const int64_t* ref_seed, int32_t n_part, int32_t k_ref,
                                  const double* half_width, const int32_t* n_grid,
                                  double* new_seeds, int64_t new_stride, void* cuda_stream)
{
    RefineGrid g;
    int64_t G = 0;
    if (!ctx || n_seeds < 0 || seed_stride < n_seeds || n_part < 0 || n_part > COMET_MAX_PARTITIONS ||
        k_ref < 1 || k_ref > COMET_MAX_REFS || make_grid(&g, &G, half_width, n_grid))
        return COMET_EINVAL;
    if (n_part == 0) return COMET_OK;
    if (!seeds || !ref_seed || !new_seeds || new_stride < (int64_t)n_part * k_ref * G) return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    const dim3 grid((unsigned)((G + 255) / 256), (unsigned)(n_part * k_ref));
    k_refine_seeds<<<grid, 256, 0, (cudaStream_t)cuda_stream>>>(seeds, seed_stride, ref_seed, k_ref, g, G, new_seeds, new_stride);
    CU(ctx, cudaGetLastError());
    return COMET_OK;
}

static int launch_classify_seeds(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int32_t charge,
                                 double bz_tesla, double step_cm, int32_t n_steps, double r_stop_cm,
                                 const double* wire_a, const double* wire_b, int32_t n_wires, const int32_t* fired_wire,
                                 const int32_t* hit_off, const double* rho, int32_t n_fired, int32_t n_hits,
                                 double cutoff_cm, const int64_t* seed_idx, int32_t n_sel, const double* rss,
                                 double* dca, uint8_t* cls, double* seed_out, double* rss_out, cudaStream_t st,
                                 const int32_t* dyn = nullptr)
{
    ClassifyArgs a;
    memset(&a, 0, sizeof(a));
    a.dyn = dyn;
    a.seeds = seeds;
    a.stride = seed_stride;
    a.qkb = COMET_KAPPA * (double)charge * bz_tesla;
    a.hk = make_stepk_host(step_cm);
    a.n_steps = n_steps;
    a.r_stop2 = r_stop_cm * r_stop_cm;
    a.wire_a = wire_a; a.wire_b = wire_b; a.n_wires = n_wires; a.fired_wire = fired_wire;
    a.W = n_fired;
    a.hit_off = hit_off;
    a.rho = rho;
    a.n_hits = n_hits;
    a.lambda = cutoff_cm;
    a.ck = nullptr; a.n_ck = 0; a.rss = nullptr;
    memset(&a.po, 0, sizeof(a.po));
    const bool field = ctx->field.B != nullptr;
    if (field) a.qkb = COMET_KAPPA * (double)charge;
    a.F = ctx->field;
    a.h_min = step_cm / 64.0;
    const size_t smem = (size_t)(n_steps + 1) * (field ? 7 : 6) * sizeof(double);
    if (field) k_classify_seeds<true><<<n_sel, 256, smem, st>>>(a, seed_idx, rss, dca, cls, seed_out, rss_out);
    else k_classify_seeds<false><<<n_sel, 256, smem, st>>>(a, seed_idx, rss, dca, cls, seed_out, rss_out);
    CU(ctx, cudaGetLastError());
    return COMET_OK;
}

extern "C" int comet_classify_seeds(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds,
                                    int32_t charge, double bz_tesla, double step_cm, int32_t n_steps,
                                    double r_stop_cm,
                                    const double* wire_a, const double* wire_b, int32_t n_wires,
                                    const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                                    int32_t n_fired, int32_t n_hits, double cutoff_cm,
                                    const int64_t* seed_idx, int32_t n_sel, double* dca, uint8_t* cls,
                                    void* cuda_stream)
{
    if (!ctx || n_seeds < 0 || seed_stride < n_seeds || bad_physics(charge, bz_tesla, step_cm, n_steps) ||
        !(r_stop_cm >= 0.0) || n_sel < 0 ||
        bad_hits(wire_a, wire_b, n_wires, fired_wire, hit_off, rho, n_fired, n_hits, cutoff_cm))
        return COMET_EINVAL;
    if (ctx->field.B && n_steps > COMET_MAX_STEPS_FIELD) return COMET_EINVAL;
    if (n_sel == 0) return COMET_OK;
    if (!seeds || !seed_idx || (n_fired > 0 && !dca) || (n_hits > 0 && !cls)) return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    return launch_classify_seeds(ctx, seeds, seed_stride, charge, bz_tesla, step_cm, n_steps, r_stop_cm, wire_a, wire_b, n_wires,
                                 fired_wire, hit_off, rho,
                                 n_fired, n_hits, cutoff_cm, seed_idx, n_sel, nullptr, dca, cls, nullptr, nullptr, st);
}

// work buffer of comet_scan_stage: two seed sets [6][S_max], rss [S_max], references [P][max(k_ref, k_final)]
static size_t stage_layout(int64_t n_seeds, int32_t n_part, int32_t k_ref, int32_t k_final, int64_t G,
                           int64_t* s_max, size_t* off_rss, size_t* off_ref)
{
    const int64_t s_new = (int64_t)n_part * k_ref * G;
    *s_max = ((n_seeds > s_new ? n_seeds : s_new) + 31) / 32 * 32;
    size_t o = 2 * 6 * sizeof(double) * (size_t)*s_max;
    *off_rss = o;
    o += sizeof(double) * (size_t)*s_max;
    *off_ref = o;
    o += sizeof(int64_t) * (size_t)n_part * (size_t)(k_ref > k_final ? k_ref : k_final);
    return (o + 255) / 256 * 256;
}

extern "C" size_t comet_stage_work_bytes(int64_t n_seeds, int32_t n_part, int32_t k_ref, int32_t k_final,
                                         const int32_t* n_grid)
{
    RefineGrid g;
    int64_t G = 0, s_max;
    size_t o1, o2;
    const double hw0[4] = {0.0, 0.0, 0.0, 0.0};
    if (n_seeds < 0 || n_part < 0 || n_part > COMET_MAX_PARTITIONS || k_ref < 1 || k_ref > COMET_MAX_REFS ||
        k_final < 1 || k_final > COMET_MAX_REFS || make_grid(&g, &G, hw0, n_grid))
        return 0;
    return stage_layout(n_seeds, n_part, k_ref, k_final, G, &s_max, &o1, &o2);
}

// comet_scan_stage; dyn != NULL (comet_scan_turns): n_fired / n_hits are the sizes the launches are made for, the
// list's real sizes and the loop's stop flag live on the device
static int scan_stage_impl(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds, int32_t z_run,
                           int32_t charge, double bz_tesla, double step_cm, int32_t n_steps, double r_stop_cm,
                           const double* wire_a, const double* wire_b, int32_t n_wires,
                           const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                           int32_t n_fired, int32_t n_hits, double cutoff_cm,
                           const int64_t* part_off, int32_t n_part,
                           const double* half_width, const int32_t* n_grid, int32_t n_iter, double shrink,
                           int32_t k_ref, int32_t k_final, void* work,
                           double* final_seed, double* final_rss, double* final_dca, uint8_t* cls,
                           void* cuda_stream, const int32_t* dyn)
{
    RefineGrid g;
    int64_t G = 0;
    if (!ctx || n_seeds < 1 || seed_stride < n_seeds || bad_physics(charge, bz_tesla, step_cm, n_steps) ||
        !(r_stop_cm >= 0.0) ||
        bad_hits(wire_a, wire_b, n_wires, fired_wire, hit_off, rho, n_fired, n_hits, cutoff_cm) ||
        n_part < 1 || n_part > COMET_MAX_PARTITIONS || !part_off || n_iter < 0 || !(shrink > 0.0) || !isfinite(shrink) ||
        k_ref < 1 || k_ref > COMET_MAX_REFS || k_final < 1 || k_final > COMET_MAX_REFS || bad_zrun(z_run) ||
        make_grid(&g, &G, half_width, n_grid) || !seeds || !work || !final_seed || !final_rss ||
        (n_fired > 0 && !final_dca) || (n_hits > 0 && !cls))
        return COMET_EINVAL;
    PartOff po;
    if (fill_partoff(&po, part_off, n_part, n_seeds, true) || po.off[0] != 0 || po.off[n_part] != n_seeds) return COMET_EINVAL;
    int64_t s_max;
    size_t off_rss, off_ref;
    stage_layout(n_seeds, n_part, k_ref, k_final, G, &s_max, &off_rss, &off_ref);
    double* set[2] = {(double*)work, (double*)work + 6 * s_max};
    double* rss = (double*)((char*)work + off_rss);
    int64_t* ref = (int64_t*)((char*)work + off_ref);
    // iteration 0 scans the caller's seeds; iteration i > 0 the set written by the refinement before it
    const double* cur = seeds;
    int64_t cur_stride = seed_stride, cur_n = n_seeds;
    int64_t po_cur[COMET_MAX_PARTITIONS + 1];
    for (int p = 0; p <= n_part; ++p) po_cur[p] = part_off[p];
    double hw[4] = {half_width[0], half_width[1], half_width[2], half_width[3]};
    int rc;
    for (int it = 0; ; ++it) {
        // (the caller's promise is about the seeds it passed: the refined sets are checked on the device)
        rc = scan_rss_impl(ctx, nullptr, nullptr, cur, cur_stride, cur_n, it == 0 ? z_run : 0, charge, bz_tesla, step_cm, n_steps,
                           r_stop_cm, wire_a, wire_b, n_wires, fired_wire, hit_off, rho, n_fired, n_hits, cutoff_cm, rss, nullptr,
                           cuda_stream, dyn, it > 0);
        if (rc) return rc;
        if (it == n_iter) break;
        rc = comet_select_references(ctx, cur, cur_stride, cur_n, rss, po_cur, n_part, hw, k_ref, ref, cuda_stream);
        if (rc) return rc;
        double* nxt = set[it & 1];
        rc = comet_refine_seeds(ctx, cur, cur_stride, cur_n, ref, n_part, k_ref, hw, n_grid, nxt, s_max, cuda_stream);
        if (rc) return rc;
        cur = nxt;
        cur_stride = s_max;
        cur_n = (int64_t)n_part * k_ref * G;
        for (int p = 0; p <= n_part; ++p) po_cur[p] = (int64_t)p * k_ref * G;
        for (int d = 0; d < 4; ++d) hw[d] = hw[d] * shrink;
    }
    rc = comet_select_references(ctx, cur, cur_stride, cur_n, rss, po_cur, n_part, hw, k_final, ref, cuda_stream);
    if (rc) return rc;
    // the wire table is the one comet_scan_rss has just written on this stream
    return launch_classify_seeds(ctx, cur, cur_stride, charge, bz_tesla, step_cm, n_steps, r_stop_cm, wire_a, wire_b, n_wires,
                                 fired_wire, hit_off, rho,
                                 n_fired, n_hits, cutoff_cm, ref, n_part * k_final, rss, final_dca, cls, final_seed,
                                 final_rss, (cudaStream_t)cuda_stream, dyn);
}

extern "C" int comet_scan_stage(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds, int32_t z_run,
                                int32_t charge, double bz_tesla, double step_cm, int32_t n_steps, double r_stop_cm,
                                const double* wire_a, const double* wire_b, int32_t n_wires,
                                const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                                int32_t n_fired, int32_t n_hits, double cutoff_cm,
                                const int64_t* part_off, int32_t n_part,
                                const double* half_width, const int32_t* n_grid, int32_t n_iter, double shrink,
                                int32_t k_ref, int32_t k_final, void* work,
                                double* final_seed, double* final_rss, double* final_dca, uint8_t* cls,
                                void* cuda_stream)
{
    return scan_stage_impl(ctx, seeds, seed_stride, n_seeds, z_run, charge, bz_tesla, step_cm, n_steps, r_stop_cm, wire_a, wire_b,
                           n_wires, fired_wire, hit_off, rho, n_fired, n_hits, cutoff_cm, part_off, n_part, half_width, n_grid,
                           n_iter, shrink, k_ref, k_final, work, final_seed, final_rss, final_dca, cls, cuda_stream, nullptr);
}

// ---------------------------------------------------------------------------------------------
// sequential stages with hit removal (readings R33-R34)
// ---------------------------------------------------------------------------------------------
extern "C" int comet_remove_hits(comet_ctx* ctx, const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                                 int32_t n_fired, int32_t n_hits, const uint8_t* cls, const int32_t* orig_in,
                                 int32_t* fired_out, int32_t* hit_off_out, double* rho_out, int32_t* orig_out,
                                 int32_t* counts, void* cuda_stream)
{
    if (!ctx || n_fired < 0 || n_hits < 0 || (n_hits & 1) || !hit_off || !hit_off_out || !counts ||
        (n_fired > 0 && (!fired_wire || !fired_out)) || (n_hits > 0 && (!rho || !cls || !rho_out)))
        return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    k_remove_hits<<<1, COMET_RM_THREADS, 0, (cudaStream_t)cuda_stream>>>(fired_wire, hit_off, rho, n_fired, cls, orig_in,
                                                                        fired_out, hit_off_out, rho_out, orig_out, counts);
    CU(ctx, cudaGetLastError());
    return COMET_OK;
}

// work buffer of comet_scan_turns: the stage work, two reduced hit lists (fired, hit_off, rho, orig), the
// stage's classification and DCAs, the two counters
struct TurnsLayout {
    size_t stage, list[2], cls, dca, counts, total;
    size_t o_fired, o_off, o_rho, o_orig;     // within a list
};
static TurnsLayout turns_layout(size_t stage_bytes, int32_t n_fired, int32_t n_hits)
{
    TurnsLayout L;
    auto up = [](size_t v) { return (v + 255) / 256 * 256; };
    L.o_fired = 0;
    L.o_off = up(sizeof(int32_t) * (size_t)n_fired);
    L.o_rho = L.o_off + up(sizeof(int32_t) * ((size_t)n_fired + 1));
    L.o_orig = L.o_rho + up(sizeof(double) * (size_t)n_hits);
    const size_t list_bytes = L.o_orig + up(sizeof(int32_t) * (size_t)n_hits);
    size_t o = up(stage_bytes);
    L.stage = 0;
    L.list[0] = o; o += list_bytes;
    L.list[1] = o; o += list_bytes;
    L.cls = o; o += up((size_t)n_hits);
    L.dca = o; o += up(sizeof(double) * (size_t)n_fired);
    L.counts = o; o += 256;
    L.total = o;
    return L;
}

extern "C" size_t comet_turns_work_bytes(int64_t max_partition_seeds, int32_t n_fired, int32_t n_hits, int32_t k_ref,
                                         const int32_t* n_grid)
{
    if (n_fired < 0 || n_hits < 0) return 0;
    const size_t sb = comet_stage_work_bytes(max_partition_seeds, 1, k_ref, 1, n_grid);
    if (!sb) return 0;
    return turns_layout(sb, n_fired, n_hits).total;
}

extern "C" int comet_scan_turns(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds, int32_t z_run,
                                int32_t charge, double bz_tesla, double step_cm, int32_t n_steps, double r_stop_cm,
                                const double* wire_a, const double* wire_b, int32_t n_wires,
                                const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                                int32_t n_fired, int32_t n_hits, double cutoff_cm,
                                const int64_t* part_off, int32_t n_part,
                                const double* half_width, const int32_t* n_grid, int32_t n_iter, double shrink,
                                int32_t k_ref, int32_t min_wires, int32_t max_tracks, void* work,
                                double* turn_seed, double* turn_rss, uint8_t* turn_cls,
                                int32_t* done, int32_t* wires_before, void* cuda_stream)
{
    if (!ctx || n_part < 1 || n_part > COMET_MAX_PARTITIONS || !part_off || !work || !turn_seed || !turn_rss ||
        (n_hits > 0 && !turn_cls) || !done || !wires_before || (n_hits & 1) || min_wires < 0 || max_tracks < 0 ||
        n_seeds < 1 || seed_stride < n_seeds || bad_zrun(z_run))
        return COMET_EINVAL;
    PartOff po;
    if (fill_partoff(&po, part_off, n_part, n_seeds, true)) return COMET_EINVAL;
    int64_t max_part = 0;
    for (int p = 0; p < n_part; ++p)
        if (po.off[p + 1] - po.off[p] > max_part) max_part = po.off[p + 1] - po.off[p];
    const size_t sb = comet_stage_work_bytes(max_part, 1, k_ref, 1, n_grid);
    if (!sb) return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const TurnsLayout L = turns_layout(sb, n_fired, n_hits);
    char* Wk = (char*)work;
    uint8_t* cls_stage = (uint8_t*)(Wk + L.cls);
    double* dca_stage = (double*)(Wk + L.dca);
    int32_t* dyn = (int32_t*)(Wk + L.counts);              // {fired wires left, entries left, stop flag, stages done}
    // nothing done yet: NaN seeds / RSS (all-ones is a NaN), empty classification
    CU(ctx, cudaMemsetAsync(turn_seed, 0xff, sizeof(double) * 6 * (size_t)n_part, st));
    CU(ctx, cudaMemsetAsync(turn_rss, 0xff, sizeof(double) * (size_t)n_part, st));
    if (n_hits) CU(ctx, cudaMemsetAsync(turn_cls, 0, (size_t)n_part * (size_t)n_hits, st));
    k_turn_init<<<1, 1, 0, st>>>(dyn, n_fired, n_hits, done, wires_before, n_part);
    // Every stage is enqueued for the event's own list sizes: after a removal the list is padded back to n_fired wires with
    // wires without entries (k_remove_hits), which no kernel finds anything on; Eq. (1) runs over the dyn[0] wires that
    // are left (k_rss_sum), and once the stop rule has fired (k_turn_gate) every kernel of the later stages returns at once.
    // No host read, no synchronisation: the loop can be captured into a CUDA graph.
    const int32_t* cur_fw = fired_wire;
    const int32_t* cur_ho = hit_off;
    const double* cur_rho = rho;
    const int32_t* cur_orig = nullptr;                   // identity
    int flip = 0;
    for (int p = n_part - 1; p >= 0; --p) {              // the last turn first
        k_turn_gate<<<1, 1, 0, st>>>(dyn, p, min_wires, max_tracks, done, wires_before);
        const int64_t np_seeds = po.off[p + 1] - po.off[p];
        const int64_t one[2] = {0, np_seeds};
        rc = scan_stage_impl(ctx, seeds + po.off[p], seed_stride, np_seeds, (z_run > 1 && po.off[p] % z_run == 0) ? z_run : 0,
                             charge, bz_tesla, step_cm, n_steps, r_stop_cm,
                             wire_a, wire_b, n_wires, cur_fw, cur_ho, cur_rho, n_fired, n_hits, cutoff_cm, one, 1,
                             half_width, n_grid, n_iter, shrink, k_ref, 1, Wk + L.stage,
                             turn_seed + 6 * (size_t)p, turn_rss + p, dca_stage, cls_stage, st, dyn);
        if (rc) return rc;
        if (n_hits) k_scatter_cls<<<(n_hits + 255) / 256, 256, 0, st>>>(cls_stage, cur_orig, n_hits, turn_cls + (size_t)p * n_hits, dyn);
        char* Lb = Wk + L.list[flip];
        int32_t* n_fw = (int32_t*)(Lb + L.o_fired);
        int32_t* n_ho = (int32_t*)(Lb + L.o_off);
        double* n_rho = (double*)(Lb + L.o_rho);
        int32_t* n_orig = (int32_t*)(Lb + L.o_orig);
        k_remove_hits<<<1, COMET_RM_THREADS, 0, st>>>(cur_fw, cur_ho, cur_rho, n_fired, cls_stage, cur_orig, n_fw, n_ho, n_rho,
                                                      n_orig, dyn, 1, dyn + 2);
        CU(ctx, cudaGetLastError());
        cur_fw = n_fw; cur_ho = n_ho; cur_rho = n_rho; cur_orig = n_orig;
        flip ^= 1;
    }
    return COMET_OK;
}

// ---------------------------------------------------------------------------------------------
// Hough-transform transverse seeding (readings R35-R37)
// ---------------------------------------------------------------------------------------------
extern "C" size_t comet_hough_work_bytes(int32_t n_events)
{
    return n_events < 0 ? 0 : sizeof(HoughWork) * (size_t)(n_events > 0 ? n_events : 1);
}

extern "C" int comet_hough_seeds(comet_ctx* ctx, const double* wire_a, const double* wire_b, int32_t n_wires,
                                 const int32_t* fired_wire, const int32_t* ev_off, int32_t n_events,
                                 const double* cos_tab, const double* sin_tab, int32_t n_phi,
                                 double rho_min, double inv_drho, int32_t n_rho,
                                 int32_t charge, double bz_tesla, double r_seed_cm, void* work,
                                 int32_t* acc, int32_t* peak, double* circle, void* cuda_stream)
{
    if (!ctx || n_events < 0 || n_events > 65535 || n_wires < 0 || n_phi < 1 || n_rho < 1 || n_rho > 32768 ||
        (int64_t)n_phi * n_rho >= ((int64_t)1 << 31) || !(inv_drho > 0.0) || !isfinite(inv_drho) || !isfinite(rho_min) ||
        !(r_seed_cm > 0.0) || (charge != 1 && charge != -1) || !isfinite(bz_tesla) || bz_tesla == 0.0 ||
        !cos_tab || !sin_tab || !ev_off || !work || (n_events > 0 && (!peak || !circle)) ||
        (n_wires > 0 && (!wire_a || !wire_b)))
        return COMET_EINVAL;
    if (n_events == 0) return COMET_OK;
    int rc = set_device(ctx);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // directions per CTA: at least one CTA per SM, and small CTAs (about COMET_HT_BINS bins in shared memory) so
    // that a batch of events runs as many short CTAs per SM rather than one or two long waves
    int64_t ctas_per_event = (ctx->n_sm + n_events - 1) / n_events;
    int D = (int)((n_phi + ctas_per_event - 1) / ctas_per_event);
    const int d_max = COMET_HT_BINS / n_rho > 0 ? COMET_HT_BINS / n_rho : 1;
    if (D > d_max) D = d_max;
    if (D < 1) D = 1;
    if (D < COMET_HT_THREADS) {                            // a divisor of the CTA size: threads keep their direction
        int p2 = 1;
        while (2 * p2 <= D) p2 *= 2;
        D = p2;
    }
    const size_t smem = (size_t)D * n_rho * sizeof(int) + 2 * COMET_HT_THREADS * sizeof(double);
    if (smem > 48 * 1024) CU(ctx, cudaFuncSetAttribute(k_hough, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CU(ctx, cudaMemsetAsync(work, 0, sizeof(HoughWork) * (size_t)n_events, st));
    const dim3 grid((unsigned)((n_phi + D - 1) / D), (unsigned)n_events);
    k_hough<<<grid, COMET_HT_THREADS, smem, st>>>(wire_a, wire_b, n_wires, fired_wire, ev_off, cos_tab, sin_tab, n_phi, D,
                                                  rho_min, inv_drho, n_rho, charge, bz_tesla, r_seed_cm, acc, peak,
                                                  circle, (HoughWork*)work);
    CU(ctx, cudaGetLastError());
    return COMET_OK;
}

// ---------------------------------------------------------------------------------------------
// half tracks (readings R38-R42)
// ---------------------------------------------------------------------------------------------
extern "C" int comet_half_hit_masks(comet_ctx* ctx, const double* wire_a, const double* wire_b, int32_t n_wires,
                                    const int32_t* fired_wire, const int32_t* hit_off, int32_t n_fired, int32_t n_hits,
                                    const double* circle, double overlap_cm, uint8_t* in_ent, uint8_t* in_exit,
                                    void* cuda_stream)
{
    if (!ctx || n_wires < 0 || n_fired < 0 || n_hits < 0 || !circle || !(overlap_cm >= 0.0) ||
        (n_fired > 0 && (!wire_a || !wire_b || !fired_wire || !hit_off)) || (n_hits > 0 && (!in_ent || !in_exit)))
        return COMET_EINVAL;
    if (n_fired == 0) return COMET_OK;
    int rc = set_device(ctx);
    if (rc) return rc;
    k_half_masks<<<(n_fired + 255) / 256, 256, 0, (cudaStream_t)cuda_stream>>>(wire_a, wire_b, n_wires, fired_wire, hit_off,
                                                                               n_fired, circle, overlap_cm, in_ent, in_exit,
                                                                               nullptr, nullptr);
    CU(ctx, cudaGetLastError());
    return COMET_OK;
}

extern "C" int comet_flip_seeds(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds,
                                double* out, int64_t out_stride, void* cuda_stream)
{
    if (!ctx || n_seeds < 0 || seed_stride < n_seeds || out_stride < n_seeds || (n_seeds > 0 && (!seeds || !out)))
        return COMET_EINVAL;
    if (n_seeds == 0) return COMET_OK;
    int rc = set_device(ctx);
    if (rc) return rc;
    k_flip_seeds<<<(unsigned)((6 * n_seeds + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(seeds, seed_stride, n_seeds, out,
                                                                                              out_stride, 0);
    CU(ctx, cudaGetLastError());
    return COMET_OK;
}

extern "C" int comet_layer_veto(comet_ctx* ctx, const uint8_t* cls, int32_t n_sel,
                                const int32_t* fired_wire, const int32_t* hit_off, int32_t n_fired, int32_t n_hits,
                                const int32_t* wire_layer, int32_t n_wires, int32_t min_layers, uint8_t* ok,
                                void* cuda_stream)
{
    if (!ctx || n_sel < 0 || n_fired < 0 || n_hits < 0 || n_wires < 0 || (n_sel > 0 && !ok) ||
        (n_sel > 0 && n_hits > 0 && !cls) || (n_fired > 0 && (!fired_wire || !hit_off || !wire_layer)))
        return COMET_EINVAL;
    if (n_sel == 0) return COMET_OK;
    int rc = set_device(ctx);
    if (rc) return rc;
    k_layer_veto<<<(n_sel + 7) / 8, 256, 0, (cudaStream_t)cuda_stream>>>(cls, n_sel, n_hits, fired_wire, hit_off, n_fired,
                                                                        wire_layer, min_layers, ok);
    CU(ctx, cudaGetLastError());
    return COMET_OK;
}

extern "C" int comet_merge_half_sets(comet_ctx* ctx, const uint8_t* cls_e, const int32_t* orig_e, const uint8_t* ok_e,
                                     int32_t k_e, int32_t h_e, const uint8_t* cls_x, const int32_t* orig_x,
                                     const uint8_t* ok_x, int32_t k_x, int32_t h_x, int32_t n_hits,
                                     uint8_t* valid, uint8_t* cls, int32_t* n_cls, void* cuda_stream)
{
    if (!ctx || k_e < 1 || k_x < 1 || k_e > 65535 || k_x > 65535 || h_e < 0 || h_x < 0 || n_hits < 0 || h_e > n_hits ||
        h_x > n_hits || !ok_e || !ok_x || !valid || !n_cls || (n_hits > 0 && !cls) || (h_e > 0 && (!cls_e || !orig_e)) ||
        (h_x > 0 && (!cls_x || !orig_x)))
        return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    k_merge_half<<<dim3((unsigned)k_x, (unsigned)k_e), 256, 0, (cudaStream_t)cuda_stream>>>(cls_e, orig_e, ok_e, h_e, cls_x, orig_x,
                                                                                           ok_x, h_x, n_hits, valid, cls, n_cls);
    CU(ctx, cudaGetLastError());
    return COMET_OK;
}

// work buffer of comet_scan_half_tracks: the stage work, the flipped exit-side seeds, the two remove masks, the
// two half lists (fired, hit_off, rho; orig goes to the caller), the stage's DCAs, the four counters
struct HalfLayout {
    size_t stage, flip, rm[2], fw[2], ho[2], rho[2], dca, counts, total;
};
static HalfLayout half_layout(size_t stage_bytes, int64_t n_exit, int32_t n_fired, int32_t n_hits, int32_t k_final)
{
    HalfLayout L;
    auto up = [](size_t v) { return (v + 255) / 256 * 256; };
    size_t o = 0;
    L.stage = o; o += up(stage_bytes);
    L.flip = o; o += up(sizeof(double) * 6 * (size_t)n_exit);
    for (int h = 0; h < 2; ++h) {
        L.rm[h] = o; o += up((size_t)n_hits);
        L.fw[h] = o; o += up(sizeof(int32_t) * (size_t)n_fired);
        L.ho[h] = o; o += up(sizeof(int32_t) * ((size_t)n_fired + 1));
        L.rho[h] = o; o += up(sizeof(double) * (size_t)n_hits);
    }
    L.dca = o; o += up(sizeof(double) * (size_t)k_final * (size_t)n_fired);
    L.counts = o; o += 256;
    L.total = o;
    return L;
}

extern "C" size_t comet_half_work_bytes(int64_t n_seeds_ent, int64_t n_seeds_exit, int32_t n_fired, int32_t n_hits,
                                        int32_t k_ref, int32_t k_final, const int32_t* n_grid)
{
    if (n_seeds_ent < 1 || n_seeds_exit < 1 || n_fired < 0 || n_hits < 0) return 0;
    const size_t sb = comet_stage_work_bytes(n_seeds_ent > n_seeds_exit ? n_seeds_ent : n_seeds_exit, 1, k_ref, k_final, n_grid);
    if (!sb) return 0;
    return half_layout(sb, n_seeds_exit, n_fired, n_hits, k_final).total;
}

static int half_tracks_impl(comet_ctx* ctx, const double* seeds_ent, int64_t stride_ent, int64_t n_ent,
                            const double* seeds_exit, int64_t stride_exit, int64_t n_exit,
                            int32_t charge, double bz_tesla, double step_cm, int32_t n_steps, double r_stop_cm,
                                      const double* wire_a, const double* wire_b, int32_t n_wires,
                                      const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                                      int32_t n_fired, int32_t n_hits, double cutoff_cm,
                                      const int32_t* wire_layer, const double* circle, double overlap_cm, int32_t min_layers,
                                      const double* half_width, const int32_t* n_grid, int32_t n_iter, double shrink,
                                      int32_t k_ref, int32_t k_final, void* work,
                                      double* half_seed, double* half_rss, uint8_t* half_ok, uint8_t* half_cls,
                                      int32_t* half_orig, int32_t* counts_host,
                                      uint8_t* valid, uint8_t* cls, int32_t* n_cls, void* cuda_stream)
{
    if (!ctx || n_ent < 1 || n_exit < 1 || stride_ent < n_ent || stride_exit < n_exit || !seeds_ent || !seeds_exit ||
        n_fired < 0 || n_hits < 0 || (n_hits & 1) ||
        !circle || !(overlap_cm >= 0.0) || !work || !half_seed || !half_rss || !half_ok || !counts_host || !valid || !n_cls ||
        !hit_off || (n_fired > 0 && (!wire_layer || !fired_wire)) || (n_hits > 0 && (!rho || !half_cls || !half_orig || !cls)))
        return COMET_EINVAL;
    const size_t sb = comet_stage_work_bytes(n_ent > n_exit ? n_ent : n_exit, 1, k_ref, k_final, n_grid);
    if (!sb) return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const HalfLayout L = half_layout(sb, n_exit, n_fired, n_hits, k_final);
    char* Wk = (char*)work;
    int32_t* counts = (int32_t*)(Wk + L.counts);
    double* flipped = (double*)(Wk + L.flip);
    double* dca_stage = (double*)(Wk + L.dca);
    // the two hit lists (R39) and the backward seeds (R38)
    if (n_fired)
        k_half_masks<<<(n_fired + 255) / 256, 256, 0, st>>>(wire_a, wire_b, n_wires, fired_wire, hit_off, n_fired, circle,
                                                            overlap_cm, nullptr, nullptr, (uint8_t*)(Wk + L.rm[0]),
                                                            (uint8_t*)(Wk + L.rm[1]));
    for (int h = 0; h < 2; ++h)
        k_remove_hits<<<1, COMET_RM_THREADS, 0, st>>>(fired_wire, hit_off, rho, n_fired, (const uint8_t*)(Wk + L.rm[h]), nullptr,
                                                      (int32_t*)(Wk + L.fw[h]), (int32_t*)(Wk + L.ho[h]),
                                                      (double*)(Wk + L.rho[h]), half_orig ? half_orig + (size_t)h * n_hits : nullptr,
                                                      counts + 2 * h);
    k_flip_seeds<<<(unsigned)((6 * n_exit + 255) / 256), 256, 0, st>>>(seeds_exit, stride_exit, n_exit, flipped, n_exit, 0);
    CU(ctx, cudaGetLastError());
    CU(ctx, cudaMemcpyAsync(counts_host, counts, 4 * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    CU(ctx, cudaStreamSynchronize(st));              // the sizes of the two lists set the launches of the scans
    const size_t side_cls = (size_t)k_final * (size_t)n_hits;
    for (int h = 0; h < 2; ++h) {
        const int32_t w = counts_host[2 * h], hh = counts_host[2 * h + 1];
        double* rho_h = (double*)(Wk + L.rho[h]);
        if (h == 1 && hh) k_negate<<<(hh + 255) / 256, 256, 0, st>>>(rho_h, hh);     // R38: left and right swap
        const int64_t ns = h == 0 ? n_ent : n_exit;
        const int64_t one[2] = {0, ns};
        double* fs = half_seed + (size_t)h * k_final * 6;
        uint8_t* cls_h = half_cls ? half_cls + (size_t)h * side_cls : nullptr;
        rc = comet_scan_stage(ctx, h == 0 ? seeds_ent : flipped, h == 0 ? stride_ent : ns, ns, 0, h == 0 ? charge : -charge, bz_tesla, step_cm, n_steps,
                              r_stop_cm, wire_a, wire_b, n_wires, (const int32_t*)(Wk + L.fw[h]), (const int32_t*)(Wk + L.ho[h]),
                              rho_h, w, hh, cutoff_cm, one, 1, half_width, n_grid, n_iter, shrink, k_ref, k_final,
                              Wk + L.stage, fs, half_rss + (size_t)h * k_final, dca_stage, cls_h, st);
        if (rc) return rc;
        if (h == 1) k_flip_seeds<<<(6 * k_final + 255) / 256, 256, 0, st>>>(fs, 0, k_final, fs, 0, 1);
        k_layer_veto<<<(k_final + 7) / 8, 256, 0, st>>>(cls_h, k_final, hh, (const int32_t*)(Wk + L.fw[h]),
                                                        (const int32_t*)(Wk + L.ho[h]), w, wire_layer, min_layers,
                                                        half_ok + (size_t)h * k_final);
    }
    k_merge_half<<<dim3((unsigned)k_final, (unsigned)k_final), 256, 0, st>>>(
        half_cls, half_orig, half_ok, counts_host[1], half_cls ? half_cls + side_cls : nullptr,
        half_orig ? half_orig + n_hits : nullptr, half_ok + k_final, counts_host[3], n_hits, valid, cls, n_cls);
    CU(ctx, cudaGetLastError());
    return COMET_OK;
}

extern "C" int comet_scan_half_tracks(comet_ctx* ctx, const double* seeds_ent, int64_t n_ent,
                                      const double* seeds_exit, int64_t n_exit,
                                      int32_t charge, double bz_tesla, double step_cm, int32_t n_steps, double r_stop_cm,
                                      const double* wire_a, const double* wire_b, int32_t n_wires,
                                      const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                                      int32_t n_fired, int32_t n_hits, double cutoff_cm,
                                      const int32_t* wire_layer, const double* circle, double overlap_cm, int32_t min_layers,
                                      const double* half_width, const int32_t* n_grid, int32_t n_iter, double shrink,
                                      int32_t k_ref, int32_t k_final, void* work,
                                      double* half_seed, double* half_rss, uint8_t* half_ok, uint8_t* half_cls,
                                      int32_t* half_orig, int32_t* counts_host,
                                      uint8_t* valid, uint8_t* cls, int32_t* n_cls, void* cuda_stream)
{
    return half_tracks_impl(ctx, seeds_ent, n_ent, n_ent, seeds_exit, n_exit, n_exit, charge, bz_tesla, step_cm, n_steps,
                            r_stop_cm, wire_a, wire_b, n_wires, fired_wire, hit_off, rho, n_fired, n_hits, cutoff_cm,
                            wire_layer, circle, overlap_cm, min_layers, half_width, n_grid, n_iter, shrink, k_ref, k_final,
                            work, half_seed, half_rss, half_ok, half_cls, half_orig, counts_host, valid, cls, n_cls,
                            cuda_stream);
}

// work buffer of comet_scan_turns_half: the half-track work, the half-track outputs of a turn, the chosen set,
// two reduced hit lists (fired, hit_off, rho, orig), the counters
struct TurnsHalfLayout {
    size_t half, hseed, hrss, hok, hcls, horig, valid, cls, ncls, best, pick, list[2], o_fired, o_off, o_rho, o_orig, total;
};
static TurnsHalfLayout turns_half_layout(size_t half_bytes, int32_t n_fired, int32_t n_hits, int32_t K)
{
    TurnsHalfLayout L;
    auto up = [](size_t v) { return (v + 255) / 256 * 256; };
    size_t o = 0;
    L.half = o; o += up(half_bytes);
    L.hseed = o; o += up(sizeof(double) * 2 * 6 * (size_t)K);
    L.hrss = o; o += up(sizeof(double) * 2 * (size_t)K);
    L.hok = o; o += up(2 * (size_t)K);
    L.hcls = o; o += up(2 * (size_t)K * (size_t)n_hits);
    L.horig = o; o += up(sizeof(int32_t) * 2 * (size_t)n_hits);
    L.valid = o; o += up((size_t)K * K);
    L.cls = o; o += up((size_t)K * K * (size_t)n_hits);
    L.ncls = o; o += up(sizeof(int32_t) * (size_t)K * K);
    L.best = o; o += up((size_t)n_hits);
    L.pick = o; o += 256;                                   // counts [2] then pick [3], read back together
    L.o_fired = 0;
    L.o_off = up(sizeof(int32_t) * (size_t)n_fired);
    L.o_rho = L.o_off + up(sizeof(int32_t) * ((size_t)n_fired + 1));
    L.o_orig = L.o_rho + up(sizeof(double) * (size_t)n_hits);
    const size_t list_bytes = L.o_orig + up(sizeof(int32_t) * (size_t)n_hits);
    L.list[0] = o; o += list_bytes;
    L.list[1] = o; o += list_bytes;
    L.total = o;
    return L;
}

extern "C" size_t comet_turns_half_work_bytes(int64_t max_seeds_ent, int64_t max_seeds_exit, int32_t n_fired, int32_t n_hits,
                                              int32_t k_ref, int32_t k_final, const int32_t* n_grid)
{
    const size_t hb = comet_half_work_bytes(max_seeds_ent, max_seeds_exit, n_fired, n_hits, k_ref, k_final, n_grid);
    if (!hb) return 0;
    return turns_half_layout(hb, n_fired, n_hits, k_final).total;
}

extern "C" int comet_scan_turns_half(comet_ctx* ctx, const double* seeds_ent, const int64_t* off_ent, int64_t n_ent,
                                     const double* seeds_exit, const int64_t* off_exit, int64_t n_exit, int32_t n_part,
                                     int32_t charge, double bz_tesla, double step_cm, int32_t n_steps, double r_stop_cm,
                                     const double* wire_a, const double* wire_b, int32_t n_wires,
                                     const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                                     int32_t n_fired, int32_t n_hits, double cutoff_cm,
                                     const int32_t* wire_layer, const double* circle, double overlap_cm, int32_t min_layers,
                                     const double* half_width, const int32_t* n_grid, int32_t n_iter, double shrink,
                                     int32_t k_ref, int32_t k_final, int32_t min_wires, int32_t max_tracks, void* work,
                                     int32_t* turn_pair, int32_t* turn_n, double* turn_seed, uint8_t* turn_cls,
                                     int32_t* done_host, int32_t* wires_before_host, void* cuda_stream)
{
    if (!ctx || n_part < 1 || n_part > COMET_MAX_PARTITIONS || !off_ent || !off_exit || !work || !turn_pair || !turn_n ||
        !turn_seed || (n_hits > 0 && !turn_cls) || !done_host || !wires_before_host || (n_hits & 1) || n_hits < 0 ||
        n_fired < 0 || min_wires < 0 || max_tracks < 0 || n_ent < 1 || n_exit < 1)
        return COMET_EINVAL;
    PartOff pe, px;
    if (fill_partoff(&pe, off_ent, n_part, n_ent, true) || fill_partoff(&px, off_exit, n_part, n_exit, true)) return COMET_EINVAL;
    int64_t max_e = 0, max_x = 0;
    for (int p = 0; p < n_part; ++p) {
        if (pe.off[p + 1] - pe.off[p] > max_e) max_e = pe.off[p + 1] - pe.off[p];
        if (px.off[p + 1] - px.off[p] > max_x) max_x = px.off[p + 1] - px.off[p];
    }
    const size_t hb = comet_half_work_bytes(max_e, max_x, n_fired, n_hits, k_ref, k_final, n_grid);
    if (!hb) return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int K = k_final;
    const TurnsHalfLayout L = turns_half_layout(hb, n_fired, n_hits, K);
    char* Wk = (char*)work;
    double* hseed = (double*)(Wk + L.hseed);
    uint8_t* v_valid = (uint8_t*)(Wk + L.valid);
    uint8_t* v_cls = (uint8_t*)(Wk + L.cls);
    int32_t* v_ncls = (int32_t*)(Wk + L.ncls);
    uint8_t* cls_best = (uint8_t*)(Wk + L.best);
    int32_t* counts = (int32_t*)(Wk + L.pick);              // counts [0..1], pick [2..4]
    // nothing done yet: pairs -1, sizes 0, NaN seeds (all-ones is a NaN), empty classification
    CU(ctx, cudaMemsetAsync(turn_pair, 0xff, sizeof(int32_t) * 2 * (size_t)n_part, st));
    CU(ctx, cudaMemsetAsync(turn_n, 0, sizeof(int32_t) * (size_t)n_part, st));
    CU(ctx, cudaMemsetAsync(turn_seed, 0xff, sizeof(double) * 12 * (size_t)n_part, st));
    if (n_hits) CU(ctx, cudaMemsetAsync(turn_cls, 0, (size_t)n_part * (size_t)n_hits, st));
    for (int p = 0; p < n_part; ++p) { done_host[p] = 0; wires_before_host[p] = 0; }
    const int32_t* cur_fw = fired_wire;
    const int32_t* cur_ho = hit_off;
    const double* cur_rho = rho;
    const int32_t* cur_orig = nullptr;                      // identity
    int32_t cur_w = n_fired, cur_h = n_hits, n_done = 0, flip = 0;
    for (int p = n_part - 1; p >= 0; --p) {                 // the last turn first
        if (cur_w < min_wires || n_done >= max_tracks) break;
        int32_t hc4[4];
        rc = half_tracks_impl(ctx, seeds_ent + pe.off[p], n_ent, pe.off[p + 1] - pe.off[p],
                              seeds_exit + px.off[p], n_exit, px.off[p + 1] - px.off[p], charge, bz_tesla, step_cm, n_steps,
                              r_stop_cm, wire_a, wire_b, n_wires, cur_fw, cur_ho, cur_rho, cur_w, cur_h, cutoff_cm, wire_layer,
                              circle, overlap_cm, min_layers, half_width, n_grid, n_iter, shrink, k_ref, K, Wk + L.half,
                              hseed, (double*)(Wk + L.hrss), (uint8_t*)(Wk + L.hok), (uint8_t*)(Wk + L.hcls),
                              (int32_t*)(Wk + L.horig), hc4, v_valid, v_cls, v_ncls, st);
        if (rc) return rc;
        wires_before_host[p] = cur_w;
        k_best_pair<<<1, 256, 0, st>>>(v_valid, v_ncls, v_cls, K, K, cur_h, hseed, K, cls_best, counts + 2,
                                       turn_pair + 2 * (size_t)p, turn_n + p, turn_seed + 12 * (size_t)p);
        if (cur_h) k_scatter_cls<<<(cur_h + 255) / 256, 256, 0, st>>>(cls_best, cur_orig, cur_h, turn_cls + (size_t)p * n_hits);
        char* Lb = Wk + L.list[flip];
        int32_t* n_fw = (int32_t*)(Lb + L.o_fired);
        int32_t* n_ho = (int32_t*)(Lb + L.o_off);
        double* n_rho = (double*)(Lb + L.o_rho);
        int32_t* n_orig = (int32_t*)(Lb + L.o_orig);
        k_remove_hits<<<1, COMET_RM_THREADS, 0, st>>>(cur_fw, cur_ho, cur_rho, cur_w, cls_best, cur_orig, n_fw, n_ho, n_rho,
                                                      n_orig, counts);
        CU(ctx, cudaGetLastError());
        int32_t hc[5];
        CU(ctx, cudaMemcpyAsync(hc, counts, sizeof(hc), cudaMemcpyDeviceToHost, st));
        CU(ctx, cudaStreamSynchronize(st));
        if (hc[2] < 0) break;                               // no valid pair: the reconstruction stops
        done_host[p] = 1;
        n_done += 1;
        cur_fw = n_fw; cur_ho = n_ho; cur_rho = n_rho; cur_orig = n_orig;
        cur_w = hc[0]; cur_h = hc[1];
        flip ^= 1;
    }
    return COMET_OK;
}

// ---------------------------------------------------------------------------------------------
// seed grids as inputs (readings R17, R44)
// ---------------------------------------------------------------------------------------------
extern "C" int32_t comet_grid_z_run(int32_t n_z)
{
    if (n_z < 1) return 0;
    int32_t r = 1;
    while (r < 32 && n_z % (2 * r) == 0) r *= 2;
    return r;
}

static int make_shape(GridShape* g, int32_t n_part, int32_t n_p, int32_t n_ct, int32_t n_phi, int32_t n_z)
{
    if (n_part < 1 || n_part > COMET_MAX_PARTITIONS || n_p < 1 || n_ct < 1 || n_phi < 1 || n_z < 1 || n_p > 65536 ||
        n_ct > 65536 || n_phi > 65536 || n_z > 65536)
        return COMET_EINVAL;
    g->n_p = n_p; g->n_ct = n_ct; g->n_phi = n_phi; g->n_z = n_z;
    g->G = (int64_t)n_p * n_ct * n_phi * n_z;
    if (g->G > ((int64_t)1 << 40)) return COMET_EINVAL;
    g->A = 2 + n_p + 2 * n_ct + 2 * n_phi + n_z;
    return COMET_OK;
}

extern "C" size_t comet_grid_axes_len(int32_t n_p, int32_t n_ct, int32_t n_phi, int32_t n_z)
{
    GridShape g;
    return make_shape(&g, 1, n_p, n_ct, n_phi, n_z) ? 0 : (size_t)g.A;
}

extern "C" int comet_seed_grid(comet_ctx* ctx, const double* axes, int32_t n_part, int32_t n_p, int32_t n_ct,
                               int32_t n_phi, int32_t n_z, double* seeds, int64_t seed_stride, void* cuda_stream)
{
    GridShape g;
    if (!ctx || make_shape(&g, n_part, n_p, n_ct, n_phi, n_z) || !axes || !seeds || seed_stride < g.G * n_part)
        return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    const int64_t total = g.G * n_part;
    k_seed_grid<<<(unsigned)((total + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(axes, g, total, seeds, seed_stride);
    CU(ctx, cudaGetLastError());
    return COMET_OK;
}

extern "C" int comet_seed_runs(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds,
                               int32_t* z_run_host, void* cuda_stream)
{
    if (!ctx || n_seeds < 0 || seed_stride < n_seeds || !z_run_host || (n_seeds > 0 && !seeds)) return COMET_EINVAL;
    *z_run_host = 32;
    if (n_seeds < 2) return COMET_OK;
    int rc = set_device(ctx);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    unsigned int* flag = ctx->zg_flag + COMET_MAX_LANES;      // a slot of its own (the lanes use [0, COMET_MAX_LANES))
    CU(ctx, cudaMemsetAsync(flag, 0xff, sizeof(unsigned int), st));
    k_zgroup_check<<<(unsigned)((n_seeds + 255) / 256), 256, 0, st>>>(seeds, seed_stride, n_seeds, flag);
    CU(ctx, cudaGetLastError());
    unsigned int f = 0;
    CU(ctx, cudaMemcpyAsync(&f, flag, sizeof(f), cudaMemcpyDeviceToHost, st));
    CU(ctx, cudaStreamSynchronize(st));
    *z_run_host = f > 32u ? 32 : (int32_t)f;
    return COMET_OK;
}

extern "C" int comet_set_geometry(comet_ctx* ctx, const double* wire_a_host, const double* wire_b_host, int32_t n_wires,
                                  void* cuda_stream)
{
    if (!ctx || n_wires < 0 || (n_wires > 0 && (!wire_a_host || !wire_b_host))) return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CU(ctx, cudaStreamSynchronize(st));
    if (ctx->geom_a) { cudaFree(ctx->geom_a); ctx->geom_a = nullptr; }
    if (ctx->geom_b) { cudaFree(ctx->geom_b); ctx->geom_b = nullptr; }
    ctx->geom_n = 0;
    if (n_wires == 0) return COMET_OK;
    const size_t bytes = sizeof(double) * 3 * (size_t)n_wires;
    cudaError_t e = cudaMalloc(&ctx->geom_a, bytes);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->geom_b, bytes);
    if (e != cudaSuccess) { ctx->last_cuda = (int)e; cudaGetLastError(); return COMET_ENOMEM; }
    CU(ctx, cudaMemcpyAsync(ctx->geom_a, wire_a_host, bytes, cudaMemcpyHostToDevice, st));
    CU(ctx, cudaMemcpyAsync(ctx->geom_b, wire_b_host, bytes, cudaMemcpyHostToDevice, st));
    CU(ctx, cudaStreamSynchronize(st));
    ctx->geom_n = n_wires;
    return COMET_OK;
}

extern "C" int comet_get_geometry(const comet_ctx* ctx, const double** wire_a_dev, const double** wire_b_dev, int32_t* n_wires)
{
    if (!ctx || !wire_a_dev || !wire_b_dev || !n_wires) return COMET_EINVAL;
    *wire_a_dev = ctx->geom_a; *wire_b_dev = ctx->geom_b; *n_wires = ctx->geom_n;
    return COMET_OK;
}

// ---------------------------------------------------------------------------------------------
// whole event from host buffers
// ---------------------------------------------------------------------------------------------
static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

static int grow(comet_ctx* ctx, void** buf, size_t* have, size_t need)
{
    if (need <= *have) return COMET_OK;
    if (*buf) { CU(ctx, cudaFree(*buf)); *buf = nullptr; *have = 0; }
    cudaError_t e = cudaMalloc(buf, need);
    if (e != cudaSuccess) { ctx->last_cuda = (int)e; *buf = nullptr; return COMET_ENOMEM; }
    *have = need;
    return COMET_OK;
}

extern "C" int comet_scan_event_host(comet_ctx* ctx, const double* seeds_host, int64_t n_seeds,
                                     int32_t charge, double bz_tesla, double step_cm, int32_t n_steps,
                                     double r_stop_cm,
                                     const double* wire_a_host, const double* wire_b_host, int32_t n_wires,
                                     const int32_t* fired_wire_host, const int32_t* hit_off_host,
                                     const double* rho_host, int32_t n_fired, int32_t n_hits, double cutoff_cm,
                                     const int64_t* part_off_host, int32_t n_part, size_t track_budget_bytes,
                                     int64_t* best_seed_host, double* best_rss_host, double* best_dca_host,
                                     uint8_t* cls_host, double* rss_host, void* cuda_stream)
{
    // wire_a_host == NULL: the geometry set with comet_set_geometry, already on the device
    const bool resident = ctx && !wire_a_host && !wire_b_host && ctx->geom_n > 0;
    if (resident) n_wires = ctx->geom_n;
    if (!ctx || n_seeds < 0 || bad_physics(charge, bz_tesla, step_cm, n_steps) || !(r_stop_cm >= 0.0) ||
        bad_hits(resident ? ctx->geom_a : wire_a_host, resident ? ctx->geom_b : wire_b_host, n_wires, fired_wire_host,
                 hit_off_host, rho_host, n_fired, n_hits, cutoff_cm) ||
        n_part < 0 || n_part > COMET_MAX_PARTITIONS || (n_seeds > 0 && !seeds_host) ||
        (n_part > 0 && (!part_off_host || !best_seed_host || !best_rss_host)) ||
        (n_part > 0 && n_fired > 0 && !best_dca_host) || (n_part > 0 && n_hits > 0 && !cls_host))
        return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // ---- carve one device slab: inputs then outputs ------------------------------------------
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
    const size_t o_seeds = take(sizeof(double) * 6 * (size_t)n_seeds);
    const size_t o_wa = take(resident ? 0 : sizeof(double) * 3 * (size_t)n_wires);
    const size_t o_wb = take(resident ? 0 : sizeof(double) * 3 * (size_t)n_wires);
    const size_t o_fw = take(sizeof(int32_t) * (size_t)n_fired);
    const size_t o_ho = take(sizeof(int32_t) * ((size_t)n_fired + 1));
    const size_t o_rho = take(sizeof(double) * (size_t)n_hits);
    const size_t o_npts = take(sizeof(int32_t) * (size_t)n_seeds);
    const size_t o_rss = take(sizeof(double) * (size_t)n_seeds);
    const size_t o_bs = take(sizeof(int64_t) * (size_t)n_part);
    const size_t o_br = take(sizeof(double) * (size_t)n_part);
    const size_t o_bd = take(sizeof(double) * (size_t)n_part * (size_t)n_fired);
    const size_t o_cls = take((size_t)n_part * (size_t)n_hits);
    rc = grow(ctx, &ctx->hbuf, &ctx->hbuf_bytes, off);
    if (rc) return rc;
    char* B = (char*)ctx->hbuf;
    double* d_seeds = (double*)(B + o_seeds);
    double* d_wa = resident ? ctx->geom_a : (double*)(B + o_wa);
    double* d_wb = resident ? ctx->geom_b : (double*)(B + o_wb);
    int32_t* d_fw = (int32_t*)(B + o_fw);
    int32_t* d_ho = (int32_t*)(B + o_ho);
    double* d_rho = (double*)(B + o_rho);
    int32_t* d_npts = (int32_t*)(B + o_npts);
    double* d_rss = (double*)(B + o_rss);
    int64_t* d_bs = (int64_t*)(B + o_bs);
    double* d_br = (double*)(B + o_br);
    double* d_bd = (double*)(B + o_bd);
    uint8_t* d_cls = (uint8_t*)(B + o_cls);
    // ---- track_budget_bytes == 0: fused A+B, no track buffer; else slabs of seeds per A+B round ----
    const bool fused = track_budget_bytes == 0;
    const size_t per_chunk = comet_track_bytes(COMET_LANES, n_steps);
    int64_t slab_chunks = fused ? 0 : (int64_t)(track_budget_bytes / per_chunk);
    if (!fused) {
        if (slab_chunks < 1) slab_chunks = 1;
        const int64_t total_chunks = n_chunks_of(n_seeds);
        if (slab_chunks > total_chunks) slab_chunks = total_chunks;
        rc = grow(ctx, &ctx->tbuf, &ctx->tbuf_bytes, (size_t)slab_chunks * per_chunk);
        if (rc) return rc;
    }
    // ---- H2D ---------------------------------------------------------------------------------
    // (fused mode uploads the seeds per sub-slab inside scan_rss_impl, overlapped with the kernels)
    if (n_seeds && !fused) CU(ctx, cudaMemcpyAsync(d_seeds, seeds_host, sizeof(double) * 6 * (size_t)n_seeds, cudaMemcpyHostToDevice, st));
    if (n_fired) {
        if (!resident) {
            CU(ctx, cudaMemcpyAsync(d_wa, wire_a_host, sizeof(double) * 3 * (size_t)n_wires, cudaMemcpyHostToDevice, st));
            CU(ctx, cudaMemcpyAsync(d_wb, wire_b_host, sizeof(double) * 3 * (size_t)n_wires, cudaMemcpyHostToDevice, st));
        }
        CU(ctx, cudaMemcpyAsync(d_fw, fired_wire_host, sizeof(int32_t) * (size_t)n_fired, cudaMemcpyHostToDevice, st));
        CU(ctx, cudaMemcpyAsync(d_ho, hit_off_host, sizeof(int32_t) * ((size_t)n_fired + 1), cudaMemcpyHostToDevice, st));
    }
    if (n_hits) CU(ctx, cudaMemcpyAsync(d_rho, rho_host, sizeof(double) * (size_t)n_hits, cudaMemcpyHostToDevice, st));
    // ---- A + B per slab, then C --------------------------------------------------------------
    if (fused && n_seeds > 0) {
        rc = scan_rss_impl(ctx, d_seeds, seeds_host, d_seeds, n_seeds, n_seeds, 0, charge, bz_tesla, step_cm, n_steps, r_stop_cm,
                           d_wa, d_wb, n_wires, d_fw, d_ho, d_rho, n_fired, n_hits, cutoff_cm, d_rss, d_npts, st);
        if (rc) return rc;
    }
    const int64_t slab_seeds = slab_chunks * COMET_LANES;
    for (int64_t s0 = 0; !fused && s0 < n_seeds; s0 += slab_seeds) {
        const int64_t ns = (n_seeds - s0 < slab_seeds) ? (n_seeds - s0) : slab_seeds;
        rc = comet_seed_extrapolate(ctx, d_seeds + s0, n_seeds, ns, charge, bz_tesla, step_cm, n_steps, r_stop_cm,
                                    ctx->tbuf, d_npts + s0, st);
        if (rc) return rc;
        rc = comet_dca_rss(ctx, ctx->tbuf, d_npts + s0, ns, n_steps, charge, bz_tesla, step_cm, d_seeds + s0, n_seeds,
                           d_wa, d_wb, n_wires, d_fw, d_ho, d_rho, n_fired, n_hits, cutoff_cm, d_rss + s0, nullptr,
                           nullptr, st);
        if (rc) return rc;
    }
    rc = comet_select_and_classify(ctx, d_seeds, n_seeds, n_seeds, charge, bz_tesla, step_cm, n_steps, r_stop_cm,
                                   d_wa, d_wb, n_wires, d_fw, d_ho, d_rho, n_fired, n_hits, cutoff_cm, d_rss,
                                   part_off_host, n_part, d_bs, d_br, d_bd, d_cls, st);
    if (rc) return rc;
    // ---- D2H ---------------------------------------------------------------------------------
    if (n_part) {
        CU(ctx, cudaMemcpyAsync(best_seed_host, d_bs, sizeof(int64_t) * (size_t)n_part, cudaMemcpyDeviceToHost, st));
        CU(ctx, cudaMemcpyAsync(best_rss_host, d_br, sizeof(double) * (size_t)n_part, cudaMemcpyDeviceToHost, st));
        if (n_fired) CU(ctx, cudaMemcpyAsync(best_dca_host, d_bd, sizeof(double) * (size_t)n_part * n_fired, cudaMemcpyDeviceToHost, st));
        if (n_hits) CU(ctx, cudaMemcpyAsync(cls_host, d_cls, (size_t)n_part * n_hits, cudaMemcpyDeviceToHost, st));
    }
    if (rss_host && n_seeds) CU(ctx, cudaMemcpyAsync(rss_host, d_rss, sizeof(double) * (size_t)n_seeds, cudaMemcpyDeviceToHost, st));
    CU(ctx, cudaStreamSynchronize(st));
    return COMET_OK;
}

// The event of comet_scan_event_host with the seed sets given as grid axes: a few KB cross the bus per event.
extern "C" int comet_scan_event_grid_submit(comet_ctx* ctx, int32_t slot, const double* axes_host, int32_t n_part, int32_t n_p,
                                            int32_t n_ct, int32_t n_phi, int32_t n_z,
                                            int32_t charge, double bz_tesla, double step_cm, int32_t n_steps,
                                            double r_stop_cm,
                                            const int32_t* fired_wire_host, const int32_t* hit_off_host,
                                            const double* rho_host, int32_t n_fired, int32_t n_hits, double cutoff_cm,
                                            void* cuda_stream)
{
    GridShape g;
    if (!ctx || slot < 0 || slot >= COMET_EVENT_SLOTS || make_shape(&g, n_part, n_p, n_ct, n_phi, n_z) || !axes_host ||
        ctx->geom_n <= 0 || bad_physics(charge, bz_tesla, step_cm, n_steps) || !(r_stop_cm >= 0.0) ||
        bad_hits(ctx->geom_a, ctx->geom_b, ctx->geom_n, fired_wire_host, hit_off_host, rho_host, n_fired, n_hits, cutoff_cm))
        return COMET_EINVAL;
    comet_ctx::EventSlot& q = ctx->slot[slot];
    if (q.pending) return COMET_EINVAL;                      // (collect the event that is in the slot first)
    int rc = set_device(ctx);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int64_t n_seeds = g.G * n_part;
    const int64_t stride = (n_seeds + 31) / 32 * 32;
    // one device slab: [inputs: axes | fired | hit_off | rho] [seeds] [rss] [outputs: best_seed | best_rss | best_dca | cls];
    // the inputs and the outputs each cross the bus as ONE copy through a pinned staging buffer of the same layout
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
    const size_t o_axes = take(sizeof(double) * (size_t)g.A * n_part);
    const size_t o_fw = take(sizeof(int32_t) * (size_t)n_fired);
    const size_t o_ho = take(sizeof(int32_t) * ((size_t)n_fired + 1));
    const size_t o_rho = take(sizeof(double) * (size_t)n_hits);
    const size_t in_bytes = off;
    const size_t o_seeds = take(sizeof(double) * 6 * (size_t)stride);
    const size_t o_rss = take(sizeof(double) * (size_t)n_seeds);
    const size_t o_out = off;
    const size_t o_bs = take(sizeof(int64_t) * (size_t)n_part);
    const size_t o_br = take(sizeof(double) * (size_t)n_part);
    const size_t o_bd = take(sizeof(double) * (size_t)n_part * (size_t)n_fired);
    const size_t o_cls = take((size_t)n_part * (size_t)n_hits);
    const size_t out_bytes = off - o_out;
    if (!q.done) CU(ctx, cudaEventCreateWithFlags(&q.done, cudaEventDisableTiming));
    if (off > q.dbuf_bytes) {
        CU(ctx, cudaDeviceSynchronize());
        rc = grow(ctx, &q.dbuf, &q.dbuf_bytes, off);
        if (rc) return rc;
    }
    if (in_bytes + out_bytes > q.hstage_bytes) {
        CU(ctx, cudaDeviceSynchronize());
        if (q.hstage) { cudaFreeHost(q.hstage); q.hstage = nullptr; q.hstage_bytes = 0; }
        cudaError_t e = cudaHostAlloc(&q.hstage, in_bytes + out_bytes, cudaHostAllocDefault);
        if (e != cudaSuccess) { ctx->last_cuda = (int)e; q.hstage = nullptr; cudaGetLastError(); return COMET_ENOMEM; }
        q.hstage_bytes = in_bytes + out_bytes;
    }
    char* B = (char*)q.dbuf;
    char* Hs = (char*)q.hstage;
    double* d_axes = (double*)(B + o_axes);
    double* d_seeds = (double*)(B + o_seeds);
    int32_t* d_fw = (int32_t*)(B + o_fw);
    int32_t* d_ho = (int32_t*)(B + o_ho);
    double* d_rho = (double*)(B + o_rho);
    double* d_rss = (double*)(B + o_rss);
    int64_t* d_bs = (int64_t*)(B + o_bs);
    double* d_br = (double*)(B + o_br);
    double* d_bd = (double*)(B + o_bd);
    uint8_t* d_cls = (uint8_t*)(B + o_cls);
    memcpy(Hs + o_axes, axes_host, sizeof(double) * (size_t)g.A * n_part);
    if (n_fired) {
        memcpy(Hs + o_fw, fired_wire_host, sizeof(int32_t) * (size_t)n_fired);
        memcpy(Hs + o_ho, hit_off_host, sizeof(int32_t) * ((size_t)n_fired + 1));
    }
    if (n_hits) memcpy(Hs + o_rho, rho_host, sizeof(double) * (size_t)n_hits);
    CU(ctx, cudaMemcpyAsync(B, Hs, in_bytes, cudaMemcpyHostToDevice, st));
    rc = comet_seed_grid(ctx, d_axes, n_part, n_p, n_ct, n_phi, n_z, d_seeds, stride, st);
    if (rc) return rc;
    // (a partition is a whole number of runs: G is a multiple of the run length)
    rc = scan_rss_impl(ctx, nullptr, nullptr, d_seeds, stride, n_seeds, comet_grid_z_run(n_z), charge, bz_tesla, step_cm,
                       n_steps, r_stop_cm, ctx->geom_a, ctx->geom_b, ctx->geom_n, d_fw, d_ho, d_rho, n_fired, n_hits,
                       cutoff_cm, d_rss, nullptr, st);
    if (rc) return rc;
    int64_t po[COMET_MAX_PARTITIONS + 1];
    for (int p = 0; p <= n_part; ++p) po[p] = (int64_t)p * g.G;
    rc = comet_select_and_classify(ctx, d_seeds, stride, n_seeds, charge, bz_tesla, step_cm, n_steps, r_stop_cm,
                                   ctx->geom_a, ctx->geom_b, ctx->geom_n, d_fw, d_ho, d_rho, n_fired, n_hits, cutoff_cm,
                                   d_rss, po, n_part, d_bs, d_br, d_bd, d_cls, st);
    if (rc) return rc;
    CU(ctx, cudaMemcpyAsync(Hs + in_bytes, B + o_out, out_bytes, cudaMemcpyDeviceToHost, st));
    CU(ctx, cudaEventRecord(q.done, st));
    q.in_bytes = in_bytes; q.o_out = o_out; q.out_bytes = out_bytes; q.o_bs = o_bs; q.o_br = o_br; q.o_bd = o_bd; q.o_cls = o_cls;
    q.o_rss = o_rss; q.n_part = n_part; q.n_fired = n_fired; q.n_hits = n_hits; q.n_seeds = n_seeds;
    q.pending = 1;
    return COMET_OK;
}

extern "C" int comet_scan_event_grid_collect(comet_ctx* ctx, int32_t slot, int64_t* best_seed_host, double* best_rss_host,
                                             double* best_dca_host, uint8_t* cls_host)
{
    if (!ctx || slot < 0 || slot >= COMET_EVENT_SLOTS) return COMET_EINVAL;
    comet_ctx::EventSlot& q = ctx->slot[slot];
    if (!q.pending || !best_seed_host || !best_rss_host || (q.n_fired > 0 && !best_dca_host) || (q.n_hits > 0 && !cls_host))
        return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    CU(ctx, cudaEventSynchronize(q.done));
    q.pending = 0;
    const char* Ho = (const char*)q.hstage + q.in_bytes;
    memcpy(best_seed_host, Ho + (q.o_bs - q.o_out), sizeof(int64_t) * (size_t)q.n_part);
    memcpy(best_rss_host, Ho + (q.o_br - q.o_out), sizeof(double) * (size_t)q.n_part);
    if (q.n_fired) memcpy(best_dca_host, Ho + (q.o_bd - q.o_out), sizeof(double) * (size_t)q.n_part * q.n_fired);
    if (q.n_hits) memcpy(cls_host, Ho + (q.o_cls - q.o_out), (size_t)q.n_part * q.n_hits);
    return COMET_OK;
}

extern "C" int comet_scan_event_grid_host(comet_ctx* ctx, const double* axes_host, int32_t n_part, int32_t n_p,
                                          int32_t n_ct, int32_t n_phi, int32_t n_z,
                                          int32_t charge, double bz_tesla, double step_cm, int32_t n_steps,
                                          double r_stop_cm,
                                          const int32_t* fired_wire_host, const int32_t* hit_off_host,
                                          const double* rho_host, int32_t n_fired, int32_t n_hits, double cutoff_cm,
                                          int64_t* best_seed_host, double* best_rss_host, double* best_dca_host,
                                          uint8_t* cls_host, double* rss_host, void* cuda_stream)
{
    if (!ctx || !best_seed_host || !best_rss_host || (n_fired > 0 && !best_dca_host) || (n_hits > 0 && !cls_host))
        return COMET_EINVAL;
    if (ctx->slot[0].pending) return COMET_EINVAL;           // (an event submitted to slot 0 is still to be collected)
    int rc = comet_scan_event_grid_submit(ctx, 0, axes_host, n_part, n_p, n_ct, n_phi, n_z, charge, bz_tesla, step_cm, n_steps,
                                          r_stop_cm, fired_wire_host, hit_off_host, rho_host, n_fired, n_hits, cutoff_cm, cuda_stream);
    if (rc) return rc;
    const comet_ctx::EventSlot& q = ctx->slot[0];
    if (rss_host)
        CU(ctx, cudaMemcpyAsync(rss_host, (const char*)q.dbuf + q.o_rss, sizeof(double) * (size_t)q.n_seeds, cudaMemcpyDeviceToHost,
                                (cudaStream_t)cuda_stream));
    rc = comet_scan_event_grid_collect(ctx, 0, best_seed_host, best_rss_host, best_dca_host, cls_host);
    if (rc) return rc;
    if (rss_host) CU(ctx, cudaStreamSynchronize((cudaStream_t)cuda_stream));
    return COMET_OK;
}

// ---------------------------------------------------------------------------------------------
// FP64 pipe peak probe
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_fp64_probe(int iters, double* sink)
{
    double a0 = threadIdx.x * 1e-9, a1 = a0 + 1.0, a2 = a0 + 2.0, a3 = a0 + 3.0;
    double a4 = a0 + 4.0, a5 = a0 + 5.0, a6 = a0 + 6.0, a7 = a0 + 7.0;
    const double m = 0.999999999, b = 1e-12;
#pragma unroll 1
    for (int i = 0; i < iters; i += 8) {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            a0 = fma(a0, m, b); a1 = fma(a1, m, b); a2 = fma(a2, m, b); a3 = fma(a3, m, b);
            a4 = fma(a4, m, b); a5 = fma(a5, m, b); a6 = fma(a6, m, b); a7 = fma(a7, m, b);
        }
    }
    const double r = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (r == 123.456) sink[0] = r;          // never true: keeps the chains alive
}

extern "C" int comet_fp64_peak_probe(comet_ctx* ctx, int32_t iters, double* sink_dev, double* n_fma, void* cuda_stream)
{
    if (!ctx || iters < 8 || !sink_dev) return COMET_EINVAL;
    int rc = set_device(ctx);
    if (rc) return rc;
    iters = (iters + 7) / 8 * 8;
    const int blocks = ctx->n_sm * 8, threads = 256;
    k_fp64_probe<<<blocks, threads, 0, (cudaStream_t)cuda_stream>>>(iters, sink_dev);
    CU(ctx, cudaGetLastError());
    if (n_fma) *n_fma = (double)blocks * threads * (double)iters * 8.0;
    return COMET_OK;
}

// ---------------------------------------------------------------------------------------------
// comet_argmin_static: the per-partition argmin of step C (reading R15) for callers that
// cannot allocate -- no ctx, no cudaMalloc: the partial minima live in a file-scope device array
// ---------------------------------------------------------------------------------------------
// Scratch of the two-stage argmin: [COMET_STATIC_MAX_PART][COMET_ARGMIN_SPLIT] partial values (doubles), then as many
// partial indices (int64): 64 KB.  Every GPU that loads the library holds it until the process exits.  In HOST code the
// name below is only a stand-in for the symbol, not a device address: host code takes the address from
// cudaGetSymbolAddress (static_scratch_ptr), device code names the array directly.
#define COMET_STATIC_SLOTS (COMET_STATIC_MAX_PART * COMET_ARGMIN_SPLIT)
#define COMET_STATIC_BYTES (COMET_STATIC_SLOTS * (sizeof(double) + sizeof(int64_t)))
#define COMET_STATIC_MAX_DEVICES 64
static __device__ __align__(256) unsigned char g_static_scratch[COMET_STATIC_BYTES];

// second stage: one warp per partition merges the partition's COMET_ARGMIN_SPLIT partial minima (lower value wins,
// equal values -> lower index: R15) -- read from the array by its name -- and writes the winner as k_select_classify does
__global__ void __launch_bounds__(32) k_argmin_static_finish(int64_t* __restrict__ best_seed, double* __restrict__ best_rss)
{
    const double* pv = reinterpret_cast<const double*>(g_static_scratch);
    const int64_t* pi = reinterpret_cast<const int64_t*>(g_static_scratch + COMET_STATIC_SLOTS * sizeof(double));
    const int p = blockIdx.x, lane = threadIdx.x;
    double v = 0.0;
    int64_t idx = -1;
    for (int b = lane; b < COMET_ARGMIN_SPLIT; b += 32) argmin_merge(v, idx, pv[p * COMET_ARGMIN_SPLIT + b], pi[p * COMET_ARGMIN_SPLIT + b]);
    for (int o = 16; o > 0; o >>= 1) {
        const double v2 = __shfl_down_sync(0xffffffffu, v, o);
        const int64_t i2 = __shfl_down_sync(0xffffffffu, idx, o);
        argmin_merge(v, idx, v2, i2);
    }
    if (lane == 0) {
        best_seed[p] = idx;
        best_rss[p] = (idx >= 0 && v != -INFINITY) ? v : __longlong_as_double(0x7ff8000000000000LL);
    }
}

// device address of g_static_scratch on the CURRENT device: resolved once per device, with that device current
static std::mutex g_static_mu;
static void* g_static_ptr[COMET_STATIC_MAX_DEVICES];
static int static_scratch_ptr(void** out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return COMET_ECUDA; }
    if (dev < 0 || dev >= COMET_STATIC_MAX_DEVICES) return COMET_EINVAL;
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[dev]) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_static_scratch) != cudaSuccess || !p) { cudaGetLastError(); return COMET_ECUDA; }
        g_static_ptr[dev] = p;
    }
    *out = g_static_ptr[dev];
    return COMET_OK;
}

extern "C" int comet_argmin_static(const double* rss, int64_t n_seeds, const int64_t* part_off, int32_t n_part,
                                   int64_t* best_seed, double* best_rss, void* cuda_stream)
{
    if (n_seeds < 0 || n_part < 0) return COMET_EINVAL;
    if (n_part > COMET_STATIC_MAX_PART) return COMET_ELIMIT;
    if (n_part == 0) return COMET_OK;
    if (!part_off || !best_seed || !best_rss) return COMET_EINVAL;
    PartOff po;
    if (fill_partoff(&po, part_off, n_part, n_seeds, false)) return COMET_EINVAL;
    if (po.off[n_part] > 0 && !rss) return COMET_EINVAL;
    void* scratch = nullptr;
    int rc = static_scratch_ptr(&scratch);
    if (rc) return rc;
    double* pv = reinterpret_cast<double*>(scratch);
    int64_t* pi = reinterpret_cast<int64_t*>(reinterpret_cast<unsigned char*>(scratch) + COMET_STATIC_SLOTS * sizeof(double));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // every slot the second stage reads is written by the first stage of the same call (an empty slice writes "none"):
    // nothing of an earlier call survives, nothing has to start at zero
    k_argmin_stage1<<<dim3(COMET_ARGMIN_SPLIT, n_part), COMET_ARGMIN_THREADS, 0, st>>>(rss, po, pv, pi);
    k_argmin_static_finish<<<n_part, 32, 0, st>>>(best_seed, best_rss);
    if (cudaGetLastError() != cudaSuccess) return COMET_ECUDA;
    return COMET_OK;
}
