// refine.cuh -- iterative seed refinement (readings R24-R28 of DESIGN.md), sm_100a.
//
//   k_select_refs     per turn partition, up to k sparse reference points: repeatedly the seed of lowest RSS
//                     (ties -> lowest index, NaN never) that is not selected yet and whose refinement box
//                     ref_d +- hw_d overlaps no selected box (|delta_d| < 2 hw_d in every dimension, strict);
//   k_refine_seeds    the finer seed set around every reference point, linear in (z, p_x, p_y, p_z);
//   k_classify_seeds  hit classification for a list of seeds (select.cuh's classify_cta).
//
// Everything stays on the device between the iterations of a stage (the paper copies seeds, tracks and RSS
// across the PCIe bus four times per iteration).  Each comparison and each grid
// value is one IEEE operation per operation of the definition, so references and seeds do not depend
// on the kernel variant or on compiler flags.
#pragma once
#include <cooperative_groups.h>
#include "common.cuh"
#include "select.cuh"

namespace comet {

#define COMET_REF_THREADS 1024
// COMET_MAX_REFS (comet.h): limit of k_ref and k_final

struct RefBox {
    double two_hw[4];           // 2 * half width of dimension d (seed component 2 + d)
};

// One CTA per partition.  Round r: every thread walks its seeds in increasing index and keeps the first one
// of strictly lowest RSS that is not blocked by the r references selected so far (the overlap test runs
// only for a seed that would become the thread's candidate); the CTA merges the candidates (ties -> lower
// index) and appends the winner.
__global__ void __launch_bounds__(COMET_REF_THREADS)
k_select_refs(const double* __restrict__ seeds, int64_t stride, const double* __restrict__ rss, PartOff po,
              RefBox box, int32_t k_ref, int64_t* __restrict__ ref_seed)
{
    __shared__ int64_t sel_idx[COMET_MAX_REFS];
    __shared__ double sel_c[COMET_MAX_REFS][4];
    __shared__ double sv[COMET_REF_THREADS / 32];
    __shared__ int64_t si[COMET_REF_THREADS / 32];
    __shared__ int64_t s_win;
    const int p = blockIdx.x;
    const int64_t lo = po.off[p], hi = po.off[p + 1];
    int64_t* out = ref_seed + (size_t)p * k_ref;
    for (int r = threadIdx.x; r < k_ref; r += blockDim.x) out[r] = -1;
    // Partitions of at most PER seeds per thread (the refined seed sets of a stage): the RSS values stay in
    // registers and a seed that overlaps a selected box is retired for good, so a round is a register-only
    // argmin, the CTA merge, and one overlap test of the live seeds against the NEW reference only -- the same
    // greedy rule (increasing (RSS, index), skip what is selected or overlaps a selected box), a quarter of the time.
    constexpr int PER = 8;
    if (hi - lo <= (int64_t)PER * COMET_REF_THREADS) {
        double rv[PER];
        unsigned dead = 0u;
#pragma unroll
        for (int j = 0; j < PER; ++j) {
            const int64_t sj = lo + threadIdx.x + (int64_t)j * COMET_REF_THREADS;
            rv[j] = sj < hi ? rss[sj] : 0.0;
            if (!(sj < hi) || rv[j] != rv[j]) dead |= 1u << j;       // out of range or NaN: never selected
        }
        for (int r = 0; r < k_ref; ++r) {
            double v = 0.0;
            int64_t idx = -1;
#pragma unroll
            for (int j = 0; j < PER; ++j)
                if (!((dead >> j) & 1u) && (idx < 0 || rv[j] < v)) { v = rv[j]; idx = lo + threadIdx.x + (int64_t)j * COMET_REF_THREADS; }
            for (int o = 16; o > 0; o >>= 1) {
                const double v2 = __shfl_down_sync(0xffffffffu, v, o);
                const int64_t i2 = __shfl_down_sync(0xffffffffu, idx, o);
                argmin_merge(v, idx, v2, i2);
            }
            if ((threadIdx.x & 31) == 0) { sv[threadIdx.x >> 5] = v; si[threadIdx.x >> 5] = idx; }
            __syncthreads();
            if (threadIdx.x < 32) {
                v = sv[threadIdx.x];
                idx = si[threadIdx.x];
                for (int o = 16; o > 0; o >>= 1) {
                    const double v2 = __shfl_down_sync(0xffffffffu, v, o);
                    const int64_t i2 = __shfl_down_sync(0xffffffffu, idx, o);
                    argmin_merge(v, idx, v2, i2);
                }
                if (threadIdx.x == 0) {
                    s_win = idx;
                    if (idx >= 0) {
                        sel_idx[r] = idx;
                        for (int d = 0; d < 4; ++d) sel_c[r][d] = seeds[(size_t)(2 + d) * stride + idx];
                        out[r] = idx;
                    }
                }
            }
            __syncthreads();
            const int64_t win = s_win;
            if (win < 0) break;
            if (r + 1 == k_ref) break;
#pragma unroll
            for (int j = 0; j < PER; ++j) {
                if ((dead >> j) & 1u) continue;
                const int64_t sj = lo + threadIdx.x + (int64_t)j * COMET_REF_THREADS;
                const bool ov = fabs(xsub(seeds[2 * stride + sj], sel_c[r][0])) < box.two_hw[0] &&
                                fabs(xsub(seeds[3 * stride + sj], sel_c[r][1])) < box.two_hw[1] &&
                                fabs(xsub(seeds[4 * stride + sj], sel_c[r][2])) < box.two_hw[2] &&
                                fabs(xsub(seeds[5 * stride + sj], sel_c[r][3])) < box.two_hw[3];
                if (ov || sj == win) dead |= 1u << j;
            }
        }
        return;
    }
    for (int r = 0; r < k_ref; ++r) {
        double v = 0.0;
        int64_t idx = -1;
        for (int64_t s = lo + threadIdx.x; s < hi; s += blockDim.x) {
            const double rs = rss[s];
            if (rs != rs) continue;
            if (idx >= 0 && !(rs < v)) continue;
            bool blocked = false;
            if (r > 0) {
                const double c0 = seeds[2 * stride + s], c1 = seeds[3 * stride + s];
                const double c2 = seeds[4 * stride + s], c3 = seeds[5 * stride + s];
                for (int q = 0; q < r && !blocked; ++q) {
                    const bool ov = fabs(xsub(c0, sel_c[q][0])) < box.two_hw[0] && fabs(xsub(c1, sel_c[q][1])) < box.two_hw[1] &&
                                    fabs(xsub(c2, sel_c[q][2])) < box.two_hw[2] && fabs(xsub(c3, sel_c[q][3])) < box.two_hw[3];
                    blocked = ov || sel_idx[q] == s;
                }
            }
            if (!blocked) { v = rs; idx = s; }
        }
        for (int o = 16; o > 0; o >>= 1) {
            const double v2 = __shfl_down_sync(0xffffffffu, v, o);
            const int64_t i2 = __shfl_down_sync(0xffffffffu, idx, o);
            argmin_merge(v, idx, v2, i2);
        }
        if ((threadIdx.x & 31) == 0) { sv[threadIdx.x >> 5] = v; si[threadIdx.x >> 5] = idx; }
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int w = 1; w < COMET_REF_THREADS / 32; ++w) argmin_merge(v, idx, sv[w], si[w]);
            s_win = idx;
            if (idx >= 0) {
                sel_idx[r] = idx;
                for (int d = 0; d < 4; ++d) sel_c[r][d] = seeds[(size_t)(2 + d) * stride + idx];
                out[r] = idx;
            }
        }
        __syncthreads();
        if (s_win < 0) break;
    }
}

// Large partitions (the first iteration of a stage: 131072 seeds per partition): the greedy rule visits the seeds in
// increasing (RSS, index), so only the seeds of lowest RSS matter -- as long as enough of them exist.  One CTA per partition:
//   1. a threshold key K* from a sample of 2048 seeds (the 16th smallest of their RSS high words, by a radix select in
//      shared memory): about 1024 seeds lie below it;
//   2. the candidates: EVERY seed whose key is below K* (they must fit the list of M = COMET_SHORT_M, else fallback),
//      compacted into shared memory;
//   3. the greedy rule on the candidates, register-resident as in k_select_refs.
// The candidates are exactly the seeds the rule visits first, so the references it finds among them are the references of
// the full rule.  If they run out before k_ref references are found (heavy overlaps, or a partition whose M smallest
// values are equal), fallback[p] = 1 and k_select_refs_cluster redoes the partition: the result never depends on M.
#define COMET_SHORT_M 2048
#define COMET_SHORT_RANK 16
__device__ __forceinline__ unsigned rss_key(double v)
{
    return (v != v) ? 0xffffffffu : (unsigned)__double2hiint(v);        // RSS >= 0: the high word orders like the value
}
__global__ void __launch_bounds__(COMET_REF_THREADS)
k_select_refs_short(const double* __restrict__ seeds, int64_t stride, const double* __restrict__ rss, PartOff po,
                    RefBox box, int32_t k_ref, int64_t* __restrict__ ref_seed, int* __restrict__ fallback)
{
    constexpr int M = COMET_SHORT_M, PER = M / COMET_REF_THREADS;
    __shared__ unsigned hist[257];
    __shared__ unsigned s_prefix, s_want, s_cnt;
    __shared__ int cand[M];
    __shared__ int64_t sel_idx[COMET_MAX_REFS];
    __shared__ double sel_c[COMET_MAX_REFS][4];
    __shared__ double sv[COMET_REF_THREADS / 32];
    __shared__ int64_t si[COMET_REF_THREADS / 32];
    __shared__ int64_t s_win;
    const int p = blockIdx.x;
    const int64_t lo = po.off[p], hi = po.off[p + 1];
    const int64_t n = hi - lo;
    int64_t* out = ref_seed + (size_t)p * k_ref;
    for (int r = threadIdx.x; r < k_ref; r += blockDim.x) out[r] = -1;
    if (threadIdx.x == 0) { s_prefix = 0u; s_want = (unsigned)M; s_cnt = 0u; fallback[p] = 0; }
    __syncthreads();
    unsigned kstar = 0xffffffffu;                           // n <= M: every seed with a number is a candidate
    if (n > M) {
        // threshold from a sample: 2 x 1024 seeds at a stride of n / 2048, the COMET_SHORT_RANK-th smallest of their keys by
        // a radix select in shared memory.  About COMET_SHORT_RANK n / 2048 seeds lie below it (1024 +- 256 for rank 16):
        // ANY threshold is correct as long as the list holds every seed below it, which is checked (cnt < M) below.
        const int64_t sstep = n / (2 * COMET_REF_THREADS);
        unsigned skey[2];
#pragma unroll
        for (int j = 0; j < 2; ++j) skey[j] = rss_key(rss[lo + (int64_t)(threadIdx.x + j * COMET_REF_THREADS) * sstep]);
        if (threadIdx.x == 0) s_want = COMET_SHORT_RANK;
        for (int shift = 24; shift >= 0; shift -= 8) {
            for (int b2 = threadIdx.x; b2 < 257; b2 += blockDim.x) hist[b2] = 0u;
            __syncthreads();
            const unsigned prefix = s_prefix;
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const bool in = shift == 24 || (skey[j] >> (shift + 8)) == (prefix >> (shift + 8));
                const unsigned digit = in ? ((skey[j] >> shift) & 255u) : 256u;
                const unsigned peers = __match_any_sync(0xffffffffu, digit);
                if (in && (int)(threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(&hist[digit], (unsigned)__popc(peers));
            }
            __syncthreads();
            if (threadIdx.x == 0) {
                unsigned want = s_want, cum = 0u;
                int d = 0;
                for (; d < 255; ++d) {
                    if (cum + hist[d] >= want) break;
                    cum += hist[d];
                }
                s_prefix = prefix | ((unsigned)d << shift);
                s_want = want - cum;
            }
            __syncthreads();
        }
        kstar = s_prefix;
    }
    for (int64_t s = lo + threadIdx.x; s < hi; s += blockDim.x) {
        if (rss_key(rss[s]) < kstar) {
            const unsigned pos = atomicAdd(&s_cnt, 1u);
            if (pos < (unsigned)M) cand[pos] = (int)(s - lo);
        }
    }
    __syncthreads();
    if (s_cnt >= (unsigned)M && n > M) {                    // (more seeds below the threshold than the list holds: the full rule)
        if (threadIdx.x == 0) fallback[p] = 1;
        return;
    }
    const int cnt = (int)min(s_cnt, (unsigned)M);
    // the greedy rule on the candidates (k_select_refs, register-resident branch)
    double rv[PER], cc[PER][4];                             // RSS and the refined components of the thread's candidates
    int64_t sj[PER];
    unsigned dead = 0u;
#pragma unroll
    for (int j = 0; j < PER; ++j) {
        const int q = threadIdx.x + j * COMET_REF_THREADS;
        sj[j] = q < cnt ? lo + cand[q] : -1;
        rv[j] = q < cnt ? rss[sj[j]] : 0.0;
        if (!(q < cnt) || rv[j] != rv[j]) dead |= 1u << j;
#pragma unroll
        for (int d = 0; d < 4; ++d) cc[j][d] = q < cnt ? seeds[(size_t)(2 + d) * stride + sj[j]] : 0.0;
    }
    int found = 0;
    for (int r = 0; r < k_ref; ++r) {
        double v = 0.0;
        int64_t idx = -1;
#pragma unroll
        for (int j = 0; j < PER; ++j)
            if (!((dead >> j) & 1u)) argmin_merge(v, idx, rv[j], sj[j]);
        for (int o = 16; o > 0; o >>= 1) {
            const double v2 = __shfl_down_sync(0xffffffffu, v, o);
            const int64_t i2 = __shfl_down_sync(0xffffffffu, idx, o);
            argmin_merge(v, idx, v2, i2);
        }
        if ((threadIdx.x & 31) == 0) { sv[threadIdx.x >> 5] = v; si[threadIdx.x >> 5] = idx; }
        __syncthreads();
        if (threadIdx.x < 32) {
            v = sv[threadIdx.x];
            idx = si[threadIdx.x];
            for (int o = 16; o > 0; o >>= 1) {
                const double v2 = __shfl_down_sync(0xffffffffu, v, o);
                const int64_t i2 = __shfl_down_sync(0xffffffffu, idx, o);
                argmin_merge(v, idx, v2, i2);
            }
            if (threadIdx.x == 0) {
                s_win = idx;
                if (idx >= 0) {
                    sel_idx[r] = idx;
                    for (int d = 0; d < 4; ++d) sel_c[r][d] = seeds[(size_t)(2 + d) * stride + idx];
                    out[r] = idx;
                }
            }
        }
        __syncthreads();
        const int64_t win = s_win;
        if (win < 0) break;
        found = r + 1;
        if (r + 1 == k_ref) break;
#pragma unroll
        for (int j = 0; j < PER; ++j) {
            if ((dead >> j) & 1u) continue;
            const bool ov = fabs(xsub(cc[j][0], sel_c[r][0])) < box.two_hw[0] && fabs(xsub(cc[j][1], sel_c[r][1])) < box.two_hw[1] &&
                            fabs(xsub(cc[j][2], sel_c[r][2])) < box.two_hw[2] && fabs(xsub(cc[j][3], sel_c[r][3])) < box.two_hw[3];
            if (ov || sj[j] == win) dead |= 1u << j;
        }
    }
    // the candidates ran out while other seeds exist: the full rule decides
    if (threadIdx.x == 0 && found < k_ref && n > M) fallback[p] = 1;
}

// The same selection by a thread-block cluster of COMET_REF_CLUSTER CTAs per partition: every CTA owns a
// slice of the partition (its RSS values staged once in shared memory when they fit), each round the CTAs
// publish their candidates in their own shared memory, synchronise the cluster, and every CTA merges the
// COMET_REF_CLUSTER candidates through distributed shared memory in rank order -- the same (value, index)
// ordering, hence the same references as k_select_refs, in a fraction of the time for large partitions.
#define COMET_REF_CLUSTER 8
#define COMET_REF_SMEM_MAX 25600        // RSS values a CTA stages in shared memory (200 KB)

template <bool SMEM>
__global__ void __cluster_dims__(COMET_REF_CLUSTER, 1, 1) __launch_bounds__(COMET_REF_THREADS)
k_select_refs_cluster(const double* __restrict__ seeds, int64_t stride, const double* __restrict__ rss, PartOff po,
                      RefBox box, int32_t k_ref, int64_t* __restrict__ ref_seed, const int* __restrict__ only_if = nullptr)
{
    if (only_if && !only_if[blockIdx.y]) return;            // (k_select_refs_short has served this partition)
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    extern __shared__ __align__(16) double srss[];
    __shared__ int64_t sel_idx[COMET_MAX_REFS];
    __shared__ double sel_c[COMET_MAX_REFS][4];
    __shared__ double sv[COMET_REF_THREADS / 32];
    __shared__ int64_t si[COMET_REF_THREADS / 32];
    __shared__ double slot_v;
    __shared__ int64_t slot_i;
    __shared__ int64_t s_win;
    const int p = blockIdx.y;
    const unsigned rank = cluster.block_rank();
    const int64_t lo = po.off[p], hi = po.off[p + 1];
    const int64_t per = (hi - lo + COMET_REF_CLUSTER - 1) / COMET_REF_CLUSTER;
    const int64_t b = min(hi, lo + per * (int64_t)rank), e = min(hi, b + per);
    int64_t* out = ref_seed + (size_t)p * k_ref;
    if (rank == 0)
        for (int r = threadIdx.x; r < k_ref; r += blockDim.x) out[r] = -1;
    if (SMEM)
        for (int64_t s = b + threadIdx.x; s < e; s += blockDim.x) srss[s - b] = rss[s];
    __syncthreads();
    for (int r = 0; r < k_ref; ++r) {
        double v = 0.0;
        int64_t idx = -1;
        for (int64_t s = b + threadIdx.x; s < e; s += blockDim.x) {
            const double rs = SMEM ? srss[s - b] : rss[s];
            if (rs != rs) continue;
            if (idx >= 0 && !(rs < v)) continue;
            bool blocked = false;
            if (r > 0) {
                const double c0 = seeds[2 * stride + s], c1 = seeds[3 * stride + s];
                const double c2 = seeds[4 * stride + s], c3 = seeds[5 * stride + s];
                for (int q = 0; q < r && !blocked; ++q) {
                    const bool ov = fabs(xsub(c0, sel_c[q][0])) < box.two_hw[0] && fabs(xsub(c1, sel_c[q][1])) < box.two_hw[1] &&
                                    fabs(xsub(c2, sel_c[q][2])) < box.two_hw[2] && fabs(xsub(c3, sel_c[q][3])) < box.two_hw[3];
                    blocked = ov || sel_idx[q] == s;
                }
            }
            if (!blocked) { v = rs; idx = s; }
        }
        for (int o = 16; o > 0; o >>= 1) {
            const double v2 = __shfl_down_sync(0xffffffffu, v, o);
            const int64_t i2 = __shfl_down_sync(0xffffffffu, idx, o);
            argmin_merge(v, idx, v2, i2);
        }
        if ((threadIdx.x & 31) == 0) { sv[threadIdx.x >> 5] = v; si[threadIdx.x >> 5] = idx; }
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int w = 1; w < COMET_REF_THREADS / 32; ++w) argmin_merge(v, idx, sv[w], si[w]);
            slot_v = v;
            slot_i = idx;
        }
        cluster.sync();                                  // every CTA's candidate is published
        if (threadIdx.x == 0) {
            double wv = 0.0;
            int64_t wi = -1;
            for (unsigned c = 0; c < COMET_REF_CLUSTER; ++c)
                argmin_merge(wv, wi, *cluster.map_shared_rank(&slot_v, c), *cluster.map_shared_rank(&slot_i, c));
            s_win = wi;
            if (wi >= 0) {
                sel_idx[r] = wi;
                for (int d = 0; d < 4; ++d) sel_c[r][d] = seeds[(size_t)(2 + d) * stride + wi];
                if (rank == 0) out[r] = wi;
            }
        }
        cluster.sync();                                  // slots are read; s_win and the new reference are visible
        if (s_win < 0) break;
    }
}

struct RefineGrid {
    double hw[4];
    double step[4];             // (2 hw) / (n - 1), 0 for n = 1
    int32_t n[4];
};

// One thread per new seed.  Slot (p, r) = blockIdx.y holds G seeds around reference ref_seed[p][r]; an
// empty slot repeats the partition's first reference (R27).
__global__ void __launch_bounds__(256)
k_refine_seeds(const double* __restrict__ seeds, int64_t stride, const int64_t* __restrict__ ref_seed,
               int32_t k_ref, RefineGrid g, int64_t G, double* __restrict__ out, int64_t out_stride)
{
    const int64_t slot = blockIdx.y;
    const int64_t gi = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gi >= G) return;
    int64_t ref = ref_seed[slot];
    if (ref < 0) ref = ref_seed[slot / k_ref * k_ref];
    if (ref < 0) return;                                  // empty partition: nothing to write
    const int64_t o = slot * G + gi;
    out[o] = seeds[ref];
    out[out_stride + o] = seeds[stride + ref];
    int64_t rem = gi;
#pragma unroll
    for (int d = 3; d >= 0; --d) {
        const int j = (int)(rem % g.n[d]);
        rem /= g.n[d];
        const double v = seeds[(size_t)(2 + d) * stride + ref];
        out[(size_t)(2 + d) * out_stride + o] = (g.n[d] > 1) ? xadd(xsub(v, g.hw[d]), xmul((double)j, g.step[d])) : v;
    }
}

// One CTA per listed seed: classification of PAPER.md:83 (classify_cta), the seed itself and its RSS.
template <bool FIELD>
__global__ void __launch_bounds__(256)
k_classify_seeds(const ClassifyArgs a, const int64_t* __restrict__ seed_idx, const double* __restrict__ rss,
                 double* __restrict__ dca, uint8_t* __restrict__ cls, double* __restrict__ seed_out,
                 double* __restrict__ rss_out)
{
    extern __shared__ __align__(16) double sm[];
    if (a.dyn && a.dyn[2]) return;                          // (the turn loop has stopped: the outputs keep their initial values)
    const int64_t idx = seed_idx[blockIdx.x];
    const double qnan = __longlong_as_double(0x7ff8000000000000LL);
    if (threadIdx.x < 6 && seed_out) seed_out[(size_t)blockIdx.x * 6 + threadIdx.x] = (idx >= 0) ? a.seeds[threadIdx.x * a.stride + idx] : qnan;
    if (threadIdx.x == 0 && rss_out) rss_out[blockIdx.x] = (idx >= 0 && rss) ? rss[idx] : qnan;
    classify_cta<FIELD>(a, idx, dca + (size_t)blockIdx.x * a.W, cls + (size_t)blockIdx.x * a.n_hits, sm);
}

}  // namespace comet
