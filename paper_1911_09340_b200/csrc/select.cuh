// select.cuh -- step C: per-partition argmin of RSS (reading R15) and hit
// classification for the winning seed (reading R13), sm_100a.
#pragma once
#include "common.cuh"

namespace comet {

struct PartOff {
    int64_t off[65];            // COMET_MAX_PARTITIONS + 1
};

#define COMET_ARGMIN_SPLIT 64   // CTAs per partition in the first argmin stage
#define COMET_ARGMIN_THREADS 256
#define COMET_ARGMIN_FUSED 16384 // partitions up to this size skip the first stage: the CTA of k_select_classify scans them
#define COMET_SEL_CK 4           // = COMET_FUSED_CK (scan_fused.cuh; checked there): rows between the scan's checkpoints

// (value, index) ordering of R15: smaller rss wins, equal rss -> lower index.  NaN never wins
// against a number (the comparison is false), exactly as the serial scan "rss[s] < rss[b]".
__device__ __forceinline__ void argmin_merge(double& v, int64_t& i, double v2, int64_t i2)
{
    if (i2 >= 0 && (i < 0 || v2 < v || (v2 == v && i2 < i))) { v = v2; i = i2; }
}

// A serial scan "b = lo; for s > lo: if (rss[s] < rss[b]) b = s" keeps the first index whose value is strictly
// smaller than every earlier one.  With NaNs the comparison is false when either side is NaN: a NaN at the first
// position of the partition stays the winner whatever follows, a NaN anywhere else never wins.  Reproduced here by
// skipping NaNs at s > lo and giving a NaN at lo the value -infinity (RSS is a sum of squares: no number is that
// small); k_select_classify turns it back into the NaN it stands for.
// one thread's share [first, first + step, ...) of [.., hi) of the partition that starts at lo, then the warp's minimum
__device__ __forceinline__ void partition_argmin(const double* __restrict__ rss, int64_t lo, int64_t first, int64_t hi,
                                                 int64_t step, double& v, int64_t& idx)
{
    v = 0.0;
    idx = -1;
    // batches of 8 loads in flight (one CTA may scan a whole partition: a load per iteration would serialise the latencies)
    constexpr int NB = 8;
    for (int64_t s0 = first; s0 < hi; s0 += NB * step) {
        double rb[NB];
#pragma unroll
        for (int q = 0; q < NB; ++q) {
            const int64_t s = s0 + q * step;
            rb[q] = s < hi ? rss[s] : __longlong_as_double(0x7ff8000000000000LL);   // (past the end: a NaN, skipped below)
        }
#pragma unroll
        for (int q = 0; q < NB; ++q) {
            const int64_t s = s0 + q * step;
            double r = rb[q];
            if (r != r) {
                if (s != lo || s >= hi) continue;
                r = -INFINITY;
            }
            if (idx < 0 || r < v) { v = r; idx = s; }   // increasing s per thread: ties keep lower s
        }
    }
    for (int o = 16; o > 0; o >>= 1) {
        const double v2 = __shfl_down_sync(0xffffffffu, v, o);
        const int64_t i2 = __shfl_down_sync(0xffffffffu, idx, o);
        argmin_merge(v, idx, v2, i2);
    }
}

__global__ void __launch_bounds__(COMET_ARGMIN_THREADS)
k_argmin_stage1(const double* __restrict__ rss, PartOff po, double* __restrict__ pv, int64_t* __restrict__ pi)
{
    const int p = blockIdx.y;
    const int64_t lo = po.off[p], hi = po.off[p + 1];
    const int64_t n = hi - lo;
    const int64_t per = (n + gridDim.x - 1) / gridDim.x;
    const int64_t b = lo + per * blockIdx.x, e = min(hi, b + per);
    double v;
    int64_t idx;
    partition_argmin(rss, lo, b + threadIdx.x, e, blockDim.x, v, idx);
    __shared__ double sv[COMET_ARGMIN_THREADS / 32];
    __shared__ int64_t si[COMET_ARGMIN_THREADS / 32];
    if ((threadIdx.x & 31) == 0) { sv[threadIdx.x >> 5] = v; si[threadIdx.x >> 5] = idx; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < COMET_ARGMIN_THREADS / 32; ++w) argmin_merge(v, idx, sv[w], si[w]);
        pv[p * gridDim.x + blockIdx.x] = v;
        pi[p * gridDim.x + blockIdx.x] = idx;
    }
}

struct ClassifyArgs {
    const double* seeds;
    int64_t stride;
    double qkb;
    StepK hk;
    int32_t n_steps;
    double r_stop2;
    const double* wire_a;      // [3][n_wires] wire end points: the lines (O4) are formed here, no table of another kernel is read
    const double* wire_b;
    int32_t n_wires;
    const int32_t* fired_wire; // [W]
    int32_t W;
    const int32_t* hit_off;
    const double* rho;
    int32_t n_hits;
    double lambda;
    const double* pv;          // stage-1 partial minima [n_part][COMET_ARGMIN_SPLIT]
    const int64_t* pi;
    int64_t* best_seed;
    double* best_rss;
    double* best_dca;
    uint8_t* cls;
    FieldMap F;                // field-map variants: the map; qkb = kappa q, hk.h = h_max
    double h_min;
    // the distinct transverse tracks of the comet_scan_rss call that produced rss (scan_zgroup.cuh), when the ctx knows
    // they are still those of `seeds`: the winner's (x, y, T_x, T_y) rows are copied instead of stepped again
    const double* ub;          // [track][u_rows][4], nullptr = record the track here
    const int32_t* np_u;
    int32_t zshift, u_rows;
    // or (uniform field, plain scan kernels) that call's checkpoints: (x, T) of every COMET_SEL_CK-th recorded state of
    // every seed, [chunk][n_ck][6][32]; the states in between are stepped by one thread per checkpoint
    const double* ck;          // nullptr = no checkpoints
    int32_t n_ck;
    const double* rss;         // partitions of at most COMET_ARGMIN_FUSED seeds: k_select_classify takes the argmin itself
    PartOff po;
    const int32_t* dyn;        // comet_scan_turns: device {.., .., stop flag}: set = write nothing
};

// CTA-wide: re-extrapolate seed `idx` into shared memory (state k at sm[k*6..]), then one thread per fired
// wire does O5..O8 + O11 in exact arithmetic: dca[i] = signed D, cls[j] = 1 for the classified entries
// (all other entries 0).  idx < 0: NaN / zeros.
// With n_grp > 1 the CTA is one of n_grp that share a seed: each rebuilds the track for itself and takes the fired wires
// [grp W / n_grp, (grp + 1) W / n_grp) and their hit entries (the search over the states is the bulk of the work and one
// CTA uses one SM).
template <bool FIELD>
__device__ __forceinline__ void classify_cta(const ClassifyArgs& a, int64_t idx, double* __restrict__ dca,
                                             uint8_t* __restrict__ cls, double* sm, int grp = 0, int n_grp = 1)
{
    constexpr int RS = FIELD ? 7 : 6;                   // row: x, T and, in a field map, the step leaving the state
    __shared__ int32_t s_np;
    __shared__ double s_c;
    const int W = a.W;
    const int w0 = (int)((int64_t)W * grp / n_grp), w1 = (int)((int64_t)W * (grp + 1) / n_grp);
    {
        // the entries of the group's wires; the first and the last group also take what lies outside every wire's range
        const int j0 = (grp == 0 || W == 0) ? 0 : a.hit_off[w0], j1 = (grp == n_grp - 1 || W == 0) ? a.n_hits : a.hit_off[w1];
        for (int j = j0 + (int)threadIdx.x; j < j1; j += blockDim.x) cls[j] = 0;
    }
    if (idx < 0) {
        for (int i = w0 + (int)threadIdx.x; i < w1; i += blockDim.x) dca[i] = __longlong_as_double(0x7ff8000000000000LL);
        return;
    }
    // The scan's tracks are taken only if they ARE this seed's: state 0 of the track / checkpoint 0 must equal the seed's own
    // initial state bit for bit (the host has compared the physics; a track is a function of its initial state and those).  A
    // buffer that was rewritten, or reused by the allocator for another seed set, falls through to the chain below.
    bool rows_ok = false, ck_ok = false;
    if (!FIELD && (a.ub || a.ck)) {
        State s0;
        (void)seed_init(a.seeds, a.stride, idx, a.qkb, s0);
        if (a.ub) {
            const double2* g0 = reinterpret_cast<const double2*>(a.ub + (size_t)(idx >> a.zshift) * (size_t)a.u_rows * 4);
            const double2 xy = __ldg(g0), tt = __ldg(g0 + 1);
            rows_ok = xy.x == s0.x0 && xy.y == s0.x1 && tt.x == s0.t0 && tt.y == s0.t1;
        } else {
            const double* o = a.ck + (size_t)(idx >> 5) * (size_t)a.n_ck * (6 * COMET_LANES) + (idx & 31);
            ck_ok = o[0] == s0.x0 && o[32] == s0.x1 && o[64] == s0.x2 && o[96] == s0.t0 && o[128] == s0.t1 && o[160] == s0.t2;
        }
    }
    if (rows_ok) {
        // the same numbers without the chain of 400-odd dependent RKN4 steps: (x, y, T_x, T_y) of every recorded state are
        // the rows of the seed's distinct transverse track, z is one addition per step (x_2' = x_2 + h T_2)
        State st;
        const double c = seed_init(a.seeds, a.stride, idx, a.qkb, st);
        const int64_t u = idx >> a.zshift;
        const int32_t np = min(max(__ldg(a.np_u + u), 1), a.n_steps + 1);
        const double2* g = reinterpret_cast<const double2*>(a.ub + (size_t)u * (size_t)a.u_rows * 4);
        for (int k = threadIdx.x; k < np; k += blockDim.x) {
            const double2 xy = __ldg(g + 2 * k), tt = __ldg(g + 2 * k + 1);
            double* o = sm + (size_t)k * RS;
            o[0] = xy.x; o[1] = xy.y; o[3] = tt.x; o[4] = tt.y; o[5] = st.t2;
        }
        if (threadIdx.x == 0) {
            s_c = c;
            s_np = np;
            const double hz = xmul(a.hk.h, st.t2);
            double z = st.x2;
            sm[2] = z;
            for (int k = 1; k < np; ++k) { z = xadd(z, hz); sm[(size_t)k * RS + 2] = z; }
        }
    } else if (ck_ok) {
        // the same numbers without the chain: thread m starts from checkpoint m (recorded state m CK, bit for bit) and steps
        // the CK - 1 states after it.  The first state in the target region ends the track (R3); the checkpoints behind it
        // were never written and whatever those threads compute is not read (pure arithmetic: nothing is addressed by it).
        constexpr int CK = COMET_SEL_CK;
        State s0;
        const double c = seed_init(a.seeds, a.stride, idx, a.qkb, s0);
        if (threadIdx.x == 0) { s_c = c; s_np = a.n_steps + 1; }
        __syncthreads();
        const double* base = a.ck + (size_t)(idx >> 5) * (size_t)a.n_ck * (6 * COMET_LANES) + (idx & 31);
        const bool use_stop = a.r_stop2 > 0.0;
        for (int m = threadIdx.x; m * CK <= a.n_steps; m += blockDim.x) {
            const double* o = base + (size_t)m * (6 * COMET_LANES);
            State st;
            st.x0 = o[0]; st.x1 = o[32]; st.x2 = o[64]; st.t0 = o[96]; st.t1 = o[128]; st.t2 = o[160];
            int first = 1 << 30;
#pragma unroll
            for (int j = 0; j < CK; ++j) {
                const int k = m * CK + j;
                if (k > a.n_steps) break;
                if (j > 0) rkn4_step(st, a.hk, c);
                double* r = sm + (size_t)k * RS;
                r[0] = st.x0; r[1] = st.x1; r[2] = st.x2; r[3] = st.t0; r[4] = st.t1; r[5] = st.t2;
                if (use_stop && k > 0 && first > k && in_target_region(st, a.r_stop2)) first = k;
            }
            if (first < (1 << 30)) atomicMin(&s_np, first + 1);
        }
    } else
    if (threadIdx.x == 0) {
        State st;
        const double c = seed_init(a.seeds, a.stride, idx, a.qkb, st);
        s_c = c;
        int32_t np = a.n_steps + 1;
        sm[0] = st.x0; sm[1] = st.x1; sm[2] = st.x2; sm[3] = st.t0; sm[4] = st.t1; sm[5] = st.t2;
        double htry = a.hk.h;
        int32_t k = 1;
        if (!FIELD) {
            // one thread, one chain of dependent operations: blocks of four steps are recorded unconditionally (rows
            // past the stop are never read) and the stop test stays off the chain, as in k_gen_unique
            const bool use_stop = a.r_stop2 > 0.0;
            for (; k + 3 <= a.n_steps; k += 4) {
                int first = 4;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    rkn4_step(st, a.hk, c);
                    double* o = sm + (size_t)(k + j) * RS;
                    o[0] = st.x0; o[1] = st.x1; o[2] = st.x2; o[3] = st.t0; o[4] = st.t1; o[5] = st.t2;
                    const double r2 = xadd(xmul(st.x0, st.x0), xmul(st.x1, st.x1));
                    const double rad = xadd(xmul(st.x0, st.t0), xmul(st.x1, st.t1));
                    const bool stop = (r2 < a.r_stop2) & (rad < 0.0) & use_stop;
                    first = (stop & (first == 4)) ? j : first;
                }
                if (first < 4) { np = k + first + 1; break; }
            }
        }
        for (; np == a.n_steps + 1 && k <= a.n_steps; ++k) {
            if (FIELD) sm[(size_t)(k - 1) * RS + 6] = adaptive_field_step(st, htry, a.hk.h, a.h_min, c, a.F);
            else rkn4_step(st, a.hk, c);
            double* o = sm + (size_t)k * RS;
            o[0] = st.x0; o[1] = st.x1; o[2] = st.x2; o[3] = st.t0; o[4] = st.t1; o[5] = st.t2;
            if (a.r_stop2 > 0.0 && in_target_region(st, a.r_stop2)) { np = k + 1; break; }
        }
        s_np = np;
    }
    __syncthreads();                                    // also orders the cls zeroing before the marks below
    const int32_t np = s_np;
    const double c = s_c;
    // O5 for every wire: the recorded states are cut into NSEG segments per wire (NSEG threads per wire), the segment
    // minima are merged in increasing row order with a strict <, i.e. the lowest row wins ties as in the serial scan
    __shared__ double s_bd[256];
    __shared__ int s_ks[256];
    const int nthr = blockDim.x;
    const int Wp = min(w1 - w0, nthr);
    const int NSEG = Wp > 0 ? nthr / Wp : 1;
    for (int i0 = w0; i0 < w1; i0 += Wp) {
        const int wi = i0 + (int)threadIdx.x % Wp, seg = (int)threadIdx.x / Wp;
        const bool on = wi < w1 && seg < NSEG;
        WireLine wl;
        int ks = 0;
        double bd = 0.0;
        if (on) {
            wl = wire_line_of(a.wire_a, a.wire_b, a.n_wires, a.fired_wire[wi]);
            const int len = (np + NSEG - 1) / NSEG;
            const int kb = seg * len, ke = min(np, kb + len);
            ks = -1;
            for (int k = kb; k < ke; ++k) {
                double u0, u1, u2;
                const double d2 = perp2_exact(sm[k * RS], sm[k * RS + 1], sm[k * RS + 2], wl, u0, u1, u2);
                if (ks < 0 || d2 < bd) { bd = d2; ks = k; }
            }
        }
        __syncthreads();
        s_bd[threadIdx.x] = bd;
        s_ks[threadIdx.x] = on ? ks : -1;
        __syncthreads();
        const int i = wi;
        if (!(on && seg == 0)) continue;
        for (int g2 = 1; g2 < NSEG; ++g2) {
            const int k2 = s_ks[g2 * Wp + (int)threadIdx.x];
            const double d2 = s_bd[g2 * Wp + (int)threadIdx.x];
            if (k2 >= 0 && (ks < 0 || d2 < bd)) { bd = d2; ks = k2; }
        }
        State st;
        st.x0 = sm[ks * RS]; st.x1 = sm[ks * RS + 1]; st.x2 = sm[ks * RS + 2];
        st.t0 = sm[ks * RS + 3]; st.t1 = sm[ks * RS + 4]; st.t2 = sm[ks * RS + 5];
        double D;
        if (FIELD) {
            const double lo = (ks > 0) ? -sm[(ks - 1) * RS + 6] : 0.0, hi = (ks < np - 1) ? sm[ks * RS + 6] : 0.0;
            D = fine_dca_field(st, lo, hi, c, a.F, wl);
        } else {
            D = fine_dca(st, ks, np, a.hk.h, c, wl);
        }
        dca[i] = D;
        int js;
        double rmin;
        (void)wire_residual(D, a.rho, a.hit_off[i], a.hit_off[i + 1], a.lambda, &js, &rmin);
        if (js >= 0 && rmin < a.lambda) cls[js] = 1;
    }
}

// gridDim.y CTAs per partition: each finishes the argmin, then classifies the winning seed on its share of the wires.
template <bool FIELD>
__global__ void __launch_bounds__(256) k_select_classify(const ClassifyArgs a)
{
    extern __shared__ __align__(16) double sm[];       // [(n_steps+1)][6]
    __shared__ int64_t s_best;
    const int p = blockIdx.x;
    const bool first_grp = blockIdx.y == 0;             // (every group finds the same winner; the first one writes it)
    if (a.rss) {
        // a small partition: the whole argmin here (same rule as k_argmin_stage1)
        __shared__ double sv[8];
        __shared__ int64_t si[8];
        double v = 0.0;
        int64_t idx = -1;
        partition_argmin(a.rss, a.po.off[p], a.po.off[p] + threadIdx.x, a.po.off[p + 1], blockDim.x, v, idx);
        if ((threadIdx.x & 31) == 0) { sv[threadIdx.x >> 5] = v; si[threadIdx.x >> 5] = idx; }
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int w = 1; w < (int)blockDim.x / 32; ++w) argmin_merge(v, idx, sv[w], si[w]);
            s_best = idx;
            if (first_grp) {
                a.best_seed[p] = idx;
                a.best_rss[p] = (idx >= 0 && v != -INFINITY) ? v : __longlong_as_double(0x7ff8000000000000LL);
            }
        }
    } else if (threadIdx.x == 0) {
        double v = 0.0;
        int64_t idx = -1;
        for (int b = 0; b < COMET_ARGMIN_SPLIT; ++b)
            argmin_merge(v, idx, a.pv[p * COMET_ARGMIN_SPLIT + b], a.pi[p * COMET_ARGMIN_SPLIT + b]);
        s_best = idx;
        if (first_grp) {
            a.best_seed[p] = idx;
            a.best_rss[p] = (idx >= 0 && v != -INFINITY) ? v : __longlong_as_double(0x7ff8000000000000LL);
        }
    }
    __syncthreads();
    classify_cta<FIELD>(a, s_best, a.best_dca + (size_t)p * a.W, a.cls + (size_t)p * a.n_hits, sm, (int)blockIdx.y, (int)gridDim.y);
}

}  // namespace comet
