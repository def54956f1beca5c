// scan_fused.cuh -- kernels A and B in one pass with the track kept on chip (sm_100a).
//
// The materialised path writes 48 bytes per recorded state to HBM (k_extrapolate runs at the HBM
// write rate) only for kernel B to read a small part of it back.  Here a warp owns one track chunk
// (32 consecutive seeds, lane = seed) from the seed to its (seed, wire) shortlist:
//
//   generate   TR RKN4 steps per lane (the definition's operations, common.cuh), the positions of the
//              TR rows go to a warp-private shared-memory tile [TR][3][32] fp64 (conflict-free, never
//              to HBM); every CK-th recorded state (x, T) is written to a small checkpoint buffer;
//   level 0    one sample per tile (row TR/2) against every fired wire.  This is the dense part, so
//              it runs with lane = WIRE: the wire's shortlist constants stay in registers for the
//              whole chunk, the 32 seeds' samples are broadcast from shared memory, and each lane
//              builds a 32-bit mask of the seeds whose tile may hold that wire's closest state
//              (Lipschitz bound of dca.cuh with the wire's far radius as the upper bound);
//   level 1    per wire with a non-empty mask (lane = seed again): the 8-row sub-block samples of
//              the tile, then row sweeps of the sub-blocks within reach, all from the tile; the best
//              (squared distance, row) of the pair so far lives in the pair workspace (L2-resident,
//              touched only by this warp);
//   finish     per wire: pairs whose closest state is farther than the far radius get e^2 = cutoff^2,
//              (chunk, wire) items with a near lane go to the work list of k_fine_ck.
//
// k_fine_ck takes the exact decision between bk-1, bk, bk+1 and runs the virtual-plane iteration
// from states it regenerates from the nearest checkpoint (at most CK-1+2 RKN steps), so every
// number that reaches a result is produced by the same operations as in the materialised path and
// by the definition: n_pts and RSS are bit-identical.
//
// RSS-only (the hot path).  Calls that ask for D or k* of every pair use the materialised path.
#pragma once
#include "common.cuh"
#include "dca.cuh"

namespace comet {

#ifndef COMET_FUSED_TR
#define COMET_FUSED_TR 32          // rows per tile (level-0 block)
#endif
#ifndef COMET_FUSED_CK
#define COMET_FUSED_CK 4           // rows between checkpoints
#endif
#ifndef COMET_FUSED_WARPS
#define COMET_FUSED_WARPS 1        // warps (chunks) per CTA
#endif
#define COMET_FUSED_QMAX 3         // wires per lane and round in level 0

struct FusedArgs {
    const double* seeds;
    int64_t stride;
    int64_t n_seeds;         // seeds of this slab
    double qkb;
    StepK hk;
    int32_t n_steps;
    double r_stop2;
    const double* wt;        // [15][W]
    int32_t W;
    const int32_t* hit_off;
    const double* rho;
    double lambda;
    int64_t SP;              // 32 * chunks of this slab: stride of bd / kb
    int32_t n_ck;            // checkpoint rows per chunk: n_steps / CK + 1
    double* ck;              // [chunks][n_ck][6][32]
    double* bd;              // [W][SP] best squared distance of the pair so far; e^2 afterwards
    int32_t* kb;             // [W][SP] its row, -1 = none / far
    int32_t* n_pts;          // [n_seeds]
    unsigned long long* items;
    unsigned int* n_items;
    unsigned long long* stats;
};

template <int Q>
__global__ void __launch_bounds__(32 * COMET_FUSED_WARPS) k_scan_fused(const FusedArgs a)
{
    constexpr int TR = COMET_FUSED_TR, CK = COMET_FUSED_CK, ROW = 3 * COMET_LANES;
    constexpr int NSUB = TR / COMET_M1;
    constexpr unsigned FULL = 0xffffffffu;
    constexpr int IMAX = 0x7fffffff;
    static_assert(TR % COMET_M1 == 0 && TR % CK == 0, "tile rows");
    extern __shared__ __align__(16) double fsm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* tile = fsm + warp * (TR * ROW);
    const int64_t chunk = (int64_t)blockIdx.x * COMET_FUSED_WARPS + warp;
    if (chunk * COMET_LANES >= a.n_seeds) return;
    const int64_t s = chunk * COMET_LANES + lane;
    const bool valid = s < a.n_seeds;
    const int W = a.W;
    const double h = a.hk.h;
    const double INF = 1.7976931348623157e308;
    const double L = COMET_LIP * h;
    const double half0 = (TR / 2) * L + COMET_SLACK, half1 = (COMET_M1 / 2) * L + COMET_SLACK;
    const double lam2 = xmul(a.lambda, a.lambda);

    State st;
    double c = 0.0;
    if (valid) {
        c = seed_init(a.seeds, a.stride, s, a.qkb, st);
    } else {
        st.x0 = st.x1 = st.x2 = 0.0;
        st.t0 = st.t1 = st.t2 = 0.0;
    }
    const bool lip_ok = fabs(c) * h <= COMET_CH_MAX;
    const unsigned nolip_mask = __ballot_sync(FULL, valid && !lip_ok);
    bool active = valid;
    int32_t np = valid ? a.n_steps + 1 : 0;
    const bool use_stop = a.r_stop2 > 0.0;

    // pair workspace of this chunk: nothing found yet
    for (int i = 0; i < W; ++i) {
        a.bd[(size_t)i * a.SP + s] = INF;
        a.kb[(size_t)i * a.SP + s] = -1;
    }

    // level-0 constants of this lane's wires (lane = wire): wire i = (r * Q + q) * 32 + lane
    const int n_rounds = (W + 32 * Q - 1) / (32 * Q);
    EvalC ec[Q];
    int thi[Q];
    auto load_round = [&](int r) {
#pragma unroll
        for (int q = 0; q < Q; ++q) {
            const int i = (r * Q + q) * 32 + lane;
            const int ii = min(i, W - 1);
            load_evalc(ec[q], a.wt, W, ii);
            const double cap = __ldg(a.wt + 14 * W + ii);
            const double t0 = cap + half0;
            thi[q] = (i < W && cap >= 0.0) ? __double2hiint(t0 * t0) : -1;
        }
    };
    if (n_rounds == 1) load_round(0);

    double* ckc = a.ck + (size_t)chunk * a.n_ck * (6 * COMET_LANES) + lane;
    const int n_tiles = (a.n_steps + TR) / TR;              // rows 0 .. n_steps
    for (int t = 0; t < n_tiles; ++t) {
        const int r0 = t * TR;
        // ---- generate rows r0 .. r0 + TR - 1 (Algorithm 1; finished lanes hold their last state) ------
#pragma unroll 2
        for (int rr = 0; rr < TR; ++rr) {
            const int k = r0 + rr;
            if (k > 0 && active) {
                rkn4_step(st, a.hk, c);
                if (use_stop && in_target_region(st, a.r_stop2)) { np = k + 1; active = false; }
            }
            if (k >= a.n_steps) active = false;
            double* tr = tile + rr * ROW + lane;
            tr[0] = st.x0; tr[32] = st.x1; tr[64] = st.x2;
            if ((rr & (CK - 1)) == 0 && k <= a.n_steps) {
                double* o = ckc + (size_t)(k / CK) * (6 * COMET_LANES);
                o[0] = st.x0; o[32] = st.x1; o[64] = st.x2; o[96] = st.t0; o[128] = st.t1; o[160] = st.t2;
            }
        }
        __syncwarp();
        const unsigned live = __ballot_sync(FULL, np > r0);  // lanes with a real row in this tile
        // ---- level 0 (lane = wire) and, per wire with candidates, level 1 + sweeps (lane = seed) ------
        for (int r = 0; r < n_rounds; ++r) {
            if (n_rounds > 1) load_round(r);
            unsigned m[Q];
#pragma unroll
            for (int q = 0; q < Q; ++q) m[q] = 0u;
            const double* sp = tile + (TR / 2) * ROW;
#pragma unroll 4
            for (int ss = 0; ss < 32; ++ss) {
                const double x0 = sp[ss], x1 = sp[32 + ss], x2 = sp[64 + ss];
#pragma unroll
                for (int q = 0; q < Q; ++q)
                    m[q] |= (unsigned)(__double2hiint(d2_fma(ec[q], x0, x1, x2)) <= thi[q]) << ss;
            }
#pragma unroll
            for (int q = 0; q < Q; ++q) {
                if (thi[q] >= 0) m[q] |= nolip_mask;
                m[q] &= live;
                unsigned any = __ballot_sync(FULL, m[q] != 0u);
                while (any) {
                    const int wl = __ffs(any) - 1;
                    any &= any - 1;
                    const unsigned mask = __shfl_sync(FULL, m[q], wl);
                    const int i = (r * Q + q) * 32 + wl;
                    // ---- wire i, lane = seed ------------------------------------------------------
                    const bool mine = (mask >> lane) & 1u;
                    const size_t pidx = (size_t)i * a.SP + s;
                    const double old = __ldcg(a.bd + pidx);           // used after the sweeps
                    EvalC w;
                    load_evalc(w, a.wt, W, i);                        // warp-uniform, L1-resident
                    const double cap = __ldg(a.wt + 14 * W + i);
                    int d1h[NSUB];
                    int m1 = IMAX;
#pragma unroll
                    for (int j = 0; j < NSUB; ++j) {
                        const double* ps = tile + (j * COMET_M1 + COMET_M1 / 2) * ROW + lane;
                        d1h[j] = __double2hiint(d2_fma(w, ps[0], ps[32], ps[64]));
                        m1 = min(m1, d1h[j]);
                    }
                    const double ub = fmin(cap, sqrt(__hiloint2double(m1 + 1, 0)));
                    const double t1 = ub + half1;
                    const int t1h = lip_ok ? __double2hiint(t1 * t1) : IMAX;
                    unsigned sub = 0u;
#pragma unroll
                    for (int j = 0; j < NSUB; ++j)
                        if (mine && d1h[j] <= t1h) sub |= 1u << j;
                    unsigned wsub = __reduce_or_sync(FULL, sub);
                    if (!wsub) continue;
                    double best = old;
                    int bk = -1;
                    while (wsub) {
                        const int j = __ffs(wsub) - 1;
                        wsub &= wsub - 1;
                        const double* pr = tile + (j * COMET_M1) * ROW + lane;
#pragma unroll
                        for (int kk = 0; kk < COMET_M1; ++kk) {
                            const double d2 = d2_fma(w, pr[kk * ROW], pr[kk * ROW + 32], pr[kk * ROW + 64]);
                            const int k = r0 + j * COMET_M1 + kk;
                            // rows at or past n_pts repeat the last state: not recorded, never taken
                            if (d2 < best && k < np) { best = d2; bk = k; }
                        }
                    }
                    if (bk >= 0) { a.bd[pidx] = best; a.kb[pidx] = bk; }
                }
            }
        }
        __syncwarp();
        if (!__any_sync(FULL, active)) break;
    }
    if (valid) a.n_pts[s] = np;
    // ---- finish: far pairs take the cutoff, (chunk, wire) items with a near lane go to k_fine_ck -------
    for (int i = 0; i < W; ++i) {
        const size_t pidx = (size_t)i * a.SP + s;
        const double bdv = __ldcg(a.bd + pidx);
        const int kbv = __ldcg(a.kb + pidx);
        const double cap = __ldg(a.wt + 14 * W + i);
        const bool near = valid && kbv >= 0 && (sqrt(bdv) <= cap || !lip_ok);
        if (__any_sync(FULL, near)) {
            if (!near && kbv >= 0) a.kb[pidx] = -1;
            if (lane == 0) a.items[atomicAdd(a.n_items, 1u)] = ((unsigned long long)chunk << 16) | (unsigned)i;
        } else {
            a.bd[pidx] = lam2;
        }
    }
}

// Persistent warps over the work list: exact decision between bk-1, bk, bk+1 on states regenerated
// from the nearest checkpoint at or before bk-1, then O6..O8 (common.cuh).
__global__ void __launch_bounds__(COMET_FINE_THREADS, COMET_FINE_MINB) k_fine_ck(const FusedArgs a)
{
    constexpr int CK = COMET_FUSED_CK;
    const int lane = threadIdx.x & 31;
    const unsigned n_items = *a.n_items;
    const unsigned n_warps = gridDim.x * (COMET_FINE_THREADS / 32);
    const int W = a.W;
    const double lam2 = xmul(a.lambda, a.lambda);
    for (unsigned it = blockIdx.x * (COMET_FINE_THREADS / 32) + (threadIdx.x >> 5); it < n_items; it += n_warps) {
        const unsigned long long item = a.items[it];
        const int64_t chunk = (int64_t)(item >> 16);
        const int i = (int)(item & 0xffffu);
        const int64_t s = chunk * COMET_LANES + lane;
        const size_t pidx = (size_t)i * a.SP + s;
        const int bk = a.kb[pidx];
        double e2 = lam2;
        if (s < a.n_seeds && bk >= 0) {
            const int np = a.n_pts[s];
            const double px = a.seeds[3 * a.stride + s], py = a.seeds[4 * a.stride + s], pz = a.seeds[5 * a.stride + s];
            const double c = xdiv(a.qkb, xsqrt(xdot3(px, py, pz, px, py, pz)));
            WireLine wl;
            wl.m0 = __ldg(a.wt + i); wl.m1 = __ldg(a.wt + W + i); wl.m2 = __ldg(a.wt + 2 * W + i);
            wl.w0 = __ldg(a.wt + 3 * W + i); wl.w1 = __ldg(a.wt + 4 * W + i); wl.w2 = __ldg(a.wt + 5 * W + i);
            const int ka = max(bk - 1, 0), kz = min(bk + 1, np - 1);
            const int kc = ka & ~(CK - 1);
            const double* o = a.ck + ((size_t)chunk * a.n_ck + (size_t)(kc / CK)) * (6 * COMET_LANES) + lane;
            State st;
            st.x0 = o[0]; st.x1 = o[32]; st.x2 = o[64]; st.t0 = o[96]; st.t1 = o[128]; st.t2 = o[160];
            for (int k = kc; k < ka; ++k) rkn4_step(st, a.hk, c);
            State bs = st;
            int ks = ka;
            double bd = 0.0;
            for (int k = ka; k <= kz; ++k) {
                double u0, u1, u2;
                const double d2 = perp2_exact(st.x0, st.x1, st.x2, wl, u0, u1, u2);
                if (k == ka || d2 < bd) { bd = d2; ks = k; bs = st; }
                if (k < kz) rkn4_step(st, a.hk, c);
            }
            const double D = fine_dca(bs, ks, np, a.hk.h, c, wl);
            const double e = wire_residual(D, a.rho, __ldg(a.hit_off + i), __ldg(a.hit_off + i + 1), a.lambda,
                                           nullptr, nullptr);
            e2 = xmul(e, e);
        }
        a.bd[pidx] = e2;
    }
}

}  // namespace comet
