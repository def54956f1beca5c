// scan_small.cuh -- kernels A + B2 for launches that cannot fill the GPU (the refined seed sets of a stage, a few
// hundred chunks; BASELINE.json configs[0]), uniform field (sm_100a).
//
// k_scan_fused gives a chunk to one warp, which alternates between generating a 16-row tile and searching it: on a
// small launch every warp is a serial chain of ~370 RKN4 steps interleaved with its search, and the SMs idle in
// between (its SPLIT variant lets four warps repeat the same chain and share the wires).  Here a CTA of four warps
// owns the chunk and the two jobs overlap:
//
//   warp 0        generates the track, tile by tile, into a double-buffered tile in shared memory (the definition's
//                 RKN4 steps, the target-region test, the checkpoints for k_fine_ck) -- one tile ahead of the search;
//   warps 1 - 3   search the tile that is ready: the level-0 test of k_scan_fused (lane = wire; a search warp takes every
//                 third wire, so that neighbouring wires -- near the same rows -- go to different warps), then the sweeps
//                 of the sub-blocks its tests opened (lane = seed), merging the pair keys with an atomic min;
//   all four      the finish of k_scan_fused, wire groups dealt round-robin.
//
// One __syncthreads per tile.  The chain of the generator (about 110 cycles per step) is what is left on the critical
// path: 24 tiles x 16 steps instead of 24 x (16 steps + the search of a tile).  Same keys, checkpoints and work list as
// k_scan_fused, hence the same n_pts and RSS bit for bit.
#pragma once
#include "scan_fused.cuh"

namespace comet {

#define COMET_SMALL_SMEM (((COMET_FUSED_WFIELDS + 1) * COMET_FUSED_WCAP + 2 * COMET_FUSED_TR * 3 * COMET_LANES) * (int)sizeof(double))

template <bool STATS>
__global__ void __launch_bounds__(128, 4) k_scan_small(const FusedArgs a)
{
    constexpr int TR = COMET_FUSED_TR, CK = COMET_FUSED_CK, ROW = 3 * COMET_LANES, CKF = 6;
    constexpr int FM1 = COMET_FUSED_M1, NSUB = TR / FM1, WCAP = COMET_FUSED_WCAP;
    constexpr int NSEARCH = 3;
    constexpr unsigned FULL = 0xffffffffu;
    if (a.dyn && a.dyn[2]) return;                          // (the turn loop has stopped)
    extern __shared__ __align__(16) double ssm[];
    __shared__ int32_t s_np[2][COMET_LANES];                // recorded states of every lane as known after each tile
    __shared__ int s_gen[2];                                // the generator goes on after this tile
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* wtab = ssm;                                     // [WFIELDS + 1][WCAP]
    double* tiles = ssm + (COMET_FUSED_WFIELDS + 1) * WCAP; // [2][TR][3][32]
    const int W = a.W;
    for (int v = threadIdx.x; v < COMET_FUSED_WFIELDS * WCAP; v += 128) {
        const int f = v / WCAP, i = v - f * WCAP;
        wtab[v] = (i < W) ? __ldg(a.wt + (size_t)(6 + f) * W + i) : -1.0;
    }
    for (int i = threadIdx.x; i < WCAP; i += 128)
        wtab[COMET_FUSED_WFIELDS * WCAP + i] = (i < W) ? wire_slope(__ldg(a.wt + (size_t)8 * W + i), __ldg(a.wt + (size_t)12 * W + i)) : 0.0;
    const int64_t chunk = blockIdx.x;
    const int64_t s = chunk * COMET_LANES + lane;
    const bool valid = s < a.n_seeds;
    const double h = a.hk.h;
    const double INF = 1.7976931348623157e308;
    const double L = COMET_LIP * h;
    const double half1 = (FM1 / 2) * L + COMET_SLACK;
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
    unsigned long long* const keys = reinterpret_cast<unsigned long long*>(a.bd);
    for (int i = warp; i < W; i += 4) keys[(size_t)i * a.SP + s] = COMET_KEY_NONE;
    const int n_tiles = (a.n_steps + TR) / TR;
    unsigned long long st_cnt[ST_N];
    if (STATS) {
#pragma unroll
        for (int j = 0; j < ST_N; ++j) st_cnt[j] = 0;
        if (valid && warp == 0) st_cnt[ST_PAIRS] = (unsigned long long)W;
    }
    // ---- generator state (warp 0) -----------------------------------------------------------------------
    bool active = valid;
    int32_t np = valid ? a.n_steps + 1 : 0;
    const bool use_stop = a.r_stop2 > 0.0;
    double* ckc = a.ck + (size_t)chunk * a.n_ck * (CKF * COMET_LANES) + lane;
    // The chain of dependent operations of a step is the generator's whole cost, so the stop test does not sit on it: blocks
    // of 4 steps are taken and stored unconditionally, the first state in the target region is only remembered, and the
    // rows after it are overwritten with it afterwards (hold-last); a lane that has stopped just repeats its last position.
    auto generate = [&](int t) {
        double* tile = tiles + (t & 1) * (TR * ROW);
        const int r0 = t * TR;
#pragma unroll 1
        for (int b = 0; b < TR; b += 4) {
            const int k0 = r0 + b;
            double* tb = tile + b * ROW + lane;
            if (active) {
                int first = 4;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int k = k0 + j;
                    if (k > 0 && k <= a.n_steps) {          // (warp-uniform: row 0 is the seed, rows past the capacity repeat the last state)
                        rkn4_step(st, a.hk, c);
                        const double r2 = xadd(xmul(st.x0, st.x0), xmul(st.x1, st.x1));
                        const double rad = xadd(xmul(st.x0, st.t0), xmul(st.x1, st.t1));
                        const bool stop = (r2 < a.r_stop2) & (rad < 0.0) & use_stop;
                        first = (stop & (first == 4)) ? j : first;
                    }
                    tb[j * ROW] = st.x0; tb[j * ROW + 32] = st.x1; tb[j * ROW + 64] = st.x2;
                    if (j == 0 && k <= a.n_steps) {
                        double* o = ckc + (size_t)(k / CK) * (CKF * COMET_LANES);
                        o[0] = st.x0; o[32] = st.x1; o[64] = st.x2; o[96] = st.t0; o[128] = st.t1; o[160] = st.t2;
                    }
                }
                if (first < 4) {
                    np = k0 + first + 1;
                    active = false;
                    st.x0 = tb[first * ROW]; st.x1 = tb[first * ROW + 32]; st.x2 = tb[first * ROW + 64];
                    for (int j = first + 1; j < 4; ++j) { tb[j * ROW] = st.x0; tb[j * ROW + 32] = st.x1; tb[j * ROW + 64] = st.x2; }
                } else if (k0 + 3 >= a.n_steps) {
                    active = false;                         // capacity reached: np stays n_steps + 1
                }
            } else {
#pragma unroll
                for (int j = 0; j < 4; ++j) { tb[j * ROW] = st.x0; tb[j * ROW + 32] = st.x1; tb[j * ROW + 64] = st.x2; }
            }
        }
        s_np[t & 1][lane] = np;
        const bool go_on = __any_sync(FULL, active);
        if (lane == 0) s_gen[t & 1] = go_on ? 1 : 0;
    };
    if (warp == 0) {
        s_np[1][lane] = np;                                 // (so that the minimum over the two buffers below is the final count)
        generate(0);
    }
    __syncthreads();
    for (int t = 0; t < n_tiles; ++t) {
        const int r0 = t * TR;
        const bool more = s_gen[t & 1] != 0 && t + 1 < n_tiles;
        if (warp == 0) {
            if (more) generate(t + 1);
        } else {
            // ---- search tile t (k_scan_fused's level 0 and sweeps) ------------------------------------------
            const double* tile = tiles + (t & 1) * (TR * ROW);
            const int32_t npt = s_np[t & 1][lane];
            const unsigned live = __ballot_sync(FULL, npt > r0);
            if (live) {
                const int rep = __ffs(live) - 1;
                const bool is_live = (live >> lane) & 1u;
                double rx[NSUB][3];
                float rxy[NSUB], rz[NSUB];
#pragma unroll
                for (int j = 0; j < NSUB; ++j) {
                    const int srow = j * FM1 + FM1 / 2;
                    const double* ps = tile + srow * ROW + lane;
                    const double s0 = ps[0], s1 = ps[32], s2 = ps[64];
                    rx[j][0] = __shfl_sync(FULL, s0, rep); rx[j][1] = __shfl_sync(FULL, s1, rep); rx[j][2] = __shfl_sync(FULL, s2, rep);
                    const double e0 = s0 - rx[j][0], e1 = s1 - rx[j][1], e2 = s2 - rx[j][2];
                    const float fxy = is_live ? __fsqrt_ru(__double2float_ru(fma(e0, e0, e1 * e1))) : 0.f;
                    const float fz = is_live ? __double2float_ru(fabs(e2)) : 0.f;
                    rxy[j] = __uint_as_float(__reduce_max_sync(FULL, __float_as_uint(fxy)));
                    rz[j] = __uint_as_float(__reduce_max_sync(FULL, __float_as_uint(fz)));
                }
                const bool any_nolip = (nolip_mask & live) != 0u;
                // every search warp takes a strided third of the wires (neighbouring wires, which tend to be near the same
                // rows, go to different warps): its level-0 tests and the sweeps they open
                for (int r = 0; r * (32 * NSEARCH) < W; ++r) {
                    unsigned sm = 0u;
                    {
                        const int i = NSEARCH * (r * 32 + lane) + (warp - 1);
                        const int ii = min(i, W - 1);
                        EvalC ec;
                        wconst_evalc(ec, wtab, a.wt, W, ii);
                        const double cap = (i < W) ? wconst(wtab, a.wt, W, 8, ii) : -1.0;
                        const double swz = (ii < WCAP) ? wtab[COMET_FUSED_WFIELDS * WCAP + ii] : wire_slope(ec.e1z, ec.e2z);
#pragma unroll
                        for (int j = 0; j < NSUB; ++j) {
                            const double spread = ((double)rxy[j] + (double)rz[j] * swz) * 1.000001;
                            const double t0 = cap + half1 + spread;
                            if (d2_fma(ec, rx[j][0], rx[j][1], rx[j][2]) <= t0 * t0) sm |= 1u << j;
                        }
                        if (any_nolip) sm = (1u << NSUB) - 1u;
                        if (cap < 0.0) sm = 0u;
                        if (STATS && cap >= 0.0) st_cnt[ST_SAMPLES] += NSUB;
                    }
                    unsigned any = __ballot_sync(FULL, sm != 0u);
                    while (any) {
                        const int wl = __ffs(any) - 1;
                        any &= any - 1;
                        unsigned wsub = __shfl_sync(FULL, sm, wl);
                        const int i = NSEARCH * (r * 32 + wl) + (warp - 1);
                        EvalC w;
                        wconst_evalc(w, wtab, a.wt, W, i);
                        double best = INF;
                        int bk = -1;
                        while (wsub) {
                            const int j = __ffs(wsub) - 1;
                            wsub &= wsub - 1;
                            const double* pr = tile + (j * FM1) * ROW + lane;
                            if (STATS) { st_cnt[ST_ROWS_EXEC] += FM1; if (is_live) st_cnt[ST_ROWS_NEEDED] += FM1; }
                            const int k0 = r0 + j * FM1;
#pragma unroll
                            for (int kk = 0; kk < FM1; ++kk) {
                                const double d2 = d2_fma(w, pr[kk * ROW], pr[kk * ROW + 32], pr[kk * ROW + 64]);
                                if (d2 < best) { best = d2; bk = k0 + kk; }
                            }
                        }
                        bk = min(bk, npt - 1);
                        if (bk >= 0 && npt > r0) atomicMin(keys + (size_t)i * a.SP + s, pack_key(best, bk));
                    }
                }
            }
        }
        __syncthreads();
        if (!more) break;
    }
    // the count only goes down (a lane stops once): the smaller of the two buffers is the one after the last tile
    np = min(s_np[0][lane], s_np[1][lane]);
    if (valid && warp == 0) { a.n_pts[s] = np; a.cw[s] = c; }
    // ---- finish (k_scan_fused's), wire groups dealt round-robin to the four warps ---------------------------
    constexpr int FB = 8, LCAP = 512;
    unsigned short* lst = reinterpret_cast<unsigned short*>(tiles) + warp * LCAP;
    int cnt = 0;
    auto flush = [&]() {
        __syncwarp();
        unsigned base = 0;
        if (lane == 0) base = atomicAdd(a.n_items, (unsigned)cnt);
        base = __shfl_sync(FULL, base, 0);
        for (int j = lane; j < cnt; j += 32) a.items[base + j] = ((unsigned long long)chunk << 16) | (unsigned)lst[j];
        cnt = 0;
        __syncwarp();
    };
    for (int i0 = warp * FB; i0 < W; i0 += 4 * FB) {
        unsigned long long kv[FB];
        double cap2[FB];
#pragma unroll
        for (int j = 0; j < FB; ++j) {
            const int i = min(i0 + j, W - 1);
            kv[j] = __ldcg(keys + (size_t)i * a.SP + s);
            const double cap = wconst(wtab, a.wt, W, 8, i);
            cap2[j] = cap * cap;
        }
#pragma unroll
        for (int j = 0; j < FB; ++j) {
            const int i = i0 + j;
            if (i < W) {
                const size_t pidx = (size_t)i * a.SP + s;
                const bool found = kv[j] != COMET_KEY_NONE;
                const bool near = valid && found && (key_d2(kv[j]) <= cap2[j] || !lip_ok);
                if (STATS && near) st_cnt[ST_FINE_NEEDED] += 1;
                if (__any_sync(FULL, near)) {
                    if (STATS) st_cnt[ST_FINE_EXEC] += 1;
                    if (!near && found) keys[pidx] = COMET_KEY_NONE;
                    if (lane == 0) lst[cnt] = (unsigned short)i;
                    if (++cnt == LCAP) flush();
                } else {
                    a.bd[pidx] = lam2;
                }
            }
        }
    }
    if (cnt) flush();
    if (STATS) {
#pragma unroll
        for (int j = 0; j < ST_N; ++j) {
            unsigned long long v = st_cnt[j];
            for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(FULL, v, o);
            if (lane == 0 && a.stats && v) atomicAdd(a.stats + j, v);
        }
    }
}

}  // namespace comet
