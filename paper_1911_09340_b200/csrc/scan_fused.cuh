// scan_fused.cuh -- kernels A and B in one pass with the track kept on chip (sm_100a).
//
// The materialised path writes 48 bytes per recorded state to HBM (k_extrapolate runs at the HBM
// write rate) only for kernel B to read a small part of it back.  Here a warp owns one track chunk
// (32 consecutive seeds, lane = seed) from the seed to its (seed, wire) shortlist:
//
//   generate   TR RKN4 steps per lane (the definition's operations, common.cuh), the positions of the
//              TR rows go to a warp-private shared-memory tile [TR][3][32] fp64 (conflict-free, never
//              to HBM); every CK-th recorded state (x, T) is written to a small checkpoint buffer;
//   level 0    one evaluation per (8-row sub-block, wire) with lane = WIRE, the wires' shortlist
//              constants coming from a table in shared memory (one copy per CTA): the sub-block sample
//              of one representative seed and the largest offset of the other seeds' samples from it
//              bound every seed's distance from below (Lipschitz bound of dca.cuh with the wire's far
//              radius as the upper bound), so a sub-block is opened for a wire only if some seed may
//              have its closest state there;
//   sweeps     per wire with open sub-blocks (lane = seed again, the wire's constants are broadcast
//              from the table): their rows are evaluated from the tile; the tile's
//              best (squared distance, row) of the pair is merged into the pair workspace with one
//              fire-and-forget 64-bit atomic min on a packed key (no read-modify-write round trip to
//              L2): key = bits(d^2) with the low 13 bits replaced by the row, so keys order by d^2
//              (to 2^-39 relative) and then by row -- enough for a shortlist whose choice is re-decided
//              exactly between bk-1, bk, bk+1;
//   finish     per wire: pairs whose closest state is farther than the far radius get e^2 = cutoff^2,
//              (chunk, wire) items with a near lane go to the work list of k_fine_ck.
//
// k_fine_ck takes the exact decision between bk-1, bk, bk+1 and runs the virtual-plane iteration
// from states it regenerates from the nearest checkpoint (at most CK-1+2 RKN steps), so every
// number that reaches a result is produced by the same operations as in the materialised path and
// by the definition: n_pts and RSS are bit-identical.
//
// RSS-only (the hot path).  Calls that ask for D or k* of every pair use the materialised path.
// Seed sets in z-runs (the first-iteration grids of the method) are served by k_gen_unique + k_scan_zrun
// (scan_zgroup.cuh, scan_zrun.cuh) and share k_fine_ck<.., ZG = true> below; this kernel serves every other seed set
// (refined sets, small calls) and the field map.
#pragma once
#include "common.cuh"
#include "dca.cuh"

namespace comet {

#ifndef COMET_FUSED_TR
#define COMET_FUSED_TR 16          // rows per tile
#endif
#ifndef COMET_FUSED_CK
#define COMET_FUSED_CK 4           // rows between checkpoints
#endif
#ifndef COMET_FUSED_WARPS
#define COMET_FUSED_WARPS 4        // warps (chunks) per CTA; they share the wire table
#endif
#ifndef COMET_FUSED_MINB
#define COMET_FUSED_MINB 4         // resident CTAs per SM the register allocation aims at
#endif
#ifndef COMET_FUSED_M1
#define COMET_FUSED_M1 8           // rows per sub-block
#endif
#ifndef COMET_FUSED_WCAP
#define COMET_FUSED_WCAP 96        // wires whose constants the shared-memory table holds (the others: L1/L2)
#endif
#define COMET_FUSED_WFIELDS 9      // e1[3] -m.e1 | e2[3] -m.e2 | far radius  (fields 6..14 of the wire table)
// the CTA's table has one more row: sqrt(1 - w_z^2) rounded up, the wire's slope against the z axis

// Packed shortlist key of a (seed, wire) pair: the bit pattern of the non-negative squared distance
// (monotone as an unsigned integer) with its 13 low mantissa bits replaced by the row (<= 4096).
#define COMET_KEY_NONE 0xffffffffffffffffull
#define COMET_KEY_KBITS 13
__device__ __forceinline__ unsigned long long pack_key(double d2, int k)
{
    return ((unsigned long long)__double_as_longlong(d2) & ~((1ull << COMET_KEY_KBITS) - 1ull)) | (unsigned long long)k;
}
__device__ __forceinline__ double key_d2(unsigned long long key)
{
    return __longlong_as_double((long long)(key & ~((1ull << COMET_KEY_KBITS) - 1ull)));
}
__device__ __forceinline__ int key_row(unsigned long long key) { return (int)(key & ((1ull << COMET_KEY_KBITS) - 1ull)); }

struct FusedArgs {
    const double* seeds;
    int64_t stride;
    int64_t n_seeds;         // seeds of this slab
    double qkb;
    StepK hk;
    int32_t n_steps;
    double r_stop2;
    const double* wt;        // [15][W]
    const float* wtf;        // [11][W] single-precision shortlist fields (k_wire_prep), for k_scan_zrun's levels A and B
    int32_t W;
    const int32_t* hit_off;
    const double* rho;
    double lambda;
    int64_t SP;              // 32 * chunks of this slab: stride of bd
    int32_t n_ck;            // checkpoint rows per chunk: n_steps / CK + 1
    double* ck;              // [chunks][n_ck][6][32]
    double* bd;              // [W][SP] packed (d^2, row) key of the pair's closest state so far; e^2 afterwards
    int32_t* n_pts;          // [n_seeds]
    double* cw;              // [SP] curvature constant c = kappa q B_z / |p| of every seed, for k_fine_ck
    double* tw;              // [SP] ZG: T_z of every seed, for k_fine_ck
    unsigned long long* items;
    unsigned int* n_items;   // [0] items listed by the scan, [1] items handed out by k_fine_ck
    unsigned long long* stats;
    FieldMap F;              // field-map variants (FIELD = true): the map, and qkb = kappa q, hk.h = h_max
    double h_min;            // h_max / 64 (R31)
    const unsigned int* zg;  // scan_zgroup.cuh: run length of the launch's seeds (device); nullptr = not checked
    int32_t zrun;            //   or the caller's promise (comet_scan_rss z_run >= 8): `zg` is then nullptr
    double* ub;              // scan_zgroup.cuh: (x_0, x_1, T_0, T_1) of the distinct transverse tracks [u / 32][u_rows][4][32]
    int32_t* np_u;           //   and their numbers of recorded states
    int32_t u_rows;          //   rows per track in ub: n_steps + 1 rounded up to whole 64-row blocks
    const int32_t* dyn;      // comet_scan_turns: device {fired wires left, entries left, stop flag}: nullptr = sizes are exact
    unsigned int* tm;        // scan_zrun.cuh: [chunks][ceil(W / 32)] bit i: k_fine_ck fills the e^2 row of wire i (else cutoff^2)
};
#define COMET_ZG_MIN 8             // smallest run length served by the ZG kernels (scan_zgroup.cuh)
__device__ __forceinline__ unsigned int zgroup_of(const unsigned int* flag)
{
    const unsigned int f = *flag;
    return f > 32u ? 32u : f;
}
// run length the ZG kernels work with: the caller's promise, else what k_zgroup_check found
__device__ __forceinline__ unsigned int zrun_of(const int32_t zrun, const unsigned int* flag)
{
    return zrun > 0 ? (unsigned int)zrun : zgroup_of(flag);
}
#define COMET_CK_FIELDS(FIELD) ((FIELD) ? 7 : 6)    // checkpoint row: x, T and, in a field map, the trial step
#ifndef COMET_FUSED_CK_FIELD
#define COMET_FUSED_CK_FIELD 4     // rows between checkpoints in a field map (1 and 2 were measured: the extra checkpoint traffic costs what the shorter replay saves)
#endif
#define COMET_CK_ROWS(FIELD) ((FIELD) ? COMET_FUSED_CK_FIELD : COMET_FUSED_CK)

// shortlist constants of wire i: from the CTA's table when it holds the wire, else from the wire table
// in global memory (warp-uniform or lane-contiguous addresses either way)
__device__ __forceinline__ double wconst(const double* wtab, const double* __restrict__ wt, int W, int f, int i)
{
    return (i < COMET_FUSED_WCAP) ? wtab[f * COMET_FUSED_WCAP + i] : __ldg(wt + (size_t)(6 + f) * W + i);
}
__device__ __forceinline__ void wconst_evalc(EvalC& w, const double* wtab, const double* __restrict__ wt, int W, int i)
{
    w.e1x = wconst(wtab, wt, W, 0, i); w.e1y = wconst(wtab, wt, W, 1, i); w.e1z = wconst(wtab, wt, W, 2, i);
    w.c1 = wconst(wtab, wt, W, 3, i);
    w.e2x = wconst(wtab, wt, W, 4, i); w.e2y = wconst(wtab, wt, W, 5, i); w.e2z = wconst(wtab, wt, W, 6, i);
    w.c2 = wconst(wtab, wt, W, 7, i);
}

// sqrt(1 - w_z^2) = sqrt(e1z^2 + e2z^2) for the orthonormal basis {e1, e2, w}, rounded up
__device__ __forceinline__ double wire_slope(double e1z, double e2z)
{
    return (double)__fsqrt_ru(__double2float_ru(fma(e1z, e1z, e2z * e2z)));
}

// (Seed sets in z-runs are served by k_scan_zrun, scan_zrun.cuh; with the run length found on the device both kernels
// are enqueued and the one that does not serve the launch returns at once.)
template <bool STATS, bool FIELD, bool SPLIT = false>
__global__ void __launch_bounds__(32 * COMET_FUSED_WARPS, COMET_FUSED_MINB) k_scan_fused(const FusedArgs a)
{
    constexpr int CKF = COMET_CK_FIELDS(FIELD);
    constexpr int TR = COMET_FUSED_TR, CK = COMET_CK_ROWS(FIELD), ROW = 3 * COMET_LANES;
    constexpr int FM1 = COMET_FUSED_M1;
    constexpr int NSUB = TR / FM1;
    constexpr int WCAP = COMET_FUSED_WCAP;
    constexpr unsigned FULL = 0xffffffffu;
    static_assert(TR % FM1 == 0 && TR % CK == 0, "tile rows");
    if (a.dyn && a.dyn[2]) return;                          // (the turn loop has stopped)
    if (!FIELD && a.zg && zgroup_of(a.zg) >= COMET_ZG_MIN) return;     // the z-run kernels serve this launch (scan_zrun.cuh)
    extern __shared__ __align__(16) double fsm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* wtab = fsm;                                     // [WFIELDS + 1][WCAP]
    double* tile = fsm + (COMET_FUSED_WFIELDS + 1) * WCAP + warp * (TR * ROW);
    const int W = a.W;
    for (int v = threadIdx.x; v < COMET_FUSED_WFIELDS * WCAP; v += 32 * COMET_FUSED_WARPS) {
        const int f = v / WCAP, i = v - f * WCAP;
        wtab[v] = (i < W) ? __ldg(a.wt + (size_t)(6 + f) * W + i) : -1.0;
    }
    for (int i = threadIdx.x; i < WCAP; i += 32 * COMET_FUSED_WARPS)
        wtab[COMET_FUSED_WFIELDS * WCAP + i] = (i < W) ? wire_slope(__ldg(a.wt + (size_t)8 * W + i), __ldg(a.wt + (size_t)12 * W + i)) : 0.0;
    __syncthreads();
    // SPLIT (small launches that cannot fill the GPU: the refined seed sets of a stage): the CTA's warps all take
    // the SAME chunk -- each generates the track for itself -- and share its wires: warp w takes the level-0 rounds
    // and the finish groups w, w + 4, ...; one chunk is then a quarter of the serial work per warp
    constexpr bool split = SPLIT;
    const int wpart = split ? warp : 0, nparts = split ? COMET_FUSED_WARPS : 1;
    const int64_t chunk = split ? (int64_t)blockIdx.x : (int64_t)blockIdx.x * COMET_FUSED_WARPS + warp;
    if (chunk * COMET_LANES >= a.n_seeds) return;
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
    // states are at most 1.001 h apart when |curvature| h <= 0.05 (in a map: with its largest |B| and h = h_max)
    const bool lip_ok = (FIELD ? fabs(c) * __ldg(a.F.bmax) * h : fabs(c) * h) <= COMET_CH_MAX;
    const unsigned nolip_mask = __ballot_sync(FULL, valid && !lip_ok);
    double htry = h;                                        // FIELD: trial step of the adaptive control (R31)
    bool active = valid;
    int32_t np = valid ? a.n_steps + 1 : 0;
    const bool use_stop = a.r_stop2 > 0.0;
    // pair workspace of this chunk: nothing found yet
    unsigned long long* const keys = reinterpret_cast<unsigned long long*>(a.bd);
    for (int i = 32 * wpart; i < W; i += 32 * nparts)      // (the wires of this warp's rounds)
        for (int q = i; q < min(i + 32, W); ++q) keys[(size_t)q * a.SP + s] = COMET_KEY_NONE;

    const int n_rounds = (W + 31) / 32;                     // level 0: wire i = r * 32 + lane
    double* ckc = a.ck + (size_t)chunk * a.n_ck * (CKF * COMET_LANES) + lane;
    const int n_tiles = (a.n_steps + TR) / TR;              // rows 0 .. n_steps
    unsigned long long st_cnt[ST_N];                        // work counters (COMET_OPT_STATS), thread-level
    if (STATS) {
#pragma unroll
        for (int j = 0; j < ST_N; ++j) st_cnt[j] = 0;
        if (valid && wpart == 0) st_cnt[ST_PAIRS] = (unsigned long long)W;
    }
#ifdef COMET_FUSED_PROF
    long long pc_gen = 0, pc_l0 = 0, pc_l1 = 0, pc_visits = 0, pc_sweeps = 0, pc_mark;
#define PC_MARK() (pc_mark = clock64())
#define PC_ADD(v) do { const long long pc_now = clock64(); v += pc_now - pc_mark; pc_mark = pc_now; } while (0)
#else
#define PC_MARK()
#define PC_ADD(v)
#endif
    for (int t = 0; t < n_tiles; ++t) {
        const int r0 = t * TR;
        PC_MARK();
        // ---- generate rows r0 .. r0 + TR - 1 (Algorithm 1; finished lanes hold their last state) ------
#pragma unroll (FIELD ? 1 : 2)
        for (int rr = 0; rr < TR; ++rr) {
            const int k = r0 + rr;
            if (k > 0 && active) {
                if (FIELD) (void)adaptive_field_step(st, htry, h, a.h_min, c, a.F);
                else rkn4_step(st, a.hk, c);
                if (use_stop && in_target_region(st, a.r_stop2)) { np = k + 1; active = false; }
            }
            if (k >= a.n_steps) active = false;
            double* tr = tile + rr * ROW + lane;
            tr[0] = st.x0; tr[32] = st.x1; tr[64] = st.x2;
            if ((rr & (CK - 1)) == 0 && k <= a.n_steps && wpart == 0) {
                double* o = ckc + (size_t)(k / CK) * (CKF * COMET_LANES);
                o[0] = st.x0; o[32] = st.x1; o[64] = st.x2; o[96] = st.t0; o[128] = st.t1; o[160] = st.t2;
                if (FIELD) o[192] = htry;
            }
        }
        __syncwarp();
        PC_ADD(pc_gen);
        const unsigned live = __ballot_sync(FULL, np > r0);  // lanes with a real row in this tile
        if (!live) break;
        // ---- level 0 (lane = wire): one evaluation per (wire, sub-block) --------------------------------
        // The sample (row M1/2) of sub-block j of every live seed lies within `spread` of the sample of
        // a representative seed -- measured perpendicular to the wire: at most rho_xy + rho_z sqrt(1 - w_z^2)
        // for offsets of at most rho_xy in (x, y) and rho_z in z -- and the distance to a line is
        // 1-Lipschitz, so no row of the sub-block of any seed is closer to the wire than
        // d(representative sample) - spread - (M1/2) L.  Sub-blocks that cannot hold a state within the
        // wire's far radius are skipped for the whole chunk; a chunk of unrelated seeds only loses pruning.
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
            // non-negative floats order like their bit patterns
            rxy[j] = __uint_as_float(__reduce_max_sync(FULL, __float_as_uint(fxy)));
            rz[j] = __uint_as_float(__reduce_max_sync(FULL, __float_as_uint(fz)));
        }
        const bool any_nolip = (nolip_mask & live) != 0u;
        for (int r = wpart; r < n_rounds; r += nparts) {
            unsigned sm = 0u;                               // bit j: sub-block j of this tile may matter to the lane's wire
            {
                const int i = r * 32 + lane;
                const int ii = min(i, W - 1);
                EvalC ec;
                wconst_evalc(ec, wtab, a.wt, W, ii);
                const double cap = (i < W) ? wconst(wtab, a.wt, W, 8, ii) : -1.0;   // far radius; < 0: no entries
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
            PC_ADD(pc_l0);
            unsigned any = __ballot_sync(FULL, sm != 0u);
            while (any) {
                const int wl = __ffs(any) - 1;
                any &= any - 1;
                unsigned wsub = __shfl_sync(FULL, sm, wl);
                const int i = r * 32 + wl;
                // ---- wire i, lane = seed: sweep the open sub-blocks row by row --------------------------
#ifdef COMET_FUSED_PROF
                pc_visits += 1;
#endif
                EvalC w;
                wconst_evalc(w, wtab, a.wt, W, i);          // broadcast
                double best = INF;
                int bk = -1;
                while (wsub) {
                    const int j = __ffs(wsub) - 1;
                    wsub &= wsub - 1;
#ifdef COMET_FUSED_PROF
                    pc_sweeps += 1;
#endif
                    const double* pr = tile + (j * FM1) * ROW + lane;
                    if (STATS) { st_cnt[ST_ROWS_EXEC] += FM1; if (is_live) st_cnt[ST_ROWS_NEEDED] += FM1; }
                    const int k0 = r0 + j * FM1;
#pragma unroll
                    for (int kk = 0; kk < FM1; ++kk) {
                        const double d2 = d2_fma(w, pr[kk * ROW], pr[kk * ROW + 32], pr[kk * ROW + 64]);
                        if (d2 < best) { best = d2; bk = k0 + kk; }
                    }
                }
                // Rows at or past n_pts repeat the last recorded state, so one of them can only tie with it (and then
                // loses to the strict <) or stand in for it from a later sub-block: the row index is clamped, the distance
                // is that state's own.  Lanes without a recorded row in this tile keep out.
                bk = min(bk, np - 1);
                if (bk >= 0 && np > r0) atomicMin(keys + (size_t)i * a.SP + s, pack_key(best, bk));
            }
            PC_ADD(pc_l1);
        }
        __syncwarp();
        if (!__any_sync(FULL, active)) break;
    }
#ifdef COMET_FUSED_PROF
    if (lane == 0 && a.stats) {
        atomicAdd(a.stats + 0, (unsigned long long)pc_gen); atomicAdd(a.stats + 1, (unsigned long long)pc_l0);
        atomicAdd(a.stats + 2, (unsigned long long)pc_l1); atomicAdd(a.stats + 3, (unsigned long long)pc_visits);
        atomicAdd(a.stats + 4, (unsigned long long)pc_sweeps);
    }
    PC_MARK();
#endif
    if (valid && wpart == 0) { a.n_pts[s] = np; a.cw[s] = c; }
    // ---- finish: far pairs take the cutoff, (chunk, wire) items with a near lane go to k_fine_ck -------
    // Keys come from L2: FB wires in flight at a time.  The items are collected in the (now free) tile
    // and appended to the work list with one reservation per LCAP items.
    constexpr int FB = 8, LCAP = 1024;
    static_assert(LCAP * (int)sizeof(unsigned short) <= TR * ROW * (int)sizeof(double), "item list fits the tile");
    unsigned short* lst = reinterpret_cast<unsigned short*>(tile);
    int cnt = 0;                                            // warp-uniform
    auto flush = [&]() {
        __syncwarp();
        unsigned base = 0;
        if (lane == 0) base = atomicAdd(a.n_items, (unsigned)cnt);
        base = __shfl_sync(FULL, base, 0);
        for (int j = lane; j < cnt; j += 32) a.items[base + j] = ((unsigned long long)chunk << 16) | (unsigned)lst[j];
        cnt = 0;
        __syncwarp();
    };
    // (SPLIT: the groups of the wires of this warp's rounds: FB divides 32)
    for (int i0 = 0; i0 < W; i0 += FB) {
        if (((i0 >> 5) % nparts) != wpart) continue;
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
                // key_d2 <= d^2 of the closest recorded state: "far" is decided on the safe side
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
#ifndef COMET_FUSED_PROF
    if (STATS) {
#pragma unroll
        for (int j = 0; j < ST_N; ++j) {
            unsigned long long v = st_cnt[j];
            for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(FULL, v, o);
            if (lane == 0 && a.stats && v) atomicAdd(a.stats + j, v);
        }
    }
#endif
#ifdef COMET_FUSED_PROF
    if (lane == 0 && a.stats) atomicAdd(a.stats + 5, (unsigned long long)(clock64() - pc_mark));
#endif
}

// Persistent warps over the work list: exact decision between bk-1, bk, bk+1 on states regenerated
// from the nearest checkpoint at or before bk-1, then O6..O8 (common.cuh).
#ifndef COMET_FINE_MINB_FIELD
#define COMET_FINE_MINB_FIELD 2    // the field-map variant needs ~2x the registers (three field look-ups per step)
#endif
// ZG = true (scan_zgroup.cuh): the candidates bk-1, bk, bk+1 are not regenerated: their (x, y, T_0, T_1) are the
// recorded states of the seed's distinct transverse track (the same numbers), z comes from the z checkpoint at or
// before bk-1 plus one addition per step.
template <bool FIELD, bool ZG = false>
__global__ void __launch_bounds__(COMET_FINE_THREADS, FIELD ? COMET_FINE_MINB_FIELD : COMET_FINE_MINB) k_fine_ck(const FusedArgs a)
{
    static_assert(!(FIELD && ZG), "the transverse motion depends on z in a field map");
    if (a.dyn && a.dyn[2]) return;                          // (the turn loop has stopped)
    if (ZG) {
        if (zrun_of(a.zrun, a.zg) < COMET_ZG_MIN) return;
    } else if (!FIELD && a.zg && zgroup_of(a.zg) >= COMET_ZG_MIN) {
        return;
    }
    const int zshift = ZG ? 31 - __clz((int)zrun_of(a.zrun, a.zg)) : 0;
    constexpr int CK = COMET_CK_ROWS(FIELD);
    constexpr int CKF = COMET_CK_FIELDS(FIELD);
    const int lane = threadIdx.x & 31;
    const unsigned n_items = *a.n_items;
    const unsigned n_warps = gridDim.x * (COMET_FINE_THREADS / 32);
    const int W = a.W;
    const double lam2 = xmul(a.lambda, a.lambda);
    // a warp's first item is its own index; the next ones are handed out by a counter -- asked for before the work on the
    // current item, so the answer is there when it is needed: items differ in cost (live lanes, iterations of O6) and the
    // grid is one wave, so a fixed share per warp would leave a fifth of the warp slots idle towards the end
    unsigned it = blockIdx.x * (COMET_FINE_THREADS / 32) + (threadIdx.x >> 5);
    while (it < n_items) {
        unsigned nxt = 0;
        if (lane == 0) nxt = n_warps + atomicAdd(a.n_items + 1, 1u);
        const unsigned long long item = a.items[it];
        const int64_t chunk = (int64_t)(item >> 16);
        const int i = (int)(item & 0xffffu);
        const int64_t s = chunk * COMET_LANES + lane;
        const size_t pidx = (size_t)i * a.SP + s;
        const unsigned long long key = reinterpret_cast<const unsigned long long*>(a.bd)[pidx];
        const int bk = key_row(key);
        double e2 = lam2;
        if (s < a.n_seeds && key != COMET_KEY_NONE) {
            const int np = a.n_pts[s];
            const double c = a.cw[s];
            WireLine wl;
            wl.m0 = __ldg(a.wt + i); wl.m1 = __ldg(a.wt + W + i); wl.m2 = __ldg(a.wt + 2 * W + i);
            wl.w0 = __ldg(a.wt + 3 * W + i); wl.w1 = __ldg(a.wt + 4 * W + i); wl.w2 = __ldg(a.wt + 5 * W + i);
            const int ka = max(bk - 1, 0), kz = min(bk + 1, np - 1);
            double D;
            if (FIELD) {
                // replay the adaptive recording from the checkpoint at or before ka - 1 up to kz + 1: the
                // candidates ka..kz with the lengths of the recorded steps into and out of them (R32)
                const int kc = max(ka - 1, 0) & ~(CK - 1);
                const double* o = a.ck + ((size_t)chunk * a.n_ck + (size_t)(kc / CK)) * (CKF * COMET_LANES) + lane;
                State st;
                st.x0 = o[0]; st.x1 = o[32]; st.x2 = o[64]; st.t0 = o[96]; st.t1 = o[128]; st.t2 = o[160];
                double h = o[192], h_in = 0.0, bs_in = 0.0, bs_out = 0.0, bd = 0.0;
                State bs = st;
                int ks = ka;
                for (int k = kc;; ++k) {
                    if (k >= ka && k <= kz) {
                        double u0, u1, u2;
                        const double d2 = perp2_exact(st.x0, st.x1, st.x2, wl, u0, u1, u2);
                        if (k == ka || d2 < bd) { bd = d2; ks = k; bs = st; bs_in = h_in; }
                    }
                    if (k > kz || k >= np - 1) break;
                    const double used = adaptive_field_step(st, h, a.hk.h, a.h_min, c, a.F);
                    if (ks == k && k >= ka) bs_out = used;
                    h_in = used;
                }
                const double lo = (ks > 0) ? -bs_in : 0.0, hi = (ks < np - 1) ? bs_out : 0.0;
                D = fine_dca_field(bs, lo, hi, c, a.F, wl);
            } else if (ZG) {
                // the distinct track's rows [u][row] = (x, y, T_x, T_y) (scan_zgroup.cuh); z from the checkpoint at or
                // before ka (one every COMET_ZR_CK rows, scan_zrun.cuh) plus one addition per step
                constexpr int CKZ = 8;
                const int kc = ka & ~(CKZ - 1);
                const int64_t u = s >> zshift;
                const double2* g = reinterpret_cast<const double2*>(a.ub + ((size_t)u * (size_t)a.u_rows + (size_t)ka) * 4);
                const double t2 = a.tw[s], hz = xmul(a.hk.h, t2);
                double z = a.ck[(size_t)chunk * a.n_ck * COMET_LANES + (size_t)(kc / CKZ) * COMET_LANES + lane];
                for (int k = kc; k < ka; ++k) z = xadd(z, hz);
                State cand[3];
#pragma unroll
                for (int j = 0; j < 3; ++j) {                // rows ka, ka + 1, ka + 2 (clamped: read, not used, past kz)
                    const double2* r = g + (size_t)min(j, kz - ka) * 2;
                    const double2 xy = __ldg(r), tt = __ldg(r + 1);
                    cand[j].x0 = xy.x; cand[j].x1 = xy.y; cand[j].t0 = tt.x; cand[j].t1 = tt.y;
                    cand[j].t2 = t2;
                }
                State bs = cand[0];
                int ks = ka;
                double bd = 0.0;
#pragma unroll
                for (int j = 0; j < 3; ++j) {
                    if (ka + j <= kz) {
                        cand[j].x2 = z;
                        double u0, u1, u2;
                        const double d2 = perp2_exact(cand[j].x0, cand[j].x1, z, wl, u0, u1, u2);
                        if (j == 0 || d2 < bd) { bd = d2; ks = ka + j; bs = cand[j]; }
                        z = xadd(z, hz);
                    }
                }
                D = fine_dca(bs, ks, np, a.hk.h, c, wl);
            } else {
                const int kc = ka & ~(CK - 1);
                const double* o = a.ck + ((size_t)chunk * a.n_ck + (size_t)(kc / CK)) * (CKF * COMET_LANES) + lane;
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
                D = fine_dca(bs, ks, np, a.hk.h, c, wl);
            }
            const double e = wire_residual(D, a.rho, __ldg(a.hit_off + i), __ldg(a.hit_off + i + 1), a.lambda,
                                           nullptr, nullptr);
            e2 = xmul(e, e);
        }
        a.bd[pidx] = e2;
        it = __shfl_sync(0xffffffffu, nxt, 0);
    }
}

}  // namespace comet
