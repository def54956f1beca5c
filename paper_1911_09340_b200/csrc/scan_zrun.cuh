// scan_zrun.cuh -- kernels A + B2 for seed sets in z-runs: the closest-state shortlist of every (seed, wire) pair
// straight from the distinct transverse tracks, with a tangent-line bound per (track, sub-block) (sm_100a).
//
// Aligned runs of ZR = 32 / NU consecutive seeds share (x, y, p) and differ only in z (scan_zgroup.cuh), so a
// track chunk of 32 seeds holds NU distinct transverse tracks.  k_gen_unique has stepped them once:
// ub[track][row] = (x, y, T_x, T_y), 32 bytes per recorded state, rows past the last state of a track repeat it up
// to the end of its 64-row block.  A warp owns a chunk from there to its shortlist keys (lane = seed in the
// sweeps, lane = wire in the tests):
//
//   z chain    every seed's own z column, one addition per recorded state (the definition's x_2' = x_2 + h T_2),
//              kept only as a checkpoint every 8th row for k_fine_ck; nothing else of the track is recomputed;
//   staging    per 64-row block the (x, y) rows of the chunk's NU tracks (2 KB for NU = 2) and the tangents of the 8
//              sub-block samples go to the warp's shared memory with cp.async, one block ahead (double buffer), so
//              the L2 latency of ub is off the path;
//   level A    (float) per 64-row block and wire: the distance of ONE sample (row 36) of each distinct track, taken at
//              the centre of the run's z range, against R_i + (z half range) sqrt(1 - w_z^2) + 36 L -- the
//              1-Lipschitz bound of dca.cuh; the wires that pass are compacted into a list;
//   level B    (float) per listed wire, 8-row sub-block and distinct track: the sample (row 4 of the sub-block) WITH ITS
//              TANGENT.  The rows of the sub-block lie within U = 4 h of arc of the sample, and a curve of
//              curvature <= |c| leaves its tangent line by at most |c| U^2 / 2 over that arc, so no row of any seed
//              of the run is closer to the wire than
//                  sqrt( min_{|u| <= U} |a + u b|^2 ) - |c| U^2 / 2 - (z half range) sqrt(1 - w_z^2),
//              a = the sample's offset from the wire and b = its tangent, both projected on the plane
//              perpendicular to the wire.  The minimum of the quadratic is taken in closed form without a
//              division.  A sub-block is opened for a wire only if that bound is within the far radius R_i: about
//              1.2 opened sub-blocks per sub-block that holds a state within R_i, against 2.5 with the one-sample
//              Lipschitz test of k_scan_fused (configs[1]);
//   sweeps     lane = seed: the rows of the opened sub-blocks are read from the staged block (one 16-byte
//              shared-memory load per row, broadcast to the seeds of the run), z = z_0 + k h T_z folded into the
//              wire's constants, 8 FP64 instructions + compare per row, best (d^2, row) merged into the pair key
//              with one atomic min as in k_scan_fused;
//   keys       a warp owns the 32 keys of a (chunk, wire) pair row: the first sweep of a wire stores them, later
//              ones (another block) merge with a fire-and-forget atomic min; a bit per wire in the warp's shared
//              memory remembers which rows exist.  Nothing is written for the wires that never pass level B;
//   finish     only the touched rows are read back: a row with a lane within the far radius becomes an item of
//              k_fine_ck, the others are dropped; the chunk's mask of rows k_fine_ck will fill goes to memory and
//              k_rss_sum adds cutoff^2 for every other wire without reading anything.
//
// Levels A and B only prune, with slack, so they run in SINGLE precision (north_star: "FP32 for the coarse search"): the
// 8 samples of a block per track are converted once per block, the wire's shortlist fields come from a float table
// (k_wire_prep: basis and offsets rounded to nearest, far radius and sqrt(1 - w_z^2) rounded up).  Rounding: a projected
// offset u = x e_x + y e_y + z e_z + c evaluated in float from rounded inputs is off by less than 5 x 2^-24 S,
// S = |x| + |y| + |z| + |c|, a distance by sqrt(2) times that, the tangent's projections by 9 x 2^-24, the closed-form minimum
// by another ~1e-5 cm; every threshold takes 32 x 2^-24 (X + |c1| + |c2|) on top, X >= |x| + |y| + |z| for every state of
// the chunk (the seeds' largest |x_0|_1 + 3.003 n_steps h), and thr^2 a factor 1 + 2e-6.  The sweeps stay in double
// precision: they choose the row, and a wrong choice between non-adjacent rows would not be repaired afterwards.
// Only shortlists are decided here (FMA-form distances, slack 1e-6 cm on every bound): k_fine_ck<ZG> re-decides
// between rows k-1, k, k+1 with the definition's exact operations, so n_pts and RSS are the bit-identical numbers
// of the plain path and of the definition.  A chunk with a lane beyond |c| h <= 0.05 opens everything.
#pragma once
#include "scan_fused.cuh"

namespace comet {

#ifndef COMET_ZR_WARPS
#define COMET_ZR_WARPS 4
#endif
#ifndef COMET_ZR_WCAP
#define COMET_ZR_WCAP 128          // wires whose constants the CTA's shared-memory table holds (the others: L1/L2)
#endif
#define COMET_ZR_CK 8              // rows between z checkpoints
#define COMET_ZR_LCAP 1024         // (chunk, wire) items collected per reservation in the finish
#ifndef COMET_ZR_MINB
#define COMET_ZR_MINB 5
#endif
#define COMET_ZR_NF (COMET_FUSED_WFIELDS + 1)
// doubles of shared memory per warp: two staged blocks of (64 rows + 8 sample tangents) x NU tracks x 2, the pass
// list (64 shorts); the item list of the finish (LCAP shorts = 256 doubles) reuses the staged blocks
// + the single-precision samples of the staged block: [8 sub-blocks][NU tracks][x, y, z, T_x, T_y, -, -, -] floats
#define COMET_ZR_WSM(NU) (2 * (64 + 8) * (NU) * 2 + 16 + 8 * (NU) * 4)
#define COMET_ZR_FF 11             // fields of the single-precision wire table (k_wire_prep)
// + the touched-wire mask: one bit per fired wire, rounded up to whole 16 bytes
#define COMET_ZR_MWD(W) ((((W) + 31) / 32 + 3) / 4 * 2)
#define COMET_ZR_SMEM_OF(NU, W, WPC, WCAP_) ((COMET_ZR_NF * (WCAP_) + (WPC) * (COMET_ZR_WSM(NU) + COMET_ZR_MWD(W))) * (int)sizeof(double) + \
                                            COMET_ZR_FF * (WCAP_) * (int)sizeof(float))
// BIGW (more fired wires than the table holds): CTAs of ONE warp and no table at all -- every wire constant comes through L1,
// 20 CTAs per SM, no warp waits for the slowest of its CTA (measured on configs[4], 972 wires: 0.973 -> 0.919 ms; with a table
// that serves every wire the four-warp CTA is the faster one: 0.340 against 0.356 ms on configs[1])
#define COMET_ZR_WPC(BIGW) ((BIGW) ? 1 : COMET_ZR_WARPS)
#define COMET_ZR_TCAP(BIGW) ((BIGW) ? 0 : COMET_ZR_WCAP)
#define COMET_ZR_SMEM(NU, W, BIGW) COMET_ZR_SMEM_OF(NU, W, COMET_ZR_WPC(BIGW), COMET_ZR_TCAP(BIGW))
// relative rounding slack of the single-precision tests: 32 x 2^-24 per unit of (|x| + |y| + |z| + |c1| + |c2|)
#define COMET_ZR_FSLACK 1.9073486e-6f
#define COMET_ZR_MARGIN 1e-6       // cm, added to every pruning threshold (FMA rounding is ~1e-13)

template <bool BIGW>
__device__ __forceinline__ double zr_const(const double* wtab, const double* __restrict__ wt, int W, int f, int i)
{
    if (!BIGW) return wtab[f * COMET_ZR_WCAP + i];
    return __ldg(wt + (size_t)(6 + f) * W + i);
}
template <bool BIGW>
__device__ __forceinline__ void zr_evalc(EvalC& w, const double* wtab, const double* __restrict__ wt, int W, int i)
{
    w.e1x = zr_const<BIGW>(wtab, wt, W, 0, i); w.e1y = zr_const<BIGW>(wtab, wt, W, 1, i); w.e1z = zr_const<BIGW>(wtab, wt, W, 2, i);
    w.c1 = zr_const<BIGW>(wtab, wt, W, 3, i);
    w.e2x = zr_const<BIGW>(wtab, wt, W, 4, i); w.e2y = zr_const<BIGW>(wtab, wt, W, 5, i); w.e2z = zr_const<BIGW>(wtab, wt, W, 6, i);
    w.c2 = zr_const<BIGW>(wtab, wt, W, 7, i);
}
template <bool BIGW>
__device__ __forceinline__ float zr_constf(const float* wtabf, const float* __restrict__ wtf, int W, int f, int i)
{
    if (!BIGW) return wtabf[f * COMET_ZR_WCAP + i];
    return __ldg(wtf + (size_t)f * W + i);
}
template <bool BIGW>
__device__ __forceinline__ double zr_slope(const double* wtab, const double* __restrict__ wt, int W, int i)
{
    if (!BIGW) return wtab[COMET_FUSED_WFIELDS * COMET_ZR_WCAP + i];
    return wire_slope(__ldg(wt + (size_t)8 * W + i), __ldg(wt + (size_t)12 * W + i));
}

template <bool STATS, int NU, bool BIGW>
__global__ void __launch_bounds__(32 * COMET_ZR_WPC(BIGW), BIGW ? 20 : COMET_ZR_MINB) k_scan_zrun(const FusedArgs a)
{
    static_assert(NU == 1 || NU == 2 || NU == 4, "runs of 32, 16 or 8 seeds");
    constexpr int ZR = 32 / NU, ZSH = (NU == 1 ? 5 : (NU == 2 ? 4 : 3));
    constexpr int WCAP = COMET_ZR_TCAP(BIGW), NF = COMET_ZR_NF, WPC = COMET_ZR_WPC(BIGW);
    constexpr int BLK = 64, SUB = 8, NSUB = BLK / SUB, SROW = 36;
    constexpr int CK = COMET_ZR_CK, LCAP = COMET_ZR_LCAP;
    constexpr int BUFD = (BLK + NSUB) * NU * 2;             // doubles per staged block: rows [64][NU][x, y], tangents [8][NU][T_x, T_y]
    constexpr unsigned FULL = 0xffffffffu;
    static_assert(LCAP * (int)sizeof(unsigned short) <= 2 * BUFD * (int)sizeof(double) || NU == 1, "item list fits the staged blocks");
    if (a.dyn && a.dyn[2]) return;                          // (the turn loop has stopped)
    if (zrun_of(a.zrun, a.zg) != (unsigned)ZR) return;      // another variant serves this launch
    extern __shared__ __align__(16) double zsm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* wtab = zsm;                                     // [NF][WCAP]
    const int W = a.W;
    const int MW = (W + 31) / 32;                           // words of the touched-wire mask
    double* stg = zsm + NF * WCAP + warp * (COMET_ZR_WSM(NU) + COMET_ZR_MWD(W));   // two staged blocks
    unsigned short* plist = reinterpret_cast<unsigned short*>(stg + 2 * BUFD);     // [64] wires that passed level A
    float* sampf = reinterpret_cast<float*>(stg + 2 * BUFD + 16);                  // [8][NU][8] samples of the current block
    unsigned* tmask = reinterpret_cast<unsigned*>(stg + 2 * BUFD + 16 + NSUB * NU * 4);   // [MW] bit i: the key row of wire i exists
    float* wtabf = reinterpret_cast<float*>(zsm + NF * WCAP + WPC * (COMET_ZR_WSM(NU) + COMET_ZR_MWD(W)));   // [FF][WCAP]
    unsigned short* lst = reinterpret_cast<unsigned short*>(stg);                  // finish: [<= LCAP] items
    constexpr int LCAPW = (NU == 1) ? (2 * BUFD * 4) : LCAP;                       // shorts the staged blocks hold
    for (int v = threadIdx.x; v < COMET_FUSED_WFIELDS * WCAP; v += 32 * WPC) {
        const int f = v / WCAP, i = v - f * WCAP;
        wtab[v] = (i < W) ? __ldg(a.wt + (size_t)(6 + f) * W + i) : -1.0;
    }
    for (int i = threadIdx.x; i < WCAP; i += 32 * WPC)
        wtab[COMET_FUSED_WFIELDS * WCAP + i] = (i < W) ? wire_slope(__ldg(a.wt + (size_t)8 * W + i), __ldg(a.wt + (size_t)12 * W + i)) : 0.0;
    for (int v = threadIdx.x; v < COMET_ZR_FF * WCAP; v += 32 * WPC) {
        const int f = v / WCAP, i = v - f * WCAP;
        wtabf[v] = (i < W) ? __ldg(a.wtf + (size_t)f * W + i) : -1.f;
    }
    __syncthreads();
    const int64_t chunk = (int64_t)blockIdx.x * WPC + warp;
    if (chunk * COMET_LANES >= a.n_seeds) return;
    const int64_t s = chunk * COMET_LANES + lane;
    const bool valid = s < a.n_seeds;
    const double h = a.hk.h;
    const double INF = 1.7976931348623157e308;
    const double L = COMET_LIP * h;
    const double U = (SUB / 2) * h * 1.000001;              // arc between a sub-block's sample and its farthest row
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
    const bool any_nolip = __any_sync(FULL, valid && !lip_ok);
    const int tl = lane >> ZSH;                             // the seed's distinct track within the chunk
    const int64_t ug0 = (chunk * COMET_LANES) >> ZSH;       // the chunk's first distinct track
    const int32_t np = valid ? __ldg(a.np_u + ug0 + tl) : 0;       // recorded states of the seed = of its transverse track
    const double hz = xmul(h, st.t2);                       // x_2' = x_2 + h T_2, T_2 constant
    const double z0 = st.x2;
    // largest |c| of the chunk, rounded up: how far a track leaves its tangent line over the arc U
    const float cf = valid ? __double2float_ru(fabs(c)) : 0.f;
    const double cmax = (double)__uint_as_float(__reduce_max_sync(FULL, __float_as_uint(cf)));
    const double dev = cmax * U * U * 0.5000005 + 1e-7;
    // per run: centre and half range of the seeds' z_0 (an invalid lane of a ragged last run stands aside)
    double zlo, zhi;
    {
        const double zfirst = __shfl_sync(FULL, z0, tl << ZSH);
        const double zv = valid ? z0 : zfirst;
        zlo = zv; zhi = zv;
#pragma unroll
        for (int o = 1; o < ZR; o <<= 1) {
            zlo = fmin(zlo, __shfl_xor_sync(FULL, zlo, o));
            zhi = fmax(zhi, __shfl_xor_sync(FULL, zhi, o));
        }
    }
    const double zc0 = 0.5 * (zlo + zhi);
    const double zh = 0.5 * (zhi - zlo) * 1.000001 + 1e-9; // |z_k(seed) - (zc0 + k hz)| <= zh for every seed of the run
    double zh_t[NU], tz_t[NU], zc_t[NU], hz_t[NU];
    int32_t np_t[NU];
    int32_t npmax = 0;
#pragma unroll
    for (int t = 0; t < NU; ++t) {
        zh_t[t] = __shfl_sync(FULL, zh, t << ZSH);
        tz_t[t] = __shfl_sync(FULL, st.t2, t << ZSH);
        zc_t[t] = __shfl_sync(FULL, zc0, t << ZSH);
        hz_t[t] = __shfl_sync(FULL, hz, t << ZSH);
        np_t[t] = __shfl_sync(FULL, np, t << ZSH);
        npmax = max(npmax, np_t[t]);
    }
    int32_t npmin = npmax;
#pragma unroll
    for (int t = 0; t < NU; ++t)
        if (np_t[t] > 0) npmin = min(npmin, np_t[t]);

    // Levels A and B are pruning tests with slack: they run in single precision (twice the rate of the FP64 pipe, half the
    // registers).  Every input is rounded to float and every operation rounds again: a projected offset
    // u = x e_x + y e_y + z e_z + c is off by less than 8 x 2^-24 (|x| + |y| + |z| + |c|), a distance by less than twice
    // that; the thresholds take COMET_ZR_FSLACK x (X + |c1| + |c2|) on top, X >= |x| + |y| + |z| of every state of the chunk.
    float zh_f[NU], tz_f[NU];
#pragma unroll
    for (int t = 0; t < NU; ++t) {
        zh_f[t] = __double2float_ru(zh_t[t]);
        tz_f[t] = (float)tz_t[t];
    }
    float xsum_f;
    {
        const float xs = valid ? __double2float_ru(fabs(st.x0) + fabs(st.x1) + fabs(st.x2)) : 0.f;
        xsum_f = __uint_as_float(__reduce_max_sync(FULL, __float_as_uint(xs))) + __double2float_ru(3.003 * (double)a.n_steps * h);
    }
    const float dev_f = __double2float_ru(dev + COMET_ZR_MARGIN), lipA_f = __double2float_ru(SROW * L + COMET_ZR_MARGIN);
    const float U_f = __double2float_ru(U * 1.000001);
    // the sample this lane converts per block: sub-block lane / NU of track lane % NU
    const int tq = lane & (NU - 1);
    const double zc_q = __shfl_sync(FULL, zc0, tq << ZSH), hz_q = __shfl_sync(FULL, hz, tq << ZSH);
    const int32_t np_q = __shfl_sync(FULL, np, tq << ZSH);

    // staging: lane l copies the pieces p = l, l + 32, ... of a block: always of track l % NU
    const int ts = lane & (NU - 1);
    const int32_t np_s = __shfl_sync(FULL, np, ts << ZSH);
    const double* const ub_s = a.ub + (size_t)(ug0 + ts) * (size_t)a.u_rows * 4;
    const unsigned stg_sh = (unsigned)__cvta_generic_to_shared(stg);
    auto stage = [&](int r0s, int buf) {
        if (r0s < npmax && np_s > r0s) {                    // (rows up to the end of a track's last 64-row block exist: hold-last)
            const double* src = ub_s + (size_t)r0s * 4;
            const unsigned dst = stg_sh + (unsigned)(buf * BUFD * 8);
#pragma unroll
            for (int m = 0; m < 2 * NU; ++m) {
                const int row = (lane >> (5 - ZSH)) + m * ZR;         // p / NU with p = lane + 32 m
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + (unsigned)((row * NU + ts) * 16)), "l"(src + (size_t)row * 4));
            }
            if (lane < NSUB * NU) {
                const int j = lane >> (5 - ZSH);
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + (unsigned)((BLK * NU + j * NU + ts) * 16)),
                             "l"(src + (size_t)(j * SUB + SUB / 2) * 4 + 2));
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    stage(0, 0);

    // pair keys of this chunk: no row exists yet
    unsigned long long* const keys = reinterpret_cast<unsigned long long*>(a.bd);
    for (int w = lane; w < MW; w += 32) tmask[w] = 0u;
    // the seed's z column (Algorithm 1 for x_2), a checkpoint every CK rows
    {
        double* ckc = a.ck + (size_t)chunk * a.n_ck * COMET_LANES + lane;
        double z = z0;
        if (np > 0) ckc[0] = z;
        int k0 = 1;
        for (; k0 + CK <= npmin; k0 += CK) {                // rows every seed of the chunk has
#pragma unroll
            for (int q = 0; q < CK; ++q) z = xadd(z, hz);
            ckc[(size_t)((k0 + CK - 1) / CK) * COMET_LANES] = z;
        }
        for (; k0 < npmax; k0 += CK) {
#pragma unroll
            for (int q = 0; q < CK; ++q) {
                const int k = k0 + q;
                if (k < np) z = xadd(z, hz);
                if (q == CK - 1 && k < np) ckc[(size_t)(k / CK) * COMET_LANES] = z;
            }
        }
    }
    if (valid) { a.n_pts[s] = np; a.cw[s] = c; a.tw[s] = st.t2; }

    unsigned long long st_cnt[ST_N];
    if (STATS) {
#pragma unroll
        for (int j = 0; j < ST_N; ++j) st_cnt[j] = 0;
        if (valid) st_cnt[ST_PAIRS] = (unsigned long long)W;
    }
    const int n_rounds = (W + 31) / 32;
    int buf = 0;
    for (int r0 = 0; r0 < npmax; r0 += BLK, buf ^= 1) {
        __syncwarp();                                       // everyone is done with the block staged two blocks ago
        stage(r0 + BLK, buf ^ 1);
        asm volatile("cp.async.wait_group 1;" ::: "memory");
        __syncwarp();
        const double* rows = stg + buf * BUFD;              // [64][NU][x, y]
        const double* tang = rows + BLK * NU * 2;           // [8][NU][T_x, T_y]
        const bool tail = r0 + BLK > npmin;                 // some track of the chunk ends in this block
        const double r0d = (double)r0;
        const double zb = fma(r0d, hz, z0);                 // the seed's z at row r0 (to rounding: shortlist only)
        // the block's 8 samples per track (row 4 of every sub-block) in single precision: position at the run's centre in z
        // (a sample past the track's last state repeats it) and tangent
        if (lane < NSUB * NU) {
            const int j = lane >> (5 - ZSH);
            const int kr = j * SUB + SUB / 2;
            const double2 xy = *reinterpret_cast<const double2*>(rows + (kr * NU + tq) * 2);
            const double2 tt = *reinterpret_cast<const double2*>(tang + (j * NU + tq) * 2);
            const double z = fma((double)(r0 + (tail ? min(kr, np_q - 1 - r0) : kr)), hz_q, zc_q);
            float4 f0;
            f0.x = (float)xy.x; f0.y = (float)xy.y; f0.z = (float)z; f0.w = (float)tt.x;
            *reinterpret_cast<float4*>(sampf + (j * NU + tq) * 8) = f0;
            sampf[(j * NU + tq) * 8 + 4] = (float)tt.y;
        }
        __syncwarp();
        int cnt = 0;
        auto level_b = [&](const unsigned short* list, int n) {
            // ---- level B (lane = listed wire): tangent-line bound per (distinct track, sub-block) ------------
            const int i = lane < n ? (int)list[lane] : -1;
            unsigned m8 = 0u;
            if (i >= 0) {
                const float e1x = zr_constf<BIGW>(wtabf, a.wtf, W, 0, i), e1y = zr_constf<BIGW>(wtabf, a.wtf, W, 1, i);
                const float e1z = zr_constf<BIGW>(wtabf, a.wtf, W, 2, i), c1 = zr_constf<BIGW>(wtabf, a.wtf, W, 3, i);
                const float e2x = zr_constf<BIGW>(wtabf, a.wtf, W, 4, i), e2y = zr_constf<BIGW>(wtabf, a.wtf, W, 5, i);
                const float e2z = zr_constf<BIGW>(wtabf, a.wtf, W, 6, i), c2 = zr_constf<BIGW>(wtabf, a.wtf, W, 7, i);
                const float cap = zr_constf<BIGW>(wtabf, a.wtf, W, 8, i), swz = zr_constf<BIGW>(wtabf, a.wtf, W, 9, i);
                const float slack = COMET_ZR_FSLACK * (xsum_f + zr_constf<BIGW>(wtabf, a.wtf, W, 10, i));
#pragma unroll
                for (int t = 0; t < NU; ++t) {
                    if (np_t[t] <= r0) continue;
                    const float thr = fmaf(zh_f[t], swz, cap) + dev_f + slack;
                    const float thr2 = thr * thr * 1.000002f;
                    const float bz1 = tz_f[t] * e1z, bz2 = tz_f[t] * e2z;
#pragma unroll
                    for (int j = 0; j < NSUB; ++j) {
                        if (np_t[t] <= r0 + j * SUB) break;          // the track has no row in this sub-block
                        const float4 p = *reinterpret_cast<const float4*>(sampf + (j * NU + t) * 8);   // x, y, z, T_x
                        const float ty = sampf[(j * NU + t) * 8 + 4];
                        const float a1 = fmaf(p.x, e1x, fmaf(p.y, e1y, fmaf(p.z, e1z, c1)));
                        const float a2 = fmaf(p.x, e2x, fmaf(p.y, e2y, fmaf(p.z, e2z, c2)));
                        const float b1 = fmaf(p.w, e1x, fmaf(ty, e1y, bz1));
                        const float b2 = fmaf(p.w, e2x, fmaf(ty, e2y, bz2));
                        const float aa = fmaf(a1, a1, a2 * a2), bb = fmaf(b1, b1, b2 * b2);
                        const float ab = fabsf(fmaf(a1, b1, a2 * b2));
                        // min over |u| <= U of |a + u b|^2 = aa - sv (2 ab - sv) / bb with sv = min(ab, U bb)
                        const float ubb = U_f * bb;
                        const float sv = ab < ubb ? ab : ubb;
                        if (fmaf(aa - thr2, bb, -(sv * fmaf(2.f, ab, -sv))) <= 0.f) m8 |= 1u << j;
                    }
                    if (STATS) st_cnt[ST_SAMPLES_B] += NSUB;
                }
                if (any_nolip) m8 = (1u << NSUB) - 1u;
            }
            unsigned any = __ballot_sync(FULL, m8 != 0u);
            while (any) {
                const int wl = __ffs(any) - 1;
                any &= any - 1;
                unsigned msub = __shfl_sync(FULL, m8, wl);
                const int iw = __shfl_sync(FULL, i, wl);
                // ---- wire iw, lane = seed: sweep the opened sub-blocks row by row ------------------------------
                EvalC w;
                zr_evalc<BIGW>(w, wtab, a.wt, W, iw);      // broadcast
                // u_c = x e_cx + y e_cy + (z e_cz + c_c) with z = zb + kr hz: the bracket is A_c + kr D_c
                const double A1 = fma(zb, w.e1z, w.c1), A2 = fma(zb, w.e2z, w.c2), D1 = hz * w.e1z, D2 = hz * w.e2z;
                double best = INF;
                int bk = -1;
                while (msub) {
                    const int j = __ffs(msub) - 1;
                    msub &= msub - 1;
                    const int k0 = r0 + j * SUB;
                    const double kd = (double)(j * SUB);
                    const double A1j = fma(kd, D1, A1), A2j = fma(kd, D2, A2);
                    const double* pr = rows + ((j * SUB) * NU + tl) * 2;
                    if (STATS) { st_cnt[ST_ROWS_EXEC] += SUB; if (np > k0) st_cnt[ST_ROWS_NEEDED] += min(SUB, np - k0); }
                    if (!tail) {
#pragma unroll
                        for (int kk = 0; kk < SUB; ++kk) {
                            const double2 xy = *reinterpret_cast<const double2*>(pr + kk * NU * 2);
                            const double u1 = fma(xy.x, w.e1x, fma(xy.y, w.e1y, fma((double)kk, D1, A1j)));
                            const double u2 = fma(xy.x, w.e2x, fma(xy.y, w.e2y, fma((double)kk, D2, A2j)));
                            const double d2 = fma(u1, u1, u2 * u2);
                            if (d2 < best) { best = d2; bk = k0 + kk; }
                        }
                    } else {
                        // the block in which a track of the chunk ends: rows past the seed's last state stay out
                        const int nr = np - k0;
#pragma unroll
                        for (int kk = 0; kk < SUB; ++kk) {
                            const double2 xy = *reinterpret_cast<const double2*>(pr + kk * NU * 2);
                            const double u1 = fma(xy.x, w.e1x, fma(xy.y, w.e1y, fma((double)kk, D1, A1j)));
                            const double u2 = fma(xy.x, w.e2x, fma(xy.y, w.e2y, fma((double)kk, D2, A2j)));
                            const double d2 = fma(u1, u1, u2 * u2);
                            if (kk < nr && d2 < best) { best = d2; bk = k0 + kk; }
                        }
                    }
                }
                // the row's first sweep stores the keys, later ones merge (the warp owns the row)
                const unsigned tw_ = tmask[iw >> 5];
                if (!((tw_ >> (iw & 31)) & 1u)) {
                    keys[(size_t)iw * a.SP + s] = bk >= 0 ? pack_key(best, bk) : COMET_KEY_NONE;
                    if (STATS) st_cnt[ST_TOUCHED] += 1;
                    __syncwarp();
                    if (lane == 0) tmask[iw >> 5] = tw_ | (1u << (iw & 31));
                    __syncwarp();
                } else if (bk >= 0) {
                    atomicMin(keys + (size_t)iw * a.SP + s, pack_key(best, bk));
                }
            }
        };
        // ---- level A (lane = wire): one sample per distinct track and block ----------------------------------
        constexpr int JA = SROW / SUB;                        // the sample of level A is sub-block 4's (row 36)
        static_assert(JA * SUB + SUB / 2 == SROW, "level A takes a sample level B has");
        for (int r = 0; r < n_rounds; ++r) {
            const int i = r * 32 + lane;
            const int ii = min(i, W - 1);
            const float e1x = zr_constf<BIGW>(wtabf, a.wtf, W, 0, ii), e1y = zr_constf<BIGW>(wtabf, a.wtf, W, 1, ii);
            const float e1z = zr_constf<BIGW>(wtabf, a.wtf, W, 2, ii), c1 = zr_constf<BIGW>(wtabf, a.wtf, W, 3, ii);
            const float e2x = zr_constf<BIGW>(wtabf, a.wtf, W, 4, ii), e2y = zr_constf<BIGW>(wtabf, a.wtf, W, 5, ii);
            const float e2z = zr_constf<BIGW>(wtabf, a.wtf, W, 6, ii), c2 = zr_constf<BIGW>(wtabf, a.wtf, W, 7, ii);
            const float cap = (i < W) ? zr_constf<BIGW>(wtabf, a.wtf, W, 8, ii) : -1.f;    // far radius; < 0: no entries
            const float swz = zr_constf<BIGW>(wtabf, a.wtf, W, 9, ii);
            const float slack = COMET_ZR_FSLACK * (xsum_f + zr_constf<BIGW>(wtabf, a.wtf, W, 10, ii));
            bool pass = false;
#pragma unroll
            for (int t = 0; t < NU; ++t) {
                if (np_t[t] <= r0) continue;
                const float4 p = *reinterpret_cast<const float4*>(sampf + (JA * NU + t) * 8);
                const float thr = fmaf(zh_f[t], swz, cap) + lipA_f + slack;
                const float u1 = fmaf(p.x, e1x, fmaf(p.y, e1y, fmaf(p.z, e1z, c1)));
                const float u2 = fmaf(p.x, e2x, fmaf(p.y, e2y, fmaf(p.z, e2z, c2)));
                pass = pass || (fmaf(u1, u1, u2 * u2) <= thr * thr * 1.000002f);
                if (STATS && cap >= 0.f) st_cnt[ST_SAMPLES] += 1;
            }
            if (any_nolip) pass = true;
            if (cap < 0.f) pass = false;
            const unsigned pm = __ballot_sync(FULL, pass);
            if (pass) plist[cnt + __popc(pm & ((1u << lane) - 1u))] = (unsigned short)i;
            cnt += __popc(pm);
            __syncwarp();
            if (cnt >= 32) {
                cnt -= 32;
                level_b(plist + cnt, 32);
                __syncwarp();
            }
        }
        if (cnt) level_b(plist, cnt);
    }
    asm volatile("cp.async.wait_all;" ::: "memory");
    __syncwarp();
    // ---- finish: the touched rows are read back; a row with a near lane is an item of k_fine_ck ---------
    constexpr int FB = 8;
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
    for (int wd = 0; wd < MW; ++wd) {
        const unsigned bits = tmask[wd];
        unsigned keep = bits;                               // rows k_fine_ck will fill
        const int nt = __popc(bits);
        __syncwarp();
        if ((bits >> lane) & 1u) plist[__popc(bits & ((1u << lane) - 1u))] = (unsigned short)(wd * 32 + lane);
        __syncwarp();
        for (int b0 = 0; b0 < nt; b0 += FB) {
            unsigned long long kv[FB];
            double cap2[FB];
            int iw[FB];
#pragma unroll
            for (int j = 0; j < FB; ++j) {
                iw[j] = (int)plist[min(b0 + j, nt - 1)];
                kv[j] = __ldcg(keys + (size_t)iw[j] * a.SP + s);
                const double cap = zr_const<BIGW>(wtab, a.wt, W, 8, iw[j]);
                cap2[j] = cap * cap;
            }
#pragma unroll
            for (int j = 0; j < FB; ++j) {
                if (b0 + j < nt) {
                    const bool found = kv[j] != COMET_KEY_NONE;
                    // key_d2 <= d^2 of the closest recorded state: "far" is decided on the safe side
                    const bool near = valid && found && (key_d2(kv[j]) <= cap2[j] || !lip_ok);
                    if (STATS && near) st_cnt[ST_FINE_NEEDED] += 1;
                    if (__any_sync(FULL, near)) {
                        if (STATS) st_cnt[ST_FINE_EXEC] += 1;
                        if (!near && found) keys[(size_t)iw[j] * a.SP + s] = COMET_KEY_NONE;
                        if (lane == 0) lst[cnt] = (unsigned short)iw[j];
                        if (++cnt == LCAPW) flush();
                    } else {
                        keep &= ~(1u << (iw[j] & 31));      // every lane is far: cutoff^2, nothing to store
                    }
                }
            }
        }
        if (lane == 0) a.tm[(size_t)chunk * MW + wd] = keep;
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
