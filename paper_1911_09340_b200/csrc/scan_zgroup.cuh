// scan_zgroup.cuh -- seed sets in which runs of ZG consecutive seeds share the transverse start (x, y, p_x, p_y,
// p_z) and differ only in z: every distinct transverse track is stepped once (sm_100a).
//
// In the uniform field (0, 0, B_z) the transverse motion does not depend on z: f(T) = c (T_y, -T_x, 0), T_z is
// constant and x_2' = x_2 + h T_2 (common.cuh, rkn4_step).  Seeds with bit-identical (x_0, x_1, p) therefore go
// through bit-identical (x_0, x_1, T_0, T_1) sequences, stop at the same recorded state, and their z sequences
// differ only by the start value, one addition per step.  The seed grids of the method ("A seed set
// was prepared by combining each component from the grids of the ranges") have z as one of the grid axes, so with z
// as the fastest index a track chunk of 32 seeds holds only 32 / ZG distinct transverse tracks.  SIMT lanes cannot
// skip duplicated work inside a warp, so the work is re-mapped: k_gen_unique (this file) steps the distinct tracks
// (lane = distinct track) and leaves (x_0, x_1, T_0, T_1) of every recorded state in ub[track][row];
// k_scan_zrun (scan_zrun.cuh; lane = seed) works from those rows and adds its own z column (one addition per
// recorded state instead of the 50 operations of the RKN4 step); k_fine_ck<.., ZG = true> (scan_fused.cuh) reads its
// three candidate states from them.  Every number is produced by the same IEEE operations as in the plain
// k_scan_fused (and the definition), so n_pts and RSS are bit-identical.
//
// Which seeds qualify: the caller's promise (comet_scan_rss z_run), else decided on the device (k_zgroup_check: the
// largest power of two ZG <= 32 such that every aligned run of ZG seeds of the launch is uniform); the z-run kernels
// run when ZG >= 8 and the plain kernel otherwise -- without a promise all are launched, the ones that are not
// needed exit at once, so the call stays asynchronous.
#pragma once
#include "scan_fused.cuh"

namespace comet {

// flag <- min(flag, largest power of two dividing every position where the transverse start changes), flag
// preset to 0xffffffff; positions that are multiples of 32 never lower it (32 is the cap).
__global__ void __launch_bounds__(256)
k_zgroup_check(const double* __restrict__ seeds, int64_t stride, int64_t n, unsigned int* __restrict__ flag)
{
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned int cand = 32u;
    if (s > 0 && s < n && (s & 31) != 0) {
        bool same = true;
        const int comp[5] = {0, 1, 3, 4, 5};
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            const long long a = __double_as_longlong(seeds[comp[j] * stride + s]);
            const long long b = __double_as_longlong(seeds[comp[j] * stride + s - 1]);
            same = same && (a == b);
        }
        if (!same) cand = (unsigned int)(s & -s);
    }
    cand = __reduce_min_sync(0xffffffffu, cand);
    if ((threadIdx.x & 31) == 0 && cand < 32u && cand < *(volatile unsigned int*)flag) atomicMin(flag, cand);
}

// One thread per distinct transverse track of the launch (unique u = seeds [u ZG, (u + 1) ZG)), one warp per CTA:
// Algorithm 1 for (x_0, x_1, T_0, T_1), every recorded state to ub [u][row] = (x_0, x_1, T_0, T_1) -- 32 bytes per state,
// the rows of a track contiguous, so that k_scan_zrun reads a sub-block of a track as 8 x 32 bytes and a sample with its
// tangent as one row --, the number of recorded states to np_u.  Rows between the last state and the end of its 64-row
// block repeat it.  A lane's rows are 32 bytes at a stride of a whole track, so the warp records 8 steps in shared memory
// and writes them out together: 256 contiguous bytes per track and flush instead of 32 scattered 32-byte stores per step.
#define COMET_GU_ROWS 8
#define COMET_GU_STRIDE (32 * 4 + 4)       // doubles per staged row (padded against bank conflicts)
template <bool STATS>
__global__ void __launch_bounds__(32) k_gen_unique(const FusedArgs a)
{
    constexpr int GR = COMET_GU_ROWS, RS = COMET_GU_STRIDE;
    constexpr unsigned FULL = 0xffffffffu;
    __shared__ __align__(16) double sm[GR * RS];
    if (a.dyn && a.dyn[2]) return;                          // (the turn loop has stopped)
    const unsigned int zg = zrun_of(a.zrun, a.zg);
    if (zg < COMET_ZG_MIN) return;                          // the plain k_scan_fused serves this launch
    const int zshift = 31 - __clz((int)zg);
    const int lane = threadIdx.x;
    const int64_t ug0 = (int64_t)blockIdx.x * 32;
    const int64_t ug = ug0 + lane;
    const int64_t su = ug << zshift;
    if ((ug0 << zshift) >= a.n_seeds) return;               // (warp-uniform)
    const bool valid = su < a.n_seeds;
    State st;
    double c = 0.0;
    if (valid) {
        c = seed_init(a.seeds, a.stride, su, a.qkb, st);
    } else {
        st.x0 = st.x1 = st.t0 = st.t1 = 0.0;
    }
    st.x2 = 0.0;                                            // z is the sweep kernel's business
    st.t2 = 0.0;
    const bool use_stop = a.r_stop2 > 0.0;
    int32_t np = valid ? a.n_steps + 1 : 1;                 // recorded states (a lane without a track records nothing new)
    bool active = valid;
    // flush of the staged rows k0 .. k0 + GR - 1: lane l writes the pieces p = l, l + 32, ... of 16 bytes; 16 consecutive
    // pieces are the 8 rows of one track (256 contiguous bytes).  Everything but the round is fixed per lane.
    const int f_row = (lane >> 1) & 7, f_half = lane & 1, f_trk = lane >> 4;
    const int64_t n_trk = (a.n_seeds + ((int64_t)1 << zshift) - 1) >> zshift;
    const int n_here = (int)min((int64_t)32, n_trk - ug0);  // tracks of this warp
    double* const f_dst = a.ub + ((size_t)(ug0 + f_trk) * (size_t)a.u_rows + (size_t)f_row) * 4 + f_half * 2;
    const double* const f_src = sm + f_row * RS + f_trk * 4 + f_half * 2;
    const size_t f_step = (size_t)2 * (size_t)a.u_rows * 4;                     // two tracks per pass
    auto flush = [&](int k0) {
        __syncwarp();
        double* d = f_dst + (size_t)k0 * 4;
#pragma unroll
        for (int i = 0; i < GR * 2; ++i) {
            if (2 * i + f_trk < n_here) *reinterpret_cast<double2*>(d + i * f_step) = *reinterpret_cast<const double2*>(f_src + i * 8);
        }
        __syncwarp();
    };
    double* const my = sm + lane * 4;
    auto put = [&](int row) {
        *reinterpret_cast<double2*>(my + row * RS) = make_double2(st.x0, st.x1);
        *reinterpret_cast<double2*>(my + row * RS + 2) = make_double2(st.t0, st.t1);
    };
    // Rows k .. k + GR - 1 per round (row 0 is the seed state).  The chain of dependent operations of a step is the whole
    // cost here (one warp per CTA, about one warp per scheduler), so nothing may sit on it: every lane takes the steps of a
    // round unconditionally -- straight-line code, the tail of one step overlaps the chain of the next -- and stages them;
    // the first state in the target region, if any, is only remembered.  Afterwards a lane that stopped (in this round or
    // before) overwrites the rows after its last state with it: the hold-last padding.
    const int n_rows = a.n_steps + 1;
    int k = 0;                                              // first row of the round
    // A round cannot hold a stop while every lane is farther outside the target region than a round's steps can cover
    // (a step moves the position by at most 1.001 h) and the capacity is not reached: such a round skips the tests.
    const double far_r = sqrt(a.r_stop2) + (GR + 1) * 1.001 * a.hk.h;
    const double far2 = far_r * far_r;
    bool quiet = false;                                     // (warp-uniform) the next round needs no test
    while (true) {
        const State hold = st;                              // (what a finished lane keeps)
        int first = GR;                                     // row of this round at which the lane stops
        if (quiet) {
#pragma unroll
            for (int j = 0; j < GR; ++j) {
                rkn4_step(st, a.hk, c);
                put(j);
            }
        } else {
#pragma unroll
            for (int j = 0; j < GR; ++j) {
                if (k + j > 0) {                            // (row 0: the seed state itself; warp-uniform)
                    rkn4_step(st, a.hk, c);
                    // in_target_region without its early exit: no branch waits for this step's position
                    const double r2 = xadd(xmul(st.x0, st.x0), xmul(st.x1, st.x1));
                    const double rad = xadd(xmul(st.x0, st.t0), xmul(st.x1, st.t1));
                    const bool stop = ((r2 < a.r_stop2) & (rad < 0.0) & use_stop) | (k + j == n_rows - 1);
                    first = (stop & (first == GR)) ? j : first;
                }
                put(j);
            }
        }
        {
            const double r2e = fma(st.x0, st.x0, st.x1 * st.x1);
            const bool lane_quiet = !active || !use_stop || r2e > far2;
            quiet = __all_sync(FULL, lane_quiet) && (k + 2 * GR < n_rows - 1);
        }
        if (!active) {
            st = hold;
            for (int j = 0; j < GR; ++j) put(j);
        } else if (first < GR) {
            // (the capacity counts as a stop at row n_steps: np = n_steps + 1 either way)
            np = k + first + 1;
            active = false;
            const double2 xy = *reinterpret_cast<const double2*>(my + first * RS), tt = *reinterpret_cast<const double2*>(my + first * RS + 2);
            st.x0 = xy.x; st.x1 = xy.y; st.t0 = tt.x; st.t1 = tt.y;
            for (int j = first + 1; j < GR; ++j) put(j);
        }
        flush(k);                                           // (u_rows is a multiple of 64: whole rounds)
        k += GR;
        // go on while a lane is still stepping, then to the end of the 64-row block of the warp's longest track
        if ((!__any_sync(FULL, active) && (k & 63) == 0) || k >= a.u_rows) break;
    }
    if (valid) {
        a.np_u[ug] = np;
        if (STATS && a.stats) atomicAdd(a.stats + ST_UNIQUE, (unsigned long long)(np - 1));
    }
}

}  // namespace comet
