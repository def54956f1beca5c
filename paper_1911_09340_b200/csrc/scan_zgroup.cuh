// scan_zgroup.cuh -- seed sets in which runs of ZG consecutive seeds share the transverse start (x, y, p_x, p_y,
// p_z) and differ only in z: every distinct transverse track is stepped once (sm_100a).
//
// In the uniform field (0, 0, B_z) the transverse motion does not depend on z: f(T) = c (T_y, -T_x, 0), T_z is
// constant and x_2' = x_2 + h T_2 (common.cuh, rkn4_step).  Seeds with bit-identical (x_0, x_1, p) therefore go
// through bit-identical (x_0, x_1, T_0, T_1) sequences, stop at the same recorded state, and their z sequences
// differ only by the start value, one addition per step.  The seed grids of the method ("A seed set
// was prepared by combining each component from the grids of the ranges") have z as one of the grid axes, so with z
// as the fastest index a track chunk of 32 seeds holds only 32 / ZG distinct transverse tracks.  SIMT lanes cannot
// skip duplicated work inside a warp, so the work is re-mapped: k_gen_unique steps the distinct tracks (lane =
// distinct track) and leaves (x_0, x_1, T_0, T_1) of every recorded state in a buffer that stays in L2;
// k_scan_fused<.., ZG = true> (lane = seed) copies its tile rows from there, adds its own z column (one addition
// per recorded state instead of the 48 operations of the RKN4 step) and goes on as before.  Every number is
// produced by the same IEEE operations as in the plain k_scan_fused (and the definition), so n_pts, checkpoints, keys
// and RSS are bit-identical.
//
// Which seeds qualify is decided on the device (k_zgroup_check: the largest power of two ZG <= 32 such that every
// aligned run of ZG seeds of the launch is uniform); the ZG kernels run when ZG >= 8 and the plain kernel
// otherwise -- all are launched, the ones that are not needed exit at once, so the call stays asynchronous.
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

// One thread per distinct transverse track of the launch (unique u = seeds [u ZG, (u + 1) ZG)): Algorithm 1 for
// (x_0, x_1, T_0, T_1), every recorded state to ub [u][row] = (x_0, x_1, T_0, T_1) -- 32 bytes per state, the rows of a
// track contiguous, so that k_scan_zrun reads a sub-block of a track as 8 x 32 bytes and a sample with its tangent as one
// row --, the number of recorded states to np_u.  Rows between the last state and the end of its 64-row block repeat it.
template <bool STATS>
__global__ void __launch_bounds__(128) k_gen_unique(const FusedArgs a)
{
    const unsigned int zg = zrun_of(a.zrun, a.zg);
    if (zg < COMET_ZG_MIN) return;                          // the plain k_scan_fused serves this launch
    const int zshift = 31 - __clz((int)zg);
    const int64_t ug = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t su = ug << zshift;
    if (su >= a.n_seeds) return;
    State st;
    const double c = seed_init(a.seeds, a.stride, su, a.qkb, st);
    st.x2 = 0.0;                                            // z is the sweep kernel's business
    st.t2 = 0.0;
    double2* o = reinterpret_cast<double2*>(a.ub + (size_t)ug * (size_t)a.u_rows * 4);
    const bool use_stop = a.r_stop2 > 0.0;
    int32_t np = a.n_steps + 1;
    o[0] = make_double2(st.x0, st.x1); o[1] = make_double2(st.t0, st.t1);
    // The chain of dependent operations of a step is the whole cost here (one warp per CTA, nothing to overlap
    // with), so the stop test must not sit on it: blocks of 4 steps are taken and recorded unconditionally -- rows
    // past the stop are overwritten by the padding below -- and the first state in the target region, if any, ends
    // the track afterwards.
    State last = st;
    int k = 1;
    for (; k + 3 <= a.n_steps; k += 4) {
        int first = 4;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            rkn4_step(st, a.hk, c);
            o[(size_t)(k + j) * 2] = make_double2(st.x0, st.x1); o[(size_t)(k + j) * 2 + 1] = make_double2(st.t0, st.t1);
            // in_target_region without its early exit: no branch waits for this step's position
            const double r2 = xadd(xmul(st.x0, st.x0), xmul(st.x1, st.x1));
            const double rad = xadd(xmul(st.x0, st.t0), xmul(st.x1, st.t1));
            const bool stop = (r2 < a.r_stop2) & (rad < 0.0) & use_stop;
            if (stop & (first == 4)) { first = j; last = st; }
        }
        if (first < 4) { np = k + first + 1; break; }
        last = st;
    }
    if (np == a.n_steps + 1)
        for (; k <= a.n_steps; ++k) {
            rkn4_step(st, a.hk, c);
            o[(size_t)k * 2] = make_double2(st.x0, st.x1); o[(size_t)k * 2 + 1] = make_double2(st.t0, st.t1);
            last = st;
            if (use_stop && in_target_region(st, a.r_stop2)) { np = k + 1; break; }
        }
    // hold-last padding up to the end of the 64-row block (u_rows is a multiple of 64)
    for (int q = np; q < ((np + 63) & ~63); ++q) {
        o[(size_t)q * 2] = make_double2(last.x0, last.x1); o[(size_t)q * 2 + 1] = make_double2(last.t0, last.t1);
    }
    a.np_u[ug] = np;
    if (STATS && a.stats) atomicAdd(a.stats + ST_UNIQUE, (unsigned long long)(np - 1));
}

}  // namespace comet
