// extrapolate.cuh -- kernel A "track recording" (Algorithm 1) for sm_100a.
//
// One thread per seed, one warp per track chunk of 32 consecutive seeds.  Every step the warp
// writes six fully coalesced 256-byte rows (3 position + 3 tangent components x 32 lanes), so the
// stores run at 100 % sector efficiency -- the paper's AoS layout reached 25 %.
// A lane that has reached the target region keeps writing its LAST recorded position up to the last
// row any lane of its chunk records ("hold-last" padding).  Kernel B can then scan or sample the
// chunk's rows without a per-lane bound: a padded row is at the same distance from any wire as the
// lane's last state, so it never wins the strict "<" of the closest-state search (ties -> lowest k)
// and it keeps the row-to-row displacement bounded by the step length, which the pruned search
// relies on.  Lanes beyond n_seeds in a ragged last chunk hold zeros.
#pragma once
#include "common.cuh"

namespace comet {

__global__ void __launch_bounds__(128)
k_extrapolate(const double* __restrict__ seeds, int64_t stride, int64_t n_seeds, double qkb, StepK hk,
              int32_t n_steps, double r_stop2, double* __restrict__ X, double* __restrict__ T,
              int32_t* __restrict__ n_pts)
{
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const int64_t chunk = s >> 5;
    const int32_t n_rows = track_rows(n_steps);
    if (chunk * COMET_LANES >= n_seeds) return;          // whole warp out of range
    bool active = s < n_seeds;
    State st;
    double c = 0.0;
    if (active) {
        c = seed_init(seeds, stride, s, qkb, st);
    } else {
        st.x0 = st.x1 = st.x2 = 0.0;
        st.t0 = st.t1 = st.t2 = 0.0;
    }
    size_t row = track_row(chunk, n_rows, 0) + lane;
    X[row] = st.x0; X[row + 32] = st.x1; X[row + 64] = st.x2;
    T[row] = st.t0; T[row + 32] = st.t1; T[row + 64] = st.t2;
    int32_t np = n_steps + 1;
    const bool use_stop = r_stop2 > 0.0;
    int32_t k = 1;
    for (; k <= n_steps; ++k) {
        if (!__any_sync(0xffffffffu, active)) break;
        row += 3 * COMET_LANES;
        if (active) {
            rkn4_step(st, hk, c);
            X[row] = st.x0; X[row + 32] = st.x1; X[row + 64] = st.x2;
            T[row] = st.t0; T[row + 32] = st.t1; T[row + 64] = st.t2;
            if (use_stop && in_target_region(st, r_stop2)) { np = k + 1; active = false; }
        } else {
            X[row] = st.x0; X[row + 32] = st.x1; X[row + 64] = st.x2;      // hold-last padding
        }
    }
    // pad the chunk to whole 64-row blocks (rows k .. next multiple of 64; they exist: n_rows % 64 == 0)
    for (; k & (COMET_ROW_PAD - 1); ++k) {
        row += 3 * COMET_LANES;
        X[row] = st.x0; X[row + 32] = st.x1; X[row + 64] = st.x2;
    }
    if (s < n_seeds) n_pts[s] = np;
}

// canonical export [seed][k][6], NaN beyond n_pts (parity tests)
__global__ void k_track_export(const double* __restrict__ X, const double* __restrict__ T,
                               const int32_t* __restrict__ n_pts, int32_t n_steps, int64_t seed_begin,
                               int64_t seed_end, double* __restrict__ out)
{
    const int32_t n_out = n_steps + 1;
    const int64_t total = (seed_end - seed_begin) * (int64_t)n_out;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total;
         i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t s = seed_begin + i / n_out;
        const int32_t k = (int32_t)(i % n_out);
        const size_t row = track_row(s >> 5, track_rows(n_steps), k) + (size_t)(s & 31);
        const bool ok = k < n_pts[s];
        const double nan = __longlong_as_double(0x7ff8000000000000LL);
        double* o = out + (size_t)i * 6;
        o[0] = ok ? X[row] : nan; o[1] = ok ? X[row + 32] : nan; o[2] = ok ? X[row + 64] : nan;
        o[3] = ok ? T[row] : nan; o[4] = ok ? T[row + 32] : nan; o[5] = ok ? T[row + 64] : nan;
    }
}

}  // namespace comet
