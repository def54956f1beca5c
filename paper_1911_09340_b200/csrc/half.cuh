// half.cuh -- the half-track scheme around the scan (readings R38-R42), sm_100a.
//
// "a turn partition was split into two half tracks whose seeds are at the CDC entrance and exit sides [...]
// forward direction from the entrance and the backward direction from the exit by flipping the charge and
// momentum.  The hits of the event were also grouped into two sets for each half track." (:230)
// "the seeds which have any missing layer without the hits were excluded.  The complete sets of classified hits
// were formed by combinatorially merging two half sets" (:236).
// The scans themselves are the kernels of comet_scan_stage (a half track ends at the apex: the target region
// of R3 with r_stop beyond the chamber, R42); this file holds the integer/byte work around them: the hit
// grouping about the apex line of the Hough circle (one fp64 decision per wire, IEEE operation by operation),
// the momentum flip, the layer veto (a 64-bit layer mask per seed) and the merge (scatter + count per pair).
#pragma once
#include "common.cuh"

namespace comet {

// R39.  One thread per fired wire: d = s (cx m_y - cy m_x) / R; entrance half iff d > -overlap, exit half
// iff d <= overlap.  in_* are the memberships, rm_* (optional) their complements for k_remove_hits.
__global__ void __launch_bounds__(256)
k_half_masks(const double* __restrict__ wire_a, const double* __restrict__ wire_b, int32_t n_wires,
             const int32_t* __restrict__ fired_wire, const int32_t* __restrict__ hit_off, int32_t W,
             const double* __restrict__ circle, double overlap,
             uint8_t* __restrict__ in_e, uint8_t* __restrict__ in_x, uint8_t* __restrict__ rm_e, uint8_t* __restrict__ rm_x)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= W) return;
    const double R = circle[0], cx = circle[1], cy = circle[2], ex = circle[3], ey = circle[4];
    const double s = xsub(xmul(cx, ey), xmul(cy, ex)) > 0.0 ? 1.0 : -1.0;
    const int wi = fired_wire[i];
    const double mx = xmul(xadd(wire_a[wi], wire_b[wi]), 0.5);
    const double my = xmul(xadd(wire_a[n_wires + wi], wire_b[n_wires + wi]), 0.5);
    const double d = s * xdiv(xsub(xmul(cx, my), xmul(cy, mx)), R);       // s = +-1: exact
    const uint8_t e = d > -overlap ? 1 : 0, x = d <= overlap ? 1 : 0;
    for (int j = hit_off[i]; j < hit_off[i + 1]; ++j) {
        if (in_e) { in_e[j] = e; in_x[j] = x; }
        if (rm_e) { rm_e[j] = 1 - e; rm_x[j] = 1 - x; }
    }
}

// R38: (x, p) -> (x, -p).  SoA [6][stride] seeds (aos == 0) or [n][6] rows (aos == 1).
__global__ void __launch_bounds__(256)
k_flip_seeds(const double* in, int64_t in_stride, int64_t n, double* out, int64_t out_stride,
             int aos)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 6 * n) return;
    if (aos) {
        out[i] = (i % 6) >= 3 ? -in[i] : in[i];
    } else {
        const int64_t c = i / n, s = i - c * n;
        const double v = in[c * in_stride + s];
        out[c * out_stride + s] = c >= 3 ? -v : v;
    }
}

__global__ void __launch_bounds__(256) k_negate(double* __restrict__ v, int32_t n)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) v[i] = -v[i];
}

// R40.  One warp per seed: OR of (1 << layer) over the wires with a classified entry; kept iff the mask is a run
// of ones from bit 0 of length >= min_layers.  Layers must lie in [0, 64).
__global__ void __launch_bounds__(256)
k_layer_veto(const uint8_t* __restrict__ cls, int32_t n_sel, int32_t H, const int32_t* __restrict__ fired_wire,
             const int32_t* __restrict__ hit_off, int32_t W, const int32_t* __restrict__ wire_layer, int32_t min_layers,
             uint8_t* __restrict__ ok)
{
    const int a = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (a >= n_sel) return;
    const uint8_t* row = cls + (size_t)a * H;
    unsigned long long mask = 0;
    for (int i = lane; i < W; i += 32) {
        int any = 0;
        for (int j = hit_off[i]; j < hit_off[i + 1]; ++j) any |= row[j];
        if (any) mask |= 1ull << (wire_layer[fired_wire[i]] & 63);
    }
    for (int o = 16; o > 0; o >>= 1) mask |= __shfl_xor_sync(0xffffffffu, mask, o);
    if (lane == 0) ok[a] = (mask != 0 && (mask & (mask + 1)) == 0 && __popcll(mask) >= min_layers) ? 1 : 0;
}

// R41.  CTA (b, a): the complete set of entrance-side seed a and exit-side seed b.
__global__ void __launch_bounds__(256)
k_merge_half(const uint8_t* __restrict__ cls_e, const int32_t* __restrict__ orig_e, const uint8_t* __restrict__ ok_e,
             int32_t He, const uint8_t* __restrict__ cls_x, const int32_t* __restrict__ orig_x,
             const uint8_t* __restrict__ ok_x, int32_t Hx, int32_t H,
             uint8_t* __restrict__ valid, uint8_t* __restrict__ cls, int32_t* __restrict__ n_cls)
{
    __shared__ int s_n[8];
    const int b = blockIdx.x, a = blockIdx.y, Kx = gridDim.x, t = threadIdx.x;
    uint8_t* row = cls + ((size_t)a * Kx + b) * H;
    const bool v = ok_e[a] && ok_x[b];
    for (int j = t; j < H; j += 256) row[j] = 0;
    __syncthreads();
    if (v) {
        for (int j = t; j < He; j += 256)
            if (cls_e[(size_t)a * He + j]) row[orig_e[j]] = 1;
        for (int j = t; j < Hx; j += 256)
            if (cls_x[(size_t)b * Hx + j]) row[orig_x[j]] = 1;
    }
    __syncthreads();
    int c = 0;
    for (int j = t; j < H; j += 256) c += row[j];
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if ((t & 31) == 0) s_n[t >> 5] = c;
    __syncthreads();
    if (t == 0) {
        int n = 0;
        for (int k = 0; k < 8; ++k) n += s_n[k];
        n_cls[a * Kx + b] = n;
        valid[a * Kx + b] = v ? 1 : 0;
    }
}

// R43.  One CTA: the valid pair with the most classified entries (ties -> the lowest a Kx + b) by a packed-key
// maximum ((n_cls + 1) in the high word, inverted flat index in the low word; 0 = no valid pair); its complete
// set goes to cls_best [H] (zeros without a pair), its two seeds, (a, b) and its size to the turn's outputs.
// pick [3]: a, b (-1 = none), n_cls -- the host reads it with the counters of the next hit list.
__global__ void __launch_bounds__(256)
k_best_pair(const uint8_t* __restrict__ valid, const int32_t* __restrict__ n_cls, const uint8_t* __restrict__ cls,
            int32_t Ke, int32_t Kx, int32_t H, const double* __restrict__ half_seed, int32_t K,
            uint8_t* __restrict__ cls_best, int32_t* __restrict__ pick, int32_t* __restrict__ turn_pair,
            int32_t* __restrict__ turn_n, double* __restrict__ turn_seed)
{
    __shared__ unsigned long long s_key[8];
    const int t = threadIdx.x;
    unsigned long long key = 0;
    for (int i = t; i < Ke * Kx; i += 256)
        if (valid[i]) {
            const unsigned long long kk = ((unsigned long long)(unsigned int)(n_cls[i] + 1) << 32) |
                                          (unsigned long long)(~(unsigned int)i);
            key = kk > key ? kk : key;
        }
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xffffffffu, key, o);
        key = other > key ? other : key;
    }
    if ((t & 31) == 0) s_key[t >> 5] = key;
    __syncthreads();
    key = s_key[0];
    for (int i = 1; i < 8; ++i) key = s_key[i] > key ? s_key[i] : key;
    const int flat = key ? (int)(~(unsigned int)(key & 0xffffffffu)) : -1;
    const int a = flat >= 0 ? flat / Kx : -1, b = flat >= 0 ? flat - a * Kx : -1;
    for (int j = t; j < H; j += 256) cls_best[j] = flat >= 0 ? cls[(size_t)flat * H + j] : 0;
    if (t == 0) {
        pick[0] = a; pick[1] = b; pick[2] = flat >= 0 ? n_cls[flat] : 0;
        if (flat >= 0) { turn_pair[0] = a; turn_pair[1] = b; turn_n[0] = n_cls[flat]; }
    }
    if (flat >= 0 && t < 12) turn_seed[t] = t < 6 ? half_seed[(size_t)a * 6 + t] : half_seed[((size_t)K + b) * 6 + (t - 6)];
}

}  // namespace comet
