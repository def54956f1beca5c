// hough.cuh -- Hough-transform transverse seeding (Fig. 10; readings R35-R37), sm_100a.
//
// "The transverse components of (theta, p_x, p_y) were extracted by finding a circle that is the transverse
// projection of a helical trajectory [...] the Hough transform was applied to the set of transverse positions
// of the fired wires."  The circle passes through the origin (R36): u = x/(x^2+y^2), v = y/(x^2+y^2) of a
// wire's midpoint (R35) lie on the line u cos(phi) + v sin(phi) = rho = 1/(2R); every fired wire votes once
// per direction phi_j in the bin floor((rho - rho_min) inv_drho).  Integer/histogram work: the votes of a
// CTA's directions are counted with shared-memory atomics (integer adds: the counts do not depend on the
// order), the peak is a packed-key maximum (votes high word, inverted flat index low word: most votes,
// ties -> the lowest j n_rho + k) taken over the votes themselves (no pass over the bins), and the last CTA of an event to finish turns the peak into the circle and
// the entrance/exit seed points (R37).  The bin of a vote is decided in fp64 with one IEEE operation per
// operation of the definition (common.cuh's arithmetic policy).
#pragma once
#include "common.cuh"

namespace comet {

#define COMET_HT_THREADS 256
#ifndef COMET_HT_BINS
#define COMET_HT_BINS 8192          // vote bins per CTA the launch aims at (more, smaller CTAs: a short tail)
#endif

struct HoughWork {                 // per event, zeroed by the API before the launch
    unsigned long long key;        // max over the CTAs of (votes << 32) | ~flat
    unsigned int done;             // CTAs of the event that have published their key
    unsigned int pad;
};

// R37: peak bin -> circle, entrance and exit seed points.  out[11] = R, cx, cy, entrance (x, y, px, py), exit.
__device__ __forceinline__ void hough_circle(int votes, int k, double cj, double sj, double rho_min, double inv_drho,
                                             int32_t charge, double bz, double r_seed, double* __restrict__ out)
{
    const double nan = __longlong_as_double(0x7ff8000000000000LL);
#pragma unroll
    for (int i = 0; i < 11; ++i) out[i] = nan;
    if (votes == 0) return;
    const double rho_s = xadd(rho_min, xdiv((double)k + 0.5, inv_drho));
    const double R = xdiv(1.0, xmul(2.0, rho_s));
    const double cx = xmul(R, cj), cy = xmul(R, sj);
    out[0] = R;
    out[1] = cx;
    out[2] = cy;
    const double rs2 = xmul(r_seed, r_seed);
    const double t = xdiv(rs2, xmul(2.0, R));              // component of the seed point along the centre direction
    const double n2 = xsub(rs2, xmul(t, t));
    if (!(n2 > 0.0)) return;                               // the circle does not reach the seed cylinder
    const double n = xsqrt(n2);
    const double sense = ((double)charge * bz > 0.0) ? -1.0 : 1.0;   // +1: counter-clockwise (electron in B_z > 0)
    const double pT = xmul(xmul(COMET_KAPPA, fabs(bz)), R);
    double pt[2][4], rad[2];
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const double sn = i == 0 ? n : -n;
        const double px = xsub(xmul(t, cj), xmul(sn, sj));
        const double py = xadd(xmul(t, sj), xmul(sn, cj));
        const double tx = sense * xdiv(-xsub(py, cy), R), ty = sense * xdiv(xsub(px, cx), R);
        pt[i][0] = px;
        pt[i][1] = py;
        pt[i][2] = xmul(pT, tx);
        pt[i][3] = xmul(pT, ty);
        rad[i] = xadd(xmul(px, tx), xmul(py, ty));
    }
    const int e = rad[0] > 0.0 ? 0 : 1;                    // the entrance is where the track moves outwards
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        out[3 + i] = e == 0 ? pt[0][i] : pt[1][i];
        out[7 + i] = e == 0 ? pt[1][i] : pt[0][i];
    }
}

// grid (ceil(n_phi / D), n_events), COMET_HT_THREADS threads, D * n_rho * 4 + 2 * COMET_HT_THREADS * 8 bytes of
// dynamic shared memory.  CTA (b, e) counts the votes of event e's wires for the directions [b D, b D + D).
__global__ void __launch_bounds__(COMET_HT_THREADS)
k_hough(const double* __restrict__ wire_a, const double* __restrict__ wire_b, int32_t n_wires,
        const int32_t* __restrict__ fired_wire, const int32_t* __restrict__ ev_off,
        const double* __restrict__ cos_tab, const double* __restrict__ sin_tab, int32_t n_phi, int32_t D,
        double rho_min, double inv_drho, int32_t n_rho, int32_t charge, double bz, double r_seed,
        int32_t* __restrict__ acc, int32_t* __restrict__ peak, double* __restrict__ circle, HoughWork* __restrict__ work)
{
    extern __shared__ __align__(16) unsigned char ht_smem[];
    double* s_u = reinterpret_cast<double*>(ht_smem);
    double* s_v = s_u + COMET_HT_THREADS;
    int* s_acc = reinterpret_cast<int*>(s_v + COMET_HT_THREADS);
    __shared__ unsigned long long s_key[COMET_HT_THREADS / 32];
    __shared__ bool s_last;
    const int t = threadIdx.x, ev = blockIdx.y;
    const int j0 = blockIdx.x * D, nd = min(D, n_phi - j0);
    const int w0 = ev_off[ev], W = ev_off[ev + 1] - w0;
    const int n_bins = nd * n_rho;
    {   // zero the rows, 16 bytes per store (s_acc is 16-byte aligned, the tail goes word by word)
        int4* z4 = reinterpret_cast<int4*>(s_acc);
        const int n4 = n_bins >> 2;
        for (int i = t; i < n4; i += COMET_HT_THREADS) z4[i] = make_int4(0, 0, 0, 0);
        for (int i = (n4 << 2) + t; i < n_bins; i += COMET_HT_THREADS) s_acc[i] = 0;
    }
    const double n_rho_d = (double)n_rho;
    // The peak is found while voting: the thread whose vote completes a bin's final count sees that count, so
    // the maximum over all votes of (count after the vote, inverted flat index) is the peak with the rule of R36.
    unsigned long long key = 0;
    const bool fixed_d = (COMET_HT_THREADS % nd) == 0;      // CTA-uniform
    const int d_fix = t % nd, w_first = t / nd, w_step = COMET_HT_THREADS / nd;
    const double c_fix = cos_tab[j0 + d_fix], s_fix = sin_tab[j0 + d_fix];
    for (int base = 0; base < W; base += COMET_HT_THREADS) {
        __syncthreads();                                   // zeroing done / previous tile consumed
        const int nt = min(COMET_HT_THREADS, W - base);
        if (t < nt) {
            const int wi = fired_wire[w0 + base + t];
            const double x = xmul(xadd(wire_a[wi], wire_b[wi]), 0.5);
            const double y = xmul(xadd(wire_a[n_wires + wi], wire_b[n_wires + wi]), 0.5);
            const double r2 = xadd(xmul(x, x), xmul(y, y));
            s_u[t] = xdiv(x, r2);
            s_v[t] = xdiv(y, r2);
        }
        __syncthreads();
        auto vote = [&](int w, int d, double cd, double sd) {
            const double rho = xadd(xmul(s_u[w], cd), xmul(s_v[w], sd));
            const double k = floor(xmul(xsub(rho, rho_min), inv_drho));
            if (k >= 0.0 && k < n_rho_d) {
                const int bin = d * n_rho + (int)k;
                const unsigned int c = (unsigned int)atomicAdd(&s_acc[bin], 1) + 1u;
                const unsigned int flat = (unsigned int)(j0 * n_rho + bin);
                const unsigned long long kk = ((unsigned long long)c << 32) | (unsigned long long)(~flat);
                key = kk > key ? kk : key;
            }
        };
        if (fixed_d) {                                     // the thread keeps its direction: tables in registers
            for (int w = w_first; w < nt; w += w_step) vote(w, d_fix, c_fix, s_fix);
        } else {
            for (int i = t; i < nt * nd; i += COMET_HT_THREADS) {
                const int w = i / nd, d = i - w * nd;
                vote(w, d, cos_tab[j0 + d], sin_tab[j0 + d]);
            }
        }
    }
    if (acc) {                                             // rows out (optional)
        __syncthreads();
        int32_t* acc_e = acc + ((size_t)ev * n_phi + j0) * n_rho;
        for (int i = t; i < n_bins; i += COMET_HT_THREADS) acc_e[i] = s_acc[i];
    }
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xffffffffu, key, o);
        key = other > key ? other : key;
    }
    if ((t & 31) == 0) s_key[t >> 5] = key;
    __syncthreads();
    if (t == 0) {
        for (int i = 1; i < COMET_HT_THREADS / 32; ++i) key = s_key[i] > key ? s_key[i] : key;
        if (key) atomicMax(&work[ev].key, key);
        __threadfence();
        s_last = atomicAdd(&work[ev].done, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!s_last || t != 0) return;
    __threadfence();
    const unsigned long long best = atomicMax(&work[ev].key, 0ull);   // atomic read of the final key
    const int votes = (int)(best >> 32);
    const unsigned int flat = best ? ~(unsigned int)(best & 0xffffffffu) : 0u;   // no votes: peak (0, 0, 0)
    const int j = (int)(flat / (unsigned int)n_rho), k = (int)(flat - (unsigned int)j * (unsigned int)n_rho);
    peak[3 * ev] = votes;
    peak[3 * ev + 1] = j;
    peak[3 * ev + 2] = k;
    hough_circle(votes, k, cos_tab[j], sin_tab[j], rho_min, inv_drho, charge, bz, r_seed, circle + 11 * (size_t)ev);
}

}  // namespace comet
