// turns.cuh -- hit removal between the sequential stages of an event (readings R33-R34), sm_100a.
//
// "The hits classified previously were excluded in the seed scanning; therefore, the number of wires gets
// reduced whenever a track is fitted."  A measured hit is the adjacent pair of ghost entries (2m, 2m+1); an
// entry leaves the list when it or its partner is classified, a wire left without entries leaves the fired
// list.  Integer work: flags, two exclusive prefix sums over the wires, an order-preserving compaction.
#pragma once
#include "common.cuh"

namespace comet {

#define COMET_RM_THREADS 1024

// One CTA.  Thread t owns a contiguous range of wires; (kept wires, kept entries) of the ranges are scanned
// across the CTA (warp shuffles + one shared-memory round), then every thread writes its wires in order.
// orig_in == nullptr means the identity (the event's own entry numbering).
__global__ void __launch_bounds__(COMET_RM_THREADS)
k_remove_hits(const int32_t* __restrict__ fired_wire, const int32_t* __restrict__ hit_off,
              const double* __restrict__ rho, int32_t W, const uint8_t* __restrict__ cls,
              const int32_t* __restrict__ orig_in, int32_t* __restrict__ fired_out,
              int32_t* __restrict__ hit_off_out, double* __restrict__ rho_out, int32_t* __restrict__ orig_out,
              int32_t* __restrict__ counts)
{
    __shared__ int s_w[COMET_RM_THREADS / 32], s_e[COMET_RM_THREADS / 32];
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    const int per = (W + COMET_RM_THREADS - 1) / COMET_RM_THREADS;
    const int w0 = min(W, t * per), w1 = min(W, w0 + per);
    int nw = 0, ne = 0;
    for (int i = w0; i < w1; ++i) {
        int c = 0;
        for (int j = hit_off[i]; j < hit_off[i + 1]; ++j) c += !(cls[j] | cls[j ^ 1]);
        nw += c > 0;
        ne += c;
    }
    // inclusive warp scans, then the warp totals
    int iw = nw, ie = ne;
    for (int o = 1; o < 32; o <<= 1) {
        const int a = __shfl_up_sync(0xffffffffu, iw, o), b = __shfl_up_sync(0xffffffffu, ie, o);
        if (lane >= o) { iw += a; ie += b; }
    }
    if (lane == 31) { s_w[warp] = iw; s_e[warp] = ie; }
    __syncthreads();
    int bw = 0, be = 0, tw = 0, te = 0;
    for (int k = 0; k < COMET_RM_THREADS / 32; ++k) {
        if (k < warp) { bw += s_w[k]; be += s_e[k]; }
        tw += s_w[k];
        te += s_e[k];
    }
    int ow = bw + iw - nw, oe = be + ie - ne;            // exclusive offsets of this thread's range
    for (int i = w0; i < w1; ++i) {
        const int e0 = oe;
        for (int j = hit_off[i]; j < hit_off[i + 1]; ++j) {
            if (!(cls[j] | cls[j ^ 1])) {
                rho_out[oe] = rho[j];
                if (orig_out) orig_out[oe] = orig_in ? orig_in[j] : j;
                ++oe;
            }
        }
        if (oe > e0) {
            fired_out[ow] = fired_wire[i];
            hit_off_out[ow] = e0;
            ++ow;
        }
    }
    if (t == 0) {
        hit_off_out[tw] = te;
        counts[0] = tw;
        counts[1] = te;
    }
}

// classification of a stage (entries of the reduced list) -> the event's own entry numbering
__global__ void __launch_bounds__(256)
k_scatter_cls(const uint8_t* __restrict__ cls, const int32_t* __restrict__ orig, int32_t H, uint8_t* __restrict__ out)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j < H && cls[j]) out[orig ? orig[j] : j] = 1;
}

}  // namespace comet
