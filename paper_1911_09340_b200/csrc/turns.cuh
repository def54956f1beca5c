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
// pad != 0 (comet_scan_turns, whose launches are sized by the event's first list): the output list is filled up to W
// wires with wires WITHOUT entries (a valid wire index, hit_off = the number of entries), so that a consumer
// launched for W wires finds nothing on them; counts[0..1] hold the real sizes.  stop: a device flag; set = do nothing.
__global__ void __launch_bounds__(COMET_RM_THREADS)
k_remove_hits(const int32_t* __restrict__ fired_wire, const int32_t* __restrict__ hit_off,
              const double* __restrict__ rho, int32_t W, const uint8_t* __restrict__ cls,
              const int32_t* __restrict__ orig_in, int32_t* __restrict__ fired_out,
              int32_t* __restrict__ hit_off_out, double* __restrict__ rho_out, int32_t* __restrict__ orig_out,
              int32_t* __restrict__ counts, int pad = 0, const int32_t* __restrict__ stop = nullptr)
{
    if (stop && *stop) return;
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
    if (pad && W > 0) {
        const int32_t any_wire = fired_wire[W - 1];
        for (int i = tw + t; i < W; i += COMET_RM_THREADS) {
            fired_out[i] = any_wire;
            hit_off_out[i + 1] = te;
        }
    }
}

// comet_scan_turns, before the stage of partition p: dyn = {fired wires left, entries left, stop flag, stages done}.
// The stage runs iff the loop has not stopped, at least min_wires fired wires are left and fewer than max_tracks stages
// are done (R34); else the stop flag is set for good and every later kernel of the loop returns at once.
__global__ void k_turn_gate(int32_t* __restrict__ dyn, int p, int32_t min_wires, int32_t max_tracks,
                            int32_t* __restrict__ done, int32_t* __restrict__ wires_before)
{
    if (dyn[2] || dyn[0] < min_wires || dyn[3] >= max_tracks) { dyn[2] = 1; return; }
    done[p] = 1;
    wires_before[p] = dyn[0];
    dyn[3] += 1;
}
__global__ void k_turn_init(int32_t* __restrict__ dyn, int32_t W, int32_t H, int32_t* __restrict__ done,
                            int32_t* __restrict__ wires_before, int n_part)
{
    dyn[0] = W; dyn[1] = H; dyn[2] = 0; dyn[3] = 0;
    for (int p = 0; p < n_part; ++p) { done[p] = 0; wires_before[p] = 0; }
}

// classification of a stage (entries of the reduced list) -> the event's own entry numbering
__global__ void __launch_bounds__(256)
k_scatter_cls(const uint8_t* __restrict__ cls, const int32_t* __restrict__ orig, int32_t H, uint8_t* __restrict__ out,
              const int32_t* __restrict__ dyn = nullptr)
{
    if (dyn) {                                              // (comet_scan_turns: the entries that are left; nothing once stopped)
        if (dyn[2]) return;
        H = dyn[1];
    }
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j < H && cls[j]) out[orig ? orig[j] : j] = 1;
}

}  // namespace comet
