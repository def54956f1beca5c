// seedgrid.cuh -- the first-iteration seed set of a turn partition built on the device from its axis tables
// ("A seed set was prepared by combining each component from the grids of the ranges"; reading R17,
// R44), sm_100a.
//
// The inputs are the grid's axes, not 6 x S doubles: per partition the seed point (x, y) on the r = 50 cm cylinder,
// the |p| values, (sin theta, cos theta) of the polar-angle axis, (cos phi0, sin phi0) of the azimuth axis and the z0
// values -- tables, as in comet_hough_seeds, so that no transcendental function is evaluated here and the products
// below are the same IEEE operations, in the same order, as in the host-side generator (comet_synth.seed_grid):
//     p_x = (|p| sin theta) cos phi0      p_y = (|p| sin theta) sin phi0      p_z = |p| cos theta
// Seed index within the partition: ((i_p n_ct + i_ct) n_phi + i_phi) n_z + i_z -- z fastest, so aligned runs of
// comet_grid_z_run(n_z) seeds differ only in z and the scan steps every distinct transverse track once.
#pragma once
#include "common.cuh"

namespace comet {

struct GridShape {
    int32_t n_p, n_ct, n_phi, n_z;
    int64_t G;               // seeds per partition
    int32_t A;               // doubles per partition in the axes table: 2 + n_p + 2 n_ct + 2 n_phi + n_z
};

// axes [n_part][A]: x, y | p [n_p] | sin theta [n_ct] | cos theta [n_ct] | cos phi0 [n_phi] | sin phi0 [n_phi] | z0 [n_z]
__global__ void __launch_bounds__(256)
k_seed_grid(const double* __restrict__ axes, GridShape g, int64_t n_total, double* __restrict__ seeds, int64_t stride)
{
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n_total) return;
    const int64_t part = s / g.G;
    int64_t r = s - part * g.G;
    const int iz = (int)(r % g.n_z); r /= g.n_z;
    const int iphi = (int)(r % g.n_phi); r /= g.n_phi;
    const int ict = (int)(r % g.n_ct);
    const int ip = (int)(r / g.n_ct);
    const double* a = axes + (size_t)part * g.A;
    const double pm = __ldg(a + 2 + ip);
    const double* act = a + 2 + g.n_p;
    const double st = __ldg(act + ict), ct = __ldg(act + g.n_ct + ict);
    const double* aph = act + 2 * g.n_ct;
    const double cf = __ldg(aph + iphi), sf = __ldg(aph + g.n_phi + iphi);
    const double z = __ldg(aph + 2 * g.n_phi + iz);
    const double pt = xmul(pm, st);
    seeds[s] = __ldg(a);
    seeds[stride + s] = __ldg(a + 1);
    seeds[2 * stride + s] = z;
    seeds[3 * stride + s] = xmul(pt, cf);
    seeds[4 * stride + s] = xmul(pt, sf);
    seeds[5 * stride + s] = xmul(pm, ct);
}

}  // namespace comet
