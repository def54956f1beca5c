// dca.cuh -- kernel B "DCA finding" + RSS (Algorithm 2; Eq. (1), :75-77), sm_100a.
//
// Mapping (differs from the paper's block = seed / thread = wire):
//   CTA  = one track chunk (32 consecutive seeds), lane = seed, so the chunk rows kernel A wrote
//          ([k][3][32] doubles = 768 B per recorded state) are read back exactly as written;
//   warp = a group of WT fired wires per pass, their line constants held in registers
//          (warp-uniform), NWARPS*WT wires per pass over the chunk's recorded states;
//   the chunk's position rows are streamed through shared memory in tiles of KT states with a
//   two-stage cp.async pipeline; every row read from shared memory is conflict-free
//   (bank = lane) and is reused by WT wire evaluations from registers.
//
// Per (seed, wire):
//   B2 shortlist: argmin_k of |perp(x_k)|^2 in the 2-vector form u = (x.e1 - m.e1, x.e2 - m.e2)
//      with {e1, e2, w} orthonormal: 8 FP64 FMA-pipe instructions + 1 compare per state;
//   B2 decision: the exact distance of DESIGN.md O5 (the definition's operation order) at k-1, k, k+1;
//   B3/B4: exact virtual-plane iteration, signed DCA and bounded residual (common.cuh);
//   B5: e^2 of the pass go through shared memory and warp 0 adds them in wire order, so RSS
//      is summed in exactly the order of Eq. (1)'s index i -- no atomics.
#pragma once
#include "common.cuh"

namespace comet {

#define COMET_WT_FIELDS 14   // m[3] w[3] | e1[3] -m.e1 | e2[3] -m.e2
#define COMET_KT 32          // recorded states per shared-memory tile
#define COMET_DCA_WARPS 8

// B1: wire prep, one thread per fired wire (once per event).
__global__ void k_wire_prep(const double* __restrict__ wire_a, const double* __restrict__ wire_b,
                            int32_t n_wires, const int32_t* __restrict__ fired_wire, int32_t W,
                            double* __restrict__ wt)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= W) return;
    const int wi = fired_wire[i];
    const double a0 = wire_a[wi], a1 = wire_a[(size_t)n_wires + wi], a2 = wire_a[2 * (size_t)n_wires + wi];
    const double b0 = wire_b[wi], b1 = wire_b[(size_t)n_wires + wi], b2 = wire_b[2 * (size_t)n_wires + wi];
    // exact line (O4): w = (b-a)/|b-a|, m = (a+b)/2
    const double d0 = xsub(b0, a0), d1 = xsub(b1, a1), d2 = xsub(b2, a2);
    const double len = xsqrt(xdot3(d0, d1, d2, d0, d1, d2));
    const double w0 = xdiv(d0, len), w1 = xdiv(d1, len), w2 = xdiv(d2, len);
    const double m0 = xmul(xadd(a0, b0), 0.5), m1 = xmul(xadd(a1, b1), 0.5), m2 = xmul(xadd(a2, b2), 0.5);
    wt[0 * W + i] = m0; wt[1 * W + i] = m1; wt[2 * W + i] = m2;
    wt[3 * W + i] = w0; wt[4 * W + i] = w1; wt[5 * W + i] = w2;
    // orthonormal basis of the plane perpendicular to w (shortlist only)
    double p0, p1, p2;
    const double f0 = fabs(w0), f1 = fabs(w1), f2 = fabs(w2);
    if (f0 <= f1 && f0 <= f2) { p0 = 0.0; p1 = -w2; p2 = w1; }          // x^ x w ... any vector _|_ w
    else if (f1 <= f2)        { p0 = w2; p1 = 0.0; p2 = -w0; }
    else                      { p0 = -w1; p1 = w0; p2 = 0.0; }
    const double pn = 1.0 / sqrt(p0 * p0 + p1 * p1 + p2 * p2);
    p0 *= pn; p1 *= pn; p2 *= pn;
    const double q0 = w1 * p2 - w2 * p1, q1 = w2 * p0 - w0 * p2, q2 = w0 * p1 - w1 * p0;
    wt[6 * W + i] = p0; wt[7 * W + i] = p1; wt[8 * W + i] = p2;
    wt[9 * W + i] = -(m0 * p0 + m1 * p1 + m2 * p2);
    wt[10 * W + i] = q0; wt[11 * W + i] = q1; wt[12 * W + i] = q2;
    wt[13 * W + i] = -(m0 * q0 + m1 * q1 + m2 * q2);
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

struct DcaArgs {
    const double* X;         // position plane
    const double* T;         // tangent plane
    const int32_t* n_pts;
    int64_t n_seeds;
    int32_t n_steps;
    double qkb;              // kappa * charge * B_z
    double h;
    const double* seeds;
    int64_t stride;
    const double* wt;        // [14][W]
    int32_t W;
    const int32_t* hit_off;
    const double* rho;
    double lambda;
    double* rss;
    double* dca;             // optional
    int32_t* kstar;          // optional
};

template <int WT>
__global__ void __launch_bounds__(COMET_DCA_WARPS * 32, 2) k_dca_rss(const DcaArgs a)
{
    constexpr int NW = COMET_DCA_WARPS;
    constexpr int WPP = NW * WT;                  // wires per pass
    constexpr int ROW = 3 * COMET_LANES;          // doubles per recorded state of a chunk
    extern __shared__ __align__(16) double smem[];
    double* stage0 = smem;                        // [2][KT][ROW]
    double* e2s = smem + 2 * COMET_KT * ROW;      // [WPP][32]

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t chunk = blockIdx.x;
    const int64_t s = chunk * COMET_LANES + lane;
    const bool valid = s < a.n_seeds;
    const int32_t n_rows = a.n_steps + 1;
    const int32_t np = valid ? a.n_pts[s] : 0;
    const int32_t kmax = __reduce_max_sync(0xffffffffu, np);
    const int n_tiles = (kmax + COMET_KT - 1) / COMET_KT;
    const size_t base = track_row(chunk, n_rows, 0);
    const double* Xc = a.X + base;
    const double* Tc = a.T + base;
    double c = 0.0;
    if (valid) {
        const double px = a.seeds[3 * a.stride + s], py = a.seeds[4 * a.stride + s], pz = a.seeds[5 * a.stride + s];
        c = xdiv(a.qkb, xsqrt(xdot3(px, py, pz, px, py, pz)));
    }
    const int W = a.W;
    const int n_pass = (W + WPP - 1) / WPP;
    double rss_acc = 0.0;

    for (int pass = 0; pass < n_pass; ++pass) {
        int wi[WT];
        double e1x[WT], e1y[WT], e1z[WT], c1[WT], e2x[WT], e2y[WT], e2z[WT], c2[WT], best[WT];
        int bk[WT];
#pragma unroll
        for (int q = 0; q < WT; ++q) {
            int i = pass * WPP + warp * WT + q;
            wi[q] = i;
            if (i >= W) i = W - 1;
            e1x[q] = __ldg(a.wt + 6 * W + i); e1y[q] = __ldg(a.wt + 7 * W + i); e1z[q] = __ldg(a.wt + 8 * W + i);
            c1[q] = __ldg(a.wt + 9 * W + i);
            e2x[q] = __ldg(a.wt + 10 * W + i); e2y[q] = __ldg(a.wt + 11 * W + i); e2z[q] = __ldg(a.wt + 12 * W + i);
            c2[q] = __ldg(a.wt + 13 * W + i);
            best[q] = 1.7976931348623157e308;
            bk[q] = 0;
        }
        // ---- B2 shortlist: stream the chunk's position rows through shared memory ----------
        auto prefetch = [&](int t) {
            const int rows = min(COMET_KT, kmax - t * COMET_KT);
            const int nvec = rows * (ROW / 2);                    // 16-byte pieces
            const double* src = Xc + (size_t)t * COMET_KT * ROW;
            double* dst = stage0 + (t & 1) * COMET_KT * ROW;
            for (int v = threadIdx.x; v < nvec; v += NW * 32) cp_async16(dst + 2 * v, src + 2 * v);
            cp_async_commit();
        };
        prefetch(0);
        for (int t = 0; t < n_tiles; ++t) {
            if (t + 1 < n_tiles) { prefetch(t + 1); cp_async_wait<1>(); }
            else { cp_async_wait<0>(); }
            __syncthreads();
            const double* sx = stage0 + (t & 1) * COMET_KT * ROW + lane;
            const int rows = min(COMET_KT, kmax - t * COMET_KT);
            const int k0 = t * COMET_KT;
#pragma unroll 4
            for (int kk = 0; kk < rows; ++kk) {
                const double x0 = sx[kk * ROW], x1 = sx[kk * ROW + 32], x2 = sx[kk * ROW + 64];
                const bool in_arc = (k0 + kk) < np;       // rows past this lane's last state hold a sentinel
#pragma unroll
                for (int q = 0; q < WT; ++q) {
                    const double u1 = fma(x0, e1x[q], fma(x1, e1y[q], fma(x2, e1z[q], c1[q])));
                    const double u2 = fma(x0, e2x[q], fma(x1, e2y[q], fma(x2, e2z[q], c2[q])));
                    const double d2 = fma(u1, u1, u2 * u2);
                    if (in_arc && d2 < best[q]) { best[q] = d2; bk[q] = k0 + kk; }
                }
            }
            __syncthreads();
        }
        // ---- B2 decision, B3, B4 per wire --------------------------------------------------
#pragma unroll
        for (int q = 0; q < WT; ++q) {
            double e2 = 0.0;
            if (valid && wi[q] < W) {
                const int i = wi[q];
                WireLine wl;
                wl.m0 = __ldg(a.wt + i); wl.m1 = __ldg(a.wt + W + i); wl.m2 = __ldg(a.wt + 2 * W + i);
                wl.w0 = __ldg(a.wt + 3 * W + i); wl.w1 = __ldg(a.wt + 4 * W + i); wl.w2 = __ldg(a.wt + 5 * W + i);
                const int ka = max(bk[q] - 1, 0), kb = min(bk[q] + 1, np - 1);
                int ks = ka;
                double bd = 0.0;
                State st;
                st.x0 = st.x1 = st.x2 = 0.0;
                for (int k = ka; k <= kb; ++k) {
                    const double* xr = Xc + (size_t)k * ROW + lane;
                    const double x0 = xr[0], x1 = xr[32], x2 = xr[64];
                    double u0, u1, u2;
                    const double d2 = perp2_exact(x0, x1, x2, wl, u0, u1, u2);
                    if (k == ka || d2 < bd) { bd = d2; ks = k; st.x0 = x0; st.x1 = x1; st.x2 = x2; }
                }
                const double* tr = Tc + (size_t)ks * ROW + lane;
                st.t0 = tr[0]; st.t1 = tr[32]; st.t2 = tr[64];
                const double D = fine_dca(st, ks, np, a.h, c, wl);
                const double e = wire_residual(D, a.rho, __ldg(a.hit_off + i), __ldg(a.hit_off + i + 1),
                                               a.lambda, nullptr, nullptr);
                e2 = xmul(e, e);
                if (a.dca) a.dca[(size_t)s * W + i] = D;
                if (a.kstar) a.kstar[(size_t)s * W + i] = ks;
            }
            e2s[(warp * WT + q) * 32 + lane] = e2;
        }
        __syncthreads();
        // ---- B5: warp 0 adds this pass's e^2 in wire order ---------------------------------
        if (warp == 0) {
            const int n_here = min(WPP, W - pass * WPP);
            for (int j = 0; j < n_here; ++j) rss_acc = xadd(rss_acc, e2s[j * 32 + lane]);
        }
        __syncthreads();
    }
    if (warp == 0 && valid) a.rss[s] = rss_acc;
}

}  // namespace comet
