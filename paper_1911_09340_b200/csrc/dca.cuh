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

#define COMET_WT_FIELDS 15   // m[3] w[3] | e1[3] -m.e1 | e2[3] -m.e2 | far radius R_i
#define COMET_KT 32          // recorded states per shared-memory tile
#define COMET_DCA_WARPS 8

// B1: wire prep, one thread per fired wire (once per event).
// Field 14 is the wire's "far radius" R_i = max_j |rho_ij| + lambda + 0.51 h + 1e-6 cm (-1 for a
// wire without entries).  The virtual-plane iteration ends on the arc between the recorded states
// k*-1 and k*+1 (R10), at an offset sigma from k* with |sigma| <= h; that point is at most |sigma| of
// arc from state k* and at most h - |sigma| from its neighbour on that side, and both are at least
// d_k* from the wire (k* is the closest recorded state), so |D| >= d_k* - h/2 (1-Lipschitz; the
// 0.01 h + 1e-6 cover the step-length excess 1.001 and the RKN error of the sub-steps).  A track whose
// every recorded state is farther than R_i therefore has |D| - |rho_ij| > lambda for every entry and
// its bounded residual is exactly lambda (pruned mode).
//
// `tight` (uniform field: recorded states exactly h of arc apart): a sharper radius from the shape of the
// distance along the track.  Let s* be the arc position of k*, d* = d_k*, and u = s - s* in the bracket of the
// iteration (|u| <= 1.001 h).  On the tangent line at k* the squared distance to the wire is the quadratic
// g(u)^2 = d*^2 + a u (u + 2 v), 0 <= a <= 1, with its minimum at u = -v; the track leaves that line by at most
// eps = |c| (1.001 h)^2 / 2 <= 0.0251 h (|c| h <= COMET_CH_MAX = 0.05; lanes beyond that take no shortcut), and the
// distance to a line is 1-Lipschitz, so the neighbours' d_k*+-1 >= d* give g(+-h) >= d* - eps, i.e.
// a h (2|v| - h) <= 2 d* eps.  Minimising g^2 over the bracket under that constraint (|v| <= h: -a v^2 with
// a v^2 <= a h^2/4 + 1.5 d* eps; |v| > h: the bracket end, -a h (2|v| - h) >= -2 d* eps) leaves
// g^2 >= d*^2 - 0.2505 h^2 - 2 d* eps everywhere in the bracket -- at a track end the missing neighbour's side is
// not in the bracket --, hence |D| >= sqrt(d*^2 - 0.2505 h^2 - 2 d* eps) - eps - 1e-6 for whatever point the
// iteration ends on.  |D| - max|rho| > lambda then follows from d* > eps + sqrt((max|rho| + lambda + eps + 1e-6)^2
// + 0.2505 h^2 + eps^2); the smaller of the two radii is used.
__global__ void k_wire_prep(const double* __restrict__ wire_a, const double* __restrict__ wire_b,
                            int32_t n_wires, const int32_t* __restrict__ fired_wire, int32_t W,
                            const int32_t* __restrict__ hit_off, const double* __restrict__ rho,
                            double lambda, double h, int tight, double* __restrict__ wt, float* __restrict__ wtf = nullptr)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= W) return;
    // exact line (O4): w = (b-a)/|b-a|, m = (a+b)/2
    const WireLine wl = wire_line_of(wire_a, wire_b, n_wires, fired_wire[i]);
    const double w0 = wl.w0, w1 = wl.w1, w2 = wl.w2, m0 = wl.m0, m1 = wl.m1, m2 = wl.m2;
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
    double rmax = -1.0;
    for (int j = hit_off[i]; j < hit_off[i + 1]; ++j) rmax = fmax(rmax, fabs(rho[j]));
    double cap = rmax + lambda + 0.51 * h + 1e-6;
    if (tight) {
        const double eps = 0.0251 * h, b = rmax + lambda + eps + 1e-6;
        cap = fmin(cap, eps + sqrt(b * b + 0.2505 * h * h + eps * eps));
    }
    wt[14 * W + i] = (rmax < 0.0) ? -1.0 : cap;
    // single-precision copy of the shortlist fields for the pruning tests of k_scan_zrun (levels A and B): the basis and
    // offsets rounded to nearest (the tests carry the rounding as slack), the far radius, sqrt(1 - w_z^2) and |c1| + |c2|
    // rounded up
    if (wtf) {
        const double c1 = -(m0 * p0 + m1 * p1 + m2 * p2), c2 = -(m0 * q0 + m1 * q1 + m2 * q2);
        wtf[0 * W + i] = (float)p0; wtf[1 * W + i] = (float)p1; wtf[2 * W + i] = (float)p2; wtf[3 * W + i] = (float)c1;
        wtf[4 * W + i] = (float)q0; wtf[5 * W + i] = (float)q1; wtf[6 * W + i] = (float)q2; wtf[7 * W + i] = (float)c2;
        wtf[8 * W + i] = (rmax < 0.0) ? -1.f : __double2float_ru(cap);
        wtf[9 * W + i] = __fsqrt_ru(__double2float_ru(fma(p2, p2, q2 * q2)));
        wtf[10 * W + i] = __double2float_ru(fabs(c1) + fabs(c2));
    }
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
    unsigned long long* stats;   // optional work counters [ST_N] (pruned kernel, COMET_OPT_STATS)
};

// B2 decision + B3 + B4 for one (seed, wire) pair given the shortlisted state bk:
// the exact distance of O5 (the definition's operation order) decides between bk-1, bk, bk+1,
// then the virtual-plane iteration, the signed DCA and the squared bounded residual.
__device__ __forceinline__ double pair_exact(const double* __restrict__ Xc, const double* __restrict__ Tc,
                                             int lane, int bk, int np, const DcaArgs& a, double c, int i,
                                             double& D, int& ks)
{
    constexpr int ROW = 3 * COMET_LANES;
    const int W = a.W;
    WireLine wl;
    wl.m0 = __ldg(a.wt + i); wl.m1 = __ldg(a.wt + W + i); wl.m2 = __ldg(a.wt + 2 * W + i);
    wl.w0 = __ldg(a.wt + 3 * W + i); wl.w1 = __ldg(a.wt + 4 * W + i); wl.w2 = __ldg(a.wt + 5 * W + i);
    const int ka = max(bk - 1, 0), kb = min(bk + 1, np - 1);
    ks = ka;
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
    D = fine_dca(st, ks, np, a.h, c, wl);
    const double e = wire_residual(D, a.rho, __ldg(a.hit_off + i), __ldg(a.hit_off + i + 1), a.lambda,
                                   nullptr, nullptr);
    return xmul(e, e);
}

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
    const int32_t n_rows = track_rows(a.n_steps);
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
                // rows past this lane's last state repeat it (hold-last): never strictly smaller
#pragma unroll
                for (int q = 0; q < WT; ++q) {
                    const double u1 = fma(x0, e1x[q], fma(x1, e1y[q], fma(x2, e1z[q], c1[q])));
                    const double u2 = fma(x0, e2x[q], fma(x1, e2y[q], fma(x2, e2z[q], c2[q])));
                    const double d2 = fma(u1, u1, u2 * u2);
                    if (d2 < best[q]) { best[q] = d2; bk[q] = k0 + kk; }
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
                double D;
                int ks;
                e2 = pair_exact(Xc, Tc, lane, bk[q], np, a, c, i, D, ks);
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

// ---------------------------------------------------------------------------------------------
// Pruned closest-state search (COMET_COARSE_PRUNED): same k*, D and RSS as the exhaustive scan.
//
// Consecutive recorded states are at most L = 1.001 h apart (an RKN step of length h with |c| h
// <= 0.05 moves the position by less than h (1 + 1e-3); hold-last padding moves it by 0), and the
// distance to a line is 1-Lipschitz, so a state j rows away from an evaluated state k has
// D_j >= D_k - j L.  With any upper bound `ub` on the answer, a block of rows whose centre sample
// has D > ub + (half block) L cannot hold the closest state and is skipped.  Two levels:
//   level 0: blocks of M0 = 64 rows, sample at row 32; pass 1 takes the minimum over the samples
//            (ub), pass 2 revisits the samples and opens the blocks that may hold the answer;
//   level 1: an opened block is cut into sub-blocks of M1 = 8 rows, sample at row 4, the running
//            minimum tightens ub, and only the sub-blocks that may hold the answer are evaluated
//            row by row (in increasing k, strict "<": lowest k wins ties, as in the exhaustive scan).
// ub is also capped by the wire's far radius R_i (k_wire_prep) when neither D nor k* is asked
// for: a pair whose every state is farther than R_i contributes exactly lambda^2 to RSS and skips
// the virtual-plane iteration.  All bounds carry an absolute slack of 1e-9 cm for the rounding of
// the FMA-form distances (~1e-13 cm).  Lanes with |c| h > 0.05 take no shortcut (ub = infinity).
//
// Three kernels, no barriers, no atomics in the data path (lane = seed of a track chunk everywhere):
//   k_coarse_pruned  warp = (chunk, group of WT wires): shortlisted state bk per pair, -1 = far
//   k_fine           warp = (chunk, wire): exact decision + virtual-plane iteration + residual -> e^2
//   k_rss_sum        thread = seed: RSS = sum of e^2 in wire order (Eq. (1))
// bk [W][SP] int32 and e^2 [W][SP] double (SP = 32 * number of chunks) live in the ctx workspace.
// ---------------------------------------------------------------------------------------------
#ifndef COMET_M0
#define COMET_M0 64
#endif
#ifndef COMET_M1
#define COMET_M1 8
#endif
#define COMET_CH_MAX 0.05
#define COMET_LIP 1.001
#define COMET_SLACK 1e-9
#define COMET_PR_WARPS 8
#ifndef COMET_COARSE_MINB
#define COMET_COARSE_MINB 3
#endif
#ifndef COMET_SWEEP_B
#define COMET_SWEEP_B 8           // rows loaded per batch in a sub-block sweep
#endif
#ifndef COMET_FINE_MINB
#define COMET_FINE_MINB 4
#endif
#ifndef COMET_FINE_THREADS
#define COMET_FINE_THREADS 256
#endif

struct EvalC {
    double e1x, e1y, e1z, c1, e2x, e2y, e2z, c2;
};
__device__ __forceinline__ void load_evalc(EvalC& w, const double* __restrict__ wt, int W, int i)
{
    w.e1x = __ldg(wt + 6 * W + i); w.e1y = __ldg(wt + 7 * W + i); w.e1z = __ldg(wt + 8 * W + i);
    w.c1 = __ldg(wt + 9 * W + i);
    w.e2x = __ldg(wt + 10 * W + i); w.e2y = __ldg(wt + 11 * W + i); w.e2z = __ldg(wt + 12 * W + i);
    w.c2 = __ldg(wt + 13 * W + i);
}
__device__ __forceinline__ double d2_fma(const EvalC& w, double x0, double x1, double x2)
{
    const double u1 = fma(x0, w.e1x, fma(x1, w.e1y, fma(x2, w.e1z, w.c1)));
    const double u2 = fma(x0, w.e2x, fma(x1, w.e2y, fma(x2, w.e2z, w.c2)));
    return fma(u1, u1, u2 * u2);
}

// optional work counters (COMET_OPT_STATS), thread-level
enum { ST_SAMPLES = 0, ST_ROWS_NEEDED, ST_ROWS_EXEC, ST_FINE_NEEDED, ST_FINE_EXEC, ST_PAIRS, ST_UNIQUE, ST_SAMPLES_B, ST_TOUCHED, ST_N };

struct PrunedArgs {
    DcaArgs d;
    int64_t n_chunks;
    int64_t SP;              // 32 * n_chunks: stride of kb / e2
    int32_t n_groups;        // ceil(W / WT)
    int32_t cap_s;           // sub-block samples the shared-memory stage holds
    int32_t full;            // dca or kstar requested: no far-pair shortcut
    int32_t* kb;             // [W][SP]
    double* e2;              // [W][SP]
    unsigned long long* items;   // work list of k_fine: (chunk << 16 | wire) of every warp-item with a near lane
    unsigned int* n_items;       // its length (zeroed before k_coarse_pruned)
};

// CTA = one track chunk.  The sub-block samples (row 8 j + 4 of every 8-row sub-block j, fp64) are
// staged in shared memory once per CTA when they fit (`cap_s` of them; else they are read from
// global memory): both sampling levels run from there, only the rows of opened sub-blocks are read
// from the track buffer.  The level-0 sample of block t is sub-block sample 8 t + 4 (row 64 t + 36,
// at most 36 rows from any row of the block).  Kernel A pads every chunk to whole 64-row blocks
// (hold-last rows), so no index is ever clamped.
//
// Thresholds are compared on the high 32 bits of the (non-negative) squared distances: hi(d) <=
// hi(thr) whenever d <= thr, so the integer test accepts a superset -- still a correct pruning --
// and the minimum over samples is tracked as the integer minimum of the high words, rounded up.
template <int WT, bool STATS, bool SMEM>
__device__ __forceinline__ void coarse_groups(const PrunedArgs& pa, const double* __restrict__ Xl,
                                              const double* sbase, int n0, int lane, int64_t s, bool lip_ok,
                                              int* s_next, unsigned long long* st_cnt)
{
    constexpr int ROW = 3 * COMET_LANES;
    constexpr int NSUB = COMET_M0 / COMET_M1;               // sub-blocks per block
    constexpr int SST = SMEM ? ROW : COMET_M1 * ROW;        // distance between sub-block samples (doubles)
    constexpr unsigned FULL = 0xffffffffu;
    constexpr int IMAX = 0x7fffffff;
    const DcaArgs& a = pa.d;
    const int W = a.W;
    const double L = COMET_LIP * a.h;
    const double INF = 1.7976931348623157e308;
    const double half0 = (COMET_M0 / 2 + COMET_M1 / 2) * L + COMET_SLACK, half1 = (COMET_M1 / 2) * L + COMET_SLACK;
    const double lam2 = xmul(a.lambda, a.lambda);

    while (true) {
        int g = 0;
        if (lane == 0) g = atomicAdd(s_next, 1);
        g = __shfl_sync(FULL, g, 0);
        if (g >= pa.n_groups) break;
        const int i0 = g * WT;
        // ---- level 0: minimum over the block samples, then the blocks within reach of it ------------
        double ub0[WT];                                     // min(sqrt(min sample), far radius)
        unsigned mask[WT];                                  // bit t % 32: block t may hold the closest state
        {
            EvalC ec[WT];
            int dh[WT], thi[WT];
#pragma unroll
            for (int q = 0; q < WT; ++q) {
                load_evalc(ec[q], a.wt, W, min(i0 + q, W - 1));
                dh[q] = IMAX;
                mask[q] = 0u;
            }
            // RSS-only calls know an upper bound before looking at anything: the far radius.  One pass.
            // Calls that want D / k* of every pair first take the minimum over the block samples.
            const double* p = sbase + (NSUB / 2) * SST;
            if (pa.full) {
#pragma unroll 2
                for (int t = 0; t < n0; ++t, p += NSUB * SST) {
                    const double x0 = p[0], x1 = p[32], x2 = p[64];
#pragma unroll
                    for (int q = 0; q < WT; ++q) dh[q] = min(dh[q], __double2hiint(d2_fma(ec[q], x0, x1, x2)));
                }
                if (STATS) st_cnt[ST_SAMPLES] += (unsigned long long)n0 * min(WT, W - i0);
            }
#pragma unroll
            for (int q = 0; q < WT; ++q) {
                const double cap = pa.full ? INF : __ldg(a.wt + 14 * W + min(i0 + q, W - 1));   // far radius R_i
                const double dm = pa.full ? __hiloint2double(dh[q] + 1, 0) : INF;   // >= the smallest sample
                ub0[q] = lip_ok ? fmin(sqrt(dm), cap) : INF;
                const double t0 = ub0[q] + half0;
                thi[q] = lip_ok ? __double2hiint(t0 * t0) : IMAX;
                if (cap < 0.0 || i0 + q >= W) thi[q] = -1;           // wire without entries / past the end
            }
            p = sbase + (NSUB / 2) * SST;
#pragma unroll 2
            for (int t = 0; t < n0; ++t, p += NSUB * SST) {
                const double x0 = p[0], x1 = p[32], x2 = p[64];
                const unsigned bit = 1u << (t & 31);
#pragma unroll
                for (int q = 0; q < WT; ++q)
                    if (__double2hiint(d2_fma(ec[q], x0, x1, x2)) <= thi[q]) mask[q] |= bit;
            }
            if (STATS) st_cnt[ST_SAMPLES] += (unsigned long long)n0 * min(WT, W - i0);
        }
        // ---- per wire: level 1 in the opened blocks, row sweeps of the opened sub-blocks ------------
#pragma unroll 1
        for (int q = 0; q < WT; ++q) {
            const int i = i0 + q;
            if (i >= W) break;
            unsigned mq = mask[0];
            double ub = ub0[0];
#pragma unroll
            for (int r = 1; r < WT; ++r)
                if (q == r) { mq = mask[r]; ub = ub0[r]; }
            unsigned wm = __reduce_or_sync(FULL, mq);       // blocks any lane of the warp wants
            if (STATS) st_cnt[ST_PAIRS] += 1;
            int bk = -1;
            if (wm) {
                const double cap = pa.full ? INF : __ldg(a.wt + 14 * W + i);
                EvalC w;
                load_evalc(w, a.wt, W, i);                           // warp-uniform, L1-resident
                double best = INF;
                while (wm) {
                    const int tb = __ffs(wm) - 1;
                    wm &= wm - 1;
                    for (int t = tb; t < n0; t += 32) {              // blocks that share the mask bit
                        const double* ps = sbase + t * (NSUB * SST);
                        int d1h[NSUB];
                        int m1 = IMAX;
#pragma unroll
                        for (int j = 0; j < NSUB; ++j) {
                            d1h[j] = __double2hiint(d2_fma(w, ps[j * SST], ps[j * SST + 32], ps[j * SST + 64]));
                            m1 = min(m1, d1h[j]);
                        }
                        if (STATS) st_cnt[ST_SAMPLES] += NSUB;
                        ub = fmin(ub, sqrt(__hiloint2double(m1 + 1, 0)));
                        const double t1 = ub + half1;
                        const int t1h = lip_ok ? __double2hiint(t1 * t1) : IMAX;
                        unsigned sub = 0u;
#pragma unroll
                        for (int j = 0; j < NSUB; ++j)
                            if (d1h[j] <= t1h) sub |= 1u << j;
                        unsigned wsub = __reduce_or_sync(FULL, sub);
                        while (wsub) {
                            const int j = __ffs(wsub) - 1;
                            wsub &= wsub - 1;
                            if (STATS) { st_cnt[ST_ROWS_EXEC] += COMET_M1; if ((sub >> j) & 1u) st_cnt[ST_ROWS_NEEDED] += COMET_M1; }
                            const int rj = (t * NSUB + j) * COMET_M1;
                            const double* pr = Xl + (size_t)(unsigned)(rj * ROW);
#pragma unroll
                            for (int k0 = 0; k0 < COMET_M1; k0 += COMET_SWEEP_B) {
                                double xr[COMET_SWEEP_B][3];
#pragma unroll
                                for (int kk = 0; kk < COMET_SWEEP_B; ++kk) {
                                    xr[kk][0] = __ldg(pr + (k0 + kk) * ROW); xr[kk][1] = __ldg(pr + (k0 + kk) * ROW + 32);
                                    xr[kk][2] = __ldg(pr + (k0 + kk) * ROW + 64);
                                }
#pragma unroll
                                for (int kk = 0; kk < COMET_SWEEP_B; ++kk) {
                                    const double d2 = d2_fma(w, xr[kk][0], xr[kk][1], xr[kk][2]);
                                    if (d2 < best) { best = d2; bk = rj + k0 + kk; }
                                }
                            }
                        }
                    }
                }
                // near <=> the closest recorded state is within the far radius (always, in full mode)
                const bool near = (bk >= 0) && (sqrt(best) <= cap || !lip_ok);
                if (!near) bk = -1;
            }
            if (STATS && bk >= 0) st_cnt[ST_FINE_NEEDED] += 1;
            // a (chunk, wire) item with a near lane goes to k_fine's work list; the others are done here
            if (__any_sync(FULL, bk >= 0)) {
                pa.kb[(size_t)i * pa.SP + s] = bk;
                if (lane == 0)
                    pa.items[atomicAdd(pa.n_items, 1u)] = ((unsigned long long)(s >> 5) << 16) | (unsigned)i;
            } else {
                pa.e2[(size_t)i * pa.SP + s] = lam2;
            }
        }
    }
}

template <int WT, bool STATS>
__global__ void __launch_bounds__(COMET_PR_WARPS * 32, COMET_COARSE_MINB) k_coarse_pruned(const PrunedArgs pa)
{
    constexpr int ROW = 3 * COMET_LANES;
    constexpr unsigned FULL = 0xffffffffu;
    extern __shared__ __align__(16) double ssm[];           // [cap_s][ROW]
    __shared__ int s_next;
    const DcaArgs& a = pa.d;
    const int lane = threadIdx.x & 31;
    const int64_t chunk = blockIdx.x;
    const int64_t s = chunk * COMET_LANES + lane;
    const bool valid = s < a.n_seeds;
    const int32_t np = valid ? a.n_pts[s] : 0;
    const int32_t kmax = __reduce_max_sync(FULL, np);
    const int n0 = (kmax + COMET_M0 - 1) / COMET_M0;        // blocks (all complete: kernel A pads)
    const int nS = n0 * (COMET_M0 / COMET_M1);
    const double* __restrict__ Xc = a.X + track_row(chunk, track_rows(a.n_steps), 0);
    const bool in_smem = nS <= pa.cap_s;                    // CTA-uniform
    if (in_smem) {
        for (int v = threadIdx.x; v < nS * (ROW / 2); v += COMET_PR_WARPS * 32) {
            const int j = v / (ROW / 2), o = (v - j * (ROW / 2)) * 2;
            cp_async16(ssm + j * ROW + o, Xc + (size_t)(j * COMET_M1 + COMET_M1 / 2) * ROW + o);
        }
        cp_async_commit();
    }
    if (threadIdx.x == 0) s_next = 0;
    double ch = 0.0;                                        // |c| h of this lane
    if (valid) {
        const double px = a.seeds[3 * a.stride + s], py = a.seeds[4 * a.stride + s], pz = a.seeds[5 * a.stride + s];
        ch = fabs(a.qkb) * a.h / sqrt(px * px + py * py + pz * pz);
    }
    const bool lip_ok = ch <= COMET_CH_MAX;                 // Lipschitz bound valid for this lane
    unsigned long long st_cnt[ST_N];
    if (STATS) {
#pragma unroll
        for (int j = 0; j < ST_N; ++j) st_cnt[j] = 0;
    }
    cp_async_wait<0>();
    __syncthreads();
    if (in_smem) coarse_groups<WT, STATS, true>(pa, Xc + lane, ssm + lane, n0, lane, s, lip_ok, &s_next, st_cnt);
    else coarse_groups<WT, STATS, false>(pa, Xc + lane, Xc + lane + (COMET_M1 / 2) * ROW, n0, lane, s, lip_ok, &s_next, st_cnt);
    if (STATS) {
#pragma unroll
        for (int j = 0; j < ST_N; ++j) {
            unsigned long long v = st_cnt[j];
            for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(FULL, v, o);
            if (lane == 0 && a.stats && v) atomicAdd(a.stats + j, v);
        }
    }
}

// Persistent warps walk the work list of (chunk, wire) items that have at least one near lane:
// B2 decision + B3 + B4 for the near lanes, lambda^2 for the others.
template <bool STATS>
__global__ void __launch_bounds__(COMET_FINE_THREADS, COMET_FINE_MINB) k_fine(const PrunedArgs pa)
{
    const DcaArgs& a = pa.d;
    const int lane = threadIdx.x & 31;
    const unsigned n_items = *pa.n_items;
    const unsigned n_warps = gridDim.x * (COMET_FINE_THREADS / 32);
    const int W = a.W;
    const int32_t n_rows = track_rows(a.n_steps);
    const double lam2 = xmul(a.lambda, a.lambda);
    for (unsigned it = blockIdx.x * (COMET_FINE_THREADS / 32) + (threadIdx.x >> 5); it < n_items; it += n_warps) {
        const unsigned long long item = pa.items[it];
        const int64_t chunk = (int64_t)(item >> 16);
        const int i = (int)(item & 0xffffu);
        const int64_t s = chunk * COMET_LANES + lane;
        const bool valid = s < a.n_seeds;
        const int bk = pa.kb[(size_t)i * pa.SP + s];
        double e2 = lam2;
        if (STATS) { if (lane == 0 && a.stats) atomicAdd(a.stats + ST_FINE_EXEC, 32ull); }
        if (valid && bk >= 0) {
            const size_t base = track_row(chunk, n_rows, 0);
            const double px = a.seeds[3 * a.stride + s], py = a.seeds[4 * a.stride + s], pz = a.seeds[5 * a.stride + s];
            const double c = xdiv(a.qkb, xsqrt(xdot3(px, py, pz, px, py, pz)));
            double D;
            int ks;
            e2 = pair_exact(a.X + base, a.T + base, lane, bk, a.n_pts[s], a, c, i, D, ks);
            if (a.dca) a.dca[(size_t)s * W + i] = D;
            if (a.kstar) a.kstar[(size_t)s * W + i] = ks;
        }
        pa.e2[(size_t)i * pa.SP + s] = e2;
    }
}

// B5: RSS_s = sum_i e^2_i in increasing wire order (Eq. (1); no atomics, cf. :374).
// tm != nullptr (scan_zrun.cuh): bit i of the chunk's mask says whether the row of wire i exists; every other pair is
// beyond the far radius and contributes cutoff^2 = lam2 without a load.
__global__ void __launch_bounds__(256) k_rss_sum(const double* __restrict__ e2, int64_t SP, int32_t W,
                                                 int64_t n_seeds, double* __restrict__ rss,
                                                 const unsigned int* __restrict__ tm, double lam2,
                                                 const unsigned int* __restrict__ zg, const int32_t* __restrict__ dyn = nullptr)
{
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n_seeds) return;
    // (comet_scan_turns: the launch is sized by the event's first list; the wires that are left come first, Eq. (1) runs over them)
    const int MW = (W + 31) / 32;                          // words per chunk of the mask (as launched)
    if (dyn) {
        if (dyn[2]) return;
        W = dyn[0];
    }
    double acc = 0.0;
    // (zg: the run length found on the device -- the mask exists only if the z-run kernel served the launch)
    if (tm && (!zg || *zg >= 8u)) {
        // (the mask is the chunk's, a warp is one chunk: the control flow below is warp-uniform.  The additions are those of
        // the plain loop, one per wire in wire order; only the bit tests of the wires without a row go)
        const unsigned int* m = tm + (size_t)(s >> 5) * MW;
        for (int wd = 0; wd * 32 < W; ++wd) {
            unsigned bits = __ldg(m + wd);
            const int n = min(32, W - wd * 32);
            if (n < 32) bits &= (1u << n) - 1u;
            if (__popc(bits) > 6) {                         // many rows: the loads of a batch of wires in flight together
#pragma unroll 4
                for (int q = 0; q < n; ++q)
                    acc = xadd(acc, ((bits >> q) & 1u) ? e2[(size_t)(wd * 32 + q) * SP + s] : lam2);
                continue;
            }
            int j = 0;
            while (bits) {
                const int jn = __ffs(bits) - 1;             // the next wire with a row
                bits &= bits - 1;
                for (; j < jn; ++j) acc = xadd(acc, lam2);
                acc = xadd(acc, e2[(size_t)(wd * 32 + jn) * SP + s]);
                j = jn + 1;
            }
            if (j == 0 && n == 32) {
#pragma unroll
                for (int q = 0; q < 32; ++q) acc = xadd(acc, lam2);
            } else {
                for (; j < n; ++j) acc = xadd(acc, lam2);
            }
        }
    } else {
        // (small launches are latency-bound: 16 loads in flight per thread)
#pragma unroll 16
        for (int i = 0; i < W; ++i) acc = xadd(acc, e2[(size_t)i * SP + s]);
    }
    rss[s] = acc;
}

}  // namespace comet
