// common.cuh -- shared device helpers of the CUDA seed x hit scan (sm_100a).
//
// Arithmetic policy.  Everything that ends up in a result (track points, k*, DCA, residuals,
// RSS) is computed with one IEEE-754 double operation per operation of the definition in
// DESIGN.md section 2, in the order written there -- the __d*_rn intrinsics are never contracted
// into FMAs by nvcc -- so the results do not depend on compiler flags or on the kernel variant.
// Only the coarse closest-point *shortlist* (dca.cuh) uses FMAs; its choice is re-decided with
// the exact distance before it is used.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define COMET_KAPPA 2.99792458      // (MeV/c)/(T cm): "0.3 B" of PAPER.md:319 Eq. (2), reading R4
#define COMET_TOL_CM 1e-9           // TOLERANCE of PAPER.md:173, reading R9
#define COMET_MAX_ITER 16
#define COMET_DEN_MIN 1e-12
#define COMET_LANES 32              // seeds per track chunk

namespace comet {

__device__ __forceinline__ double xmul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double xadd(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double xsub(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ double xdiv(double a, double b) { return __ddiv_rn(a, b); }
__device__ __forceinline__ double xsqrt(double a) { return __dsqrt_rn(a); }
// a0*b0 + a1*b1 + a2*b2 evaluated left to right
__device__ __forceinline__ double xdot3(double a0, double a1, double a2, double b0, double b1, double b2)
{
    return xadd(xadd(xmul(a0, b0), xmul(a1, b1)), xmul(a2, b2));
}

struct State {          // one recorded track parameter: position (cm) and unit tangent
    double x0, x1, x2, t0, t1, t2;
};

// Step constants for a step of signed length h: h, h/2, h*h/6, h/6 (each one IEEE operation).
struct StepK {
    double h, hh, hh6, h6;
};
__host__ __device__ __forceinline__ StepK make_stepk_host(double h)
{
    StepK k;
    k.h = h;
    k.hh = h / 2.0;
    k.hh6 = (h * h) / 6.0;
    k.h6 = h / 6.0;
    return k;
}
// a / 6.0 correctly rounded without the division sequence: with y = RN(1/6), q = RN(a y), the exact
// residual r = a - 6 q (one FMA) and q' = RN(q + r y) give RN(a / 6) (Markstein's theorem; 6 has no
// hard-case significand).  Checked against a / 6.0 on 2e9 random doubles.
__device__ __forceinline__ double div6(double a)
{
    const double y = 1.0 / 6.0;
    const double q = xmul(a, y);
    const double r = fma(-6.0, q, a);
    return fma(r, y, q);
}
__device__ __forceinline__ StepK make_stepk(double h)
{
    StepK k;
    k.h = h;
    k.hh = xmul(h, 0.5);                 // == h / 2.0 exactly
    k.hh6 = div6(xmul(h, h));            // == (h * h) / 6.0
    k.h6 = div6(h);                      // == h / 6.0
    return k;
}

// One classical 4th-order Runge-Kutta-Nystrom step in the uniform field (0,0,B_z)
// (reading R1):  f(T) = c (T_y, -T_x, 0),
//   k1=f(T) k2=f(T+h/2 k1) k3=f(T+h/2 k2) k4=f(T+h k3)
//   x' = x + h T + h^2/6 (k1+k2+k3)      T' = T + h/6 (k1 + 2 k2 + 2 k3 + k4)
// The z components of k are zero: x2' = x2 + h T2, T2' = T2.  T is not renormalised.
__device__ __forceinline__ void rkn4_step(State& s, const StepK& k, double c)
{
    const double k1x = xmul(c, s.t1), k1y = -xmul(c, s.t0);
    double ax = xadd(s.t0, xmul(k.hh, k1x)), ay = xadd(s.t1, xmul(k.hh, k1y));
    const double k2x = xmul(c, ay), k2y = -xmul(c, ax);
    ax = xadd(s.t0, xmul(k.hh, k2x));
    ay = xadd(s.t1, xmul(k.hh, k2y));
    const double k3x = xmul(c, ay), k3y = -xmul(c, ax);
    ax = xadd(s.t0, xmul(k.h, k3x));
    ay = xadd(s.t1, xmul(k.h, k3y));
    const double k4x = xmul(c, ay), k4y = -xmul(c, ax);
    s.x0 = xadd(xadd(s.x0, xmul(k.h, s.t0)), xmul(k.hh6, xadd(xadd(k1x, k2x), k3x)));
    s.x1 = xadd(xadd(s.x1, xmul(k.h, s.t1)), xmul(k.hh6, xadd(xadd(k1y, k2y), k3y)));
    s.x2 = xadd(s.x2, xmul(k.h, s.t2));
    // k1 + 2 k2 + 2 k3 + k4 left to right: 2 k is exact, so fma(2, k2, k1) == RN(k1 + RN(2 k2)) bit for bit
    s.t0 = xadd(s.t0, xmul(k.h6, xadd(fma(2.0, k3x, fma(2.0, k2x, k1x)), k4x)));
    s.t1 = xadd(s.t1, xmul(k.h6, xadd(fma(2.0, k3y, fma(2.0, k2y, k1y)), k4y)));
}

// Seed -> initial state and curvature constant c = kappa q B_z / |p| (A1; qkb = kappa*q*B_z).
__device__ __forceinline__ double seed_init(const double* __restrict__ seeds, int64_t stride, int64_t s,
                                            double qkb, State& st)
{
    const double px = seeds[3 * stride + s], py = seeds[4 * stride + s], pz = seeds[5 * stride + s];
    const double P = xsqrt(xdot3(px, py, pz, px, py, pz));
    st.x0 = seeds[s];
    st.x1 = seeds[stride + s];
    st.x2 = seeds[2 * stride + s];
    st.t0 = xdiv(px, P);
    st.t1 = xdiv(py, P);
    st.t2 = xdiv(pz, P);
    return xdiv(qkb, P);
}

// target region test of reading R3 on a recorded state
__device__ __forceinline__ bool in_target_region(const State& s, double r_stop2)
{
    const double r2 = xadd(xmul(s.x0, s.x0), xmul(s.x1, s.x1));
    if (!(r2 < r_stop2)) return false;                  // the usual case: x.T is not needed
    const double rad = xadd(xmul(s.x0, s.t0), xmul(s.x1, s.t1));
    return rad < 0.0;
}

// Track buffer: plane [n_chunks][n_rows][3][32]; index of (chunk, k, component 0, lane 0).
// n_rows = track_rows(n_steps): n_steps + 1 recorded states rounded up to a multiple of 64 rows, so
// that kernel A can pad every chunk to whole 64-row blocks (hold-last) for the pruned search.
#define COMET_ROW_PAD 64
__device__ __host__ __forceinline__ int32_t track_rows(int32_t n_steps)
{
    return (n_steps + COMET_ROW_PAD) & ~(COMET_ROW_PAD - 1);
}
__device__ __host__ __forceinline__ size_t track_row(int64_t chunk, int32_t n_rows, int32_t k)
{
    return ((size_t)chunk * (size_t)n_rows + (size_t)k) * (size_t)(3 * COMET_LANES);
}

// Exact wire line (O4): unit direction w and midpoint m.
struct WireLine {
    double m0, m1, m2, w0, w1, w2;
};

// O4: the line of wire `wi` from its end points (SoA [3][n_wires]): w = (b - a) / |b - a|, m = (a + b) / 2
__device__ __forceinline__ WireLine wire_line_of(const double* __restrict__ wire_a, const double* __restrict__ wire_b,
                                                 int32_t n_wires, int wi)
{
    const double a0 = wire_a[wi], a1 = wire_a[(size_t)n_wires + wi], a2 = wire_a[2 * (size_t)n_wires + wi];
    const double b0 = wire_b[wi], b1 = wire_b[(size_t)n_wires + wi], b2 = wire_b[2 * (size_t)n_wires + wi];
    const double d0 = xsub(b0, a0), d1 = xsub(b1, a1), d2 = xsub(b2, a2);
    const double len = xsqrt(xdot3(d0, d1, d2, d0, d1, d2));
    WireLine wl;
    wl.w0 = xdiv(d0, len); wl.w1 = xdiv(d1, len); wl.w2 = xdiv(d2, len);
    wl.m0 = xmul(xadd(a0, b0), 0.5); wl.m1 = xmul(xadd(a1, b1), 0.5); wl.m2 = xmul(xadd(a2, b2), 0.5);
    return wl;
}

// exact squared perpendicular distance from the wire line to x (O4/O5)
__device__ __forceinline__ double perp2_exact(double x0, double x1, double x2, const WireLine& wl,
                                              double& u0, double& u1, double& u2)
{
    const double d0 = xsub(x0, wl.m0), d1 = xsub(x1, wl.m1), d2 = xsub(x2, wl.m2);
    const double t = xdot3(d0, d1, d2, wl.w0, wl.w1, wl.w2);
    u0 = xsub(d0, xmul(t, wl.w0));
    u1 = xsub(d1, xmul(t, wl.w1));
    u2 = xsub(d2, xmul(t, wl.w2));
    return xdot3(u0, u1, u2, u0, u1, u2);
}

// O6 + O7: virtual-plane iteration from recorded state `s` (index kstar of n_pts) and signed DCA.
__device__ __forceinline__ double fine_dca(State s, int kstar, int n_pts, double h, double c,
                                           const WireLine& wl)
{
    const double lo = (kstar > 0) ? -h : 0.0;
    const double hi = (kstar < n_pts - 1) ? h : 0.0;
    double sigma = 0.0;
#pragma unroll 1
    for (int it = 0; it < COMET_MAX_ITER; ++it) {
        const double tw = xdot3(s.t0, s.t1, s.t2, wl.w0, wl.w1, wl.w2);
        const double n0 = xsub(s.t0, xmul(tw, wl.w0));
        const double n1 = xsub(s.t1, xmul(tw, wl.w1));
        const double n2 = xsub(s.t2, xmul(tw, wl.w2));
        const double den = xdot3(s.t0, s.t1, s.t2, n0, n1, n2);
        if (den < COMET_DEN_MIN) break;
        const double mx0 = xsub(wl.m0, s.x0), mx1 = xsub(wl.m1, s.x1), mx2 = xsub(wl.m2, s.x2);
        double delta = xdiv(xdot3(mx0, mx1, mx2, n0, n1, n2), den);
        double target = xadd(sigma, delta);
        if (target < lo) target = lo;
        if (target > hi) target = hi;
        delta = xsub(target, sigma);
        if (fabs(delta) < COMET_TOL_CM) break;
        const StepK k = make_stepk(delta);
        rkn4_step(s, k, c);
        sigma = xadd(sigma, delta);
    }
    double u0, u1, u2;
    const double d2 = perp2_exact(s.x0, s.x1, s.x2, wl, u0, u1, u2);
    const double c0 = xsub(xmul(s.t1, wl.w2), xmul(s.t2, wl.w1));
    const double c1 = xsub(xmul(s.t2, wl.w0), xmul(s.t0, wl.w2));
    const double c2 = xsub(xmul(s.t0, wl.w1), xmul(s.t1, wl.w0));
    const double side = xdot3(u0, u1, u2, c0, c1, c2);
    const double dist = xsqrt(d2);
    return (side >= 0.0) ? dist : -dist;
}

// ---------------------------------------------------------------------------------------------
// Inhomogeneous field map + adaptive step (readings R29-R32).
// ---------------------------------------------------------------------------------------------
struct FieldMap {
    const double* B;        // [nx][ny][nz][3] Tesla, node (i,j,k) at o + (i dx, j dy, k dz); nullptr = uniform field
    int32_t n[3];
    double o[3], d[3];
    double tol, tol32;      // step tolerance of R31 and tol / 32
    double inv[3];          // 1 / d when every d is a power of two (pow2 = 1): then (x - o) * inv IS the IEEE quotient
    int32_t pow2;           // (x - o) / d, bit for bit -- scaling by a power of two is exact -- at a tenth of its cost
    const double* bmax;     // device scalar: largest |B| of the map (for the step-length bound of the pruning)
};

__device__ __forceinline__ double lerp1(double a, double b, double f) { return xadd(a, xmul(f, xsub(b, a))); }

// R29: trilinear interpolation, z then y then x; outside the grid the edge value.
__device__ __forceinline__ void field_at(const FieldMap& F, double x0, double x1, double x2,
                                         double& b0, double& b1, double& b2)
{
    const double xs[3] = {x0, x1, x2};
    int idx[3];
    double f[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double df = xsub(xs[a], F.o[a]);
        const double t = F.pow2 ? xmul(df, F.inv[a]) : xdiv(df, F.d[a]);
        double fl = floor(t);
        if (fl < 0.0) fl = 0.0;
        if (fl > (double)(F.n[a] - 2)) fl = (double)(F.n[a] - 2);
        idx[a] = (int)fl;
        double fr = xsub(t, fl);
        if (fr < 0.0) fr = 0.0;
        if (fr > 1.0) fr = 1.0;
        f[a] = fr;
    }
    double out[3];
    const size_t sy = (size_t)F.n[2] * 3, sx = (size_t)F.n[1] * sy;
    const double* p = F.B + (size_t)idx[0] * sx + (size_t)idx[1] * sy + (size_t)idx[2] * 3;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double v00 = lerp1(__ldg(p + c), __ldg(p + c + 3), f[2]);
        const double v01 = lerp1(__ldg(p + sy + c), __ldg(p + sy + c + 3), f[2]);
        const double v10 = lerp1(__ldg(p + sx + c), __ldg(p + sx + c + 3), f[2]);
        const double v11 = lerp1(__ldg(p + sx + sy + c), __ldg(p + sx + sy + c + 3), f[2]);
        out[c] = lerp1(lerp1(v00, v01, f[1]), lerp1(v10, v11, f[1]), f[0]);
    }
    b0 = out[0]; b1 = out[1]; b2 = out[2];
}

// k = cq (T x B)
__device__ __forceinline__ void lorentz_rhs(double t0, double t1, double t2, double b0, double b1, double b2,
                                            double cq, double& k0, double& k1, double& k2)
{
    k0 = xmul(cq, xsub(xmul(t1, b2), xmul(t2, b1)));
    k1 = xmul(cq, xsub(xmul(t2, b0), xmul(t0, b2)));
    k2 = xmul(cq, xsub(xmul(t0, b1), xmul(t1, b0)));
}

// R30: one Nystrom RK4 step of signed length h in the field map; returns the error estimate EST.
__device__ __forceinline__ double rkn4_field_step(State& s, double h, double cq, const FieldMap& F)
{
    const double hh = xmul(h, 0.5), h2 = xmul(h, h);
    const double hh8 = xmul(h2, 0.125), hh2 = xmul(h2, 0.5), hh6 = div6(h2), h6 = div6(h);
    const double x[3] = {s.x0, s.x1, s.x2}, T[3] = {s.t0, s.t1, s.t2};
    double b0, b1, b2, k1[3], k2[3], k3[3], k4[3];
    field_at(F, x[0], x[1], x[2], b0, b1, b2);
    lorentz_rhs(T[0], T[1], T[2], b0, b1, b2, cq, k1[0], k1[1], k1[2]);
    field_at(F, xadd(xadd(x[0], xmul(hh, T[0])), xmul(hh8, k1[0])), xadd(xadd(x[1], xmul(hh, T[1])), xmul(hh8, k1[1])),
             xadd(xadd(x[2], xmul(hh, T[2])), xmul(hh8, k1[2])), b0, b1, b2);
    lorentz_rhs(xadd(T[0], xmul(hh, k1[0])), xadd(T[1], xmul(hh, k1[1])), xadd(T[2], xmul(hh, k1[2])), b0, b1, b2, cq,
                k2[0], k2[1], k2[2]);
    lorentz_rhs(xadd(T[0], xmul(hh, k2[0])), xadd(T[1], xmul(hh, k2[1])), xadd(T[2], xmul(hh, k2[2])), b0, b1, b2, cq,
                k3[0], k3[1], k3[2]);
    field_at(F, xadd(xadd(x[0], xmul(h, T[0])), xmul(hh2, k3[0])), xadd(xadd(x[1], xmul(h, T[1])), xmul(hh2, k3[1])),
             xadd(xadd(x[2], xmul(h, T[2])), xmul(hh2, k3[2])), b0, b1, b2);
    lorentz_rhs(xadd(T[0], xmul(h, k3[0])), xadd(T[1], xmul(h, k3[1])), xadd(T[2], xmul(h, k3[2])), b0, b1, b2, cq,
                k4[0], k4[1], k4[2]);
    double est = 0.0, xn[3], tn[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) est = xadd(est, fabs(xadd(xsub(xsub(k1[i], k2[i]), k3[i]), k4[i])));
    est = xmul(h2, est);
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        xn[i] = xadd(xadd(x[i], xmul(h, T[i])), xmul(hh6, xadd(xadd(k1[i], k2[i]), k3[i])));
        tn[i] = xadd(T[i], xmul(h6, xadd(fma(2.0, k3[i], fma(2.0, k2[i], k1[i])), k4[i])));
    }
    s.x0 = xn[0]; s.x1 = xn[1]; s.x2 = xn[2];
    s.t0 = tn[0]; s.t1 = tn[1]; s.t2 = tn[2];
    return est;
}

// R31: one recorded step with the adaptive step control.  `h` is the trial step on entry and the next trial
// step on exit; returns the length of the step taken.
__device__ __forceinline__ double adaptive_field_step(State& s, double& h, double h_max, double h_min, double cq,
                                                      const FieldMap& F)
{
    State t;
    double est;
    for (;;) {
        t = s;
        est = rkn4_field_step(t, h, cq, F);
        if (est > F.tol && h > h_min) { h = xmul(h, 0.5); continue; }
        break;
    }
    s = t;
    const double used = h;
    if (est < F.tol32 && h < h_max) h = xmul(2.0, h);
    return used;
}

// O6 + O7 in the field map: the bracket [lo, hi] is given by the recorded steps around k* (R32).
__device__ __forceinline__ double fine_dca_field(State s, double lo, double hi, double cq, const FieldMap& F,
                                                 const WireLine& wl)
{
    double sigma = 0.0;
#pragma unroll 1
    for (int it = 0; it < COMET_MAX_ITER; ++it) {
        const double tw = xdot3(s.t0, s.t1, s.t2, wl.w0, wl.w1, wl.w2);
        const double n0 = xsub(s.t0, xmul(tw, wl.w0));
        const double n1 = xsub(s.t1, xmul(tw, wl.w1));
        const double n2 = xsub(s.t2, xmul(tw, wl.w2));
        const double den = xdot3(s.t0, s.t1, s.t2, n0, n1, n2);
        if (den < COMET_DEN_MIN) break;
        const double mx0 = xsub(wl.m0, s.x0), mx1 = xsub(wl.m1, s.x1), mx2 = xsub(wl.m2, s.x2);
        double delta = xdiv(xdot3(mx0, mx1, mx2, n0, n1, n2), den);
        double target = xadd(sigma, delta);
        if (target < lo) target = lo;
        if (target > hi) target = hi;
        delta = xsub(target, sigma);
        if (fabs(delta) < COMET_TOL_CM) break;
        (void)rkn4_field_step(s, delta, cq, F);
        sigma = xadd(sigma, delta);
    }
    double u0, u1, u2;
    const double d2 = perp2_exact(s.x0, s.x1, s.x2, wl, u0, u1, u2);
    const double c0 = xsub(xmul(s.t1, wl.w2), xmul(s.t2, wl.w1));
    const double c1 = xsub(xmul(s.t2, wl.w0), xmul(s.t0, wl.w2));
    const double c2 = xsub(xmul(s.t0, wl.w1), xmul(s.t1, wl.w0));
    const double side = xdot3(u0, u1, u2, c0, c1, c2);
    const double dist = xsqrt(d2);
    return (side >= 0.0) ? dist : -dist;
}

// O8: bounded residual of one wire; *jstar = lowest entry index attaining the minimum (-1: none).
__device__ __forceinline__ double wire_residual(double D, const double* __restrict__ rho, int j0, int j1,
                                                double lambda, int* jstar, double* rmin_out)
{
    int js = -1;
    double rmin = 0.0;
    for (int j = j0; j < j1; ++j) {
        const double r = fabs(xsub(D, __ldg(rho + j)));
        if (js < 0 || r < rmin) { rmin = r; js = j; }
    }
    if (jstar) *jstar = js;
    if (rmin_out) *rmin_out = rmin;
    if (js < 0) return lambda;
    return (rmin < lambda) ? rmin : lambda;
}

}  // namespace comet
