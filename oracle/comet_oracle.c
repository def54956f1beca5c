/*
 * comet_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU restatement of the seed x hit scan of arXiv 1911.09340
 * ("GPU-accelerated event reconstruction for the COMET Phase-I experiment"),
 * written from the paper (citations are /root/reference/PAPER.md line numbers)
 * with the readings R1..R23 listed in DESIGN.md.  It shares no code with the
 * CUDA path under paper_1911_09340_b200/ and must never be imported, linked or
 * called by it: only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may use it.
 *
 * Shape: the paper's CPU function, Algorithm 3: one task per
 * seed = record the track (Algorithm 1's loop), then for every
 * wire find the recorded state closest to it and iterate the virtual-plane
 * extrapolation (Algorithm 2, prose :103, :216), accumulate
 * the squared bounded residual of Eq. (1).  OpenMP runs over
 * seeds only, so results do not depend on the thread count.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (no fast-math, no
 * contraction: every operation below is one IEEE-754 double operation in the
 * order written).
 *
 * Parity pins (tests/test_oracle_*_pins.py, tests/test_oracle_golden.py): closed-form helix radius / angular
 * advance / pitch, |T| conservation, straight-line limit, reversibility, axial
 * wire closed form, brute-force dense sampling, rotation / translation / endpoint
 * swap symmetries, truth-seed RSS = injected smearing, RSS bounds, brute-force
 * argmin and classification.  No function here is "parity unpinned".
 *
 * Units: cm, MeV/c, Tesla, charge in e.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* R4: "0.3 B" of PAPER.md:319 Eq. (2), in (MeV/c)/(T cm). */
#define ORACLE_KAPPA 2.99792458
/* R9: TOLERANCE of PAPER.md:173 and the iteration cap. */
#define ORACLE_TOL_CM 1e-9
#define ORACLE_MAX_ITER 16

typedef struct {
    double x[3];
    double T[3];
} ostate;

/* f(T) = c (T x z_hat) = c (Ty, -Tx, 0): the uniform-B_z equation of motion (O1). */
static void field_rhs(const double T[3], double c, double k[3])
{
    k[0] = c * T[1];
    k[1] = -(c * T[0]);
    k[2] = 0.0;
}

/* O2 / R1: one classical 4th-order Runge-Kutta-Nystrom step of signed length h
 * (method of ref [7]).  T is not renormalised. */
static void rkn4_step(ostate* s, double h, double c)
{
    double k1[3], k2[3], k3[3], k4[3], t[3];
    int i;
    field_rhs(s->T, c, k1);
    for (i = 0; i < 3; ++i) t[i] = s->T[i] + (h / 2.0) * k1[i];
    field_rhs(t, c, k2);
    for (i = 0; i < 3; ++i) t[i] = s->T[i] + (h / 2.0) * k2[i];
    field_rhs(t, c, k3);
    for (i = 0; i < 3; ++i) t[i] = s->T[i] + h * k3[i];
    field_rhs(t, c, k4);
    for (i = 0; i < 3; ++i) {
        s->x[i] = s->x[i] + h * s->T[i] + ((h * h) / 6.0) * (k1[i] + k2[i] + k3[i]);
    }
    for (i = 0; i < 3; ++i) {
        s->T[i] = s->T[i] + (h / 6.0) * (k1[i] + 2.0 * k2[i] + 2.0 * k3[i] + k4[i]);
    }
}

/* O1 + O3: Algorithm 1.  pts has room for n_steps+1 states.
 * R3: targetRegion = first recorded point with r < r_stop moving inward. */
static int record_track(const double seed[6], int charge, double bz, double h, int n_steps,
                        double r_stop, ostate* pts)
{
    double P = sqrt(seed[3] * seed[3] + seed[4] * seed[4] + seed[5] * seed[5]);
    double c = ORACLE_KAPPA * (double)charge * bz / P;
    int k, n_pts = n_steps + 1;
    pts[0].x[0] = seed[0]; pts[0].x[1] = seed[1]; pts[0].x[2] = seed[2];
    pts[0].T[0] = seed[3] / P; pts[0].T[1] = seed[4] / P; pts[0].T[2] = seed[5] / P;
    for (k = 1; k <= n_steps; ++k) {
        pts[k] = pts[k - 1];
        rkn4_step(&pts[k], h, c);
        if (r_stop > 0.0) {
            double r2 = pts[k].x[0] * pts[k].x[0] + pts[k].x[1] * pts[k].x[1];
            double rad = pts[k].x[0] * pts[k].T[0] + pts[k].x[1] * pts[k].T[1];
            if (r2 < r_stop * r_stop && rad < 0.0) { n_pts = k + 1; break; }
        }
    }
    return n_pts;
}

static double dot3(const double a[3], const double b[3])
{
    return a[0] * b[0] + a[1] * b[1] + a[2] * b[2];
}

/* O4: perp(x) = (x - m) - ((x - m) . w) w, the vector from the infinite wire line
 * (R5) to x, measured from the wire midpoint m. */
static void perp_to_wire(const double x[3], const double m[3], const double w[3], double u[3])
{
    double d[3], t;
    int i;
    for (i = 0; i < 3; ++i) d[i] = x[i] - m[i];
    t = dot3(d, w);
    for (i = 0; i < 3; ++i) u[i] = d[i] - t * w[i];
}

/* O5..O7: Algorithm 2 lines 6-15 for one (track, wire): returns the signed DCA,
 * writes the index of the closest recorded state to *kstar_out. */
static double wire_dca(const ostate* pts, int n_pts, double h, double c,
                       const double m[3], const double w[3], int* kstar_out)
{
    int k, kstar = 0, it;
    double best = 0.0, u[3], sigma = 0.0, lo, hi, cross[3], side, dist;
    ostate s;
    /* O5 / R6: closest recorded state, squared perpendicular distance, ties -> lowest k
     * ("Find state (in params) closest to geom"). */
    for (k = 0; k < n_pts; ++k) {
        double d2;
        perp_to_wire(pts[k].x, m, w, u);
        d2 = dot3(u, u);
        if (k == 0 || d2 < best) { best = d2; kstar = k; }
    }
    /* O6 / R7, R8, R10: virtual plane through the wire whose normal is the part of
     * the momentum direction perpendicular to the wire; step by the
     * path length to that plane; total offset kept inside [s_{k*-1}, s_{k*+1}]. */
    s = pts[kstar];
    lo = (kstar > 0) ? -h : 0.0;
    hi = (kstar < n_pts - 1) ? h : 0.0;
    for (it = 0; it < ORACLE_MAX_ITER; ++it) {
        double nv[3], tw, den, mx[3], delta, target;
        int i;
        tw = dot3(s.T, w);
        for (i = 0; i < 3; ++i) nv[i] = s.T[i] - tw * w[i];
        den = dot3(s.T, nv);
        if (den < 1e-12) break;
        for (i = 0; i < 3; ++i) mx[i] = m[i] - s.x[i];
        delta = dot3(mx, nv) / den;
        target = sigma + delta;
        if (target < lo) target = lo;
        if (target > hi) target = hi;
        delta = target - sigma;
        if (fabs(delta) < ORACLE_TOL_CM) break;
        rkn4_step(&s, delta, c);
        sigma = sigma + delta;
    }
    /* O7 / R16: signed DCA, + when u . (T x w) >= 0. */
    perp_to_wire(s.x, m, w, u);
    cross[0] = s.T[1] * w[2] - s.T[2] * w[1];
    cross[1] = s.T[2] * w[0] - s.T[0] * w[2];
    cross[2] = s.T[0] * w[1] - s.T[1] * w[0];
    side = dot3(u, cross);
    dist = sqrt(dot3(u, u));
    if (kstar_out) *kstar_out = kstar;
    return (side >= 0.0) ? dist : -dist;
}

/* O4: unit direction and midpoint of fired wire i. */
static void wire_line(const double* wire_a, const double* wire_b, int n_wires, int wi,
                      double m[3], double w[3])
{
    double d[3], len;
    int i;
    for (i = 0; i < 3; ++i) d[i] = wire_b[(size_t)i * n_wires + wi] - wire_a[(size_t)i * n_wires + wi];
    len = sqrt(dot3(d, d));
    for (i = 0; i < 3; ++i) {
        w[i] = d[i] / len;
        m[i] = (wire_a[(size_t)i * n_wires + wi] + wire_b[(size_t)i * n_wires + wi]) / 2.0;
    }
}

/* O8: bounded residual of one wire, Eq. (1): min over the wire's hit
 * entries (ghosts explicit, R12) of |D - rho_j|, capped at lambda.  *jstar = lowest
 * index attaining the minimum (-1 when the wire has no entries). */
static double wire_residual(double D, const double* rho, int j0, int j1, double lambda,
                            int* jstar, double* rmin_out)
{
    int j, js = -1;
    double rmin = 0.0;
    for (j = j0; j < j1; ++j) {
        double r = fabs(D - rho[j]);
        if (js < 0 || r < rmin) { rmin = r; js = j; }
    }
    if (jstar) *jstar = js;
    if (rmin_out) *rmin_out = rmin;
    if (js < 0) return lambda;
    return (rmin < lambda) ? rmin : lambda;
}

/* One seed of Algorithm 3 given its recorded track. */
static double seed_rss(const ostate* pts, int n_pts, double h, double c,
                       const double* wire_a, const double* wire_b, int n_wires,
                       const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                       int n_fired, double lambda, double* dca_row, int32_t* kstar_row)
{
    double rss = 0.0;
    int i;
    for (i = 0; i < n_fired; ++i) {            /* O9: increasing wire order */
        double m[3], w[3], D, e;
        int ks;
        wire_line(wire_a, wire_b, n_wires, fired_wire[i], m, w);
        D = wire_dca(pts, n_pts, h, c, m, w, &ks);
        e = wire_residual(D, rho, hit_off[i], hit_off[i + 1], lambda, NULL, NULL);
        rss = rss + e * e;
        if (dca_row) dca_row[i] = D;
        if (kstar_row) kstar_row[i] = ks;
    }
    return rss;
}

static double seed_curvature(const double* seeds, int64_t n_seeds, int64_t s, int charge, double bz,
                             double seed[6])
{
    int i;
    double P;
    for (i = 0; i < 6; ++i) seed[i] = seeds[(size_t)i * n_seeds + s];
    P = sqrt(seed[3] * seed[3] + seed[4] * seed[4] + seed[5] * seed[5]);
    return ORACLE_KAPPA * (double)charge * bz / P;
}

/* ------------------------------------------------------------------------ */
/* exported                                                                 */
/* ------------------------------------------------------------------------ */

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* Algorithm 1 alone: track [n_seeds][n_steps+1][6] = x,y,z,Tx,Ty,Tz (NaN beyond n_pts). */
void oracle_extrapolate(const double* seeds, int64_t n_seeds, int charge, double bz,
                        double step, int n_steps, double r_stop,
                        double* track, int32_t* n_pts)
{
    int64_t s;
#pragma omp parallel for schedule(dynamic, 16)
    for (s = 0; s < n_seeds; ++s) {
        ostate* pts = (ostate*)malloc(sizeof(ostate) * (size_t)(n_steps + 1));
        double seed[6];
        int k, np;
        (void)seed_curvature(seeds, n_seeds, s, charge, bz, seed);
        np = record_track(seed, charge, bz, step, n_steps, r_stop, pts);
        n_pts[s] = np;
        for (k = 0; k <= n_steps; ++k) {
            double* o = track + ((size_t)s * (size_t)(n_steps + 1) + (size_t)k) * 6;
            int i;
            for (i = 0; i < 3; ++i) {
                o[i] = (k < np) ? pts[k].x[i] : NAN;
                o[3 + i] = (k < np) ? pts[k].T[i] : NAN;
            }
        }
        free(pts);
    }
}

/* Algorithm 3 over all seeds: rss[n_seeds]; optional dca[n_seeds][n_fired] (signed),
 * kstar[n_seeds][n_fired], n_pts[n_seeds]. */
void oracle_scan(const double* seeds, int64_t n_seeds, int charge, double bz,
                 double step, int n_steps, double r_stop,
                 const double* wire_a, const double* wire_b, int n_wires,
                 const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                 int n_fired, double cutoff,
                 double* rss, double* dca, int32_t* kstar, int32_t* n_pts)
{
    int64_t s;
#pragma omp parallel
    {
        ostate* pts = (ostate*)malloc(sizeof(ostate) * (size_t)(n_steps + 1));
#pragma omp for schedule(dynamic, 16)
        for (s = 0; s < n_seeds; ++s) {
            double seed[6];
            double c = seed_curvature(seeds, n_seeds, s, charge, bz, seed);
            int np = record_track(seed, charge, bz, step, n_steps, r_stop, pts);
            if (n_pts) n_pts[s] = np;
            rss[s] = seed_rss(pts, np, step, c, wire_a, wire_b, n_wires, fired_wire, hit_off, rho,
                              n_fired, cutoff,
                              dca ? dca + (size_t)s * (size_t)n_fired : NULL,
                              kstar ? kstar + (size_t)s * (size_t)n_fired : NULL);
        }
        free(pts);
    }
}

/* O10 + O11: per partition the lowest-index argmin of rss, then the
 * classification rule of PAPER.md:83 for that seed: on every fired wire the closest
 * hit entry is classified iff its residual is < lambda (R13 strict).
 * best_dca [n_part][n_fired], cls [n_part][n_hits] (0/1). */
void oracle_select_classify(const double* seeds, int64_t n_seeds, int charge, double bz,
                            double step, int n_steps, double r_stop,
                            const double* wire_a, const double* wire_b, int n_wires,
                            const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                            int n_fired, int n_hits, double cutoff,
                            const double* rss, const int64_t* part_off, int n_part,
                            int64_t* best_seed, double* best_rss, double* best_dca, uint8_t* cls)
{
    int p;
    ostate* pts = (ostate*)malloc(sizeof(ostate) * (size_t)(n_steps + 1));
    for (p = 0; p < n_part; ++p) {
        int64_t s, b = -1;
        double seed[6], c;
        int np, i;
        for (s = part_off[p]; s < part_off[p + 1]; ++s) {
            if (b < 0 || rss[s] < rss[b]) b = s;
        }
        best_seed[p] = b;
        memset(cls + (size_t)p * (size_t)n_hits, 0, (size_t)n_hits);
        if (b < 0) {
            best_rss[p] = NAN;
            for (i = 0; i < n_fired; ++i) best_dca[(size_t)p * n_fired + i] = NAN;
            continue;
        }
        best_rss[p] = rss[b];
        c = seed_curvature(seeds, n_seeds, b, charge, bz, seed);
        np = record_track(seed, charge, bz, step, n_steps, r_stop, pts);
        for (i = 0; i < n_fired; ++i) {
            double m[3], w[3], D, rmin;
            int js;
            wire_line(wire_a, wire_b, n_wires, fired_wire[i], m, w);
            D = wire_dca(pts, np, step, c, m, w, NULL);
            best_dca[(size_t)p * n_fired + i] = D;
            (void)wire_residual(D, rho, hit_off[i], hit_off[i + 1], cutoff, &js, &rmin);
            if (js >= 0 && rmin < cutoff) cls[(size_t)p * (size_t)n_hits + js] = 1;
        }
    }
    free(pts);
}

/* Single RKN4 step exposed for the pin tests (state = x,y,z,Tx,Ty,Tz; c = kappa q Bz / |p|). */
void oracle_rkn4_step(double* state6, double h, double c)
{
    ostate s;
    int i;
    for (i = 0; i < 3; ++i) { s.x[i] = state6[i]; s.T[i] = state6[3 + i]; }
    rkn4_step(&s, h, c);
    for (i = 0; i < 3; ++i) { state6[i] = s.x[i]; state6[3 + i] = s.T[i]; }
}

double oracle_kappa(void) { return ORACLE_KAPPA; }

/* ------------------------------------------------------------------------------------------
 * Iterative seed refinement (readings R24-R27 of DESIGN.md).
 *
 * "several seeds with the lowest RSS are selected as reference points for the next seed
 * scanning, where new seeds are fetched in their vicinity and with a finer granularity. [...]
 * the selected seeds are ensured to be sparse enough to avoid overlaps between new seed sets
 * from each reference point."
 *
 * The scanned seed components are the paper's (z, p_x, p_y, p_z) at fixed (x, y), i.e. fixed
 * azimuth on the R = 50 cm cylinder: dimension d = 0..3 is seed component 2 + d.
 * The new seed set of a reference point is the box ref_d +- half_width_d; two boxes overlap iff
 * |ref_a,d - ref_b,d| < 2 half_width_d in every dimension (strict).
 * ------------------------------------------------------------------------------------------ */

/* 1 iff the refinement boxes around seeds a and b overlap (R25). */
static int boxes_overlap(const double* seeds, int64_t n_seeds, int64_t a, int64_t b, const double* half_width)
{
    int d;
    for (d = 0; d < 4; ++d) {
        const double* comp = seeds + (size_t)(2 + d) * (size_t)n_seeds;
        const double two_hw = 2.0 * half_width[d];
        if (!(fabs(comp[a] - comp[b]) < two_hw)) return 0;
    }
    return 1;
}

/* O12: per partition, up to k_ref reference points: repeatedly the seed of lowest RSS (ties ->
 * lowest index; NaN never) among those that are not selected yet and whose box overlaps no
 * selected box.  ref_seed [n_part][k_ref], -1 where no seed is left. */
void oracle_select_references(const double* seeds, int64_t n_seeds, const double* rss,
                              const int64_t* part_off, int n_part, const double* half_width,
                              int k_ref, int64_t* ref_seed)
{
    int p, r, q;
    for (p = 0; p < n_part; ++p) {
        int64_t* sel = ref_seed + (size_t)p * (size_t)k_ref;
        for (r = 0; r < k_ref; ++r) sel[r] = -1;
        for (r = 0; r < k_ref; ++r) {
            int64_t s, best = -1;
            for (s = part_off[p]; s < part_off[p + 1]; ++s) {
                int blocked = 0;
                if (rss[s] != rss[s]) continue;
                for (q = 0; q < r && !blocked; ++q)
                    if (sel[q] == s || boxes_overlap(seeds, n_seeds, s, sel[q], half_width)) blocked = 1;
                if (blocked) continue;
                if (best < 0 || rss[s] < rss[best]) best = s;
            }
            if (best < 0) break;
            sel[r] = best;
        }
    }
}

/* O13: the new seed set.  Slot (p, r) holds G = n_grid[0] n_grid[1] n_grid[2] n_grid[3] seeds
 * around reference ref_seed[p][r] (an empty slot repeats the partition's first reference, R27):
 * component 2 + d takes the n_grid[d] values lo + j step, lo = ref_d - half_width_d,
 * step = (2 half_width_d) / (n_grid[d] - 1)   (n_grid[d] = 1: the reference's own value);
 * (x, y) are the reference's.  Seed index within the slot: ((j0 n1 + j1) n2 + j2) n3 + j3.
 * new_seeds is SoA [6][n_part k_ref G]. */
void oracle_refine_seeds(const double* seeds, int64_t n_seeds, const int64_t* ref_seed, int n_part,
                         int k_ref, const double* half_width, const int32_t* n_grid,
                         double* new_seeds)
{
    const int64_t G = (int64_t)n_grid[0] * n_grid[1] * n_grid[2] * n_grid[3];
    const int64_t S_new = (int64_t)n_part * k_ref * G;
    int p, r, d;
    for (p = 0; p < n_part; ++p) {
        for (r = 0; r < k_ref; ++r) {
            int64_t ref = ref_seed[(size_t)p * k_ref + r];
            int64_t g, base = ((int64_t)p * k_ref + r) * G;
            double lo[4], stp[4];
            if (ref < 0) ref = ref_seed[(size_t)p * k_ref];
            for (d = 0; d < 4; ++d) {
                const double v = seeds[(size_t)(2 + d) * (size_t)n_seeds + ref];
                if (n_grid[d] > 1) {
                    lo[d] = v - half_width[d];
                    stp[d] = (2.0 * half_width[d]) / (double)(n_grid[d] - 1);
                } else {
                    lo[d] = v;
                    stp[d] = 0.0;
                }
            }
            for (g = 0; g < G; ++g) {
                int64_t rem = g;
                int j[4];
                for (d = 3; d >= 0; --d) { j[d] = (int)(rem % n_grid[d]); rem /= n_grid[d]; }
                new_seeds[0 * S_new + base + g] = seeds[0 * (size_t)n_seeds + ref];
                new_seeds[1 * S_new + base + g] = seeds[1 * (size_t)n_seeds + ref];
                for (d = 0; d < 4; ++d)
                    new_seeds[(size_t)(2 + d) * S_new + base + g] = lo[d] + (double)j[d] * stp[d];
            }
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * Inhomogeneous field map and adaptive step ("RKN method [7] with an adaptive step
 * size that adjusts to the roughness of the magnetic field", :99 "BFields in the grid format",
 * :135-136; readings R29-R32 of DESIGN.md).  Separate functions: the uniform-field ones above
 * stay as pinned.
 * ------------------------------------------------------------------------------------------ */
typedef struct {
    const double* B;     /* [nx][ny][nz][3] Tesla, node (i,j,k) at o + (i dx, j dy, k dz) */
    int n[3];
    double o[3], d[3];
} ofield;

static double lerp1(double a, double b, double f) { return a + f * (b - a); }

/* R29: trilinear interpolation, z then y then x; outside the grid the edge value (clamped). */
static void field_at(const ofield* F, const double x[3], double B[3])
{
    int idx[3], a, c;
    double f[3];
    for (a = 0; a < 3; ++a) {
        double t = (x[a] - F->o[a]) / F->d[a];
        double fl = floor(t);
        if (fl < 0.0) fl = 0.0;
        if (fl > (double)(F->n[a] - 2)) fl = (double)(F->n[a] - 2);
        idx[a] = (int)fl;
        f[a] = t - fl;
        if (f[a] < 0.0) f[a] = 0.0;
        if (f[a] > 1.0) f[a] = 1.0;
    }
    for (c = 0; c < 3; ++c) {
        double v[2][2];
        int di, dj;
        for (di = 0; di < 2; ++di)
            for (dj = 0; dj < 2; ++dj) {
                size_t base = (((size_t)(idx[0] + di) * F->n[1] + (size_t)(idx[1] + dj)) * F->n[2] + (size_t)idx[2]) * 3 + c;
                v[di][dj] = lerp1(F->B[base], F->B[base + 3], f[2]);
            }
        B[c] = lerp1(lerp1(v[0][0], v[0][1], f[1]), lerp1(v[1][0], v[1][1], f[1]), f[0]);
    }
}

/* k = cq (T x B), cq = kappa q / |p|. */
static void lorentz_rhs(const double T[3], const double B[3], double cq, double k[3])
{
    k[0] = cq * (T[1] * B[2] - T[2] * B[1]);
    k[1] = cq * (T[2] * B[0] - T[0] * B[2]);
    k[2] = cq * (T[0] * B[1] - T[1] * B[0]);
}

/* R30: one Nystrom RK4 step of signed length h in the field map: field at x, at the midpoint
 * x + h/2 T + h^2/8 k1 (used for k2 and k3) and at the end point x + h T + h^2/2 k3.  Returns the
 * error estimate EST = h^2 (|k1-k2-k3+k4|_x + |.|_y + |.|_z) of the method of ref [7]. */
static double rkn4_field_step(ostate* s, double h, double cq, const ofield* F)
{
    double B[3], k1[3], k2[3], k3[3], k4[3], t[3], xm[3], est = 0.0;
    int i;
    field_at(F, s->x, B);
    lorentz_rhs(s->T, B, cq, k1);
    for (i = 0; i < 3; ++i) xm[i] = s->x[i] + (h / 2.0) * s->T[i] + ((h * h) / 8.0) * k1[i];
    field_at(F, xm, B);
    for (i = 0; i < 3; ++i) t[i] = s->T[i] + (h / 2.0) * k1[i];
    lorentz_rhs(t, B, cq, k2);
    for (i = 0; i < 3; ++i) t[i] = s->T[i] + (h / 2.0) * k2[i];
    lorentz_rhs(t, B, cq, k3);
    for (i = 0; i < 3; ++i) xm[i] = s->x[i] + h * s->T[i] + ((h * h) / 2.0) * k3[i];
    field_at(F, xm, B);
    for (i = 0; i < 3; ++i) t[i] = s->T[i] + h * k3[i];
    lorentz_rhs(t, B, cq, k4);
    for (i = 0; i < 3; ++i) est = est + fabs(((k1[i] - k2[i]) - k3[i]) + k4[i]);
    est = (h * h) * est;
    for (i = 0; i < 3; ++i) s->x[i] = s->x[i] + h * s->T[i] + ((h * h) / 6.0) * (k1[i] + k2[i] + k3[i]);
    for (i = 0; i < 3; ++i) s->T[i] = s->T[i] + (h / 6.0) * (k1[i] + 2.0 * k2[i] + 2.0 * k3[i] + k4[i]);
    return est;
}

/* R31: Algorithm 1 with the adaptive step.  The trial step starts at h_max; a step whose EST
 * exceeds tol is retried with half the length (not below h_max/64); after an accepted step with
 * EST < tol/32 the trial step doubles (not above h_max).  hs[k] = length of the step from state
 * k to state k+1.  Stop rule R3 as in record_track. */
static int record_track_field(const double seed[6], int charge, const ofield* F, double h_max, int n_steps,
                              double r_stop, double tol, ostate* pts, double* hs)
{
    double P = sqrt(seed[3] * seed[3] + seed[4] * seed[4] + seed[5] * seed[5]);
    double cq = ORACLE_KAPPA * (double)charge / P;
    double h = h_max, h_min = h_max / 64.0;
    int k, n_pts = n_steps + 1;
    pts[0].x[0] = seed[0]; pts[0].x[1] = seed[1]; pts[0].x[2] = seed[2];
    pts[0].T[0] = seed[3] / P; pts[0].T[1] = seed[4] / P; pts[0].T[2] = seed[5] / P;
    for (k = 1; k <= n_steps; ++k) {
        double est;
        for (;;) {
            pts[k] = pts[k - 1];
            est = rkn4_field_step(&pts[k], h, cq, F);
            if (est > tol && h > h_min) { h = h / 2.0; continue; }
            break;
        }
        hs[k - 1] = h;
        if (est < tol / 32.0 && h < h_max) h = 2.0 * h;
        if (r_stop > 0.0) {
            double r2 = pts[k].x[0] * pts[k].x[0] + pts[k].x[1] * pts[k].x[1];
            double rad = pts[k].x[0] * pts[k].T[0] + pts[k].x[1] * pts[k].T[1];
            if (r2 < r_stop * r_stop && rad < 0.0) { n_pts = k + 1; break; }
        }
    }
    return n_pts;
}

/* O5..O7 in the field map: as wire_dca, the sub-steps are field steps (PAPER.md:180
 * "RKN(state, distance, BFields)") and the bracket is the two recorded steps around k* (R32). */
static double wire_dca_field(const ostate* pts, const double* hs, int n_pts, double cq, const ofield* F,
                             const double m[3], const double w[3], int* kstar_out)
{
    int k, kstar = 0, it;
    double best = 0.0, u[3], sigma = 0.0, lo, hi, cross[3], side, dist;
    ostate s;
    for (k = 0; k < n_pts; ++k) {
        double d2;
        perp_to_wire(pts[k].x, m, w, u);
        d2 = dot3(u, u);
        if (k == 0 || d2 < best) { best = d2; kstar = k; }
    }
    s = pts[kstar];
    lo = (kstar > 0) ? -hs[kstar - 1] : 0.0;
    hi = (kstar < n_pts - 1) ? hs[kstar] : 0.0;
    for (it = 0; it < ORACLE_MAX_ITER; ++it) {
        double nv[3], tw, den, mx[3], delta, target;
        int i;
        tw = dot3(s.T, w);
        for (i = 0; i < 3; ++i) nv[i] = s.T[i] - tw * w[i];
        den = dot3(s.T, nv);
        if (den < 1e-12) break;
        for (i = 0; i < 3; ++i) mx[i] = m[i] - s.x[i];
        delta = dot3(mx, nv) / den;
        target = sigma + delta;
        if (target < lo) target = lo;
        if (target > hi) target = hi;
        delta = target - sigma;
        if (fabs(delta) < ORACLE_TOL_CM) break;
        (void)rkn4_field_step(&s, delta, cq, F);
        sigma = sigma + delta;
    }
    perp_to_wire(s.x, m, w, u);
    cross[0] = s.T[1] * w[2] - s.T[2] * w[1];
    cross[1] = s.T[2] * w[0] - s.T[0] * w[2];
    cross[2] = s.T[0] * w[1] - s.T[1] * w[0];
    side = dot3(u, cross);
    dist = sqrt(dot3(u, u));
    if (kstar_out) *kstar_out = kstar;
    return (side >= 0.0) ? dist : -dist;
}

static ofield make_field(const double* B, const int32_t* n, const double* o, const double* d)
{
    ofield F;
    int a;
    F.B = B;
    for (a = 0; a < 3; ++a) { F.n[a] = n[a]; F.o[a] = o[a]; F.d[a] = d[a]; }
    return F;
}

/* pins */
void oracle_field_at(const double* B, const int32_t* n, const double* o, const double* d,
                     const double* x3, double* out3)
{
    ofield F = make_field(B, n, o, d);
    field_at(&F, x3, out3);
}

double oracle_rkn4_field_step(const double* B, const int32_t* n, const double* o, const double* d,
                              double* state6, double h, double cq)
{
    ofield F = make_field(B, n, o, d);
    ostate s;
    double est;
    int i;
    for (i = 0; i < 3; ++i) { s.x[i] = state6[i]; s.T[i] = state6[3 + i]; }
    est = rkn4_field_step(&s, h, cq, &F);
    for (i = 0; i < 3; ++i) { state6[i] = s.x[i]; state6[3 + i] = s.T[i]; }
    return est;
}

/* Algorithm 1 in the field map: track [n_seeds][n_steps+1][6] (NaN beyond n_pts), n_pts [n_seeds],
 * hs [n_seeds][n_steps] step lengths (NaN beyond n_pts-1). */
void oracle_extrapolate_field(const double* seeds, int64_t n_seeds, int charge,
                              const double* B, const int32_t* n, const double* o, const double* d,
                              double h_max, int n_steps, double r_stop, double tol,
                              double* track, int32_t* n_pts, double* hs_out)
{
    ofield F = make_field(B, n, o, d);
    int64_t s;
#pragma omp parallel for schedule(dynamic, 16)
    for (s = 0; s < n_seeds; ++s) {
        ostate* pts = (ostate*)malloc(sizeof(ostate) * (size_t)(n_steps + 1));
        double* hs = (double*)malloc(sizeof(double) * (size_t)n_steps);
        double seed[6];
        int i, k, np;
        for (i = 0; i < 6; ++i) seed[i] = seeds[(size_t)i * n_seeds + s];
        np = record_track_field(seed, charge, &F, h_max, n_steps, r_stop, tol, pts, hs);
        n_pts[s] = np;
        for (k = 0; k <= n_steps; ++k) {
            double* row = track + ((size_t)s * (size_t)(n_steps + 1) + (size_t)k) * 6;
            for (i = 0; i < 3; ++i) {
                row[i] = (k < np) ? pts[k].x[i] : NAN;
                row[3 + i] = (k < np) ? pts[k].T[i] : NAN;
            }
            if (k < n_steps) hs_out[(size_t)s * n_steps + k] = (k < np - 1) ? hs[k] : NAN;
        }
        free(pts);
        free(hs);
    }
}

/* Algorithm 3 in the field map (as oracle_scan). */
void oracle_scan_field(const double* seeds, int64_t n_seeds, int charge,
                       const double* B, const int32_t* n, const double* o, const double* d,
                       double h_max, int n_steps, double r_stop, double tol,
                       const double* wire_a, const double* wire_b, int n_wires,
                       const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                       int n_fired, double cutoff, double* rss, double* dca, int32_t* kstar, int32_t* n_pts)
{
    ofield F = make_field(B, n, o, d);
    int64_t s;
#pragma omp parallel for schedule(dynamic, 16)
    for (s = 0; s < n_seeds; ++s) {
        ostate* pts = (ostate*)malloc(sizeof(ostate) * (size_t)(n_steps + 1));
        double* hs = (double*)malloc(sizeof(double) * (size_t)n_steps);
        double seed[6], P, cq, acc = 0.0;
        int i, np;
        for (i = 0; i < 6; ++i) seed[i] = seeds[(size_t)i * n_seeds + s];
        P = sqrt(seed[3] * seed[3] + seed[4] * seed[4] + seed[5] * seed[5]);
        cq = ORACLE_KAPPA * (double)charge / P;
        np = record_track_field(seed, charge, &F, h_max, n_steps, r_stop, tol, pts, hs);
        if (n_pts) n_pts[s] = np;
        for (i = 0; i < n_fired; ++i) {
            double m[3], w[3], D, e;
            int ks;
            wire_line(wire_a, wire_b, n_wires, fired_wire[i], m, w);
            D = wire_dca_field(pts, hs, np, cq, &F, m, w, &ks);
            e = wire_residual(D, rho, hit_off[i], hit_off[i + 1], cutoff, NULL, NULL);
            acc = acc + e * e;
            if (dca) dca[(size_t)s * n_fired + i] = D;
            if (kstar) kstar[(size_t)s * n_fired + i] = ks;
        }
        rss[s] = acc;
        free(pts);
        free(hs);
    }
}

/* O11 in the field map for the listed seeds: dca [n_sel][n_fired], cls [n_sel][n_hits]. */
void oracle_classify_seeds_field(const double* seeds, int64_t n_seeds, int charge,
                                 const double* B, const int32_t* n, const double* o, const double* d,
                                 double h_max, int n_steps, double r_stop, double tol,
                                 const double* wire_a, const double* wire_b, int n_wires,
                                 const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                                 int n_fired, int n_hits, double cutoff,
                                 const int64_t* seed_idx, int n_sel, double* dca, uint8_t* cls)
{
    ofield F = make_field(B, n, o, d);
    ostate* pts = (ostate*)malloc(sizeof(ostate) * (size_t)(n_steps + 1));
    double* hs = (double*)malloc(sizeof(double) * (size_t)n_steps);
    int q;
    for (q = 0; q < n_sel; ++q) {
        int64_t s = seed_idx[q];
        double seed[6], P, cq;
        int i, np;
        memset(cls + (size_t)q * (size_t)n_hits, 0, (size_t)n_hits);
        if (s < 0) {
            for (i = 0; i < n_fired; ++i) dca[(size_t)q * n_fired + i] = NAN;
            continue;
        }
        for (i = 0; i < 6; ++i) seed[i] = seeds[(size_t)i * n_seeds + s];
        P = sqrt(seed[3] * seed[3] + seed[4] * seed[4] + seed[5] * seed[5]);
        cq = ORACLE_KAPPA * (double)charge / P;
        np = record_track_field(seed, charge, &F, h_max, n_steps, r_stop, tol, pts, hs);
        for (i = 0; i < n_fired; ++i) {
            double m[3], w[3], D, rmin;
            int js;
            wire_line(wire_a, wire_b, n_wires, fired_wire[i], m, w);
            D = wire_dca_field(pts, hs, np, cq, &F, m, w, NULL);
            dca[(size_t)q * n_fired + i] = D;
            (void)wire_residual(D, rho, hit_off[i], hit_off[i + 1], cutoff, &js, &rmin);
            if (js >= 0 && rmin < cutoff) cls[(size_t)q * (size_t)n_hits + js] = 1;
        }
    }
    free(pts);
    free(hs);
}
