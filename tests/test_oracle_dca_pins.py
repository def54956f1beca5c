"""Pins for the oracle's DCA finder (O4-O7; PAPER.md:150-185 Algorithm 2, prose :103, :216).

Expected values never come from the oracle's own formulas: they are the textbook
line-line distance (B = 0), the closed form for an axial wire (distance from the
helix axis minus the radius), a dense brute-force sampling of the analytic helix,
hand-computed toy cases, and symmetries of the geometry.
"""
import math

import numpy as np
import pytest

from oracle import comet_oracle as O

KAPPA = 2.99792458


def _seed(x, p):
    return np.array([[x[0]], [x[1]], [x[2]], [p[0]], [p[1]], [p[2]]], dtype=np.float64)


def _wires(a_list, b_list):
    """SoA [3][n] endpoint arrays from lists of 3-vectors."""
    return (np.ascontiguousarray(np.array(a_list, dtype=np.float64).T),
            np.ascontiguousarray(np.array(b_list, dtype=np.float64).T))


def _scan_dca(seeds, q, bz, h, n, r_stop, wa, wb, cutoff=0.1, rho=None):
    """Signed DCA of every wire (one dummy hit entry each) to every seed's track."""
    W = wa.shape[1]
    fired = np.arange(W, dtype=np.int32)
    hit_off = np.arange(W + 1, dtype=np.int32)
    if rho is None:
        rho = np.zeros(W)
    return O.scan(seeds, q, bz, h, n, r_stop, wa, wb, fired, hit_off, rho, cutoff,
                  want_dca=True, want_kstar=True, want_npts=True)


def _helix_xy(x0, T0, c, s):
    """Analytic transverse position/tangent at arc length s (complex numbers)."""
    t = (T0[0] + 1j * T0[1]) * np.exp(-1j * c * s)
    x = (x0[0] + 1j * x0[1]) + (T0[0] + 1j * T0[1]) * (1 - np.exp(-1j * c * s)) / (1j * c)
    return x, t


def test_sign_convention_and_magnitude_hand_case():
    """Straight track along +x through the origin, wire parallel to z through (3, +1):
    closest approach at x = 3, distance 1.  u = x - wire = (0,-1,0), T x w = x^ x z^ = -y^,
    so u . (T x w) = +1 and the signed DCA is +1 (reading R16).  Wire at y = -2 gives -2."""
    wa, wb = _wires([[3, 1, -50], [3, -2, -50]], [[3, 1, 50], [3, -2, 50]])
    r = _scan_dca(_seed([0, 0, 0], [100, 0, 0]), -1, 0.0, 0.5, 40, 0.0, wa, wb)
    assert abs(r["dca"][0, 0] - 1.0) < 1e-14
    assert abs(r["dca"][0, 1] + 2.0) < 1e-14
    assert r["kstar"][0, 0] == 6 and r["kstar"][0, 1] == 6        # x_k = 0.5 k -> k = 6 at x = 3
    # swapping the endpoints flips w and therefore the sign
    r2 = _scan_dca(_seed([0, 0, 0], [100, 0, 0]), -1, 0.0, 0.5, 40, 0.0, wb, wa)
    np.testing.assert_allclose(r2["dca"], -r["dca"], rtol=0, atol=1e-15)


def test_closest_recorded_state_tie_goes_to_lowest_k():
    """Wire at x = 3.25 is exactly midway between recorded x = 3.0 (k = 6) and 3.5 (k = 7)."""
    wa, wb = _wires([[3.25, 1, -50]], [[3.25, 1, 50]])
    r = _scan_dca(_seed([0, 0, 0], [100, 0, 0]), -1, 0.0, 0.5, 40, 0.0, wa, wb)
    assert r["kstar"][0, 0] == 6
    assert abs(r["dca"][0, 0] - 1.0) < 1e-14


def test_zero_field_matches_textbook_line_line_distance():
    rng = np.random.default_rng(7)
    x0 = np.array([50.0, 1.0, -3.0])
    p = np.array([60.0, 70.0, 40.0])
    T = p / np.linalg.norm(p)
    a_list, b_list, expect = [], [], []
    for _ in range(40):
        # wires that cross the region the 100 cm long track passes through
        s_c = rng.uniform(10, 90)
        foot = x0 + s_c * T + rng.normal(0, 1.0, 3)
        w = np.array([rng.normal(0, 0.05), rng.normal(0, 0.05), 1.0])
        w /= np.linalg.norm(w)
        a, b = foot - 75 * w, foot + 80 * w
        a_list.append(a)
        b_list.append(b)
        m = 0.5 * (a + b)
        n = np.cross(T, w)
        expect.append(np.dot(x0 - m, n) / np.linalg.norm(n))     # signed: u . (T x w)/|T x w|
    wa, wb = _wires(a_list, b_list)
    r = _scan_dca(_seed(x0, p), -1, 0.0, 0.5, 200, 0.0, wa, wb)
    np.testing.assert_allclose(r["dca"][0], np.array(expect), rtol=0, atol=1e-12)


@pytest.mark.parametrize("pmag,ct,h,n,tol", [(104.0, 0.6, 0.5, 400, 4e-9), (103.5, 0.2, 0.25, 1200, 5e-10)])
def test_axial_wire_closed_form(pmag, ct, h, n, tol):
    """For a wire parallel to B the DCA of a helix is | |centre - wire|_xy - R | exactly;
    the RKN4 track differs from the helix by its global error only."""
    phi = 1.1
    st = math.sqrt(1 - ct * ct)
    x0 = np.array([50.0 * math.cos(0.2), 50.0 * math.sin(0.2), -10.0])
    p = pmag * np.array([st * math.cos(phi), st * math.sin(phi), ct])
    q, bz = -1, 1.0
    c = KAPPA * q * bz / pmag
    T0 = p / pmag
    R = st / abs(c)
    centre = np.array([x0[0] + T0[1] / c, x0[1] - T0[0] / c])
    # axial wires placed near points of the first 60 % of the arc, 0.05..0.7 cm off the circle
    a_list, b_list, expect = [], [], []
    for i, frac in enumerate(np.linspace(0.05, 0.6, 12)):
        s = frac * n * h
        xs, _ = _helix_xy(x0, T0, c, s)
        radial = np.array([xs.real, xs.imag]) - centre
        radial /= np.linalg.norm(radial)
        off = (0.05 + 0.06 * i) * (1 if i % 2 == 0 else -1)
        wxy = centre + (R + off) * radial
        a_list.append([wxy[0], wxy[1], -75.0])
        b_list.append([wxy[0], wxy[1], 75.0])
        expect.append(abs(off))
    wa, wb = _wires(a_list, b_list)
    r = _scan_dca(_seed(x0, p), q, bz, h, n, 0.0, wa, wb)
    d = r["dca"][0]
    np.testing.assert_allclose(np.abs(d), np.array(expect), rtol=0, atol=tol)
    # electron in +B_z turns counter-clockwise: T x z^ points away from the centre,
    # u = x - wire points towards the centre for a wire outside the circle => negative sign
    assert np.all(np.sign(d) == -np.sign([0.05 + 0.06 * i if i % 2 == 0 else -(0.05 + 0.06 * i)
                                          for i in range(12)]))


def test_stereo_wires_against_dense_brute_force():
    """Minimum over a 1e-4 cm sampling of the ANALYTIC helix of the point-line distance
    (cross-product form), for tilted wires."""
    pmag, ct, phi = 104.0, 0.55, 0.9
    st = math.sqrt(1 - ct * ct)
    x0 = np.array([50.0, 0.0, 2.0])
    p = pmag * np.array([st * math.cos(phi), st * math.sin(phi), ct])
    q, bz, h, n = -1, 1.0, 0.5, 160
    c = KAPPA * q * bz / pmag
    T0 = p / pmag
    rng = np.random.default_rng(11)
    a_list, b_list = [], []
    for s_c in (12.0, 25.3, 41.7, 60.2):
        xs, _ = _helix_xy(x0, T0, c, s_c)
        foot = np.array([xs.real, xs.imag, x0[2] + T0[2] * s_c]) + rng.normal(0, 0.3, 3)
        w = np.array([rng.normal(0, 0.04), rng.normal(0, 0.04), 1.0])
        w /= np.linalg.norm(w)
        a_list.append(foot - 70 * w)
        b_list.append(foot + 70 * w)
    wa, wb = _wires(a_list, b_list)
    r = _scan_dca(_seed(x0, p), q, bz, h, n, 0.0, wa, wb)
    s = np.arange(0.0, n * h, 1e-4)
    xs, _ = _helix_xy(x0, T0, c, s)
    pos = np.stack([xs.real, xs.imag, x0[2] + T0[2] * s], axis=1)
    for i in range(4):
        a, b = np.array(a_list[i]), np.array(b_list[i])
        w = (b - a) / np.linalg.norm(b - a)
        dist = np.linalg.norm(np.cross(pos - a, w), axis=1)
        # sampling error <= (1e-4/2)^2 / (2 d) curvature term: far below 1e-7 for d ~ 0.1..1 cm
        assert abs(abs(r["dca"][0, i]) - dist.min()) < 2e-8


def test_rigid_motion_invariance():
    """Rotating everything about z (the field axis) or translating along z leaves D unchanged."""
    pmag, ct, phi = 103.5, 0.3, 0.4
    st = math.sqrt(1 - ct * ct)
    x0 = np.array([50.0, 0.0, -20.0])
    p = pmag * np.array([st * math.cos(phi), st * math.sin(phi), ct])
    rng = np.random.default_rng(3)
    c = KAPPA * -1 * 1.0 / pmag
    T0 = p / pmag
    a_list, b_list = [], []
    for s_c in rng.uniform(5, 100, 16):
        xs, _ = _helix_xy(x0, T0, c, s_c)
        foot = np.array([xs.real, xs.imag, x0[2] + T0[2] * s_c]) + rng.normal(0, 0.4, 3)
        w = np.array([rng.normal(0, 0.04), rng.normal(0, 0.04), 1.0])
        w /= np.linalg.norm(w)
        a_list.append(foot - 75 * w)
        b_list.append(foot + 75 * w)
    wa, wb = _wires(a_list, b_list)
    base = _scan_dca(_seed(x0, p), -1, 1.0, 0.25, 480, 0.0, wa, wb)["dca"][0]
    ang, dz = 1.2345, 17.0
    Rz = np.array([[math.cos(ang), -math.sin(ang), 0], [math.sin(ang), math.cos(ang), 0], [0, 0, 1]])
    shift = np.array([0, 0, dz])
    wa2 = np.ascontiguousarray(Rz @ wa + shift[:, None])
    wb2 = np.ascontiguousarray(Rz @ wb + shift[:, None])
    moved = _scan_dca(_seed(Rz @ x0 + shift, Rz @ p), -1, 1.0, 0.25, 480, 0.0, wa2, wb2)["dca"][0]
    np.testing.assert_allclose(moved, base, rtol=0, atol=2e-12)
    # mirror in the xz-plane with charge flip is also a symmetry of the equation of motion;
    # it reverses handedness, so the signed DCA changes sign
    Mx = np.diag([1.0, -1.0, 1.0])
    mir = _scan_dca(_seed(Mx @ x0, Mx @ p), +1, 1.0, 0.25, 480, 0.0,
                    np.ascontiguousarray(Mx @ wa), np.ascontiguousarray(Mx @ wb))["dca"][0]
    np.testing.assert_allclose(mir, -base, rtol=0, atol=2e-12)


def test_arc_end_clamp_gives_distance_from_last_recorded_point():
    """Reading R10: the search never leaves the recorded arc.  A straight 10 cm track along +x
    and an axial wire beyond its end at x = 14: the closest point of the arc is its end."""
    wa, wb = _wires([[14, 3, -50], [-5, 2, -50]], [[14, 3, 50], [-5, 2, 50]])
    r = _scan_dca(_seed([0, 0, 0], [100, 0, 0]), -1, 0.0, 0.5, 20, 0.0, wa, wb)
    assert r["kstar"][0, 0] == 20 and r["kstar"][0, 1] == 0
    assert abs(abs(r["dca"][0, 0]) - 5.0) < 1e-13         # hypot(4, 3)
    assert abs(abs(r["dca"][0, 1]) - math.hypot(5, 2)) < 1e-13


def test_kstar_is_argmin_of_point_line_distance_over_recorded_points():
    """k* against numpy's argmin of the cross-product distance over the exported track."""
    from comet_synth import make_config, event_seeds
    ev = make_config(0)[0]
    seeds, _ = event_seeds(ev)
    seeds = np.ascontiguousarray(seeds[:, ::257])
    track, n_pts = O.extrapolate(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop)
    r = O.scan(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a, ev.geom.wire_b,
               ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, want_kstar=True, want_npts=True, want_dca=True)
    np.testing.assert_array_equal(r["n_pts"], n_pts)
    a = ev.geom.wire_a[:, ev.fired_wire].T
    b = ev.geom.wire_b[:, ev.fired_wire].T
    w = (b - a) / np.linalg.norm(b - a, axis=1, keepdims=True)
    for s in range(seeds.shape[1]):
        pts = track[s, :n_pts[s], 0:3]
        d = np.linalg.norm(np.cross(pts[:, None, :] - 0.5 * (a + b)[None], w[None]), axis=2)   # [k][wire]
        ks = np.argmin(d, axis=0)
        np.testing.assert_array_equal(r["kstar"][s], ks)
        # refined DCA never exceeds the distance at the closest recorded point
        assert np.all(np.abs(r["dca"][s]) <= d[ks, np.arange(len(ks))] + 1e-12)
