"""Pins for the oracle's extrapolator (O1-O3; Algorithm 1).

None of these re-types the RKN4 formula: the expected values come from the
closed-form helix in a uniform B_z (radius p_T/(kappa B), angular advance c s,
constant pitch -- PAPER.md:319 Eq. (2)), from invariants (|T| = 1, T_z constant,
straight line at B = 0, reversibility under charge + momentum flip,
PAPER.md:230) and from hand-computed numbers.
"""
import math

import numpy as np
import pytest

from oracle import comet_oracle as O

KAPPA = 2.99792458   # typed here on purpose: pins the oracle's constant (reading R4)


def _seed(x, p):
    return np.array([[x[0]], [x[1]], [x[2]], [p[0]], [p[1]], [p[2]]], dtype=np.float64)


def test_kappa_is_speed_of_light_constant():
    # R = p_T / (0.3 B) with p in GeV/c, B in T, R in m == 0.299792458
    assert O.kappa() == KAPPA
    assert abs(O.kappa() / 10.0 - 0.299792458) < 1e-15


@pytest.mark.parametrize("pmag,ct,h,n,tol", [
    (104.0, 0.6, 0.5, 400, 6e-8),
    (103.5, 0.2, 0.25, 1200, 7e-9),
    (104.0, 0.15, 0.2, 1600, 3e-9),
    (60.0, 0.3, 0.25, 1200, 6e-8),
])
def test_track_follows_closed_form_helix(pmag, ct, h, n, tol):
    """Every recorded point lies on the analytic helix at arc length k h."""
    phi = 0.7
    st = math.sqrt(1 - ct * ct)
    x0 = np.array([50.0 * math.cos(0.3), 50.0 * math.sin(0.3), -12.0])
    p = pmag * np.array([st * math.cos(phi), st * math.sin(phi), ct])
    q, bz = -1, 1.0
    track, n_pts = O.extrapolate(_seed(x0, p), q, bz, h, n, 0.0)
    assert n_pts[0] == n + 1
    T0 = p / pmag
    c = KAPPA * q * bz / pmag
    s = h * np.arange(n + 1)
    # rotation of the transverse tangent by the angle -c s, written with complex numbers
    t_xy = (T0[0] + 1j * T0[1]) * np.exp(-1j * c * s)
    # integral of the tangent: x(s) = x0 + T0_xy (1 - exp(-i c s)) / (i c)
    x_xy = (x0[0] + 1j * x0[1]) + (T0[0] + 1j * T0[1]) * (1 - np.exp(-1j * c * s)) / (1j * c)
    assert np.max(np.abs(track[0, :, 0] - x_xy.real)) < tol
    assert np.max(np.abs(track[0, :, 1] - x_xy.imag)) < tol
    assert np.max(np.abs(track[0, :, 2] - (x0[2] + T0[2] * s))) < 1e-11
    assert np.max(np.abs(track[0, :, 3] - t_xy.real)) < tol
    assert np.max(np.abs(track[0, :, 4] - t_xy.imag)) < tol


def test_radius_and_turn_direction():
    """Transverse radius = p_T/(kappa |B|); an electron (q = -1) in +B_z turns counter-clockwise
    seen from +z (F = q v x B: v = +x, B = +z gives F = -q y = +y for q = -1)."""
    pmag, ct = 100.0, 0.0
    x0 = np.array([0.0, 0.0, 0.0])
    p = np.array([pmag, 0.0, 0.0])
    track, _ = O.extrapolate(_seed(x0, p), -1, 1.0, 0.1, 2200, 0.0)
    R = pmag / KAPPA          # 33.356... cm
    # circle centre must be at (0, +R): all points at distance R from it
    d = np.hypot(track[0, :, 0] - 0.0, track[0, :, 1] - R)
    assert np.max(np.abs(d - R)) < 1e-9
    assert track[0, 10, 1] > 0.0                     # bends towards +y
    # positron bends the other way
    track_p, _ = O.extrapolate(_seed(x0, p), +1, 1.0, 0.1, 50, 0.0)
    assert track_p[0, 10, 1] < 0.0
    np.testing.assert_allclose(track_p[0, :, 1], -track[0, :51, 1], rtol=0, atol=1e-15)
    # one full revolution takes 2 pi R of arc: the track returns to the start
    k_rev = 2 * math.pi * R / 0.1
    k0 = int(round(k_rev))
    assert np.hypot(track[0, k0, 0], track[0, k0, 1]) < abs(k_rev - k0) * 0.1 + 1e-6


def test_pitch():
    """Delta z per revolution = 2 pi R_3D cos(theta) with R_3D = |p|/(kappa B)."""
    pmag, ct = 103.5, 0.2
    st = math.sqrt(1 - ct * ct)
    p = pmag * np.array([st, 0.0, ct])
    h = 0.05
    turn_arc = 2 * math.pi * pmag / KAPPA             # arc length of one revolution
    n = int(turn_arc / h) + 2
    track, _ = O.extrapolate(_seed([0, 0, 0], p), -1, 1.0, h, n, 0.0)
    # find where phi of the tangent completes a revolution by interpolation on T_y sign
    ty = track[0, :, 4]
    k = np.nonzero((ty[1:-1] < 0) & (ty[2:] >= 0))[0]   # electron: T_y goes +,then -, back to 0 at 2 pi
    assert k.size >= 1
    k = k[-1] + 1
    f = -ty[k] / (ty[k + 1] - ty[k])
    z_turn = track[0, k, 2] + f * (track[0, k + 1, 2] - track[0, k, 2])
    assert abs(z_turn - turn_arc * ct) < 1e-6


def test_tangent_norm_and_tz_invariants():
    pmag, ct, phi = 104.0, 0.55, 2.1
    st = math.sqrt(1 - ct * ct)
    p = pmag * np.array([st * math.cos(phi), st * math.sin(phi), ct])
    track, _ = O.extrapolate(_seed([50, 0, 3], p), -1, 1.0, 0.5, 400, 0.0)
    T = track[0, :, 3:6]
    assert np.max(np.abs(np.linalg.norm(T, axis=1) - 1.0)) < 2e-11     # reading R1: no renormalisation
    assert np.all(T[:, 2] == T[0, 2])                                   # bit-constant
    assert T[0, 2] == p[2] / math.sqrt(p[0] * p[0] + p[1] * p[1] + p[2] * p[2])
    z = track[0, :, 2]
    assert np.max(np.abs(z - (3 + T[0, 2] * 0.5 * np.arange(401)))) < 1e-12


def test_zero_field_is_a_straight_line():
    p = np.array([30.0, -40.0, 12.0])
    x0 = np.array([1.0, 2.0, 3.0])
    track, n_pts = O.extrapolate(_seed(x0, p), -1, 0.0, 0.5, 100, 0.0)
    T0 = p / np.linalg.norm(p)
    expect = x0[None, :] + 0.5 * np.arange(101)[:, None] * T0[None, :]
    assert np.max(np.abs(track[0, :, 0:3] - expect)) < 1e-13
    assert np.max(np.abs(track[0, :, 3:6] - T0[None, :])) == 0.0


def test_reversibility_backward_half_track():
    """Flip charge and momentum at the end point and step back: returns to the start
    (the paper's backward half track)."""
    pmag, ct, phi = 104.0, 0.6, 0.4
    st = math.sqrt(1 - ct * ct)
    x0 = np.array([50.0, 0.0, -5.0])
    p = pmag * np.array([st * math.cos(phi), st * math.sin(phi), ct])
    n, h = 400, 0.5
    fwd, _ = O.extrapolate(_seed(x0, p), -1, 1.0, h, n, 0.0)
    xe, Te = fwd[0, n, 0:3], fwd[0, n, 3:6]
    bwd, _ = O.extrapolate(_seed(xe, -pmag * Te), +1, 1.0, h, n, 0.0)
    assert np.max(np.abs(bwd[0, n, 0:3] - x0)) < 2e-7
    # and every intermediate point is revisited
    assert np.max(np.abs(bwd[0, ::-1, 0:3] - fwd[0, :, 0:3])) < 2e-7


def test_single_step_hand_computed():
    """One RKN4 step of a 90-degree-ish arc against the analytic circle: local error O((c h)^5).
    Expected numbers are computed from sin/cos, not from the RKN formula."""
    c, h = 0.03, 1.0
    s = O.rkn4_step([0, 0, 0, 1, 0, 0], h, c)
    # dT/ds = c (Ty, -Tx, 0): T = (cos cs, -sin cs), x = (sin cs / c, (cos cs - 1)/c)
    assert abs(s[3] - math.cos(c * h)) < (c * h) ** 5 / 100
    assert abs(s[4] + math.sin(c * h)) < (c * h) ** 5 / 100
    assert abs(s[0] - math.sin(c * h) / c) < (c * h) ** 5 / c
    assert abs(s[1] - (math.cos(c * h) - 1) / c) < (c * h) ** 5 / c
    # 4th order: halving h cuts the one-step tangent error ~32x
    e1 = abs(O.rkn4_step([0, 0, 0, 1, 0, 0], 2.0, 0.2)[3] - math.cos(0.4))
    e2 = abs(O.rkn4_step([0, 0, 0, 1, 0, 0], 1.0, 0.2)[3] - math.cos(0.2))
    assert 20 < e1 / e2 < 90
    # negative step is the inverse direction along the same circle
    b = O.rkn4_step([0, 0, 0, 1, 0, 0], -h, c)
    # (local position error of the Nystrom form is c^4 h^5 / 120 = 6.7e-9 cm here)
    assert abs(b[0] + math.sin(c * h) / c) < (c * h) ** 5 / c / 100
    assert abs(b[1] - (math.cos(c * h) - 1) / c) < (c * h) ** 5 / c / 100
    # and mirrors the forward step exactly: x -> -x, y -> y, Tx -> Tx, Ty -> -Ty
    assert b[0] == -s[0] and b[1] == s[1] and b[3] == s[3] and b[4] == -s[4]


def test_target_region_stop_rule():
    """Reading R3: recording stops at the first point with r < r_stop moving inward."""
    pmag, ct = 104.0, 0.2
    st = math.sqrt(1 - ct * ct)
    # start on r = 50 moving outward at 30 degrees to the radial direction
    x0 = np.array([50.0, 0.0, 0.0])
    a = math.radians(30)
    p = pmag * np.array([st * math.cos(a), st * math.sin(a), ct])
    h, n = 0.25, 1200
    full, n_full = O.extrapolate(_seed(x0, p), -1, 1.0, h, n, 0.0)
    cut, n_cut = O.extrapolate(_seed(x0, p), -1, 1.0, h, n, 50.0)
    assert n_full[0] == n + 1 and 2 <= n_cut[0] < n + 1
    r = np.hypot(full[0, :, 0], full[0, :, 1])
    rad = full[0, :, 0] * full[0, :, 3] + full[0, :, 1] * full[0, :, 4]
    inside = np.nonzero((r[1:] < 50.0) & (rad[1:] < 0.0))[0] + 1
    assert n_cut[0] == inside[0] + 1
    k = n_cut[0]
    np.testing.assert_array_equal(cut[0, :k], full[0, :k])
    assert np.all(np.isnan(cut[0, k:]))
    # an inward-moving seed that starts inside r_stop stops after the first step
    p_in = pmag * np.array([-st, 0.0, ct])
    _, n_in = O.extrapolate(_seed([49.0, 0.0, 0.0], p_in), -1, 1.0, h, n, 50.0)
    assert n_in[0] == 2
