"""Pins for the oracle's field-map path (trilinear field, Nystrom RK4 in the map, adaptive step, DCA;
PAPER.md:77, :99, :135-136; readings R29-R32).

Independent references: scipy's RegularGridInterpolator for the field, scipy's DOP853 integrator of the
Lorentz-force equation in that interpolated field for the trajectory and for the DCA (dense sampling), and the
already pinned uniform-field oracle for the limit of a uniform map.
"""
import numpy as np
import pytest
from scipy.integrate import solve_ivp
from scipy.interpolate import RegularGridInterpolator

from comet_synth import event_seeds, make_config, solenoid_map, uniform_map
from oracle import comet_oracle as O

KAPPA = 2.99792458


def _interp(field):
    B, o, d = field
    axes = [o[a] + d[a] * np.arange(B.shape[a]) for a in range(3)]
    f = RegularGridInterpolator(axes, B, method="linear", bounds_error=False, fill_value=None)
    lo, hi = np.array([a[0] for a in axes]), np.array([a[-1] for a in axes])
    return lambda x: f(np.clip(x, lo, hi))[0]


def _reference_track(field, seed, charge, s_end, dense=False):
    bf = _interp(field)
    P = np.linalg.norm(seed[3:])
    cq = KAPPA * charge / P
    rhs = lambda s, y: np.concatenate([y[3:], cq * np.cross(y[3:], bf(y[:3]))])
    y0 = np.concatenate([seed[:3], seed[3:] / P])
    return solve_ivp(rhs, [0.0, s_end], y0, method="DOP853", rtol=1e-12, atol=1e-13, dense_output=dense)


@pytest.fixture(scope="module")
def cfg0():
    ev = make_config(0)[0]
    seeds, _ = event_seeds(ev, shape=(2, 2, 2, 2))
    return ev, seeds


def test_field_at_is_trilinear_and_clamped():
    F = solenoid_map()
    bf = _interp(F)
    rng = np.random.default_rng(0)
    for x in rng.uniform(-95, 95, size=(200, 3)):
        np.testing.assert_allclose(O.field_at(F, x), bf(x), rtol=0, atol=1e-14)
    B, o, d = F
    np.testing.assert_array_equal(O.field_at(F, o + d * np.array([3, 5, 7])), B[3, 5, 7])           # a node
    np.testing.assert_allclose(O.field_at(F, o + d * np.array([3.5, 5, 7])), 0.5 * (B[3, 5, 7] + B[4, 5, 7]), atol=1e-16)
    np.testing.assert_array_equal(O.field_at(F, [500.0, -500.0, 1e4]), B[-1, 0, -1])               # outside: the edge value
    # the generator's map is a solenoid: B_z ~ b0 in the centre, weaker at the ends, B_r pointing outwards there
    assert abs(O.field_at(F, [0, 0, 0])[2] - 1.0) < 1e-3
    assert O.field_at(F, [0, 0, 92.0])[2] < 0.6 and O.field_at(F, [40.0, 0, 80.0])[0] > 0.01


def test_uniform_map_reproduces_the_uniform_field_oracle(cfg0):
    ev, seeds = cfg0
    args = (ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff)
    for bz in (1.0, 0.73):
        ru = O.scan(seeds, ev.charge, bz, ev.step, ev.n_steps, ev.r_stop, *args, want_dca=True, want_kstar=True, want_npts=True)
        rf = O.scan_field(seeds, ev.charge, uniform_map(bz), ev.step, ev.n_steps, ev.r_stop, 1e-3, *args,
                          want_dca=True, want_kstar=True, want_npts=True)
        np.testing.assert_array_equal(ru["n_pts"], rf["n_pts"])
        np.testing.assert_array_equal(ru["kstar"], rf["kstar"])
        np.testing.assert_allclose(rf["dca"], ru["dca"], rtol=0, atol=1e-11)
        np.testing.assert_allclose(rf["rss"], ru["rss"], rtol=1e-9)
    # one step: same state as the uniform step, and the step estimate of a pure rotation is tiny
    st = np.array([50.0, 1.0, 2.0, 0.6, 0.64, 0.48])
    s1, est = O.rkn4_field_step(uniform_map(1.0), st, 0.5, -KAPPA / 104.0)
    np.testing.assert_allclose(s1, O.rkn4_step(st, 0.5, -KAPPA * 1.0 / 104.0), rtol=0, atol=1e-15)
    assert 0.0 < est < 1e-5


def test_field_track_against_dop853(cfg0):
    ev, seeds = cfg0
    F = solenoid_map()
    seed = seeds[:, 3].copy()
    seed[2] = 55.0                                  # start where the field is rough
    errs = []
    for h in (0.5, 0.25, 0.125):
        tr, npt, hs = O.extrapolate_field(seed.reshape(6, 1), ev.charge, F, h, int(60 / h), 0.0, 1e9)   # tol huge: fixed step
        assert np.all(hs[0, :npt[0] - 1] == h)
        ref = _reference_track(F, seed, ev.charge, 60.0)
        errs.append(np.abs(tr[0, npt[0] - 1, :3] - ref.y[:3, -1]).max())
        assert abs(np.linalg.norm(tr[0, npt[0] - 1, 3:]) - 1.0) < 1e-9                                  # |T| conserved
    # (the trilinear field has kinks at the cell faces, so the order is below 4)
    assert errs[0] < 1e-4 and errs[2] < errs[1] < errs[0] and errs[2] < 2e-6


def test_adaptive_step_control(cfg0):
    ev, seeds = cfg0
    F = solenoid_map()
    sd = seeds[:, :4].copy()
    sd[2] = [0.0, 30.0, 55.0, 65.0]
    h_max, n = 0.5, 300
    P = np.linalg.norm(sd[3:], axis=0)
    worst = []
    for tol in (1e-5, 1e-7, 1e-9):
        tr, npt, hs = O.extrapolate_field(sd, ev.charge, F, h_max, n, 0.0, tol)
        err = []
        for s in range(4):
            k = npt[s] - 1
            h = hs[s, :k]
            assert np.all(np.isin(h, h_max / 2.0 ** np.arange(7)))                   # halvings of h_max, never below h_max/64
            # every accepted step meets the tolerance unless it is already the shortest one;
            # a step shorter than its predecessor was forced by a rejected longer one
            for j in range(k):
                _, est = O.rkn4_field_step(F, tr[s, j], h[j], KAPPA * ev.charge / P[s])
                assert est <= tol or h[j] == h_max / 64
                if j > 0 and h[j] < h[j - 1]:
                    _, est2 = O.rkn4_field_step(F, tr[s, j], 2 * h[j], KAPPA * ev.charge / P[s])
                    assert est2 > tol
            ref = _reference_track(F, sd[:, s], ev.charge, float(h.sum()))
            err.append(np.abs(tr[s, k, :3] - ref.y[:3, -1]).max())
        worst.append(max(err))
    assert worst[2] < worst[1] < worst[0] and worst[2] < 2e-7                        # a tighter tolerance buys accuracy
    # rougher field -> shorter steps: the track started near the end plate takes shorter steps than the central one
    tr, npt, hs = O.extrapolate_field(sd, ev.charge, F, h_max, n, 0.0, 1e-7)
    assert np.nanmean(hs[3]) < np.nanmean(hs[0])
    # a huge tolerance is the fixed-step recording
    tr2, npt2, hs2 = O.extrapolate_field(sd, ev.charge, F, h_max, n, 0.0, 1e9)
    assert np.all(hs2[~np.isnan(hs2)] == h_max)


def test_step_error_estimate_closed_forms():
    """R31's error estimate EST = h^2 sum_xyz |k1 - k2 - k3 + k4| pinned against numbers that do not come from the
    oracle's own step: (a) in a uniform field the four slopes of R30 are powers of the rotation generator
    J T = (T_y, -T_x, 0) applied to T -- k1 = w J T, k2 = k1 + (h/2) w^2 J^2 T, k3 = k2 + (h^2/4) w^3 J^3 T,
    k4 = k1 + h w^2 J^2 T + (h^2/2) w^3 J^3 T + (h^3/4) w^4 J^4 T, w = cq B_z -- so k1 - k2 - k3 + k4 =
    (h^2/4) w^3 J^3 T + (h^3/4) w^4 J^4 T with J^2 = -1 in the transverse plane: a closed form in which any other
    sign pattern of the four slopes leaves a term of order h w^2, four orders of magnitude larger;  (b) in the
    field B = (0, 0, b0 + g x), which the trilinear map holds exactly, k1..k4 are written out with numpy cross
    products at the three positions of R30 (start, midpoint with k1, end point with k3)."""
    # (a) uniform field
    for (bz, P, q, h, T) in [(1.0, 104.0, -1, 0.5, [0.6, 0.3, 0.2]), (0.8, 60.0, 1, 0.25, [-0.1, 0.9, 0.3]),
                             (1.2, 95.0, -1, 0.125, [0.7, -0.7, 0.1])]:
        T = np.array(T) / np.linalg.norm(T)
        cq = KAPPA * q / P
        w = cq * bz
        _, est = O.rkn4_field_step(uniform_map(bz), np.concatenate([[3.0, -2.0, 5.0], T]), h, cq)
        a, b = h * h * w ** 3 / 4.0, h ** 3 * w ** 4 / 4.0
        expect = h * h * (abs(-a * T[1] + b * T[0]) + abs(a * T[0] + b * T[1]))
        assert expect > 0.0
        np.testing.assert_allclose(est, expect, rtol=1e-7)
        for signs in [(1, 1, -1, -1), (1, -1, 1, -1), (1, 1, 1, 1), (1, -1, -1, -1), (-1, 1, 1, 1)]:
            # what a mis-signed combination would give (k's from the closed forms above): far from EST
            JT = np.array([T[1], -T[0], 0.0]); Tp = np.array([T[0], T[1], 0.0])
            k1 = w * JT
            k2 = k1 - (h / 2) * w ** 2 * Tp
            k3 = k2 - (h * h / 4) * w ** 3 * JT
            k4 = k1 - h * w ** 2 * Tp - (h * h / 2) * w ** 3 * JT + (h ** 3 / 4) * w ** 4 * Tp
            wrong = h * h * np.abs(signs[0] * k1 + signs[1] * k2 + signs[2] * k3 + signs[3] * k4).sum()
            assert abs(wrong - est) > 100.0 * est
    # (b) linear gradient along x: B_z = b0 + g x (exact under trilinear interpolation)
    b0, g = 0.9, 0.004
    d = np.array([8.0, 8.0, 8.0]); o = np.array([-96.0, -96.0, -96.0]); n = 25
    B = np.zeros((n, n, n, 3))
    B[..., 2] = (b0 + g * (o[0] + d[0] * np.arange(n)))[:, None, None]
    F = (B, o, d)
    bfield = lambda x: np.array([0.0, 0.0, b0 + g * x[0]])
    rng = np.random.default_rng(5)
    for _ in range(6):
        x = rng.uniform(-60.0, 60.0, 3)
        T = rng.normal(size=3); T /= np.linalg.norm(T)
        h = float(rng.choice([0.5, 0.25, -0.3]))
        cq = KAPPA * float(rng.choice([-1, 1])) / rng.uniform(60.0, 110.0)
        k1 = cq * np.cross(T, bfield(x))
        bm = bfield(x + h / 2 * T + h * h / 8 * k1)
        k2 = cq * np.cross(T + h / 2 * k1, bm)
        k3 = cq * np.cross(T + h / 2 * k2, bm)
        k4 = cq * np.cross(T + h * k3, bfield(x + h * T + h * h / 2 * k3))
        s1, est = O.rkn4_field_step(F, np.concatenate([x, T]), h, cq)
        np.testing.assert_allclose(est, h * h * np.abs(k1 - k2 - k3 + k4).sum(), rtol=1e-6)
        np.testing.assert_allclose(s1[:3], x + h * T + h * h / 6 * (k1 + k2 + k3), rtol=0, atol=1e-13)
        np.testing.assert_allclose(s1[3:], T + h / 6 * (k1 + 2 * k2 + 2 * k3 + k4), rtol=0, atol=1e-14)
    # the gradient shows up in EST at the order the closed form predicts: with T along x and a weak field the
    # second difference of the acceleration along the step is k1 - 2 k(h/2) + k(h) ~ 0 for a linear B(x), so EST
    # stays at the uniform-field size, while a kink of the map (a cell face crossed by the step) raises it
    Bk = B.copy()
    Bk[n // 2:, :, :, 2] += 0.05 * (d[0] * np.arange(n - n // 2))[:, None, None] / d[0]
    x0 = np.array([o[0] + d[0] * (n // 2) - 0.2, 1.0, 2.0]); T0 = np.array([1.0, 0.0, 0.0])
    _, e_lin = O.rkn4_field_step(F, np.concatenate([x0, T0]), 0.5, KAPPA / 100.0)
    _, e_kink = O.rkn4_field_step((Bk, o, d), np.concatenate([x0, T0]), 0.5, KAPPA / 100.0)
    assert e_kink > 20.0 * e_lin


def test_field_dca_against_dense_sampling(cfg0):
    ev, seeds = cfg0
    F = solenoid_map()
    seed = seeds[:, 5].copy()
    h, n = 0.25, 400
    out = O.scan_field(seed.reshape(6, 1), ev.charge, F, h, n, 0.0, 1e-8, ev.geom.wire_a, ev.geom.wire_b,
                       ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, want_dca=True, want_kstar=True, want_npts=True)
    tr, npt, hs = O.extrapolate_field(seed.reshape(6, 1), ev.charge, F, h, n, 0.0, 1e-8)
    arc = float(np.nansum(hs[0]))
    ref = _reference_track(F, seed, ev.charge, arc, dense=True)
    s = np.linspace(0.0, arc, 200001)
    X = ref.sol(s)[:3].T
    checked = 0
    for i, wi in enumerate(ev.fired_wire):
        a, b = ev.geom.wire_a[:, wi], ev.geom.wire_b[:, wi]
        w = (b - a) / np.linalg.norm(b - a)
        m = 0.5 * (a + b)
        dlt = X - m
        u = dlt - np.outer(dlt @ w, w)
        dist = np.linalg.norm(u, axis=1)
        j = int(np.argmin(dist))
        if j in (0, len(s) - 1) or dist[j] > 3.0:
            continue                                   # closest approach at an arc end or far away: other tests
        assert abs(abs(out["dca"][0, i]) - dist[j]) < 2e-6
        T = ref.sol(s[j])[3:]
        assert np.sign(out["dca"][0, i]) == np.sign(u[j] @ np.cross(T, w))
        checked += 1
    assert checked >= 10


def test_classify_seeds_field_is_the_rule_of_o11(cfg0):
    ev, seeds = cfg0
    F = solenoid_map()
    args = (ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff)
    sc = O.scan_field(seeds, ev.charge, F, ev.step, ev.n_steps, ev.r_stop, 1e-7, *args, want_dca=True)
    idx = np.array([3, -1, 9], dtype=np.int64)
    c = O.classify_seeds_field(seeds, idx, ev.charge, F, ev.step, ev.n_steps, ev.r_stop, 1e-7, *args)
    np.testing.assert_array_equal(c["dca"][[0, 2]], sc["dca"][[3, 9]])
    assert np.isnan(c["dca"][1]).all() and c["cls"][1].sum() == 0
    for q, s in ((0, 3), (2, 9)):
        exp = np.zeros(ev.n_hits, dtype=np.uint8)
        for i in range(ev.n_fired):
            j0, j1 = ev.hit_off[i], ev.hit_off[i + 1]
            res = np.abs(sc["dca"][s, i] - ev.rho[j0:j1])
            if res.size and res.min() < ev.cutoff:
                exp[j0 + int(np.argmin(res))] = 1
        np.testing.assert_array_equal(c["cls"][q], exp)
