"""Pins for the oracle's Hough-transform transverse seeding (Fig. 10; readings R35-R37)."""
import numpy as np

from comet_synth import event_seeds, hough_tables, make_config
from oracle import comet_oracle as O

KAPPA = 2.99792458


def _wires_on_circle(R, phi_c, n, rng, jitter=0.0):
    """Fake 'wires' (vertical segments) whose midpoints lie on the circle of radius R through the origin."""
    cx, cy = R * np.cos(phi_c), R * np.sin(phi_c)
    a = rng.uniform(0, 2 * np.pi, n)
    x = cx + R * np.cos(a) + rng.normal(0, jitter, n)
    y = cy + R * np.sin(a) + rng.normal(0, jitter, n)
    keep = np.hypot(x, y) > 20.0                       # away from the origin, like the chamber
    x, y = x[keep], y[keep]
    wa = np.stack([x, y, np.full(x.size, -75.0)])
    wb = np.stack([x, y, np.full(x.size, 75.0)])
    return wa, wb, np.arange(x.size, dtype=np.int32)


def test_conformal_map_turns_circles_through_the_origin_into_lines():
    rng = np.random.default_rng(0)
    wa, wb, fw = _wires_on_circle(33.0, 1.1, 50, rng)
    x, y = wa[0], wa[1]
    u, v = x / (x * x + y * y), y / (x * x + y * y)
    np.testing.assert_allclose(u * np.cos(1.1) + v * np.sin(1.1), 1.0 / 66.0, atol=1e-15)


def test_exact_circle_is_recovered_within_one_bin():
    rng = np.random.default_rng(1)
    c, s = hough_tables(256)
    rmin, rmax, n_rho = 1 / 120.0, 1 / 40.0, 128
    inv = n_rho / (rmax - rmin)
    for R, j_c in ((33.0, 40), (28.5, 200), (45.0, 3)):
        phi_c = 2 * np.pi * j_c / 256
        wa, wb, fw = _wires_on_circle(R, phi_c, 60, rng)
        out = O.hough_seeds(wa, wb, fw, c, s, rmin, inv, n_rho, -1, 1.0, 50.0)
        votes, j, k = out["peak"]
        assert votes == fw.size and j == j_c                      # every wire votes for the true direction and bin
        assert k == int(np.floor((1 / (2 * R) - rmin) * inv))
        assert abs(out["R"] - R) < R * R * 2 / inv                # dR = 2 R^2 d(rho), within one bin
        assert out["acc"].sum() <= fw.size * 256 and out["acc"].dtype == np.int32
        # ties -> the lowest flat index
        assert (out["acc"].ravel() == votes).argmax() == j * n_rho + k


def test_seed_points_and_momenta_geometry_and_rotation_sense():
    rng = np.random.default_rng(2)
    c, s = hough_tables(256)
    rmin, rmax, n_rho = 1 / 120.0, 1 / 40.0, 256
    inv = n_rho / (rmax - rmin)
    wa, wb, fw = _wires_on_circle(33.0, 2 * np.pi * 77 / 256, 80, rng)
    for charge, bz in ((-1, 1.0), (+1, 1.0), (-1, -0.8)):
        out = O.hough_seeds(wa, wb, fw, c, s, rmin, inv, n_rho, charge, bz, 50.0)
        R, ctr = out["R"], out["centre"]
        assert abs(np.hypot(*ctr) - R) < 1e-12                    # the circle passes through the origin
        for key, outward in (("entrance", True), ("exit", False)):
            x, y, px, py = out[key]
            assert abs(np.hypot(x, y) - 50.0) < 1e-12 and abs(np.hypot(x - ctr[0], y - ctr[1]) - R) < 1e-12
            assert abs((x - ctr[0]) * px + (y - ctr[1]) * py) < 1e-9          # tangent
            assert abs(np.hypot(px, py) - KAPPA * abs(bz) * R) < 1e-10        # p_T = kappa |B| R
            assert (x * px + y * py > 0) == outward
        # the sense of rotation agrees with the (pinned) extrapolator: a track started at the entrance with the
        # Hough momentum stays on the Hough circle and arrives at the exit point
        x, y, px, py = out["entrance"]
        seed = np.array([x, y, 0.0, px, py, 20.0]).reshape(6, 1)
        tr, npt = O.extrapolate(seed, charge, bz, 0.25, 1200, 50.0)
        pts = tr[0, :npt[0], :2]
        assert np.abs(np.hypot(pts[:, 0] - ctr[0], pts[:, 1] - ctr[1]) - R).max() < 1e-6
        assert np.hypot(*(pts[-1] - out["exit"][:2])) < 0.3          # stops within a step of the exit point


def test_hough_on_a_synthetic_event_is_a_coarse_seed():
    """configs[1]: the vertex is a few cm off the axis, so the through-origin circle is approximate -- the seed
    must still land within the windows the scan is given (paper: 0.02 rad, 3.2 MeV/c with its own finder)."""
    ev = make_config(1)[0]
    c, s = hough_tables(256)
    rmin, rmax, n_rho = 1 / 120.0, 1 / 40.0, 128
    out = O.hough_seeds(ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, c, s, rmin, n_rho / (rmax - rmin), n_rho,
                        ev.charge, ev.bz, 50.0)
    p = ev.partitions[0]
    pT = ev.pmag * np.sqrt(1 - p.cos_theta ** 2)
    assert out["peak"][0] >= 15
    assert abs(np.hypot(*out["entrance"][2:]) - pT) < 8.0
    d_theta = np.angle(np.exp(1j * (np.arctan2(out["entrance"][1], out["entrance"][0]) - p.theta_e)))
    assert abs(d_theta) < 0.12
    # no fired wires: no peak
    none = O.hough_seeds(ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire[:0], c, s, rmin, 1000.0, n_rho, -1, 1.0, 50.0)
    assert none["peak"][0] == 0 and np.isnan(none["entrance"]).all()
