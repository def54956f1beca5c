"""The far radius of the pruned searches (k_wire_prep), checked on the oracle's own numbers.

The CUDA path gives a (seed, wire) pair the residual lambda without running the virtual-plane iteration when the
closest recorded state is farther from the wire than R = min(rho_max + lambda + 0.51 h,
eps + sqrt((rho_max + lambda + eps)^2 + 0.2505 h^2 + eps^2)) (+1e-6), eps = 0.0251 h (uniform field, |c| h <= 0.05).
That rests on |D| >= sqrt(d*^2 - 0.2505 h^2 - 2 d* eps) - eps for the D the method computes from the closest
recorded state at distance d*.  Here the inequality and the decision are checked on every pair of samples of
configs 0, 1 and 4 with D, k* and the track taken from the oracle (no CUDA code involved)."""
import numpy as np
import pytest

from comet_synth import event_seeds, make_config
from oracle import comet_oracle as O

KAPPA = 2.99792458


@pytest.mark.parametrize("cfg,n_sub", [(0, 1500), (1, 1200), (4, 250)])
def test_far_radius_is_safe_on_the_oracles_numbers(cfg, n_sub):
    ev = make_config(cfg)[0]
    seeds, _ = event_seeds(ev)
    idx = np.sort(np.random.default_rng(7).permutation(seeds.shape[1])[:n_sub])
    sd = np.ascontiguousarray(seeds[:, idx])
    r = O.scan(sd, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire,
               ev.hit_off, ev.rho, ev.cutoff, want_dca=True, want_kstar=True)
    tr, _ = O.extrapolate(sd, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop)
    wa, wb = ev.geom.wire_a[:, ev.fired_wire], ev.geom.wire_b[:, ev.fired_wire]
    w = wb - wa
    w /= np.linalg.norm(w, axis=0)
    m = (wa + wb) / 2
    S, W = r["kstar"].shape
    x = tr[np.arange(S)[:, None], r["kstar"], :3]                   # the closest recorded state of every pair
    d = x - m.T[None]
    perp = d - np.einsum("swc,cw->sw", d, w)[..., None] * w.T[None]
    d_star = np.linalg.norm(perp, axis=2)
    h = ev.step
    eps = 0.0251 * h
    assert np.all(np.abs(KAPPA * ev.charge * ev.bz / np.linalg.norm(sd[3:6], axis=0)) * h <= 0.05)
    D = np.abs(r["dca"])
    lower = np.sqrt(np.maximum(d_star ** 2 - 0.2505 * h * h - 2 * d_star * eps, 0.0)) - eps - 1e-6
    assert (D - lower).min() > 0.0                                   # the inequality behind the radius
    rho_max = np.array([np.abs(ev.rho[ev.hit_off[i]:ev.hit_off[i + 1]]).max() for i in range(W)])
    b = rho_max + ev.cutoff + eps + 1e-6
    radius = np.minimum(rho_max + ev.cutoff + 0.51 * h + 1e-6, eps + np.sqrt(b * b + 0.2505 * h * h + eps * eps))
    far = d_star > radius[None, :]
    assert far.sum() > 0.5 * far.size * (cfg != 0) and (~far).sum() > 0
    assert np.all((D - rho_max[None, :])[far] > ev.cutoff)            # every far pair's residual is the cutoff
    window = far & (d_star <= (rho_max + ev.cutoff + 0.51 * h + 1e-6)[None, :])
    assert window.sum() > 0                                          # pairs only the sharper radius calls far
