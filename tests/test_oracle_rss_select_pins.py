"""Pins for the oracle's residual / RSS / argmin / classification (O8-O11;
PAPER.md:75-83 Eq. (1) and the classification rule).

Expected values: the smearing the generator injected (truth seed), exact bounds and
monotonicity of Eq. (1), hand-computed toy events, and brute-force numpy loops that
start from signed DCAs only.
"""
import numpy as np
import pytest

from comet_synth import event_seeds, make_config, truth_seed
from oracle import comet_oracle as O


def _scan(ev, seeds, cutoff=None, rho=None, **kw):
    return O.scan(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a, ev.geom.wire_b,
                  ev.fired_wire, ev.hit_off, ev.rho if rho is None else rho,
                  ev.cutoff if cutoff is None else cutoff, **kw)


def _select(ev, seeds, rss, part_off, cutoff=None):
    return O.select_classify(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a,
                             ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.rho,
                             ev.cutoff if cutoff is None else cutoff, rss, part_off)


@pytest.mark.parametrize("cfg,rel", [(0, 3e-5), (1, 3e-6)])
def test_truth_seed_rss_equals_injected_smearing(cfg, rel, cfg0_event, cfg1_event):
    """A seed equal to the generating truth gives per-wire residuals equal to the injected
    smear (PAPER.md:294 smearing; north_star invariant)."""
    ev = cfg0_event if cfg == 0 else cfg1_event
    lam = ev.cutoff
    for p in range(len(ev.partitions)):
        seeds = truth_seed(ev, p).reshape(6, 1)
        r = _scan(ev, seeds, want_dca=True)
        D = r["dca"][0]
        expect, n_checked = 0.0, 0
        for i in range(ev.n_fired):
            js = range(ev.hit_off[i], ev.hit_off[i + 1])
            own = [j for j in js if ev.hit_turn[j] == p and ev.hit_real[j]]
            if own:
                j = own[0]
                # signed truth DCA agrees with the oracle's (RKN4 global error only)
                assert abs(D[i] - ev.hit_true_dca[j]) < 1e-9
                # the generator's drift r = |true DCA| + eps (clamped at 0)
                res = [abs(ev.hit_true_dca[j] - ev.rho[jj]) for jj in js]
                expect += min(min(res), lam) ** 2
                n_checked += 1
            else:
                # wire fired by another turn only: whatever the oracle found, bounded by lambda
                res = [abs(D[i] - ev.rho[jj]) for jj in js]
                expect += min(min(res), lam) ** 2
        assert n_checked >= 15
        assert abs(r["rss"][0] - expect) <= rel * expect
        # and the part that is pure injected smear: sum over single-hit wires of eps^2
        pure = [(abs(ev.rho[ev.hit_off[i]]) - abs(ev.hit_true_dca[ev.hit_off[i]])) ** 2
                for i in range(ev.n_fired)
                if ev.hit_off[i + 1] - ev.hit_off[i] == 2 and ev.hit_turn[ev.hit_off[i]] == p
                and abs(ev.rho[ev.hit_off[i]]) > 0]
        got = [min(abs(abs(D[i]) - abs(ev.rho[ev.hit_off[i]])), lam) ** 2
               for i in range(ev.n_fired)
               if ev.hit_off[i + 1] - ev.hit_off[i] == 2 and ev.hit_turn[ev.hit_off[i]] == p
               and abs(ev.rho[ev.hit_off[i]]) > 0]
        if pure:
            np.testing.assert_allclose(np.minimum(pure, lam * lam), got, rtol=0, atol=5e-10)


def test_rss_bounds_monotonicity_and_ghost_symmetry(cfg0_event):
    ev = cfg0_event
    seeds, _ = event_seeds(ev)
    seeds = np.ascontiguousarray(seeds[:, ::37])
    W = ev.n_fired
    prev = None
    for lam in (0.02, 0.05, 0.1, 0.2, 0.8):
        rss = _scan(ev, seeds, cutoff=lam)["rss"]
        assert np.all(rss >= 0.0) and np.all(rss <= W * lam * lam * (1 + 1e-15))
        if prev is not None:
            assert np.all(rss >= prev)           # non-decreasing in lambda, term by term
        prev = rss
    base = _scan(ev, seeds)["rss"]
    flipped = _scan(ev, seeds, rho=-ev.rho)["rss"]   # both ghosts present: set of rho per wire unchanged
    np.testing.assert_array_equal(base, flipped)


def test_far_seed_gives_exactly_W_lambda_squared(cfg0_event):
    ev = cfg0_event
    far = truth_seed(ev, 0).reshape(6, 1).copy()
    far[2, 0] += 60.0                                  # 60 cm along z: nowhere near any fired wire's DCA
    far[3:5, 0] *= -1.0
    lam = ev.cutoff
    r = _scan(ev, np.ascontiguousarray(far))
    expect = 0.0
    for _ in range(ev.n_fired):
        expect = expect + lam * lam
    assert r["rss"][0] == expect


def test_eq1_from_signed_dca_bruteforce(cfg1_event):
    """RSS, argmin and classification recomputed by plain Python loops from the signed DCAs."""
    ev = cfg1_event
    seeds, part_off = event_seeds(ev, shape=(4, 3, 3, 3))
    r = _scan(ev, seeds, want_dca=True)
    lam = ev.cutoff
    S = seeds.shape[1]
    rss = np.zeros(S)
    for s in range(S):
        acc = 0.0
        for i in range(ev.n_fired):
            best = min(abs(r["dca"][s, i] - ev.rho[j]) for j in range(ev.hit_off[i], ev.hit_off[i + 1]))
            acc += min(best, lam) ** 2
        rss[s] = acc
    np.testing.assert_allclose(r["rss"], rss, rtol=1e-14, atol=0)
    sel = _select(ev, seeds, r["rss"], part_off)
    P = len(part_off) - 1
    for p in range(P):
        lo, hi = part_off[p], part_off[p + 1]
        b = lo + int(np.argmin(r["rss"][lo:hi]))          # numpy argmin = first occurrence
        assert sel["best_seed"][p] == b
        assert sel["best_rss"][p] == r["rss"][b]
        np.testing.assert_array_equal(sel["best_dca"][p], r["dca"][b])
        cls = np.zeros(ev.n_hits, dtype=np.uint8)
        for i in range(ev.n_fired):
            js = list(range(ev.hit_off[i], ev.hit_off[i + 1]))
            res = [abs(r["dca"][b, i] - ev.rho[j]) for j in js]
            jm = js[int(np.argmin(res))]
            if min(res) < lam:
                cls[jm] = 1
        np.testing.assert_array_equal(sel["cls"][p], cls)
        # at most one classified entry per (partition, wire), all with residual < lambda
        for i in range(ev.n_fired):
            assert sel["cls"][p][ev.hit_off[i]:ev.hit_off[i + 1]].sum() <= 1


def test_argmin_ties_and_permutation():
    """Tie -> lowest seed index (reading R15); permuting seeds permutes the result."""
    ev = make_config(0)[0]
    seeds, _ = event_seeds(ev, shape=(3, 2, 2, 2))
    S = seeds.shape[1]
    r = _scan(ev, seeds)
    # duplicate the whole set: every rss value appears twice, the first copy must win
    dup = np.ascontiguousarray(np.concatenate([seeds, seeds], axis=1))
    r2 = _scan(ev, dup)
    np.testing.assert_array_equal(r2["rss"][:S], r["rss"])
    np.testing.assert_array_equal(r2["rss"][S:], r["rss"])
    sel = _select(ev, dup, r2["rss"], np.array([0, 2 * S], dtype=np.int64))
    assert sel["best_seed"][0] == int(np.argmin(r["rss"]))
    # two partitions over the two copies: second partition's winner is the same seed + S
    sel2 = _select(ev, dup, r2["rss"], np.array([0, S, 2 * S], dtype=np.int64))
    assert sel2["best_seed"][1] == sel2["best_seed"][0] + S
    np.testing.assert_array_equal(sel2["cls"][0], sel2["cls"][1])
    perm = np.random.default_rng(5).permutation(S)
    rp = _scan(ev, np.ascontiguousarray(seeds[:, perm]))
    np.testing.assert_array_equal(rp["rss"], r["rss"][perm])


def test_classification_toy_event_hand_computed():
    """Straight track along +x at y = 0 (B = 0); three axial wires at y = +1, -2, +0.5 with
    hand-picked drift entries; lambda = 0.1."""
    wa = np.ascontiguousarray(np.array([[3, 1, -50], [5, -2, -50], [7, 0.5, -50]], dtype=np.float64).T)
    wb = np.ascontiguousarray(np.array([[3, 1, 50], [5, -2, 50], [7, 0.5, 50]], dtype=np.float64).T)
    fired = np.array([0, 1, 2], dtype=np.int32)
    # signed DCAs are +1, -2, +0.5 (see test_oracle_dca_pins sign case)
    # wire 0: entries +-1.03            -> closest +1.03, residual 0.03  -> classified
    # wire 1: entries +-1.85, +-2.3     -> closest -1.85, residual 0.15  -> NOT classified (> lambda)
    # wire 2: entries +-0.9, +-0.45     -> closest +0.45, residual 0.05  -> classified
    rho = np.array([1.03, -1.03, 1.85, -1.85, 2.3, -2.3, 0.9, -0.9, 0.45, -0.45])
    hit_off = np.array([0, 2, 6, 10], dtype=np.int32)
    seeds = np.array([[0.0], [0.0], [0.0], [100.0], [0.0], [0.0]])
    lam = 0.1
    r = O.scan(seeds, -1, 0.0, 0.5, 40, 0.0, wa, wb, fired, hit_off, rho, lam, want_dca=True)
    expect = 0.03 ** 2 + lam ** 2 + 0.05 ** 2
    assert abs(r["rss"][0] - expect) < 1e-15
    sel = O.select_classify(seeds, -1, 0.0, 0.5, 40, 0.0, wa, wb, fired, hit_off, rho, lam, r["rss"],
                            np.array([0, 1], dtype=np.int64))
    np.testing.assert_array_equal(sel["cls"][0], [1, 0, 0, 0, 0, 0, 0, 0, 1, 0])
    # strict '<' (reading R13): residual exactly lambda is not classified
    rho2 = rho.copy()
    rho2[0], rho2[1] = 1.0 + lam, -(1.0 + lam)
    sel2 = O.select_classify(seeds, -1, 0.0, 0.5, 40, 0.0, wa, wb, fired, hit_off, rho2, 1.0 + lam - 1.0,
                             r["rss"], np.array([0, 1], dtype=np.int64))
    assert sel2["cls"][0][0] == 0
    # r = 0: both ghosts tie, the lower index is the classified one (reading R12)
    rho3 = rho.copy()
    rho3[0], rho3[1] = 0.0, -0.0
    sel3 = O.select_classify(seeds, -1, 0.0, 0.5, 40, 0.0, wa, wb, fired, hit_off, rho3, 1.5, r["rss"],
                             np.array([0, 1], dtype=np.int64))
    assert sel3["cls"][0][0] == 1 and sel3["cls"][0][1] == 0


def test_truth_seed_classifies_its_own_hits(cfg1_event):
    """With the truth seed as the only seed of a partition, the classified entries are the
    real-side entries of that turn whose smear is below lambda (plus nothing from far turns)."""
    ev = cfg1_event
    for p in range(len(ev.partitions)):
        seeds = truth_seed(ev, p).reshape(6, 1)
        r = _scan(ev, seeds)
        sel = _select(ev, seeds, r["rss"], np.array([0, 1], dtype=np.int64))
        cls = sel["cls"][0].astype(bool)
        own_real = (ev.hit_turn == p) & (ev.hit_real == 1)
        eps = np.abs(np.abs(ev.rho) - np.abs(ev.hit_true_dca))
        must = own_real & (eps < ev.cutoff - 1e-6)
        # an own hit can lose only to another entry on the same wire that is even closer
        lost = must & ~cls
        for j in np.nonzero(lost)[0]:
            i = np.searchsorted(ev.hit_off, j, side="right") - 1
            assert cls[ev.hit_off[i]:ev.hit_off[i + 1]].sum() == 1
        assert (must & cls).sum() >= 0.8 * must.sum()      # the rest lost to a closer entry (checked above)
        # purity against truth labels (metric definition of)
        assert (cls & (ev.hit_turn == p)).sum() >= 0.8 * cls.sum()
