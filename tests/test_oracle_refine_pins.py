"""Pins for the oracle's iterative seed refinement (O12, O13, scan_stage).

The paper prints no numbers for this step, so the pins are hand-computed toy cases, a brute force written
differently (sort + walk instead of repeated minimum), invariants of the selection rule, numpy's linspace,
and the physics: refining around the lowest-RSS seeds must move the best seed towards the generating truth.
"""
import numpy as np
import pytest

from comet_synth import event_seeds, make_config, truth_seed
from oracle import comet_oracle as O


def _toy_seeds(z, px=None, py=None, pz=None):
    n = len(z)
    s = np.zeros((6, n))
    s[0], s[1] = 50.0, 0.0
    s[2] = z
    s[3] = 0.0 if px is None else px
    s[4] = 100.0 if py is None else py
    s[5] = 20.0 if pz is None else pz
    return s


def test_select_references_hand_case():
    # boxes of half width 1 overlap iff |dz| < 2 (strict): walking in RSS order 1, 2, 3, 4, 0:
    # 1 taken; 2 overlaps 1; 3 is exactly 2 away from 1 -> taken; 4 taken; 0 overlaps 1.
    seeds = _toy_seeds([0.0, 1.0, 2.0, 3.0, 10.0])
    rss = np.array([5.0, 1.0, 2.0, 3.0, 4.0])
    po = np.array([0, 5])
    assert O.select_references(seeds, rss, po, [1, 1, 1, 1], 3).tolist() == [[1, 3, 4]]
    assert O.select_references(seeds, rss, po, [1, 1, 1, 1], 5).tolist() == [[1, 3, 4, -1, -1]]
    # a wider box swallows seed 3 as well
    assert O.select_references(seeds, rss, po, [1.01, 1, 1, 1], 3).tolist() == [[1, 4, -1]]
    # boxes must overlap in EVERY dimension: separating seed 2 in p_x frees it
    seeds2 = _toy_seeds([0.0, 1.0, 2.0, 3.0, 10.0], px=[0, 0, 2.0, 0, 0])
    assert O.select_references(seeds2, rss, po, [1, 1, 1, 1], 3).tolist() == [[1, 2, 3]]


def test_select_references_ties_nan_and_zero_width():
    seeds = _toy_seeds([0.0, 5.0, 10.0, 15.0])
    po = np.array([0, 4])
    # ties -> lowest index; NaN is never a reference
    assert O.select_references(seeds, np.array([2.0, 1.0, 1.0, np.nan]), po, [1, 1, 1, 1], 4).tolist() == [[1, 2, 0, -1]]
    # zero width: nothing overlaps, but a seed is never selected twice
    same = _toy_seeds([1.0, 1.0, 1.0])
    assert O.select_references(same, np.array([3.0, 2.0, 1.0]), np.array([0, 3]), [0, 0, 0, 0], 4).tolist() == [[2, 1, 0, -1]]
    # empty partition
    assert O.select_references(seeds, np.ones(4), np.array([0, 0, 4]), [1, 1, 1, 1], 2).tolist() == [[-1, -1], [0, 1]]


def _greedy_sorted(seeds, rss, lo, hi, hw, k):
    """The same rule written as sort + walk (the paper's wording: go down the list of lowest-RSS seeds)."""
    idx = [s for s in range(lo, hi) if not np.isnan(rss[s])]
    idx.sort(key=lambda s: (rss[s], s))
    sel = []
    for s in idx:
        if len(sel) == k:
            break
        if all(any(not (abs(seeds[2 + d, s] - seeds[2 + d, t]) < 2.0 * hw[d]) for d in range(4)) for t in sel):
            sel.append(s)
    return sel + [-1] * (k - len(sel))


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_select_references_brute_force_and_invariants(seed):
    rng = np.random.default_rng(seed)
    n = 600
    s = np.zeros((6, n))
    s[2:] = rng.integers(0, 7, size=(4, n)) * np.array([[0.5], [1.0], [1.0], [2.0]])   # a grid: many exact ties of |d| = 2 hw
    rss = rng.integers(0, 40, size=n).astype(float) * 0.01
    rss[rng.integers(0, n, 5)] = np.nan
    po = np.array([0, 250, 250, 600])
    hw = np.array([0.5, 1.0, 1.5, 2.0])
    k = 9
    ref = O.select_references(s, rss, po, hw, k)
    for p in range(3):
        assert ref[p].tolist() == _greedy_sorted(s, rss, po[p], po[p + 1], hw, k)
        sel = [x for x in ref[p] if x >= 0]
        for i, a in enumerate(sel):          # pairwise sparse
            for b in sel[:i]:
                assert any(abs(s[2 + d, a] - s[2 + d, b]) >= 2 * hw[d] for d in range(4))
        if sel:                              # maximal: every better seed that was passed over is blocked
            last = sel[-1]
            for t in range(po[p], po[p + 1]):
                if t in sel or np.isnan(rss[t]) or (rss[t], t) > (rss[last], last):
                    continue
                assert any(all(abs(s[2 + d, t] - s[2 + d, b]) < 2 * hw[d] for d in range(4)) for b in sel)
    # k = 1 is the argmin of O10
    r1 = O.select_references(s, np.nan_to_num(rss, nan=9.0), po, hw, 1)
    assert r1[0, 0] == np.lexsort((np.arange(250), np.nan_to_num(rss, nan=9.0)[:250]))[0]


def test_refine_seeds_against_linspace_and_hand_order():
    rng = np.random.default_rng(3)
    seeds = rng.normal(size=(6, 40)) * 10
    ref = np.array([[7, 11, -1], [30, -1, -1]], dtype=np.int64)
    hw = np.array([1.5, 0.25, 2.0, 0.0])
    ng = np.array([4, 3, 2, 1], dtype=np.int32)
    new, po = O.refine_seeds(seeds, ref, hw, ng)
    G = 24
    assert new.shape == (6, 2 * 3 * G) and po.tolist() == [0, 3 * G, 6 * G]
    for p in range(2):
        for r in range(3):
            src = ref[p, r] if ref[p, r] >= 0 else ref[p, 0]      # an empty slot repeats the first reference
            blk = new[:, (p * 3 + r) * G:(p * 3 + r + 1) * G]
            assert np.all(blk[0] == seeds[0, src]) and np.all(blk[1] == seeds[1, src])
            axes = [np.linspace(seeds[2 + d, src] - hw[d], seeds[2 + d, src] + hw[d], ng[d]) if ng[d] > 1
                    else np.array([seeds[2 + d, src]]) for d in range(4)]
            grid = np.stack(np.meshgrid(*axes, indexing="ij"), axis=0).reshape(4, G)   # last dimension fastest
            np.testing.assert_allclose(blk[2:], grid, rtol=0, atol=1e-13)
            assert blk[5, 0] == seeds[5, src]                                          # n = 1: the value itself
            assert blk[2, 0] == seeds[2, src] - hw[0]                                  # first point is lo exactly
    # hand order: index ((j0 n1 + j1) n2 + j2) n3 + j3 -> seed 1 differs from seed 0 in p_y, seed 2 in p_x
    b0 = new[:, :G]
    assert b0[4, 1] > b0[4, 0] and b0[3, 1] == b0[3, 0]
    assert b0[3, 2] > b0[3, 0] and b0[2, 2] == b0[2, 0]
    assert b0[2, 6] > b0[2, 0]


def test_new_seed_sets_of_selected_references_do_not_overlap():
    rng = np.random.default_rng(4)
    n = 300
    s = np.zeros((6, n))
    s[2:] = rng.uniform(-3, 3, size=(4, n))
    rss = rng.uniform(size=n)
    hw = np.array([0.6, 0.5, 0.7, 0.4])
    ref = O.select_references(s, rss, np.array([0, n]), hw, 6)
    assert (ref >= 0).all()
    new, _ = O.refine_seeds(s, ref, hw, np.array([3, 3, 3, 3], dtype=np.int32))
    G = 81
    for a in range(6):
        for b in range(a):
            A, B = new[2:, a * G:(a + 1) * G], new[2:, b * G:(b + 1) * G]
            gap = np.maximum(A.min(axis=1) - B.max(axis=1), B.min(axis=1) - A.max(axis=1))
            assert gap.max() >= -1e-12        # separated (or touching) in at least one dimension


def test_stage_moves_the_best_seed_towards_the_truth():
    ev = make_config(0)[0]
    seeds, po = event_seeds(ev)
    args = (ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire,
            ev.hit_off, ev.rho, ev.cutoff)
    rss0 = O.scan(seeds, *args)["rss"]
    b0 = int(np.argmin(rss0))
    hw = np.array([1.2, 1.0, 1.0, 4.0])
    out = O.scan_stage(seeds, po, *args, half_width=hw, n_grid=[3, 5, 5, 5], n_iter=3, shrink=0.5, k_ref=4, k_final=3)
    assert out["final_seed"].shape == (1, 3, 6) and out["cls"].shape == (1, 3, ev.n_hits)
    best = out["final_seed"][0, 0]
    truth = truth_seed(ev, 0)
    scale = np.array([1.0, 1.0, 1.0, 1.0])
    d0 = np.linalg.norm((seeds[2:, b0] - truth[2:]) / scale)
    d1 = np.linalg.norm((best[2:] - truth[2:]) / scale)
    assert out["final_rss"][0, 0] <= rss0[b0] * (1 + 1e-9)
    assert out["final_rss"][0, 0] < 0.7 * rss0[b0]
    assert d1 < d0
    # the finally selected seeds are sorted by RSS and classify at least as many hits as the coarse best seed
    fr = out["final_rss"][0]
    assert np.all(np.diff(fr[~np.isnan(fr)]) >= 0)
    c0 = O.classify_seeds(seeds, [b0], *args)["cls"].sum()
    assert out["cls"][0, 0].sum() >= c0
    # classification of a listed seed is the O11 rule: it equals select_classify on that seed alone
    one = O.select_classify(np.ascontiguousarray(best.reshape(6, 1)), *args, np.zeros(1), np.array([0, 1]))
    assert np.array_equal(one["cls"][0], out["cls"][0, 0])
    np.testing.assert_array_equal(one["best_dca"][0], out["final_dca"][0, 0])
