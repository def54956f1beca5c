"""Regression pin: the oracle on BASELINE.json configs[0] against tests/golden/cfg0_oracle.json
(written by tests/golden/make_golden.py from the oracle alone)."""
import json
import os

import numpy as np

from comet_synth import event_seeds
from oracle import comet_oracle as O

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg0_oracle.json")


def test_cfg0_matches_golden(cfg0_event):
    ev = cfg0_event
    g = json.load(open(GOLD))
    seeds, part_off = event_seeds(ev)
    assert seeds.shape[1] == g["n_seeds"] and ev.n_fired == g["n_fired"] and ev.n_hits == g["n_hits"]
    r = O.scan(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a, ev.geom.wire_b,
               ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, want_npts=True)
    sel = O.select_classify(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a,
                            ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, r["rss"], part_off)
    assert int(r["n_pts"].sum()) == g["n_pts_sum"]
    assert [int(v) for v in sel["best_seed"]] == g["best_seed"]
    order = np.argsort(r["rss"], kind="stable")
    assert [int(v) for v in order[:5]] == g["lowest5_seeds"]
    np.testing.assert_allclose(r["rss"][order[:5]], [float.fromhex(v) for v in g["lowest5_rss"]], rtol=1e-13)
    np.testing.assert_allclose(sel["best_dca"][0], [float.fromhex(v) for v in g["best_dca"]], rtol=1e-12, atol=1e-14)
    assert [int(j) for j in np.nonzero(sel["cls"][0])[0]] == g["classified_entries"]


def test_thread_count_does_not_change_results(cfg0_event):
    """the CPU result is deterministic for an arbitrary number of threads."""
    ev = cfg0_event
    seeds, _ = event_seeds(ev)
    seeds = np.ascontiguousarray(seeds[:, ::5])
    args = (seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a, ev.geom.wire_b,
            ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff)
    n0 = O.max_threads()
    try:
        O.set_threads(1)
        a = O.scan(*args, want_dca=True)
        O.set_threads(max(2, n0))
        b = O.scan(*args, want_dca=True)
    finally:
        O.set_threads(n0)
    np.testing.assert_array_equal(a["rss"], b["rss"])
    np.testing.assert_array_equal(a["dca"], b["dca"])
