"""Pins for the oracle's hit removal and sequential stage loop (readings R33-R34)."""
import numpy as np

from comet_synth import event_seeds, make_config
from oracle import comet_oracle as O


def test_remove_hits_hand_case():
    fired = np.array([10, 11, 12, 13], dtype=np.int32)
    hit_off = np.array([0, 2, 6, 6, 8], dtype=np.int32)          # wire 12 has no entries to begin with
    rho = np.array([0.1, -0.1, 0.2, -0.2, 0.3, -0.3, 0.4, -0.4])
    cls = np.array([0, 1, 0, 0, 1, 0, 0, 0], dtype=np.uint8)     # the -0.1 ghost and the +0.3 ghost are classified
    fw, ho, rh, src = O.remove_hits(fired, hit_off, rho, cls)
    # wire 10 loses its only hit (both ghosts) and goes; wire 11 keeps the 0.2 pair; wire 12 goes; wire 13 stays
    assert fw.tolist() == [11, 13] and ho.tolist() == [0, 2, 4]
    assert rh.tolist() == [0.2, -0.2, 0.4, -0.4] and src.tolist() == [2, 3, 6, 7]
    # nothing classified: only the wire without entries goes
    fw, ho, rh, src = O.remove_hits(fired, hit_off, rho, np.zeros(8, dtype=np.uint8))
    assert fw.tolist() == [10, 11, 13] and ho.tolist() == [0, 2, 6, 8] and src.tolist() == list(range(8))


def test_remove_hits_vectorised_restatement():
    rng = np.random.default_rng(1)
    counts = rng.integers(0, 4, size=300) * 2
    hit_off = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    H = int(hit_off[-1])
    rho = rng.normal(size=H)
    cls = (rng.uniform(size=H) < 0.2).astype(np.uint8)
    fired = rng.permutation(5000)[:300].astype(np.int32)
    fw, ho, rh, src = O.remove_hits(fired, hit_off, rho, cls)
    gone = cls.astype(bool) | cls.reshape(-1, 2)[:, ::-1].reshape(-1).astype(bool)      # entry or its partner
    wire_of = np.repeat(np.arange(300), counts)
    keep = ~gone
    np.testing.assert_array_equal(src, np.flatnonzero(keep))
    np.testing.assert_array_equal(rh, rho[keep])
    left = np.bincount(wire_of[keep], minlength=300)
    np.testing.assert_array_equal(fw, fired[left > 0])
    np.testing.assert_array_equal(ho, np.concatenate([[0], np.cumsum(left[left > 0])]))
    assert np.all(ho % 2 == 0)                                     # pairs stay pairs: the result can be reduced again


def test_stage_loop_takes_turns_apart():
    ev = make_config(1)[0]
    seeds, po = event_seeds(ev, shape=(6, 6, 6, 6))
    args = (ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire,
            ev.hit_off, ev.rho, ev.cutoff)
    kw = dict(half_width=[1.2, 1.0, 1.0, 2.0], n_grid=[3, 3, 3, 3], n_iter=2, shrink=0.5, k_ref=4)
    out = O.scan_turns(seeds, po, *args, **kw)
    P = len(po) - 1
    assert out["done"].all()
    # the last turn is scanned first against all wires; every later stage sees fewer wires
    wb = out["wires_before"]
    assert wb[P - 1] == ev.n_fired and np.all(np.diff(wb[::-1]) < 0)
    # a hit is given to one turn only, ghosts never both
    cls = out["turn_cls"].astype(int)
    assert cls.sum(axis=0).max() == 1
    pair = cls.sum(axis=0).reshape(-1, 2).sum(axis=1)
    assert pair.max() == 1
    # physics: most hits a stage classifies belong to its turn (truth labels of the generator)
    turn_of_entry = np.asarray(ev.hit_turn)                      # per entry
    for p in range(P):
        got = turn_of_entry[cls[p].astype(bool)]
        assert got.size >= 15 and np.mean(got == p) > 0.8
    # the first stage is the plain stage of scan_stage on the full hit list
    sub = np.ascontiguousarray(seeds[:, po[P - 1]:po[P]])
    st = O.scan_stage(sub, np.array([0, sub.shape[1]]), *args, k_final=1, **kw)
    np.testing.assert_array_equal(out["turn_seed"][P - 1], st["final_seed"][0, 0])
    np.testing.assert_array_equal(out["turn_cls"][P - 1], st["cls"][0, 0])
    # stopping rules
    few = O.scan_turns(seeds, po, *args, max_tracks=1, **kw)
    assert few["done"].tolist() == [False] * (P - 1) + [True]
    none = O.scan_turns(seeds, po, *args, min_wires=ev.n_fired + 1, **kw)
    assert not none["done"].any()
