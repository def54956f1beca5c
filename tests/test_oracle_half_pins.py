"""Pins for the oracle's half-track scheme (readings R38-R42)."""
import numpy as np

from comet_synth import hough_tables, make_config, truth_seed
from oracle import comet_oracle as O

R_HALF = 1.0e3          # R42: a target region beyond the chamber = stop at the apex


def _exit_seed(ev, part):
    """The generating truth at the partition's inward r = 50 crossing (closed-form helix of the generator)."""
    h, pt = ev.helix(), ev.partitions[part]
    return np.concatenate([h.position(np.asarray(pt.s_out)), ev.pmag * h.tangent(np.asarray(pt.s_out))])


def test_backward_extrapolation_retraces_the_forward_helix():
    """Flipping the charge AND the momentum runs the same helix backwards (time reversal): the backward track
    from the truth exit state lies on the generator's closed-form helix at s_out - k h.  Flipping only one of
    the two gives a circle of the opposite curvature and misses by centimetres."""
    ev = make_config(1)[0]
    h = ev.helix()
    for part in range(len(ev.partitions)):
        pt = ev.partitions[part]
        back = O.flip_seeds(_exit_seed(ev, part).reshape(6, 1))
        tr, n = O.extrapolate(back, -ev.charge, ev.bz, ev.step, ev.n_steps, 0.0)
        k = np.arange(200)
        want = h.position(pt.s_out - ev.step * k)
        assert np.abs(tr[0, :200, :3] - want).max() < 1e-8
        # the tangent recorded on the way back is minus the forward tangent
        assert np.abs(tr[0, :200, 3:] + h.tangent(pt.s_out - ev.step * k)).max() < 1e-9
        for q, sd in ((ev.charge, back), (-ev.charge, _exit_seed(ev, part).reshape(6, 1))):
            wrong, _ = O.extrapolate(sd, q, ev.bz, ev.step, ev.n_steps, 0.0)
            assert np.abs(wrong[0, 150, :2] - want[150, :2]).max() > 1.0
    np.testing.assert_array_equal(O.flip_seeds(O.flip_seeds(back)), back)


def test_half_track_ends_at_the_apex():
    """R42: with the target region beyond the chamber the recording stops at the first state that moves inwards:
    k = ceil(s_apex / h) with s_apex the arc length at which x.T changes sign on the closed-form helix; the forward
    half from the entrance and the backward half from the exit meet there (their arc lengths add up to the turn)."""
    from scipy.optimize import brentq
    ev = make_config(1)[0]
    h = ev.helix()
    for part in range(len(ev.partitions)):
        pt = ev.partitions[part]

        def radial(s):
            x, t = h.position(np.asarray(s)), h.tangent(np.asarray(s))
            return float(x[0] * t[0] + x[1] * t[1])
        s_apex = brentq(radial, pt.s_in + 1.0, pt.s_out - 1.0, xtol=1e-12)
        fwd = truth_seed(ev, part).reshape(6, 1)
        _, n_f = O.extrapolate(fwd, ev.charge, ev.bz, ev.step, ev.n_steps, R_HALF)
        assert n_f[0] == int(np.ceil((s_apex - pt.s_in) / ev.step)) + 1
        back = O.flip_seeds(_exit_seed(ev, part).reshape(6, 1))
        _, n_b = O.extrapolate(back, -ev.charge, ev.bz, ev.step, ev.n_steps, R_HALF)
        assert n_b[0] == int(np.ceil((pt.s_out - s_apex) / ev.step)) + 1
        assert abs((n_f[0] + n_b[0] - 2) * ev.step - (pt.s_out - pt.s_in)) < 2 * ev.step


def _fake_wires(xy):
    xy = np.asarray(xy, np.float64)
    wa = np.stack([xy[:, 0], xy[:, 1], np.full(len(xy), -75.0)])
    wb = np.stack([xy[:, 0], xy[:, 1], np.full(len(xy), 75.0)])
    return wa, wb


def test_half_hit_masks_hand_case_and_restatement():
    # circle centred on the +x axis (R = 40): the dividing line is the x axis; entrance point below it
    circle = np.array([40.0, 40.0, 0.0, 30.0, -40.0, 0, 0, 30.0, 40.0, 0, 0])
    wa, wb = _fake_wires([(60, -5), (60, 5), (70, -0.5), (70, 0.5), (75, 0.0)])
    fired = np.arange(5, dtype=np.int32)
    hit_off = np.array([0, 2, 4, 8, 10, 12], dtype=np.int32)
    e, x = O.half_hit_masks(wa, wb, fired, hit_off, 12, circle, 0.0)
    assert e.tolist() == [1, 1, 0, 0, 1, 1, 1, 1, 0, 0, 0, 0]          # y < 0: the entrance side
    assert x.tolist() == [0, 0, 1, 1, 0, 0, 0, 0, 1, 1, 1, 1]          # y >= 0 (on the line -> exit)
    e, x = O.half_hit_masks(wa, wb, fired, hit_off, 12, circle, 1.0)   # 1 cm band: wires 2, 3, 4 in both
    assert e.tolist() == [1, 1, 0, 0, 1, 1, 1, 1, 1, 1, 1, 1]
    assert x.tolist() == [0, 0, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1]
    # entrance on the other side: the sets swap (the line itself stays with the exit)
    circle2 = circle.copy()
    circle2[3:5] = (30.0, 40.0)
    e2, x2 = O.half_hit_masks(wa, wb, fired, hit_off, 12, circle2, 0.0)
    assert e2.tolist() == [0, 0, 1, 1, 0, 0, 0, 0, 1, 1, 0, 0] and x2.tolist() == [1, 1, 0, 0, 1, 1, 1, 1, 0, 0, 1, 1]
    # vectorised restatement on a real event with a rotated circle; without overlap the sets partition the entries
    ev = make_config(1)[0]
    c, s = hough_tables(256)
    hs = O.hough_seeds(ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, c, s, 1 / 120.0, 128 * 120.0 * 40 / 80, 128,
                       ev.charge, ev.bz, 50.0)
    circ = np.concatenate([[hs["R"]], hs["centre"], hs["entrance"], hs["exit"]])
    for ov in (0.0, 3.0):
        e, x = O.half_hit_masks(ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.n_hits, circ, ov)
        m = (ev.geom.wire_a[:2, ev.fired_wire] + ev.geom.wire_b[:2, ev.fired_wire]) / 2
        chat = circ[1:3] / np.hypot(*circ[1:3])
        d = chat[0] * m[1] - chat[1] * m[0]                             # distance from the origin-centre line
        side_e = np.sign(chat[0] * circ[4] - chat[1] * circ[3])
        cnt = np.diff(ev.hit_off)
        clear = np.abs(np.abs(d) - ov) > 1e-9
        np.testing.assert_array_equal(e[np.repeat(clear, cnt)], np.repeat(side_e * d > -ov, cnt)[np.repeat(clear, cnt)])
        np.testing.assert_array_equal(x[np.repeat(clear, cnt)], np.repeat(side_e * d <= ov, cnt)[np.repeat(clear, cnt)])
        if ov == 0.0:
            assert np.all(e + x == 1)
        else:
            assert np.all(e + x >= 1) and np.any(e + x == 2)
    # no circle: nothing is grouped
    e, x = O.half_hit_masks(ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.n_hits, np.full(11, np.nan), 1.0)
    assert not e.any() and not x.any()


def test_layer_veto_hand_cases_and_restatement():
    layer = np.array([0, 0, 1, 2, 3, 3, 5], dtype=np.int32)            # 7 wires
    fired = np.array([0, 2, 3, 4, 6], dtype=np.int32)                   # layers 0, 1, 2, 3, 5
    hit_off = np.array([0, 2, 4, 6, 8, 10], dtype=np.int32)
    rows = np.array([
        [1, 0, 0, 1, 1, 0, 0, 0, 0, 0],     # layers 0, 1, 2: contiguous from 0 -> kept
        [1, 0, 0, 0, 1, 0, 0, 0, 0, 0],     # 0, 2: layer 1 missing
        [0, 0, 1, 0, 1, 0, 0, 0, 0, 0],     # 1, 2: layer 0 missing
        [0, 0, 0, 0, 0, 0, 0, 0, 0, 0],     # nothing classified
        [1, 0, 1, 0, 1, 0, 1, 0, 0, 1],     # 0, 1, 2, 3, 5: layer 4 missing
        [1, 1, 0, 0, 0, 0, 0, 0, 0, 0],     # layer 0 only
    ], dtype=np.uint8)
    assert O.layer_veto(rows, fired, hit_off, layer, 1).tolist() == [1, 0, 0, 0, 0, 1]
    assert O.layer_veto(rows, fired, hit_off, layer, 3).tolist() == [1, 0, 0, 0, 0, 0]
    assert O.layer_veto(rows, fired, hit_off, layer, 4).tolist() == [0, 0, 0, 0, 0, 0]
    rng = np.random.default_rng(5)
    geom = make_config(0)[0].geom
    fired = np.sort(rng.permutation(geom.n_wires)[:150]).astype(np.int32)
    cnt = 2 * rng.integers(1, 3, size=150)
    hit_off = np.concatenate([[0], np.cumsum(cnt)]).astype(np.int32)
    lay_of_entry = np.repeat(geom.layer[fired], cnt)
    cls = (rng.uniform(size=(40, hit_off[-1])) < rng.uniform(0.0, 0.2, size=(40, 1))).astype(np.uint8)
    cls[:8] = lay_of_entry[None, :] <= np.arange(8)[:, None] + 3      # some rows that pass
    got = O.layer_veto(cls, fired, hit_off, geom.layer, 4)
    for a in range(40):
        present = np.bincount(lay_of_entry[cls[a].astype(bool)], minlength=20) > 0
        n_lead = 20 if present.all() else int(np.argmin(present))      # leading run of hit layers
        want = present.any() and present.sum() == n_lead and n_lead >= 4
        assert got[a] == int(want)
    assert got[:8].all() and not got.all()


def test_merge_half_sets_hand_case_and_invariants():
    cls_e = np.array([[1, 0, 1, 0], [0, 1, 0, 0]], dtype=np.uint8)
    orig_e = np.array([0, 1, 4, 5], dtype=np.int32)
    cls_x = np.array([[0, 1], [1, 0], [1, 1]], dtype=np.uint8)
    orig_x = np.array([4, 7], dtype=np.int32)
    m = O.merge_half_sets(cls_e, orig_e, [1, 1], cls_x, orig_x, [1, 0, 1], 8)
    assert m["valid"].tolist() == [[1, 0, 1], [1, 0, 1]]
    assert m["cls"][0, 0].tolist() == [1, 0, 0, 0, 1, 0, 0, 1]
    assert m["cls"][0, 2].tolist() == [1, 0, 0, 0, 1, 0, 0, 1]          # entry 4 from both halves counts once
    assert m["cls"][1, 2].tolist() == [0, 1, 0, 0, 1, 0, 0, 1]
    assert not m["cls"][:, 1].any()
    assert m["n_cls"].tolist() == [[3, 0, 3], [2, 0, 3]]
    rng = np.random.default_rng(9)
    He, Hx, H = 30, 26, 60
    oe, ox = np.sort(rng.permutation(H)[:He]).astype(np.int32), np.sort(rng.permutation(H)[:Hx]).astype(np.int32)
    ce, cx = (rng.uniform(size=(5, He)) < 0.3).astype(np.uint8), (rng.uniform(size=(4, Hx)) < 0.3).astype(np.uint8)
    ok_e, ok_x = np.array([1, 0, 1, 1, 1]), np.array([1, 1, 0, 1])
    m = O.merge_half_sets(ce, oe, ok_e, cx, ox, ok_x, H)
    np.testing.assert_array_equal(m["valid"], np.outer(ok_e, ok_x))
    for a in range(5):
        for b in range(4):
            want = set(oe[ce[a].astype(bool)]) | set(ox[cx[b].astype(bool)]) if ok_e[a] and ok_x[b] else set()
            assert set(np.flatnonzero(m["cls"][a, b])) == want and m["n_cls"][a, b] == len(want)


def test_two_truth_half_tracks_cover_the_turn():
    """On a synthetic turn the forward half from the truth entrance and the backward half from the truth exit,
    each against its own hit set (3 cm overlap around the Hough apex line), classify true entries only and
    together every hit the full-length truth track classifies."""
    ev = make_config(0)[0]
    c, s = hough_tables(256)
    hs = O.hough_seeds(ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, c, s, 1 / 120.0, 128 / (1 / 40.0 - 1 / 120.0), 128,
                       ev.charge, ev.bz, 50.0)
    circ = np.concatenate([[hs["R"]], hs["centre"], hs["entrance"], hs["exit"]])
    args = (ev.bz, ev.step, ev.n_steps, R_HALF, ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.rho,
            ev.cutoff, ev.geom.layer, circ, 3.0, 3)
    kw = dict(half_width=[0.0, 0.0, 0.0, 0.0], n_grid=[1, 1, 1, 1], n_iter=0, shrink=1.0, k_ref=1, k_final=1)
    se, sx = truth_seed(ev, 0).reshape(6, 1), _exit_seed(ev, 0).reshape(6, 1)
    out = O.scan_half_tracks(se, sx, ev.charge, *args, **kw)
    np.testing.assert_array_equal(out["ent"]["final_seed"][0], se[:, 0])
    np.testing.assert_array_equal(out["ext"]["final_seed"][0], sx[:, 0])           # returned in the forward convention
    full = O.classify_seeds(se, [0], ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a, ev.geom.wire_b,
                            ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff)["cls"][0].astype(bool)
    assert full.sum() >= 15
    assert out["ent"]["ok"][0] == 1 and out["ext"]["ok"][0] == 1 and out["valid"].tolist() == [[1]]
    merged = out["cls"][0, 0].astype(bool)
    assert np.all(ev.hit_real[merged] == 1)                                        # true entries only
    assert np.all(merged[full])                                                    # the halves cover the turn
    assert out["n_cls"][0, 0] == merged.sum()
    for key in ("ent", "ext"):                                                     # each half contributes
        assert out[key]["cls"][0].sum() >= 5
    # the sign of the drift on the way back matters: with +rho the backward half picks the ghosts
    ex = out["ext"]
    bad = O.scan_stage(O.flip_seeds(sx), np.array([0, 1]), -ev.charge, ev.bz, ev.step, ev.n_steps, R_HALF, ev.geom.wire_a,
                       ev.geom.wire_b, ex["fired_wire"], ex["hit_off"], ev.rho[ex["orig"]], ev.cutoff, **kw)
    picked = ex["orig"][bad["cls"][0, 0].astype(bool)]
    assert picked.size >= 5 and np.mean(ev.hit_real[picked]) < 0.5


def test_best_pair_hand_cases():
    valid = np.array([[1, 0, 1], [1, 1, 0]], dtype=np.uint8)
    n = np.array([[5, 99, 7], [7, 6, 50]], dtype=np.int32)
    assert O.best_pair(valid, n) == 2                     # 7 at (0, 2) and (1, 0): the lower flat index; 99 and 50 are not valid
    assert O.best_pair(np.zeros((2, 3), np.uint8), n) == -1
    assert O.best_pair(np.ones((2, 3), np.uint8), n) == 1
    assert O.best_pair(np.ones((1, 1), np.uint8), np.zeros((1, 1), np.int32)) == 0       # a valid empty set still counts
    rng = np.random.default_rng(4)
    for _ in range(50):
        v, m = (rng.uniform(size=(4, 5)) < 0.5).astype(np.uint8), rng.integers(0, 6, size=(4, 5)).astype(np.int32)
        key = np.where(v.ravel() > 0, m.ravel(), -1)
        want = int(np.argmax(key)) if key.max() >= 0 else -1                             # first maximum
        assert O.best_pair(v, m) == want


def _turn_seed_sets(ev, shape_e=(5, 5, 5, 4), shape_x=(5, 5, 4, 5)):
    from comet_synth import seed_grid
    pr = tuple(ev.spec["p_range"])
    se, sx = [], []
    for p in range(len(ev.partitions)):
        se.append(seed_grid(ev, p, shape_e, pr, ct_hw=0.15))
        x, T = _exit_seed(ev, p)[:3], _exit_seed(ev, p)[3:] / ev.pmag
        g = seed_grid(ev, p, shape_x, pr, ct_hw=0.15)                # the partition's grid moved to the exit state
        pt = ev.partitions[p]
        rot = np.arctan2(T[1], T[0]) - pt.phi
        px, py = g[3].copy(), g[4].copy()
        g[0], g[1], g[2] = x[0], x[1], g[2] + (x[2] - pt.z)
        g[3], g[4] = px * np.cos(rot) - py * np.sin(rot), px * np.sin(rot) + py * np.cos(rot)
        sx.append(g)
    off = lambda blocks: np.concatenate([[0], np.cumsum([b.shape[1] for b in blocks])]).astype(np.int64)
    return np.concatenate(se, axis=1), off(se), np.concatenate(sx, axis=1), off(sx)


def test_event_loop_with_half_tracks_takes_turns_apart():
    ev = make_config(1)[0]
    c, s = hough_tables(256)
    hs = O.hough_seeds(ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, c, s, 1 / 120.0, 128 / (1 / 40.0 - 1 / 120.0), 128,
                       ev.charge, ev.bz, 50.0)
    circ = np.concatenate([[hs["R"]], hs["centre"], hs["entrance"], hs["exit"]])
    se, oe, sx, ox = _turn_seed_sets(ev)
    args = (ev.charge, ev.bz, ev.step, ev.n_steps, R_HALF, ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, ev.hit_off,
            ev.rho, ev.cutoff, ev.geom.layer, circ, 3.0, 3)
    kw = dict(half_width=[1.0, 1.2, 1.2, 1.5], n_grid=[3, 3, 3, 3], n_iter=2, shrink=0.5, k_ref=3, k_final=3)
    out = O.scan_turns_half(se, oe, sx, ox, *args, min_wires=10, **kw)
    P = len(oe) - 1
    assert out["done"].all() and (out["turn_pair"] >= 0).all()
    wb = out["wires_before"]
    assert wb[P - 1] == ev.n_fired and np.all(np.diff(wb[::-1]) < 0)       # fewer wires for every earlier turn
    cls = out["turn_cls"].astype(int)
    assert cls.sum(axis=0).max() == 1                                      # a hit entry goes to one turn only
    assert cls.sum(axis=0).reshape(-1, 2).sum(axis=1).max() == 1           # never both ghosts of a hit
    turn = np.asarray(ev.hit_turn)
    for p in range(P):
        got = turn[cls[p].astype(bool)]
        assert got.size == out["turn_n"][p] >= 30 and np.mean(got == p) > 0.75
    # the first stage is scan_half_tracks on the full list with best_pair's choice
    ht = O.scan_half_tracks(se[:, oe[P - 1]:oe[P]], sx[:, ox[P - 1]:ox[P]], *args, **kw)
    a, b = divmod(O.best_pair(ht["valid"], ht["n_cls"]), 3)
    assert tuple(out["turn_pair"][P - 1]) == (a, b)
    np.testing.assert_array_equal(out["turn_cls"][P - 1], ht["cls"][a, b])
    np.testing.assert_array_equal(out["turn_seed"][P - 1, 0], ht["ent"]["final_seed"][a])
    np.testing.assert_array_equal(out["turn_seed"][P - 1, 1], ht["ext"]["final_seed"][b])
    # stopping rules: max_tracks, min_wires, and a turn without a valid pair (a veto nothing passes)
    one = O.scan_turns_half(se, oe, sx, ox, *args, min_wires=10, max_tracks=1, **kw)
    assert one["done"].tolist() == [False] * (P - 1) + [True]
    none = O.scan_turns_half(se, oe, sx, ox, *args, min_wires=ev.n_fired + 1, **kw)
    assert not none["done"].any() and not none["wires_before"].any()
    veto = O.scan_turns_half(se, oe, sx, ox, *args[:-1], 21, min_wires=10, **kw)
    assert not veto["done"].any() and veto["wires_before"].tolist() == [0] * (P - 1) + [ev.n_fired]
    assert not veto["turn_cls"].any() and np.isnan(veto["turn_seed"]).all()
