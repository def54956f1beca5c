"""Half-track scheme on the device vs the oracle through the C ABI (needs one B200): comet_half_hit_masks,
comet_flip_seeds, comet_layer_veto, comet_merge_half_sets and the whole comet_scan_half_tracks.

Byte and index work is compared for identity; the finally selected seeds, their RSS and the hit grouping are
fp64 results of the same IEEE operations on both sides and are compared bit for bit (RSS: 1e-9 relative is the
bar of BASELINE.json, identity is what is observed)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from comet_synth import hough_tables, make_config, seed_grid, truth_seed  # noqa: E402
from oracle import comet_oracle as O  # noqa: E402

R_HALF = 1.0e3


@pytest.fixture(scope="module")
def comet():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_1911_09340_b200 import Comet
    from paper_1911_09340_b200.build import build
    build()
    c = Comet(0)
    yield c
    c.close()


def _dev(a, dt=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dt is not None:
        t = t.to(dt)
    return t.cuda()


def _same_f64(a, b):
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
    ok = ~np.isnan(b)
    return a.shape == b.shape and np.array_equal(np.isnan(a), np.isnan(b)) and np.array_equal(a[ok], b[ok])


def _circle(ev, n_rho=128):
    c, s = hough_tables(256)
    hs = O.hough_seeds(ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, c, s, 1 / 120.0, n_rho / (1 / 40.0 - 1 / 120.0),
                       n_rho, ev.charge, ev.bz, 50.0)
    return np.concatenate([[hs["R"]], hs["centre"], hs["entrance"], hs["exit"]])


def _exit_state(ev, part):
    h, pt = ev.helix(), ev.partitions[part]
    return h.position(np.asarray(pt.s_out)), h.tangent(np.asarray(pt.s_out))


def _exit_grid(ev, part, shape, p_range, rng_hw=(0.15, 0.04, 4.0)):
    """Exit-side seed grid (physical momenta) around the truth exit state, same axes as comet_synth.seed_grid."""
    x, T = _exit_state(ev, part)
    n_p, n_ct, n_phi, n_z = shape
    pa = np.linspace(p_range[0], p_range[1], n_p)
    ca = np.linspace(T[2] - rng_hw[0], T[2] + rng_hw[0], n_ct)
    phi = np.arctan2(T[1], T[0])
    fa = np.linspace(phi - rng_hw[1], phi + rng_hw[1], n_phi)
    za = np.linspace(x[2] - rng_hw[2], x[2] + rng_hw[2], n_z)
    P, C, F, Z = (v.ravel() for v in np.meshgrid(pa, ca, fa, za, indexing="ij"))
    S = np.sqrt(1.0 - C * C)
    return np.ascontiguousarray(np.stack([np.full(P.size, x[0]), np.full(P.size, x[1]), Z,
                                          P * S * np.cos(F), P * S * np.sin(F), P * C]))


@pytest.mark.parametrize("cfg,overlap", [(1, 0.0), (1, 3.0), (4, 1.5)])
def test_half_hit_masks_identical(comet, cfg, overlap):
    ev = make_config(cfg)[0]
    circ = _circle(ev)
    ref_e, ref_x = O.half_hit_masks(ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.n_hits, circ, overlap)
    ge, gx = comet.half_hit_masks(_dev(ev.geom.wire_a), _dev(ev.geom.wire_b), _dev(ev.fired_wire), _dev(ev.hit_off),
                                  ev.n_hits, _dev(circ), overlap)
    assert np.array_equal(ge.cpu().numpy(), ref_e) and np.array_equal(gx.cpu().numpy(), ref_x)
    assert ref_e.any() and ref_x.any()
    # no circle: nothing grouped
    ge, gx = comet.half_hit_masks(_dev(ev.geom.wire_a), _dev(ev.geom.wire_b), _dev(ev.fired_wire), _dev(ev.hit_off),
                                  ev.n_hits, _dev(np.full(11, np.nan)), overlap)
    assert not ge.any().item() and not gx.any().item()


def test_flip_seeds_identical(comet):
    rng = np.random.default_rng(3)
    seeds = rng.normal(size=(6, 1000 + 37))
    seeds[3, 5] = 0.0
    got = comet.flip_seeds(_dev(seeds)).cpu().numpy()
    ref = O.flip_seeds(seeds)
    assert np.array_equal(got.view(np.int64), ref.view(np.int64))            # signed zeros included


def test_layer_veto_identical(comet):
    rng = np.random.default_rng(5)
    geom = make_config(0)[0].geom
    fired = np.sort(rng.permutation(geom.n_wires)[:333]).astype(np.int32)
    cnt = 2 * rng.integers(1, 3, size=fired.size)
    hit_off = np.concatenate([[0], np.cumsum(cnt)]).astype(np.int32)
    H = int(hit_off[-1])
    lay = np.repeat(geom.layer[fired], cnt)
    cls = (rng.uniform(size=(75, H)) < rng.uniform(0.0, 0.3, size=(75, 1))).astype(np.uint8)
    cls[:20] = lay[None, :] <= np.arange(20)[:, None]
    cls[20] = 0
    for min_layers in (1, 4, 12):
        ref = O.layer_veto(cls, fired, hit_off, geom.layer, min_layers)
        got = comet.layer_veto(_dev(cls), _dev(fired), _dev(hit_off), _dev(geom.layer), min_layers).cpu().numpy()
        assert np.array_equal(got, ref)
        assert ref[:20].sum() == 20 - (min_layers - 1) and ref[20] == 0


def test_merge_half_sets_identical(comet):
    rng = np.random.default_rng(9)
    H, He, Hx = 700, 390, 410                                     # rows longer than one pass of the CTA
    oe = np.sort(rng.permutation(H)[:He]).astype(np.int32)
    ox = np.sort(rng.permutation(H)[:Hx]).astype(np.int32)
    ce = (rng.uniform(size=(10, He)) < 0.2).astype(np.uint8)
    cx = (rng.uniform(size=(7, Hx)) < 0.2).astype(np.uint8)
    ok_e = (rng.uniform(size=10) < 0.7).astype(np.uint8)
    ok_x = (rng.uniform(size=7) < 0.7).astype(np.uint8)
    ref = O.merge_half_sets(ce, oe, ok_e, cx, ox, ok_x, H)
    got = comet.merge_half_sets(_dev(ce), _dev(oe), _dev(ok_e), _dev(cx), _dev(ox), _dev(ok_x), H)
    for k in ("valid", "cls", "n_cls"):
        assert np.array_equal(got[k].cpu().numpy(), ref[k]), k
    assert ref["valid"].any() and not ref["valid"].all()


def _compare_half_tracks(got, ref, H):
    for key in ("ent", "ext"):
        g, r = got[key], ref[key]
        assert g["n_fired"] == r["fired_wire"].size, key
        assert np.array_equal(g["orig"].cpu().numpy(), r["orig"]), key
        assert _same_f64(g["final_seed"].cpu().numpy(), r["final_seed"]), key
        assert _same_f64(g["final_rss"].cpu().numpy(), r["final_rss"]), key
        assert np.array_equal(g["cls"].cpu().numpy(), r["cls"]), key
        assert np.array_equal(g["ok"].cpu().numpy(), r["ok"]), key
    for k in ("valid", "cls", "n_cls"):
        assert np.array_equal(got[k].cpu().numpy(), ref[k]), k


@pytest.mark.parametrize("cfg,overlap,k_final", [(0, 3.0, 3), (1, 3.0, 4), (1, 0.0, 2)])
def test_scan_half_tracks_identical(comet, cfg, overlap, k_final):
    """A first turn as two half tracks: grids around the truth entrance and exit states, two refinements, k_final
    finally selected seeds per side, layer veto and merge -- everything identical to the oracle."""
    ev = make_config(cfg)[0]
    circ = _circle(ev)
    sp = ev.spec
    p_range = tuple(sp["p_range"])
    se = seed_grid(ev, 0, (6, 5, 5, 4), p_range, ct_range=sp.get("ct_range"), ct_hw=sp.get("ct_hw", 0.15))
    sx = _exit_grid(ev, 0, (5, 5, 4, 5), p_range)
    kw = dict(half_width=[1.0, 1.2, 1.2, 1.5], n_grid=[3, 3, 3, 3], n_iter=2, shrink=0.5, k_ref=3, k_final=k_final)
    ref = O.scan_half_tracks(se, sx, ev.charge, ev.bz, ev.step, ev.n_steps, R_HALF, ev.geom.wire_a, ev.geom.wire_b,
                             ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, ev.geom.layer, circ, overlap, 3, **kw)
    got = comet.scan_half_tracks(_dev(se), _dev(sx), ev.charge, ev.bz, ev.step, ev.n_steps, R_HALF,
                                 _dev(ev.geom.wire_a), _dev(ev.geom.wire_b), _dev(ev.fired_wire), _dev(ev.hit_off),
                                 _dev(ev.rho), ev.cutoff, _dev(ev.geom.layer), _dev(circ), overlap, 3, **kw)
    torch.cuda.synchronize()
    _compare_half_tracks(got, ref, ev.n_hits)
    # physics of the synthetic turn: both halves classify hits of the first turn, the best pair is valid
    assert ref["ent"]["cls"][0].sum() >= 5 and ref["ext"]["cls"][0].sum() >= 5
    turn = np.asarray(ev.hit_turn)
    best = ref["cls"][0, 0].astype(bool)
    if ref["valid"][0, 0]:
        assert np.mean(turn[best] == 0) > 0.8


def test_scan_half_tracks_without_a_circle(comet, cfg0_event):
    """NaN circle: both hit lists are empty, every seed ties at RSS 0, nothing is classified, no pair is valid."""
    ev = cfg0_event
    se = truth_seed(ev, 0).reshape(6, 1).repeat(4, axis=1)
    se[2] += np.arange(4)
    circ = np.full(11, np.nan)
    kw = dict(half_width=[1.0, 1.0, 1.0, 1.0], n_grid=[2, 2, 2, 2], n_iter=1, shrink=0.5, k_ref=2, k_final=2)
    ref = O.scan_half_tracks(se, se, ev.charge, ev.bz, ev.step, ev.n_steps, R_HALF, ev.geom.wire_a, ev.geom.wire_b,
                             ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, ev.geom.layer, circ, 1.0, 3, **kw)
    got = comet.scan_half_tracks(_dev(se), _dev(se), ev.charge, ev.bz, ev.step, ev.n_steps, R_HALF,
                                 _dev(ev.geom.wire_a), _dev(ev.geom.wire_b), _dev(ev.fired_wire), _dev(ev.hit_off),
                                 _dev(ev.rho), ev.cutoff, _dev(ev.geom.layer), _dev(circ), 1.0, 3, **kw)
    torch.cuda.synchronize()
    _compare_half_tracks(got, ref, ev.n_hits)
    assert got["ent"]["n_fired"] == 0 and not got["valid"].any().item() and not got["cls"].any().item()


def test_scan_half_tracks_full_size_as_benchmarked(comet, cfg1_event):
    """configs[1], turn 0, in the configuration bench.py's `seeding.half_tracks` leg times: the full 131072-seed grid
    per side (the partition's grid at the entrance, the same grid moved to the truth exit state), 3 refinements of
    10 references x 5^4 seeds per side, 10 finally selected seeds per side, 10 x 10 merge -- identical to the oracle."""
    ev = cfg1_event
    circ = _circle(ev)
    sp = ev.spec
    se = seed_grid(ev, 0, sp["grid"], tuple(sp["p_range"]), ct_range=sp.get("ct_range"), ct_hw=sp.get("ct_hw", 0.15))
    assert se.shape[1] == 131072
    x_out, t_out = _exit_state(ev, 0)
    pt = ev.partitions[0]
    sx = se.copy()
    sx[0], sx[1] = x_out[0], x_out[1]
    sx[2] += x_out[2] - pt.z
    rot = np.arctan2(t_out[1], t_out[0]) - pt.phi
    px, py = sx[3].copy(), sx[4].copy()
    sx[3], sx[4] = px * np.cos(rot) - py * np.sin(rot), px * np.sin(rot) + py * np.cos(rot)
    kw = dict(half_width=[0.6, 0.5, 0.5, 1.0], n_grid=[5, 5, 5, 5], n_iter=3, shrink=0.5, k_ref=10, k_final=10)
    got = comet.scan_half_tracks(_dev(se), _dev(sx), ev.charge, ev.bz, ev.step, ev.n_steps, R_HALF,
                                 _dev(ev.geom.wire_a), _dev(ev.geom.wire_b), _dev(ev.fired_wire), _dev(ev.hit_off),
                                 _dev(ev.rho), ev.cutoff, _dev(ev.geom.layer), _dev(circ), 3.0, 3, **kw)
    torch.cuda.synchronize()
    ref = O.scan_half_tracks(se, sx, ev.charge, ev.bz, ev.step, ev.n_steps, R_HALF, ev.geom.wire_a, ev.geom.wire_b,
                             ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, ev.geom.layer, circ, 3.0, 3, **kw)
    _compare_half_tracks(got, ref, ev.n_hits)
    assert ref["valid"].sum() >= 50 and ref["n_cls"].max() >= 40


def test_half_track_argument_errors(comet, cfg0_event):
    from paper_1911_09340_b200 import CometError
    ev = cfg0_event
    wa, wb, fw, ho, rho = (_dev(ev.geom.wire_a), _dev(ev.geom.wire_b), _dev(ev.fired_wire), _dev(ev.hit_off), _dev(ev.rho))
    circ, lay = _dev(_circle(ev)), _dev(ev.geom.layer)
    se = _dev(truth_seed(ev, 0).reshape(6, 1))
    good = dict(half_width=[1.0, 1.0, 1.0, 1.0], n_grid=[2, 2, 2, 2], n_iter=1, shrink=0.5, k_ref=2, k_final=2)
    with pytest.raises(CometError):                                  # negative overlap
        comet.half_hit_masks(wa, wb, fw, ho, ev.n_hits, circ, -1.0)
    with pytest.raises(CometError):                                  # negative overlap in the whole call
        comet.scan_half_tracks(se, se, ev.charge, ev.bz, ev.step, ev.n_steps, R_HALF, wa, wb, fw, ho, rho, ev.cutoff,
                               lay, circ, -0.5, 3, **good)
    with pytest.raises(CometError):                                  # an odd number of entries breaks the ghost pairs (R33)
        comet.scan_half_tracks(se, se, ev.charge, ev.bz, ev.step, ev.n_steps, R_HALF, wa, wb, fw, ho, rho[:-1].contiguous(),
                               ev.cutoff, lay, circ, 1.0, 3, **good)
    with pytest.raises(CometError):                                  # grid sizes out of range
        comet.scan_half_tracks(se, se, ev.charge, ev.bz, ev.step, ev.n_steps, R_HALF, wa, wb, fw, ho, rho, ev.cutoff,
                               lay, circ, 1.0, 3, **dict(good, n_grid=[0, 2, 2, 2]))
    with pytest.raises(CometError):                                  # half lists longer than the event
        comet.merge_half_sets(_dev(np.zeros((1, 8), np.uint8)), _dev(np.arange(8, dtype=np.int32)), _dev(np.ones(1, np.uint8)),
                              _dev(np.zeros((1, 2), np.uint8)), _dev(np.arange(2, dtype=np.int32)), _dev(np.ones(1, np.uint8)), 4)


def _turn_seed_sets(ev, shape_e=(5, 5, 5, 4), shape_x=(5, 5, 4, 5)):
    pr = tuple(ev.spec["p_range"])
    se = [seed_grid(ev, p, shape_e, pr, ct_hw=0.15) for p in range(len(ev.partitions))]
    sx = [_exit_grid(ev, p, shape_x, pr) for p in range(len(ev.partitions))]
    off = lambda blocks: np.concatenate([[0], np.cumsum([b.shape[1] for b in blocks])]).astype(np.int64)
    return (np.ascontiguousarray(np.concatenate(se, axis=1)), off(se),
            np.ascontiguousarray(np.concatenate(sx, axis=1)), off(sx))


def _compare_turns_half(got, ref):
    assert got["done"].tolist() == ref["done"].tolist()
    assert got["wires_before"].tolist() == ref["wires_before"].tolist()
    assert np.array_equal(got["turn_pair"].cpu().numpy(), ref["turn_pair"])
    assert np.array_equal(got["turn_n"].cpu().numpy(), ref["turn_n"])
    assert np.array_equal(got["turn_cls"].cpu().numpy(), ref["turn_cls"])
    assert _same_f64(got["turn_seed"].cpu().numpy(), ref["turn_seed"])


@pytest.mark.parametrize("cfg", [1, 4])
def test_event_loop_with_half_tracks_identical(comet, cfg):
    """Fig. 13 with half tracks: three turns, last first, the chosen complete set's hits removed in between; pairs,
    sets, seeds, wire counts and stopping decisions identical to the oracle (configs[4]: 1000 noise wires)."""
    ev = make_config(cfg)[0]
    circ = _circle(ev)
    se, oe, sx, ox = _turn_seed_sets(ev)
    phys = (ev.charge, ev.bz, ev.step, ev.n_steps, R_HALF)
    kw = dict(half_width=[1.0, 1.2, 1.2, 1.5], n_grid=[3, 3, 3, 3], n_iter=2, shrink=0.5, k_ref=3, k_final=3)
    dargs = (_dev(ev.geom.wire_a), _dev(ev.geom.wire_b), _dev(ev.fired_wire), _dev(ev.hit_off), _dev(ev.rho), ev.cutoff,
             _dev(ev.geom.layer), _dev(circ))
    hargs = (ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, ev.geom.layer, circ)
    for extra in (dict(min_wires=10), dict(min_wires=10, max_tracks=2), dict(min_wires=ev.n_fired + 1)):
        ref = O.scan_turns_half(se, oe, sx, ox, *phys, *hargs, 3.0, 3, **kw, **extra)
        got = comet.scan_turns_half(_dev(se), oe, _dev(sx), ox, *phys, *dargs, 3.0, 3, **kw, **extra)
        torch.cuda.synchronize()
        _compare_turns_half(got, ref)
    assert ref["done"].sum() == 0
    # a veto nothing passes: the first turn has no valid pair and the loop stops there
    ref = O.scan_turns_half(se, oe, sx, ox, *phys, *hargs, 3.0, 21, min_wires=10, **kw)
    got = comet.scan_turns_half(_dev(se), oe, _dev(sx), ox, *phys, *dargs, 3.0, 21, min_wires=10, **kw)
    torch.cuda.synchronize()
    _compare_turns_half(got, ref)
    assert not ref["done"].any() and ref["wires_before"][-1] == ev.n_fired
