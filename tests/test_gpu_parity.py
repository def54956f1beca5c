"""CUDA path vs CPU oracle, element by element, through the C ABI (needs one B200).

Bars (BASELINE.json north_star; R23):
  * n_pts, k*, best seed, classified set: identical;
  * track points: the CUDA extrapolator performs the definition's IEEE operations one by one, so
    they are compared for bit equality (and reported), with 1e-12 relative as the hard bar;
  * DCA: |delta| <= 1e-9 * max(|ref|, 1e-3 cm); RSS: 1e-9 relative.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from comet_synth import event_seeds, make_config, truth_seed  # noqa: E402
from oracle import comet_oracle as O  # noqa: E402

DCA_REL, DCA_FLOOR, RSS_REL = 1e-9, 1e-3, 1e-9


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


class DevEvent:
    def __init__(self, ev, seeds):
        self.ev = ev
        self.seeds_h = np.ascontiguousarray(seeds)
        self.seeds = _dev(seeds)
        self.wire_a, self.wire_b = _dev(ev.geom.wire_a), _dev(ev.geom.wire_b)
        self.fired, self.hit_off, self.rho = _dev(ev.fired_wire), _dev(ev.hit_off), _dev(ev.rho)

    def phys(self):
        ev = self.ev
        return (ev.charge, ev.bz, ev.step, ev.n_steps)

    def hits(self):
        return (self.wire_a, self.wire_b, self.fired, self.hit_off, self.rho)


def _oracle_scan(ev, seeds, cutoff=None, r_stop=None, **kw):
    return O.scan(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop if r_stop is None else r_stop,
                  ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.rho,
                  ev.cutoff if cutoff is None else cutoff, **kw)


def _check_dca(got, ref):
    tol = DCA_REL * np.maximum(np.abs(ref), DCA_FLOOR)
    bad = np.abs(got - ref) > tol
    assert not bad.any(), "DCA mismatch: %d of %d, worst %.3e" % (bad.sum(), bad.size, np.abs(got - ref).max())


def _check_rss(got, ref):
    rel = np.abs(got - ref) / np.maximum(np.abs(ref), 1e-300)
    assert rel.max() <= RSS_REL, "RSS mismatch: worst relative %.3e" % rel.max()


# ------------------------------------------------------------------------------------------------
# kernel A
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("r_stop", [50.0, 0.0])
def test_extrapolate_matches_oracle_cfg0(comet, cfg0_event, r_stop):
    ev = cfg0_event
    seeds, _ = event_seeds(ev)
    seeds = np.ascontiguousarray(seeds[:, :1000])           # 31 full chunks + a ragged tail of 8
    d = DevEvent(ev, seeds)
    track, n_pts = comet.seed_extrapolate(d.seeds, ev.charge, ev.bz, ev.step, ev.n_steps, r_stop)
    got = comet.track_export(track, n_pts, seeds.shape[1], ev.n_steps).cpu().numpy()
    ref, ref_n = O.extrapolate(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, r_stop)
    np.testing.assert_array_equal(n_pts.cpu().numpy(), ref_n)
    assert np.array_equal(np.isnan(got), np.isnan(ref))
    m = ~np.isnan(ref)
    np.testing.assert_allclose(got[m], ref[m], rtol=1e-12, atol=1e-12)
    assert np.array_equal(got[m], ref[m]), "track not bit-identical (max |d| %.3e)" % np.abs(got[m] - ref[m]).max()


def test_extrapolate_seed_range_and_positron(comet, cfg1_event):
    ev = cfg1_event
    seeds, _ = event_seeds(ev, shape=(4, 4, 4, 5))          # 3 * 320 seeds
    d = DevEvent(ev, seeds)
    S = seeds.shape[1]
    b, e = 96, 96 + 333
    track, n_pts = comet.seed_extrapolate(d.seeds, +1, 0.7, ev.step, ev.n_steps, 0.0, seed_range=(b, e))
    got = comet.track_export(track, n_pts, e - b, ev.n_steps).cpu().numpy()
    ref, ref_n = O.extrapolate(np.ascontiguousarray(seeds[:, b:e]), +1, 0.7, ev.step, ev.n_steps, 0.0)
    np.testing.assert_array_equal(n_pts.cpu().numpy(), ref_n)
    assert np.array_equal(got, ref)
    assert S == 960


# ------------------------------------------------------------------------------------------------
# kernel B
# ------------------------------------------------------------------------------------------------
MODES = ["pruned", "exhaustive"]


def _set_mode(comet, mode):
    from paper_1911_09340_b200.binding import COARSE_EXHAUSTIVE, COARSE_PRUNED, OPT_COARSE_SEARCH
    comet.set_option(OPT_COARSE_SEARCH, COARSE_PRUNED if mode == "pruned" else COARSE_EXHAUSTIVE)


def _run_b(comet, d, cutoff=None, r_stop=None, mode="pruned", full=True, **kw):
    """Kernel A + kernel B.  full=True asks for D and k* of every pair; full=False is the RSS-only
    call the whole path makes (in pruned mode it also skips provably-far pairs)."""
    ev = d.ev
    r_stop = ev.r_stop if r_stop is None else r_stop
    _set_mode(comet, mode)
    track, n_pts = comet.seed_extrapolate(d.seeds, ev.charge, ev.bz, ev.step, ev.n_steps, r_stop)
    out = comet.dca_rss(track, n_pts, d.seeds, *d.phys(), *d.hits(), ev.cutoff if cutoff is None else cutoff,
                        want_dca=full, want_kstar=full, **kw)
    torch.cuda.synchronize()
    _set_mode(comet, "pruned")
    return {k: v.cpu().numpy() for k, v in out.items()}, n_pts.cpu().numpy()


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("r_stop", [50.0, 0.0])
def test_dca_rss_matches_oracle_cfg0_full(comet, cfg0_event, r_stop, mode):
    """All 8192 seeds x 32 wires of configs[0]: 256 chunks, 1 pass of 32 wires."""
    ev = cfg0_event
    seeds, _ = event_seeds(ev)
    d = DevEvent(ev, seeds)
    got, n_pts = _run_b(comet, d, r_stop=r_stop, mode=mode)
    ref = _oracle_scan(ev, seeds, r_stop=r_stop, want_dca=True, want_kstar=True, want_npts=True)
    np.testing.assert_array_equal(n_pts, ref["n_pts"])
    np.testing.assert_array_equal(got["kstar"], ref["kstar"])
    _check_dca(got["dca"], ref["dca"])
    _check_rss(got["rss"], ref["rss"])
    # stronger than the bar: same operations in the same order
    assert np.array_equal(got["dca"], ref["dca"])
    assert np.array_equal(got["rss"], ref["rss"])
    # the RSS-only call (pruned mode: far pairs take the cutoff without the plane iteration)
    got2, _ = _run_b(comet, d, r_stop=r_stop, mode=mode, full=False)
    assert np.array_equal(got2["rss"], ref["rss"])


@pytest.mark.parametrize("mode", MODES)
def test_dca_rss_cfg1_ragged(comet, cfg1_event, mode):
    """71 fired wires (3 passes of 24), truth seeds first, 2000-odd seeds with a ragged last chunk."""
    ev = cfg1_event
    seeds, _ = event_seeds(ev)
    ts = np.stack([truth_seed(ev, i) for i in range(len(ev.partitions))], axis=1)
    seeds = np.ascontiguousarray(np.concatenate([ts, seeds[:, ::191]], axis=1))
    assert seeds.shape[1] % 32 != 0
    d = DevEvent(ev, seeds)
    got, n_pts = _run_b(comet, d, mode=mode)
    ref = _oracle_scan(ev, seeds, want_dca=True, want_kstar=True, want_npts=True)
    np.testing.assert_array_equal(n_pts, ref["n_pts"])
    np.testing.assert_array_equal(got["kstar"], ref["kstar"])
    _check_dca(got["dca"], ref["dca"])
    _check_rss(got["rss"], ref["rss"])
    assert np.array_equal(got["rss"], ref["rss"])
    got2, _ = _run_b(comet, d, mode=mode, full=False)
    assert np.array_equal(got2["rss"], ref["rss"])


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("n_fired", [1, 7, 33, 97, 300])
def test_dca_rss_wire_counts(comet, cfg1_event, n_fired, mode):
    """Every wires-per-warp instantiation (1..4), partly filled last passes / wire groups, and more
    wires than one e^2 staging pass of the pruned kernel holds (256)."""
    import copy
    ev = copy.copy(cfg1_event)
    ev.fired_wire = cfg1_event.fired_wire[:min(n_fired, cfg1_event.n_fired)].copy()
    if n_fired > cfg1_event.n_fired:        # pad with unfired wires that carry no entries
        extra = np.setdiff1d(np.arange(ev.geom.n_wires, dtype=np.int32), cfg1_event.fired_wire)[:n_fired - cfg1_event.n_fired]
        ev.fired_wire = np.concatenate([cfg1_event.fired_wire, extra]).astype(np.int32)
        ev.hit_off = np.concatenate([cfg1_event.hit_off, np.full(extra.size, cfg1_event.hit_off[-1], dtype=np.int32)])
        ev.rho = cfg1_event.rho
    else:
        ev.hit_off = cfg1_event.hit_off[:n_fired + 1].copy()
        ev.rho = cfg1_event.rho[:ev.hit_off[-1]].copy()
    seeds, _ = event_seeds(ev, shape=(3, 3, 4, 4))
    d = DevEvent(ev, seeds)
    got, _ = _run_b(comet, d, mode=mode)
    ref = _oracle_scan(ev, seeds, want_dca=True, want_kstar=True)
    np.testing.assert_array_equal(got["kstar"], ref["kstar"])
    _check_dca(got["dca"], ref["dca"])
    _check_rss(got["rss"], ref["rss"])
    got2, _ = _run_b(comet, d, mode=mode, full=False)
    assert np.array_equal(got2["rss"], ref["rss"])


# ------------------------------------------------------------------------------------------------
# kernels A + B fused (comet_scan_rss): track on chip, same numbers
# ------------------------------------------------------------------------------------------------
def _run_fused(comet, d, cutoff=None, r_stop=None):
    ev = d.ev
    out = comet.scan_rss(d.seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop if r_stop is None else r_stop,
                         *d.hits(), ev.cutoff if cutoff is None else cutoff)
    torch.cuda.synchronize()
    return out["rss"].cpu().numpy(), out["n_pts"].cpu().numpy()


@pytest.mark.parametrize("r_stop", [50.0, 0.0])
def test_fused_matches_oracle_cfg0_full(comet, cfg0_event, r_stop):
    ev = cfg0_event
    seeds, _ = event_seeds(ev)
    d = DevEvent(ev, seeds)
    rss, n_pts = _run_fused(comet, d, r_stop=r_stop)
    ref = _oracle_scan(ev, seeds, r_stop=r_stop, want_npts=True)
    np.testing.assert_array_equal(n_pts, ref["n_pts"])
    _check_rss(rss, ref["rss"])
    assert np.array_equal(rss, ref["rss"])


def test_fused_cfg1_ragged(comet, cfg1_event):
    ev = cfg1_event
    seeds, _ = event_seeds(ev)
    ts = np.stack([truth_seed(ev, i) for i in range(len(ev.partitions))], axis=1)
    seeds = np.ascontiguousarray(np.concatenate([ts, seeds[:, ::191]], axis=1))
    assert seeds.shape[1] % 32 != 0
    d = DevEvent(ev, seeds)
    rss, n_pts = _run_fused(comet, d)
    ref = _oracle_scan(ev, seeds, want_npts=True)
    np.testing.assert_array_equal(n_pts, ref["n_pts"])
    assert np.array_equal(rss, ref["rss"])
    # a seed range of the same array, no n_pts wanted
    out = comet.scan_rss(d.seeds, *d.phys()[:3], ev.n_steps, ev.r_stop, *d.hits(), ev.cutoff, want_npts=False,
                         seed_range=(64, 64 + 777))
    assert out["n_pts"] is None
    assert np.array_equal(out["rss"].cpu().numpy(), ref["rss"][64:64 + 777])


@pytest.mark.parametrize("n_fired", [1, 7, 33, 65, 97, 300])
def test_fused_wire_counts(comet, cfg1_event, n_fired):
    """Every wires-per-lane instantiation of level 0 (1, 2, 3), several rounds, wires without entries."""
    import copy
    ev = copy.copy(cfg1_event)
    ev.fired_wire = cfg1_event.fired_wire[:min(n_fired, cfg1_event.n_fired)].copy()
    if n_fired > cfg1_event.n_fired:
        extra = np.setdiff1d(np.arange(ev.geom.n_wires, dtype=np.int32), cfg1_event.fired_wire)[:n_fired - cfg1_event.n_fired]
        ev.fired_wire = np.concatenate([cfg1_event.fired_wire, extra]).astype(np.int32)
        ev.hit_off = np.concatenate([cfg1_event.hit_off, np.full(extra.size, cfg1_event.hit_off[-1], dtype=np.int32)])
        ev.rho = cfg1_event.rho
    else:
        ev.hit_off = cfg1_event.hit_off[:n_fired + 1].copy()
        ev.rho = cfg1_event.rho[:ev.hit_off[-1]].copy()
    seeds, _ = event_seeds(ev, shape=(3, 3, 4, 4))
    d = DevEvent(ev, seeds)
    rss, n_pts = _run_fused(comet, d)
    ref = _oracle_scan(ev, seeds, want_npts=True)
    np.testing.assert_array_equal(n_pts, ref["n_pts"])
    assert np.array_equal(rss, ref["rss"])


def test_fused_high_occupancy_cutoffs_and_odd_steps(comet):
    """configs[4] (~970 fired wires: 11 level-0 rounds) at three cutoffs; then a step count that is
    not a multiple of the tile or the checkpoint interval, without the target-region stop."""
    ev = make_config(4)[0]
    seeds, _ = event_seeds(ev, shape=(4, 4, 4, 4))
    d = DevEvent(ev, seeds)
    for lam in ev.spec["cutoffs"]:
        rss, _ = _run_fused(comet, d, cutoff=lam)
        ref = _oracle_scan(ev, seeds, cutoff=lam)
        assert np.array_equal(rss, ref["rss"]), lam
    import copy
    ev2 = copy.copy(ev)
    ev2.n_steps = 333
    d2 = DevEvent(ev2, seeds)
    rss, n_pts = _run_fused(comet, d2, r_stop=0.0)
    ref = _oracle_scan(ev2, seeds, r_stop=0.0, want_npts=True)
    np.testing.assert_array_equal(n_pts, ref["n_pts"])
    assert np.array_equal(rss, ref["rss"])


@pytest.mark.parametrize("lanes", [1, 3, 8])
def test_fused_internal_stream_lanes(comet, cfg1_event, lanes):
    """comet_scan_rss cuts a slab into sub-slabs on internal streams (COMET_OPT_LANES): same numbers."""
    from paper_1911_09340_b200.binding import OPT_LANES
    ev = cfg1_event
    seeds, _ = event_seeds(ev)
    seeds = np.ascontiguousarray(seeds[:, :3 * 4 * 148 * 32 + 77])      # several sub-slabs and a ragged tail
    d = DevEvent(ev, seeds)
    old = comet.get_option(OPT_LANES)
    try:
        comet.set_option(OPT_LANES, lanes)
        rss, n_pts = _run_fused(comet, d)
        rss2, _ = _run_fused(comet, d)                                  # back to back on the same workspace
    finally:
        comet.set_option(OPT_LANES, old)
    sample = np.arange(0, seeds.shape[1], 37)
    ref = _oracle_scan(ev, np.ascontiguousarray(seeds[:, sample]), want_npts=True)
    np.testing.assert_array_equal(n_pts[sample], ref["n_pts"])
    assert np.array_equal(rss[sample], ref["rss"])
    assert np.array_equal(rss, rss2)
    comet.set_option(OPT_LANES, 1)
    try:
        rss1, _ = _run_fused(comet, d)
    finally:
        comet.set_option(OPT_LANES, old)
    assert np.array_equal(rss, rss1)


def test_fused_unrelated_seeds_in_a_chunk(comet, cfg1_event):
    """The sub-block test bounds a chunk's seeds by a representative one: shuffled seeds (a chunk then
    mixes partitions and far-apart grid points) only lose pruning, never correctness."""
    ev = cfg1_event
    seeds, _ = event_seeds(ev)
    rng = np.random.default_rng(5)
    pick = rng.permutation(seeds.shape[1])[:2048 + 13]
    seeds = np.ascontiguousarray(seeds[:, pick])
    d = DevEvent(ev, seeds)
    rss, n_pts = _run_fused(comet, d)
    ref = _oracle_scan(ev, seeds, want_npts=True)
    np.testing.assert_array_equal(n_pts, ref["n_pts"])
    assert np.array_equal(rss, ref["rss"])


def test_fused_no_wires(comet, cfg0_event):
    ev = cfg0_event
    seeds, _ = event_seeds(ev, shape=(2, 2, 2, 5))
    d = DevEvent(ev, seeds)
    out = comet.scan_rss(d.seeds, *d.phys(), ev.r_stop, d.wire_a, d.wire_b,
                         torch.zeros(0, dtype=torch.int32, device="cuda"),
                         torch.zeros(1, dtype=torch.int32, device="cuda"),
                         torch.zeros(0, dtype=torch.float64, device="cuda"), ev.cutoff)
    torch.cuda.synchronize()
    assert torch.all(out["rss"] == 0.0)
    _, ref_n = O.extrapolate(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop)
    np.testing.assert_array_equal(out["n_pts"].cpu().numpy(), ref_n)


def test_dca_rss_no_wires_and_no_seeds(comet, cfg0_event):
    ev = cfg0_event
    seeds, _ = event_seeds(ev, shape=(2, 2, 2, 5))
    d = DevEvent(ev, seeds)
    track, n_pts = comet.seed_extrapolate(d.seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop)
    empty_i = torch.zeros(0, dtype=torch.int32, device="cuda")
    out = comet.dca_rss(track, n_pts, d.seeds, *d.phys(), d.wire_a, d.wire_b, empty_i,
                        torch.zeros(1, dtype=torch.int32, device="cuda"),
                        torch.zeros(0, dtype=torch.float64, device="cuda"), ev.cutoff)
    assert torch.all(out["rss"] == 0.0)
    # zero seeds: nothing to do, no error
    z = torch.zeros((6, 0), dtype=torch.float64, device="cuda")
    t0, n0 = comet.seed_extrapolate(z, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop)
    assert n0.numel() == 0


def test_high_occupancy_cutoff_sweep(comet):
    """configs[4]: ~1000 noise hits; D is cutoff-independent, RSS and classification are not."""
    ev = make_config(4)[0]
    seeds, part_off = event_seeds(ev, shape=(4, 4, 4, 4))
    d = DevEvent(ev, seeds)
    ref_d = None
    for lam in ev.spec["cutoffs"]:
        got, _ = _run_b(comet, d, cutoff=lam)
        ref = _oracle_scan(ev, seeds, cutoff=lam, want_dca=True, want_kstar=True)
        np.testing.assert_array_equal(got["kstar"], ref["kstar"])
        _check_dca(got["dca"], ref["dca"])
        _check_rss(got["rss"], ref["rss"])
        for mode in MODES:
            got2, _ = _run_b(comet, d, cutoff=lam, mode=mode, full=False)
            assert np.array_equal(got2["rss"], ref["rss"]), mode
        if ref_d is not None:
            assert np.array_equal(got["dca"], ref_d)
        ref_d = got["dca"]
        sel = comet.select_and_classify(d.seeds, *d.phys(), ev.r_stop, *d.hits(), lam,
                                        torch.from_numpy(got["rss"]).cuda(), part_off)
        rs = O.select_classify(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a,
                               ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.rho, lam, ref["rss"], part_off)
        np.testing.assert_array_equal(sel["best_seed"].cpu().numpy(), rs["best_seed"])
        np.testing.assert_array_equal(sel["cls"].cpu().numpy(), rs["cls"])


# ------------------------------------------------------------------------------------------------
# step C and the whole path
# ------------------------------------------------------------------------------------------------
def _check_select(sel, ref, ev, cutoff):
    np.testing.assert_array_equal(sel["best_seed"].cpu().numpy(), ref["best_seed"])
    _check_rss(sel["best_rss"].cpu().numpy(), ref["best_rss"])
    bd, rd = sel["best_dca"].cpu().numpy(), ref["best_dca"]
    _check_dca(bd, rd)
    cls, rcls = sel["cls"].cpu().numpy(), ref["cls"]
    if not np.array_equal(cls, rcls):
        # only entries whose residual lies within 1e-9 cm of the cutoff may differ
        for p, j in zip(*np.nonzero(cls != rcls)):
            i = np.searchsorted(ev.hit_off, j, side="right") - 1
            assert abs(abs(rd[p, i] - ev.rho[j]) - cutoff) < 1e-9


def test_whole_path_cfg0(comet, cfg0_event):
    ev = cfg0_event
    seeds, part_off = event_seeds(ev)
    d = DevEvent(ev, seeds)
    out = comet.scan_event(d.seeds, part_off, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff)
    ref = _oracle_scan(ev, seeds)
    _check_rss(out["rss"].cpu().numpy(), ref["rss"])
    rs = O.select_classify(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a,
                           ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, ref["rss"], part_off)
    _check_select(out, rs, ev, ev.cutoff)
    # slabbed processing (track buffer smaller than the seed set) gives the same numbers
    out2 = comet.scan_event(d.seeds, part_off, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff, slab_seeds=1000)
    assert torch.equal(out2["rss"], out["rss"]) and torch.equal(out2["cls"], out["cls"])
    assert torch.equal(out2["best_seed"], out["best_seed"])
    # the default is the fused path (track on chip); the track-buffer path gives the same numbers
    out3 = comet.scan_event(d.seeds, part_off, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff, fused=False)
    assert torch.equal(out3["rss"], out["rss"]) and torch.equal(out3["n_pts"], out["n_pts"])


def test_select_ties_and_empty_partition(comet, cfg0_event):
    ev = cfg0_event
    seeds, _ = event_seeds(ev, shape=(3, 2, 2, 2))
    S = seeds.shape[1]
    dup = np.ascontiguousarray(np.concatenate([seeds, seeds], axis=1))
    d = DevEvent(ev, dup)
    part_off = np.array([0, S, S, 2 * S], dtype=np.int64)      # middle partition is empty
    out = comet.scan_event(d.seeds, part_off, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff)
    bs = out["best_seed"].cpu().numpy()
    assert bs[1] == -1 and bs[2] == bs[0] + S
    assert torch.all(out["cls"][1] == 0) and torch.isnan(out["best_rss"][1])
    one = comet.select_and_classify(d.seeds, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff, out["rss"],
                                    np.array([0, 2 * S], dtype=np.int64))
    assert int(one["best_seed"][0]) == int(bs[0])              # tie between the copies -> lower index


def test_select_with_nan_rss_follows_the_serial_rule(comet, cfg0_event):
    """NaN in RSS (a degenerate seed with |p| = 0): the serial argmin "rss[s] < rss[b]" keeps a NaN at the first
    position of a partition and never takes one anywhere else.  Positions chosen to hit the first element of a
    CTA's range, of a thread's stride and interior ones, in partitions long enough for all 64 CTAs of stage 1."""
    ev = cfg0_event
    seeds, _ = event_seeds(ev, shape=(16, 8, 8, 8))
    S = seeds.shape[1]
    d = DevEvent(ev, seeds)
    rng = np.random.default_rng(11)
    rss = rng.uniform(0.1, 1.0, S)
    part_off = np.array([0, 3000, 3001, S], dtype=np.int64)
    per = (S - 3001 + 63) // 64
    for s in (1, 2, 255, 256, 257, 2999, 3001 + per, 3001 + per + 256, 3001 + 5 * per + 3, S - 1):
        rss[s] = np.nan
    rss[300] = 0.01                                         # the winner of partition 0 sits behind NaNs of its thread
    rss[3001 + per + 512] = 0.02                            # and so does the winner of partition 2 (same thread as two NaNs)
    cases = [rss.copy()]
    first_nan = rss.copy()
    first_nan[0] = np.nan                                   # NaN at a partition's first position wins it
    first_nan[3000] = np.nan                                # one-seed partition holding a NaN
    cases.append(first_nan)
    for r in cases:
        out = comet.select_and_classify(d.seeds, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff,
                                        torch.from_numpy(r).cuda(), part_off)
        rs = O.select_classify(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a,
                               ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, r, part_off)
        np.testing.assert_array_equal(out["best_seed"].cpu().numpy(), rs["best_seed"])
        np.testing.assert_array_equal(out["best_rss"].cpu().numpy(), rs["best_rss"])
        np.testing.assert_array_equal(out["cls"].cpu().numpy(), rs["cls"])
        np.testing.assert_array_equal(out["best_dca"].cpu().numpy(), rs["best_dca"])


def test_whole_path_host_buffers(comet, cfg0_event):
    ev = cfg0_event
    seeds, part_off = event_seeds(ev)
    out = comet.scan_event_host(torch.from_numpy(seeds).pin_memory(), part_off, ev.charge, ev.bz, ev.step,
                                ev.n_steps, ev.r_stop, ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire,
                                ev.hit_off, ev.rho, ev.cutoff, want_rss=True,
                                track_budget_bytes=40 << 20)       # forces several slabs
    ref = _oracle_scan(ev, seeds)
    _check_rss(out["rss"].numpy(), ref["rss"])
    rs = O.select_classify(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a,
                           ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, ref["rss"], part_off)
    np.testing.assert_array_equal(out["best_seed"].numpy(), rs["best_seed"])
    np.testing.assert_array_equal(out["cls"].numpy(), rs["cls"])


def test_argument_errors(comet, cfg0_event):
    from paper_1911_09340_b200 import CometError
    ev = cfg0_event
    seeds, _ = event_seeds(ev, shape=(2, 2, 2, 4))
    d = DevEvent(ev, seeds)
    with pytest.raises(CometError):
        comet.seed_extrapolate(d.seeds, ev.charge, ev.bz, -1.0, ev.n_steps, ev.r_stop)      # step <= 0
    with pytest.raises(CometError):
        comet.seed_extrapolate(d.seeds, 0, ev.bz, ev.step, ev.n_steps, ev.r_stop)           # charge 0
    with pytest.raises(CometError):
        comet.seed_extrapolate(d.seeds, ev.charge, ev.bz, ev.step, 5000, ev.r_stop)         # > COMET_MAX_STEPS
    with pytest.raises(CometError):
        comet.seed_extrapolate(d.seeds.cpu(), ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop)


# ------------------------------------------------------------------------------------------------
# full-size configurations (the launch configuration bench.py times) and the remaining configs
# ------------------------------------------------------------------------------------------------
def _oracle_select(ev, seeds, rss, part_off, cutoff=None):
    return O.select_classify(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a,
                             ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.rho,
                             ev.cutoff if cutoff is None else cutoff, rss, part_off)


def test_full_cfg1_as_benchmarked(comet, cfg1_event):
    """configs[1] at full size (3 x 131072 seeds x 71 wires), default (pruned) mode, device-resident
    inputs exactly as bench.py runs it: every RSS, the best seeds and the classified set."""
    ev = cfg1_event
    seeds, part_off = event_seeds(ev)
    assert seeds.shape[1] == 3 * 131072
    d = DevEvent(ev, seeds)
    out = comet.scan_event(d.seeds, part_off, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff)
    torch.cuda.synchronize()
    ref = _oracle_scan(ev, seeds, want_npts=True)
    np.testing.assert_array_equal(out["n_pts"].cpu().numpy(), ref["n_pts"])
    got = out["rss"].cpu().numpy()
    _check_rss(got, ref["rss"])
    assert np.array_equal(got, ref["rss"])
    _check_select(out, _oracle_select(ev, seeds, ref["rss"], part_off), ev, ev.cutoff)


def test_pair_workspace_slabs(comet, cfg0_event):
    """A pair workspace smaller than the problem: comet_dca_rss walks seed slabs, same numbers."""
    from paper_1911_09340_b200 import Comet
    ev = cfg0_event
    seeds, part_off = event_seeds(ev)
    d = DevEvent(ev, seeds)
    c2 = Comet(0)
    try:
        c2.reserve(5 * 32 * ev.n_fired)                    # 5 chunks per slab -> 52 slabs, ragged last one
        out = c2.scan_event(d.seeds, part_off, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff)
        ref = comet.scan_event(d.seeds, part_off, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff)
        assert torch.equal(out["rss"], ref["rss"]) and torch.equal(out["cls"], ref["cls"])
        assert torch.equal(out["best_seed"], ref["best_seed"])
        track, n_pts = c2.seed_extrapolate(d.seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop)
        full = c2.dca_rss(track, n_pts, d.seeds, *d.phys(), *d.hits(), ev.cutoff, want_dca=True, want_kstar=True)
        oref = _oracle_scan(ev, seeds, want_dca=True, want_kstar=True)
        np.testing.assert_array_equal(full["kstar"].cpu().numpy(), oref["kstar"])
        assert np.array_equal(full["dca"].cpu().numpy(), oref["dca"])
    finally:
        c2.close()


def test_cfg2_batch_of_events_on_streams():
    """configs[2]: independent events (1-4 turns, |p| in [60,105]) in flight on several streams, one
    context per stream; reduced seed grid so that the oracle finishes in seconds."""
    from paper_1911_09340_b200 import Comet
    events = make_config(2, n_events=6)
    n_str = 3
    ctxs = [Comet(0) for _ in range(n_str)]
    streams = [torch.cuda.Stream() for _ in range(n_str)]
    try:
        outs, inputs = [], []
        for k, ev in enumerate(events):
            seeds, part_off = event_seeds(ev, shape=(6, 4, 4, 6))
            d = DevEvent(ev, seeds)
            st = streams[k % n_str]
            st.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(st):
                outs.append(ctxs[k % n_str].scan_event(d.seeds, part_off, *d.phys(), ev.r_stop, *d.hits(),
                                                       ev.cutoff, stream=st))
            inputs.append((ev, seeds, part_off, d))
        torch.cuda.synchronize()
        assert len({len(ev.partitions) for ev in events}) > 1          # a mix of turn counts
        for (ev, seeds, part_off, _), out in zip(inputs, outs):
            ref = _oracle_scan(ev, seeds)
            assert np.array_equal(out["rss"].cpu().numpy(), ref["rss"])
            _check_select(out, _oracle_select(ev, seeds, ref["rss"], part_off), ev, ev.cutoff)
    finally:
        for c in ctxs:
            c.close()


def test_cfg3_large_scan_in_slabs(comet):
    """configs[3] (4 turns, 1600 steps of 0.2 cm): the track buffer of the full grid does not fit in
    HBM, so seeds go through a bounded track workspace.  Reduced grid, element by element."""
    ev = make_config(3)[0]
    assert len(ev.partitions) == 4 and ev.n_steps == 1600
    seeds, part_off = event_seeds(ev, shape=(8, 4, 8, 16))             # 4 x 4096 seeds
    out = comet.scan_event_host(torch.from_numpy(seeds).pin_memory(), part_off, ev.charge, ev.bz, ev.step,
                                ev.n_steps, ev.r_stop, ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire,
                                ev.hit_off, ev.rho, ev.cutoff, want_rss=True,
                                track_budget_bytes=300 << 20)          # ~3800 seeds per slab
    ref = _oracle_scan(ev, seeds)
    assert np.array_equal(out["rss"].numpy(), ref["rss"])
    rs = _oracle_select(ev, seeds, ref["rss"], part_off)
    np.testing.assert_array_equal(out["best_seed"].numpy(), rs["best_seed"])
    np.testing.assert_array_equal(out["cls"].numpy(), rs["cls"])


def _sampled_full_size_check(comet, ev, seeds, part_off, n_sample, cutoff=None, budget=8 << 30):
    """Whole path at full size through the host-buffer entry point (run length found on the device); a sample of
    RSS, the contenders for the best seed and the winners' D / classified sets against the oracle
    (parity_checks.check_event_against_oracle)."""
    cutoff = ev.cutoff if cutoff is None else cutoff
    S = seeds.shape[1]
    out = comet.scan_event_host(torch.from_numpy(seeds).pin_memory(), part_off, ev.charge, ev.bz, ev.step,
                                ev.n_steps, ev.r_stop, ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire,
                                ev.hit_off, ev.rho, cutoff, want_rss=True, track_budget_bytes=budget)
    from parity_checks import check_event_against_oracle
    got = {k: out[k].numpy() for k in ("best_seed", "best_rss", "best_dca", "cls")}
    check_event_against_oracle(ev, seeds, tuple(ev.spec["grid"]), part_off, out["rss"].numpy(), got, n_sample,
                               np.random.default_rng(S % 1000 + int(budget > 0)), cutoff=cutoff)
    return out


@pytest.mark.parametrize("budget", [0, 8 << 30], ids=["fused", "track8GiB"])
def test_full_cfg3_sampled(comet, budget):
    """configs[3] at full size: 4 x 1048576 seeds, 1600 steps; fused (track on chip, checkpoint
    slabs) and through 8 GiB track slabs."""
    ev = make_config(3)[0]
    seeds, part_off = event_seeds(ev)
    assert seeds.shape[1] == 4 * 1048576
    _sampled_full_size_check(comet, ev, seeds, part_off, n_sample=4096, budget=budget)


@pytest.mark.parametrize("budget", [0, 8 << 30], ids=["fused", "track8GiB"])
def test_full_cfg4_sampled(comet, budget):
    """configs[4] at full size: 3 x 131072 seeds against ~970 fired wires, three cutoffs."""
    ev = make_config(4)[0]
    seeds, part_off = event_seeds(ev)
    assert seeds.shape[1] == 3 * 131072 and ev.n_fired > 900
    for lam in ev.spec["cutoffs"]:
        _sampled_full_size_check(comet, ev, seeds, part_off, n_sample=1024, cutoff=lam, budget=budget)


def test_seed_sharded_scan_two_ranks_emulated(comet, cfg1_event):
    """The seed-sharded N > 1 flow on one GPU: each 'rank' scans only its chunk-aligned seed ranges
    (one after the other here, no kernel waits on another), the local winners are merged with the
    rule of sharding.merge_best, every rank classifies the winners itself.  Same result as one rank."""
    from paper_1911_09340_b200.sharding import local_best, shard_partitions
    ev = cfg1_event
    seeds, part_off = event_seeds(ev, shape=(5, 4, 4, 7))             # 560 seeds per partition: ragged chunks
    d = DevEvent(ev, seeds)
    one = comet.scan_event(d.seeds, part_off, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff)
    world, P = 2, len(part_off) - 1
    loc = []
    for rank in range(world):
        ranges = shard_partitions(part_off, rank, world)
        rss = torch.full((seeds.shape[1],), float("nan"), dtype=torch.float64, device="cuda")
        for b, e in ranges:
            if e > b:
                track, n_pts = comet.seed_extrapolate(d.seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop,
                                                      seed_range=(b, e))
                comet.dca_rss(track, n_pts, d.seeds, *d.phys(), *d.hits(), ev.cutoff, rss=rss[b:e],
                              seed_range=(b, e))
        loc.append(local_best(rss, ranges))
    gv = torch.minimum(loc[0][0], loc[1][0])
    big = torch.iinfo(torch.int64).max
    gi = torch.minimum(torch.where(loc[0][0] == gv, loc[0][1], big), torch.where(loc[1][0] == gv, loc[1][1], big))
    assert torch.equal(gi, one["best_seed"]) and torch.equal(gv, one["best_rss"])
    winners = d.seeds[:, gi].contiguous()                              # [6][P]
    sel = comet.select_and_classify(winners, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff, gv.contiguous(),
                                    np.arange(P + 1, dtype=np.int64))
    assert torch.equal(sel["cls"], one["cls"]) and torch.equal(sel["best_dca"], one["best_dca"])


# ------------------------------------------------------------------------------------------------
# iterative seed refinement (comet_select_references, comet_refine_seeds, comet_classify_seeds,
# comet_scan_stage): bit-identical references, seeds, RSS and classification
# ------------------------------------------------------------------------------------------------
def _ev_args(ev):
    return (ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire,
            ev.hit_off, ev.rho, ev.cutoff)


@pytest.mark.parametrize("k_ref", [1, 5, 64])
def test_select_references_matches_oracle(comet, k_ref):
    rng = np.random.default_rng(11)
    n = 5000
    s = np.zeros((6, n))
    s[2:] = rng.integers(0, 9, size=(4, n)) * np.array([[0.5], [1.0], [1.0], [2.0]])     # exact |d| = 2 hw ties
    rss = rng.integers(0, 300, size=n).astype(float) * 0.01                               # many RSS ties
    rss[rng.integers(0, n, 20)] = np.nan
    po = np.array([0, 1, 1, 1900, 5000])                                                  # a 1-seed and an empty partition
    hw = np.array([0.5, 1.0, 1.5, 2.0])
    ref = comet.select_references(_dev(s), _dev(rss), po, hw, k_ref)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(ref.cpu().numpy(), O.select_references(s, rss, po, hw, k_ref))


@pytest.mark.parametrize("n", [20000, 150000, 300000])
def test_select_references_large_partitions(comet, n):
    """One CTA (<= 16384 seeds), a cluster with RSS staged in shared memory, a cluster reading global memory."""
    rng = np.random.default_rng(n)
    s = np.zeros((6, n + 700))
    s[2:] = rng.integers(0, 12, size=(4, n + 700)) * np.array([[0.5], [1.0], [1.0], [2.0]])
    rss = rng.integers(0, 2000, size=n + 700).astype(float) * 0.001
    rss[rng.integers(0, n, 50)] = np.nan
    po = np.array([0, n, n + 700])
    hw = np.array([0.5, 1.0, 1.0, 2.0])
    ref = comet.select_references(_dev(s), _dev(rss), po, hw, 12)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(ref.cpu().numpy(), O.select_references(s, rss, po, hw, 12))


@pytest.mark.parametrize("case", ["all_equal", "few_small", "sample_misses", "one_box", "nan_heavy"])
def test_select_references_shortlist_fallbacks(comet, case):
    """Large partitions take their references from the seeds below a sampled RSS threshold (k_select_refs_short) and fall
    back to the full rule when that list cannot decide: every seed equal, fewer distinct small values than references,
    a sample that misses the small values (more seeds below the threshold than the list holds), every seed in one box
    (one reference only), mostly NaN."""
    rng = np.random.default_rng(7)
    n = 70000
    s = np.zeros((6, n))
    s[2:] = rng.normal(size=(4, n)) * np.array([[3.0], [5.0], [5.0], [8.0]])
    rss = rng.uniform(0.5, 2.0, n)
    if case == "all_equal":
        rss[:] = 0.71
    elif case == "few_small":
        rss[:] = 0.71
        rss[rng.integers(0, n, 5)] = 0.1
    elif case == "sample_misses":
        rss[:] = rng.uniform(0.1, 0.2, n)
        rss[::n // 2048] = 5.0                               # the sampled positions hold the largest values
    elif case == "one_box":
        s[2:] = 0.0
    elif case == "nan_heavy":
        rss[rng.random(n) < 0.97] = np.nan
    po = np.array([0, n])
    hw = np.array([0.5, 1.0, 1.0, 2.0])
    ref = comet.select_references(_dev(s), _dev(rss), po, hw, 12)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(ref.cpu().numpy(), O.select_references(s, rss, po, hw, 12))


def test_select_references_cfg1_rss(comet, cfg1_event):
    ev = cfg1_event
    seeds, po = event_seeds(ev)
    d = DevEvent(ev, seeds)
    rss, _ = _run_fused(comet, d)
    hw = np.array([0.6, 0.5, 0.5, 1.5])
    ref = comet.select_references(d.seeds, _dev(rss), po, hw, 10)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(ref.cpu().numpy(), O.select_references(seeds, rss, po, hw, 10))


def test_refine_seeds_matches_oracle(comet):
    rng = np.random.default_rng(12)
    seeds = rng.normal(size=(6, 300)) * 20
    ref = np.array([[7, 11, -1, 5], [250, -1, -1, -1], [3, 4, 5, 6]], dtype=np.int64)
    hw = np.array([1.5, 0.25, 2.0, 0.0])
    for ng in ([4, 3, 2, 1], [1, 1, 1, 1], [5, 7, 3, 9]):
        new, po = comet.refine_seeds(_dev(seeds), _dev(ref), hw, ng)
        torch.cuda.synchronize()
        exp, epo = O.refine_seeds(seeds, ref, hw, ng)
        assert np.array_equal(new.cpu().numpy(), exp)
        np.testing.assert_array_equal(po, epo)


def test_classify_seeds_matches_oracle(comet, cfg0_event):
    ev = cfg0_event
    seeds, _ = event_seeds(ev)
    d = DevEvent(ev, seeds)
    idx = np.array([5, -1, 8191, 670, 670], dtype=np.int64)
    out = comet.classify_seeds(d.seeds, _dev(idx), *d.phys(), ev.r_stop, *d.hits(), ev.cutoff)
    torch.cuda.synchronize()
    ref = O.classify_seeds(seeds, idx, *_ev_args(ev))
    np.testing.assert_array_equal(out["cls"].cpu().numpy(), ref["cls"])
    np.testing.assert_array_equal(out["dca"].cpu().numpy(), ref["dca"])               # bit-identical, NaN rows included


@pytest.mark.parametrize("n_iter", [0, 3])
def test_scan_stage_matches_oracle_cfg0(comet, cfg0_event, n_iter):
    ev = cfg0_event
    seeds, po = event_seeds(ev)
    d = DevEvent(ev, seeds)
    kw = dict(half_width=[1.2, 1.0, 1.0, 4.0], n_grid=[3, 5, 5, 5], n_iter=n_iter, shrink=0.5, k_ref=4, k_final=10)
    out = comet.scan_stage(d.seeds, po, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff, **kw)
    torch.cuda.synchronize()
    ref = O.scan_stage(seeds, po, *_ev_args(ev), **kw)
    np.testing.assert_array_equal(out["final_seed"].cpu().numpy(), ref["final_seed"])
    np.testing.assert_array_equal(out["final_rss"].cpu().numpy(), ref["final_rss"])
    np.testing.assert_array_equal(out["cls"].cpu().numpy(), ref["cls"])
    _check_dca(np.nan_to_num(out["final_dca"].cpu().numpy()), np.nan_to_num(ref["final_dca"]))


def test_scan_stage_cfg1_three_partitions(comet, cfg1_event):
    """Three turn partitions at once, a coarse first set (every 8th seed of the configs[1] grid), two refinements."""
    ev = cfg1_event
    seeds, po = event_seeds(ev)
    n_per = seeds.shape[1] // 3
    seeds = np.ascontiguousarray(np.concatenate([seeds[:, p * n_per:(p + 1) * n_per:8] for p in range(3)], axis=1))
    po = np.arange(4, dtype=np.int64) * (n_per // 8)
    d = DevEvent(ev, seeds)
    kw = dict(half_width=[0.6, 0.5, 0.5, 1.0], n_grid=[3, 4, 4, 3], n_iter=2, shrink=0.5, k_ref=6, k_final=10)
    out = comet.scan_stage(d.seeds, po, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff, **kw)
    torch.cuda.synchronize()
    ref = O.scan_stage(seeds, po, *_ev_args(ev), **kw)
    np.testing.assert_array_equal(out["final_seed"].cpu().numpy(), ref["final_seed"])
    np.testing.assert_array_equal(out["final_rss"].cpu().numpy(), ref["final_rss"])
    np.testing.assert_array_equal(out["cls"].cpu().numpy(), ref["cls"])


def test_refinement_argument_errors(comet, cfg0_event):
    from paper_1911_09340_b200 import CometError
    ev = cfg0_event
    seeds, po = event_seeds(ev, shape=(2, 2, 2, 2))
    d = DevEvent(ev, seeds)
    rss = torch.zeros(seeds.shape[1], dtype=torch.float64, device="cuda")
    with pytest.raises(CometError):
        comet.select_references(d.seeds, rss, po, [1, 1, 1, 1], 65)
    with pytest.raises(CometError):
        comet.select_references(d.seeds, rss, po, [1, -1, 1, 1], 2)
    with pytest.raises(CometError):
        comet.refine_seeds(d.seeds, torch.zeros((1, 2), dtype=torch.int64, device="cuda"), [1, 1, 1, 1], [2, 0, 2, 2])
    with pytest.raises(CometError):          # an empty partition
        comet.scan_stage(d.seeds, [0, 0, seeds.shape[1]], *d.phys(), ev.r_stop, *d.hits(), ev.cutoff,
                         half_width=[1, 1, 1, 1], n_grid=[2, 2, 2, 2], n_iter=1, shrink=0.5, k_ref=2, k_final=2)


# ------------------------------------------------------------------------------------------------
# inhomogeneous field map + adaptive step (comet_set_field): bit-identical to the oracle's field path
# ------------------------------------------------------------------------------------------------
@pytest.fixture()
def field_comet():
    from paper_1911_09340_b200 import Comet
    c = Comet(0)
    yield c
    c.close()


def _set_map(c, F, tol):
    B, o, d = F
    t = _dev(B)
    c.set_field(t, o, d, tol)
    return t


@pytest.mark.parametrize("tol", [1e-5, 1e-7, 1e-9])
def test_field_scan_matches_oracle_cfg0(field_comet, cfg0_event, tol):
    from comet_synth import solenoid_map
    c, ev = field_comet, cfg0_event
    seeds, po = event_seeds(ev)
    seeds = np.ascontiguousarray(seeds[:, :2048 + 19])
    seeds[2, 1000:] += 40.0                       # part of the seeds start near the end plate, where the steps halve
    d = DevEvent(ev, seeds)
    F = solenoid_map()
    _set_map(c, F, tol)
    out = c.scan_rss(d.seeds, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff)
    torch.cuda.synchronize()
    ref = O.scan_field(seeds, ev.charge, F, ev.step, ev.n_steps, ev.r_stop, tol, ev.geom.wire_a, ev.geom.wire_b,
                       ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, want_npts=True)
    np.testing.assert_array_equal(out["n_pts"].cpu().numpy(), ref["n_pts"])
    assert np.array_equal(out["rss"].cpu().numpy(), ref["rss"])
    tr, npt, hs = O.extrapolate_field(seeds[:, 1500:1600], ev.charge, F, ev.step, ev.n_steps, ev.r_stop, tol)
    if tol < 1e-6:
        assert np.nanmin(hs) < ev.step            # the case does exercise the step control


def test_field_uniform_map_equals_uniform_path(field_comet, cfg0_event):
    from comet_synth import uniform_map
    c, ev = field_comet, cfg0_event
    seeds, po = event_seeds(ev, shape=(4, 4, 4, 4))
    d = DevEvent(ev, seeds)
    a = c.scan_rss(d.seeds, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff)
    rss_u, np_u = a["rss"].clone(), a["n_pts"].clone()
    keep = _set_map(c, uniform_map(ev.bz), 1e-3)
    b = c.scan_rss(d.seeds, ev.charge, 123.0, ev.step, ev.n_steps, ev.r_stop, *d.hits(), ev.cutoff)   # bz ignored
    torch.cuda.synchronize()
    assert torch.equal(np_u, b["n_pts"])
    np.testing.assert_allclose(b["rss"].cpu().numpy(), rss_u.cpu().numpy(), rtol=1e-9)
    # the materialised track is a uniform-field path
    from paper_1911_09340_b200 import CometError
    with pytest.raises(CometError):
        c.seed_extrapolate(d.seeds, *d.phys(), ev.r_stop)
    c.set_field(None)
    c.seed_extrapolate(d.seeds, *d.phys(), ev.r_stop)
    del keep


def test_field_classify_and_stage_match_oracle(field_comet, cfg0_event):
    from comet_synth import solenoid_map
    c, ev = field_comet, cfg0_event
    seeds, po = event_seeds(ev, shape=(6, 4, 4, 4))
    d = DevEvent(ev, seeds)
    F, tol = solenoid_map(), 1e-7
    keep = _set_map(c, F, tol)
    fargs = (ev.charge, F, ev.step, ev.n_steps, ev.r_stop, tol, ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire,
             ev.hit_off, ev.rho, ev.cutoff)
    idx = np.array([0, 17, -1, seeds.shape[1] - 1], dtype=np.int64)
    got = c.classify_seeds(d.seeds, _dev(idx), *d.phys(), ev.r_stop, *d.hits(), ev.cutoff)
    ref = O.classify_seeds_field(seeds, idx, *fargs)
    ref["dca"][2] = np.nan
    np.testing.assert_array_equal(got["dca"].cpu().numpy(), ref["dca"])
    np.testing.assert_array_equal(got["cls"].cpu().numpy(), ref["cls"])
    # whole path A + B + C
    out = c.scan_event(d.seeds, po, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff)
    rs = O.scan_field(seeds, *fargs)["rss"]
    best = int(np.argmin(rs))
    assert np.array_equal(out["rss"].cpu().numpy(), rs)
    assert out["best_seed"].cpu().tolist() == [best]
    np.testing.assert_array_equal(out["cls"].cpu().numpy()[0], O.classify_seeds_field(seeds, [best], *fargs)["cls"][0])
    # a stage with two refinements
    kw = dict(half_width=[1.2, 1.0, 1.0, 4.0], n_grid=[3, 3, 3, 3], n_iter=2, shrink=0.5, k_ref=3, k_final=4)
    so = c.scan_stage(d.seeds, po, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff, **kw)
    torch.cuda.synchronize()
    sr = O.scan_stage(seeds, po, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a, ev.geom.wire_b,
                      ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, field=F, rkn_tol=tol, **kw)
    np.testing.assert_array_equal(so["final_seed"].cpu().numpy(), sr["final_seed"])
    np.testing.assert_array_equal(so["final_rss"].cpu().numpy(), sr["final_rss"])
    np.testing.assert_array_equal(so["cls"].cpu().numpy(), sr["cls"])
    del keep


@pytest.mark.parametrize("spacing", [(3.0, 5.0, 2.5), (4.0, 4.0, 6.0), (2.0, 8.0, 0.5)])
def test_field_map_spacings_division_and_exact_scaling(field_comet, cfg0_event, spacing):
    """The cell coordinate (x - o) / d of R29 is an IEEE division; when all three spacings are powers of two the
    kernels scale by 1 / d instead (the same number, bit for bit).  Both branches, and a map in which only some
    axes have such a spacing (division), against the oracle's division: RSS, n_pts, winner and classification."""
    from comet_synth import solenoid_map
    c, ev = field_comet, cfg0_event
    seeds, po = event_seeds(ev, shape=(5, 4, 4, 4))
    d = DevEvent(ev, seeds)
    F, tol = solenoid_map(spacing=spacing), 1e-7
    keep = _set_map(c, F, tol)
    fargs = (ev.charge, F, ev.step, ev.n_steps, ev.r_stop, tol, ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire,
             ev.hit_off, ev.rho, ev.cutoff)
    out = c.scan_event(d.seeds, po, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff)
    ref = O.scan_field(seeds, *fargs, want_npts=True)
    assert np.array_equal(out["rss"].cpu().numpy(), ref["rss"])
    assert np.array_equal(out["n_pts"].cpu().numpy(), ref["n_pts"])
    best = int(np.argmin(ref["rss"]))
    assert out["best_seed"].cpu().tolist() == [best]
    rc = O.classify_seeds_field(seeds, [best], *fargs)
    np.testing.assert_array_equal(out["cls"].cpu().numpy()[0], rc["cls"][0])
    np.testing.assert_array_equal(out["best_dca"].cpu().numpy()[0], rc["dca"][0])
    del keep


def test_field_scan_cfg1_ragged_three_partitions(field_comet, cfg1_event):
    from comet_synth import solenoid_map
    c, ev = field_comet, cfg1_event
    seeds, _ = event_seeds(ev)
    seeds = np.ascontiguousarray(seeds[:, ::97])
    d = DevEvent(ev, seeds)
    F, tol = solenoid_map(), 1e-8
    keep = _set_map(c, F, tol)
    out = c.scan_rss(d.seeds, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff)
    torch.cuda.synchronize()
    ref = O.scan_field(seeds, ev.charge, F, ev.step, ev.n_steps, ev.r_stop, tol, ev.geom.wire_a, ev.geom.wire_b,
                       ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, want_npts=True)
    np.testing.assert_array_equal(out["n_pts"].cpu().numpy(), ref["n_pts"])
    assert np.array_equal(out["rss"].cpu().numpy(), ref["rss"])
    del keep


def test_scan_path_is_capturable_in_a_cuda_graph(comet, cfg1_event):
    """comet_scan_rss forks into the ctx's internal streams and joins them with events, and nothing on the hot
    path allocates or synchronises: the whole A + B + C sequence can be captured once and replayed."""
    ev = cfg1_event
    seeds, po = event_seeds(ev)
    seeds = np.ascontiguousarray(seeds[:, :4 * 4 * 148 * 32])
    po = [0, seeds.shape[1]]
    d = DevEvent(ev, seeds)
    S = seeds.shape[1]
    rss = torch.empty(S, dtype=torch.float64, device="cuda")
    n_pts = torch.empty(S, dtype=torch.int32, device="cuda")
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        comet.scan_rss(d.seeds, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff, rss=rss, n_pts=n_pts, stream=st)   # grows the workspace
        ref = comet.select_and_classify(d.seeds, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff, rss, po, stream=st)
    st.synchronize()
    rss_ref, best_ref, cls_ref = rss.clone(), ref["best_seed"].clone(), ref["cls"].clone()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=st):
        comet.scan_rss(d.seeds, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff, rss=rss, n_pts=n_pts, stream=st)
        out = comet.select_and_classify(d.seeds, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff, rss, po, stream=st)
    for _ in range(2):
        rss.zero_()
        out["cls"].zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(rss, rss_ref)
        assert torch.equal(out["best_seed"], best_ref) and torch.equal(out["cls"], cls_ref)


# ------------------------------------------------------------------------------------------------
# sequential stages with hit removal (comet_remove_hits, comet_scan_turns)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n_wires_case", [0, 1, 300, 5000])
def test_remove_hits_matches_oracle(comet, n_wires_case):
    rng = np.random.default_rng(21 + n_wires_case)
    W = n_wires_case
    counts = rng.integers(0, 4, size=W) * 2
    hit_off = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    H = int(hit_off[-1])
    rho = rng.normal(size=H)
    cls = (rng.uniform(size=H) < 0.25).astype(np.uint8)
    fired = rng.permutation(20000)[:W].astype(np.int32)
    orig = rng.permutation(H).astype(np.int32)
    for og in (None, orig):
        got = comet.remove_hits(_dev(fired), _dev(hit_off), _dev(rho), _dev(cls), None if og is None else _dev(og))
        fw, ho, rh, src = O.remove_hits(fired, hit_off, rho, cls)
        np.testing.assert_array_equal(got["fired_wire"].cpu().numpy(), fw)
        np.testing.assert_array_equal(got["hit_off"].cpu().numpy(), ho)
        np.testing.assert_array_equal(got["rho"].cpu().numpy(), rh)
        np.testing.assert_array_equal(got["orig"].cpu().numpy(), src if og is None else og[src])
        assert got["counts"] == (fw.size, rh.size)


def test_scan_turns_matches_oracle_cfg1(comet, cfg1_event):
    ev = cfg1_event
    seeds, po = event_seeds(ev, shape=(6, 6, 6, 6))
    d = DevEvent(ev, seeds)
    kw = dict(half_width=[1.2, 1.0, 1.0, 2.0], n_grid=[3, 3, 3, 3], n_iter=2, shrink=0.5, k_ref=4)
    for extra in ({}, {"max_tracks": 2}, {"min_wires": 50}):
        out = comet.scan_turns(d.seeds, po, *d.phys(), ev.r_stop, *d.hits(), ev.cutoff, **kw, **extra)
        torch.cuda.synchronize()
        ref = O.scan_turns(seeds, po, *_ev_args(ev), **kw, **extra)
        np.testing.assert_array_equal(out["done"], ref["done"])
        np.testing.assert_array_equal(out["wires_before"], ref["wires_before"])
        np.testing.assert_array_equal(out["turn_seed"].cpu().numpy(), ref["turn_seed"])
        np.testing.assert_array_equal(out["turn_rss"].cpu().numpy(), ref["turn_rss"])
        np.testing.assert_array_equal(out["turn_cls"].cpu().numpy(), ref["turn_cls"])
