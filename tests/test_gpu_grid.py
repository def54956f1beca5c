"""Seed grids as inputs, the z_run promise, workspace reservation + CUDA-graph capture of a cold context, and
BASELINE.json configs[2] at full size on streams -- CUDA path vs CPU oracle through the C ABI (needs one B200).

Everything is compared for bit equality: the CUDA path performs the definition's IEEE operations one by one
(DESIGN.md section 6); the hard bars of north_star (1e-9 relative) are implied.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from comet_synth import event_axes, event_seeds, make_config  # noqa: E402
from oracle import comet_oracle as O  # noqa: E402,F401
from parity_checks import check_event_against_oracle, oracle_scan as _oracle_scan, oracle_select as _oracle_select  # noqa: E402


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


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _hits(ev):
    return (_dev(ev.geom.wire_a), _dev(ev.geom.wire_b), _dev(ev.fired_wire), _dev(ev.hit_off), _dev(ev.rho))


# ------------------------------------------------------------------------------------------------
# comet_seed_grid / comet_seed_runs
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,shape", [(0, None), (1, None), (1, (3, 5, 7, 6)), (2, (2, 1, 1, 24)), (0, (1, 1, 1, 1))])
def test_seed_grid_is_the_host_generator_bit_for_bit(comet, cfg, shape):
    ev = make_config(cfg)[0]
    seeds, part_off = event_seeds(ev, shape=shape)
    axes, shp, po = event_axes(ev, shape=shape)
    np.testing.assert_array_equal(po, part_off)
    stride = seeds.shape[1] + 40                               # a stride larger than the set
    buf = torch.full((6, stride), float("nan"), dtype=torch.float64, device="cuda")
    got = comet.seed_grid(_dev(axes), shp, seeds=buf)
    torch.cuda.synchronize()
    g = got.cpu().numpy()
    assert np.array_equal(g[:, :seeds.shape[1]], seeds)
    assert np.isnan(g[:, seeds.shape[1]:]).all()               # nothing written past the set
    # the run length the grid promises is what the device finds in the seeds
    found = comet.seed_runs(got[:, :seeds.shape[1]].contiguous())
    promised = comet.grid_z_run(shp[3])
    assert promised == {8: 8, 16: 16, 6: 2, 24: 8, 1: 1}[shp[3]]
    assert found >= promised and found in (1, 2, 4, 8, 16, 32)


def test_seed_runs_on_irregular_sets(comet):
    rng = np.random.default_rng(3)
    s = rng.normal(size=(6, 1000))
    assert comet.seed_runs(_dev(s)) == 1
    s2 = np.repeat(rng.normal(size=(6, 40)), 16, axis=1)
    s2[2] = rng.normal(size=640)                               # runs of 16 that differ only in z
    assert comet.seed_runs(_dev(s2)) == 16
    s3 = s2.copy()
    s3[4, 16 * 7 + 8:16 * 8] += 1e-13                          # one run broken in the middle: 8
    assert comet.seed_runs(_dev(s3)) == 8
    s4 = s2.copy()
    s4[0, 16 * 9 + 3] = np.nextafter(s4[0, 16 * 9 + 3], 1e9)   # one bit in x at an odd position: 1
    assert comet.seed_runs(_dev(s4)) == 1
    assert comet.seed_runs(_dev(np.repeat(rng.normal(size=(6, 3)), 64, axis=1))) == 32
    assert comet.seed_runs(_dev(s[:, :1])) == 32


# ------------------------------------------------------------------------------------------------
# the z_run promise: the same numbers with the run length promised, found on the device, or not used
# ------------------------------------------------------------------------------------------------
def test_z_run_promise_gives_the_same_numbers(comet, cfg1_event):
    from paper_1911_09340_b200.binding import OPT_STATS, OPT_ZGROUP
    ev = cfg1_event
    axes, shp, part_off = event_axes(ev, shape=(8, 8, 16, 16))      # 16384 seeds per partition: 1536 chunks, z-run kernels
    seeds = comet.seed_grid(_dev(axes), shp)
    hits = _hits(ev)
    phys = (ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop)
    outs = {}
    for zr in (0, 16, 8, 1):
        comet.set_option(OPT_STATS, 1)
        comet.read_stats(reset=True)
        o = comet.scan_rss(seeds, *phys, *hits, ev.cutoff, z_run=zr)
        st = comet.read_stats(reset=True)
        comet.set_option(OPT_STATS, 0)
        assert (st["unique_states"] > 0) == (zr != 1)          # which kernels served the call
        outs[zr] = (o["rss"].cpu().numpy(), o["n_pts"].cpu().numpy(), st["unique_states"])
    assert outs[8][2] == 2 * outs[16][2]                       # runs of 8: every track stepped twice
    for zr in (16, 8, 1):
        assert np.array_equal(outs[zr][0], outs[0][0]) and np.array_equal(outs[zr][1], outs[0][1])
    # (without the counters: the multi-lane launch configuration of the timed path)
    o = comet.scan_rss(seeds, *phys, *hits, ev.cutoff, z_run=16)
    assert np.array_equal(o["rss"].cpu().numpy(), outs[0][0])
    h = seeds.cpu().numpy()
    idx = np.arange(0, h.shape[1], 37)
    ref = _oracle_scan(ev, np.ascontiguousarray(h[:, idx]))
    assert np.array_equal(outs[0][0][idx], ref["rss"])
    with pytest.raises(Exception):
        comet.scan_rss(seeds, *phys, *hits, ev.cutoff, z_run=12)    # not a power of two
    comet.set_option(OPT_ZGROUP, 1)


@pytest.mark.parametrize("n_z,cut,r_stop,n_steps", [(32, 0, 50.0, None), (8, 0, 50.0, None), (16, 5, 50.0, None), (8, 3, 0.0, 150),
                                                    (16, 0, 1.0e3, None), (32, 31, 50.0, 40)])
def test_z_run_kernel_variants_with_the_promise(comet, cfg1_event, n_z, cut, r_stop, n_steps):
    """k_scan_zrun's three variants (1, 2 or 4 distinct tracks per chunk) with the run length PROMISED, on sets that
    end inside a run and inside a chunk, without a stop (r_stop = 0: every track uses the whole capacity), with the
    apex stop (r_stop beyond the chamber), and with fewer steps than one 64-row block."""
    from paper_1911_09340_b200.binding import OPT_ZGROUP
    from comet_synth import seed_grid
    ev = cfg1_event
    sp = ev.spec
    seeds = seed_grid(ev, 0, (3, 4, 5, n_z), tuple(sp["p_range"]), ct_hw=sp.get("ct_hw", 0.15))
    seeds = np.ascontiguousarray(seeds[:, :seeds.shape[1] - cut])
    ns = ev.n_steps if n_steps is None else n_steps
    ref = O.scan(seeds, ev.charge, ev.bz, ev.step, ns, r_stop, ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, ev.hit_off,
                 ev.rho, ev.cutoff, want_npts=True)
    comet.set_option(OPT_ZGROUP, 2)
    try:
        o = comet.scan_rss(_dev(seeds), ev.charge, ev.bz, ev.step, ns, r_stop, *_hits(ev), ev.cutoff, z_run=min(n_z, 32))
        torch.cuda.synchronize()
    finally:
        comet.set_option(OPT_ZGROUP, 1)
    assert np.array_equal(o["n_pts"].cpu().numpy(), ref["n_pts"])
    assert np.array_equal(o["rss"].cpu().numpy(), ref["rss"])


def test_z_run_kernels_without_hits_and_with_empty_wires(comet, cfg1_event):
    """No fired wire at all (RSS = 0), and a hit list in which some fired wires have no entries (they contribute cutoff^2
    and are never swept)."""
    from paper_1911_09340_b200.binding import OPT_ZGROUP
    ev = cfg1_event
    seeds, _ = event_seeds(ev, shape=(4, 4, 4, 16))
    d = _dev(seeds)
    wa, wb = _dev(ev.geom.wire_a), _dev(ev.geom.wire_b)
    phys = (ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop)
    comet.set_option(OPT_ZGROUP, 2)
    try:
        e32, ef = torch.zeros(0, dtype=torch.int32, device="cuda"), torch.zeros(0, dtype=torch.float64, device="cuda")
        o = comet.scan_rss(d, *phys, wa, wb, e32, torch.zeros(1, dtype=torch.int32, device="cuda"), ef, ev.cutoff, z_run=16)
        torch.cuda.synchronize()
        ref = O.scan(seeds, *phys, ev.geom.wire_a, ev.geom.wire_b, np.zeros(0, np.int32), np.zeros(1, np.int32), np.zeros(0),
                     ev.cutoff, want_npts=True)
        assert np.array_equal(o["rss"].cpu().numpy(), ref["rss"]) and float(o["rss"].abs().max()) == 0.0
        assert np.array_equal(o["n_pts"].cpu().numpy(), ref["n_pts"])
        # every third fired wire loses its entries
        keep = np.ones(ev.n_fired, bool)
        keep[::3] = False
        cnt = np.where(keep, np.diff(ev.hit_off), 0)
        ho = np.zeros(ev.n_fired + 1, np.int32)
        ho[1:] = np.cumsum(cnt)
        rho = np.concatenate([ev.rho[ev.hit_off[i]:ev.hit_off[i + 1]] for i in range(ev.n_fired) if keep[i]])
        o = comet.scan_rss(d, *phys, wa, wb, _dev(ev.fired_wire), _dev(ho), _dev(rho), ev.cutoff, z_run=16)
        torch.cuda.synchronize()
        ref = O.scan(seeds, *phys, ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, ho, rho, ev.cutoff)
        assert np.array_equal(o["rss"].cpu().numpy(), ref["rss"])
    finally:
        comet.set_option(OPT_ZGROUP, 1)


# ------------------------------------------------------------------------------------------------
# comet_reserve_scan: the first call of a cold context neither allocates nor synchronises -- it can be captured
# ------------------------------------------------------------------------------------------------
def test_cold_context_first_call_captured_in_a_graph(cfg1_event):
    from paper_1911_09340_b200 import Comet, CometError
    ev = cfg1_event
    axes, shp, part_off = event_axes(ev, shape=(16, 16, 16, 16))    # 6144 chunks: four sub-slab lanes
    S = int(part_off[-1])
    hits = _hits(ev)
    phys = (ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop)
    d_axes = _dev(axes)
    side = torch.cuda.Stream()
    cold = Comet(0)
    try:
        seeds = torch.empty((6, S), dtype=torch.float64, device="cuda")
        rss = torch.empty(S, dtype=torch.float64, device="cuda")
        n_pts = torch.empty(S, dtype=torch.int32, device="cuda")
        torch.cuda.synchronize()
        # without a reservation the call would have to grow its workspace: refused during capture
        g0 = torch.cuda.CUDAGraph()
        with pytest.raises(CometError):
            with torch.cuda.graph(g0, stream=side):
                cold.scan_rss(seeds, *phys, *hits, ev.cutoff, rss=rss, n_pts=n_pts, z_run=16, stream=side)
        torch.cuda.synchronize()
        cold.reserve_scan(S, ev.n_steps, ev.n_fired, z_run=16)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            cold.seed_grid(d_axes, shp, seeds=seeds, stream=side)
            cold.scan_rss(seeds, *phys, *hits, ev.cutoff, rss=rss, n_pts=n_pts, z_run=16, stream=side)
            sel = cold.select_and_classify(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, *hits, ev.cutoff, rss,
                                           part_off, stream=side)
        rss.fill_(-1.0)
        g.replay()
        torch.cuda.synchronize()
        r1 = rss.cpu().numpy().copy()
        b1 = sel["best_seed"].cpu().numpy().copy()
        rss.fill_(-2.0)
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(rss.cpu().numpy(), r1)
        h = seeds.cpu().numpy()
        ref = _oracle_scan(ev, h)
        assert np.array_equal(r1, ref["rss"])
        rs = _oracle_select(ev, h, ref["rss"], part_off)
        np.testing.assert_array_equal(b1, rs["best_seed"])
        np.testing.assert_array_equal(sel["cls"].cpu().numpy(), rs["cls"])
    finally:
        cold.close()


def test_turn_loop_replayed_from_a_graph(cfg1_event):
    """comet_scan_turns enqueues a whole event -- three stages with refinements and hit removal, list sizes and the
    stop rule on the device -- without a host read: captured once into a CUDA graph on a cold context (workspace
    reserved), replayed twice, identical to the oracle's loop, also when the stop rule fires before the last stage."""
    from paper_1911_09340_b200 import Comet
    ev = cfg1_event
    axes, shp, part_off = event_axes(ev, shape=(8, 8, 16, 16))           # 16384 seeds per partition: the z-run kernels
    seeds_h, _ = event_seeds(ev, shape=(8, 8, 16, 16))
    hits = _hits(ev)
    kw = dict(half_width=[1.2, 1.0, 1.0, 2.0], n_grid=[3, 3, 3, 3], n_iter=2, shrink=0.5, k_ref=4)
    args = (ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, ev.hit_off,
            ev.rho, ev.cutoff)
    side = torch.cuda.Stream()
    for extra in ({}, {"max_tracks": 2}, {"min_wires": 50}):
        cold = Comet(0)
        try:
            seeds = cold.seed_grid(_dev(axes), shp)
            cold.reserve_scan(int(part_off[1]), ev.n_steps, ev.n_fired, z_run=16)
            torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=side):
                out = cold.scan_turns(seeds, part_off, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, *hits, ev.cutoff,
                                      stream=side, z_run=16, sync=False, **kw, **extra)
            ref = O.scan_turns(seeds_h, part_off, *args, **kw, **extra)
            for _ in range(2):
                for k in ("turn_seed", "turn_rss"):
                    out[k].fill_(7.0)
                g.replay()
                torch.cuda.synchronize()
                np.testing.assert_array_equal(out["done_dev"].cpu().numpy().astype(bool), ref["done"])
                np.testing.assert_array_equal(out["wires_before_dev"].cpu().numpy(), ref["wires_before"])
                np.testing.assert_array_equal(out["turn_seed"].cpu().numpy(), ref["turn_seed"])
                np.testing.assert_array_equal(out["turn_rss"].cpu().numpy(), ref["turn_rss"])
                np.testing.assert_array_equal(out["turn_cls"].cpu().numpy(), ref["turn_cls"])
        finally:
            cold.close()


# ------------------------------------------------------------------------------------------------
# comet_scan_event_grid_host
# ------------------------------------------------------------------------------------------------
def test_grid_host_event_matches_oracle(comet, cfg0_event):
    ev = cfg0_event
    comet.set_geometry(ev.geom.wire_a, ev.geom.wire_b)
    axes, shp, part_off = event_axes(ev)
    seeds, _ = event_seeds(ev)
    out = comet.scan_event_grid_host(torch.from_numpy(axes).pin_memory(), shp, ev.charge, ev.bz, ev.step, ev.n_steps,
                                     ev.r_stop, ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, want_rss=True)
    ref = _oracle_scan(ev, seeds)
    assert np.array_equal(out["rss"].numpy(), ref["rss"])
    rs = _oracle_select(ev, seeds, ref["rss"], part_off)
    np.testing.assert_array_equal(out["best_seed"].numpy(), rs["best_seed"])
    np.testing.assert_array_equal(out["best_rss"].numpy(), rs["best_rss"])
    np.testing.assert_array_equal(out["cls"].numpy(), rs["cls"])
    np.testing.assert_array_equal(out["best_dca"].numpy(), rs["best_dca"])
    # the seeds-from-host entry point with the resident geometry: the same
    out2 = comet.scan_event_host(torch.from_numpy(seeds).pin_memory(), part_off, ev.charge, ev.bz, ev.step, ev.n_steps,
                                 ev.r_stop, None, None, ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, want_rss=True)
    assert np.array_equal(out2["rss"].numpy(), ref["rss"])
    np.testing.assert_array_equal(out2["cls"].numpy(), rs["cls"])


@pytest.mark.parametrize("z_run,shape", [(16, (8, 8, 32, 16)), (1, (4, 4, 4, 4))])
def test_select_does_not_reuse_tracks_of_rewritten_seeds(cfg1_event, z_run, shape):
    """The seed buffer of the last scan is rewritten in place (as an allocator that hands the same address out again would
    do): comet_select_and_classify must not classify with the tracks that scan left in the context.  State 0 of the
    reused track is compared with the seed itself on the device; the winner's track is stepped again."""
    from paper_1911_09340_b200 import Comet
    ev = cfg1_event
    seeds_a, part_off = event_seeds(ev, shape=shape)
    # other seeds of the same shape: the grid mirrored in its momentum axis and shifted in z
    seeds_b = np.ascontiguousarray(seeds_a[:, ::-1]).copy()
    seeds_b[2] += 0.37
    d, hits = _dev(seeds_a), _hits(ev)
    phys = (ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop)
    a, b = Comet(0), Comet(0)
    try:
        a.scan_rss(d, *phys, *hits, ev.cutoff, z_run=z_run)
        torch.cuda.synchronize()
        d.copy_(_dev(seeds_b))                              # same buffer, other seeds
        rss_b = b.scan_rss(d, *phys, *hits, ev.cutoff, z_run=1)["rss"]
        got = a.select_and_classify(d, *phys, *hits, ev.cutoff, rss_b, part_off)
        ref = b.select_and_classify(d, *phys, *hits, ev.cutoff, rss_b, part_off)
        torch.cuda.synchronize()
        for k in ("best_seed", "best_rss", "best_dca", "cls"):
            assert np.array_equal(got[k].cpu().numpy(), ref[k].cpu().numpy(), equal_nan=True), k
        win = got["best_seed"].cpu().numpy()
        rs = O.classify_seeds(seeds_b, win, *phys, ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff)
        np.testing.assert_array_equal(got["best_dca"].cpu().numpy(), rs["dca"])
        np.testing.assert_array_equal(got["cls"].cpu().numpy(), rs["cls"])
    finally:
        a.close()
        b.close()


def test_events_in_flight_through_submit_and_collect(comet):
    """comet_scan_event_grid_submit / _collect: six different events (configs[2]: one to four partitions, different hit
    lists) through the two slots, the next one submitted before the last one is collected; every result equals the
    synchronous call's and the oracle's; a slot refuses a second event and an empty slot refuses a collect."""
    from paper_1911_09340_b200 import CometError
    evs = make_config(2, n_events=6)
    shape = (3, 4, 4, 16)
    comet.set_geometry(evs[0].geom.wire_a, evs[0].geom.wire_b)
    args = []
    for ev in evs:
        axes, shp, part_off = event_axes(ev, shape=shape)
        args.append((ev, axes, shp, part_off))
    sync = [comet.scan_event_grid_host(torch.from_numpy(a), shp, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop,
                                       ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff) for ev, a, shp, _ in args]
    sync = [{k: v.clone() for k, v in o.items()} for o in sync]
    sub = lambda k: comet.scan_event_grid_submit(k % 2, torch.from_numpy(args[k][1]), args[k][2], args[k][0].charge, args[k][0].bz,
                                                 args[k][0].step, args[k][0].n_steps, args[k][0].r_stop, args[k][0].fired_wire,
                                                 args[k][0].hit_off, args[k][0].rho, args[k][0].cutoff)
    with pytest.raises(CometError):
        comet.scan_event_grid_collect(0, (1, 1, 1))
    sizes, got = {}, {}
    sizes[0] = sub(0)
    with pytest.raises(CometError):
        sub(0)                                              # the slot is taken (nothing is enqueued)
    for k in range(1, len(args)):
        sizes[k] = sub(k)
        got[k - 1] = comet.scan_event_grid_collect((k - 1) % 2, sizes[k - 1])
    got[len(args) - 1] = comet.scan_event_grid_collect((len(args) - 1) % 2, sizes[len(args) - 1])
    for k, (ev, axes, shp, part_off) in enumerate(args):
        for key in ("best_seed", "best_rss", "best_dca", "cls"):
            assert np.array_equal(got[k][key].numpy(), sync[k][key].numpy(), equal_nan=True), (k, key)
        seeds, _ = event_seeds(ev, shape=shape)
        ref = _oracle_scan(ev, seeds)
        rs = _oracle_select(ev, seeds, ref["rss"], part_off)
        np.testing.assert_array_equal(got[k]["best_seed"].numpy(), rs["best_seed"])
        np.testing.assert_array_equal(got[k]["cls"].numpy(), rs["cls"])
        np.testing.assert_array_equal(got[k]["best_dca"].numpy(), rs["best_dca"])


def test_full_cfg2_batch_on_streams_as_benchmarked():
    """BASELINE.json configs[2] at full size, the way bench.py's batch leg runs it: the events' full grids (131072
    seeds per partition, 1-4 turns, |p| from 60 to 105 MeV/c) built on the device from their axes, scanned with the
    promised run length (z-run kernels, sub-slab lanes) on 2 streams with one context each, all in flight together.
    The first 32 of the 256 events are checked against the oracle one by one (the bench asserts that the batch of
    256 reproduces the single-stream results)."""
    from paper_1911_09340_b200 import Comet
    n_events, n_str = 32, 2
    events = make_config(2, n_events=n_events)
    # (momenta below ~80 MeV/c do not reach 5 layers and are redrawn, R19: the accepted ones span 82..105)
    assert len({len(ev.partitions) for ev in events}) == 4 and min(ev.pmag for ev in events) < 85 < 100 < max(ev.pmag for ev in events)
    ctxs = [Comet(0) for _ in range(n_str)]
    streams = [torch.cuda.Stream() for _ in range(n_str)]
    wa, wb = _dev(events[0].geom.wire_a), _dev(events[0].geom.wire_b)
    try:
        items, outs = [], []
        for ev in events:
            axes, shp, part_off = event_axes(ev)
            items.append((ev, _dev(axes), shp, part_off, _dev(ev.fired_wire), _dev(ev.hit_off), _dev(ev.rho)))
        for q in ctxs:
            q.reserve_scan(4 * 131072, events[0].n_steps, 250, z_run=16)
        torch.cuda.synchronize()
        for k, (ev, d_axes, shp, part_off, fw, ho, rho) in enumerate(items):
            q, st = ctxs[k % n_str], streams[k % n_str]
            with torch.cuda.stream(st):
                seeds = q.seed_grid(d_axes, shp, stream=st)
                o = q.scan_event(seeds, part_off, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, wa, wb, fw, ho, rho,
                                 ev.cutoff, stream=st, z_run=q.grid_z_run(shp[3]))
                o["seeds"] = seeds
                outs.append(o)
        torch.cuda.synchronize()
        rng = np.random.default_rng(2)
        for (ev, _, shp, part_off, *_), o in zip(items, outs):
            seeds_h, po = event_seeds(ev)
            assert np.array_equal(o["seeds"].cpu().numpy(), seeds_h) and np.array_equal(po, part_off)
            got = {k: o[k].cpu().numpy() for k in ("best_seed", "best_rss", "best_dca", "cls")}
            check_event_against_oracle(ev, seeds_h, shp, part_off, o["rss"].cpu().numpy(), got, 768, rng)
    finally:
        for c in ctxs:
            c.close()


@pytest.mark.parametrize("cfg", [3, 4])
def test_full_cfg3_cfg4_grid_path(comet, cfg):
    """configs[3] (4 x 1048576 seeds, 1600 steps) and configs[4] (~970 fired wires, three cutoffs) at full size
    through the device-resident grid path of bench.py, with the oracle-side contender check."""
    ev = make_config(cfg)[0]
    axes, shp, part_off = event_axes(ev)
    seeds_h, _ = event_seeds(ev)
    wa, wb, fw, ho, rho = _hits(ev)
    seeds = comet.seed_grid(_dev(axes), shp)
    rng = np.random.default_rng(cfg)
    for lam in ev.spec.get("cutoffs", (ev.cutoff,)):
        o = comet.scan_event(seeds, part_off, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, wa, wb, fw, ho, rho,
                             lam, z_run=comet.grid_z_run(shp[3]))
        torch.cuda.synchronize()
        got = {k: o[k].cpu().numpy() for k in ("best_seed", "best_rss", "best_dca", "cls")}
        check_event_against_oracle(ev, seeds_h, shp, part_off, o["rss"].cpu().numpy(), got, 2048 if cfg == 3 else 1024,
                                   rng, cutoff=lam)


# ------------------------------------------------------------------------------------------------
# step C after a plain scan: the winner's track from the scan's checkpoints (select.cuh)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n_steps,r_stop,n_seeds", [(None, None, 997), (41, 0.0, 256), (40, 0.0, 100), (43, None, 64),
                                                    (None, 70.0, 300), (7, None, 33), (3, 0.0, 32)])
def test_select_after_a_plain_scan_uses_its_checkpoints(cfg0_event, n_steps, r_stop, n_seeds):
    """comet_select_and_classify right after comet_scan_rss of the same seed buffer (plain kernels: a small set) rebuilds
    the winners' tracks from the scan's checkpoints -- one thread per checkpoint instead of one chain -- and skips the wire
    table and, for small partitions, the first argmin stage.  Same winners, RSS, D and classified sets as a context that
    has not seen the scan (the chain), and as the oracle; tracks that stop early, at a checkpoint row, one row after it,
    or fill the capacity; a ragged last chunk; a partition that starts inside a chunk."""
    from paper_1911_09340_b200 import Comet
    ev = cfg0_event
    n_steps = ev.n_steps if n_steps is None else n_steps
    r_stop = ev.r_stop if r_stop is None else r_stop
    seeds, _ = event_seeds(ev)
    rng = np.random.default_rng(11)
    pick = np.sort(rng.choice(seeds.shape[1], n_seeds, replace=False))
    seeds = np.ascontiguousarray(seeds[:, pick])
    part_off = [0, n_seeds // 3 + 1, n_seeds]
    d, hits = _dev(seeds), _hits(ev)
    phys = (ev.charge, ev.bz, ev.step, n_steps, r_stop)
    a, b = Comet(0), Comet(0)
    try:
        o = a.scan_rss(d, *phys, *hits, ev.cutoff)
        sa = a.select_and_classify(d, *phys, *hits, ev.cutoff, o["rss"], part_off)
        sb = b.select_and_classify(d, *phys, *hits, ev.cutoff, o["rss"], part_off)
        torch.cuda.synchronize()
        for k in ("best_seed", "best_rss", "best_dca", "cls"):
            assert np.array_equal(sa[k].cpu().numpy(), sb[k].cpu().numpy(), equal_nan=True), k
        ref = O.select_classify(seeds, *phys, ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff,
                                o["rss"].cpu().numpy(), part_off)
        assert np.array_equal(sa["best_seed"].cpu().numpy(), ref["best_seed"])
        assert np.array_equal(sa["best_dca"].cpu().numpy(), ref["best_dca"], equal_nan=True)
        assert np.array_equal(sa["cls"].cpu().numpy().astype(bool), np.asarray(ref["cls"]).astype(bool))
        # the track lengths the checkpoints stand for span the cases named above
        np_w = o["n_pts"].cpu().numpy()[ref["best_seed"]]
        assert np.all(np_w >= 1) and np.all(np_w <= n_steps + 1)
    finally:
        a.close()
        b.close()
