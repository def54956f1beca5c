"""COMET_OPT_ZGROUP (scan_zgroup.cuh): seeds in runs that differ only in z share their transverse track.

k_zgroup_check finds the run length on the device, k_gen_unique steps every distinct transverse track once and
k_scan_fused<.., ZG> adds the z column.  The results must not depend on which path ran: n_pts and RSS are compared
with the oracle bit for bit, for run lengths 8, 16 and 32, ragged seed counts, a seed set without runs (the plain
kernel must take over) and with the option switched off; the work counter `unique_states` shows which path ran.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from comet_synth import event_seeds, make_config, seed_grid  # noqa: E402
from oracle import comet_oracle as O  # noqa: E402


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


def _scan(comet, ev, seeds, zgroup, r_stop=None):
    from paper_1911_09340_b200.binding import OPT_STATS, OPT_ZGROUP
    S = seeds.shape[1]
    rss = torch.empty(S, dtype=torch.float64, device="cuda")
    n_pts = torch.empty(S, dtype=torch.int32, device="cuda")
    comet.set_option(OPT_ZGROUP, 2 if zgroup else 0)        # 2: also for calls below the size threshold of the default
    comet.set_option(OPT_STATS, 1)
    comet.read_stats(reset=True)
    try:
        comet.scan_rss(_dev(seeds), ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop if r_stop is None else r_stop,
                       _dev(ev.geom.wire_a), _dev(ev.geom.wire_b), _dev(ev.fired_wire), _dev(ev.hit_off), _dev(ev.rho),
                       ev.cutoff, rss=rss, n_pts=n_pts)
        st = comet.read_stats(reset=True)
    finally:
        comet.set_option(OPT_STATS, 0)
        comet.set_option(OPT_ZGROUP, 1)
    return rss.cpu().numpy(), n_pts.cpu().numpy(), st


def _oracle(ev, seeds, r_stop=None):
    return O.scan(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop if r_stop is None else r_stop, ev.geom.wire_a,
                  ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, want_npts=True)


@pytest.mark.parametrize("n_z,n_seeds", [(8, 8 * 8 * 8 * 4), (16, 2048), (16, 2048 - 5), (32, 1024 + 32 + 7), (64, 1024)])
def test_z_runs_identical_to_the_oracle(comet, cfg1_event, n_z, n_seeds):
    """Grids with z as the fastest axis (run length n_z); seed counts that end inside a run and inside a chunk."""
    ev = cfg1_event
    sp = ev.spec
    seeds = seed_grid(ev, 1, (8, 4, 4, n_z), tuple(sp["p_range"]), ct_hw=sp.get("ct_hw", 0.15))[:, :n_seeds]
    seeds = np.ascontiguousarray(seeds)
    ref = _oracle(ev, seeds)
    rss, n_pts, st = _scan(comet, ev, seeds, 1)
    assert np.array_equal(n_pts, ref["n_pts"]) and np.array_equal(rss, ref["rss"])
    run = min(n_z, 32)
    # the z-run kernels served the call: one RKN4 step per recorded state of every run's first seed
    assert st["unique_states"] == int((ref["n_pts"][::run].astype(np.int64) - 1).sum())
    rss0, n_pts0, st0 = _scan(comet, ev, seeds, 0)
    assert st0["unique_states"] == 0
    assert np.array_equal(rss0, rss) and np.array_equal(n_pts0, n_pts)
    # the z-run kernel prunes with its own bound (tangent line per distinct track, scan_zrun.cuh): the same pairs reach
    # the virtual-plane iteration -- a pair whose closest state sits on the far radius to 1e-12 could differ --, with fewer rows swept
    assert st["pairs"] == st0["pairs"] and abs(st["fine_needed"] - st0["fine_needed"]) <= 2
    assert st["rows_executed"] <= st0["rows_executed"]


@pytest.mark.parametrize("case", ["runs_of_4", "one_odd_seed", "shuffled", "apex_stop"])
def test_fallback_and_mixed_sets(comet, cfg1_event, case):
    ev = cfg1_event
    sp = ev.spec
    pr = tuple(sp["p_range"])
    r_stop = None
    if case == "runs_of_4":
        seeds = seed_grid(ev, 0, (8, 4, 8, 4), pr, ct_hw=0.15)       # z-runs shorter than 8: the plain kernel
        expect_zg = False
    elif case == "one_odd_seed":
        seeds = seed_grid(ev, 0, (4, 4, 4, 16), pr, ct_hw=0.15).copy()
        seeds[3, 777] *= 1.0000001                                    # one seed breaks its run
        expect_zg = False
    elif case == "shuffled":
        seeds = seed_grid(ev, 0, (4, 4, 4, 16), pr, ct_hw=0.15)
        seeds = seeds[:, np.random.default_rng(3).permutation(seeds.shape[1])]
        expect_zg = False
    else:
        seeds = seed_grid(ev, 2, (4, 4, 4, 16), pr, ct_hw=0.15)      # half tracks: the target region beyond the chamber
        r_stop = 1.0e3
        expect_zg = True
    seeds = np.ascontiguousarray(seeds)
    ref = _oracle(ev, seeds, r_stop)
    rss, n_pts, st = _scan(comet, ev, seeds, 1, r_stop)
    assert np.array_equal(n_pts, ref["n_pts"]) and np.array_equal(rss, ref["rss"])
    assert (st["unique_states"] > 0) == expect_zg


def test_full_cfg1_both_paths_agree(comet, cfg1_event):
    """The benchmarked event (3 x 131072 seeds, runs of 16): the z-run path against the plain path, every seed."""
    ev = cfg1_event
    seeds, _ = event_seeds(ev)
    rss1, n1, st1 = _scan(comet, ev, seeds, 1)
    rss0, n0, st0 = _scan(comet, ev, seeds, 0)
    assert np.array_equal(rss1, rss0) and np.array_equal(n1, n0)
    assert st1["unique_states"] * 16 == int(n1.astype(np.int64).sum()) - seeds.shape[1] and st0["unique_states"] == 0


def test_small_calls_take_the_plain_kernels_by_default(comet, cfg0_event):
    """configs[0] (8192 seeds in runs of 8) is below the size threshold of COMET_OPT_ZGROUP = 1."""
    from paper_1911_09340_b200.binding import OPT_STATS
    ev = cfg0_event
    seeds, _ = event_seeds(ev)
    comet.set_option(OPT_STATS, 1)
    comet.read_stats(reset=True)
    try:
        comet.scan_rss(_dev(seeds), ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, _dev(ev.geom.wire_a), _dev(ev.geom.wire_b),
                       _dev(ev.fired_wire), _dev(ev.hit_off), _dev(ev.rho), ev.cutoff)
        st = comet.read_stats(reset=True)
    finally:
        comet.set_option(OPT_STATS, 0)
    assert st["unique_states"] == 0 and st["pairs"] == seeds.shape[1] * ev.n_fired


def test_turn_loop_at_full_size_runs_partitions_through_the_z_run_kernels(comet, cfg1_event):
    """comet_scan_turns on the full configs[1] grids: every stage scans ONE partition of the caller's seed array
    (a pointer offset with the whole array's stride, 4096 chunks: above the size threshold), against a hit list that
    shrinks from stage to stage -- turn seeds, RSS and classified sets identical to the oracle's loop."""
    ev = cfg1_event
    seeds, po = event_seeds(ev)
    kw = dict(half_width=[0.6, 0.5, 0.5, 1.0], n_grid=[3, 3, 3, 3], n_iter=1, shrink=0.5, k_ref=4)
    args = (ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop)
    ref = O.scan_turns(seeds, po, *args, ev.geom.wire_a, ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, **kw)
    got = comet.scan_turns(_dev(seeds), po, *args, _dev(ev.geom.wire_a), _dev(ev.geom.wire_b), _dev(ev.fired_wire),
                           _dev(ev.hit_off), _dev(ev.rho), ev.cutoff, **kw)
    torch.cuda.synchronize()
    assert got["done"].tolist() == ref["done"].tolist() and ref["done"].all()
    assert got["wires_before"].tolist() == ref["wires_before"].tolist()
    assert np.array_equal(got["turn_seed"].cpu().numpy(), ref["turn_seed"])
    assert np.array_equal(got["turn_rss"].cpu().numpy(), ref["turn_rss"])
    assert np.array_equal(got["turn_cls"].cpu().numpy(), ref["turn_cls"])


@pytest.mark.parametrize("shift", [(0.0, 0.0, 0.0), (3000.0, -2000.0, 5000.0), (-40000.0, 25000.0, 8000.0),
                                   (1.0e6, -2.0e6, 5.0e5), (1.0e7, 2.0e7, -1.5e7)])
def test_single_precision_pruning_far_from_the_origin(comet, cfg1_event, shift):
    """Levels A and B of k_scan_zrun prune in single precision with the rounding carried as slack proportional to the
    size of the coordinates.  The whole event -- wires and seeds -- is moved away from the origin, up to 2e7 cm, where a
    float resolves 1-2 cm (the drift circles are 0.1-0.8 cm, the far radii about 1 cm): without the slack the tests drop
    near pairs there (checked once with COMET_ZR_FSLACK = 0: the last case fails on RSS; the far radius is itself
    conservative by more than 0.1 cm, so smaller shifts do not show it); with it RSS and n_pts stay bit-identical to the
    oracle's on the same shifted inputs (no target region: it is centred on the origin).  Up to 4e4 cm the pruning still
    prunes; at 2e7 cm the slack opens everything (rows of the last 64-row block included), which is the correct answer."""
    import copy
    ev = copy.deepcopy(cfg1_event)
    sp = ev.spec
    sh = np.asarray(shift)
    seeds = seed_grid(ev, 1, (8, 4, 4, 16), tuple(sp["p_range"]), ct_hw=sp.get("ct_hw", 0.15))
    seeds = np.ascontiguousarray(seeds)
    seeds[0:3] += sh[:, None]
    ev.geom.wire_a[:] = ev.geom.wire_a + sh[:, None]
    ev.geom.wire_b[:] = ev.geom.wire_b + sh[:, None]
    ev.n_steps = 400
    ref = _oracle(ev, seeds, r_stop=0.0)
    rss, n_pts, st = _scan(comet, ev, seeds, 1, r_stop=0.0)
    assert st["unique_states"] > 0                              # the z-run kernels served the launch
    assert np.array_equal(n_pts, ref["n_pts"])
    assert np.array_equal(rss, ref["rss"])
    assert float(np.min(rss)) < ev.n_fired * ev.cutoff ** 2     # some seed is near some wire: the comparison is not vacuous
    assert st["rows_executed"] < (0.25 if max(abs(v) for v in shift) < 1e5 else 1.2) * seeds.shape[1] * ev.n_fired * 401
