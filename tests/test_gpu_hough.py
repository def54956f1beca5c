"""comet_hough_seeds (k_hough) vs the oracle's hough_seeds through the C ABI (needs one B200).

Integer work: the accumulator and the peak are compared for identity.  The bin of a vote and the circle are
fp64 decisions taken with the same IEEE operations on both sides (R36-R37), so the circle and the
seed points are compared bit for bit as well (NaN where the oracle has NaN).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from comet_synth import hough_tables, make_config  # noqa: E402
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


def _dev(a, dt=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dt is not None:
        t = t.to(dt)
    return t.cuda()


def _same(a, b):
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
    return a.shape == b.shape and np.array_equal(a.view(np.int64)[~np.isnan(b)], b.view(np.int64)[~np.isnan(b)]) \
        and np.array_equal(np.isnan(a), np.isnan(b))


def _run_and_compare(comet, geom_a, geom_b, fired_lists, n_phi, rho_lo, rho_hi, n_rho, charge, bz, r_seed=50.0,
                     want_acc=True):
    c, s = hough_tables(n_phi)
    inv = n_rho / (rho_hi - rho_lo)
    ev_off = np.zeros(len(fired_lists) + 1, dtype=np.int32)
    ev_off[1:] = np.cumsum([len(f) for f in fired_lists])
    fired = np.concatenate([np.asarray(f, np.int32) for f in fired_lists]) if ev_off[-1] else np.zeros(0, np.int32)
    got = comet.hough_seeds(_dev(geom_a), _dev(geom_b), _dev(fired), _dev(ev_off), _dev(c), _dev(s), rho_lo, inv,
                            n_rho, charge, bz, r_seed, want_acc=want_acc)
    torch.cuda.synchronize()
    peak, circle = got["peak"].cpu().numpy(), got["circle"].cpu().numpy()
    acc = got["acc"].cpu().numpy() if want_acc else None
    for e, f in enumerate(fired_lists):
        ref = O.hough_seeds(geom_a, geom_b, np.asarray(f, np.int32), c, s, rho_lo, inv, n_rho, charge, bz, r_seed)
        if want_acc:
            assert np.array_equal(acc[e], ref["acc"]), "event %d: accumulator differs" % e
        assert tuple(int(v) for v in peak[e]) == ref["peak"], "event %d: peak %s vs %s" % (e, peak[e], ref["peak"])
        exp = np.concatenate([[ref["R"]], ref["centre"], ref["entrance"], ref["exit"]])
        assert _same(circle[e], exp), "event %d: circle %s vs %s" % (e, circle[e], exp)
    return peak, circle


def test_hough_cfg1_event_identical(comet, cfg1_event):
    ev = cfg1_event
    peak, circle = _run_and_compare(comet, ev.geom.wire_a, ev.geom.wire_b, [ev.fired_wire], 256, 1 / 120.0, 1 / 40.0,
                                    128, ev.charge, ev.bz)
    assert peak[0, 0] >= 15 and np.isfinite(circle[0]).all()


@pytest.mark.parametrize("n_phi,n_rho", [(1000, 300), (37, 1), (2048, 512), (5, 20000)])
def test_hough_batch_with_empty_and_ragged_shapes(comet, n_phi, n_rho):
    """A batch of config-2 events (1-4 turns, 20-240 fired wires) with an empty event in the middle; direction
    counts that do not divide into the CTAs, one bin only, and rows larger than the default shared memory."""
    evs = make_config(2, n_events=7)
    lists = [e.fired_wire for e in evs[:3]] + [np.zeros(0, np.int32)] + [e.fired_wire for e in evs[3:]]
    g = evs[0].geom
    for charge, bz in ((-1, 1.0), (+1, 0.9)):
        _run_and_compare(comet, g.wire_a, g.wire_b, lists, n_phi, 1 / 150.0, 1 / 30.0, n_rho, charge, bz)


def test_hough_high_occupancy_several_wire_tiles(comet):
    """configs[4]: ~1100 fired wires = several 256-wire tiles with a ragged tail; many equal-vote bins (ties)."""
    ev = make_config(4)[0]
    assert ev.fired_wire.size > 600
    _run_and_compare(comet, ev.geom.wire_a, ev.geom.wire_b, [ev.fired_wire, ev.fired_wire[:257], ev.fired_wire[:1]],
                     256, 1 / 120.0, 1 / 40.0, 64, ev.charge, ev.bz)


def test_hough_circle_not_reaching_the_seed_radius_and_votes_out_of_range(comet, cfg1_event):
    ev = cfg1_event
    # rho window far above any wire: no votes at all
    peak, circle = _run_and_compare(comet, ev.geom.wire_a, ev.geom.wire_b, [ev.fired_wire], 64, 1.0, 2.0, 16,
                                    ev.charge, ev.bz)
    assert tuple(peak[0]) == (0, 0, 0) and np.isnan(circle[0]).all()
    # r_seed beyond the circle's diameter: R and the centre are given, the seed points are NaN
    peak, circle = _run_and_compare(comet, ev.geom.wire_a, ev.geom.wire_b, [ev.fired_wire], 256, 1 / 120.0, 1 / 40.0,
                                    128, ev.charge, ev.bz, r_seed=200.0)
    assert peak[0, 0] > 0 and np.isfinite(circle[0, :3]).all() and np.isnan(circle[0, 3:]).all()


def test_hough_whole_config2_batch_peaks_only(comet):
    """All 256 events of configs[2] in one launch, accumulator not written; peaks and circles identical."""
    evs = make_config(2)
    g = evs[0].geom
    _run_and_compare(comet, g.wire_a, g.wire_b, [e.fired_wire for e in evs], 256, 1 / 150.0, 1 / 30.0, 128, -1, 1.0,
                     want_acc=False)


def test_hough_argument_errors(comet, cfg1_event):
    from paper_1911_09340_b200 import CometError
    ev = cfg1_event
    c, s = hough_tables(16)
    a, b = _dev(ev.geom.wire_a), _dev(ev.geom.wire_b)
    fw, off = _dev(ev.fired_wire), _dev(np.array([0, ev.fired_wire.size], np.int32))
    for kw in (dict(n_rho=0), dict(n_rho=40000), dict(inv_drho=0.0), dict(charge=0), dict(bz=0.0), dict(r_seed=-1.0)):
        args = dict(rho_min=0.01, inv_drho=1000.0, n_rho=32, charge=-1, bz=1.0, r_seed=50.0)
        args.update(kw)
        with pytest.raises(CometError):
            comet.hough_seeds(a, b, fw, off, _dev(c), _dev(s), **args)
