"""comet_argmin_static: the per-partition argmin of step C without a context and without any allocation inside the
library (its scratch is a file-scope device array) -- against the existing path, comet_select_and_classify, which
keeps the same partial minima in the context's cudaMalloc'ed workspace.  Bit equality (integer indices; the values are
copies of RSS entries).  Collected last on purpose (needs one B200)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from comet_synth import event_seeds, make_config  # noqa: E402


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _serial_argmin(rss, part_off):
    """The rule of reading R15 written out: b = lo; for s > lo: if rss[s] < rss[b]: b = s."""
    best, val = [], []
    for lo, hi in zip(part_off[:-1], part_off[1:]):
        if hi == lo:
            best.append(-1)
            val.append(np.nan)
            continue
        b = lo
        for s in range(lo + 1, hi):
            if rss[s] < rss[b]:
                b = s
        best.append(b)
        val.append(rss[b])
    return np.array(best, dtype=np.int64), np.array(val)


def test_argmin_static_equals_the_context_path_on_two_calls_in_a_row():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_1911_09340_b200 import Comet, CometError, argmin_static
    from paper_1911_09340_b200.build import build
    build()
    ev = make_config(0)[0]
    seeds, _ = event_seeds(ev, shape=(8, 8, 16, 16))            # 16384 seeds
    S = seeds.shape[1]
    c = Comet(0)
    try:
        d = _dev(seeds)
        hits = (_dev(ev.geom.wire_a), _dev(ev.geom.wire_b), _dev(ev.fired_wire), _dev(ev.hit_off), _dev(ev.rho))
        phys = (ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop)
        rss = c.scan_rss(d, *phys, *hits, ev.cutoff)["rss"]
        # call 1: three ragged partitions, one of them empty; call 2 right behind it on the same stream: other
        # partitions and a changed RSS (ties at the minimum, a NaN that must not win, a NaN at a partition's first seed)
        po1 = [0, 5000, 5000, S - 7, S]
        rss2 = rss.clone()
        m = float(rss.min().item())
        rss2[[123, 4567, 9000, S - 1]] = m * 0.5
        rss2[77] = float("nan")
        rss2[6000] = float("nan")
        po2 = [0, 100, 6000, 6001, 12000, S]
        out1 = argmin_static(rss, po1)
        out2 = argmin_static(rss2, po2)
        torch.cuda.synchronize()
        for r, po, out in ((rss, po1, out1), (rss2, po2, out2)):
            ref = c.select_and_classify(d, *phys, *hits, ev.cutoff, r, po)
            torch.cuda.synchronize()
            assert np.array_equal(out["best_seed"].cpu().numpy(), ref["best_seed"].cpu().numpy())
            assert np.array_equal(out["best_rss"].cpu().numpy(), ref["best_rss"].cpu().numpy(), equal_nan=True)
            bs, bv = _serial_argmin(r.cpu().numpy(), po)
            assert np.array_equal(out["best_seed"].cpu().numpy(), bs)
        # the same call again into the caller's own outputs: the array's old contents do not matter
        bs_buf = torch.full((8,), -7, dtype=torch.int64, device="cuda")
        br_buf = torch.zeros(8, dtype=torch.float64, device="cuda")
        argmin_static(rss, po1, best_seed=bs_buf, best_rss=br_buf)
        torch.cuda.synchronize()
        assert np.array_equal(bs_buf.cpu().numpy()[:4], out1["best_seed"].cpu().numpy())
        assert np.array_equal(br_buf.cpu().numpy()[:4], out1["best_rss"].cpu().numpy(), equal_nan=True)
        assert bs_buf.cpu().numpy()[4:].tolist() == [-7] * 4
        # the limit: 64 partitions pass, 65 are refused with the limit's message and nothing is written
        po64 = np.linspace(0, S, 65).astype(np.int64)
        o64 = argmin_static(rss, po64)
        torch.cuda.synchronize()
        assert np.array_equal(o64["best_seed"].cpu().numpy(), _serial_argmin(rss.cpu().numpy(), po64.tolist())[0])
        po65 = np.linspace(0, S, 66).astype(np.int64)
        with pytest.raises(CometError, match="limit of the statically allocated scratch"):
            argmin_static(rss, po65)
        with pytest.raises(CometError, match="invalid argument"):
            argmin_static(rss, [0, S + 1])
    finally:
        c.close()
