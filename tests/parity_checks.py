"""Checks shared by the GPU parity tests: what the CPU oracle can decide on its own about a full-size event."""
import numpy as np

from oracle import comet_oracle as O


def oracle_scan(ev, seeds, cutoff=None):
    return O.scan(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a, ev.geom.wire_b,
                  ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff if cutoff is None else cutoff)


def oracle_select(ev, seeds, rss, part_off, cutoff=None):
    return O.select_classify(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a,
                             ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.rho,
                             ev.cutoff if cutoff is None else cutoff, rss, part_off)


def check_event_against_oracle(ev, seeds, shape, part_off, rss, out, n_sample, rng, cutoff=None, n_top=192, reach=2):
    """`rss` [S], out = best_seed / best_rss / best_dca / cls of the CUDA path (numpy), `seeds` the host grid.
    (1) RSS of a sample -- strided, random, and the seeds around every chunk-of-32, 4096-chunk and partition boundary
    the launch configuration can cut at -- equals the oracle's;  (2) per partition the oracle scans the `n_top` seeds
    the device ranks lowest AND the (2 reach + 1)^4 grid neighbourhood of the winner: their RSS are equal, the winner
    is the oracle's own lowest-index argmin over them, so a wrongly high RSS next to the winner cannot hide;  (3) the
    winner's RSS, D and classified set against the oracle."""
    S = seeds.shape[1]
    P = len(part_off) - 1
    bnd = []
    for p in range(P + 1):
        bnd += list(range(int(part_off[p]) - 2, int(part_off[p]) + 2))
    for c in rng.integers(1, max(2, S // 32), 24):
        bnd += [32 * int(c) - 1, 32 * int(c)]
    for q in range(1, 16):                                      # cuts of a slab into up to 8 sub-slabs / lanes
        c = (S // 32) * q // 16 * 32
        bnd += [c - 1, c, c + 1]
    idx = np.concatenate([np.arange(0, S, max(1, S // (n_sample // 2))), rng.integers(0, S, n_sample // 2), np.array(bnd)])
    idx = np.unique(idx[(idx >= 0) & (idx < S)])
    ref = oracle_scan(ev, np.ascontiguousarray(seeds[:, idx]), cutoff=cutoff)
    assert np.array_equal(rss[idx], ref["rss"]), "sampled RSS differ from the oracle"
    lam = ev.cutoff if cutoff is None else cutoff
    assert rss.min() >= 0.0 and rss.max() <= ev.n_fired * lam * lam * (1 + 1e-12)
    n_p, n_ct, n_phi, n_z = shape
    for p in range(P):
        lo, hi = int(part_off[p]), int(part_off[p + 1])
        b = int(out["best_seed"][p])
        assert lo <= b < hi
        top = lo + np.argsort(rss[lo:hi], kind="stable")[:n_top]
        r = b - lo
        iz, r = r % n_z, r // n_z
        ip_, r = r % n_phi, r // n_phi
        ic, ipp = r % n_ct, r // n_ct
        rng_ = lambda c, n: np.arange(max(0, c - reach), min(n, c + reach + 1))
        A, Bc, C, D = np.meshgrid(rng_(ipp, n_p), rng_(ic, n_ct), rng_(ip_, n_phi), rng_(iz, n_z), indexing="ij")
        nb = lo + (((A * n_ct + Bc) * n_phi + C) * n_z + D).ravel()
        cand = np.unique(np.concatenate([top, nb, [b]]))
        rc = oracle_scan(ev, np.ascontiguousarray(seeds[:, cand]), cutoff=cutoff)
        assert np.array_equal(rss[cand], rc["rss"]), "contenders' RSS differ from the oracle"
        assert int(cand[np.argmin(rc["rss"])]) == b, "the oracle ranks another contender first"   # first minimum = lowest index
        assert rss[b] == rss[lo:hi].min() and b == lo + int(np.argmin(rss[lo:hi]))
        one = np.ascontiguousarray(seeds[:, b:b + 1])
        r1 = oracle_scan(ev, one, cutoff=cutoff)
        rs = oracle_select(ev, one, r1["rss"], np.array([0, 1], dtype=np.int64), cutoff=cutoff)
        assert float(out["best_rss"][p]) == float(r1["rss"][0])
        assert np.array_equal(out["best_dca"][p], rs["best_dca"][0])
        np.testing.assert_array_equal(out["cls"][p], rs["cls"][0])


