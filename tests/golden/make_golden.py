"""Writes tests/golden/cfg0_oracle.json from the CPU oracle ONLY (never from the CUDA path).

Run:  python tests/golden/make_golden.py
The file is a regression pin of the oracle on BASELINE.json configs[0] (seed 1): a later change
to the oracle's arithmetic must regenerate it and justify the change in its commit message.
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from comet_synth import event_seeds, make_config  # noqa: E402
from oracle import comet_oracle as O  # noqa: E402


def main():
    ev = make_config(0)[0]
    seeds, part_off = event_seeds(ev)
    r = O.scan(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a, ev.geom.wire_b,
               ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, want_npts=True)
    sel = O.select_classify(seeds, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a,
                            ev.geom.wire_b, ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, r["rss"], part_off)
    order = np.argsort(r["rss"], kind="stable")
    out = {
        "source": "oracle/comet_oracle.c via tests/golden/make_golden.py; BASELINE.json configs[0], rng seed 1",
        "n_seeds": int(seeds.shape[1]), "n_fired": ev.n_fired, "n_hits": ev.n_hits,
        "n_pts_min": int(r["n_pts"].min()), "n_pts_max": int(r["n_pts"].max()),
        "n_pts_sum": int(r["n_pts"].sum()),
        "best_seed": [int(v) for v in sel["best_seed"]],
        "best_rss": [float.hex(float(v)) for v in sel["best_rss"]],
        "lowest5_seeds": [int(v) for v in order[:5]],
        "lowest5_rss": [float.hex(float(v)) for v in r["rss"][order[:5]]],
        "rss_sum": float.hex(float(np.sum(r["rss"]))),
        "classified_entries": [int(j) for j in np.nonzero(sel["cls"][0])[0]],
        "best_dca": [float.hex(float(v)) for v in sel["best_dca"][0]],
    }
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg0_oracle.json"), "w") as f:
        json.dump(out, f, indent=1)
        f.write("\n")


if __name__ == "__main__":
    main()
