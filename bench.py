#!/usr/bin/env python
"""bench.py -- throughput of the seed x hit scan on BASELINE.json configs[1], one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1] [--path fused|materialised]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A step is one pass of the whole hot path over one synthetic event whose inputs are resident in HBM:
comet_scan_rss (kernels A + B fused, track on chip; default) or comet_seed_extrapolate + comet_dca_rss
(--path materialised), then comet_select_and_classify.  `value` is
seed x fired-wire DCA evaluations per second over all ranks (each rank scans its own replica of the
event: weak scaling, no data-path collective).  `e2e` is the same metric through
comet_scan_event_host with pinned HOST buffers (H2D of the inputs and D2H of the results inside the
timed region).  `roofline` is for the longest kernel of the step, timed live with CUDA events on its stream.
`--impl reference` times the CPU oracle (oracle/) on the host cores on a bounded sample.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "seed_hit_dca_evals_per_s"
UNIT = "DCA evals/s (seed x fired-wire pairs)"

# FP64 pipe model of k_dca_rss: per (seed, wire, recorded state) the shortlist
# issues 9 FP64-pipe instructions (6 DFMA + DMUL + DFMA + DSETP); per (seed, wire) the exact decision
# + virtual-plane iteration + residual issue about FINE_INSTR more.  FLOPs are pipe slots x 2.
SHORTLIST_INSTR = 9
FINE_INSTR = 600
# 148 SMs x 64 FP64 FMA lanes x 2 flop x 1.965 GHz (B200_PROFILING.md: 148 SMs, clocks.max.sm 1965 MHz)
FP64_PEAK_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
# FP64-pipe instructions per recorded state in kernel A: the RKN4 step of reading R1 is 48 IEEE operations
# (44 issued: the two exact doublings ride on FMAs) + 4 for the target-region test of R3
GEN_INSTR = 48
# refinement recipe of the `stage` entry (R26): box half widths about one step of the configs[1] grid
STAGE_HALF_WIDTH = [0.6, 0.5, 0.5, 1.0]
STAGE_GRID = [5, 5, 5, 5]
# `field` entry: step tolerance of R31 and the FP64-pipe instructions of one attempted Nystrom step in the map
FIELD_TOL = 1e-7
FIELD_STEP_INSTR = 420
# `seeding` entry: Hough accumulator (R36): directions, rho bins, rho window in 1/cm (R from 15 to 75 cm)
HOUGH_N_PHI, HOUGH_N_RHO, HOUGH_RHO = 256, 128, (1.0 / 150.0, 1.0 / 30.0)
# dram__bytes_read.sum + dram__bytes_write.sum per launch on configs[1] (profiles/r1d_full_scan_fused_fine_ck.txt: plain kernels)
TRAFFIC_BYTES = {"k_scan_fused": 347658496 + 2243479000, "k_fine_ck": 681160960 + 80465000}
# the same with COMET_OPT_ZGROUP (profiles/r1h_full_zgroup.txt): k_gen_unique + k_scan_fused<ZG>, k_fine_ck<ZG>
TRAFFIC_BYTES_ZG = {"k_scan_fused": 17152768 + 235757056 + 338066432 + 661437952, "k_fine_ck": 471857920 + 72980736}


def _event(cfg):
    from comet_synth import event_seeds, make_config
    ev = make_config(cfg)[0]
    seeds, part_off = event_seeds(ev)
    return ev, seeds, part_off


def _workload_name(cfg, ev, seeds, part_off):
    return ("BASELINE.json configs[%d]: %d partition(s) x %d seeds, %d fired wires / %d hit entries, "
            "%d steps x %.3g cm, r_stop %.0f cm, cutoff %.3g cm"
            % (cfg, len(part_off) - 1, seeds.shape[1] // (len(part_off) - 1), ev.n_fired, ev.n_hits,
               ev.n_steps, ev.step, ev.r_stop, ev.cutoff))


# --------------------------------------------------------------------------------------------------
# CPU oracle legs
# --------------------------------------------------------------------------------------------------
def _oracle_time(ev, seeds, part_off, n_sample):
    """Seconds the oracle needs for A+B on the first n_sample seeds plus C on them."""
    from oracle import comet_oracle as O
    sub = np.ascontiguousarray(seeds[:, :n_sample])
    t0 = time.perf_counter()
    r = O.scan(sub, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a, ev.geom.wire_b,
               ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff)
    O.select_classify(sub, ev.charge, ev.bz, ev.step, ev.n_steps, ev.r_stop, ev.geom.wire_a, ev.geom.wire_b,
                      ev.fired_wire, ev.hit_off, ev.rho, ev.cutoff, r["rss"],
                      np.array([0, n_sample], dtype=np.int64))
    return time.perf_counter() - t0


def _oracle_sample_size(ev, seeds, part_off, target_s):
    S = seeds.shape[1]
    probe = min(S, 4096)
    t = _oracle_time(ev, seeds, part_off, probe)
    n = int(min(S, max(probe, probe * target_s / max(t, 1e-6))))
    return max(32, n // 32 * 32)


def cpu_baseline(ev, seeds, part_off, target_s=15.0):
    from oracle import comet_oracle as O
    n = _oracle_sample_size(ev, seeds, part_off, target_s)
    t = _oracle_time(ev, seeds, part_off, n)
    return {"value": n * ev.n_fired / t, "unit": UNIT, "cores": O.max_threads(), "kind": "oracle",
            "sample": "first %d of %d seeds of the same event (A+B+C), %.1f s" % (n, seeds.shape[1], t),
            "events_per_s_extrapolated": 1.0 / (t * seeds.shape[1] / n)}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import comet_oracle as O
    ev, seeds, part_off = _event(args.config)
    n = _oracle_sample_size(ev, seeds, part_off, 4.0)
    for _ in range(args.warmup):
        _oracle_time(ev, seeds, part_off, n)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _oracle_time(ev, seeds, part_off, n)
    dt = (time.perf_counter() - t0) / args.steps
    value = n * ev.n_fired / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": _workload_name(args.config, ev, seeds, part_off),
                   "note": "CPU oracle (oracle/comet_oracle.c, gcc -O2, OpenMP over seeds) on the host cores; "
                           "each step scans a bounded sample of the event's seeds"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": O.max_threads(), "kind": "oracle",
                         "sample": "first %d of %d seeds per step (A+B+C)" % (n, seeds.shape[1])},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# --------------------------------------------------------------------------------------------------
# clocks
# --------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "50"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.f.read().splitlines():
            c = [x.strip() for x in ln.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1])); pw.append(float(c[2]))
            except ValueError:
                continue
            for nm, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), power_w_max=float(max(pw)),
                       reasons=sorted(reasons), samples=len(sm))
        return out


# --------------------------------------------------------------------------------------------------
# CUDA legs
# --------------------------------------------------------------------------------------------------
def _time_steps(fn, n, stream):
    import torch
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(n):
        out = fn()
    e1.record(stream)
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / n, out


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1911_09340_b200 import Comet
    from paper_1911_09340_b200.binding import COARSE_EXHAUSTIVE, COARSE_PRUNED, OPT_COARSE_SEARCH, OPT_LANES, OPT_STATS, OPT_TIMING, OPT_ZGROUP
    from paper_1911_09340_b200.build import build

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        build()
    if world > 1:
        dist.barrier()
    torch.cuda.set_device(local)
    ev, seeds, part_off = _event(args.config)
    S, W, H, P = seeds.shape[1], ev.n_fired, ev.n_hits, len(part_off) - 1
    fused = args.path == "fused"
    c = Comet(local)
    c.set_option(OPT_ZGROUP, 1 if args.zgroup else 0)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    d_seeds, d_wa, d_wb = dev(seeds), dev(ev.geom.wire_a), dev(ev.geom.wire_b)
    d_fw, d_ho, d_rho = dev(ev.fired_wire), dev(ev.hit_off), dev(ev.rho)
    n_pts = torch.empty(S, dtype=torch.int32, device="cuda")
    rss = torch.empty(S, dtype=torch.float64, device="cuda")
    phys = (ev.charge, ev.bz, ev.step, ev.n_steps)
    hits = (d_wa, d_wb, d_fw, d_ho, d_rho)
    stream = torch.cuda.current_stream()
    track = None

    call_events = []                     # CUDA events on the stream around the A + B call of every timed step

    def step_fused():
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        c.scan_rss(d_seeds, *phys, ev.r_stop, *hits, ev.cutoff, rss=rss, n_pts=n_pts)
        e1.record(stream)
        call_events.append((e0, e1))
        return c.select_and_classify(d_seeds, *phys, ev.r_stop, *hits, ev.cutoff, rss, part_off)

    def step_mat():
        c.seed_extrapolate(d_seeds, *phys, ev.r_stop, track=track, n_pts=n_pts)
        c.dca_rss(track, n_pts, d_seeds, *phys, *hits, ev.cutoff, rss=rss)
        return c.select_and_classify(d_seeds, *phys, ev.r_stop, *hits, ev.cutoff, rss, part_off)

    if not fused:
        track = torch.empty(c.track_bytes(S, ev.n_steps), dtype=torch.uint8, device="cuda")
    step = step_fused if fused else step_mat
    knames = ("k_scan_fused", "k_fine_ck", "k_rss_sum") if fused else ("k_coarse_pruned", "k_fine", "k_rss_sum")

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    torch.cuda.synchronize()
    del call_events[:]
    ms_per_step, out = _time_steps(step, args.steps, stream)
    if world > 1:
        dist.barrier()
    clocks = sampler.stop() if sampler else None
    ms_call = float(np.mean([a.elapsed_time(b) for a, b in call_events])) if call_events else None
    # per-kernel device times: the library brackets its kernels with CUDA events; with this option
    # comet_scan_rss runs its sub-slabs one after the other on the caller's stream (kernels in isolation)
    c.set_option(OPT_TIMING, 1)
    _time_steps(step, min(args.steps, 32), stream)
    ktimes = c.read_timing(knames)
    c.set_option(OPT_TIMING, 0)
    if world > 1:
        t = torch.tensor([ms_per_step], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_per_step = float(t.item())
    pairs = float(S) * W
    value = world * pairs / (ms_per_step * 1e-3)
    n_states = float(n_pts.sum().item())
    best = out["best_seed"].cpu().numpy().tolist()
    n_cls = int(out["cls"].sum().item())
    rss_main = rss.clone()

    # ---- work counters (one untimed extra pass) -------------------------------------------------
    c.set_option(OPT_STATS, 1)
    c.read_stats(reset=True)
    if fused:
        c.scan_rss(d_seeds, *phys, ev.r_stop, *hits, ev.cutoff, rss=rss, n_pts=n_pts)
    else:
        c.dca_rss(track, n_pts, d_seeds, *phys, *hits, ev.cutoff, rss=rss)
    stats = c.read_stats(reset=True)
    c.set_option(OPT_STATS, 0)

    # ---- the other path and the exhaustive closest-state search, for comparison (untimed region) ----
    n_cmp = 1 + min(args.steps, 5)
    ms_other, paths_agree, ms_exh, exh_agree = None, None, None, None
    compare = c.track_bytes(S, ev.n_steps) <= (48 << 30)     # configs[3]'s track (322 GB) does not fit: no comparison
    if compare:
        if track is None:
            track = torch.empty(c.track_bytes(S, ev.n_steps), dtype=torch.uint8, device="cuda")
        other_step = step_mat if fused else step_fused
        other_step()
        ms_other, _ = _time_steps(other_step, n_cmp, stream)
        paths_agree = bool(torch.equal(rss, rss_main))
        c.seed_extrapolate(d_seeds, *phys, ev.r_stop, track=track, n_pts=n_pts)
        c.set_option(OPT_COARSE_SEARCH, COARSE_EXHAUSTIVE)
        exh = lambda: c.dca_rss(track, n_pts, d_seeds, *phys, *hits, ev.cutoff, rss=rss)
        exh()
        ms_exh, _ = _time_steps(exh, n_cmp, stream)
        exh_agree = bool(torch.equal(rss, rss_main))
        c.set_option(OPT_COARSE_SEARCH, COARSE_PRUNED)
    track = None
    torch.cuda.empty_cache()

    # ---- a whole stage: scan + 3 on-device refinements + final selection + classification ----
    stage = None
    if fused:
        skw = dict(half_width=STAGE_HALF_WIDTH, n_grid=STAGE_GRID, n_iter=3, shrink=0.5, k_ref=10, k_final=10)
        so = c.scan_stage(d_seeds, part_off, *phys, ev.r_stop, *hits, ev.cutoff, **skw)
        swork = so["work"]
        ms_stage, so = _time_steps(lambda: c.scan_stage(d_seeds, part_off, *phys, ev.r_stop, *hits, ev.cutoff, work=swork, **skw),
                                   n_cmp, stream)
        g = int(np.prod(STAGE_GRID))
        stage = {"ms_per_stage": ms_stage, "iterations": 4,
                 "seeds_per_iteration": [S] + [P * 10 * g] * 3,
                 "dca_evals_per_s": (S + 3 * P * 10 * g) * W / (ms_stage * 1e-3),
                 "best_rss_first_iteration": out["best_rss"].cpu().numpy().tolist(),
                 "best_rss_final": so["final_rss"][:, 0].cpu().numpy().tolist(),
                 "recipe": "comet_scan_stage: k_ref 10, half widths %s (z cm, px, py, pz MeV/c) halved per iteration, "
                           "grid %s per reference, 10 finally selected seeds per partition classified" % (STAGE_HALF_WIDTH, STAGE_GRID)}
        del swork, so

    # ---- the same event in an inhomogeneous field map with the adaptive step (R29-R32) ----
    field = None
    if fused and args.field:
        from comet_synth import solenoid_map
        fB, fo, fd = solenoid_map()
        d_map = dev(fB)
        c.set_field(d_map, fo, fd, FIELD_TOL)
        step_fused()
        ms_field, fo_out = _time_steps(step_fused, max(2, n_cmp // 2), stream)
        st_field = float(n_pts.sum().item())
        c.set_option(OPT_TIMING, 1)
        _time_steps(step_fused, 2, stream)
        kt_field = c.read_timing(knames)
        c.set_option(OPT_TIMING, 0)
        c.set_field(None)
        field = {"ms_per_step": ms_field, "dca_evals_per_s": pairs / (ms_field * 1e-3), "rkn_tol_cm": FIELD_TOL,
                 "recorded_states_per_seed": st_field / S, "kernels_serial_ms": kt_field,
                 "best_seed": fo_out["best_seed"].cpu().numpy().tolist(),
                 "map": "comet_synth.solenoid_map(): %s nodes, %.0f cm spacing, B_z falling off towards the end plates"
                        % ("x".join(str(v) for v in fB.shape[:3]), fd[0]),
                 "fp64_model": "about %d FP64-pipe instructions per attempted step (3 trilinear look-ups of 3 components, "
                               "4 cross products, error estimate)" % FIELD_STEP_INSTR,
                 "k_scan_fused_tflops_model": 2.0 * FIELD_STEP_INSTR * st_field / (kt_field["k_scan_fused"] * 1e-3) / 1e12}
        del d_map

    # ---- seeding workloads of SURVEY 8(f): Hough transform (NEXT #4) and one turn as two half tracks (NEXT #3) ----
    seeding = None
    if fused and args.seeding:
        from comet_synth import hough_tables, make_config
        evs = make_config(2, n_events=32)
        lists = [e.fired_wire for e in evs] * 8                      # 256 events: the first 32 of configs[2], 8 times
        ev_off = np.zeros(len(lists) + 1, dtype=np.int32)
        ev_off[1:] = np.cumsum([f.size for f in lists])
        ct, stb = hough_tables(HOUGH_N_PHI)
        inv = HOUGH_N_RHO / (HOUGH_RHO[1] - HOUGH_RHO[0])
        hargs = (d_wa, d_wb, dev(np.concatenate(lists)), dev(ev_off), dev(ct), dev(stb), HOUGH_RHO[0], inv, HOUGH_N_RHO,
                 -1, 1.0, 50.0)
        c.hough_seeds(*hargs, want_acc=False)
        ms_h, _ = _time_steps(lambda: c.hough_seeds(*hargs, want_acc=False), 20, stream)
        votes = float(ev_off[-1]) * HOUGH_N_PHI
        # the call is shorter than its launch path from Python: replayed from a CUDA graph the device time shows
        hg = torch.cuda.CUDAGraph()
        with torch.cuda.graph(hg):
            hg_out = c.hough_seeds(*hargs, want_acc=False)
        hg.replay()
        ms_hg, _ = _time_steps(hg.replay, 50, stream)
        # one turn of this event as two half tracks: Hough circle of the event, grids at the entrance and exit points
        one = dev(np.array([0, ev.n_fired], dtype=np.int32))
        ho1 = c.hough_seeds(d_wa, d_wb, d_fw, one, dev(ct), dev(stb), HOUGH_RHO[0], inv, HOUGH_N_RHO, ev.charge, ev.bz, 50.0,
                            want_acc=False)
        n0 = int(part_off[1])
        se = d_seeds[:, :n0].contiguous()
        hx, pt = ev.helix(), ev.partitions[0]
        x_out = hx.position(np.asarray(pt.s_out))
        t_out = hx.tangent(np.asarray(pt.s_out))
        sx_h = seeds[:, :n0].copy()                                  # the same grid shape, moved to the exit state
        sx_h[0], sx_h[1] = x_out[0], x_out[1]
        sx_h[2] += x_out[2] - pt.z
        rot = np.arctan2(t_out[1], t_out[0]) - pt.phi
        px, py = sx_h[3].copy(), sx_h[4].copy()
        sx_h[3], sx_h[4] = px * np.cos(rot) - py * np.sin(rot), px * np.sin(rot) + py * np.cos(rot)
        sx = dev(sx_h)
        hkw = dict(half_width=STAGE_HALF_WIDTH, n_grid=STAGE_GRID, n_iter=3, shrink=0.5, k_ref=10, k_final=10)
        d_layer, d_circ = dev(ev.geom.layer), ho1["circle"][0].contiguous()
        hfn = lambda: c.scan_half_tracks(se, sx, *phys, 1.0e3, *hits, ev.cutoff, d_layer, d_circ, 3.0, 3, **hkw)
        hfn()
        hfn()
        ms_half, hout_ = _time_steps(hfn, 10, stream)
        seeding = {"hough": {"ms_per_launch": ms_h, "events": len(lists), "fired_wires": int(ev_off[-1]),
                             "ms_per_graph_replay": ms_hg, "votes_per_s": votes / (ms_hg * 1e-3),
                             "events_per_s": len(lists) / (ms_hg * 1e-3),
                             "accumulator": "%d directions x %d rho bins per event, kept in shared memory (not written out)"
                                            % (HOUGH_N_PHI, HOUGH_N_RHO),
                             "workload": "256 events in one launch: the first 32 events of configs[2], 8 times"},
                   "half_tracks": {"ms_per_turn": ms_half, "seeds_per_side": n0, "k_final": 10,
                                   "valid_pairs": int(hout_["valid"].sum().item()),
                                   "best_pair_hits": int(hout_["n_cls"][0, 0].item()),
                                   "recipe": "comet_scan_half_tracks on turn 0 of the event: Hough circle -> two hit lists "
                                             "(3 cm overlap), the partition's grid at the entrance and the same grid moved to "
                                             "the truth exit state, 3 refinements per side, layer veto (>= 3 layers), 10 x 10 merge"}}
        del hout_, se, sx, hg, hg_out

    # ---- configs[2]: a batch of independent events in flight on streams (one context per stream) ----
    batch = None
    if fused and args.batch > 0:
        from comet_synth import event_seeds, make_config
        bevs = make_config(2, n_events=args.batch)
        n_str = 2
        bctx = [Comet(local) for _ in range(n_str)]
        for q in bctx:
            q.set_option(OPT_ZGROUP, 1 if args.zgroup else 0)
        bstr = [torch.cuda.Stream() for _ in range(n_str)]
        items = []
        for bev in bevs:
            bs, bpo = event_seeds(bev)
            items.append((bev, dev(bs), bpo, dev(bev.fired_wire), dev(bev.hit_off), dev(bev.rho)))

        def run_batch():
            for q in bstr:
                q.wait_stream(stream)
            res = []
            for k, (bev, bs, bpo, bfw, bho, brho) in enumerate(items):
                q = bstr[k % n_str]
                with torch.cuda.stream(q):
                    res.append(bctx[k % n_str].scan_event(bs, bpo, bev.charge, bev.bz, bev.step, bev.n_steps, bev.r_stop,
                                                          d_wa, d_wb, bfw, bho, brho, bev.cutoff, stream=q))
            for q in bstr:
                stream.wait_stream(q)
            return res
        run_batch()
        run_batch()
        torch.cuda.synchronize()
        ms_batch, _ = _time_steps(run_batch, 6, stream)
        b_parts = sum(len(it[2]) - 1 for it in items)
        b_pairs = sum(float(it[1].shape[1]) * it[0].n_fired for it in items)
        batch = {"events": len(items), "partitions": b_parts, "ms_per_batch": ms_batch,
                 "events_per_s": len(items) / (ms_batch * 1e-3), "dca_evals_per_s": b_pairs / (ms_batch * 1e-3),
                 "workload": "the first %d events of BASELINE.json configs[2] (1-4 turns, |p| in [60, 105] MeV/c, 131072 seeds "
                             "per partition), device-resident, %d streams with one context each" % (len(items), n_str)}
        for q in bctx:
            q.close()
        del items, bctx

    # ---- e2e: host buffers through comet_scan_event_host -------------------------------------
    pin = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a)).to(dt).pin_memory()
    h = dict(seeds=pin(seeds, torch.float64), wa=pin(ev.geom.wire_a, torch.float64), wb=pin(ev.geom.wire_b, torch.float64),
             fw=pin(ev.fired_wire, torch.int32), ho=pin(ev.hit_off, torch.int32), rho=pin(ev.rho, torch.float64))
    budget = 0 if fused else 8 << 30
    hout = None

    def e2e_step():
        nonlocal hout
        hout = c.scan_event_host(h["seeds"], part_off, *phys, ev.r_stop, h["wa"], h["wb"], h["fw"], h["ho"], h["rho"],
                                 ev.cutoff, out=hout, track_budget_bytes=budget)

    for _ in range(max(1, min(args.warmup, 3))):
        e2e_step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    w0 = time.perf_counter()
    for _ in range(args.steps):
        e2e_step()
    e2e_s = (time.perf_counter() - w0) / args.steps
    if world > 1:
        t = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    h2d = sum(int(v.numel() * v.element_size()) for v in h.values())
    d2h = sum(int(v.numel() * v.element_size()) for v in hout.values())
    assert hout["best_seed"].numpy().tolist() == best

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    # ---- FP64 pipe peak, measured live ---------------------------------------------------------
    n_fma = c.fp64_peak_probe(8 * 4096)
    torch.cuda.synchronize()
    pe0, pe1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    best_ms = 1e30
    for _ in range(5):
        pe0.record(stream); c.fp64_peak_probe(8 * 4096); pe1.record(stream)
        torch.cuda.synchronize()
        best_ms = min(best_ms, pe0.elapsed_time(pe1))
    peak_measured = 2 * n_fma / (best_ms * 1e-3) / 1e12
    peak = FP64_PEAK_NOMINAL_TFLOPS
    ev_needed = stats["samples"] + stats["rows_needed"]
    ev_exec = stats["samples"] + stats["rows_executed"]
    gen = GEN_INSTR * n_states if fused else 0.0
    # z-runs (scan_zgroup.cuh): the RKN4 step is executed once per distinct transverse track and every seed adds its z
    uniq = float(stats.get("unique_states", 0))
    gen_exec = (GEN_INSTR * uniq + n_states) if (fused and uniq > 0) else gen
    fl = {knames[0]: 2.0 * (gen + SHORTLIST_INSTR * ev_needed), knames[1]: 2.0 * FINE_INSTR * stats["fine_needed"]}
    # k_fine_ck<ZG> reads the three candidate states instead of regenerating them (about 3.5 RKN4 steps of the 600)
    fine_exec = (FINE_INSTR - 168) if (fused and uniq > 0) else FINE_INSTR
    fl_exec = {knames[0]: 2.0 * (gen_exec + SHORTLIST_INSTR * ev_exec), knames[1]: 2.0 * fine_exec * stats["fine_executed"]}
    kernels = {"timed_over": "%d steps after the timed region with COMET_OPT_TIMING (CUDA events recorded by the library "
                             "on its stream; kernels run one after the other)" % ktimes["n_calls"]}
    kernels.update({k: {"ms_per_launch": ktimes[k], "achieved": fl[k] / (ktimes[k] * 1e-3) / 1e12,
                        "frac": fl[k] / (ktimes[k] * 1e-3) / 1e12 / peak,
                        "achieved_executed": fl_exec[k] / (ktimes[k] * 1e-3) / 1e12,
                        "share_of_step": ktimes[k] / ms_per_step} for k in fl})
    kernels["k_rss_sum"] = {"ms_per_launch": ktimes["k_rss_sum"], "bound": "hbm",
                            "achieved_gbs": (pairs * 8 + S * 8) / (ktimes["k_rss_sum"] * 1e-3) / 1e9}
    kernel = max(fl, key=lambda k: ktimes[k])
    if fused and ms_call is not None:
        # the timed region runs k_scan_fused and k_fine_ck of different sub-slabs concurrently: the roofline entry
        # is the A + B call as launched there (both kernels' algorithmic work over the call's device time)
        lanes = 4 if (c.get_option(OPT_ZGROUP) and (S + 31) // 32 >= 1024) else c.get_option(OPT_LANES)
        top = {"kernel": "k_scan_fused + k_fine_ck (comet_scan_rss: sub-slabs on %d internal streams)" % lanes,
               "achieved": (fl[knames[0]] + fl[knames[1]]) / (ms_call * 1e-3) / 1e12, "ms_per_launch": ms_call,
               "achieved_executed": (fl_exec[knames[0]] + fl_exec[knames[1]]) / (ms_call * 1e-3) / 1e12,
               "timed": "CUDA events on the caller's stream around every comet_scan_rss of the timed region",
               "traffic": (sum((TRAFFIC_BYTES_ZG if uniq > 0 else TRAFFIC_BYTES).values())) if args.config == 1 else None}
    else:
        top = {"kernel": kernel, "achieved": kernels[kernel]["achieved"], "ms_per_launch": ktimes[kernel],
               "timed": kernels["timed_over"], "traffic": None}
    model = ("FP64-pipe slots x 2 of the work the path needs (thread-level counters, comet_read_stats): "
             + ("%d per recorded state (RKN4 step + target-region test, Alg. 1), " % GEN_INSTR if fused else "")
             + "%d per shortlist evaluation (sub-block sample or swept row); %s: %d per (seed, wire) pair that runs "
               "the virtual-plane iteration" % (SHORTLIST_INSTR, knames[1], FINE_INSTR)
             + ("; `achieved` counts the RKN4 step once per (seed, recorded state) -- SURVEY 8(d)'s unit -- although with "
                "COMET_OPT_ZGROUP the library executes it once per distinct transverse track (%.0f of %.0f states) plus one "
                "z addition per (seed, state): `achieved_executed` counts what is executed" % (uniq, n_states) if uniq > 0 else ""))
    flops_exh = 2.0 * (SHORTLIST_INSTR * n_states * W + FINE_INSTR * pairs)
    if fused:
        # k_wire_prep, then k_scan_fused + k_fine_ck + k_rss_sum per sub-slab (the library's rule: up to
        # COMET_OPT_LANES sub-slabs of at least 2 CTAs of 4 chunks per SM), then k_wire_prep, k_argmin_stage1, k_select_classify
        chunks = (S + 31) // 32
        zg_on = bool(c.get_option(OPT_ZGROUP)) and chunks >= 1024        # the library's size threshold for the z-run kernels
        n_sub = 4 if zg_on else c.get_option(OPT_LANES)
        n_sm = torch.cuda.get_device_properties(local).multi_processor_count
        while n_sub > 1 and chunks // n_sub < 4 * n_sm * 2:
            n_sub -= 1
        # per sub-slab: k_scan_fused, k_fine_ck, k_rss_sum; with COMET_OPT_ZGROUP also k_zgroup_check, k_gen_unique and the ZG
        # variants of the first two (the variants that do not serve the launch exit at once)
        launches_per_step = 1 + (7 if zg_on else 3) * n_sub + 3
    else:
        launches_per_step = 8
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": _workload_name(args.config, ev, seeds, part_off),
                   "path": ("fused: comet_scan_rss (track on chip) + comet_select_and_classify" if fused else
                            "materialised: comet_seed_extrapolate + comet_dca_rss + comet_select_and_classify"),
                   "l2": (("working set larger than L2 (126 MB): every step rewrites %.2f GB of distinct-track rows, %.2f GB of z "
                           "checkpoints and %.2f GB of (seed, wire) pair keys and rereads them"
                           % (uniq * 32 / 1e9, n_states * 2 / 1e9, pairs * 8 / 1e9)) if uniq > 0 else
                          ("working set larger than L2 (126 MB): every step rewrites %.1f GB of checkpoints and %.2f GB of "
                           "(seed, wire) pair keys and rereads them" % (n_states * 12 / 1e9, pairs * 8 / 1e9))) if fused else
                         ("inputs larger than L2 (126 MB): every step rewrites the recorded part of the track buffer "
                          "(%.1f GB) and kernel B rereads it" % (n_states * 48 / 1e9)),
                   "parallelism": "one replica of the event per GPU (event-level sharding, no collective)"},
        "events_per_s": world / (ms_per_step * 1e-3),
        "result": {"best_seed": best, "classified_entries": n_cls, "recorded_states_per_seed": n_states / S},
        "e2e": {"value": world * pairs / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_s * 1e3,
                "api": "comet_scan_event_host, pinned host buffers" + ("" if fused else ", %d GiB track slab" % (budget >> 30))},
        "gpu_launches": launches_per_step * args.steps,
        "clocks": clocks,
        "stage": stage,
        "field": field,
        "seeding": seeding,
        "batch": batch,
        "roofline": {"kernel": top["kernel"], "bound": "alu", "achieved": top["achieved"], "peak": peak,
                     "unit": "TFLOP/s", "frac": top["achieved"] / peak, "traffic": top["traffic"],
                     "timed": top["timed"],
                     "peak_source": "derived: 148 SMs x 64 FP64 FMA lanes x 2 x 1.965 GHz (MEASURED_PEAKS.json has no FP64 figure)",
                     "peak_measured_dfma_probe": peak_measured,
                     "frac_of_measured": top["achieved"] / peak_measured,
                     "achieved_executed": top.get("achieved_executed"),
                     "frac_executed": (top["achieved_executed"] / peak) if top.get("achieved_executed") else None,
                     "ms_per_launch": top["ms_per_launch"], "share_of_step": top["ms_per_launch"] / ms_per_step,
                     "model": model, "kernels": kernels, "work_counters": stats,
                     "other_path": {"path": "materialised" if fused else "fused", "ms_per_step": ms_other,
                                    "rss_bit_identical": paths_agree},
                     "exhaustive_search": None if ms_exh is None else
                                          {"kernel": "k_dca_rss", "ms_per_launch": ms_exh, "rss_bit_identical": exh_agree,
                                           "achieved": flops_exh / (ms_exh * 1e-3) / 1e12,
                                           "frac": flops_exh / (ms_exh * 1e-3) / 1e12 / peak,
                                           "model": "%d per (seed, wire, recorded state) + %d per (seed, wire)"
                                                    % (SHORTLIST_INSTR, FINE_INSTR)}},
    }
    if args.cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(ev, seeds, part_off)
    print(json.dumps(line))
    c.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--path", choices=["fused", "materialised"], default="fused")
    ap.add_argument("--no-cpu-baseline", dest="cpu_baseline", action="store_false")
    ap.add_argument("--no-field", dest="field", action="store_false", help="skip the field-map leg")
    ap.add_argument("--batch", type=int, default=16, help="events of configs[2] in the batch leg (0 = skip)")
    ap.add_argument("--no-zgroup", dest="zgroup", action="store_false",
                    help="COMET_OPT_ZGROUP = 0: every seed runs its own RKN4 steps even where runs of seeds differ only in z")
    ap.add_argument("--no-seeding", dest="seeding", action="store_false", help="skip the Hough / half-track legs")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
