"""ctypes wrapper around oracle/comet_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference legs may import this.  It never imports paper_1911_09340_b200.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "comet_oracle.c")
_LIB = os.path.join(_HERE, "libcomet_oracle.so")
_lib = None

_F64 = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_I32 = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_I64 = np.ctypeslib.ndpointer(dtype=np.int64, flags="C_CONTIGUOUS")
_U8 = np.ctypeslib.ndpointer(dtype=np.uint8, flags="C_CONTIGUOUS")


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off -fopenmp: one IEEE double operation per written operation."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC",
               "-Wall", "-Wextra", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        c_int, c_i64, c_dbl, vp = ctypes.c_int, ctypes.c_int64, ctypes.c_double, ctypes.c_void_p
        L.oracle_max_threads.restype = c_int
        L.oracle_set_threads.argtypes = [c_int]
        L.oracle_kappa.restype = c_dbl
        L.oracle_rkn4_step.argtypes = [_F64, c_dbl, c_dbl]
        L.oracle_extrapolate.argtypes = [_F64, c_i64, c_int, c_dbl, c_dbl, c_int, c_dbl, _F64, _I32]
        L.oracle_scan.argtypes = [_F64, c_i64, c_int, c_dbl, c_dbl, c_int, c_dbl,
                                  _F64, _F64, c_int, _I32, _I32, _F64, c_int, c_dbl,
                                  _F64, vp, vp, vp]
        L.oracle_select_classify.argtypes = [_F64, c_i64, c_int, c_dbl, c_dbl, c_int, c_dbl,
                                             _F64, _F64, c_int, _I32, _I32, _F64, c_int, c_int, c_dbl,
                                             _F64, _I64, c_int, _I64, _F64, _F64, _U8]
        fld = [_F64, _I32, _F64, _F64]
        L.oracle_field_at.argtypes = fld + [_F64, _F64]
        L.oracle_rkn4_field_step.argtypes = fld + [_F64, c_dbl, c_dbl]
        L.oracle_rkn4_field_step.restype = c_dbl
        L.oracle_extrapolate_field.argtypes = [_F64, c_i64, c_int] + fld + [c_dbl, c_int, c_dbl, c_dbl, _F64, _I32, _F64]
        L.oracle_scan_field.argtypes = [_F64, c_i64, c_int] + fld + [c_dbl, c_int, c_dbl, c_dbl,
                                        _F64, _F64, c_int, _I32, _I32, _F64, c_int, c_dbl, _F64, vp, vp, vp]
        L.oracle_classify_seeds_field.argtypes = [_F64, c_i64, c_int] + fld + [c_dbl, c_int, c_dbl, c_dbl,
                                                  _F64, _F64, c_int, _I32, _I32, _F64, c_int, c_int, c_dbl,
                                                  _I64, c_int, _F64, _U8]
        L.oracle_select_references.argtypes = [_F64, c_i64, _F64, _I64, c_int, _F64, c_int, _I64]
        L.oracle_refine_seeds.argtypes = [_F64, c_i64, _I64, c_int, c_int, _F64, _I32, _F64]
        _lib = L
    return _lib


def max_threads() -> int:
    return int(lib().oracle_max_threads())


def set_threads(n: int) -> None:
    lib().oracle_set_threads(int(n))


def kappa() -> float:
    return float(lib().oracle_kappa())


def rkn4_step(state6, h: float, c: float) -> np.ndarray:
    s = np.ascontiguousarray(state6, dtype=np.float64).copy()
    lib().oracle_rkn4_step(s, float(h), float(c))
    return s


def _c(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


def extrapolate(seeds, charge, bz, step, n_steps, r_stop):
    """Algorithm 1.  seeds [6][S] -> (track [S][n_steps+1][6], n_pts [S])."""
    seeds = _c(seeds, np.float64)
    S = seeds.shape[1]
    track = np.empty((S, n_steps + 1, 6))
    n_pts = np.empty(S, dtype=np.int32)
    lib().oracle_extrapolate(seeds, S, int(charge), float(bz), float(step), int(n_steps),
                             float(r_stop), track, n_pts)
    return track, n_pts


def scan(seeds, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire, hit_off, rho,
         cutoff, want_dca=False, want_kstar=False, want_npts=False):
    """Algorithm 3 over all seeds -> dict(rss[, dca, kstar, n_pts])."""
    seeds = _c(seeds, np.float64)
    wire_a, wire_b = _c(wire_a, np.float64), _c(wire_b, np.float64)
    fired_wire, hit_off, rho = _c(fired_wire, np.int32), _c(hit_off, np.int32), _c(rho, np.float64)
    S, W = seeds.shape[1], fired_wire.shape[0]
    out = {"rss": np.empty(S)}
    dca = np.empty((S, W)) if want_dca else None
    ks = np.empty((S, W), dtype=np.int32) if want_kstar else None
    npt = np.empty(S, dtype=np.int32) if want_npts else None
    ptr = lambda a: a.ctypes.data_as(ctypes.c_void_p) if a is not None else None
    lib().oracle_scan(seeds, S, int(charge), float(bz), float(step), int(n_steps), float(r_stop),
                      wire_a, wire_b, wire_a.shape[1], fired_wire, hit_off, rho, W, float(cutoff),
                      out["rss"], ptr(dca), ptr(ks), ptr(npt))
    if want_dca:
        out["dca"] = dca
    if want_kstar:
        out["kstar"] = ks
    if want_npts:
        out["n_pts"] = npt
    return out


def select_classify(seeds, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire, hit_off,
                    rho, cutoff, rss, part_off):
    """O10 + O11 -> dict(best_seed [P], best_rss [P], best_dca [P][W], cls [P][H])."""
    seeds = _c(seeds, np.float64)
    wire_a, wire_b = _c(wire_a, np.float64), _c(wire_b, np.float64)
    fired_wire, hit_off, rho = _c(fired_wire, np.int32), _c(hit_off, np.int32), _c(rho, np.float64)
    rss, part_off = _c(rss, np.float64), _c(part_off, np.int64)
    S, W, H, P = seeds.shape[1], fired_wire.shape[0], rho.shape[0], part_off.shape[0] - 1
    best_seed = np.empty(P, dtype=np.int64)
    best_rss = np.empty(P)
    best_dca = np.empty((P, W))
    cls = np.zeros((P, H), dtype=np.uint8)
    lib().oracle_select_classify(seeds, S, int(charge), float(bz), float(step), int(n_steps),
                                 float(r_stop), wire_a, wire_b, wire_a.shape[1], fired_wire, hit_off,
                                 rho, W, H, float(cutoff), rss, part_off, P,
                                 best_seed, best_rss, best_dca, cls)
    return {"best_seed": best_seed, "best_rss": best_rss, "best_dca": best_dca, "cls": cls}


def select_references(seeds, rss, part_off, half_width, k_ref):
    """O12: sparse lowest-RSS reference points -> int64 [P][k_ref], -1 = none."""
    seeds, rss, part_off = _c(seeds, np.float64), _c(rss, np.float64), _c(part_off, np.int64)
    hw = _c(half_width, np.float64)
    P = part_off.shape[0] - 1
    ref = np.empty((P, int(k_ref)), dtype=np.int64)
    lib().oracle_select_references(seeds, seeds.shape[1], rss, part_off, P, hw, int(k_ref), ref)
    return ref


def refine_seeds(seeds, ref_seed, half_width, n_grid):
    """O13: the finer seed set around every reference -> (seeds [6][P k G], part_off)."""
    seeds, ref_seed = _c(seeds, np.float64), _c(ref_seed, np.int64)
    hw, ng = _c(half_width, np.float64), _c(n_grid, np.int32)
    P, K = ref_seed.shape
    G = int(np.prod(ng.astype(np.int64)))
    new = np.empty((6, P * K * G))
    lib().oracle_refine_seeds(seeds, seeds.shape[1], ref_seed, P, K, hw, ng, new)
    return new, np.arange(P + 1, dtype=np.int64) * (K * G)


def classify_seeds(seeds, idx, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire, hit_off, rho,
                   cutoff):
    """O11 for the listed seeds -> dict(dca [n][W], cls [n][H]); idx < 0 -> NaN / zeros.
    Each listed seed is scored as a partition of its own by select_classify."""
    seeds = _c(seeds, np.float64)
    idx = np.asarray(idx, dtype=np.int64).ravel()
    W, H = len(fired_wire), len(rho)
    dca = np.full((idx.size, W), np.nan)
    cls = np.zeros((idx.size, H), dtype=np.uint8)
    ok = np.flatnonzero(idx >= 0)
    if ok.size:
        sub = np.ascontiguousarray(seeds[:, idx[ok]])
        r = select_classify(sub, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire, hit_off, rho,
                            cutoff, np.zeros(ok.size), np.arange(ok.size + 1, dtype=np.int64))
        dca[ok], cls[ok] = r["best_dca"], r["cls"]
    return {"dca": dca, "cls": cls}


def scan_stage(seeds, part_off, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire, hit_off, rho,
               cutoff, half_width, n_grid, n_iter, shrink, k_ref, k_final, field=None, rkn_tol=None):
    """One *stage* (the seed scanning of a turn, several *iterations*), every turn
    partition at once (R14).  Iteration 0 scans the given seeds; each of the n_iter further iterations
    picks k_ref sparse reference points (box half_width), scans the finer sets around them, and
    multiplies half_width by `shrink`.  The k_final finally selected seeds ("finally
    selected 10 seeds") are picked by the same rule with the last half_width and classified.
    -> dict(final_seed [P][k_final][6] (NaN = none), final_rss, final_dca, cls, history)."""
    seeds = _c(seeds, np.float64)
    part_off = _c(part_off, np.int64)
    hw = np.array(half_width, dtype=np.float64)
    args = (charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire, hit_off, rho, cutoff)
    if field is not None:        # the same stage in a field map (R29-R32): bz is not used
        fargs = (charge, field, step, n_steps, r_stop, rkn_tol, wire_a, wire_b, fired_wire, hit_off, rho, cutoff)
        scan_ = lambda sd: scan_field(sd, *fargs)
        classify_ = lambda sd, idx: classify_seeds_field(sd, idx, *fargs)
    else:
        scan_ = lambda sd: scan(sd, *args)
        classify_ = lambda sd, idx: classify_seeds(sd, idx, *args)
    history = []
    rss = scan_(seeds)["rss"]
    for _ in range(int(n_iter)):
        ref = select_references(seeds, rss, part_off, hw, k_ref)
        history.append({"ref_rss": np.where(ref >= 0, rss[np.maximum(ref, 0)], np.nan), "half_width": hw.copy()})
        seeds, part_off = refine_seeds(seeds, ref, hw, n_grid)
        rss = scan_(seeds)["rss"]
        hw = hw * float(shrink)
    fin = select_references(seeds, rss, part_off, hw, k_final)
    P = fin.shape[0]
    final_seed = np.full((P, int(k_final), 6), np.nan)
    ok = fin >= 0
    final_seed[ok] = seeds[:, fin[ok]].T
    final_rss = np.where(ok, rss[np.maximum(fin, 0)], np.nan)
    c = classify_(seeds, fin)
    W, H = len(fired_wire), len(rho)
    return {"final_seed": final_seed, "final_rss": final_rss, "final_dca": c["dca"].reshape(P, int(k_final), W),
            "cls": c["cls"].reshape(P, int(k_final), H), "history": history}


# ---- inhomogeneous field map + adaptive step (readings R29-R32) -------------------
def _fld(field):
    """field = (B [nx][ny][nz][3], origin [3], spacing [3]) -> ctypes arguments."""
    B, o, d = field
    B = _c(B, np.float64)
    return B, np.array(B.shape[:3], dtype=np.int32), _c(o, np.float64), _c(d, np.float64)


def field_at(field, x):
    out = np.empty(3)
    lib().oracle_field_at(*_fld(field), _c(x, np.float64), out)
    return out


def rkn4_field_step(field, state6, h, cq):
    """One Nystrom RK4 step in the field map -> (new state, EST)."""
    s = np.array(state6, dtype=np.float64)
    est = lib().oracle_rkn4_field_step(*_fld(field), s, float(h), float(cq))
    return s, float(est)


def extrapolate_field(seeds, charge, field, h_max, n_steps, r_stop, tol):
    seeds = _c(seeds, np.float64)
    S = seeds.shape[1]
    track = np.empty((S, n_steps + 1, 6))
    n_pts = np.empty(S, dtype=np.int32)
    hs = np.empty((S, n_steps))
    lib().oracle_extrapolate_field(seeds, S, int(charge), *_fld(field), float(h_max), int(n_steps), float(r_stop),
                                   float(tol), track, n_pts, hs)
    return track, n_pts, hs


def scan_field(seeds, charge, field, h_max, n_steps, r_stop, tol, wire_a, wire_b, fired_wire, hit_off, rho,
               cutoff, want_dca=False, want_kstar=False, want_npts=False):
    seeds = _c(seeds, np.float64)
    wire_a, wire_b = _c(wire_a, np.float64), _c(wire_b, np.float64)
    fired_wire, hit_off, rho = _c(fired_wire, np.int32), _c(hit_off, np.int32), _c(rho, np.float64)
    S, W = seeds.shape[1], fired_wire.shape[0]
    out = {"rss": np.empty(S)}
    dca = np.empty((S, W)) if want_dca else None
    ks = np.empty((S, W), dtype=np.int32) if want_kstar else None
    npt = np.empty(S, dtype=np.int32) if want_npts else None
    ptr = lambda a: a.ctypes.data_as(ctypes.c_void_p) if a is not None else None
    lib().oracle_scan_field(seeds, S, int(charge), *_fld(field), float(h_max), int(n_steps), float(r_stop), float(tol),
                            wire_a, wire_b, wire_a.shape[1], fired_wire, hit_off, rho, W, float(cutoff),
                            out["rss"], ptr(dca), ptr(ks), ptr(npt))
    if want_dca:
        out["dca"] = dca
    if want_kstar:
        out["kstar"] = ks
    if want_npts:
        out["n_pts"] = npt
    return out


def classify_seeds_field(seeds, idx, charge, field, h_max, n_steps, r_stop, tol, wire_a, wire_b, fired_wire,
                         hit_off, rho, cutoff):
    seeds = _c(seeds, np.float64)
    wire_a, wire_b = _c(wire_a, np.float64), _c(wire_b, np.float64)
    fired_wire, hit_off, rho = _c(fired_wire, np.int32), _c(hit_off, np.int32), _c(rho, np.float64)
    idx = _c(np.asarray(idx, dtype=np.int64).ravel(), np.int64)
    W, H = fired_wire.shape[0], rho.shape[0]
    dca = np.empty((idx.size, W))
    cls = np.zeros((idx.size, H), dtype=np.uint8)
    lib().oracle_classify_seeds_field(seeds, seeds.shape[1], int(charge), *_fld(field), float(h_max), int(n_steps),
                                      float(r_stop), float(tol), wire_a, wire_b, wire_a.shape[1], fired_wire,
                                      hit_off, rho, W, H, float(cutoff), idx, idx.size, dca, cls)
    return {"dca": dca, "cls": cls}


# ---- sequential stages with hit removal (readings R33-R34) ---------------------------
def remove_hits(fired_wire, hit_off, rho, cls):
    """"The hits classified previously were excluded in the seed scanning; therefore, the number of wires
    gets reduced whenever a track is fitted".  A measured hit is the adjacent pair of ghost
    entries (2m, 2m+1) (R12, R33): an entry goes when it or its partner is classified; a wire left without
    entries goes too.  -> (fired_wire, hit_off, rho, src) with src[j'] = old index of kept entry j'."""
    fired_wire, hit_off, rho = np.asarray(fired_wire), np.asarray(hit_off), np.asarray(rho)
    cls = np.asarray(cls).astype(bool)
    H = rho.shape[0]
    assert H % 2 == 0 and np.all(hit_off % 2 == 0)
    new_fw, new_off, new_rho, src = [], [0], [], []
    for i in range(fired_wire.shape[0]):                 # plain loops: wire by wire, entry by entry
        kept = []
        for j in range(hit_off[i], hit_off[i + 1]):
            if not (cls[j] or cls[j ^ 1]):
                kept.append(j)
        if kept:
            new_fw.append(fired_wire[i])
            new_rho.extend(rho[j] for j in kept)
            src.extend(kept)
            new_off.append(new_off[-1] + len(kept))
    return (np.array(new_fw, dtype=np.int32), np.array(new_off, dtype=np.int32),
            np.array(new_rho, dtype=np.float64), np.array(src, dtype=np.int32))


def scan_turns(seeds, part_off, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire, hit_off, rho,
               cutoff, half_width, n_grid, n_iter, shrink, k_ref, min_wires=30, max_tracks=5):
    """The stage loop of PAPER.md:256 without the fit: the last turn partition first; each stage scans its
    partition's seeds against the hits that are left (scan_stage with one finally selected seed), classifies
    the hits of its best seed, removes them (remove_hits) and moves to the previous turn; it stops when fewer
    than min_wires fired wires are left or max_tracks stages are done (R34).
    -> dict(turn_seed [P][6], turn_rss [P], turn_cls [P][H] in the ORIGINAL entry numbering, done [P] bool,
            wires_before [P])."""
    seeds = _c(seeds, np.float64)
    part_off = np.asarray(part_off, dtype=np.int64)
    P, H = part_off.shape[0] - 1, len(rho)
    fw, ho, rh = np.asarray(fired_wire, np.int32), np.asarray(hit_off, np.int32), np.asarray(rho, np.float64)
    orig = np.arange(H, dtype=np.int32)
    out = {"turn_seed": np.full((P, 6), np.nan), "turn_rss": np.full(P, np.nan),
           "turn_cls": np.zeros((P, H), dtype=np.uint8), "done": np.zeros(P, dtype=bool),
           "wires_before": np.zeros(P, dtype=np.int32)}
    n_done = 0
    for p in range(P - 1, -1, -1):
        if fw.shape[0] < min_wires or n_done >= max_tracks:
            break
        sub = np.ascontiguousarray(seeds[:, part_off[p]:part_off[p + 1]])
        st = scan_stage(sub, np.array([0, sub.shape[1]], dtype=np.int64), charge, bz, step, n_steps, r_stop,
                        wire_a, wire_b, fw, ho, rh, cutoff, half_width, n_grid, n_iter, shrink, k_ref, 1)
        out["turn_seed"][p], out["turn_rss"][p] = st["final_seed"][0, 0], st["final_rss"][0, 0]
        out["wires_before"][p], out["done"][p] = fw.shape[0], True
        cls = st["cls"][0, 0]
        out["turn_cls"][p, orig[cls.astype(bool)]] = 1
        fw, ho, rh, src = remove_hits(fw, ho, rh, cls)
        orig = orig[src]
        n_done += 1
    return out


# ---- Hough-transform transverse seeding (Fig. 10; readings R35-R37) -----------------
def hough_seeds(wire_a, wire_b, fired_wire, cos_tab, sin_tab, rho_min, inv_drho, n_rho, charge, bz, r_seed):
    """"The transverse components (theta, p_x, p_y) were extracted by finding a circle that is the transverse
    projection of a helical trajectory [...] the Hough transform was applied to the set of transverse positions
    of the fired wires".  R35: a wire's transverse position is the (x, y) of its midpoint.
    R36: the circle passes through the origin (the stopping target on the axis), so u = x/(x^2+y^2),
    v = y/(x^2+y^2) maps it to the line u cos(phi) + v sin(phi) = rho with rho = 1/(2R) and phi the azimuth of
    the circle's centre; every fired wire votes once per direction phi_j (tables given) in the bin
    floor((rho - rho_min) inv_drho) if that lies in [0, n_rho); the peak is the bin of most votes, ties -> the
    lowest j n_rho + k.  R37: R = 1/(2 rho*) with rho* the bin centre, centre R (cos, sin); the seed points are
    the two intersections with the cylinder r = r_seed, p_T = kappa |B_z| R along the tangent in the sense of
    rotation of the particle; the entrance is the one where the track moves outwards.
    -> dict(acc [n_phi][n_rho] int32, peak (votes, j, k), R, centre [2], entrance [4] (x, y, px, py), exit [4])."""
    wire_a, wire_b = np.asarray(wire_a, np.float64), np.asarray(wire_b, np.float64)
    cos_tab, sin_tab = np.asarray(cos_tab, np.float64), np.asarray(sin_tab, np.float64)
    n_phi = cos_tab.shape[0]
    acc = np.zeros((n_phi, int(n_rho)), dtype=np.int32)
    for wi in np.asarray(fired_wire):
        x = (wire_a[0, wi] + wire_b[0, wi]) / 2.0
        y = (wire_a[1, wi] + wire_b[1, wi]) / 2.0
        r2 = x * x + y * y
        u, v = x / r2, y / r2
        for j in range(n_phi):
            rho = u * cos_tab[j] + v * sin_tab[j]
            k = np.floor((rho - rho_min) * inv_drho)
            if 0.0 <= k < n_rho:
                acc[j, int(k)] += 1
    flat = acc.ravel()
    best = int(np.argmax(flat))                            # first maximum = lowest j n_rho + k
    j, k = divmod(best, int(n_rho))
    out = {"acc": acc, "peak": (int(flat[best]), j, k)}
    nan4 = np.full(4, np.nan)
    if flat[best] == 0:
        out.update(R=np.nan, centre=np.full(2, np.nan), entrance=nan4, exit=nan4.copy())
        return out
    rho_s = rho_min + (k + 0.5) / inv_drho
    R = 1.0 / (2.0 * rho_s)
    cx, cy = R * cos_tab[j], R * sin_tab[j]
    out.update(R=R, centre=np.array([cx, cy]))
    t = (r_seed * r_seed) / (2.0 * R)                      # component of the seed point along the centre direction
    n2 = r_seed * r_seed - t * t
    if not (n2 > 0.0):
        out.update(entrance=nan4, exit=nan4.copy())         # the circle does not reach the seed cylinder
        return out
    n = np.sqrt(n2)
    sense = -1.0 if (charge * bz) > 0.0 else 1.0            # +1: counter-clockwise (electron in B_z > 0)
    pT = KAPPA_ * abs(bz) * R
    pts = []
    for sgn in (1.0, -1.0):
        px_ = t * cos_tab[j] - sgn * n * sin_tab[j]
        py_ = t * sin_tab[j] + sgn * n * cos_tab[j]
        tx, ty = -(py_ - cy) / R, (px_ - cx) / R            # counter-clockwise tangent
        tx, ty = sense * tx, sense * ty
        pts.append((px_, py_, pT * tx, pT * ty, px_ * tx + py_ * ty))
    ent, ext = (pts[0], pts[1]) if pts[0][4] > 0.0 else (pts[1], pts[0])
    out.update(entrance=np.array(ent[:4]), exit=np.array(ext[:4]))
    return out


# ---- half tracks (readings R38-R42) --------------------------------------------
def flip_seeds(seeds):
    """"The track extrapolation was done in the forward direction from the entrance and the backward direction
    from the exit by flipping the charge and momentum".  R38: the backward seed of an exit-side
    seed (x, p) is (x, -p), extrapolated with the charge -q (the caller passes -charge).  The signed DCA of a
    wire is measured against the track's direction of travel, so on the way back it has the opposite sign:
    the backward scan is run against -rho (scan_half_tracks does that)."""
    out = np.array(seeds, dtype=np.float64, copy=True)
    out[3:6] = -out[3:6]
    return out


def half_hit_masks(wire_a, wire_b, fired_wire, hit_off, n_hits, circle, overlap):
    """"The hits of the event were also grouped into two sets for each half track".  R39: the
    two half tracks meet at the apex of the transverse circle found by the Hough transform (circle = R, centre
    x, y, entrance x, y, ...: hough_seeds' output), which lies on the line from the origin through the centre.
    With m the (x, y) of a wire's midpoint, d = (cx m_y - cy m_x) / R is its signed distance from that line and
    s = +1 if cx e_y - cy e_x > 0 else -1 the side of the entrance point e: the wire's entries belong to the
    entrance half iff s d > -overlap and to the exit half iff s d <= overlap.
    -> (in_ent [n_hits] uint8, in_exit [n_hits] uint8)."""
    wire_a, wire_b = np.asarray(wire_a, np.float64), np.asarray(wire_b, np.float64)
    circle = np.asarray(circle, np.float64)
    R, cx, cy, ex, ey = circle[0], circle[1], circle[2], circle[3], circle[4]
    s = 1.0 if (cx * ey - cy * ex) > 0.0 else -1.0
    in_e = np.zeros(int(n_hits), dtype=np.uint8)
    in_x = np.zeros(int(n_hits), dtype=np.uint8)
    for i, wi in enumerate(np.asarray(fired_wire)):
        mx = (wire_a[0, wi] + wire_b[0, wi]) / 2.0
        my = (wire_a[1, wi] + wire_b[1, wi]) / 2.0
        d = s * ((cx * my - cy * mx) / R)
        for j in range(hit_off[i], hit_off[i + 1]):
            in_e[j] = 1 if d > -overlap else 0
            in_x[j] = 1 if d <= overlap else 0
    return in_e, in_x


def layer_veto(cls, fired_wire, hit_off, wire_layer, min_layers):
    """"the seeds which have any missing layer without the hits were excluded".  R40: a half
    track starts in front of the first layer, so it crosses the layers 0 .. l_max, l_max the highest layer
    with a classified hit of this seed: the seed is kept iff every one of those layers has a classified hit
    and there are at least min_layers of them.  cls [K][H] -> ok [K] uint8."""
    cls = np.atleast_2d(np.asarray(cls)).astype(bool)
    wire_layer = np.asarray(wire_layer)
    ok = np.zeros(cls.shape[0], dtype=np.uint8)
    for a in range(cls.shape[0]):
        layers = set()
        for i, wi in enumerate(np.asarray(fired_wire)):
            for j in range(hit_off[i], hit_off[i + 1]):
                if cls[a, j]:
                    layers.add(int(wire_layer[wi]))
        if layers:
            l_max = max(layers)
            ok[a] = 1 if (all(l in layers for l in range(l_max + 1)) and l_max + 1 >= min_layers) else 0
    return ok


def merge_half_sets(cls_e, orig_e, ok_e, cls_x, orig_x, ok_x, n_hits):
    """"The complete sets of classified hits were formed by combinatorially merging two half sets, one of which
    is from each direction".  R41: pair (a, b) of an entrance-side seed a and an exit-side seed
    b is valid iff both passed the layer veto; its complete set is the union of the two half sets in the
    event's own entry numbering (orig_* map the entries of the half lists back).
    -> dict(valid [Ke][Kx] uint8, cls [Ke][Kx][n_hits] uint8 (zeros where not valid), n_cls [Ke][Kx] int32)."""
    cls_e, cls_x = np.atleast_2d(np.asarray(cls_e)), np.atleast_2d(np.asarray(cls_x))
    Ke, Kx = cls_e.shape[0], cls_x.shape[0]
    valid = np.zeros((Ke, Kx), dtype=np.uint8)
    cls = np.zeros((Ke, Kx, int(n_hits)), dtype=np.uint8)
    n_cls = np.zeros((Ke, Kx), dtype=np.int32)
    for a in range(Ke):
        for b in range(Kx):
            if not (ok_e[a] and ok_x[b]):
                continue
            valid[a, b] = 1
            for j in range(cls_e.shape[1]):
                if cls_e[a, j]:
                    cls[a, b, orig_e[j]] = 1
            for j in range(cls_x.shape[1]):
                if cls_x[b, j]:
                    cls[a, b, orig_x[j]] = 1
            n_cls[a, b] = int(cls[a, b].sum())
    return {"valid": valid, "cls": cls, "n_cls": n_cls}


def scan_half_tracks(seeds_e, seeds_x, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire, hit_off, rho,
                     cutoff, wire_layer, circle, overlap, min_layers, half_width, n_grid, n_iter, shrink, k_ref,
                     k_final):
    """One turn partition as two half tracks (R38-R42): the hits are grouped by
    half_hit_masks; the entrance-side seeds are scanned forwards against the entrance set, the exit-side
    seeds backwards (flip_seeds, -charge) against the exit set, each by scan_stage with k_final finally
    selected seeds (paper: 10 per side); seeds with a missing layer are vetoed; the half sets are merged
    combinatorially.  R42: a half track ends at the apex, the first recorded state that moves inwards --
    this is the target region of R3 with r_stop beyond the chamber (the caller passes e.g. 1e3 cm).
    The exit-side final seeds are returned in the physical (forward) convention.
    -> dict(ent / ext: dict(final_seed [K][6], final_rss [K], cls [K][H_half], ok [K], orig [H_half],
            fired_wire, hit_off), valid, cls, n_cls)."""
    H = len(rho)
    in_e, in_x = half_hit_masks(wire_a, wire_b, fired_wire, hit_off, H, circle, overlap)
    out = {}
    for key, keep, sd, q in (("ent", in_e, np.asarray(seeds_e, np.float64), charge),
                             ("ext", in_x, flip_seeds(seeds_x), -charge)):
        fw, ho, rh, src = remove_hits(fired_wire, hit_off, rho, 1 - keep)
        if key == "ext":
            rh = -rh            # R38: the reversed tangent swaps left and right, so the signed drift changes sign
        st = scan_stage(np.ascontiguousarray(sd), np.array([0, sd.shape[1]], dtype=np.int64), q, bz, step, n_steps,
                        r_stop, wire_a, wire_b, fw, ho, rh, cutoff, half_width, n_grid, n_iter, shrink, k_ref, k_final)
        fs = st["final_seed"][0]
        if key == "ext":
            fs = flip_seeds(fs.T).T
        cls = st["cls"][0]
        out[key] = {"final_seed": fs, "final_rss": st["final_rss"][0], "cls": cls, "orig": src, "fired_wire": fw,
                    "hit_off": ho, "ok": layer_veto(cls, fw, ho, wire_layer, min_layers)}
    m = merge_half_sets(out["ent"]["cls"], out["ent"]["orig"], out["ent"]["ok"],
                        out["ext"]["cls"], out["ext"]["orig"], out["ext"]["ok"], H)
    out.update(m)
    return out


def best_pair(valid, n_cls):
    """R43: the complete set that goes on -- the paper keeps the one whose fit has the highest NDF;
    without the fit, the valid pair with the most classified entries, ties -> the lowest a K_x + b; -1 = none."""
    valid, n_cls = np.asarray(valid), np.asarray(n_cls)
    best, arg = -1, -1
    for a in range(valid.shape[0]):
        for b in range(valid.shape[1]):
            if valid[a, b] and n_cls[a, b] > best:
                best, arg = int(n_cls[a, b]), a * valid.shape[1] + b
    return arg


def scan_turns_half(seeds_e, off_e, seeds_x, off_x, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire,
                    hit_off, rho, cutoff, wire_layer, circle, overlap, min_layers, half_width, n_grid, n_iter, shrink,
                    k_ref, k_final, min_wires=30, max_tracks=5):
    """The event loop of Fig. 13 with half tracks and without the fits: the last turn partition
    first; scan_half_tracks of the turn's entrance- and exit-side seed sets against the hits that are left; the
    complete set of best_pair (R43) is the turn's, its hits are removed (remove_hits) before the previous turn;
    the loop stops when fewer than min_wires fired wires are left, max_tracks turns are done (R34) or a turn has
    no valid pair (":244 If the fitting results were not converged for any of the complete sets, the event
    reconstruction process was stopped").  The transverse seed (the circle) is the same for every turn (:256).
    -> dict(turn_pair [P][2] (-1 = none), turn_n [P], turn_cls [P][H] in the event's own numbering,
            turn_seed [P][2][6] (entrance, exit), done [P], wires_before [P])."""
    seeds_e, seeds_x = _c(seeds_e, np.float64), _c(seeds_x, np.float64)
    off_e, off_x = np.asarray(off_e, np.int64), np.asarray(off_x, np.int64)
    P, H, K = off_e.shape[0] - 1, len(rho), int(k_final)
    fw, ho, rh = np.asarray(fired_wire, np.int32), np.asarray(hit_off, np.int32), np.asarray(rho, np.float64)
    orig = np.arange(H, dtype=np.int32)
    out = {"turn_pair": np.full((P, 2), -1, dtype=np.int32), "turn_n": np.zeros(P, dtype=np.int32),
           "turn_cls": np.zeros((P, H), dtype=np.uint8), "turn_seed": np.full((P, 2, 6), np.nan),
           "done": np.zeros(P, dtype=bool), "wires_before": np.zeros(P, dtype=np.int32)}
    n_done = 0
    for p in range(P - 1, -1, -1):
        if fw.shape[0] < min_wires or n_done >= max_tracks:
            break
        se = np.ascontiguousarray(seeds_e[:, off_e[p]:off_e[p + 1]])
        sx = np.ascontiguousarray(seeds_x[:, off_x[p]:off_x[p + 1]])
        ht = scan_half_tracks(se, sx, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fw, ho, rh, cutoff, wire_layer,
                              circle, overlap, min_layers, half_width, n_grid, n_iter, shrink, k_ref, k_final)
        out["wires_before"][p] = fw.shape[0]
        arg = best_pair(ht["valid"], ht["n_cls"])
        if arg < 0:
            break
        a, b = divmod(arg, K)
        cls = ht["cls"][a, b]
        out["turn_pair"][p], out["turn_n"][p], out["done"][p] = (a, b), ht["n_cls"][a, b], True
        out["turn_seed"][p, 0], out["turn_seed"][p, 1] = ht["ent"]["final_seed"][a], ht["ext"]["final_seed"][b]
        out["turn_cls"][p, orig[cls.astype(bool)]] = 1
        fw, ho, rh, src = remove_hits(fw, ho, rh, cls)
        orig = orig[src]
        n_done += 1
    return out


KAPPA_ = 2.99792458     # R4
