"""Truth events, hits with left/right ghosts and seed grids for BASELINE.json's configs.

Recipe (stated in DESIGN.md "Input recipe"; stands in for the paper's Geant4
samples, which are not available):

* truth = one closed-form helix (no scattering, no energy loss) from a vertex
  with r < 10 cm;
* a *turn partition* is the arc between an outward and the next inward crossing
  of r = 50 cm (the paper's seed radius) that lies inside
  |z| < 75 cm;
* every wire whose true distance of closest approach to a partition's arc is
  below 0.8 cm gets one hit with drift r = max(0, DCA + N(0, sigma)); each hit
  is stored as two entries, rho = +r and rho = -r (PAPER.md:37 ghosts);
* the paper's preselection (>= 5 layers, < 250 fired wires) is
  applied and the event redrawn from the same RNG stream until it passes;
* seeds: Cartesian grid over (|p|, cos theta, phi0, z0) at the entrance point
  (50 cos theta_e, 50 sin theta_e, z0), index ((ip*n_ct+ict)*n_phi+iphi)*n_z+iz.
"""
from dataclasses import dataclass, field
from typing import List, Optional, Sequence, Tuple

import numpy as np

from .geometry import CDCGeometry, cdc_geometry
from .helix import Helix

R_SEED = 50.0          # cm
HIT_DCA_MAX = 0.8      # cm, BASELINE.json configs[0]
SIGMA_DRIFT = 0.02     # cm, BASELINE.json configs[0]


@dataclass
class Partition:
    index: int
    s_in: float
    s_out: float
    x_in: np.ndarray        # [3] truth position at the outward r = 50 crossing
    T_in: np.ndarray        # [3] truth unit tangent there
    theta_e: float          # azimuth of x_in
    phi: float              # azimuth of T_in
    cos_theta: float        # T_z
    z: float                # x_in[2]


@dataclass
class Event:
    geom: CDCGeometry
    bz: float
    charge: int
    pmag: float
    vertex: np.ndarray
    p0: np.ndarray
    partitions: List[Partition]
    fired_wire: np.ndarray      # int32 [n_fired], strictly increasing
    hit_off: np.ndarray         # int32 [n_fired+1]
    rho: np.ndarray             # float64 [n_hits], signed drift (+r / -r)
    hit_turn: np.ndarray        # int32 [n_hits], truth partition, -1 = noise
    hit_real: np.ndarray        # uint8 [n_hits], 1 = the entry on the true side
    hit_true_dca: np.ndarray    # float64 [n_hits], signed truth DCA (NaN for noise)
    step: float
    n_steps: int
    cutoff: float
    r_stop: float = R_SEED
    n_trials: int = 1
    layers_hit: int = 0
    spec: dict = field(default_factory=dict)

    @property
    def n_fired(self) -> int:
        return int(self.fired_wire.shape[0])

    @property
    def n_hits(self) -> int:
        return int(self.rho.shape[0])

    def helix(self) -> Helix:
        return Helix(self.vertex, self.p0, self.charge, self.bz)


# ----------------------------------------------------------------------------
# truth helix -> partitions
# ----------------------------------------------------------------------------
def _find_partitions(h: Helix, half_len: float, max_parts: int = 8) -> Tuple[List[Partition], bool]:
    """Consecutive passages through r > R_SEED that lie fully inside |z| < half_len.

    Returns (partitions, first_inside): scanning starts at the vertex and stops
    at the first passage that is not fully inside.
    """
    from scipy.optimize import brentq

    tz = h.T0[2]
    if tz <= 0:
        return [], False
    s_max = (half_len + 10.0 - h.x0[2]) / tz
    s_max = min(s_max, 2.0 * np.pi / abs(h.c) * (max_parts + 2))
    ds = 0.05
    s = np.arange(0.0, s_max + ds, ds)
    pos = h.position(s)
    f = np.hypot(pos[:, 0], pos[:, 1]) - R_SEED

    def g(t):
        q = h.position(np.asarray(t))
        return float(np.hypot(q[0], q[1]) - R_SEED)

    sign = f > 0
    idx = np.nonzero(sign[1:] != sign[:-1])[0]
    crossings = [(brentq(g, s[i], s[i + 1], xtol=1e-13, rtol=1e-15), bool(sign[i + 1])) for i in idx]
    parts: List[Partition] = []
    k = 0
    # pair (outward, inward)
    while k + 1 < len(crossings) and len(parts) < max_parts:
        (s_in, out0), (s_out, out1) = crossings[k], crossings[k + 1]
        if not out0:       # starts with an inward crossing (vertex outside r=50 cannot happen, r<10)
            k += 1
            continue
        assert not out1
        x_in = h.position(np.asarray(s_in))
        x_out = h.position(np.asarray(s_out))
        if not (abs(x_in[2]) < half_len and abs(x_out[2]) < half_len):
            break
        T_in = h.tangent(np.asarray(s_in))
        parts.append(Partition(
            index=len(parts), s_in=float(s_in), s_out=float(s_out),
            x_in=x_in, T_in=T_in,
            theta_e=float(np.arctan2(x_in[1], x_in[0])),
            phi=float(np.arctan2(T_in[1], T_in[0])),
            cos_theta=float(T_in[2]), z=float(x_in[2])))
        k += 2
    # was there a further passage that is (partly) inside the chamber length?
    more_inside = False
    if k + 1 < len(crossings):
        x_in = h.position(np.asarray(crossings[k][0]))
        more_inside = abs(x_in[2]) < half_len
    return parts, more_inside


# ----------------------------------------------------------------------------
# truth DCA of every wire to one partition's arc
# ----------------------------------------------------------------------------
def _wire_lines(geom: CDCGeometry):
    a = geom.wire_a.T
    b = geom.wire_b.T
    d = b - a
    w = d / np.linalg.norm(d, axis=1, keepdims=True)
    m = 0.5 * (a + b)
    return m, w


def _perp(delta, w):
    return delta - np.sum(delta * w, axis=-1, keepdims=True) * w


def _true_dca(h: Helix, part: Partition, m: np.ndarray, w: np.ndarray, dca_max: float):
    """Signed truth DCA of wires that come within dca_max of the partition arc.

    Returns (wire_idx, signed_dca).  1-D minimisation on the closed-form helix:
    coarse sampling every 0.2 cm, then Newton on d/ds |u|^2/2 = u . T.
    """
    ds = 0.2
    n = max(2, int(np.ceil((part.s_out - part.s_in) / ds)) + 1)
    s = np.linspace(part.s_in, part.s_out, n)
    pos = h.position(s)                                   # [n,3]
    best = np.full(m.shape[0], np.inf)
    best_s = np.zeros(m.shape[0])
    for i0 in range(0, n, 64):
        P = pos[i0:i0 + 64]
        u = _perp(P[:, None, :] - m[None, :, :], w[None, :, :])
        d2 = np.sum(u * u, axis=-1)                       # [chunk, n_wires]
        j = np.argmin(d2, axis=0)
        v = d2[j, np.arange(m.shape[0])]
        upd = v < best
        best[upd] = v[upd]
        best_s[upd] = s[i0 + j[upd]]
    cand = np.nonzero(best < (dca_max + 0.25) ** 2)[0]
    if cand.size == 0:
        return cand, np.zeros(0)
    sc = best_s[cand]
    mc, wc = m[cand], w[cand]
    for _ in range(12):
        X = h.position(sc)
        T = h.tangent(sc)
        u = _perp(X - mc, wc)
        dT = h.c * np.stack([T[:, 1], -T[:, 0], np.zeros_like(sc)], axis=-1)
        Tp = _perp(T, wc)
        g = np.sum(u * T, axis=-1)
        gp = np.sum(Tp * Tp, axis=-1) + np.sum(u * dT, axis=-1)
        sc = np.clip(sc - g / gp, part.s_in, part.s_out)
    X = h.position(sc)
    T = h.tangent(sc)
    u = _perp(X - mc, wc)
    dist = np.linalg.norm(u, axis=-1)
    side = np.sum(u * np.cross(T, wc), axis=-1)
    signed = np.where(side >= 0, dist, -dist)
    keep = dist < dca_max
    return cand[keep], signed[keep]


# ----------------------------------------------------------------------------
# one event
# ----------------------------------------------------------------------------
def make_event(rng: np.random.Generator, *, pmag, cos_theta: Tuple[float, float],
               vertex_z: Tuple[float, float], n_turns, step: float, n_steps: int,
               cutoff: float, bz: float = 1.0, charge: int = -1,
               vertex_r: float = 10.0, n_noise: int = 0,
               geom: Optional[CDCGeometry] = None, max_trials: int = 100000,
               spec: Optional[dict] = None) -> Event:
    """Draw truth electrons until one passes the acceptance + preselection.

    pmag: float or (lo, hi) for a uniform draw.  n_turns: int (exactly that many
    partitions fully inside, the next one not) or (lo, hi) (any count in range).
    """
    geom = geom or cdc_geometry()
    m, w = _wire_lines(geom)
    for trial in range(1, max_trials + 1):
        p = float(rng.uniform(*pmag)) if isinstance(pmag, (tuple, list)) else float(pmag)
        ct = float(rng.uniform(*cos_theta))
        phi = float(rng.uniform(0.0, 2.0 * np.pi))
        rv = vertex_r * np.sqrt(rng.uniform())
        av = rng.uniform(0.0, 2.0 * np.pi)
        zv = float(rng.uniform(*vertex_z))
        vertex = np.array([rv * np.cos(av), rv * np.sin(av), zv])
        st = np.sqrt(1.0 - ct * ct)
        p0 = p * np.array([st * np.cos(phi), st * np.sin(phi), ct])
        h = Helix(vertex, p0, charge, bz)
        parts, more = _find_partitions(h, geom.half_len)
        if isinstance(n_turns, (tuple, list)):
            if not (n_turns[0] <= len(parts) <= n_turns[1]):
                continue
        elif n_turns == 1:
            # single passage wanted: the first passage is the event (BASELINE configs[0])
            if len(parts) < 1:
                continue
            parts = parts[:1]
        else:
            if len(parts) != n_turns or more:
                continue
        wires, dcas, turns = [], [], []
        for part in parts:
            wi, sd = _true_dca(h, part, m, w, HIT_DCA_MAX)
            wires.append(wi)
            dcas.append(sd)
            turns.append(np.full(wi.shape, part.index, dtype=np.int32))
        wires = np.concatenate(wires)
        dcas = np.concatenate(dcas)
        turns = np.concatenate(turns)
        layers_hit = np.unique(geom.layer[wires]).size if wires.size else 0
        n_fired_real = np.unique(wires).size
        if layers_hit < 5 or n_fired_real >= 250:
            continue
        # drift radii (smearing drawn only for accepted events would change the
        # stream with acceptance; draw here, after the cuts, in wire order)
        order = np.lexsort((turns, wires))
        wires, dcas, turns = wires[order], dcas[order], turns[order]
        r = np.maximum(0.0, np.abs(dcas) + rng.normal(0.0, SIGMA_DRIFT, size=dcas.shape))
        if n_noise:
            nw = rng.integers(0, geom.n_wires, size=n_noise)
            nr = rng.uniform(0.0, HIT_DCA_MAX, size=n_noise)
            wires = np.concatenate([wires, nw])
            r = np.concatenate([r, nr])
            dcas = np.concatenate([dcas, np.full(n_noise, np.nan)])
            turns = np.concatenate([turns, np.full(n_noise, -1, dtype=np.int32)])
            order = np.argsort(wires, kind="stable")
            wires, r, dcas, turns = wires[order], r[order], dcas[order], turns[order]
        fired, counts = np.unique(wires, return_counts=True)
        hit_off = np.zeros(fired.size + 1, dtype=np.int32)
        hit_off[1:] = 2 * np.cumsum(counts)
        rho = np.empty(2 * r.size)
        rho[0::2] = r
        rho[1::2] = -r
        hit_turn = np.repeat(turns, 2).astype(np.int32)
        true_d = np.repeat(dcas, 2)
        real = np.zeros(2 * r.size, dtype=np.uint8)
        real[0::2] = (dcas >= 0)
        real[1::2] = (dcas < 0)
        return Event(
            geom=geom, bz=bz, charge=charge, pmag=p, vertex=vertex, p0=p0,
            partitions=parts, fired_wire=fired.astype(np.int32), hit_off=hit_off,
            rho=rho, hit_turn=hit_turn, hit_real=real, hit_true_dca=true_d,
            step=step, n_steps=n_steps, cutoff=cutoff, r_stop=R_SEED,
            n_trials=trial, layers_hit=int(layers_hit), spec=dict(spec or {}))
    raise RuntimeError("no accepted event in %d trials" % max_trials)


# ----------------------------------------------------------------------------
# seeds
# ----------------------------------------------------------------------------
def truth_seed(ev: Event, part: int) -> np.ndarray:
    """[6] the generating truth at the partition's entrance: x (cm), p (MeV/c)."""
    pt = ev.partitions[part]
    return np.concatenate([pt.x_in, ev.pmag * pt.T_in])


def seed_axes(ev: Event, part: int, shape: Sequence[int], p_range: Tuple[float, float],
              ct_range: Optional[Tuple[float, float]] = None, ct_hw: float = 0.15,
              phi_hw: float = 0.04, z_hw: float = 4.0) -> dict:
    """The axis tables of one partition's seed grid (readings R17, R44): inclusive linspaces of
    |p| over p_range, cos theta over ct_range or truth +- ct_hw, phi0 over truth +- phi_hw, z0 over truth +- z_hw,
    with the tables derived from them (sin theta, cos phi0, sin phi0) and the seed point (x, y) on r = 50 cm."""
    pt = ev.partitions[part]
    n_p, n_ct, n_phi, n_z = (int(v) for v in shape)
    if ct_range is None:
        ct_range = (pt.cos_theta - ct_hw, pt.cos_theta + ct_hw)
    ca = np.linspace(ct_range[0], ct_range[1], n_ct)
    fa = np.linspace(pt.phi - phi_hw, pt.phi + phi_hw, n_phi)
    return {"xy": np.array([R_SEED * np.cos(pt.theta_e), R_SEED * np.sin(pt.theta_e)]),
            "p": np.linspace(p_range[0], p_range[1], n_p),
            "sin_theta": np.sqrt(1.0 - ca * ca), "cos_theta": ca,
            "cos_phi": np.cos(fa), "sin_phi": np.sin(fa),
            "z": np.linspace(pt.z - z_hw, pt.z + z_hw, n_z)}


def pack_axes(ax: dict) -> np.ndarray:
    """The layout of comet_seed_grid's `axes` argument (include/comet.h):
    x, y | p | sin theta | cos theta | cos phi0 | sin phi0 | z0."""
    return np.concatenate([ax["xy"], ax["p"], ax["sin_theta"], ax["cos_theta"], ax["cos_phi"], ax["sin_phi"], ax["z"]])


def grid_from_axes(ax: dict) -> np.ndarray:
    """SoA seeds [6][S] from the axis tables: index ((i_p n_ct + i_ct) n_phi + i_phi) n_z + i_z (z fastest),
    p_x = (|p| sin theta) cos phi0, p_y = (|p| sin theta) sin phi0, p_z = |p| cos theta (one multiplication each,
    in this order)."""
    ip, ic, jf, iz = np.meshgrid(np.arange(ax["p"].size), np.arange(ax["cos_theta"].size),
                                 np.arange(ax["cos_phi"].size), np.arange(ax["z"].size), indexing="ij")
    ip, ic, jf, iz = ip.ravel(), ic.ravel(), jf.ravel(), iz.ravel()
    P = ax["p"][ip]
    PS = P * ax["sin_theta"][ic]
    seeds = np.empty((6, P.size))
    seeds[0] = ax["xy"][0]
    seeds[1] = ax["xy"][1]
    seeds[2] = ax["z"][iz]
    seeds[3] = PS * ax["cos_phi"][jf]
    seeds[4] = PS * ax["sin_phi"][jf]
    seeds[5] = P * ax["cos_theta"][ic]
    return seeds


def seed_grid(ev: Event, part: int, shape: Sequence[int], p_range: Tuple[float, float],
              ct_range: Optional[Tuple[float, float]] = None, ct_hw: float = 0.15,
              phi_hw: float = 0.04, z_hw: float = 4.0) -> np.ndarray:
    """SoA seeds [6][S] for one partition (reading R17): the grid of seed_axes."""
    return grid_from_axes(seed_axes(ev, part, shape, p_range, ct_range, ct_hw, phi_hw, z_hw))


def _grid_args(ev: Event, shape):
    sp = ev.spec
    shape = tuple(shape or sp["grid"])
    p_range = tuple(sp["p_range"]) if "p_range" in sp else (ev.pmag - sp["p_hw"], ev.pmag + sp["p_hw"])
    return shape, p_range, sp.get("ct_range"), sp.get("ct_hw", 0.15)


def event_axes(ev: Event, shape: Optional[Sequence[int]] = None):
    """The axes of all partitions' grids: (axes [P][A] as comet_seed_grid takes them, shape, part_off [P+1])."""
    shape, p_range, ct_range, ct_hw = _grid_args(ev, shape)
    rows = [pack_axes(seed_axes(ev, i, shape, p_range, ct_range=ct_range, ct_hw=ct_hw)) for i in range(len(ev.partitions))]
    G = int(np.prod(shape))
    return np.ascontiguousarray(np.stack(rows)), shape, np.arange(len(rows) + 1, dtype=np.int64) * G


def event_seeds(ev: Event, shape: Optional[Sequence[int]] = None):
    """All partitions' grids concatenated: (seeds [6][S], part_off int64 [P+1])."""
    sp = ev.spec
    shape = tuple(shape or sp["grid"])
    if "p_range" in sp:
        p_range = tuple(sp["p_range"])
    else:
        p_range = (ev.pmag - sp["p_hw"], ev.pmag + sp["p_hw"])
    blocks = [seed_grid(ev, i, shape, p_range, ct_range=sp.get("ct_range"),
                        ct_hw=sp.get("ct_hw", 0.15)) for i in range(len(ev.partitions))]
    part_off = np.zeros(len(blocks) + 1, dtype=np.int64)
    part_off[1:] = np.cumsum([b.shape[1] for b in blocks])
    return np.ascontiguousarray(np.concatenate(blocks, axis=1)), part_off


# ----------------------------------------------------------------------------
# BASELINE.json configs (index 0..4)
# ----------------------------------------------------------------------------
CONFIG_SPECS = {
    0: dict(name="cfg0_tiny", rng_seed=1, n_events=1, pmag=104.0, cos_theta=(0.5, 0.7),
            vertex_z=(-30.0, 30.0), n_turns=1, grid=(16, 8, 8, 8), p_range=(98.0, 110.0),
            ct_range=(0.45, 0.75), n_steps=400, step=0.5, cutoff=0.1, n_noise=0),
    1: dict(name="cfg1_signal3turn", rng_seed=1001, n_events=1, pmag=103.5, cos_theta=(0.10, 0.25),
            vertex_z=(-70.0, -50.0), n_turns=3, grid=(32, 16, 16, 16), p_range=(95.0, 110.0),
            ct_hw=0.15, n_steps=1200, step=0.25, cutoff=0.1, n_noise=0),
    2: dict(name="cfg2_batch256", rng_seed=1002, n_events=256, pmag=(60.0, 105.0), cos_theta=(0.10, 0.70),
            vertex_z=(-70.0, 30.0), n_turns=(1, 4), grid=(32, 16, 16, 16), p_hw=7.5,
            ct_hw=0.15, n_steps=1200, step=0.25, cutoff=0.1, n_noise=0),
    3: dict(name="cfg3_largescan", rng_seed=1003, n_events=1, pmag=104.0, cos_theta=(0.10, 0.25),
            vertex_z=(-70.0, -50.0), n_turns=4, grid=(64, 32, 32, 16), p_range=(95.0, 110.0),
            ct_hw=0.15, n_steps=1600, step=0.2, cutoff=0.1, n_noise=0),
    4: dict(name="cfg4_highocc", rng_seed=1004, n_events=1, pmag=103.5, cos_theta=(0.10, 0.25),
            vertex_z=(-70.0, -50.0), n_turns=3, grid=(32, 16, 16, 16), p_range=(95.0, 110.0),
            ct_hw=0.15, n_steps=1200, step=0.25, cutoff=0.1, cutoffs=(0.05, 0.1, 0.2), n_noise=1000),
}


def config_spec(idx: int) -> dict:
    return dict(CONFIG_SPECS[idx])


def make_config(idx: int, n_events: Optional[int] = None) -> List[Event]:
    """Events of BASELINE.json configs[idx] (seed grids are built by event_seeds)."""
    sp = config_spec(idx)
    rng = np.random.default_rng(sp["rng_seed"])
    geom = cdc_geometry()
    n = sp["n_events"] if n_events is None else n_events
    out = []
    for _ in range(n):
        out.append(make_event(
            rng, pmag=sp["pmag"], cos_theta=sp["cos_theta"], vertex_z=sp["vertex_z"],
            n_turns=sp["n_turns"], step=sp["step"], n_steps=sp["n_steps"], cutoff=sp["cutoff"],
            n_noise=sp["n_noise"], geom=geom, spec=sp))
    return out
