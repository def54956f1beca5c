"""ctypes binding of libcomet.so (include/comet.h): argument marshalling only.

torch supplies device memory (`tensor.data_ptr()`) and streams (`torch.cuda.Stream.cuda_stream`);
every step of the path runs inside the library's CUDA kernels.  There is no fallback: a missing
library or a failing call raises CometError.
"""
import ctypes
import os
from typing import Optional, Sequence

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))

EXPORTED_SYMBOLS = [
    "comet_create", "comet_destroy", "comet_status_string", "comet_last_cuda_error",
    "comet_set_option", "comet_get_option", "comet_track_bytes", "comet_seed_extrapolate",
    "comet_track_export", "comet_dca_rss", "comet_select_and_classify", "comet_scan_event_host",
    "comet_fp64_peak_probe", "comet_read_stats", "comet_reserve", "comet_read_timing", "comet_scan_rss",
    "comet_select_references", "comet_refine_seeds", "comet_classify_seeds", "comet_stage_work_bytes",
    "comet_scan_stage", "comet_set_field", "comet_remove_hits", "comet_turns_work_bytes", "comet_scan_turns",
    "comet_hough_work_bytes", "comet_hough_seeds", "comet_half_hit_masks", "comet_flip_seeds", "comet_layer_veto",
    "comet_merge_half_sets", "comet_half_work_bytes", "comet_scan_half_tracks",
    "comet_turns_half_work_bytes", "comet_scan_turns_half",
    "comet_reserve_scan", "comet_seed_grid", "comet_grid_axes_len", "comet_grid_z_run", "comet_seed_runs",
    "comet_set_geometry", "comet_get_geometry", "comet_scan_event_grid_host",
    "comet_scan_event_grid_submit", "comet_scan_event_grid_collect", "comet_argmin_static",
]

COMET_CHUNK = 32
OPT_COARSE_SEARCH = 1
COARSE_EXHAUSTIVE = 0
COARSE_PRUNED = 1
OPT_STATS = 2
OPT_TIMING = 3
OPT_LANES = 4
OPT_ZGROUP = 5
STATS_FIELDS = ("samples", "rows_needed", "rows_executed", "fine_needed", "fine_executed", "pairs", "unique_states",
                "samples_b", "touched")


class CometError(RuntimeError):
    pass


def lib_path() -> str:
    return os.path.join(_HERE, "libcomet.so")


_lib = None


def load_library():
    """dlopen the in-tree libcomet.so and declare the signatures of include/comet.h."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise CometError("%s is missing: build it with `python -m paper_1911_09340_b200.build` "
                         "(there is no CPU fallback)" % path)
    L = ctypes.CDLL(path)
    vp, i32, i64, dbl, sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_double, ctypes.c_size_t
    L.comet_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int]
    L.comet_destroy.argtypes = [vp]
    L.comet_status_string.argtypes = [ctypes.c_int]
    L.comet_status_string.restype = ctypes.c_char_p
    L.comet_last_cuda_error.argtypes = [vp]
    L.comet_set_option.argtypes = [vp, ctypes.c_int, ctypes.c_int]
    L.comet_get_option.argtypes = [vp, ctypes.c_int, ctypes.POINTER(ctypes.c_int)]
    L.comet_track_bytes.argtypes = [i64, i32]
    L.comet_track_bytes.restype = sz
    L.comet_seed_extrapolate.argtypes = [vp, vp, i64, i64, i32, dbl, dbl, i32, dbl, vp, vp, vp]
    L.comet_track_export.argtypes = [vp, vp, vp, i64, i32, i64, i64, vp, vp]
    L.comet_dca_rss.argtypes = [vp, vp, vp, i64, i32, i32, dbl, dbl, vp, i64,
                                vp, vp, i32, vp, vp, vp, i32, i32, dbl, vp, vp, vp, vp]
    L.comet_scan_rss.argtypes = [vp, vp, i64, i64, i32, i32, dbl, dbl, i32, dbl,
                                 vp, vp, i32, vp, vp, vp, i32, i32, dbl, vp, vp, vp]
    L.comet_select_and_classify.argtypes = [vp, vp, i64, i64, i32, dbl, dbl, i32, dbl,
                                            vp, vp, i32, vp, vp, vp, i32, i32, dbl,
                                            vp, vp, i32, vp, vp, vp, vp, vp]
    L.comet_scan_event_host.argtypes = [vp, vp, i64, i32, dbl, dbl, i32, dbl,
                                        vp, vp, i32, vp, vp, vp, i32, i32, dbl,
                                        vp, i32, sz, vp, vp, vp, vp, vp, vp]
    L.comet_fp64_peak_probe.argtypes = [vp, i32, vp, ctypes.POINTER(dbl), vp]
    L.comet_reserve.argtypes = [vp, i64]
    L.comet_read_timing.argtypes = [vp, ctypes.POINTER(ctypes.c_float), i32, ctypes.POINTER(i32)]
    L.comet_read_stats.argtypes = [vp, ctypes.POINTER(ctypes.c_uint64), i32, i32, vp]
    L.comet_remove_hits.argtypes = [vp, vp, vp, vp, i32, i32, vp, vp, vp, vp, vp, vp, vp, vp]
    L.comet_turns_work_bytes.argtypes = [i64, i32, i32, i32, vp]
    L.comet_turns_work_bytes.restype = sz
    L.comet_scan_turns.argtypes = [vp, vp, i64, i64, i32, i32, dbl, dbl, i32, dbl,
                                   vp, vp, i32, vp, vp, vp, i32, i32, dbl,
                                   vp, i32, vp, vp, i32, dbl, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp]
    L.comet_hough_work_bytes.argtypes = [i32]
    L.comet_hough_work_bytes.restype = sz
    L.comet_hough_seeds.argtypes = [vp, vp, vp, i32, vp, vp, i32, vp, vp, i32, dbl, dbl, i32, i32, dbl, dbl,
                                    vp, vp, vp, vp, vp]
    L.comet_half_hit_masks.argtypes = [vp, vp, vp, i32, vp, vp, i32, i32, vp, dbl, vp, vp, vp]
    L.comet_flip_seeds.argtypes = [vp, vp, i64, i64, vp, i64, vp]
    L.comet_layer_veto.argtypes = [vp, vp, i32, vp, vp, i32, i32, vp, i32, i32, vp, vp]
    L.comet_merge_half_sets.argtypes = [vp, vp, vp, vp, i32, i32, vp, vp, vp, i32, i32, i32, vp, vp, vp, vp]
    L.comet_half_work_bytes.argtypes = [i64, i64, i32, i32, i32, i32, vp]
    L.comet_half_work_bytes.restype = sz
    L.comet_scan_half_tracks.argtypes = [vp, vp, i64, vp, i64, i32, dbl, dbl, i32, dbl,
                                         vp, vp, i32, vp, vp, vp, i32, i32, dbl,
                                         vp, vp, dbl, i32, vp, vp, i32, dbl, i32, i32, vp,
                                         vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    L.comet_turns_half_work_bytes.argtypes = [i64, i64, i32, i32, i32, i32, vp]
    L.comet_turns_half_work_bytes.restype = sz
    L.comet_scan_turns_half.argtypes = [vp, vp, vp, i64, vp, vp, i64, i32, i32, dbl, dbl, i32, dbl,
                                        vp, vp, i32, vp, vp, vp, i32, i32, dbl,
                                        vp, vp, dbl, i32, vp, vp, i32, dbl, i32, i32, i32, i32, vp,
                                        vp, vp, vp, vp, vp, vp, vp]
    L.comet_set_field.argtypes = [vp, vp, vp, vp, vp, dbl, vp]
    L.comet_select_references.argtypes = [vp, vp, i64, i64, vp, vp, i32, vp, i32, vp, vp]
    L.comet_refine_seeds.argtypes = [vp, vp, i64, i64, vp, i32, i32, vp, vp, vp, i64, vp]
    L.comet_classify_seeds.argtypes = [vp, vp, i64, i64, i32, dbl, dbl, i32, dbl,
                                       vp, vp, i32, vp, vp, vp, i32, i32, dbl, vp, i32, vp, vp, vp]
    L.comet_stage_work_bytes.argtypes = [i64, i32, i32, i32, vp]
    L.comet_stage_work_bytes.restype = sz
    L.comet_scan_stage.argtypes = [vp, vp, i64, i64, i32, i32, dbl, dbl, i32, dbl,
                                   vp, vp, i32, vp, vp, vp, i32, i32, dbl,
                                   vp, i32, vp, vp, i32, dbl, i32, i32, vp, vp, vp, vp, vp, vp]
    L.comet_reserve_scan.argtypes = [vp, i64, i32, i32, i32]
    L.comet_seed_grid.argtypes = [vp, vp, i32, i32, i32, i32, i32, vp, i64, vp]
    L.comet_grid_axes_len.argtypes = [i32, i32, i32, i32]
    L.comet_grid_axes_len.restype = sz
    L.comet_grid_z_run.argtypes = [i32]
    L.comet_grid_z_run.restype = i32
    L.comet_seed_runs.argtypes = [vp, vp, i64, i64, ctypes.POINTER(i32), vp]
    L.comet_set_geometry.argtypes = [vp, vp, vp, i32, vp]
    L.comet_get_geometry.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.POINTER(i32)]
    L.comet_scan_event_grid_host.argtypes = [vp, vp, i32, i32, i32, i32, i32, i32, dbl, dbl, i32, dbl,
                                             vp, vp, vp, i32, i32, dbl, vp, vp, vp, vp, vp, vp]
    L.comet_scan_event_grid_submit.argtypes = [vp, i32, vp, i32, i32, i32, i32, i32, i32, dbl, dbl, i32, dbl,
                                               vp, vp, vp, i32, i32, dbl, vp]
    L.comet_scan_event_grid_collect.argtypes = [vp, i32, vp, vp, vp, vp]
    L.comet_argmin_static.argtypes = [vp, i64, vp, i32, vp, vp, vp]
    for name in EXPORTED_SYMBOLS:
        if name not in ("comet_status_string", "comet_track_bytes", "comet_stage_work_bytes", "comet_turns_work_bytes",
                        "comet_hough_work_bytes", "comet_half_work_bytes", "comet_grid_axes_len", "comet_grid_z_run",
                        "comet_turns_half_work_bytes"):
            getattr(L, name).restype = ctypes.c_int
    _lib = L
    return L


def _stream_ptr(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def _dev(t: Optional[torch.Tensor], dtype, name: str, device) -> int:
    """data_ptr of a contiguous CUDA tensor of the given dtype on `device` (0 for None)."""
    if t is None:
        return 0
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise CometError("%s must be a contiguous CUDA tensor of dtype %s" % (name, dtype))
    if t.device.index != device:
        raise CometError("%s is on cuda:%s, the context is on cuda:%d" % (name, t.device.index, device))
    return int(t.data_ptr())


STATIC_MAX_PART = 64        # COMET_STATIC_MAX_PART


def argmin_static(rss, part_off: Sequence[int], best_seed=None, best_rss=None, stream=None):
    """comet_argmin_static: per-partition lowest-index argmin of `rss` (CUDA float64 [S]) on rss's device, without a
    context and without any allocation inside the library; the outputs are the caller's (int64 [P], float64 [P] CUDA
    tensors; made here with torch when not given).  All calls on a device share one static scratch array: calls that
    can overlap on the GPU race."""
    L = load_library()
    if not torch.cuda.is_available():
        raise CometError("no CUDA device: the seed x hit scan has no CPU implementation")
    if not isinstance(rss, torch.Tensor) or not rss.is_cuda:
        raise CometError("rss must be a CUDA tensor")
    d = rss.device.index
    po = np.ascontiguousarray(np.asarray(part_off, dtype=np.int64))
    P = po.shape[0] - 1
    with torch.cuda.device(d):
        if best_seed is None:
            best_seed = torch.empty(P, dtype=torch.int64, device=rss.device)
        if best_rss is None:
            best_rss = torch.empty(P, dtype=torch.float64, device=rss.device)
        if best_seed.numel() < P or best_rss.numel() < P:
            raise CometError("best_seed / best_rss hold fewer than %d partitions" % P)
        rc = L.comet_argmin_static(_dev(rss, torch.float64, "rss", d), int(rss.numel()), po.ctypes.data, P,
                                   _dev(best_seed, torch.int64, "best_seed", d), _dev(best_rss, torch.float64, "best_rss", d),
                                   _stream_ptr(stream))
    if rc != 0:
        raise CometError("libcomet: %s (status %d)" % (L.comet_status_string(rc).decode(), rc))
    return {"best_seed": best_seed, "best_rss": best_rss}


class Comet:
    """One comet_ctx (one per stream).  Methods mirror the C entry points."""

    def __init__(self, device: int = 0):
        self._L = load_library()
        if not torch.cuda.is_available():
            raise CometError("no CUDA device: the seed x hit scan has no CPU implementation")
        self.device = int(device)
        h = ctypes.c_void_p()
        self._check(self._L.comet_create(ctypes.byref(h), self.device), None)
        self._h = h

    # -- plumbing ---------------------------------------------------------------------------
    def _check(self, rc: int, h=True):
        if rc != 0:
            msg = self._L.comet_status_string(rc).decode()
            cu = self._L.comet_last_cuda_error(self._h) if h and getattr(self, "_h", None) else 0
            raise CometError("libcomet: %s (status %d, cudaError %d)" % (msg, rc, cu))

    def close(self):
        if getattr(self, "_h", None):
            torch.cuda.synchronize(self.device)
            self._L.comet_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_option(self, option: int, value: int):
        self._check(self._L.comet_set_option(self._h, int(option), int(value)))

    def get_option(self, option: int) -> int:
        v = ctypes.c_int()
        self._check(self._L.comet_get_option(self._h, int(option), ctypes.byref(v)))
        return v.value

    def set_field(self, field=None, origin=None, spacing=None, rkn_tol=1e-7, stream=None):
        """comet_set_field: `field` is a CUDA tensor [nx][ny][nz][3] (Tesla) that must stay alive while it
        is set; None returns to the uniform field."""
        if field is None:
            self._field = None
            self._check(self._L.comet_set_field(self._h, 0, 0, 0, 0, 0.0, 0))
            return
        n = np.ascontiguousarray(np.asarray(field.shape[:3], dtype=np.int32))
        o = np.ascontiguousarray(np.asarray(origin, dtype=np.float64))
        d = np.ascontiguousarray(np.asarray(spacing, dtype=np.float64))
        if field.dim() != 4 or field.shape[3] != 3:
            raise CometError("field must be [nx][ny][nz][3]")
        self._check(self._L.comet_set_field(self._h, _dev(field, torch.float64, "field", self.device), n.ctypes.data,
                                            o.ctypes.data, d.ctypes.data, float(rkn_tol), _stream_ptr(stream)))
        self._field = field

    def reserve(self, max_pairs_per_launch: int):
        """Pre-allocates the pruned search's (seed, wire) pair workspace (12 bytes per pair)."""
        self._check(self._L.comet_reserve(self._h, int(max_pairs_per_launch)))

    def reserve_scan(self, n_seeds: int, n_steps: int, n_fired: int, z_run: int = 0):
        """comet_reserve_scan: sizes every workspace of comet_scan_rss & co.; later calls do not allocate."""
        self._check(self._L.comet_reserve_scan(self._h, int(n_seeds), int(z_run), int(n_steps), int(n_fired)))

    def read_timing(self, names=("k_coarse_pruned", "k_fine", "k_rss_sum", "k_gen_unique")) -> dict:
        """Mean device milliseconds per kernel of the latest (<= 64) seed slabs of comet_dca_rss (pruned:
        k_coarse_pruned, k_fine, k_rss_sum) or comet_scan_rss (k_scan_fused, k_fine_ck, k_rss_sum) made
        with OPT_TIMING = 1 (waits for them).  `names` labels the three slots."""
        buf = (ctypes.c_float * 4)()
        n = ctypes.c_int32()
        self._check(self._L.comet_read_timing(self._h, buf, 4, ctypes.byref(n)))
        out = {k: float(v) for k, v in zip(names, buf)}
        out["n_calls"] = int(n.value)
        return out

    def read_stats(self, reset: bool = True, stream=None) -> dict:
        """Work counters of the pruned comet_dca_rss calls made with OPT_STATS = 1 (synchronises)."""
        buf = (ctypes.c_uint64 * len(STATS_FIELDS))()
        self._check(self._L.comet_read_stats(self._h, buf, len(STATS_FIELDS), int(bool(reset)), _stream_ptr(stream)))
        return dict(zip(STATS_FIELDS, (int(v) for v in buf)))

    def track_bytes(self, n_seeds: int, n_steps: int) -> int:
        return int(self._L.comet_track_bytes(int(n_seeds), int(n_steps)))

    def _tdev(self):
        return torch.device("cuda", self.device)

    # -- kernel A ---------------------------------------------------------------------------
    def seed_extrapolate(self, seeds, charge, bz, step, n_steps, r_stop, track=None, n_pts=None,
                         seed_range=None, stream=None):
        """seeds: CUDA float64 [6][S].  Returns (track uint8 buffer, n_pts int32 [n])."""
        S = seeds.shape[1]
        b, e = (0, S) if seed_range is None else seed_range
        n = e - b
        base = _dev(seeds, torch.float64, "seeds", self.device)
        need = self.track_bytes(n, n_steps)
        if track is None:
            track = torch.empty(max(need, 16), dtype=torch.uint8, device=self._tdev())
        elif track.numel() * track.element_size() < need:
            raise CometError("track buffer too small: %d < %d bytes" % (track.numel() * track.element_size(), need))
        if n_pts is None:
            n_pts = torch.empty(n, dtype=torch.int32, device=self._tdev())
        self._check(self._L.comet_seed_extrapolate(
            self._h, base + 8 * b, S, n, int(charge), float(bz), float(step), int(n_steps), float(r_stop),
            int(track.data_ptr()), _dev(n_pts, torch.int32, "n_pts", self.device), _stream_ptr(stream)))
        return track, n_pts

    def track_export(self, track, n_pts, n_seeds, n_steps, seed_begin=0, seed_end=None, stream=None):
        seed_end = n_seeds if seed_end is None else seed_end
        out = torch.empty((seed_end - seed_begin, n_steps + 1, 6), dtype=torch.float64, device=self._tdev())
        self._check(self._L.comet_track_export(
            self._h, int(track.data_ptr()), _dev(n_pts, torch.int32, "n_pts", self.device), int(n_seeds),
            int(n_steps), int(seed_begin), int(seed_end), int(out.data_ptr()), _stream_ptr(stream)))
        return out

    # -- kernel B ---------------------------------------------------------------------------
    def dca_rss(self, track, n_pts, seeds, charge, bz, step, n_steps, wire_a, wire_b, fired_wire, hit_off,
                rho, cutoff, rss=None, want_dca=False, want_kstar=False, seed_range=None, stream=None):
        S = seeds.shape[1]
        b, e = (0, S) if seed_range is None else seed_range
        n = e - b
        W, H = int(fired_wire.shape[0]), int(rho.shape[0])
        d = self.device
        if rss is None:
            rss = torch.empty(n, dtype=torch.float64, device=self._tdev())
        dca = torch.empty((n, W), dtype=torch.float64, device=self._tdev()) if want_dca else None
        ks = torch.empty((n, W), dtype=torch.int32, device=self._tdev()) if want_kstar else None
        self._check(self._L.comet_dca_rss(
            self._h, int(track.data_ptr()), _dev(n_pts, torch.int32, "n_pts", d), n, int(n_steps), int(charge),
            float(bz), float(step), _dev(seeds, torch.float64, "seeds", d) + 8 * b, S,
            _dev(wire_a, torch.float64, "wire_a", d), _dev(wire_b, torch.float64, "wire_b", d),
            int(wire_a.shape[1]), _dev(fired_wire, torch.int32, "fired_wire", d),
            _dev(hit_off, torch.int32, "hit_off", d), _dev(rho, torch.float64, "rho", d), W, H, float(cutoff),
            _dev(rss, torch.float64, "rss", d), _dev(dca, torch.float64, "dca", d),
            _dev(ks, torch.int32, "kstar", d), _stream_ptr(stream)))
        out = {"rss": rss}
        if want_dca:
            out["dca"] = dca
        if want_kstar:
            out["kstar"] = ks
        return out

    # -- kernels A + B fused, track on chip ---------------------------------------------------
    def scan_rss(self, seeds, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire, hit_off, rho,
                 cutoff, rss=None, n_pts=None, want_npts=True, seed_range=None, stream=None, z_run=0):
        """comet_scan_rss: RSS (and n_pts) of seeds[:, b:e] without a track buffer."""
        S = seeds.shape[1]
        b, e = (0, S) if seed_range is None else seed_range
        n = e - b
        W, H = int(fired_wire.shape[0]), int(rho.shape[0])
        d = self.device
        if rss is None:
            rss = torch.empty(n, dtype=torch.float64, device=self._tdev())
        if n_pts is None and want_npts:
            n_pts = torch.empty(n, dtype=torch.int32, device=self._tdev())
        self._check(self._L.comet_scan_rss(
            self._h, _dev(seeds, torch.float64, "seeds", d) + 8 * b, S, n, int(z_run), int(charge), float(bz), float(step),
            int(n_steps), float(r_stop),
            _dev(wire_a, torch.float64, "wire_a", d), _dev(wire_b, torch.float64, "wire_b", d),
            int(wire_a.shape[1]), _dev(fired_wire, torch.int32, "fired_wire", d),
            _dev(hit_off, torch.int32, "hit_off", d), _dev(rho, torch.float64, "rho", d), W, H, float(cutoff),
            _dev(rss, torch.float64, "rss", d), _dev(n_pts, torch.int32, "n_pts", d), _stream_ptr(stream)))
        return {"rss": rss, "n_pts": n_pts}

    # -- step C -----------------------------------------------------------------------------
    def select_and_classify(self, seeds, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire,
                            hit_off, rho, cutoff, rss, part_off: Sequence[int], stream=None):
        S = seeds.shape[1]
        W, H = int(fired_wire.shape[0]), int(rho.shape[0])
        po = np.ascontiguousarray(np.asarray(part_off, dtype=np.int64))
        P = po.shape[0] - 1
        d, td = self.device, self._tdev()
        best_seed = torch.empty(P, dtype=torch.int64, device=td)
        best_rss = torch.empty(P, dtype=torch.float64, device=td)
        best_dca = torch.empty((P, W), dtype=torch.float64, device=td)
        cls = torch.empty((P, H), dtype=torch.uint8, device=td)
        self._check(self._L.comet_select_and_classify(
            self._h, _dev(seeds, torch.float64, "seeds", d), S, S, int(charge), float(bz), float(step),
            int(n_steps), float(r_stop),
            _dev(wire_a, torch.float64, "wire_a", d), _dev(wire_b, torch.float64, "wire_b", d),
            int(wire_a.shape[1]), _dev(fired_wire, torch.int32, "fired_wire", d),
            _dev(hit_off, torch.int32, "hit_off", d), _dev(rho, torch.float64, "rho", d), W, H, float(cutoff),
            _dev(rss, torch.float64, "rss", d), po.ctypes.data, P,
            int(best_seed.data_ptr()), int(best_rss.data_ptr()), int(best_dca.data_ptr()), int(cls.data_ptr()),
            _stream_ptr(stream)))
        return {"best_seed": best_seed, "best_rss": best_rss, "best_dca": best_dca, "cls": cls}

    # -- iterative seed refinement ------------------------------------------------------------
    def select_references(self, seeds, rss, part_off, half_width, k_ref, stream=None):
        """comet_select_references -> int64 [P][k_ref] (device), -1 = none."""
        S = seeds.shape[1]
        po = np.ascontiguousarray(np.asarray(part_off, dtype=np.int64))
        hw = np.ascontiguousarray(np.asarray(half_width, dtype=np.float64))
        P, d = po.shape[0] - 1, self.device
        ref = torch.empty((P, int(k_ref)), dtype=torch.int64, device=self._tdev())
        self._check(self._L.comet_select_references(
            self._h, _dev(seeds, torch.float64, "seeds", d), S, S, _dev(rss, torch.float64, "rss", d),
            po.ctypes.data, P, hw.ctypes.data, int(k_ref), int(ref.data_ptr()), _stream_ptr(stream)))
        return ref

    def refine_seeds(self, seeds, ref_seed, half_width, n_grid, stream=None):
        """comet_refine_seeds -> (new seeds [6][P k G] (device), part_off of the new set)."""
        S = seeds.shape[1]
        hw = np.ascontiguousarray(np.asarray(half_width, dtype=np.float64))
        ng = np.ascontiguousarray(np.asarray(n_grid, dtype=np.int32))
        P, K = int(ref_seed.shape[0]), int(ref_seed.shape[1])
        G, d = int(np.prod(ng.astype(np.int64))), self.device
        new = torch.empty((6, P * K * G), dtype=torch.float64, device=self._tdev())
        self._check(self._L.comet_refine_seeds(
            self._h, _dev(seeds, torch.float64, "seeds", d), S, S, _dev(ref_seed, torch.int64, "ref_seed", d), P, K,
            hw.ctypes.data, ng.ctypes.data, int(new.data_ptr()), P * K * G, _stream_ptr(stream)))
        return new, np.arange(P + 1, dtype=np.int64) * (K * G)

    def classify_seeds(self, seeds, seed_idx, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire,
                       hit_off, rho, cutoff, stream=None):
        S, n = seeds.shape[1], int(seed_idx.numel())
        W, H, d, td = int(fired_wire.shape[0]), int(rho.shape[0]), self.device, self._tdev()
        dca = torch.empty((n, W), dtype=torch.float64, device=td)
        cls = torch.empty((n, H), dtype=torch.uint8, device=td)
        self._check(self._L.comet_classify_seeds(
            self._h, _dev(seeds, torch.float64, "seeds", d), S, S, int(charge), float(bz), float(step),
            int(n_steps), float(r_stop),
            _dev(wire_a, torch.float64, "wire_a", d), _dev(wire_b, torch.float64, "wire_b", d),
            int(wire_a.shape[1]), _dev(fired_wire, torch.int32, "fired_wire", d),
            _dev(hit_off, torch.int32, "hit_off", d), _dev(rho, torch.float64, "rho", d), W, H, float(cutoff),
            _dev(seed_idx, torch.int64, "seed_idx", d), n, int(dca.data_ptr()), int(cls.data_ptr()),
            _stream_ptr(stream)))
        return {"dca": dca, "cls": cls}

    def stage_work_bytes(self, n_seeds, n_part, k_ref, k_final, n_grid) -> int:
        ng = np.ascontiguousarray(np.asarray(n_grid, dtype=np.int32))
        return int(self._L.comet_stage_work_bytes(int(n_seeds), int(n_part), int(k_ref), int(k_final), ng.ctypes.data))

    def scan_stage(self, seeds, part_off, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire, hit_off,
                   rho, cutoff, half_width, n_grid, n_iter, shrink, k_ref, k_final, work=None, stream=None, z_run=0):
        """comet_scan_stage: a whole stage (scan, n_iter refinements, final selection, classification)."""
        S = seeds.shape[1]
        po = np.ascontiguousarray(np.asarray(part_off, dtype=np.int64))
        hw = np.ascontiguousarray(np.asarray(half_width, dtype=np.float64))
        ng = np.ascontiguousarray(np.asarray(n_grid, dtype=np.int32))
        P, W, H = po.shape[0] - 1, int(fired_wire.shape[0]), int(rho.shape[0])
        d, td = self.device, self._tdev()
        if work is None:
            nb = self.stage_work_bytes(S, P, k_ref, k_final, ng)
            if nb == 0:
                raise CometError("comet_stage_work_bytes: invalid arguments")
            work = torch.empty(nb, dtype=torch.uint8, device=td)
        out = {"final_seed": torch.empty((P, int(k_final), 6), dtype=torch.float64, device=td),
               "final_rss": torch.empty((P, int(k_final)), dtype=torch.float64, device=td),
               "final_dca": torch.empty((P, int(k_final), W), dtype=torch.float64, device=td),
               "cls": torch.empty((P, int(k_final), H), dtype=torch.uint8, device=td), "work": work}
        self._check(self._L.comet_scan_stage(
            self._h, _dev(seeds, torch.float64, "seeds", d), S, S, int(z_run), int(charge), float(bz), float(step),
            int(n_steps), float(r_stop),
            _dev(wire_a, torch.float64, "wire_a", d), _dev(wire_b, torch.float64, "wire_b", d),
            int(wire_a.shape[1]), _dev(fired_wire, torch.int32, "fired_wire", d),
            _dev(hit_off, torch.int32, "hit_off", d), _dev(rho, torch.float64, "rho", d), W, H, float(cutoff),
            po.ctypes.data, P, hw.ctypes.data, ng.ctypes.data, int(n_iter), float(shrink), int(k_ref), int(k_final),
            int(work.data_ptr()), int(out["final_seed"].data_ptr()), int(out["final_rss"].data_ptr()),
            int(out["final_dca"].data_ptr()), int(out["cls"].data_ptr()), _stream_ptr(stream)))
        return out

    # -- sequential stages with hit removal -------------------------------------------------------
    def remove_hits(self, fired_wire, hit_off, rho, cls, orig=None, stream=None):
        """comet_remove_hits -> dict(fired_wire, hit_off, rho, orig, counts) (device; sliced to the new sizes,
        which costs one synchronisation)."""
        W, H, d, td = int(fired_wire.shape[0]), int(rho.shape[0]), self.device, self._tdev()
        fo = torch.empty(W, dtype=torch.int32, device=td)
        ho = torch.empty(W + 1, dtype=torch.int32, device=td)
        ro = torch.empty(H, dtype=torch.float64, device=td)
        oo = torch.empty(H, dtype=torch.int32, device=td)
        cnt = torch.empty(2, dtype=torch.int32, device=td)
        self._check(self._L.comet_remove_hits(
            self._h, _dev(fired_wire, torch.int32, "fired_wire", d), _dev(hit_off, torch.int32, "hit_off", d),
            _dev(rho, torch.float64, "rho", d), W, H, _dev(cls, torch.uint8, "cls", d), _dev(orig, torch.int32, "orig", d),
            int(fo.data_ptr()), int(ho.data_ptr()), int(ro.data_ptr()), int(oo.data_ptr()), int(cnt.data_ptr()),
            _stream_ptr(stream)))
        nw, nh = (int(v) for v in cnt.cpu().tolist())
        return {"fired_wire": fo[:nw], "hit_off": ho[:nw + 1], "rho": ro[:nh], "orig": oo[:nh], "counts": (nw, nh)}

    def scan_turns(self, seeds, part_off, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire, hit_off,
                   rho, cutoff, half_width, n_grid, n_iter, shrink, k_ref, min_wires=30, max_tracks=5, stream=None,
                   z_run=0, work=None, sync=True):
        """comet_scan_turns: the last turn first, hits of a stage's best seed removed before the previous turn."""
        S = seeds.shape[1]
        po = np.ascontiguousarray(np.asarray(part_off, dtype=np.int64))
        hw = np.ascontiguousarray(np.asarray(half_width, dtype=np.float64))
        ng = np.ascontiguousarray(np.asarray(n_grid, dtype=np.int32))
        P, W, H = po.shape[0] - 1, int(fired_wire.shape[0]), int(rho.shape[0])
        d, td = self.device, self._tdev()
        nb = int(self._L.comet_turns_work_bytes(int(np.diff(po).max()), W, H, int(k_ref), ng.ctypes.data))
        if nb == 0:
            raise CometError("comet_turns_work_bytes: invalid arguments")
        if work is None:
            work = torch.empty(nb, dtype=torch.uint8, device=td)
        out = {"work": work, "turn_seed": torch.empty((P, 6), dtype=torch.float64, device=td),
               "turn_rss": torch.empty(P, dtype=torch.float64, device=td),
               "turn_cls": torch.empty((P, H), dtype=torch.uint8, device=td)}
        done = torch.empty(P, dtype=torch.int32, device=td)
        wb = torch.empty(P, dtype=torch.int32, device=td)
        self._check(self._L.comet_scan_turns(
            self._h, _dev(seeds, torch.float64, "seeds", d), S, S, int(z_run), int(charge), float(bz), float(step),
            int(n_steps), float(r_stop),
            _dev(wire_a, torch.float64, "wire_a", d), _dev(wire_b, torch.float64, "wire_b", d),
            int(wire_a.shape[1]), _dev(fired_wire, torch.int32, "fired_wire", d),
            _dev(hit_off, torch.int32, "hit_off", d), _dev(rho, torch.float64, "rho", d), W, H, float(cutoff),
            po.ctypes.data, P, hw.ctypes.data, ng.ctypes.data, int(n_iter), float(shrink), int(k_ref),
            int(min_wires), int(max_tracks), int(work.data_ptr()), int(out["turn_seed"].data_ptr()),
            int(out["turn_rss"].data_ptr()), int(out["turn_cls"].data_ptr()), int(done.data_ptr()), int(wb.data_ptr()),
            _stream_ptr(stream)))
        out["done_dev"], out["wires_before_dev"] = done, wb
        if sync:                                             # (the call itself only enqueues: reading the flags back waits for it)
            out["done"], out["wires_before"] = done.cpu().numpy().astype(bool), wb.cpu().numpy()
        return out

    # -- Hough-transform transverse seeding --------------------------------------------------------
    def hough_seeds(self, wire_a, wire_b, fired_wire, ev_off, cos_tab, sin_tab, rho_min, inv_drho, n_rho,
                    charge, bz, r_seed, want_acc=True, stream=None):
        """comet_hough_seeds for a batch of events (fired_wire concatenated, ev_off [n_events+1]) ->
        dict(acc [E][n_phi][n_rho] or None, peak [E][3], circle [E][11]) (device)."""
        d, td = self.device, self._tdev()
        E, n_phi = int(ev_off.shape[0]) - 1, int(cos_tab.shape[0])
        work = torch.empty(int(self._L.comet_hough_work_bytes(E)), dtype=torch.uint8, device=td)
        out = {"acc": torch.empty((E, n_phi, int(n_rho)), dtype=torch.int32, device=td) if want_acc else None,
               "peak": torch.empty((E, 3), dtype=torch.int32, device=td),
               "circle": torch.empty((E, 11), dtype=torch.float64, device=td)}
        self._check(self._L.comet_hough_seeds(
            self._h, _dev(wire_a, torch.float64, "wire_a", d), _dev(wire_b, torch.float64, "wire_b", d),
            int(wire_a.shape[1]), _dev(fired_wire, torch.int32, "fired_wire", d), _dev(ev_off, torch.int32, "ev_off", d),
            E, _dev(cos_tab, torch.float64, "cos_tab", d), _dev(sin_tab, torch.float64, "sin_tab", d), n_phi,
            float(rho_min), float(inv_drho), int(n_rho), int(charge), float(bz), float(r_seed),
            int(work.data_ptr()), _dev(out["acc"], torch.int32, "acc", d), int(out["peak"].data_ptr()),
            int(out["circle"].data_ptr()), _stream_ptr(stream)))
        out["_work"] = work          # keeps the buffer alive until the caller drops the result
        return out

    # -- half tracks -----------------------------------------------------------------------------
    def half_hit_masks(self, wire_a, wire_b, fired_wire, hit_off, n_hits, circle, overlap, stream=None):
        """comet_half_hit_masks -> (in_ent, in_exit) uint8 [n_hits] (device)."""
        d, td = self.device, self._tdev()
        ie = torch.zeros(int(n_hits), dtype=torch.uint8, device=td)
        ix = torch.zeros(int(n_hits), dtype=torch.uint8, device=td)
        self._check(self._L.comet_half_hit_masks(
            self._h, _dev(wire_a, torch.float64, "wire_a", d), _dev(wire_b, torch.float64, "wire_b", d),
            int(wire_a.shape[1]), _dev(fired_wire, torch.int32, "fired_wire", d), _dev(hit_off, torch.int32, "hit_off", d),
            int(fired_wire.shape[0]), int(n_hits), _dev(circle, torch.float64, "circle", d), float(overlap),
            int(ie.data_ptr()), int(ix.data_ptr()), _stream_ptr(stream)))
        return ie, ix

    def flip_seeds(self, seeds, stream=None):
        """comet_flip_seeds -> new SoA [6][S] tensor with the momentum negated."""
        S = int(seeds.shape[1])
        out = torch.empty_like(seeds)
        self._check(self._L.comet_flip_seeds(self._h, _dev(seeds, torch.float64, "seeds", self.device), S, S,
                                             int(out.data_ptr()), S, _stream_ptr(stream)))
        return out

    def layer_veto(self, cls, fired_wire, hit_off, wire_layer, min_layers, stream=None):
        """comet_layer_veto: cls [n_sel][n_hits] -> ok uint8 [n_sel] (device)."""
        d = self.device
        n_sel, H = int(cls.shape[0]), int(cls.shape[1])
        ok = torch.empty(n_sel, dtype=torch.uint8, device=self._tdev())
        self._check(self._L.comet_layer_veto(
            self._h, _dev(cls, torch.uint8, "cls", d), n_sel, _dev(fired_wire, torch.int32, "fired_wire", d),
            _dev(hit_off, torch.int32, "hit_off", d), int(fired_wire.shape[0]), H,
            _dev(wire_layer, torch.int32, "wire_layer", d), int(wire_layer.shape[0]), int(min_layers),
            int(ok.data_ptr()), _stream_ptr(stream)))
        return ok

    def merge_half_sets(self, cls_e, orig_e, ok_e, cls_x, orig_x, ok_x, n_hits, stream=None):
        """comet_merge_half_sets -> dict(valid [Ke][Kx], cls [Ke][Kx][n_hits], n_cls [Ke][Kx]) (device)."""
        d, td = self.device, self._tdev()
        Ke, He, Kx, Hx = int(cls_e.shape[0]), int(cls_e.shape[1]), int(cls_x.shape[0]), int(cls_x.shape[1])
        out = {"valid": torch.empty((Ke, Kx), dtype=torch.uint8, device=td),
               "cls": torch.empty((Ke, Kx, int(n_hits)), dtype=torch.uint8, device=td),
               "n_cls": torch.empty((Ke, Kx), dtype=torch.int32, device=td)}
        self._check(self._L.comet_merge_half_sets(
            self._h, _dev(cls_e, torch.uint8, "cls_e", d), _dev(orig_e, torch.int32, "orig_e", d),
            _dev(ok_e, torch.uint8, "ok_e", d), Ke, He, _dev(cls_x, torch.uint8, "cls_x", d),
            _dev(orig_x, torch.int32, "orig_x", d), _dev(ok_x, torch.uint8, "ok_x", d), Kx, Hx, int(n_hits),
            int(out["valid"].data_ptr()), int(out["cls"].data_ptr()), int(out["n_cls"].data_ptr()), _stream_ptr(stream)))
        return out

    def scan_half_tracks(self, seeds_e, seeds_x, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire,
                         hit_off, rho, cutoff, wire_layer, circle, overlap, min_layers, half_width, n_grid, n_iter,
                         shrink, k_ref, k_final, stream=None):
        """comet_scan_half_tracks -> dict(ent / ext: dict(final_seed [K][6], final_rss [K], ok [K], cls [K][H_half],
        orig [H_half], n_fired), valid, cls, n_cls) (device tensors)."""
        d, td = self.device, self._tdev()
        hw = np.ascontiguousarray(np.asarray(half_width, dtype=np.float64))
        ng = np.ascontiguousarray(np.asarray(n_grid, dtype=np.int32))
        Se, Sx, W, H, K = int(seeds_e.shape[1]), int(seeds_x.shape[1]), int(fired_wire.shape[0]), int(rho.shape[0]), int(k_final)
        nb = int(self._L.comet_half_work_bytes(Se, Sx, W, H, int(k_ref), K, ng.ctypes.data))
        if nb == 0:
            raise CometError("comet_half_work_bytes: invalid arguments")
        work = torch.empty(nb, dtype=torch.uint8, device=td)
        hs = torch.empty((2, K, 6), dtype=torch.float64, device=td)
        hr = torch.empty((2, K), dtype=torch.float64, device=td)
        hok = torch.empty((2, K), dtype=torch.uint8, device=td)
        hcls = torch.empty((2, K * H), dtype=torch.uint8, device=td)
        horig = torch.empty((2, H), dtype=torch.int32, device=td)
        counts = np.zeros(4, dtype=np.int32)
        out = {"valid": torch.empty((K, K), dtype=torch.uint8, device=td),
               "cls": torch.empty((K, K, H), dtype=torch.uint8, device=td),
               "n_cls": torch.empty((K, K), dtype=torch.int32, device=td)}
        self._check(self._L.comet_scan_half_tracks(
            self._h, _dev(seeds_e, torch.float64, "seeds_e", d), Se, _dev(seeds_x, torch.float64, "seeds_x", d), Sx,
            int(charge), float(bz), float(step), int(n_steps), float(r_stop),
            _dev(wire_a, torch.float64, "wire_a", d), _dev(wire_b, torch.float64, "wire_b", d), int(wire_a.shape[1]),
            _dev(fired_wire, torch.int32, "fired_wire", d), _dev(hit_off, torch.int32, "hit_off", d),
            _dev(rho, torch.float64, "rho", d), W, H, float(cutoff),
            _dev(wire_layer, torch.int32, "wire_layer", d), _dev(circle, torch.float64, "circle", d), float(overlap),
            int(min_layers), hw.ctypes.data, ng.ctypes.data, int(n_iter), float(shrink), int(k_ref), K,
            int(work.data_ptr()), int(hs.data_ptr()), int(hr.data_ptr()), int(hok.data_ptr()), int(hcls.data_ptr()),
            int(horig.data_ptr()), counts.ctypes.data, int(out["valid"].data_ptr()), int(out["cls"].data_ptr()),
            int(out["n_cls"].data_ptr()), _stream_ptr(stream)))
        for h, key in enumerate(("ent", "ext")):
            w, hh = int(counts[2 * h]), int(counts[2 * h + 1])
            out[key] = {"final_seed": hs[h], "final_rss": hr[h], "ok": hok[h], "cls": hcls[h, :K * hh].view(K, hh),
                        "orig": horig[h, :hh], "n_fired": w}
        out["_work"] = work
        return out

    def scan_turns_half(self, seeds_e, off_e, seeds_x, off_x, charge, bz, step, n_steps, r_stop, wire_a, wire_b,
                        fired_wire, hit_off, rho, cutoff, wire_layer, circle, overlap, min_layers, half_width, n_grid,
                        n_iter, shrink, k_ref, k_final, min_wires=30, max_tracks=5, stream=None):
        """comet_scan_turns_half: the event loop of Fig. 13 with half tracks (last turn first, the best complete set's
        hits removed before the previous turn)."""
        d, td = self.device, self._tdev()
        oe = np.ascontiguousarray(np.asarray(off_e, dtype=np.int64))
        ox = np.ascontiguousarray(np.asarray(off_x, dtype=np.int64))
        hw = np.ascontiguousarray(np.asarray(half_width, dtype=np.float64))
        ng = np.ascontiguousarray(np.asarray(n_grid, dtype=np.int32))
        P, W, H = oe.shape[0] - 1, int(fired_wire.shape[0]), int(rho.shape[0])
        Se, Sx = int(seeds_e.shape[1]), int(seeds_x.shape[1])
        nb = int(self._L.comet_turns_half_work_bytes(int(np.diff(oe).max()), int(np.diff(ox).max()), W, H, int(k_ref),
                                                     int(k_final), ng.ctypes.data))
        if nb == 0:
            raise CometError("comet_turns_half_work_bytes: invalid arguments")
        work = torch.empty(nb, dtype=torch.uint8, device=td)
        out = {"turn_pair": torch.empty((P, 2), dtype=torch.int32, device=td),
               "turn_n": torch.empty(P, dtype=torch.int32, device=td),
               "turn_seed": torch.empty((P, 2, 6), dtype=torch.float64, device=td),
               "turn_cls": torch.empty((P, H), dtype=torch.uint8, device=td)}
        done = np.zeros(P, dtype=np.int32)
        wb = np.zeros(P, dtype=np.int32)
        self._check(self._L.comet_scan_turns_half(
            self._h, _dev(seeds_e, torch.float64, "seeds_e", d), oe.ctypes.data, Se,
            _dev(seeds_x, torch.float64, "seeds_x", d), ox.ctypes.data, Sx, P,
            int(charge), float(bz), float(step), int(n_steps), float(r_stop),
            _dev(wire_a, torch.float64, "wire_a", d), _dev(wire_b, torch.float64, "wire_b", d), int(wire_a.shape[1]),
            _dev(fired_wire, torch.int32, "fired_wire", d), _dev(hit_off, torch.int32, "hit_off", d),
            _dev(rho, torch.float64, "rho", d), W, H, float(cutoff),
            _dev(wire_layer, torch.int32, "wire_layer", d), _dev(circle, torch.float64, "circle", d), float(overlap),
            int(min_layers), hw.ctypes.data, ng.ctypes.data, int(n_iter), float(shrink), int(k_ref), int(k_final),
            int(min_wires), int(max_tracks), int(work.data_ptr()), int(out["turn_pair"].data_ptr()),
            int(out["turn_n"].data_ptr()), int(out["turn_seed"].data_ptr()), int(out["turn_cls"].data_ptr()),
            done.ctypes.data, wb.ctypes.data, _stream_ptr(stream)))
        out["done"], out["wires_before"] = done.astype(bool), wb
        return out

    # -- whole event, device-resident inputs --------------------------------------------------
    def scan_event(self, seeds, part_off, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire,
                   hit_off, rho, cutoff, track=None, n_pts=None, rss=None, slab_seeds=None, stream=None,
                   fused=True, z_run=0):
        """A, B and C.  fused=True (default): comet_scan_rss, the track stays on chip.  fused=False:
        comet_seed_extrapolate + comet_dca_rss through a track buffer in HBM (per slab of seeds when
        the buffer is smaller than the whole set)."""
        S = seeds.shape[1]
        if fused and track is None and slab_seeds is None:
            if rss is None:
                rss = torch.empty(S, dtype=torch.float64, device=self._tdev())
            if n_pts is None:
                n_pts = torch.empty(S, dtype=torch.int32, device=self._tdev())
            self.scan_rss(seeds, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire, hit_off, rho,
                          cutoff, rss=rss, n_pts=n_pts, stream=stream, z_run=z_run)
            out = self.select_and_classify(seeds, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire,
                                           hit_off, rho, cutoff, rss, part_off, stream=stream)
            out["rss"] = rss
            out["n_pts"] = n_pts
            return out
        if slab_seeds is None:
            slab_seeds = S
        slab_seeds = max(COMET_CHUNK, (int(slab_seeds) // COMET_CHUNK) * COMET_CHUNK)
        if rss is None:
            rss = torch.empty(S, dtype=torch.float64, device=self._tdev())
        if n_pts is None:
            n_pts = torch.empty(S, dtype=torch.int32, device=self._tdev())
        if track is None:
            track = torch.empty(self.track_bytes(min(S, slab_seeds), n_steps), dtype=torch.uint8, device=self._tdev())
        for b in range(0, S, slab_seeds):
            e = min(S, b + slab_seeds)
            self.seed_extrapolate(seeds, charge, bz, step, n_steps, r_stop, track=track, n_pts=n_pts[b:e],
                                  seed_range=(b, e), stream=stream)
            self.dca_rss(track, n_pts[b:e], seeds, charge, bz, step, n_steps, wire_a, wire_b, fired_wire,
                         hit_off, rho, cutoff, rss=rss[b:e], seed_range=(b, e), stream=stream)
        out = self.select_and_classify(seeds, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire,
                                       hit_off, rho, cutoff, rss, part_off, stream=stream)
        out["rss"] = rss
        out["n_pts"] = n_pts
        return out

    # -- whole event, host buffers ------------------------------------------------------------
    def scan_event_host(self, seeds, part_off, charge, bz, step, n_steps, r_stop, wire_a, wire_b, fired_wire,
                        hit_off, rho, cutoff, out=None, want_rss=False, track_budget_bytes=0, stream=None):
        """All arrays are HOST torch tensors (pinned for asynchronous copies) or numpy arrays."""
        def host(a, dt):
            t = a if isinstance(a, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(a))
            if t.is_cuda or t.dtype != dt or not t.is_contiguous():
                raise CometError("host array must be a contiguous CPU tensor of dtype %s" % dt)
            return t
        seeds = host(seeds, torch.float64)
        if wire_a is not None:                               # None: the geometry of set_geometry
            wire_a, wire_b = host(wire_a, torch.float64), host(wire_b, torch.float64)
        fired_wire, hit_off, rho = host(fired_wire, torch.int32), host(hit_off, torch.int32), host(rho, torch.float64)
        po = host(np.asarray(part_off, dtype=np.int64) if not isinstance(part_off, torch.Tensor) else part_off,
                  torch.int64)
        S, W, H, P = seeds.shape[1], fired_wire.shape[0], rho.shape[0], po.shape[0] - 1
        if out is None:
            out = {"best_seed": torch.empty(P, dtype=torch.int64).pin_memory(),
                   "best_rss": torch.empty(P, dtype=torch.float64).pin_memory(),
                   "best_dca": torch.empty((P, W), dtype=torch.float64).pin_memory(),
                   "cls": torch.empty((P, H), dtype=torch.uint8).pin_memory()}
            if want_rss:
                out["rss"] = torch.empty(S, dtype=torch.float64).pin_memory()
        rss_ptr = out["rss"].data_ptr() if "rss" in out else 0
        self._check(self._L.comet_scan_event_host(
            self._h, seeds.data_ptr(), S, int(charge), float(bz), float(step), int(n_steps), float(r_stop),
            wire_a.data_ptr() if wire_a is not None else 0, wire_b.data_ptr() if wire_a is not None else 0,
            int(wire_a.shape[1]) if wire_a is not None else 0, fired_wire.data_ptr(), hit_off.data_ptr(),
            rho.data_ptr(), W, H, float(cutoff), po.data_ptr(), P, int(track_budget_bytes),
            out["best_seed"].data_ptr(), out["best_rss"].data_ptr(), out["best_dca"].data_ptr(),
            out["cls"].data_ptr(), rss_ptr, _stream_ptr(stream)))
        return out

    # -- seed grids as inputs -------------------------------------------------------------------
    def grid_z_run(self, n_z: int) -> int:
        return int(self._L.comet_grid_z_run(int(n_z)))

    def seed_grid(self, axes, shape, seeds=None, stream=None):
        """comet_seed_grid: axes CUDA float64 [P][A], shape = (n_p, n_ct, n_phi, n_z) -> seeds [6][P G] (device)."""
        n_p, n_ct, n_phi, n_z = (int(v) for v in shape)
        A = int(self._L.comet_grid_axes_len(n_p, n_ct, n_phi, n_z))
        if A == 0 or axes.dim() != 2 or axes.shape[1] != A:
            raise CometError("axes must be [n_part][%d] for this grid shape" % A)
        P = int(axes.shape[0])
        S = P * n_p * n_ct * n_phi * n_z
        if seeds is None:
            seeds = torch.empty((6, S), dtype=torch.float64, device=self._tdev())
        self._check(self._L.comet_seed_grid(self._h, _dev(axes, torch.float64, "axes", self.device), P, n_p, n_ct, n_phi,
                                            n_z, _dev(seeds, torch.float64, "seeds", self.device), int(seeds.shape[1]),
                                            _stream_ptr(stream)))
        return seeds

    def seed_runs(self, seeds, stream=None) -> int:
        """comet_seed_runs: the z_run of a seed set (synchronises)."""
        v = ctypes.c_int32()
        self._check(self._L.comet_seed_runs(self._h, _dev(seeds, torch.float64, "seeds", self.device), int(seeds.shape[1]),
                                            int(seeds.shape[1]), ctypes.byref(v), _stream_ptr(stream)))
        return int(v.value)

    def set_geometry(self, wire_a, wire_b, stream=None):
        """comet_set_geometry: HOST arrays [3][n_wires]; returns the device copies as CUDA tensors' addresses."""
        wa = torch.from_numpy(np.ascontiguousarray(np.asarray(wire_a, dtype=np.float64)))
        wb = torch.from_numpy(np.ascontiguousarray(np.asarray(wire_b, dtype=np.float64)))
        self._check(self._L.comet_set_geometry(self._h, wa.data_ptr(), wb.data_ptr(), int(wa.shape[1]), _stream_ptr(stream)))

    def scan_event_grid_host(self, axes, shape, charge, bz, step, n_steps, r_stop, fired_wire, hit_off, rho, cutoff,
                             out=None, want_rss=False, stream=None):
        """comet_scan_event_grid_host: axes HOST [P][A] (pinned for asynchronous copies), the event's hits HOST."""
        def host(a, dt):
            t = a if isinstance(a, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(a))
            if t.is_cuda or t.dtype != dt or not t.is_contiguous():
                raise CometError("host array must be a contiguous CPU tensor of dtype %s" % dt)
            return t
        axes = host(axes, torch.float64)
        fired_wire, hit_off, rho = host(fired_wire, torch.int32), host(hit_off, torch.int32), host(rho, torch.float64)
        n_p, n_ct, n_phi, n_z = (int(v) for v in shape)
        P, W, H = int(axes.shape[0]), int(fired_wire.shape[0]), int(rho.shape[0])
        S = P * n_p * n_ct * n_phi * n_z
        if out is None:
            out = {"best_seed": torch.empty(P, dtype=torch.int64).pin_memory(),
                   "best_rss": torch.empty(P, dtype=torch.float64).pin_memory(),
                   "best_dca": torch.empty((P, W), dtype=torch.float64).pin_memory(),
                   "cls": torch.empty((P, H), dtype=torch.uint8).pin_memory()}
            if want_rss:
                out["rss"] = torch.empty(S, dtype=torch.float64).pin_memory()
        rss_ptr = out["rss"].data_ptr() if "rss" in out else 0
        self._check(self._L.comet_scan_event_grid_host(
            self._h, axes.data_ptr(), P, n_p, n_ct, n_phi, n_z, int(charge), float(bz), float(step), int(n_steps),
            float(r_stop), fired_wire.data_ptr(), hit_off.data_ptr(), rho.data_ptr(), W, H, float(cutoff),
            out["best_seed"].data_ptr(), out["best_rss"].data_ptr(), out["best_dca"].data_ptr(),
            out["cls"].data_ptr(), rss_ptr, _stream_ptr(stream)))
        return out

    def scan_event_grid_submit(self, slot, axes, shape, charge, bz, step, n_steps, r_stop, fired_wire, hit_off, rho, cutoff,
                               stream=None):
        """comet_scan_event_grid_submit: enqueue one event (HOST arrays, copied before the call returns) into `slot`."""
        def host(a, dt):
            t = a if isinstance(a, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(a))
            if t.is_cuda or t.dtype != dt or not t.is_contiguous():
                raise CometError("host array must be a contiguous CPU tensor of dtype %s" % dt)
            return t
        axes = host(axes, torch.float64)
        fired_wire, hit_off, rho = host(fired_wire, torch.int32), host(hit_off, torch.int32), host(rho, torch.float64)
        n_p, n_ct, n_phi, n_z = (int(v) for v in shape)
        P, W, H = int(axes.shape[0]), int(fired_wire.shape[0]), int(rho.shape[0])
        self._check(self._L.comet_scan_event_grid_submit(
            self._h, int(slot), axes.data_ptr(), P, n_p, n_ct, n_phi, n_z, int(charge), float(bz), float(step), int(n_steps),
            float(r_stop), fired_wire.data_ptr(), hit_off.data_ptr(), rho.data_ptr(), W, H, float(cutoff), _stream_ptr(stream)))
        return (P, W, H)

    def scan_event_grid_collect(self, slot, sizes, out=None):
        """comet_scan_event_grid_collect: wait for the event in `slot`; `sizes` is what the submit returned."""
        P, W, H = sizes
        if out is None:
            out = {"best_seed": torch.empty(P, dtype=torch.int64), "best_rss": torch.empty(P, dtype=torch.float64),
                   "best_dca": torch.empty((P, W), dtype=torch.float64), "cls": torch.empty((P, H), dtype=torch.uint8)}
        self._check(self._L.comet_scan_event_grid_collect(
            self._h, int(slot), out["best_seed"].data_ptr(), out["best_rss"].data_ptr(), out["best_dca"].data_ptr(),
            out["cls"].data_ptr()))
        return out

    # -- measurement helper -------------------------------------------------------------------
    def fp64_peak_probe(self, iters: int, sink=None, stream=None) -> float:
        """Enqueues the DFMA loop; returns the number of FP64 FMA instructions (thread-level) it runs."""
        if sink is None:
            sink = torch.zeros(1, dtype=torch.float64, device=self._tdev())
        self._sink = sink
        n = ctypes.c_double()
        self._check(self._L.comet_fp64_peak_probe(self._h, int(iters), int(sink.data_ptr()), ctypes.byref(n),
                                                  _stream_ptr(stream)))
        return n.value
