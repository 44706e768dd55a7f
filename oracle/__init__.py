"""ORACLE — TEST INFRASTRUCTURE ONLY (ctypes wrapper of oracle/velo_oracle.cpp).

Only tests/, `__graft_entry__.smoke()` and bench.py's `cpu_baseline` / `--impl reference` legs may import this
package.  It shares nothing with `paper_1912_09161_b200/csrc` and never imports the CUDA binding.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "velo_oracle.cpp")
_LIB = os.path.join(_HERE, "_velo_oracle.so")

# Default cuts (reading R5).
DEFAULT_PARAMS = dict(w_seed_phi16=512, w_fwd_phi16=512, max_slope=0.4, s_seed=2.0 ** -6, s_fwd=2.0 ** -4,
                      s_weak=2.0 ** -7, max_skipped=1)

STATUS_BAD_HEADER, STATUS_BAD_SP, STATUS_TOO_MANY_CLUSTERS = 1, 2, 4


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-shared", "-fPIC", "-pthread",
                               "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


class _Params(ctypes.Structure):
    _fields_ = [("w_seed_phi16", ctypes.c_int32), ("w_fwd_phi16", ctypes.c_int32), ("max_slope", ctypes.c_float),
                ("s_seed", ctypes.c_float), ("s_fwd", ctypes.c_float), ("s_weak", ctypes.c_float),
                ("max_skipped", ctypes.c_int32)]


class _Geometry(ctypes.Structure):
    _fields_ = [("n_sensors", ctypes.c_uint32), ("n_modules", ctypes.c_uint32), ("n_layers", ctypes.c_uint32),
                ("n_cols", ctypes.c_uint32), ("n_rows", ctypes.c_uint32), ("pitch_mm", ctypes.c_float),
                ("sensor_module", ctypes.c_void_p), ("module_layer", ctypes.c_void_p),
                ("sensor_ltg", ctypes.c_void_p), ("params", _Params)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        L.oracle_mix32.restype = ctypes.c_uint32
        L.oracle_mix32.argtypes = [ctypes.c_uint32]
        L.oracle_atan2_poly.restype = ctypes.c_float
        L.oracle_atan2_poly.argtypes = [ctypes.c_float, ctypes.c_float]
        L.oracle_phi16.restype = ctypes.c_int32
        L.oracle_phi16.argtypes = [ctypes.c_float, ctypes.c_float]
        L.oracle_scatter.restype = ctypes.c_float
        L.oracle_scatter.argtypes = [ctypes.c_void_p] * 3
        L.oracle_fit.argtypes = [ctypes.c_uint32] + [ctypes.c_void_p] * 4
        L.oracle_kalman.argtypes = [ctypes.c_uint32] + [ctypes.c_void_p] * 5 + [ctypes.c_double, ctypes.c_void_p]
        L.oracle_pvs.argtypes = [ctypes.c_uint32] + [ctypes.c_void_p] * 9 + [ctypes.c_int]
        L.oracle_pv_candidates.restype = ctypes.c_uint32
        L.oracle_pv_candidates.argtypes = [ctypes.c_uint32] + [ctypes.c_void_p] * 8 + [ctypes.c_uint32]
        L.oracle_run.restype = ctypes.c_void_p
        L.oracle_run.argtypes = [ctypes.POINTER(_Geometry), ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint32,
                                 ctypes.c_uint32]
        L.oracle_run_hits.restype = ctypes.c_void_p
        L.oracle_run_hits.argtypes = [ctypes.POINTER(_Params), ctypes.c_uint32] + [ctypes.c_void_p] * 4 + [
            ctypes.c_uint32, ctypes.c_void_p]
        L.oracle_set_cluster_regions.argtypes = [ctypes.c_uint32, ctypes.c_uint32]
        L.oracle_free.argtypes = [ctypes.c_void_p]
        L.oracle_total.restype = ctypes.c_uint64
        L.oracle_total.argtypes = [ctypes.c_void_p, ctypes.c_int]
        L.oracle_export_clusters.argtypes = [ctypes.c_void_p, ctypes.c_uint32] + [ctypes.c_void_p] * 12
        L.oracle_export_tracks.argtypes = [ctypes.c_void_p] + [ctypes.c_void_p] * 7
        L.oracle_export_pixels.argtypes = [ctypes.c_void_p] + [ctypes.c_void_p] * 3
        L.oracle_export_near_cut.argtypes = [ctypes.c_void_p] + [ctypes.c_void_p] * 3
        _lib = L
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data


def make_params(params: dict | None = None) -> _Params:
    d = dict(DEFAULT_PARAMS)
    if params:
        d.update(params)
    return _Params(**d)


@dataclass
class Clusters:
    """Compacted SoA cluster output in the C-ABI layout (include/allen_velo.h)."""

    event_offsets: np.ndarray
    layer_offsets: np.ndarray
    key: np.ndarray
    n_pixels: np.ndarray
    sum_col: np.ndarray
    sum_row: np.ndarray
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    phi16: np.ndarray
    checksum: np.ndarray
    status: np.ndarray


@dataclass
class Tracks:
    event_offsets: np.ndarray
    hit_offsets: np.ndarray
    hits: np.ndarray
    x0: np.ndarray
    y0: np.ndarray
    tx: np.ndarray
    ty: np.ndarray

    def hit_sets(self, e: int) -> list[tuple[int, ...]]:
        """Canonical form of event e's tracks: sorted list of sorted hit tuples."""
        t0, t1 = int(self.event_offsets[e]), int(self.event_offsets[e + 1])
        return sorted(tuple(sorted(int(h) for h in self.hits[self.hit_offsets[t]:self.hit_offsets[t + 1]]))
                      for t in range(t0, t1))


@dataclass
class Result:
    clusters: Clusters
    tracks: Tracks
    near_cut_per_event: np.ndarray
    near_cut_hit_event: np.ndarray
    near_cut_hit_index: np.ndarray
    pix_event: np.ndarray | None = None
    pix_key: np.ndarray | None = None
    pix_cluster: np.ndarray | None = None


def _export(L, h, n_events: int, n_layers: int, with_pixels: bool) -> Result:
    nc, nt, nh = L.oracle_total(h, 0), L.oracle_total(h, 1), L.oracle_total(h, 2)
    npix, nnc = L.oracle_total(h, 3), L.oracle_total(h, 4)
    u32, f32 = np.uint32, np.float32
    c = Clusters(np.zeros(n_events + 1, u32), np.zeros(n_events * n_layers + 1, u32), np.zeros(nc, u32),
                 np.zeros(nc, u32), np.zeros(nc, u32), np.zeros(nc, u32), np.zeros(nc, f32), np.zeros(nc, f32),
                 np.zeros(nc, f32), np.zeros(nc, np.int16), np.zeros(nc, u32), np.zeros(n_events, u32))
    L.oracle_export_clusters(h, n_layers, _p(c.event_offsets), _p(c.layer_offsets), _p(c.key), _p(c.n_pixels),
                             _p(c.sum_col), _p(c.sum_row), _p(c.x), _p(c.y), _p(c.z), _p(c.phi16), _p(c.checksum),
                             _p(c.status))
    t = Tracks(np.zeros(n_events + 1, u32), np.zeros(nt + 1, u32), np.zeros(nh, np.uint16), np.zeros(nt, f32),
               np.zeros(nt, f32), np.zeros(nt, f32), np.zeros(nt, f32))
    L.oracle_export_tracks(h, _p(t.event_offsets), _p(t.hit_offsets), _p(t.hits), _p(t.x0), _p(t.y0), _p(t.tx),
                           _p(t.ty))
    nce, nhe, nhi = np.zeros(n_events, u32), np.zeros(nnc, u32), np.zeros(nnc, u32)
    L.oracle_export_near_cut(h, _p(nce), _p(nhe), _p(nhi))
    res = Result(c, t, nce, nhe, nhi)
    if with_pixels:
        res.pix_event, res.pix_key, res.pix_cluster = np.zeros(npix, u32), np.zeros(npix, u32), np.zeros(npix, u32)
        L.oracle_export_pixels(h, _p(res.pix_event), _p(res.pix_key), _p(res.pix_cluster))
    return res


def reconstruct(geometry, raw: np.ndarray, event_offsets: np.ndarray, params: dict | None = None,
                n_threads: int = 1, with_pixels: bool = False, export: bool = True,
                cluster_regions: tuple[int, int] = (0, 0)) -> Result | None:
    """Run the oracle over a batch.  `geometry` is a workload.Geometry-like object (duck-typed).
    cluster_regions = (sp_cols, sp_rows): the local clustering variant of P:179 (R11): clusters are the
    connected components inside regions of that many super-pixels; (0, 0) = exact connected components."""
    L = lib()
    L.oracle_set_cluster_regions(int(cluster_regions[0]), int(cluster_regions[1]))
    smod = np.ascontiguousarray(geometry.sensor_module, np.uint16)
    mlay = np.ascontiguousarray(geometry.module_layer, np.uint16)
    ltg = np.ascontiguousarray(geometry.sensor_ltg, np.float32)
    g = _Geometry(geometry.n_sensors, geometry.n_modules, geometry.n_layers, geometry.n_cols, geometry.n_rows,
                  geometry.pitch_mm, _p(smod), _p(mlay), _p(ltg), make_params(params))
    raw = np.ascontiguousarray(raw, np.uint8)
    off = np.ascontiguousarray(event_offsets, np.uint32)
    n_events = len(off) - 1
    h = L.oracle_run(ctypes.byref(g), _p(raw), _p(off), n_events, n_threads)
    try:
        return _export(L, h, n_events, geometry.n_layers, with_pixels) if export else None
    finally:
        L.oracle_free(h)
        L.oracle_set_cluster_regions(0, 0)


def search_hits(x, y, z, phi16, layer_offsets, params: dict | None = None) -> Result:
    """O5 + O6 on caller-given hits of one event (already in normative order)."""
    L = lib()
    x, y, z = (np.ascontiguousarray(a, np.float32) for a in (x, y, z))
    phi16 = np.ascontiguousarray(phi16, np.int16)
    lo = np.ascontiguousarray(layer_offsets, np.uint32)
    P = make_params(params)
    h = L.oracle_run_hits(ctypes.byref(P), len(x), _p(x), _p(y), _p(z), _p(phi16), len(lo) - 1, _p(lo))
    try:
        return _export(L, h, 1, len(lo) - 1, False)
    finally:
        L.oracle_free(h)


def phi16(x: float, y: float) -> int:
    return int(lib().oracle_phi16(x, y))


def atan2_poly(x: float, y: float) -> float:
    return float(lib().oracle_atan2_poly(x, y))


def mix32(v: int) -> int:
    return int(lib().oracle_mix32(v))


def scatter(a, b, c) -> float:
    a, b, c = (np.ascontiguousarray(v, np.float32) for v in (a, b, c))
    return float(lib().oracle_scatter(_p(a), _p(b), _p(c)))


def fit(x, y, z) -> np.ndarray:
    x, y, z = (np.ascontiguousarray(a, np.float32) for a in (x, y, z))
    out = np.zeros(4, np.float32)
    lib().oracle_fit(len(x), _p(x), _p(y), _p(z), _p(out))
    return out


def kalman(hit_offsets, abs_hits, x, y, z, pitch: float) -> np.ndarray:
    """O7 (R9): simple Kalman fit of every track; hits are indices into x, y, z, in order of addition.
    Returns [n_tracks, 12] float64: x, y, tx, ty, z, chi2, C00x, C01x, C11x, C00y, C01y, C11y at the last hit."""
    ho = np.ascontiguousarray(hit_offsets, np.uint32)
    hits = np.ascontiguousarray(abs_hits, np.uint32)
    x, y, z = (np.ascontiguousarray(a, np.float32) for a in (x, y, z))
    out = np.zeros((len(ho) - 1, 12), np.float64)
    lib().oracle_kalman(len(ho) - 1, _p(ho), _p(hits), _p(x), _p(y), _p(z), float(pitch), _p(out))
    return out


def kalman_of(result: "Result", pitch: float) -> np.ndarray:
    """O7 for every track of an oracle.Result (event-local hit indices resolved to absolute cluster indices)."""
    t, c = result.tracks, result.clusters
    n_per_event = np.diff(t.event_offsets.astype(np.int64))
    ev_of_track = np.repeat(np.arange(len(n_per_event)), n_per_event)
    ev_of_hit = np.repeat(ev_of_track, np.diff(t.hit_offsets.astype(np.int64)))
    abs_hits = c.event_offsets[ev_of_hit].astype(np.int64) + t.hits
    return kalman(t.hit_offsets, abs_hits, c.x, c.y, c.z, pitch)


PV_MAX = 32


def find_pvs(track_offsets, x0, y0, tx, ty, kal, iterations: int = 8):
    """O8 (R10): primary vertices per event from the straight-line fit (seeding histogram) and the Kalman
    states (weighted fit).  Returns (vertices [n_events, 32, 8] float64, counts [n_events], candidates [n_events])."""
    to = np.ascontiguousarray(track_offsets, np.uint32)
    x0, y0, tx, ty = (np.ascontiguousarray(a, np.float32) for a in (x0, y0, tx, ty))
    kal = np.ascontiguousarray(kal, np.float64)
    n = len(to) - 1
    out = np.zeros((n, PV_MAX, 8), np.float64)
    counts, cands = np.zeros(n, np.uint32), np.zeros(n, np.uint32)
    lib().oracle_pvs(n, _p(to), _p(x0), _p(y0), _p(tx), _p(ty), _p(kal), _p(out), _p(counts), _p(cands), iterations)
    return out, counts, cands


def pv_candidates(x0, y0, tx, ty, kal, cap: int = 300):
    """O8 for ONE event with every candidate as it stands before the duplicate removal of step 4 (R10).
    Returns (vertices [n, 8], candidates [m, 6]: z_seed, x, y, z, sum_w, ok)."""
    x0, y0, tx, ty = (np.ascontiguousarray(a, np.float32) for a in (x0, y0, tx, ty))
    kal = np.ascontiguousarray(kal, np.float64)
    out, cand, m = np.zeros((PV_MAX, 8), np.float64), np.zeros((cap, 6), np.float64), ctypes.c_uint32(0)
    n = lib().oracle_pv_candidates(len(x0), _p(x0), _p(y0), _p(tx), _p(ty), _p(kal), _p(out), ctypes.byref(m), _p(cand),
                                   cap)
    return out[:n], cand[:min(m.value, cap)]


def pvs_of(result: "Result", pitch: float):
    t = result.tracks
    return find_pvs(t.event_offsets, t.x0, t.y0, t.tx, t.ty, kalman_of(result, pitch))
