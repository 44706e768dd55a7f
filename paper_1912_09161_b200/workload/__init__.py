"""Seeded synthetic inputs: geometry G0, event generator, raw-bank packer.

Input generation only — none of the reconstruction arithmetic lives here.  Both the CPU oracle
(`oracle/`) and the CUDA path consume what this module produces; neither shares code with it.
Recipe and citations: DESIGN.md "Input recipe" (BASELINE.json `configs`;
PAPER.md:96 for nu=6, PAPER.md:165 for 26 planes, PAPER.md:240 for 2<eta<5).
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "velo_gen.cpp")
_LIB = os.path.join(_HERE, "_velo_gen.so")

BASE_SEED = 0x19120916


def build(force: bool = False) -> str:
    """Compile the generator (g++) next to its source if missing or stale."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


# ----------------------------------------------------------------------------------------------
# Geometry G0 (VELO-like, not the real survey): 26 stations x (right, left) module x 2 sensors.
# ----------------------------------------------------------------------------------------------

STATION_Z = np.array(
    [-290.0, -265.0, -240.0, -215.0]
    + [-150.0 + 25.0 * i for i in range(18)]
    + [350.0, 450.0, 600.0, 737.5]
)
N_COLS, N_ROWS, PITCH_MM = 768, 256, 0.055
HALF_GAP_MM = 4.0  # square beam hole |x|,|y| < 4 mm
LEFT_DZ_MM = 12.5


@dataclass
class Geometry:
    """Host description of the detector handed to `allen_velo_create` and to the oracle."""

    n_sensors: int
    n_modules: int
    n_layers: int
    n_cols: int
    n_rows: int
    pitch_mm: float
    sensor_module: np.ndarray  # u16 [n_sensors]
    module_layer: np.ndarray  # u16 [n_modules]
    sensor_ltg: np.ndarray  # f32 [n_sensors, 9] row-major local->global
    # generator-side (double precision) description of the same sensors
    sensor_frame: np.ndarray = field(repr=False, default=None)  # f64 [n_sensors, 7]: ox, oy, ecx, ecy, erx, ery, z

    def sensor_layer(self) -> np.ndarray:
        return self.module_layer[self.sensor_module]


def geometry_g0() -> Geometry:
    return _pinwheel_stations(STATION_Z, LEFT_DZ_MM)


def _pinwheel_stations(station_z, left_dz) -> Geometry:
    # (origin, e_col, e_row) of the four pinwheel sensors of a station: R0, R1 (right module), L0, L1 (left).
    g = HALF_GAP_MM
    frames = [
        ((-g, g), (1.0, 0.0), (0.0, 1.0)),  # R0: col -> +x, row -> +y
        ((g, g), (0.0, -1.0), (1.0, 0.0)),  # R1: col -> -y, row -> +x
        ((g, -g), (-1.0, 0.0), (0.0, -1.0)),  # L0: col -> -x, row -> -y
        ((-g, -g), (0.0, 1.0), (-1.0, 0.0)),  # L1: col -> +y, row -> -x
    ]
    n_st = len(station_z)
    n_modules, n_sensors = 2 * n_st, 4 * n_st
    sensor_module = np.zeros(n_sensors, np.uint16)
    module_layer = np.zeros(n_modules, np.uint16)
    ltg = np.zeros((n_sensors, 9), np.float32)
    frame = np.zeros((n_sensors, 7), np.float64)
    for k in range(n_st):
        for side in range(2):
            m = 2 * k + side
            module_layer[m] = k
            zm = station_z[k] + (left_dz if side else 0.0)
            for j in range(2):
                s = 2 * m + j
                (ox, oy), (ecx, ecy), (erx, ery) = frames[2 * side + j]
                sensor_module[s] = m
                ltg[s] = [ecx, erx, ox, ecy, ery, oy, 0.0, 0.0, zm]
                frame[s] = [ox, oy, ecx, ecy, erx, ery, zm]
    return Geometry(n_sensors, n_modules, n_st, N_COLS, N_ROWS, PITCH_MM, sensor_module, module_layer, ltg, frame)


def geometry_variant(kind: str) -> Geometry:
    """Other detector descriptions the C ABI admits (include/allen_velo.h: 3 <= n_layers <= 64, at most 8 sensors per
    layer, other sensor sizes), built from G0's sensor frames; for tests beyond the one geometry the benchmarks use.

    "g52": 52 stations (G0's and one more 12.5 mm behind each, left modules 5 mm behind the right ones): 52 layers;
    "g13": two stations per layer (13 layers of 8 sensors at four different z);
    "coarse": G0 with sensors of 384 x 128 pixels of 0.11 mm (same area, a quarter of the pixels);
    "shuffled": G0 with the sensors (= raw banks) numbered in a fixed random order, so that the banks of a layer's
                sensors are scattered over the raw event instead of following one another.
    """
    g = geometry_g0()
    if kind == "g52":
        g = _pinwheel_stations(np.sort(np.concatenate([STATION_Z, STATION_Z + 12.5])), 5.0)
    elif kind == "g13":
        g.module_layer = (np.arange(g.n_modules, dtype=np.uint16) // 4).astype(np.uint16)
        g.n_layers = g.n_modules // 4
    elif kind == "coarse":
        g.n_cols, g.n_rows, g.pitch_mm = N_COLS // 2, N_ROWS // 2, 2.0 * PITCH_MM
    elif kind == "shuffled":
        perm = np.random.default_rng(20191209).permutation(g.n_sensors)  # new sensor i is G0's sensor perm[i]
        g.sensor_module = np.ascontiguousarray(g.sensor_module[perm])
        g.sensor_ltg = np.ascontiguousarray(g.sensor_ltg[perm])
        g.sensor_frame = np.ascontiguousarray(g.sensor_frame[perm])
    else:
        raise ValueError(kind)
    return g


# ----------------------------------------------------------------------------------------------
# Event generator
# ----------------------------------------------------------------------------------------------


class _Config(ctypes.Structure):
    _fields_ = [
        ("seed", ctypes.c_uint64),
        ("first_event", ctypes.c_uint64),
        ("n_events", ctypes.c_uint32),
        ("fixed_pv", ctypes.c_int32),
        ("nu", ctypes.c_double),
        ("fixed_tracks", ctypes.c_int32),
        ("mean_tracks", ctypes.c_double),
        ("noise_occ", ctypes.c_double),
        ("hit_eff", ctypes.c_double),
        ("charge_sharing", ctypes.c_int32),
        ("scatter_sigma", ctypes.c_double),
        ("displaced_frac", ctypes.c_double),
        ("displaced_mean", ctypes.c_double),
        ("isolate", ctypes.c_int32),
        ("shuffle_sp", ctypes.c_int32),
        ("n_sensors", ctypes.c_uint32),
        ("n_modules", ctypes.c_uint32),
        ("n_cols", ctypes.c_uint32),
        ("n_rows", ctypes.c_uint32),
        ("pitch", ctypes.c_double),
    ]


# BASELINE.json configs 0..3 (config 4 = config 2's generator at several batch sizes).
CONFIGS = {
    0: dict(n_events=16, fixed_pv=1, fixed_tracks=20, noise_occ=0.0, hit_eff=1.0, charge_sharing=0,
            scatter_sigma=0.0, displaced_frac=0.0, isolate=1, nu=1.0),
    1: dict(n_events=1000, nu=6.0, noise_occ=1e-4, hit_eff=0.99, charge_sharing=1,
            scatter_sigma=0.0, displaced_frac=0.0),
    2: dict(n_events=10000, nu=6.0, noise_occ=1e-4, hit_eff=0.99, charge_sharing=1,
            scatter_sigma=1e-4, displaced_frac=0.1),
    3: dict(n_events=10000, nu=12.0, noise_occ=2e-4, hit_eff=0.99, charge_sharing=1,
            scatter_sigma=1e-4, displaced_frac=0.1),
}


@dataclass
class Batch:
    """One generated batch: raw bytes + offsets (the method's input) and the generator truth."""

    config: int
    seed: int
    geometry: Geometry
    raw: np.ndarray  # u8, 16-byte multiples per event
    event_offsets: np.ndarray  # u32 [n_events+1], bytes
    particles: dict  # arrays per particle
    pixels: dict  # arrays per (pixel, source)
    pvs: dict

    @property
    def n_events(self) -> int:
        return len(self.event_offsets) - 1

    def sha(self) -> str:
        h = hashlib.sha256()
        h.update(self.event_offsets.tobytes())
        h.update(self.raw.tobytes())
        return h.hexdigest()[:16]

    def n_sp_words(self) -> int:
        """Total super-pixel words in the batch (read from the event headers)."""
        w = self.raw.view(np.uint32)
        return int(w[(self.event_offsets[:-1] // 4) + 2].sum())

    def select(self, events) -> "Batch":
        """A new batch holding the given events (by index, any order); truth is re-indexed."""
        events = np.asarray(events, dtype=np.int64)
        parts = [self.raw[self.event_offsets[e]:self.event_offsets[e + 1]] for e in events]
        sizes = np.array([len(p) for p in parts], dtype=np.uint64)
        off = np.zeros(len(events) + 1, np.uint32)
        off[1:] = np.cumsum(sizes)
        raw = np.concatenate(parts) if parts else np.zeros(0, np.uint8)
        remap = -np.ones(self.n_events, np.int64)
        remap[events] = np.arange(len(events))

        def sub(table, key):
            keep = remap[table[key]] >= 0
            out = {k: v[keep].copy() for k, v in table.items()}
            out[key] = remap[out[key]].astype(np.uint32)
            return out, keep

        pixels, _ = sub(self.pixels, "event")
        particles, keep_p = sub(self.particles, "event")
        new_pid = -np.ones(len(keep_p) + 1, np.int64)  # last slot serves particle == -1
        new_pid[:-1][keep_p] = np.arange(int(keep_p.sum()))
        pixels["particle"] = new_pid[pixels["particle"]].astype(np.int32)
        pvs, _ = sub(self.pvs, "event")
        return Batch(self.config, self.seed, self.geometry, raw, off, particles, pixels, pvs)


def generate(config: int, n_events: int | None = None, batch_index: int = 0, first_event: int = 0,
             geometry: Geometry | None = None, shuffle_sp: bool = True, **overrides) -> Batch:
    """Generate one batch of BASELINE.json config `config` (0..3).

    seed = 0x19120916 + 1000*config + batch_index; every event owns the Philox stream `first_event + e`.
    """
    geo = geometry or geometry_g0()
    lib = ctypes.CDLL(build())
    lib.velo_gen_run.restype = ctypes.c_void_p
    lib.velo_gen_run.argtypes = [ctypes.POINTER(_Config), ctypes.c_void_p, ctypes.c_void_p]
    lib.velo_gen_free.argtypes = [ctypes.c_void_p]
    lib.velo_gen_size.restype = ctypes.c_uint64
    lib.velo_gen_size.argtypes = [ctypes.c_void_p, ctypes.c_int]
    lib.velo_gen_ptr.restype = ctypes.c_void_p
    lib.velo_gen_ptr.argtypes = [ctypes.c_void_p, ctypes.c_int]

    p = dict(CONFIGS[config])
    p.update(overrides)
    if n_events is not None:
        p["n_events"] = n_events
    seed = BASE_SEED + 1000 * config + batch_index
    cfg = _Config(
        seed=seed, first_event=first_event, n_events=p["n_events"],
        fixed_pv=p.get("fixed_pv", 0), nu=p["nu"], fixed_tracks=p.get("fixed_tracks", 0),
        mean_tracks=p.get("mean_tracks", 25.0), noise_occ=p["noise_occ"], hit_eff=p["hit_eff"],
        charge_sharing=p["charge_sharing"], scatter_sigma=p["scatter_sigma"],
        displaced_frac=p["displaced_frac"], displaced_mean=p.get("displaced_mean", 5.0),
        isolate=p.get("isolate", 0), shuffle_sp=int(shuffle_sp),
        n_sensors=geo.n_sensors, n_modules=geo.n_modules, n_cols=geo.n_cols, n_rows=geo.n_rows,
        pitch=geo.pitch_mm,
    )
    frame = np.ascontiguousarray(geo.sensor_frame, np.float64)
    smod = np.ascontiguousarray(geo.sensor_module, np.uint16)
    h = lib.velo_gen_run(ctypes.byref(cfg), frame.ctypes.data, smod.ctypes.data)
    try:
        def arr(what, dtype, count):
            if count == 0:
                return np.zeros(0, dtype)
            ptr = lib.velo_gen_ptr(h, what)
            buf = (ctypes.c_char * (count * np.dtype(dtype).itemsize)).from_address(ptr)
            return np.frombuffer(buf, dtype=dtype).copy()

        n_raw, n_off = lib.velo_gen_size(h, 0), lib.velo_gen_size(h, 1)
        n_p, n_x, n_v = lib.velo_gen_size(h, 2), lib.velo_gen_size(h, 3), lib.velo_gen_size(h, 4)
        raw = arr(0, np.uint8, n_raw)
        off = arr(1, np.uint32, n_off)
        particles = dict(
            event=arr(10, np.uint32, n_p), pv=arr(11, np.int32, n_p), displaced=arr(12, np.uint8, n_p),
            ox=arr(13, np.float64, n_p), oy=arr(14, np.float64, n_p), oz=arr(15, np.float64, n_p),
            tx=arr(16, np.float64, n_p), ty=arr(17, np.float64, n_p),
            n_crossings=arr(18, np.uint32, n_p), n_hits=arr(19, np.uint32, n_p),
        )
        pixels = dict(
            event=arr(20, np.uint32, n_x), sensor=arr(21, np.uint16, n_x), col=arr(22, np.uint16, n_x),
            row=arr(23, np.uint16, n_x), particle=arr(24, np.int32, n_x), main=arr(25, np.uint8, n_x),
        )
        pvs = dict(event=arr(30, np.uint32, n_v), x=arr(31, np.float64, n_v), y=arr(32, np.float64, n_v),
                   z=arr(33, np.float64, n_v))
    finally:
        lib.velo_gen_free(h)
    return Batch(config, seed, geo, raw, off, particles, pixels, pvs)


def pack_events(geometry: Geometry, events: list[list[tuple[int, int, int]]], shuffle_seed: int | None = None):
    """Pack hand-made events (lists of (sensor, col, row) fired pixels) into raw format v1.

    Pure-Python twin of the C++ packer for tests that need specific pixel patterns.
    Returns (raw u8 array, event_offsets u32 array).
    """
    rng = np.random.default_rng(shuffle_seed) if shuffle_seed is not None else None
    chunks, offsets = [], [0]
    for pix in events:
        banks: list[dict[tuple[int, int], int]] = [dict() for _ in range(geometry.n_sensors)]
        for s, c, r in pix:
            key = (c >> 1, r >> 2)
            banks[s][key] = banks[s].get(key, 0) | (1 << (4 * (c & 1) + (r & 3)))
        words = [0x56454C4F, geometry.n_sensors, sum(len(b) for b in banks), 0]
        off = 0
        for b in banks:
            words.append(off)
            off += len(b)
        words.append(off)
        while len(words) % 4:
            words.append(0)
        for b in banks:
            sp = [((spc << 14) | (spr << 8) | hm) for (spc, spr), hm in sorted(b.items())]
            if rng is not None:
                sp = list(rng.permutation(np.array(sp, dtype=np.uint64)).astype(np.uint64)) if sp else sp
            words.extend(int(w) for w in sp)
        while len(words) % 4:
            words.append(0)
        a = np.array(words, dtype=np.uint32)
        chunks.append(a.view(np.uint8))
        offsets.append(offsets[-1] + a.nbytes)
    raw = np.concatenate(chunks) if chunks else np.zeros(0, np.uint8)
    return raw, np.array(offsets, dtype=np.uint32)
