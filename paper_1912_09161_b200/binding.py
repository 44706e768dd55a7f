"""Thin ctypes binding of the C ABI in include/allen_velo.h — argument marshalling only.

Same names as the C entry points.  PyTorch supplies device memory and streams; every step of the path runs in the
CUDA kernels of `csrc/`.  There is no CPU fallback: a missing shared object or a missing CUDA device raises.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("ALLEN_VELO_LIB") or os.path.join(_HERE, "_allen_velo.so")  # override: an alternative build

OK, ERR_INVALID, ERR_CUDA, ERR_WORKSPACE = 0, -1, -2, -3
STATUS_BAD_HEADER, STATUS_BAD_SP, STATUS_TOO_MANY_CLUSTERS = 1, 2, 4
STATUS_CLUSTER_CAPACITY, STATUS_TRACK_CAPACITY, STATUS_STAGE_OVERFLOW = 8, 16, 32


class allen_velo_params_t(ctypes.Structure):
    _fields_ = [("w_seed_phi16", ctypes.c_int32), ("w_fwd_phi16", ctypes.c_int32), ("max_slope", ctypes.c_float),
                ("s_seed", ctypes.c_float), ("s_fwd", ctypes.c_float), ("s_weak", ctypes.c_float),
                ("max_skipped", ctypes.c_int32)]


class allen_velo_geometry_t(ctypes.Structure):
    _fields_ = [("n_sensors", ctypes.c_uint32), ("n_modules", ctypes.c_uint32), ("n_layers", ctypes.c_uint32),
                ("n_cols", ctypes.c_uint32), ("n_rows", ctypes.c_uint32), ("pitch_mm", ctypes.c_float),
                ("sensor_module", ctypes.c_void_p), ("module_layer", ctypes.c_void_p),
                ("sensor_ltg", ctypes.c_void_p), ("params", allen_velo_params_t)]


class allen_velo_clusters_t(ctypes.Structure):
    _fields_ = [("capacity", ctypes.c_uint32)] + [(n, ctypes.c_void_p) for n in (
        "event_offsets", "layer_offsets", "key", "n_pixels", "sum_col", "sum_row", "x", "y", "z", "phi16",
        "checksum", "status")]


class allen_velo_tracks_t(ctypes.Structure):
    _fields_ = [("capacity_tracks", ctypes.c_uint32), ("capacity_hits", ctypes.c_uint32)] + [
        (n, ctypes.c_void_p) for n in ("event_offsets", "hit_offsets", "hits", "x0", "y0", "tx", "ty", "kalman")]


class allen_velo_vertices_t(ctypes.Structure):
    _fields_ = [("max_per_event", ctypes.c_uint32), ("n_vertices", ctypes.c_void_p), ("vertices", ctypes.c_void_p)]


_lib = None


_debug_lib = None


def load_library(debug: bool = False):
    """dlopen the in-tree extension (debug=True: the build with bounds checks, _allen_velo_debug.so).  Raises if it has
    not been built (no fallback)."""
    global _lib, _debug_lib
    if (_debug_lib if debug else _lib) is None:
        path = os.path.join(_HERE, "_allen_velo_debug.so") if debug else LIB_PATH
        if not os.path.exists(path):
            raise RuntimeError(f"CUDA extension {path} is missing: run `python -m paper_1912_09161_b200.build` "
                               "(or __graft_entry__.build()); there is no CPU fallback")
        L = ctypes.CDLL(path)
        L.allen_velo_default_params.argtypes = [ctypes.POINTER(allen_velo_params_t)]
        L.allen_velo_default_params.restype = None
        L.allen_velo_create.argtypes = [ctypes.POINTER(allen_velo_geometry_t), ctypes.POINTER(ctypes.c_void_p)]
        L.allen_velo_create.restype = ctypes.c_int
        L.allen_velo_workspace_bytes.argtypes = [ctypes.c_void_p, ctypes.c_uint32, ctypes.c_size_t]
        L.allen_velo_workspace_bytes.restype = ctypes.c_size_t
        L.allen_velo_set_workspace.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t]
        L.allen_velo_set_workspace.restype = ctypes.c_int
        L.allen_velo_set_occupancy_hint.argtypes = [ctypes.c_void_p, ctypes.c_uint32]
        L.allen_velo_set_occupancy_hint.restype = ctypes.c_int
        L.allen_velo_set_vertex_output.argtypes = [ctypes.c_void_p, ctypes.POINTER(allen_velo_vertices_t)]
        L.allen_velo_set_vertex_output.restype = ctypes.c_int
        L.allen_velo_reconstruct.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint32,
                                             ctypes.c_void_p, ctypes.POINTER(allen_velo_clusters_t),
                                             ctypes.POINTER(allen_velo_tracks_t)]
        L.allen_velo_reconstruct.restype = ctypes.c_int
        L.allen_velo_enable_timing.argtypes = [ctypes.c_void_p, ctypes.c_uint32]
        L.allen_velo_enable_timing.restype = ctypes.c_int
        L.allen_velo_kernel_count.argtypes = []
        L.allen_velo_kernel_count.restype = ctypes.c_uint32
        L.allen_velo_kernel_name.argtypes = [ctypes.c_uint32]
        L.allen_velo_kernel_name.restype = ctypes.c_char_p
        L.allen_velo_kernel_times.argtypes = [ctypes.c_void_p, ctypes.c_uint32, ctypes.c_void_p]
        L.allen_velo_kernel_times.restype = ctypes.c_int
        L.allen_velo_last_launch_count.argtypes = [ctypes.c_void_p]
        L.allen_velo_last_launch_count.restype = ctypes.c_uint32
        L.allen_velo_set_cluster_regions.argtypes = [ctypes.c_void_p, ctypes.c_uint32, ctypes.c_uint32]
        L.allen_velo_set_cluster_regions.restype = ctypes.c_int
        L.allen_velo_debug_track_counters.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
        L.allen_velo_debug_track_counters.restype = ctypes.c_int
        L.allen_velo_last_error.argtypes = [ctypes.c_void_p]
        L.allen_velo_last_error.restype = ctypes.c_char_p
        L.allen_velo_destroy.argtypes = [ctypes.c_void_p]
        L.allen_velo_destroy.restype = None
        L.allen_velo_debug_fault.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
        L.allen_velo_debug_fault.restype = ctypes.c_int
        L.allen_velo_debug_checks_compiled.argtypes = []
        L.allen_velo_debug_checks_compiled.restype = ctypes.c_int
        L.allen_velo_offsets_noalloc.argtypes = [ctypes.c_void_p, ctypes.c_uint32, ctypes.c_void_p, ctypes.c_void_p,
                                                 ctypes.c_char_p, ctypes.c_size_t]
        L.allen_velo_offsets_noalloc.restype = ctypes.c_int
        if debug:
            _debug_lib = L
        else:
            _lib = L
    return _debug_lib if debug else _lib


NOALLOC_MAX_COUNTS = 4194304  # ALLEN_VELO_NOALLOC_MAX_COUNTS
ERR_TOO_LARGE = -4


def offsets_noalloc(counts, n: int, offsets, stream=None) -> tuple[int, str]:
    """include/allen_velo_noalloc.h: offsets[0..n] = exclusive prefix sum of counts[0..n) with the scan's scratch in the
    library's static device array (no handle, no workspace, no allocation).  `counts` / `offsets`: uint32-sized device
    tensors (int32 views); only pointers are passed.  Returns (return code, error text).  One call at a time per device."""
    lib = load_library()
    text = ctypes.create_string_buffer(256)
    s = ctypes.c_void_p(stream.cuda_stream) if stream is not None else None
    rc = lib.allen_velo_offsets_noalloc(ctypes.c_void_p(counts.data_ptr()) if counts is not None else None, n,
                                        ctypes.c_void_p(offsets.data_ptr()) if offsets is not None else None, s, text, 256)
    return int(rc), text.value.decode()


def allen_velo_default_params() -> allen_velo_params_t:
    p = allen_velo_params_t()
    load_library().allen_velo_default_params(ctypes.byref(p))
    return p


@dataclass
class ClusterBuffers:
    """Caller-owned device tensors for `out_clusters` (torch), plus the marshalled struct."""
    capacity: int
    event_offsets: "torch.Tensor"
    layer_offsets: "torch.Tensor"
    key: "torch.Tensor"
    n_pixels: "torch.Tensor"
    sum_col: "torch.Tensor"
    sum_row: "torch.Tensor"
    x: "torch.Tensor"
    y: "torch.Tensor"
    z: "torch.Tensor"
    phi16: "torch.Tensor"
    checksum: "torch.Tensor | None"
    status: "torch.Tensor"

    def struct(self) -> allen_velo_clusters_t:
        s = allen_velo_clusters_t()
        s.capacity = self.capacity
        for name in ("event_offsets", "layer_offsets", "key", "n_pixels", "sum_col", "sum_row", "x", "y", "z",
                     "phi16", "status"):
            setattr(s, name, getattr(self, name).data_ptr())
        s.checksum = self.checksum.data_ptr() if self.checksum is not None else None
        return s


@dataclass
class TrackBuffers:
    capacity_tracks: int
    capacity_hits: int
    event_offsets: "torch.Tensor"
    hit_offsets: "torch.Tensor"
    hits: "torch.Tensor"
    x0: "torch.Tensor"
    y0: "torch.Tensor"
    tx: "torch.Tensor"
    ty: "torch.Tensor"
    kalman: "torch.Tensor | None" = None

    def struct(self) -> allen_velo_tracks_t:
        s = allen_velo_tracks_t()
        s.capacity_tracks, s.capacity_hits = self.capacity_tracks, self.capacity_hits
        for name in ("event_offsets", "hit_offsets", "hits", "x0", "y0", "tx", "ty"):
            setattr(s, name, getattr(self, name).data_ptr())
        s.kalman = self.kalman.data_ptr() if self.kalman is not None else None
        return s


def alloc_outputs(n_events: int, n_layers: int, cluster_capacity: int, track_capacity: int, hit_capacity: int,
                  device, with_checksum: bool = True, with_kalman: bool = False):
    """Allocate output tensors with torch (device memory only; int32 storage stands for u32, int16 for u16)."""
    import torch

    i32, f32, i16 = torch.int32, torch.float32, torch.int16
    z = lambda n, dt: torch.zeros(max(int(n), 1), dtype=dt, device=device)
    c = ClusterBuffers(cluster_capacity, z(n_events + 1, i32), z(n_events * n_layers + 1, i32),
                       z(cluster_capacity, i32), z(cluster_capacity, i32), z(cluster_capacity, i32),
                       z(cluster_capacity, i32), z(cluster_capacity, f32), z(cluster_capacity, f32),
                       z(cluster_capacity, f32), z(cluster_capacity, i16),
                       z(cluster_capacity, i32) if with_checksum else None, z(n_events, i32))
    t = TrackBuffers(track_capacity, hit_capacity, z(n_events + 1, i32), z(track_capacity + 1, i32),
                     z(hit_capacity, i16), z(track_capacity, f32), z(track_capacity, f32), z(track_capacity, f32),
                     z(track_capacity, f32), z(12 * track_capacity, f32) if with_kalman else None)
    return c, t


class AllenVelo:
    """RAII wrapper of the handle: allen_velo_create / set_workspace / reconstruct / destroy."""

    def __init__(self, geometry, params: dict | None = None, debug: bool = False):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_1912_09161_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self._lib = load_library(debug)
        p = allen_velo_default_params()
        for k, v in (params or {}).items():
            setattr(p, k, v)
        self._smod = np.ascontiguousarray(geometry.sensor_module, np.uint16)
        self._mlay = np.ascontiguousarray(geometry.module_layer, np.uint16)
        self._ltg = np.ascontiguousarray(geometry.sensor_ltg, np.float32)
        g = allen_velo_geometry_t(geometry.n_sensors, geometry.n_modules, geometry.n_layers, geometry.n_cols,
                                  geometry.n_rows, geometry.pitch_mm, self._smod.ctypes.data, self._mlay.ctypes.data,
                                  self._ltg.ctypes.data, p)
        self.n_layers = geometry.n_layers
        h = ctypes.c_void_p()
        rc = self._lib.allen_velo_create(ctypes.byref(g), ctypes.byref(h))
        if rc != OK:
            raise RuntimeError(f"allen_velo_create failed with {rc}")
        self._h = h
        self._ws = None

    def workspace_bytes(self, n_events: int, raw_bytes: int) -> int:
        return int(self._lib.allen_velo_workspace_bytes(self._h, n_events, raw_bytes))

    def set_occupancy_hint(self, n_events: int, raw_bytes: int) -> None:
        """Tell the library the average SP words per (event, layer) of the batches to come (performance only)."""
        per_layer = raw_bytes // 4 // max(1, n_events * self.n_layers)
        if self._lib.allen_velo_set_occupancy_hint(self._h, per_layer) != OK:
            raise RuntimeError("allen_velo_set_occupancy_hint failed")

    def set_vertex_output(self, n_vertices=None, vertices=None) -> None:
        """Primary vertices (optional): `n_vertices` int32 [n_events], `vertices` float32 [n_events, slots, 8] CUDA
        tensors the caller keeps alive; None switches the output off."""
        if vertices is None:
            rc = self._lib.allen_velo_set_vertex_output(self._h, None)
            self._pv = None
        else:
            s = allen_velo_vertices_t(int(vertices.shape[1]), n_vertices.data_ptr(), vertices.data_ptr())
            rc = self._lib.allen_velo_set_vertex_output(self._h, ctypes.byref(s))
            self._pv = (n_vertices, vertices)
        if rc != OK:
            raise RuntimeError(f"allen_velo_set_vertex_output failed with {rc}: {self.last_error()}")

    def set_workspace(self, tensor) -> None:
        """`tensor`: a torch uint8 CUDA tensor the caller keeps alive (kept referenced here too)."""
        rc = self._lib.allen_velo_set_workspace(self._h, tensor.data_ptr(), tensor.numel() * tensor.element_size())
        if rc != OK:
            raise RuntimeError(f"allen_velo_set_workspace failed with {rc}: {self.last_error()}")
        self._ws = tensor

    def reconstruct(self, raw_banks, event_offsets, n_events: int, stream, out_clusters: ClusterBuffers,
                    out_tracks: TrackBuffers) -> int:
        """Enqueue on `stream` (a torch.cuda.Stream or None for the current stream).  Returns the C return code."""
        import torch

        s = stream if stream is not None else torch.cuda.current_stream()
        cs, ts = out_clusters.struct(), out_tracks.struct()
        return int(self._lib.allen_velo_reconstruct(self._h, raw_banks.data_ptr(), event_offsets.data_ptr(), n_events,
                                                    ctypes.c_void_p(s.cuda_stream), ctypes.byref(cs), ctypes.byref(ts)))

    def enable_timing(self, n_calls: int) -> None:
        rc = self._lib.allen_velo_enable_timing(self._h, n_calls)
        if rc != OK:
            raise RuntimeError(f"allen_velo_enable_timing failed with {rc}")

    def kernel_names(self) -> list[str]:
        return [self._lib.allen_velo_kernel_name(i).decode() for i in range(self._lib.allen_velo_kernel_count())]

    def kernel_times(self, call: int) -> np.ndarray:
        out = np.zeros(self._lib.allen_velo_kernel_count(), np.float32)
        rc = self._lib.allen_velo_kernel_times(self._h, call, out.ctypes.data)
        if rc != OK:
            raise RuntimeError(f"allen_velo_kernel_times failed with {rc}: {self.last_error()}")
        return out

    def last_launch_count(self) -> int:
        return int(self._lib.allen_velo_last_launch_count(self._h))

    def set_cluster_regions(self, sp_cols: int, sp_rows: int) -> None:
        """Local clustering variant (R11); (0, 0) = exact connected components."""
        rc = self._lib.allen_velo_set_cluster_regions(self._h, sp_cols, sp_rows)
        if rc != OK:
            raise RuntimeError(f"allen_velo_set_cluster_regions -> {rc}: {self.last_error()}")

    def debug_fault(self) -> int:
        """Highest code of a failed bounds check since the last call (debug build; 0 = none).  Synchronises."""
        out = ctypes.c_uint32(0)
        rc = self._lib.allen_velo_debug_fault(self._h, ctypes.byref(out))
        if rc != OK:
            raise RuntimeError(f"allen_velo_debug_fault -> {rc}")
        return int(out.value)

    def checks_compiled(self) -> bool:
        return bool(self._lib.allen_velo_debug_checks_compiled())

    def track_counters(self) -> dict:
        """List sizes of the track search of the last call (include/allen_velo_debug.h; synchronises the device)."""
        out = (ctypes.c_uint32 * 16)()
        rc = self._lib.allen_velo_debug_track_counters(self._h, out)
        if rc != OK:
            raise RuntimeError(f"allen_velo_debug_track_counters -> {rc}")
        return dict(follow=[int(out[0]), int(out[1]), int(out[2])], second_pass=[int(out[12]), int(out[13])])

    def last_error(self) -> str:
        return self._lib.allen_velo_last_error(self._h).decode()

    def destroy(self) -> None:
        if getattr(self, "_h", None):
            self._lib.allen_velo_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def reconstruct_batch(velo: AllenVelo, raw: np.ndarray, event_offsets: np.ndarray, device="cuda:0",
                      with_checksum: bool = True, cluster_capacity: int | None = None,
                      track_capacity: int | None = None, hit_capacity: int | None = None, with_kalman: bool = False,
                      with_vertices: bool = False):
    """Convenience for tests/smoke: copy a host batch to the device, run the path once, return host copies.

    Host<->device copies and the final synchronise happen here, outside the C ABI.  Returns (clusters, tracks)
    as dicts of numpy arrays in the ABI layout (u32/u16 views restored).
    """
    import torch

    n_events = len(event_offsets) - 1
    raw_bytes = int(raw.size)
    d_raw = torch.from_numpy(np.ascontiguousarray(raw)).to(device) if raw_bytes else torch.zeros(16, dtype=torch.uint8, device=device)
    d_off = torch.from_numpy(np.ascontiguousarray(event_offsets).view(np.int32)).to(device)
    ccap = cluster_capacity if cluster_capacity is not None else raw_bytes // 2 + 16  # <= 2 clusters per SP word
    tcap = track_capacity if track_capacity is not None else ccap // 3 + 16
    hcap = hit_capacity if hit_capacity is not None else ccap
    oc, ot = alloc_outputs(n_events, velo.n_layers, ccap, tcap, hcap, device, with_checksum, with_kalman)
    ws = torch.empty(velo.workspace_bytes(n_events, raw_bytes), dtype=torch.uint8, device=device)
    velo.set_workspace(ws)
    velo.set_occupancy_hint(n_events, raw_bytes)
    if with_vertices:
        d_nv = torch.zeros(max(n_events, 1), dtype=torch.int32, device=device)
        d_pv = torch.zeros((max(n_events, 1), 32, 8), dtype=torch.float32, device=device)
        velo.set_vertex_output(d_nv, d_pv)
    try:
        rc = velo.reconstruct(d_raw, d_off, n_events, None, oc, ot)
    finally:
        if with_vertices:
            velo.set_vertex_output(None, None)
    if rc != OK:
        raise RuntimeError(f"allen_velo_reconstruct failed with {rc}: {velo.last_error()}")
    torch.cuda.synchronize()

    def host(t, dt):
        return t.cpu().numpy().view(dt)

    u32, u16 = np.uint32, np.uint16
    nc = int(host(oc.event_offsets, u32)[n_events])
    clusters = dict(event_offsets=host(oc.event_offsets, u32), layer_offsets=host(oc.layer_offsets, u32),
                    status=host(oc.status, u32)[:n_events], n=nc)
    for name, dt in (("key", u32), ("n_pixels", u32), ("sum_col", u32), ("sum_row", u32), ("x", np.float32),
                     ("y", np.float32), ("z", np.float32), ("phi16", np.int16)):
        clusters[name] = host(getattr(oc, name), dt)[:min(nc, ccap)]
    clusters["checksum"] = host(oc.checksum, u32)[:min(nc, ccap)] if with_checksum else None
    te = host(ot.event_offsets, u32)
    nt = int(te[n_events])
    ho = host(ot.hit_offsets, u32)[:min(nt, tcap) + 1]
    nh = int(ho[-1]) if nt <= tcap else 0
    tracks = dict(event_offsets=te, hit_offsets=ho, hits=host(ot.hits, u16)[:min(nh, hcap)], n=nt)
    for name in ("x0", "y0", "tx", "ty"):
        tracks[name] = host(getattr(ot, name), np.float32)[:min(nt, tcap)]
    if with_kalman:
        tracks["kalman"] = host(ot.kalman, np.float32).reshape(-1, 12)[:min(nt, tcap)]
    if with_vertices:
        tracks["n_vertices"] = d_nv.cpu().numpy().view(np.uint32)[:n_events]
        tracks["vertices"] = d_pv.cpu().numpy()[:n_events]
    return clusters, tracks


class StreamedVelo:
    """Host-to-host reconstruction of a large batch in chunks on several CUDA streams (the paper's host loop
    gives every thread its own stream and ~1000-event batches so that copies and kernels of different batches overlap).

    Every stream owns a handle, device input/output buffers, a workspace and pinned host buffers for the track output.
    `reconstruct` cuts the batch into chunks of `chunk_events`, and for each chunk enqueues on its stream: H2D of the
    raw banks and offsets, allen_velo_reconstruct, D2H of the offsets; once those arrive (the host waits for THIS stream
    only, the others keep working) the D2H of exactly the tracks found.  All arithmetic runs in the CUDA kernels; this
    class only moves bytes and calls the C ABI.
    """

    def __init__(self, geometry, chunk_events: int, max_chunk_raw_bytes: int, n_streams: int = 2, device="cuda:0",
                 params: dict | None = None, prioritise: bool = False):
        import torch

        self.device, self.chunk_events, self.n_layers = torch.device(device), int(chunk_events), geometry.n_layers
        self.max_raw = (int(max_chunk_raw_bytes) + 15) // 16 * 16
        ccap = self.max_raw // 4 + 4096          # clusters <= SP words (x2 only for adversarial input: flagged, not UB)
        tcap, hcap = ccap // 3 + 16, ccap
        self.slots = []
        for _ in range(n_streams):
            v = AllenVelo(geometry, params)
            oc, ot = alloc_outputs(self.chunk_events, self.n_layers, ccap, tcap, hcap, self.device, with_checksum=False)
            ws = torch.empty(v.workspace_bytes(self.chunk_events, self.max_raw), dtype=torch.uint8, device=self.device)
            v.set_workspace(ws)
            v.set_occupancy_hint(self.chunk_events, self.max_raw)
            pin = lambda n, dt: torch.empty(max(int(n), 1), dtype=dt).pin_memory()
            self.slots.append(dict(
                velo=v, oc=oc, ot=ot, stream=torch.cuda.Stream(device=self.device),
                d_raw=torch.empty(self.max_raw, dtype=torch.uint8, device=self.device),
                d_off=torch.empty(self.chunk_events + 1, dtype=torch.int32, device=self.device),
                h_off=pin(self.chunk_events + 1, torch.int32), h_te=pin(self.chunk_events + 1, torch.int32),
                h_st=pin(self.chunk_events, torch.int32), h_ho=pin(tcap + 1, torch.int32), h_tot=pin(1, torch.int32),
                tcap=tcap,
                h_hits=pin(hcap, torch.int16), h_fit=[pin(tcap, torch.float32) for _ in range(4)],
                pending=None))
        self.h2d_bytes = self.d2h_bytes = 0

    def _finish(self, s):
        """Second half of a chunk: sizes have arrived -> fetch exactly the tracks found."""
        import torch

        p = s["pending"]
        if p is None:
            return None
        s["stream"].synchronize()
        n = p["n_events"]
        nt, nh = int(s["h_te"][n]), int(s["h_tot"][0])  # both totals came with the offsets: one wait per chunk
        with torch.cuda.stream(s["stream"]):
            s["h_ho"][:nt + 1].copy_(s["ot"].hit_offsets[:nt + 1], non_blocking=True)
            for hb, db in zip(s["h_fit"], (s["ot"].x0, s["ot"].y0, s["ot"].tx, s["ot"].ty)):
                hb[:nt].copy_(db[:nt], non_blocking=True)
            s["h_hits"][:nh].copy_(s["ot"].hits[:nh], non_blocking=True)
        self.d2h_bytes += 4 * (n + 1) + 4 * n + 4 + 4 * (nt + 1) + 16 * nt + 2 * nh
        s["pending"] = None
        return dict(first_event=p["first"], n_events=n, n_tracks=nt, n_hits=nh)

    def reconstruct(self, h_raw, h_event_offsets, on_chunk=None, chunk_sizes=None):
        """h_raw: pinned uint8 tensor (raw format v1, events back to back); h_event_offsets: int64/int32 numpy array
        [n_events+1].  Calls on_chunk(info, slot) when a chunk's tracks are on their way to the slot's pinned buffers
        (valid after slot['stream'].synchronize()).  `chunk_sizes`: events of the first chunks (each <= chunk_events; the
        rest of the batch goes in chunks of chunk_events) — a short first chunk gets the GPU started while the next
        ones are still being copied.  Returns the list of chunk infos."""
        import torch

        off = np.asarray(h_event_offsets).astype(np.int64)
        n_events = len(off) - 1
        self.h2d_bytes = self.d2h_bytes = 0
        infos = []
        firsts, at = [], 0
        for size in list(chunk_sizes or []):
            if not 0 < int(size) <= self.chunk_events:
                raise ValueError("chunk_sizes entries must be in [1, chunk_events]")
            if at < n_events:
                firsts.append((at, min(at + int(size), n_events)))
                at = firsts[-1][1]
        while at < n_events:
            firsts.append((at, min(at + self.chunk_events, n_events)))
            at = firsts[-1][1]
        for k, (first, last) in enumerate(firsts):
            s = self.slots[k % len(self.slots)]
            done = self._finish(s)  # the slot's previous chunk (the other slots keep running meanwhile)
            if done is not None:
                infos.append(done)
                if on_chunk:
                    on_chunk(done, s)
            n = last - first
            b0, b1 = int(off[first]), int(off[last])
            if b1 - b0 > self.max_raw:
                raise ValueError("chunk larger than max_chunk_raw_bytes")
            s["stream"].synchronize()  # the slot's host staging buffers are free again
            s["h_off"][:n + 1] = torch.from_numpy((off[first:last + 1] - b0).astype(np.int32))
            with torch.cuda.stream(s["stream"]):
                s["d_raw"][:b1 - b0].copy_(h_raw[b0:b1], non_blocking=True)
                s["d_off"][:n + 1].copy_(s["h_off"][:n + 1], non_blocking=True)
                rc = s["velo"].reconstruct(s["d_raw"], s["d_off"], n, s["stream"], s["oc"], s["ot"])
                if rc != OK:
                    raise RuntimeError(f"allen_velo_reconstruct failed with {rc}: {s['velo'].last_error()}")
                s["h_te"][:n + 1].copy_(s["ot"].event_offsets[:n + 1], non_blocking=True)
                s["h_st"][:n].copy_(s["oc"].status[:n], non_blocking=True)
                s["h_tot"].copy_(s["ot"].hit_offsets[s["tcap"]:s["tcap"] + 1], non_blocking=True)
            self.h2d_bytes += (b1 - b0) + 4 * (n + 1)
            s["pending"] = dict(first=first, n_events=n)
        for s in self.slots:
            done = self._finish(s)
            if done is not None:
                infos.append(done)
                if on_chunk:
                    on_chunk(done, s)
        for s in self.slots:
            s["stream"].synchronize()
        return sorted(infos, key=lambda i: i["first_event"])

    def destroy(self):
        for s in self.slots:
            s["velo"].destroy()
        self.slots = []
