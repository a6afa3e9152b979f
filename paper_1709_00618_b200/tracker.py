"""Thin Python binding of libtpctrk.so (include/tpc_tracker.h): argument marshalling only.

PyTorch is used for device memory and streams; every step of the hot path runs in the library's CUDA kernels.
There is no fallback: if the shared library is missing or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtpctrk.so")

CAND_MAX_HITS = 10
N_COUNTS = 16
N_STAGES = 6
STAGE_NAMES = ("bin", "neighbours", "chains", "fit", "follow", "select")
ERRORS = {-1: "TPC_ERR_ARG", -2: "TPC_ERR_GEOMETRY", -3: "TPC_ERR_WORKSPACE", -4: "TPC_ERR_CUDA",
          -5: "TPC_ERR_CAPACITY", -6: "TPC_ERR_INPUT", -7: "TPC_ERR_LIMIT"}

EXPORTS = ("tpc_tracker_create", "tpc_tracker_destroy", "tpc_workspace_bytes", "tpc_set_workspace", "tpc_set_stream",
           "tpc_track_sectors", "tpc_check_counts", "tpc_last_launch_count", "tpc_set_stage_timing",
           "tpc_stage_times_ms", "tpc_last_error", "tpc_track_sectors_host", "tpc_set_work_counters",
           "tpc_set_input_layout", "tpc_pipeline_create", "tpc_pipeline_destroy", "tpc_pipeline_run",
           "tpc_merge_refit", "tpc_estimate_vertices", "tpc_start_hits_static")
STATIC_MAX_CLUSTERS = 1 << 27                        # TPC_STATIC_MAX_CLUSTERS
VTX_MAX_PER_WINDOW = 64
INPUT_LAYOUTS = {"xyzw": 0, "yz": 1, "i16": 2}       # TPC_INPUT_*
LAYOUT_BYTES = {"xyzw": 16, "yz": 8, "i16": 4}
I16_Y_STEP, I16_Z_STEP = 1.0 / 256.0, 1.0 / 64.0     # TPC_I16_*_STEP


class TpcError(RuntimeError):
    pass


class Params(C.Structure):
    _fields_ = [("nf_win_y", C.c_float), ("nf_win_z", C.c_float), ("nf_d2_max", C.c_float),
                ("cand_min_hits", C.c_int32), ("cand_max_hits", C.c_int32), ("kf_p0", C.c_float * 5),
                ("kf_gate_sigma", C.c_float), ("kf_win_max", C.c_float), ("kf_max_gap", C.c_int32),
                ("kf_max_sinphi", C.c_float), ("kf_edge_margin", C.c_float), ("sel_min_hits", C.c_int32),
                ("grid_cell_z", C.c_float), ("grid_cells_y", C.c_int32), ("nf_bridge_rows", C.c_int32)]


class Geometry(C.Structure):
    _fields_ = [("n_rows", C.c_int32), ("row_x", C.POINTER(C.c_float)), ("sectors_per_event", C.c_int32),
                ("half_angle_rad", C.c_float), ("z_lo", C.c_float), ("z_hi", C.c_float), ("sigma_y", C.c_float),
                ("sigma_z", C.c_float), ("params", Params)]


_OUT_PTRS = ("link_up_raw", "link_dn_raw", "link_up", "link_dn")


class Output(C.Structure):
    _fields_ = [("link_up_raw", C.c_void_p), ("link_dn_raw", C.c_void_p), ("link_up", C.c_void_p),
                ("link_dn", C.c_void_p), ("start_hits", C.c_void_p), ("start_capacity", C.c_int64),
                ("cand_hits", C.c_void_p), ("cand_n", C.c_void_p), ("cand_capacity", C.c_int64),
                ("tl_params", C.c_void_p), ("tl_cov", C.c_void_p), ("tl_chi2", C.c_void_p), ("tl_nhits", C.c_void_p),
                ("tl_rows", C.c_void_p), ("tl_hits", C.c_void_p), ("tl_capacity", C.c_int64),
                ("trk_params", C.c_void_p), ("trk_cov", C.c_void_p), ("trk_chi2", C.c_void_p),
                ("trk_xref", C.c_void_p), ("trk_cand_id", C.c_void_p), ("trk_nhits", C.c_void_p),
                ("trk_sector", C.c_void_p), ("trk_hit_offset", C.c_void_p), ("trk_hits", C.c_void_p),
                ("trk_capacity", C.c_int64), ("trk_hits_capacity", C.c_int64), ("cluster_owner", C.c_void_p),
                ("counts", C.c_void_p)]


class Phase2Output(C.Structure):
    _fields_ = [("seg_next", C.c_void_p), ("seg_prev", C.c_void_p), ("seg_ok", C.c_void_p), ("seg_params", C.c_void_p),
                ("seg_cov", C.c_void_p), ("seg_chi2", C.c_void_p), ("mtrk_first", C.c_void_p), ("mtrk_nseg", C.c_void_p),
                ("mtrk_nhits", C.c_void_p), ("mtrk_ok", C.c_void_p), ("mtrk_params", C.c_void_p),
                ("mtrk_cov", C.c_void_p), ("mtrk_chi2", C.c_void_p), ("mtrk_capacity", C.c_int64),
                ("counts2", C.c_void_p)]


class VertexOutput(C.Structure):
    _fields_ = [("trk_zv", C.c_void_p), ("trk_dca", C.c_void_p), ("trk_vtx", C.c_void_p), ("vtx_z", C.c_void_p),
                ("vtx_window", C.c_void_p), ("vtx_ntracks", C.c_void_p), ("vtx_capacity", C.c_int64),
                ("counts3", C.c_void_p)]


class Slot(C.Structure):
    _fields_ = [("clusters", C.c_void_p), ("row_offsets", C.c_void_p), ("max_clusters", C.c_int64),
                ("max_instances", C.c_int32), ("out", Output), ("workspace", C.c_void_p),
                ("workspace_bytes", C.c_size_t)]


class HostOutput(C.Structure):
    _fields_ = [("trk_params", C.c_void_p), ("trk_cov", C.c_void_p), ("trk_nhits", C.c_void_p),
                ("trk_sector", C.c_void_p), ("trk_hit_offset", C.c_void_p), ("trk_hits", C.c_void_p),
                ("cluster_owner", C.c_void_p), ("trk_capacity", C.c_int64), ("trk_hits_capacity", C.c_int64),
                ("totals", C.c_int64 * 16), ("n_chunks", C.c_int64), ("n_launches", C.c_int64),
                ("h2d_bytes", C.c_int64), ("d2h_bytes", C.c_int64), ("h2d_ms", C.c_float), ("compute_ms", C.c_float),
                ("d2h_ms", C.c_float), ("wall_ms", C.c_float)]


_lib = None


def load_library():
    """dlopen libtpctrk.so and declare the prototypes.  Raises if the library has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise TpcError(f"{LIB_PATH} not found: build it with `python -m paper_1709_00618_b200.build` "
                       "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    lib.tpc_tracker_create.argtypes = [C.POINTER(Geometry), C.c_float, C.POINTER(C.c_void_p)]
    lib.tpc_tracker_create.restype = C.c_int
    lib.tpc_tracker_destroy.argtypes = [C.c_void_p]
    lib.tpc_tracker_destroy.restype = None
    lib.tpc_workspace_bytes.argtypes = [C.c_void_p, C.c_int64, C.c_int64]
    lib.tpc_workspace_bytes.restype = C.c_size_t
    lib.tpc_set_workspace.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t]
    lib.tpc_set_stream.argtypes = [C.c_void_p, C.c_void_p]
    lib.tpc_track_sectors.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int64, C.POINTER(Output)]
    lib.tpc_check_counts.argtypes = [C.POINTER(C.c_int64), C.POINTER(Output)]
    lib.tpc_last_launch_count.argtypes = [C.c_void_p]
    lib.tpc_last_launch_count.restype = C.c_int32
    lib.tpc_set_stage_timing.argtypes = [C.c_void_p, C.c_int32]
    lib.tpc_set_work_counters.argtypes = [C.c_void_p, C.c_int32]
    lib.tpc_set_input_layout.argtypes = [C.c_void_p, C.c_int32]
    lib.tpc_stage_times_ms.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_float)]
    lib.tpc_last_error.argtypes = [C.c_void_p]
    lib.tpc_last_error.restype = C.c_char_p
    lib.tpc_track_sectors_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int64, C.c_int32,
                                           C.POINTER(Slot), C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p,
                                           C.POINTER(HostOutput)]
    lib.tpc_merge_refit.argtypes = [C.c_void_p, C.POINTER(Phase2Output)]
    lib.tpc_estimate_vertices.argtypes = [C.c_void_p, C.POINTER(Phase2Output), C.POINTER(VertexOutput)]
    lib.tpc_pipeline_create.argtypes = [C.c_void_p, C.POINTER(Slot), C.c_int32, C.POINTER(C.c_void_p)]
    lib.tpc_pipeline_destroy.argtypes = [C.c_void_p]
    lib.tpc_pipeline_destroy.restype = None
    lib.tpc_pipeline_run.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int64, C.c_int32,
                                     C.POINTER(HostOutput)]
    lib.tpc_start_hits_static.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_int64, C.c_void_p,
                                          C.c_void_p]
    _lib = lib
    return lib


def start_hits_static(link_up, link_dn, start_hits, n_start, *, n_clusters=None, stream=None):
    """tpc_start_hits_static on torch CUDA tensors; asynchronous on `stream` (default: torch's current stream).

    The one call of the library that needs neither a workspace nor a Tracker: it is meant for callers that have no
    way to allocate device memory (a component of a framework that handed out all GPU memory at start-up, a real-time
    loop where cudaMalloc's device-wide synchronisation is not acceptable).  Its scratch memory is an array built into
    the library, shared by every call on that GPU: calls must not overlap on the device, and at most
    STATIC_MAX_CLUSTERS links are accepted (TPC_ERR_LIMIT beyond that).  link_up / link_dn: int32 [n] cleaned links;
    start_hits: int32 [capacity] or None (count only); n_start: int64 [1] receives the required count.
    Make the first call on a device before starting any stream capture there (one-time address look-up).
    """
    import torch
    lib = load_library()
    n = int(link_up.numel() if n_clusters is None else n_clusters)
    s = stream if stream is not None else torch.cuda.current_stream(link_up.device)
    with torch.cuda.device(link_up.device):
        rc = lib.tpc_start_hits_static(C.c_void_p(link_up.data_ptr()), C.c_void_p(link_dn.data_ptr()), n,
                                       C.c_void_p(start_hits.data_ptr() if start_hits is not None else None),
                                       int(start_hits.numel()) if start_hits is not None else 0,
                                       C.c_void_p(n_start.data_ptr()), C.c_void_p(s.cuda_stream))
    if rc != 0:
        raise TpcError(f"tpc_start_hits_static: {ERRORS.get(rc, rc)}: {lib.tpc_last_error(None).decode()}")


def make_geometry(row_x: np.ndarray, *, z_lo=0.0, z_hi=250.0, sigma_y=0.1, sigma_z=0.1, sectors_per_event=36,
                  half_angle_rad=float(np.deg2rad(10.0)), **params):
    """Returns (Geometry, keep-alive row_x array).  Unknown tunables raise; omitted ones take the defaults."""
    rx = np.ascontiguousarray(row_x, dtype=np.float32)
    g = Geometry()
    g.n_rows = len(rx)
    g.row_x = rx.ctypes.data_as(C.POINTER(C.c_float))
    g.sectors_per_event = sectors_per_event
    g.half_angle_rad = half_angle_rad
    g.z_lo, g.z_hi, g.sigma_y, g.sigma_z = z_lo, z_hi, sigma_y, sigma_z
    names = {f[0] for f in Params._fields_}
    for k, v in params.items():
        if k not in names:
            raise TypeError(f"unknown tracker parameter {k!r}")
        if k == "kf_p0":
            for i in range(5):
                g.params.kf_p0[i] = v[i]
        else:
            setattr(g.params, k, v)
    return g, rx


@dataclass
class TrackResult:
    """Host copies (numpy) of one call's outputs; fields not requested are None."""
    counts: np.ndarray
    link_up_raw: np.ndarray = None
    link_dn_raw: np.ndarray = None
    link_up: np.ndarray = None
    link_dn: np.ndarray = None
    start_hits: np.ndarray = None
    cand_hits: np.ndarray = None
    cand_n: np.ndarray = None
    tl_params: np.ndarray = None
    tl_cov: np.ndarray = None
    tl_chi2: np.ndarray = None
    tl_nhits: np.ndarray = None
    tl_rows: np.ndarray = None
    tl_hits: np.ndarray = None
    trk_params: np.ndarray = None
    trk_cov: np.ndarray = None
    trk_chi2: np.ndarray = None
    trk_xref: np.ndarray = None
    trk_cand_id: np.ndarray = None
    trk_nhits: np.ndarray = None
    trk_sector: np.ndarray = None
    trk_hit_offset: np.ndarray = None
    trk_hits: np.ndarray = None
    cluster_owner: np.ndarray = None

    @property
    def n_start(self): return int(self.counts[0])
    @property
    def n_cand(self): return int(self.counts[1])
    @property
    def n_tracklets(self): return int(self.counts[2])
    @property
    def n_tracks(self): return int(self.counts[3])
    @property
    def n_track_hits(self): return int(self.counts[4])


class Tracker:
    """tpc_tracker_create(geometry, Bz) + workspace/stream plumbing with torch tensors."""

    def __init__(self, row_x, bz, *, device="cuda:0", **geom_kw):
        import torch
        if not torch.cuda.is_available():
            raise TpcError("no CUDA device: the TPC tracker has no CPU path")
        self._torch = torch
        self.device = torch.device(device)
        self.lib = load_library()
        self.n_rows = len(row_x)
        geom, self._rx = make_geometry(row_x, **geom_kw)
        h = C.c_void_p()
        with torch.cuda.device(self.device):
            rc = self.lib.tpc_tracker_create(C.byref(geom), C.c_float(bz), C.byref(h))
        if rc != 0:
            raise TpcError(f"tpc_tracker_create: {ERRORS.get(rc, rc)}: {self.lib.tpc_last_error(None).decode()}")
        self._h = h
        self._ws = None
        self._out_keep = None
        self.input_layout = "xyzw"

    @classmethod
    def for_event(cls, ev, **kw):
        from . import datagen
        return cls(ev.row_x, ev.bz, z_lo=ev.z_lo, z_hi=ev.z_hi, sigma_y=ev.sigma_y,
                   sigma_z=ev.sigma_z, **kw)

    def close(self):
        if getattr(self, "_h", None):
            self.lib.tpc_tracker_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, what):
        if rc != 0:
            raise TpcError(f"{what}: {ERRORS.get(rc, rc)}: {self.lib.tpc_last_error(self._h).decode()}")

    def workspace_bytes(self, max_clusters, max_inst):
        return int(self.lib.tpc_workspace_bytes(self._h, int(max_clusters), int(max_inst)))

    def reserve(self, max_clusters, max_inst):
        """Allocate (with torch) and attach a workspace large enough for these sizes."""
        need = self.workspace_bytes(max_clusters, max_inst)
        if self._ws is None or self._ws.numel() < need:
            self._ws = self._torch.empty(need, dtype=self._torch.uint8, device=self.device)
        self._check(self.lib.tpc_set_workspace(self._h, C.c_void_p(self._ws.data_ptr()), self._ws.numel()),
                    "tpc_set_workspace")

    def set_stream(self, stream=None):
        s = stream if stream is not None else self._torch.cuda.current_stream(self.device)
        self._check(self.lib.tpc_set_stream(self._h, C.c_void_p(s.cuda_stream)), "tpc_set_stream")

    def set_stage_timing(self, enable=True):
        self._check(self.lib.tpc_set_stage_timing(self._h, 1 if enable else 0), "tpc_set_stage_timing")

    def set_work_counters(self, enable=True):
        """counts[6..9] (S5 transports / updates / examined clusters / searches) are only filled when enabled."""
        self._check(self.lib.tpc_set_work_counters(self._h, 1 if enable else 0), "tpc_set_work_counters")

    def set_input_layout(self, layout="xyzw"):
        """`clusters` of the track calls: "xyzw" float32 [N,4]; "yz" float32 [N,2]; "i16" int16 [N,2] fixed point."""
        self.input_layout = layout
        self._check(self.lib.tpc_set_input_layout(self._h, INPUT_LAYOUTS[layout]), "tpc_set_input_layout")

    def stage_times_ms(self, age=0):
        """Milliseconds per stage of the timed call `age` calls back (0 = last)."""
        buf = (C.c_float * N_STAGES)()
        self._check(self.lib.tpc_stage_times_ms(self._h, int(age), buf), "tpc_stage_times_ms")
        return dict(zip(STAGE_NAMES, [float(x) for x in buf]))

    @property
    def last_launch_count(self):
        return int(self.lib.tpc_last_launch_count(self._h))

    # ---- device-level call: torch tensors in, torch tensors out, asynchronous ------------------------------------
    def alloc_outputs(self, n_clusters, *, debug=False, cand_capacity=None, trk_capacity=None):
        """Device output buffers as a dict of torch tensors (+ the ctypes struct).  debug=True adds every parity array."""
        t = self._torch
        dev = self.device
        n = max(int(n_clusters), 1)
        cc = int(cand_capacity if cand_capacity is not None else n // 4 + 1)
        tc = int(trk_capacity if trk_capacity is not None else n // 10 + 1)
        i32, f32, i64 = t.int32, t.float32, t.int64
        bufs = dict(counts=t.zeros(N_COUNTS, dtype=i64, device=dev),
                    trk_params=t.empty((tc, 5), dtype=f32, device=dev), trk_cov=t.empty((tc, 15), dtype=f32, device=dev),
                    trk_chi2=t.empty(tc, dtype=f32, device=dev), trk_xref=t.empty(tc, dtype=f32, device=dev),
                    trk_cand_id=t.empty(tc, dtype=i32, device=dev), trk_nhits=t.empty(tc, dtype=i32, device=dev),
                    trk_sector=t.empty(tc, dtype=i32, device=dev), trk_hit_offset=t.empty(tc + 1, dtype=i64, device=dev),
                    trk_hits=t.empty(n, dtype=i32, device=dev), cluster_owner=t.empty(n, dtype=i32, device=dev))
        if debug:
            for k in _OUT_PTRS:
                bufs[k] = t.empty(n, dtype=i32, device=dev)
            bufs.update(start_hits=t.empty(n, dtype=i32, device=dev),
                        cand_hits=t.empty((cc, CAND_MAX_HITS), dtype=i32, device=dev),
                        cand_n=t.empty(cc, dtype=i32, device=dev),
                        tl_params=t.empty((cc, 5), dtype=f32, device=dev), tl_cov=t.empty((cc, 15), dtype=f32, device=dev),
                        tl_chi2=t.empty(cc, dtype=f32, device=dev), tl_nhits=t.empty(cc, dtype=i32, device=dev),
                        tl_rows=t.empty((cc, 3), dtype=i32, device=dev),
                        tl_hits=t.empty((cc, self.n_rows), dtype=i32, device=dev))
        o = Output()
        for k, v in bufs.items():
            setattr(o, k, v.data_ptr())
        o.start_capacity = n if debug else 0
        o.cand_capacity = cc if debug else 0
        o.tl_capacity = cc if debug else 0
        o.trk_capacity = tc
        o.trk_hits_capacity = n
        return bufs, o

    def track_sectors_device(self, clusters, row_offsets, n_inst, out_struct):
        """tpc_track_sectors on device tensors (float32 [N,4], int32 [n_inst*R+1]); asynchronous."""
        n = int(clusters.shape[0])
        self._check(self.lib.tpc_track_sectors(self._h, C.c_void_p(clusters.data_ptr()),
                                               C.c_void_p(row_offsets.data_ptr()), int(n_inst), n,
                                               C.byref(out_struct)), "tpc_track_sectors")

    # ---- phase 2: sector merger + refit on the final tracks of the last track_sectors call ------------------------
    def alloc_phase2(self, n_tracks):
        """Device buffers for tpc_merge_refit sized for n_tracks final tracks (+ the ctypes struct)."""
        t = self._torch
        dev = self.device
        n = max(int(n_tracks), 1)
        i32, f32, i64 = t.int32, t.float32, t.int64
        bufs = dict(seg_next=t.empty(n, dtype=i32, device=dev), seg_prev=t.empty(n, dtype=i32, device=dev),
                    seg_ok=t.empty(n, dtype=i32, device=dev), seg_params=t.empty((n, 5), dtype=f32, device=dev),
                    seg_cov=t.empty((n, 15), dtype=f32, device=dev), seg_chi2=t.empty(n, dtype=f32, device=dev),
                    mtrk_first=t.empty(n, dtype=i32, device=dev), mtrk_nseg=t.empty(n, dtype=i32, device=dev),
                    mtrk_nhits=t.empty(n, dtype=i32, device=dev), mtrk_ok=t.empty(n, dtype=i32, device=dev),
                    mtrk_params=t.empty((n, 5), dtype=f32, device=dev), mtrk_cov=t.empty((n, 15), dtype=f32, device=dev),
                    mtrk_chi2=t.empty(n, dtype=f32, device=dev), counts2=t.zeros(4, dtype=i64, device=dev))
        o = Phase2Output()
        for k, v in bufs.items():
            setattr(o, k, v.data_ptr())
        o.mtrk_capacity = n
        return bufs, o

    def merge_refit_device(self, out_struct):
        """tpc_merge_refit on the tracks of the last track call of this tracker; asynchronous."""
        self._check(self.lib.tpc_merge_refit(self._h, C.byref(out_struct)), "tpc_merge_refit")

    def alloc_vertices(self, n_merged, n_windows):
        """Device buffers for tpc_estimate_vertices (+ the ctypes struct)."""
        t = self._torch
        dev = self.device
        n, nv = max(int(n_merged), 1), max(int(n_windows), 1) * VTX_MAX_PER_WINDOW
        bufs = dict(trk_zv=t.empty(n, dtype=t.float32, device=dev), trk_dca=t.empty(n, dtype=t.float32, device=dev),
                    trk_vtx=t.empty(n, dtype=t.int32, device=dev), vtx_z=t.empty(nv, dtype=t.float32, device=dev),
                    vtx_window=t.empty(nv, dtype=t.int32, device=dev), vtx_ntracks=t.empty(nv, dtype=t.int32, device=dev),
                    counts3=t.zeros(2, dtype=t.int64, device=dev))
        o = VertexOutput()
        for k, v in bufs.items():
            setattr(o, k, v.data_ptr())
        o.vtx_capacity = nv
        return bufs, o

    def estimate_vertices_device(self, phase2_struct, out_struct):
        """tpc_estimate_vertices on the merged tracks of the last merge_refit call; asynchronous."""
        self._check(self.lib.tpc_estimate_vertices(self._h, C.byref(phase2_struct), C.byref(out_struct)),
                    "tpc_estimate_vertices")

    def merge_refit(self, n_tracks, vertices_for_windows=0):
        """numpy results of phase 2 for the last track_sectors() call (its workspace is still attached); with
        vertices_for_windows = n also the vertex estimate (tpc_estimate_vertices) under the key "vertices"."""
        t = self._torch
        with t.cuda.device(self.device):
            bufs, o = self.alloc_phase2(n_tracks)
            self.merge_refit_device(o)
            vb = None
            if vertices_for_windows:
                vb, vo = self.alloc_vertices(n_tracks, vertices_for_windows)
                self.estimate_vertices_device(o, vo)
            t.cuda.synchronize(self.device)
        c2 = bufs["counts2"].cpu().numpy()
        nm = int(c2[0])
        res = {k: v.cpu().numpy()[:(nm if k.startswith("mtrk") else n_tracks)] for k, v in bufs.items() if k != "counts2"}
        res["counts2"] = c2
        if vb is not None:
            c3 = vb["counts3"].cpu().numpy()
            nv = int(c3[0])
            res["vertices"] = {k: v.cpu().numpy()[:(nv if k.startswith("vtx") else nm)] for k, v in vb.items()
                               if k != "counts3"}
            res["vertices"]["counts3"] = c3
        return res

    # ---- convenience: numpy in, numpy out (used by the parity tests) ----------------------------------------------
    def track_sectors(self, clusters: np.ndarray, row_offsets: np.ndarray, n_inst: int, *, debug=False,
                      cand_capacity=None, trk_capacity=None) -> TrackResult:
        t = self._torch
        if self.input_layout == "i16":
            cl = t.from_numpy(np.ascontiguousarray(clusters, np.int16).reshape(-1, 2)).to(self.device)
        else:
            cl = t.from_numpy(np.ascontiguousarray(clusters, np.float32)
                              .reshape(-1, 4 if self.input_layout == "xyzw" else 2)).to(self.device)
        ro = t.from_numpy(np.ascontiguousarray(row_offsets, np.int32)).to(self.device)
        n = int(cl.shape[0])
        self._last_inputs = (cl, ro)  # tpc_merge_refit reads the row offsets of the last call: keep them alive
        with t.cuda.device(self.device):
            self.reserve(n, n_inst)
            self.set_stream()
            bufs, o = self.alloc_outputs(n, debug=debug, cand_capacity=cand_capacity, trk_capacity=trk_capacity)
            self.track_sectors_device(cl, ro, n_inst, o)
            t.cuda.synchronize(self.device)
        counts = bufs["counts"].cpu().numpy()
        cnt = (C.c_int64 * N_COUNTS)(*[int(x) for x in counts])
        rc = self.lib.tpc_check_counts(cnt, C.byref(o))
        if rc != 0:
            raise TpcError(f"tpc_check_counts: {ERRORS.get(rc, rc)} counts={counts.tolist()}")
        res = TrackResult(counts=counts)
        nt, nh, nc, ns = res.n_tracks, res.n_track_hits, res.n_cand, res.n_start
        cut = dict(trk_params=nt, trk_cov=nt, trk_chi2=nt, trk_xref=nt, trk_cand_id=nt, trk_nhits=nt, trk_sector=nt,
                   trk_hit_offset=nt + 1, trk_hits=nh, cluster_owner=n, link_up_raw=n, link_dn_raw=n, link_up=n,
                   link_dn=n, start_hits=ns, cand_hits=nc, cand_n=nc, tl_params=nc, tl_cov=nc, tl_chi2=nc, tl_nhits=nc,
                   tl_rows=nc, tl_hits=nc)
        for k, v in bufs.items():
            if k != "counts":
                setattr(res, k, v[:cut[k]].cpu().numpy())
        return res


class HostPipeline:
    """Buffers and the persistent pipeline handle for tpc_pipeline_run: `n_slots` device slots (torch), each with its
    own workspace, and pinned host result arrays for the outputs named in `want`.

    The chunk loop, the stream/event choreography and every copy are inside the C library; this class only owns
    memory and marshals pointers."""

    RESULTS = ("trk_params", "trk_cov", "trk_nhits", "trk_sector", "trk_hit_offset", "trk_hits", "cluster_owner")

    def __init__(self, tracker: Tracker, max_chunk_clusters: int, inst_per_chunk: int, total_clusters: int, *,
                 n_slots=2, trk_frac=0.05, want=RESULTS, slot_workspaces=True):
        t = tracker._torch
        self.trk = tracker
        self.inst_per_chunk = int(inst_per_chunk)
        dev = tracker.device
        n = max(int(max_chunk_clusters), 1)
        tc = int(n * trk_frac) + 64
        i32, f32, i64, u8 = t.int32, t.float32, t.int64, t.uint8
        self._keep = []
        self.slots = (Slot * n_slots)()
        ws_bytes = tracker.workspace_bytes(n, self.inst_per_chunk)
        shapes = dict(trk_params=((tc, 5), f32), trk_cov=((tc, 15), f32), trk_nhits=((tc,), i32),
                      trk_sector=((tc,), i32), trk_hit_offset=((tc + 1,), i64), trk_hits=((n,), i32),
                      cluster_owner=((n,), i32))
        with t.cuda.device(dev):
            for s in range(n_slots):
                b = dict(clusters=t.empty(n * LAYOUT_BYTES[tracker.input_layout], dtype=u8, device=dev),
                         row_offsets=t.empty(self.inst_per_chunk * tracker.n_rows + 1, dtype=i32, device=dev),
                         counts=t.zeros(N_COUNTS, dtype=i64, device=dev))
                for k in want:
                    b[k] = t.empty(shapes[k][0], dtype=shapes[k][1], device=dev)
                if slot_workspaces:
                    b["workspace"] = t.empty(ws_bytes, dtype=u8, device=dev)
                self._keep.append(b)
                sl = self.slots[s]
                sl.clusters, sl.row_offsets = b["clusters"].data_ptr(), b["row_offsets"].data_ptr()
                sl.max_clusters, sl.max_instances = n, self.inst_per_chunk
                sl.out.counts = b["counts"].data_ptr()
                for k in want:
                    setattr(sl.out, k, b[k].data_ptr())
                sl.out.trk_capacity, sl.out.trk_hits_capacity = tc, n
                if slot_workspaces:
                    sl.workspace, sl.workspace_bytes = b["workspace"].data_ptr(), ws_bytes
            if not slot_workspaces:
                tracker.reserve(n, self.inst_per_chunk)
        N = max(int(total_clusters), 1)
        T = int(N * trk_frac) + 64
        hshapes = dict(trk_params=((T, 5), f32), trk_cov=((T, 15), f32), trk_nhits=((T,), i32), trk_sector=((T,), i32),
                       trk_hit_offset=((T + 1,), i64), trk_hits=((N,), i32), cluster_owner=((N,), i32))
        self.host = {k: t.empty(hshapes[k][0], dtype=hshapes[k][1], pin_memory=True) for k in want}
        self.hout = HostOutput()
        for k, v in self.host.items():
            setattr(self.hout, k, v.data_ptr())
        self.hout.trk_capacity, self.hout.trk_hits_capacity = T, N
        self.n_slots = n_slots
        h = C.c_void_p()
        with t.cuda.device(dev):
            tracker._check(tracker.lib.tpc_pipeline_create(tracker._h, self.slots, n_slots, C.byref(h)),
                           "tpc_pipeline_create")
        self._p = h

    def close(self):
        if getattr(self, "_p", None):
            self.trk.lib.tpc_pipeline_destroy(self._p)
            self._p = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def run(self, h_clusters, h_row_offsets, n_inst):
        """h_clusters: pinned torch tensor of the tracker's input layout ([N,4] f32 / [N,2] f32 / [N,2] i16);
        h_row_offsets: pinned int32 [n_inst*R+1].  Blocks.  Returns a snapshot (plain Python numbers) of what the
        call wrote into its tpc_host_output_t."""
        tr = self.trk
        n = int(h_clusters.shape[0])
        with tr._torch.cuda.device(tr.device):
            rc = tr.lib.tpc_pipeline_run(self._p, C.c_void_p(h_clusters.data_ptr()),
                                         C.c_void_p(h_row_offsets.data_ptr()), int(n_inst), n, self.inst_per_chunk,
                                         C.byref(self.hout))
        tr._check(rc, "tpc_pipeline_run")
        ho = self.hout
        return dict(totals=[int(x) for x in ho.totals], n_chunks=int(ho.n_chunks), n_launches=int(ho.n_launches),
                    h2d_bytes=int(ho.h2d_bytes), d2h_bytes=int(ho.d2h_bytes), h2d_ms=float(ho.h2d_ms),
                    compute_ms=float(ho.compute_ms), d2h_ms=float(ho.d2h_ms), wall_ms=float(ho.wall_ms))
