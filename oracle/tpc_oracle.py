"""ctypes wrapper around oracle/tpc_oracle.c (plain C, gcc).  TEST INFRASTRUCTURE, not product.

Builds liboracle_tpc.so next to the source on first use (gcc -O2 -ffp-contract=off, no fast-math).
Every function here only marshals numpy arrays; all arithmetic is in the C file, which cites the
passages it follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tpc_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_tpc.so")

CAND_MAX = 10


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
               "-Wall", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class Config(C.Structure):
    _fields_ = [
        ("n_rows", C.c_int32), ("row_x", C.POINTER(C.c_float)), ("sectors_per_event", C.c_int32),
        ("half_angle_rad", C.c_float), ("z_lo", C.c_float), ("z_hi", C.c_float), ("sigma_y", C.c_float),
        ("sigma_z", C.c_float), ("nf_win_y", C.c_float), ("nf_win_z", C.c_float), ("nf_d2_max", C.c_float),
        ("cand_min_hits", C.c_int32), ("cand_max_hits", C.c_int32), ("kf_p0", C.c_double * 5),
        ("kf_gate_sigma", C.c_double), ("kf_win_max", C.c_double), ("kf_max_gap", C.c_int32),
        ("kf_max_sinphi", C.c_double), ("kf_edge_margin", C.c_double), ("sel_min_hits", C.c_int32),
        ("grid_cell_y", C.c_float), ("grid_cell_z", C.c_float), ("bz", C.c_double),
        ("nf_bridge_rows", C.c_int32), ("pad_", C.c_int32),
    ]


class Tracklet(C.Structure):
    _fields_ = [("ok", C.c_int32), ("nhits", C.c_int32), ("first_row", C.c_int32), ("last_row", C.c_int32),
                ("ref_row", C.c_int32), ("p", C.c_double * 5), ("cov", C.c_double * 15), ("chi2", C.c_double)]


TRACKLET_DTYPE = np.dtype([("ok", "<i4"), ("nhits", "<i4"), ("first_row", "<i4"), ("last_row", "<i4"),
                           ("ref_row", "<i4"), ("_pad", "<i4"), ("p", "<f8", (5,)), ("cov", "<f8", (15,)),
                           ("chi2", "<f8")])

FIT_DTYPE = np.dtype([("ok", "<i4"), ("nhits", "<i4"), ("nseg", "<i4"), ("first_row", "<i4"), ("p", "<f8", (5,)),
                      ("cov", "<f8", (15,)), ("chi2", "<f8")])


class Segment(C.Structure):
    _fields_ = [("sector", C.c_int32), ("n", C.c_int32), ("rows", C.POINTER(C.c_int32)), ("y", C.POINTER(C.c_float)),
                ("z", C.POINTER(C.c_float))]


@dataclass
class Phase2Result:
    seg_fit: np.ndarray    # FIT_DTYPE [n_tracks]: refit of every final track alone (kept hits only)
    seg_next: np.ndarray   # [n_tracks] track that continues this one outward in the neighbouring sector, or -1
    seg_prev: np.ndarray
    m_first: np.ndarray    # [n_merged] innermost segment (track index) of every merged track, ascending
    m_fit: np.ndarray      # FIT_DTYPE [n_merged]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        assert _lib.orc_sizeof_tracklet() == C.sizeof(Tracklet) == TRACKLET_DTYPE.itemsize
        assert _lib.orc_sizeof_config() == C.sizeof(Config)
        _lib.orc_update.restype = C.c_double
        _lib.orc_phase2.restype = C.c_int64
        _lib.orc_vertices.restype = C.c_int64
        assert _lib.orc_sizeof_fit() == FIT_DTYPE.itemsize and _lib.orc_sizeof_segment() == C.sizeof(Segment)
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


@dataclass
class OracleResult:
    link_up_raw: np.ndarray
    link_dn_raw: np.ndarray
    link_up: np.ndarray
    link_dn: np.ndarray
    start_hits: np.ndarray
    cand_hits: np.ndarray  # [n_cand, 10]
    cand_n: np.ndarray
    tracklets: np.ndarray  # TRACKLET_DTYPE [n_cand]
    tracklet_hits: np.ndarray  # [n_cand, n_rows] global cluster index or -1
    cluster_owner: np.ndarray  # [N] final track index or -1
    trk_cand: np.ndarray  # [n_tracks]
    trk_hit_offset: np.ndarray  # [n_tracks+1]
    trk_hits: np.ndarray


class Oracle:
    """Holds the configuration (SURVEY.md 8(c) constants are the defaults) and exposes the stages."""

    def __init__(self, row_x, bz, *, z_lo=0.0, z_hi=250.0, sigma_y=0.1, sigma_z=0.1, sectors_per_event=36,
                 half_angle_rad=float(np.deg2rad(10.0)), nf_win_y=2.0, nf_win_z=2.5, nf_d2_max=1.0, cand_min_hits=4,
                 cand_max_hits=CAND_MAX, kf_p0=(1.0, 1.0, 0.1, 0.1, 10.0), kf_gate_sigma=4.0, kf_win_max=3.0,
                 kf_max_gap=5, kf_max_sinphi=0.95, kf_edge_margin=2.0, sel_min_hits=10, grid_cell_y=4.0,
                 grid_cell_z=5.0, nf_bridge_rows=0):
        self._row_x = np.ascontiguousarray(row_x, dtype=np.float32)
        c = Config()
        c.n_rows = len(self._row_x)
        c.row_x = _p(self._row_x, C.c_float)
        c.sectors_per_event = sectors_per_event
        c.half_angle_rad = half_angle_rad
        c.z_lo, c.z_hi, c.sigma_y, c.sigma_z = z_lo, z_hi, sigma_y, sigma_z
        c.nf_win_y, c.nf_win_z, c.nf_d2_max = nf_win_y, nf_win_z, nf_d2_max
        c.cand_min_hits, c.cand_max_hits = cand_min_hits, cand_max_hits
        for i in range(5):
            c.kf_p0[i] = kf_p0[i]
        c.kf_gate_sigma, c.kf_win_max, c.kf_max_gap = kf_gate_sigma, kf_win_max, kf_max_gap
        c.kf_max_sinphi, c.kf_edge_margin, c.sel_min_hits = kf_max_sinphi, kf_edge_margin, sel_min_hits
        c.grid_cell_y, c.grid_cell_z, c.bz = grid_cell_y, grid_cell_z, bz
        c.nf_bridge_rows = int(nf_bridge_rows)
        self.cfg = c
        self.n_rows = c.n_rows
        self.bz = bz
        self.c_b = -0.00299792458 * bz

    @classmethod
    def for_event(cls, ev, **kw):
        return cls(ev.row_x, ev.bz, z_lo=ev.z_lo, z_hi=ev.z_hi, sigma_y=ev.sigma_y,
                   sigma_z=ev.sigma_z, **kw)

    # ---- stages -------------------------------------------------------------------------------------------
    def neighbours(self, clusters, row_offsets, n_inst, use_grid=True):
        cl = np.ascontiguousarray(clusters, np.float32)
        ro = np.ascontiguousarray(row_offsets, np.int32)
        n = cl.shape[0]
        up = np.empty(max(n, 1), np.int32)
        dn = np.empty(max(n, 1), np.int32)
        lib().orc_neighbours(C.byref(self.cfg), _p(cl, C.c_float), _p(ro, C.c_int32), C.c_int32(n_inst),
                             C.c_int32(1 if use_grid else 0), _p(up, C.c_int32), _p(dn, C.c_int32))
        return up[:n], dn[:n]

    def clean(self, up, dn):
        n = len(up)
        up = np.ascontiguousarray(up, np.int32)
        dn = np.ascontiguousarray(dn, np.int32)
        cu = np.empty(max(n, 1), np.int32)
        cd = np.empty(max(n, 1), np.int32)
        lib().orc_clean(C.c_int64(n), _p(up, C.c_int32), _p(dn, C.c_int32), _p(cu, C.c_int32), _p(cd, C.c_int32))
        return cu[:n], cd[:n]

    def candidates(self, cu, cd):
        n = len(cu)
        cu = np.ascontiguousarray(cu, np.int32)
        cd = np.ascontiguousarray(cd, np.int32)
        cnt = np.zeros(2, np.int64)
        M = self.cfg.cand_max_hits
        lib().orc_candidates(C.byref(self.cfg), C.c_int64(n), _p(cu, C.c_int32), _p(cd, C.c_int32), None,
                             C.c_int64(0), None, None, C.c_int64(0), _p(cnt, C.c_int64))
        ns, nc = int(cnt[0]), int(cnt[1])
        sh = np.empty(max(ns, 1), np.int32)
        ch = np.empty((max(nc, 1), M), np.int32)
        cn = np.empty(max(nc, 1), np.int32)
        lib().orc_candidates(C.byref(self.cfg), C.c_int64(n), _p(cu, C.c_int32), _p(cd, C.c_int32),
                             _p(sh, C.c_int32), C.c_int64(ns), _p(ch, C.c_int32), _p(cn, C.c_int32), C.c_int64(nc),
                             _p(cnt, C.c_int64))
        return sh[:ns], ch[:nc], cn[:nc]

    def follow(self, clusters, row_offsets, n_inst, cand_hits, cand_n, use_grid=True):
        cl = np.ascontiguousarray(clusters, np.float32)
        ro = np.ascontiguousarray(row_offsets, np.int32)
        ch = np.ascontiguousarray(cand_hits, np.int32)
        cn = np.ascontiguousarray(cand_n, np.int32)
        nc = len(cn)
        tl = np.zeros(max(nc, 1), TRACKLET_DTYPE)
        th = np.full((max(nc, 1), self.n_rows), -1, np.int32)
        if nc:
            lib().orc_follow(C.byref(self.cfg), _p(cl, C.c_float), _p(ro, C.c_int32), C.c_int32(n_inst),
                             _p(ch, C.c_int32), _p(cn, C.c_int32), C.c_int64(nc), C.c_int32(1 if use_grid else 0),
                             C.cast(tl.ctypes.data, C.POINTER(Tracklet)), _p(th, C.c_int32))
        return tl[:nc], th[:nc]

    def select(self, n_clusters, tracklets, tracklet_hits):
        nc = len(tracklets)
        tl = np.ascontiguousarray(tracklets)
        th = np.ascontiguousarray(tracklet_hits, np.int32)
        owner = np.empty(max(n_clusters, 1), np.int32)
        tc = np.empty(max(nc, 1), np.int32)
        tho = np.zeros(nc + 2, np.int64)
        thl = np.empty(max(n_clusters, 1), np.int32)
        cnt = np.zeros(2, np.int64)
        lib().orc_select(C.byref(self.cfg), C.c_int64(n_clusters), C.cast(tl.ctypes.data, C.POINTER(Tracklet)),
                         _p(th, C.c_int32), C.c_int64(nc), _p(owner, C.c_int32), _p(tc, C.c_int32),
                         _p(tho, C.c_int64), _p(thl, C.c_int32), C.c_int64(max(nc, 1)), C.c_int64(max(n_clusters, 1)),
                         _p(cnt, C.c_int64))
        nt, nh = int(cnt[0]), int(cnt[1])
        return owner[:n_clusters], tc[:nt], tho[:nt + 1], thl[:nh]

    def track(self, clusters, row_offsets, n_inst, use_grid=True) -> OracleResult:
        up, dn = self.neighbours(clusters, row_offsets, n_inst, use_grid)
        cu, cd = self.clean(up, dn)
        sh, ch, cn = self.candidates(cu, cd)
        tl, th = self.follow(clusters, row_offsets, n_inst, ch, cn, use_grid)
        owner, tc, tho, thl = self.select(len(clusters), tl, th)
        return OracleResult(up, dn, cu, cd, sh, ch, cn, tl, th, owner, tc, tho, thl)

    def track_count(self, clusters, row_offsets, n_inst, n_threads=1):
        """Whole chain per instance, totals only (the timed cpu_baseline entry)."""
        cl = np.ascontiguousarray(clusters, np.float32)
        ro = np.ascontiguousarray(row_offsets, np.int32)
        cnt = np.zeros(5, np.int64)
        lib().orc_track_count(C.byref(self.cfg), _p(cl, C.c_float), _p(ro, C.c_int32), C.c_int32(n_inst),
                              C.c_int32(n_threads), _p(cnt, C.c_int64))
        return dict(n_start=int(cnt[0]), n_cand=int(cnt[1]), n_tracklets=int(cnt[2]), n_tracks=int(cnt[3]),
                    n_track_hits=int(cnt[4]))

    # ---- filter pieces (for the pins) -----------------------------------------------------------------------
    def transport(self, p, P, dx, want_jac=False):
        p = np.ascontiguousarray(p, np.float64)
        P = np.ascontiguousarray(P, np.float64).reshape(25)
        p1 = np.empty(5)
        P1 = np.empty(25)
        F = np.empty(25)
        rc = lib().orc_transport(_p(p, C.c_double), _p(P, C.c_double), C.c_double(dx), C.c_double(self.c_b),
                                 C.c_double(self.cfg.kf_max_sinphi), _p(p1, C.c_double), _p(P1, C.c_double),
                                 _p(F, C.c_double))
        if rc:
            return None
        return (p1, P1.reshape(5, 5), F.reshape(5, 5)) if want_jac else (p1, P1.reshape(5, 5))

    def update(self, p, P, ym, zm):
        p = np.array(p, np.float64)
        P = np.array(P, np.float64).reshape(25)
        sy2 = float(self.cfg.sigma_y) ** 2
        sz2 = float(self.cfg.sigma_z) ** 2
        chi2 = lib().orc_update(_p(p, C.c_double), _p(P, C.c_double), C.c_double(ym), C.c_double(zm),
                                C.c_double(sy2), C.c_double(sz2))
        return p, P.reshape(5, 5), chi2

    def seed(self, x, y, z):
        x = np.ascontiguousarray(x, np.float64)
        y = np.ascontiguousarray(y, np.float64)
        z = np.ascontiguousarray(z, np.float64)
        p = np.empty(5)
        lib().orc_seed(_p(x, C.c_double), _p(y, C.c_double), _p(z, C.c_double), C.c_double(self.c_b),
                       _p(p, C.c_double))
        return p


    # ---- phase 2: sector merger + refit -------------------------------------------------
    def rotate(self, p, P, x, alpha, want_jac=False):
        """State on the plane x of one sector frame -> state in the frame rotated by +alpha (reading M2).  Returns
        (p1, P1, x1[, J]) or None."""
        p = np.ascontiguousarray(p, np.float64)
        P = np.ascontiguousarray(P, np.float64).reshape(25)
        p1, P1, J = np.empty(5), np.empty(25), np.empty(25)
        x1 = C.c_double()
        rc = lib().orc_rotate(_p(p, C.c_double), _p(P, C.c_double), C.c_double(x), C.c_double(alpha),
                              C.c_double(self.c_b), C.c_double(self.cfg.kf_max_sinphi), _p(p1, C.c_double),
                              _p(P1, C.c_double), C.byref(x1), _p(J, C.c_double))
        if rc:
            return None
        out = (p1, P1.reshape(5, 5), x1.value)
        return out + (J.reshape(5, 5),) if want_jac else out

    def refit_chain(self, segments):
        """segments: list of (sector, rows, y, z) inside out, rows increasing (readings M1, M4).  Returns a FIT_DTYPE
        record."""
        keep, segs = [], (Segment * len(segments))()
        for i, (sec, rows, y, z) in enumerate(segments):
            r = np.ascontiguousarray(rows, np.int32)
            yy = np.ascontiguousarray(y, np.float32)
            zz = np.ascontiguousarray(z, np.float32)
            keep.append((r, yy, zz))
            segs[i].sector, segs[i].n = int(sec), len(r)
            segs[i].rows, segs[i].y, segs[i].z = _p(r, C.c_int32), _p(yy, C.c_float), _p(zz, C.c_float)
        f = np.zeros(1, FIT_DTYPE)
        lib().orc_refit_chain(C.byref(self.cfg), segs, C.c_int(len(segments)), C.c_void_p(f.ctypes.data))
        return f[0]

    def phase2(self, clusters, row_offsets, n_inst, res: "OracleResult") -> Phase2Result:
        """Merger + refit on the final tracks of `res` (an OracleResult of the same input)."""
        ro = np.ascontiguousarray(row_offsets, np.int32)
        nt = len(res.trk_cand)
        inst = (np.searchsorted(ro[::self.n_rows], res.cand_hits[res.trk_cand, 0], side="right") - 1).astype(np.int32) \
            if nt else np.zeros(0, np.int32)
        return self.phase2_on_tracks(clusters, row_offsets, n_inst, inst, res.trk_hit_offset, res.trk_hits)

    def phase2_on_tracks(self, clusters, row_offsets, n_inst, trk_inst, trk_hit_offset, trk_hits) -> Phase2Result:
        """Merger + refit (orc_phase2) on ANY list of final tracks of this input: sector instance per track, CSR
        offsets and kept hits (global cluster indices, rows increasing).  The GPU parity tests pass the GPU's own
        S6 output here, so that phase 2 is compared on identical tracks at sizes where S5 near-ties flip."""
        cl = np.ascontiguousarray(clusters, np.float32)
        ro = np.ascontiguousarray(row_offsets, np.int32)
        nt = len(trk_inst)
        inst = np.ascontiguousarray(trk_inst, np.int32)
        off = np.ascontiguousarray(trk_hit_offset, np.int64)
        hits = np.ascontiguousarray(trk_hits, np.int32)
        seg_fit = np.zeros(max(nt, 1), FIT_DTYPE)
        m_fit = np.zeros(max(nt, 1), FIT_DTYPE)
        nxt = np.full(max(nt, 1), -1, np.int32)
        prv = np.full(max(nt, 1), -1, np.int32)
        mf = np.full(max(nt, 1), -1, np.int32)
        nm = lib().orc_phase2(C.byref(self.cfg), _p(cl, C.c_float), _p(ro, C.c_int32), C.c_int32(n_inst),
                              C.c_int64(nt), _p(inst, C.c_int32), _p(off, C.c_int64), _p(hits, C.c_int32),
                              C.c_void_p(seg_fit.ctypes.data), _p(nxt, C.c_int32), _p(prv, C.c_int32),
                              _p(mf, C.c_int32), C.c_void_p(m_fit.ctypes.data)) if nt else 0
        return Phase2Result(seg_fit[:nt], nxt[:nt], prv[:nt], mf[:nm], m_fit[:nm])


    # ---- time-coordinate tracking: vertex estimate (readings T1-T3) -----------------------
    def track_vertex_z(self, p, x):
        """(z_v, dca) of a state p on the plane x: closest approach to the beam line (reading T1)."""
        p = np.ascontiguousarray(p, np.float64)
        zv, dca = C.c_double(), C.c_double()
        lib().orc_track_vertex_z(_p(p, C.c_double), C.c_double(x), C.c_double(self.c_b), C.byref(zv), C.byref(dca))
        return zv.value, dca.value

    def vertices(self, p2: "Phase2Result", m_inst, vtx_cap=4096):
        """Readings T1-T3 on the merged tracks of phase2().  m_inst: sector instance of every merged track's innermost
        segment.  Returns dict(trk_zv, trk_dca, trk_vtx, vtx_z, vtx_window, vtx_ntracks)."""
        nm = len(p2.m_first)
        fit = np.ascontiguousarray(p2.m_fit)
        inst = np.ascontiguousarray(m_inst, np.int32)
        zv, dca = np.zeros(max(nm, 1)), np.zeros(max(nm, 1))
        tv = np.full(max(nm, 1), -1, np.int32)
        vz = np.zeros(vtx_cap)
        vw = np.zeros(vtx_cap, np.int32)
        vn = np.zeros(vtx_cap, np.int32)
        nv = lib().orc_vertices(C.byref(self.cfg), C.c_int64(nm), C.c_void_p(fit.ctypes.data), _p(inst, C.c_int32),
                                _p(zv, C.c_double), _p(dca, C.c_double), _p(tv, C.c_int32), _p(vz, C.c_double),
                                _p(vw, C.c_int32), _p(vn, C.c_int32), C.c_int64(vtx_cap)) if nm else 0
        assert nv <= vtx_cap
        return dict(trk_zv=zv[:nm], trk_dca=dca[:nm], trk_vtx=tv[:nm], vtx_z=vz[:nv], vtx_window=vw[:nv],
                    vtx_ntracks=vn[:nv])


def unpack_cov(c15):
    P = np.zeros((5, 5))
    k = 0
    for i in range(5):
        for j in range(i + 1):
            P[i, j] = P[j, i] = c15[k]
            k += 1
    return P
