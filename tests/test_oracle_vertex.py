"""Pins for the oracle's time-coordinate vertex estimate (oracle/tpc_oracle.c orc_track_vertex_z, orc_vertices;
DESIGN.md readings T1-T3; "the tracking will run in time coordinate first to estimate the vertex and only
then convert to spacial coordinates").

Independent references: the generator's closed-form helix (a track from the beam line has its closest approach AT its
origin), a brute-force scan of the helix for the closest approach of displaced tracks, the drift offsets the generator
applied to each collision of a CFG:4 window, truth labels, and hand-placed z_v values for the peak rule."""
import numpy as np
import pytest

from oracle.tpc_oracle import FIT_DTYPE, Oracle, Phase2Result
from paper_1709_00618_b200 import datagen as dg

RX = dg.row_x()
BZ = 0.5


def test_tracks_from_the_beam_line_point_back_to_their_origin():
    trk = dict(pt=np.array([0.25, 0.6, 3.0, 1.0]), eta=np.array([0.5, -0.8, 0.1, 0.7]), q=np.array([1.0, -1.0, 1.0, -1.0]),
               phi0=np.array([0.10, 0.25, 0.17, 0.30]), x0=np.zeros(4), y0=np.zeros(4), z0=np.array([0.0, 7.5, -3.0, 120.0]))
    for bz in (BZ, 0.0, -0.3):
        o = Oracle(RX, bz)
        for i in range(4):
            for x in (85.0, 130.0, 240.0):
                st = dg.local_truth_state(trk, i, x, bz)
                if not np.all(np.isfinite(st)) or abs(st[2]) > 0.95:
                    continue
                zv, dca = o.track_vertex_z(st, x)
                assert abs(zv - trk["z0"][i]) < 1e-8 and abs(dca) < 1e-8, (bz, i, x, zv, dca)


def test_displaced_tracks_against_a_brute_force_scan_of_the_helix():
    """Origin off the beam line: closest approach found by scanning the helix (generator's closed form at many planes,
    then a parabola through the three best samples)."""
    trk = dict(pt=np.array([0.5, 1.5, 0.8]), eta=np.array([0.4, -0.6, 0.2]), q=np.array([1.0, -1.0, -1.0]),
               phi0=np.array([0.15, 0.22, 0.12]), x0=np.array([6.0, -4.0, 10.0]), y0=np.array([8.0, 5.0, -12.0]),
               z0=np.array([3.0, -2.0, 1.0]))
    o = Oracle(RX, BZ)
    for i in range(3):
        xs = np.linspace(-40.0, 60.0, 20001)
        st = np.array([dg.local_truth_state(trk, i, x, BZ) for x in xs])
        ok = np.all(np.isfinite(st), axis=1) & (np.abs(st[:, 2]) < 0.999)
        r2 = np.where(ok, xs ** 2 + st[:, 0] ** 2, np.inf)
        k = int(np.argmin(r2))
        # parabolic refinement in the plane position
        a, b, c = r2[k - 1], r2[k], r2[k + 1]
        dx = 0.5 * (a - c) / (a - 2 * b + c) * (xs[1] - xs[0])
        sb = dg.local_truth_state(trk, i, xs[k] + dx, BZ)
        want_dca, want_z = np.hypot(xs[k] + dx, sb[0]), sb[1]
        zv, dca = o.track_vertex_z(dg.local_truth_state(trk, i, 120.0, BZ), 120.0)
        assert abs(abs(dca) - want_dca) < 1e-5 and abs(zv - want_z) < 1e-4, (i, dca, want_dca, zv, want_z)
        # the sign of dca is the side of the beam line: positive when it lies to the right of the direction of flight
        # (v = position across the direction, measured to the left, is positive at the closest approach)
        s, x, y = sb[2], xs[k] + dx, sb[0]
        assert np.sign(dca) == np.sign(-x * s + y * np.sqrt(1 - s * s))


def _fake_phase2(zvs, nhits=50, ok=1, dca=0.0):
    """Merged tracks whose z_v is zvs by construction: straight tracks (k = 0, sinPhi = 0, dz/ds = 0) at row 20 with
    y = dca -> u = x, v = dca, ds = -u, z_v = z."""
    fit = np.zeros(len(zvs), FIT_DTYPE)
    fit["ok"], fit["nhits"], fit["nseg"], fit["first_row"] = ok, nhits, 1, 20
    fit["p"][:, 1] = zvs
    fit["p"][:, 0] = dca
    e = np.zeros(0, np.int32)
    return Phase2Result(fit, e, e, np.arange(len(zvs), dtype=np.int32), fit)


def test_peak_rule_on_hand_placed_tracks():
    o = Oracle(RX, BZ, z_lo=-250.0, z_hi=500.0)
    rng = np.random.default_rng(2)
    a = 40.1 + rng.uniform(-0.05, 0.05, 12)
    b = 45.1 + rng.uniform(-0.05, 0.05, 12)   # 5 cm away: a second vertex
    few = -100.0 + rng.uniform(-0.05, 0.05, 9)  # 9 < 10: no vertex
    far = np.array([60.0])
    p2 = _fake_phase2(np.concatenate([a, b, few, far]))
    v = o.vertices(p2, np.zeros(len(p2.m_first), np.int32))
    assert len(v["vtx_z"]) == 2 and np.allclose(v["vtx_z"], [a.mean(), b.mean()], atol=1e-9)
    assert list(v["vtx_ntracks"]) == [12, 12] and np.all(v["trk_vtx"][:12] == 0) and np.all(v["trk_vtx"][12:24] == 1)
    assert np.all(v["trk_vtx"][24:] == -1)
    # two windows: vertices are per window (instances 0..35 and 36..71), listed window by window; a track is only
    # assigned to a vertex of its own window
    inst = np.concatenate([np.zeros(12, np.int32), np.full(22, 36, np.int32)])
    v = o.vertices(p2, inst)
    assert list(v["vtx_window"]) == [0, 1] and np.allclose(v["vtx_z"], [a.mean(), b.mean()], atol=1e-9)
    p2b = _fake_phase2(np.concatenate([a, a + 1.0]))
    v = o.vertices(p2b, np.concatenate([np.zeros(12, np.int32), np.full(12, 36, np.int32)]))
    assert list(v["vtx_window"]) == [0, 1] and np.all(v["trk_vtx"][:12] == 0) and np.all(v["trk_vtx"][12:] == 1)
    # resolution of the rule: the seed is the maximum of the 3-bin sums over +-4 bins, so two equally populated
    # collisions 3 cm apart are ONE seed (the lower one); its position averages the tracks within 1.5 cm only
    p2c = _fake_phase2(np.concatenate([a, a + 3.0]))
    v = o.vertices(p2c, np.zeros(24, np.int32))
    assert len(v["vtx_z"]) == 1 and np.isclose(v["vtx_z"][0], a.mean(), atol=1e-9)
    # a plateau: 5 tracks in one bin and 5 in the next -> one seed (the lower bin), vertex = mean of all ten
    lo, hi = 10.0 + 0.1, 10.5 + 0.1
    p2 = _fake_phase2(np.concatenate([np.full(5, lo), np.full(5, hi)]))
    v = o.vertices(p2, np.zeros(10, np.int32))
    assert len(v["vtx_z"]) == 1 and np.isclose(v["vtx_z"][0], 0.5 * (lo + hi))
    # tracks that are not vertex-like (few hits, large dca, failed fit) do not vote but are assigned within 3 cm
    z = np.concatenate([np.full(12, 5.0), [5.5, 7.9, 8.1]])
    p2 = _fake_phase2(z)
    p2.m_fit["nhits"][12:] = 12
    v = o.vertices(p2, np.zeros(len(z), np.int32))
    assert len(v["vtx_z"]) == 1 and np.isclose(v["vtx_z"][0], 5.0) and list(v["trk_vtx"][12:]) == [0, 0, -1]
    p2 = _fake_phase2(np.full(15, 5.0), dca=3.5)  # |dca| > 3 cm: not vertex-like -> no votes, no vertex
    assert len(o.vertices(p2, np.zeros(15, np.int32))["vtx_z"]) == 0


def test_drift_window_vertices_are_the_generated_drift_offsets():
    """CFG:4: five collisions, each shifted in z by its drift offset; every collision's primaries come from z = 0, so
    its vertex in the time-like coordinate IS the offset.  All collisions with >= 30 reconstructed tracks are found,
    to 0.05 cm, and tracks go to the vertex of their own collision."""
    ev = dg.drift_window(seed=4005, mean_tracks=300.0, cap_tracks=800)
    o = Oracle.for_event(ev)
    r = o.track(ev.clusters, ev.row_offsets, ev.n_inst)
    p2 = o.phase2(ev.clusters, ev.row_offsets, ev.n_inst, r)
    R = ev.n_rows
    inst = np.searchsorted(ev.row_offsets[::R], r.cand_hits[r.trk_cand, 0], side="right") - 1
    v = o.vertices(p2, inst[p2.m_first])
    shifts = np.unique(ev.truth["z_shift"])
    n_gen = np.array([(ev.truth["z_shift"] == s).sum() for s in shifts])
    assert len(shifts) == 5
    found = [np.abs(v["vtx_z"] - s).min() < 0.05 for s in shifts]
    assert all(f for f, n in zip(found, n_gen) if n >= 60), (v["vtx_z"], shifts, n_gen)
    assert len(v["vtx_z"]) <= 5 and np.all(np.diff(v["vtx_z"]) > 0)
    # purity: the drift offset of a track's truth particle equals its vertex
    lab = np.array([ev.labels[r.trk_hits[r.trk_hit_offset[t]]] for t in p2.m_first])
    has = (v["trk_vtx"] >= 0) & (lab >= 0)
    good = np.abs(ev.truth["z_shift"][lab[has]] - v["vtx_z"][v["trk_vtx"][has]]) < 0.1
    assert has.sum() > 0.9 * len(lab) and good.mean() > 0.99
    assert v["vtx_ntracks"].sum() == (v["trk_vtx"] >= 0).sum()
