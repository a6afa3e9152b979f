"""Pins for the oracle's non-uniform pad-row pitch (reading A5'; "non-uniform pad-row
pitch with the weighted second difference").  Geometry: 63 rows of 0.75 cm, 64 of 1.0 cm, 32 of 1.5 cm.

What fixes the answer without retyping the oracle's formula: three collinear points have zero deviation whatever the
row steps, so straight tracks must link through both pitch boundaries even when they are steep enough that the plain
(unweighted) second difference would exceed the cut there; the window is a slope bound, so the same steep track must
be found in the 1.5 cm rows where it moves further than the fixed window of the default reading; grid == brute
force; noise-free helices are recovered with all hits and their generating parameters; and on equally spaced rows
nothing changes at all."""
import numpy as np
import pytest

from oracle.tpc_oracle import Oracle
from paper_1709_00618_b200 import datagen as dg

RX3 = dg.row_x_three_pad_sizes()
RX = dg.row_x()


def _event_from_rows(rows_yz, rx):
    cl, ro = [], [0]
    for r in range(len(rx)):
        for (y, z) in rows_yz.get(r, []):
            cl.append((rx[r], y, z, 0.0))
        ro.append(len(cl))
    return np.array(cl, np.float32).reshape(-1, 4), np.array(ro, np.int32)


def test_geometry_has_three_pad_sizes():
    d = np.diff(RX3.astype(np.float64))
    assert len(RX3) == 159 and np.allclose(d[:63], 0.75) and np.allclose(d[63:127], 1.0) and np.allclose(d[127:], 1.5)


@pytest.mark.parametrize("sy,sz", [(0.3, 0.5), (-1.0, 2.2), (1.2, -2.0)])
def test_straight_tracks_link_through_the_pitch_boundaries(sy, sz):
    """One straight track, one cluster per row.  Slopes (1.0, 2.2): at the 1.0 -> 1.5 cm boundary the plain second
    difference would be (0.5, 1.1) cm -> D = 1.46 > 1 (no link), and in the 1.5 cm rows the track moves 3.3 cm in z
    per row, beyond the fixed 2.5 cm window.  With reading A5' every interior hit links to its two neighbours."""
    x = RX3.astype(np.float64)
    rows = {r: [(sy * (x[r] - x[20]), 100.0 + sz * (x[r] - x[80]))] for r in range(20, 150)}
    cl, ro = _event_from_rows(rows, RX3)
    o = Oracle(RX3, 0.0)
    for use_grid in (True, False):
        up, dn = o.neighbours(cl, ro, 1, use_grid=use_grid)
        n = len(cl)
        assert np.array_equal(up[1:n - 1], np.arange(2, n)) and np.array_equal(dn[1:n - 1], np.arange(0, n - 2))
        assert up[0] == -1 and up[n - 1] == -1  # the end hits have no pair
    cu, cd = o.clean(up, dn)
    start, ch, cn = o.candidates(cu, cd)
    assert len(start) == 1 and start[0] == 1  # one chain over the whole track


def test_deviation_is_measured_from_the_line_not_from_the_mean():
    """Row 127 sits at the 1.0 -> 1.5 cm boundary (dd = 1.0, du = 1.5).  Its hit is displaced by e from the line
    (slope 1) through its partners in rows 126 and 128.  Reading A5' normalises the deviation so that equal steps give
    the plain second difference: wu = 2 dd / (du + dd) = 0.8, wd = 1.2, and a displacement e of the middle hit gives
    wu (1.5 - e) - wd (1 + e) = -2 e whatever the slope.  Cut D <= 1 -> linked iff |e| <= 0.5 cm, as for equal steps.
    (Unweighted, the slope alone would contribute 0.5 cm and the cut would sit at e = -0.25 / +0.75.)"""
    x = RX3.astype(np.float64)
    assert np.isclose(x[127] - x[126], 1.0) and np.isclose(x[128] - x[127], 1.5)
    for axis in (0, 1):
        for e, linked in ((0.45, True), (0.55, False), (-0.45, True), (-0.55, False)):
            def pt(r, off=0.0):
                v = 1.0 * (x[r] - x[127]) + off
                return (v, 50.0) if axis == 0 else (0.0, 50.0 + v)
            rows = {126: [pt(126)], 127: [pt(127, e)], 128: [pt(128)]}
            cl, ro = _event_from_rows(rows, RX3)
            up, dn = Oracle(RX3, 0.0).neighbours(cl, ro, 1)
            assert (up[1] == 2 and dn[1] == 0) == linked, (axis, e)


def test_grid_equals_brute_force_with_three_pad_sizes():
    rng = np.random.default_rng(31)
    rows = {}
    for r in range(55, 140):  # spans both boundaries
        n = rng.integers(3, 30)
        y = np.concatenate([rng.uniform(-6, 6, n), rng.uniform(-25, 25, 5)])
        z = np.concatenate([rng.uniform(100, 112, n), rng.uniform(0, 250, 5)])
        rows[r] = list(zip(y, z))
    cl, ro = _event_from_rows(rows, RX3)
    for cells in [(4.0, 5.0), (1.5, 2.0)]:
        o = Oracle(RX3, 0.5, grid_cell_y=cells[0], grid_cell_z=cells[1])
        ug, dg_ = o.neighbours(cl, ro, 1, use_grid=True)
        ub, db = o.neighbours(cl, ro, 1, use_grid=False)
        assert np.array_equal(ug, ub) and np.array_equal(dg_, db)
    assert (ug >= 0).sum() > 200


@pytest.mark.parametrize("bz", [0.5, 0.0])
def test_noise_free_tracks_recovered_with_three_pad_sizes(bz):
    rng = np.random.default_rng(41)
    n = 12
    trk = dict(pt=rng.uniform(0.8, 3.0, n), eta=np.linspace(0.05, 0.85, n), q=np.where(np.arange(n) % 2, 1.0, -1.0),
               phi0=rng.uniform(0.12, 0.23, n), x0=np.zeros(n), y0=np.zeros(n), z0=np.zeros(n))
    ev = dg.from_tracks(trk, bz=bz, rx=RX3)
    assert np.array_equal(ev.row_x, RX3) and np.all(np.isin(ev.clusters[:, 0], RX3))
    o = Oracle.for_event(ev)
    r = o.track(ev.clusters, ev.row_offsets, 1)
    labs = ev.labels
    assert len(r.trk_cand) == len(np.unique(labs))
    t64 = {k: np.asarray(v, float) for k, v in trk.items()}
    for t in range(len(r.trk_cand)):
        hits = r.trk_hits[r.trk_hit_offset[t]:r.trk_hit_offset[t + 1]]
        lab = labs[hits[0]]
        assert np.all(labs[hits] == lab) and len(hits) == (labs == lab).sum()
        tl = r.tracklets[r.trk_cand[t]]
        truth = dg.local_truth_state(t64, int(lab), float(RX3[tl["ref_row"]]), bz)
        if bz == 0.0:
            truth[4] = 0.0
        assert np.allclose(tl["p"], truth, rtol=1e-5, atol=2e-6), (tl["p"] - truth)


def test_equally_spaced_rows_keep_the_default_reading_bit_for_bit():
    """The step factors snap to exactly 1 on rows that pass the uniformity test, and x * 1.0f is exact: perturbing the
    uniform radii below that tolerance must not change a single link."""
    ev = dg.single_sector(seed=1041)
    u0, d0 = Oracle(RX, 0.5).neighbours(ev.clusters, ev.row_offsets, 1)
    rx_p = (RX.astype(np.float64) + np.random.default_rng(1).uniform(-2e-5, 2e-5, len(RX))).astype(np.float32)
    u1, d1 = Oracle(rx_p, 0.5).neighbours(ev.clusters, ev.row_offsets, 1)
    assert np.array_equal(u0, u1) and np.array_equal(d0, d1)
