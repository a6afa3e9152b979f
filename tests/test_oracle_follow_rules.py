"""Pins for the oracle's S5 pick-up and stop rules (oracle/tpc_oracle.c pickup(), follow_dir(); DESIGN.md readings
A9/A10; "extrapolates the trajectory through the TPC sector volume to pick up additional clusters").

Every case is a hand-placed Bz = 0 straight track with zero smear whose answer is evident from the rule itself:
which of several clusters inside the gate is attached (the nearest), which of two exact duplicates (the lowest local
index), where the gate ends (4 sigma, capped at 3 cm), how many consecutive empty rows are tolerated (5, and a hit
resets the count), and where a track that leaves the wedge stops (the first row with |y| > x tan(10 deg) + 2 cm).
The candidate is given to orc_follow directly, so S2-S4 play no part.  The last test is the weighted-least-squares
pin of the filter arithmetic: in the linear regime the sequential filter must equal a one-shot regression (numpy)
with the prior folded in.
"""
import numpy as np
import pytest

from oracle.tpc_oracle import Oracle, unpack_cov
from paper_1709_00618_b200 import datagen as dg

RX = dg.row_x()
TAN10 = float(np.tan(np.deg2rad(10.0)))


class Line:
    """Straight track y = y0 + my (x - x_ref), z = z0 + mz (x - x_ref); one cluster per row in `rows`."""

    def __init__(self, rows, *, y0=1.0, my=0.05, z0=100.0, mz=0.3, x_ref=float(RX[0])):
        self.y0, self.my, self.z0, self.mz, self.x_ref = y0, my, z0, mz, x_ref
        self.rows = {int(r): [self.at(r)] for r in rows}  # row -> list of (y, z); the track's own cluster first

    def at(self, r, dy=0.0, dz=0.0):
        x = float(RX[r])
        return (self.y0 + self.my * (x - self.x_ref) + dy, self.z0 + self.mz * (x - self.x_ref) + dz)

    def drop(self, rows):
        for r in rows:
            self.rows.pop(int(r), None)
        return self

    def event(self):
        cl, ro, first = [], [0], {}
        for r in range(len(RX)):
            first[r] = len(cl)
            for (y, z) in self.rows.get(r, []):
                cl.append((RX[r], y, z, 0.0))
            ro.append(len(cl))
        return np.array(cl, np.float32).reshape(-1, 4), np.array(ro, np.int32), first


def _follow(line, cand_rows, **okw):
    """Follow the candidate made of the FIRST cluster of each row in cand_rows.  Returns (tracklet, hits[R], first
    global index per row)."""
    cl, ro, first = line.event()
    o = Oracle(RX, 0.0, **okw)
    ch = np.full((1, 10), -1, np.int32)
    ch[0, :len(cand_rows)] = [first[r] for r in cand_rows]
    for use_grid in (True, False):  # the grid is an acceleration structure: both searches must agree
        tl, th = o.follow(cl, ro, 1, ch, np.array([len(cand_rows)], np.int32), use_grid=use_grid)
        if use_grid:
            ref = (tl.copy(), th.copy())
        else:
            assert np.array_equal(th, ref[1]) and tl["nhits"][0] == ref[0]["nhits"][0]
    assert tl["ok"][0] == 1
    return tl[0], th[0], first


CAND = list(range(60, 70))


def test_complete_track_is_followed_both_ways():
    t, h, first = _follow(Line(range(30, 121)), CAND)
    assert t["nhits"] == 91 and t["first_row"] == 30 and t["last_row"] == 120 and t["ref_row"] == 30
    assert all(h[r] == first[r] for r in range(30, 121)) and np.all(h[:30] == -1) and np.all(h[121:] == -1)


# ---------------------------------------------------------------- pickup(): nearest, ties, gate

@pytest.mark.parametrize("extra_first", [False, True])
def test_nearest_of_two_clusters_in_the_gate_is_attached(extra_first):
    """Row 85 holds the track's cluster and a second one 0.2 cm away in y (inside the >= 0.4 cm gate): the nearer
    one (distance 0) is attached wherever it sits in the row."""
    ln = Line(range(30, 121))
    ln.rows[85] = [ln.at(85, dy=0.2), ln.at(85)] if extra_first else [ln.at(85), ln.at(85, dy=0.2)]
    t, h, first = _follow(ln, CAND)
    assert h[85] == first[85] + (1 if extra_first else 0)
    assert t["nhits"] == 91


def test_nearer_impostor_wins_over_the_displaced_true_cluster():
    """Distances 0.05 cm (z) against 0.15 cm (y): the metric is Euclidean in (y, z), the smaller one wins."""
    ln = Line(range(30, 121))
    ln.rows[85] = [ln.at(85, dy=0.15), ln.at(85, dz=-0.05)]
    _, h, first = _follow(ln, CAND)
    assert h[85] == first[85] + 1
    ln.rows[85] = [ln.at(85, dy=0.15, dz=0.15), ln.at(85, dy=-0.2)]  # 0.212 against 0.2: not a per-axis maximum rule
    _, h, first = _follow(ln, CAND)
    assert h[85] == first[85] + 1


def test_exact_duplicates_attach_the_lowest_local_index():
    ln = Line(range(30, 121))
    ln.rows[85] = [ln.at(85, dy=0.3), ln.at(85), ln.at(85), ln.at(85)]  # duplicates at local indices 1, 2, 3
    ln.rows[40] = [ln.at(40), ln.at(40)]                                # and in the downward phase
    _, h, first = _follow(ln, CAND)
    assert h[85] == first[85] + 1 and h[40] == first[40]


def test_gate_is_four_sigma_of_the_predicted_residual():
    """sigma = 0.1 cm: the gate is 4 sqrt(P + 0.01) >= 0.4 cm, and < 0.57 cm once the prediction error is below the
    cluster error (it is, after ten hits).  A lone cluster 0.39 cm off is attached, one 0.6 cm off is not."""
    for off, attached in ((0.39, True), (-0.39, True), (0.6, False), (-0.6, False)):
        for axis in ("y", "z"):
            ln = Line(range(30, 121))
            ln.rows[85] = [ln.at(85, dy=off) if axis == "y" else ln.at(85, dz=off)]
            _, h, first = _follow(ln, CAND)
            assert (h[85] == first[85]) == attached, (off, axis)
            assert h[86] == first[86]  # one empty row does not stop the track


def test_gate_is_capped_at_three_centimetres():
    """sigma = 1 cm makes 4 sigma >= 4 cm, so the cap (kf_win_max = 3 cm) is the gate: 2.9 cm in, 3.1 cm out."""
    for off, attached in ((2.9, True), (3.1, False), (-2.9, True), (-3.1, False)):
        for axis in ("y", "z"):
            ln = Line(range(30, 121), y0=0.0, my=0.0)
            ln.rows[85] = [ln.at(85, dy=off) if axis == "y" else ln.at(85, dz=off)]
            _, h, first = _follow(ln, CAND, sigma_y=1.0, sigma_z=1.0)
            assert (h[85] == first[85]) == attached, (off, axis)
    # and the cap is the parameter: 2 cm
    ln = Line(range(30, 121), y0=0.0, my=0.0)
    ln.rows[85] = [ln.at(85, dy=2.5)]
    _, h, _ = _follow(ln, CAND, sigma_y=1.0, sigma_z=1.0, kf_win_max=2.0)
    assert h[85] == -1


# ---------------------------------------------------------------- follow_dir(): gap counter, edge stop

def test_five_empty_rows_are_bridged_six_stop_the_track_upward():
    t, h, first = _follow(Line(range(30, 121)).drop(range(80, 85)), CAND)  # rows 80..84 empty
    assert t["last_row"] == 120 and t["nhits"] == 91 - 5 and all(h[r] == first[r] for r in range(85, 121))
    t, h, first = _follow(Line(range(30, 121)).drop(range(80, 86)), CAND)  # rows 80..85 empty
    assert t["last_row"] == 79 and np.all(h[80:] == -1)
    assert t["nhits"] == 79 - 30 + 1 and t["first_row"] == 30  # the downward phase is unaffected


def test_five_empty_rows_are_bridged_six_stop_the_track_downward():
    t, h, first = _follow(Line(range(30, 121)).drop(range(45, 50)), CAND)  # rows 45..49 empty
    assert t["first_row"] == 30 and t["ref_row"] == 30 and t["nhits"] == 91 - 5
    assert all(h[r] == first[r] for r in range(30, 45))
    t, h, first = _follow(Line(range(30, 121)).drop(range(44, 50)), CAND)  # rows 44..49 empty
    assert t["first_row"] == 50 and t["ref_row"] == 50 and np.all(h[:50] == -1)
    assert t["nhits"] == 120 - 50 + 1 and t["last_row"] == 120


def test_a_hit_resets_the_gap_counter():
    """5 empty rows, one hit, 5 empty rows: the track continues (the counter is consecutive rows, not a total)."""
    ln = Line(range(30, 121)).drop(range(80, 85)).drop(range(86, 91))
    t, h, first = _follow(ln, CAND)
    assert h[85] == first[85] and t["last_row"] == 120 and t["nhits"] == 91 - 10
    ln = Line(range(30, 121)).drop(range(34, 39)).drop(range(40, 45))
    t, h, first = _follow(ln, CAND)
    assert h[39] == first[39] and t["first_row"] == 30 and t["nhits"] == 91 - 10


def test_gap_limit_is_the_parameter():
    t, _, _ = _follow(Line(range(30, 121)).drop(range(80, 83)), CAND, kf_max_gap=2)  # 3 empty rows > 2
    assert t["last_row"] == 79
    t, _, _ = _follow(Line(range(30, 121)).drop(range(80, 82)), CAND, kf_max_gap=2)  # 2 empty rows
    assert t["last_row"] == 120


def test_track_stops_at_the_first_row_beyond_the_sector_edge_margin():
    """y = 0.45 (x - 100): |y| <= x tan(10 deg) + 2 cm holds up to row 84 (by 0.17 cm) and fails at row 85 (by
    0.11 cm).  Clusters keep lying on the line beyond the edge; none of them may be attached."""
    ln = Line(range(20, 110), y0=0.0, my=0.45, x_ref=100.0, z0=50.0, mz=0.2)
    x = RX.astype(np.float64)
    inside = np.abs(0.45 * (x - 100.0)) <= x * TAN10 + 2.0
    assert inside[84] and not inside[85]
    t, h, first = _follow(ln, list(range(40, 50)))
    assert t["last_row"] == 84 and np.all(h[85:] == -1) and all(h[r] == first[r] for r in range(20, 85))
    # mirrored in y, and a wider margin moves the stop outward: 0.45 (x-100) = x tan10 + 4 at x = 179.05 -> row 91
    ln = Line(range(20, 110), y0=0.0, my=-0.45, x_ref=100.0, z0=50.0, mz=0.2)
    t, h, _ = _follow(ln, list(range(40, 50)))
    assert t["last_row"] == 84
    inside4 = np.abs(0.45 * (x - 100.0)) <= x * TAN10 + 4.0
    t, h, _ = _follow(ln, list(range(40, 50)), kf_edge_margin=4.0)
    assert t["last_row"] == int(np.flatnonzero(inside4)[-1]) == 91


def test_track_stops_at_the_detector_ends():
    t, h, _ = _follow(Line(range(0, 159)), list(range(70, 80)))
    assert t["first_row"] == 0 and t["last_row"] == 158 and t["nhits"] == 159


# ---------------------------------------------------------------- weighted least squares == sequential filter

def test_filter_equals_one_shot_weighted_least_squares_in_the_linear_regime():
    """Bz = 0.  Hits lie on a straight line L0 up to residuals of 1e-6 cm, so the model is linear over the spread of
    the estimates (the neglected terms are O(1e-12)).  Then the sequential filter (seed as prior mean, P0 as prior
    covariance, transport + two scalar updates per hit) must equal the one-shot weighted least-squares solution
    with the prior folded in, computed here with numpy from the line geometry:
        y(x) = y + (x - x0) tan(phi),  z(x) = z + t (x - x0) / cos(phi),  d tan(phi)/d sin(phi) = 1/cos^3(phi)."""
    rng = np.random.default_rng(5)
    o = Oracle(RX, 0.0, sigma_y=0.1, sigma_z=0.12)
    s0, t0 = 0.3, 0.6
    c = np.sqrt(1.0 - s0 * s0)
    rows = np.arange(20, 60)
    xs = RX[rows].astype(np.float64)
    d = xs - xs[0]
    yL, zL = 2.0 + d * s0 / c, 80.0 + t0 * d / c
    eps = 1e-6
    ry, rz = eps * rng.normal(size=len(xs)), eps * rng.normal(size=len(xs))
    y, z = yL + ry, zL + rz
    n = len(xs)
    sel = [0, n // 2, n - 1]
    p = o.seed(xs[sel], y[sel], z[sel])
    p_seed = p.copy()
    P = np.diag([1.0, 1.0, 0.1, 0.1, 10.0])
    p, P, _ = o.update(p, P, y[0], z[0])
    for j in range(1, n):
        p, P = o.transport(p, P, xs[j] - xs[j - 1])
        p, P, _ = o.update(p, P, y[j], z[j])
    # one-shot regression for delta = (dy, dz, ds, dt) at x0, relative to L0
    A, B, Cc = d / c ** 3, t0 * d * s0 / c ** 3, d / c
    J = np.zeros((2 * n, 4))
    J[0::2, 0] = 1.0; J[0::2, 2] = A
    J[1::2, 1] = 1.0; J[1::2, 2] = B; J[1::2, 3] = Cc
    sy2, sz2 = float(np.float32(0.1)) ** 2, float(np.float32(0.12)) ** 2
    W = np.diag(np.tile([1.0 / sy2, 1.0 / sz2], n))
    r = np.empty(2 * n); r[0::2] = ry; r[1::2] = rz
    Pinv0 = np.diag(1.0 / np.array([1.0, 1.0, 0.1, 0.1]))
    d_seed = p_seed[:4] - np.array([yL[0], zL[0], s0, t0])
    Cov = np.linalg.inv(Pinv0 + J.T @ W @ J)
    delta = Cov @ (Pinv0 @ d_seed + J.T @ W @ r)
    T = np.eye(4)  # delta at x0 -> delta at the last row
    T[0, 2] = A[-1]; T[1, 2] = B[-1]; T[1, 3] = Cc[-1]
    want = T @ delta
    got = p[:4] - np.array([yL[-1], zL[-1], s0, t0])
    assert np.all(np.abs(want) > 1e-9)  # the comparison is not vacuous
    assert np.allclose(got, want, rtol=2e-5, atol=1e-12), (got, want)
    Cw = T @ Cov @ T.T
    sd = np.sqrt(np.diag(Cw))
    assert np.max(np.abs(P[:4, :4] - Cw) / np.outer(sd, sd)) < 1e-6  # every entry, on the scale of its variances
    # q/pt is decoupled without field: it keeps its seed value and its prior variance
    assert p[4] == p_seed[4] and P[4, 4] == 10.0 and np.all(P[4, :4] == 0.0)
