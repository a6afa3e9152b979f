"""Pins for the oracle's S2 class-1 links (nf_bridge_rows = 1: a single missing row is bridged; reading A2',
SURVEY.md 8(f) NEXT-1).  Brute force, hand-placed configurations whose answer is evident, and invariants -- none of
them retypes the oracle's formula."""
import numpy as np
import pytest

from oracle.tpc_oracle import Oracle
from paper_1709_00618_b200 import datagen as dg

RX = dg.row_x()


def _event_from_rows(rows_yz, n_rows=159):
    cl, ro = [], [0]
    for r in range(n_rows):
        for (y, z) in rows_yz.get(r, []):
            cl.append((RX[r], y, z, 0.0))
        ro.append(len(cl))
    return np.array(cl, np.float32).reshape(-1, 4), np.array(ro, np.int32)


def _rows_of(ro, n):
    return np.repeat(np.arange(len(ro) - 1), np.diff(ro))[:n]


@pytest.mark.parametrize("seed", [11, 12])
def test_bridged_grid_equals_brute_force(seed):
    """Sparse random rows (so that many hits lack an adjacent pair) with a dense blob: grid search == O(N^2) search."""
    rng = np.random.default_rng(seed)
    rows = {}
    for r in range(20, 60):
        if rng.random() < 0.25:
            continue  # empty row
        n = rng.integers(0, 25)
        y = np.concatenate([rng.uniform(-5, 5, n), rng.uniform(-20, 20, 4)])
        z = np.concatenate([rng.uniform(100, 110, n), rng.uniform(0, 250, 4)])
        rows[r] = list(zip(y, z))
    cl, ro = _event_from_rows(rows)
    for cells in [(4.0, 5.0), (1.5, 2.0)]:
        o = Oracle(RX, 0.5, nf_bridge_rows=1, grid_cell_y=cells[0], grid_cell_z=cells[1])
        ug, dg_ = o.neighbours(cl, ro, 1, use_grid=True)
        ub, db = o.neighbours(cl, ro, 1, use_grid=False)
        assert np.array_equal(ug, ub) and np.array_equal(dg_, db)
    u0, _ = Oracle(RX, 0.5).neighbours(cl, ro, 1)
    assert (ug >= 0).sum() > (u0 >= 0).sum() > 50  # bridging adds links; the case is not vacuous


def test_adjacent_pairs_are_never_replaced():
    """Class 1 is tried only for hits WITHOUT an admissible adjacent pair: every link of the default reading stays."""
    ev = dg.single_sector(seed=1021, eff=0.9)
    u0, d0 = Oracle.for_event(ev).neighbours(ev.clusters, ev.row_offsets, 1)
    u1, d1 = Oracle.for_event(ev, nf_bridge_rows=1).neighbours(ev.clusters, ev.row_offsets, 1)
    has = u0 >= 0
    assert np.array_equal(u1[has], u0[has]) and np.array_equal(d1[has], d0[has])
    rows = _rows_of(ev.row_offsets, ev.n_clusters)
    new = (u1 >= 0) & ~has
    assert new.sum() > 100
    # a bridged pair spans exactly three rows: (r+1, r-2) or (r+2, r-1)
    assert np.all(rows[u1[new]] - rows[d1[new]] == 3)
    assert np.all(np.isin(rows[u1[new]] - rows[new], (1, 2)))


def test_straight_line_with_one_missing_cluster_chains_through():
    """Noise-free straight line (Bz = 0 geometry: y, z linear in x), the cluster of row 50 removed.  Default reading:
    the chain breaks (hits 48 | 52 are its ends).  Bridged: hits 49 and 51 link across the gap with D ~ 0, the links
    are mutual, and one chain covers rows 31..69."""
    rows = {r: [(0.02 * (RX[r] - 85.0) - 3.0, 0.5 * (RX[r] - 85.0) + 20.0)] for r in range(30, 71) if r != 50}
    cl, ro = _event_from_rows(rows)
    row_of = _rows_of(ro, len(cl))
    idx = {int(r): i for i, r in enumerate(row_of)}
    for bridge, n_start in ((0, 2), (1, 1)):
        o = Oracle(RX, 0.0, nf_bridge_rows=bridge)
        up, dn = o.neighbours(cl, ro, 1)
        cu, cd = o.clean(up, dn)
        start, _, cn = o.candidates(cu, cd)
        assert len(start) == n_start
        if bridge:
            assert up[idx[49]] == idx[51] and dn[idx[49]] == idx[48]
            assert dn[idx[51]] == idx[49] and up[idx[51]] == idx[52]
            assert cu[idx[49]] == idx[51] and cd[idx[51]] == idx[49]
            assert start[0] == idx[31]
        else:
            assert up[idx[49]] == -1 and up[idx[51]] == -1
            assert sorted(row_of[start]) == [31, 52]


def test_two_missing_rows_are_not_bridged():
    rows = {r: [(1.0, 50.0 + 0.3 * r)] for r in range(30, 71) if r not in (50, 51)}
    cl, ro = _event_from_rows(rows)
    o = Oracle(RX, 0.0, nf_bridge_rows=1)
    up, dn = o.neighbours(cl, ro, 1)
    cu, cd = o.clean(up, dn)
    start, _, _ = o.candidates(cu, cd)
    assert len(start) == 2


def test_class1_cut_scales_with_the_spacing():
    """Middle hit displaced by e from the line through its partners (rows r+1 and r-2): the deviation of reading A2' is
    dd*(u-h) - du*(h-d) = -3e, cut at 2.25 * D2MAX = 2.25 cm^2 -> linked iff |e| <= 0.5 cm."""
    for e, linked in ((0.45, True), (0.55, False)):
        rows = {40: [(0.0, 100.0)], 42: [(e, 100.0)], 43: [(0.0, 100.0)]}
        cl, ro = _event_from_rows(rows)
        up, dn = Oracle(RX, 0.0, nf_bridge_rows=1).neighbours(cl, ro, 1)
        assert (up[1] == 2 and dn[1] == 0) == linked


def test_bridging_halves_the_candidates_and_keeps_the_tracks():
    """CFG:2-like event (efficiency 0.95): far fewer candidates (clone work), about the same final tracks."""
    ev = dg.full_event(seed=2011, n_prim=300)
    a = Oracle.for_event(ev).track(ev.clusters, ev.row_offsets, ev.n_inst)
    b = Oracle.for_event(ev, nf_bridge_rows=1).track(ev.clusters, ev.row_offsets, ev.n_inst)
    assert len(b.cand_n) < 0.6 * len(a.cand_n)
    assert abs(len(b.trk_cand) - len(a.trk_cand)) <= 0.03 * len(a.trk_cand)
    assert (b.cluster_owner >= 0).sum() >= 0.98 * (a.cluster_owner >= 0).sum()


def test_exact_tie_between_the_two_kinds_prefers_the_pair_with_the_near_upper_partner():
    """Reading A2': minimum over (D, du, u, d).  Hit h = (0, 100) in row 50; row 51 holds u1 = 1.5 (local index 1,
    behind a far-away cluster), row 49 d1 = 1.5, row 48 d2 = -3, row 52 u2 = -3 (local index 0).  The adjacent pair
    (u1, d1) deviates by 3 cm -> inadmissible; both bridged pairs are exactly straight:
        (du, dd) = (1, 2): 2 (u1 - h) - (h - d2) = 3 - 3 = 0;   (2, 1): (u2 - h) - 2 (h - d1) = -3 + 3 = 0.
    The tie goes to du = 1 although the other pair's upper partner has the lower local index."""
    def links(d2_y):
        rows = {48: [(d2_y, 100.0)], 49: [(1.5, 100.0)], 50: [(0.0, 100.0)], 51: [(-15.0, 100.0), (1.5, 100.0)],
                52: [(-3.0, 100.0)]}
        cl, ro = _event_from_rows(rows)
        idx = {(int(r), k): int(ro[r]) + k for r in rows for k in range(len(rows[r]))}
        for use_grid in (True, False):
            up, dn = Oracle(RX, 0.0, nf_bridge_rows=1).neighbours(cl, ro, 1, use_grid=use_grid)
            got = (int(up[idx[50, 0]]), int(dn[idx[50, 0]]))
            assert use_grid or got == first
            first = got
        up0, _ = Oracle(RX, 0.0).neighbours(cl, ro, 1)
        assert up0[idx[50, 0]] == -1  # no admissible adjacent pair: class 1 is what links it
        return got, idx

    got, idx = links(-3.0)
    assert got == (idx[51, 1], idx[48, 0])
    # D decides before the kind does: with d2 = -3.25 the (1, 2) pair deviates by 0.25 cm, the (2, 1) pair by 0
    got, idx = links(-3.25)
    assert got == (idx[52, 0], idx[49, 0])
