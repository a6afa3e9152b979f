"""Pins for the oracle's Cellular-Automaton stages S1-S4 (SURVEY.md 8(c) "What pins the oracle").

None of these retypes the oracle's formula: they use brute force, hand-placed configurations whose answer is
evident, generator truth labels, and structural invariants.
"""
import numpy as np
import pytest

from oracle.tpc_oracle import Oracle
from paper_1709_00618_b200 import datagen as dg

RX = dg.row_x()


def _event_from_rows(rows_yz, n_rows=159):
    """rows_yz: dict row -> list of (y, z). One instance."""
    cl, ro = [], [0]
    for r in range(n_rows):
        for (y, z) in rows_yz.get(r, []):
            cl.append((RX[r], y, z, 0.0))
        ro.append(len(cl))
    return np.array(cl, np.float32).reshape(-1, 4), np.array(ro, np.int32)


def _orc(**kw):
    return Oracle(RX, 0.5, **kw)


# ---------------------------------------------------------------- S1+S2: grid search == brute force

@pytest.mark.parametrize("seed", [1, 2, 3])
def test_grid_equals_brute_force_random(seed):
    rng = np.random.default_rng(seed)
    rows = {}
    for r in range(30, 50):
        n = rng.integers(0, 60)
        # dense blob so that windows hold many pairs, plus far-away hits
        y = np.concatenate([rng.uniform(-6, 6, n), rng.uniform(-20, 20, 5)])
        z = np.concatenate([rng.uniform(100, 112, n), rng.uniform(0, 250, 5)])
        rows[r] = list(zip(y, z))
    cl, ro = _event_from_rows(rows)
    o = _orc()
    ug, dg_ = o.neighbours(cl, ro, 1, use_grid=True)
    ub, db = o.neighbours(cl, ro, 1, use_grid=False)
    assert np.array_equal(ug, ub) and np.array_equal(dg_, db)
    assert (ug >= 0).sum() > 100  # the case is not vacuous


def test_grid_equals_brute_force_adversarial():
    """Duplicated hits, hits exactly on the window edges, hits on bin boundaries, hits outside the grid range."""
    rows = {}
    base = [(0.0, 100.0), (0.0, 100.0), (4.0, 105.0), (-3.0, 95.0), (1.0, 100.0)]
    for r in range(10, 16):
        rows[r] = list(base)
    # exactly on the window edge of (0,100): dy = 2.0, dz = 2.5 ; and just outside
    rows[12] += [(2.0, 102.5), (-2.0, 97.5), (np.nextafter(np.float32(2.0), np.float32(3)), 100.0)]
    rows[11] += [(2.0, 102.5), (0.0, 102.5), (-2.0, 100.0), (0.0, 97.5)]
    rows[13] += [(0.0, 97.5), (2.0, 100.0), (1e3, 100.0), (0.0, -1e3), (0.0, 1e4)]  # far outside the grid
    cl, ro = _event_from_rows(rows)
    for cells in [(4.0, 5.0), (1.0, 1.0), (50.0, 300.0)]:
        o = _orc(grid_cell_y=cells[0], grid_cell_z=cells[1])
        ug, dg_ = o.neighbours(cl, ro, 1, use_grid=True)
        ub, db = o.neighbours(cl, ro, 1, use_grid=False)
        assert np.array_equal(ug, ub) and np.array_equal(dg_, db)


def test_grid_equals_brute_force_both_sides_cfg2_sectors():
    """z<0 side (mirrored grid origin) and a drift-window z range."""
    ev = dg.drift_window(seed=4003, mean_tracks=40.0)
    o = Oracle.for_event(ev)
    ug, dg_ = o.neighbours(ev.clusters, ev.row_offsets, ev.n_inst, use_grid=True)
    ub, db = o.neighbours(ev.clusters, ev.row_offsets, ev.n_inst, use_grid=False)
    assert np.array_equal(ug, ub) and np.array_equal(dg_, db)
    assert (ug >= 0).sum() > 1000


# ---------------------------------------------------------------- S2: hand-placed configurations

def test_hand_placed_straight_vs_kinked():
    """Row 20 hit A at (0,50). Up row has u0 on the straight line and u1 off it; down row d0 on the line.
    The straight pair must win; link indices are global."""
    rows = {19: [(-0.5, 49.0)], 20: [(0.0, 50.0)], 21: [(0.9, 51.0), (0.5, 51.0)]}
    cl, ro = _event_from_rows(rows)
    up, dn = _orc().neighbours(cl, ro, 1)
    # global indices: row19 -> 0, row20 -> 1, row21 -> 2,3 ; (0.5,51) continues the line exactly
    assert up[1] == 3 and dn[1] == 0
    assert up[0] == -1 and dn[0] == -1  # row 19 hit has nothing below it
    assert up[2] == -1 and up[3] == -1


def test_hand_placed_d2_cut_and_window():
    # second difference: ey = (yu - y) - (y - yd).  yd=-1, y=0, yu=0 -> ey = -1 -> D = 1.0 -> admissible (<=)
    rows = {19: [(-1.0, 50.0)], 20: [(0.0, 50.0)], 21: [(0.0, 50.0)]}
    cl, ro = _event_from_rows(rows)
    up, dn = _orc().neighbours(cl, ro, 1)
    assert up[1] == 2 and dn[1] == 0
    # just beyond the cut
    rows[19] = [(np.float32(-1.001), 50.0)]
    cl, ro = _event_from_rows(rows)
    up, dn = _orc().neighbours(cl, ro, 1)
    assert up[1] == -1 and dn[1] == -1
    # straight but outside the y window (|dy| = 2.1 > 2.0) -> no link although D = 0
    rows = {19: [(-2.1, 50.0)], 20: [(0.0, 50.0)], 21: [(2.1, 50.0)]}
    cl, ro = _event_from_rows(rows)
    up, dn = _orc().neighbours(cl, ro, 1)
    assert up[1] == -1
    # z window 2.5: exactly on it is inside
    rows = {19: [(0.0, 47.5)], 20: [(0.0, 50.0)], 21: [(0.0, 52.5)]}
    cl, ro = _event_from_rows(rows)
    up, dn = _orc().neighbours(cl, ro, 1)
    assert up[1] == 2 and dn[1] == 0


def test_tie_break_lowest_index():
    """Duplicated up and down hits give equal D: the lowest (u, d) indices must be chosen."""
    rows = {19: [(0.0, 50.0), (0.0, 50.0)], 20: [(0.0, 50.0)], 21: [(0.0, 50.0), (0.0, 50.0), (0.0, 50.0)]}
    cl, ro = _event_from_rows(rows)
    up, dn = _orc().neighbours(cl, ro, 1)
    assert dn[2] == 0 and up[2] == 3
    # symmetric pairs with the same D: (u=3,d=1) and (u=4,d=0) -> lowest u first
    rows = {19: [(-0.5, 50.0), (0.5, 50.0)], 20: [(0.0, 50.0)], 21: [(-0.5, 50.0), (0.5, 50.0)]}
    cl, ro = _event_from_rows(rows)
    up, dn = _orc().neighbours(cl, ro, 1)
    assert up[2] == 3 and dn[2] == 1  # u=3 is (-0.5): straight partner is d=(+0.5) = index 1


def test_first_and_last_row_never_link():
    rows = {r: [(0.0, 50.0)] for r in range(159)}
    cl, ro = _event_from_rows(rows)
    up, dn = _orc().neighbours(cl, ro, 1)
    assert up[0] == -1 and dn[0] == -1 and up[158] == -1 and dn[158] == -1
    assert np.all(up[1:158] == np.arange(2, 159)) and np.all(dn[1:158] == np.arange(0, 157))


# ---------------------------------------------------------------- S2 metric on generated tracks (truth labels)

def _well_separated_tracks(n, seed, pt_lo=0.8):
    rng = np.random.default_rng(seed)
    return dict(pt=rng.uniform(pt_lo, 3.0, n), eta=np.linspace(0.05, 0.85, n), q=np.where(np.arange(n) % 2, 1.0, -1.0),
                phi0=rng.uniform(0.12, 0.23, n), x0=np.zeros(n), y0=np.zeros(n), z0=np.zeros(n))


@pytest.mark.parametrize("bz", [0.0, 0.5])
def test_noise_free_tracks_link_to_own_neighbours(bz):
    trk = _well_separated_tracks(12, 5)
    ev = dg.from_tracks(trk, bz=bz)
    o = Oracle.for_event(ev)
    up, dn = o.neighbours(ev.clusters, ev.row_offsets, 1)
    lab = ev.labels
    rows = np.searchsorted(ev.row_offsets, np.arange(ev.n_clusters), side="right") - 1
    n_int = 0
    for h in range(ev.n_clusters):
        same = lab == lab[h]
        has_up = np.any(same & (rows == rows[h] + 1))
        has_dn = np.any(same & (rows == rows[h] - 1))
        if has_up and has_dn and 1 <= rows[h] <= 157:
            n_int += 1
            assert up[h] >= 0 and lab[up[h]] == lab[h] and rows[up[h]] == rows[h] + 1
            assert dn[h] >= 0 and lab[dn[h]] == lab[h] and rows[dn[h]] == rows[h] - 1
            # straightness: D of the chosen pair is rounding-size for lines, sagitta^2-size for helices
            y, z = ev.clusters[h, 1].astype(np.float64), ev.clusters[h, 2].astype(np.float64)
            ey = (ev.clusters[up[h], 1] - y) - (y - ev.clusters[dn[h], 1])
            ez = (ev.clusters[up[h], 2] - z) - (z - ev.clusters[dn[h], 2])
            assert ey * ey + ez * ez < (1e-8 if bz == 0.0 else 1e-3)
    assert n_int > 1000


# ---------------------------------------------------------------- S3 / S4 invariants

def test_cleaning_and_chain_invariants_cfg1():
    ev = dg.single_sector()
    o = Oracle.for_event(ev)
    up, dn = o.neighbours(ev.clusters, ev.row_offsets, 1)
    cu, cd = o.clean(up, dn)
    n = ev.n_clusters
    idx = np.arange(n)
    # mutual: cu[h]=u <=> cd[u]=h
    m = cu >= 0
    assert np.array_equal(cd[cu[m]], idx[m])
    m = cd >= 0
    assert np.array_equal(cu[cd[m]], idx[m])
    # cleaned links are a subset of raw links
    assert np.all((cu == up) | (cu == -1)) and np.all((cd == dn) | (cd == -1))
    # in/out degree <= 1
    assert len(np.unique(cu[cu >= 0])) == (cu >= 0).sum()
    assert (cu >= 0).sum() < (up >= 0).sum()  # something was actually cleaned away
    sh, ch, cn = o.candidates(cu, cd)
    rows = np.searchsorted(ev.row_offsets, idx, side="right") - 1
    assert np.all(np.diff(sh) > 0) and np.all(np.diff(ch[:, 0]) > 0)  # canonical order
    assert np.all((cn >= 4) & (cn <= 10))
    for c in range(len(cn)):
        hits = ch[c, :cn[c]]
        assert np.all(ch[c, cn[c]:] == -1)
        assert cd[hits[0]] == -1 and np.all(np.diff(rows[hits]) == 1)
        assert np.all(cu[hits[:-1]] == hits[1:])
    # chains partition the linked hits: every hit with a cleaned link lies on exactly one chain from a start hit
    seen = np.zeros(n, int)
    for s in sh:
        h = s
        while h >= 0:
            seen[h] += 1
            h = cu[h]
    linked = (cu >= 0) | (cd >= 0)
    assert np.array_equal(seen > 0, linked) and seen.max() == 1
    # candidates are exactly the start hits whose chain has >= 4 hits
    lens = []
    for s in sh:
        L, h = 0, s
        while h >= 0:
            L += 1
            h = cu[h]
        lens.append(L)
    assert np.array_equal(sh[np.array(lens) >= 4], ch[:, 0])


def test_one_chain_per_noise_free_track():
    """Full-efficiency noise-free track with m hits in consecutive rows -> exactly one chain of m-2 hits."""
    trk = _well_separated_tracks(10, 9)
    ev = dg.from_tracks(trk, bz=0.5)
    o = Oracle.for_event(ev)
    up, dn = o.neighbours(ev.clusters, ev.row_offsets, 1)
    cu, cd = o.clean(up, dn)
    sh, ch, cn = o.candidates(cu, cd)
    labs = ev.labels
    assert len(sh) == len(np.unique(labs))
    for s in sh:
        L, h = 0, s
        while h >= 0:
            assert labs[h] == labs[s]
            L += 1
            h = cu[h]
        assert L == (labs == labs[s]).sum() - 2
    assert np.all(cn == 10)


def test_empty_and_tiny_inputs():
    o = _orc()
    cl = np.zeros((0, 4), np.float32)
    ro = np.zeros(160, np.int32)
    r = o.track(cl, ro, 1)
    assert len(r.link_up) == 0 and len(r.cand_n) == 0 and len(r.trk_cand) == 0
    cl, ro = _event_from_rows({5: [(0.0, 1.0)]})
    r = o.track(cl, ro, 1)
    assert r.link_up_raw[0] == -1 and r.cluster_owner[0] == -1
