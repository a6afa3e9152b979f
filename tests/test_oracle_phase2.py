"""Pins for the oracle's phase 2: sector merger + refit (oracle/tpc_oracle.c orc_rotate, orc_refit_chain, orc_phase2;
DESIGN.md readings M1-M4; "merges the track segments found in the individual sectors to final tracks and
performs a track refit").

Independent references: the generator's closed-form helix expressed in the frames of two neighbouring sectors
(dg.local_truth_state with a sector argument), central finite differences, hand-placed straight tracks whose
matching answer is evident from the rule, generator truth labels, and pull statistics."""
from types import SimpleNamespace

import numpy as np
import pytest

from oracle.tpc_oracle import Oracle, unpack_cov
from paper_1709_00618_b200 import datagen as dg

RX = dg.row_x()
BZ = 0.5
A20 = float(np.deg2rad(20.0))


def _orc(bz=BZ, **kw):
    kw.setdefault("sigma_y", 0.1)
    kw.setdefault("sigma_z", 0.1)
    return Oracle(RX, bz, **kw)


def _rand_cov(rng):
    A = rng.normal(size=(5, 5)) * np.array([0.1, 0.1, 0.01, 0.01, 0.05])[:, None]
    return A @ A.T + np.diag([1e-4, 1e-4, 1e-6, 1e-6, 1e-5])


# ---------------------------------------------------------------- M2: rotation between sector frames

def test_rotation_then_transport_equals_the_helix_in_the_neighbouring_frame():
    trk = dict(pt=np.array([0.35, 1.2, 0.2]), eta=np.array([0.4, -0.7, 0.1]), q=np.array([1.0, -1.0, -1.0]),
               phi0=np.array([0.30, 0.33, 0.36]), x0=np.array([0.0, 3.0, -2.0]), y0=np.array([0.0, 1.0, 2.0]),
               z0=np.array([0.0, 5.0, -3.0]))
    o = _orc()
    for i in range(3):
        for s_from, s_to in ((0, 1), (1, 0), (5, 4), (0, 17), (17, 0)):
            for xa, xb in ((100.0, 110.0), (150.0, 149.0)):
                t = {k: v.copy() for k, v in trk.items()}
                t["phi0"] = trk["phi0"] + s_from * A20  # keep the track near the frames in question
                sa = dg.local_truth_state(t, i, xa, BZ, sector=s_from)
                sb = dg.local_truth_state(t, i, xb, BZ, sector=s_to)
                d = (s_to - s_from + 9) % 18 - 9
                if not (abs(sa[2]) <= 0.8 and abs(sb[2]) <= 0.8):  # also skips NaN (plane not reached)
                    continue
                p1, P1, x1 = o.rotate(sa, np.eye(5), xa, d * A20)
                got, _ = o.transport(p1, P1, xb - x1)
                assert np.allclose(got, sb, rtol=0, atol=1e-9), (i, s_from, s_to, got - sb)


def test_rotation_jacobian_vs_central_finite_differences():
    """J is the derivative of 'state on the old plane -> state on the (fixed) new plane': perturb, rotate, bring the
    result back to the nominal new plane with the (separately pinned) transport, difference."""
    o = _orc()
    rng = np.random.default_rng(3)
    for alpha in (A20, -A20):
        for _ in range(10):
            p = np.array([rng.uniform(-30, 30), rng.uniform(0, 250), rng.uniform(-0.4, 0.4), rng.uniform(-1, 1),
                          rng.uniform(-3, 3)])
            x = rng.uniform(90, 240)
            P = _rand_cov(rng)
            p1, P1, x1, J = o.rotate(p, P, x, alpha, want_jac=True)
            Jn = np.zeros((5, 5))
            for j in range(5):
                h = [1e-3, 1e-3, 1e-5, 1e-5, 1e-2][j]

                def at(hh):
                    a = p.copy(); a[j] += hh
                    q, Q, xq = o.rotate(a, P, x, alpha)
                    return o.transport(q, Q, x1 - xq)[0]
                cd = lambda hh: (at(hh) - at(-hh)) / (2 * hh)  # noqa: E731
                Jn[:, j] = (4.0 * cd(0.5 * h) - cd(h)) / 3.0
            assert np.max(np.abs(J - Jn) - 1e-5 * np.abs(Jn)) < 2e-8, (J - Jn)
            assert np.allclose(P1, J @ P @ J.T, rtol=1e-12, atol=1e-18)


def test_rotation_forth_and_back_is_the_identity():
    o = _orc()
    rng = np.random.default_rng(4)
    p = np.array([12.0, 80.0, 0.25, 0.6, -1.4])
    P = _rand_cov(rng)
    p1, P1, x1 = o.rotate(p, P, 130.0, A20)
    p2, P2, x2 = o.rotate(p1, P1, x1, -A20)
    assert np.isclose(x2, 130.0, atol=1e-12) and np.allclose(p2, p, atol=1e-12)
    assert np.allclose(P2, P, rtol=1e-10, atol=1e-16)
    assert o.rotate([0, 0, 0.9, 0, 0], np.eye(5), 100.0, -A20) is None  # sin(phi + 20 deg) > 0.95


# ---------------------------------------------------------------- M1: refit of the kept hits

def _one_track_hits(trk, i, rows, bz=BZ, sector=0):
    st = np.array([dg.local_truth_state(trk, i, float(RX[r]), bz, sector=sector) for r in rows])
    return st[:, 0].astype(np.float32), st[:, 1].astype(np.float32), st


def test_refit_reproduces_the_generating_helix_and_uses_only_the_kept_hits():
    trk = dict(pt=np.array([0.5, 2.0, 1.0]), eta=np.array([0.5, -0.3, 0.8]), q=np.array([1.0, -1.0, 1.0]),
               phi0=np.array([0.16, 0.2, 0.18]), x0=np.zeros(3), y0=np.zeros(3), z0=np.zeros(3))
    o = _orc()
    for i in range(3):
        rows = np.arange(20, 130)
        y, z, st = _one_track_hits(trk, i, rows)
        f = o.refit_chain([(0, rows, y, z)])
        assert f["ok"] == 1 and f["nhits"] == len(rows) and f["first_row"] == 20 and f["nseg"] == 1
        assert np.allclose(f["p"], st[0], rtol=1e-5, atol=2e-6), f["p"] - st[0]
        # five hits displaced by 0.3 cm: the fit over all hits is pulled, the fit over the kept hits is not
        yb = y.copy()
        yb[40:45] += 0.3
        pulled = o.refit_chain([(0, rows, yb, z)])
        assert abs(pulled["p"][0] - st[0][0]) > 1e-3
        keep = np.ones(len(rows), bool)
        keep[40:45] = False
        g = o.refit_chain([(0, rows[keep], yb[keep], z[keep])])
        assert g["nhits"] == keep.sum() and np.allclose(g["p"], st[0], rtol=1e-5, atol=2e-6)
        # sparse kept hits (every third row) and a short track
        h = o.refit_chain([(0, rows[::3], y[::3], z[::3])])
        assert np.allclose(h["p"], st[0], rtol=1e-5, atol=2e-6)
        s = o.refit_chain([(0, rows[:10], y[:10], z[:10])])
        assert s["ok"] == 1 and np.allclose(s["p"][:4], st[0][:4], rtol=1e-4, atol=1e-4)


def test_chain_refit_across_a_sector_boundary_reproduces_the_helix():
    """Hits of one helix given as two segments in the frames of sectors 0 and 1 (exact, fp32-rounded): the chain fit
    equals the helix at the innermost hit in sector 0's frame, and its covariance is that of ONE fit over all hits
    (smaller than the fit of the inner segment alone)."""
    trk = dict(pt=np.array([0.6]), eta=np.array([0.4]), q=np.array([1.0]), phi0=np.array([0.33]), x0=np.zeros(1),
               y0=np.zeros(1), z0=np.zeros(1))
    o = _orc()
    rows_a, rows_b = np.arange(10, 70), np.arange(70, 140)
    ya, za, sta = _one_track_hits(trk, 0, rows_a, sector=0)
    yb, zb, stb = _one_track_hits(trk, 0, rows_b, sector=1)
    assert np.all(np.abs(stb[:, 2]) < 0.9)
    f = o.refit_chain([(0, rows_a, ya, za), (1, rows_b, yb, zb)])
    assert f["ok"] == 1 and f["nseg"] == 2 and f["nhits"] == 130 and f["first_row"] == 10
    assert np.allclose(f["p"], sta[0], rtol=1e-5, atol=2e-6), f["p"] - sta[0]
    alone = o.refit_chain([(0, rows_a, ya, za)])
    assert f["cov"][14] < 0.5 * alone["cov"][14]  # q/pt is better known with the outer 70 hits
    assert f["chi2"] < 1e-3 * 2 * 130


def test_pulls_of_single_and_merged_fits():
    """Smeared hits (0.1 cm): pulls of the chain fit ~ N(0,1) for one-segment and two-segment tracks; this exercises
    the rotated covariance (M2) in the way the statistics see it."""
    rng = np.random.default_rng(9)
    o = _orc()
    pulls = {1: [], 2: []}
    for it in range(400):
        trk = dict(pt=np.array([rng.uniform(0.4, 2.0)]), eta=np.array([rng.uniform(-0.8, 0.8)]),
                   q=np.array([rng.choice([-1.0, 1.0])]), phi0=np.array([rng.uniform(0.30, 0.40)]), x0=np.zeros(1),
                   y0=np.zeros(1), z0=np.zeros(1))
        rows_a, rows_b = np.arange(5, 75), np.arange(75, 150)
        ya, za, sta = _one_track_hits(trk, 0, rows_a, sector=0)
        yb, zb, stb = _one_track_hits(trk, 0, rows_b, sector=1)
        if not (np.abs(sta[:, 2]).max() <= 0.7 and np.abs(stb[:, 2]).max() <= 0.7):
            continue
        n = lambda v: (v.astype(np.float64) + rng.normal(0, 0.1, len(v))).astype(np.float32)  # noqa: E731
        for nseg, segs in ((1, [(0, rows_a, n(ya), n(za))]), (2, [(0, rows_a, n(ya), n(za)), (1, rows_b, n(yb), n(zb))])):
            f = o.refit_chain(segs)
            assert f["ok"] == 1
            pulls[nseg].append((f["p"] - sta[0]) / np.sqrt(np.diag(unpack_cov(f["cov"]))))
    for nseg in (1, 2):
        pl = np.array(pulls[nseg])
        assert len(pl) > 250
        assert np.all(np.abs(pl.mean(0)) < 0.2), (nseg, pl.mean(0))
        assert np.all(np.abs(pl.std(0) - 1.0) < 0.15), (nseg, pl.std(0))


# ---------------------------------------------------------------- M3 / M4: matching on hand-placed straight tracks

def _straight_two_sector_event(bz=0.0, z_shift_b=0.0, drop_b_rows=0, split_row=80, extra_b=None, extra_a=None):
    """One straight track (Bz = 0) that leaves sector 0 through its upper edge at `split_row`: hits of rows
    10..split_row-1 in sector 0's frame, rows split_row..150 in sector 1's frame.  Returns the Event-like tuple and the
    fake S6 result phase 2 consumes."""
    x = RX.astype(np.float64)
    # global line: through (x0, y0) = (85, 5) in sector 0's frame with slope my; z linear in the path
    my, mz = 0.12, 0.4
    ya = 5.0 + my * (x - 85.0)
    za = 30.0 + mz * (x - 85.0)
    rows_a = np.arange(10, split_row)
    rows_b = np.arange(split_row + drop_b_rows, 150)
    # the same line in sector 1's frame: intersect with the planes x' = RX[r]
    ca, sa = np.cos(A20), np.sin(A20)
    # points on the line: (X, Y) = (t, 5 + my (t - 85)) in frame 0;  x' = X ca + Y sa = RX[r]  ->  solve for t
    t = (x[rows_b] - (5.0 - my * 85.0) * sa) / (ca + my * sa)
    Yb = 5.0 + my * (t - 85.0)
    yb = -t * sa + Yb * ca
    zb = 30.0 + mz * (t - 85.0) + z_shift_b
    tracks = [(0, rows_a, ya[rows_a], za[rows_a]), (1, rows_b, yb, zb)]
    if extra_b is not None:
        tracks.append(extra_b(rows_b, yb, zb))
    if extra_a is not None:
        tracks.append(extra_a(rows_a, ya[rows_a], za[rows_a]))
    R = len(RX)
    n_inst = 36
    per_slab = {}
    for ti, (sec, rows, yy, zz) in enumerate(tracks):
        for r, y_, z_ in zip(rows, yy, zz):
            per_slab.setdefault(sec * R + int(r), []).append((RX[int(r)], y_, z_, float(ti)))
    cl, ro, where = [], [0], {}
    for slab in range(n_inst * R):
        for rec in per_slab.get(slab, []):
            where[(int(rec[3]), slab % R)] = len(cl)
            cl.append(rec)
        ro.append(len(cl))
    cl = np.array(cl, np.float32).reshape(-1, 4)
    ro = np.array(ro, np.int32)
    hits, off, first = [], [0], []
    for ti, (sec, rows, yy, zz) in enumerate(tracks):
        hits += [where[(ti, int(r))] for r in rows]
        off.append(len(hits))
        first.append(hits[off[-2]])
    cand_hits = np.full((len(tracks), 10), -1, np.int32)
    cand_hits[:, 0] = first
    res = SimpleNamespace(trk_cand=np.arange(len(tracks), dtype=np.int32), cand_hits=cand_hits,
                          trk_hit_offset=np.array(off, np.int64), trk_hits=np.array(hits, np.int32))
    return cl, ro, n_inst, res


def test_straight_track_across_a_sector_edge_is_merged():
    cl, ro, n_inst, res = _straight_two_sector_event()
    o = _orc(bz=0.0)
    p2 = o.phase2(cl, ro, n_inst, res)
    assert list(p2.seg_next) == [1, -1] and list(p2.seg_prev) == [-1, 0]
    assert list(p2.m_first) == [0] and p2.m_fit["nseg"][0] == 2 and p2.m_fit["nhits"][0] == 70 + 70
    # the merged fit is the straight line in sector 0's frame at row 10
    assert np.allclose(p2.m_fit["p"][0][:2], [5.0 + 0.12 * (RX[10] - 85.0), 30.0 + 0.4 * (RX[10] - 85.0)], atol=1e-4)
    assert np.isclose(p2.m_fit["p"][0][2], 0.12 / np.hypot(1.0, 0.12), atol=1e-5)


def test_matching_cuts_gap_and_side():
    o = _orc(bz=0.0)
    for dz, linked in ((1.9, True), (2.1, False), (-1.9, True), (-2.1, False)):
        cl, ro, n, res = _straight_two_sector_event(z_shift_b=dz)
        assert (o.phase2(cl, ro, n, res).seg_next[0] == 1) == linked, dz
    for drop, linked in ((9, True), (10, False)):  # first_row(B) - last_row(A) = 1 + drop
        cl, ro, n, res = _straight_two_sector_event(drop_b_rows=drop)
        assert (o.phase2(cl, ro, n, res).seg_next[0] == 1) == linked, drop
    # B must START after A ends: a segment that overlaps A's rows is not a continuation
    cl, ro, n, res = _straight_two_sector_event(drop_b_rows=-5)
    assert o.phase2(cl, ro, n, res).seg_next[0] == -1


def test_best_candidate_wins_and_the_choice_must_be_mutual():
    """Two continuations in sector 1: the true one and a copy shifted by 0.5 cm in z.  A picks the nearer (the true
    one); the copy also picks A as its best predecessor but is not A's choice -> it stays unlinked."""
    def extra(rows_b, yb, zb):
        return (1, rows_b, yb, zb + 0.5)
    cl, ro, n, res = _straight_two_sector_event(extra_b=extra)
    p2 = _orc(bz=0.0).phase2(cl, ro, n, res)
    assert list(p2.seg_next) == [1, -1, -1] and list(p2.seg_prev) == [-1, 0, -1]
    assert list(p2.m_first) == [0, 2] and list(p2.m_fit["nseg"]) == [2, 1]
    # exact duplicate of the continuation: the tie goes to the lower track index
    cl, ro, n, res = _straight_two_sector_event(extra_b=lambda r, y, z: (1, r, y, z))
    p2 = _orc(bz=0.0).phase2(cl, ro, n, res)
    assert list(p2.seg_next) == [1, -1, -1]


def test_two_inner_segments_compete_for_one_continuation():
    """The inner segment twice (track 2 = a copy of track 0 shifted by 0.3 cm in z): both pick B as successor, B picks
    the nearer one; only the mutual choice becomes a link, and B has exactly one predecessor."""
    cl, ro, n, res = _straight_two_sector_event(extra_a=lambda r, y, z: (0, r, y, z + 0.3))
    p2 = _orc(bz=0.0).phase2(cl, ro, n, res)
    assert list(p2.seg_next) == [1, -1, -1] and list(p2.seg_prev) == [-1, 0, -1]
    assert list(p2.m_first) == [0, 2]
    # exact copy: the tie goes to the lower track index
    cl, ro, n, res = _straight_two_sector_event(extra_a=lambda r, y, z: (0, r, y, z))
    p2 = _orc(bz=0.0).phase2(cl, ro, n, res)
    assert list(p2.seg_next) == [1, -1, -1] and list(p2.seg_prev) == [-1, 0, -1]


# ---------------------------------------------------------------- end to end against generator truth

def test_event_segments_of_one_particle_are_joined_and_nothing_else():
    """Noise-free full event (zero smear, tracker sigma 0.1): every link joins two segments of the same generated
    particle; most multi-sector particles are fully chained; merged hit counts add up."""
    ev = dg.full_event(seed=2201, n_prim=300, eff=1.0, sigma_y=0.0, sigma_z=0.0, noise=0.0)
    o = Oracle(ev.row_x, ev.bz, sigma_y=0.1, sigma_z=0.1)
    r = o.track(ev.clusters, ev.row_offsets, ev.n_inst)
    p2 = o.phase2(ev.clusters, ev.row_offsets, ev.n_inst, r)
    nt = len(r.trk_cand)
    lab = np.array([ev.labels[r.trk_hits[r.trk_hit_offset[t]]] for t in range(nt)])
    linked = np.flatnonzero(p2.seg_next >= 0)
    assert len(linked) > 200 and np.all(lab[linked] == lab[p2.seg_next[linked]])
    assert np.array_equal(p2.seg_prev[p2.seg_next[linked]], linked)  # links are mutual
    assert len(p2.m_first) == nt - len(linked) and np.all(np.diff(p2.m_first) > 0)
    nh = np.diff(r.trk_hit_offset)
    for m, t in enumerate(p2.m_first):
        tot, x, k = 0, t, 0
        while x >= 0:
            tot, x, k = tot + nh[x], p2.seg_next[x], k + 1
        assert p2.m_fit["nseg"][m] == k and (p2.m_fit["ok"][m] == 0 or p2.m_fit["nhits"][m] == tot)
    multi = sum(1 for v in np.bincount(lab) if v > 1)
    assert len(linked) >= 0.9 * (nt - len(np.unique(lab))) and multi > 100
    # merged fits reproduce the generating helix at the innermost row of the innermost segment
    t64 = {k: np.asarray(v, float) for k, v in ev.truth.items() if k != "primary"}
    R = ev.n_rows
    inst_of = np.searchsorted(ev.row_offsets[::R], r.cand_hits[r.trk_cand, 0], side="right") - 1
    checked = 0
    for m, t in enumerate(p2.m_first):
        f = p2.m_fit[m]
        if not f["ok"] or f["nseg"] < 2:
            continue
        truth = dg.local_truth_state(t64, int(lab[t]), float(RX[f["first_row"]]), ev.bz, sector=int(inst_of[t]) % 18)
        if inst_of[t] % 36 >= 18:
            continue  # generator's z < 0 side uses the same frame; keep the check on one side for brevity
        assert np.allclose(f["p"], truth, rtol=2e-5, atol=5e-6), (m, f["p"] - truth)
        checked += 1
    assert checked > 50
