"""GPU-vs-oracle comparison helpers (tests only).  The oracle is oracle/tpc_oracle.c; the GPU path is reached only
through the C ABI (paper_1709_00618_b200.tracker)."""
import numpy as np

from oracle.tpc_oracle import Oracle

# BASELINE.json north_star: "matched tracks must have fitted parameters within 1e-3 relative / 1e-4 absolute".
PAR_RTOL = 1e-3
PAR_ATOL = 1e-4
MIN_SHARED = 0.995  # ">= 99.5 % of hit assignments" shared with the oracle
# north_star fixes no tolerance for the covariance and chi2; DESIGN.md section 3 ("Tolerances beyond the five
# parameters") derives these from the fp32 arithmetic: every covariance entry within COV_TOL of the scale of its two
# variances, chi2 within CHI2_RTOL relative + CHI2_ATOL.
COV_TOL = 1e-3
CHI2_RTOL = 5e-4
CHI2_ATOL = 5e-4


def run_oracle(ev, **kw):
    o = Oracle.for_event(ev, **kw)
    return o.track(ev.clusters, ev.row_offsets, ev.n_inst)


def assert_ca_bit_exact(g, o):
    """S2, S3, S4: integer results are unique -> bit-exact."""
    assert np.array_equal(g.link_up_raw, o.link_up_raw), "raw up links differ"
    assert np.array_equal(g.link_dn_raw, o.link_dn_raw), "raw down links differ"
    assert np.array_equal(g.link_up, o.link_up), "cleaned up links differ"
    assert np.array_equal(g.link_dn, o.link_dn), "cleaned down links differ"
    assert np.array_equal(g.start_hits, o.start_hits), "start hits differ"
    assert g.n_start == len(o.start_hits) and g.n_cand == len(o.cand_n)
    assert np.array_equal(g.cand_n, o.cand_n), "candidate lengths differ"
    assert np.array_equal(g.cand_hits, o.cand_hits), "candidate hit lists differ"


def tracklet_report(g, o):
    """S5 comparison per candidate id (ids are identical on both sides because candidates are bit-exact)."""
    ok_o = o.tracklets["ok"].astype(bool)
    ok_g = g.tl_nhits > 0
    both = ok_o & ok_g
    same_hits = np.all(g.tl_hits == o.tracklet_hits, axis=1)
    att_o = o.tracklet_hits >= 0
    shared = ((g.tl_hits == o.tracklet_hits) & att_o)[both].sum()
    total = max(att_o[both].sum(), (g.tl_hits >= 0)[both].sum())
    ident = both & same_hits
    po = o.tracklets["p"][ident]
    pg = g.tl_params[ident].astype(np.float64)
    excess = np.abs(pg - po) / (PAR_ATOL + PAR_RTOL * np.abs(po))  # <= 1 means inside the tolerance
    # covariance (packed lower triangle, 15 entries) on the scale of the two variances involved; chi2
    co = o.tracklets["cov"][ident]
    cg = g.tl_cov[ident].astype(np.float64)
    ii = np.array([i for i in range(5) for j in range(i + 1)])
    jj = np.array([j for i in range(5) for j in range(i + 1)])
    diag = np.array([0, 2, 5, 9, 14])
    scale = np.sqrt(co[:, diag[ii]] * co[:, diag[jj]])
    cov_excess = np.abs(cg - co) / (COV_TOL * scale) if co.size else np.zeros((0, 15))
    xo = o.tracklets["chi2"][ident]
    xg = g.tl_chi2[ident].astype(np.float64)
    chi2_excess = np.abs(xg - xo) / (CHI2_ATOL + CHI2_RTOL * xo) if xo.size else np.zeros(0)
    return dict(worst_cov_excess=float(cov_excess.max()) if cov_excess.size else 0.0,
                worst_chi2_excess=float(chi2_excess.max()) if chi2_excess.size else 0.0,
                ref_rows_equal=bool(np.array_equal(g.tl_rows[ident][:, 2], o.tracklets["ref_row"][ident])),
                n_cand=len(ok_o), ok_mismatch=int((ok_o != ok_g).sum()), identical_hit_lists=int(ident.sum()),
                n_both=int(both.sum()), shared_frac=float(shared / max(total, 1)),
                worst_param_excess=float(excess.max()) if excess.size else 0.0,
                worst_by_param=excess.max(axis=0).tolist() if excess.size else [0.0] * 5,
                nhits_equal=bool(np.array_equal(g.tl_nhits[ident], o.tracklets["nhits"][ident])),
                rows_equal=bool(np.array_equal(g.tl_rows[ident][:, 0], o.tracklets["first_row"][ident])
                                and np.array_equal(g.tl_rows[ident][:, 1], o.tracklets["last_row"][ident])))


def final_track_report(g, o, n_clusters):
    """S6: share of identical final cluster->track assignments, with tracks matched by candidate id."""
    own_g = np.full(n_clusters, -1, np.int64)
    own_o = np.full(n_clusters, -1, np.int64)
    m = g.cluster_owner >= 0
    own_g[m] = g.trk_cand_id[g.cluster_owner[m]]
    m = o.cluster_owner >= 0
    own_o[m] = o.trk_cand[o.cluster_owner[m]]
    assigned = (own_g >= 0) | (own_o >= 0)
    same = (own_g == own_o) & assigned
    return dict(n_tracks_gpu=int(g.n_tracks), n_tracks_oracle=int(len(o.trk_cand)),
                shared_assign_frac=float(same.sum() / max(assigned.sum(), 1)),
                tracks_identical=bool(np.array_equal(g.trk_cand_id, o.trk_cand)))


def assert_final_track_records(g, o, row_offsets, n_rows, row_x):
    """Everything S6 returns per final track against the oracle, tracks matched by candidate id:
    trk_params / trk_cov / trk_chi2 are the tracklet's (S6 does not refit, S6) -> bit-identical to the
    GPU's own tracklet outputs, which tracklet_report() compares with the oracle; trk_xref = x of the oracle's
    reference row exactly; trk_sector = sector instance of the candidate's start hit exactly; trk_nhits = the
    oracle's kept hits for every common track whose hit list is the same on both sides."""
    cid = g.trk_cand_id
    assert np.array_equal(g.trk_params, g.tl_params[cid]) and np.array_equal(g.trk_cov, g.tl_cov[cid])
    assert np.array_equal(g.trk_chi2, g.tl_chi2[cid])
    tl = o.tracklets[cid]
    ok = tl["ok"].astype(bool)  # a GPU-only tracklet (A12/A13 threshold flips) has no oracle record
    assert np.array_equal(g.trk_xref[ok], np.asarray(row_x, np.float32)[tl["ref_row"][ok]])
    inst_of_hit = np.searchsorted(np.asarray(row_offsets)[::n_rows], o.cand_hits[cid, 0], side="right") - 1
    assert np.array_equal(g.trk_sector, inst_of_hit.astype(np.int32))
    # kept hits: compare per track on the tracks both sides have
    common, ig, io = np.intersect1d(cid, o.trk_cand, return_indices=True)
    kept_o = np.diff(o.trk_hit_offset)[io]
    kept_g = g.trk_nhits[ig]
    same_list = np.array([np.array_equal(g.trk_hits[g.trk_hit_offset[a]:g.trk_hit_offset[a + 1]],
                                         o.trk_hits[o.trk_hit_offset[b]:o.trk_hit_offset[b + 1]])
                          for a, b in zip(ig, io)], bool) if len(common) else np.zeros(0, bool)
    # trk_nhits against the oracle's kept counts on the common tracks whose TRACKLET hit lists agree: the two
    # selectors then start from the same tracklet, and the kept count can only differ where a competing tracklet
    # differs (a flipped near-tie of S5 elsewhere changes who claims a shared cluster).  Counted, bounded and returned.
    same_tl0 = np.all(g.tl_hits[common] == o.tracklet_hits[common], axis=1) if len(common) else np.zeros(0, bool)
    nhits_diff = int((kept_g[same_tl0] != kept_o[same_tl0]).sum())
    # observed on the B200: 0 everywhere except 1 of 18,014 on the CFG:3 central event -> observed + 1, scaled with size
    assert nhits_diff <= 2 + same_tl0.sum() // 20000, (nhits_diff, int(same_tl0.sum()))
    assert np.all(kept_g[same_list] == np.diff(g.trk_hit_offset)[ig][same_list])
    # north_star: "matched tracks must have fitted parameters within 1e-3 relative / 1e-4 absolute" -- the FINAL tracks
    # (tracklet_report applies the same bar to every tracklet, final or not).  Matched = same candidate id and the
    # tracklet's hit list identical on both sides, so the two fits saw the same measurements.
    same_tl = np.all(g.tl_hits[common] == o.tracklet_hits[common], axis=1) if len(common) else np.zeros(0, bool)
    pg = g.trk_params[ig][same_tl].astype(np.float64)
    po = o.tracklets["p"][common][same_tl]
    ex = np.abs(pg - po) / (PAR_ATOL + PAR_RTOL * np.abs(po))
    return dict(common_tracks=int(len(common)), identical_track_hit_lists=int(same_list.sum()),
                same_tracklet_tracks=int(same_tl0.sum()), trk_nhits_differ=nhits_diff,
                worst_track_param_excess=float(ex.max()) if ex.size else 0.0)


def assert_final_consistency(g, n_clusters):
    """Internal consistency of the S6 outputs (holds at any size)."""
    nt = g.n_tracks
    off = g.trk_hit_offset
    assert off[0] == 0 and off[nt] == g.n_track_hits and np.all(np.diff(off) == g.trk_nhits)
    assert np.all(g.trk_nhits >= 10)
    assert np.all(np.diff(g.trk_cand_id) > 0)
    owner = g.cluster_owner
    assert owner.shape[0] == n_clusters
    trk_of_hit = np.repeat(np.arange(nt), g.trk_nhits)
    assert np.array_equal(owner[g.trk_hits], trk_of_hit)
    assert (owner >= 0).sum() == g.n_track_hits  # every owned cluster is listed exactly once
