"""GPU parity with S2 row bridging on (nf_bridge_rows = 1, reading A2' / SURVEY 8(f) NEXT-1): same bar as the default
reading -- links, cleaned links, start hits and candidates bit-exact, tracklets and final tracks within tolerance."""
import dataclasses
import json
import os

import numpy as np
import pytest

from paper_1709_00618_b200 import datagen as dg

from parity_util import (MIN_SHARED, assert_ca_bit_exact, assert_final_consistency, assert_final_track_records,
                         final_track_report, run_oracle, tracklet_report)

pytestmark = pytest.mark.gpu


def _gpu(ev, **kw):
    from paper_1709_00618_b200 import Tracker
    trk = Tracker.for_event(ev, **kw)
    res = trk.track_sectors(ev.clusters, ev.row_offsets, ev.n_inst, debug=True)
    trk.close()
    return res


def _parity(ev, label, max_ok_mismatch=0):
    o = run_oracle(ev, nf_bridge_rows=1)
    g = _gpu(ev, nf_bridge_rows=1)
    assert_ca_bit_exact(g, o)
    tr = tracklet_report(g, o)
    fr = final_track_report(g, o, ev.n_clusters)
    assert_final_consistency(g, ev.n_clusters)
    # the same bar as the default reading (test_gpu_edge._check): covariance, chi2, reference rows and every trk_*
    # record, not only links, parameters and assignments
    rec = assert_final_track_records(g, o, ev.row_offsets, ev.n_rows, dg.row_x(ev.n_rows))
    os.makedirs("gpurun_out", exist_ok=True)
    with open("gpurun_out/parity_report.jsonl", "a") as f:
        f.write(json.dumps(dict(case=label, n_clusters=ev.n_clusters, **tr, **fr, **rec)) + "\n")
    assert tr["ok_mismatch"] <= max_ok_mismatch, tr
    assert tr["shared_frac"] >= MIN_SHARED and tr["worst_param_excess"] <= 1.0, tr
    assert rec["worst_track_param_excess"] <= 1.0, rec
    assert tr["nhits_equal"] and tr["rows_equal"] and tr["ref_rows_equal"], tr
    assert tr["worst_cov_excess"] <= 1.0 and tr["worst_chi2_excess"] <= 1.0, tr
    assert fr["shared_assign_frac"] >= MIN_SHARED, fr
    return g, o


def test_bridge_cfg1_low_efficiency():
    g, o = _parity(dg.single_sector(seed=1031, eff=0.9), "bridge_cfg1_eff0.9")
    base = _gpu(dg.single_sector(seed=1031, eff=0.9))
    assert g.n_cand < 0.7 * base.n_cand  # the point of the reading: fewer clone candidates


def test_bridge_cfg2_and_cfg3_like():
    _parity(dg.full_event(seed=2001), "bridge_cfg2")
    _parity(dg.full_event(seed=3002, n_prim=800, sec_frac=0.2, sigma_z=0.12, noise=0.10), "bridge_cfg3_small")


def test_bridge_small_drift_windows_batch():
    evs = [dg.drift_window(seed=5201 + i, mean_tracks=200.0, cap_tracks=500) for i in range(2)]
    _parity(dg.concat_events(evs), "bridge_cfg4_small_batch")


def test_bridge_duplicates_and_edges():
    """Every cluster twice (all ties, also between the two class-1 kinds) and bridged links next to rows 0 / R-1."""
    ev = dg.single_sector(seed=1032, n_tracks=60, eff=0.85)
    rows = np.repeat(np.arange(ev.n_rows), np.diff(ev.row_offsets))
    order = np.argsort(np.concatenate([rows, rows]), kind="stable")
    cl = np.concatenate([ev.clusters, ev.clusters])[order]
    ro = np.concatenate([[0], np.cumsum(np.bincount(rows, minlength=ev.n_rows) * 2)]).astype(np.int32)
    dup = dataclasses.replace(ev, clusters=np.ascontiguousarray(cl), row_offsets=ro,
                              labels=np.full(len(cl), -1, np.int32), truth={})
    _parity(dup, "bridge_duplicates")


def test_bridge_full_size_window():
    ev = dg.drift_window(seed=5001)
    _parity(ev, "bridge_cfg4_full_window", max_ok_mismatch=1)  # observed 0 of 2.0 M clusters' tracklets, + 1
