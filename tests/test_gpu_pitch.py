"""GPU parity with a non-uniform pad-row pitch (reading A5'): 63 rows of 0.75 cm,
64 of 1.0 cm, 32 of 1.5 cm.  Same bar as the default geometry: links, start hits and candidates bit-exact, tracklets
and final tracks within the north_star tolerances."""
import numpy as np
import pytest

from paper_1709_00618_b200 import datagen as dg

from parity_util import (MIN_SHARED, assert_ca_bit_exact, assert_final_consistency, assert_final_track_records,
                         final_track_report, run_oracle, tracklet_report)

pytestmark = pytest.mark.gpu
RX3 = dg.row_x_three_pad_sizes()


def _parity(ev):
    from paper_1709_00618_b200 import Tracker
    assert np.array_equal(ev.row_x, RX3)
    o = run_oracle(ev)
    trk = Tracker.for_event(ev)
    g = trk.track_sectors(ev.clusters, ev.row_offsets, ev.n_inst, debug=True)
    trk.close()
    assert_ca_bit_exact(g, o)
    tr = tracklet_report(g, o)
    fr = final_track_report(g, o, ev.n_clusters)
    assert_final_consistency(g, ev.n_clusters)
    rec = assert_final_track_records(g, o, ev.row_offsets, ev.n_rows, ev.row_x)
    assert tr["ok_mismatch"] == 0 and tr["shared_frac"] >= MIN_SHARED and tr["worst_param_excess"] <= 1.0, tr
    assert tr["nhits_equal"] and tr["rows_equal"] and tr["ref_rows_equal"], tr
    assert tr["worst_cov_excess"] <= 1.0 and tr["worst_chi2_excess"] <= 1.0, tr
    assert rec["worst_track_param_excess"] <= 1.0 and fr["shared_assign_frac"] >= MIN_SHARED, (rec, fr)
    return g, o


def test_single_sector_three_pad_sizes():
    g, o = _parity(dg.single_sector(seed=1051, rx=RX3))
    assert g.n_tracks > 50


def test_steep_straight_tracks_cross_the_pitch_boundaries():
    """Bz = 0, slopes up to the window's bound: chains must run through both boundaries (one candidate per track)."""
    n = 10
    trk = dict(pt=np.full(n, 2.0), eta=np.linspace(0.1, 1.3, n), q=np.ones(n), phi0=np.linspace(0.05, 0.30, n),
               x0=np.zeros(n), y0=np.zeros(n), z0=np.zeros(n))
    ev = dg.from_tracks(trk, bz=0.0, rx=RX3, sigma_y=0.03, sigma_z=0.03)
    g, o = _parity(ev)
    assert g.n_cand == len(np.unique(ev.labels)) == g.n_tracks


def test_full_event_three_pad_sizes_both_sides():
    _parity(dg.full_event(seed=2051, n_prim=600, sec_frac=0.2, noise=0.10, rx=RX3))


def test_bridging_is_rejected_with_non_uniform_pitch():
    from paper_1709_00618_b200 import Tracker
    from paper_1709_00618_b200.tracker import TpcError
    with pytest.raises(TpcError, match="GEOMETRY"):
        Tracker(RX3, 0.5, nf_bridge_rows=1)
