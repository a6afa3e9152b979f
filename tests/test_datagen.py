"""Generator checks: CSR consistency, determinism, sizes of BASELINE.json configs."""
import numpy as np

from paper_1709_00618_b200 import datagen as dg


def _check_csr(ev):
    ro = ev.row_offsets
    assert ro.dtype == np.int32 and ro[0] == 0 and ro[-1] == ev.n_clusters
    assert len(ro) == ev.n_inst * ev.n_rows + 1
    assert np.all(np.diff(ro) >= 0)
    rx = dg.row_x(ev.n_rows)
    rows = (np.searchsorted(ro, np.arange(ev.n_clusters), side="right") - 1) % ev.n_rows
    assert np.array_equal(ev.clusters[:, 0], rx[rows])
    assert ev.clusters.dtype == np.float32 and ev.clusters.shape[1] == 4
    assert np.array_equal(ev.clusters[:, 3].astype(np.int32), ev.labels)


def test_cfg1_size_and_determinism():
    a = dg.single_sector()
    b = dg.single_sector()
    _check_csr(a)
    assert np.array_equal(a.clusters, b.clusters) and np.array_equal(a.row_offsets, b.row_offsets)
    assert 6000 < a.n_clusters < 14000  # ~10 k clusters
    assert a.clusters[:, 2].min() > -1.0  # z >= 0 side (up to smear)
    c = dg.single_sector(seed=1002)
    assert not np.array_equal(a.clusters[:100], c.clusters[:100])


def test_cfg2_size_and_sides():
    ev = dg.full_event()
    _check_csr(ev)
    assert 120_000 < ev.n_clusters < 180_000  # ~150 k
    inst = (np.searchsorted(ev.row_offsets, np.arange(ev.n_clusters), side="right") - 1) // ev.n_rows
    z = ev.clusters[:, 2]
    assert np.all(z[inst < 18] > -1.0) and np.all(z[inst >= 18] < 1.0)
    # inside the wedge (up to smear)
    assert np.all(np.abs(ev.clusters[:, 1]) <= ev.clusters[:, 0] * np.tan(dg.HALF_ANGLE_RAD) + 1.0)


def test_cfg4_shift_range():
    ev = dg.drift_window(seed=4002, mean_tracks=300.0)
    _check_csr(ev)
    assert ev.z_lo == -250.0 and ev.z_hi == 500.0
    inst = (np.searchsorted(ev.row_offsets, np.arange(ev.n_clusters), side="right") - 1) // ev.n_rows
    z = ev.clusters[:, 2]
    assert z[inst < 18].min() >= -251.0 and z[inst < 18].max() <= 501.0
    assert z[inst >= 18].min() >= -501.0 and z[inst >= 18].max() <= 251.0


def test_batch_concat():
    b = dg.window_batch(2, seed0=5001, mean_tracks=100.0)
    _check_csr(b)
    assert b.n_inst == 72
    assert b.labels.max() < len(b.truth["pt"])


def test_truth_state_on_helix():
    """local_truth_state agrees with the generated (zero-smear) clusters: y, z at each row."""
    trk = dict(pt=[0.8, 1.5], eta=[0.3, 0.6], q=[1.0, -1.0], phi0=[0.17, 0.2], x0=[0.0, 0.0], y0=[0.0, 0.0],
               z0=[0.0, 0.0])
    ev, y64, z64 = dg.from_tracks(trk, bz=0.5, fp64_coords=True)
    t = {k: np.asarray(v, float) for k, v in trk.items()}
    for i in range(ev.n_clusters):
        s = dg.local_truth_state(t, int(ev.labels[i]), float(ev.clusters[i, 0]), 0.5)
        assert abs(s[0] - y64[i]) < 1e-9 and abs(s[1] - z64[i]) < 1e-9


def test_quantise_i16_round_trip_and_resolution():
    """16-bit fixed-point input format (TPC_INPUT_I16): decode(encode(ev)) is within half a step of the fp32 input,
    the decoded values are exact multiples of the steps, and re-encoding the decoded event gives the same counts."""
    ev = dg.drift_window(seed=4003, mean_tracks=100.0, cap_tracks=300)
    q, evq = dg.quantise_i16(ev)
    assert q.dtype == np.int16 and q.shape == (ev.n_clusters, 2)
    dy = evq.clusters[:, 1].astype(np.float64) - ev.clusters[:, 1]
    dz = evq.clusters[:, 2].astype(np.float64) - ev.clusters[:, 2]
    assert np.abs(dy).max() <= 0.5 / 256 + 1e-6 and np.abs(dz).max() <= 0.5 / 64 + 1e-5
    assert np.all(evq.clusters[:, 1] * 256 == np.rint(evq.clusters[:, 1] * 256))
    q2, evq2 = dg.quantise_i16(evq)
    assert np.array_equal(q2, q) and np.array_equal(evq2.clusters, evq.clusters)
    assert np.array_equal(evq.row_offsets, ev.row_offsets) and np.array_equal(evq.clusters[:, 0], ev.clusters[:, 0])
    # both z sides are used and the unsigned z count spans most of its range for -250..500 cm windows
    qz = q[:, 1].view(np.uint16)
    assert qz.min() < 2000 and qz.max() > 40000
