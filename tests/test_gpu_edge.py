"""GPU edge cases and full-size parity: empty and ragged inputs, exact duplicates (tie-breaks), dense spots (the slow
paths of S2 and S5), capacity overflow, and the bench's own workload (full CFG:4 windows) against the oracle."""
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
    create_kw = {k: kw.pop(k) for k in list(kw) if k.startswith("grid_")}  # tracker parameters; the rest per call
    trk = Tracker.for_event(ev, **create_kw)
    res = trk.track_sectors(ev.clusters, ev.row_offsets, ev.n_inst, debug=True, **kw)
    trk.close()
    return res


def _rebuild(ev, clusters, rows, inst=None):
    """An Event with the given clusters; rows (and instances) say where each goes.  Order inside a row = given order."""
    inst = np.zeros(len(rows), np.int64) if inst is None else np.asarray(inst, np.int64)
    slab = inst * ev.n_rows + np.asarray(rows, np.int64)
    order = np.argsort(slab, kind="stable")
    ro = np.zeros(ev.n_inst * ev.n_rows + 1, np.int32)
    np.add.at(ro, slab + 1, 1)
    ro = np.cumsum(ro).astype(np.int32)
    cl = np.ascontiguousarray(clusters[order], np.float32)
    return dataclasses.replace(ev, clusters=cl, row_offsets=ro, labels=np.full(len(cl), -1, np.int32), truth={})


def _rows_of(ev):
    return np.repeat(np.arange(ev.n_inst * ev.n_rows), np.diff(ev.row_offsets)) % ev.n_rows


def _check(ev, max_ok_mismatch=0, **gpu_kw):
    o = run_oracle(ev)
    g = _gpu(ev, **gpu_kw)
    assert_ca_bit_exact(g, o)
    tr = tracklet_report(g, o)
    fr = final_track_report(g, o, ev.n_clusters)
    assert_final_consistency(g, ev.n_clusters)
    rec = assert_final_track_records(g, o, ev.row_offsets, ev.n_rows, dg.row_x(ev.n_rows))
    os.makedirs("gpurun_out", exist_ok=True)
    with open("gpurun_out/parity_report.jsonl", "a") as f:
        f.write(json.dumps(dict(case=ev.name, n_clusters=ev.n_clusters, **tr, **fr, **rec)) + "\n")
    assert tr["ok_mismatch"] <= max_ok_mismatch, tr
    assert tr["shared_frac"] >= MIN_SHARED and tr["worst_param_excess"] <= 1.0, tr
    assert rec["worst_track_param_excess"] <= 1.0, rec
    assert tr["nhits_equal"] and tr["rows_equal"] and tr["ref_rows_equal"], tr
    assert tr["worst_cov_excess"] <= 1.0 and tr["worst_chi2_excess"] <= 1.0, tr
    if fr["n_tracks_gpu"] or fr["n_tracks_oracle"]:
        assert fr["shared_assign_frac"] >= MIN_SHARED, fr
    return g, o


def test_empty_input():
    ev = dg.single_sector(seed=1001)
    empty = _rebuild(ev, ev.clusters[:0], np.zeros(0, np.int64))
    g = _gpu(empty)
    assert g.counts[:6].tolist() == [0, 0, 0, 0, 0, 0]
    assert g.cluster_owner.shape == (0,) and g.trk_hit_offset[0] == 0


def test_ragged_rows_few_hits():
    """Most rows empty: hits only in rows 0..14 and 140..158, one row with a single hit."""
    ev = dg.single_sector(seed=1011)
    rows = _rows_of(ev)
    keep = (rows <= 14) | (rows >= 140)
    keep[np.flatnonzero(rows == 3)[1:]] = False
    rag = _rebuild(ev, ev.clusters[keep], rows[keep])
    g, o = _check(rag)
    assert g.n_tracks == len(o.trk_cand) and g.n_tracks > 0


def test_short_tracks_only_no_final_track():
    """Tracks of 8 rows: candidates and tracklets exist, but no tracklet reaches sel_min = 10 hits."""
    ev = dg.single_sector(seed=1012, noise=0.0)
    rows = _rows_of(ev)
    keep = (rows >= 40) & (rows < 48)
    sh = _rebuild(ev, ev.clusters[keep], rows[keep])
    g, o = _check(sh)
    assert g.n_cand > 0 and g.n_tracks == 0 and np.all(g.cluster_owner == -1)


def test_exact_duplicates_tie_breaks():
    """Every cluster twice: every D and every pick-up distance ties exactly, so the lowest-index rules decide."""
    ev = dg.single_sector(seed=1013, n_tracks=60)
    rows = _rows_of(ev)
    cl = np.concatenate([ev.clusters, ev.clusters])
    dup = _rebuild(ev, cl, np.concatenate([rows, rows]))
    _check(dup)


def test_dense_spot_slow_paths():
    """> 4 window hits in the neighbour rows and > 3 hits in the follower's gate: the loops behind the in-line paths."""
    ev = dg.single_sector(seed=1014, n_tracks=40)
    rows = _rows_of(ev)
    rng = np.random.default_rng(77)
    extra_rows = np.repeat(np.arange(60, 75), 12)
    x = dg.row_x(ev.n_rows)[extra_rows]
    blob = np.stack([x, rng.uniform(-1.0, 1.0, len(x)), rng.uniform(99.0, 101.5, len(x)),
                     np.full(len(x), -1.0)], axis=1).astype(np.float32)
    dense = _rebuild(ev, np.concatenate([ev.clusters, blob]), np.concatenate([rows, extra_rows]))
    _check(dense)


@pytest.mark.parametrize("grid", [{}, {"grid_cell_z": 0.7}, {"grid_cell_z": 0.7, "grid_cells_y": 3}])
def test_duplicated_dense_spot_ties_in_the_slow_paths(grid):
    """The dense spot with EVERY cluster duplicated: exact ties among more hits than the in-line paths hold (S2: more
    than four window hits per neighbour row; S5: ties beyond the fourth hit of the gate and, with z bins narrower than
    the gate, in the loop over the bins in between), all resolved by the lowest local index as in the oracle."""
    ev = dg.single_sector(seed=1014, n_tracks=40)
    rows = _rows_of(ev)
    rng = np.random.default_rng(78)
    extra_rows = np.repeat(np.arange(60, 75), 8)
    x = dg.row_x(ev.n_rows)[extra_rows]
    blob = np.stack([x, rng.uniform(-1.0, 1.0, len(x)), rng.uniform(99.0, 101.5, len(x)),
                     np.full(len(x), -1.0)], axis=1).astype(np.float32)
    cl = np.concatenate([ev.clusters, blob])
    rw = np.concatenate([rows, extra_rows])
    dup = _rebuild(ev, np.concatenate([cl, cl]), np.concatenate([rw, rw]))
    _check(dup, **grid)


def test_capacity_overflow_is_reported_not_written():
    from paper_1709_00618_b200 import Tracker
    from paper_1709_00618_b200.tracker import TpcError
    ev = dg.single_sector(seed=1001)
    full = _gpu(ev)
    assert full.n_tracks > 4
    trk = Tracker.for_event(ev)
    with pytest.raises(TpcError, match="CAPACITY"):
        trk.track_sectors(ev.clusters, ev.row_offsets, ev.n_inst, trk_capacity=3)
    trk.close()


def test_full_size_drift_windows_against_oracle():
    """The bench's workload at full size: three full CFG:4 windows (5 overlapping events each, 108 sector instances:
    enough slabs for the two-level scan of the long-input path), in the launch configuration bench.py times (one
    tpc_track_sectors call on the batch)."""
    evs = [dg.drift_window(seed=5001 + i) for i in range(3)]
    batch = dg.concat_events(evs)
    assert batch.n_clusters > 1_000_000
    # A tracklet exists or not by threshold tests on the fitted state (|sinPhi| <= 0.95 in a transport): fp64 in the
    # oracle, fp32 in the kernels (A12/A13), so at this size a handful of the ~130 k candidates may fall on
    # the other side; they count against the 99.5 % shared-assignment bar like any other difference.
    # Observed: 1 of 130,252 candidates (round 1); the allowance is observed + 1.
    g, o = _check(batch, max_ok_mismatch=2)
    assert abs(g.n_tracks - len(o.trk_cand)) <= 2


def test_compact_inputs_and_host_pipeline_against_oracle_full_window():
    """One full CFG:4 window through every input layout and both entry points, each compared with the ORACLE:
    (y, z) pairs (TPC_INPUT_YZ) must reproduce the float4 result bit for bit; 16-bit fixed point (TPC_INPUT_I16) is
    compared with the oracle run on the decoded coordinates (the quantisation is applied before either side sees the
    clusters, so links and candidates stay bit-exact); the chunked host pipeline returns the same job-wide arrays."""
    import torch
    from paper_1709_00618_b200 import Tracker
    from paper_1709_00618_b200.tracker import HostPipeline
    ev = dg.drift_window(seed=5003)
    assert ev.n_clusters > 300_000
    g_ref, o_ref = _check(ev, max_ok_mismatch=1)
    q, ev_q = dg.quantise_i16(ev)
    assert np.abs(ev_q.clusters[:, 1:3] - ev.clusters[:, 1:3]).max() <= 0.5 / 64 + 1e-4
    o_q = run_oracle(ev_q)
    R = ev.n_rows
    for layout, data, o in (("yz", np.ascontiguousarray(ev.clusters[:, 1:3]), o_ref), ("i16", q, o_q)):
        trk = Tracker.for_event(ev)
        trk.set_input_layout(layout)
        g = trk.track_sectors(data, ev.row_offsets, ev.n_inst, debug=True)
        assert_ca_bit_exact(g, o)
        tr = tracklet_report(g, o)
        fr = final_track_report(g, o, ev.n_clusters)
        assert_final_consistency(g, ev.n_clusters)
        assert_final_track_records(g, o, ev.row_offsets, R, dg.row_x(R))
        assert tr["ok_mismatch"] <= 1 and tr["shared_frac"] >= MIN_SHARED and tr["worst_param_excess"] <= 1.0, tr
        assert tr["worst_cov_excess"] <= 1.0 and tr["worst_chi2_excess"] <= 1.0, tr
        assert fr["shared_assign_frac"] >= MIN_SHARED, fr
        if layout == "yz":  # same (y, z) as the float4 call: identical bits
            for k in ("link_up_raw", "cand_hits", "tl_hits", "tl_params", "tl_cov", "trk_params", "cluster_owner"):
                assert np.array_equal(getattr(g, k), getattr(g_ref, k)), k
        # the chunked host pipeline on this layout: 7 chunks of 6 sector instances (the last one ragged), 3 slots
        h_in = torch.from_numpy(data).pin_memory()
        h_ro = torch.from_numpy(ev.row_offsets).pin_memory()
        ipc = 5
        mx = max(int(ev.row_offsets[min(i + ipc, ev.n_inst) * R] - ev.row_offsets[i * R])
                 for i in range(0, ev.n_inst, ipc))
        pipe = HostPipeline(trk, mx, ipc, ev.n_clusters, n_slots=3)
        ho = pipe.run(h_in, h_ro, ev.n_inst)
        nt, nh = ho["totals"][3], ho["totals"][4]
        assert nt == g.n_tracks and nh == g.n_track_hits
        assert ho["h2d_bytes"] == data.itemsize * 2 * ev.n_clusters + 4 * (ev.n_inst * R + ho["n_chunks"])
        own = pipe.host["cluster_owner"].numpy()[:ev.n_clusters]
        assert np.array_equal(own, g.cluster_owner)
        assert np.array_equal(pipe.host["trk_hits"].numpy()[:nh], g.trk_hits)
        assert np.array_equal(pipe.host["trk_params"].numpy()[:nt], g.trk_params)
        # ... and directly against the oracle: final assignment by candidate id
        own_o = np.where(o.cluster_owner >= 0, o.trk_cand[np.maximum(o.cluster_owner, 0)], -1)
        own_g = np.where(own >= 0, g.trk_cand_id[np.maximum(own, 0)], -1)
        assigned = (own_o >= 0) | (own_g >= 0)
        assert ((own_o == own_g) & assigned).sum() >= MIN_SHARED * assigned.sum()
        pipe.close()
        trk.close()


def test_host_pipeline_capacity_overflow_reports_totals():
    """Host result arrays too small for the job: the run still visits every chunk, returns
    TPC_ERR_CAPACITY (not a CUDA error from unrecorded events) and hout.totals hold the required sizes; the chunks
    downloaded before the arrays filled up are intact; a second run on the same pipeline behaves the same, and a
    pipeline with enough room gives the full result afterwards.  Slot (device) capacity overflow likewise."""
    import ctypes as C
    import torch
    from paper_1709_00618_b200 import Tracker
    from paper_1709_00618_b200.tracker import HostPipeline
    ev = dg.full_event(seed=2001)
    R = ev.n_rows
    trk = Tracker.for_event(ev)
    g = trk.track_sectors(ev.clusters, ev.row_offsets, ev.n_inst)
    h_in = torch.from_numpy(ev.clusters).pin_memory()
    h_ro = torch.from_numpy(ev.row_offsets).pin_memory()
    ipc = 4  # 9 chunks on 2 slots: the overflow falls both inside and after the first n_slots chunks
    mx = max(int(ev.row_offsets[min(i + ipc, ev.n_inst) * R] - ev.row_offsets[i * R]) for i in range(0, ev.n_inst, ipc))
    per_chunk = [int(((g.trk_sector >= i) & (g.trk_sector < i + ipc)).sum()) for i in range(0, ev.n_inst, ipc)]
    assert min(per_chunk) > 0
    for fit_chunks in (0, 3):
        pipe = HostPipeline(trk, mx, ipc, ev.n_clusters, n_slots=2)
        cap = sum(per_chunk[:fit_chunks]) + per_chunk[fit_chunks] // 2  # chunk `fit_chunks` no longer fits
        pipe.hout.trk_capacity = cap
        for _ in range(2):
            pipe.host["trk_nhits"].fill_(-5)
            with torch.cuda.device(trk.device):
                rc = trk.lib.tpc_pipeline_run(pipe._p, C.c_void_p(h_in.data_ptr()), C.c_void_p(h_ro.data_ptr()),
                                              ev.n_inst, ev.n_clusters, ipc, C.byref(pipe.hout))
            assert rc == -5, (rc, trk.lib.tpc_last_error(trk._h))
            assert int(pipe.hout.totals[3]) == g.n_tracks and int(pipe.hout.totals[4]) == g.n_track_hits
            assert int(pipe.hout.n_chunks) == len(per_chunk)
            done = sum(per_chunk[:fit_chunks])
            got = pipe.host["trk_nhits"].numpy()
            assert np.array_equal(got[:done], g.trk_nhits[:done]) and np.all(got[done:cap] == -5)
        pipe.close()
    # device-side (slot) track capacity too small: same contract
    pipe = HostPipeline(trk, mx, ipc, ev.n_clusters, n_slots=2)
    for s in range(2):
        pipe.slots[s].out.trk_capacity = max(per_chunk) // 2
    with torch.cuda.device(trk.device):
        h = C.c_void_p()
        assert trk.lib.tpc_pipeline_create(trk._h, pipe.slots, 2, C.byref(h)) == 0  # slots are copied at creation
        rc = trk.lib.tpc_pipeline_run(h, C.c_void_p(h_in.data_ptr()), C.c_void_p(h_ro.data_ptr()), ev.n_inst,
                                      ev.n_clusters, ipc, C.byref(pipe.hout))
        trk.lib.tpc_pipeline_destroy(h)
    assert rc == -5 and int(pipe.hout.totals[3]) == g.n_tracks
    pipe.close()
    # enough room: the whole job
    pipe = HostPipeline(trk, mx, ipc, ev.n_clusters, n_slots=2)
    ho = pipe.run(h_in, h_ro, ev.n_inst)
    assert ho["totals"][3] == g.n_tracks
    assert np.array_equal(pipe.host["trk_nhits"].numpy()[:g.n_tracks], g.trk_nhits)
    pipe.close()
    # the pipeline's chunks leave nothing for phase 2: the state of the tpc_track_sectors call above is stale now
    from paper_1709_00618_b200.tracker import TpcError
    with pytest.raises(TpcError, match="ARG"):
        trk.merge_refit(g.n_tracks)
    trk.close()


def test_i16_layout_is_refused_for_rows_wider_than_its_y_range():
    """TPC_INPUT_I16 holds |y| < 128 cm: a geometry whose outermost row is wider cannot use it."""
    from paper_1709_00618_b200 import Tracker
    from paper_1709_00618_b200.tracker import TpcError
    ok = Tracker(np.linspace(85.0, 247.0, 159).astype(np.float32), 0.5)
    ok.set_input_layout("i16")
    ok.close()
    wide = Tracker(np.linspace(85.0, 730.0, 159).astype(np.float32), 0.5)  # 730 tan(10 deg) + 0.5 = 129.2 cm
    with pytest.raises(TpcError, match="128 cm"):
        wide.set_input_layout("i16")
    wide.set_input_layout("yz")
    wide.close()


def test_full_size_central_event_against_oracle():
    """CFG:3 at full size: 8,000 primaries + 20 % secondaries, 10 % noise, ~1.5 M clusters, ~260 hits per row."""
    ev = dg.central_event(seed=3001)
    assert ev.n_clusters > 1_000_000
    _check(ev, max_ok_mismatch=2)  # observed 1 of 73,605 tracklets (A12/A13 threshold in fp32 vs fp64), + 1


def test_dense_rows_unstaged_neighbour_search():
    """Rows of 700-1000 hits (2,000 tracks in one sector): every row exceeds the 382 hits of S2's shared-memory row
    buffers, so all three rows of a slab are read in place; more than two hits per thread in S1."""
    ev = dg.single_sector(seed=1031, n_tracks=2000)
    n_row = np.diff(ev.row_offsets)
    assert (n_row[:-2] + n_row[2:]).max() > 1024 and n_row.max() > 600
    _check(ev)


def test_rows_around_the_staging_buffer_size():
    """1,000 tracks in one sector: 44 rows above and 115 rows below the 382 hits of S2's row buffers, so slabs mix rows
    that arrive by bulk copy with rows read in place (own row, row above, row below in every combination)."""
    ev = dg.single_sector(seed=1032, n_tracks=1000)
    n_row = np.diff(ev.row_offsets)
    big = n_row > 382
    assert big.sum() > 20 and (~big).sum() > 20
    assert (big[1:] != big[:-1]).any()  # at least one staged row next to an unstaged one
    _check(ev)


def test_many_nearly_empty_instances():
    """3,600 sector instances with a handful of tracks each: the per-instance bookkeeping (cell tables, slab scans,
    candidate bases) at a large instance count and tiny rows."""
    evs = [dg.full_event(seed=2100 + i, n_prim=12, noise=0.0) for i in range(100)]
    batch = dg.concat_events(evs)
    assert batch.n_inst == 3600
    g, o = _check(batch)
    assert g.n_tracks > 500


def test_cell_table_index_beyond_32_bits():
    """1,728 sector instances with the finest row grid (16,384 cells per row): instances x rows x cells = 4.5e9 > 2^32
    table entries (9 GB), beyond a 32-bit ENTRY index (it wrapped silently; the follower now indexes the
    table by its 32-byte row units, 16 entries each, and the call rejects jobs beyond 2^32 units -- next test)."""
    from paper_1709_00618_b200 import Tracker
    evs = [dg.full_event(seed=2300 + i, n_prim=12, noise=0.0) for i in range(48)]
    batch = dg.concat_events(evs)
    assert batch.n_inst == 1728
    o = run_oracle(batch)
    trk = Tracker.for_event(batch, grid_cells_y=64, grid_cell_z=0.98)
    assert trk.workspace_bytes(batch.n_clusters, batch.n_inst) > 8.5e9  # the table alone: 1728 * 159 * 16400 * 2 B
    g = trk.track_sectors(batch.clusters, batch.row_offsets, batch.n_inst, debug=True)
    trk.close()
    assert_ca_bit_exact(g, o)
    tr = tracklet_report(g, o)
    assert tr["ok_mismatch"] == 0 and tr["shared_frac"] >= MIN_SHARED and tr["worst_param_excess"] <= 1.0, tr
    assert np.array_equal(g.trk_cand_id, o.trk_cand) and g.n_tracks > 200


def test_row_longer_than_16_bit_limit_is_flagged():
    """A pad row with more than 65,535 clusters cannot be indexed by the 16-bit local positions: the call flags it
    (counts[5] bit 0 -> TPC_ERR_INPUT from tpc_check_counts), stays inside its buffers and leaves the tracker usable."""
    from paper_1709_00618_b200 import Tracker
    from paper_1709_00618_b200.tracker import TpcError
    ev = dg.single_sector(seed=1001)
    rows = _rows_of(ev)
    rng = np.random.default_rng(3)
    n_big = 66_000
    x = np.full(n_big, dg.row_x(ev.n_rows)[100])
    blob = np.stack([x, rng.uniform(-30, 30, n_big), rng.uniform(0, 250, n_big), np.full(n_big, -1.0)],
                    axis=1).astype(np.float32)
    big = _rebuild(ev, np.concatenate([ev.clusters, blob]), np.concatenate([rows, np.full(n_big, 100)]))
    assert np.diff(big.row_offsets).max() > 65_535
    trk = Tracker.for_event(big)
    with pytest.raises(TpcError, match="TPC_ERR_INPUT"):
        trk.track_sectors(big.clusters, big.row_offsets, big.n_inst, debug=True)
    ok = trk.track_sectors(ev.clusters, ev.row_offsets, ev.n_inst, debug=True)  # same handle, legal input
    o = run_oracle(ev)
    assert_ca_bit_exact(ok, o)
    trk.close()


def test_null_row_offsets_is_rejected():
    """n_sector_instances > 0 with row_offsets == NULL must be an argument error, not a device fault."""
    import ctypes as C
    import torch
    from paper_1709_00618_b200 import Tracker
    ev = dg.single_sector(seed=1001)
    trk = Tracker.for_event(ev)
    trk.reserve(16, 1)
    trk.set_stream()
    bufs, out = trk.alloc_outputs(16)
    rc = trk.lib.tpc_track_sectors(trk._h, None, None, 1, 0, C.byref(out))
    assert rc == -1
    torch.cuda.synchronize()
    trk.close()


def test_cell_table_beyond_the_follower_index_is_rejected():
    """30,000 sector instances with the finest row grid: 30,000 x 159 rows x 1,025 units of 32 bytes = 4.9e9 >= 2^32,
    more than the follower's 32-bit unit index covers (a 156 GB table): TPC_ERR_ARG before anything is touched."""
    import ctypes as C
    import torch
    from paper_1709_00618_b200 import Tracker
    ev = dg.single_sector(seed=1001)
    trk = Tracker.for_event(ev, grid_cells_y=64, grid_cell_z=0.98)
    trk.reserve(16, 1)
    trk.set_stream()
    bufs, out = trk.alloc_outputs(16)
    dummy = torch.zeros(64, dtype=torch.int32, device="cuda")
    rc = trk.lib.tpc_track_sectors(trk._h, dummy.data_ptr(), dummy.data_ptr(), 30_000, 16, C.byref(out))
    assert rc == -1
    ok = trk.lib.tpc_track_sectors(trk._h, dummy.data_ptr(), dummy.data_ptr(), 20_000, 16, C.byref(out))
    assert ok != -1  # 20,000 instances pass the argument checks (and fail later: the workspace is far too small)
    torch.cuda.synchronize()
    trk.close()


def test_twenty_drift_windows_against_oracle():
    """20 full CFG:4 windows in one call (720 sector instances, ~23 M clusters): the parameter tolerance at a fifth of
    the bench size (the worst excess grows with the sample; DESIGN.md section 6 quotes this figure)."""
    evs = [dg.drift_window(seed=5001 + i) for i in range(20)]
    batch = dg.concat_events(evs)
    assert batch.n_clusters > 15_000_000
    # A12/A13 threshold flips: observed 1 per ~130 k candidates -> ~8 expected in ~1 M; allowance 12
    g, o = _check(batch, max_ok_mismatch=12)
    assert abs(g.n_tracks - len(o.trk_cand)) <= 8


_FULL = {}  # shared with the forked workers of the all-windows comparison below (copy-on-write, nothing pickled)


def _window_tracklet_excess(w):
    """Worker: the oracle on window w of the bench batch alone, its tracklets against the GPU's slice for that window.
    Returns plain numbers."""
    from oracle.tpc_oracle import Oracle
    from parity_util import PAR_ATOL, PAR_RTOL
    b, R = _FULL["batch"], _FULL["R"]
    lo, hi = int(b.row_offsets[36 * w * R]), int(b.row_offsets[36 * (w + 1) * R])
    ro = (b.row_offsets[36 * w * R:36 * (w + 1) * R + 1] - lo).astype(np.int32)
    o = Oracle.for_event(b).track(b.clusters[lo:hi], ro, 36)
    c0, c1 = (int(x) for x in np.searchsorted(_FULL["cand_first"], [lo, hi]))
    if c1 - c0 != len(o.cand_n):
        return dict(window=w, cand_mismatch=1)
    th = _FULL["tl_hits"][c0:c1]
    th = np.where(th >= 0, th - lo, -1)
    ok_o, ok_g = o.tracklets["ok"].astype(bool), _FULL["tl_nhits"][c0:c1] > 0
    same = np.all(th == o.tracklet_hits, axis=1) & ok_o & ok_g
    pg = _FULL["tl_params"][c0:c1][same].astype(np.float64)
    po = o.tracklets["p"][same]
    ex = (np.abs(pg - po) / (PAR_ATOL + PAR_RTOL * np.abs(po))).max(axis=1) if same.any() else np.zeros(0)
    nh = o.tracklets["nhits"][same]
    over = ex > 1.0
    return dict(window=w, cand_mismatch=0, tracklets=int(ok_o.sum()), ok_flips=int((ok_o != ok_g).sum()),
                identical_lists=int(same.sum()), beyond_tol=int(over.sum()), worst=float(ex.max()) if ex.size else 0.0,
                beyond_tol_max_nhits=int(nh[over].max()) if over.any() else 0)


def test_full_bench_batch_sampled_instances_against_oracle():
    """BASELINE.json configs[4] at FULL size, in the launch configuration bench.py times: 100 drift windows (3,600
    sector instances, 116 M clusters) in ONE tpc_track_sectors call.  Sector instances are independent, so the oracle
    can compute any one of them alone: twelve sampled instances (first, last, both z sides, the largest) are compared
    output by output -- links, start hits and candidates bit-exact; tracklet hit lists, parameters, covariance, chi2;
    final assignment -- plus the properties that hold at any size for the whole batch.  Then (round 3) EVERY window
    goes through the oracle in a process pool and all 5.15 M tracklets are held to the north_star parameter bar, and
    tpc_merge_refit on the call's 1.39 M final tracks is compared on three sampled windows."""
    import sys
    import torch
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import bench
    from oracle.tpc_oracle import Oracle
    from paper_1709_00618_b200 import Tracker
    from parity_util import COV_TOL, PAR_ATOL, PAR_RTOL
    evs, batch = bench.make_batch(100, 5001, 0)
    N, S, R = batch.n_clusters, batch.n_inst, batch.n_rows
    assert S == 3600 and N > 100_000_000
    trk = Tracker.for_event(batch)
    dev = trk.device
    d_cl = torch.from_numpy(batch.clusters).to(dev)
    d_ro = torch.from_numpy(batch.row_offsets).to(dev)
    trk.reserve(N, S)
    trk.set_stream()
    bufs, out = trk.alloc_outputs(N, debug=True, trk_capacity=N // 20 + 64)
    trk.track_sectors_device(d_cl, d_ro, S, out)
    torch.cuda.synchronize(dev)
    counts = bufs["counts"].cpu().numpy()
    n_start, n_cand, n_tl, n_trk, n_thits = (int(x) for x in counts[:5])
    assert counts[5] == 0 and n_cand > 5_000_000 and n_trk > 1_300_000
    # whole-batch properties (any size)
    off = bufs["trk_hit_offset"][:n_trk + 1].cpu().numpy()
    nh = bufs["trk_nhits"][:n_trk].cpu().numpy()
    assert off[0] == 0 and off[n_trk] == n_thits and np.array_equal(np.diff(off), nh) and nh.min() >= 10
    cid = bufs["trk_cand_id"][:n_trk].cpu().numpy()
    assert np.all(np.diff(cid) > 0)
    assert int((bufs["cluster_owner"] >= 0).sum()) == n_thits
    cand_first = bufs["cand_hits"][:n_cand, 0].cpu().numpy()
    assert np.all(np.diff(cand_first) > 0)
    start_hits = bufs["start_hits"][:n_start].cpu().numpy()
    inst_sizes = np.diff(batch.row_offsets[::R])
    sample = sorted({0, 1, 17, 18, 35, 36, 1799, 1800, 3564, 3599, int(np.argmax(inst_sizes)), int(np.argmin(inst_sizes))})
    worst = 0.0
    for inst in sample:
        lo, hi = int(batch.row_offsets[inst * R]), int(batch.row_offsets[(inst + 1) * R])
        ro1 = (batch.row_offsets[inst * R:(inst + 1) * R + 1] - lo).astype(np.int32)
        # the instance alone, as instance `inst % 36` of a one-window problem (its z side must survive): pad with
        # empty instances in front
        k = inst % 36
        ro_pad = np.concatenate([np.zeros(k * R, np.int32), ro1, np.full((35 - k) * R, ro1[-1], np.int32)])
        orc = Oracle.for_event(batch)
        o = orc.track(batch.clusters[lo:hi], ro_pad, 36)

        def reb(a):  # device slice of a per-cluster index array, re-based to the instance
            v = a[lo:hi].cpu().numpy()
            return np.where(v >= 0, v - lo, -1)
        assert np.array_equal(reb(bufs["link_up_raw"]), o.link_up_raw) and np.array_equal(reb(bufs["link_dn_raw"]), o.link_dn_raw)
        assert np.array_equal(reb(bufs["link_up"]), o.link_up) and np.array_equal(reb(bufs["link_dn"]), o.link_dn)
        s0, s1 = np.searchsorted(start_hits, [lo, hi])
        assert np.array_equal(start_hits[s0:s1] - lo, o.start_hits)
        c0, c1 = np.searchsorted(cand_first, [lo, hi])
        assert c1 - c0 == len(o.cand_n)
        ch = bufs["cand_hits"][c0:c1].cpu().numpy()
        assert np.array_equal(np.where(ch >= 0, ch - lo, -1), o.cand_hits)
        assert np.array_equal(bufs["cand_n"][c0:c1].cpu().numpy(), o.cand_n)
        th = bufs["tl_hits"][c0:c1].cpu().numpy()
        th = np.where(th >= 0, th - lo, -1)
        nhg = bufs["tl_nhits"][c0:c1].cpu().numpy()
        ok_o = o.tracklets["ok"].astype(bool)
        assert np.array_equal(nhg > 0, ok_o)
        same = np.all(th == o.tracklet_hits, axis=1) & ok_o
        assert same.sum() >= MIN_SHARED * ok_o.sum()
        pg = bufs["tl_params"][c0:c1].cpu().numpy().astype(np.float64)[same]
        po = o.tracklets["p"][same]
        ex = np.abs(pg - po) / (PAR_ATOL + PAR_RTOL * np.abs(po))
        worst = max(worst, float(ex.max()))
        assert ex.max() <= 1.0
        cg = bufs["tl_cov"][c0:c1].cpu().numpy().astype(np.float64)[same]
        co = o.tracklets["cov"][same]
        ii = np.array([i for i in range(5) for j in range(i + 1)])
        jj = np.array([j for i in range(5) for j in range(i + 1)])
        diag = np.array([0, 2, 5, 9, 14])
        assert (np.abs(cg - co) / (COV_TOL * np.sqrt(co[:, diag[ii]] * co[:, diag[jj]]))).max() <= 1.0
        # final assignment of this instance's clusters, tracks matched by candidate id
        own = bufs["cluster_owner"][lo:hi].cpu().numpy()
        own_g = np.where(own >= 0, cid[np.maximum(own, 0)] - c0, -1)
        own_o = np.where(o.cluster_owner >= 0, o.trk_cand[np.maximum(o.cluster_owner, 0)], -1)
        assigned = (own_g >= 0) | (own_o >= 0)
        assert ((own_g == own_o) & assigned).sum() >= MIN_SHARED * assigned.sum()
    os.makedirs("gpurun_out", exist_ok=True)
    with open("gpurun_out/parity_report.jsonl", "a") as f:
        f.write(json.dumps(dict(case="cfg5_full_100_windows_sampled", n_clusters=N, instances=sample,
                                worst_param_excess=worst, n_cand=n_cand, n_tracks=n_trk)) + "\n")
    # ---- every window of the call against the oracle ("show that the north_star tolerance holds on all
    # 5.2 M tracklets of the headline workload, or state the measured exceedance rate").  Windows are independent: the
    # oracle runs them one per worker process; the GPU's tracklet arrays are shared with the workers by fork.
    import multiprocessing as mp
    _FULL.update(batch=batch, R=R, cand_first=cand_first, tl_hits=bufs["tl_hits"][:n_cand].cpu().numpy(),
                 tl_nhits=bufs["tl_nhits"][:n_cand].cpu().numpy(), tl_params=bufs["tl_params"][:n_cand].cpu().numpy())
    with mp.get_context("fork").Pool(min(os.cpu_count() or 1, 32)) as pool:
        per_win = pool.map(_window_tracklet_excess, range(100), chunksize=1)
    _FULL.clear()
    tot = {k: int(sum(r.get(k, 0) for r in per_win)) for k in ("cand_mismatch", "tracklets", "ok_flips",
                                                                "identical_lists", "beyond_tol")}
    tot["worst"] = max(r.get("worst", 0.0) for r in per_win)
    tot["beyond_tol_max_nhits"] = max(r.get("beyond_tol_max_nhits", 0) for r in per_win)
    with open("gpurun_out/parity_report.jsonl", "a") as f:
        f.write(json.dumps(dict(case="cfg5_full_100_windows_ALL_tracklets", **tot)) + "\n")
    assert tot["cand_mismatch"] == 0  # candidates are bit-exact in every window
    # observed: 1 one-sided tracklet of 5,149,574 (A12/A13 threshold in fp32 vs fp64) -> observed + 1
    assert tot["identical_lists"] >= MIN_SHARED * tot["tracklets"] and tot["ok_flips"] <= 2, tot
    # the north_star bar (1e-3 relative / 1e-4 absolute) on every tracklet with the same hit list on both sides:
    # measured on the B200 in round 3: 0 of 5,149,552 beyond the bar, worst 0.72; allowance =
    # observed + 1, and what exceeds must stay near the bar
    assert tot["beyond_tol"] <= 1 and tot["worst"] <= 2.0, tot
    # ---- phase 2 at the size bench.py times it: tpc_merge_refit on all 1.39 M final tracks of this call, compared
    # with the oracle on three sampled WINDOWS (36 instances each: links never leave a window).  The oracle's phase 2
    # gets the GPU's own final tracks of the window, so S5 near-tie flips do not stand in the way.
    from test_gpu_phase2 import _phase2_compare
    p2bufs, p2o = trk.alloc_phase2(n_trk)
    trk.merge_refit_device(p2o)
    torch.cuda.synchronize(dev)
    c2 = p2bufs["counts2"].cpu().numpy()
    assert c2[0] == n_trk - c2[1] and c2[1] > 500_000
    sec = bufs["trk_sector"][:n_trk].cpu().numpy()
    hits = bufs["trk_hits"]
    mfirst = p2bufs["mtrk_first"][:int(c2[0])].cpu().numpy()
    for w in (0, 57, 99):
        t0, t1 = (int(x) for x in np.searchsorted(sec, [36 * w, 36 * (w + 1)]))
        lo, hi = int(batch.row_offsets[36 * w * R]), int(batch.row_offsets[36 * (w + 1) * R])
        ro_w = (batch.row_offsets[36 * w * R:36 * (w + 1) * R + 1] - lo).astype(np.int32)
        off_w = off[t0:t1 + 1] - off[t0]
        hits_w = hits[int(off[t0]):int(off[t1])].cpu().numpy() - lo
        q = Oracle.for_event(batch).phase2_on_tracks(batch.clusters[lo:hi], ro_w, 36, sec[t0:t1] - 36 * w, off_w, hits_w)
        m0, m1 = (int(x) for x in np.searchsorted(mfirst, [t0, t1]))

        def loc(name, a, b, shift=None):
            v = p2bufs[name][a:b].cpu().numpy()
            return np.where(v >= 0, v - shift, -1) if shift is not None else v
        pw = {k: loc(k, t0, t1) for k in ("seg_ok", "seg_params", "seg_cov", "seg_chi2")}
        pw.update(seg_next=loc("seg_next", t0, t1, t0), seg_prev=loc("seg_prev", t0, t1, t0))
        pw.update({k: loc(k, m0, m1) for k in ("mtrk_nseg", "mtrk_nhits", "mtrk_ok", "mtrk_params", "mtrk_cov")})
        pw["mtrk_first"] = loc("mtrk_first", m0, m1, t0)
        assert pw["seg_next"].max() < t1 - t0  # a link never leaves its window
        pw["counts2"] = np.array([m1 - m0, int((pw["seg_next"] >= 0).sum())])
        rep = _phase2_compare(pw, q, t1 - t0, min_links=3000)
        assert rep["chains_3plus_compared"] >= 1, rep
    trk.close()
