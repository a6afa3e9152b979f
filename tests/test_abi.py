"""The C-ABI library loads and exports every symbol include/tpc_tracker.h declares; host-only entry points behave
as the header says.  No compute calls (no GPU needed)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "tpc_tracker.h")


@pytest.fixture(scope="module")
def lib():
    from paper_1709_00618_b200 import build, tracker
    build.build()
    return tracker.load_library()


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tpc_[a-z_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    from paper_1709_00618_b200 import tracker
    names = _declared_functions()
    assert len(names) >= 12
    for n in names:
        assert hasattr(lib, n), f"{n} declared in tpc_tracker.h but not exported by libtpctrk.so"
    assert sorted(tracker.EXPORTS) == names, "binding and header disagree on the entry points"


def test_binding_structs_match_header_sizes():
    from paper_1709_00618_b200 import tracker
    # tpc_params_t: 3 f + 2 i + 5 f + 2 f + 1 i + 2 f + 1 i + 1 f + 2 i = 19 words
    assert C.sizeof(tracker.Params) == 19 * 4
    raw = 8 + 8 + 4 * 6 + C.sizeof(tracker.Params)  # n_rows(+pad), ptr, spe..sigma, params
    assert C.sizeof(tracker.Geometry) == (raw + 7) // 8 * 8  # tail padding to the pointer alignment
    assert C.sizeof(tracker.Output) % 8 == 0
    # tpc_slot_t: 2 ptr + int64 + int32(+pad) + tpc_output_t + ptr + size_t
    assert C.sizeof(tracker.Slot) == 8 * 4 + C.sizeof(tracker.Output) + 16
    # tpc_phase2_output_t: 13 ptr + int64 + ptr
    assert C.sizeof(tracker.Phase2Output) == 8 * 15
    assert C.sizeof(tracker.VertexOutput) == 8 * 8
    # tpc_host_output_t: 7 ptr + 2 int64 + 16 int64 + 4 int64 + 4 float
    assert C.sizeof(tracker.HostOutput) == 8 * (7 + 2 + 16 + 4) + 16


def test_no_cpu_fallback_without_device(lib):
    import torch
    from paper_1709_00618_b200 import Tracker, TpcError, datagen
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(TpcError):
        Tracker(datagen.row_x(), 0.5)


def test_geometry_validation_is_host_side(lib):
    from paper_1709_00618_b200 import tracker
    rx = np.linspace(85.0, 247.0, 159).astype(np.float32)
    flat = rx.copy()
    flat[50] = flat[49]  # not strictly increasing
    uneven = rx.copy()
    uneven[50] += 0.3  # non-uniform pitch: accepted (reading A5') unless row bridging (reading A2') is asked for
    for arr, n, want, kw in ((flat, 159, -2, {}), (rx, 2, -2, {}), (rx[::-1].copy(), 159, -2, {}),
                             (uneven, 159, -2, dict(nf_bridge_rows=1))):
        geom, keep = tracker.make_geometry(arr[:n] if n < len(arr) else arr, **kw)
        geom.n_rows = n
        h = C.c_void_p()
        rc = lib.tpc_tracker_create(C.byref(geom), C.c_float(0.5), C.byref(h))
        assert rc == want and not h.value
        assert len(lib.tpc_last_error(None)) > 0
    assert lib.tpc_tracker_create(None, C.c_float(0.5), None) == -1


def test_check_counts_host_logic(lib):
    from paper_1709_00618_b200 import tracker
    o = tracker.Output()
    o.trk_capacity, o.trk_hits_capacity = 10, 100
    o.trk_hits = 0x1000  # any non-NULL value: the function only compares pointers with NULL
    o.cluster_owner = 0x1000
    cnt = (C.c_int64 * 16)()
    cnt[3], cnt[4] = 10, 100
    assert lib.tpc_check_counts(cnt, C.byref(o)) == 0
    cnt[3] = 11
    assert lib.tpc_check_counts(cnt, C.byref(o)) == -5
    cnt[3], cnt[4] = 10, 101
    assert lib.tpc_check_counts(cnt, C.byref(o)) == -5
    cnt[4], cnt[5] = 100, 1
    assert lib.tpc_check_counts(cnt, C.byref(o)) == -6
    assert lib.tpc_check_counts(None, C.byref(o)) == -1


def test_null_handle_calls_fail_cleanly(lib):
    assert lib.tpc_set_stream(None, None) == -1
    assert lib.tpc_set_workspace(None, None, 0) == -1
    assert lib.tpc_workspace_bytes(None, 100, 1) == 0
    assert lib.tpc_last_launch_count(None) == 0
    lib.tpc_tracker_destroy(None)
