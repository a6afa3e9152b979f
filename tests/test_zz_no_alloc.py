"""tpc_start_hits_static, the library's one entry point that allocates nothing, against the regular path.

Some users of the library cannot allocate device memory: their process runs inside a framework that took the whole
GPU at start-up and only passes them fixed buffers, or they sit in an online loop where a cudaMalloc (which
synchronises the whole device) is not allowed.  For them the start-hit search of S4 exists in a form whose scratch
memory is an array compiled into the library (include/tpc_tracker.h).  That array is shared by all calls and keeps
what the previous call left in it, so the thing to prove here is that a call's result does not depend on what ran
before: the same entry point is called several times in a row, on inputs of different sizes, and every result must
equal `start_hits` / counts[0] of tpc_track_sectors bit for bit (integer work: no tolerance).

The file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here must
not hide the parity tests.  It passes alone in a fresh process (the first call does the one-time address look-up)
and after the other tests (the tracker has used the GPU before).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1709_00618_b200 import build
    build.build()
    return torch


def _regular_path(ev):
    """Cleaned links and start hits of the existing path (tpc_track_sectors with the debug outputs)."""
    from paper_1709_00618_b200 import Tracker
    trk = Tracker.for_event(ev)
    g = trk.track_sectors(ev.clusters, ev.row_offsets, ev.n_inst, debug=True)
    trk.close()
    return g


def _static(torch, link_up, link_dn, capacity=None, offset=0):
    """One call of the no-allocation entry point; `offset` shifts the device arrays off their 16-byte alignment."""
    from paper_1709_00618_b200 import tracker
    dev = torch.device("cuda:0")
    n = len(link_up)
    up = torch.empty(n + offset, dtype=torch.int32, device=dev)[offset:]
    dn = torch.empty(n + offset, dtype=torch.int32, device=dev)[offset:]
    up.copy_(torch.from_numpy(link_up))
    dn.copy_(torch.from_numpy(link_dn))
    cap = n if capacity is None else capacity
    out = torch.full((max(cap, 1),), -7, dtype=torch.int32, device=dev)
    cnt = torch.full((1,), -7, dtype=torch.int64, device=dev)
    tracker.start_hits_static(up, dn, out[:cap] if cap > 0 else None, cnt, n_clusters=n)
    torch.cuda.synchronize(dev)
    return out.cpu().numpy(), int(cnt.item())


def test_static_start_hits_equal_the_regular_path_on_calls_in_a_row(torch_cuda):
    from paper_1709_00618_b200 import datagen
    big = datagen.full_event(seed=2001)      # CFG:2: ~150 k clusters = ~70 tiles, several look-back windows, ragged tail
    small = datagen.single_sector(seed=1001)  # CFG:1: a few tiles
    g_big, g_small = _regular_path(big), _regular_path(small)
    assert g_big.n_start > 1000 and g_small.n_start > 50 and len(g_big.link_up) % 2048 != 0
    # big, small, big again: the second and third call find the status words of the call before them in the array
    for g in (g_big, g_small, g_big, g_big):
        out, n_start = _static(torch_cuda, g.link_up, g.link_dn)
        assert n_start == g.n_start
        assert np.array_equal(out[:n_start], g.start_hits)
        assert np.all(out[n_start:] == -7), "nothing is written beyond the count"
    # arrays that are not 16-byte aligned take the scalar loads; same result
    out, n_start = _static(torch_cuda, g_small.link_up, g_small.link_dn, offset=1)
    assert n_start == g_small.n_start and np.array_equal(out[:n_start], g_small.start_hits)


def test_static_start_hits_capacity_limit_and_empty_input(torch_cuda):
    from paper_1709_00618_b200 import datagen, tracker
    torch = torch_cuda
    g = _regular_path(datagen.single_sector(seed=1002))
    # too small an output: what fits is written, the count is the required one
    cap = g.n_start // 2
    out, n_start = _static(torch, g.link_up, g.link_dn, capacity=cap)
    assert n_start == g.n_start and np.array_equal(out[:cap], g.start_hits[:cap])
    # count only
    _, n_start = _static(torch, g.link_up, g.link_dn, capacity=0)
    assert n_start == g.n_start
    # no clusters: the count is cleared
    _, n_start = _static(torch, np.zeros(0, np.int32), np.zeros(0, np.int32))
    assert n_start == 0
    # beyond the built-in array: refused before anything is enqueued, with a text that names the limit
    dev = torch.device("cuda:0")
    dummy = torch.zeros(8, dtype=torch.int32, device=dev)
    cnt = torch.full((1,), -7, dtype=torch.int64, device=dev)
    with pytest.raises(tracker.TpcError, match="TPC_ERR_LIMIT.*TPC_STATIC_MAX_CLUSTERS"):
        tracker.start_hits_static(dummy, dummy, dummy, cnt, n_clusters=tracker.STATIC_MAX_CLUSTERS + 1)
    torch.cuda.synchronize(dev)
    assert int(cnt.item()) == -7
    # and the call after the refusal works as before
    out, n_start = _static(torch, g.link_up, g.link_dn)
    assert n_start == g.n_start and np.array_equal(out[:n_start], g.start_hits)
