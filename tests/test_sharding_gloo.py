"""N > 1 host logic on CPU: world_size-2 gloo.  The data path has no collective; what is
covered here is the partition of sector instances, that a shard is a self-contained tracker input whose results are the
corresponding slice of the whole job (checked with the CPU oracle standing in for the per-rank tracker), and the
max/sum reduction the bench contract asks for."""
import os

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1709_00618_b200 import datagen as dg
from paper_1709_00618_b200 import sharding as sh


def test_window_seeds_are_disjoint():
    a, b = sh.window_seeds(4, 5001, 0), sh.window_seeds(4, 5001, 1)
    assert a == [5001, 5002, 5003, 5004] and b == [5005, 5006, 5007, 5008]


def test_partition_covers_everything_once():
    evs = [dg.drift_window(seed=5201 + i, mean_tracks=30.0 * (i + 1), cap_tracks=200) for i in range(5)]
    batch = dg.concat_events(evs)
    for world in (1, 2, 3, 4, 8):
        parts = [sh.partition_instances(batch.row_offsets, batch.n_inst, batch.n_rows, world, r) for r in range(world)]
        assert parts[0][0] == 0 and parts[0][2] == 0
        for (i0, ni, c0, nc), (j0, _, d0, _) in zip(parts[:-1], parts[1:]):
            assert i0 + ni == j0 and c0 + nc == d0
        i0, ni, c0, nc = parts[-1]
        assert i0 + ni == batch.n_inst and c0 + nc == batch.n_clusters
        assert all(p[0] % 36 == 0 for p in parts)


def _worker(rank, world, port, tmp):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle.tpc_oracle import Oracle
        evs = [dg.drift_window(seed=5301 + i, mean_tracks=40.0, cap_tracks=120) for i in range(4)]
        batch = dg.concat_events(evs)
        i0, ni, c0, nc = sh.partition_instances(batch.row_offsets, batch.n_inst, batch.n_rows, world, rank)
        cl, ro = sh.local_problem(batch.clusters, batch.row_offsets, batch.n_rows, i0, ni)
        assert cl.shape[0] == nc and ro[0] == 0 and ro[-1] == nc
        o = Oracle.for_event(batch)
        res = o.track(cl, ro, ni)
        counts = np.zeros(16, np.int64)
        counts[1], counts[3] = len(res.cand_n), len(res.trk_cand)
        allc = sh.gather_counts(counts)
        assert allc.shape == (world, 16)
        ms, n = sh.combine_step(10.0 + rank, nc)
        assert ms == 10.0 + world - 1 and n == batch.n_clusters
        # the shard's owner array, shifted by the tracks of the lower ranks, is the slice of the whole-job result
        base = int(allc[:rank, 3].sum())
        own = np.where(res.cluster_owner >= 0, res.cluster_owner + base, -1)
        np.save(os.path.join(tmp, f"own{rank}.npy"), own)
        dist.barrier()
        if rank == 0:
            whole = o.track(batch.clusters, batch.row_offsets, batch.n_inst)
            got = np.concatenate([np.load(os.path.join(tmp, f"own{r}.npy")) for r in range(world)])
            assert np.array_equal(got, whole.cluster_owner)
            assert int(allc[:, 3].sum()) == len(whole.trk_cand) and int(allc[:, 1].sum()) == len(whole.cand_n)
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo(tmp_path):
    port = 29500 + (os.getpid() % 2000)
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)


def _strong_worker(rank, world, port, tmp):
    """bench.py's --scaling strong code path (shard_job -> track -> gather_counts / combine_step) with the oracle
    standing in for the per-rank GPU tracker."""
    import sys
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle.tpc_oracle import Oracle
        evs = [dg.drift_window(seed=5401 + i, mean_tracks=25.0 * (1 + i % 3), cap_tracks=120) for i in range(5)]
        batch = dg.concat_events(evs)
        my_evs, local, shard = bench.shard_job(evs, batch, world, rank)
        assert sum(e.n_clusters for e in my_evs) == local.n_clusters == shard["n_clusters"]
        assert local.n_inst == 36 * len(my_evs) and local.row_offsets[0] == 0
        assert np.array_equal(local.clusters, batch.clusters[shard["cluster0"]:shard["cluster0"] + shard["n_clusters"]])
        o = Oracle.for_event(batch)
        res = o.track(local.clusters, local.row_offsets, local.n_inst)
        counts = np.zeros(16, np.int64)
        counts[1], counts[3], counts[4] = len(res.cand_n), len(res.trk_cand), len(res.trk_hits)
        allc = sh.gather_counts(counts)
        ms, n = sh.combine_step(5.0 + 2 * rank, local.n_clusters)
        assert n == batch.n_clusters and ms == 5.0 + 2 * (world - 1)  # whole job over the slowest rank
        base = int(allc[:rank, 3].sum())
        np.save(os.path.join(tmp, f"sown{rank}.npy"), np.where(res.cluster_owner >= 0, res.cluster_owner + base, -1))
        dist.barrier()
        if rank == 0:
            whole = o.track(batch.clusters, batch.row_offsets, batch.n_inst)
            got = np.concatenate([np.load(os.path.join(tmp, f"sown{r}.npy")) for r in range(world)])
            assert np.array_equal(got, whole.cluster_owner)
            assert int(allc[:, 3].sum()) == len(whole.trk_cand) and int(allc[:, 4].sum()) == len(whole.trk_hits)
    finally:
        dist.destroy_process_group()


def test_bench_strong_scaling_path_world_size_2_gloo(tmp_path):
    port = 31500 + (os.getpid() % 2000)
    mp.spawn(_strong_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
