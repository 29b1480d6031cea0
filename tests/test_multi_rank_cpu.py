"""The N > 1 path of bench.py on CPU: two processes over gloo (channels shard with no
data-path collective; only the step time (max) and the work counters (sum) are reduced).  The oracle stands in for
the GPU library on each rank: a channel table split over two ranks, each keyed by its global channel offset, reproduces
the single-process run bit for bit -- the partition-independence that makes replicas over channel ranges correct."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _worker(rank, world, port, tmp):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import oracle
    from paper_2110_15640_b200 import workloads as wl
    grid, opac, prm = wl.cfg2(nlon=8, nlat=4, nlev=10, nbands=1, ng=4, packets=2000)
    n_per = 2                                              # channels per rank
    c0 = bench.rank_chan0(rank, n_per)
    mine = {k: (v[c0:c0 + n_per] if isinstance(v, np.ndarray) and v.shape[:1] == (4,) else v) for k, v in opac.items()}
    mine["chan0"] = c0
    res = oracle.run_albedo(grid, mine, prm, want_event_count=True)
    np.save(os.path.join(tmp, "flux_%d.npy" % rank), res["flux_sum"])
    np.save(os.path.join(tmp, "evc_%d.npy" % rank), res["event_count"])
    ms, (events,) = bench.reduce_over_ranks(10.0 + 5.0 * rank, [res["counters"]["events"]], world)
    if rank == 0:
        np.save(os.path.join(tmp, "reduced.npy"), np.array([ms, events]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_shard_channels_and_reduce_over_gloo(tmp_path):
    import torch.multiprocessing as mp
    import oracle
    from paper_2110_15640_b200 import workloads as wl
    port = 29600 + os.getpid() % 300
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    grid, opac, prm = wl.cfg2(nlon=8, nlat=4, nlev=10, nbands=1, ng=4, packets=2000)
    full = oracle.run_albedo(grid, opac, prm, want_event_count=True)
    flux = np.concatenate([np.load(tmp_path / "flux_0.npy"), np.load(tmp_path / "flux_1.npy")], axis=0)
    evc = np.concatenate([np.load(tmp_path / "evc_0.npy"), np.load(tmp_path / "evc_1.npy")], axis=0)
    assert np.array_equal(flux, full["flux_sum"]) and np.array_equal(evc, full["event_count"])
    ms, events = np.load(tmp_path / "reduced.npy")
    assert ms == 15.0                                      # max over ranks
    assert events == full["counters"]["events"]            # sum over ranks


def test_single_rank_reduce_is_identity():
    import bench
    assert bench.reduce_over_ranks(3.5, [1, 2], 1) == (3.5, [1.0, 2.0])
    assert bench.rank_chan0(3, 176) == 528
