"""N > 1 host logic (replicas only: DESIGN.md §1) on CPU with the gloo backend, world_size 2.

The data path has no collective; what crosses ranks is bookkeeping: shard bounds, per-rank seeds, max-over-ranks timing, summed unit
counts and the summed basin histogram.  Nothing here touches the CUDA library or the oracle."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2508_15522_b200 import inputs, shard


def test_replica_shard_partitions_exactly():
    for n_total in (0, 1, 7, 64, 4096, 16384, 8191):
        for world in (1, 2, 3, 4, 8):
            spans = [shard.replica_shard(n_total, world, r) for r in range(world)]
            assert spans[0][0] == 0 and sum(c for _, c in spans) == n_total
            for (f0, c0), (f1, _) in zip(spans, spans[1:]):
                assert f0 + c0 == f1
            counts = [c for _, c in spans]
            assert max(counts) - min(counts) <= 1
    with pytest.raises(ValueError):
        shard.replica_shard(10, 2, 2)


def test_rank_seeds_are_distinct_and_batches_differ():
    seeds = {shard.rank_seed(1001, r, s) for r in range(8) for s in (0, 10, 11)}
    assert len(seeds) == 24
    topo = inputs.benzene()
    a = inputs.place_replicas(topo, 4, 11.28, 11.28, 0.0, shard.rank_seed(1000, 0, 10))
    b = inputs.place_replicas(topo, 4, 11.28, 11.28, 0.0, shard.rank_seed(1000, 1, 10))
    assert a.shape == b.shape and np.abs(a - b).max() > 0.1
    assert np.array_equal(a, inputs.place_replicas(topo, 4, 11.28, 11.28, 0.0, shard.rank_seed(1000, 0, 10)))


def test_basin_histogram_counts():
    e = np.array([-1.234, -1.226, -1.2251, -0.5, 7.0, -9.0, np.nan])
    h = shard.basin_histogram(e, -2.0, 0.0, 0.01)
    assert h.shape == (200,) and h.sum() == 6 and h.dtype == np.int64
    assert h[76] == 1 and h[77] == 2 and h[150] == 1 and h[199] == 1 and h[0] == 1


def test_single_process_reductions_are_identity():
    assert shard.max_over_ranks(3.5) == 3.5
    assert np.array_equal(shard.sum_over_ranks(np.array([1, 2, 3])), np.array([1, 2, 3]))
    v, ms = shard.aggregate_throughput(1000.0, 500.0)
    assert v == 2000.0 and ms == 500.0


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # strong-scaling shard of config 0's 64 replicas: each rank takes its slice of one seeded batch
        cfg = inputs.config(0)
        first, count = shard.replica_shard(cfg["n_rep"], world, rank)
        mine = cfg["pos"][first:first + count]
        # stand-in "relaxed energies": a deterministic function of the slice (no method arithmetic)
        energies = -1.0 - 0.001 * np.arange(first, first + count)
        hist = shard.sum_over_ranks(shard.basin_histogram(energies, -1.1, -0.9, 0.01))
        units = shard.sum_over_ranks(np.array([count * 1000], np.int64))
        ms = shard.max_over_ranks(10.0 + 5.0 * rank)
        value, ms2 = shard.aggregate_throughput(count * 1000, 10.0 + 5.0 * rank)
        checksum = shard.sum_over_ranks(np.array([float(np.sum(mine, dtype=np.float64))]))
        dist.barrier()
        np.savez(os.path.join(out_dir, "rank%d.npz" % rank), hist=hist, units=units, ms=ms, value=value, ms2=ms2, checksum=checksum,
                 first=first, count=count)
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    r = [np.load(tmp_path / ("rank%d.npz" % k)) for k in range(world)]
    cfg = inputs.config(0)
    # both ranks hold the same reduced values
    for key in ("hist", "units", "ms", "value", "ms2", "checksum"):
        assert np.array_equal(r[0][key], r[1][key]), key
    assert int(r[0]["first"]) == 0 and int(r[1]["first"]) == 32 and int(r[0]["count"]) + int(r[1]["count"]) == cfg["n_rep"]
    assert int(r[0]["units"][0]) == 64000
    assert float(r[0]["ms"]) == 15.0 and float(r[0]["ms2"]) == 15.0                 # max over ranks
    assert abs(float(r[0]["value"]) - 64000 / 15e-3) < 1e-6
    single = shard.basin_histogram(-1.0 - 0.001 * np.arange(64), -1.1, -0.9, 0.01)   # the unsharded histogram
    assert np.array_equal(r[0]["hist"], single) and single.sum() == 64
    assert abs(float(r[0]["checksum"][0]) - float(np.sum(cfg["pos"], dtype=np.float64))) < 1e-6
