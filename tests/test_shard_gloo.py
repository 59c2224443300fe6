"""The N > 1 path on CPU: two gloo ranks shard a photon-id range, each produces the tallies of its shard, one
all-reduce sums them, and the sum equals the one-rank tallies bit for bit.  The per-shard tallies come from the oracle
here (test infrastructure; there is no GPU in this container) — what is under test is the host logic the GPU path uses
unchanged: shard_range + allreduce_tallies + photon_id_offset semantics."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2507_11603_b200 import shard
from paper_2507_11603_b200 import workloads as W


def test_shard_range_partitions_exactly():
    for n in (0, 1, 7, 1000, 10**6 + 3):
        for world in (1, 2, 3, 8):
            ranges = [shard.shard_range(n, r, world) for r in range(world)]
            assert ranges[0][0] == 0 and sum(c for _, c in ranges) == n
            for (o0, c0), (o1, _) in zip(ranges, ranges[1:]):
                assert o0 + c0 == o1
            assert max(c for _, c in ranges) - min(c for _, c in ranges) <= 1
    with pytest.raises(ValueError):
        shard.shard_range(10, 2, 2)


def _worker(rank, world, port, n, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import thor_oracle
        w = W.static_sphere(n=16, tau0=30.0, T=1e4, n_photons=n)
        off, cnt = shard.shard_range(n, rank, world)
        r = thor_oracle.run(w["grid"], w["sources"], dict(w["opts"], photon_id_offset=off), cnt, w["seed"])
        spec = torch.from_numpy(r["spectrum"].astype(np.int64))
        hist = torch.from_numpy(r["nscat_hist"].astype(np.int64))
        cnts = torch.tensor([r["counters"][k] for k in thor_oracle.COUNTER_NAMES], dtype=torch.int64)
        shard.allreduce_tallies([spec, hist, cnts])
        if rank == 0:
            torch.save(dict(spec=spec, hist=hist, cnts=cnts), out)
    finally:
        dist.destroy_process_group()


def test_two_rank_shards_sum_to_the_single_rank_run(tmp_path, oracle):
    n, world = 3001, 2
    out = str(tmp_path / "sum.pt")
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(world, port, n, out), nprocs=world, join=True)
    got = torch.load(out)
    w = W.static_sphere(n=16, tau0=30.0, T=1e4, n_photons=n)
    ref = oracle.run(w["grid"], w["sources"], w["opts"], n, w["seed"])
    assert np.array_equal(got["spec"].numpy(), ref["spectrum"].astype(np.int64))
    assert np.array_equal(got["hist"].numpy(), ref["nscat_hist"].astype(np.int64))
    assert [int(v) for v in got["cnts"]] == [ref["counters"][k] for k in oracle.COUNTER_NAMES]
    assert int(got["cnts"][0]) + int(got["cnts"][1]) + int(got["cnts"][2]) + int(got["cnts"][3]) == n
