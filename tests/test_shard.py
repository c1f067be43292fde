"""Host logic of the multi-GPU form of the path ("each of N ranks traces 1/N of the
rays, results added at the end"): ray-index shares are disjoint and cover the range; the gather/add of the monitor
arrays is one sum-reduce.  Runs with the gloo backend, world_size 2, on CPU; the per-rank tallies come from the
oracle (rays are keyed by index, so two shares summed must equal one run over the whole range)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2410_08747_b200.shard import ray_range, reduce_tallies


def test_ray_range_strong_partitions_exactly():
    for n in (0, 1, 7, 1000, 10**9 + 7):
        for world in (1, 2, 3, 8):
            spans = [ray_range(r, world, n, "strong") for r in range(world)]
            assert spans[0][0] == 0 and sum(c for _, c in spans) == n
            for (f0, c0), (f1, _) in zip(spans, spans[1:]):
                assert f0 + c0 == f1                                  # contiguous, disjoint
            assert max(c for _, c in spans) - min(c for _, c in spans) <= 1


def test_ray_range_weak_windows_are_disjoint():
    spans = [ray_range(r, 4, 1000, "weak") for r in range(4)]
    assert spans == [(0, 1000), (1000, 1000), (2000, 1000), (3000, 1000)]
    with pytest.raises(ValueError):
        ray_range(4, 4, 10)
    with pytest.raises(ValueError):
        ray_range(0, 2, 10, "sideways")


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_total, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import workloads as W
    from oracle import oracle as O
    inst = W.config0()
    first, count = ray_range(rank, world, n_total, "strong")
    o = O.trace(inst, first=first, n=count)
    t = [torch.from_numpy(o["N"][0].astype(np.int64)), torch.from_numpy(o["P"][0].copy()), torch.from_numpy(o["P2"][0].copy())]
    reduce_tallies(t)                                                 # all-reduce: every rank ends with the sum
    if rank == 0:
        q.put([x.numpy() for x in t])
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_shares_sum_to_the_whole_run_gloo():
    import workloads as W
    from oracle import oracle as O
    n_total = 40_001
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, n_total, q)) for r in range(2)]
    for p in procs:
        p.start()
    N, P, P2 = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    whole = O.trace(W.config0(), first=0, n=n_total)
    assert np.array_equal(N.astype(np.uint64), whole["N"][0])        # integer counts exact
    assert np.allclose(P, whole["P"][0], rtol=1e-13, atol=0) and np.allclose(P2, whole["P2"][0], rtol=1e-13, atol=0)
    assert int(N.sum()) == whole["detected"]
