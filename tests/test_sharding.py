"""Multi-rank path on CPU (gloo, world_size 2): every rank generates ITS slice of the seeded
workload, evaluates it (here with the oracle, standing in for its GPU), and the gathered
result must equal the single-process evaluation of the whole workload -- i.e. the slicing
and the counter-based generator are consistent, and no rank needs another rank's data."""
import os
import socket

import numpy as np
import pytest

from paper_2502_07060_b200 import inputs, sharding


def test_slices_partition_the_batch():
    for total in (0, 1, 7, 64, 1000):
        for world in (1, 2, 3, 8):
            got = [sharding.strong_slice(r, world, total) for r in range(world)]
            assert got[0][0] == 0 and sum(c for _, c in got) == total
            for (s0, c0), (s1, _) in zip(got, got[1:]):
                assert s1 == s0 + c0
            assert max(c for _, c in got) - min(c for _, c in got) <= 1
    assert sharding.weak_slice(3, 4, 100) == (300, 100)
    with pytest.raises(ValueError):
        sharding.weak_slice(2, 2, 10)


def test_generator_slices_are_independent():
    whole = inputs.make_fp_inputs(6, 5, 96, seed=4)
    for start, count in [(0, 40), (40, 56)]:
        part = inputs.make_fp_inputs(6, 5, count, seed=4, start=start)
        assert np.array_equal(part[0], whole[0][start:start + count])
        assert np.array_equal(part[1], whole[1][start:start + count])


def _worker(rank, world, port, mode, q):
    import torch
    import torch.distributed as dist
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        if mode == "weak":
            start, count = sharding.weak_slice(rank, world, 50)
        else:
            start, count = sharding.strong_slice(rank, world, 101)
        mom, pol, _ = inputs.make_fp_inputs(7, 5, count, seed=9, start=start)
        out = oracle.amplitudes(oracle.FP31, mom, pol, threads=1).astype(np.int64)
        # the only communication: gathering results (and the timing max in bench.py)
        sizes = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
        dist.all_gather(sizes, torch.tensor([count]))
        mx = int(max(s.item() for s in sizes))
        pad = torch.zeros(mx, dtype=torch.int64)
        pad[:count] = torch.from_numpy(out)
        bufs = [torch.zeros(mx, dtype=torch.int64) for _ in range(world)]
        dist.all_gather(bufs, pad)
        t = torch.tensor([float(rank + 1)], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)        # bench.py's max-over-ranks timing
        if rank == 0:
            full = np.concatenate([b.numpy()[:int(s.item())] for b, s in zip(bufs, sizes)])
            q.put((full, float(t.item())))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("mode", ["weak", "strong"])
def test_two_ranks_reproduce_the_whole_batch(oracle_mod, mode):
    import torch.multiprocessing as mp
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, mode, q)) for r in range(2)]
    for p in procs:
        p.start()
    full, tmax = q.get(timeout=120)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    total = 100 if mode == "weak" else 101
    mom, pol, _ = inputs.make_fp_inputs(7, 5, total, seed=9)
    ref = oracle_mod.amplitudes(oracle_mod.FP31, mom, pol, threads=2).astype(np.int64)
    assert np.array_equal(full, ref)
    assert tmax == 2.0
