"""N > 1 host logic with world_size-2 gloo on CPU: the element ranges partition the
tensor, chunk boundaries are warp-tile aligned, and the timing reduction is a max over ranks."""
import importlib.util
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _sharding():
    # load the module by path: importing the package would need libfusefss.so, which these tests do not
    spec = importlib.util.spec_from_file_location("ffs_sharding", os.path.join(ROOT, "paper_2606_09551_b200", "sharding.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def test_shard_ranges_partition():
    S = _sharding()
    for total in (1, 31, 32, 33, 4096, 393216, 22544384, 1000003):
        for world in (1, 2, 3, 8):
            pos = 0
            for r in range(world):
                first, n = S.shard_range(total, r, world)
                assert first == pos and n >= 0
                assert first % 32 == 0 or first == total
                pos += n
            assert pos == total
    with pytest.raises(ValueError):
        S.shard_range(10, 2, 2)


def _worker(rank, world, port, total, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    S = _sharding()
    first, n = S.shard_range(total, rank, world)
    mine = torch.tensor([first, n], dtype=torch.int64)
    got = [torch.zeros(2, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(got, mine)
    t = S.max_over_ranks(10.0 + rank)                       # "device time" of this rank
    if rank == 0:
        out.put(([g.tolist() for g in got], t))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    total, world, port = 393216 + 17, 2, 29517 + os.getpid() % 1000
    procs = [ctx.Process(target=_worker, args=(r, world, port, total, out)) for r in range(world)]
    for p in procs:
        p.start()
    ranges, tmax = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert ranges[0][0] == 0 and ranges[0][0] + ranges[0][1] == ranges[1][0]
    assert ranges[1][0] + ranges[1][1] == total and ranges[1][0] % 32 == 0
    assert tmax == 11.0
