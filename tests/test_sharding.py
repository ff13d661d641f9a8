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


# ---- the N > 1 paths of bench.py on ONE GPU: two processes over gloo (NCCL refuses two ranks on one device) ------------------------------
def _bench_line(extra, nproc=1, port=0):
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    common = ["--workload", "gelu", "--count", "65536", "--steps", "2", "--warmup", "3", "--no-cpu", "--no-e2e", "--no-sp", "--no-configs", "--no-probes"]
    if nproc == 1:
        cmd = [sys.executable, os.path.join(root, "bench.py"), "--gpus", "1"] + common + extra
    else:
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(nproc), "--master-addr", "127.0.0.1",
               "--master-port", str(port), os.path.join(root, "bench.py"), "--gpus", str(nproc), "--backend", "gloo", "--same-gpu"] + common + extra
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=900, cwd=root)
    assert out.returncode == 0, out.stderr[-3000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout[-2000:]
    return json.loads(lines[0])


@pytest.mark.gpu
def test_bench_multi_rank_paths_on_one_gpu():
    """bench.py's strong-scaling, replica and party-per-process legs have only ever had one GPU to run on.  Two processes sharing cuda:0 over a
    gloo group run the same code (sharding.shard_range, max-over-ranks timing, the per-round exchange of two_party.run_party); the outputs they
    leave must reconstruct to the same values as the one-process run: equal 32-bit checksums of y0 + y1."""
    one = _bench_line([])
    ref = one["output_checksum"]["value"]
    strong = _bench_line(["--scaling", "strong"], nproc=2, port=29731)
    assert strong["n_gpus"] == 2 and strong["scaling"] == "strong" and "gloo" in strong["config"]["backend"]
    assert strong["output_checksum"]["value"] == ref
    weak = _bench_line([], nproc=2, port=29732)
    assert weak["scaling"] == "weak" and weak["output_checksum"]["value"] == ref          # rank 0's replica = the one-process tensor (seed 0)
    assert weak["strong_scaling_leg"]["output_checksum"] == ref and weak["strong_scaling_leg"]["value"] > 0
    two = _bench_line(["--two-party"], nproc=2, port=29733)
    assert two["scaling"] == "two-party" and two["rounds"] >= 1 and two["online_bytes_sent_per_party_per_step"] > 0
    assert two["output_checksum"]["value"] == ref
