"""Party-per-process online phase with a REAL exchange (world_size-2 gloo on CPU): rank b holds party
b's key only, runs paper_2606_09551_b200/two_party.run_party (the product's host loop) with the oracle as compute
backend, and the two ranks' outputs equal the single-process run of both parties."""
import importlib.util
import os

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _two_party():
    spec = importlib.util.spec_from_file_location("ffs_two_party", os.path.join(ROOT, "paper_2606_09551_b200", "two_party.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def _setup(variant):
    import sys
    sys.path.insert(0, ROOT)
    import oracle
    from workloads import specs, tensors
    spec = specs.toy(12, 4)
    if variant & 1:
        spec = specs.shared_prefix(spec)
    if variant & 2:
        spec = specs.input_masked_mul(spec)
    P = oracle.Program(spec)
    rng = np.random.default_rng(4)
    count = 70
    x = rng.integers(0, 1 << 12, count, dtype=np.uint64)
    r_in = rng.integers(0, 1 << 12, count, dtype=np.uint64)
    r_out = rng.integers(0, 1 << 12, 2 * count, dtype=np.uint64).reshape(2, count)
    keys = P.keygen(r_in, r_out, 5)
    return P, keys, (x + r_in) & np.uint64(4095)


def _worker(rank, port, variant, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE="2")
    dist.init_process_group("gloo", rank=rank, world_size=2)
    T = _two_party()
    P, keys, xhat = _setup(variant)
    y, z, sent = T.run_party(P, rank, keys[rank], xhat,
                             to_tensor=lambda a: torch.from_numpy(a),
                             from_tensor=lambda t, a: t.numpy(),
                             new_msg=lambda nb: np.zeros(nb, np.uint8))
    out.put((rank, np.array(y), np.array(z), sent))
    dist.barrier()
    dist.destroy_process_group()


def _run(variant):
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29600 + os.getpid() % 300 + variant
    procs = [ctx.Process(target=_worker, args=(r, port, variant, out)) for r in (0, 1)]
    for p in procs:
        p.start()
    got = dict((r, (y, z, s)) for r, y, z, s in (out.get(timeout=180), out.get(timeout=180)))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    P, keys, xhat = _setup(variant)
    exp = P.run_gate(keys[0], keys[1], xhat)
    for b in (0, 1):
        assert np.array_equal(got[b][0], exp["y"][b]) and np.array_equal(got[b][1], exp["z"][b])
        assert got[b][2] == P.msg_total(xhat.size)                      # bytes actually sent = counted online message bytes


def test_two_party_exchange_variant0():
    _run(0)


def test_two_party_exchange_variant3():
    _run(3)
