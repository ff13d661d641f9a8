"""Party-per-process online phase with a REAL exchange (world_size-2 gloo on CPU): rank b holds party
b's key only, runs paper_2606_09551_b200/two_party.run_party (the product's host loop) with the oracle as compute
backend, and the two ranks' outputs equal the single-process run of both parties."""
import importlib.util
import os

import numpy as np
import pytest
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


# ---- the CUDA path, party per process (-m gpu): two processes share the one GPU, gloo group, pinned-host staging -----------
def _cuda_setup(variant):
    import sys
    sys.path.insert(0, ROOT)
    from workloads import specs, tensors
    name = "gelu" if variant < 16 else "shift_relu"
    spec = specs.CONFIGS[name]()
    v = variant % 16
    if v & 1:
        spec = specs.shared_prefix(spec)
    if v & 2:
        spec = specs.input_masked_mul(spec)
    if v & 8:
        spec = specs.early_termination(spec)
    inp = tensors.inputs(name, spec, count=777, seed=6)
    return spec, inp


def _cuda_worker(rank, port, variant, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE="2")
    import sys
    sys.path.insert(0, ROOT)
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=2)
    import paper_2606_09551_b200 as F
    from paper_2606_09551_b200 import two_party as T
    spec, inp = _cuda_setup(variant)
    P = F.Program(spec)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.int64)).cuda()
    keys = P.keygen(dev(inp["r_in"]), dev(inp["r_out"]), 5)        # the dealer's output; this rank keeps ITS bundle only
    key = keys[rank].clone()
    del keys
    l0 = F.launch_count()
    y, z, sent = T.run_party_cuda(P, rank, key, dev(inp["xhat"]))
    torch.cuda.synchronize()
    out.put((rank, y.cpu().numpy().view(np.uint64), z.cpu().numpy().view(np.uint64), sent, F.launch_count() - l0))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.gpu
@pytest.mark.parametrize("variant", [0, 3, 9, 16])
def test_two_party_cuda(variant):
    """Each party in its own process with its own key bundle only, the library's kernels as compute backend, a real exchange of
    every round's opening buffer: both ranks' output shares equal the oracle's single-process run bit for bit, and the bytes
    sent equal the counted online message bytes."""
    import oracle
    assert torch.cuda.is_available()
    import __graft_entry__ as g
    g.build()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29900 + os.getpid() % 300 + variant
    procs = [ctx.Process(target=_cuda_worker, args=(r, port, variant, out)) for r in (0, 1)]
    for p in procs:
        p.start()
    got = dict((r, (y, z, s, l)) for r, y, z, s, l in (out.get(timeout=600), out.get(timeout=600)))
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    spec, inp = _cuda_setup(variant)
    O = oracle.Program(spec)
    k0, k1 = O.keygen(inp["r_in"], inp["r_out"], 5)
    exp = O.run_gate(k0, k1, inp["xhat"])
    na = O.shape["n_out_a"]
    for b in (0, 1):
        assert np.array_equal(got[b][0][:na], exp["y"][b]), (variant, b)
        if O.shape["n_out_b"]:
            assert np.array_equal(got[b][1], exp["z"][b]), (variant, b)
        assert got[b][2] == O.msg_total(inp["xhat"].size)
        assert got[b][3] > 0                                            # the library's kernels ran in that process
