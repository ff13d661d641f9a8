"""Party-per-process online phase (the paper's own layout: one GPU per party).

Rank b of a 2-rank `torch.distributed` group plays party b: it holds ITS key bundle only, evaluates the two FSS calls
locally (no interaction) and runs the post-processing rounds through the per-round C-ABI call `fusefss_post`,
exchanging each round's opening buffer with its peer: NCCL send/recv of the device buffers over NVLink when the two ranks own
two GPUs, or -- two processes sharing ONE GPU, gloo group -- staged through pinned host memory.
Host logic only -- `prog` is any object with the Program interface (eval_cmp / eval_lut / post / post_rounds /
post_msg_bytes / shape): the library's Program on GPUs (tests/test_two_party.py::test_two_party_cuda, bench.py --two-party),
the oracle's in the CPU-only gloo tests.
"""
from __future__ import annotations


def exchange(mine, peer: int, rank: int):
    """Swap one message buffer with the peer (the lower rank sends first); returns the peer's buffer, on mine's device.
    A CUDA buffer over a gloo group is staged through pinned host memory."""
    import torch
    import torch.distributed as dist
    staged = mine.is_cuda and dist.get_backend() != "nccl"
    out = torch.empty(mine.shape, dtype=mine.dtype, pin_memory=True) if staged else mine
    if staged:
        out.copy_(mine, non_blocking=False)
    theirs = torch.empty_like(out)
    if rank < peer:
        dist.send(out, dst=peer)
        dist.recv(theirs, src=peer)
    else:
        dist.recv(theirs, src=peer)
        dist.send(out, dst=peer)
    return theirs.to(mine.device, non_blocking=False) if staged else theirs


def run_party(prog, party: int, key, xhat, to_tensor, from_tensor, new_msg):
    """Online phase of one party.  to_tensor / from_tensor convert a message buffer to / from a torch tensor for the
    exchange; new_msg(nbytes) allocates a zeroed message buffer of the backend's kind.  Returns (y, z, bytes_sent)."""
    bits = prog.eval_cmp(party, key, xhat) if prog.shape["T"] else None
    coeff = prog.eval_lut(party, key, xhat) if prog.shape["has_lut"] else None
    count = int(xhat.numel() if hasattr(xhat, "numel") else xhat.size)
    rounds = prog.post_rounds()
    sizes = [prog.post_msg_bytes(count, q) for q in range(rounds)]
    total = max(1, sum(sizes))
    mine, theirs = new_msg(total), new_msg(total)
    sent, off = 0, 0
    for q in range(rounds):
        prog.post(party, key, xhat, bits, coeff, q, theirs, mine)           # writes this party's openings of round q
        if sizes[q]:
            seg = to_tensor(mine)[off:off + sizes[q]].contiguous()
            got = exchange(seg, 1 - party, party)
            t = to_tensor(theirs)
            t[off:off + sizes[q]] = got
            theirs = from_tensor(t, theirs)
            sent += sizes[q]
        off += sizes[q]
    y, z = prog.post(party, key, xhat, bits, coeff, rounds, theirs, mine)
    return y, z, sent


def run_party_cuda(prog, party: int, key, xhat):
    """run_party for the library's Program: message buffers are CUDA uint8 tensors."""
    import torch
    return run_party(prog, party, key, xhat, to_tensor=lambda t: t, from_tensor=lambda t, old: t,
                     new_msg=lambda nb: torch.zeros(max(256, nb), dtype=torch.uint8, device="cuda"))


def bench(F, torch, dist, args, rank, world, M):
    """bench.py --two-party (N = 2, one GPU per party): both ranks derive the key pair from the same dealer seed, rank b
    keeps party b's bundle; timed = the online phase (this party's FSS calls + the post-processing rounds with a real NCCL
    exchange of every round's opening buffer), max over the two ranks."""
    import numpy as np
    from workloads import specs, tensors
    if world != 2:
        return {"two_party": "needs exactly 2 ranks (one GPU per party)", "n_gpus": world}
    name = args.workload
    spec = specs.CONFIGS[name]()
    v = args.variant
    if v & 1:
        spec = specs.shared_prefix(spec)
    if v & 2:
        spec = specs.input_masked_mul(spec)
    if v & 4:
        spec = specs.public_point_horner(spec)
    if v & 8:
        spec = specs.early_termination(spec)
    P = F.Program(spec)
    count = args.count or min(tensors.FULL_COUNT[name], 1 << 20)
    free_b, _ = torch.cuda.mem_get_info()
    while 2 * P.key_bytes(count) > 0.8 * free_b:
        count //= 2
    inp = tensors.inputs(name, spec, count=count, seed=0)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.int64)).cuda()
    keys = P.keygen(dev(inp["r_in"]), dev(inp["r_out"]), 0)
    key = keys[rank]
    del keys
    xhat = dev(inp["xhat"])
    ev = lambda: torch.cuda.Event(enable_timing=True)
    for _ in range(args.warmup):
        run_party_cuda(P, rank, key, xhat)
    torch.cuda.synchronize(); dist.barrier(); torch.cuda.synchronize()
    a, b = ev(), ev()
    a.record()
    for _ in range(args.steps):
        y, z, sent = run_party_cuda(P, rank, key, xhat)
    b.record()
    torch.cuda.synchronize(); dist.barrier(); torch.cuda.synchronize()
    nccl = dist.get_backend() == "nccl"
    t = torch.tensor([a.elapsed_time(b)], device="cuda" if nccl else "cpu", dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms = float(t.item()) / args.steps
    # reconstruct on rank 0: the two parties' output shares must add up to the plaintext gate (the check a user of the online phase would make)
    y_other = exchange(y.contiguous(), 1 - rank, rank)
    mask = (1 << spec.n) - 1
    rec = y[0] + y_other[0]
    if spec.n < 64:
        rec = rec & mask
    checksum = int((rec & 0xFFFFFFFF).sum().item()) & 0xFFFFFFFF
    how = "NCCL send/recv of the device buffers" if nccl else "gloo, staged through pinned host memory (two processes; a stand-in for NVLink when both ranks share one GPU)"
    return {"metric": "online elements/s, one process per party (FSS calls + post-processing rounds with a real exchange: %s)" % how, "value": count / (ms * 1e-3),
            "unit": "elements/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "two-party", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
            "config": {"workload": f"{name} n={spec.n} f={spec.f} count={count}", "construction": f"variant {v}", "parallelism": "party b on GPU b, send/recv of the opening buffers"},
            "online_bytes_sent_per_party_per_step": sent, "rounds": P.post_rounds(), "exchange": how,
            "output_checksum": {"value": checksum, "what": "sum over elements of (y0 + y1 mod 2^n) mod 2^32, y1 received from the peer"}}
