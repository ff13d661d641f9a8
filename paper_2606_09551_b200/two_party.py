"""Party-per-process online phase (the paper's own layout: one GPU per party).

Rank b of a 2-rank `torch.distributed` group plays party b: it holds ITS key bundle only, evaluates the two FSS calls
locally (no interaction) and runs the post-processing rounds through the per-round C-ABI call `fusefss_post`,
exchanging each round's opening buffer with its peer (NCCL over NVLink on two GPUs; gloo in the CPU test).
Host logic only -- `prog` is any object with the Program interface (eval_cmp / eval_lut / post / post_rounds /
post_msg_bytes / shape); the library's Program on GPUs, the oracle's in tests/test_two_party.py.
"""
from __future__ import annotations


def exchange(mine, peer: int, rank: int):
    """Swap one message buffer with the peer (the lower rank sends first); returns the peer's buffer."""
    import torch
    import torch.distributed as dist
    theirs = torch.empty_like(mine)
    if rank < peer:
        dist.send(mine, dst=peer)
        dist.recv(theirs, src=peer)
    else:
        dist.recv(theirs, src=peer)
        dist.send(mine, dst=peer)
    return theirs


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
