"""fusefss_post_fused_noalloc: the fused post-processing pass for hosts of this library that must not allocate device memory.

Who that is: an inference server whose own allocator has already claimed almost all of HBM (a cudaMalloc from a library then
fails or breaks the server's accounting), an online two-party loop that cannot absorb the device-wide synchronisation a
first-use cudaMalloc causes, a party process held to a device-memory quota fixed in advance.  For them the interpreter's
instruction table sits in a 48 KB array inside the library image (FUSEFSS_NOALLOC_MAX_INS = 2048 instructions, one array per
GPU, shared by every call) instead of a buffer malloc'ed on first use; longer programs are refused with FUSEFSS_E_STATIC.

What is checked here: the new entry point writes exactly the shares fusefss_post_fused writes -- integer ring arithmetic, so
the bar is bit-exact, as everywhere in tests/ -- on two calls in a row, on a second program that overwrites the shared table in
between, and on a program close to the size limit; and the limit itself.  All calls run on one stream: overlapping calls would
race on the table, which the header documents.

The file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first failure and a problem here must not
hide the parity tests.  It builds its own inputs and keeps no state, so it passes alone in a fresh process as well as after
the rest of the suite."""
import dataclasses
import os

import numpy as np
import pytest

from helpers import mask_of
from workloads import specs, tensors

E_COUNT, E_STATIC, MAX_INS = -4, -10, 2048


def _long_phi(k):
    """plain_default with a Phi of k + 5 nodes: acc = y_0, then k times acc += y_0 (so the output is (k + 1) y_0), plus the
    predicate bit passed through.  k picks the length of the lowered program; no method arithmetic lives here."""
    s = specs.plain_default(8, 3)
    phi = [(specs.PHI_A_Y, 0, 0, 0, 0), (specs.PHI_A_Y, 1, 0, 0, 0)]
    acc = 1
    for i in range(k):
        nxt = 1 + (i + 1) % 2
        phi.append((specs.PHI_A_ADD, nxt, acc, 0, 0))
        acc = nxt
    phi += [(specs.PHI_A_OUT, 0, acc, 0, 0), (specs.PHI_B_Z, 0, 0, 0, 0), (specs.PHI_B_OUT, 0, 0, 0, 0)]
    return dataclasses.replace(s, name=f"long_phi_{k}", phi=phi, n_out_a=1, n_out_b=1)


def test_size_limit_needs_no_gpu():
    """The limit is checked on the host before any CUDA call and before `count`, so count = 0 probes it: a program that fits
    answers E_COUNT, one that does not answers E_STATIC with a message that names the limit.  (Dummy non-null pointers: the call
    returns before it would touch them.)"""
    import __graft_entry__ as g
    g.build()
    import paper_2606_09551_b200 as F
    probe = lambda P: F.lib.fusefss_post_fused_noalloc(P._h, 1, 1, 1, None, None, None, None, 0, None, None, None, None, None)
    assert probe(F.Program(specs.gelu())) == E_COUNT
    assert probe(F.Program(_long_phi(MAX_INS - 100))) == E_COUNT
    too_long = F.Program(_long_phi(MAX_INS + 50))
    assert probe(too_long) == E_STATIC
    header = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "fusefss.h")
    assert f"#define FUSEFSS_NOALLOC_MAX_INS {MAX_INS}" in open(header).read()
    assert b"FUSEFSS_NOALLOC_MAX_INS" in F.lib.fusefss_strerror(E_STATIC)
    assert F.lib.fusefss_post_fused_noalloc(None, 1, 1, 1, None, None, None, None, 8, None, None, None, None, None) == -1


@pytest.fixture(scope="module")
def F():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; the product has no CPU fallback"
    import __graft_entry__ as g
    g.build()
    import paper_2606_09551_b200 as F
    return F


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int64)).cuda()


def _host(t):
    return t.cpu().numpy().view(np.uint64).copy()


class _Case:
    """One gate instance on the device: keys, both parties' FSS outputs and the EXISTING path's post-processing result."""

    def __init__(self, F, spec, count, seed):
        import torch
        rng = np.random.default_rng(seed)
        m = mask_of(spec.n)
        u = lambda k: (rng.integers(0, 1 << 63, size=k, dtype=np.uint64) * np.uint64(2) + rng.integers(0, 2, size=k, dtype=np.uint64)) & m
        self.P = P = F.Program(spec)
        self.count, self.na = count, max(1, P.shape["n_out_a"])
        x, r_in, r_out = u(count), u(count), u(self.na * count).reshape(self.na, count)
        self.xhat = _dev((x + r_in) & m)
        self.k0, self.k1 = P.keygen(_dev(r_in), _dev(r_out), seed=seed + 11)
        self.bits, self.coeff = P.eval_fused_both(self.k0, self.k1, self.xhat)
        ref = P.post_fused(self.k0, self.k1, self.xhat, self.bits[0], self.bits[1], self.coeff[0], self.coeff[1])
        torch.cuda.synchronize()
        self.ref = [_host(t) for t in ref]
        self.has_z = P.shape["n_out_b"] > 0

    def noalloc(self):
        """one call of the new entry point into poisoned output tensors (a kernel that wrote nothing cannot pass)"""
        import torch
        outs = [torch.full((self.na, self.count), -0x0123456789ABCDEF, dtype=torch.int64, device="cuda") for _ in (0, 1)]
        outs += [torch.full((self.count,), -0x0123456789ABCDEF, dtype=torch.int64, device="cuda") for _ in (0, 1)]
        self.P.post_fused_noalloc(self.k0, self.k1, self.xhat, self.bits[0], self.bits[1], self.coeff[0], self.coeff[1], outs)
        return outs

    def check(self, outs, what):
        import torch
        torch.cuda.synchronize()
        n_a = self.P.shape["n_out_a"]
        for b in (0, 1):
            assert np.array_equal(_host(outs[b])[:n_a], self.ref[b][:n_a]), f"{self.P.spec.name}: y{b} differs ({what})"
            if self.has_z:
                assert np.array_equal(_host(outs[2 + b]), self.ref[2 + b]), f"{self.P.spec.name}: z{b} differs ({what})"


CASES = [
    ("gelu", specs.gelu, 1000),                                            # Protocol 3, Beaver products, ragged tail
    ("gelu_sp", lambda: specs.shared_prefix(specs.gelu()), 777),            # single-key construction
    ("toy_masked", lambda: specs.toy(8, 3, True), 300),                     # AND / B2A / kappa, masked outputs
    ("a2b64", lambda: specs.a2b_demo(64, 12), 70),                          # interactive A2B: the shared-memory instantiation
    ("long_phi", lambda: _long_phi(MAX_INS - 100), 257),                    # a table close to the 48 KB limit
]


@pytest.mark.gpu
@pytest.mark.parametrize("name,mk,count", CASES, ids=[c[0] for c in CASES])
def test_noalloc_matches_post_fused_twice(F, name, mk, count):
    """Two calls in a row on the same stream, each compared with fusefss_post_fused bit for bit."""
    c = _Case(F, mk(), count, seed=5)
    first = c.noalloc()
    second = c.noalloc()                                  # issued before the first is checked: back to back on the stream
    c.check(first, "first call")
    c.check(second, "second call")


@pytest.mark.gpu
def test_noalloc_table_is_rewritten_per_call(F):
    """The table keeps the previous call's program.  A long program, then a short one, then the long one again, all queued on one
    stream without a host wait in between: every call must have run its OWN program."""
    a = _Case(F, _long_phi(1500), 513, seed=1)
    b = _Case(F, specs.relu(16, 8), 2048, seed=2)
    c = _Case(F, specs.toy(8, 3), 100, seed=3)
    outs = [(a, a.noalloc()), (b, b.noalloc()), (c, c.noalloc()), (a, a.noalloc()), (b, b.noalloc())]
    for i, (case, o) in enumerate(outs):
        case.check(o, f"call {i} of the interleaved sequence")


@pytest.mark.gpu
def test_noalloc_rejects_and_keeps_working(F):
    """An over-long program is refused with a clear error on the GPU box too, and the refusal leaves the table usable."""
    with pytest.raises(F.FuseFSSError, match="FUSEFSS_NOALLOC_MAX_INS"):
        big = _Case.__new__(_Case)
        big.P = F.Program(_long_phi(MAX_INS + 50))
        d = _dev(np.zeros(8, np.uint64))
        big.P.post_fused_noalloc(d, d, d, d, d, d, d, (d, d, d, d))
    ok = _Case(F, specs.gelu(), 64, seed=9)
    ok.check(ok.noalloc(), "after a rejected call")
