"""Softmax vector block composed from compiled gates (App. G).
CPU: the oracle composition (oracle/blocks.py) reconstructs, stage by stage, the plaintext fixed-point pipeline,
and that pipeline approximates the real softmax within a stated bound.  GPU: the library's block
(paper_2606_09551_b200/blocks.py: C-ABI calls only) matches the oracle composition share for share."""
import numpy as np
import pytest

from workloads import specs


def _specs(variant):
    mk = {"nexp": specs.nexp(), "tr_e": specs.shift_relu(64, 20), "recip": specs.recip(), "tr_t": specs.shift_relu(64, 28),
          "tr_y": specs.shift_relu(64, 24)}
    out = {}
    for k, s in mk.items():
        if variant & 1:
            s = specs.shared_prefix(s)
        if variant & 2:
            s = specs.input_masked_mul(s)
        if variant & 4:
            s = specs.public_point_horner(s)
        out[k] = s
    return out


def _inputs(rows, cols, seed):
    rng = np.random.default_rng(seed)
    xr = np.maximum(-20.0, -4.0 * rng.exponential(1.0, size=(rows, cols)))      # config 3: max-subtracted scores
    xr[:, 0] = 0.0                                                               # the row maximum
    x = np.floor(xr.reshape(-1) * 4096 + 0.5).astype(np.int64).view(np.uint64)
    U = lambda k: rng.integers(0, 1 << 63, size=k, dtype=np.uint64) * np.uint64(2) + rng.integers(0, 2, size=k, dtype=np.uint64)
    x0 = U(x.size)
    masks = dict(nexp=U(x.size), tr_e=U(x.size), recip=U(rows), tr_t=U(rows), tr_y=U(x.size))
    return xr, x, x0, x - x0, masks


@pytest.mark.parametrize("variant", [0, 3, 7])
def test_oracle_block_reconstructs_plaintext_pipeline(orc, variant):
    from oracle import blocks
    rows, cols = 4, 24
    progs = {k: orc.Program(s) for k, s in _specs(variant).items()}
    xr, x, x0, x1, masks = _inputs(rows, cols, 3)
    out = blocks.softmax(progs, x0, x1, masks, rows, cols, seed=100)
    pl = blocks.softmax_plain(progs, x, rows, cols)
    for k in ("e", "f", "s", "t", "u", "p", "y"):
        assert np.array_equal(out[k][0] + out[k][1], pl[k]), k
    y = pl["y"].astype(np.float64).reshape(rows, cols) / 4096.0
    ref = np.exp(xr) / np.exp(xr).sum(axis=1, keepdims=True)
    assert np.abs(y - ref).max() <= 2.0 ** -9                                    # stated bound of the fixed-point block
    assert np.all(np.abs(y.sum(axis=1) - 1.0) <= 2.0 ** -7)


@pytest.mark.gpu
@pytest.mark.parametrize("variant,rows,cols", [(3, 5, 40), (0, 3, 33), (1, 12, 128), (7, 4, 48)])
def test_gpu_block_matches_oracle_composition(orc, variant, rows, cols):
    import torch
    import __graft_entry__ as g
    g.build()
    from oracle import blocks as oblocks
    from paper_2606_09551_b200 import blocks as gblocks
    assert torch.cuda.is_available()
    xr, x, x0, x1, masks = _inputs(rows, cols, 7)
    progs = {k: orc.Program(s) for k, s in _specs(variant).items()}
    exp = oblocks.softmax(progs, x0, x1, masks, rows, cols, seed=40)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.int64)).cuda()
    B = gblocks.Softmax(rows, cols, variant)
    B.keygen({k: dev(v) for k, v in masks.items()}, seed=40)
    got = B.run(dev(x0), dev(x1))
    torch.cuda.synchronize()
    host = lambda t: t.cpu().numpy().view(np.uint64).reshape(-1)
    for k in ("e", "f", "s", "t", "u", "p", "y"):
        for b in (0, 1):
            assert np.array_equal(host(got[k][b]), exp[k][b]), (k, b)
    pl = oblocks.softmax_plain(progs, x, rows, cols)
    assert np.array_equal(host(got["y"][0]) + host(got["y"][1]), pl["y"])
    assert B.rounds() > 0 and B.online_bytes_per_party() > 0 and B.key_bytes_per_party() > 0


# ---- LayerNorm block (mean / variance reductions + rsqrt gate + signed truncation gates) ---------------------------
def _ln_specs(variant, k):
    mk = {"mean": specs.ars(64, k), "var": specs.ars(64, k + 12), "rsqrt": specs.rsqrt(), "tr_g": specs.ars(64, 24),
          "tr_y": specs.ars(64, 24)}
    out = {}
    for kk, s in mk.items():
        if variant & 1:
            s = specs.shared_prefix(s)
        if variant & 2:
            s = specs.input_masked_mul(s)
        out[kk] = s
    return out


def _ln_inputs(rows, d, seed):
    rng = np.random.default_rng(seed)
    xr = rng.normal(rng.normal(0.0, 1.0, size=(rows, 1)), rng.uniform(0.5, 3.0, size=(rows, 1)), size=(rows, d))
    x = np.floor(xr.reshape(-1) * 4096 + 0.5).astype(np.int64).view(np.uint64)
    U = lambda k: rng.integers(0, 1 << 63, size=k, dtype=np.uint64) * np.uint64(2) + rng.integers(0, 2, size=k, dtype=np.uint64)
    x0 = U(x.size)
    masks = dict(mean=U(rows), var=U(rows), rsqrt=U(rows), tr_g=U(rows), tr_y=U(x.size))
    return x, x0, x - x0, masks


@pytest.mark.parametrize("variant", [0, 3])
def test_oracle_layernorm_reconstructs_plaintext_pipeline(orc, variant):
    from oracle import blocks
    rows, d = 4, 32
    progs = {k: orc.Program(s) for k, s in _ln_specs(variant, 5).items()}
    x, x0, x1, masks = _ln_inputs(rows, d, 5)
    out = blocks.layernorm(progs, x0, x1, masks, rows, d, seed=77)
    pl = blocks.layernorm_plain(progs, x, rows, d)
    for k in ("m", "c", "q", "v", "g", "h", "p", "y"):
        assert np.array_equal(out[k][0] + out[k][1], pl[k]), k
    y = pl["y"].view(np.int64).astype(np.float64).reshape(rows, d) / 4096.0
    xq = x.view(np.int64).astype(np.float64).reshape(rows, d) / 4096.0
    ref = (xq - xq.mean(axis=1, keepdims=True)) / xq.std(axis=1, keepdims=True)
    assert np.abs(y - ref).max() <= 0.03                     # rsqrt spline: <= 0.5 % relative on a value of magnitude <= ~4


@pytest.mark.gpu
@pytest.mark.parametrize("variant,rows,d", [(3, 5, 64), (0, 2, 32), (1, 9, 1024)])
def test_gpu_layernorm_matches_oracle_composition(orc, variant, rows, d):
    import torch
    import __graft_entry__ as g
    g.build()
    from oracle import blocks as oblocks
    from paper_2606_09551_b200 import blocks as gblocks
    x, x0, x1, masks = _ln_inputs(rows, d, 11)
    progs = {k: orc.Program(s) for k, s in _ln_specs(variant, d.bit_length() - 1).items()}
    exp = oblocks.layernorm(progs, x0, x1, masks, rows, d, seed=21)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.int64)).cuda()
    B = gblocks.LayerNorm(rows, d, variant)
    B.keygen({k: dev(v) for k, v in masks.items()}, seed=21)
    got = B.run(dev(x0), dev(x1))
    torch.cuda.synchronize()
    host = lambda t: t.cpu().numpy().view(np.uint64).reshape(-1)
    for k in ("m", "c", "q", "v", "g", "h", "p", "y"):
        for b in (0, 1):
            assert np.array_equal(host(got[k][b]), exp[k][b]), (k, b)
    pl = oblocks.layernorm_plain(progs, x, rows, d)
    assert np.array_equal(host(got["y"][0]) + host(got["y"][1]), pl["y"])


# ---- gate -> gate edges through the opened masked output yhat = y + r_out (online step 6) ----------
def _fused(specs_by_stage, edges):
    import dataclasses
    return {k: (dataclasses.replace(s, mask_output=True) if k in edges else s) for k, s in specs_by_stage.items()}


@pytest.mark.parametrize("variant", [0, 3])
def test_oracle_fused_output_opening(orc, variant):
    """nExp / Recip compiled with mask_output and keyed with r_out = the next gate's r_in: the opened yhat is that gate's xhat.
    The pipeline still reconstructs the plaintext one at every stage (the masked stages after removing their public-to-the-
    dealer mask), and the downstream shares equal the unfused composition's from the truncation gates' outputs on."""
    from oracle import blocks
    rows, cols = 3, 20
    xr, x, x0, x1, masks = _inputs(rows, cols, 9)
    progs = {k: orc.Program(s) for k, s in _fused(_specs(variant), ("nexp", "recip")).items()}
    out = blocks.softmax(progs, x0, x1, masks, rows, cols, seed=50, fused_open=True)
    pl = blocks.softmax_plain({k: orc.Program(s) for k, s in _specs(variant).items()}, x, rows, cols)
    assert np.array_equal(out["e"][0] + out["e"][1] - masks["tr_e"], pl["e"])         # yhat - r_out = y
    assert np.array_equal(out["t"][0] + out["t"][1] - masks["tr_t"], pl["t"])
    for k in ("f", "s", "u", "p", "y"):
        assert np.array_equal(out[k][0] + out[k][1], pl[k]), k
    ln = {k: orc.Program(s) for k, s in _fused(_ln_specs(variant, 5), ("rsqrt",)).items()}
    x, x0, x1, masks = _ln_inputs(4, 32, 6)
    out = blocks.layernorm(ln, x0, x1, masks, 4, 32, seed=60, fused_open=True)
    pl = blocks.layernorm_plain({k: orc.Program(s) for k, s in _ln_specs(variant, 5).items()}, x, 4, 32)
    assert np.array_equal(out["g"][0] + out["g"][1] - masks["tr_g"], pl["g"])
    for k in ("m", "c", "q", "v", "h", "p", "y"):
        assert np.array_equal(out[k][0] + out[k][1], pl[k]), k


@pytest.mark.gpu
@pytest.mark.parametrize("variant", [0, 3])
def test_gpu_fused_output_opening(orc, variant):
    import torch
    import __graft_entry__ as g
    g.build()
    from oracle import blocks as oblocks
    from paper_2606_09551_b200 import blocks as gblocks
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.int64)).cuda()
    host = lambda t: t.cpu().numpy().view(np.uint64).reshape(-1)
    rows, cols = 5, 40
    xr, x, x0, x1, masks = _inputs(rows, cols, 12)
    progs = {k: orc.Program(s) for k, s in _fused(_specs(variant), ("nexp", "recip")).items()}
    exp = oblocks.softmax(progs, x0, x1, masks, rows, cols, seed=41, fused_open=True)
    B = gblocks.Softmax(rows, cols, variant, fused_open=True)
    B.keygen({k: dev(v) for k, v in masks.items()}, seed=41)
    got = B.run(dev(x0), dev(x1))
    torch.cuda.synchronize()
    for k in ("e", "f", "s", "t", "u", "p", "y"):
        for b in (0, 1):
            assert np.array_equal(host(got[k][b]), exp[k][b]), (k, b)
    rows, d = 3, 64
    x, x0, x1, masks = _ln_inputs(rows, d, 13)
    progs = {k: orc.Program(s) for k, s in _fused(_ln_specs(variant, 6), ("rsqrt",)).items()}
    exp = oblocks.layernorm(progs, x0, x1, masks, rows, d, seed=22, fused_open=True)
    B = gblocks.LayerNorm(rows, d, variant, fused_open=True)
    B.keygen({k: dev(v) for k, v in masks.items()}, seed=22)
    got = B.run(dev(x0), dev(x1))
    torch.cuda.synchronize()
    for k in ("m", "c", "q", "v", "g", "h", "p", "y"):
        for b in (0, 1):
            assert np.array_equal(host(got[k][b]), exp[k][b]), (k, b)
