"""GPU parity (-m gpu): the CUDA path, called through the C ABI, against the CPU oracle element by element on
the same seeded inputs.  Integer ring arithmetic => the bar is BIT-EXACT: key buffers, both parties' eval_cmp
words and eval_lut coefficient shares, every round's opened messages, the output shares, and the
reconstruction against the plaintext G(x) (Lemma 4.5 / Thm 4.6)."""
import os

import numpy as np
import pytest

from helpers import mask_of, pack_bits, pmap
from workloads import specs, tensors

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def F():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; the product has no CPU fallback"
    import __graft_entry__ as g
    g.build()
    import paper_2606_09551_b200 as F
    return F


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int64)).cuda()


def host(t):
    return t.cpu().numpy().view(np.uint64)


def _parity(F, orc, spec, x, r_in, r_out, seed, check_plain=True, first_elem=0):
    import torch
    n, count = spec.n, x.size
    xhat = (x + r_in) & mask_of(n)
    P, O = F.Program(spec), orc.Program(spec)
    na = P.shape["n_out_a"]
    r_out = r_out.reshape(-1)[: max(1, na) * count].reshape(max(1, na), count)
    k0, k1 = P.alloc_keys(count)
    k0.zero_(); k1.zero_()                                   # padding bytes are unspecified; zero them to compare whole buffers
    P.keygen(dev(r_in), dev(r_out), seed, first_elem, keys=(k0, k1))
    ok0, ok1 = O.keygen(r_in, r_out, seed, first_elem)
    torch.cuda.synchronize()
    assert np.array_equal(k0.cpu().numpy(), ok0), spec.name + ": party-0 key bytes"
    assert np.array_equal(k1.cpu().numpy(), ok1), spec.name + ": party-1 key bytes"
    got = P.run_gate(k0, k1, dev(xhat))
    exp = O.run_gate(ok0, ok1, xhat)
    for b in (0, 1):
        if P.shape["T"]:
            assert np.array_equal(host(got["bits"][b]), exp["bits"][b]), spec.name + ": eval_cmp"
        if P.shape["has_lut"]:
            assert np.array_equal(host(got["coeff"][b]), exp["coeff"][b]), spec.name + ": eval_lut"
        tot = P.msg_total(count)
        assert np.array_equal(got["msg"][b].cpu().numpy()[:tot], exp["msg"][b][:tot]), spec.name + ": opened messages"
        assert np.array_equal(host(got["y"][b])[:na], exp["y"][b]), spec.name + ": y shares"
        if P.shape["n_out_b"]:
            assert np.array_equal(host(got["z"][b]), exp["z"][b]), spec.name + ": z shares"
    # the fused two-call evaluation == the separate calls, bit for bit
    for b, k in ((0, k0), (1, k1)):
        if P.shape["T"] or P.shape["has_lut"]:
            fb, fc = P.eval_fused(b, k, dev(xhat))
            if P.shape["T"]:
                assert np.array_equal(host(fb), exp["bits"][b]), spec.name + ": eval_fused bits"
            if P.shape["has_lut"]:
                assert np.array_equal(host(fc), exp["coeff"][b]), spec.name + ": eval_fused coeff"
    if P.shape["T"] or P.shape["has_lut"]:                  # both parties in one call
        bb, cc = P.eval_fused_both(k0, k1, dev(xhat))
        for b in (0, 1):
            if P.shape["T"]:
                assert np.array_equal(host(bb[b]), exp["bits"][b]), spec.name + ": eval_fused_both bits"
            if P.shape["has_lut"]:
                assert np.array_equal(host(cc[b]), exp["coeff"][b]), spec.name + ": eval_fused_both coeff"
    # fused post == per-round post, bit for bit
    y0, y1, z0, z1 = P.post_fused(k0, k1, dev(xhat), got["bits"][0], got["bits"][1], got["coeff"][0], got["coeff"][1])
    assert np.array_equal(host(y0)[:na], exp["y"][0]) and np.array_equal(host(y1)[:na], exp["y"][1])
    if P.shape["n_out_b"]:
        assert np.array_equal(host(z0), exp["z"][0]) and np.array_equal(host(z1), exp["z"][1])
    if check_plain:
        ye, ze = O.plain_G(x, r_in)
        if spec.mask_output:
            ye = (ye + r_out[: ye.shape[0]]) & mask_of(n)
        assert np.array_equal((host(y0)[:na] + host(y1)[:na]) & mask_of(n), ye), spec.name + ": reconstruction"
        if P.shape["n_out_b"]:
            assert np.array_equal(host(z0) ^ host(z1), pack_bits(ze))
    return P, (k0, k1)


def test_aes_core_fips197(F):
    """The device T-table core against the FIPS-197 vectors (tests/golden/fips197_aes128.txt)."""
    path = os.path.join(os.path.dirname(__file__), "golden", "fips197_aes128.txt")
    n = 0
    for line in open(path):
        line = line.split("#")[0].split()
        if len(line) == 3:
            key, pt, ct = (bytes.fromhex(v) for v in line)
            assert F.aes_kat(key, pt) == ct
            n += 1
    assert n >= 2


def test_bitsliced_aes_matches_fips197_and_the_table_core(F):
    """The bitsliced core (timed against the T-table core, DESIGN 5.2): block 0 = the FIPS-197 vector, the other 31 blocks
    against the device T-table core, which the test above pins to the standard."""
    path = os.path.join(os.path.dirname(__file__), "golden", "fips197_aes128.txt")
    key, pt, ct = [bytes.fromhex(v) for v in [l for l in open(path) if l.strip() and not l.startswith("#")][0].split()]
    rng = np.random.default_rng(3)
    blocks = [pt] + [bytes(rng.integers(0, 256, 16, dtype=np.uint8)) for _ in range(31)]
    out = F.bitslice_kat(key, b"".join(blocks))
    assert out[:16] == ct
    for k in (1, 2, 17, 31):
        assert out[16 * k:16 * k + 16] == F.aes_kat(key, blocks[k])


SMALL = [lambda: specs.relu(8, 4), lambda: specs.toy(8, 3), lambda: specs.toy(8, 3, True), specs.plain_default,
         specs.single_interval, specs.no_bits, specs.full_partition, lambda: specs.shift_relu(8, 3),
         lambda: specs.toy(12, 4), lambda: specs.relu(12, 6), lambda: specs.ars(8, 3), lambda: specs.ars(12, 5),
         lambda: specs.tiny_ring(1), lambda: specs.tiny_ring(2)]


SMALL_SP = [(lambda mk=mk: specs.shared_prefix(mk())) for mk in SMALL]


SMALL_XM = [(lambda mk=mk: specs.input_masked_mul(mk())) for mk in SMALL[:4] + SMALL[7:9] + SMALL_SP[:4] + SMALL_SP[7:9]]


SMALL_XP = [(lambda mk=mk: specs.public_point_horner(mk())) for mk in SMALL[1:4] + SMALL[5:6] + SMALL[8:9] + SMALL_SP[1:4] + SMALL_SP[5:6] + SMALL_SP[8:9]]


SMALL_ET = [(lambda mk=mk: specs.early_termination(mk())) for mk in SMALL[:5] + SMALL[7:] + SMALL_SP[:5] + SMALL_SP[7:] + SMALL_XM[:2] + SMALL_XP[-2:]]


SMALL_DENSE = [(lambda mk=mk: specs.dense_table(mk())) for mk in SMALL[:4] + SMALL[5:9]] + \
              [lambda: specs.early_termination(specs.dense_table(specs.shift_relu(8, 3))), lambda: specs.input_masked_mul(specs.dense_table(specs.toy(8, 3)))]


# the A2B node (DESIGN 15): bit 0 local, bits j >= 1 through a masked opening and a j-bit comparison key
SMALL_A2B = [lambda: specs.a2b_demo(8, 3), lambda: specs.shared_prefix(specs.a2b_demo(8, 3)), lambda: specs.early_termination(specs.a2b_demo(8, 3)),
             lambda: specs.early_termination(specs.shared_prefix(specs.a2b_demo(12, 4))), lambda: specs.input_masked_mul(specs.a2b_demo(12, 4))]


@pytest.fixture
def knobs(F):
    """fusefss_debug_set knobs, restored after the test"""
    def set_(**kw):
        for k, v in kw.items():
            F.debug_set(k, v)
    yield set_
    F.debug_set("force_g", 0); F.debug_set("small_kernels", 1); F.debug_set("eval_threads", 1024); F.debug_set("gen_quad", 1); F.debug_set("sp_split", 1); F.debug_set("coop", 1)


@pytest.mark.parametrize("mk", SMALL + SMALL_SP + SMALL_XM + SMALL_XP + SMALL_ET + SMALL_DENSE + SMALL_A2B)
@pytest.mark.parametrize("mode", ["auto", "g1", "g2_big"])
def test_small_rings_all_masks(F, orc, mk, mode, knobs):
    """Every mask r (both Protocol 3 branches, incl. beta_0 = 0 and the dummy split) at n <= 8; a ragged count.
    auto: the launch configuration the library picks (small launches: every tree on its own warp, 256-thread kernels, in-kernel
    zeroing + atomics; the dealer's quad-lane kernel k_gen_vec_quad; at these sizes the lane-split single-key kernel k_eval_sp_split); g1: one warp walks all trees of an element (no atomics); g2_big: two tree groups with the 1024-thread
    instantiations (the code path of large tensors whose last wave is split)."""
    if mode == "g1":
        knobs(force_g=1, gen_quad=0, sp_split=0)            # and the lane-per-element kernels instead of the quad-lane dealer / lane-split evaluation
    if mode == "g2_big":
        knobs(force_g=2, small_kernels=0)
    spec = mk()
    N = 1 << spec.n
    rng = np.random.default_rng(5)
    if N <= 256:
        r_in = np.concatenate([np.arange(N, dtype=np.uint64), rng.integers(0, N, 37, dtype=np.uint64)])
    else:
        r_in = np.concatenate([np.array([0, 1, N - 1, N // 2, N // 2 - 1, N - 3], dtype=np.uint64),
                               (np.uint64(N) - np.array(spec.alpha, dtype=np.uint64)) & mask_of(spec.n),
                               rng.integers(0, N, 300, dtype=np.uint64)])
    x = rng.integers(0, N, r_in.size, dtype=np.uint64)
    r_out = rng.integers(0, N, 4 * r_in.size, dtype=np.uint64)
    _parity(F, orc, spec, x, r_in, r_out, seed=11)


CONFIGS = [("relu16", 4096), ("gelu", 700), ("nexp", 330), ("recip", 130), ("shift_relu", 1500), ("rsqrt", 100),
           ("silu", 131)]


@pytest.mark.parametrize("variant", [0, 1, 2, 3, 4, 5, 8, 9])
@pytest.mark.parametrize("name,count", CONFIGS)
def test_config_parity(F, orc, name, count, variant):
    """BASELINE.json's configs on their seeded synthetic inputs (workloads/tensors.py), several 32-element tiles
    and a ragged tail; config 1 at its full size.  variant 1 = the single-key shared-prefix construction, whose
    kernel shares tree prefixes between nearby points while the oracle walks every point from the root."""
    spec = specs.CONFIGS[name]()
    if variant & 1:
        spec = specs.shared_prefix(spec)
        count = min(4096, count * 4)
    if variant & 2:
        spec = specs.input_masked_mul(spec)                 # one opening per product with x (DESIGN 10)
        count = max(33, count // 4)
    if variant & 4:
        spec = specs.public_point_horner(spec)              # Horner in the public xhat, zero Beaver rounds (DESIGN 11)
        count = max(33, count // 2)
    if variant & 8:
        spec = specs.early_termination(spec)                # bit trees cut 7 levels early (DESIGN 13)
    inp = tensors.inputs(name, spec, count=count, seed=0)
    _parity(F, orc, spec, inp["x"], inp["r_in"], inp["r_out"], seed=0)


@pytest.mark.parametrize("variant", [0, 1, 5, 9])
@pytest.mark.parametrize("name,count", [("relu16", 4096), ("recip", 130), ("rsqrt", 40), ("gelu", 333)])
def test_no_cooperative_launch_fallback(F, orc, name, count, variant, knobs):
    """Small launches accumulate the trees / points of an element with atomics from several warps and zero the outputs in-kernel behind
    a cooperative-launch grid barrier.  Where the context refuses that launch (cudaErrorCooperativeLaunchTooLarge: MPS thread percentage,
    SM partitions) the library clears the outputs with cudaMemsetAsync and launches normally; the "coop" = 0 knob takes that road on
    purpose.  Same bits: the three evaluation kernels (k_eval_p3, k_eval_sp, k_eval_sp_split at the tiny counts) against the oracle."""
    knobs(coop=0)
    spec = specs.CONFIGS[name]()
    if variant & 1:
        spec = specs.shared_prefix(spec)
    if variant & 4:
        spec = specs.public_point_horner(spec)
    if variant & 8:
        spec = specs.early_termination(spec)
    inp = tensors.inputs(name, spec, count=count, seed=6)
    _parity(F, orc, spec, inp["x"], inp["r_in"], inp["r_out"], seed=2)


def test_prepare_then_no_first_use_allocation(F):
    """fusefss_prepare uploads the program's tables (2 MB for this dense-table program); with every tensor allocated beforehand, the dealer,
    evaluation and post-processing calls that follow leave the device's free memory where it was: nothing allocates on first use."""
    import torch
    spec = specs.dense_table(specs.shared_prefix(specs.relu(16, 8)))
    P = F.Program(spec)
    count = 64
    inp = tensors.inputs("relu16", spec, count=count, seed=1)
    r_in, r_out, xhat = dev(inp["r_in"]), dev(inp["r_out"]), dev(inp["xhat"])
    keys = P.alloc_keys(count)
    I = lambda *shape: torch.empty(shape, dtype=torch.int64, device="cuda")
    bits, coeff = [I(count), I(count)], [I(P.shape["p"], count), I(P.shape["p"], count)]
    outs = (I(1, count), I(1, count), I(count), I(count))
    F.Program(specs.relu(16, 8)).prepare()                   # per-device constants and module load are behind us
    torch.cuda.synchronize()
    P.prepare()
    P.prepare()                                              # idempotent
    free1 = torch.cuda.mem_get_info()[0]
    P.keygen(r_in, r_out, 3, keys=keys)
    P.eval_fused_both(keys[0], keys[1], xhat, bits, coeff)
    P.post_fused(keys[0], keys[1], xhat, bits[0], bits[1], coeff[0], coeff[1], outs=outs)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free1
    y = (host(outs[0])[0] + host(outs[1])[0]) & mask_of(16)
    x = inp["x"]
    assert np.array_equal(y, np.where(x < (1 << 15), x, 0))  # ReLU on the 16-bit ring (App. N)


def test_dense_table_relu16(F, orc):
    """config 1 (ReLU, n = 16) in the dense-table representation: 65,536-point full-domain evaluation per element and party; the
    oracle walks every point from the root, so a few dozen elements (a tile, a ragged tail, both parties in one launch)."""
    spec = specs.dense_table(specs.relu(16, 8))
    inp = tensors.inputs("relu16", spec, count=41, seed=4)
    inp["x"][:4] = np.array([0, 1 << 15, (1 << 15) - 1, (1 << 16) - 1], dtype=np.uint64)
    inp["r_in"][4:8] = np.array([0, 1, (1 << 16) - 1, 1 << 15], dtype=np.uint64)
    _parity(F, orc, spec, inp["x"], inp["r_in"], inp["r_out"], seed=3)


@pytest.mark.parametrize("variant", [0, 1, 8, 9])
def test_a2b_n64(F, orc, variant):
    """A2B nodes on the 64-bit ring (63-, 12- and 1-bit comparison keys inside the post-processing kernels), several tiles and a
    ragged tail; x on the interval boundaries and around the sign change."""
    spec = specs.a2b_demo(64, 12)
    if variant & 1:
        spec = specs.shared_prefix(spec)
    if variant & 8:
        spec = specs.early_termination(spec)
    rng = np.random.default_rng(21)
    u = lambda k: rng.integers(0, 1 << 63, size=k, dtype=np.uint64) * np.uint64(2) + rng.integers(0, 2, size=k, dtype=np.uint64)
    count = 333
    x, r_in = u(count), u(count)
    a = np.array(spec.alpha, dtype=np.uint64)
    edge = np.concatenate([a, a - np.uint64(1), np.array([0, 1, 2**63, 2**63 - 1, 2**64 - 1], dtype=np.uint64)])
    x[: edge.size] = edge
    r_in[edge.size: edge.size + 3] = np.array([0, 2**64 - 1, 2**63], dtype=np.uint64)
    _parity(F, orc, spec, x, r_in, u(count), seed=6)


@pytest.mark.parametrize("variant", [0, 1])
def test_edge_masks_n64(F, orc, variant):
    """n = 64 corner masks: r = 0 (beta_0 = 0 branch + dummy split), r = -alpha_i (a translated start lands on 0),
    r = 2^64-1, and x at the interval boundaries; for variant 1 also xhat values whose cluster of points straddles
    a 2^tail_bits boundary (two different prefixes) and wraps around 2^64."""
    spec = specs.gelu()
    if variant:
        spec = specs.shared_prefix(spec)
    a = np.array(spec.alpha, dtype=np.uint64)
    r_in = np.concatenate([np.array([0, 1, 2**64 - 1, 2**63, 2**63 - 1], dtype=np.uint64), (np.uint64(0) - a), (np.uint64(0) - a) + np.uint64(1)])
    x = np.resize(np.concatenate([a, a - np.uint64(1), np.array([0, 2**64 - 1], dtype=np.uint64)]), r_in.size)
    if variant:                                            # xhat = x + r near multiples of 2^16 and near 0 / 2^64
        xh = np.array([0, 1, 2**64 - 1, 2**16, 2**16 - 1, 2**16 + 1, 3 * 2**16 + 5, 2**63, 2**63 + 2**15, 2**64 - 2**14, 2**14, 5 * 2**17 - 3],
                      dtype=np.uint64)
        r_in = np.concatenate([r_in, np.arange(xh.size, dtype=np.uint64) * np.uint64(0x9E3779B97F4A7C15)])
        x = np.concatenate([x, xh - r_in[-xh.size:]])
    r_out = np.arange(r_in.size, dtype=np.uint64)
    _parity(F, orc, spec, x, r_in, r_out, seed=9)


@pytest.mark.parametrize("count", [1, 2, 31, 32, 33])
@pytest.mark.parametrize("variant", [0, 1])
def test_degenerate_counts(F, orc, count, variant):
    """one element, a pair, and the counts around one 32-lane tile (the quad-lane dealer kernel works on 8-element tiles, the evaluation
    on 32-element tiles; dead lanes shadow the last element and must store nothing)"""
    spec = specs.CONFIGS["gelu"]()
    if variant:
        spec = specs.shared_prefix(spec)
    inp = tensors.inputs("gelu", spec, count=count, seed=5)
    _parity(F, orc, spec, inp["x"], inp["r_in"], inp["r_out"], seed=8)


def test_chunked_keygen_equals_one_shot(F, orc):
    """Randomness is derived from the GLOBAL element index (DESIGN 4.5): keygen of [40, 140) as its own chunk
    produces the same per-element material as the one-shot run (compared through the oracle's chunk)."""
    spec = specs.CONFIGS["shift_relu"]()
    inp = tensors.inputs("shift_relu", spec, count=140, seed=1)
    sl = slice(40, 140)
    _parity(F, orc, spec, inp["x"][sl], inp["r_in"][sl], inp["r_out"][:, sl], seed=4, first_elem=40)


def test_gate_host_end_to_end(F, orc):
    """fusefss_gate_host (host buffers, chunked) == oracle outputs; chunk boundary inside the tensor."""
    import torch
    spec = specs.CONFIGS["gelu"]()
    count, chunk = 300, 128
    inp = tensors.inputs("gelu", spec, count=count, seed=2)
    P, O = F.Program(spec), orc.Program(spec)
    ws = torch.empty(P.workspace_bytes(chunk), dtype=torch.uint8, device="cuda")
    y0, y1, z0, z1 = P.gate_host(inp["r_in"], inp["r_out"], inp["xhat"], 5, chunk, ws)
    ye, ze = O.plain_G(inp["x"], inp["r_in"])
    assert np.array_equal(y0[:1] + y1[:1], ye)
    assert np.array_equal(z0 ^ z1, pack_bits(ze))
    # shares themselves: chunked keygen with global indices == the oracle's one-shot keygen
    ok0, ok1 = O.keygen(inp["r_in"], inp["r_out"], 5)
    exp = O.run_gate(ok0, ok1, inp["xhat"])
    assert np.array_equal(y0[:1], exp["y"][0]) and np.array_equal(y1[:1], exp["y"][1])
    assert np.array_equal(z0, exp["z"][0]) and np.array_equal(z1, exp["z"][1])


@pytest.mark.parametrize("mk,count,chunk", [(lambda: specs.shared_prefix(specs.gelu()), 1000, 96), (lambda: specs.toy(8, 3, True), 777, 64),
                                            (lambda: specs.shift_relu(), 2050, 1024)])
def test_gate_host_many_chunks(F, orc, mk, count, chunk):
    """fusefss_gate_host double-buffers its input / output arrays over an internal copy stream: many chunks, a ragged last one, pinned
    host buffers (truly asynchronous copies), masked outputs (r_out travels too); every share equals the oracle's one-shot run, twice in
    a row through the same workspace."""
    import torch
    spec = mk()
    rng = np.random.default_rng(17)
    N = 1 << spec.n if spec.n < 64 else None
    u = (lambda k: rng.integers(0, N, k, dtype=np.uint64)) if N else \
        (lambda k: rng.integers(0, 1 << 63, size=k, dtype=np.uint64) * np.uint64(2) + rng.integers(0, 2, size=k, dtype=np.uint64))
    P, O = F.Program(spec), orc.Program(spec)
    na = max(1, P.shape["n_out_a"])
    x, r_in, r_out = u(count), u(count), u(na * count).reshape(na, count)
    xhat = (x + r_in) & mask_of(spec.n)
    pin = lambda a: torch.from_numpy(a.view(np.int64)).pin_memory().numpy().view(np.uint64)
    ws = torch.empty(P.workspace_bytes(chunk), dtype=torch.uint8, device="cuda")
    ok0, ok1 = O.keygen(r_in, r_out, 5)
    exp = O.run_gate(ok0, ok1, xhat)
    for _ in range(2):
        y0, y1, z0, z1 = P.gate_host(pin(r_in), pin(r_out), pin(xhat), 5, chunk, ws)
        assert np.array_equal(y0[:P.shape["n_out_a"]], exp["y"][0]) and np.array_equal(y1[:P.shape["n_out_a"]], exp["y"][1])
        if P.shape["n_out_b"]:
            assert np.array_equal(z0, exp["z"][0]) and np.array_equal(z1, exp["z"][1])


FULL = [("relu16", 0), ("relu16", 1), ("relu16", 8), ("shift_relu", 8), ("shift_relu", 9), ("gelu", 8), ("gelu", 0), ("gelu", 1), ("gelu", 5), ("nexp", 0), ("nexp", 1), ("recip", 0), ("recip", 1),
        ("shift_relu", 0), ("shift_relu", 1), ("rsqrt", 0), ("rsqrt", 3), ("silu", 0), ("silu", 1)]


@pytest.mark.parametrize("name,variant", FULL)
def test_full_size_sampled(F, orc, name, variant):
    """Every BASELINE.json config at its FULL size in the launch configuration bench.py times (keygen in its three
    parts, fusefss_eval_fused_both, post_fused; config 5 / variant 0 as one 704,512-element chunk at a non-zero global
    offset, as in the chunked run -- test_silu_all_chunks covers every chunk).  The oracle recomputes a sample of several
    hundred elements one by one on all host cores (its keygen is deterministic in the GLOBAL element index), and the
    reconstruction property G(x) is checked on a 20,000-element prefix."""
    import gc
    import torch
    gc.collect()
    torch.cuda.empty_cache()                                  # the big configs need most of the 180 GB
    spec = specs.CONFIGS[name]()
    if variant & 1:
        spec = specs.shared_prefix(spec)
    if variant & 2:
        spec = specs.input_masked_mul(spec)
    if variant & 4:
        spec = specs.public_point_horner(spec)
    if variant & 8:
        spec = specs.early_termination(spec)
    count = tensors.FULL_COUNT[name]
    first = 0
    if name == "silu" and not variant & 1:                    # does not fit resident: bench.py streams chunks of this size
        first, count = 3 * 704512, 704512
    inp = tensors.inputs(name, spec, count=first + count if first else count, seed=0)
    sl = slice(first, first + count)
    x, r_in, r_out, xhat = inp["x"][sl], inp["r_in"][sl], np.ascontiguousarray(inp["r_out"][:, sl]), inp["xhat"][sl]
    P, O = F.Program(spec), orc.Program(spec)
    keys = P.alloc_keys(count)
    for parts in (1, 2, 4):
        P.keygen(dev(r_in), dev(r_out), 0, first, keys=keys, parts=parts)
    k0, k1 = keys
    xh = dev(xhat)
    T, lut = P.shape["T"], P.shape["has_lut"]
    bits, coeff = P.eval_fused_both(k0, k1, xh)              # ONE launch: both parties, both FSS calls (what bench.py times)
    y0, y1, z0, z1 = P.post_fused(k0, k1, xh, bits[0], bits[1], coeff[0], coeff[1])
    torch.cuda.synchronize()
    # the oracle recomputes a sample element by element on all host cores (its keygen is deterministic in the GLOBAL index):
    # the tile edges at both ends, a 96-element run across the middle, and a few hundred random elements
    rng = np.random.default_rng(1)
    n_s = {"silu": 160, "gelu": 320, "nexp": 320}.get(name, 480)
    mid = count // 2 // 32 * 32
    idx = np.unique(np.concatenate([[0, 1, 31, 32, 33, count - 1, count - 2, count - 33], np.arange(mid - 48, mid + 48), rng.integers(0, count, n_s)]))
    idx = idx[(idx >= 0) & (idx < count)]
    hb = [host(t) if t is not None else None for t in bits]
    hc = [host(t) if t is not None else None for t in coeff]
    hy, hz = [host(y0), host(y1)], [host(z0), host(z1)]

    def one(e):
        e = int(e)
        ok0, ok1 = O.keygen(r_in[e:e + 1], r_out[:, e:e + 1], 0, first_elem=first + e)
        exp = O.run_gate(ok0, ok1, xhat[e:e + 1])
        for b in (0, 1):
            if T:
                assert hb[b][e] == exp["bits"][b][0], (name, variant, e)
            if lut:
                assert np.array_equal(hc[b].reshape(P.shape["p"], -1)[:, e], exp["coeff"][b][:, 0]), (name, variant, e)
            assert hy[b].reshape(-1, count)[0, e] == exp["y"][b][0, 0], (name, variant, e)
            if P.shape["n_out_b"]:
                assert hz[b][e] == exp["z"][b][0], (name, variant, e)
    pmap(one, idx, threads=True)
    # property at full size: shares reconstruct to the plaintext operator on a prefix
    k = min(20000, count)
    ye, ze = O.plain_G(x[:k], r_in[:k])
    assert np.array_equal((host(y0)[0, :k] + host(y1)[0, :k]) & mask_of(spec.n), ye[0])
    if P.shape["n_out_b"]:
        assert np.array_equal(host(z0)[:k] ^ host(z1)[:k], pack_bits(ze))


def test_silu_all_chunks(F, orc):
    """config 5 (SiLU, 22,544,384 elements, Protocol 3) exactly as bench.py streams it: 32 chunks of 704,512 elements through ONE
    pair of key buffers (overwritten per chunk), global element indices.  From every chunk the first and last tile edges and a few
    random elements are kept and recomputed by the oracle one by one (~700 elements across all 31 chunk boundaries); the
    reconstruction property G(x) is checked on a 65,536-element stride sample of the whole tensor."""
    import gc
    import torch
    gc.collect()
    torch.cuda.empty_cache()
    spec = specs.CONFIGS["silu"]()
    total, chunk = tensors.FULL_COUNT["silu"], 704512
    inp = tensors.inputs("silu", spec, count=total, seed=0)
    P, O = F.Program(spec), orc.Program(spec)
    k0, k1 = P.alloc_keys(chunk)
    rng = np.random.default_rng(7)
    stride = total // 65536
    keep_idx, keep = [], {"bits": [[], []], "coeff": [[], []], "y": [[], []], "z": [[], []]}
    prop_y, prop_z, prop_idx = [], [], []
    for first in range(0, total, chunk):
        c = min(chunk, total - first)
        sl = slice(first, first + c)
        r_in, r_out, xh = dev(inp["r_in"][sl]), dev(np.ascontiguousarray(inp["r_out"][:, sl])), dev(inp["xhat"][sl])
        P.keygen(r_in, r_out, 0, first, keys=(k0, k1))
        bits, coeff = P.eval_fused_both(k0, k1, xh)
        y0, y1, z0, z1 = P.post_fused(k0, k1, xh, bits[0], bits[1], coeff[0], coeff[1])
        loc = np.unique(np.concatenate([[0, 1, 31, 32, c - 33, c - 32, c - 2, c - 1], rng.integers(0, c, 14)]))
        li = torch.from_numpy(loc).cuda()
        keep_idx.append(first + loc)
        for b, (bb, cc, yy, zz) in enumerate(((bits[0], coeff[0], y0, z0), (bits[1], coeff[1], y1, z1))):
            keep["bits"][b].append(host(bb[li])); keep["coeff"][b].append(host(cc[:, li].contiguous()))
            keep["y"][b].append(host(yy[0, li])); keep["z"][b].append(host(zz[li]))
        pl = np.arange((-first) % stride, c, stride)
        pi = torch.from_numpy(pl).cuda()
        prop_idx.append(first + pl)
        prop_y.append((host(y0[0, pi]) + host(y1[0, pi])) & mask_of(spec.n)); prop_z.append(host(z0[pi]) ^ host(z1[pi]))
    torch.cuda.synchronize()
    idx = np.concatenate(keep_idx)
    got = {k: [np.concatenate(v[b], axis=-1) for b in (0, 1)] for k, v in keep.items()}

    def one(i):
        e = int(idx[i])
        ok0, ok1 = O.keygen(inp["r_in"][e:e + 1], np.ascontiguousarray(inp["r_out"][:, e:e + 1]), 0, first_elem=e)
        exp = O.run_gate(ok0, ok1, inp["xhat"][e:e + 1])
        for b in (0, 1):
            assert got["bits"][b][i] == exp["bits"][b][0], (e, "bits")
            assert np.array_equal(got["coeff"][b][:, i], exp["coeff"][b][:, 0]), (e, "coeff")
            assert got["y"][b][i] == exp["y"][b][0, 0], (e, "y")
            assert got["z"][b][i] == exp["z"][b][0], (e, "z")
    pmap(one, range(idx.size), threads=True)
    pidx = np.concatenate(prop_idx)
    ye, ze = O.plain_G(inp["x"][pidx], inp["r_in"][pidx])
    assert np.array_equal(np.concatenate(prop_y), ye[0])
    assert np.array_equal(np.concatenate(prop_z), pack_bits(ze))


@pytest.mark.parametrize("mk,count", [(specs.limits, 45), (lambda: specs.early_termination(specs.limits()), 37),
                                      (lambda: specs.shared_prefix(specs.limits(n_pred=1)), 70), (specs.limits_piecewise, 100),
                                      (lambda: specs.shared_prefix(specs.limits_piecewise()), 100)])
def test_compiled_limits(F, orc, mk, count):
    """Gate types AT the compiled limits (workloads.specs.limits: m = 63 intervals -> 63 lookup trees, p = 8 payload words, T = 64 atoms
    filling the packed comparison word, 63 output bits, 66 live bit registers; limits_piecewise: 32 AND gates = 64 opened bits = one full
    message bit word in one round): keys, both calls, every round's messages, shares and reconstruction, ragged count."""
    spec = mk()
    rng = np.random.default_rng(31)
    u = lambda k: rng.integers(0, 1 << 63, size=k, dtype=np.uint64) * np.uint64(2) + rng.integers(0, 2, size=k, dtype=np.uint64)
    x = u(count)
    a = np.array(spec.alpha, dtype=np.uint64)
    x[:20] = np.concatenate([a[:10], a[-10:] - np.uint64(1)])
    r_in = u(count)
    r_in[20:23] = np.array([0, 2**64 - 1, 2**63], dtype=np.uint64)
    _parity(F, orc, spec, x, r_in, u(2 * count), seed=13)


@pytest.mark.parametrize("variant", [0, 1, 5])
def test_many_scattered_boundaries(F, orc, variant):
    """m = 39 intervals spread over the whole ring (M = 40 lookup intervals for Protocol 3; 39 single-point clusters for
    the single-key construction -- no prefix to share): parity on a ragged count."""
    N = 1 << 64
    alpha = [(i + 1) * (N // 40) + 17 * i for i in range(38)]
    spec = specs._mk("many", 64, 12, alpha, [[[3 * i + 1, i]] for i in range(39)], n_out_a=1)
    if variant & 1:
        spec = specs.shared_prefix(spec)
    if variant & 4:
        spec = specs.public_point_horner(spec)
    rng = np.random.default_rng(8)
    u = lambda k: rng.integers(0, 1 << 63, size=k, dtype=np.uint64) * np.uint64(2) + rng.integers(0, 2, size=k, dtype=np.uint64)
    count = 45
    x = u(count)
    x[:38] = np.array(alpha, dtype=np.uint64) - np.uint64(1)
    _parity(F, orc, spec, x, u(count), u(count), seed=2)
