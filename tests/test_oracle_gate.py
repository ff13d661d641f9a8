"""Tier B (keyed algorithm) pinned to Tier A (plaintext semantics) and Tier A pinned to closed forms.
Lemma 4.5 / Thm 4.6: reconstructing the two parties' outputs gives G(x) for EVERY
x and EVERY mask r.  Exhaustive (every x, every r) at n = 8 for every spec; at n = 12 all x with sampled r (incl. r = 0,
r = -alpha_i, r = N-1) and all r with sampled x (incl. every alpha_i, alpha_i - 1).  The loops run on all host cores
(tests/helpers.pmap: the oracle's C calls release the GIL); the oracle itself is single-threaded."""
import os

import numpy as np
import pytest

from helpers import all_r_keys, check_all_r, check_pairs, corner_inputs, corner_masks, mask_of, pack_bits, pmap
from workloads import specs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _signed(v, n):
    v = v.astype(np.int64)
    return np.where(v >= (1 << (n - 1)), v - (1 << n), v)


SPECS8 = [lambda: specs.relu(8, 4), lambda: specs.toy(8, 3), lambda: specs.toy(8, 3, True),
          lambda: specs.plain_default(8, 3), lambda: specs.single_interval(8, 3), lambda: specs.no_bits(8, 3),
          lambda: specs.full_partition(3), lambda: specs.shift_relu(8, 3)]
SPECS12 = [lambda: specs.relu(12, 6), lambda: specs.shift_relu(12, 4), lambda: specs.toy(12, 4)]


@pytest.mark.parametrize("mk", SPECS8)
def test_reconstruct_equals_plaintext_exhaustive_n8(orc, mk):
    """EVERY x and EVERY mask r at n = 8 (65,536 instances per spec; full_partition: n = 3): the gate's outputs, the packed
    comparison's bits and the interval lookup's payload all reconstruct to their plain definitions."""
    spec = mk()
    check_all_r(orc, spec, range(1 << spec.n))


@pytest.mark.parametrize("mk", SPECS12)
def test_reconstruct_all_x_sampled_r_n12(orc, mk):
    """n = 12: all 4,096 x for each of >= 8 masks, among them r = 0, r = -alpha_i (beta_0 = 0 branch), r = N-1."""
    spec = mk()
    N = 1 << spec.n
    rs = corner_masks(spec, extra=4, seed=12)
    assert len(rs) >= 8
    x = np.tile(np.arange(N, dtype=np.uint64), len(rs))
    r = np.repeat(np.array(rs, dtype=np.uint64), N)
    check_pairs(orc, spec, x, r)


@pytest.mark.parametrize("mk", SPECS12)
def test_reconstruct_all_r_sampled_x_n12(orc, mk):
    """n = 12: all 4,096 masks r for x on / just below / just above every alpha_i, the ring's ends, the sign change."""
    spec = mk()
    check_all_r(orc, spec, corner_inputs(spec, extra=3, seed=12))


@pytest.mark.parametrize("n", [1, 2])
@pytest.mark.parametrize("variant", [0, 1, 8, 9, 3, 5])
def test_tiny_rings_exhaustive(orc, n, variant):
    """Z_2 and Z_4 (M = min(m + 1, 2^n) binds: P:579): every x and every r, both constructions and the variant bits."""
    spec = specs.tiny_ring(n)
    if variant & 1:
        spec = specs.shared_prefix(spec)
    if variant & 2:
        spec = specs.input_masked_mul(spec)
    if variant & 4:
        spec = specs.public_point_horner(spec)
    if variant & 8:
        spec = specs.early_termination(spec)
    check_all_r(orc, spec, range(1 << n))


def test_appendix_N_relu_golden(orc):
    """App. N: shape (T, M, p, #Beaver), atoms, and semantics (max(x,0), MSB(x))."""
    gold = {}
    for line in open(os.path.join(GOLD, "appN_relu.txt")):
        line = line.split("#")[0].split()
        if line:
            gold[line[0]] = [int(v) for v in line[1:]]
    for n, f in ((8, 4), (12, 6), (16, 8), (64, 12)):
        spec = specs.relu(n, f)
        P = orc.Program(spec)
        for key in ("T", "M", "p", "M_A", "M_B", "G_mix"):
            assert P.shape[key] == gold[key][0], key
        assert spec.m == gold["m"][0]
        assert [int(v) for v in spec.coeff[0].reshape(-1)] == gold["P0"]
        assert [int(v) for v in spec.coeff[1].reshape(-1)] == gold["P1"]
        assert P.shape["k"] == [n, n]
        a0, a1 = P.atom(0), P.atom(1)
        assert (a0["is_theta"], a1["is_theta"], a1["beta"], a0["c"], a1["c"]) == (0, 1, 1 << (n - 1), 0, 0)
    n = 8
    P = orc.Program(specs.relu(8, 4))
    xs = np.arange(256, dtype=np.uint64)
    y, z = P.plain_G(xs, np.zeros(256, np.uint64))
    assert np.array_equal(_signed(y[0], n), np.maximum(_signed(xs, n), 0))
    assert np.array_equal(z[0], (xs >= 128).astype(np.uint8))


@pytest.mark.parametrize("n,f", [(8, 3), (12, 4)])
def test_shift_relu_closed_form(orc, n, f):
    """config 4a semantics: y = max(0, floor(x_signed / 2^f)) for all x, r; wrap bit two ways agree."""
    P = orc.Program(specs.shift_relu(n, f))
    N = 1 << n
    xs = np.arange(N, dtype=np.uint64)
    for r in (range(N) if n == 8 else [0, 1, N // 2, N - 1, 1234, 3001]):
        rv = np.full(N, r, dtype=np.uint64)
        y, z = P.plain_G(xs, rv)
        assert np.array_equal(y[0].astype(np.int64), np.maximum(0, _signed(xs, n) >> f))
        assert np.array_equal(z[0], (xs >= N // 2).astype(np.uint8))
        assert np.array_equal(z[1], z[2])                            # AND-path wrap bit == r-atom wrap bit
        assert np.array_equal(z[1], (((xs + rv) & mask_of(n)) < rv).astype(np.uint8))


@pytest.mark.parametrize("variant", [0, 9])
def test_a2b_node(orc, variant):
    """A2B (reading DESIGN 15 = bit extraction): every x and every r at n = 8 reconstructs Tier A, and Tier A's
    extracted bits are what they claim to be (closed forms on the cleartext: MSB(x), bit f of y_0, LSB(x + y_0))."""
    spec = specs.a2b_demo(8, 3)
    if variant & 1:
        spec = specs.shared_prefix(spec)
    if variant & 8:
        spec = specs.early_termination(spec)
    P = check_all_r(orc, spec, range(256), seed=43)
    assert P.shape["G_mix"] == 1 + 3 and P.post_rounds() == 4            # one B2A + three preprocessed A2B (the LSB one is local)
    assert P.online_bits() == 8 + 2 * 8 + 3 * 8 + 1                       # xhat + the Horner Beaver product + three A2B openings + one B2A bit
    x = np.arange(256, dtype=np.uint64)
    y, z = P.plain_G(x, np.zeros(256, np.uint64))
    y0 = np.array([int(P.plain_F(int(v))[0][0]) for v in x], dtype=np.uint64)
    assert np.array_equal(z[0], (x >= 128).astype(np.uint8))
    assert np.array_equal(z[1], ((y0 >> np.uint64(3)) & np.uint64(1)).astype(np.uint8))
    assert np.array_equal(z[2], (((x + y0) & np.uint64(255)) & np.uint64(1)).astype(np.uint8))
    check_pairs(orc, specs.a2b_demo(12, 4) if not variant else specs.early_termination(specs.shared_prefix(specs.a2b_demo(12, 4))),
                np.tile(np.arange(0, 4096, 7, dtype=np.uint64), 3), np.repeat(np.array([0, 4095, 1234], dtype=np.uint64), 586), seed=44)


def test_shape_is_mask_independent(orc):
    """Prop. I.3: (T, M, p), key length and layout depend on (program, count) only."""
    spec = specs.toy(8, 3)
    P = orc.Program(spec)
    sizes = {P.key_bytes(c) for c in (1, 31, 32, 33, 1000)}
    assert len(sizes) >= 3
    kb = P.key_bytes(16)
    for r0 in (0, 1, 255, 224):                                      # incl. r = -alpha_i (beta_0 = 0 branch)
        k0, k1 = P.keygen(np.full(16, r0, np.uint64), None, 3)
        assert k0.size == kb and k1.size == kb
    for other in (specs.relu(64, 12), specs.gelu(), specs.shift_relu()):
        Q = orc.Program(other)
        assert Q.key_bytes(7) == Q.key_bytes(7)


def test_chunked_keygen_equals_one_shot(orc):
    """randomness is derived from the GLOBAL element index, so chunks reproduce the one-shot keys."""
    spec = specs.shift_relu(12, 4)
    P = orc.Program(spec)
    rng = np.random.default_rng(0)
    r = rng.integers(0, 4096, 96, dtype=np.uint64)
    xh = rng.integers(0, 4096, 96, dtype=np.uint64)
    k0, k1 = P.keygen(r, None, 9)
    full = P.run_gate(k0, k1, xh)
    for lo, hi in ((0, 40), (40, 96)):
        c0, c1 = P.keygen(r[lo:hi], None, 9, first_elem=lo)
        part = P.run_gate(c0, c1, xh[lo:hi])
        for b in (0, 1):
            assert np.array_equal(part["y"][b], full["y"][b][:, lo:hi])
            assert np.array_equal(part["bits"][b], full["bits"][b][lo:hi])
            assert np.array_equal(part["coeff"][b], full["coeff"][b][:, lo:hi])


def test_single_party_shares_look_uniform(orc):
    """guards against a degenerate "share = value" bug: chi^2 of party-0 output share at n = 8."""
    spec = specs.relu(8, 4)
    P = orc.Program(spec)
    rng = np.random.default_rng(5)
    cnt = 8192
    r = rng.integers(0, 256, cnt, dtype=np.uint64)
    x = np.full(cnt, 3, np.uint64)
    k0, k1 = P.keygen(r, None, 77)
    out = P.run_gate(k0, k1, (x + r) & np.uint64(255))
    for arr in (out["y"][0][0], out["coeff"][0][0], out["coeff"][1][1]):
        h = np.bincount(arr.astype(np.int64), minlength=256)
        chi2 = ((h - cnt / 256) ** 2 / (cnt / 256)).sum()
        assert chi2 < 400, chi2                                       # 255 dof: mean 255, sd ~22.6
    ones = int((out["bits"][0] & np.uint64(1)).sum())
    assert 0.45 < ones / cnt < 0.55


def test_complexity_accounting_table(orc):
    """App. O counts per config, as listed in DESIGN.md."""
    exp = {"relu16": (2, 3, 2, 1, 0, 0), "gelu": (5, 11, 3, 2, 0, 0), "nexp": (0, 19, 2, 1, 0, 0),
           "recip": (0, 19, 3, 2, 0, 0), "shift_relu": (3, 3, 1, 1, 1, 2), "rsqrt": (0, 15, 3, 2, 0, 0),
           "silu": (5, 27, 3, 2, 0, 0)}
    for name, want in exp.items():
        P = orc.Program(specs.CONFIGS[name]())
        got = tuple(P.shape[k] for k in ("T", "M", "p", "M_A", "M_B", "G_mix"))
        assert got == want, (name, got)
    P = orc.Program(specs.shift_relu())
    assert P.shape["k"] == [64, 64, 12] and P.post_rounds() == 3
    assert P.online_bits() == 64 + 2 * 64 + 2 + 2


def ill_formed_specs():
    """(why, spec) pairs that both compilers must reject."""
    import copy
    out = []
    s = specs.relu(8, 4); s.alpha = [0]; out.append(("boundary 0", s))
    s = specs.toy(8, 3); s.alpha = [40, 40, 200]; out.append(("boundaries not strictly increasing", s))
    s = specs.toy(8, 3); s.alpha = [40, 100, 256]; out.append(("boundary >= 2^n", s))
    s = specs.toy(8, 3); s.nodes = list(s.nodes); s.nodes[2] = (specs.BN_C, 0, 0, 0, 0, 300); out.append(("C_beta with beta > 2^n", s))
    s = specs.toy(8, 3); s.nodes = list(s.nodes); s.nodes[0] = (specs.BN_D, 3, 0, 0, 0, 9); out.append(("D_gamma with gamma > 2^f", s))
    s = specs.toy(8, 3); s.nodes = list(s.nodes); s.nodes[0] = (specs.BN_D, 9, 0, 0, 0, 1); out.append(("D width > n", s))
    s = specs.toy(8, 3); s.nodes = list(s.nodes); s.nodes[3] = (specs.BN_AND, 0, 0, 5, 0, 0); out.append(("operand does not precede", s))
    s = specs.toy(8, 3); s.kappa_b = [(specs.KB_R_BIT, 8)]; out.append(("kappa^B bit index >= n", s))
    s = specs.toy(8, 3); s.kappa_a = [(specs.KA_R_SHR, 64)]; out.append(("kappa^A shift >= 64", s))
    s = specs.toy(8, 3); s.kappa_a = [(specs.KA_R_SHR, 1)] * 9; out.append(("more than 8 kappa^A", s))
    s = specs.toy(8, 3); s.phi = [(specs.PHI_B_XHAT, d, 8, b, i) if (op, a) == (specs.PHI_B_XHAT, 1) else (op, d, a, b, i) for (op, d, a, b, i) in s.phi]
    out.append(("xhat bit index >= n", s))
    s = specs.shift_relu(8, 3); s.phi = [(op, d, a, 8 if op == specs.PHI_B_ANDPUB else b, i) for (op, d, a, b, i) in s.phi]; out.append(("ANDPUB bit index >= n", s))
    s = specs.toy(8, 3); s.phi = [o for o in s.phi if not (o[0] == specs.PHI_A_OUT and o[1] == 1)]; out.append(("arithmetic output never written", s))
    s = specs.toy(8, 3); s.phi = s.phi + [(specs.PHI_B_OUT, 0, 7, 0, 0)]; out.append(("bit output written twice", s))
    s = specs.toy(8, 3); s.phi = s.phi + [(99, 0, 0, 0, 0)]; out.append(("unknown Phi op", s))
    return out


def test_rejects_ill_formed(orc):
    for why, s in ill_formed_specs():
        with pytest.raises(ValueError):
            orc.Program(s)
            pytest.fail("accepted: " + why)
    orc.Program(specs.toy(8, 3))


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("n,f", [(8, 3), (12, 5)])
def test_ars_gate_closed_form(orc, n, f, variant):
    """Signed truncation gate (workloads.specs.ars): with the gate input x' = x + 2^{n-1}, the shares reconstruct to
    floor(x_signed / 2^f) for every x and every mask r (closed form; SURVEY C7 truncation identity)."""
    spec = specs.ars(n, f)
    if variant:
        spec = specs.shared_prefix(spec)
    P = orc.Program(spec)
    N = 1 << n
    r_in, (k0, k1) = all_r_keys(P, n, 21)

    def one(x):
        xs = x - N if x >= N // 2 else x
        want = np.uint64((xs >> f) % N)
        xp = np.full(N, (x + N // 2) % N, dtype=np.uint64)               # x' = x + 2^{n-1}
        out = P.run_gate(k0, k1, (xp + r_in) & mask_of(n))
        assert np.all(((out["y"][0] + out["y"][1]) & mask_of(n)) == want), (n, f, x)
    pmap(one, range(N) if n == 8 else sorted(set(list(range(0, N, 37)) + [N - 1, N // 2, N // 2 - 1, N // 2 + 1, (1 << f) - 1, 1 << f])))
    if n == 12:                                                          # and every x for a few masks
        rs = np.array([0, 1, N - 1, N // 2, N // 2 - 1, 1234, 3001, (1 << f) - 1], dtype=np.uint64)
        x = np.tile(np.arange(N, dtype=np.uint64), rs.size)
        r = np.repeat(rs, N)
        ka, kb = P.keygen(r, None, 22)
        out = P.run_gate(ka, kb, (((x + np.uint64(N // 2)) & mask_of(n)) + r) & mask_of(n))
        xs = x.astype(np.int64)
        xs = np.where(xs >= N // 2, xs - N, xs)
        assert np.array_equal((out["y"][0][0] + out["y"][1][0]) & mask_of(n), ((xs >> f) % N).astype(np.uint64))
