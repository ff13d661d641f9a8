"""Single-key shared-prefix construction (variant 1) -- oracle pins.
One DCF key f_{r_k,1} per view width, evaluated at the public points (xhat + delta) mod 2^k:
  I[view_{k,c}(x) < beta] = e - b + a,  h = (xhat + c) mod 2^k, e = I[h < beta], b = I[h < r_k], a = I[(h - beta) mod 2^k < r_k].
Pinned by brute force: the identity itself, and reconstruction of both calls and of the whole gate to the
plaintext F(x) / G(x) for EVERY x and EVERY mask r at n = 8 (all specs, all variant bits); at n = 12 all x for the corner
masks and all r for the corner inputs (tests/helpers.py: corner_masks, corner_inputs)."""
import numpy as np
import pytest

from helpers import all_r_keys, check_all_r, check_pairs, corner_inputs, corner_masks, mask_of, pack_bits
from workloads import specs


def test_identity_exhaustive():
    k = 6
    N = 1 << k
    r, h = np.meshgrid(np.arange(N), np.arange(N), indexing="ij")
    x = (h - r) % N
    for c in (0, 5, N - 3):
        hp, xp = (h + c) % N, (x + c) % N
        b = (hp < r).astype(np.int64)
        for beta in range(1, N):
            e = (hp < beta).astype(np.int64)
            a = (((hp - beta) % N) < r).astype(np.int64)
            want = (xp < beta).astype(np.int64)
            assert np.array_equal(want, e - b + a)
            assert np.array_equal(want, e ^ b ^ a)


SPECS8 = [lambda: specs.relu(8, 4), lambda: specs.toy(8, 3), lambda: specs.toy(8, 3, True),
          lambda: specs.plain_default(8, 3), lambda: specs.single_interval(8, 3), lambda: specs.no_bits(8, 3),
          lambda: specs.full_partition(3), lambda: specs.shift_relu(8, 3)]
SPECS12 = [lambda: specs.relu(12, 6), lambda: specs.shift_relu(12, 4), lambda: specs.toy(12, 4)]


@pytest.mark.parametrize("mk", SPECS8)
def test_sp_reconstruct_equals_plaintext_exhaustive_n8(orc, mk):
    """EVERY x and EVERY mask r at n = 8: gate outputs = G(x); atoms = the predicates themselves (Def I.1 with c_t = -beta_t,
    theta_t = r); the lookup = the active interval's payload (Def I.2)."""
    spec = specs.shared_prefix(mk())
    check_all_r(orc, spec, range(1 << spec.n), seed=13)


@pytest.mark.parametrize("mk", SPECS12)
def test_sp_reconstruct_all_x_sampled_r_n12(orc, mk):
    spec = specs.shared_prefix(mk())
    N = 1 << spec.n
    rs = corner_masks(spec, extra=4, seed=13)
    assert len(rs) >= 8
    check_pairs(orc, spec, np.tile(np.arange(N, dtype=np.uint64), len(rs)), np.repeat(np.array(rs, dtype=np.uint64), N), seed=13)


@pytest.mark.parametrize("mk", SPECS12)
def test_sp_reconstruct_all_r_sampled_x_n12(orc, mk):
    spec = specs.shared_prefix(mk())
    check_all_r(orc, spec, corner_inputs(spec, extra=3, seed=13), seed=13)


def test_sp_shapes_and_key_size(orc):
    """Shape depends on the spec only (Prop. I.3): one n-bit key (p = 1) + one key per narrower view; the key is
    ~20-48x smaller than the Protocol-3 construction's."""
    for mk, ratio in ((specs.gelu, 15), (specs.silu, 35)):
        s1 = specs.shared_prefix(mk())
        P0, P1 = orc.Program(mk()), orc.Program(s1)
        assert P1.shape["n_kb"] == 0 and P1.shape["M"] == s1.m
        assert (P1.shape["M_A"], P1.shape["rounds"]) == (P0.shape["M_A"], P0.shape["rounds"])
        per = P1.key_bytes(1 << 16) / (1 << 16)
        assert per == 16 + 64 * 24 + 8 + 8 + 3 * 8 * P1.shape["M_A"]
        assert P0.key_bytes(1 << 16) / (1 << 16) > ratio * per


def test_sp_share_is_not_the_value(orc):
    """A single party's comparison bits look uniform (guards against a degenerate share = value bug)."""
    spec = specs.shared_prefix(specs.relu(8, 4))
    P = orc.Program(spec)
    r_in, (k0, k1) = all_r_keys(P, 8, 3)
    xhat = (np.uint64(77) + r_in) & mask_of(8)
    b0 = P.eval_cmp(0, k0, xhat) & np.uint64(1)
    assert 80 < int(b0.sum()) < 176


# ---- variant bit 1: input-masked products ------------------------------------------
_slow = lambda mk: pytest.param(mk, marks=pytest.mark.slow)
XM = [_slow(lambda: specs.relu(8, 4)), lambda: specs.toy(8, 3), _slow(lambda: specs.toy(8, 3, True)), _slow(lambda: specs.plain_default(8, 3)),
      _slow(lambda: specs.no_bits(8, 3)), lambda: specs.shift_relu(8, 3)]


@pytest.mark.parametrize("sp", [0, 1])
@pytest.mark.parametrize("mk", XM)
def test_xmul_reconstruct_exhaustive_n8(orc, mk, sp):
    """y * x with x = xhat - r_in opens one element instead of two; the gate still reconstructs to G(x) for
    every x and r, with both constructions."""
    spec = specs.input_masked_mul(specs.shared_prefix(mk()) if sp else mk())
    check_all_r(orc, spec, range(1 << spec.n), seed=17)


def test_xmul_online_bytes(orc):
    """Online bytes per element per party: n/8 (xhat) + n/8 per product with x (2n/8 for a general Beaver)."""
    g0, g1 = orc.Program(specs.gelu()), orc.Program(specs.input_masked_mul(specs.gelu()))
    assert g0.online_bits() == 64 + 2 * 2 * 64 and g1.online_bits() == 64 + 2 * 64
    assert g1.post_msg_bytes(1024, 0) * 2 == g0.post_msg_bytes(1024, 0)
    assert g0.key_bytes(4096) - g1.key_bytes(4096) == 2 * 8 * 4096          # (b, c) instead of (a, b, c) per product


# ---- variant bit 2: payload = coefficients of P_i(X - r_in), Horner in the public xhat -------
XP = [lambda: specs.toy(8, 3), _slow(lambda: specs.toy(8, 3, True)), lambda: specs.plain_default(8, 3), _slow(lambda: specs.no_bits(8, 3))]


@pytest.mark.parametrize("sp", [0, 1])
@pytest.mark.parametrize("mk", XP)
def test_xpoly_reconstruct_exhaustive_n8(orc, mk, sp):
    spec = specs.public_point_horner(specs.shared_prefix(mk()) if sp else mk())
    check_all_r(orc, spec, range(1 << spec.n), seed=17)      # the lookup returns shifted coefficients: only atoms + outputs are pinned


@pytest.mark.parametrize("variant", [pytest.param(2, marks=pytest.mark.slow), 3, pytest.param(4, marks=pytest.mark.slow), 5])
def test_variant_bits_n12(orc, variant):
    """variant bits 1 / 2 at n = 12: every x for the corner masks, every r for the corner inputs."""
    spec = specs.toy(12, 4)
    if variant & 1:
        spec = specs.shared_prefix(spec)
    if variant & 2:
        spec = specs.input_masked_mul(spec)
    if variant & 4:
        spec = specs.public_point_horner(spec)
    N = 1 << spec.n
    rs = corner_masks(spec, extra=1, seed=variant)
    check_pairs(orc, spec, np.tile(np.arange(N, dtype=np.uint64), len(rs)), np.repeat(np.array(rs, dtype=np.uint64), N), seed=19)
    check_all_r(orc, spec, corner_inputs(spec, extra=0, seed=variant)[::2], seed=19)


# ---- variant bit 3: early-terminated bit trees ------------------------------------------------
ET = [_slow(lambda: specs.relu(8, 4)), lambda: specs.toy(8, 3), _slow(lambda: specs.toy(8, 3, True)), _slow(lambda: specs.plain_default(8, 3)),
      lambda: specs.single_interval(8, 3), lambda: specs.shift_relu(8, 3)]


@pytest.mark.parametrize("sp", [0, 1])
@pytest.mark.parametrize("mk", ET)
def test_early_termination_reconstruct_exhaustive_n8(orc, mk, sp):
    """Every x and every r at n = 8 with early-terminated bit trees (k = 8: one level + leaf block; k = 3: leaf block only):
    gate outputs, atoms and lookup reconstruct to their plain definitions, with both constructions."""
    spec = specs.early_termination(specs.shared_prefix(mk()) if sp else mk())
    check_all_r(orc, spec, range(1 << spec.n), seed=23)


@pytest.mark.parametrize("variant", [8, pytest.param(9, marks=pytest.mark.slow), 15])
def test_early_termination_n12(orc, variant):
    spec = specs.toy(12, 4)
    if variant & 1:
        spec = specs.shared_prefix(spec)
    if variant & 2:
        spec = specs.input_masked_mul(spec)
    if variant & 4:
        spec = specs.public_point_horner(spec)
    spec = specs.early_termination(spec)
    N = 1 << spec.n
    rs = corner_masks(spec, extra=1, seed=variant)
    check_pairs(orc, spec, np.tile(np.arange(N, dtype=np.uint64), len(rs)), np.repeat(np.array(rs, dtype=np.uint64), N), seed=29)
    check_all_r(orc, spec, corner_inputs(spec, extra=0, seed=variant)[::2], seed=29)


def test_early_termination_key_size(orc):
    """bit tree on k bits: 16 (root) + 16 max(k-7,0) (levels) + 16 (leaf block) + 8 (VCW bits) bytes instead of 16(k+1) + 8;
    shape (T, M, p, rounds, online bits) unchanged."""
    for mk in (specs.gelu, specs.shift_relu, lambda: specs.shared_prefix(specs.shift_relu())):
        s0 = mk()
        P0, P1 = orc.Program(s0), orc.Program(specs.early_termination(s0))
        assert P0.shape == P1.shape and P0.online_bits() == P1.online_bits()
        c = 1 << 16
        if s0.variant & 1:
            saved = 16 * (12 - 5 - 1)                                  # the 12-bit tree: 5 levels + leaf instead of 12
        else:
            saved = sum(16 * (k - max(k - 7, 0) - 1) for k in P0.shape["k"])
        assert P0.key_bytes(c) - P1.key_bytes(c) == saved * c


# ---- variant bit 4: dense-table ("DPF-LUT") lookup by full-domain evaluation ------------------------
DENSE = [lambda: specs.relu(8, 4), _slow(lambda: specs.toy(8, 3)), _slow(lambda: specs.plain_default(8, 3)), _slow(lambda: specs.no_bits(8, 3)),
         _slow(lambda: specs.shift_relu(8, 3)), lambda: specs.full_partition(3)]


@pytest.mark.parametrize("mk", DENSE)
def test_dense_table_reconstruct_exhaustive_n8(orc, mk):
    """Every x and every r at n = 8: the lookup evaluated on all 2^n points of the single key reconstructs the active interval's
    payload, the atoms and the gate outputs their plain definitions."""
    spec = specs.dense_table(mk())
    check_all_r(orc, spec, range(1 << spec.n), seed=37)


def test_dense_table_n12_and_shape(orc):
    spec = specs.dense_table(specs.toy(12, 4))
    N = 1 << spec.n
    rs = corner_masks(spec, extra=2, seed=3)
    xs = corner_inputs(spec, extra=2, seed=3)
    rng = np.random.default_rng(3)
    x = np.array([xs[i % len(xs)] for i in range(96)], dtype=np.uint64)
    r = np.array([rs[(i * 7) % len(rs)] for i in range(96)], dtype=np.uint64)
    x[64:], r[64:] = rng.integers(0, N, 32, dtype=np.uint64), rng.integers(0, N, 32, dtype=np.uint64)
    P = check_pairs(orc, spec, x, r, seed=41, chunk=12)
    P1 = orc.Program(specs.shared_prefix(specs.toy(12, 4)))
    assert P.key_bytes(4096) == P1.key_bytes(4096) and P.shape == P1.shape         # the same single key; only the evaluation differs
    with pytest.raises(ValueError):
        orc.Program(specs.dense_table(specs.gelu()))                                # n = 64: no dense table
    import dataclasses
    with pytest.raises(ValueError):
        orc.Program(dataclasses.replace(specs.toy(8, 3), variant=16))               # needs the single-key construction


def test_xpoly_shape(orc):
    """No Beaver multiplication and no round is left for a pure spline: online = the xhat opening only."""
    for mk in (specs.gelu, specs.silu, specs.nexp, specs.rsqrt):
        P = orc.Program(specs.public_point_horner(mk()))
        assert (P.shape["M_A"], P.shape["rounds"]) == (0, 0) and P.online_bits() == 64
