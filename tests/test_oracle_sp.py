"""Single-key shared-prefix construction (variant 1) -- oracle pins.
One DCF key f_{r_k,1} per view width, evaluated at the public points (xhat + delta) mod 2^k:
  I[view_{k,c}(x) < beta] = e - b + a,  h = (xhat + c) mod 2^k, e = I[h < beta], b = I[h < r_k], a = I[(h - beta) mod 2^k < r_k].
Pinned by brute force: the identity itself, and reconstruction of both calls and of the whole gate to the
plaintext F(x) / G(x) for every x and every mask r at n = 8 (sampled at n = 12)."""
import numpy as np
import pytest

from helpers import all_r_keys, mask_of, pack_bits
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


def _check_all_r(orc, spec, xs, seed=13):
    P = orc.Program(spec)
    n = spec.n
    N = 1 << n
    na = P.shape["n_out_a"]
    r_out = (np.arange(N * max(1, na), dtype=np.uint64) * np.uint64(2654435761)) & mask_of(n)
    r_in, (k0, k1) = all_r_keys(P, n, seed, r_out)
    for x in xs:
        xv = np.full(N, x, dtype=np.uint64)
        xhat = (xv + r_in) & mask_of(n)
        out = P.run_gate(k0, k1, xhat)
        ye, ze = P.plain_G(xv, r_in)
        if spec.mask_output:
            ye = (ye + r_out.reshape(-1, N)[: ye.shape[0]]) & mask_of(n)
        assert np.array_equal((out["y"][0] + out["y"][1]) & mask_of(n), ye), (spec.name, x)
        if P.shape["n_out_b"]:
            assert np.array_equal(out["z"][0] ^ out["z"][1], pack_bits(ze)), (spec.name, x)
        for t in range(P.shape["T"]):                       # Def I.1 with c_t = -beta_t, theta = r
            a = P.atom(t)
            K = np.uint64((1 << a["k"]) - 1)
            got = ((out["bits"][0] ^ out["bits"][1]) >> np.uint64(t)) & np.uint64(1)
            if a["is_theta"]:
                want = (((xv & K) + np.uint64(a["c"])) & K) < np.uint64(a["beta"])
            else:
                want = (((xhat & K) + np.uint64(a["c"])) & K) < (r_in & K)
            assert np.array_equal(got, want.astype(np.uint64)), (spec.name, t)
        if P.shape["has_lut"]:                               # Def I.2: the active interval's payload
            c = (out["coeff"][0] + out["coeff"][1]) & mask_of(n)
            i_star = np.searchsorted(np.array([0] + spec.alpha), np.uint64(x), side="right") - 1
            pay = np.concatenate([spec.coeff[i_star].reshape(-1), spec.aux[i_star].reshape(-1)]) & mask_of(n)
            assert np.array_equal(c, np.repeat(pay[:, None], N, axis=1)), (spec.name, x)
    return P


SPECS8 = [lambda: specs.relu(8, 4), lambda: specs.toy(8, 3), lambda: specs.toy(8, 3, True),
          lambda: specs.plain_default(8, 3), lambda: specs.single_interval(8, 3), lambda: specs.no_bits(8, 3),
          lambda: specs.full_partition(3), lambda: specs.shift_relu(8, 3)]


@pytest.mark.parametrize("mk", SPECS8)
def test_sp_reconstruct_equals_plaintext_exhaustive_n8(orc, mk):
    spec = specs.shared_prefix(mk())
    N = 1 << spec.n
    xs = range(N) if spec.name.startswith(("relu_n8", "shift_relu_n8", "full_n3")) else list(range(0, N, 5)) + [N - 1, N // 2, N // 2 - 1]
    _check_all_r(orc, spec, xs)


@pytest.mark.parametrize("mk", [lambda: specs.relu(12, 6), lambda: specs.shift_relu(12, 4), lambda: specs.toy(12, 4)])
def test_sp_reconstruct_n12(orc, mk):
    spec = specs.shared_prefix(mk())
    rng = np.random.default_rng(12)
    xs = [0, 2047, 2048, 4095] + [int(v) for v in rng.integers(0, 4096, 1)]
    _check_all_r(orc, spec, xs)


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
XM = [lambda: specs.relu(8, 4), lambda: specs.toy(8, 3), lambda: specs.toy(8, 3, True), lambda: specs.plain_default(8, 3),
      lambda: specs.no_bits(8, 3), lambda: specs.shift_relu(8, 3)]


@pytest.mark.parametrize("sp", [0, 1])
@pytest.mark.parametrize("mk", XM)
def test_xmul_reconstruct_exhaustive_n8(orc, mk, sp):
    """y * x with x = xhat - r_in opens one element instead of two; the gate still reconstructs to G(x) for
    every x and r, with both constructions."""
    spec = specs.input_masked_mul(specs.shared_prefix(mk()) if sp else mk())
    N = 1 << spec.n
    _check_all_r(orc, spec, list(range(0, N, 5)) + [N - 1]) if sp else _check_plain_only(orc, spec, list(range(0, N, 5)) + [N - 1])


def _check_plain_only(orc, spec, xs, seed=17):
    P = orc.Program(spec)
    n = spec.n
    N = 1 << n
    na = P.shape["n_out_a"]
    r_out = (np.arange(N * max(1, na), dtype=np.uint64) * np.uint64(40503)) & mask_of(n)
    r_in, (k0, k1) = all_r_keys(P, n, seed, r_out)
    for x in xs:
        xv = np.full(N, x, dtype=np.uint64)
        out = P.run_gate(k0, k1, (xv + r_in) & mask_of(n))
        ye, ze = P.plain_G(xv, r_in)
        if spec.mask_output:
            ye = (ye + r_out.reshape(-1, N)[: ye.shape[0]]) & mask_of(n)
        assert np.array_equal((out["y"][0] + out["y"][1]) & mask_of(n), ye), (spec.name, x)
        if P.shape["n_out_b"]:
            assert np.array_equal(out["z"][0] ^ out["z"][1], pack_bits(ze)), (spec.name, x)


def test_xmul_online_bytes(orc):
    """Online bytes per element per party: n/8 (xhat) + n/8 per product with x (2n/8 for a general Beaver)."""
    g0, g1 = orc.Program(specs.gelu()), orc.Program(specs.input_masked_mul(specs.gelu()))
    assert g0.online_bits() == 64 + 2 * 2 * 64 and g1.online_bits() == 64 + 2 * 64
    assert g1.post_msg_bytes(1024, 0) * 2 == g0.post_msg_bytes(1024, 0)
    assert g0.key_bytes(4096) - g1.key_bytes(4096) == 2 * 8 * 4096          # (b, c) instead of (a, b, c) per product


# ---- variant bit 2: payload = coefficients of P_i(X - r_in), Horner in the public xhat -------
XP = [lambda: specs.toy(8, 3), lambda: specs.toy(8, 3, True), lambda: specs.plain_default(8, 3), lambda: specs.no_bits(8, 3)]


@pytest.mark.parametrize("sp", [0, 1])
@pytest.mark.parametrize("mk", XP)
def test_xpoly_reconstruct_exhaustive_n8(orc, mk, sp):
    spec = specs.public_point_horner(specs.shared_prefix(mk()) if sp else mk())
    N = 1 << spec.n
    _check_plain_only(orc, spec, list(range(0, N, 5)) + [N - 1])


def test_xpoly_shape(orc):
    """No Beaver multiplication and no round is left for a pure spline: online = the xhat opening only."""
    for mk in (specs.gelu, specs.silu, specs.nexp, specs.rsqrt):
        P = orc.Program(specs.public_point_horner(mk()))
        assert (P.shape["M_A"], P.shape["rounds"]) == (0, 0) and P.online_bits() == 64
