"""Differential tests on RANDOM operator specifications (random partitions, polynomials, predicate DAGs, Phi
programs; tests/helpers.random_spec): the two independent compilers agree on every shape, the oracle's keyed
algorithm reconstructs the plaintext G(x) (Thm 4.6), and (-m gpu) the CUDA path matches the
oracle bit for bit -- for all variant flag combinations."""
import numpy as np
import pytest

from helpers import mask_of, pack_bits, random_spec

VARIANTS = [0, 1, 2, 3, 4, 5, 7, 8, 9, 15]


@pytest.fixture(scope="module")
def F():
    import __graft_entry__ as g
    g.build()
    import paper_2606_09551_b200 as F
    return F


def test_compilers_agree_on_random_specs(F, orc):
    n_ok = 0
    for seed in range(120):
        for v in VARIANTS:
            s = random_spec(seed, v)
            P, O = F.Program(s), orc.Program(s)
            assert P.shape == O.shape, (seed, v)
            assert all(P.atom(t) == O.atom(t) for t in range(P.shape["T"])), (seed, v)
            assert all(P.key_bytes(c) == O.key_bytes(c) for c in (1, 33, 1000)), (seed, v)
            assert P.post_rounds() == O.post_rounds() and P.online_bits() == O.online_bits(), (seed, v)
            assert all(P.post_msg_bytes(77, q) == O.post_msg_bytes(77, q) for q in range(P.post_rounds())), (seed, v)
            n_ok += 1
    assert n_ok == 120 * len(VARIANTS)


def _inputs(spec, count, seed):
    rng = np.random.default_rng(seed)
    n = spec.n
    u = lambda k: rng.integers(0, 1 << 63, size=k, dtype=np.uint64) * np.uint64(2) + rng.integers(0, 2, size=k, dtype=np.uint64)
    x, r_in = u(count) & mask_of(n), u(count) & mask_of(n)
    edges = np.array(([0] + spec.alpha) * 2, dtype=np.uint64)[:count]      # x on and just below the interval boundaries
    x[: edges.size] = edges
    x[edges.size: 2 * edges.size] = ((edges - np.uint64(1)) & mask_of(n))[: max(0, count - edges.size)]
    r_out = u(count * max(1, spec.n_out_a or spec.r)) & mask_of(n)
    return x, r_in, r_out


@pytest.mark.parametrize("seed", range(24))
def test_oracle_reconstructs_random_specs(orc, seed):
    for v in (0, 1, 3, 5, 8, 15):                       # every variant for every seed (A2B nodes and the et / all-bits variants included)
        spec = random_spec(seed, v)
        P = orc.Program(spec)
        count = 48
        x, r_in, r_out = _inputs(spec, count, seed)
        na = P.shape["n_out_a"]
        r_out = r_out[: max(1, na) * count].reshape(max(1, na), count)
        k0, k1 = P.keygen(r_in, r_out, seed)
        out = P.run_gate(k0, k1, (x + r_in) & mask_of(spec.n))
        ye, ze = P.plain_G(x, r_in)
        if spec.mask_output:
            ye = (ye + r_out[: ye.shape[0]]) & mask_of(spec.n)
        assert np.array_equal((out["y"][0] + out["y"][1]) & mask_of(spec.n), ye), (seed, v)
        if P.shape["n_out_b"]:
            assert np.array_equal(out["z"][0] ^ out["z"][1], pack_bits(ze)), (seed, v)


@pytest.mark.gpu
@pytest.mark.parametrize("seed", range(16))
def test_gpu_matches_oracle_on_random_specs(F, orc, seed):
    import torch
    from test_gpu_parity import _parity
    assert torch.cuda.is_available()
    for v in VARIANTS:
        spec = random_spec(seed, v)
        x, r_in, r_out = _inputs(spec, 75, seed + 1000)
        _parity(F, orc, spec, x, r_in, r_out, seed=seed)
