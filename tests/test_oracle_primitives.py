"""Pins for the oracle's primitives: AES-128 vs FIPS-197, the DCF truth table by brute force,
Protocol 3's post-conditions, the masked-rewrite lemmas.  None of these re-types an oracle formula:
they compare against the public standard, plain definitions (u < alpha), or exhaustive identities."""
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_aes128_fips197(orc):
    rows = [l.split() for l in open(os.path.join(GOLD, "fips197_aes128.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 2
    for key, pt, ct in rows:
        assert orc.aes128_encrypt(bytes.fromhex(key), bytes.fromhex(pt)).hex() == ct


def test_prg_is_davies_meyer_of_fips_aes(orc):
    # PRG_i(s, tau) = AES_{K_i}(s^tau) ^ (s^tau), K_i = (i,1,2,..,15): pinned through the KAT-checked AES
    s = bytes(range(100, 116))
    for i in range(4):
        for tau in range(3):
            x = bytes([s[0] ^ tau]) + s[1:]
            key = bytes([i]) + bytes(range(1, 16))
            ct = orc.aes128_encrypt(key, x)
            assert orc.prg(i, s, tau) == bytes(a ^ b for a, b in zip(ct, x))


def test_dcf_bit_exhaustive_k8(orc):
    """every (alpha, u) at k = 8: Eval_0 xor Eval_1 = I[u < alpha]; alpha = 0 never fires."""
    us = np.arange(256, dtype=np.uint64)
    rng = np.random.default_rng(1)
    ones = 0
    for alpha in range(256):
        s0, s1 = rng.bytes(16), rng.bytes(16)
        o0, o1 = orc.dcf_bit_pair(8, alpha, s0, s1, us)
        assert np.array_equal(o0 ^ o1, (us < alpha).astype(np.uint8)), alpha
        ones += int(o0.sum())
    assert 0.4 < ones / 65536 < 0.6          # a single party's share is not the value itself


@pytest.mark.parametrize("k", [1, 2, 5, 12])
def test_dcf_bit_other_widths(orc, k):
    us = np.arange(1 << k, dtype=np.uint64)
    rng = np.random.default_rng(k)
    alphas = range(1 << k) if k <= 5 else rng.integers(0, 1 << k, 24)
    for alpha in alphas:
        o0, o1 = orc.dcf_bit_pair(k, int(alpha), rng.bytes(16), rng.bytes(16), us)
        assert np.array_equal(o0 ^ o1, (us < int(alpha)).astype(np.uint8))


@pytest.mark.parametrize("k", [1, 2, 3, 5, 6, 7, 8, 9, 10, 12])
def test_dcf_bit_early_termination_truth_table(orc, k):
    """Early-terminated bit-DCF (variant bit 3, DESIGN 13): Eval_0 xor Eval_1 = I[u < alpha] for every (alpha, u) at k <= 9
    (k <= 7: the whole function is one leaf block; k = 8, 9: 1-2 levels + leaf), all u for sampled alpha at k = 10, 12."""
    from helpers import pmap
    K = 1 << k
    us = np.arange(K, dtype=np.uint64)
    rng0 = np.random.default_rng(k)
    alphas = range(K) if k <= 9 else sorted({0, 1, K - 1, K // 2, 127, 128, 129, K - 128, K - 127} | {int(v) for v in rng0.integers(0, K, 40)})

    def one(alpha):
        rng = np.random.default_rng([k, alpha])
        o0, o1 = orc.dcf_bit_pair_et(k, int(alpha), rng.bytes(16), rng.bytes(16), us)
        assert np.array_equal(o0 ^ o1, (us < int(alpha)).astype(np.uint8)), (k, alpha)
        return int(o0.sum())
    ones = sum(pmap(one, alphas))
    if k >= 5:
        assert 0.35 < ones / (len(alphas) * K) < 0.65    # a single party's share is not the value itself


def test_dcf_bit_early_termination_k64_edges(orc):
    rng = np.random.default_rng(17)
    top = (1 << 64) - 1
    for alpha in [0, 1, 127, 128, 1 << 63, top, top - 127, (1 << 63) + 12345, 0x0123456789ABCDEF]:
        near = [alpha + d for d in range(-130, 131, 13) if 0 <= alpha + d <= top]
        us = np.array([0, 1, 127, 128, 1 << 63, top] + near, dtype=np.uint64)
        o0, o1 = orc.dcf_bit_pair_et(64, alpha, rng.bytes(16), rng.bytes(16), us)
        assert np.array_equal(o0 ^ o1, np.array([int(int(u) < alpha) for u in us], dtype=np.uint8)), alpha


def test_dcf_bit_k64_edges(orc):
    rng = np.random.default_rng(7)
    top = (1 << 64) - 1
    for alpha in [0, 1, 1 << 63, top, (1 << 63) + 12345, 0x0123456789ABCDEF]:
        us = np.array([0, 1, alpha - 1 if alpha else 0, alpha, min(alpha + 1, top), 1 << 63, top], dtype=np.uint64)
        o0, o1 = orc.dcf_bit_pair(64, alpha, rng.bytes(16), rng.bytes(16), us)
        exp = np.array([int(int(u) < alpha) for u in us], dtype=np.uint8)
        assert np.array_equal(o0 ^ o1, exp)


@pytest.mark.parametrize("n,p", [(8, 1), (8, 2), (8, 3), (8, 7), (16, 2)])
def test_dcf_vec_exhaustive_k8(orc, n, p):
    """every (alpha, u) at k = 8, payload in (Z_2^n)^p: Eval_0 + Eval_1 = beta * I[u < alpha]."""
    from helpers import pmap
    us = np.arange(256, dtype=np.uint64)
    mask = np.uint64((1 << n) - 1)

    def one(alpha):
        rng = np.random.default_rng([n, p, alpha])
        beta = rng.integers(0, 1 << n, p, dtype=np.uint64)
        o0, o1 = orc.dcf_vec_pair(8, n, p, alpha, beta, rng.bytes(16), rng.bytes(16), us)
        exp = np.where((us < alpha)[:, None], beta[None, :], np.uint64(0))
        assert np.array_equal((o0 + o1) & mask, exp), alpha
        return int(o0[:, 0].sum() & mask)
    shares = pmap(one, range(256))
    assert len(set(shares)) > 100            # a single party's share is not the value itself (256 draws mod 2^n)


@pytest.mark.parametrize("n,p,k", [(12, 3, 12), (64, 3, 12), (64, 8, 10)])
def test_dcf_vec_all_u_sampled_alpha(orc, n, p, k):
    """k = 10 / 12 input bits: all u for sampled alpha (incl. 0, 1, 2^k - 1, 2^{k-1})."""
    from helpers import pmap
    K = 1 << k
    us = np.arange(K, dtype=np.uint64)
    mask = np.uint64((1 << n) - 1) if n < 64 else np.uint64(0xFFFFFFFFFFFFFFFF)
    rng0 = np.random.default_rng(k * 100 + p)

    def one(alpha):
        rng = np.random.default_rng([n, p, alpha])
        beta = rng.integers(0, 1 << 63, p, dtype=np.uint64) * np.uint64(2) + np.uint64(1)
        beta &= mask
        o0, o1 = orc.dcf_vec_pair(k, n, p, alpha, beta, rng.bytes(16), rng.bytes(16), us)
        exp = np.where((us < alpha)[:, None], beta[None, :], np.uint64(0))
        assert np.array_equal((o0 + o1) & mask, exp), alpha
    pmap(one, [0, 1, K - 1, K // 2, K // 2 - 1] + [int(v) for v in rng0.integers(0, K, 11)])


def test_dcf_vec_k64(orc):
    rng = np.random.default_rng(3)
    for alpha in [1, 1 << 63, (1 << 64) - 1, 0xDEADBEEF12345678]:
        beta = rng.integers(0, 1 << 64, 3, dtype=np.uint64, endpoint=False)
        us = np.array([0, alpha - 1, alpha, (1 << 64) - 1, 1 << 62], dtype=np.uint64)
        o0, o1 = orc.dcf_vec_pair(64, 64, 3, alpha, beta, rng.bytes(16), rng.bytes(16), us)
        for i, u in enumerate(us):
            exp = beta if int(u) < alpha else np.zeros(3, np.uint64)
            assert np.array_equal(o0[i] + o1[i], exp)


# ---- the lemmas, exhaustively at n = 8 (pins the readings G1-G5 of DESIGN.md) ---------------------
def test_lemma_4_3_and_E1_exhaustive():
    n = 8
    N = 1 << n
    x = np.arange(N)[:, None]
    r = np.arange(N)[None, :]
    for k in (8, 3):                      # k = n: Lemma 4.3; k = f: Lemma E.1
        K = 1 << k
        xh = (x + r) % N % K
        rk = r % K
        for beta in range(0, K + 1):
            theta = (rk + beta) % K
            w = (rk + beta >= K)          # carry with >= (reading G3)
            lhs = (x % K) < beta
            rhs = (xh < theta) ^ (xh < rk) ^ w
            assert np.array_equal(np.broadcast_to(lhs, rhs.shape), rhs), (k, beta)


def test_interval_indicator_corollary_and_J3():
    n = 8
    N = 1 << n
    x = np.arange(N)[:, None]
    r = np.arange(N)[None, :]
    xh = (x + r) % N
    a0, a1 = 37, 200                      # corollary PAPER.md:157-161
    w0, w1 = (r + a0 >= N), (r + a1 >= N)
    rhs = (xh < (a1 + r) % N) ^ (xh < (a0 + r) % N) ^ w1 ^ w0
    assert np.array_equal(np.broadcast_to((x >= a0) & (x < a1), rhs.shape), rhs)
    s = N // 2                            # MSB(x + c)
    for c in (0, 5, 129, 255):
        xc = (xh + c) % N
        pred = (xc < (r + s) % N) ^ (xc < r) ^ (r + s >= N)
        assert np.array_equal(np.broadcast_to(((x + c) % N) >= s, pred.shape), ~pred)


# ---- Protocol 3 ---------------------------------------------------------------
@pytest.mark.parametrize("n,alpha", [(8, [128]), (8, [33, 128, 253]), (8, [1, 2, 3, 255]), (12, [512, 2048, 2049, 4000]),
                                     (3, [1, 2, 3, 4, 5, 6, 7]), (2, [1, 2])])
def test_protocol3_postconditions(orc, n, alpha):
    N = 1 << n
    m = len(alpha) + 1
    full = [0] + alpha + [N]
    branches = set()
    xs = np.arange(N) if n <= 8 else np.random.default_rng(0).integers(0, N, 64)
    interval_of = np.searchsorted(np.array(full), np.arange(N), side="right") - 1
    for r in range(N):
        B, ord_, M = orc.protocol3(n, alpha, r)
        assert M == min(m + 1, N)                                   # line 2
        B = B[:M] + [N]                                             # B_M = 2^n (truncated to 64 bits by the test entry)
        assert len(B) == M + 1 and len(ord_) == M and B[0] == 0
        assert all(B[j] < B[j + 1] for j in range(M)), (r, B)
        assert len(set(ord_)) == m and sorted(set(ord_)) == list(range(m))   # <= 1 duplicate
        branches.add((alpha and (N - r) % N in full[:-1]) or (not alpha))
        xh = (xs + r) % N
        j = np.searchsorted(np.array(B), xh, side="right") - 1      # lookup interval of xhat
        assert np.array_equal(np.array(ord_)[j], interval_of[xs]), r
    assert branches == {True, False} or m == N or n == 2
