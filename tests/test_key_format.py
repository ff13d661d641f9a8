"""The oracle's key buffer against the WRITTEN key format, without the GPU in the loop.

DESIGN.md 4.4 (layout) and 4.5 (deterministic randomness R(e, slot)) are this build's readings of what the paper leaves open; both the
oracle and the CUDA path implement them, and the GPU parity tests compare the two byte for byte.  This file ties the format to the
text instead of to either implementation: offsets are computed here from the rules of 4.4, values from 4.5 with nothing but the
FIPS-197-pinned block cipher (oracle.aes128_encrypt, tests/test_oracle_primitives.py), and the oracle's buffer has to hold exactly
those words there.  A section moved, a slot renumbered, or low / high halves swapped in either document or code fails here."""
import numpy as np
import pytest

from workloads import specs

COUNT, SEED, FIRST = 37, 0x1234ABCD, 1000          # a ragged count (padding matters), a global element offset (chunked keygen)


def _up(x):
    return (x + 255) // 256 * 256


def _R(orc, e, slot):
    """DESIGN 4.5: R(e, slot) = AES128_{seed || ~seed}(LE64(e) || LE64(slot))"""
    key = SEED.to_bytes(8, "little") + (~SEED & (2 ** 64 - 1)).to_bytes(8, "little")
    return orc.aes128_encrypt(key, e.to_bytes(8, "little") + slot.to_bytes(8, "little"))


def _words(buf, off, count=COUNT):
    return np.frombuffer(buf[off:off + 8 * count].tobytes(), dtype=np.uint64)


@pytest.mark.parametrize("mk", [lambda: specs.relu(16, 8), specs.gelu, lambda: specs.toy(8, 3, True), specs.recip],
                         ids=["relu16", "gelu", "toy_masked", "recip"])
def test_oracle_keys_follow_the_written_format(orc, mk):
    spec = mk()
    O = orc.Program(spec)
    sh, n = O.shape, spec.n
    mask = (1 << n) - 1
    rng = np.random.default_rng(1)
    u = lambda k: (rng.integers(0, 1 << 63, size=k, dtype=np.uint64) * np.uint64(2) + rng.integers(0, 2, size=k, dtype=np.uint64)) & np.uint64(mask)
    na = max(1, sh["n_out_a"])
    r_in, r_out = u(COUNT), u(na * COUNT).reshape(na, COUNT)
    k0, k1 = O.keygen(r_in, r_out, SEED, FIRST)
    s16, s8 = _up(16 * COUNT), _up(8 * COUNT)
    lo = lambda b: int.from_bytes(b[:8], "little") & mask
    hi = lambda b: int.from_bytes(b[8:], "little") & mask

    # 4.4: the T bit trees come first -- root [s16], k_t level arrays [s16], one [s8] word of VCW bits each
    off, tree_off = 0, []
    for t in range(sh["T"]):
        tree_off.append(off)
        off += s16 * (1 + sh["k"][t]) + s8
    # 4.5: root of tree t, party b = R(e, 0x1000 + 2t + b) with its two low bits cleared; bit 0 then carries the final-CW bit
    for t in sorted({0, sh["T"] - 1} & set(range(sh["T"]))):
        for b, kb in ((0, k0), (1, k1)):
            got = np.frombuffer(kb[tree_off[t]:tree_off[t] + 16 * COUNT].tobytes(), dtype=np.uint8).reshape(COUNT, 16)
            exp = np.frombuffer(b"".join(_R(orc, FIRST + e, 0x1000 + 2 * t + b) for e in range(COUNT)), dtype=np.uint8).reshape(COUNT, 16)
            assert np.array_equal(got[:, 1:], exp[:, 1:]) and np.array_equal(got[:, 0] & 0xFC, exp[:, 0] & 0xFC), (spec.name, t, b)
            assert not (got[:, 0] & 2).any()
    # 4.4: then c_b[p][s8] and the M-1 vector trees: root [s16], n levels of {sCW [s16], VCW [p][s8]}, fin [p][s8]
    if sh["has_lut"]:
        p = sh["p"]
        off += p * s8 + (sh["M"] - 1) * (s16 + n * (s16 + p * s8) + p * s8)
    # [r_in] [s8]: party 0 holds the low 8 bytes of R(e, 0x4000), party 1 the difference
    w0, w1 = _words(k0, off), _words(k1, off)
    exp0 = np.array([lo(_R(orc, FIRST + e, 0x4000)) for e in range(COUNT)], dtype=np.uint64)
    assert np.array_equal(w0, exp0), spec.name + ": [r_in]_0"
    assert np.array_equal((w0 + w1) & np.uint64(mask), r_in), spec.name + ": [r_in]_0 + [r_in]_1 = r_in"
    off += s8
    # [r_out][n_out_a][s8] if the outputs are masked: share j of party 0 = low 8 bytes of R(e, 0x4100 + j)
    if spec.mask_output:
        for j in range(sh["n_out_a"]):
            y0, y1 = _words(k0, off + j * s8), _words(k1, off + j * s8)
            assert np.array_equal(y0, np.array([lo(_R(orc, FIRST + e, 0x4100 + j)) for e in range(COUNT)], dtype=np.uint64))
            assert np.array_equal((y0 + y1) & np.uint64(mask), r_out[j]), spec.name + ": r_out shares"
        off += sh["n_out_a"] * s8
    # kappa^A [.][s8], one [s8] word of kappa^B bits if the gate has any, then Beaver (a, b, c)[M_A][3][s8]
    off += len(spec.kappa_a) * s8 + (s8 if sh["n_kb"] > 0 else 0)
    for i in range(sh["M_A"]):
        ab = [_R(orc, FIRST + e, 0x6000 + i) for e in range(COUNT)]
        ab0 = [_R(orc, FIRST + e, 0x6800 + i) for e in range(COUNT)]
        c0 = [_R(orc, FIRST + e, 0x7000 + i) for e in range(COUNT)]
        want = [([lo(v) for v in ab0], [(lo(a) - lo(v)) & mask for a, v in zip(ab, ab0)]),
                ([hi(v) for v in ab0], [(hi(a) - hi(v)) & mask for a, v in zip(ab, ab0)]),
                ([lo(v) for v in c0], [(lo(a) * hi(a) - lo(v)) & mask for a, v in zip(ab, c0)])]
        for j, (e0, e1) in enumerate(want):
            o = off + (3 * i + j) * s8
            assert np.array_equal(_words(k0, o), np.array(e0, dtype=np.uint64)), (spec.name, "Beaver", i, j, 0)
            assert np.array_equal(_words(k1, o), np.array(e1, dtype=np.uint64)), (spec.name, "Beaver", i, j, 1)
    assert off + 3 * sh["M_A"] * s8 <= O.key_bytes(COUNT)
