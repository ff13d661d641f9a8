#!/usr/bin/env python
"""Generates bitslice_sbox.cuh: the AES S-box (FIPS-197 5.1.1) as a straight-line Boolean circuit on eight 32-bit bit-planes,
for the bitsliced-AES probe (fusefss_bitslice_probe; "T-tables or a bitsliced design, chosen by measurement").

Derivation (own; the textbook composite-field method): GF(2^8) = GF(2)[x]/(x^8+x^4+x^3+x+1) is isomorphic to the tower
GF(((2^2)^2)^2) with  z^2 = z + 1  over GF(2),  y^2 = y + z  over GF(2^2)  and  w^2 = w + LAM  over GF(2^4) (LAM found by
search).  The script finds a root of the AES polynomial in the tower (=> the 8x8 change-of-basis matrices), evaluates the inverse
x -> x^254 symbolically there -- for a = ah w + al:  d = ah^2 LAM + ah al + al^2,  a^-1 = (ah d^-1) w + (ah + al) d^-1 -- with
every bit a node of a hash-consed XOR/AND DAG, maps back, applies the affine layer, checks all 256 inputs against the S-box
computed from its definition, and prints the circuit.  Run:  python gen_bitslice_sbox.py > bitslice_sbox.cuh
"""
from __future__ import annotations

import sys


# ---- plain GF arithmetic (numbers) for the search and the final check ---------------------------------------------------------
def gf256_mul(a, b):
    p = 0
    for _ in range(8):
        if b & 1:
            p ^= a
        hi = a & 0x80
        a = (a << 1) & 0xFF
        if hi:
            a ^= 0x1B
        b >>= 1
    return p


def sbox_def(x):
    inv = 0
    if x:
        for y in range(1, 256):
            if gf256_mul(x, y) == 1:
                inv = y
                break
    r = inv
    for s in range(1, 5):
        r ^= ((inv << s) | (inv >> (8 - s))) & 0xFF
    return r ^ 0x63


# tower arithmetic on integers: GF(4) elements 0..3 (bit1 = z coefficient), GF(16) = (h, l) GF(4) pairs packed h<<2|l,
# GF(256) = (H, L) GF(16) pairs packed H<<4|L
def g4_mul(a, b):
    a1, a0, b1, b0 = a >> 1, a & 1, b >> 1, b & 1
    hh, ll = a1 & b1, a0 & b0
    mid = ((a1 ^ a0) & (b1 ^ b0)) ^ ll                       # a1 b0 + a0 b1 + a1 b1
    return ((mid) << 1) | (ll ^ hh)                            # z^2 = z + 1


def g16_mul(a, b, ):
    ah, al, bh, bl = a >> 2, a & 3, b >> 2, b & 3
    hh, ll = g4_mul(ah, bh), g4_mul(al, bl)
    mid = g4_mul(ah ^ al, bh ^ bl) ^ ll                        # ah bl + al bh + ah bh
    return ((mid) << 2) | (ll ^ g4_mul(hh, 2))                 # y^2 = y + z   (z = 2)


def g256_mul(a, b, lam):
    ah, al, bh, bl = a >> 4, a & 15, b >> 4, b & 15
    hh, ll = g16_mul(ah, bh), g16_mul(al, bl)
    mid = g16_mul(ah ^ al, bh ^ bl) ^ ll
    return (mid << 4) | (ll ^ g16_mul(hh, lam))                # w^2 = w + lam


def towers():
    """every (lam, powers of a root): lam makes w^2 + w + lam irreducible over GF(16), the root solves x^8+x^4+x^3+x+1 = 0 in
    the tower; each choice gives a different (equally valid) circuit -- the generator keeps the smallest."""
    for lam in range(1, 16):
        if any(g16_mul(t, t) ^ t ^ lam == 0 for t in range(16)):
            continue                                           # reducible
        for r in range(2, 256):
            pw = [1]
            for _ in range(8):
                pw.append(g256_mul(pw[-1], r, lam))
            if pw[8] ^ pw[4] ^ pw[3] ^ pw[1] ^ pw[0] == 0:
                yield lam, pw[:8]


# ---- symbolic XOR/AND DAG with hash-consing ---------------------------------------------------------------------------------
class Dag:
    def __init__(self):
        self.nodes = []            # (op, a, b); op in 'in', 'xor', 'and', 'not'
        self.memo = {}

    def _mk(self, op, a, b=-1):
        if op in ("xor", "and") and a > b:
            a, b = b, a
        key = (op, a, b)
        if key not in self.memo:
            self.nodes.append(key)
            self.memo[key] = len(self.nodes) - 1
        return self.memo[key]

    def inp(self, i):
        return self._mk("in", i)

    def xor(self, a, b):
        if a is None:
            return b
        if b is None:
            return a
        if a == b:
            return None
        return self._mk("xor", a, b)

    def and_(self, a, b):
        if a is None or b is None:
            return None
        if a == b:
            return a
        return self._mk("and", a, b)

    def not_(self, a):
        return self._mk("not", a)


def s4_mul(D, a, b):                                           # GF(4): a = (a1, a0)
    hh, ll = D.and_(a[0], b[0]), D.and_(a[1], b[1])
    mid = D.xor(D.and_(D.xor(a[0], a[1]), D.xor(b[0], b[1])), ll)
    return (mid, D.xor(ll, hh))


def s4_scale_z(D, a):                                          # a * z: (a1 z + a0) z = (a1 + a0) z + a1
    return (D.xor(a[0], a[1]), a[0])


def s4_sq(D, a):                                               # a^2 = a1 z^2 + a0 = a1 z + (a1 + a0)
    return (a[0], D.xor(a[0], a[1]))


def s4_add(D, a, b):
    return (D.xor(a[0], b[0]), D.xor(a[1], b[1]))


def s16_mul(D, a, b):                                          # GF(16): a = (ah, al), GF(4) pairs
    hh, ll = s4_mul(D, a[0], b[0]), s4_mul(D, a[1], b[1])
    mid = s4_add(D, s4_mul(D, s4_add(D, a[0], a[1]), s4_add(D, b[0], b[1])), ll)
    return (mid, s4_add(D, ll, s4_scale_z(D, hh)))


def s16_add(D, a, b):
    return (s4_add(D, a[0], b[0]), s4_add(D, a[1], b[1]))


def s16_sq(D, a):                                              # (ah y + al)^2 = ah^2 (y + z) + al^2
    h2, l2 = s4_sq(D, a[0]), s4_sq(D, a[1])
    return (h2, s4_add(D, l2, s4_scale_z(D, h2)))


def s16_inv(D, a):                                             # d = ah^2 z + ah al + al^2 in GF(4); d^-1 = d^2
    ah, al = a
    d = s4_add(D, s4_add(D, s4_scale_z(D, s4_sq(D, ah)), s4_mul(D, ah, al)), s4_sq(D, al))
    di = s4_sq(D, d)
    return (s4_mul(D, ah, di), s4_mul(D, s4_add(D, ah, al), di))


def s16_mul_const(D, a, c):
    """a * c for a constant c in GF(16): linear map, built from the images of the basis"""
    bits = [a[0][0], a[0][1], a[1][0], a[1][1]]               # weights 8, 4, 2, 1
    out = [None] * 4
    for i, w in enumerate((8, 4, 2, 1)):
        img = g16_mul(w, c)
        for j, ww in enumerate((8, 4, 2, 1)):
            if img & ww:
                out[j] = D.xor(out[j], bits[i])
    return ((out[0], out[1]), (out[2], out[3]))


def build(lam, pw):
    # tower element of the AES byte with bit i set = root^i; columns of the AES->tower matrix
    D = Dag()
    x = [D.inp(i) for i in range(8)]                           # x[i] = bit i of the input byte (plane i)
    t = [None] * 8                                             # tower bits, t[j] = bit j of the packed tower number
    for i in range(8):
        for j in range(8):
            if (pw[i] >> j) & 1:
                t[j] = D.xor(t[j], x[i])
    a_h = ((t[7], t[6]), (t[5], t[4]))
    a_l = ((t[3], t[2]), (t[1], t[0]))
    d = s16_add(D, s16_add(D, s16_mul_const(D, s16_sq(D, a_h), lam), s16_mul(D, a_h, a_l)), s16_sq(D, a_l))
    di = s16_inv(D, d)
    r_h, r_l = s16_mul(D, a_h, di), s16_mul(D, s16_add(D, a_h, a_l), di)
    rt = [r_l[1][1], r_l[1][0], r_l[0][1], r_l[0][0], r_h[1][1], r_h[1][0], r_h[0][1], r_h[0][0]]   # tower bits 0..7
    # tower -> AES basis: invert the matrix numerically (image of every tower unit vector)
    to_aes = {}
    for v in range(256):
        tw = 0
        for i in range(8):
            if (v >> i) & 1:
                tw ^= pw[i]
        to_aes[tw] = v
    inv_bits = [None] * 8
    for j in range(8):
        img = to_aes[1 << j]
        for i in range(8):
            if (img >> i) & 1:
                inv_bits[i] = D.xor(inv_bits[i], rt[j])
    out = []
    for i in range(8):                                         # affine layer: b_i = a_i + a_{i+4} + a_{i+5} + a_{i+6} + a_{i+7} + c_i
        v = None
        for k in (0, 4, 5, 6, 7):
            v = D.xor(v, inv_bits[(i + k) % 8])
        out.append((v, (0x63 >> i) & 1))
    return D, out, lam


def evaluate(D, out, byte):
    val = [0] * len(D.nodes)
    for i, (op, a, b) in enumerate(D.nodes):
        if op == "in":
            val[i] = (byte >> a) & 1
        elif op == "xor":
            val[i] = val[a] ^ val[b]
        elif op == "and":
            val[i] = val[a] & val[b]
        else:
            val[i] = val[a] ^ 1
    r = 0
    for i, (v, c) in enumerate(out):
        r |= ((0 if v is None else val[v]) ^ c) << i
    return r


def live_nodes(D, out):
    """only the nodes the outputs reach"""
    live = set()
    stack = [v for v, _ in out if v is not None]
    while stack:
        v = stack.pop()
        if v in live:
            continue
        live.add(v)
        op, a, b = D.nodes[v]
        if op != "in":
            stack.append(a)
            if b >= 0:
                stack.append(b)
    return live


def main():
    best = None
    for lam_, pw in towers():
        D_, out_, _ = build(lam_, pw)
        gates = sum(1 for v in live_nodes(D_, out_) if D_.nodes[v][0] != "in")
        if best is None or gates < best[0]:
            best = (gates, D_, out_, lam_)
    _, D, out, lam = best
    for b in range(256):
        assert evaluate(D, out, b) == sbox_def(b), b
    live = live_nodes(D, out)
    n_xor = sum(1 for v in live if D.nodes[v][0] == "xor")
    n_and = sum(1 for v in live if D.nodes[v][0] == "and")
    w = sys.stdout.write
    w("// bitslice_sbox.cuh -- GENERATED by gen_bitslice_sbox.py (composite-field S-box, checked against FIPS-197 5.1.1 for all 256\n")
    w("// inputs by the generator).  %d XOR + %d AND + 4 NOT on 32-bit planes; lam = %d.  Do not edit.\n" % (n_xor, n_and, lam))
    w("#pragma once\n#include <cstdint>\nnamespace fsk {\n")
    w("constexpr int kBitsliceSboxXor = %d, kBitsliceSboxAnd = %d;\n" % (n_xor, n_and))
    w("// in/out: x[i] = plane of bit i of the byte, for 32 blocks\n")
    w("__device__ __forceinline__ void bitslice_sbox(uint32_t (&x)[8]) {\n")
    for v in sorted(live):
        op, a, b = D.nodes[v]
        if op == "in":
            w("    const uint32_t n%d = x[%d];\n" % (v, a))
        elif op == "xor":
            w("    const uint32_t n%d = n%d ^ n%d;\n" % (v, a, b))
        elif op == "and":
            w("    const uint32_t n%d = n%d & n%d;\n" % (v, a, b))
    for i, (v, c) in enumerate(out):
        w("    x[%d] = %sn%d;\n" % (i, "~" if c else "", v))
    w("}\n}  // namespace fsk\n")


if __name__ == "__main__":
    main()
