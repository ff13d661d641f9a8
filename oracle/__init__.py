"""CPU oracle for the FuseFSS hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes loader around ``oracle/fusefss_oracle.c`` (plain C, built with gcc by
``oracle.build()`` / ``__graft_entry__.build()``).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package; it shares no code with ``paper_2606_09551_b200``.
See the header of ``fusefss_oracle.c`` for citations and DESIGN.md sections 3-4.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fusefss_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O3, single thread, no OpenMP, no intrinsics)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O3", "-std=gnu11", "-shared", "-fPIC", "-o", _LIB, _SRC])
    return _LIB


class _BitNode(C.Structure):
    _fields_ = [("kind", C.c_uint8), ("k", C.c_uint8), ("lhs", C.c_uint16), ("rhs", C.c_uint16),
                ("value_is_2k", C.c_uint8), ("pad", C.c_uint8), ("value", C.c_uint64)]


class _Kappa(C.Structure):
    _fields_ = [("kind", C.c_uint8), ("arg", C.c_uint8)]


class _PhiOp(C.Structure):
    _fields_ = [("op", C.c_uint8), ("dst", C.c_uint8), ("a", C.c_uint8), ("b", C.c_uint8),
                ("pad", C.c_uint32), ("imm", C.c_uint64)]


class _Spec(C.Structure):
    _fields_ = [(k, C.c_uint32) for k in (
        "n", "frac_bits", "m", "r", "d", "p_aux", "ell", "n_nodes", "n_kappa_a", "n_kappa_b", "phi_len",
        "n_out_a", "n_out_b", "mask_output", "variant")] + [
        ("alpha", C.c_void_p), ("coeff", C.c_void_p), ("aux", C.c_void_p), ("nodes", C.c_void_p),
        ("bit_root", C.c_void_p), ("kappa_a", C.c_void_p), ("kappa_b", C.c_void_p), ("phi", C.c_void_p)]


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.orc_compile.restype = C.c_void_p
        L.orc_compile.argtypes = [C.c_void_p]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_key_bytes.restype = C.c_size_t
        L.orc_key_bytes.argtypes = [C.c_void_p, C.c_size_t]
        L.orc_post_msg_bytes.restype = C.c_size_t
        L.orc_post_msg_bytes.argtypes = [C.c_void_p, C.c_size_t, C.c_int]
        L.orc_post_rounds.restype = C.c_int
        L.orc_post_rounds.argtypes = [C.c_void_p]
        L.orc_online_bits.restype = C.c_size_t
        L.orc_online_bits.argtypes = [C.c_void_p]
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None and a.size else None


def _u64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.uint64))


class _SpecHolder:
    """Marshals a workloads.specs.OpSpec into the oracle's own C struct (keeps the arrays alive)."""

    def __init__(self, s):
        self.alpha = _u64(s.alpha)
        self.coeff = _u64(s.coeff).reshape(-1)
        self.aux = _u64(s.aux).reshape(-1)
        self.nodes = (_BitNode * max(1, len(s.nodes)))()
        for i, (kind, k, lhs, rhs, is2k, value) in enumerate(s.nodes):
            self.nodes[i] = _BitNode(kind, k, lhs, rhs, is2k, 0, value)
        self.bit_root = np.ascontiguousarray(np.asarray(s.bit_root, dtype=np.uint16)).reshape(-1)
        self.ka = (_Kappa * max(1, len(s.kappa_a)))(*[_Kappa(*k) for k in s.kappa_a])
        self.kb = (_Kappa * max(1, len(s.kappa_b)))(*[_Kappa(*k) for k in s.kappa_b])
        self.phi = (_PhiOp * max(1, len(s.phi)))()
        for i, (op, dst, a, b, imm) in enumerate(s.phi):
            self.phi[i] = _PhiOp(op, dst, a, b, 0, imm & 0xFFFFFFFFFFFFFFFF)
        self.c = _Spec(s.n, s.f, s.m, s.r, s.d, s.p_aux, s.ell, len(s.nodes), len(s.kappa_a), len(s.kappa_b),
                       len(s.phi), s.n_out_a, s.n_out_b, int(s.mask_output), int(getattr(s, "variant", 0)),
                       _p(self.alpha), _p(self.coeff), _p(self.aux), C.cast(self.nodes, C.c_void_p),
                       _p(self.bit_root), C.cast(self.ka, C.c_void_p), C.cast(self.kb, C.c_void_p),
                       C.cast(self.phi, C.c_void_p))


SHAPE_KEYS = ("T", "M", "p", "M_A", "M_B", "G_mix", "rounds", "n_out_a", "n_out_b", "has_lut", "n_kb")


class Program:
    """Compiled gate type (oracle side)."""

    def __init__(self, spec):
        self.spec = spec
        self._h = _SpecHolder(spec)
        self._p = lib().orc_compile(C.byref(self._h.c))
        if not self._p:
            raise ValueError("oracle: ill-formed operator specification")
        out = (C.c_int * 11)()
        ks = (C.c_int * 64)()
        lib().orc_shape(C.c_void_p(self._p), out, ks)
        self.shape = dict(zip(SHAPE_KEYS, list(out)))
        self.shape["k"] = list(ks)[: self.shape["T"]]

    def __del__(self):
        if getattr(self, "_p", None):
            lib().orc_destroy(C.c_void_p(self._p))
            self._p = None

    def atom(self, t):
        out = (C.c_uint64 * 4)()
        lib().orc_atom(C.c_void_p(self._p), t, out)
        return dict(k=int(out[0]), c=int(out[1]), is_theta=int(out[2]), beta=int(out[3]))

    def key_bytes(self, count):
        return lib().orc_key_bytes(C.c_void_p(self._p), count)

    def post_rounds(self):
        return lib().orc_post_rounds(C.c_void_p(self._p))

    def post_msg_bytes(self, count, rnd):
        return lib().orc_post_msg_bytes(C.c_void_p(self._p), count, rnd)

    def online_bits(self):
        return lib().orc_online_bits(C.c_void_p(self._p))

    def keygen(self, r_in, r_out, seed, first_elem=0):
        r_in = _u64(r_in)
        count = r_in.size
        n_out = self.shape["n_out_a"]
        r_out = _u64(r_out).reshape(-1) if r_out is not None else np.zeros(n_out * count, np.uint64)
        kb = self.key_bytes(count)
        k0 = np.zeros(kb, np.uint8)
        k1 = np.zeros(kb, np.uint8)
        lib().orc_keygen(C.c_void_p(self._p), _p(r_in), _p(r_out), C.c_uint64(seed), C.c_uint64(first_elem),
                         C.c_size_t(count), _p(k0), _p(k1))
        return k0, k1

    def eval_cmp(self, party, key, xhat):
        xhat = _u64(xhat)
        out = np.zeros(xhat.size, np.uint64)
        lib().orc_eval_cmp(party, C.c_void_p(self._p), _p(key), _p(xhat), C.c_size_t(xhat.size), _p(out))
        return out

    def eval_lut(self, party, key, xhat):
        xhat = _u64(xhat)
        out = np.zeros((self.shape["p"], xhat.size), np.uint64)
        lib().orc_eval_lut(party, C.c_void_p(self._p), _p(key), _p(xhat), C.c_size_t(xhat.size), _p(out))
        return out

    def msg_total(self, count):
        return sum(self.post_msg_bytes(count, q) for q in range(self.post_rounds()))

    def post(self, party, key, xhat, bits, coeff, rnd, msg_in, msg_out):
        """One party, one round.  msg_in = the OTHER party's message buffer, msg_out = this party's
        (both cover all rounds).  rnd == rounds -> returns (y [n_out_a, count], z words [count])."""
        xhat = _u64(xhat)
        count = xhat.size
        y = np.zeros((max(1, self.shape["n_out_a"]), count), np.uint64)
        z = np.zeros(count, np.uint64)
        lib().orc_post(party, C.c_void_p(self._p), _p(key), _p(xhat), _p(_u64(bits)), _p(_u64(coeff).reshape(-1)),
                       C.c_size_t(count), rnd, _p(msg_in), _p(msg_out), _p(y), _p(z))
        return y[: self.shape["n_out_a"]], z

    def run_gate(self, key0, key1, xhat):
        """Both parties, all rounds (the online procedure of P:868-875 after the xhat opening)."""
        xhat = _u64(xhat)
        count = xhat.size
        keys = (key0, key1)
        bits = [self.eval_cmp(b, keys[b], xhat) for b in (0, 1)]
        coeff = [self.eval_lut(b, keys[b], xhat) for b in (0, 1)]
        R = self.post_rounds()
        tot = max(1, self.msg_total(count))
        msg = [np.zeros(tot, np.uint8), np.zeros(tot, np.uint8)]
        for q in range(R):
            for b in (0, 1):
                self.post(b, keys[b], xhat, bits[b], coeff[b], q, msg[1 - b], msg[b])
        outs = [self.post(b, keys[b], xhat, bits[b], coeff[b], R, msg[1 - b], msg[b]) for b in (0, 1)]
        return dict(bits=bits, coeff=coeff, msg=msg, y=[outs[0][0], outs[1][0]], z=[outs[0][1], outs[1][1]])

    def rin_shares(self, key, count):
        out = np.zeros(count, np.uint64)
        lib().orc_rin_shares(C.c_void_p(self._p), _p(key), C.c_size_t(count), _p(out))
        return out

    # ---- Tier A -------------------------------------------------------------------------------
    def plain_G(self, x, r):
        x = _u64(x)
        r = _u64(r)
        na, nb = self.shape["n_out_a"], self.shape["n_out_b"]
        ys = np.zeros((x.size, max(1, na)), np.uint64)
        zs = np.zeros((x.size, max(1, nb)), np.uint8)
        f = lib().orc_plain_G
        sp = C.byref(self._h.c)
        for i in range(x.size):
            f(sp, C.c_uint64(int(x[i])), C.c_uint64(int(r[i])), C.c_void_p(ys[i].ctypes.data), C.c_void_p(zs[i].ctypes.data))
        return ys[:, :na].T.copy(), zs[:, :nb].T.copy()

    def plain_F(self, x, r=0):
        s = self.spec
        y = np.zeros(max(1, s.r), np.uint64)
        z = np.zeros(max(1, s.ell), np.uint8)
        aux = np.zeros(max(1, s.p_aux), np.uint64)
        lib().orc_plain_F(C.byref(self._h.c), C.c_uint64(int(x)), C.c_uint64(int(r)), _p(y), _p(z), _p(aux))
        return y[: s.r], z[: s.ell], aux[: s.p_aux]


# ---- primitives exposed for the pins -----------------------------------------------------------
def aes128_encrypt(key: bytes, block: bytes) -> bytes:
    out = C.create_string_buffer(16)
    lib().orc_aes128_encrypt(key, block, out)
    return out.raw


def prg(i: int, s: bytes, tau: int) -> bytes:
    out = C.create_string_buffer(16)
    lib().orc_prg(i, s, tau, out)
    return out.raw


def dcf_bit_pair(k, alpha, seed0: bytes, seed1: bytes, us):
    us = _u64(us)
    o0 = np.zeros(us.size, np.uint8)
    o1 = np.zeros(us.size, np.uint8)
    lib().orc_dcf_bit_pair(k, C.c_uint64(alpha), seed0, seed1, _p(us), us.size, _p(o0), _p(o1))
    return o0, o1


def dcf_bit_pair_et(k, alpha, seed0: bytes, seed1: bytes, us):
    """early-terminated bit-DCF (variant bit 3)"""
    us = _u64(us)
    o0 = np.zeros(us.size, np.uint8)
    o1 = np.zeros(us.size, np.uint8)
    lib().orc_dcf_bit_pair_et(k, C.c_uint64(alpha), seed0, seed1, _p(us), us.size, _p(o0), _p(o1))
    return o0, o1


def dcf_vec_pair(k, n, p, alpha, beta, seed0: bytes, seed1: bytes, us):
    us = _u64(us)
    beta = _u64(beta)
    o0 = np.zeros((us.size, p), np.uint64)
    o1 = np.zeros((us.size, p), np.uint64)
    lib().orc_dcf_vec_pair(k, n, p, C.c_uint64(alpha), _p(beta), seed0, seed1, _p(us), us.size, _p(o0), _p(o1))
    return o0, o1


def dealer_rand(seed, first, count, slot):
    lo = np.zeros(count, np.uint64)
    hi = np.zeros(count, np.uint64)
    lib().orc_dealer_rand(C.c_uint64(seed), C.c_uint64(first), C.c_size_t(count), C.c_uint64(slot), _p(lo), _p(hi))
    return lo, hi


def protocol3(n, alpha_interior, r):
    a = _u64(alpha_interior)
    m = a.size + 1
    B = np.zeros(m + 3, np.uint64)
    ord_ = np.zeros(m + 2, np.int32)
    M = C.c_int()
    lib().orc_protocol3(n, m, _p(a), C.c_uint64(r), _p(B), _p(ord_), C.byref(M))
    return [int(v) for v in B[: M.value + 1]], [int(v) for v in ord_[: M.value]], M.value
