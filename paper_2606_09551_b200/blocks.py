"""Vector blocks composed from compiled gates (App. G).

softmax over max-subtracted scores:  e = nExp(x) -> truncate -> s = sum_i e_i -> t = Recip(s) -> truncate ->
y_i = e_i * t (Beaver) -> truncate.  The max reduction is not compiled by the method and is not here.
This module only ORCHESTRATES C-ABI calls (argument marshalling): every step -- masked openings, the gates'
keygen / FSS evaluation / post-processing, row sums, Beaver products -- runs in libfusefss kernels.
Both parties run on one GPU; the bytes they would exchange are counted.
"""
from __future__ import annotations

import numpy as np

from . import Program, _check, _ptr, _stream, lib

STAGES = ("nexp", "tr_e", "recip", "tr_t", "tr_y")

_M64 = (1 << 64) - 1


def _stage_seed(seed: int, block: int, stage: int) -> int:
    """Per-stage dealer seed (DESIGN 12): splitmix64's finaliser over seed + 0x9E3779B97F4A7C15 (16 block + stage + 1); block 1 =
    softmax, 2 = LayerNorm.  Keeps the stages of a block and different blocks under one block seed on unrelated randomness."""
    z = (seed + 0x9E3779B97F4A7C15 * (16 * block + stage + 1)) & _M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
    return z ^ (z >> 31)


# gate -> gate edges: the producer is compiled with mask_output and keyed with r_out = the consumer's r_in, so that the opened
# yhat of the producer IS the consumer's xhat (online step 6; masked-wire invariant P:89-91)
FUSED_EDGES = {"nexp": "tr_e", "recip": "tr_t"}
LN_FUSED_EDGES = {"rsqrt": "tr_g"}


def softmax_specs(variant: int = 3, n: int = 64, f: int = 12, fused_open: bool = False):
    """Gate types of the block: nExp (out scale 2f+8), arithmetic shifts by 20 / 28 / 24 bits (as shift+ReLU gates:
    every value here is non-negative), Recip (out scale 3f+16).  Scales: e at 32 -> 12; t at 52 -> 24; e*t at 36 -> 12."""
    from workloads import specs as S
    mk = {"nexp": S.nexp(n, f), "tr_e": S.shift_relu(n, 20), "recip": S.recip(n, f), "tr_t": S.shift_relu(n, 28),
          "tr_y": S.shift_relu(n, 24)}
    out = {}
    for k, s in mk.items():
        if variant & 1:
            s = S.shared_prefix(s)
        if variant & 2:
            s = S.input_masked_mul(s)
        if variant & 4:
            s = S.public_point_horner(s)
        if fused_open and k in FUSED_EDGES:
            import dataclasses
            s = dataclasses.replace(s, mask_output=True)
        out[k] = s
    return out


class Softmax:
    """rows x cols block.  `keygen(masks, seed)` is the dealer; `run(x0, x1)` the online phase of both parties."""

    def __init__(self, rows: int, cols: int, variant: int = 3, fused_open: bool = False):
        import torch
        self.rows, self.cols, self.N = rows, cols, rows * cols
        self.edges = FUSED_EDGES if fused_open else {}
        self.specs = softmax_specs(variant, fused_open=fused_open)
        self.progs = {k: Program(s) for k, s in self.specs.items()}
        self.n = 64
        self.counts = {"nexp": self.N, "tr_e": self.N, "recip": rows, "tr_t": rows, "tr_y": self.N}
        self.keys = {k: self.progs[k].alloc_keys(c) for k, c in self.counts.items()}
        tb = lib.fusefss_mul_triple_bytes(self.N)
        self.triples = (torch.empty(tb, dtype=torch.uint8, device="cuda"), torch.empty(tb, dtype=torch.uint8, device="cuda"))
        i64 = lambda *shape: torch.empty(shape, dtype=torch.int64, device="cuda")
        self.buf = {k: dict(xhat=i64(c), bits=[i64(c), i64(c)], coeff=[i64(self.progs[k].shape["p"], c) for _ in (0, 1)],
                            out=(i64(1, c), i64(1, c), i64(c), i64(c))) for k, c in self.counts.items()}
        self.s = [i64(rows), i64(rows)]
        self.prod = [i64(self.N), i64(self.N)]

    # ---- dealer ----------------------------------------------------------------------------------
    def keygen(self, masks, seed: int):
        """masks[stage] = device uint64 tensor of fresh input masks r_in for that gate instance."""
        for i, k in enumerate(STAGES):
            st_seed = _stage_seed(seed, 1, (1, 2, 3, 4, 6)[i])
            r_out = masks[self.edges[k]].reshape(1, -1) if k in self.edges else None     # r_out(k) = r_in(consumer)
            self.progs[k].keygen(masks[k], r_out, st_seed, 0, keys=self.keys[k])
        _check(lib.fusefss_mul_keygen(self.n, _stage_seed(seed, 1, 5), 0, self.N, _ptr(self.triples[0]), _ptr(self.triples[1]), _stream()))

    # ---- online ----------------------------------------------------------------------------------
    def _gate(self, k, x0, x1, offset=0, opened=False):
        """opened: (x0, x1) are the producer's shares of yhat = y + r_out with r_out = this gate's r_in: xhat = their sum"""
        P, (k0, k1), b, c = self.progs[k], self.keys[k], self.buf[k], self.counts[k]
        if opened:
            _check(lib.fusefss_open_output(self.n, _ptr(x0), _ptr(x1), c, offset, _ptr(b["xhat"]), _stream()))
        else:
            _check(lib.fusefss_share_open(P._h, _ptr(k0), _ptr(k1), _ptr(x0), _ptr(x1), c, offset, _ptr(b["xhat"]), _stream()))
        P.eval_fused_both(k0, k1, b["xhat"], b["bits"] if P.shape["T"] else None, b["coeff"] if P.shape["has_lut"] else None)
        y0, y1, _, _ = P.post_fused(k0, k1, b["xhat"], b["bits"][0], b["bits"][1], b["coeff"][0], b["coeff"][1], outs=b["out"])
        return y0[0], y1[0]

    def run(self, x0, x1):
        """x0, x1: additive shares [rows*cols] of the max-subtracted scores at scale 2^12.  Returns shares of softmax at 2^12."""
        e0, e1 = self._gate("nexp", x0, x1)
        f0, f1 = self._gate("tr_e", e0, e1, opened="nexp" in self.edges)
        for b, fb in ((0, f0), (1, f1)):
            _check(lib.fusefss_row_sum(self.n, _ptr(fb), self.rows, self.cols, _ptr(self.s[b]), _stream()))
        t0, t1 = self._gate("recip", self.s[0], self.s[1])
        u0, u1 = self._gate("tr_t", t0, t1, opened="recip" in self.edges)
        _check(lib.fusefss_mul_fused(self.n, _ptr(f0), _ptr(f1), _ptr(u0), _ptr(u1), _ptr(self.triples[0]), _ptr(self.triples[1]),
                                     self.N, self.cols, _ptr(self.prod[0]), _ptr(self.prod[1]), _stream()))
        y0, y1 = self._gate("tr_y", self.prod[0], self.prod[1])
        return dict(e=(e0, e1), f=(f0, f1), s=tuple(self.s), t=(t0, t1), u=(u0, u1), p=tuple(self.prod), y=(y0, y1))

    # ---- accounting ------------------------------------------------------------------------------
    def online_bytes_per_party(self) -> int:
        """openings of every gate input + the gates' own post-processing messages + 2 ring elements per Beaver product"""
        total = sum(self.progs[k].online_bits() // 8 * c for k, c in self.counts.items())
        total -= sum(self.n // 8 * self.counts[consumer] for consumer in self.edges.values())   # a fused wire is opened once: the producer's yhat IS the consumer's xhat
        return total + 16 * self.N

    def key_bytes_per_party(self) -> int:
        return sum(self.progs[k].key_bytes(c) for k, c in self.counts.items()) + lib.fusefss_mul_triple_bytes(self.N)

    def rounds(self) -> int:
        return sum(1 + self.progs[k].post_rounds() for k in STAGES) + 1


def _apply_variant(s, variant):
    from workloads import specs as S
    if variant & 1:
        s = S.shared_prefix(s)
    if variant & 2:
        s = S.input_masked_mul(s)
    if variant & 4:
        s = S.public_point_horner(s)
    return s


class LayerNorm(Softmax):
    """rows x d block, d = 2^k, no affine parameters, inputs at scale 2^12 (App. G: mean / variance reductions are linear,
    rsqrt is a compiled gate; config 4b):  mu = ARS_k(sum x); c = x - mu; v = ARS_{k+12}(sum c^2); g = rsqrt(v) (scale 2^48)
    -> ARS_24; y = ARS_24(c * g).  The signed truncations are `workloads.specs.ars` gates fed with xhat + 2^63."""
    LN_STAGES = ("mean", "var", "rsqrt", "tr_g", "tr_y")
    HALF = 1 << 63

    def __init__(self, rows: int, d: int, variant: int = 3, fused_open: bool = False):
        import dataclasses
        import torch
        from workloads import specs as S
        self.edges = LN_FUSED_EDGES if fused_open else {}
        k = d.bit_length() - 1
        if d != 1 << k:
            raise ValueError("LayerNorm block: d must be a power of two (the mean is a truncation gate)")
        self.rows, self.cols, self.N, self.n = rows, d, rows * d, 64
        mk = {"mean": S.ars(64, k), "var": S.ars(64, k + 12), "rsqrt": S.rsqrt(64, 12), "tr_g": S.ars(64, 24), "tr_y": S.ars(64, 24)}
        self.specs = {kk: _apply_variant(s, variant) for kk, s in mk.items()}
        for kk in self.edges:
            self.specs[kk] = dataclasses.replace(self.specs[kk], mask_output=True)
        self.progs = {kk: Program(s) for kk, s in self.specs.items()}
        self.counts = {"mean": rows, "var": rows, "rsqrt": rows, "tr_g": rows, "tr_y": self.N}
        self.keys = {kk: self.progs[kk].alloc_keys(c) for kk, c in self.counts.items()}
        tb = lib.fusefss_mul_triple_bytes(self.N)
        u8 = lambda: torch.empty(tb, dtype=torch.uint8, device="cuda")
        self.triples_sq, self.triples = (u8(), u8()), (u8(), u8())
        i64 = lambda *shape: torch.empty(shape, dtype=torch.int64, device="cuda")
        self.buf = {kk: dict(xhat=i64(c), bits=[i64(c), i64(c)], coeff=[i64(self.progs[kk].shape["p"], c) for _ in (0, 1)],
                             out=(i64(1, c), i64(1, c), i64(c), i64(c))) for kk, c in self.counts.items()}
        self.s = [i64(rows), i64(rows)]
        self.ssq = [i64(rows), i64(rows)]
        self.c = [i64(self.N), i64(self.N)]
        self.sq = [i64(self.N), i64(self.N)]
        self.prod = [i64(self.N), i64(self.N)]

    def keygen(self, masks, seed: int):
        for kk, off in zip(self.LN_STAGES, (1, 3, 4, 5, 7)):
            r_out = masks[self.edges[kk]].reshape(1, -1) if kk in self.edges else None
            self.progs[kk].keygen(masks[kk], r_out, _stage_seed(seed, 2, off), 0, keys=self.keys[kk])
        _check(lib.fusefss_mul_keygen(self.n, _stage_seed(seed, 2, 2), 0, self.N, _ptr(self.triples_sq[0]), _ptr(self.triples_sq[1]), _stream()))
        _check(lib.fusefss_mul_keygen(self.n, _stage_seed(seed, 2, 6), 0, self.N, _ptr(self.triples[0]), _ptr(self.triples[1]), _stream()))

    def run(self, x0, x1):
        H, st = self.HALF, _stream()
        for b, xb in ((0, x0), (1, x1)):
            _check(lib.fusefss_row_sum(self.n, _ptr(xb), self.rows, self.cols, _ptr(self.s[b]), st))
        m0, m1 = self._gate("mean", self.s[0], self.s[1], H)
        for b, (xb, mb) in enumerate(((x0, m0), (x1, m1))):
            _check(lib.fusefss_sub_bcast(self.n, _ptr(xb), _ptr(mb), self.N, self.cols, _ptr(self.c[b]), st))
        c0, c1 = self.c
        _check(lib.fusefss_mul_fused(self.n, _ptr(c0), _ptr(c1), _ptr(c0), _ptr(c1), _ptr(self.triples_sq[0]), _ptr(self.triples_sq[1]),
                                     self.N, 1, _ptr(self.sq[0]), _ptr(self.sq[1]), st))
        for b in (0, 1):
            _check(lib.fusefss_row_sum(self.n, _ptr(self.sq[b]), self.rows, self.cols, _ptr(self.ssq[b]), st))
        v0, v1 = self._gate("var", self.ssq[0], self.ssq[1], H)
        g0, g1 = self._gate("rsqrt", v0, v1)
        h0, h1 = self._gate("tr_g", g0, g1, H, opened="rsqrt" in self.edges)
        _check(lib.fusefss_mul_fused(self.n, _ptr(c0), _ptr(c1), _ptr(h0), _ptr(h1), _ptr(self.triples[0]), _ptr(self.triples[1]),
                                     self.N, self.cols, _ptr(self.prod[0]), _ptr(self.prod[1]), st))
        y0, y1 = self._gate("tr_y", self.prod[0], self.prod[1], H)
        return dict(m=(m0, m1), c=(c0, c1), q=tuple(self.sq), v=(v0, v1), g=(g0, g1), h=(h0, h1), p=tuple(self.prod), y=(y0, y1))

    def online_bytes_per_party(self) -> int:
        fused = sum(self.n // 8 * self.counts[consumer] for consumer in self.edges.values())     # a fused wire is opened once
        return sum(self.progs[k].online_bits() // 8 * c for k, c in self.counts.items()) - fused + 2 * 16 * self.N

    def key_bytes_per_party(self) -> int:
        return sum(self.progs[k].key_bytes(c) for k, c in self.counts.items()) + 2 * lib.fusefss_mul_triple_bytes(self.N)

    def rounds(self) -> int:
        return sum(1 + self.progs[k].post_rounds() for k in self.LN_STAGES) + 2


def bench(F, torch, steps: int = 3):
    """bench.py --blocks: dealer and online time of the softmax block (config 3's shape, 12 heads x 128 rows of 128) and of the
    LayerNorm block (config 4b's shape, 1024 tokens x d = 1024); CUDA events, both parties on one GPU."""
    ev = lambda: torch.cuda.Event(enable_timing=True)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.int64)).cuda()
    rng = np.random.default_rng(5)
    U = lambda k: rng.integers(0, 1 << 63, size=k, dtype=np.uint64) * np.uint64(2) + rng.integers(0, 2, size=k, dtype=np.uint64)
    out = {}

    def time_block(B, masks, x0d, x1d):
        for _ in range(3):
            B.keygen(masks, 9); res = B.run(x0d, x1d)
        torch.cuda.synchronize()
        e = [ev() for _ in range(3)]
        e[0].record()
        for _ in range(steps):
            B.keygen(masks, 9)
        e[1].record()
        for _ in range(steps):
            res = B.run(x0d, x1d)
        e[2].record()
        torch.cuda.synchronize()
        return res, e[0].elapsed_time(e[1]) / steps, e[1].elapsed_time(e[2]) / steps

    rows, cols = 12 * 128, 128
    xr = np.maximum(-20.0, -4.0 * rng.exponential(1.0, size=(rows, cols))); xr[:, 0] = 0.0
    xq = np.floor(xr.reshape(-1) * 4096 + 0.5).astype(np.int64).view(np.uint64)
    x0h = U(xq.size)
    masks = {k: dev(U(c)) for k, c in (("nexp", xq.size), ("tr_e", xq.size), ("recip", rows), ("tr_t", rows), ("tr_y", xq.size))}
    blk = {}
    for v, fo in ((3, False), (3, True), (0, False)):       # fo: gate -> gate edges through the opened yhat (DESIGN 16)
        B = Softmax(rows, cols, v, fused_open=fo)
        res, t_deal, t_on = time_block(B, masks, dev(x0h), dev(xq - x0h))
        y = (res["y"][0] + res["y"][1]).cpu().numpy().astype(np.float64).reshape(rows, cols) / 4096.0
        ref = np.exp(xr) / np.exp(xr).sum(axis=1, keepdims=True)
        blk["variant_%d%s" % (v, "_fused_open" if fo else "")] = {"rows": rows, "cols": cols, "dealer_ms": t_deal, "online_ms": t_on, "online_elems_per_s": rows * cols / (t_on * 1e-3),
                                 "key_bytes_per_elem_per_party": B.key_bytes_per_party() / (rows * cols),
                                 "online_bytes_per_elem_per_party": B.online_bytes_per_party() / (rows * cols), "rounds": B.rounds(),
                                 "max_abs_err_vs_float_softmax": float(np.abs(y - ref).max())}
        del B
        torch.cuda.empty_cache()
    out["softmax_block"] = blk
    rows, d = 1024, 1024
    xr = rng.normal(0.0, 2.0, size=(rows, d))
    xq = np.floor(xr.reshape(-1) * 4096 + 0.5).astype(np.int64).view(np.uint64)
    x0h = U(xq.size)
    masks = {k: dev(U(c)) for k, c in (("mean", rows), ("var", rows), ("rsqrt", rows), ("tr_g", rows), ("tr_y", xq.size))}
    xf = xq.view(np.int64).astype(np.float64).reshape(rows, d) / 4096.0
    ref = (xf - xf.mean(axis=1, keepdims=True)) / xf.std(axis=1, keepdims=True)
    out["layernorm_block"] = {}
    for fo in (False, True):
        B = LayerNorm(rows, d, 3, fused_open=fo)
        res, t_deal, t_on = time_block(B, masks, dev(x0h), dev(xq - x0h))
        y = (res["y"][0] + res["y"][1]).cpu().numpy().astype(np.float64).reshape(rows, d) / 4096.0
        out["layernorm_block"]["variant_3" + ("_fused_open" if fo else "")] = {
            "rows": rows, "d": d, "dealer_ms": t_deal, "online_ms": t_on, "online_elems_per_s": rows * d / (t_on * 1e-3),
            "key_bytes_per_elem_per_party": B.key_bytes_per_party() / (rows * d),
            "online_bytes_per_elem_per_party": B.online_bytes_per_party() / (rows * d), "rounds": B.rounds(),
            "max_abs_err_vs_float_layernorm": float(np.abs(y - ref).max())}
        del B
        torch.cuda.empty_cache()
    return out
