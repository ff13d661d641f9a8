"""Oracle composition of the softmax vector block (TEST INFRASTRUCTURE; App. G):
e_i = nExp(x_i) -> truncate -> s = sum_i e_i -> t = Recip(s) -> truncate -> y_i = e_i * t (Beaver) -> truncate.
Every scalar gate is the oracle's own Program (keygen, the two FSS calls, post-processing); the linear steps and
the Beaver product are written out in numpy.  The max reduction is not part of the method: inputs are
max-subtracted scores."""
from __future__ import annotations

import numpy as np

import oracle

SLOT_MUL_AB, SLOT_MUL_AB0, SLOT_MUL_C0 = 0xA000, 0xA001, 0xA002
BLOCK_SOFTMAX, BLOCK_LAYERNORM = 1, 2


def stage_seed(seed, block, stage):
    """Dealer seed of stage `stage` of a block instance (DESIGN 12): a counter-based derivation -- the splitmix64 output function
    applied to seed + golden * (16 block + stage + 1) -- so that stages of one block, and the softmax and LayerNorm blocks keyed with
    the same block seed, draw unrelated randomness (seed + small offsets collided across blocks)."""
    m = (1 << 64) - 1
    z = (int(seed) + 0x9E3779B97F4A7C15 * (16 * block + stage + 1)) & m
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & m
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & m
    return z ^ (z >> 31)


def gate(P, x0, x1, r_in, seed, first=0, offset=0, r_out=None, opened=False):
    """One compiled gate on additively shared inputs: Protocol 1 (masked opening), then the online procedure.
    `offset` = public constant added to the gate input (2^63 for the signed truncation gate workloads.specs.ars).
    r_out: output mask of a gate compiled with mask_output (its outputs are then shares of yhat = y + r_out).
    opened: (x0, x1) are the producer's shares of yhat with r_out(producer) = this gate's r_in, so xhat = x0 + x1 (step 6)."""
    count = x0.size
    k0, k1 = P.keygen(r_in, None if r_out is None else r_out.reshape(1, -1), seed, first)
    if opened:
        xhat = x0 + x1 + np.uint64(offset)
    else:
        xhat = x0 + P.rin_shares(k0, count) + x1 + P.rin_shares(k1, count) + np.uint64(offset)   # n = 64: wraps mod 2^64
    out = P.run_gate(k0, k1, xhat)
    return out["y"][0][0], out["y"][1][0], xhat


def beaver_mul(x0, x1, y0, y1, cols, seed, first=0):
    """z = x * y with y broadcast over `cols` consecutive elements; triples from R(e, 0xA000..)."""
    count = x0.size
    a, b = oracle.dealer_rand(seed, first, count, SLOT_MUL_AB)
    a0, b0 = oracle.dealer_rand(seed, first, count, SLOT_MUL_AB0)
    c0, _ = oracle.dealer_rand(seed, first, count, SLOT_MUL_C0)
    c = a * b
    a1, b1, c1 = a - a0, b - b0, c - c0
    yi = np.arange(count) // cols
    E = (x0 - a0) + (x1 - a1)
    Fv = (y0[yi] - b0) + (y1[yi] - b1)
    return E * Fv + E * b0 + Fv * a0 + c0, E * b1 + Fv * a1 + c1


def softmax(progs, x0, x1, masks, rows, cols, seed, fused_open=False):
    """progs / masks: dicts with the stages 'nexp', 'tr_e', 'recip', 'tr_t', 'tr_y' (oracle Programs / r_in arrays).
    fused_open: nExp and Recip are mask_output gates keyed with r_out = the following truncation gate's r_in; their opened
    yhat is that gate's xhat (then out['e'], out['t'] are shares of the MASKED values)."""
    fo = fused_open
    SS = lambda stage: stage_seed(seed, BLOCK_SOFTMAX, stage)
    with np.errstate(over="ignore"):
        e0, e1, _ = gate(progs["nexp"], x0, x1, masks["nexp"], SS(1), r_out=masks["tr_e"] if fo else None)
        f0, f1, _ = gate(progs["tr_e"], e0, e1, masks["tr_e"], SS(2), opened=fo)
        s0, s1 = f0.reshape(rows, cols).sum(axis=1, dtype=np.uint64), f1.reshape(rows, cols).sum(axis=1, dtype=np.uint64)
        t0, t1, _ = gate(progs["recip"], s0, s1, masks["recip"], SS(3), r_out=masks["tr_t"] if fo else None)
        u0, u1, _ = gate(progs["tr_t"], t0, t1, masks["tr_t"], SS(4), opened=fo)
        p0, p1 = beaver_mul(f0, f1, u0, u1, cols, SS(5))
        y0, y1, _ = gate(progs["tr_y"], p0, p1, masks["tr_y"], SS(6))
    return dict(e=(e0, e1), f=(f0, f1), s=(s0, s1), t=(t0, t1), u=(u0, u1), p=(p0, p1), y=(y0, y1))


def softmax_plain(progs, x, rows, cols):
    """Tier A: the same pipeline on cleartext fixed-point values (exact integer semantics of every stage)."""
    z = np.zeros(x.size, np.uint64)
    with np.errstate(over="ignore"):
        e = progs["nexp"].plain_G(x, z)[0][0]
        f = progs["tr_e"].plain_G(e, z)[0][0]
        s = f.reshape(rows, cols).sum(axis=1, dtype=np.uint64)
        zr = np.zeros(rows, np.uint64)
        t = progs["recip"].plain_G(s, zr)[0][0]
        u = progs["tr_t"].plain_G(t, zr)[0][0]
        p = f * np.repeat(u, cols)
        y = progs["tr_y"].plain_G(p, z)[0][0]
    return dict(e=e, f=f, s=s, t=t, u=u, p=p, y=y)


HALF = 1 << 63


def layernorm(progs, x0, x1, masks, rows, d, seed, fused_open=False):
    """LayerNorm without affine parameters on rows of length d = 2^k at scale 2^12 (App. G: mean / variance reductions
    are linear, rsqrt is a compiled gate):  mu = ARS_k(sum x); c = x - mu; v = ARS_{k+12}(sum c^2); g = rsqrt(v) (scale
    2^48) -> ARS_24; y = ARS_24(c * g).  progs / masks: stages 'mean', 'var', 'rsqrt', 'tr_g', 'tr_y'."""
    SS = lambda stage: stage_seed(seed, BLOCK_LAYERNORM, stage)
    with np.errstate(over="ignore"):
        rs = lambda a: a.reshape(rows, d).sum(axis=1, dtype=np.uint64)
        m0, m1, _ = gate(progs["mean"], rs(x0), rs(x1), masks["mean"], SS(1), offset=HALF)
        c0, c1 = x0 - np.repeat(m0, d), x1 - np.repeat(m1, d)
        q0, q1 = beaver_mul(c0, c1, c0, c1, 1, SS(2))
        v0, v1, _ = gate(progs["var"], rs(q0), rs(q1), masks["var"], SS(3), offset=HALF)
        g0, g1, _ = gate(progs["rsqrt"], v0, v1, masks["rsqrt"], SS(4), r_out=masks["tr_g"] if fused_open else None)
        h0, h1, _ = gate(progs["tr_g"], g0, g1, masks["tr_g"], SS(5), offset=HALF, opened=fused_open)
        p0, p1 = beaver_mul(c0, c1, h0, h1, d, SS(6))
        y0, y1, _ = gate(progs["tr_y"], p0, p1, masks["tr_y"], SS(7), offset=HALF)
    return dict(m=(m0, m1), c=(c0, c1), q=(q0, q1), v=(v0, v1), g=(g0, g1), h=(h0, h1), p=(p0, p1), y=(y0, y1))


def layernorm_plain(progs, x, rows, d):
    """Tier A: the same pipeline on cleartext fixed-point values."""
    zr, z = np.zeros(rows, np.uint64), np.zeros(x.size, np.uint64)
    H = np.uint64(HALF)
    with np.errstate(over="ignore"):
        rs = lambda a: a.reshape(rows, d).sum(axis=1, dtype=np.uint64)
        m = progs["mean"].plain_G(rs(x) + H, zr)[0][0]
        c = x - np.repeat(m, d)
        q = c * c
        v = progs["var"].plain_G(rs(q) + H, zr)[0][0]
        g = progs["rsqrt"].plain_G(v, zr)[0][0]
        h = progs["tr_g"].plain_G(g + H, zr)[0][0]
        p = c * np.repeat(h, d)
        y = progs["tr_y"].plain_G(p + H, z)[0][0]
    return dict(m=m, c=c, q=q, v=v, g=g, h=h, p=p, y=y)
