"""Operator specifications (Def 4.1) and post-processing programs (Def 4.2,
PAPER.md:131-137, App. H) for BASELINE.json's configs -- INPUT DATA ONLY.

This module serves both the CPU oracle and the CUDA library (they each marshal an `OpSpec` into
their own C struct).  It holds none of the method's arithmetic: it only describes operators
(partitions, fixed-point spline coefficient tables, predicate DAGs, Phi bytecode).  The spline
tables are fitted here (the paper prints none) with a minimax LP per piece.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

# ---- encoding constants of the specification language (mirrors include/fusefss.h) -------------
BN_CONST, BN_C, BN_D, BN_MSB, BN_CARRY, BN_NOT, BN_XOR, BN_AND, BN_OR = range(9)
KA_R_SHR, KB_R_BIT = 1, 2
(PHI_A_CONST, PHI_A_X, PHI_A_Y, PHI_A_KAPPA, PHI_A_XHAT_SHR, PHI_A_ADD, PHI_A_SUB, PHI_A_MULC, PHI_A_MUL,
 PHI_A_B2A, PHI_A_OUT, PHI_A_AUX) = range(1, 13)
(PHI_B_CONST, PHI_B_Z, PHI_B_KAPPA, PHI_B_XHAT, PHI_B_NOT, PHI_B_XOR, PHI_B_AND, PHI_B_OR, PHI_B_ANDPUB,
 PHI_B_OUT, PHI_B_A2B) = range(32, 43)

U64 = (1 << 64) - 1


@dataclass
class OpSpec:
    name: str
    n: int
    f: int
    alpha: list            # m-1 interior boundaries (python ints), strictly increasing in (0, 2^n)
    coeff: np.ndarray      # uint64 [m, r, d+1], high degree first
    aux: np.ndarray        # uint64 [m, p_aux]
    nodes: list = field(default_factory=list)     # (kind, k, lhs, rhs, value_is_2k, value)
    bit_root: np.ndarray = None                   # uint16 [m, ell]
    kappa_a: list = field(default_factory=list)   # (kind, arg)
    kappa_b: list = field(default_factory=list)
    phi: list = field(default_factory=list)       # (op, dst, a, b, imm)
    n_out_a: int = 0
    n_out_b: int = 0
    mask_output: bool = False
    out_frac: int = 0      # fractional bits of the arithmetic outputs (metadata for decode)
    domain: tuple = None   # real interval on which the spline error is stated
    func: object = None    # real function approximated (metadata for tests)
    variant: int = 0       # bit 0: single-key shared-prefix construction (DESIGN 9); bit 1: input-masked products (10); bit 2: Horner in xhat (11); bit 3: early-terminated bit trees (13)

    @property
    def m(self):
        return len(self.alpha) + 1

    @property
    def r(self):
        return int(self.coeff.shape[1])

    @property
    def d(self):
        return int(self.coeff.shape[2]) - 1

    @property
    def p_aux(self):
        return int(self.aux.shape[1])

    @property
    def ell(self):
        return 0 if self.bit_root is None else int(self.bit_root.shape[1])


def _ring(v, n):
    return int(v) & ((1 << n) - 1)


def _mk(name, n, f, alpha, coeff_int, nodes=(), bit_root_cols=0, **kw):
    """coeff_int: nested python ints [m][r][d+1] (may be negative)."""
    m = len(alpha) + 1
    c = np.array([[[_ring(v, n) for v in poly] for poly in piece] for piece in coeff_int], dtype=np.uint64)
    aux = kw.pop("aux", None)
    aux = np.zeros((m, 0), np.uint64) if aux is None else np.array(aux, dtype=np.uint64).reshape(m, -1)
    bit_root = kw.pop("bit_root", None)
    if bit_root is None:
        bit_root = np.zeros((m, 0), np.uint16)
    else:
        bit_root = np.array(bit_root, dtype=np.uint16).reshape(m, -1)
    return OpSpec(name=name, n=n, f=f, alpha=[int(a) for a in alpha], coeff=c, aux=aux, nodes=list(nodes),
                  bit_root=bit_root, **kw)


# ---- spline fitting (input preparation; minimax LP per piece, sequential coefficient rounding) ---
def _fit_piece(func, lo, hi, d, f, g, npts=2049):
    """Degree-d minimax fit of func on real [lo, hi]; coefficient of x^k quantised to scale
    2^((d+1-k) f + g).  Returns python ints, high degree first."""
    from scipy.optimize import linprog

    xs = np.linspace(lo, hi, npts)
    ys = np.array([func(float(x)) for x in xs])
    fixed = {}
    for k in range(d, -1, -1):
        free = list(range(k, -1, -1))
        resid = ys - sum(fixed[j] * xs ** j for j in fixed) if fixed else ys
        V = np.stack([xs ** j for j in free], axis=1)
        nv = len(free)
        A = np.block([[V, -np.ones((npts, 1))], [-V, -np.ones((npts, 1))]])
        b = np.concatenate([resid, -resid])
        cost = np.zeros(nv + 1)
        cost[-1] = 1.0
        res = linprog(cost, A_ub=A, b_ub=b, bounds=[(None, None)] * nv + [(0, None)], method="highs")
        if res.status != 0:
            raise RuntimeError("spline LP failed")
        scale = 2.0 ** ((d + 1 - k) * f + g)
        fixed[k] = math.floor(res.x[0] * scale + 0.5) / scale
    return [int(round(fixed[k] * 2.0 ** ((d + 1 - k) * f + g))) for k in range(d, -1, -1)]


def _const_piece(value, d, f, g):
    return [0] * d + [int(math.floor(value * 2.0 ** ((d + 1) * f + g) + 0.5))]


def _identity_piece(d, f, g):
    c = [0] * (d + 1)
    c[d - 1] = 1 << (d * f + g)
    return c


def _enc(v, f):
    return int(math.floor(v * (1 << f) + 0.5))


_CACHE = {}


def _cached(key, fn):
    if key not in _CACHE:
        _CACHE[key] = fn()
    return _CACHE[key]


# ---- config 1: App. N signed ReLU -----------------------------------------
def relu(n=16, f=8):
    N = 1 << n
    nodes = [(BN_MSB, 0, 0, 0, 0, 0)]                       # z = MSB(x)
    phi = [(PHI_A_Y, 0, 0, 0, 0), (PHI_A_Y, 1, 1, 0, 0), (PHI_A_X, 2, 0, 0, 0),
           (PHI_A_MUL, 3, 0, 2, 0), (PHI_A_ADD, 4, 3, 1, 0), (PHI_A_OUT, 0, 4, 0, 0),
           (PHI_B_Z, 0, 0, 0, 0), (PHI_B_OUT, 0, 0, 0, 0)]
    return _mk(f"relu_n{n}", n, f, [N // 2], [[[1], [0]], [[0], [0]]], nodes=nodes, bit_root=[[0], [0]],
               phi=phi, n_out_a=1, n_out_b=1, out_frac=f)


# ---- sign / |x|<c / x>c predicate bits shared by GeLU and SiLU (all XOR-only, Lemma D.1) --------
def _act_bits(n, cF):
    N = 1 << n
    H = N >> 1
    nodes = [(BN_C, 0, 0, 0, 0, H), (BN_NOT, 0, 0, 0, 0, 0),            # 1: sign = not C_{2^{n-1}}
             (BN_C, 0, 0, 0, 0, cF), (BN_C, 0, 0, 0, 0, N - cF + 1),
             (BN_NOT, 0, 3, 0, 0, 0), (BN_XOR, 0, 2, 4, 0, 0),          # 5: |x| < c
             (BN_C, 0, 0, 0, 0, cF + 1), (BN_XOR, 0, 0, 6, 0, 0)]       # 7: x > c
    return nodes, [1, 5, 7]


def _activation(name, func, n, f, half_width, pieces_per_side, g=0):
    d = 2
    N = 1 << n
    F = 1 << f
    edges_pos = [_enc(half_width * i / pieces_per_side, f) for i in range(pieces_per_side + 1)]
    alpha, coeff = [], []
    for i in range(pieces_per_side):                                     # [0, c): fitted pieces
        coeff.append([_fit_piece(func, edges_pos[i] / F, edges_pos[i + 1] / F, d, f, g)])
        alpha.append(edges_pos[i + 1])
    coeff.append([_identity_piece(d, f, g)])                             # [c, 2^{n-1}): identity tail
    alpha.append(N >> 1)
    coeff.append([_const_piece(0.0, d, f, g)])                           # [2^{n-1}, N-c): zero tail
    alpha.append(N - edges_pos[-1])
    for i in range(pieces_per_side, 0, -1):                              # [N-c, N): negative pieces
        coeff.append([_fit_piece(func, -edges_pos[i] / F, -edges_pos[i - 1] / F, d, f, g)])
        if i > 1:
            alpha.append(N - edges_pos[i - 1])
    nodes, roots = _act_bits(n, edges_pos[-1])
    m = len(alpha) + 1
    return _mk(name, n, f, alpha, coeff, nodes=nodes, bit_root=[roots] * m, n_out_a=1, n_out_b=3,
               out_frac=3 * f + g, domain=(-half_width - 1.0, half_width + 1.0), func=func)


def _gelu(x):
    return 0.5 * x * (1.0 + math.erf(x / math.sqrt(2.0)))


def _silu(x):
    return x / (1.0 + math.exp(-x))


def gelu(n=64, f=12):
    """config 2: 8 degree-2 pieces on [-4, 4] + identity / zero tails (m = 10), 3 predicate bits."""
    return _cached(("gelu", n, f), lambda: _activation(f"gelu_n{n}", _gelu, n, f, 4.0, 4))


def silu(n=64, f=12):
    """config 5: 24 degree-2 pieces on [-8, 8] + tails (m = 26), 3 predicate bits."""
    return _cached(("silu", n, f), lambda: _activation(f"silu_n{n}", _silu, n, f, 8.0, 12))


# ---- config 3: softmax helpers -----------------------------------------------------------------
def nexp(n=64, f=12):
    """nExp(x) = e^x for x <= 0: [0, 2^63) -> 1 (clamp), [2^63, N-16F) -> 0, 16 degree-1 pieces on
    [-16, 0) with breakpoints equalising the linear-interpolation error (m = 18).  No bits."""
    def build():
        d, g = 1, 8
        N, F = 1 << n, 1 << f
        u0 = math.exp(-8.0)
        xs = [2.0 * math.log(u0 + i * (1.0 - u0) / 16) for i in range(17)]
        edges = sorted({-_enc(-x, f) for x in xs})                      # negative integers (scaled), ascending
        edges[0], edges[-1] = -16 * F, 0
        coeff = [[_const_piece(1.0, d, f, g)], [_const_piece(0.0, d, f, g)]]
        alpha = [N >> 1, N + edges[0]]
        for i in range(len(edges) - 1):
            coeff.append([_fit_piece(math.exp, edges[i] / F, edges[i + 1] / F, d, f, g)])
            if i + 1 < len(edges) - 1:
                alpha.append(N + edges[i + 1])
        return _mk(f"nexp_n{n}", n, f, alpha, coeff, n_out_a=1, out_frac=2 * f + g, domain=(-20.0, 0.0),
                   func=lambda x: math.exp(min(x, 0.0)) if x >= -16.0 else 0.0)
    return _cached(("nexp", n, f), build)


def _geometric_spline(name, func, n, f, lo, hi, pieces, g, lo_val, hi_val):
    d = 2
    N, F = 1 << n, 1 << f
    edges = [_enc(lo * (hi / lo) ** (i / pieces), f) for i in range(pieces + 1)]
    coeff = [[_const_piece(lo_val, d, f, g)]]
    alpha = [edges[0]]
    for i in range(pieces):
        coeff.append([_fit_piece(func, edges[i] / F, edges[i + 1] / F, d, f, g)])
        alpha.append(edges[i + 1])
    coeff.append([_const_piece(hi_val, d, f, g)])
    return _mk(name, n, f, alpha, coeff, n_out_a=1, out_frac=3 * f + g, domain=(lo, hi), func=func)


def recip(n=64, f=12):
    """1/s on [1, 128]: 16 geometric degree-2 pieces + clamps (m = 18)."""
    return _cached(("recip", n, f), lambda: _geometric_spline(
        f"recip_n{n}", lambda s: 1.0 / s, n, f, 1.0, 128.0, 16, 16, 1.0, 1.0 / 128.0))


def rsqrt(n=64, f=12):
    """v^-1/2 on [2^-6, 2^6]: 12 octave degree-2 pieces + clamps (m = 14)."""
    return _cached(("rsqrt", n, f), lambda: _geometric_spline(
        f"rsqrt_n{n}", lambda v: v ** -0.5, n, f, 2.0 ** -6, 2.0 ** 6, 12, 12, 8.0, 0.125))


# ---- config 4a: arithmetic right shift by f fused with ReLU ----------------------------------------
def shift_relu(n=64, f=12):
    """y = max(0, x >>_arith f).  F_coeff returns a in {1, 0} (App. N style, p = 1); helper bits:
    z0 = MSB(x), z1 = carry of the low f bits of x + r, z2 = wrap bit of x + r (cross-check only).
    Phi: w = (a&b) ^ ((a^b) & ~c) with a = MSB(x), b = MSB(r) in kappa^B, c = MSB(xhat) public (1 AND);
    u = (xhat >> f) - [r >> f] - B2A(t) + 2^{n-f} B2A(w); y = a * u (1 Beaver)."""
    N = 1 << n
    nodes = [(BN_MSB, 0, 0, 0, 0, 0), (BN_CARRY, f, 0, 0, 0, 0), (BN_CARRY, n, 0, 0, 0, 0)]
    phi = [
        (PHI_B_Z, 0, 0, 0, 0), (PHI_B_KAPPA, 1, 0, 0, 0),
        (PHI_B_AND, 2, 0, 1, 0), (PHI_B_XOR, 3, 0, 1, 0), (PHI_B_ANDPUB, 4, 3, n - 1, 1), (PHI_B_XOR, 5, 2, 4, 0),
        (PHI_B_Z, 6, 1, 0, 0),
        (PHI_A_XHAT_SHR, 0, f, 0, 0), (PHI_A_KAPPA, 1, 0, 0, 0), (PHI_A_B2A, 2, 6, 0, 0), (PHI_A_B2A, 3, 5, 0, 0),
        (PHI_A_MULC, 4, 3, 0, (1 << (n - f)) & U64),
        (PHI_A_SUB, 5, 0, 1, 0), (PHI_A_SUB, 6, 5, 2, 0), (PHI_A_ADD, 7, 6, 4, 0),
        (PHI_A_Y, 8, 0, 0, 0), (PHI_A_MUL, 9, 8, 7, 0), (PHI_A_OUT, 0, 9, 0, 0),
        (PHI_B_OUT, 0, 0, 0, 0), (PHI_B_OUT, 1, 5, 0, 0), (PHI_B_Z, 7, 2, 0, 0), (PHI_B_OUT, 2, 7, 0, 0),
    ]
    return _mk(f"shift_relu_n{n}", n, f, [N // 2], [[[1]], [[0]]], nodes=nodes, bit_root=[[0, 1, 2]] * 2,
               kappa_a=[(KA_R_SHR, f)], kappa_b=[(KB_R_BIT, n - 1)], phi=phi, n_out_a=1, n_out_b=3, out_frac=f)


def ars(n=64, f=12):
    """Signed truncation y = x >>_arith f (the rescale between fixed-point multiplications):
    ARS_f(x) = LRS_f(x + 2^{n-1}) - 2^{n-1-f}.  The gate's input is x' = x + 2^{n-1}: the caller adds the public
    constant 2^{n-1} to the masked value (xhat' = xhat + 2^{n-1}, same mask).  No interval lookup (m = 1).
    LRS_f(x') = (xhat' >> f) - (r >> f) - t + 2^{n-f} w with t = carry of the low f bits, w = wrap of x' + r."""
    nodes = [(BN_MSB, 0, 0, 0, 0, 0), (BN_CARRY, f, 0, 0, 0, 0), (BN_CARRY, n, 0, 0, 0, 0)]
    phi = [
        (PHI_B_Z, 0, 0, 0, 0), (PHI_B_KAPPA, 1, 0, 0, 0),
        (PHI_B_AND, 2, 0, 1, 0), (PHI_B_XOR, 3, 0, 1, 0), (PHI_B_ANDPUB, 4, 3, n - 1, 1), (PHI_B_XOR, 5, 2, 4, 0),
        (PHI_B_Z, 6, 1, 0, 0),
        (PHI_A_XHAT_SHR, 0, f, 0, 0), (PHI_A_KAPPA, 1, 0, 0, 0), (PHI_A_B2A, 2, 6, 0, 0), (PHI_A_B2A, 3, 5, 0, 0),
        (PHI_A_MULC, 4, 3, 0, (1 << (n - f)) & U64),
        (PHI_A_SUB, 5, 0, 1, 0), (PHI_A_SUB, 6, 5, 2, 0), (PHI_A_ADD, 7, 6, 4, 0),
        (PHI_A_CONST, 8, 0, 0, 1 << (n - 1 - f)), (PHI_A_SUB, 9, 7, 8, 0), (PHI_A_OUT, 0, 9, 0, 0),
    ]
    return _mk(f"ars{f}_n{n}", n, f, [], [[[0]]], nodes=nodes, bit_root=[[0, 1, 2]],
               kappa_a=[(KA_R_SHR, f)], kappa_b=[(KB_R_BIT, n - 1)], phi=phi, n_out_a=1, n_out_b=0, out_frac=0)


# ---- a small "kitchen sink" spec for the exhaustive n = 8 / 12 brute force -------------------------
def toy(n=8, f=3, mask_output=False):
    """Exercises everything the grammar allows at brute-force size: 4 uneven intervals, r = 2 degree-2
    polynomials, one aux constant, piecewise-different Boolean outputs (Lemma D.2 normalisation with
    ANDs), D_{gamma,f}, MSB(x+c), OR/AND, sentinels, a Phi with a Beaver product, B2A and kappa."""
    N = 1 << n
    a1, a2, a3 = N // 8 + 1, N // 2, N - 3
    coeff = [[[1, 2, 3], [0, 0, 5]], [[0, 1, -1], [2, -3, 4]], [[3, 0, 0], [0, 7, 0]], [[-1, -1, -1], [0, 0, 0]]]
    aux = [[11], [22], [33], [44]]
    nodes = [
        (BN_D, f, 0, 0, 0, 3),                 # 0: (x mod 2^f) < 3
        (BN_MSB, 0, 0, 0, 0, 5),               # 1: MSB(x + 5)
        (BN_C, 0, 0, 0, 0, N // 4),            # 2: x < N/4
        (BN_AND, 0, 0, 1, 0, 0),               # 3
        (BN_OR, 0, 2, 3, 0, 0),                # 4
        (BN_C, 0, 0, 0, 1, 0),                 # 5: C_{2^n} sentinel = 1
        (BN_XOR, 0, 5, 0, 0, 0),               # 6: not D
        (BN_CONST, 0, 0, 0, 0, 0),             # 7: 0
        (BN_D, f, 0, 0, 1, 0),                 # 8: D_{2^f,f} sentinel = 1
        (BN_CARRY, f, 0, 0, 0, 0),             # 9: low-f carry of x + r
        (BN_MSB, 0, 0, 0, 0, 0),               # 10: MSB(x)
    ]
    bit_root = [[4, 0, 9], [4, 6, 9], [4, 7, 9], [4, 8, 9]]   # bit 1 is piecewise, bits 0 and 2 uniform
    phi = [
        (PHI_A_Y, 0, 0, 0, 0), (PHI_A_Y, 1, 1, 0, 0), (PHI_A_AUX, 2, 0, 0, 0),
        (PHI_A_MUL, 3, 0, 1, 0), (PHI_A_ADD, 4, 3, 2, 0),
        (PHI_B_Z, 0, 0, 0, 0), (PHI_B_Z, 1, 1, 0, 0), (PHI_B_Z, 2, 2, 0, 0), (PHI_B_KAPPA, 3, 0, 0, 0),
        (PHI_B_XOR, 4, 0, 3, 0), (PHI_B_OR, 5, 4, 1, 0), (PHI_B_XHAT, 6, 1, 0, 0), (PHI_B_AND, 7, 5, 6, 0),
        (PHI_A_B2A, 5, 7, 0, 0), (PHI_A_MULC, 6, 5, 0, 9), (PHI_A_KAPPA, 7, 0, 0, 0),
        (PHI_A_ADD, 8, 4, 6, 0), (PHI_A_SUB, 9, 8, 7, 0), (PHI_A_XHAT_SHR, 10, 2, 0, 0), (PHI_A_ADD, 11, 9, 10, 0),
        (PHI_A_CONST, 12, 0, 0, 17), (PHI_A_ADD, 13, 11, 12, 0), (PHI_A_X, 14, 0, 0, 0), (PHI_A_SUB, 15, 13, 14, 0),
        (PHI_A_OUT, 0, 15, 0, 0), (PHI_A_OUT, 1, 0, 0, 0),
        (PHI_B_OUT, 0, 7, 0, 0), (PHI_B_OUT, 1, 1, 0, 0), (PHI_B_OUT, 2, 2, 0, 0), (PHI_B_NOT, 8, 0, 0, 0),
        (PHI_B_OUT, 3, 8, 0, 0),
    ]
    return _mk(f"toy_n{n}", n, f, [a1, a2, a3], coeff, nodes=nodes, bit_root=bit_root, aux=aux,
               kappa_a=[(KA_R_SHR, 2)], kappa_b=[(KB_R_BIT, 1)], phi=phi, n_out_a=2, n_out_b=4,
               mask_output=mask_output, out_frac=f)


def a2b_demo(n=8, f=3):
    """Exercises the A2B node (App. H: "A2B : [x] -> <b> for a suitable extracted bit b"; DESIGN 15): Phi extracts
    the sign of the gate input itself (bit n-1 of x), bit f of the degree-1 spline output y_0, the low bit of y_0 + x (local), and
    feeds an extracted bit back into arithmetic through B2A.  m = 3 intervals, one predicate bit."""
    N = 1 << n
    nodes = [(BN_C, 0, 0, 0, 0, N // 3)]
    phi = [
        (PHI_A_X, 0, 0, 0, 0), (PHI_A_Y, 1, 0, 0, 0), (PHI_A_ADD, 2, 0, 1, 0),
        (PHI_B_A2B, 0, 0, n - 1, 0),          # B0 = MSB(x)
        (PHI_B_A2B, 1, 1, f, 0),              # B1 = bit f of y_0
        (PHI_B_A2B, 2, 2, 0, 0),              # B2 = LSB(x + y_0)   (local)
        (PHI_B_Z, 3, 0, 0, 0), (PHI_B_XOR, 4, 0, 3, 0),
        (PHI_A_B2A, 3, 1, 0, 0), (PHI_A_MULC, 4, 3, 0, 5), (PHI_A_ADD, 5, 4, 1, 0),
        (PHI_B_A2B, 5, 5, 1, 0),              # B5 = bit 1 of (5 B1 + y_0): an A2B after a B2A, two rounds later
        (PHI_A_OUT, 0, 5, 0, 0),
        (PHI_B_OUT, 0, 0, 0, 0), (PHI_B_OUT, 1, 1, 0, 0), (PHI_B_OUT, 2, 2, 0, 0), (PHI_B_OUT, 3, 4, 0, 0), (PHI_B_OUT, 4, 5, 0, 0),
    ]
    return _mk(f"a2b_n{n}", n, f, [N // 4, N // 2 + 3], [[[3, 1]], [[-2, 7]], [[1, -5]]], nodes=nodes, bit_root=[[0]] * 3,
               phi=phi, n_out_a=1, n_out_b=5, out_frac=2 * f)


def tiny_ring(n=1):
    """The smallest rings (n = 1: Z_2, two intervals, M = min(m + 1, 2^n) = 2; n = 2: three intervals, M = 4 = the whole ring):
    degree-1 pieces, a threshold bit and the MSB.  Degenerate-size edge case for both constructions."""
    m = 2 if n == 1 else 3
    nodes = [(BN_C, 0, 0, 0, 0, 1), (BN_MSB, 0, 0, 0, 0, 0)]
    return _mk(f"tiny_n{n}", n, 0, [1] if n == 1 else [1, 3], [[[i + 1, 1 - i]] for i in range(m)], nodes=nodes, bit_root=[[0, 1]] * m,
               n_out_a=1, out_frac=0)


def limits(n=64, m=63, r=2, d=3, n_pred=63):
    """A gate type AT the compiled limits (fusefss.h: m < 64, p <= 8, T <= 64, 64 output bits): m = 63 intervals spread over the ring,
    r = 2 polynomials of degree 3 (p = 8 payload words) and 63 distinct thresholds C_beta, each its own output bit:
    T = 1 r-atom + 63 theta-atoms = 64.  Stress / edge-case input, not an operator of the paper."""
    N = 1 << n
    alpha = [(i + 1) * (N // (m + 1)) + 3 * i for i in range(m - 1)]
    coeff = [[[(7 * i + 3 * j + k + 1) * (1 if (i + k) % 3 else -1) for k in range(d + 1)] for j in range(r)] for i in range(m)]
    nodes = [(BN_C, 0, 0, 0, 0, (t + 1) * (N // (n_pred + 2)) + 5 * t + 1) for t in range(n_pred)]
    return _mk(f"limits_m{m}_p{r * (d + 1)}_T{n_pred + 1}", n, 12, alpha, coeff, nodes=nodes, bit_root=[list(range(n_pred))] * m,
               n_out_a=r, out_frac=12)


def limits_piecewise(n=64, m=32):
    """m = 32 intervals with ONE piecewise output bit: Lemma D.2 spends m = 32 AND gates on it, all in one round -- 64 opened bits,
    exactly one message bit word (the per-round limit); the 31 boundary comparisons become atoms."""
    N = 1 << n
    alpha = [(i + 1) * (N // (m + 1)) + i for i in range(m - 1)]
    nodes = [(BN_C, 0, 0, 0, 0, N // 5 + 11), (BN_NOT, 0, 0, 0, 0, 0)]
    return _mk(f"limits_pw_m{m}", n, 12, alpha, [[[i + 1, -i]] for i in range(m)], nodes=nodes, bit_root=[[i % 2] for i in range(m)],
               n_out_a=1, out_frac=12)


def plain_default(n=8, f=3):
    """No Phi (default: outputs are F's y and z), r = 1 degree-1, m = 3, one piecewise bit."""
    N = 1 << n
    nodes = [(BN_C, 0, 0, 0, 0, 5), (BN_MSB, 0, 0, 0, 0, 0), (BN_CONST, 0, 0, 0, 0, 1)]
    return _mk(f"plain_n{n}", n, f, [7, N // 2 + 1], [[[2, 1]], [[0, 9]], [[-1, 0]]], nodes=nodes,
               bit_root=[[0], [1], [2]], n_out_a=1, n_out_b=1, out_frac=2 * f)


def single_interval(n=8, f=3):
    """m = 1: the interval lookup is omitted; one predicate bit."""
    nodes = [(BN_C, 0, 0, 0, 0, 100 % (1 << n) or 1)]
    return _mk(f"single_n{n}", n, f, [], [[[3, 1]]], nodes=nodes, bit_root=[[0]], n_out_a=1, n_out_b=1,
               out_frac=2 * f)


def no_bits(n=8, f=3):
    """T = 0: the packed comparison is omitted."""
    N = 1 << n
    return _mk(f"nobits_n{n}", n, f, [N // 4, N // 2], [[[1, 0]], [[2, 1]], [[0, 3]]], n_out_a=1, out_frac=2 * f)


def full_partition(n=3):
    """m = N: M = N, no padding possible (Protocol 3 line 2 / line 12)."""
    N = 1 << n
    return _mk(f"full_n{n}", n, 0, list(range(1, N)), [[[i * 3 + 1]] for i in range(N)], n_out_a=1)


def shared_prefix(spec):
    """The same operator compiled with the single-key, multi-point construction."""
    import dataclasses
    return dataclasses.replace(spec, variant=1, name=spec.name + "_sp")


def input_masked_mul(spec):
    """The same operator with variant bit 1: products with the gate input x open ONE ring element."""
    import dataclasses
    return dataclasses.replace(spec, variant=spec.variant | 2, name=spec.name + "_xm")


def public_point_horner(spec):
    """Variant bit 2: the lookup returns the coefficients of P_i(X - r_in), Horner runs in the public xhat -- zero
    Beaver rounds for the spline."""
    import dataclasses
    return dataclasses.replace(spec, variant=spec.variant | 4, name=spec.name + "_xp")


def early_termination(spec):
    """Variant bit 3: the bit-DCF trees stop max(k-7, 0) levels deep and read the output bit out of a 128-bit leaf block
    (DESIGN.md section 13)."""
    import dataclasses
    return dataclasses.replace(spec, variant=spec.variant | 8, name=spec.name + "_et")


def dense_table(spec):
    """Variant bits 0 + 4: the interval lookup in the dense-table ("DPF-LUT") representation -- the single key
    f_{r,1} evaluated on the whole domain of 2^n points (n <= 16); cost and shape depend on n only."""
    import dataclasses
    return dataclasses.replace(spec, variant=spec.variant | 17, name=spec.name + "_dense")


CONFIGS = {
    "relu16": lambda: relu(16, 8),
    "gelu": gelu,
    "nexp": nexp,
    "recip": recip,
    "shift_relu": shift_relu,
    "rsqrt": rsqrt,
    "silu": silu,
}
