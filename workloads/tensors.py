"""Seeded synthetic inputs with the shapes / distributions of BASELINE.json's configs (SURVEY.md
section 8(d)).  They stand in for the BERT / GPT-2 / LLaMA activations the paper measures on
(PAPER.md:253, 463-465); no dataset item is reproduced.  Holds no method arithmetic: x is quantised
with the fixed tie rule floor(2^f x + 0.5) (reading S8), masks are uniform n-bit words, and
xhat = x + r_in mod 2^n is Protocol 1's output, i.e. the boundary input of the hot path.
"""
from __future__ import annotations

import numpy as np


def _mask(n):
    return np.uint64((1 << n) - 1) if n < 64 else np.uint64(0xFFFFFFFFFFFFFFFF)


def quantise(xr: np.ndarray, f: int, n: int) -> np.ndarray:
    q = np.floor(xr * float(1 << f) + 0.5).astype(np.int64)
    return q.view(np.uint64) & _mask(n)


def uniform_ring(rng, count, n):
    return rng.integers(0, 1 << 64, size=count, dtype=np.uint64, endpoint=False) & _mask(n) if n == 64 else \
        rng.integers(0, 1 << n, size=count, dtype=np.uint64)


def masks(count: int, n: int, seed: int, n_out: int = 1):
    """(r_in[count], r_out[n_out, count]) -- fresh uniform masks per wire."""
    rng = np.random.default_rng(seed + 1)
    return uniform_ring(rng, count, n), uniform_ring(rng, count * n_out, n).reshape(n_out, count)


def xhat_of(x, r_in, n):
    return (x + r_in) & _mask(n)


# (config name, full element count, generator of real-valued inputs)
def _gen(name, rng, count):
    if name == "relu16":
        return rng.integers(-(1 << 15), 1 << 15, size=count).astype(np.float64) / 256.0
    if name == "gelu":                       # 128 x 3072, N(0, 2^2)
        return rng.normal(0.0, 2.0, size=count)
    if name == "nexp":                       # 12 x 128 x 128 max-subtracted scores
        return np.maximum(-20.0, -4.0 * rng.exponential(1.0, size=count))
    if name == "recip":                      # 12 x 128 row sums of nExp outputs: in [1, 128]
        s = np.exp(np.maximum(-20.0, -4.0 * rng.exponential(1.0, size=(count, 128))))
        s[:, 0] = 1.0                        # the row maximum contributes e^0
        return s.sum(axis=1)
    if name == "shift_relu":                 # 1024 x 4096 matmul outputs at scale 2f, N(0, 3^2)
        return rng.normal(0.0, 3.0, size=count)
    if name == "rsqrt":                      # 1024 variances, log-uniform on [2^-6, 2^6]
        return 2.0 ** rng.uniform(-6.0, 6.0, size=count)
    if name == "silu":                       # 2048 x 11008, N(0, 3^2)
        return rng.normal(0.0, 3.0, size=count)
    raise KeyError(name)


FULL_COUNT = {"relu16": 4096, "gelu": 128 * 3072, "nexp": 12 * 128 * 128, "recip": 12 * 128,
              "shift_relu": 1024 * 4096, "rsqrt": 1024, "silu": 2048 * 11008}
IN_FRAC = {"shift_relu": 24}


def inputs(name: str, spec, count: int | None = None, seed: int = 0):
    """Returns dict(x, r_in, r_out, xhat) of uint64 arrays for config `name` (count defaults to full)."""
    count = FULL_COUNT[name] if count is None else count
    rng = np.random.default_rng(seed)
    xr = _gen(name, rng, count)
    x = quantise(xr, IN_FRAC.get(name, spec.f), spec.n)
    r_in, r_out = masks(count, spec.n, seed, max(1, spec.n_out_a))
    return dict(x=x, r_in=r_in, r_out=r_out, xhat=xhat_of(x, r_in, spec.n), real=xr)
