"""Shared test helpers (no method arithmetic beyond plain reconstruction)."""
import numpy as np


def mask_of(n):
    return np.uint64((1 << n) - 1) if n < 64 else np.uint64(0xFFFFFFFFFFFFFFFF)


def pack_bits(z):
    """z: uint8 [n_bits, count] -> uint64 words with bit j = z[j]."""
    w = np.zeros(z.shape[1], np.uint64)
    for j in range(z.shape[0]):
        w |= z[j].astype(np.uint64) << np.uint64(j)
    return w


def all_r_keys(P, n, seed, r_out=None):
    """One element per mask value r = 0..2^n-1 (keys depend on r only, so each x reuses them)."""
    N = 1 << n
    r_in = np.arange(N, dtype=np.uint64)
    return r_in, P.keygen(r_in, r_out, seed)
