"""The plaintext spline of every config vs the real function it approximates, over every representable
input of the stated domain (Tier A, A3): stated maximum absolute errors."""
import numpy as np
import pytest

from workloads import specs

# name, lo, hi, stride, bound
CASES = [("gelu", -6.0, 6.0, 1, 2.0 ** -8), ("silu", -10.0, 10.0, 1, 2.0 ** -8), ("nexp", -20.0, 0.0, 1, 2.0 ** -9),
         ("recip", 1.0, 128.0, 3, 2.0 ** -10), ("rsqrt", 2.0 ** -6, 2.0 ** 6, 1, 2.5e-2)]


@pytest.mark.parametrize("name,lo,hi,stride,bound", CASES)
def test_spline_error(orc, name, lo, hi, stride, bound):
    spec = specs.CONFIGS[name]()
    P = orc.Program(spec)
    f = spec.f
    xs = np.arange(int(lo * (1 << f)), int(hi * (1 << f)) + 1, stride, dtype=np.int64)
    y, _ = P.plain_G(xs.view(np.uint64), np.zeros(xs.size, np.uint64))
    got = y[0].view(np.int64).astype(np.float64) / 2.0 ** spec.out_frac
    ref = np.array([spec.func(v / (1 << f)) for v in xs])
    assert np.abs(got - ref).max() <= bound


def test_gelu_bits_plain(orc):
    spec = specs.gelu()
    P = orc.Program(spec)
    F = 1 << 12
    xs = np.array([0, 1, 4 * F - 1, 4 * F, 4 * F + 1, -1, -4 * F + 1, -4 * F, -4 * F - 1, 1 << 40, -(1 << 40)],
                  dtype=np.int64)
    _, z = P.plain_G(xs.view(np.uint64), np.zeros(xs.size, np.uint64))
    assert list(z[0]) == [int(v < 0) for v in xs]
    assert list(z[1]) == [int(abs(int(v)) < 4 * F) for v in xs]
    assert list(z[2]) == [int(v > 4 * F) for v in xs]
