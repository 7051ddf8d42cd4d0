"""Host-side checks of arithmetic identities the CUDA kernels rely on (no GPU, no oracle import
needed for the arithmetic itself): each identity is proved here in exact rational arithmetic."""
from fractions import Fraction

import numpy as np


def _rn32(fr):
    """Round a non-negative Fraction to the nearest binary32 (ties to even, subnormals included)."""
    if fr == 0:
        return np.float32(0)
    e = fr.numerator.bit_length() - fr.denominator.bit_length()
    if Fraction(2) ** e > fr:
        e -= 1
    if Fraction(2) ** (e + 1) <= fr:
        e += 1
    q = max(e, -126) - 23                      # exponent of one ulp
    scaled = fr / Fraction(2) ** q
    n = scaled.numerator // scaled.denominator
    rem = scaled - n
    if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and (n & 1)):
        n += 1
    return np.float32(float(Fraction(n) * Fraction(2) ** q))


def test_rn32_helper_matches_numpy_on_doubles():
    rng = np.random.default_rng(0)
    for v in np.abs(rng.standard_normal(2000)) * 10.0 ** rng.integers(-44, 38, 2000):
        assert _rn32(Fraction(float(v))).view(np.uint32) == np.float32(v).view(np.uint32)


def test_div6_of_a_bf16_value_in_three_ops_is_the_ieee_quotient():
    """quant_math.cuh::div6_bf16: q0 = x*c, r = fma(-6, q0, x), q = fma(r, c, q0) with c = fl(1/6)
    equals fl(x / 6) (Q4, `amax_b / 6`) for EVERY finite non-negative bf16 x."""
    c = Fraction(float(np.float32(1) / np.float32(6)))
    for b in range(0, 0x7F80):
        x = Fraction(float(np.uint32(b << 16).view(np.float32)))
        want = _rn32(x / 6)
        q0 = Fraction(float(_rn32(x * c)))
        r_exact = x - 6 * q0                   # fma: one rounding of the exact value (may be negative)
        r = Fraction(float(_rn32(abs(r_exact)))) * (1 if r_exact >= 0 else -1)
        q = _rn32(q0 + r * c)
        assert q.view(np.uint32) == want.view(np.uint32), hex(b)
    # and the plain product x * fl(1/6) is NOT enough (guards against a test that cannot fail)
    x = (np.arange(0x0080, 0x7F80, dtype=np.uint32) << 16).view(np.float32)
    assert np.any((x * (np.float32(1) / np.float32(6))).astype(np.float32) != (x / np.float32(6)).astype(np.float32))
