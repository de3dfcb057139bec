"""Correctly rounded binary32 arithmetic from exact rationals (test helper).

Used to pin the oracle's O4 finalisation to the mathematics instead of to
another float implementation: every operation of O4 is "exact real result,
rounded once to nearest-even binary32".  Nothing here calls numpy/C float
division or sqrt; float32 values are only *decoded* from their bit patterns.
"""
from fractions import Fraction
import struct


def f32_from_bits(b: int) -> Fraction:
    s = -1 if b >> 31 else 1
    e = (b >> 23) & 0xFF
    m = b & 0x7FFFFF
    assert e != 0xFF
    if e == 0:
        return s * Fraction(m, 1 << 149)
    return s * Fraction((1 << 23) | m) * Fraction(2) ** (e - 150)


def bits_of_float(x: float) -> int:
    return struct.unpack("<I", struct.pack("<f", x))[0]


def round_f32(x: Fraction) -> int:
    """Bit pattern of the binary32 nearest to the exact rational x (ties to even)."""
    if x == 0:
        return 0
    sign = 0
    if x < 0:
        sign, x = 0x80000000, -x
    lo, hi = 0, 0x7F7FFFFF          # positive finite patterns are ordered like their values
    while hi - lo > 1:
        mid = (lo + hi) // 2
        if f32_from_bits(mid) <= x:
            lo = mid
        else:
            hi = mid
    a, b = f32_from_bits(lo), f32_from_bits(hi)
    if x - a < b - x:
        r = lo
    elif x - a > b - x:
        r = hi
    else:
        r = lo if (lo & 1) == 0 else hi
    return sign | r


def sqrt_f32(bits: int) -> int:
    """Correctly rounded binary32 sqrt of the non-negative binary32 `bits`."""
    x = f32_from_bits(bits)
    assert x >= 0
    if x == 0:
        return 0
    lo, hi = 0, 0x7F7FFFFF
    while hi - lo > 1:
        mid = (lo + hi) // 2
        v = f32_from_bits(mid)
        if v * v <= x:
            lo = mid
        else:
            hi = mid
    a, b = f32_from_bits(lo), f32_from_bits(hi)
    m = (a + b) / 2                  # sqrt(x) < m  <=>  x < m*m ; a tie is impossible for sqrt
    return lo if x < m * m else hi


def finalize_exact(Q, Sp, St, Spp, Stt, p_c, t_c):
    """O4 from exact arithmetic.  Returns 4 bit patterns (pad_mean,time_mean,sigma_pad,sigma_time)."""
    fQ = f32_from_bits(round_f32(Fraction(Q)))
    out = []
    for S, c in ((Sp, p_c), (St, t_c)):
        fS = f32_from_bits(round_f32(Fraction(S)))
        d = f32_from_bits(round_f32(fS / fQ))
        out.append(round_f32(f32_from_bits(round_f32(Fraction(c))) + d))
    for S2, S1 in ((Spp, Sp), (Stt, St)):
        V = Q * S2 - S1 * S1
        assert V >= 0
        fV = round_f32(Fraction(V))
        r = f32_from_bits(sqrt_f32(fV))
        out.append(round_f32(r / fQ))
    return out
