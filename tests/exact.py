"""Exact-arithmetic helpers for pinning the oracle (test-side only, independent of oracle/ and of
the CUDA library): IEEE-754 binary32 values as Fractions and round-to-nearest-even back."""
from fractions import Fraction
import struct


def f32_bits(x: float) -> int:
    return struct.unpack("<I", struct.pack("<f", x))[0]


def bits_f32(u: int) -> float:
    return struct.unpack("<f", struct.pack("<I", u & 0xFFFFFFFF))[0]


def frac_of_f32(x: float) -> Fraction:
    return Fraction(float(x))          # every finite float is an exact rational


def round_to_f32_bits(q: Fraction) -> int:
    """Round an exact rational to the nearest binary32 (ties to even); normal/subnormal range only."""
    if q == 0:
        return 0
    sign = 0x80000000 if q < 0 else 0
    q = abs(q)
    # find e with 2^e <= q < 2^(e+1)
    e = q.numerator.bit_length() - q.denominator.bit_length()
    if Fraction(2) ** e > q:
        e -= 1
    if Fraction(2) ** (e + 1) <= q:
        e += 1
    e_eff = max(e, -126)
    scaled = q / Fraction(2) ** (e_eff - 23)      # significand in units of the last place
    lo = scaled.numerator // scaled.denominator
    rem = scaled - lo
    if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and (lo & 1)):
        lo += 1
    if e >= -126:
        if lo == (1 << 24):
            lo >>= 1
            e_eff += 1
        assert e_eff <= 127
        return sign | ((e_eff + 127) << 23) | (lo - (1 << 23))
    # subnormal (lo < 2^23) or rounds up to the smallest normal (lo == 2^23, encodes correctly)
    return sign | lo


def fused_step_bits(a: float, y: float, b: float) -> int:
    """fmaf(a, y, b) by definition: exact a*y+b, rounded once."""
    return round_to_f32_bits(frac_of_f32(a) * frac_of_f32(y) + frac_of_f32(b))


def round_f32_to_bf16_bits(x: float) -> int:
    """RNE of a finite binary32 to bfloat16 by exact arithmetic on the bit pattern."""
    u = f32_bits(x)
    hi, lo = u >> 16, u & 0xFFFF
    if lo > 0x8000 or (lo == 0x8000 and (hi & 1)):
        hi += 1
    return hi & 0xFFFF
