"""Exact rational helpers for the tests (Python `fractions` / big integers only).

Independent of both oracle/ and the CUDA path: this is the "something other than itself" that pins the oracle.
CPython's int/int true division is correctly rounded, so float(Fraction) is round-to-nearest-even.
"""
from fractions import Fraction
import math


def F(x) -> Fraction:
    return Fraction(float(x))


def fsum_exact(values) -> Fraction:
    t = Fraction(0)
    for v in values:
        t += Fraction(float(v))
    return t


def round_to_limbs(v: Fraction, limbs: int):
    """limb_l = RN(v - limb_0 - ... - limb_{l-1}), l = 0..limbs-1."""
    out = []
    for _ in range(limbs):
        f = float(v)
        out.append(f)
        v -= Fraction(f)
    return out


def ulp(x: float) -> float:
    return math.ulp(x)


def round_half_even(q: Fraction) -> int:
    return round(q)  # Python's round() on a Fraction rounds half to even


def nearest_digits(value: Fraction, E: int, Q: int, bits: int = 13):
    """Signed-digit expansion by exact nearest rounding: D_q = RN(R_q / u_q), R_{q+1} = R_q - D_q u_q.
    Also returns min over q of the distance of R_q/u_q from a tie (x.5)."""
    digits, R, margin = [], value, Fraction(1)
    for q in range(Q):
        u = Fraction(2) ** (E - bits * (q + 1))
        t = R / u
        margin = min(margin, abs(abs(t - math.floor(t)) - Fraction(1, 2)))
        D = round_half_even(t)
        digits.append(D)
        R -= D * u
    return digits, R, margin
