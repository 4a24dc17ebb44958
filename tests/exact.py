"""Exact rational arithmetic helpers for the oracle pins: correctly rounded IEEE results from Fractions.

Independent of oracle/ and of the CUDA path: used to restate, with exact arithmetic and ONE explicit
rounding per IEEE operation, what a fused multiply-add / subtract / divide must return bit for bit.
"""
from __future__ import annotations

import math
from fractions import Fraction

import numpy as np


def rn(x: Fraction, prec: int, emin: int) -> Fraction:
    """Round-to-nearest-even of the exact rational x to a binary float with `prec` significand bits and
    minimum normal exponent emin (binary64: 53, -1022; binary32: 24, -126).  Returns the exact value."""
    if x == 0:
        return Fraction(0)
    s = -1 if x < 0 else 1
    a = -x if x < 0 else x
    e = a.numerator.bit_length() - a.denominator.bit_length()        # 2^(e-1) <= a < 2^(e+1)
    if Fraction(2) ** e > a:
        e -= 1                                                     # now 2^e <= a < 2^(e+1)
    e = max(e, emin)                                               # subnormal range: fixed quantum
    q = Fraction(2) ** (e - prec + 1)                              # ulp
    m = a / q
    f = m.numerator // m.denominator
    r = m - f
    if r > Fraction(1, 2) or (r == Fraction(1, 2) and (f & 1)):
        f += 1
    return s * f * q


def rn64(x: Fraction) -> Fraction:
    return rn(x, 53, -1022)


def rn32(x: Fraction) -> Fraction:
    return rn(x, 24, -126)


def F(x) -> Fraction:
    """Exact value of a numpy / python float."""
    return Fraction(float(x))


def wrap_exact(x: Fraction) -> Fraction:
    """The oracle's wrap on the exactly-representable double x: w = RN64(x - floor(x)); 1.0 -> 0.0."""
    w = rn64(x - math.floor(x))
    return Fraction(0) if w >= 1 else w


def to_f64(x: Fraction) -> np.float64:
    return np.float64(x.numerator / x.denominator)                 # exact: x is representable


def to_f32(x: Fraction) -> np.float32:
    return np.float32(x.numerator / x.denominator)                 # exact: x is representable in binary32
