"""Exact Wigner symbols for the oracle (TEST INFRASTRUCTURE, see oracle/__init__.py).

Every symbol is evaluated from its textbook Racah single-sum formula with the
sum carried in exact rational arithmetic (``fractions.Fraction``); only the
final square root of the rational prefactor is taken in floating point, so a
returned value is the correctly rounded symbol up to ~2 ulp.  All angular
momenta are passed DOUBLED (``two_j = 2*j``) so that half-integers are ints.

Used by ``oracle.channels`` for the coefficients g of (A4).

Pins (tests/test_oracle_wigner.py): sympy.physics.wigner (library routine),
the closed forms {a b c; 0 c b} = (-1)^{a+b+c}/sqrt((2b+1)(2c+1)),
<a 0 b 0|a+b 0> closed form, orthogonality sums of 6j and CG.
"""
from fractions import Fraction
from functools import lru_cache
from math import factorial, sqrt


def _tri_ok(a2, b2, c2):
    """Triangle rule on doubled momenta, including the integer-sum rule."""
    return (a2 + b2 + c2) % 2 == 0 and abs(a2 - b2) <= c2 <= a2 + b2


def _delta2(a2, b2, c2):
    """Delta(abc)^2 = (a+b-c)!(a-b+c)!(-a+b+c)!/(a+b+c+1)! as a Fraction."""
    return Fraction(
        factorial((a2 + b2 - c2) // 2) * factorial((a2 - b2 + c2) // 2) * factorial((-a2 + b2 + c2) // 2),
        factorial((a2 + b2 + c2) // 2 + 1),
    )


@lru_cache(maxsize=None)
def six_j(j1, j2, j3, j4, j5, j6):
    """{j1 j2 j3; j4 j5 j6}, arguments doubled.  Racah's formula."""
    if not (_tri_ok(j1, j2, j3) and _tri_ok(j1, j5, j6) and _tri_ok(j4, j2, j6) and _tri_ok(j4, j5, j3)):
        return 0.0
    a1 = (j1 + j2 + j3) // 2
    a2 = (j1 + j5 + j6) // 2
    a3 = (j4 + j2 + j6) // 2
    a4 = (j4 + j5 + j3) // 2
    b1 = (j1 + j2 + j4 + j5) // 2
    b2 = (j2 + j3 + j5 + j6) // 2
    b3 = (j3 + j1 + j6 + j4) // 2
    total = Fraction(0)
    for t in range(max(a1, a2, a3, a4), min(b1, b2, b3) + 1):
        term = Fraction(
            factorial(t + 1),
            factorial(t - a1) * factorial(t - a2) * factorial(t - a3) * factorial(t - a4)
            * factorial(b1 - t) * factorial(b2 - t) * factorial(b3 - t),
        )
        total += -term if t % 2 else term
    d2 = _delta2(j1, j2, j3) * _delta2(j1, j5, j6) * _delta2(j4, j2, j6) * _delta2(j4, j5, j3)
    # sign(total) * sqrt(total^2 * d2), evaluated once in floating point
    val = sqrt(float(total * total * d2))
    return val if total >= 0 else -val


@lru_cache(maxsize=None)
def nine_j(j1, j2, j3, j4, j5, j6, j7, j8, j9):
    """{j1 j2 j3; j4 j5 j6; j7 j8 j9} (rows), doubled arguments, as the sum over
    one 6j triple product: sum_x (-1)^{2x}(2x+1){j1 j4 j7; j8 j9 x}{j2 j5 j8; j4 x j6}{j3 j6 j9; x j1 j2}."""
    for (a, b, c) in ((j1, j2, j3), (j4, j5, j6), (j7, j8, j9), (j1, j4, j7), (j2, j5, j8), (j3, j6, j9)):
        if not _tri_ok(a, b, c):
            return 0.0
    lo = max(abs(j1 - j9), abs(j4 - j8), abs(j2 - j6))
    hi = min(j1 + j9, j4 + j8, j2 + j6)
    total = 0.0
    for x in range(lo, hi + 1, 2):
        sgn = -1.0 if x % 2 else 1.0
        total += sgn * (x + 1) * six_j(j1, j4, j7, j8, j9, x) * six_j(j2, j5, j8, j4, x, j6) * six_j(j3, j6, j9, x, j1, j2)
    return total


@lru_cache(maxsize=None)
def cg000(a, b, c):
    """<a 0 b 0 | c 0> for INTEGER (not doubled) a, b, c.
    = (-1)^{a-b} sqrt(2c+1) (a b c; 0 0 0), with the closed form of the 3j symbol."""
    if (a + b + c) % 2 or not (abs(a - b) <= c <= a + b):
        return 0.0
    g = (a + b + c) // 2
    three_j_sq = Fraction(
        factorial(2 * g - 2 * a) * factorial(2 * g - 2 * b) * factorial(2 * g - 2 * c), factorial(2 * g + 1)
    ) * Fraction(factorial(g), factorial(g - a) * factorial(g - b) * factorial(g - c)) ** 2
    three_j = sqrt(float(three_j_sq)) * (-1.0 if g % 2 else 1.0)
    return (-1.0 if (a - b) % 2 else 1.0) * sqrt(2 * c + 1.0) * three_j
