"""Pins for oracle/wigner.py: library routine (sympy), closed forms, orthogonality."""
import itertools
import math

import pytest

from oracle import wigner


def test_six_j_against_sympy():
    from sympy.physics.wigner import wigner_6j
    from sympy import Rational

    def sym(args):
        try:
            return float(wigner_6j(*[Rational(a, 2) for a in args]))
        except ValueError:  # sympy raises where the symbol vanishes by the triangle rules
            return 0.0

    n = 0
    for args in itertools.product(range(0, 5), repeat=6):
        if sum(args) % 3 or n > 400:  # thin the grid
            continue
        ref = sym(args)
        assert wigner.six_j(*args) == pytest.approx(ref, abs=1e-14)
        n += 1
    # a few larger ones that occur for j<=3, J=7/2
    for args in [(8, 6, 6, 4, 8, 10), (7, 5, 4, 3, 6, 3), (6, 8, 4, 8, 6, 10), (3, 7, 6, 5, 3, 4),
                 (7, 5, 4, 3, 5, 4), (9, 7, 4, 3, 5, 6)]:
        ref = sym(args)
        assert wigner.six_j(*args) == pytest.approx(ref, abs=1e-14)


def test_six_j_closed_form():
    # {a b c; 0 c b} = (-1)^{a+b+c} / sqrt((2b+1)(2c+1))
    for a, b, c in [(1, 1, 1), (2, 1, 1), (2, 2, 1), (3, 2, 2), (4, 3, 2)]:
        val = wigner.six_j(2 * a, 2 * b, 2 * c, 0, 2 * c, 2 * b)
        assert val == pytest.approx((-1) ** (a + b + c) / math.sqrt((2 * b + 1) * (2 * c + 1)), abs=1e-15)


def test_six_j_orthogonality():
    # sum_x (2x+1)(2f+1) {a b x; c d f}{a b x; c d g} = delta_fg
    a, b, c, d = 3, 4, 5, 2  # doubled
    for f in range(abs(a - d), a + d + 1, 2):
        for g in range(abs(a - d), a + d + 1, 2):
            if (b + c + f) % 2 or (b + c + g) % 2:
                continue
            s = sum((x + 1) * (f + 1) * wigner.six_j(a, b, x, c, d, f) * wigner.six_j(a, b, x, c, d, g)
                    for x in range(abs(a - b), a + b + 1, 2))
            ok_f = abs(b - c) <= f <= b + c
            assert s == pytest.approx(1.0 if (f == g and ok_f) else 0.0, abs=1e-13)


def test_nine_j_against_sympy():
    from sympy.physics.wigner import wigner_9j
    from sympy import Rational

    cases = [
        (2, 2, 4, 2, 1, 3, 2, 3, 1), (4, 2, 2, 2, 1, 3, 2, 3, 1), (0, 2, 2, 0, 1, 1, 0, 1, 1),
        (4, 2, 4, 4, 1, 5, 4, 3, 1), (6, 2, 4, 2, 1, 3, 4, 3, 1), (2, 0, 2, 4, 1, 3, 2, 1, 3),
        (4, 2, 6, 6, 1, 7, 8, 3, 7), (8, 2, 6, 4, 1, 5, 6, 1, 7),
    ]
    for args in cases:
        ref = float(wigner_9j(*[Rational(a, 2) for a in args], prec=40))
        assert wigner.nine_j(*args) == pytest.approx(ref, abs=1e-14)


def test_cg000_against_sympy_and_closed_form():
    from sympy.physics.wigner import clebsch_gordan

    for a in range(0, 6):
        for b in range(0, 6):
            for c in range(abs(a - b), a + b + 1):
                ref = float(clebsch_gordan(a, b, c, 0, 0, 0))
                assert wigner.cg000(a, b, c) == pytest.approx(ref, abs=1e-14)
    # <a0 b0|a+b 0> = (a+b)!/(a! b!) sqrt((2a)!(2b)!/(2a+2b)!)
    f = math.factorial
    for a, b in [(1, 1), (2, 1), (3, 2), (4, 4)]:
        cf = f(a + b) / (f(a) * f(b)) * math.sqrt(f(2 * a) * f(2 * b) / f(2 * a + 2 * b))
        assert wigner.cg000(a, b, a + b) == pytest.approx(cf, rel=1e-14)
