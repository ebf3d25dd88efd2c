"""Pins P1-P3 for oracle/cg_exact.py: closed forms, symmetries, exact
orthonormality.  None of these re-type the Racah sum."""
import os
from fractions import Fraction
from math import factorial as f, sqrt

import pytest

from oracle.cg_exact import cg_exact, cg_exact_square, CGTable

GOLD = os.path.join(os.path.dirname(__file__), "golden", "cg_closed_forms.txt")


def test_golden_closed_forms():
    n = 0
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        tj1, tm1, tj2, tm2, tJ, tM, sg, num, den = (int(x) for x in line.split())
        s, sq = cg_exact_square(tj1, tm1, tj2, tm2, tJ, tM)
        assert s == sg, line
        assert sq == Fraction(num, den), line
        assert cg_exact(tj1, tm1, tj2, tm2, tJ, tM) == pytest.approx(sg * sqrt(num / den), abs=1e-16)
        n += 1
    assert n == 28


def test_stretched_and_j0_and_scalar():
    for tj1 in range(0, 12):
        for tj2 in range(0, 12):
            assert cg_exact_square(tj1, tj1, tj2, tj2, tj1 + tj2, tj1 + tj2) == (1, 1)
        for tm in range(-tj1, tj1 + 1, 2):
            # <j m j -m|0 0> = (-1)^(j-m)/sqrt(2j+1)
            s, sq = cg_exact_square(tj1, tm, tj1, -tm, 0, 0)
            assert sq == Fraction(1, tj1 + 1)
            assert s == (-1 if ((tj1 - tm) // 2) & 1 else 1)
            # <j m 0 0|j m> = 1
            assert cg_exact_square(tj1, tm, 0, 0, tj1, tm) == (1, 1)


def test_maximal_J_closed_form():
    # J = j1+j2: sqrt[(2j1)!(2j2)!(J+M)!(J-M)! / ((2J)!(j1+m1)!(j1-m1)!(j2+m2)!(j2-m2)!)], positive
    for tj1 in range(0, 10):
        for tj2 in range(0, 10):
            tJ = tj1 + tj2
            for tm1 in range(-tj1, tj1 + 1, 2):
                for tm2 in range(-tj2, tj2 + 1, 2):
                    tM = tm1 + tm2
                    h = lambda x: x // 2
                    want = Fraction(f(tj1) * f(tj2) * f(h(tJ + tM)) * f(h(tJ - tM)),
                                    f(tJ) * f(h(tj1 + tm1)) * f(h(tj1 - tm1)) * f(h(tj2 + tm2)) * f(h(tj2 - tm2)))
                    assert cg_exact_square(tj1, tm1, tj2, tm2, tJ, tM) == (1, want)


def _signed(s, sq):
    return s, sq


def test_symmetries():
    for tj1 in range(0, 8):
        for tj2 in range(0, 8):
            for tJ in range(abs(tj1 - tj2), tj1 + tj2 + 1, 2):
                ph = -1 if ((tj1 + tj2 - tJ) // 2) & 1 else 1
                for tm1 in range(-tj1, tj1 + 1, 2):
                    for tm2 in range(-tj2, tj2 + 1, 2):
                        s, sq = cg_exact_square(tj1, tm1, tj2, tm2, tJ, tm1 + tm2)
                        s2, sq2 = cg_exact_square(tj2, tm2, tj1, tm1, tJ, tm1 + tm2)
                        s3, sq3 = cg_exact_square(tj1, -tm1, tj2, -tm2, tJ, -tm1 - tm2)
                        assert sq == sq2 == sq3
                        assert s2 == ph * s and s3 == ph * s


def test_selection_rules_are_zero():
    assert cg_exact(3, 1, 1, 1, 4, 0) == 0.0       # M != m1+m2
    assert cg_exact(3, 1, 1, 1, 6, 2) == 0.0       # triangle
    assert cg_exact(3, 1, 1, 1, 3, 2) == 0.0       # parity of 2J
    assert cg_exact(2, 2, 2, 2, 2, 4) == 0.0       # |M| > J
    assert cg_exact(3, 5, 1, -1, 4, 4) == 0.0      # |m1| > j1


def _signed_sqrt_products_sum(terms):
    """sum_i s_i*sqrt(a_i)*t_i*sqrt(b_i), exactly: each sqrt(a_i*b_i) is written r*sqrt(q) with q a
    square-free integer (the numbers are factorial-smooth, so trial division terminates), the
    rational coefficients are collected per q.  Returns the rational part (q = 1) and asserts that
    every irrational part cancels exactly."""
    acc = {}
    for (s, a), (t, b) in terms:
        if s == 0 or t == 0:
            continue
        p = a * b
        n = p.numerator * p.denominator          # sqrt(num/den) = sqrt(num*den)/den
        r, q, d = 1, 1, 2
        while d * d <= n:
            while n % (d * d) == 0:
                n //= d * d
                r *= d
            if n % d == 0:
                n //= d
                q *= d
            d += 1
        q *= n
        acc[q] = acc.get(q, Fraction(0)) + s * t * Fraction(r, p.denominator)
    for q, v in acc.items():
        if q != 1:
            assert v == 0, (q, v)
    return acc.get(1, Fraction(0))


def test_orthonormality_exact():
    # sum_{m1 m2} C(J M) C(J' M) = delta_JJ' ; sum_J C(m1 m2) C(m1' m2') = delta delta -- exact rationals
    for tj1 in range(0, 7):
        for tj2 in range(0, 7):
            Js = list(range(abs(tj1 - tj2), tj1 + tj2 + 1, 2))
            for tM in range(-(tj1 + tj2), tj1 + tj2 + 1, 2):
                pairs = [(tm1, tM - tm1) for tm1 in range(-tj1, tj1 + 1, 2) if abs(tM - tm1) <= tj2]
                for J in Js:
                    for Jp in Js:
                        if abs(tM) > J or abs(tM) > Jp:
                            continue
                        if J == Jp:
                            tot = sum(cg_exact_square(tj1, a, tj2, b, J, tM)[1] for a, b in pairs)
                            assert tot == 1
                        else:
                            tot = _signed_sqrt_products_sum(
                                [(cg_exact_square(tj1, a, tj2, b, J, tM), cg_exact_square(tj1, a, tj2, b, Jp, tM))
                                 for a, b in pairs])
                            assert tot == 0
                for (a, b) in pairs:
                    for (c, d) in pairs:
                        tot = _signed_sqrt_products_sum(
                            [(cg_exact_square(tj1, a, tj2, b, J, tM), cg_exact_square(tj1, c, tj2, d, J, tM))
                             for J in Js])
                        assert tot == (1 if (a, b) == (c, d) else 0)


def test_table_matches_function():
    t = CGTable([(3, 5), (4, 3), (1, 1), (0, 1), (2, 1)])
    for (tj1, tj2) in [(3, 5), (4, 3), (1, 1), (0, 1), (2, 1)]:
        for tJ in range(abs(tj1 - tj2), tj1 + tj2 + 1, 2):
            for tm1 in range(-tj1, tj1 + 1, 2):
                for tm2 in range(-tj2, tj2 + 1, 2):
                    assert t.get(tj1, tm1, tj2, tm2, tJ, tm1 + tm2) == cg_exact(tj1, tm1, tj2, tm2, tJ, tm1 + tm2)
