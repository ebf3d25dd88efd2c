"""ORACLE (test infrastructure, not product code) -- exact Clebsch-Gordan coefficients.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this.  It shares no code with paper_1412_5989_b200/csrc.

The paper gives no formula for the projection matrix D ("D is developed from a series
of angular momentum and isospin coupling coefficients"); the reading
(Q1/Q2) is the Condon-Shortley Clebsch-Gordan coefficient
in Racah's closed form, evaluated here in EXACT rational arithmetic:

  <j1 m1 j2 m2 | J M> = delta(M, m1+m2) * sqrt(P) * S
  P = (2J+1) (j1+j2-J)! (j1-j2+J)! (-j1+j2+J)! / (j1+j2+J+1)!
      * (J+M)! (J-M)! (j1-m1)! (j1+m1)! (j2-m2)! (j2+m2)!
  S = sum_k (-1)^k / [ k! (j1+j2-J-k)! (j1-m1-k)! (j2+m2-k)! (J-j2+m1+k)! (J-j1-m2+k)! ]

P and S are Fractions; the value is sign(S) * sqrt(P*S^2) with P*S^2 converted to the
nearest double (Python's int/int true division is correctly rounded) and one
``math.sqrt`` (<= 1 ulp total).  All arguments are DOUBLED integers (tj = 2j, tm = 2m).

Pinned (tests/test_oracle_cg.py) by closed forms, symmetries and exact orthonormality.
"""
from __future__ import annotations

from fractions import Fraction
from functools import lru_cache
from math import factorial, sqrt

import numpy as np


def cg_allowed(tj1: int, tm1: int, tj2: int, tm2: int, tJ: int, tM: int) -> bool:
    """Integer selection rules of the coefficient (everything that makes it identically 0)."""
    if tm1 + tm2 != tM:
        return False
    if tJ < abs(tj1 - tj2) or tJ > tj1 + tj2 or ((tj1 + tj2 + tJ) & 1):
        return False
    if abs(tm1) > tj1 or abs(tm2) > tj2 or abs(tM) > tJ:
        return False
    if ((tj1 + tm1) & 1) or ((tj2 + tm2) & 1) or ((tJ + tM) & 1):
        return False
    return True


def cg_exact_square(tj1: int, tm1: int, tj2: int, tm2: int, tJ: int, tM: int):
    """(sign, P*S^2) with sign in {-1, 0, +1} and P*S^2 an exact Fraction."""
    return _cg_exact_square(int(tj1), int(tm1), int(tj2), int(tm2), int(tJ), int(tM))   # no numpy ints


@lru_cache(maxsize=None)
def _cg_exact_square(tj1: int, tm1: int, tj2: int, tm2: int, tJ: int, tM: int):
    if not cg_allowed(tj1, tm1, tj2, tm2, tJ, tM):
        return 0, Fraction(0)
    f = factorial
    h = lambda x: x // 2  # all arguments below are even by the selection rules
    a = h(tj1 + tj2 - tJ)
    b = h(tj1 - tm1)
    c = h(tj2 + tm2)
    d = h(tJ - tj2 + tm1)
    e = h(tJ - tj1 - tm2)
    P = Fraction((tJ + 1) * f(a) * f(h(tj1 - tj2 + tJ)) * f(h(-tj1 + tj2 + tJ)), f(h(tj1 + tj2 + tJ) + 1))
    P *= f(h(tJ + tM)) * f(h(tJ - tM)) * f(b) * f(h(tj1 + tm1)) * f(h(tj2 - tm2)) * f(c)
    S = Fraction(0)
    for k in range(max(0, -d, -e), min(a, b, c) + 1):
        term = Fraction(1, f(k) * f(a - k) * f(b - k) * f(c - k) * f(d + k) * f(e + k))
        S += -term if (k & 1) else term
    if S == 0:
        return 0, Fraction(0)
    return (1 if S > 0 else -1), P * S * S


def cg_exact(tj1: int, tm1: int, tj2: int, tm2: int, tJ: int, tM: int) -> float:
    """<j1 m1 j2 m2 | J M>, Condon-Shortley, as the double nearest (<= 1 ulp) to the exact value."""
    s, sq = cg_exact_square(tj1, tm1, tj2, tm2, tJ, tM)
    if s == 0:
        return 0.0
    return s * sqrt(sq.numerator / sq.denominator)


class CGTable:
    """Flat table of exact CGs for a set of (2j1, 2j2) pairs, for the C oracle.

    Block (tj1, tj2) holds [iJ][i1][i2] with iJ = (tJ - |tj1-tj2|)/2, i1 = (tm1+tj1)/2,
    i2 = (tm2+tj2)/2, value <j1 m1 j2 m2 | J m1+m2> (0 where |m1+m2| > J).
    ``off[tj1 * dim2 + tj2]`` is the block start or -1."""

    def __init__(self, pairs):
        pairs = sorted(set((int(a), int(b)) for a, b in pairs))
        self.dim1 = max(p[0] for p in pairs) + 1
        self.dim2 = max(p[1] for p in pairs) + 1
        self.off = np.full(self.dim1 * self.dim2, -1, dtype=np.int64)
        chunks = []
        pos = 0
        for (tj1, tj2) in pairs:
            nJ = min(tj1, tj2) + 1
            blk = np.zeros((nJ, tj1 + 1, tj2 + 1))
            for iJ in range(nJ):
                tJ = abs(tj1 - tj2) + 2 * iJ
                for i1 in range(tj1 + 1):
                    tm1 = 2 * i1 - tj1
                    for i2 in range(tj2 + 1):
                        tm2 = 2 * i2 - tj2
                        blk[iJ, i1, i2] = cg_exact(tj1, tm1, tj2, tm2, tJ, tm1 + tm2)
            self.off[tj1 * self.dim2 + tj2] = pos
            chunks.append(blk.ravel())
            pos += blk.size
        self.val = np.concatenate(chunks)

    def get(self, tj1, tm1, tj2, tm2, tJ, tM) -> float:
        if not cg_allowed(tj1, tm1, tj2, tm2, tJ, tM):
            return 0.0
        o = self.off[tj1 * self.dim2 + tj2]
        assert o >= 0
        iJ = (tJ - abs(tj1 - tj2)) // 2
        return float(self.val[o + (iJ * (tj1 + 1) + (tm1 + tj1) // 2) * (tj2 + 1) + (tm2 + tj2) // 2])


def pairs_needed_2b(twoj_orb) -> list:
    tjs = sorted(set(int(x) for x in twoj_orb))
    return [(a, b) for a in tjs for b in tjs] + [(1, 1)]


def pairs_needed_3b(twoj_orb) -> list:
    tjs = sorted(set(int(x) for x in twoj_orb))
    pairs = [(a, b) for a in tjs for b in tjs]
    tjmax = max(tjs)
    pairs += [(2 * J12, c) for J12 in range(0, tjmax + 1) for c in tjs]
    pairs += [(1, 1), (0, 1), (2, 1)]
    return pairs
