"""ORACLE (test infrastructure, not product code) -- the step that follows the transformation in MFDn.

PAPER.md:93 ("we must thus also store which many-body element the request pertains to so that it can be added to
the correct many-body element ... the 3-body element is added with a specific phase, which must also be stored with
the request") and PAPER.md:97 ("iterates through the returned three-body elements in the chunk, multiplies them by
the stored phases, and adds them to the array of many-body elements at the stored locations"):

    for i in request order:   H[loc[i]] += phase[i] * v[i]

written out as exactly that loop, in fp64.  A location outside [0, h_len) is skipped (SURVEY.md 8(f) NEXT-1 reading:
the paper does not say; a buffer entry cannot point outside the array it was made for).  Only tests/ may import this.
"""
from __future__ import annotations

import numpy as np


def accumulate(values, loc, phase, h_len: int) -> np.ndarray:
    """H[loc[i]] += phase[i] * values[i] for i = 0, 1, ... (request order); phase None means +1 everywhere."""
    H = [0.0] * int(h_len)
    for i in range(len(values)):
        l = int(loc[i])
        if 0 <= l < h_len:
            H[l] += (1.0 if phase is None else float(phase[i])) * float(values[i])
    return np.asarray(H, dtype=np.float64)
