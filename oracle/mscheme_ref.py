"""ORACLE (test infrastructure, not product code) -- the coupled-JT -> M-scheme
transformation written out as its definition, in plain Python, one request at a time.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this.  It shares no code with paper_1412_5989_b200/csrc.

What it computes (section 3.1): "an element in the new basis is a linear
combination of elements from the old basis, weighted by the projections in D"
(A' = D^T A D), D "developed from a series of angular momentum and isospin coupling
coefficients"; only the block of A belonging to the request's orbitals contributes and
its elements are reached "with a set of nested loops over coupled angular momentum and
isospin values".  The paper prints no formula; the formulas below are the reading fixed
in DESIGN.md ("Readings", Q1-Q7):

3-body, canonically ordered bra (alpha beta gamma) on orbitals a<=b<=c, ket (delta eps
zeta) on d<=e<=f:
  <abg|V|dez> = sum_{J,T} sum_{J12,T12} sum_{J12',T12'}  B * K * V^{JT}[(abc J12 T12),(def J12' T12')]
  B = <ja ma jb mb|J12 M12> <J12 M12 jc mc|J M> <1/2 ta 1/2 tb|T12 MT12> <T12 MT12 1/2 tc|T MT>
  K = the same with (d e f; delta eps zeta; J12' T12').
2-body, canonically ordered bra (alpha beta) on a<=b, ket (gamma delta) on c<=d:
  <ab|V|gd> = sqrt((1+d_ab)(1+d_cd)) sum_{J,T} <ja ma jb mb|J M><1/2 ta 1/2 tb|T MT>
                                              <jc mc jd md|J M><1/2 tc 1/2 td|T MT> V^{JT}_{ab,cd}

Per request (C2): 1 decode, 2 selection rules S1..S7 (integer only; they define ``mask``),
3 canonicalise (stable sort by (orbital, SPS) ascending, sign = parity of the
permutation), 4 direct sum in the fixed loop order J, T, J12, T12, J12', T12' (ascending),
plain fp64 accumulation, times sign (and the 2-body sqrt factor).

Pinned by tests/test_oracle_pins.py (identity/projector tables, J^2 / J12^2 / T^2 / T12^2
operator tables built from ladder operators with no CG code, trace identity, round trip,
conservation, hermiticity, exchange antisymmetry, brute-force counts).
"""
from __future__ import annotations

from math import sqrt

import numpy as np


class Table2B:
    """Channel-major 2-body table + lookup (J,T,par) -> channel, (a,b) -> row."""

    def __init__(self, t):
        self.t = t
        self.chan = {}
        self.row = []
        s0 = 0
        for c in range(len(t.chan_J)):
            self.chan[(int(t.chan_J[c]), int(t.chan_T[c]), int(t.chan_par[c]))] = c
            d = int(t.chan_dim[c])
            self.row.append({(int(t.state_a[s0 + r]), int(t.state_b[s0 + r])): r for r in range(d)})
            s0 += d
        self.tuples = set(k for r in self.row for k in r)

    def value(self, c, r, q):
        return float(self.t.values[int(self.t.chan_off[c]) + r * int(self.t.chan_dim[c]) + q])


class Table3B:
    """Channel-major 3-body table + lookup (2J,2T,par) -> channel, (a,b,c,J12,T12) -> row."""

    def __init__(self, t):
        self.t = t
        self.e3max = int(t.e3max)
        self.chan = {}
        self.row = []
        s0 = 0
        for c in range(len(t.chan_twoJ)):
            self.chan[(int(t.chan_twoJ[c]), int(t.chan_twoT[c]), int(t.chan_par[c]))] = c
            d = int(t.chan_dim[c])
            self.row.append({(int(t.state_a[s0 + r]), int(t.state_b[s0 + r]), int(t.state_c[s0 + r]),
                              int(t.state_J12[s0 + r]), int(t.state_T12[s0 + r])): r for r in range(d)})
            s0 += d
        self.tuples = set(k[:3] for r in self.row for k in r)
        self.max_twoJ = max(k[0] for k in self.chan) if self.chan else 0

    def value(self, c, r, q):
        return float(self.t.values[int(self.t.chan_off[c]) + r * int(self.t.chan_dim[c]) + q])


def _canonicalise(basis, sps):
    """Stable sort by (orbital, SPS) ascending; sign = (-1)^inversions (C2 step 3)."""
    key = [(int(basis.sps_orb[s]), int(s)) for s in sps]
    inv = 0
    for i in range(len(key)):
        for j in range(i + 1, len(key)):
            if key[i] > key[j]:
                inv += 1
    order = sorted(range(len(key)), key=lambda i: key[i])
    return [int(sps[i]) for i in order], (-1 if (inv & 1) else 1)


def mscheme_2b_one(basis, tab: Table2B, cg, req):
    """One 2-body request (bra0, bra1, ket0, ket1) -> (value, mask, n_terms, bad).
    ``cg(tj1,tm1,tj2,tm2,tJ,tM)`` is the coupling coefficient provider."""
    req = [int(x) for x in req]
    if any(s < 0 or s >= basis.n_sps for s in req):
        return 0.0, 0, 0, 1
    bra, ket = req[:2], req[2:]
    if bra[0] == bra[1] or ket[0] == ket[1]:                                    # S1 Pauli
        return 0.0, 0, 0, 0
    tm = lambda ss: sum(int(basis.sps_twom[s]) for s in ss)
    tt = lambda ss: sum(int(basis.sps_twotz[s]) for s in ss)
    pp = lambda ss: sum(int(basis.l[basis.sps_orb[s]]) for s in ss) & 1
    if tm(bra) != tm(ket) or tt(bra) != tt(ket) or pp(bra) != pp(ket):          # S2 S3 S4
        return 0.0, 0, 0, 0
    bra, sb = _canonicalise(basis, bra)
    ket, sk = _canonicalise(basis, ket)
    a, b = (int(basis.sps_orb[s]) for s in bra)
    c, d = (int(basis.sps_orb[s]) for s in ket)
    if (a, b) not in tab.tuples or (c, d) not in tab.tuples:                    # S6
        return 0.0, 0, 0, 0
    ja, jb, jc, jd = (int(basis.twoj[o]) for o in (a, b, c, d))
    ma, mb = (int(basis.sps_twom[s]) for s in bra)
    mc, md = (int(basis.sps_twom[s]) for s in ket)
    ta, tb = (int(basis.sps_twotz[s]) for s in bra)
    tc, td = (int(basis.sps_twotz[s]) for s in ket)
    twoM, twoMT, par = ma + mb, ta + tb, pp(bra)
    total, nterms = 0.0, 0
    for J in range(0, (max(ja + jb, jc + jd)) // 2 + 1):
        if 2 * J < abs(twoM) or 2 * J < abs(ja - jb) or 2 * J > ja + jb or 2 * J < abs(jc - jd) or 2 * J > jc + jd:
            continue
        for T in (0, 1):
            if 2 * T < abs(twoMT):
                continue
            ch = tab.chan.get((J, T, par))
            if ch is None:
                continue
            r = tab.row[ch].get((a, b))
            q = tab.row[ch].get((c, d))
            if r is None or q is None:
                continue
            B = cg(ja, ma, jb, mb, 2 * J, twoM) * cg(1, ta, 1, tb, 2 * T, twoMT)
            K = cg(jc, mc, jd, md, 2 * J, twoM) * cg(1, tc, 1, td, 2 * T, twoMT)
            total += B * K * tab.value(ch, r, q)
            nterms += 1
    if nterms == 0:                                                              # S7
        return 0.0, 0, 0, 0
    norm = sqrt((2.0 if a == b else 1.0) * (2.0 if c == d else 1.0))
    return sb * sk * norm * total, 1, nterms, 0


def mscheme_3b_one(basis, tab: Table3B, cg, req):
    """One 3-body request (bra0..2, ket0..2) -> (value, mask, n_terms, bad)."""
    req = [int(x) for x in req]
    if any(s < 0 or s >= basis.n_sps for s in req):
        return 0.0, 0, 0, 1
    bra, ket = req[:3], req[3:]
    if len(set(bra)) != 3 or len(set(ket)) != 3:                                # S1 Pauli
        return 0.0, 0, 0, 0
    tm = lambda ss: sum(int(basis.sps_twom[s]) for s in ss)
    tt = lambda ss: sum(int(basis.sps_twotz[s]) for s in ss)
    pp = lambda ss: sum(int(basis.l[basis.sps_orb[s]]) for s in ss) & 1
    ee = lambda ss: sum(int(2 * basis.n[basis.sps_orb[s]] + basis.l[basis.sps_orb[s]]) for s in ss)
    if tm(bra) != tm(ket) or tt(bra) != tt(ket) or pp(bra) != pp(ket):          # S2 S3 S4
        return 0.0, 0, 0, 0
    if ee(bra) > tab.e3max or ee(ket) > tab.e3max:                              # S5
        return 0.0, 0, 0, 0
    bra, sb = _canonicalise(basis, bra)
    ket, sk = _canonicalise(basis, ket)
    a, b, c = (int(basis.sps_orb[s]) for s in bra)
    d, e, f = (int(basis.sps_orb[s]) for s in ket)
    if (a, b, c) not in tab.tuples or (d, e, f) not in tab.tuples:              # S6
        return 0.0, 0, 0, 0
    ja, jb, jc, jd, je, jf = (int(basis.twoj[o]) for o in (a, b, c, d, e, f))
    ma, mb, mc = (int(basis.sps_twom[s]) for s in bra)
    md, me, mf = (int(basis.sps_twom[s]) for s in ket)
    ta, tb, tc = (int(basis.sps_twotz[s]) for s in bra)
    td, te, tf = (int(basis.sps_twotz[s]) for s in ket)
    twoM, twoMT, par = ma + mb + mc, ta + tb + tc, pp(bra)
    total, nterms = 0.0, 0
    for twoJ in range(1, tab.max_twoJ + 1, 2):
        if twoJ < abs(twoM):
            continue
        for twoT in (1, 3):
            if twoT < abs(twoMT):
                continue
            ch = tab.chan.get((twoJ, twoT, par))
            if ch is None:
                continue
            rows = tab.row[ch]
            for J12 in range(abs(ja - jb) // 2, (ja + jb) // 2 + 1):
                if 2 * J12 < abs(ma + mb) or twoJ < abs(2 * J12 - jc) or twoJ > 2 * J12 + jc:
                    continue
                for T12 in (0, 1):
                    if 2 * T12 < abs(ta + tb) or twoT < abs(2 * T12 - 1) or twoT > 2 * T12 + 1:
                        continue
                    r = rows.get((a, b, c, J12, T12))
                    if r is None:
                        continue
                    B = (cg(ja, ma, jb, mb, 2 * J12, ma + mb) * cg(2 * J12, ma + mb, jc, mc, twoJ, twoM)
                         * cg(1, ta, 1, tb, 2 * T12, ta + tb) * cg(2 * T12, ta + tb, 1, tc, twoT, twoMT))
                    for J12p in range(abs(jd - je) // 2, (jd + je) // 2 + 1):
                        if 2 * J12p < abs(md + me) or twoJ < abs(2 * J12p - jf) or twoJ > 2 * J12p + jf:
                            continue
                        for T12p in (0, 1):
                            if 2 * T12p < abs(td + te) or twoT < abs(2 * T12p - 1) or twoT > 2 * T12p + 1:
                                continue
                            q = rows.get((d, e, f, J12p, T12p))
                            if q is None:
                                continue
                            K = (cg(jd, md, je, me, 2 * J12p, md + me) * cg(2 * J12p, md + me, jf, mf, twoJ, twoM)
                                 * cg(1, td, 1, te, 2 * T12p, td + te) * cg(2 * T12p, td + te, 1, tf, twoT, twoMT))
                            total += B * K * tab.value(ch, r, q)
                            nterms += 1
    if nterms == 0:                                                              # S7
        return 0.0, 0, 0, 0
    return sb * sk * total, 1, nterms, 0


def mscheme_batch(basis, table, cg, req):
    """All requests of ``req`` (int [n][4] or [n][6]) -> (values f64[n], mask u8[n],
    n_terms i64[n], bad_count)."""
    req = np.asarray(req)
    three = req.shape[1] == 6
    tab = Table3B(table) if three else Table2B(table)
    one = mscheme_3b_one if three else mscheme_2b_one
    n = req.shape[0]
    val = np.zeros(n)
    mask = np.zeros(n, np.uint8)
    nt = np.zeros(n, np.int64)
    bad = 0
    for i in range(n):
        v, m, t, b = one(basis, tab, cg, req[i])
        val[i], mask[i], nt[i] = v, m, t
        bad += b
    return val, mask, nt, bad
