"""Pins P4-P9 for the transform oracle (oracle/mscheme_ref.py, oracle/mscheme_oracle.c).

The paper prints no matrix element (PAPER.md has no table of values), so the oracle is pinned
by what the mathematics fixes:
  P5 identity / pair-antisymmetriser tables      -> Kronecker deltas
  P6 J^2, J12^2, T^2, T12^2 operator tables      -> matrices built from j_z and ladder operators,
                                                    with NO Clebsch-Gordan code involved
  P4 trace identity, P7 round trip (inverse sum), P8 conservation / hermiticity / antisymmetry,
  P9 brute-force counts (tests/golden/counts.txt).
A dropped term, wrong sign/phase, wrong coupling order or transposed operand fails P5/P6.
"""
import os
from math import sqrt

import numpy as np
import pytest

from paper_1412_5989_b200 import workloads as W
from oracle import cg_exact, mscheme_c, mscheme_ref

GOLD = os.path.join(os.path.dirname(__file__), "golden", "counts.txt")


def golden_counts():
    out = {}
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        out[k] = int(v)
    return out


# ------------------------------------------------------------ ladder-operator machinery (no CG)
def _jz_jp(tj):
    """j_z and j_+ on the basis m = -j..j (ascending): <m+1|j+|m> = sqrt(j(j+1) - m(m+1))."""
    j = tj / 2.0
    ms = [(-tj + 2 * i) / 2.0 for i in range(tj + 1)]
    jz = np.diag(ms)
    jp = np.zeros((tj + 1, tj + 1))
    for i, m in enumerate(ms[:-1]):
        jp[i + 1, i] = sqrt(j * (j + 1) - m * (m + 1))
    return jz, jp


def total_j_squared(tjs, which):
    """(sum_{i in which} j_i)^2 on the product basis of angular momenta tjs (first index slowest)."""
    dims = [t + 1 for t in tjs]
    def embed(op, i):
        mats = [np.eye(d) for d in dims]
        mats[i] = op
        out = mats[0]
        for m in mats[1:]:
            out = np.kron(out, m)
        return out
    N = int(np.prod(dims))
    Jz, Jp = np.zeros((N, N)), np.zeros((N, N))
    for i in which:
        jz, jp = _jz_jp(tjs[i])
        Jz += embed(jz, i)
        Jp += embed(jp, i)
    Jm = Jp.T
    return Jz @ Jz + 0.5 * (Jp @ Jm + Jm @ Jp)


def _fill_diag(table, fn):
    """table.values <- diag(fn(channel index, state index)) per channel."""
    table.values[:] = 0.0
    s0 = 0
    for c in range(table.n_chan):
        d = int(table.chan_dim[c])
        blk = table.block(c)
        for r in range(d):
            blk[r, r] = fn(c, s0 + r)
        s0 += d


def _midx(b, sps_list):
    """index of the (m...) tuple in the product basis, m ascending per particle, first particle slowest."""
    idx = 0
    for s in sps_list:
        tj = int(b.twoj[b.sps_orb[s]])
        idx = idx * (tj + 1) + (int(b.sps_twom[s]) + tj) // 2
    return idx


def _tidx(b, sps_list):
    idx = 0
    for s in sps_list:
        idx = idx * 2 + (int(b.sps_twotz[s]) + 1) // 2
    return idx


# ----------------------------------------------------------------------------- 2-body pins
@pytest.fixture(scope="module")
def cfg0():
    return W.make_config(0)


@pytest.fixture(scope="module")
def cfg2():
    return W.make_config(2)


def _expected_2b_operator(b, req, spatial, which):
    """Antisymmetrised 2-particle element <ab|O|cd> - <ab|O|dc> of a one-plus-two-body operator O that
    is a product  (angular part) x (isospin part)  acting on distinguishable-particle product states."""
    out = np.zeros(len(req))
    cache = {}
    for i, (p, q, r, s) in enumerate(req):
        tot = 0.0
        for sgn, (x, y) in ((1, (r, s)), (-1, (s, r))):
            if b.sps_orb[p] != b.sps_orb[x] or b.sps_orb[q] != b.sps_orb[y]:
                continue
            tjs = (int(b.twoj[b.sps_orb[p]]), int(b.twoj[b.sps_orb[q]]))
            if which == "J":
                if (b.sps_twotz[p], b.sps_twotz[q]) != (b.sps_twotz[x], b.sps_twotz[y]):
                    continue
                if tjs not in cache:
                    cache[tjs] = total_j_squared(tjs, (0, 1))
                tot += sgn * cache[tjs][_midx(b, (p, q)), _midx(b, (x, y))]
            elif which == "T":
                if (b.sps_twom[p], b.sps_twom[q]) != (b.sps_twom[x], b.sps_twom[y]):
                    continue
                if "T" not in cache:
                    cache["T"] = total_j_squared((1, 1), (0, 1))
                tot += sgn * cache["T"][_tidx(b, (p, q)), _tidx(b, (x, y))]
            else:  # identity
                if p == x and q == y:
                    tot += sgn
        out[i] = tot
    return out


@pytest.mark.parametrize("which", ["1", "J", "T"])
def test_2b_operator_tables(cfg0, which):
    """P5/P6: V^{JT} = 1, J(J+1), T(T+1) (times identity) must decouple to the antisymmetrised
    m-scheme matrix of 1, (j1+j2)^2, (t1+t2)^2 built from ladder operators."""
    b = cfg0.basis
    t = W.coupled_2b(b, 0, "zeros")
    f = {"1": lambda c, s: 1.0, "J": lambda c, s: t.chan_J[c] * (t.chan_J[c] + 1.0),
         "T": lambda c, s: t.chan_T[c] * (t.chan_T[c] + 1.0)}[which]
    _fill_diag(t, f)
    req = cfg0.requests()
    # add non-canonical particle orders (sign path)
    rng = np.random.default_rng(5)
    sw = req[rng.choice(len(req), 2000, replace=False)].copy()
    sw[:1000, [0, 1]] = sw[:1000, [1, 0]]
    sw[500:1500, [2, 3]] = sw[500:1500, [3, 2]]
    req = np.concatenate([req, sw])
    val, mask, _, bad = mscheme_c.mscheme(b, t, req)
    want = _expected_2b_operator(b, req, None, which)
    assert bad == 0
    assert np.max(np.abs(val - want)) < 5e-14
    assert np.all(val[mask == 0] == 0.0)


def test_2b_trace_identity(cfg0):
    """P4: sum over canonical m-states on orbitals (a,b) of <ab|V|ab> = sum_{JT}(2J+1)(2T+1)V^{JT}_{ab,ab}."""
    b, t = cfg0.basis, cfg0.table
    ms = cfg0.ms.states
    diag = np.concatenate([ms, ms], axis=1)
    val, mask, _, _ = mscheme_c.mscheme(b, t, diag)
    oa, ob = b.sps_orb[ms[:, 0]], b.sps_orb[ms[:, 1]]
    s0 = 0
    want = {}
    for c in range(t.n_chan):
        d = int(t.chan_dim[c])
        blk = t.block(c)
        for r in range(d):
            k = (int(t.state_a[s0 + r]), int(t.state_b[s0 + r]))
            want[k] = want.get(k, 0.0) + (2 * t.chan_J[c] + 1) * (2 * t.chan_T[c] + 1) * blk[r, r]
        s0 += d
    for (a, bb), w in want.items():
        got = val[(oa == a) & (ob == bb)].sum()
        assert got == pytest.approx(w, abs=1e-12)


def test_2b_round_trip(cfg0):
    """P7: coupling the oracle's m-scheme output back with the inverse CG sum recovers V^{JT}."""
    b, t = cfg0.basis, cfg0.table
    cg = cg_exact.cg_exact
    sps_of = {o: [s for s in range(b.n_sps) if b.sps_orb[s] == o] for o in range(b.n_orb)}
    rng = np.random.default_rng(7)
    s_start = np.concatenate([[0], np.cumsum(t.chan_dim)])
    checked = 0
    for c in rng.permutation(t.n_chan)[:8]:
        J, T = int(t.chan_J[c]), int(t.chan_T[c])
        d = int(t.chan_dim[c])
        for r in range(d):
            for q in rng.permutation(d)[:3]:
                a, bb = int(t.state_a[s_start[c] + r]), int(t.state_b[s_start[c] + r])
                cc, dd = int(t.state_a[s_start[c] + q]), int(t.state_b[s_start[c] + q])
                tM, tMT = 2 * J - 2 * (r % (J + 1)), 0 if T == 0 else 2 * ((r % 3) - 1)   # any |M|<=J, |MT|<=T
                reqs, wts = [], []
                for p in sps_of[a]:
                    for p2 in sps_of[bb]:
                        wb = (cg(int(b.twoj[a]), int(b.sps_twom[p]), int(b.twoj[bb]), int(b.sps_twom[p2]), 2 * J, tM)
                              * cg(1, int(b.sps_twotz[p]), 1, int(b.sps_twotz[p2]), 2 * T, tMT))
                        if wb == 0.0:
                            continue
                        for x in sps_of[cc]:
                            for y in sps_of[dd]:
                                wk = (cg(int(b.twoj[cc]), int(b.sps_twom[x]), int(b.twoj[dd]), int(b.sps_twom[y]), 2 * J, tM)
                                      * cg(1, int(b.sps_twotz[x]), 1, int(b.sps_twotz[y]), 2 * T, tMT))
                                if wk != 0.0:
                                    reqs.append((p, p2, x, y))
                                    wts.append(wb * wk)
                val, _, _, _ = mscheme_c.mscheme(b, t, np.array(reqs, np.int32))
                norm = sqrt((2.0 if a == bb else 1.0) * (2.0 if cc == dd else 1.0))
                back = float(np.dot(val, wts)) / norm
                assert back == pytest.approx(t.block(c)[r, q], abs=1e-13)
                checked += 1
    assert checked > 50


def test_2b_conservation_hermiticity_antisymmetry(cfg0):
    """P8."""
    b, t = cfg0.basis, cfg0.table
    rng = np.random.default_rng(11)
    req = rng.integers(0, b.n_sps, size=(20000, 4)).astype(np.int32)
    val, mask, nt, bad = mscheme_c.mscheme(b, t, req)
    M = b.sps_twom[req]
    Tz = b.sps_twotz[req]
    P = b.l[b.sps_orb[req]]
    viol = ((M[:, 0] + M[:, 1] != M[:, 2] + M[:, 3]) | (Tz[:, 0] + Tz[:, 1] != Tz[:, 2] + Tz[:, 3])
            | (((P[:, 0] + P[:, 1] + P[:, 2] + P[:, 3]) & 1) == 1) | (req[:, 0] == req[:, 1]) | (req[:, 2] == req[:, 3]))
    assert viol.sum() > 1000 and (~viol).sum() > 100
    assert np.all(val[viol] == 0.0) and np.all(mask[viol] == 0)
    herm, *_ = mscheme_c.mscheme(b, t, req[:, [2, 3, 0, 1]])
    assert np.max(np.abs(herm - val)) < 1e-14
    swap, mask2, _, _ = mscheme_c.mscheme(b, t, req[:, [1, 0, 2, 3]])
    assert np.array_equal(swap, -val) and np.array_equal(mask2, mask)
    # out-of-range indices: value 0, mask 0, counted
    bad_req = req[:10].copy()
    bad_req[::2, 1] = b.n_sps
    bad_req[1::2, 2] = -1
    v, m, _, nb = mscheme_c.mscheme(b, t, bad_req)
    assert nb == 10 and np.all(v == 0.0) and np.all(m == 0)


# ----------------------------------------------------------------------------- 3-body pins
def _expected_3b_operator(b, req, which):
    """Same-tuple product-basis element of 1, (ja+jb+jc)^2, (ja+jb)^2, (ta+tb+tc)^2, (ta+tb)^2 for canonical
    requests on DISTINCT orbitals a<b<c; 0 when the orbital tuples differ."""
    out = np.zeros(len(req))
    cache = {}
    for i, r in enumerate(req):
        bra, ket = r[:3], r[3:]
        if tuple(b.sps_orb[bra]) != tuple(b.sps_orb[ket]):
            continue
        same_m = tuple(b.sps_twom[bra]) == tuple(b.sps_twom[ket])
        same_t = tuple(b.sps_twotz[bra]) == tuple(b.sps_twotz[ket])
        if which == "1":
            out[i] = 1.0 if (same_m and same_t) else 0.0
        elif which in ("J", "J12"):
            if not same_t:
                continue
            tjs = tuple(int(x) for x in b.twoj[b.sps_orb[bra]])
            k = (tjs, which)
            if k not in cache:
                cache[k] = total_j_squared(tjs, (0, 1, 2) if which == "J" else (0, 1))
            out[i] = cache[k][_midx(b, bra), _midx(b, ket)]
        else:
            if not same_m:
                continue
            if which not in cache:
                cache[which] = total_j_squared((1, 1, 1), (0, 1, 2) if which == "T" else (0, 1))
            out[i] = cache[which][_tidx(b, bra), _tidx(b, ket)]
    return out


@pytest.mark.parametrize("which", ["1", "J", "J12", "T", "T12"])
def test_3b_operator_tables(cfg2, which):
    """P5/P6 for tuples a<b<c (distinct orbitals): fixes Condon-Shortley phases, the coupling order
    [(ab)J12 c]J and [(ta tb)T12 tc]T, and which pair couples first."""
    b = cfg2.basis
    t = W.coupled_3b(b, 4, 2, "zeros")
    f = {"1": lambda c, s: 1.0,
         "J": lambda c, s: (t.chan_twoJ[c] / 2.0) * (t.chan_twoJ[c] / 2.0 + 1.0),
         "T": lambda c, s: (t.chan_twoT[c] / 2.0) * (t.chan_twoT[c] / 2.0 + 1.0),
         "J12": lambda c, s: t.state_J12[s] * (t.state_J12[s] + 1.0),
         "T12": lambda c, s: t.state_T12[s] * (t.state_T12[s] + 1.0)}[which]
    _fill_diag(t, f)
    req = cfg2.requests()
    ob, ok = b.sps_orb[req[:, :3]], b.sps_orb[req[:, 3:]]
    distinct = ((ob[:, 0] < ob[:, 1]) & (ob[:, 1] < ob[:, 2]) & (ok[:, 0] < ok[:, 1]) & (ok[:, 1] < ok[:, 2]))
    same = np.all(ob == ok, axis=1)
    other = np.nonzero(distinct & ~same)[0]
    other = other[np.random.default_rng(3).choice(len(other), 20000, replace=False)]
    req = np.concatenate([req[distinct & same], req[other]])
    val, mask, _, _ = mscheme_c.mscheme(b, t, req)
    want = _expected_3b_operator(b, req, which)
    assert np.count_nonzero(want) > 2000
    assert np.max(np.abs(val - want)) < 5e-14


def test_3b_identity_with_repeated_orbitals(cfg2):
    """a=b: only J12+T12 odd is listed, so the identity table is the pair antisymmetriser
    (1-P12)/2 on the first two particles; for canonical requests that is delta/2.
    b=c (a<b): nothing is excluded, identity -> plain delta."""
    b = cfg2.basis
    t = W.coupled_3b(b, 4, 2, "zeros")
    _fill_diag(t, lambda c, s: 1.0)
    req = cfg2.requests()
    ob, ok = b.sps_orb[req[:, :3]], b.sps_orb[req[:, 3:]]
    same_tuple = np.all(ob == ok, axis=1)
    val, mask, _, _ = mscheme_c.mscheme(b, t, req)
    eq = np.all(req[:, :3] == req[:, 3:], axis=1)
    ab = ob[:, 0] == ob[:, 1]
    want = np.where(eq, np.where(ab, 0.5, 1.0), 0.0)
    assert np.max(np.abs(val - want)[same_tuple]) < 5e-14
    assert np.max(np.abs(val[~same_tuple])) == 0.0 or np.max(np.abs(val[~same_tuple])) < 5e-14
    # permuting particles multiplies by the permutation sign
    sub = req[eq & ~ab][:2000]
    perm = sub[:, [1, 0, 2, 3, 4, 5]]
    v2, *_ = mscheme_c.mscheme(b, t, perm)
    assert np.allclose(v2, -1.0, atol=5e-14)
    perm = sub[:, [1, 2, 0, 5, 3, 4]]      # two cyclic (even) permutations
    v3, *_ = mscheme_c.mscheme(b, t, perm)
    assert np.allclose(v3, 1.0, atol=5e-14)


def _small_3b():
    b = W.ho_basis(1)
    return b, W.coupled_3b(b, 3, 99)


def test_3b_trace_and_round_trip_tiny():
    """P4 + P7 on a tiny basis (e<=1, E3max=3), tuples with b<c (for b=c a random table is not
    recoupling-consistent, so the raw all-orderings sum is not what canonical requests
    return).  Round trip: V^{JT}[(abc J12 T12),(def J12' T12')] = sum_{all m,tz} B K <abg|V|dez>."""
    b, t = _small_3b()
    cg = cg_exact.cg_exact
    sps_of = {o: [s for s in range(b.n_sps) if b.sps_orb[s] == o] for o in range(b.n_orb)}
    s_start = np.concatenate([[0], np.cumsum(t.chan_dim)])

    def weights(orbs, J12, T12, tJ, tT, tM, tMT):
        out = []
        ja, jb, jc = (int(b.twoj[o]) for o in orbs)
        for p in sps_of[orbs[0]]:
            for q in sps_of[orbs[1]]:
                for r in sps_of[orbs[2]]:
                    m = [int(b.sps_twom[s]) for s in (p, q, r)]
                    z = [int(b.sps_twotz[s]) for s in (p, q, r)]
                    w = (cg(ja, m[0], jb, m[1], 2 * J12, m[0] + m[1]) * cg(2 * J12, m[0] + m[1], jc, m[2], tJ, tM)
                         * cg(1, z[0], 1, z[1], 2 * T12, z[0] + z[1]) * cg(2 * T12, z[0] + z[1], 1, z[2], tT, tMT))
                    if w != 0.0:
                        out.append(((p, q, r), w))
        return out

    rng = np.random.default_rng(1)
    checked = 0
    for c in range(t.n_chan):
        tJ, tT = int(t.chan_twoJ[c]), int(t.chan_twoT[c])
        d = int(t.chan_dim[c])
        st = [(int(t.state_a[s_start[c] + r]), int(t.state_b[s_start[c] + r]), int(t.state_c[s_start[c] + r]),
               int(t.state_J12[s_start[c] + r]), int(t.state_T12[s_start[c] + r])) for r in range(d)]
        ok_rows = [r for r in range(d) if st[r][1] < st[r][2]]
        for r in rng.permutation(ok_rows)[:4]:
            for q in rng.permutation(ok_rows)[:3]:
                tM = tJ - 2 * int(rng.integers(0, tJ + 1))
                tMT = tT - 2 * int(rng.integers(0, tT + 1))
                wb = weights(st[r][:3], st[r][3], st[r][4], tJ, tT, tM, tMT)
                wk = weights(st[q][:3], st[q][3], st[q][4], tJ, tT, tM, tMT)
                reqs = np.array([x + y for x, _ in wb for y, _ in wk], np.int32)
                wts = np.array([u * v for _, u in wb for _, v in wk])
                val, *_ = mscheme_c.mscheme(b, t, reqs)
                assert float(np.dot(val, wts)) == pytest.approx(t.block(c)[r, q], abs=1e-13)
                checked += 1
    assert checked > 40
    # trace identity for tuples a<b<c: sum over canonical m-states = sum (2J+1)(2T+1) V[chi,chi]
    ms = W.mstates(b, 3, 3).states
    orb = b.sps_orb[ms]
    val, *_ = mscheme_c.mscheme(b, t, np.concatenate([ms, ms], axis=1))
    want = {}
    s0 = 0
    for c in range(t.n_chan):
        blk = t.block(c)
        for r in range(int(t.chan_dim[c])):
            k = (int(t.state_a[s0 + r]), int(t.state_b[s0 + r]), int(t.state_c[s0 + r]))
            want[k] = want.get(k, 0.0) + (t.chan_twoJ[c] + 1) * (t.chan_twoT[c] + 1) * blk[r, r]
        s0 += int(t.chan_dim[c])
    n = 0
    for (a, bb, cc), w in want.items():
        if a < bb < cc:
            got = val[(orb[:, 0] == a) & (orb[:, 1] == bb) & (orb[:, 2] == cc)].sum()
            assert got == pytest.approx(w, abs=1e-12)
            n += 1
    assert n >= 1


def test_3b_conservation_hermiticity_pair_antisymmetry(cfg2):
    """P8."""
    b, t = cfg2.basis, cfg2.table
    rng = np.random.default_rng(13)
    allreq = cfg2.requests()
    req = np.concatenate([rng.integers(0, 40, size=(20000, 6)).astype(np.int32),   # mostly violating
                          allreq[rng.choice(len(allreq), 5000, replace=False)]])   # conserving
    val, mask, nt, bad = mscheme_c.mscheme(b, t, req)
    M, Tz, L = b.sps_twom[req], b.sps_twotz[req], b.l[b.sps_orb[req]]
    E = b.e[b.sps_orb[req]]
    viol = ((M[:, :3].sum(1) != M[:, 3:].sum(1)) | (Tz[:, :3].sum(1) != Tz[:, 3:].sum(1)) | ((L.sum(1) & 1) == 1)
            | (E[:, :3].sum(1) > 4) | (E[:, 3:].sum(1) > 4)
            | (req[:, 0] == req[:, 1]) | (req[:, 0] == req[:, 2]) | (req[:, 1] == req[:, 2])
            | (req[:, 3] == req[:, 4]) | (req[:, 3] == req[:, 5]) | (req[:, 4] == req[:, 5]))
    assert viol.sum() > 1000 and (~viol).sum() > 200
    assert np.all(val[viol] == 0.0) and np.all(mask[viol] == 0)
    herm, *_ = mscheme_c.mscheme(b, t, req[:, [3, 4, 5, 0, 1, 2]])
    assert np.max(np.abs(herm - val)) < 1e-13
    # any particle permutation = permutation sign (canonicalisation), bitwise
    odd, m2, *_ = mscheme_c.mscheme(b, t, req[:, [0, 2, 1, 3, 4, 5]])
    assert np.array_equal(odd, -val) and np.array_equal(m2, mask)
    even, *_ = mscheme_c.mscheme(b, t, req[:, [2, 0, 1, 4, 5, 3]])
    assert np.array_equal(even, val)
    # global tz flip leaves the value unchanged (species label immaterial)
    flip = req.copy()
    for k in range(6):
        s = req[:, k]
        o, tz = b.sps_orb[s], b.sps_twotz[s]
        first = np.searchsorted(b.sps_orb, o)               # first SPS of that orbital (tz=+1 block)
        nm = b.twoj[o] + 1
        flip[:, k] = np.where(tz == 1, s + nm, s - nm)
    vf, mf, *_ = mscheme_c.mscheme(b, t, flip)
    # ... except where two particles tie on orbitals b = c: there the SPS tie-break picks which
    # particle couples first and a random table is not recoupling-consistent
    so_b, so_k = np.sort(b.sps_orb[req[:, :3]], axis=1), np.sort(b.sps_orb[req[:, 3:]], axis=1)
    notie = (so_b[:, 1] < so_b[:, 2]) & (so_k[:, 1] < so_k[:, 2])
    assert notie.sum() > 5000 and np.count_nonzero(val[notie]) > 500
    assert np.array_equal(mf[notie], mask[notie]) and np.max(np.abs(vf - val)[notie]) < 1e-13


# ----------------------------------------------------------------------------- counts + C vs Python
def test_counts_and_python_agreement(cfg0, cfg2):
    """P9 + the C oracle equals the pure-Python definition request by request."""
    g = golden_counts()
    for cfg in (cfg0, cfg2):
        i = cfg.index
        tb = cfg.table
        assert cfg.basis.n_sps == g[f"cfg{i}.sps"]
        assert tb.n_chan == g[f"cfg{i}.channels"] and tb.chan_dim.max() == g[f"cfg{i}.max_dim"]
        assert tb.values.size == g[f"cfg{i}.coupled_elements"]
        assert cfg.ms.n_states == g[f"cfg{i}.mstates"] and cfg.ms.n_sec == g[f"cfg{i}.sectors"]
        assert cfg.ms.sec_size.max() == g[f"cfg{i}.largest_sector"]
        assert cfg.ms.n_conserving_pairs == g[f"cfg{i}.conserving_pairs"]
        req = cfg.requests()
        val, mask, nt, bad = mscheme_c.mscheme(cfg.basis, tb, req)
        assert int(mask.sum()) == g[f"cfg{i}.mask1"]
        assert int(nt.sum()) == g[f"cfg{i}.total_terms"]
        assert bad == 0
        # hermiticity over the full (symmetric) request set: value(bra,ket) == value(ket,bra)
        A = cfg.body
        swapped, *_ = mscheme_c.mscheme(cfg.basis, tb, np.concatenate([req[:, A:], req[:, :A]], axis=1))
        assert np.max(np.abs(swapped - val)) < 1e-13
        idx = np.random.default_rng(i).choice(len(req), 400, replace=False)
        cg = mscheme_c.cg_table_for(cfg.basis, A)
        v2, m2, n2, _ = mscheme_ref.mscheme_batch(cfg.basis, tb, cg.get, req[idx])
        assert np.array_equal(v2, val[idx]) and np.array_equal(m2, mask[idx]) and np.array_equal(n2, nt[idx])
        # and with on-the-fly exact coefficients instead of the table
        v3, *_ = mscheme_ref.mscheme_batch(cfg.basis, tb, cg_exact.cg_exact, req[idx[:100]])
        assert np.array_equal(v3, val[idx[:100]])


def test_structure_counts_large_configs():
    g = golden_counts()
    for i, (emax, body) in ((1, (8, 2)), (3, (8, 3))):
        b = W.ho_basis(emax)
        if body == 2:
            keys, states = W.structure_2b(b)
            ms = W.mstates(b, 2)
        else:
            keys, states = W.structure_3b(b, 8)
            ms = W.mstates(b, 3, 8)
        dims = np.array([len(s) for s in states], np.int64)
        assert b.n_sps == g[f"cfg{i}.sps"] and len(keys) == g[f"cfg{i}.channels"]
        assert dims.max() == g[f"cfg{i}.max_dim"] and int((dims ** 2).sum()) == g[f"cfg{i}.coupled_elements"]
        assert ms.n_states == g[f"cfg{i}.mstates"] and ms.n_sec == g[f"cfg{i}.sectors"]
        assert ms.sec_size.max() == g[f"cfg{i}.largest_sector"]
        if i == 3:
            assert ms.n_conserving_pairs == g["cfg3.conserving_pairs"]


# --------------------------------------------------------------------------------- NEXT-1: the accumulate step
def test_accumulate_definition_pins():
    """oracle/accumulate_ref.py against what the definition fixes without re-typing it: one request per location gives
    phase * v; one location for all requests gives the exactly rounded sum (math.fsum) within n ulp; the total is
    conserved; out-of-range locations are dropped; numpy's unbuffered add.at (a library routine) agrees."""
    import math
    from oracle.accumulate_ref import accumulate
    from paper_1412_5989_b200 import workloads as Wl
    rng = np.random.default_rng(3)
    n = 5000
    v = rng.standard_normal(n)
    ph = np.where(rng.random(n) < 0.5, 1.0, -1.0)
    H = accumulate(v, np.arange(n), ph, n)
    assert np.array_equal(H, ph * v)
    H = accumulate(v, np.arange(n)[::-1], None, n)
    assert np.array_equal(H, v[::-1])
    H = accumulate(v, np.zeros(n, np.int64), ph, 3)
    assert H[1] == 0.0 and H[2] == 0.0
    assert abs(H[0] - math.fsum(ph * v)) <= n * np.finfo(float).eps * float(np.sum(np.abs(v)))
    loc, phase = Wl.many_body_targets(n, 700, seed=1)
    assert loc.min() >= 0 and loc.max() < 700 and set(np.unique(phase)) == {-1.0, 1.0}
    assert 2.5 < n / (1 + np.count_nonzero(np.diff(loc))) < 6.0          # runs of mean length about 4
    H = accumulate(v, loc, phase, 700)
    assert abs(math.fsum(H) - math.fsum(phase * v)) <= 1e-12
    ref = np.zeros(700)
    np.add.at(ref, loc, phase * v)
    assert np.array_equal(H, ref)
    bad = loc.copy()
    bad[::7] = -1
    bad[3::11] = 700
    keep = (bad >= 0) & (bad < 700)
    assert np.array_equal(accumulate(v, bad, phase, 700), accumulate(v[keep], bad[keep], phase[keep], 700))
