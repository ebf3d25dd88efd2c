"""Seeded synthetic inputs for the coupled-JT -> M-scheme transformation.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_1412_5989_b200/csrc``).  It holds *none of the method's arithmetic*:
no Clebsch-Gordan coefficient, no channel sum, no canonicalisation sign.  It only
lays out inputs: the single-particle basis, the *shape* of the coupled-JT tables
(which states are listed in which channel -- PAPER.md:59 "only these
potentially-nonzero elements are stored"), N(0,1) table values, and request
streams ("a 3-body element request takes the form of a set of six SPS
indices").  Imports numpy only.

Conventions (SURVEY.md section 8 top):
  orbital  o = (n, l, 2j), e = 2n + l, ordered by (e, l, 2j) ascending, 0-based
  SPS      s = (o, 2m, 2tz), orbital-major, then 2tz = +1, -1, then 2m ascending
  2-body coupled state  (a <= b ; J, T, parity),  a == b only if J + T odd
  3-body coupled state  (a <= b <= c, J12, T12 ; 2J, 2T, parity),
                        e_a+e_b+e_c <= E3max, a == b only if J12 + T12 odd
The five configs are BASELINE.json's ``configs[0..4]``.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

# --------------------------------------------------------------------------- basis


@dataclass
class Basis:
    """Orbitals and SPS as flat int32 arrays (PAPER.md:77 'flattened several arrays')."""
    n: np.ndarray
    l: np.ndarray
    twoj: np.ndarray
    sps_orb: np.ndarray
    sps_twom: np.ndarray
    sps_twotz: np.ndarray

    @property
    def n_orb(self) -> int:
        return int(self.n.shape[0])

    @property
    def n_sps(self) -> int:
        return int(self.sps_orb.shape[0])

    @property
    def e(self) -> np.ndarray:
        return 2 * self.n + self.l


def ho_basis(emax: int) -> Basis:
    """Harmonic-oscillator orbitals with 2n+l <= emax, and their SPS (protons+neutrons)."""
    orbs = []
    for e in range(emax + 1):
        for l in range(e % 2, e + 1, 2):
            for twoj in (2 * l - 1, 2 * l + 1):
                if twoj > 0:
                    orbs.append(((e - l) // 2, l, twoj))
    orbs.sort(key=lambda o: (2 * o[0] + o[1], o[1], o[2]))
    n = np.array([o[0] for o in orbs], dtype=np.int32)
    l = np.array([o[1] for o in orbs], dtype=np.int32)
    tj = np.array([o[2] for o in orbs], dtype=np.int32)
    so, sm, st = [], [], []
    for o, (_, _, twoj) in enumerate(orbs):
        for twotz in (1, -1):
            for twom in range(-twoj, twoj + 1, 2):
                so.append(o)
                sm.append(twom)
                st.append(twotz)
    return Basis(n, l, tj, np.array(so, np.int32), np.array(sm, np.int32), np.array(st, np.int32))


# ------------------------------------------------------------------ coupled tables


@dataclass
class Coupled2B:
    """Channel-major 2-body table in exactly the layout ``mfdn_coupled_upload_2b`` takes."""
    chan_J: np.ndarray
    chan_T: np.ndarray
    chan_par: np.ndarray      # 0 = even (+), 1 = odd (-)
    chan_dim: np.ndarray
    chan_off: np.ndarray      # int64 offsets into values
    state_a: np.ndarray
    state_b: np.ndarray
    values: np.ndarray        # float64, sum(chan_dim**2)

    @property
    def n_chan(self) -> int:
        return int(self.chan_J.shape[0])

    def block(self, c: int) -> np.ndarray:
        d = int(self.chan_dim[c])
        o = int(self.chan_off[c])
        return self.values[o:o + d * d].reshape(d, d)

    def state_range(self, c: int):
        s0 = int(np.sum(self.chan_dim[:c]))
        return s0, s0 + int(self.chan_dim[c])


@dataclass
class Coupled3B:
    """Channel-major 3-body table in exactly the layout ``mfdn_coupled_upload_3b`` takes."""
    e3max: int
    chan_twoJ: np.ndarray
    chan_twoT: np.ndarray
    chan_par: np.ndarray
    chan_dim: np.ndarray
    chan_off: np.ndarray
    state_a: np.ndarray
    state_b: np.ndarray
    state_c: np.ndarray
    state_J12: np.ndarray
    state_T12: np.ndarray
    values: np.ndarray

    @property
    def n_chan(self) -> int:
        return int(self.chan_twoJ.shape[0])

    def block(self, c: int) -> np.ndarray:
        d = int(self.chan_dim[c])
        o = int(self.chan_off[c])
        return self.values[o:o + d * d].reshape(d, d)

    def state_range(self, c: int):
        s0 = int(np.sum(self.chan_dim[:c]))
        return s0, s0 + int(self.chan_dim[c])


def _symmetric_normal(rng: np.random.Generator, dims) -> tuple[np.ndarray, np.ndarray]:
    """Per channel: draw the upper triangle incl. diagonal row-major from N(0,1), mirror."""
    dims = np.asarray(dims, dtype=np.int64)
    off = np.zeros(len(dims), dtype=np.int64)
    if len(dims):
        off[1:] = np.cumsum(dims[:-1] ** 2)
    vals = np.empty(int(np.sum(dims ** 2)), dtype=np.float64)
    for c, d in enumerate(dims):
        d = int(d)
        iu = np.triu_indices(d)
        m = np.zeros((d, d))
        m[iu] = rng.standard_normal(iu[0].shape[0])
        m = m + np.triu(m, 1).T
        vals[off[c]:off[c] + d * d] = m.ravel()
    return off, vals


def structure_2b(basis: Basis):
    """List of channels (J,T,par) -> list of (a,b), ascending everywhere."""
    tj, l = basis.twoj, basis.l
    chans: dict[tuple[int, int, int], list[tuple[int, int]]] = {}
    for a in range(basis.n_orb):
        for b in range(a, basis.n_orb):
            par = int((l[a] + l[b]) & 1)
            for J in range(abs(int(tj[a]) - int(tj[b])) // 2, (int(tj[a]) + int(tj[b])) // 2 + 1):
                for T in (0, 1):
                    if a == b and ((J + T) & 1) == 0:
                        continue
                    chans.setdefault((J, T, par), []).append((a, b))
    keys = sorted(chans)
    return keys, [sorted(chans[k]) for k in keys]


def coupled_2b(basis: Basis, seed: int, values: str = "normal") -> Coupled2B:
    keys, states = structure_2b(basis)
    dims = [len(s) for s in states]
    if values == "normal":
        off, vals = _symmetric_normal(np.random.default_rng(seed), dims)
    else:  # "zeros": structure only, caller fills
        off, _ = _offsets(dims)
        vals = np.zeros(int(np.sum(np.asarray(dims, np.int64) ** 2)))
    sa = np.array([s[0] for st in states for s in st], np.int32)
    sb = np.array([s[1] for st in states for s in st], np.int32)
    return Coupled2B(np.array([k[0] for k in keys], np.int32), np.array([k[1] for k in keys], np.int32),
                     np.array([k[2] for k in keys], np.int32), np.array(dims, np.int32), off, sa, sb, vals)


def _offsets(dims):
    dims = np.asarray(dims, dtype=np.int64)
    off = np.zeros(len(dims), dtype=np.int64)
    if len(dims):
        off[1:] = np.cumsum(dims[:-1] ** 2)
    return off, None


def tuples_3b(basis: Basis, e3max: int):
    """Orbital triples a<=b<=c with e_a+e_b+e_c <= E3max, ascending."""
    e = basis.e
    out = []
    for a in range(basis.n_orb):
        for b in range(a, basis.n_orb):
            for c in range(b, basis.n_orb):
                if e[a] + e[b] + e[c] <= e3max:
                    out.append((a, b, c))
    return out


def structure_3b(basis: Basis, e3max: int):
    """List of channels (2J,2T,par) -> list of (a,b,c,J12,T12), ascending everywhere."""
    tj, l = basis.twoj, basis.l
    chans: dict[tuple[int, int, int], list[tuple[int, int, int, int, int]]] = {}
    for (a, b, c) in tuples_3b(basis, e3max):
        ja, jb, jc = int(tj[a]), int(tj[b]), int(tj[c])
        par = int((l[a] + l[b] + l[c]) & 1)
        for J12 in range(abs(ja - jb) // 2, (ja + jb) // 2 + 1):
            for T12 in (0, 1):
                if a == b and ((J12 + T12) & 1) == 0:
                    continue
                for twoJ in range(abs(2 * J12 - jc), 2 * J12 + jc + 1, 2):
                    for twoT in range(abs(2 * T12 - 1), 2 * T12 + 2, 2):
                        chans.setdefault((twoJ, twoT, par), []).append((a, b, c, J12, T12))
    keys = sorted(chans)
    return keys, [sorted(chans[k]) for k in keys]


def coupled_3b(basis: Basis, e3max: int, seed: int, values: str = "normal") -> Coupled3B:
    keys, states = structure_3b(basis, e3max)
    dims = [len(s) for s in states]
    if values == "normal":
        off, vals = _symmetric_normal(np.random.default_rng(seed), dims)
    else:
        off, _ = _offsets(dims)
        vals = np.zeros(int(np.sum(np.asarray(dims, np.int64) ** 2)))
    cols = [np.array([s[i] for st in states for s in st], np.int32) for i in range(5)]
    return Coupled3B(e3max, np.array([k[0] for k in keys], np.int32), np.array([k[1] for k in keys], np.int32),
                     np.array([k[2] for k in keys], np.int32), np.array(dims, np.int32), off, *cols, vals)


# ------------------------------------------------------------------ m-scheme states


@dataclass
class MStates:
    """Canonical m-scheme A-particle states (ascending SPS index inside a state),
    grouped into (M, Tz, parity) sectors.  ``states`` is sector-major."""
    states: np.ndarray       # int32 [n_states][A]
    sec_start: np.ndarray    # int64 [n_sec + 1]
    sec_key: np.ndarray      # int32 [n_sec][3]  = (2M, 2Tz, par), ascending

    @property
    def n_states(self) -> int:
        return int(self.states.shape[0])

    @property
    def n_sec(self) -> int:
        return int(self.sec_key.shape[0])

    @property
    def sec_size(self) -> np.ndarray:
        return np.diff(self.sec_start)

    @property
    def n_conserving_pairs(self) -> int:
        return int(np.sum(self.sec_size.astype(np.int64) ** 2))


def mstates(basis: Basis, A: int, emax_sum: int | None = None, e_single_max: int | None = None) -> MStates:
    """All A-tuples (A = 2 or 3) of distinct SPS, s0 < s1 [< s2], optionally with
    sum of e <= emax_sum and each e <= e_single_max, sorted into sectors."""
    e_s = basis.e[basis.sps_orb].astype(np.int64)
    l_s = basis.l[basis.sps_orb].astype(np.int64)
    m_s = basis.sps_twom.astype(np.int64)
    t_s = basis.sps_twotz.astype(np.int64)
    ok = np.ones(basis.n_sps, bool) if e_single_max is None else (e_s <= e_single_max)
    idx = np.nonzero(ok)[0]
    if A == 2:
        i, j = np.triu_indices(len(idx), 1)
        tup = np.stack([idx[i], idx[j]], axis=1)
    else:
        parts = []
        # enumerate per first index to bound memory
        for p, s0 in enumerate(idx):
            rest = idx[p + 1:]
            if len(rest) < 2:
                continue
            if emax_sum is not None:
                rest = rest[e_s[rest] + e_s[s0] <= emax_sum]
                if len(rest) < 2:
                    continue
            i, j = np.triu_indices(len(rest), 1)
            t = np.stack([np.full(i.shape, s0), rest[i], rest[j]], axis=1)
            if emax_sum is not None:
                t = t[e_s[t].sum(axis=1) <= emax_sum]
            parts.append(t)
        tup = np.concatenate(parts, axis=0)
    if emax_sum is not None and A == 2:
        tup = tup[e_s[tup].sum(axis=1) <= emax_sum]
    M = m_s[tup].sum(axis=1)
    Tz = t_s[tup].sum(axis=1)
    par = l_s[tup].sum(axis=1) & 1
    order = np.lexsort(tuple(tup[:, k] for k in range(A - 1, -1, -1)) + (par, Tz, M))
    tup, M, Tz, par = tup[order], M[order], Tz[order], par[order]
    key = np.stack([M, Tz, par], axis=1)
    change = np.nonzero(np.any(key[1:] != key[:-1], axis=1))[0] + 1
    start = np.concatenate([[0], change, [len(tup)]]).astype(np.int64)
    return MStates(tup.astype(np.int32), start, key[start[:-1]].astype(np.int32))


# ------------------------------------------------------------------ request streams


def all_conserving_pairs(ms: MStates) -> np.ndarray:
    """Every ordered (bra, ket) pair with equal (M, Tz, parity): lexicographic in
    (sector, bra, ket).  int32 [n][2A]."""
    out = []
    for s in range(ms.n_sec):
        st = ms.states[ms.sec_start[s]:ms.sec_start[s + 1]]
        n = st.shape[0]
        bra = np.repeat(st, n, axis=0)
        ket = np.tile(st, (n, 1))
        out.append(np.concatenate([bra, ket], axis=1))
    return np.ascontiguousarray(np.concatenate(out, axis=0), dtype=np.int32)


_CHUNK = 1 << 20


def sampled_pairs(ms: MStates, n: int, seed: int, start: int = 0, permute_frac: float = 0.0,
                  ms_low: MStates | None = None, low_frac: float = 0.0, workers: int = 0) -> np.ndarray:
    """``n`` requests of the stream ``seed`` beginning at request index ``start``.

    The stream is defined chunk-wise (chunks of 2^20, chunk k drawn from
    ``default_rng([seed, k])``) so that any window can be produced without drawing
    the whole stream.  Each request: sector ~ n_s^2, bra and ket independently uniform
    in the sector.  With ``ms_low``/``low_frac`` (config 4, Q17): with
    probability ``low_frac`` the pair is drawn the same way from ``ms_low`` instead.
    ``permute_frac`` of the requests get their bra and ket particle lists randomly
    permuted (exercises the sign path; parity runs only)."""
    A = ms.states.shape[1]
    out = np.empty((n, 2 * A), dtype=np.int32)
    jobs = []   # (chunk, first row of the chunk wanted, one past the last, destination row)
    pos = 0
    k = start // _CHUNK
    while pos < n:
        c0 = k * _CHUNK
        lo = max(start, c0) - c0
        hi = min(start + n, c0 + _CHUNK) - c0
        jobs.append((k, lo, hi, pos))
        pos += hi - lo
        k += 1

    def fill(job):
        k, lo, hi, pos = job
        out[pos:pos + hi - lo] = _sample_chunk(ms, seed, k, permute_frac, ms_low, low_frac)[lo:hi]

    if workers > 1 and len(jobs) > 1:   # chunks are independent streams: the result does not depend on `workers`
        from concurrent.futures import ThreadPoolExecutor
        with ThreadPoolExecutor(workers) as ex:
            list(ex.map(fill, jobs))
    else:
        for job in jobs:
            fill(job)
    return out


def _draw(ms: MStates, rng: np.random.Generator, n: int) -> np.ndarray:
    size = ms.sec_size.astype(np.float64)
    cdf = np.cumsum(size * size)
    cdf /= cdf[-1]
    sec = np.minimum(np.searchsorted(cdf, rng.random(n), side="right"), ms.n_sec - 1)
    ns = ms.sec_size[sec]
    bra = ms.sec_start[sec] + np.minimum((rng.random(n) * ns).astype(np.int64), ns - 1)
    ket = ms.sec_start[sec] + np.minimum((rng.random(n) * ns).astype(np.int64), ns - 1)
    return np.concatenate([ms.states[bra], ms.states[ket]], axis=1)


def _sample_chunk(ms, seed, k, permute_frac, ms_low, low_frac) -> np.ndarray:
    rng = np.random.default_rng([seed, k])
    A = ms.states.shape[1]
    req = _draw(ms, rng, _CHUNK)
    if ms_low is not None and low_frac > 0.0:
        low = _draw(ms_low, rng, _CHUNK)
        pick = rng.random(_CHUNK) < low_frac
        req[pick] = low[pick]
    if permute_frac > 0.0:
        sel = np.nonzero(rng.random(_CHUNK) < permute_frac)[0]
        for side in (0, 1):
            perm = np.argsort(rng.random((len(sel), A)), axis=1)
            blk = req[sel, side * A:(side + 1) * A]
            req[sel, side * A:(side + 1) * A] = np.take_along_axis(blk, perm, axis=1)
    return req.astype(np.int32)


# ------------------------------------------------------------------------- configs


@dataclass
class Config:
    index: int
    name: str
    body: int                 # 2 or 3
    basis: Basis
    table: object             # Coupled2B or Coupled3B
    ms: MStates
    n_requests: int
    all_pairs: bool
    seed_req: int
    ms_low: MStates | None = None
    low_frac: float = 0.0
    n_batches: int = 1
    extra: dict = field(default_factory=dict)

    def requests(self, n: int | None = None, start: int = 0, permute_frac: float = 0.0, workers: int = 0) -> np.ndarray:
        """``workers`` > 1: chunks of the stream drawn by that many host threads (same result)."""
        if self.all_pairs:
            r = all_conserving_pairs(self.ms)
            return r if n is None else r[start:start + n]
        n = self.n_requests if n is None else n
        return sampled_pairs(self.ms, n, self.seed_req, start, permute_frac, self.ms_low, self.low_frac, workers)


def make_config(index: int, table_values: str = "normal") -> Config:
    """BASELINE.json configs[index]; table seed = index, request seed = 1000 + index."""
    if index == 0:
        b = ho_basis(2)
        return Config(0, "2b_emax2_all", 2, b, coupled_2b(b, 0, table_values), mstates(b, 2), 0, True, 1000)
    if index == 1:
        b = ho_basis(8)
        return Config(1, "2b_emax8_2^26", 2, b, coupled_2b(b, 1, table_values), mstates(b, 2), 1 << 26, False, 1001)
    if index == 2:
        b = ho_basis(4)
        return Config(2, "3b_E3max4_all", 3, b, coupled_3b(b, 4, 2, table_values), mstates(b, 3, 4), 0, True, 1002)
    if index == 3:
        b = ho_basis(8)
        return Config(3, "3b_E3max8_2^26", 3, b, coupled_3b(b, 8, 3, table_values), mstates(b, 3, 8), 1 << 26, False, 1003)
    if index == 4:
        b = ho_basis(6)
        ms = mstates(b, 3, 10)
        low = mstates(b, 3, 10, e_single_max=2)
        return Config(4, "3b_E3max10_e6_16x2^24", 3, b, coupled_3b(b, 10, 4, table_values), ms, 1 << 28, False, 1004,
                      ms_low=low, low_frac=0.7, n_batches=16)
    raise ValueError(f"no config {index}")


def many_body_targets(n: int, h_len: int, seed: int, mean_run: float = 4.0):
    """Where MFDn would add the n results (every buffered request carries the many-body element it
    pertains to and a phase): consecutive requests belong to one many-body element in runs of geometric length (mean
    `mean_run`; the recursive loop of PAPER.md:91 asks for the 3-body elements of one many-body element one after the
    other), the element of a run is uniform in [0, h_len), the phase of a request is +1 or -1.  Seeded, no arithmetic of
    the method.  Returns (loc int64 [n], phase float64 [n])."""
    rng = np.random.default_rng([777, seed])
    heads = rng.random(n) < 1.0 / mean_run
    if n:
        heads[0] = True
    run_id = np.cumsum(heads) - 1
    targets = rng.integers(0, h_len, size=int(run_id[-1]) + 1 if n else 0, dtype=np.int64)
    loc = targets[run_id] if n else np.zeros(0, np.int64)
    phase = np.where(rng.random(n) < 0.5, 1.0, -1.0)
    return np.ascontiguousarray(loc, np.int64), np.ascontiguousarray(phase, np.float64)

