"""ORACLE (test infrastructure, not product code) -- ctypes loader for mscheme_oracle.c.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this.  ``build()`` compiles the C file with gcc (no CUDA); the coupling
coefficients are the exact ones of oracle/cg_exact.py.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

from . import cg_exact

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mscheme_oracle.c")
_LIB = os.path.join(_HERE, "libmscheme_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"])
    return _LIB


class _Basis(C.Structure):
    _fields_ = [("n_orb", C.c_int), ("orb_n", C.c_void_p), ("orb_l", C.c_void_p), ("orb_twoj", C.c_void_p),
                ("n_sps", C.c_int), ("sps_orb", C.c_void_p), ("sps_twom", C.c_void_p), ("sps_twotz", C.c_void_p),
                ("cg_dim1", C.c_int), ("cg_dim2", C.c_int), ("cg_off", C.c_void_p), ("cg_val", C.c_void_p)]


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_num_threads.restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


_cg_cache: dict = {}


def cg_table_for(basis, body: int) -> cg_exact.CGTable:
    key = (body, tuple(sorted(set(int(x) for x in basis.twoj))))
    if key not in _cg_cache:
        pairs = cg_exact.pairs_needed_3b(basis.twoj) if body == 3 else cg_exact.pairs_needed_2b(basis.twoj)
        _cg_cache[key] = cg_exact.CGTable(pairs)
    return _cg_cache[key]


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def mscheme(basis, table, req, n_threads: int = 0, cg: cg_exact.CGTable | None = None):
    """Oracle transform of all requests -> (values f64[n], mask u8[n], n_terms i64[n], bad_count)."""
    lib = _load()
    req = np.ascontiguousarray(req, dtype=np.int32)
    body = req.shape[1] // 2
    cg = cg or cg_table_for(basis, body)
    keep = [_i32(basis.n), _i32(basis.l), _i32(basis.twoj), _i32(basis.sps_orb), _i32(basis.sps_twom),
            _i32(basis.sps_twotz), np.ascontiguousarray(cg.off, np.int64), np.ascontiguousarray(cg.val, np.float64)]
    b = _Basis(basis.n_orb, _p(keep[0]), _p(keep[1]), _p(keep[2]), basis.n_sps, _p(keep[3]), _p(keep[4]), _p(keep[5]),
               cg.dim1, cg.dim2, _p(keep[6]), _p(keep[7]))
    n = req.shape[0]
    out = np.zeros(n, np.float64)
    mask = np.zeros(n, np.uint8)
    nt = np.zeros(n, np.int64)
    bad = C.c_int64(0)
    vals = np.ascontiguousarray(table.values, np.float64)
    off = np.ascontiguousarray(table.chan_off, np.int64)
    if body == 2:
        arrs = [_i32(table.chan_J), _i32(table.chan_T), _i32(table.chan_par), _i32(table.chan_dim), off,
                _i32(table.state_a), _i32(table.state_b)]
        rc = lib.oracle_mscheme_2b(C.byref(b), C.c_int(len(arrs[0])), *[_p(a) for a in arrs], _p(vals),
                                   C.c_int64(n), _p(req), _p(out), _p(mask), _p(nt), C.byref(bad), C.c_int(n_threads))
    else:
        arrs = [_i32(table.chan_twoJ), _i32(table.chan_twoT), _i32(table.chan_par), _i32(table.chan_dim), off,
                _i32(table.state_a), _i32(table.state_b), _i32(table.state_c), _i32(table.state_J12),
                _i32(table.state_T12)]
        rc = lib.oracle_mscheme_3b(C.byref(b), C.c_int(int(table.e3max)), C.c_int(len(arrs[0])),
                                   *[_p(a) for a in arrs], _p(vals), C.c_int64(n), _p(req), _p(out), _p(mask),
                                   _p(nt), C.byref(bad), C.c_int(n_threads))
    assert rc == 0
    return out, mask, nt, int(bad.value)
