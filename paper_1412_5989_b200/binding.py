"""Thin ctypes binding of libmfdn_b200.so (include/mfdn_b200.h): same names, argument
marshalling only.  Every step of the path runs in the CUDA kernels of the library; there is no
CPU fallback -- if the library cannot be loaded this module raises.

PyTorch is used by callers for device memory and streams only; tensors are passed as
``data_ptr()`` and streams as ``torch.cuda.current_stream().cuda_stream``.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmfdn_b200.so")

MFDN_OK, MFDN_ERR_ARG, MFDN_ERR_STATE, MFDN_ERR_CUDA, MFDN_ERR_OOM, MFDN_ERR_TABLE = 0, -1, -2, -3, -4, -5
MFDN_PRESORTED, MFDN_FORCE_NAIVE, MFDN_FORCE_DENSE, MFDN_ONE_PASS_SORT, MFDN_REQ_U16 = 1, 2, 4, 8, 16
MFDN_FORCE_SORT = 32
MFDN_OPT_SLAB_FP32 = 1

# every symbol include/mfdn_b200.h declares
SYMBOLS = ["mfdn_orbitals_init", "mfdn_cg_build", "mfdn_cg_download", "mfdn_coupled_upload_2b",
           "mfdn_coupled_upload_3b", "mfdn_mscheme_2b", "mfdn_mscheme_3b", "mfdn_bad_request_count",
           "mfdn_info", "mfdn_group_keys", "mfdn_last_error", "mfdn_destroy", "mfdn_mscheme_host", "mfdn_profile",
           "mfdn_profile_read", "mfdn_fp64_peak", "mfdn_mscheme_accumulate_2b", "mfdn_mscheme_accumulate_3b",
           "mfdn_mscheme_block_len_3b", "mfdn_mscheme_blocks_3b", "mfdn_option", "mfdn_multi_client", "mfdn_mscheme_static"]
MFDN_STATIC_SCRATCH_BYTES = 32 << 20

_lib = None


class MfdnError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"mfdn status {code}: {msg}")
        self.code = code


def lib():
    """Load the shared library (no CUDA call is made by loading it)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1412_5989_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64, u32 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint32
        L.mfdn_orbitals_init.argtypes = [C.POINTER(vp), C.c_int, i32, vp, vp, vp, i32, vp, vp, vp]
        L.mfdn_cg_build.argtypes = [vp, vp]
        L.mfdn_cg_download.argtypes = [vp, C.c_int, vp, i64, C.POINTER(i64)]
        L.mfdn_coupled_upload_2b.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, vp, vp, C.c_int, vp]
        L.mfdn_coupled_upload_3b.argtypes = [vp, i32, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, C.c_int, vp]
        for f in (L.mfdn_mscheme_2b, L.mfdn_mscheme_3b):
            f.argtypes = [vp, i64, vp, vp, vp, vp, C.POINTER(C.c_size_t), u32, vp]
        for f in (L.mfdn_mscheme_accumulate_2b, L.mfdn_mscheme_accumulate_3b):
            f.argtypes = [vp, i64, vp, vp, vp, vp, i64, vp, vp, C.POINTER(C.c_size_t), u32, vp]
        L.mfdn_option.argtypes = [vp, C.c_int, i64]
        L.mfdn_multi_client.argtypes = [vp, C.c_int, i64, vp, vp, vp, i64, C.c_int, u32, C.POINTER(C.c_double)]
        L.mfdn_mscheme_block_len_3b.argtypes = [vp, vp, C.POINTER(i64)]
        L.mfdn_mscheme_blocks_3b.argtypes = [vp, i64, vp, vp, vp, vp, C.POINTER(C.c_size_t), vp]
        L.mfdn_mscheme_host.argtypes = [vp, C.c_int, i64, vp, vp, vp, vp, C.POINTER(C.c_size_t), u32, i64]
        L.mfdn_mscheme_static.argtypes = [vp, C.c_int, i64, vp, vp, vp, u32, vp]
        L.mfdn_profile.argtypes = [vp, C.c_int]
        L.mfdn_profile_read.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(i64)]
        L.mfdn_fp64_peak.argtypes = [vp, C.POINTER(C.c_double)]
        L.mfdn_bad_request_count.argtypes = [vp, vp]
        L.mfdn_bad_request_count.restype = i64
        L.mfdn_info.argtypes = [vp, C.c_int]
        L.mfdn_info.restype = i64
        L.mfdn_group_keys.argtypes = [vp, C.c_int, i64, vp, vp, vp]
        L.mfdn_last_error.argtypes = [vp]
        L.mfdn_last_error.restype = C.c_char_p
        L.mfdn_destroy.argtypes = [vp]
        L.mfdn_destroy.restype = None
        _lib = L
    return _lib


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _hp(a):
    return a.ctypes.data_as(C.c_void_p)


def _check(ctx, rc):
    if rc != MFDN_OK:
        msg = lib().mfdn_last_error(ctx).decode() if ctx else ""
        raise MfdnError(rc, msg)


def _stream(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    return C.c_void_p(int(stream))


def mfdn_orbitals_init(device, n, l, twoj, sps_orb, sps_twom, sps_twotz):
    arrs = [_i32(x) for x in (n, l, twoj, sps_orb, sps_twom, sps_twotz)]
    ctx = C.c_void_p()
    rc = lib().mfdn_orbitals_init(C.byref(ctx), int(device), len(arrs[0]), _hp(arrs[0]), _hp(arrs[1]), _hp(arrs[2]),
                                  len(arrs[3]), _hp(arrs[3]), _hp(arrs[4]), _hp(arrs[5]))
    if rc != MFDN_OK:
        raise MfdnError(rc, "mfdn_orbitals_init")
    return ctx


def mfdn_cg_build(ctx, stream=None):
    _check(ctx, lib().mfdn_cg_build(ctx, _stream(stream)))


def mfdn_cg_download(ctx, stage):
    n = C.c_int64(0)
    _check(ctx, lib().mfdn_cg_download(ctx, stage, None, 0, C.byref(n)))
    out = np.empty(n.value, np.float64)
    _check(ctx, lib().mfdn_cg_download(ctx, stage, _hp(out), n.value, C.byref(n)))
    return out


def _values_ptr(values):
    """numpy array (host) or torch CUDA tensor (device) -> (pointer, on_device, keepalive)."""
    if isinstance(values, np.ndarray):
        v = np.ascontiguousarray(values, np.float64)
        return _hp(v), 0, v
    assert values.is_cuda and values.is_contiguous() and values.dtype.itemsize == 8
    return C.c_void_p(values.data_ptr()), 1, values


def mfdn_coupled_upload_2b(ctx, chan_J, chan_T, chan_par, chan_dim, chan_off, state_a, state_b, values, stream=None):
    a = [_i32(x) for x in (chan_J, chan_T, chan_par, chan_dim)]
    off = np.ascontiguousarray(chan_off, np.int64)
    s = [_i32(x) for x in (state_a, state_b)]
    ptr, dev, keep = _values_ptr(values)
    _check(ctx, lib().mfdn_coupled_upload_2b(ctx, len(a[0]), *[_hp(x) for x in a], _hp(off), *[_hp(x) for x in s],
                                             ptr, dev, _stream(stream)))


def mfdn_coupled_upload_3b(ctx, e3max, chan_twoJ, chan_twoT, chan_par, chan_dim, chan_off, state_a, state_b, state_c,
                           state_J12, state_T12, values, stream=None):
    a = [_i32(x) for x in (chan_twoJ, chan_twoT, chan_par, chan_dim)]
    off = np.ascontiguousarray(chan_off, np.int64)
    s = [_i32(x) for x in (state_a, state_b, state_c, state_J12, state_T12)]
    ptr, dev, keep = _values_ptr(values)
    _check(ctx, lib().mfdn_coupled_upload_3b(ctx, int(e3max), len(a[0]), *[_hp(x) for x in a], _hp(off),
                                             *[_hp(x) for x in s], ptr, dev, _stream(stream)))


def _mscheme(fn, ctx, n, d_req, d_out, d_mask, d_work, work_bytes, flags, stream):
    wb = C.c_size_t(int(work_bytes))
    rc = fn(ctx, int(n), C.c_void_p(d_req), C.c_void_p(d_out), C.c_void_p(d_mask), C.c_void_p(d_work), C.byref(wb),
            int(flags), _stream(stream) if d_work else C.c_void_p(0))
    _check(ctx, rc)
    return wb.value


def mfdn_mscheme_2b(ctx, n, d_req, d_out, d_mask, d_work, work_bytes, flags=0, stream=None):
    """Raw call: device pointers as ints (0 = NULL).  Returns work_bytes (query when d_work == 0)."""
    return _mscheme(lib().mfdn_mscheme_2b, ctx, n, d_req, d_out, d_mask, d_work, work_bytes, flags, stream)


def mfdn_mscheme_3b(ctx, n, d_req, d_out, d_mask, d_work, work_bytes, flags=0, stream=None):
    return _mscheme(lib().mfdn_mscheme_3b, ctx, n, d_req, d_out, d_mask, d_work, work_bytes, flags, stream)


def mfdn_mscheme_accumulate(ctx, body, n, d_req, d_loc, d_phase, d_H, h_len, d_mask, d_work, work_bytes, flags=0, stream=None):
    """Raw call of mfdn_mscheme_accumulate_2b/3b: device pointers as ints (0 = NULL).  Returns work_bytes."""
    fn = lib().mfdn_mscheme_accumulate_3b if body == 3 else lib().mfdn_mscheme_accumulate_2b
    wb = C.c_size_t(int(work_bytes))
    _check(ctx, fn(ctx, int(n), C.c_void_p(d_req), C.c_void_p(d_loc), C.c_void_p(d_phase), C.c_void_p(d_H), int(h_len),
                   C.c_void_p(d_mask), C.c_void_p(d_work), C.byref(wb), int(flags), _stream(stream) if d_work else C.c_void_p(0)))
    return wb.value


def mfdn_mscheme_block_len_3b(ctx, orbitals):
    """Number of doubles of the block of the orbital tuples orbitals = (a, b, c, d, e, f)."""
    o = np.ascontiguousarray(orbitals, np.int32)
    assert o.shape == (6,)
    n = C.c_int64(0)
    _check(ctx, lib().mfdn_mscheme_block_len_3b(ctx, _hp(o), C.byref(n)))
    return n.value


def mfdn_mscheme_blocks_3b(ctx, h_orbitals, h_off, d_out, d_work, work_bytes, stream=None):
    """Raw call: h_orbitals int32 [n][6] and h_off int64 [n] are numpy arrays, d_out / d_work device pointers as ints."""
    o = np.ascontiguousarray(h_orbitals, np.int32).reshape(-1, 6)
    off = np.ascontiguousarray(h_off, np.int64)
    wb = C.c_size_t(int(work_bytes))
    _check(ctx, lib().mfdn_mscheme_blocks_3b(ctx, len(o), _hp(o), _hp(off), C.c_void_p(d_out), C.c_void_p(d_work), C.byref(wb),
                                            _stream(stream) if d_work else C.c_void_p(0)))
    return wb.value


def mfdn_multi_client(ctx, body, n, d_req, d_out, d_mask, chunk, n_threads, flags=0):
    """Measurement hook: n_threads native host threads with own streams push chunks through the context.  Returns seconds."""
    sec = C.c_double(0.0)
    _check(ctx, lib().mfdn_multi_client(ctx, int(body), int(n), C.c_void_p(d_req), C.c_void_p(d_out), C.c_void_p(d_mask),
                                        int(chunk), int(n_threads), int(flags), C.byref(sec)))
    return sec.value


def mfdn_mscheme_host(ctx, body, n, h_req, h_out, h_mask, d_work, work_bytes, flags=0, chunk=0):
    """Host-buffer wrapper: h_* are host addresses (ints, 0 = NULL).  Returns work_bytes."""
    wb = C.c_size_t(int(work_bytes))
    _check(ctx, lib().mfdn_mscheme_host(ctx, int(body), int(n), C.c_void_p(h_req), C.c_void_p(h_out), C.c_void_p(h_mask),
                                        C.c_void_p(d_work), C.byref(wb), int(flags), int(chunk)))
    return wb.value


def mfdn_mscheme_static(ctx, body, n, d_req, d_out, d_mask, flags=0, stream=None):
    """The allocation-free call: scratch from the library's own static device array (MFDN_STATIC_SCRATCH_BYTES)."""
    _check(ctx, lib().mfdn_mscheme_static(ctx, int(body), int(n), C.c_void_p(d_req), C.c_void_p(d_out), C.c_void_p(d_mask),
                                          int(flags), _stream(stream) if n else C.c_void_p(0)))


def mfdn_profile(ctx, enable):
    _check(ctx, lib().mfdn_profile(ctx, int(bool(enable))))


def mfdn_profile_read(ctx):
    a, b, u, n = C.c_double(0), C.c_double(0), C.c_double(0), C.c_int64(0)
    _check(ctx, lib().mfdn_profile_read(ctx, C.byref(a), C.byref(b), C.byref(u), C.byref(n)))
    return a.value, b.value, u.value, n.value


def mfdn_fp64_peak(ctx):
    t = C.c_double(0)
    _check(ctx, lib().mfdn_fp64_peak(ctx, C.byref(t)))
    return t.value


def mfdn_group_keys(ctx, body, n, d_req, d_key, stream=None):
    _check(ctx, lib().mfdn_group_keys(ctx, int(body), int(n), C.c_void_p(d_req), C.c_void_p(d_key), _stream(stream)))


def mfdn_bad_request_count(ctx, stream=None):
    return int(lib().mfdn_bad_request_count(ctx, _stream(stream)))


def mfdn_info(ctx, which):
    return int(lib().mfdn_info(ctx, int(which)))


def mfdn_destroy(ctx):
    lib().mfdn_destroy(ctx)


# ---------------------------------------------------------------------------------------------
class Context:
    """Lifecycle helper around the C calls above (marshalling only)."""

    def __init__(self, basis, device=0):
        import torch
        self.torch = torch
        self.device = device
        self.ctx = mfdn_orbitals_init(device, basis.n, basis.l, basis.twoj, basis.sps_orb, basis.sps_twom,
                                      basis.sps_twotz)
        with torch.cuda.device(device):
            mfdn_cg_build(self.ctx)
        self._work = None

    def option(self, option, value=1):
        """mfdn_option (e.g. MFDN_OPT_SLAB_FP32), before upload()."""
        _check(self.ctx, lib().mfdn_option(self.ctx, int(option), int(value)))
        return self

    def upload(self, table):
        with self.torch.cuda.device(self.device):
            if hasattr(table, "state_c"):
                mfdn_coupled_upload_3b(self.ctx, table.e3max, table.chan_twoJ, table.chan_twoT, table.chan_par,
                                       table.chan_dim, table.chan_off, table.state_a, table.state_b, table.state_c,
                                       table.state_J12, table.state_T12, table.values)
            else:
                mfdn_coupled_upload_2b(self.ctx, table.chan_J, table.chan_T, table.chan_par, table.chan_dim,
                                       table.chan_off, table.state_a, table.state_b, table.values)
        return self

    def work_bytes(self, body, n, flags=0):
        fn = mfdn_mscheme_3b if body == 3 else mfdn_mscheme_2b
        return fn(self.ctx, n, 0, 0, 0, 0, 0, flags)

    def mscheme(self, d_req, d_out=None, d_mask=None, flags=0, work=None, stream=None):
        """d_req: CUDA int32 tensor [n][4] or [n][6].  Returns (d_out f64[n], d_mask u8[n])."""
        torch = self.torch
        assert d_req.is_cuda and d_req.is_contiguous()
        if d_req.dtype in (torch.uint16, torch.int16):
            flags |= MFDN_REQ_U16            # compact requests: 16-bit SPS indices
        else:
            assert d_req.dtype == torch.int32 and not flags & MFDN_REQ_U16
        n, width = d_req.shape
        body = width // 2
        if d_out is None:
            d_out = torch.empty(n, dtype=torch.float64, device=d_req.device)
        if d_mask is None:
            d_mask = torch.empty(n, dtype=torch.uint8, device=d_req.device)
        need = self.work_bytes(body, n, flags)
        if work is None:
            if self._work is None or self._work.numel() < need:
                self._work = torch.empty(max(need, 256), dtype=torch.uint8, device=d_req.device)
            work = self._work
        assert work.numel() >= need
        fn = mfdn_mscheme_3b if body == 3 else mfdn_mscheme_2b
        fn(self.ctx, n, d_req.data_ptr(), d_out.data_ptr(), d_mask.data_ptr(), work.data_ptr(), work.numel(), flags,
           stream)
        return d_out, d_mask

    def mscheme_static(self, d_req, d_out, d_mask, flags=0, stream=None):
        """mfdn_mscheme_static: the caller passes inputs and outputs, the scratch is the library's static array."""
        torch = self.torch
        assert d_req.is_cuda and d_req.is_contiguous() and d_out.is_cuda and d_mask.is_cuda
        if d_req.dtype in (torch.uint16, torch.int16):
            flags |= MFDN_REQ_U16
        n, width = d_req.shape
        with torch.cuda.device(self.device):
            mfdn_mscheme_static(self.ctx, width // 2, n, d_req.data_ptr(), d_out.data_ptr(), d_mask.data_ptr(), flags, stream)
        return d_out, d_mask

    def accumulate(self, d_req, d_loc, d_phase, d_H, d_mask=None, flags=0, work=None, stream=None):
        """d_H[d_loc[i]] += d_phase[i] * v_i.  d_loc: CUDA int64 [n]; d_phase: CUDA float64 [n] or None;
        d_H: CUDA float64, updated in place.  Returns d_mask."""
        torch = self.torch
        assert d_req.is_cuda and d_req.is_contiguous()
        if d_req.dtype in (torch.uint16, torch.int16):
            flags |= MFDN_REQ_U16
        else:
            assert d_req.dtype == torch.int32 and not flags & MFDN_REQ_U16
        assert d_loc.is_cuda and d_loc.dtype == torch.int64 and d_loc.is_contiguous() and d_loc.numel() == d_req.shape[0]
        assert d_phase is None or (d_phase.is_cuda and d_phase.dtype == torch.float64 and d_phase.is_contiguous())
        assert d_H.is_cuda and d_H.dtype == torch.float64 and d_H.is_contiguous()
        n, width = d_req.shape
        body = width // 2
        if d_mask is None:
            d_mask = torch.empty(n, dtype=torch.uint8, device=d_req.device)
        need = mfdn_mscheme_accumulate(self.ctx, body, n, 0, 0, 0, 0, 0, 0, 0, 0, flags)
        if work is None:
            if self._work is None or self._work.numel() < need:
                self._work = torch.empty(max(need, 256), dtype=torch.uint8, device=d_req.device)
            work = self._work
        assert work.numel() >= need
        mfdn_mscheme_accumulate(self.ctx, body, n, d_req.data_ptr(), d_loc.data_ptr(), d_phase.data_ptr() if d_phase is not None else 0,
                                d_H.data_ptr(), d_H.numel(), d_mask.data_ptr(), work.data_ptr(), work.numel(), flags, stream)
        return d_mask

    def blocks(self, orbitals, stream=None):
        """Dense block mode: orbitals int [n][6].  Returns (d_out f64 on the GPU, offsets int64 [n + 1]) -- block k is
        d_out[offsets[k]:offsets[k + 1]] in the layout include/mfdn_b200.h states."""
        torch = self.torch
        o = np.ascontiguousarray(orbitals, np.int32).reshape(-1, 6)
        lens = np.array([mfdn_mscheme_block_len_3b(self.ctx, r) for r in o], np.int64)
        off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
        d_out = torch.empty(max(int(off[-1]), 1), dtype=torch.float64, device=f"cuda:{self.device}")
        need = mfdn_mscheme_blocks_3b(self.ctx, o, off[:-1], 0, 0, 0)
        work = torch.empty(max(need, 256), dtype=torch.uint8, device=f"cuda:{self.device}")
        mfdn_mscheme_blocks_3b(self.ctx, o, off[:-1], d_out.data_ptr(), work.data_ptr(), work.numel(), stream)
        self._block_work = work          # stays alive until the stream has consumed it
        return d_out[:int(off[-1])], off

    def mscheme_host(self, h_req, h_out=None, h_mask=None, flags=0, chunk=0):
        """h_req: CPU int32 tensor [n][4|6] (pinned recommended).  Returns (h_out, h_mask) CPU tensors."""
        torch = self.torch
        assert (not h_req.is_cuda) and h_req.is_contiguous()
        if h_req.dtype in (torch.uint16, torch.int16):
            flags |= MFDN_REQ_U16
        else:
            assert h_req.dtype == torch.int32 and not flags & MFDN_REQ_U16
        n, width = h_req.shape
        if h_out is None:
            h_out = torch.empty(n, dtype=torch.float64).pin_memory()
        if h_mask is None:
            h_mask = torch.empty(n, dtype=torch.uint8).pin_memory()
        need = mfdn_mscheme_host(self.ctx, width // 2, n, 0, 0, 0, 0, 0, flags, chunk)
        if getattr(self, "_hwork", None) is None or self._hwork.numel() < need:
            self._hwork = torch.empty(max(need, 256), dtype=torch.uint8, device=f"cuda:{self.device}")
        mfdn_mscheme_host(self.ctx, width // 2, n, h_req.data_ptr(), h_out.data_ptr(), h_mask.data_ptr(),
                          self._hwork.data_ptr(), self._hwork.numel(), flags, chunk)
        return h_out, h_mask

    def group_keys(self, d_req):
        torch = self.torch
        n, width = d_req.shape
        keys = torch.empty(n, dtype=torch.int32, device=d_req.device)
        mfdn_group_keys(self.ctx, width // 2, n, d_req.data_ptr(), keys.data_ptr())
        return keys

    def bad_request_count(self):
        return mfdn_bad_request_count(self.ctx)

    def close(self):
        if self.ctx:
            mfdn_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
