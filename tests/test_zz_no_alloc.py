"""mfdn_mscheme_static, the allocation-free call (include/mfdn_b200.h): its scratch is a static device array inside the
library instead of caller memory.  Checked against the existing path (mfdn_mscheme_2b/3b with caller scratch, itself
checked against the oracle in test_gpu_parity.py) on two calls in a row that share the array, and against the oracle
on a sample.  Collected last (file name), so a failure here hides no other test under `pytest -x`."""
import numpy as np
import pytest

from paper_1412_5989_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-12   # |delta| <= TOL * max|V|, the bar of test_gpu_parity.py; the mask is compared bit for bit


@pytest.fixture(scope="module")
def torch():
    import torch
    return torch


@pytest.fixture(scope="module")
def B():
    from paper_1412_5989_b200 import binding
    return binding


def _compare(cfg, got, gmask, want, wmask):
    vmax = float(np.max(np.abs(cfg.table.values)))
    assert np.array_equal(gmask, wmask), f"mask differs at {np.nonzero(gmask != wmask)[0][:10]}"
    err = float(np.max(np.abs(got - want)))
    assert err <= TOL * vmax, f"max|delta| {err:.3e} > {TOL * vmax:.3e}"
    assert np.all(got[gmask == 0] == 0.0) and not np.any(np.signbit(got[gmask == 0]))


def test_static_scratch_two_calls_in_a_row(torch, B):
    """Config 3 (3-body, E3max = 8) on the group-sort path, which is the one that uses scratch: two different request
    windows one after the other on one stream (the second call finds the first one's records, histogram and work
    items in the array), one-pass and two-pass sort.  No device memory is allocated between the calls."""
    cfg = W.make_config(3)
    ctx = B.Context(cfg.basis, 0).upload(cfg.table)
    n = (1 << 17) + 77                                     # several tiles and a ragged tail
    windows = [cfg.requests(n, start=0, permute_frac=0.01), cfg.requests(n - 4099, start=3 * n, permute_frac=0.01)]
    d_reqs = [torch.from_numpy(np.ascontiguousarray(r, np.int32)).cuda() for r in windows]
    for flags in (B.MFDN_ONE_PASS_SORT, B.MFDN_FORCE_SORT):
        need = ctx.work_bytes(3, n, flags)
        assert 256 < need <= B.MFDN_STATIC_SCRATCH_BYTES   # the path really uses scratch, and it fits the array
        # the existing path first (its outputs and scratch come from torch's allocator)
        ref = []
        for d_req in d_reqs:
            out, mask = ctx.mscheme(d_req, flags=flags)
            torch.cuda.synchronize()
            ref.append((out.cpu().numpy(), mask.cpu().numpy()))
        outs = [torch.full((len(r),), -7.0, dtype=torch.float64, device="cuda") for r in windows]
        masks = [torch.full((len(r),), 9, dtype=torch.uint8, device="cuda") for r in windows]
        B.mfdn_mscheme_static(ctx.ctx, 3, 0, 0, 0, 0, flags)            # set-up call: looks up the array's device address
        ctx.mscheme_static(d_reqs[0], outs[0], masks[0], flags)         # also loads the kernels of this path, if not yet
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        ctx.mscheme_static(d_reqs[1], outs[1], masks[1], flags)         # second call in a row on the same array
        ctx.mscheme_static(d_reqs[0], outs[0], masks[0], flags)         # and the first window again, on top of the second
        torch.cuda.synchronize()
        # the scratch of these calls would be >= 12 MB; 1 MiB of slack for anything the driver does on its own
        assert torch.cuda.mem_get_info()[0] >= free0 - (1 << 20), "device memory was allocated during mfdn_mscheme_static"
        for k in range(2):
            got, gmask = outs[k].cpu().numpy(), masks[k].cpu().numpy()
            _compare(cfg, got, gmask, *ref[k])
            assert np.array_equal(got, ref[k][0])                       # same kernels, same operation order: bit for bit
    # the default flags (thread per request at this size: no scratch needed) go through the same entry point
    out, mask = ctx.mscheme(d_reqs[0])
    ctx.mscheme_static(d_reqs[0], outs[0], masks[0], 0)
    torch.cuda.synchronize()
    _compare(cfg, outs[0].cpu().numpy(), masks[0].cpu().numpy(), out.cpu().numpy(), mask.cpu().numpy())
    # and a sample against the oracle
    from oracle import mscheme_c
    sel = np.random.default_rng(5).choice(len(windows[0]), 1 << 12, replace=False)
    want, wmask, _, _ = mscheme_c.mscheme(cfg.basis, cfg.table, windows[0][sel])
    _compare(cfg, outs[0].cpu().numpy()[sel], masks[0].cpu().numpy()[sel], want, wmask)


def test_static_scratch_limit_and_2body(torch, B):
    """A batch that needs more than the array holds is rejected with a clear error and nothing is launched; body = 2."""
    cfg3 = W.make_config(2)
    ctx3 = B.Context(cfg3.basis, 0).upload(cfg3.table)
    req = cfg3.requests()
    reps = -(-(1 << 20) // len(req))
    big = np.tile(req, (reps, 1))[: 1 << 20]               # 2^20 requests on the sort path: ~50 MB of scratch
    assert ctx3.work_bytes(3, len(big), B.MFDN_FORCE_SORT) > B.MFDN_STATIC_SCRATCH_BYTES
    d_req = torch.from_numpy(np.ascontiguousarray(big, np.int32)).cuda()
    out = torch.full((len(big),), -7.0, dtype=torch.float64, device="cuda")
    mask = torch.full((len(big),), 9, dtype=torch.uint8, device="cuda")
    with pytest.raises(B.MfdnError) as e:
        ctx3.mscheme_static(d_req, out, mask, B.MFDN_FORCE_SORT)
    assert e.value.code == B.MFDN_ERR_OOM and "static array holds" in str(e.value)
    torch.cuda.synchronize()
    assert float(out.min()) == -7.0 and int(mask.min()) == 9          # untouched
    with pytest.raises(B.MfdnError):
        B.mfdn_mscheme_static(ctx3.ctx, 4, 16, d_req.data_ptr(), out.data_ptr(), mask.data_ptr(), 0)   # body must be 2 or 3
    # 2-body, all pairs of config 0, forced onto the sort path (the 2-body default needs no scratch), twice in a row
    cfg2 = W.make_config(0)
    ctx2 = B.Context(cfg2.basis, 0).upload(cfg2.table)
    d2 = torch.from_numpy(np.ascontiguousarray(cfg2.requests(), np.int32)).cuda()
    for flags in (B.MFDN_FORCE_SORT, B.MFDN_ONE_PASS_SORT, 0):
        r_out, r_mask = ctx2.mscheme(d2, flags=flags)
        for _ in range(2):
            o = torch.full((len(d2),), -7.0, dtype=torch.float64, device="cuda")
            m = torch.full((len(d2),), 9, dtype=torch.uint8, device="cuda")
            ctx2.mscheme_static(d2, o, m, flags)
            torch.cuda.synchronize()
            _compare(cfg2, o.cpu().numpy(), m.cpu().numpy(), r_out.cpu().numpy(), r_mask.cpu().numpy())
