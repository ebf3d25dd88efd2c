"""GPU parity tests proper: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Bars (BASELINE.json north_star): max|delta| <= 1e-12 * max|V| in fp64;
selection mask bit-exact."""
import numpy as np
import pytest

from paper_1412_5989_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-12
# 0 = the library's own choice by batch size (thread-per-request for 2-body and small 3-body batches, group sort above)
MODES = {"auto": 0, "naive": 2, "one_pass_sort": 8, "two_pass_sort": 32}


@pytest.fixture(scope="module")
def torch():
    import torch
    return torch


@pytest.fixture(scope="module")
def B():
    from paper_1412_5989_b200 import binding
    return binding


@pytest.fixture(scope="module")
def oracle():
    from oracle import mscheme_c
    return mscheme_c


_cfg_cache = {}


def get_cfg(i):
    if i not in _cfg_cache:
        _cfg_cache[i] = W.make_config(i)
    return _cfg_cache[i]


_ctx_cache = {}


def get_ctx(B, i):
    if i not in _ctx_cache:
        cfg = get_cfg(i)
        _ctx_cache[i] = B.Context(cfg.basis, 0).upload(cfg.table)
    return _ctx_cache[i]


def run_gpu(torch, ctx, req, flags=0):
    d_req = torch.from_numpy(np.ascontiguousarray(req, np.int32)).cuda()
    out, mask = ctx.mscheme(d_req, flags=flags)
    torch.cuda.synchronize()
    return out.cpu().numpy(), mask.cpu().numpy()


def presort(torch, ctx, req):
    d_req = torch.from_numpy(np.ascontiguousarray(req, np.int32)).cuda()
    keys = ctx.group_keys(d_req).cpu().numpy().view(np.uint32)
    order = np.argsort(keys, kind="stable")
    return req[order], order


def check(cfg, got, gmask, want, wmask):
    vmax = float(np.max(np.abs(cfg.table.values)))
    assert np.array_equal(gmask, wmask), f"mask differs at {np.nonzero(gmask != wmask)[0][:10]}"
    err = float(np.max(np.abs(got - want))) if len(got) else 0.0
    assert err <= TOL * vmax, f"max|delta| {err:.3e} > {TOL * vmax:.3e}"
    assert np.all(got[gmask == 0] == 0.0)
    assert not np.any(np.signbit(got[gmask == 0]))


# --------------------------------------------------------------------------------- CG tables
@pytest.mark.parametrize("emax", [2, 8])
def test_cg_tables_match_exact(torch, B, emax):
    """A1: every entry of the device tables against exact-rational values (gate 1e-15)."""
    from oracle.cg_exact import cg_exact
    basis = W.ho_basis(emax)
    ctx = B.Context(basis, 0)
    nj = (int(basis.twoj.max()) + 1) // 2
    rng = np.random.default_rng(0)
    for stage in (1, 2):
        tab = B.mfdn_cg_download(ctx.ctx, stage)
        pos = 0
        worst = 0.0
        firsts = [2 * a + 1 for a in range(nj)] if stage == 1 else [2 * J for J in range(2 * nj)]
        for tj1 in firsts:
            for tj2 in [2 * b + 1 for b in range(nj)]:
                nJ = min(tj1, tj2) + 1
                cnt = (tj1 + 1) * (tj2 + 1) * nJ
                blk = tab[pos:pos + cnt].reshape(nJ, tj1 + 1, tj2 + 1)
                pos += cnt
                # all entries for small blocks, a random sample for big ones (exact arithmetic is slow)
                idx = np.ndindex(blk.shape) if cnt <= 400 else \
                    [np.unravel_index(k, blk.shape) for k in rng.choice(cnt, 150, replace=False)]
                for (iJ, i1, i2) in idx:
                    tm1, tm2, tJ = 2 * i1 - tj1, 2 * i2 - tj2, abs(tj1 - tj2) + 2 * iJ
                    worst = max(worst, abs(blk[iJ, i1, i2] - cg_exact(tj1, tm1, tj2, tm2, tJ, tm1 + tm2)))
        assert pos == len(tab)
        assert worst <= 1e-15, f"stage {stage}: max CG error {worst:.2e}"
    ctx.close()


# --------------------------------------------------------------------------------- whole small configs
@pytest.mark.parametrize("mode", list(MODES) + ["presorted", "sort_presorted", "dense", "dense_presorted"])
@pytest.mark.parametrize("idx", [0, 2])
def test_all_pairs_configs(torch, B, oracle, idx, mode):
    cfg = get_cfg(idx)
    ctx = get_ctx(B, idx)
    req = cfg.requests()
    if mode.startswith("dense") and cfg.body == 2:           # the dense-block path (H5') is 3-body only
        with pytest.raises(B.MfdnError) as e:
            run_gpu(torch, ctx, req[:100], B.MFDN_FORCE_DENSE)
        assert e.value.code == B.MFDN_ERR_ARG
        return
    want, wmask, _, _ = oracle.mscheme(cfg.basis, cfg.table, req)
    if mode.endswith("presorted"):
        flags = B.MFDN_PRESORTED | (B.MFDN_FORCE_DENSE if mode.startswith("dense") else 0) | (B.MFDN_FORCE_SORT if mode.startswith("sort") else 0)
        sreq, order = presort(torch, ctx, req)
        got, gmask = run_gpu(torch, ctx, sreq, flags)
        check(cfg, got, gmask, want[order], wmask[order])
    elif mode == "dense":
        got, gmask = run_gpu(torch, ctx, req, B.MFDN_FORCE_DENSE)
        check(cfg, got, gmask, want, wmask)
    else:
        got, gmask = run_gpu(torch, ctx, req, MODES[mode])
        check(cfg, got, gmask, want, wmask)
    assert ctx.bad_request_count() == 0


# --------------------------------------------------------------------------------- sampled large configs
@pytest.mark.parametrize("idx,n", [(1, 1 << 20), (3, (1 << 19) + 77), (4, 1 << 18)])
def test_sampled_configs_prefix(torch, B, oracle, idx, n):
    """First n requests of the stream (with 1% randomly permuted particle lists: sign path), all modes."""
    cfg = get_cfg(idx)
    ctx = get_ctx(B, idx)
    req = cfg.requests(n, permute_frac=0.01)
    want, wmask, nt, _ = oracle.mscheme(cfg.basis, cfg.table, req)
    assert 0.85 < wmask.mean() < 1.0
    for mode, flags in MODES.items():
        got, gmask = run_gpu(torch, ctx, req, flags)
        check(cfg, got, gmask, want, wmask)
    if cfg.body == 3:      # dense-block path wherever a group's blocks fit (sparse requests: correct, not fast)
        got, gmask = run_gpu(torch, ctx, req, B.MFDN_FORCE_DENSE)
        check(cfg, got, gmask, want, wmask)
    sreq, order = presort(torch, ctx, req)
    for flags in (B.MFDN_PRESORTED, B.MFDN_PRESORTED | B.MFDN_FORCE_SORT):     # the library's choice / the group-sort path
        got, gmask = run_gpu(torch, ctx, sreq, flags)
        check(cfg, got, gmask, want[order], wmask[order])


# --------------------------------------------------------------------------------- edge cases
@pytest.mark.parametrize("idx", [0, 2])
def test_edge_sizes_and_bad_indices(torch, B, oracle, idx):
    cfg = get_cfg(idx)
    ctx = get_ctx(B, idx)
    allreq = cfg.requests()
    rng = np.random.default_rng(9)
    # ragged sizes around the warp, the block and the sort tile (8192 requests: last tile of 1, full, full + 1)
    for n in (0, 1, 31, 32, 33, 127, 128, 129, 4097, 8191, 8192, 8193, 16385):
        req = allreq[rng.choice(len(allreq), n, replace=False)] if n else allreq[:0]
        want, wmask, _, _ = oracle.mscheme(cfg.basis, cfg.table, req)
        for flags in (0, 2, 8, 32):
            got, gmask = run_gpu(torch, ctx, req, flags)
            check(cfg, got, gmask, want, wmask)
    # random (mostly forbidden) requests, duplicates inside bra/ket, and out-of-range SPS indices
    width = allreq.shape[1]
    req = rng.integers(0, cfg.basis.n_sps, size=(20000, width)).astype(np.int32)
    req[:200, 0] = cfg.basis.n_sps
    req[200:300, width - 1] = -1
    req[300:400, 1] = 2 ** 31 - 1
    before = ctx.bad_request_count()
    want, wmask, _, nbad = oracle.mscheme(cfg.basis, cfg.table, req)
    got, gmask = run_gpu(torch, ctx, req, 2)
    check(cfg, got, gmask, want, wmask)
    assert ctx.bad_request_count() - before == nbad == 400
    for flags in (0, 8, 32):
        got, gmask = run_gpu(torch, ctx, req, flags)
        check(cfg, got, gmask, want, wmask)
    # one hot bucket: the same request many times over (every copy lands in one run of the partition), plus a few others
    req = np.concatenate([np.repeat(allreq[len(allreq) // 2][None, :], 30000, axis=0), allreq[rng.choice(len(allreq), 3000, replace=False)]])
    req = req[rng.permutation(len(req))]
    want, wmask, _, _ = oracle.mscheme(cfg.basis, cfg.table, req)
    for flags in (0, 8, 32):
        got, gmask = run_gpu(torch, ctx, req, flags)
        check(cfg, got, gmask, want, wmask)
    # mask pointer may be NULL
    d_req = torch.from_numpy(allreq[:1000].copy()).cuda()
    out = torch.empty(1000, dtype=torch.float64, device="cuda")
    body = width // 2
    fn = B.mfdn_mscheme_3b if body == 3 else B.mfdn_mscheme_2b
    need = fn(ctx.ctx, 1000, 0, 0, 0, 0, 0, 0)
    work = torch.empty(need, dtype=torch.uint8, device="cuda")
    fn(ctx.ctx, 1000, d_req.data_ptr(), out.data_ptr(), 0, work.data_ptr(), need, 0)
    torch.cuda.synchronize()
    want, *_ = oracle.mscheme(cfg.basis, cfg.table, allreq[:1000])
    assert np.max(np.abs(out.cpu().numpy() - want)) <= TOL * np.max(np.abs(cfg.table.values))


def test_order_chunk_and_stream_invariance(torch, B):
    """Element values are independent of one another and of request order: any
    permutation or chunking gives bitwise identical per-request results."""
    cfg = get_cfg(2)
    ctx = get_ctx(B, 2)
    req = cfg.requests()
    rng = np.random.default_rng(4)
    req = req[rng.choice(len(req), 200000, replace=False)]
    base, bmask = run_gpu(torch, ctx, req, B.MFDN_FORCE_SORT)
    perm = rng.permutation(len(req))
    got, gmask = run_gpu(torch, ctx, req[perm], B.MFDN_FORCE_SORT)
    assert np.array_equal(got, base[perm]) and np.array_equal(gmask, bmask[perm])
    # every path does the same operations in the same order: the library's choice of path by batch size is invisible
    for flags in (0, B.MFDN_FORCE_NAIVE, B.MFDN_ONE_PASS_SORT):
        other, omask = run_gpu(torch, ctx, req, flags)
        assert np.array_equal(other, base) and np.array_equal(omask, bmask), flags
    # chunks of ~20 000 (the paper's buffer size) on two streams, by the library's choice and by the sort path
    d_req = torch.from_numpy(req).cuda()
    for flags in (0, B.MFDN_FORCE_SORT):
        out = torch.empty(len(req), dtype=torch.float64, device="cuda")
        mask = torch.empty(len(req), dtype=torch.uint8, device="cuda")
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        need = ctx.work_bytes(3, 20000, flags)
        works = [torch.empty(need, dtype=torch.uint8, device="cuda") for _ in streams]
        torch.cuda.synchronize()
        for k, lo in enumerate(range(0, len(req), 20000)):
            hi = min(lo + 20000, len(req))
            s = streams[k % 2]
            with torch.cuda.stream(s):
                ctx.mscheme(d_req[lo:hi], out[lo:hi], mask[lo:hi], flags, works[k % 2], s.cuda_stream)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), base) and np.array_equal(mask.cpu().numpy(), bmask)


def test_call_order_and_table_validation(torch, B):
    cfg = get_cfg(0)
    b = cfg.basis
    ctx = B.mfdn_orbitals_init(0, b.n, b.l, b.twoj, b.sps_orb, b.sps_twom, b.sps_twotz)
    t = cfg.table
    args = (t.chan_J, t.chan_T, t.chan_par, t.chan_dim, t.chan_off, t.state_a, t.state_b, t.values)
    with pytest.raises(B.MfdnError) as e:
        B.mfdn_coupled_upload_2b(ctx, *args)
    assert e.value.code == B.MFDN_ERR_STATE
    B.mfdn_cg_build(ctx)
    with pytest.raises(B.MfdnError) as e:
        B.mfdn_mscheme_2b(ctx, 10, 0, 0, 0, 0, 0)
    assert e.value.code == B.MFDN_ERR_STATE
    bad_T = t.chan_T.copy()
    bad_T[0] = 1 - bad_T[0]                      # breaks "a == b only with J+T odd" or duplicates a channel
    with pytest.raises(B.MfdnError) as e:
        B.mfdn_coupled_upload_2b(ctx, t.chan_J, bad_T, *args[2:])
    assert e.value.code == B.MFDN_ERR_TABLE
    bad_a = t.state_a.copy()
    bad_a[3] = b.n_orb
    with pytest.raises(B.MfdnError) as e:
        B.mfdn_coupled_upload_2b(ctx, *args[:5], bad_a, *args[6:])
    assert e.value.code == B.MFDN_ERR_TABLE
    B.mfdn_coupled_upload_2b(ctx, *args)        # a failed upload leaves the context usable
    B.mfdn_destroy(ctx)


# --------------------------------------------------------------------------------- full size, bench launch config
def test_full_size_config3_sampled(torch, B, oracle):
    """2^26 requests of config 3 in the configuration bench.py times (one call, internal sort and PRESORTED),
    checked on 2^16 sampled outputs the oracle computes one by one + properties that hold at any size."""
    cfg = get_cfg(3)
    ctx = get_ctx(B, 3)
    n = 1 << 26
    req = cfg.requests(n)
    d_req = torch.from_numpy(req).cuda()
    out, mask = ctx.mscheme(d_req, flags=0)
    torch.cuda.synchronize()
    sample = np.random.default_rng(77).choice(n, 1 << 16, replace=False)
    sample.sort()
    want, wmask, _, _ = oracle.mscheme(cfg.basis, cfg.table, req[sample])
    ds = torch.from_numpy(sample).cuda()
    check(cfg, out[ds].cpu().numpy(), mask[ds].cpu().numpy(), want, wmask)
    frac = float(mask.float().mean())
    assert 0.975 < frac < 0.985                       # ~98.1% of sampled pairs have mask 1
    assert bool((out[mask == 0] == 0).all())
    # hermiticity at full size: swap bra and ket
    d_swapped = torch.cat([d_req[:, 3:], d_req[:, :3]], dim=1).contiguous()
    out2, mask2 = ctx.mscheme(d_swapped, flags=0)
    torch.cuda.synchronize()
    assert bool((mask2 == mask).all())
    assert float((out2 - out).abs().max()) <= TOL * float(np.max(np.abs(cfg.table.values)))
    del d_swapped, out2, mask2
    # PRESORTED on the key-ordered multiset gives bitwise the same values
    keys = ctx.group_keys(d_req)
    order = torch.argsort(keys.view(torch.int32).to(torch.int64) & 0xFFFFFFFF)
    d_sorted = d_req[order].contiguous()
    out3, mask3 = ctx.mscheme(d_sorted, flags=B.MFDN_PRESORTED)
    torch.cuda.synchronize()
    assert bool((out3 == out[order]).all()) and bool((mask3 == mask[order]).all())


def test_3b_upload_rules(torch, B):
    """3-body upload validation: a tuple with more than 4096 m-states does not fit the 12-bit state index of the
    packed record and is refused; a state above E3max is refused; the context stays usable."""
    b = W.ho_basis(8)
    ctx = B.mfdn_orbitals_init(0, b.n, b.l, b.twoj, b.sps_orb, b.sps_twom, b.sps_twotz)
    B.mfdn_cg_build(ctx)
    big = int(np.argmax(b.twoj))                      # 0k17/2: (2j+1)^3 = 5832 m-states for the triple (big, big, big)
    assert (int(b.twoj[big]) + 1) ** 3 > 4096
    one = np.array([1], np.int32)
    args = dict(chan_twoJ=[17], chan_twoT=[1], chan_par=[0], chan_dim=one, chan_off=np.array([0], np.int64),
                state_a=[big], state_b=[big], state_c=[big], state_J12=[0], state_T12=[1], values=np.ones(1))
    with pytest.raises(B.MfdnError) as e:
        B.mfdn_coupled_upload_3b(ctx, 24, **args)
    assert e.value.code == B.MFDN_ERR_TABLE
    with pytest.raises(B.MfdnError) as e:
        B.mfdn_coupled_upload_3b(ctx, 8, **args)      # e_a + e_b + e_c = 24 > E3max = 8
    assert e.value.code == B.MFDN_ERR_TABLE
    small = W.coupled_3b(b, 2, 5)                     # a failed upload leaves the context usable
    B.mfdn_coupled_upload_3b(ctx, 2, small.chan_twoJ, small.chan_twoT, small.chan_par, small.chan_dim, small.chan_off,
                             small.state_a, small.state_b, small.state_c, small.state_J12, small.state_T12, small.values)
    B.mfdn_destroy(ctx)


# --------------------------------------------------------------------------------- synthetic bases: rarely taken kernel paths
def _custom_basis(orbs):
    """Basis of the listed (n, l, 2j) orbitals, SPS laid out like workloads.ho_basis."""
    n = np.array([o[0] for o in orbs], np.int32)
    l = np.array([o[1] for o in orbs], np.int32)
    tj = np.array([o[2] for o in orbs], np.int32)
    so, sm, st = [], [], []
    for o, (_, _, twoj) in enumerate(orbs):
        for twotz in (1, -1):
            for twom in range(-twoj, twoj + 1, 2):
                so.append(o)
                sm.append(twom)
                st.append(twotz)
    return W.Basis(n, l, tj, np.array(so, np.int32), np.array(sm, np.int32), np.array(st, np.int32))


def _check_all_modes(torch, B, oracle, basis, table, req):
    cfg = type("Cfg", (), {"table": table})
    ctx = B.Context(basis, 0).upload(table)
    want, wmask, _, _ = oracle.mscheme(basis, table, req)
    assert wmask.mean() > 0.5
    for flags in (0, B.MFDN_FORCE_SORT, B.MFDN_ONE_PASS_SORT, B.MFDN_FORCE_NAIVE, B.MFDN_FORCE_DENSE):
        got, gmask = run_gpu(torch, ctx, req, flags)
        check(cfg, got, gmask, want, wmask)
    sreq, order = presort(torch, ctx, req)
    for flags in (B.MFDN_PRESORTED, B.MFDN_PRESORTED | B.MFDN_FORCE_SORT):
        got, gmask = run_gpu(torch, ctx, sreq, flags)
        check(cfg, got, gmask, want[order], wmask[order])
    ctx.close()


def test_wide_j_blocks_generic_branch(torch, B, oracle):
    """Tuples (0g9/2, 0g9/2, 0g9/2) and (0g9/2, 0g9/2, 0h11/2) have TEN J12 rows at J = 9/2 resp. 11/2: the J blocks
    wider than 8 take the generic branch of k_transform3 (dispatch code 25), and their isospin-combined slabs
    (about 600 cells per bin) are staged four bins at a time (five rounds per work item).  No config of
    BASELINE.json reaches either path (at most 8 rows per (tuple, J))."""
    basis = _custom_basis([(0, 4, 9), (0, 5, 11)])
    table = W.coupled_3b(basis, 13, 11)
    ms = W.mstates(basis, 3, 13)
    req = W.sampled_pairs(ms, 60000, 2011, permute_frac=0.02)
    _check_all_modes(torch, B, oracle, basis, table, req)


def test_oversized_group_plane(torch, B, oracle):
    """The triple of three 0j15/2 orbitals has 4096 m-states (accepted) and a group plane of more than 2000 cells:
    too large for the staged path even four bins at a time.  Such groups are evaluated in chunks by the
    direct kernel (k_transform3_small) -- an error-free, capacity-free route, never a hang."""
    basis = _custom_basis([(0, 7, 15)])
    table = W.coupled_3b(basis, 21, 12)
    ms = W.mstates(basis, 3, 21)
    req = W.sampled_pairs(ms, 20000, 2012, permute_frac=0.02)
    _check_all_modes(torch, B, oracle, basis, table, req)


# --------------------------------------------------------------------------------- full size, bench launch configs of configs 1 and 4
def test_full_size_config1_sampled(torch, B, oracle):
    """BASELINE.json config 1 at its full size: 2^26 two-body requests, unsorted and MFDN_PRESORTED, checked on 2^16
    sampled outputs the oracle computes one by one."""
    cfg = get_cfg(1)
    ctx = get_ctx(B, 1)
    n = 1 << 26
    req = cfg.requests(n)
    d_req = torch.from_numpy(req).cuda()
    out, mask = ctx.mscheme(d_req, flags=0)                      # the library's choice: thread-per-request for 2-body
    torch.cuda.synchronize()
    sample = np.sort(np.random.default_rng(78).choice(n, 1 << 16, replace=False))
    want, wmask, _, _ = oracle.mscheme(cfg.basis, cfg.table, req[sample])
    ds = torch.from_numpy(sample).cuda()
    check(cfg, out[ds].cpu().numpy(), mask[ds].cpu().numpy(), want, wmask)
    out_s, mask_s = ctx.mscheme(d_req, flags=B.MFDN_FORCE_SORT)   # group sort, two-pass partition
    torch.cuda.synchronize()
    assert bool((out_s == out).all()) and bool((mask_s == mask).all())
    del out_s, mask_s
    assert 0.93 < float(mask.float().mean()) < 0.955       # ~94.3% of sampled pairs have mask 1
    assert bool((out[mask == 0] == 0).all())
    keys = ctx.group_keys(d_req)
    order = torch.argsort(keys.view(torch.int32).to(torch.int64) & 0xFFFFFFFF)
    del keys
    d_sorted = d_req[order].contiguous()
    del d_req
    for flags in (B.MFDN_PRESORTED, B.MFDN_PRESORTED | B.MFDN_FORCE_SORT):   # thread per request / group-sort kernels
        out3, mask3 = ctx.mscheme(d_sorted, flags=flags)
        torch.cuda.synchronize()
        assert bool((out3 == out[order]).all()) and bool((mask3 == mask[order]).all())


def test_full_size_config4_batches(torch, B, oracle):
    """BASELINE.json config 4 in the shape bench/report time it: 2^28 requests as 16 batches of 2^24, issued round-robin
    on two streams with their own scratch; every batch checked on 2^16 sampled outputs against the oracle."""
    cfg = get_cfg(4)
    ctx = get_ctx(B, 4)
    nb, n = 16, 1 << 24
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    need = ctx.work_bytes(3, n)
    bufs = [dict(req=torch.empty((n, 6), dtype=torch.int32, device="cuda"), out=torch.empty(n, dtype=torch.float64, device="cuda"),
                 mask=torch.empty(n, dtype=torch.uint8, device="cuda"), work=torch.empty(need, dtype=torch.uint8, device="cuda"))
            for _ in streams]
    pending = [None, None]
    rng = np.random.default_rng(79)
    mask_frac = []

    def verify(slot):
        b, req, sample = pending[slot]
        streams[slot].synchronize()
        ds = torch.from_numpy(sample).cuda()
        want, wmask, _, _ = oracle.mscheme(cfg.basis, cfg.table, req[sample])
        check(cfg, bufs[slot]["out"][ds].cpu().numpy(), bufs[slot]["mask"][ds].cpu().numpy(), want, wmask)
        mask_frac.append(float(bufs[slot]["mask"].float().mean()))
        pending[slot] = None

    for b in range(nb):
        slot = b % 2
        if pending[slot] is not None:
            verify(slot)
        req = cfg.requests(n, start=b * n)
        s = streams[slot]
        with torch.cuda.stream(s):
            bufs[slot]["req"].copy_(torch.from_numpy(req), non_blocking=False)
            ctx.mscheme(bufs[slot]["req"], bufs[slot]["out"], bufs[slot]["mask"], 0, bufs[slot]["work"], s.cuda_stream)
        pending[slot] = (b, req, np.sort(rng.choice(n, 1 << 16, replace=False)))
    for slot in range(2):
        if pending[slot] is not None:
            verify(slot)
    assert len(mask_frac) == nb and all(0.98 < f <= 1.0 for f in mask_frac)   # ~99.4%


def test_multi_client_threads(torch, B):
    """Several host threads share one context, each with its own stream and scratch, shipping ~20 000-request chunks
    (PAPER.md:93 buffer size, :103 'each OpenMP thread uses a separate stream'); profiling on, so the event
    bookkeeping is exercised too.  Results are bitwise those of one big call."""
    import threading
    cfg = get_cfg(2)
    ctx = get_ctx(B, 2)
    req = cfg.requests()
    rng = np.random.default_rng(14)
    req = req[rng.choice(len(req), 400000, replace=False)]
    base, bmask = run_gpu(torch, ctx, req, B.MFDN_FORCE_SORT)
    d_req = torch.from_numpy(req).cuda()
    out = torch.empty(len(req), dtype=torch.float64, device="cuda")
    mask = torch.empty(len(req), dtype=torch.uint8, device="cuda")
    chunk, nthreads = 20000, 4
    call_flags = [0, B.MFDN_FORCE_SORT]      # thread t uses call_flags[t % 2]: the library's choice and the sort path side by side
    chunks = [(lo, min(lo + chunk, len(req))) for lo in range(0, len(req), chunk)]
    errors = []
    torch.cuda.synchronize()
    B.mfdn_profile(ctx.ctx, 1)

    def client(t):
        try:
            torch.cuda.set_device(0)
            s = torch.cuda.Stream()
            work = torch.empty(ctx.work_bytes(3, chunk, call_flags[t % 2]), dtype=torch.uint8, device="cuda")
            for k in range(t, len(chunks), nthreads):
                lo, hi = chunks[k]
                ctx.mscheme(d_req[lo:hi], out[lo:hi], mask[lo:hi], call_flags[t % 2], work, s.cuda_stream)
            s.synchronize()
        except Exception as e:      # noqa: BLE001 - reported by the main thread
            errors.append(e)

    threads = [threading.Thread(target=client, args=(t,)) for t in range(nthreads)]
    for th in threads:
        th.start()
    for th in threads:
        th.join()
    torch.cuda.synchronize()
    B.mfdn_profile(ctx.ctx, 0)
    _, _, _, calls = B.mfdn_profile_read(ctx.ctx)
    assert not errors, errors
    assert calls == len(chunks)
    assert np.array_equal(out.cpu().numpy(), base) and np.array_equal(mask.cpu().numpy(), bmask)
    # the same with native host threads (mfdn_multi_client, the measurement hook of report.py --chunks)
    for flags in (0, B.MFDN_FORCE_SORT):
        out.zero_()
        mask.zero_()
        sec = B.mfdn_multi_client(ctx.ctx, 3, len(req), d_req.data_ptr(), out.data_ptr(), mask.data_ptr(), 20000, 6, flags)
        assert sec > 0.0
        assert np.array_equal(out.cpu().numpy(), base) and np.array_equal(mask.cpu().numpy(), bmask)


# --------------------------------------------------------------------------------- NEXT-1: fused accumulate epilogue
@pytest.mark.gpu
@pytest.mark.parametrize("idx", [0, 2])
def test_accumulate_epilogue(torch, B, oracle, idx):
    """H[loc[i]] += phase[i] * v[i] against oracle/accumulate_ref.py applied to the ORACLE's values, on every
    path: default (fused into the last gather pass), one-pass sort, pre-sorted, naive.  Tolerance: each value is within
    1e-12 max|V| of the oracle's and an element sums at most m of them in an order that is not fixed, so
    |dH| <= 1e-12 * max|V| * m (m = largest number of requests on one element)."""
    from oracle.accumulate_ref import accumulate
    cfg = get_cfg(idx)
    ctx = get_ctx(B, idx)
    rng = np.random.default_rng(21)
    allreq = cfg.requests()
    for n, h_len in ((0, 5), (1, 1), (33, 7), (8193, 1500), (min(len(allreq), 60000), 9000)):
        req = allreq[rng.choice(len(allreq), n, replace=False)] if n else allreq[:0]
        loc, phase = W.many_body_targets(n, h_len, seed=n)
        if n > 100:
            loc[::13] = -1                      # skipped entries
            loc[5::17] = h_len
        want, wmask, _, _ = oracle.mscheme(cfg.basis, cfg.table, req)
        m = max(1, int(np.bincount(loc[(loc >= 0) & (loc < h_len)], minlength=1).max())) if n else 1
        tol = TOL * float(np.max(np.abs(cfg.table.values))) * m
        d_req = torch.from_numpy(np.ascontiguousarray(req, np.int32)).cuda()
        d_loc, d_phase = torch.from_numpy(loc).cuda(), torch.from_numpy(phase).cuda()
        for flags, ph in ((0, True), (B.MFDN_FORCE_SORT, True), (B.MFDN_FORCE_SORT, False), (B.MFDN_ONE_PASS_SORT, True), (B.MFDN_FORCE_NAIVE, True)):
            H0 = rng.standard_normal(h_len)     # the target is updated, not overwritten
            d_H = torch.from_numpy(H0.copy()).cuda()
            mask = ctx.accumulate(d_req, d_loc, d_phase if ph else None, d_H, flags=flags)
            torch.cuda.synchronize()
            ref = H0 + accumulate(want, loc, phase if ph else None, h_len)
            assert np.array_equal(mask.cpu().numpy(), wmask)
            assert float(np.max(np.abs(d_H.cpu().numpy() - ref))) <= tol + 1e-15 * np.max(np.abs(H0))
        if n > 100:                             # pre-sorted input: the targets travel with their requests
            sreq, order = presort(torch, ctx, req)
            d_H = torch.zeros(h_len, dtype=torch.float64, device="cuda")
            ctx.accumulate(torch.from_numpy(sreq).cuda(), torch.from_numpy(loc[order].copy()).cuda(),
                           torch.from_numpy(phase[order].copy()).cuda(), d_H, flags=B.MFDN_PRESORTED)
            torch.cuda.synchronize()
            assert float(np.max(np.abs(d_H.cpu().numpy() - accumulate(want, loc, phase, h_len)))) <= tol


# --------------------------------------------------------------------------------- NEXT-2: dense block mode
def _expected_block(cfg, oracle, orbs):
    """The block of include/mfdn_b200.h's mfdn_mscheme_blocks_3b, built from the header's words alone: enumerate the entries
    in the stated order, ask the ORACLE for those that are ordered Slater determinants, +0.0 elsewhere."""
    b = cfg.basis
    tj = np.asarray(b.twoj)
    sps = {(int(o), int(m), int(t)): k for k, (o, m, t) in enumerate(zip(b.sps_orb, b.sps_twom, b.sps_twotz))}
    listed = set(zip(cfg.table.state_a.tolist(), cfg.table.state_b.tolist(), cfg.table.state_c.tolist()))
    bra, ket = tuple(int(x) for x in orbs[:3]), tuple(int(x) for x in orbs[3:])
    lpar = lambda t: sum(int(b.l[o]) for o in t) & 1
    if bra not in listed or ket not in listed or lpar(bra) != lpar(ket):
        return np.zeros(0)
    sj = lambda t: int(sum(tj[o] for o in t))
    # common J (triangle ranges of both tuples); the library says "no common J" -> empty
    def jrange(t):
        ja, jb, jc = (int(tj[o]) for o in t)
        lo = min(abs(2 * J12 - jc) for J12 in range(abs(ja - jb) // 2, (ja + jb) // 2 + 1))
        return lo, ja + jb + jc
    (lb, hb), (lk, hk) = jrange(bra), jrange(ket)
    if max(lb, lk) > min(hb, hk):
        return np.zeros(0)
    mm = min(sj(bra), sj(ket))
    def mstates(t, twoM):     # (ia, ib, ic) of the given M in ascending (ia, ib) order
        ja, jb, jc = (int(tj[o]) for o in t)
        return [(ia, ib, ic) for ia in range(ja + 1) for ib in range(jb + 1) for ic in range(jc + 1)
                if 2 * (ia + ib + ic) - (ja + jb + jc) == twoM]
    pats = [(pb, pk) for pb in range(8) for pk in range(8) if bin(pb).count("1") == bin(pk).count("1")]
    def side(t, st, pat):     # SPS indices of an ordered Slater determinant, or None
        idx = []
        for o, i, bit in zip(t, st, ((pat >> 2) & 1, (pat >> 1) & 1, pat & 1)):
            k = sps.get((o, 2 * i - int(tj[o]), 1 if bit else -1))
            if k is None:
                return None
            idx.append(k)
        for p in range(2):
            if t[p] == t[p + 1] and not idx[p] < idx[p + 1]:
                return None
        return idx
    reqs, where, total = [], [], 0
    for mi in range(mm + 1):
        twoM = 2 * mi - mm
        rows, cols = mstates(bra, twoM), mstates(ket, twoM)
        for pb, pk in pats:
            for r, sb in enumerate(rows):
                ib = side(bra, sb, pb)
                for cidx, sk in enumerate(cols):
                    ik = side(ket, sk, pk)
                    if ib is not None and ik is not None:
                        reqs.append(ib + ik)
                        where.append(total + r * len(cols) + cidx)
            total += len(rows) * len(cols)
    out = np.zeros(total)
    if reqs:
        want, _, _, _ = oracle.mscheme(cfg.basis, cfg.table, np.asarray(reqs, np.int32))
        out[np.asarray(where)] = want
    return out


@pytest.mark.gpu
def test_dense_block_mode(torch, B, oracle):
    """mfdn_mscheme_blocks_3b against the oracle, entry by entry, for tuple pairs with distinct and repeated orbitals (a == b,
    b == c, a == b == c), equal tuples, the other parity (empty block), an unlisted tuple (empty block)."""
    cfg = get_cfg(2)
    ctx = get_ctx(B, 2)
    tup = sorted(set(zip(cfg.table.state_a.tolist(), cfg.table.state_b.tolist(), cfg.table.state_c.tolist())))
    kinds = {}
    for t in tup:
        kinds.setdefault((t[0] == t[1], t[1] == t[2]), []).append(t)
    rng = np.random.default_rng(8)
    picks = [kinds[k][int(rng.integers(len(kinds[k])))] for k in sorted(kinds)] + [tup[int(i)] for i in rng.choice(len(tup), 6, replace=False)]
    groups = [a + b for a in picks[:6] for b in picks[2:8]] + [picks[0] + picks[0]]
    n_orb = cfg.basis.n_orb
    unlisted = next((a, b, c) for a in range(n_orb) for b in range(a, n_orb) for c in range(b, n_orb) if (a, b, c) not in set(tup))
    groups.append(unlisted + tup[0])
    d_out, off = ctx.blocks(np.asarray(groups, np.int32))
    torch.cuda.synchronize()
    got = d_out.cpu().numpy()
    vmax = float(np.max(np.abs(cfg.table.values)))
    n_nonempty = 0
    for k, g in enumerate(groups):
        want = _expected_block(cfg, oracle, g)
        blk = got[off[k]:off[k + 1]]
        assert len(blk) == len(want), (g, len(blk), len(want))
        if len(want):
            n_nonempty += 1
            assert float(np.max(np.abs(blk - want))) <= TOL * vmax, g
            assert np.all(blk[want == 0.0] == 0.0) and not np.any(np.signbit(blk[want == 0.0])), g
    assert n_nonempty >= 10 and len(_expected_block(cfg, oracle, groups[-1])) == 0
    with pytest.raises(B.MfdnError) as e:
        ctx.blocks(np.asarray([[1, 0, 2, 0, 1, 2]], np.int32))     # not ascending
    assert e.value.code == B.MFDN_ERR_ARG


# --------------------------------------------------------------------------------- compact requests
@pytest.mark.gpu
@pytest.mark.parametrize("idx", [0, 2])
def test_compact_u16_requests(torch, B, oracle, idx):
    """MFDN_REQ_U16: the same requests as 16-bit SPS indices give the same values and masks bit for bit, on the device paths
    and through the host wrapper; out-of-range indices are still caught."""
    cfg = get_cfg(idx)
    ctx = get_ctx(B, idx)
    rng = np.random.default_rng(31)
    allreq = cfg.requests()
    req = allreq[rng.choice(len(allreq), min(len(allreq), 30011), replace=False)].copy()
    req[:50, 0] = cfg.basis.n_sps            # out of range
    want, wmask, _, nbad = oracle.mscheme(cfg.basis, cfg.table, req)
    r16 = np.ascontiguousarray(req.astype(np.uint16))
    before = ctx.bad_request_count()
    for flags in (0, B.MFDN_FORCE_SORT, B.MFDN_ONE_PASS_SORT, B.MFDN_FORCE_NAIVE):
        got32, m32 = run_gpu(torch, ctx, req, flags)
        out, mask = ctx.mscheme(torch.from_numpy(r16).cuda(), flags=flags)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), got32) and np.array_equal(mask.cpu().numpy(), m32)
        check(cfg, out.cpu().numpy(), mask.cpu().numpy(), want, wmask)
    assert ctx.bad_request_count() - before == 8 * nbad == 400
    h_out, h_mask = ctx.mscheme_host(torch.from_numpy(r16).pin_memory(), chunk=7000)
    check(cfg, h_out.numpy(), h_mask.numpy(), want, wmask)


# --------------------------------------------------------------------------------- NEXT-4: fp32-stored slabs
@pytest.mark.gpu
@pytest.mark.parametrize("idx", [2, 3])
def test_fp32_stored_slabs(torch, B, oracle, idx):
    """MFDN_OPT_SLAB_FP32: the isospin-combined slabs are stored in fp32, sums stay fp64.  Mask bit-exact; values within the
    bound the header states: a stored value is within 2^-24 * 5 max|V| of the fp64 one (five isospin terms, weights <= 1) and
    a request sums at most `cells` of them with coefficient products <= 1.  Every path that reads the slabs is checked
    (work-item kernel, small groups, dense blocks, block mode); the table memory shrinks as stated."""
    cfg = get_cfg(idx)
    ctx64 = get_ctx(B, idx)
    ctx = B.Context(cfg.basis, 0).option(B.MFDN_OPT_SLAB_FP32).upload(cfg.table)
    assert B.mfdn_info(ctx.ctx, 8) <= 0.6 * B.mfdn_info(ctx64.ctx, 8)      # half, up to the 16-byte rounding per group
    with pytest.raises(B.MfdnError) as e:
        ctx.option(B.MFDN_OPT_SLAB_FP32, 0)             # too late
    assert e.value.code == B.MFDN_ERR_STATE
    req = cfg.requests() if cfg.all_pairs else cfg.requests(1 << 18, permute_frac=0.01)
    if len(req) > 300000:
        req = req[np.random.default_rng(2).choice(len(req), 300000, replace=False)]
    want, wmask, nt, _ = oracle.mscheme(cfg.basis, cfg.table, req)
    vmax = float(np.max(np.abs(cfg.table.values)))
    cells = max(1, int(np.max(nt)))                      # coupled terms of a request: upper bound for its cells
    tol = 2.0 ** -24 * 5 * vmax * cells
    worst = 0.0
    for flags in (0, B.MFDN_FORCE_SORT, B.MFDN_ONE_PASS_SORT, B.MFDN_FORCE_DENSE):
        got, gmask = run_gpu(torch, ctx, req, flags)
        assert np.array_equal(gmask, wmask)
        err = float(np.max(np.abs(got - want)))
        assert err <= tol, (flags, err, tol)
        assert np.all(got[gmask == 0] == 0.0)
        worst = max(worst, err)
    assert worst > 1e-11 * vmax                          # it really is the fp32-stored table
    got, gmask = run_gpu(torch, ctx, req, B.MFDN_FORCE_NAIVE)    # reads the fp64 planes
    check(cfg, got, gmask, want, wmask)
    tup = sorted(set(zip(cfg.table.state_a.tolist(), cfg.table.state_b.tolist(), cfg.table.state_c.tolist())))
    g = np.asarray([tup[3] + tup[5], tup[0] + tup[0]], np.int32)
    a, off = ctx.blocks(g)
    b, off64 = ctx64.blocks(g)
    torch.cuda.synchronize()
    assert np.array_equal(off, off64) and float((a - b).abs().max()) <= tol
    ctx.close()

