#!/usr/bin/env python
"""Per-config report: elements/s and roofline fractions of the five BASELINE.json workloads on
one GPU, device-resident requests, whole call (selection + group sort + transform + store) timed with CUDA events.

    python -m paper_1412_5989_b200.report [--configs 0,1,2,3,4] [--reps 20] [--check 14] > report.md
    python -m paper_1412_5989_b200.report --chunks           # multi-client operation: chunk size x host threads (NEXT-3)
    python -m paper_1412_5989_b200.report --dense            # dense-block path (H5') against the default path, by request density

Configs 0 and 2 are small ("ALL conserving pairs"): they are latency measurements, an L2 flush (a 256 MiB memset)
runs between repetitions.  Configs 1 and 3: 2^26 requests per call, unsorted and pre-ordered by mfdn_group_keys.
Config 4: 16 batches of 2^24 requests issued round-robin on two streams.  Algorithmic bytes/flops per request are
SURVEY.md 8(d)'s figures (the same table bench.py uses).  `measure()` is what bench.py calls for its `configs` block;
with check > 0 it also compares 2^check sampled outputs of the timed launch configuration with the CPU oracle (the
caller passes the oracle module: this package never imports it)."""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

ALG = {  # bytes (pre-sorted / extra when unsorted) and direct-sum flops per request
    0: (16 + 8 + 1 + 0.3, 100.0, 20.0), 1: (16 + 8 + 1 + 0.6, 100.0, 40.0), 2: (24 + 8 + 1 + 0.2, 100.0, 110.0),
    3: (24 + 8 + 1 + 2.3, 100.0, 290.0), 4: (24 + 8 + 1 + 20.0, 100.0, 430.0),
}


def hbm_peak():
    peaks = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks):
        return float(json.load(open(peaks))["hbm_gbs"]), "measured"
    return 6650.0, "fallback"


def measure(idx, reps=20, check=0, oracle=None, fp64_peak=None, log2n=26, flush=None, workers=0):
    """Times config idx (unsorted and MFDN_PRESORTED), returns a dict.  check > 0: max|delta| and mask equality against
    `oracle.mscheme` on 2^check sampled requests of the first timed batch (unsorted launch)."""
    import torch
    from paper_1412_5989_b200 import binding as B, workloads as W
    hbm, hbm_src = hbm_peak()
    cfg = W.make_config(idx)
    ctx = B.Context(cfg.basis, 0).upload(cfg.table)
    if fp64_peak is None:
        fp64_peak = B.mfdn_fp64_peak(ctx.ctx)
    body = cfg.body
    if idx == 4:
        nb, per = 16, 1 << 24
        host = [cfg.requests(per, start=k * per, workers=workers) for k in range(nb)]
    elif cfg.all_pairs:
        host = [cfg.requests()]
    else:
        host = [cfg.requests(1 << log2n, workers=workers)]
    batches = [torch.from_numpy(h).cuda() for h in host]
    n_call = batches[0].shape[0]
    n_total = sum(b.shape[0] for b in batches)
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    outs = [torch.empty(n_call, dtype=torch.float64, device="cuda") for _ in streams]
    masks = [torch.empty(n_call, dtype=torch.uint8, device="cuda") for _ in streams]
    works = [torch.empty(max(ctx.work_bytes(body, n_call, 0), ctx.work_bytes(body, n_call, B.MFDN_PRESORTED)), dtype=torch.uint8, device="cuda") for _ in streams]   # both modes timed below
    small = n_total * 8 * body < (200 << 20)
    if small and flush is None:
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def one_pass(reqs, flags):
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for s in streams:
            s.wait_stream(torch.cuda.current_stream())
        for k, r in enumerate(reqs):
            s = streams[k % 2]
            with torch.cuda.stream(s):
                ctx.mscheme(r, outs[k % 2], masks[k % 2], flags, works[k % 2], s.cuda_stream)
        for s in streams:
            torch.cuda.current_stream().wait_stream(s)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)

    def timed(reqs, flags):
        for _ in range(3):
            one_pass(reqs, flags)
        t = []
        for _ in range(reps):
            if small:
                flush.zero_()
            t.append(one_pass(reqs, flags))
        return statistics.median(t)

    one_pass(batches[:1], 0)
    frac_mask = float(masks[0].sum(dtype=torch.int64).item()) / n_call   # first call's share of requests with mask = 1
    res = {"workload": cfg.name, "requests": n_total, "calls": len(batches), "mask1_fraction": frac_mask}
    if check and oracle is not None:
        ns = min(1 << check, n_call)
        sample = np.sort(np.random.default_rng(1234 + idx).choice(n_call, ns, replace=False))
        want, wmask, _, _ = oracle.mscheme(cfg.basis, cfg.table, host[0][sample])
        ds = torch.from_numpy(sample).cuda()
        got, gmask = outs[0][ds].cpu().numpy(), masks[0][ds].cpu().numpy()
        vmax = float(np.max(np.abs(cfg.table.values)))
        res["oracle_check"] = {"sampled": int(ns), "max_abs_delta": float(np.max(np.abs(got - want))), "tolerance": 1e-12 * vmax,
                               "mask_bit_exact": bool(np.array_equal(gmask, wmask))}
    ms_u = timed(batches, 0)
    sorted_batches = []
    for r in batches:
        keys = ctx.group_keys(r)
        order = torch.argsort(keys.to(torch.int64) & 0xFFFFFFFF)
        sorted_batches.append(r[order].contiguous())
        del keys, order
    del batches
    ms_p = timed(sorted_batches, B.MFDN_PRESORTED)
    b_pre, b_sort, flops = ALG[idx]
    for mode, ms, byts in (("unsorted", ms_u, b_pre + b_sort), ("presorted", ms_p, b_pre)):
        t_h = byts * n_total / (hbm * 1e9) * 1e3
        t_a = flops * n_total / (fp64_peak * 1e12) * 1e3
        roof, which = (t_h, "hbm") if t_h >= t_a else (t_a, "alu")
        res[mode] = {"ms": ms, "elements_per_s": n_total / ms * 1e3, "alg_bytes_per_request": byts, "alg_flops_per_request": flops,
                     "roof_ms": {"hbm": t_h, "alu": t_a}, "applicable": which, "frac_of_roof": roof / ms}
    ctx.close()
    del sorted_batches, outs, masks, works
    torch.cuda.empty_cache()
    return res


def dense_table(reps=10):
    """Dense-block path (MFDN_FORCE_DENSE, step H5') against the default path on pre-sorted input, by request density:
    config 2 (ALL pairs) thinned at random, and all ordered pairs of twelve mid-size sectors of config 3 thinned likewise."""
    import torch
    from paper_1412_5989_b200 import binding as B, workloads as W
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def timed(ctx, d_req, flags):
        n = d_req.shape[0]
        out = torch.empty(n, dtype=torch.float64, device="cuda")
        mask = torch.empty(n, dtype=torch.uint8, device="cuda")
        work = torch.empty(ctx.work_bytes(3, n, flags), dtype=torch.uint8, device="cuda")
        for _ in range(3):
            ctx.mscheme(d_req, out, mask, flags, work)
        torch.cuda.synchronize()
        ts, tt = [], []
        for _ in range(reps):
            flush.zero_()
            B.mfdn_profile(ctx.ctx, 1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            ctx.mscheme(d_req, out, mask, flags, work)
            e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
            tt.append(B.mfdn_profile_read(ctx.ctx)[1])
            B.mfdn_profile(ctx.ctx, 0)
        return statistics.median(ts), statistics.median(tt), out

    print("| workload | density | requests | default: call ms | default: transform ms | dense: call ms | dense: transform + dense kernels ms | max abs diff |")
    print("|---|---|---|---|---|---|---|---|")
    for idx in (2, 3):
        cfg = W.make_config(idx)
        ctx = B.Context(cfg.basis, 0).upload(cfg.table)
        if idx == 2:
            allreq, name = cfg.requests(), "config 2, all pairs"
        else:
            ms = cfg.ms
            sz = ms.sec_size
            pick = [s for s in np.argsort(sz) if 300 <= sz[s] <= 700][:12]
            parts = []
            for s in pick:
                st = ms.states[ms.sec_start[s]:ms.sec_start[s + 1]]
                k = st.shape[0]
                parts.append(np.concatenate([np.repeat(st, k, 0), np.tile(st, (k, 1))], 1))
            allreq, name = np.ascontiguousarray(np.concatenate(parts), np.int32), "config 3 basis, all pairs of 12 sectors"
        rng = np.random.default_rng(5)
        for f in (1.0, 0.5, 0.25, 0.12, 0.06):
            req = allreq if f == 1.0 else allreq[rng.random(len(allreq)) < f]
            d = torch.from_numpy(req).cuda()
            keys = ctx.group_keys(d)
            ds = d[torch.argsort(keys.to(torch.int64) & 0xFFFFFFFF)].contiguous()
            a = timed(ctx, ds, B.MFDN_PRESORTED | B.MFDN_FORCE_SORT)     # the work-item kernels of the group-sort path
            b = timed(ctx, ds, B.MFDN_PRESORTED | B.MFDN_FORCE_DENSE)
            print(f"| {name} | {f:.2f} | {len(req)} | {a[0]:.3f} | {a[1]:.3f} | {b[0]:.3f} | {b[1]:.3f} | {float((a[2] - b[2]).abs().max()):.1e} |")
        ctx.close()


def chunk_table(idx=3, total_log2=22):
    """Multi-client operation (SURVEY.md 8(f) NEXT-3; PAPER.md:93 buffers of ~20 000 requests, :103 one stream per OpenMP
    thread): T native host threads (mfdn_multi_client), each with its own stream and scratch, push chunks of a fixed size through
    one context until 2^total_log2 requests are done; wall-clock throughput of the whole job, device-resident requests; the
    result is checked bitwise against one big call."""
    import torch
    from paper_1412_5989_b200 import binding as B, workloads as W
    cfg = W.make_config(idx)
    ctx = B.Context(cfg.basis, 0).upload(cfg.table)
    n = 1 << total_log2
    d_req = torch.from_numpy(cfg.requests(n, workers=os.cpu_count() or 1)).cuda()
    out = torch.empty(n, dtype=torch.float64, device="cuda")
    mask = torch.empty(n, dtype=torch.uint8, device="cuda")
    base, bmask = ctx.mscheme(d_req, flags=B.MFDN_FORCE_SORT)
    base, bmask = base.clone(), bmask.clone()
    print("| chunk (requests) | " + " | ".join(f"{t} thread{'s' if t > 1 else ''}: elements/s" for t in (1, 2, 4, 8, 16)) + " |")
    print("|---|---|---|---|---|---|")
    for lg in (10, 12, 14, 15, 16, 18, 20, 22):
        cells = []
        for nthreads in (1, 2, 4, 8, 16):
            best = 0.0
            for _ in range(3):
                out.zero_()
                sec = B.mfdn_multi_client(ctx.ctx, cfg.body, n, d_req.data_ptr(), out.data_ptr(), mask.data_ptr(), 1 << lg, nthreads)
                best = max(best, n / sec)
            assert torch.equal(out, base) and torch.equal(mask, bmask), "chunked result differs from the single call"
            cells.append(f"{best:.3e}")
        print(f"| 2^{lg} = {1 << lg} | " + " | ".join(cells) + " |")
    ctx.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="0,1,2,3,4")
    ap.add_argument("--reps", type=int, default=20)
    ap.add_argument("--dense", action="store_true")
    ap.add_argument("--chunks", action="store_true", help="multi-client table: chunk size x host threads (config 3)")
    args = ap.parse_args()
    import torch
    from paper_1412_5989_b200 import binding as B, workloads as W
    if args.dense:
        return dense_table()
    if args.chunks:
        return chunk_table()
    hbm, hbm_src = hbm_peak()
    ctx = B.Context(W.make_config(0).basis, 0)
    fp64 = B.mfdn_fp64_peak(ctx.ctx)
    ctx.close()
    rows = [measure(int(x), args.reps, fp64_peak=fp64) for x in args.configs.split(",")]
    print(f"fp64 peak (measured DFMA micro-benchmark) {fp64:.1f} TFLOP/s; HBM peak {hbm:.1f} GB/s ({hbm_src}); "
          f"{torch.cuda.get_device_name(0)}; median of {args.reps} repetitions after 3 warm-ups\n")
    print("| workload | input | requests | calls | ms | elements/s | alg. B/req | alg. flops/req | HBM roof ms | fp64 roof ms | applicable | fraction of roof | mask = 1 |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    for r in rows:
        for mode in ("unsorted", "presorted"):
            m = r[mode]
            print(f"| {r['workload']} | {mode} | {r['requests']} | {r['calls']} | {m['ms']:.3f} | {m['elements_per_s']:.3e} | {m['alg_bytes_per_request']:.1f} | "
                  f"{m['alg_flops_per_request']:.0f} | {m['roof_ms']['hbm']:.3f} | {m['roof_ms']['alu']:.3f} | {m['applicable']} | {m['frac_of_roof']:.3f} | {r['mask1_fraction']:.4f} |")


if __name__ == "__main__":
    sys.path.insert(0, ROOT)
    main()
