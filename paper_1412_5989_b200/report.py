#!/usr/bin/env python
"""Per-config report: elements/s and roofline fractions of the five BASELINE.json workloads on
one GPU, device-resident requests, whole call (selection + group sort + transform + store) timed with CUDA events.

    python -m paper_1412_5989_b200.report [--configs 0,1,2,3,4] [--reps 20] > report.md

Configs 0 and 2 are small ("ALL conserving pairs"): they are latency measurements, an L2 flush (a 256 MiB memset)
runs between repetitions.  Configs 1 and 3: 2^26 requests per call, unsorted and pre-ordered by mfdn_group_keys.
Config 4: 16 batches of 2^24 requests issued round-robin on two streams.  Algorithmic bytes/flops per request are
SURVEY.md 8(d)'s figures (the same table bench.py uses)."""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

ALG = {  # bytes (pre-sorted / unsorted) and direct-sum flops per request
    0: (16 + 8 + 1 + 0.3, 100.0, 20.0), 1: (16 + 8 + 1 + 0.6, 100.0, 40.0), 2: (24 + 8 + 1 + 0.2, 100.0, 110.0),
    3: (24 + 8 + 1 + 2.3, 100.0, 290.0), 4: (24 + 8 + 1 + 20.0, 100.0, 430.0),
}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="0,1,2,3,4")
    ap.add_argument("--reps", type=int, default=20)
    args = ap.parse_args()
    import torch
    from paper_1412_5989_b200 import binding as B, workloads as W

    peaks = os.path.join(ROOT, "MEASURED_PEAKS.json")
    hbm = float(json.load(open(peaks))["hbm_gbs"]) if os.path.exists(peaks) else 6650.0
    hbm_src = "measured" if os.path.exists(peaks) else "fallback"
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    rows = []
    fp64 = None
    for idx in [int(x) for x in args.configs.split(",")]:
        cfg = W.make_config(idx)
        ctx = B.Context(cfg.basis, 0).upload(cfg.table)
        if fp64 is None:
            fp64 = B.mfdn_fp64_peak(ctx.ctx)
        body = cfg.body
        if idx == 4:
            nb, per = 16, 1 << 24
            batches = [torch.from_numpy(cfg.requests(per, start=k * per)).cuda() for k in range(nb)]
        elif cfg.all_pairs:
            batches = [torch.from_numpy(cfg.requests()).cuda()]
        else:
            batches = [torch.from_numpy(cfg.requests(1 << 26)).cuda()]
        n_call = batches[0].shape[0]
        n_total = sum(b.shape[0] for b in batches)
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        outs = [torch.empty(n_call, dtype=torch.float64, device="cuda") for _ in streams]
        masks = [torch.empty(n_call, dtype=torch.uint8, device="cuda") for _ in streams]
        works = [torch.empty(ctx.work_bytes(body, n_call, 0), dtype=torch.uint8, device="cuda") for _ in streams]

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
            for _ in range(args.reps):
                if n_total * 8 * body < (200 << 20):
                    flush.zero_()
                t.append(one_pass(reqs, flags))
            return statistics.median(t)

        one_pass(batches[:1], 0)
        frac_mask = float(masks[0].sum(dtype=torch.int64).item()) / n_call   # first call's share of requests with mask = 1
        ms_u = timed(batches, 0)
        sorted_batches = []
        for r in batches:
            keys = ctx.group_keys(r)
            order = torch.argsort(keys.to(torch.int64) & 0xFFFFFFFF)
            sorted_batches.append(r[order].contiguous())
            del keys, order
        ms_p = timed(sorted_batches, B.MFDN_PRESORTED)
        b_pre, b_sort, flops = ALG[idx]
        for mode, ms, byts in (("unsorted", ms_u, b_pre + b_sort), ("pre-sorted", ms_p, b_pre)):
            t_h = byts * n_total / (hbm * 1e9) * 1e3
            t_a = flops * n_total / (fp64 * 1e12) * 1e3
            roof, which = (t_h, "hbm") if t_h >= t_a else (t_a, "alu")
            rows.append((cfg.name, mode, n_total, len(batches), ms, n_total / ms * 1e3, byts, flops, t_h, t_a, which, roof / ms, frac_mask))
        ctx.close()
        del batches, sorted_batches, outs, masks, works
        torch.cuda.empty_cache()
    print(f"fp64 peak (measured DFMA micro-benchmark) {fp64:.1f} TFLOP/s; HBM peak {hbm:.1f} GB/s ({hbm_src}); "
          f"{torch.cuda.get_device_name(0)}; median of {args.reps} repetitions after 3 warm-ups\n")
    print("| workload | input | requests | calls | ms | elements/s | alg. B/req | alg. flops/req | HBM roof ms | fp64 roof ms | applicable | fraction of roof | mask = 1 |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    for r in rows:
        print(f"| {r[0]} | {r[1]} | {r[2]} | {r[3]} | {r[4]:.3f} | {r[5]:.3e} | {r[6]:.1f} | {r[7]:.0f} | {r[8]:.3f} | {r[9]:.3f} | {r[10]} | {r[11]:.3f} | {r[12]:.4f} |")


if __name__ == "__main__":
    sys.path.insert(0, ROOT)
    main()
