#!/usr/bin/env python
"""bench.py -- coupled-JT -> M-scheme transformation throughput on B200 (BASELINE.json metric).

One "step" = one pass of the whole hot path (H1 decode/selection/canonicalise/key, H2 group sort,
H3-H6 locate/stage/channel-sum/store incl. the gather back to request order) over one batch of synthetic requests:
config 3 = 3-body, E3max = 8, 2^26 requests sampled uniformly from the conserving pairs, arriving
UNSORTED and device-resident.  Prints ONE JSON line (see README/DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--log2n 26]
    python bench.py --impl reference ...      # the CPU oracle, as it stands, on the host cores

N > 1 (torchrun): every rank runs its own window of the request stream on its own GPU (the path has
no exchange step; tables are replicated) -> weak scaling, value = sum of requests / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "M-scheme 3-body elements/sec at E3max=8 (fp64)"
UNIT = "elements/s"

# Algorithmic work per request:
#   bytes: request in + value out + mask out + amortised slab; flops: direct channel sum
ALG = {
    1: {"bytes_presorted": 16 + 8 + 1 + 0.6, "bytes_unsorted": 16 + 8 + 1 + 0.6 + 100, "flops": 40.0},
    3: {"bytes_presorted": 24 + 8 + 1 + 2.3, "bytes_unsorted": 24 + 8 + 1 + 2.3 + 100, "flops": 290.0},
    4: {"bytes_presorted": 24 + 8 + 1 + 20.0, "bytes_unsorted": 24 + 8 + 1 + 20.0 + 100, "flops": 430.0},
    0: {"bytes_presorted": 16 + 8 + 1 + 0.3, "bytes_unsorted": 16 + 8 + 1 + 0.3 + 100, "flops": 20.0},
    2: {"bytes_presorted": 24 + 8 + 1 + 0.2, "bytes_unsorted": 24 + 8 + 1 + 0.2 + 100, "flops": 110.0},
}
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # 148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz = 37.2


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap,power.draw"

    def __init__(self, gpu_index):
        self.proc = None
        self.gpu = gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for k, nme in enumerate(names):
                if f[2 + k].lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def host_requests(cfg, n, start):
    if cfg.all_pairs:
        r = cfg.requests()
        reps = (n + len(r) - 1) // len(r)
        return np.ascontiguousarray(np.tile(r, (reps, 1))[:n])
    return cfg.requests(n, start=start, workers=os.cpu_count() or 1)


def cpu_baseline(cfg, n_sample, threads=0):
    """The oracle as it stands, timed on the host cores on the first n_sample requests of the stream."""
    from oracle import mscheme_c
    req = host_requests(cfg, n_sample, 0)
    mscheme_c.cg_table_for(cfg.basis, cfg.body)           # exact tables prebuilt (not timed)
    mscheme_c.mscheme(cfg.basis, cfg.table, req[:1024], threads)
    t0 = time.perf_counter()
    mscheme_c.mscheme(cfg.basis, cfg.table, req, threads)
    dt = time.perf_counter() - t0
    cores = threads or mscheme_c.num_threads()
    return n_sample / dt, cores, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1412_5989_b200 import workloads as W
    cfg = W.make_config(args.config)
    args.ref_log2n = 21 if args.ref_log2n is None else args.ref_log2n
    n_sample = 1 << args.ref_log2n
    from oracle import mscheme_c
    req = host_requests(cfg, n_sample, 0)
    mscheme_c.cg_table_for(cfg.basis, cfg.body)
    for _ in range(args.warmup):
        mscheme_c.mscheme(cfg.basis, cfg.table, req[: max(1024, n_sample // 16)])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        mscheme_c.mscheme(cfg.basis, cfg.table, req)
    dt = (time.perf_counter() - t0) / args.steps
    val = n_sample / dt
    cores = mscheme_c.num_threads()
    sample = f"first 2^{args.ref_log2n} requests of the config-{args.config} stream per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "requests_per_step": n_sample, "kind": "CPU oracle (oracle/mscheme_oracle.c)"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--log2n", type=int, default=26)
    ap.add_argument("--ref-log2n", type=int, default=None,
                    help="log2 of the CPU-oracle sample (default: 25 for the cpu_baseline leg, 21 per step of --impl reference)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="skip the per-config block (all five BASELINE.json workloads)")
    ap.add_argument("--config-reps", type=int, default=10)
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_1412_5989_b200 import binding as B, build, shard, workloads as W

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    torch.cuda.set_device(local)
    if local == 0:
        build.build()
    if world > 1:
        dist.barrier()

    cfg = W.make_config(args.config)
    body = cfg.body
    n = 1 << args.log2n
    ctx = B.Context(cfg.basis, local).upload(cfg.table)
    h_req = torch.from_numpy(host_requests(cfg, n, shard.rank_window(rank, world, n)[0])).pin_memory()
    d_req = h_req.cuda(non_blocking=True)
    d_out = torch.empty(n, dtype=torch.float64, device="cuda")
    d_mask = torch.empty(n, dtype=torch.uint8, device="cuda")
    need = max(ctx.work_bytes(body, n, 0), ctx.work_bytes(body, n, B.MFDN_PRESORTED))   # both modes are timed with this scratch
    work = torch.empty(need, dtype=torch.uint8, device="cuda")
    torch.cuda.synchronize()
    stream = torch.cuda.current_stream()

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def timed(flags, req, steps, warmup, sampler=None):
        if sampler:
            sampler.start()          # nvidia-smi needs a few 100 ms to come up: start before the warm-up steps
        for _ in range(warmup):
            ctx.mscheme(req, d_out, d_mask, flags, work)
        sync_all()
        l0 = B.mfdn_info(ctx.ctx, 6)
        B.mfdn_profile(ctx.ctx, 1)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(steps):
            ctx.mscheme(req, d_out, d_mask, flags, work)
        e1.record(stream)
        sync_all()
        clocks = sampler.stop() if sampler else None
        B.mfdn_profile(ctx.ctx, 0)
        ms_sort, ms_tr, ms_un, calls = B.mfdn_profile_read(ctx.ctx)
        ms = shard.max_over_ranks(e0.elapsed_time(e1) / steps, "cuda")
        k = max(calls, 1)
        return ms, ms_sort / k, ms_tr / k, ms_un / k, B.mfdn_info(ctx.ctx, 6) - l0, clocks

    # ---- headline: whole path on unsorted device-resident input
    sampler = ClockSampler(local)
    ms, ms_sort, ms_tr, ms_un, launches, clocks = timed(0, d_req, args.steps, args.warmup, sampler)
    n_mask = int(d_mask.sum(dtype=torch.int64).item())
    frac_mask = n_mask / n
    # 2^14 sampled outputs of the timed launch configuration against the CPU oracle (rank 0, N = 1)
    headline_check = None
    do_configs = world == 1 and not args.no_configs
    if do_configs:
        from oracle import mscheme_c
        sample = np.sort(np.random.default_rng(1234 + args.config).choice(n, min(n, 1 << 14), replace=False))
        want, wmask, _, _ = mscheme_c.mscheme(cfg.basis, cfg.table, h_req.numpy()[sample])
        ds = torch.from_numpy(sample).cuda()
        got, gmask = d_out[ds].cpu().numpy(), d_mask[ds].cpu().numpy()
        headline_check = {"sampled": int(len(sample)), "max_abs_delta": float(np.max(np.abs(got - want))),
                          "tolerance": 1e-12 * float(np.max(np.abs(cfg.table.values))), "mask_bit_exact": bool(np.array_equal(gmask, wmask))}
    # ---- NEXT-1: the same step with the results accumulated into a many-body array instead of returned
    accum = None
    if world == 1:
        h_len = 1 << 24
        loc, phase = W.many_body_targets(n, h_len, seed=args.config)
        d_loc, d_phase = torch.from_numpy(loc).cuda(), torch.from_numpy(phase).cuda()
        d_H = torch.zeros(h_len, dtype=torch.float64, device="cuda")
        awork = torch.empty(B.mfdn_mscheme_accumulate(ctx.ctx, body, n, 0, 0, 0, 0, 0, 0, 0, 0, 0), dtype=torch.uint8, device="cuda")
        for _ in range(args.warmup):
            ctx.accumulate(d_req, d_loc, d_phase, d_H, d_mask, 0, awork)
        d_H.zero_()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        ctx.accumulate(d_req, d_loc, d_phase, d_H, d_mask, 0, awork)
        e1.record(stream)
        torch.cuda.synchronize()
        # property that holds at any size: the accumulated array equals a library index_add of the returned values
        ref = torch.zeros(h_len, dtype=torch.float64, device="cuda").index_add_(0, d_loc, d_phase * d_out)
        accum = {"ms_per_step": e0.elapsed_time(e1), "value": n / (e0.elapsed_time(e1) * 1e-3), "unit": UNIT, "h_len": h_len,
                 "targets": "runs of geometric length (mean 4) on uniform elements, phases +-1 (workloads.many_body_targets)",
                 "max_abs_delta_vs_index_add_of_returned_values": float((d_H - ref).abs().max().item()),
                 "api": "mfdn_mscheme_accumulate_3b" if body == 3 else "mfdn_mscheme_accumulate_2b"}
        del d_loc, d_phase, d_H, awork, ref, loc, phase
    # ---- the same multiset pre-ordered by the library's group key (MFDN_PRESORTED): transform proper
    keys = ctx.group_keys(d_req)
    order = torch.argsort(keys.to(torch.int64) & 0xFFFFFFFF)
    d_sorted = d_req[order].contiguous()
    del keys, order
    ms_p, ms_sort_p, ms_tr_p, _, _, _ = timed(B.MFDN_PRESORTED, d_sorted, args.steps, args.warmup)
    del d_sorted
    # ---- end to end through the C ABI with HOST buffers (H2D + D2H inside the timed region)
    h_out = torch.empty(n, dtype=torch.float64).pin_memory()
    h_mask = torch.empty(n, dtype=torch.uint8).pin_memory()
    ctx.mscheme_host(h_req, h_out, h_mask)
    sync_all()
    t0 = time.perf_counter()
    for _ in range(args.e2e_steps):
        ctx.mscheme_host(h_req, h_out, h_mask)
    e2e_s = (time.perf_counter() - t0) / args.e2e_steps
    e2e_s = shard.max_over_ranks(e2e_s, "cuda")
    assert int(h_mask.sum(dtype=torch.int64).item()) == n_mask, "host-buffer path disagrees with device path"
    # the same call with compact requests (MFDN_REQ_U16: 16-bit SPS indices, half the host-to-device bytes; the call is PCIe-bound)
    e2e16_s = None
    if cfg.basis.n_sps <= 65536:
        h_req16 = torch.from_numpy(h_req.numpy().astype(np.uint16)).pin_memory()
        ref_out = h_out.clone()
        ctx.mscheme_host(h_req16, h_out, h_mask)
        sync_all()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            ctx.mscheme_host(h_req16, h_out, h_mask)
        e2e16_s = shard.max_over_ranks((time.perf_counter() - t0) / args.e2e_steps, "cuda")
        assert torch.equal(ref_out, h_out), "compact-request path disagrees with the int32 path"
        del h_req16, ref_out
    fp64_peak = B.mfdn_fp64_peak(ctx.ctx)
    # ---- all five BASELINE.json workloads inside the same run (same clocks record): whole call, unsorted and MFDN_PRESORTED
    configs = None
    if do_configs:
        from paper_1412_5989_b200 import report
        ctx.close()
        del d_req, d_out, d_mask, work, h_out, h_mask
        torch.cuda.empty_cache()
        configs = {}
        for idx in (0, 1, 2, 4):
            if idx != args.config:
                configs[str(idx)] = report.measure(idx, reps=args.config_reps, check=14, oracle=mscheme_c, fp64_peak=fp64_peak,
                                                   workers=os.cpu_count() or 1)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    hbm_peak, peak_src = measured_peaks()
    alg = ALG[args.config]
    t_tr = ms_tr * 1e-3
    flops_rate = alg["flops"] * n / t_tr / 1e12
    # the transform kernel moves request + outputs + slab (+ order array and gather sectors when sorted internally)
    gbs_tr = alg["bytes_presorted"] * n / t_tr / 1e9
    roof_hbm_ms = alg["bytes_presorted"] * n / (hbm_peak * 1e9) * 1e3
    roof_alu_ms = alg["flops"] * n / (fp64_peak * 1e12) * 1e3
    # figures taken from the ncu --set full capture of the dominant kernel (profiles/dram_traffic.txt names the capture, its
    # command and the commit it was made at; a capture cannot run inside a timed bench)
    prof = {}
    tp = os.path.join(ROOT, "profiles", "dram_traffic.txt")
    if os.path.exists(tp):
        for line in open(tp):
            f = line.split("#")[0].split()
            if len(f) >= 2:
                prof[f[0]] = f[1]
    traffic = float(prof[f"k_transform{body}_dram_bytes_per_launch"]) if f"k_transform{body}_dram_bytes_per_launch" in prof else None
    exec_flops = float(prof.get(f"k_transform{body}_executed_flops_per_request", "nan"))
    out = {
        "metric": METRIC, "value": world * n / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "requests_per_step_per_gpu": n, "input_order": "unsorted (stream order)",
                   "input_residency": "device", "l2": "inputs (%.2f GiB) exceed L2; no flush" % (n * 8 * body / 2 ** 30),
                   "mask1_fraction": frac_mask, "parallelism": "replicas, request stream sharded by rank" if world > 1 else "single GPU"},
        "clocks": clocks, "gpu_launches": int(launches),
        "e2e": ({"value": world * n / e2e16_s, "unit": UNIT, "h2d_bytes_per_step": n * 4 * body,
                 "d2h_bytes_per_step": n * 9, "ms_per_step": e2e16_s * 1e3, "steps": args.e2e_steps,
                 "api": "mfdn_mscheme_host, flag MFDN_REQ_U16: requests as 16-bit SPS indices (pinned host buffers, 4 streams, "
                        "2^22-request chunks); both directions of the PCIe link are what bounds it",
                 "int32_requests": {"value": world * n / e2e_s, "ms_per_step": e2e_s * 1e3, "h2d_bytes_per_step": n * 8 * body}}
                if e2e16_s else
                {"value": world * n / e2e_s, "unit": UNIT, "h2d_bytes_per_step": n * 8 * body,
                 "d2h_bytes_per_step": n * 9, "ms_per_step": e2e_s * 1e3, "steps": args.e2e_steps,
                 "api": "mfdn_mscheme_host (pinned host buffers, 4 streams, 2^22-request chunks)"}),
        "breakdown_ms": {"group_sort_H1_H2": ms_sort, "transform_H3_H5": ms_tr, "gather_to_request_order_H6": ms_un,
                         "presorted": {"keys_items_H1_H3": ms_sort_p, "transform_H3_H6": ms_tr_p}},
        "presorted": {"value": world * n / (ms_p * 1e-3), "unit": UNIT, "ms_per_step": ms_p,
                      "note": "same multiset pre-ordered by mfdn_group_keys, flag MFDN_PRESORTED"},
        "roofline": {"kernel": f"k_transform{body}" + (" + k_transform3_small (groups of <= 16 records)" if body == 3 else "") + ": dominant kernel of the unsorted step; CUDA events on the launch stream", "bound": "alu",
                     "achieved": flops_rate, "peak": fp64_peak, "unit": "TFLOP/s", "frac": flops_rate / fp64_peak,
                     "traffic": traffic, "traffic_source": {"file": "profiles/dram_traffic.txt", "capture": prof.get("capture"),
                                                            "commit": prof.get("commit")},
                     "flops_per_request": alg["flops"],
                     "note": "frac = ALGORITHMIC flops of the direct channel sum (SURVEY.md 8(d)) / kernel time / measured DFMA peak; "
                             "the kernel executes fewer (isospin-combined slabs are built at upload), see `as_built`",
                     "as_built": {"executed_flops_per_request": exec_flops,
                                  "frac_alu_executed": (exec_flops * n / t_tr / 1e12 / fp64_peak) if exec_flops == exec_flops else None,
                                  "applicable_bound": "hbm", "frac_hbm": gbs_tr / hbm_peak,
                                  "limiter_measured": prof.get(f"k_transform{body}_limiter")},
                     "peak_source": "measured DFMA micro-benchmark (mfdn_fp64_peak); nominal %.1f" % FP64_NOMINAL_TFLOPS,
                     "hbm": {"achieved": gbs_tr, "peak": hbm_peak, "unit": "GB/s", "frac": gbs_tr / hbm_peak,
                             "bytes_per_request": alg["bytes_presorted"], "peak_source": peak_src},
                     "roof_ms": {"alu": roof_alu_ms, "hbm": roof_hbm_ms, "kernel": ms_tr},
                     "presorted_kernel_ms": ms_tr_p,
                     "presorted_frac_alu": alg["flops"] * n / (ms_tr_p * 1e-3) / 1e12 / fp64_peak},
    }
    if not args.no_cpu_baseline:
        args.ref_log2n = 25 if args.ref_log2n is None else args.ref_log2n
        n_s = 1 << args.ref_log2n
        v, cores, dt = cpu_baseline(cfg, n_s)
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                               "note": "definition-order checker (oracle/mscheme_oracle.c), never tuned: a reported baseline, not a CPU implementation",
                               "sample": f"first 2^{args.ref_log2n} requests of the same stream, {dt:.1f} s"}
    if accum is not None:
        out["accumulate_epilogue"] = accum
    if configs is not None:
        b_pre, b_uns, fl = alg["bytes_presorted"], alg["bytes_unsorted"], alg["flops"]
        mine = {"workload": cfg.name, "requests": n, "calls": 1, "mask1_fraction": frac_mask, "oracle_check": headline_check}
        for mode, t, byts in (("unsorted", ms, b_uns), ("presorted", ms_p, b_pre)):
            t_h, t_a = byts * n / (hbm_peak * 1e9) * 1e3, fl * n / (fp64_peak * 1e12) * 1e3
            mine[mode] = {"ms": t, "elements_per_s": n / t * 1e3, "alg_bytes_per_request": byts, "alg_flops_per_request": fl,
                          "roof_ms": {"hbm": t_h, "alu": t_a}, "applicable": "hbm" if t_h >= t_a else "alu", "frac_of_roof": max(t_h, t_a) / t}
        configs[str(args.config)] = mine
        out["configs"] = {k: configs[k] for k in sorted(configs)}
    out["context"] = "paper (Titan, K20): 2.2-2.7x matrix-construction, 1.2-1.4x whole-run speedup; not a target"
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
