#!/usr/bin/env python
"""bench.py — throughput of the matrix-element hot path (BASELINE.json metric: matrix elements/sec on one
B200 for g g -> t t~ g g, FP64 headline, mixed and FP32 beside it, and the fraction of the FP roofline).

One "step" = one me_compute pass (external wavefunctions, currents, diagram
amplitudes, jamps, colour sum, helicity sum) over one batch of seeded synthetic RAMBO events.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--quick]

N > 1 is launched by torch.distributed.run (one rank per GPU); every rank takes its own page-aligned shard
of N x 524288 events (weak scaling, no data-path collective).
`--impl reference` times the CPU oracle (oracle/) on the host cores on a bounded sample of the same workload.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import inputs  # noqa: E402

HEADLINE = 3                      # index into inputs.CONFIGS: g g -> t t~ g g, 524288 events, seed 3
NOMINAL_MHZ = 1965.0
N_SM = 148
# peaks derived from unit counts x clock: 64 FP64 FMA and 128 FP32 FMA per clock per SM
PEAK_TFLOPS = {"fp64": N_SM * 64 * 2 * NOMINAL_MHZ * 1e-6, "fp32": N_SM * 128 * 2 * NOMINAL_MHZ * 1e-6}
PAPER_V100 = {"gg_ttxgg": {"fp64": 4.21e5, "fp32": 8.77e5}, "gg_ttxggg": {"fp64": 9.51e3, "mixed": 1.19e4, "fp32": 2.41e4}}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *a):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"], "samples": 0}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}


def oracle_rate(proc, p, target_seconds=15.0):
    """MEs/s of the oracle as it stands on all host cores, on a bounded sample of the events in p."""
    import oracle
    oracle.build()
    cores = oracle.max_threads()
    n0 = min(len(p), 256 * cores)
    t0 = time.perf_counter(); oracle.me(proc, p[:n0]); dt = time.perf_counter() - t0
    n = int(min(len(p), max(n0, target_seconds * n0 / max(dt, 1e-6))))
    t0 = time.perf_counter(); oracle.me(proc, p[:n]); dt = time.perf_counter() - t0
    return n / dt, cores, n, dt


def run_reference(args):
    """--impl reference: the CPU oracle, rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    cfg = inputs.CONFIGS[HEADLINE]
    cores = oracle.max_threads()
    # bounded sample per step: the first 1024*cores events of the seeded config (host Philox + RAMBO of the oracle)
    nsample = 1024 * cores
    p, _ = oracle.events(cfg["process"], nsample, cfg["seed"])
    for _ in range(args.warmup):
        oracle.me(cfg["process"], p[:8 * cores])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.me(cfg["process"], p)
    dt = time.perf_counter() - t0
    v = nsample * args.steps / dt
    sample = "first %d events of the %d-event config per step" % (nsample, cfg["events"])
    print(json.dumps({
        "impl": "reference", "metric": "matrix elements/sec (g g -> t t~ g g, FP64)", "value": v, "unit": "MEs/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg["label"] + ", %d RAMBO events, sqrt(s)=1500 GeV, seed %d" % (cfg["events"], cfg["seed"]), "sample": sample},
        "cpu_baseline": {"value": v, "unit": "MEs/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "MEs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--quick", action="store_true", help="headline workload only (no other processes, no oracle leg)")
    ap.add_argument("--events", type=int, default=0, help="override events per GPU (default: the config's)")
    ap.add_argument("--sweep", action="store_true", help="add throughput vs batch size (8192 .. config size) and 1/2/4 concurrent streams "
                                                         "to the JSON line (PAPER.md line 65 / Fig. 1: plateau and GPU sharing)")
    ap.add_argument("--config", type=int, default=HEADLINE, choices=[1, 2, 3, 4],
                    help="index into inputs.CONFIGS of the timed workload (default 3 = g g -> t t~ g g, the BASELINE.json metric; "
                         "others are for profiling a single process, e.g. --quick --config 4)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import numpy as np
    import torch
    import paper_2303_18244_b200 as me
    from paper_2303_18244_b200.shard import shard_range

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl")
    me.lib()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    HL = args.config
    cfg = inputs.CONFIGS[HL]
    per_gpu = args.events or cfg["events"]
    first, n = shard_range(per_gpu * world, rank, world)
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2

    def setup(proc, n, first):
        c = inputs.CONFIGS[proc]
        ctx = me.MEContext(proc)
        rnd = me.me_philox_uniform(c["seed"], first, n, c["nfinal"])
        mom, wt = ctx.me_rambo(inputs.SQRT_S, rnd)
        del rnd
        ctx.me_filter_helicities(mom, 32)
        return ctx, mom

    def timed(ctx, mom, n, prec, steps, warmup, host=None):
        """-> (total ms over `steps`, per-step list); L2 flushed (untimed) before every step; CUDA events on the launch stream"""
        out = torch.empty(n, dtype=torch.float64, device="cuda")
        for _ in range(warmup):                 # warm-up through the same entry as the timed steps (first-call allocations are not steady state)
            if host is None:
                ctx.me_compute(mom, n, prec, out=out)
            else:
                ctx.me_compute_host(host, n, prec, stream=stream)
        barrier()
        per = []
        for _ in range(steps):
            flush.zero_()
            e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            if host is None:
                ctx.me_compute(mom, n, prec, out=out, stream=stream)
            else:
                ctx.me_compute_host(host, n, prec, stream=stream)
            e1.record(stream)
            e1.synchronize()
            per.append(e0.elapsed_time(e1))
        barrier()
        return sum(per), per

    def allmax(x):
        if dist is None:
            return x
        t = torch.tensor([x], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    # ------------------------------------------------------------------ headline: g g -> t t~ g g
    ctx, mom = setup(HL, n, first)
    info = ctx.info
    ngood = bin(ctx.me_filter_helicities(mom, 32)[0]).count("1")
    flops_alg = info.flops_per_helicity[0] * ngood + info.flops_per_event_fixed[0]
    flops_exe = info.flops_executed_per_helicity[0] * ngood + info.flops_per_event_fixed[0]
    results = {}
    with ClockSampler(local) as clk:
        total_ms, per = timed(ctx, mom, n, me.ME_FP64, args.steps, args.warmup)
    clocks = clk.summary()
    total_ms = allmax(total_ms)
    value = per_gpu * world * args.steps / (total_ms * 1e-3)
    ms_kernel = statistics.mean(per)
    per_step_launches = info.nkernels * ((ngood + 31) // 32 if HL == 4 else 1)    # cfg 5: 3 diagram kernels + colour sum per 32-helicity chunk (ME_HEL_CHUNK)
    launches = args.steps * per_step_launches
    results[cfg["name"]] = {"fp64": {"MEs_per_s": n * args.steps / (sum(per) * 1e-3), "ms_per_step": ms_kernel}}
    # measured FMA-chain peaks (register-resident microkernel, same box, same run)
    peak_meas = {"fp64": me.me_fma_peak(1), "fp32": me.me_fma_peak(0)}
    ach = flops_alg * n / (ms_kernel * 1e-3) * 1e-12
    roofline = {"bound": "alu", "kernel": "k_%s<double,double,TM=true>" % cfg["name"] + (" (+ colour sum)" if HL == 4 else ""), "achieved": ach, "peak": PEAK_TFLOPS["fp64"], "unit": "TFLOP/s",
                "frac": ach / PEAK_TFLOPS["fp64"],
                # dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of this kernel at the full config, from the committed
                # ncu --set full capture (profiles/r1_ttxgg_fp64_tmem.md: 101.6 MB read + 5.5 MB written); algorithmic bytes = 200 B/event = 104.9 MB
                "traffic": 107.1e6 if (HL == 3 and n == 524288) else None,
                "traffic_source": "profiles/r1_ttxgg_fp64_tmem.md" if (HL == 3 and n == 524288) else None,
                "peak_source": "derived: 148 SM x 64 FP64 FMA/clk x 2 x 1.965 GHz (B200_PROFILING.md clocks; no FP64 entry in MEASURED_PEAKS.json)",
                "peak_measured_fma_chain": peak_meas["fp64"], "frac_of_measured": ach / peak_meas["fp64"],
                "flops_per_event_algorithmic": flops_alg, "flops_per_event_executed": flops_exe,
                "achieved_executed": flops_exe * n / (ms_kernel * 1e-3) * 1e-12}
    # other precisions of the headline workload
    for pname in [q for q in ("mixed", "fp32") if q in cfg["precisions"]]:
        t, pp = timed(ctx, mom, n, me.PRECISIONS[pname], args.steps, args.warmup)
        launches += args.steps * per_step_launches
        ms = statistics.mean(pp)
        results[cfg["name"]][pname] = {"MEs_per_s": n / (ms * 1e-3), "ms_per_step": ms}
    a32 = flops_alg * n / (results[cfg["name"]]["fp32"]["ms_per_step"] * 1e-3) * 1e-12
    roofline["fp32"] = {"achieved": a32, "peak": PEAK_TFLOPS["fp32"], "frac": a32 / PEAK_TFLOPS["fp32"],
                        "peak_measured_fma_chain": peak_meas["fp32"], "frac_of_measured": a32 / peak_meas["fp32"]}
    # optional exact symmetry (include/me.h ME_OPT_PARITY_PAIRING): half the helicities, same number; NOT the headline
    ctx.me_set_option(me.ME_OPT_PARITY_PAIRING, 1)
    t, pp = timed(ctx, mom, n, me.ME_FP64, args.steps, args.warmup)
    ctx.me_set_option(me.ME_OPT_PARITY_PAIRING, 0)
    launches += args.steps * info.nkernels * ((ngood // 2 + 31) // 32 if HL == 4 else 1)
    results[cfg["name"]]["fp64_parity_pairing"] = {"MEs_per_s": n / (statistics.mean(pp) * 1e-3), "ms_per_step": statistics.mean(pp)}
    if args.sweep and world == 1:
        sweep = {"batch": {}, "streams": {}}
        nb = 8192
        while nb <= n:
            t, pp = timed(ctx, mom, nb, me.ME_FP64, 5, 2)
            sweep["batch"][str(nb)] = nb / (min(pp) * 1e-3)
            nb *= 2
        # several streams sharing the GPU, each computing its own slice of the batch (the paper shares a V100 between processes)
        for ns in (1, 2, 4, 8):
            for nb in (8192, 32768):
                if ns * nb > n:
                    continue
                streams = [torch.cuda.Stream() for _ in range(ns)]
                ppages = ctx.momenta_numel(nb)
                outs = [torch.empty(nb, dtype=torch.float64, device="cuda") for _ in range(ns)]
                torch.cuda.synchronize()
                best = 1e30
                for rep in range(4):
                    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                    e0.record()
                    for k, st in enumerate(streams):
                        st.wait_event(e0)
                        ctx.me_compute(mom[k * ppages:(k + 1) * ppages], nb, me.ME_FP64, out=outs[k], stream=st)
                    for st in streams:
                        torch.cuda.current_stream().wait_stream(st)
                    e1.record(); e1.synchronize()
                    best = min(best, e0.elapsed_time(e1))
                sweep["streams"]["%dx%d" % (ns, nb)] = ns * nb / (best * 1e-3)
        results["sweep_fp64_MEs_per_s"] = sweep
        # helicity / leading-colour selection: per-helicity pass + per-event-helicity jamp pass, all in lockstep
        ns = min(n, 131072)
        ctx.me_select_helicity_color(mom, ns, seed=1)
        torch.cuda.synchronize(); t0 = time.perf_counter()
        ctx.me_select_helicity_color(mom, ns, seed=1)
        torch.cuda.synchronize()
        results["select_helicity_color_events_per_s"] = ns / (time.perf_counter() - t0)
    # ------------------------------------------------------------------ end to end: HOST buffers through the public call
    host = mom.cpu().pin_memory()
    e2e_ms, _ = timed(ctx, mom, n, me.ME_FP64, args.steps, 3, host=host)
    e2e_ms = allmax(e2e_ms)
    e2e = {"value": per_gpu * world * args.steps / (e2e_ms * 1e-3), "unit": "MEs/s", "h2d_bytes_per_step": host.numel() * 8,
           "d2h_bytes_per_step": n * 8, "api": "C-ABI me_compute_host (pinned host momenta -> sliced H2D overlapped with the kernels -> pinned host MEs)"}
    # me_compute_host cuts the batch in slices of 6 x 128 events per SM, one me_compute (per_step_launches kernels) each
    host_slice = 6 * 128 * torch.cuda.get_device_properties(local).multi_processor_count
    launches += args.steps * per_step_launches * ((n + host_slice - 1) // host_slice)
    line = {
        "metric": "matrix elements/sec (%s, FP64)" % cfg["label"], "value": value, "unit": "MEs/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "%s, %d RAMBO events per GPU, sqrt(s)=1500 GeV, Philox seed %d, %d good helicities" % (cfg["label"], per_gpu, cfg["seed"], ngood),
                   "events_per_gpu": per_gpu, "l2": "flushed between timed steps (256 MiB memset, untimed)", "parallelism": "events sharded, no collective"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline,
        "paper_context": {"hardware": "1x V100, CUDA 11.7 (PAPER.md Table 1/3)", "MEs_per_s": PAPER_V100},
    }
    # ------------------------------------------------------------------ the oracle timed beside it (rank 0, N = 1)
    if rank == 0 and world == 1 and not args.quick:
        nb = n
        p = inputs.aosoa_to_aos(mom[: ctx.momenta_numel(nb)].cpu().numpy(), nb, cfg["npar"], info.page)
        rate, cores, ns, dt = oracle_rate(cfg["process"], p)
        line["cpu_baseline"] = {"value": rate, "unit": "MEs/s", "cores": cores, "kind": "oracle",
                                "sample": "first %d of the %d events (%.1f s of CPU work)" % (ns, per_gpu, dt)}
    ctx.close(); del mom, host
    # ------------------------------------------------------------------ the other processes (context numbers; not the headline)
    if world == 1 and not args.quick:
        for proc in [q for q in (1, 2, 3, 4) if q != HL]:
            c = inputs.CONFIGS[proc]
            cx, mm = setup(proc, c["events"], 0)
            ng = bin(cx.me_filter_helicities(mm, 32)[0]).count("1")
            fl = cx.info.flops_per_helicity[0] * ng + cx.info.flops_per_event_fixed[0]
            results[c["name"]] = {}
            reps = 2 if proc == 4 else 5
            for pname in c["precisions"]:
                t, pp = timed(cx, mm, c["events"], me.PRECISIONS[pname], reps, 1)
                ms = statistics.mean(pp)
                pk = "fp32" if pname == "fp32" else "fp64"
                results[c["name"]][pname] = {"MEs_per_s": c["events"] / (ms * 1e-3), "ms_per_step": ms,
                                             "frac_of_%s_peak" % pk: fl * c["events"] / (ms * 1e-3) * 1e-12 / PEAK_TFLOPS[pk]}
            cx.close(); del mm
    line["results"] = results
    if rank == 0:
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
