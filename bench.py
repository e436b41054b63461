#!/usr/bin/env python
"""bench.py — throughput of the matrix-element hot path (BASELINE.json metric: matrix elements/sec on one
B200 for g g -> t t~ g g, FP64 headline, mixed and FP32 beside it, and the fraction of the FP roofline).

One "step" = one me_compute pass (external wavefunctions, currents, diagram
amplitudes, jamps, colour sum, helicity sum) over one batch of seeded synthetic RAMBO events.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--quick]

N > 1: one rank per GPU, every rank takes its own page-aligned shard of N x 524288 events (weak scaling, no data-path
collective).  Launched by torch.distributed.run (RANK / WORLD_SIZE in the environment) it is one of the ranks;
started plainly as `python bench.py --gpus N` it re-executes itself under torch.distributed.run with N ranks on 127.0.0.1.
`--impl reference` times the CPU oracle (oracle/) on the host cores on a bounded sample of the same workload.

Numbers that come from a profile rather than from this run (DRAM traffic per launch, executed-flop counts by opcode) are read
from the committed table profiles/r2_kernel_metrics.csv (written from ncu captures; the commands are in the .md beside it),
keyed by kernel, workload and batch size, and are labelled with that source in the JSON line.
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


def profile_metrics():
    """rows of profiles/r2_kernel_metrics.csv: {(process name, precision, option, events): {column: float}}"""
    import csv
    path = os.path.join(ROOT, "profiles", "r2_kernel_metrics.csv")
    out = {}
    if os.path.exists(path):
        with open(path) as f:
            for row in csv.DictReader(l for l in f if not l.startswith("#")):
                key = (row["process"], row["precision"], row["option"], int(row["events"]))
                out[key] = {k: float(v) for k, v in row.items() if k not in ("process", "precision", "option", "events", "kernel", "source") and v != ""}
                out[key]["source"] = row["source"]; out[key]["kernel"] = row["kernel"]
    return out


def ncu_flops_per_event(m):
    """executed ALU flops per event from the ncu opcode counts of one launch: add + mul + 2 fma (thread-level, predicated-on), both
    precisions added (the FP32 kernels form their propagator denominators in FP64).  The tensor-core flops of the colour-sum
    kernels (instruction count x instruction shape) are another unit with another peak: reported beside, never added in."""
    return (m.get("dadd", 0) + m.get("dmul", 0) + 2 * m.get("dfma", 0) + m.get("fadd", 0) + m.get("fmul", 0) + 2 * m.get("ffma", 0)) / m["events_per_launch"]


def ncu_fields(m, n, ms, peak):
    """the keys a result row takes from its row of profiles/r2_kernel_metrics.csv"""
    fe = ncu_flops_per_event(m)
    return {"flops_per_event_ncu": fe, "frac_ncu": fe * n / (ms * 1e-3) * 1e-12 / peak,
            "tensor_flops_per_event_ncu": m.get("tensor_flops", 0) / m["events_per_launch"],
            "traffic": m.get("dram_bytes"), "traffic_algorithmic": m.get("algorithmic_bytes"), "profile_source": m["source"]}


def respawn_under_torchrun(args):
    """`python bench.py --gpus N` without a torchrun environment: start N ranks on this node (127.0.0.1) and return their exit code"""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0)); port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus), "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


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
    ap.add_argument("--no-sweep", action="store_true", help="skip the short batch-size / shared-GPU sweep of the default run")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return respawn_under_torchrun(args)
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
    # algorithmic flops per event of the DEFAULT path: with current sharing (on by default where a sharing kernel exists, include/me.h
    # ME_OPT_SHARE_CURRENTS) every current is counted once per distinct helicity assignment of its own legs (SURVEY.md line 493:
    # "re-count algorithmic flops when enabled"); flops_unshared is the count with every current once per helicity
    flops_unshared = info.flops_per_helicity[0] * ngood + info.flops_per_event_fixed[0]
    shared_default = info.flops_per_event_shared > 0 and ngood == info.ncomb
    flops_alg = info.flops_per_event_shared if shared_default else flops_unshared
    flops_exe = info.flops_executed_per_event_shared if shared_default else info.flops_executed_per_helicity[0] * ngood + info.flops_per_event_fixed[0]
    results = {}
    prof = profile_metrics()
    with ClockSampler(local) as clk:
        total_ms, per = timed(ctx, mom, n, me.ME_FP64, args.steps, args.warmup)
    clocks = clk.summary()
    total_ms = allmax(total_ms)
    value = per_gpu * world * args.steps / (total_ms * 1e-3)
    ms_kernel = statistics.mean(per)
    per_step_launches = me.launches_per_pass(info, ngood)
    launches = args.steps * per_step_launches
    results[cfg["name"]] = {"fp64": {"MEs_per_s": n * args.steps / (sum(per) * 1e-3), "ms_per_step": ms_kernel}}
    # measured FMA-chain peaks (register-resident microkernel, same box, same run)
    peak_meas = {"fp64": me.me_fma_peak(1), "fp32": me.me_fma_peak(0)}

    def roof(pname, ms, flops_per_event, option="-"):
        """roofline numbers of one timed variant: algorithmic flops / CUDA-event time against the derived and the measured FMA peak;
        where the committed ncu table has this (process, precision, option, n), also the executed flops by opcode and the DRAM traffic"""
        pk = "fp32" if pname == "fp32" else "fp64"
        ach = flops_per_event * n / (ms * 1e-3) * 1e-12
        r = {"achieved": ach, "peak": PEAK_TFLOPS[pk], "frac": ach / PEAK_TFLOPS[pk], "peak_measured_fma_chain": peak_meas[pk],
             "frac_of_measured": ach / peak_meas[pk], "flops_per_event_algorithmic": flops_per_event}
        m = prof.get((cfg["name"], pname, option, n))
        if m is not None:
            r.update(ncu_fields(m, n, ms, PEAK_TFLOPS[pk])); r["kernel"] = m["kernel"]
        return r

    roofline = {"bound": "alu", "unit": "TFLOP/s", "kernel": "k_%s<double,double,TM=true,SH=%s>" % (cfg["name"], "true" if shared_default else "false") + (" (+ colour sum)" if HL == 4 else ""),
                "flops_per_event_unshared_algorithm": flops_unshared,
                "frac_counting_unshared_algorithm": flops_unshared * n / (ms_kernel * 1e-3) * 1e-12 / PEAK_TFLOPS["fp64"],
                "traffic": None, "traffic_source": None,
                "peak_source": "derived: 148 SM x 64 FP64 FMA/clk x 2 x 1.965 GHz (B200_PROFILING.md clocks; no FP64 entry in MEASURED_PEAKS.json)",
                "flops_per_event_executed": flops_exe, "achieved_executed": flops_exe * n / (ms_kernel * 1e-3) * 1e-12,
                "frac_executed": flops_exe * n / (ms_kernel * 1e-3) * 1e-12 / PEAK_TFLOPS["fp64"]}
    roofline.update(roof("fp64", ms_kernel, flops_alg, option="shared_currents" if shared_default else "-"))
    if "profile_source" in roofline:        # dram__bytes_read.sum + dram__bytes_write.sum of ONE launch at this batch size, from the committed ncu capture
        roofline["traffic_source"] = roofline["profile_source"]
    # other precisions of the headline workload
    for pname in [q for q in ("mixed", "fp32") if q in cfg["precisions"]]:
        t, pp = timed(ctx, mom, n, me.PRECISIONS[pname], args.steps, args.warmup)
        launches += args.steps * per_step_launches
        ms = statistics.mean(pp)
        results[cfg["name"]][pname] = {"MEs_per_s": n / (ms * 1e-3), "ms_per_step": ms}
        roofline[pname] = roof(pname, ms, flops_alg, option="shared_currents" if shared_default else "-")
    # options of include/me.h that reduce the work exactly; reported beside the headline, NEVER as the headline
    #   ME_OPT_PARITY_PAIRING: half the helicities, each counted twice;
    #   ME_OPT_SHARE_CURRENTS: sub-tree currents re-evaluated only when their own helicities change (own algorithmic flop count)
    def timed_option(key, opts, pname, flops_per_event, nhel_pass):
        nonlocal launches
        defaults = {me.ME_OPT_PARITY_PAIRING: 0, me.ME_OPT_SHARE_CURRENTS: 1}
        for o, v in opts.items():
            ctx.me_set_option(o, v)
        t, pp = timed(ctx, mom, n, me.PRECISIONS[pname], args.steps, args.warmup)
        for o in opts:
            ctx.me_set_option(o, defaults[o])
        launches += args.steps * me.launches_per_pass(info, nhel_pass)
        ms = statistics.mean(pp)
        results[cfg["name"]][key] = {"MEs_per_s": n / (ms * 1e-3), "ms_per_step": ms}
        if flops_per_event:
            results[cfg["name"]][key]["roofline"] = roof(pname, ms, flops_per_event, option="-")
    timed_option("fp64_parity_pairing", {me.ME_OPT_PARITY_PAIRING: 1}, "fp64", None, ngood // 2)
    if shared_default:          # the same workload with current sharing switched off: every current once per helicity
        for pname in cfg["precisions"]:
            timed_option("%s_unshared" % pname, {me.ME_OPT_SHARE_CURRENTS: 0}, pname, flops_unshared, ngood)
    if world == 1 and not args.sweep and not args.no_sweep and HL == 3:
        # short form of --sweep in every default run (Fig. 1): throughput against batch
        # size, and 1 / 2 / 4 / 8 producers sharing the GPU, each with its own context and stream and a batch of 8192 events
        sw = {"batch": {}, "streams_x_8192": {}}
        nsm = torch.cuda.get_device_properties(local).multi_processor_count
        nb = 8192
        while nb <= n:
            t, pp = timed(ctx, mom, nb, me.ME_FP64, 3, 1)
            launches += 4 * me.launches_per_pass(info, ngood, nb, nsm)
            sw["batch"][str(nb)] = nb / (min(pp) * 1e-3)
            nb *= 4
        ctxs = [ctx] + [me.MEContext(HL) for _ in range(7)]
        for c in ctxs[1:]:
            c.me_set_helicities(ctx.me_filter_helicities(mom, 32)[0])
        words = ctx.momenta_numel(8192)
        outs = [torch.empty(8192, dtype=torch.float64, device="cuda") for _ in range(8)]
        sts = [torch.cuda.Stream() for _ in range(8)]
        for ns in (1, 2, 4, 8):
            best = 1e30
            for rep in range(4):
                torch.cuda.synchronize()
                e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                e0.record()
                for k in range(ns):
                    sts[k].wait_event(e0)
                    ctxs[k].me_compute(mom[k * words:(k + 1) * words], 8192, me.ME_FP64, out=outs[k], stream=sts[k])
                for k in range(ns):
                    torch.cuda.current_stream().wait_stream(sts[k])
                e1.record(); e1.synchronize()
                best = min(best, e0.elapsed_time(e1))
                launches += ns * me.launches_per_pass(info, ngood, 8192, nsm)
            sw["streams_x_8192"][str(ns)] = ns * 8192 / (best * 1e-3)
        for c in ctxs[1:]:
            c.close()
        results["sweep_fp64_MEs_per_s"] = sw
    if args.sweep and world == 1:
        sweep = {"batch": {}, "streams": {}}
        sweep_ctxs = [ctx]
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
                while len(sweep_ctxs) < ns:            # one context per producer: calls on ONE context are ordered on the device (include/me.h)
                    sweep_ctxs.append(me.MEContext(HL)); sweep_ctxs[-1].me_set_helicities(ctx.me_filter_helicities(mom, 32)[0])
                ppages = ctx.momenta_numel(nb)
                outs = [torch.empty(nb, dtype=torch.float64, device="cuda") for _ in range(ns)]
                torch.cuda.synchronize()
                best = 1e30
                for rep in range(4):
                    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                    e0.record()
                    for k, st in enumerate(streams):
                        st.wait_event(e0)
                        sweep_ctxs[k].me_compute(mom[k * ppages:(k + 1) * ppages], nb, me.ME_FP64, out=outs[k], stream=st)
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
    launches += (args.steps + 3) * per_step_launches * ((n + host_slice - 1) // host_slice)
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
            fl_un = cx.info.flops_per_helicity[0] * ng + cx.info.flops_per_event_fixed[0]
            sh = cx.info.flops_per_event_shared > 0 and ng == cx.info.ncomb          # default path shares currents: its own algorithmic count
            fl = cx.info.flops_per_event_shared if sh else fl_un
            fx = cx.info.flops_executed_per_event_shared if sh else cx.info.flops_executed_per_helicity[0] * ng + cx.info.flops_per_event_fixed[0]
            results[c["name"]] = {}
            reps = 2 if proc == 4 else 5
            for pname in c["precisions"]:
                t, pp = timed(cx, mm, c["events"], me.PRECISIONS[pname], reps, 1)
                ms = statistics.mean(pp)
                pk = "fp32" if pname == "fp32" else "fp64"
                results[c["name"]][pname] = {"MEs_per_s": c["events"] / (ms * 1e-3), "ms_per_step": ms,
                                             "flops_per_event_algorithmic": fl, "flops_per_event_executed": fx, "flops_per_event_unshared_algorithm": fl_un,
                                             "frac_counting_unshared_algorithm": fl_un * c["events"] / (ms * 1e-3) * 1e-12 / PEAK_TFLOPS[pk],
                                             "frac_of_%s_peak" % pk: fl * c["events"] / (ms * 1e-3) * 1e-12 / PEAK_TFLOPS[pk],
                                             "frac_of_%s_peak_executed" % pk: fx * c["events"] / (ms * 1e-3) * 1e-12 / PEAK_TFLOPS[pk]}
                m = prof.get((c["name"], pname, "shared_currents" if sh else "-", c["events"]))
                if m is not None:
                    results[c["name"]][pname].update(ncu_fields(m, c["events"], ms, PEAK_TFLOPS[pk]))
                launches += (reps + 1) * me.launches_per_pass(cx.info, ng)
            cx.close(); del mm
    line["results"] = results
    if rank == 0:
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    sys.exit(main() or 0)
