#!/usr/bin/env python
"""bench.py — throughput of the batched harmonic sum (arXiv 1812.02647 eqs. 1-4) on B200, one JSON line.

A "step" is one pass of the whole hot path over one batch of synthetic spectra: hs_execute of each of the four
variants (standard, Max, freq-bin, Greedy) at Hmax = 32 in the workload's output mode.  The default workload is
BASELINE.json configs[2] (4096 spectra x 2^18 bins, Exp(1)-1 noise + 1 % injected combs, reduced output), the
configuration the metric is quoted on.  `value` = bins/s, one bin = one output bin of one variant, i.e.
variants x batch x nbins / step time, inputs resident in HBM; `e2e` = the same through hs_execute_host with pinned
host buffers (host<->device copies inside the timed region).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]
                    [--workload config2|config1|config3|allh|plane|complex]
                    [--batch B] [--variants standard,max,freqbin,greedy] [--algo auto|direct|tiled] [--no-e2e]

N > 1: one rank per GPU, every rank runs the same batch shape on its own seeded data (weak scaling, spectra are
independent: no data-path collective); time = max over ranks.  Launched under torchrun by the driver; started plainly
with --gpus N > 1 it re-launches itself under torch.distributed.run with N ranks (and fails if the box has fewer GPUs).
`--impl reference` times the CPU oracle (oracle/hs_oracle.c) on a bounded sample of the same workload on rank 0.
The non-headline workloads time the rows of SURVEY.md section 8(f): allh = every integer H up to 64 (hs_plan_create_ex),
plane = the 2-D sum over an f-fdot plane (hs_plan_create_2d), complex = the fused power-spectrum front end
(hs_execute_complex); each against its own algorithmic bytes.
"""
from __future__ import annotations

import argparse
import concurrent.futures
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

VARIANTS = ["standard", "max", "freqbin", "greedy"]
WORKLOADS = {
    # name: (batch, nbins, out_mode, description)
    "config2": (4096, 1 << 18, "reduced", "configs[2]: 4096 x 2^18 Exp(1)-1 noise, 1% combs, reduced output"),
    "config1": (256, 1 << 18, "both", "configs[1] shape: 256 x 2^18, full and reduced output (Exp(1)-1 stand-in noise)"),
    "config3": (8, 1 << 23, "full", "configs[3]: 8 x 2^23 Exp(1)-1 noise, one comb each, full output"),
    # SURVEY.md section 8(f) rows (not the headline): Exp(1)-1 noise
    "allh": (256, 1 << 18, "reduced", "8(f)-3: 256 x 2^18, every integer H = 1..64, reduced output"),
    "plane": (8, 1 << 18, "reduced", "8(f)-4: 8 f-fdot planes of 129 drifts x 2^18 bins, 2-D sum, Hmax 32, reduced output"),
    "complex": (1024, 1 << 18, "reduced", "8(f)-1: 1024 x 2^18 complex Fourier series -> |F|^2 -> harmonic sum, Hmax 32, reduced output"),
}
PLANE_ROWS = 129
BYTES_PER_BIN = {"reduced": 4 + 5, "full": 4 + 4 * 6, "both": 4 + 4 * 6 + 5}   # SURVEY.md section 8(d), Hmax = 32
PAPER_GPU_OVER_CPU = {"standard": 250, "greedy": 704, "freqbin": 110, "max": 177}   # PAPER.md:66-71, Table 1 (hardware not stated)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="config2", choices=sorted(WORKLOADS))
    ap.add_argument("--batch", type=int, default=0, help="override the batch (non-headline; recorded in config)")
    ap.add_argument("--variants", default=",".join(VARIANTS))
    ap.add_argument("--algo", default="auto", choices=["auto", "direct", "tiled", "twophase", "gather", "grouped"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="budget of the cpu_baseline leg")
    ap.add_argument("--candidates-threshold", type=float, default=25.0,
                    help="also time hs_execute_candidates at this threshold (0: skip); reported under \"candidates\"")
    ap.add_argument("--sweep", default="", choices=["", "scaling"],
                    help="scaling: configs[4] throughput sweep over Hmax and spectrum length (one JSON line per point)")
    ap.add_argument("--sweep-gib", type=float, default=16.0, help="fp32 input per sweep point (configs[4]: 16 GiB)")
    return ap.parse_args()


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(variant, workload, algo):
    """DRAM bytes per launch from the committed ncu capture (profiles/ncu_traffic.json), or None."""
    try:
        return json.load(open(os.path.join(ROOT, "profiles", "ncu_traffic.json")))[f"{workload}/{variant}/{algo}"]
    except Exception:
        return None


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
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
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            f = [t.strip() for t in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                smax.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(names, f[3:7]):
                if v == "Active":
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_per_variant(x_rows, variants, threads, gpu_bins_per_s):
    """the oracle's bins/s per variant on 1 thread (one spectrum) and spectra-parallel on all host
    threads (the paper's CPU strategy), beside the paper's Table 1 ratios."""
    import oracle
    oracle.build()
    R, N = x_rows.shape
    out = {}
    for v in variants:
        t0 = time.perf_counter()
        oracle.harmonic_sum(x_rows[0], 32, v, want_sums=False, want_reduced=True)
        one = N / (time.perf_counter() - t0)
        rows = min(R, threads)
        t0 = time.perf_counter()
        with concurrent.futures.ThreadPoolExecutor(max_workers=threads) as ex:
            list(ex.map(lambda r: oracle.harmonic_sum(x_rows[r], 32, v, want_sums=False, want_reduced=True), range(rows)))
        allc = rows * N / (time.perf_counter() - t0)
        out[v] = {"bins_per_s_1_thread": one, "bins_per_s_all_threads": allc, "spectra_timed": rows,
                  "gpu_over_cpu_all_threads": (gpu_bins_per_s[v] / allc) if v in gpu_bins_per_s else None,
                  "paper_gpu_over_cpu": PAPER_GPU_OVER_CPU.get(v)}
    return out


def oracle_rate(x_rows, variants, seconds, threads):
    """Oracle throughput (bins/s, one bin = one output bin of one variant) on whole spectra of x_rows [R][N],
    spectra-parallel over `threads` host threads (the paper's CPU strategy; ctypes releases the GIL)."""
    import oracle
    oracle.build()
    R, N = x_rows.shape
    jobs = [(r, v) for r in range(R) for v in variants]
    t0 = time.perf_counter()
    done = 0

    def work(job):
        r, v = job
        oracle.harmonic_sum(x_rows[r], 32, v, want_sums=False, want_reduced=True)
        return N

    with concurrent.futures.ThreadPoolExecutor(max_workers=threads) as ex:
        futs = []
        for job in jobs:
            futs.append(ex.submit(work, job))
        for f in futs:
            done += f.result()
            if time.perf_counter() - t0 > seconds * 4:
                break
    dt = time.perf_counter() - t0
    return done / dt, dt, done


def oracle_rate_ext(wl, x, variants, seconds, threads, scale, gpu_bins_per_s):
    """cpu_baseline of the SURVEY.md section 8(f) workloads: the extension oracle as it stands (oracle/hs_oracle_ext.c; for
    `complex` its power spectrum followed by oracle/hs_oracle.c), one variant after the other, each for its share of
    `seconds`, tasks spread over `threads` host threads (ctypes releases the GIL).  A task is
        allh     512 consecutive bins at a seeded random place in one of the first 4 spectra, all 64 levels (hsx_points_all:
                 a whole 2^18-bin spectrum of eq. 2 is minutes of work, every level being summed from scratch);
        plane    one whole f-fdot plane, reduced output (hsx_harmonic_sum_2d);
        complex  one whole spectrum: hsx_power_spectrum, then hso_harmonic_sum at Hmax 32, reduced output.
    Returns (bins/s over all variants, per-variant dict, threads actually used, description of the sample, seconds)."""
    import threading

    import numpy as np

    import oracle
    from oracle import ext
    oracle.build()
    ext.build()
    per, total_bins, total_dt, used = {}, 0, 0.0, 1
    for v in variants:
        budget = seconds / len(variants)
        if wl == "allh":
            rows, chunk = x[:4].cpu().numpy(), 512
            rng = np.random.default_rng(1)
            places = [(int(rng.integers(0, rows.shape[0])), int(rng.integers(0, rows.shape[1] - chunk))) for _ in range(1 << 16)]
            sample = f"runs of {chunk} consecutive bins at seeded random places in the first {rows.shape[0]} spectra, 64 levels each"

            def run(job, v=v, rows=rows, chunk=chunk):
                ext.points_all(rows, 64, v, np.full(chunk, job[0]), np.arange(job[1], job[1] + chunk))
                return chunk
        elif wl == "plane":
            planes = x[:min(x.shape[0], threads)].cpu().numpy()
            places = list(range(planes.shape[0]))
            sample = f"the first {planes.shape[0]} whole planes of {planes.shape[1]} x {planes.shape[2]} bins"

            def run(job, v=v, planes=planes):
                ext.harmonic_sum_2d(planes[job], 32, v, want_sums=False)
                return planes[job].size
        else:
            F = x[:min(x.shape[0], 256)].cpu().numpy()
            places = list(range(F.shape[0]))
            sample = f"up to {F.shape[0]} whole spectra of {F.shape[1]} bins: power spectrum, then the harmonic sum"

            def run(job, v=v, F=F):
                oracle.harmonic_sum(ext.power_spectrum(F[job], scale), 32, v, want_sums=False, want_reduced=True)
                return F.shape[1]
        it, lock, done = iter(places), threading.Lock(), []
        t0 = time.perf_counter()

        def worker():
            n = 0
            while time.perf_counter() - t0 < budget:
                with lock:
                    job = next(it, None)
                if job is None:
                    break
                n += run(job)
            done.append(n)

        nthreads = min(threads, len(places))
        pool = [threading.Thread(target=worker) for _ in range(nthreads)]
        for t in pool:
            t.start()
        for t in pool:
            t.join()
        dt = time.perf_counter() - t0
        bins = sum(done)
        used = max(used, nthreads)
        per[v] = {"bins_per_s_all_threads": bins / dt, "bins_timed": bins, "seconds": dt, "threads": nthreads,
                  "gpu_over_cpu_all_threads": (gpu_bins_per_s[v] / (bins / dt)) if v in gpu_bins_per_s and bins else None}
        total_bins += bins
        total_dt += dt
    return total_bins / total_dt, per, used, sample, total_dt


def cpu_sample_rows(seconds, threads, nbins, variants, cap=64):
    # ~0.7 s of single-thread work per 2^18-bin spectrum for the four variants together
    per_spectrum = 0.7 * (nbins / float(1 << 18)) * len(variants) / 4.0
    return max(1, min(cap, int(seconds * threads / per_spectrum)))


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores, on a bounded sample of the workload per step."""
    import numpy as np
    import workloads as W
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    batch, nbins, out_mode, desc = WORKLOADS[args.workload]
    variants = args.variants.split(",")
    threads = os.cpu_count() or 1
    total_steps = max(1, args.steps + args.warmup)
    rows = cpu_sample_rows(max(2.0, 120.0 / total_steps), threads, nbins, variants)
    cfg = {"config2": 2, "config1": 2, "config3": 3}[args.workload]
    x, _ = W.comb_batch_numpy(cfg, list(range(rows)), nbins, 0.01 if cfg == 2 else 1.0,
                              50.0 if cfg == 2 else 1000.0, 5000.0 if cfg == 2 else 100000.0, 0.10 if cfg == 2 else 0.03)
    for _ in range(args.warmup):
        oracle_rate(x[:max(1, rows // 4)], variants, 1e9, threads)
    t0 = time.perf_counter()
    bins = 0
    for _ in range(args.steps):
        _, _, done = oracle_rate(x, variants, 1e9, threads)
        bins += done
    dt = time.perf_counter() - t0
    value = bins / dt
    sample = f"{rows} whole spectra of {nbins} bins x {len(variants)} variants per step (of {batch} in the workload)"
    line = {"impl": "reference", "metric": "harmonic_sum_bins_per_s", "value": value, "unit": "bins/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": desc, "batch": batch, "nbins": nbins, "Hmax": 32, "out_mode": out_mode,
                       "variants": variants, "note": "CPU oracle on a bounded sample per step"},
            "cpu_baseline": {"value": value, "unit": "bins/s", "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": "bins/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_scaling(args):
    """--sweep scaling: BASELINE.json configs[4], scaling part.  Exp(1)-1 noise, nbins = 2^16 .. 2^24, batch sized to
    --sweep-gib of fp32 input, Hmax = 2 .. 32, reduced output; per point and variant the median CUDA-event time of 5
    launches after 3 warm-ups.  One JSON line per point (not the driver's contract line)."""
    import torch

    import workloads as W
    from paper_1812_02647_b200 import binding as hs
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    peak, _ = measured_peak()
    variants = args.variants.split(",")
    words = int(args.sweep_gib * (1 << 30)) // 4
    x_all = W.exp_noise_torch(1, words, 4, dev).view(-1)
    vmax_all = torch.empty(words, dtype=torch.float32, device=dev)
    amax_all = torch.empty(words, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    for lg in range(16, 25):
        nbins = 1 << lg
        batch = max(1, words // nbins)
        x, vmax, amax = (t[:batch * nbins].view(batch, nbins) for t in (x_all, vmax_all, amax_all))
        for Hmax in (2, 4, 8, 16, 32):
            point = {"sweep": "scaling", "nbins": nbins, "batch": batch, "Hmax": Hmax, "out_mode": "reduced",
                     "input_GiB": batch * nbins * 4 / 2**30, "per_variant": {}}
            for v in variants:
                p = hs.hs_plan_create(nbins, batch, Hmax, v, "reduced")
                p.ensure_workspace(dev)
                ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(5)]
                for _ in range(3):
                    p.hs_execute(x, None, vmax, amax, stream)
                for e0, e1 in ev:
                    e0.record(stream)
                    p.hs_execute(x, None, vmax, amax, stream)
                    e1.record(stream)
                torch.cuda.synchronize()
                ms = statistics.median(e0.elapsed_time(e1) for e0, e1 in ev)
                gbs = 9.0 * batch * nbins / (ms * 1e-3) / 1e9
                point["per_variant"][v] = {"ms": ms, "bins_per_s": batch * nbins / (ms * 1e-3), "eff_GBps": gbs,
                                           "frac_of_measured_peak": gbs / peak, "launches": p.launches(),
                                           "workspace_MiB": round(p.workspace_bytes() / 2**20)}
                p.hs_destroy()
                del p
            print(json.dumps(point), flush=True)


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    if args.sweep == "scaling":
        return run_scaling(args)

    import numpy as np
    import torch
    import torch.distributed as dist

    import workloads as W
    from paper_1812_02647_b200 import binding as hs
    from paper_1812_02647_b200.shard import max_over_ranks_ms, sum_over_ranks

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # started plainly: one rank per GPU under torch.distributed.run, or a clean failure (never an n_gpus: 1 line)
        have = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if have < args.gpus:
            print(json.dumps({"error": f"--gpus {args.gpus} asked for, {have} CUDA device(s) visible", "n_gpus": have}), flush=True)
            sys.exit(2)
        port = 29500 + (os.getpid() % 2000)
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        sys.exit(subprocess.call(cmd))
    if args.gpus != world:
        print(json.dumps({"error": f"--gpus {args.gpus} but WORLD_SIZE is {world}"}), flush=True)
        sys.exit(2)
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = torch.device("cuda", local_rank)

    batch, nbins, out_mode, desc = WORKLOADS[args.workload]
    if args.batch:
        batch = args.batch
    variants = args.variants.split(",")
    headline_workload = args.workload in ("config2", "config1", "config3")
    wl = args.workload
    if wl == "plane":
        variants = [v for v in variants if v in ("standard", "freqbin")]      # the 2-D sum is defined for eqs. 1 and 3
    Hmax = 64 if wl == "allh" else 32
    L = 64 if wl == "allh" else 6
    rows = PLANE_ROWS if wl == "plane" else 1                                   # rows of one batch entry
    bins_per_entry = nbins * rows

    # ---- inputs, resident in HBM (seeded; every rank draws its own batch: weak scaling) -----------------------------
    cfg = {"config2": 2, "config1": 2, "config3": 3, "allh": 5, "plane": 6, "complex": 7}[wl]
    scale = float(np.float32(1.0 / 312500.0))
    if wl == "complex":
        g = torch.Generator(device=dev).manual_seed(W.S0 + cfg + 100 * rank)
        x = torch.randn((batch, nbins, 2), generator=g, device=dev) * float(np.sqrt(312500.0 / 2))   # |F|^2 scale ~ Exp(1)
    else:
        x = W.exp_noise_torch(batch * rows, nbins, cfg + 100 * rank, dev)
        if wl == "config3":
            W.inject_combs_torch(x, 3, 1.0, 1000.0, 100000.0, 0.03)
        elif wl in ("config2", "config1"):
            W.inject_combs_torch(x, 2, 0.01, 50.0, 5000.0, 0.10)
        if rows > 1:
            x = x.view(batch, rows, nbins)
    oshape = (batch, nbins) if rows == 1 else (batch, rows, nbins)
    sums = torch.empty((batch, L) + oshape[1:], dtype=torch.float32, device=dev) if out_mode in ("full", "both") else None
    vmax = torch.empty(oshape, dtype=torch.float32, device=dev) if out_mode in ("reduced", "both") else None
    amax = torch.empty(oshape, dtype=torch.uint8, device=dev) if out_mode in ("reduced", "both") else None
    plans = {}
    for v in variants:
        if wl == "allh":
            p = hs.hs_plan_create_ex(nbins, batch, Hmax, v, out_mode, "all", "c2")
        elif wl == "plane":
            p = hs.hs_plan_create_2d(nbins, rows, batch, Hmax, v, out_mode)
        else:
            p = hs.hs_plan_create(nbins, batch, 32, v, out_mode)
            ok = not (args.algo in ("twophase", "grouped") and v not in ("max", "freqbin")) and not (args.algo == "gather" and v not in ("freqbin", "greedy"))
            p.set_algo(args.algo if ok else "auto")
        p.ensure_workspace(dev)
        plans[v] = p
    algo_names = {hs.HS_ALGO_DIRECT: "direct", hs.HS_ALGO_TILED: "tiled", hs.HS_ALGO_GENERAL: "general"}
    stream = torch.cuda.current_stream()

    def step(events=None):
        for v in variants:
            if events is not None:
                events[v][0].record(stream)
            if wl == "complex":
                plans[v].hs_execute_complex(x, scale, sums, vmax, amax, stream)
            else:
                plans[v].hs_execute(x, sums, vmax, amax, stream)
            if events is not None:
                events[v][1].record(stream)

    for _ in range(max(3, args.warmup)):
        step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()

    # ---- timed region: exactly K steps, CUDA events on the launching stream, clocks sampled meanwhile --------------
    sampler = ClockSampler(local_rank) if rank == 0 else None
    per_step_events = [{v: (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for v in variants}
                       for _ in range(args.steps)]
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    for k in range(args.steps):
        step(per_step_events[k])
    ev1.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    clocks = sampler.stop() if sampler else None
    for v in variants:
        plans[v].device_status(stream)                       # no kernel of the timed region gave up a wait (else it raises)
    local_ms = ev0.elapsed_time(ev1)
    total_ms = max_over_ranks_ms(local_ms, dist if world > 1 else None)
    ms_per_step = total_ms / args.steps
    bins_per_step = float(len(variants)) * batch * bins_per_entry * world
    value = bins_per_step / (ms_per_step * 1e-3)

    per_variant_ms = {v: statistics.mean(e[v][0].elapsed_time(e[v][1]) for e in per_step_events) for v in variants}
    per_variant_best = {v: min(e[v][0].elapsed_time(e[v][1]) for e in per_step_events) for v in variants}
    peak, peak_src = measured_peak()
    bpb = BYTES_PER_BIN[out_mode] if headline_workload else {"allh": 4 + 5, "plane": 4 + 5, "complex": 8 + 5}[wl]
    nbins_eff = bins_per_entry                               # output bins per batch entry
    per_variant = {}
    default_kernels = {"standard": "rb_kernel", "max": "gr_kernel", "freqbin": "il_persistent_kernel",
                       "greedy": "hs_greedy_gather_kernel"}
    WAIT_WORDS = {"gr_kernel": "[group-barrier waits that had to spin, polls, -, -]",
                  "il_persistent_kernel": "[times a CTA found neither of its tickets runnable, polls of those, -, -]"}
    for v in variants:
        gbs = bpb * batch * nbins_eff / (per_variant_ms[v] * 1e-3) / 1e9
        per_variant[v] = {"ms": per_variant_ms[v], "best_ms": per_variant_best[v],
                          "bins_per_s": batch * nbins_eff / (per_variant_ms[v] * 1e-3), "eff_GBps": gbs,
                          "frac_of_measured_peak": gbs / peak, "frac_of_nominal_8TBps": gbs / 8000.0,
                          "algo": algo_names[plans[v].algo], "launches": plans[v].launches()}
        ws = plans[v]._ws
        if ws is not None and ws.numel() >= 64 and v != "standard":
            # wait statistics of the persistent kernels' control block (hs_internal.cuh: words 2.. of the workspace)
            c = ws[:64].view(torch.int32).cpu().tolist()
            per_variant[v]["waits"] = {"kernel": default_kernels.get(v), "error_flag": c[1], "words_2_to_5": c[2:6],
                                       "meaning": WAIT_WORDS.get(default_kernels.get(v), "?"),
                                       "workspace_MiB": round(plans[v].workspace_bytes() / 2**20)}
    dominant = max(variants, key=lambda v: per_variant_ms[v])
    dom_algo = per_variant[dominant]["algo"]
    kname = default_kernels[dominant] if (args.algo == "auto" and args.workload == "config2") else dom_algo
    if wl in ("allh", "plane"):
        kname = "hs_allh_kernel" if wl == "allh" else "hs_2d_kernel"
    traffic = ncu_traffic(dominant, args.workload, dom_algo)
    roofline = {"bound": "hbm", "kernel": f"{kname} ({dominant}, eq. {1 + VARIANTS.index(dominant) if dominant in VARIANTS else 0})", "achieved": per_variant[dominant]["eff_GBps"],
                "peak": peak, "unit": "GB/s", "frac": per_variant[dominant]["eff_GBps"] / peak,
                "traffic": traffic,
                "traffic_source": ("profiles/ncu_traffic.json: dram__bytes_read.sum + dram__bytes_write.sum of one ncu --set full "
                                   "capture of this kernel on this workload (re-captured whenever a default kernel changes; "
                                   "not measured in this run)") if traffic is not None else None,
                "algorithmic_bytes_per_launch": bpb * batch * nbins_eff, "algorithmic_bytes_per_bin": bpb,
                "peak_source": peak_src}

    if rank != 0 and world > 1:
        # other ranks still take part in the e2e collectives below
        pass

    # ---- fused back end: hs_execute_candidates, 4 B/bin of HBM traffic instead of 9 -------------------
    cand_line = None
    if out_mode == "reduced" and args.candidates_threshold > 0 and headline_workload:
        cap = 1 << 22
        d_cand = torch.empty((cap, 4), dtype=torch.int32, device=dev)
        d_count = torch.zeros(1, dtype=torch.int64, device=dev)
        cand_line = {"threshold": args.candidates_threshold, "algorithmic_bytes_per_bin": 4, "per_variant": {}}
        for v in variants:
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(max(3, args.steps))]
            for _ in range(3):
                plans[v].hs_execute_candidates(x, args.candidates_threshold, d_cand, cap, d_count, stream)
            for e0, e1 in ev:
                e0.record(stream)
                plans[v].hs_execute_candidates(x, args.candidates_threshold, d_cand, cap, d_count, stream)
                e1.record(stream)
            torch.cuda.synchronize()
            ms = statistics.mean(e0.elapsed_time(e1) for e0, e1 in ev)
            cand_line["per_variant"][v] = {"ms": ms, "bins_per_s": batch * nbins / (ms * 1e-3), "found": int(d_count.item()),
                                           "eff_GBps": 4.0 * batch * nbins / (ms * 1e-3) / 1e9,
                                           "frac_of_measured_peak": 4.0 * batch * nbins / (ms * 1e-3) / 1e9 / peak}
        del d_cand

    # ---- e2e: the same step through hs_execute_host with pinned host buffers -------------------------------------------
    e2e = None
    if not args.no_e2e and not headline_workload:
        e2e = {"value": None, "unit": "bins/s", "unavailable": "the end-to-end leg is timed on the headline workloads only"}
    elif not args.no_e2e:
        ok, why = 1, ""
        try:
            slab = max(1, min(batch, (1 << 26) // nbins))          # 256 MiB of input per slab
            h_x = torch.empty((batch, nbins), dtype=torch.float32, pin_memory=True)
            h_x.copy_(x)
            h_sums = torch.empty((batch, L, nbins), dtype=torch.float32, pin_memory=True) if sums is not None else None
            h_max = torch.empty((batch, nbins), dtype=torch.float32, pin_memory=True) if vmax is not None else None
            h_amax = torch.empty((batch, nbins), dtype=torch.uint8, pin_memory=True) if amax is not None else None
            stagings = {}
            for v in variants:
                st = torch.empty(plans[v].host_staging_bytes(slab), dtype=torch.uint8, device=dev)
                plans[v].set_host_staging(st, slab)
                stagings[v] = st
        except (RuntimeError, MemoryError) as exc:     # e.g. no room for the pinned host buffers: report, do not fail the line
            ok, why = 0, str(exc).splitlines()[0][:200]
        if world > 1:                                  # every rank takes the same branch (the timed part has a barrier)
            flag = torch.tensor([ok], dtype=torch.int32, device=dev)
            dist.all_reduce(flag, op=dist.ReduceOp.MIN)
            ok = int(flag.item())
        if not ok:
            e2e = {"value": None, "unit": "bins/s", "unavailable": why or "another rank could not allocate its host buffers"}
        else:

            def host_step():
                for v in variants:
                    plans[v].hs_execute_host(h_x, h_sums, h_max, h_amax, stream)

            host_step()
            torch.cuda.synchronize()
            if world > 1:
                dist.barrier()
            t0 = time.perf_counter()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(args.e2e_steps):
                host_step()
            e1.record(stream)
            torch.cuda.synchronize()
            wall_ms = (time.perf_counter() - t0) * 1e3
            e2e_ms = max_over_ranks_ms(max(e0.elapsed_time(e1), wall_ms), dist if world > 1 else None) / args.e2e_steps
            h2d = len(variants) * batch * nbins * 4
            d2h = len(variants) * batch * nbins * (bpb - 4)
            e2e = {"value": bins_per_step / (e2e_ms * 1e-3), "unit": "bins/s", "h2d_bytes_per_step": h2d,
                   "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms, "steps": args.e2e_steps,
                   "slab_spectra": slab, "checksum_max": float(h_max[0, :16].sum()) if h_max is not None else None}
            del stagings

    # ---- cpu_baseline: the oracle on a bounded sample of the same workload (rank 0, N = 1 only) ------------------------
    cpu = None
    if rank == 0 and world == 1 and args.cpu_seconds > 0 and headline_workload:
        threads = os.cpu_count() or 1
        crows = cpu_sample_rows(args.cpu_seconds, threads, nbins, variants, cap=256)   # (a few seconds on 16 threads)
        crows = min(crows, batch)
        x_rows = x[:crows].cpu().numpy()
        rate, dt, done = oracle_rate(x_rows, variants, args.cpu_seconds, threads)
        cpu = {"value": rate, "unit": "bins/s", "cores": threads, "kind": "oracle",
               "sample": f"first {crows} spectra of the batch x {len(variants)} variants, whole spectra, {dt:.1f} s",
               "gpu_over_cpu": value / rate, "cpu_model": cpu_model(),
               "flags": "gcc -std=c99 -O2 (no -ffast-math), fp64, one spectrum per task (PAPER.md:27)",
               "per_variant": oracle_per_variant(x_rows, variants, threads, {v: per_variant[v]["bins_per_s"] for v in variants}),
               "paper_context": "PAPER.md:66-71 Table 1 GPU/CPU speed-ups (hardware not stated): standard 250x, Greedy 704x, freq-bin 110x, Max 177x"}
    elif rank == 0 and world == 1 and args.cpu_seconds > 0:
        threads = os.cpu_count() or 1
        rate, per_cpu, used, sample, dt = oracle_rate_ext(wl, x, variants, args.cpu_seconds, threads, scale,
                                                          {v: per_variant[v]["bins_per_s"] for v in variants})
        cpu = {"value": rate, "unit": "bins/s", "cores": used, "kind": "oracle", "sample": f"{sample}; {dt:.1f} s in all",
               "gpu_over_cpu": value / rate, "cpu_model": cpu_model(),
               "flags": "gcc -std=c99 -O2 (no -ffast-math), fp64 (the power spectrum in fp32), oracle/hs_oracle_ext.c as it stands",
               "per_variant": per_cpu}

    if rank == 0:
        line = {"metric": "harmonic_sum_bins_per_s", "value": value, "unit": "bins/s", "n_gpus": world,
                "steps": args.steps, "warmup": max(3, args.warmup), "warmup_requested": args.warmup, "ms_per_step": ms_per_step,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": desc, "batch_per_gpu": batch, "nbins": nbins, "Hmax": Hmax, "out_mode": out_mode,
                           "variants": variants, "algo": args.algo, "headline": headline_workload and not args.batch,
                           "l2": f"input {x.numel() * 4 / 2**20:.0f} MiB per variant launch vs 126 MB L2"
                                 + ("" if x.numel() * 4 > (1 << 28) else " (fits: not a headline size)"),
                           "parallelism": f"dp{world} (batch shards, no collective)",
                           "input_checksum_spectrum0": W.checksum(x[:1].reshape(1, -1)[:, :nbins].cpu().numpy())},
                "eff_GBps": value * bpb / 1e9 / world, "frac_of_measured_peak": value * bpb / 1e9 / world / peak,
                "frac_of_nominal_8TBps": value * bpb / 1e9 / world / 8000.0,
                "per_variant": per_variant, "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "candidates": cand_line,
                "gpu_launches": sum(plans[v].launches() for v in variants) * args.steps, "clocks": clocks,
                "paper_context": "PAPER.md:66-71 Table 1 GPU/CPU speed-ups 250x/704x/110x/177x (std/greedy/freq-bin/max), "
                                 "hardware not stated"}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
