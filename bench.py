#!/usr/bin/env python
"""bench.py — n-gluon |M|^2 events/s on B200 (BASELINE.json metric), one JSON line on stdout.

A "step" is one pass of the whole hot path (load event, external currents, recursion, closure / colour assembly,
store) over one batch of synthetic events.  Default workload: BASELINE.json configs[1]
(n = 6 gluons, colour-dressed recursion with sampled helicities and colour flows, 2^20 RAMBO events).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 0..4] [--n n] [--events N] [--kernel k]
  python bench.py --impl reference ...      # the CPU oracle on the host cores (bounded sample per step)

Multi-GPU (torchrun): events are independent, so each rank evaluates its own batch of the
same size with no data-path collective (weak scaling); timing is max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

# Algorithmic FP64 work per event of the colour-dressed recursion with sampled discrete colours (SURVEY.md §8d,
# mean over sampled colour assignments), and of the colour-ordered configs.
CDBG_FLOP_PER_EVENT = {4: 2.1e3, 5: 8.4e3, 6: 2.5e4, 7: 7.0e4, 8: 2.2e5, 9: 6.4e5, 10: 1.9e6, 11: 5.1e6, 12: 1.46e7}
COBG_FLOP_PER_EVENT = {0: 2.6e4, 2: 1.41e6 + 5.8e4}     # config 0 (n=4 helsum), config 2 (n=7 + colour form)
# DRAM bytes of the dominant kernel's launches of one step are NOT measured here: when profiles/ holds the table
# written from an `ncu --set full` capture of the same command, the matching row is quoted with the file's name.
TRAFFIC_CSV = os.path.join("profiles", "r02_dram_traffic.csv")     # kernel,n,events,bytes_per_step,source
CONFIG_N = {0: 4, 1: 6, 2: 7, 3: 9}
CONFIG_EVENTS = {0: 1024, 1: 1 << 20, 2: 1 << 18, 3: 1 << 18, 4: 1 << 16}
COBG_N8_EVENTS = 1 << 14      # extra line: colour-ordered n = 8 (720 orderings, 720 x 720 colour matrix)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=1, help="index into BASELINE.json configs (default 1)")
    ap.add_argument("--n", type=int, default=None, help="gluon multiplicity for the sweep config 4")
    ap.add_argument("--events", type=int, default=None, help="override the number of events per step and GPU")
    ap.add_argument("--kernel", type=int, default=0, help="BG_OPT_KERNEL (0 auto, 1 generic, 2 class programs)")
    ap.add_argument("--lanes", type=int, default=None, help="BG_OPT_LANES (lanes per event, class-program kernel)")
    ap.add_argument("--smem-limit", type=int, default=None, help="BG_OPT_SMEM_LIMIT in bytes (spill threshold)")
    ap.add_argument("--device-gen", action="store_true",
                    help="also time generate-on-device + evaluate per step (bg_generate, SURVEY NEXT-4; PAPER.md:L259)")
    ap.add_argument("--continuous", action="store_true",
                    help="CDBG configs with continuous colour / polarisation states (Eq. 5-14, SURVEY NEXT-1)")
    ap.add_argument("--lc", action="store_true", help="configs 0 / 2 in leading-colour mode (Eq. 33, SURVEY NEXT-3)")
    ap.add_argument("--comc", action="store_true",
                    help="colour-dressed configs through BG_COMC_GIVEN (Eq. 19 with colour-ordered currents, SURVEY NEXT-2; n <= 9)")
    ap.add_argument("--precision", type=int, default=None, help="BG_OPT_PRECISION (1 = double-double reference path)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-configs", action="store_true",
                    help="skip the compact measurements of the other BASELINE.json configs (C1, C3, C4, C5 n = 4..12)")
    return ap.parse_args()


def ncu_traffic(kernel: str, n: int, N: int):
    """bytes per step of the dominant kernel from the committed ncu table, or (None, None)."""
    path = os.path.join(ROOT, TRAFFIC_CSV)
    if not os.path.exists(path):
        return None, None
    import csv
    with open(path) as f:
        for row in csv.DictReader(f):
            if row["kernel"] == kernel and int(row["n"]) == n and int(row["events"]) == N:
                return float(row["bytes_per_step"]), f"{TRAFFIC_CSV}: {row['source']}"
    return None, None


def truth_sample_size(n: int, N: int) -> int:
    """events of a config compared with the long-double oracle inside the bench (bounded CPU time)."""
    return min(N, {4: 16384, 5: 16384, 6: 16384, 7: 8192, 8: 4096, 9: 2048, 10: 512, 11: 192, 12: 64}[n])


def measure_next_rows(bg, wl, dev, steps: int = 3):
    """Sweep lines for the SURVEY 8(f) rows beside the BASELINE configs: events/s (device-resident inputs, FP64 kernels)
    of the continuous colour / polarisation states (NEXT-1), the colour-ordered Monte Carlo of Eq. 19 (NEXT-2), the
    leading-colour approximation of Eq. 33 (NEXT-3) and the no-allocation entry point, on small synthetic batches;
    their parity tests are tests/test_gpu_parity.py and tests/test_zz_no_alloc.py."""
    import torch
    stream = torch.cuda.current_stream()
    sh = stream.cuda_stream

    def rate(call, N):
        for _ in range(2):
            call()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(steps):
            call()
        e1.record(stream)
        torch.cuda.synchronize()
        return {"events": N, "events_per_s": N * steps / (e0.elapsed_time(e1) * 1e-3)}

    rows = {"continuous_states": {}, "co_mc": {}, "leading_colour_helgiven": {}, "no_alloc_entry_point": {}}
    for n in range(4, 11):          # BG_CDBG_CONTINUOUS, real arithmetic
        N = max(1 << 10, (1 << 17) >> (2 * (n - 4)))
        mom = wl.rambo(n, N, seed=1, stream=900 + n)
        phi, eta = wl.continuous_states(n, N, seed=1, stream=900 + n)
        sphi, seta = wl.continuous_to_soa(phi, eta)
        d = [torch.from_numpy(x).to(dev) for x in (wl.to_soa(mom=mom), sphi, seta)]
        out = torch.empty(N, dtype=torch.float64, device=dev)
        ctx = bg.bg_init(n, bg.BG_CDBG_CONTINUOUS)
        try:
            bg.bg_reserve(ctx, N)
            rows["continuous_states"][str(n)] = rate(lambda: bg.bg_eval_continuous(ctx, sh, N, d[0], d[1], d[2], out), N)
        finally:
            bg.bg_destroy(ctx)
    for mode, key, nmax in ((bg.BG_COMC_GIVEN, "co_mc", 9), (bg.BG_COBG_HELGIVEN_LC, "leading_colour_helgiven", 8)):
        for n in range(4, nmax + 1):
            N = max(1 << 10, (1 << 18) >> (2 * (n - 4)))
            ev = wl.config_events(4, N=N, n=n)
            d_mom = torch.from_numpy(wl.to_soa(mom=ev.mom)).to(dev)
            d_hel = torch.from_numpy(wl.to_soa(hel=ev.hel)).to(dev)
            d_col = torch.from_numpy(wl.to_soa(col=ev.col)).to(dev) if mode & bg.BG_COL_GIVEN else None
            out = torch.empty(N, dtype=torch.float64, device=dev)
            ctx = bg.bg_init(n, mode)
            try:
                bg.bg_reserve(ctx, N)
                rows[key][str(n)] = rate(lambda: bg.bg_eval(ctx, sh, N, d_mom, d_hel, d_col, out), N)
            finally:
                bg.bg_destroy(ctx)
    bg.bg_static_setup()
    for n in (6, 8):                # bg_eval_static: thread-per-event kernel, scratch in the fixed device array
        N = bg.bg_static_max_events(n)
        ev = wl.config_events(4, N=N, n=n)
        d = [torch.from_numpy(x).to(dev) for x in (wl.to_soa(mom=ev.mom), wl.to_soa(hel=ev.hel), wl.to_soa(col=ev.col))]
        out = torch.empty(N, dtype=torch.float64, device=dev)
        rows["no_alloc_entry_point"][str(n)] = rate(lambda: bg.bg_eval_static(sh, n, N, d[0], d[1], d[2], out), N)
    return rows


def measure_config(bg, wl, oracle_mod, dev, config: int, n: int, steps: int, peak_tf: float, with_cpu: bool):
    """Compact measurement of one BASELINE.json config on the current device (N = 1): events/s of the default path,
    the FP64-only path beside it, the FP64 kernel's roofline fraction, the conditioning flag's cost, the CPU oracle
    (all cores / one core) and parity against the long-double oracle on a stated sample."""
    import torch
    cobg8 = config == 2 and n == 8
    N = COBG_N8_EVENTS if cobg8 else CONFIG_EVENTS[config]
    ev = wl.config_events(4, N=N, n=8) if cobg8 else wl.config_events(config, N=N, n=n if config == 4 else None)
    mode = mode_for(config)
    flop = COBG_FLOP_PER_EVENT[config] if config in (0, 2) else CDBG_FLOP_PER_EVENT[n]
    if cobg8:       # 720 orderings x (C(8,3) V3 + C(8,4) V4) at 158 / 178 flop + 2 x 720^2 MAC (SURVEY 8d counting)
        flop = 720 * (56 * 158 + 70 * 178) + 4.0 * 720 * 720
    d_mom = torch.from_numpy(wl.to_soa(mom=ev.mom)).to(dev)
    d_hel = None if ev.hel is None or (mode & bg.BG_HEL_SUM) else torch.from_numpy(wl.to_soa(hel=ev.hel)).to(dev)
    d_col = None if not (mode & bg.BG_COL_GIVEN) else torch.from_numpy(wl.to_soa(col=ev.col)).to(dev)
    d_out = torch.empty(N, dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream()
    sh = stream.cuda_stream
    ctx = bg.bg_init(n, mode)
    res = {"workload": ("COBG full colour (extra)" if cobg8 else {0: "C1", 2: "C3", 3: "C4", 4: "C5"}.get(config, "C2")) + f" n={n}", "n": n, "events": N}
    try:
        bg.bg_reserve(ctx, N)
        auto = config != 0 and not (config == 4 and n == 4)     # (n = 4 CDBG: the default is FP64 alone)

        def timed(precision):
            if auto:
                bg.bg_set_option(ctx, bg.BG_OPT_PRECISION, precision)
            for _ in range(3):
                bg.bg_eval(ctx, sh, N, d_mom, d_hel, d_col, d_out)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(steps):
                bg.bg_eval(ctx, sh, N, d_mom, d_hel, d_col, d_out)
            e1.record(stream)
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / steps
            bg.bg_set_option(ctx, bg.BG_OPT_TIMING, 1)
            kms, rms, fl, tw = [], [], 0, 0
            for _ in range(min(steps, 5)):
                bg.bg_eval(ctx, sh, N, d_mom, d_hel, d_col, d_out)
                kms.append(bg.bg_last_kernel_ms(ctx))
                fl, r = bg.bg_last_refined(ctx)
                tw = bg.bg_last_twin(ctx)
                rms.append(r)
            bg.bg_set_option(ctx, bg.BG_OPT_TIMING, 0)
            return ms, float(np.mean(kms)), float(np.mean(rms)), fl, tw
        ms, kms, rms, fl, tw = timed(2)
        got = d_out.cpu().numpy()
        res.update({"events_per_s": N / (ms * 1e-3), "ms_per_step": ms, "kernel_ms": kms,
                    "gpu_launches_per_step": bg.bg_last_launch_count(ctx), "kernel": bg.bg_last_kernel_name(ctx),
                    "current_bytes_per_event": bg.bg_current_bytes_per_event(ctx)})
        fp64_kms = kms - rms
        res["roofline"] = {"bound": "alu", "flop_per_event": flop, "fp64_kernel_ms": fp64_kms,
                           "achieved": flop * N / (fp64_kms * 1e-3) * 1e-12, "unit": "TFLOP/s",
                           "frac": flop * N / (fp64_kms * 1e-3) * 1e-12 / peak_tf}
        if config == 0:
            res["note"] = "1024 events: one 13 us launch, launch-latency bound (SURVEY 8d); FP64 alone meets 1e-11"
        if config == 2 and not cobg8:
            a, b, dmax = bg.bg_colour_form_probe(n, N, 3)
            res["colour_form_probe"] = {"dfma_row_dots_ms": a, "dmma_m8n8k4_ms": b, "max_rel_diff": dmax,
                                        "note": "step a7 alone on synthetic amplitudes (bg_colour_form_probe); the production "
                                                "kernel keeps the fused DFMA form (DESIGN.md 5.2)"}
        if auto:
            ms0, kms0, _, _, _ = timed(0)
            res["precision_auto"] = {"flagged_frac": fl / N, "second_fp64_frac": tw / N, "reevaluation_ms": rms,
                                     "overhead_pct": 100.0 * (ms / ms0 - 1.0),
                                     "fp64_only_events_per_s": N / (ms0 * 1e-3), "fp64_only_ms_per_step": ms0}
            bg.bg_set_option(ctx, bg.BG_OPT_PRECISION, 2)
    finally:
        bg.bg_destroy(ctx)
    if with_cpu:
        S = truth_sample_size(n, N)
        sub = ev.head(S)
        if config == 0:
            truth = oracle_mod.cobg_full_colour(sub.mom, None, prec="long double")
        elif cobg8:
            truth, S = None, 0        # the oracle's Gell-Mann colour matrix is out of reach at n = 8 (tests/: amplitudes + Eq. 17)
        elif config == 2:
            S = min(S, 1024)
            sub = ev.head(S)
            truth = oracle_mod.cobg_full_colour(sub.mom, sub.hel, prec="long double")
        else:
            truth = oracle_mod.cdbg(sub.mom, sub.hel, sub.col, prec="long double")
        if truth is not None:
            err = np.abs(got[:S] - truth) / np.abs(truth)
            res["parity"] = {"max_rel_err_vs_long_double": float(err.max()), "median": float(np.median(err)),
                             "n_over_1e-11": int(np.sum(err > 1e-11)), "sample": f"first {S} events"}
        if cobg8:
            return res

        class A:
            pass
        a = A()
        a.config = config
        cpu = {}
        for label, threads, budget in (("all_cores", 0, 1.0), ("one_core", 1, 1.0)):
            S2 = max(16, int(cpu_sample_size(a, n, N) * (budget / 15.0) / (1 if threads == 0 else oracle_mod.max_threads())))
            S2 = min(S2, N)
            sample = ev.head(S2)
            t0 = time.perf_counter()
            reps = 0
            while reps < 1 or (time.perf_counter() - t0 < 0.5 and reps < 1000):
                oracle_eval(a, sample, threads)
                reps += 1
            dt = time.perf_counter() - t0
            cpu[label] = {"events_per_s": S2 * reps / dt, "cores": oracle_mod.max_threads() if threads == 0 else 1,
                          "sample": f"first {S2} events x {reps}"}
        res["cpu_baseline"] = cpu
    return res



def workload_desc(args):
    n = CONFIG_N.get(args.config, args.n)
    if n is None:
        raise SystemExit("--config 4 needs --n")
    N = args.events or CONFIG_EVENTS[args.config]
    if args.config in (0, 2) and args.lc:
        import math
        # (n-1)! orderings x (C(n,3) V3 + C(n,4) V4) at 158 / 178 flop, x 2^n helicities when summed
        flop = math.factorial(n - 1) * (math.comb(n, 3) * 158 + math.comb(n, 4) * 178) * (16 if args.config == 0 else 1)
    elif args.config in (0, 2):
        flop = COBG_FLOP_PER_EVENT[args.config]
    else:
        flop = CDBG_FLOP_PER_EVENT[n]
    names = {0: "C1 n=4 COBG helicity-summed full-colour", 1: "C2 n=6 CDBG sampled helicity+colour",
             2: "C3 n=7 COBG sampled helicity full-colour (120x120)", 3: "C4 n=9 CDBG sampled helicity+colour",
             4: f"C5 n={n} CDBG sampled helicity+colour"}
    return n, N, flop, names[args.config]


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {"hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4)}
        while not self._stop_evt.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.01)

    def stop(self):
        self._stop_evt.set()
        if self.is_alive():
            self.join(timeout=2)
        med = int(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def make_events(args, n, N, rank):
    from paper_2106_06507_b200 import workload as wl
    return wl.config_events(args.config, N=N, n=n if args.config == 4 else None, first_event=rank * N)


def max_over_ranks(value: float, world: int, dev) -> float:
    """Multi-GPU numbers are the maximum over ranks (the slowest rank defines the step)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def mode_for(config, lc=False):
    import paper_2106_06507_b200 as bg
    if lc:
        return {0: bg.BG_COBG_HELSUM_LC, 2: bg.BG_COBG_HELGIVEN_LC}[config]
    return {0: bg.BG_COBG_HELSUM_FULLCOLOR, 2: bg.BG_COBG_HELGIVEN_FULLCOLOR}.get(config, bg.BG_CDBG_GIVEN)


def oracle_eval(args, ev, threads=0):
    import oracle
    if args.config == 0:
        return oracle.cobg_full_colour(ev.mom, None, threads=threads)
    if args.config == 2:
        return oracle.cobg_full_colour(ev.mom, ev.hel, threads=threads)
    return oracle.cdbg(ev.mom, ev.hel, ev.col, threads=threads)


def cpu_sample_size(args, n, N):
    """Events per oracle timing sample: about 10-30 s of CPU work (single-core estimates per event)."""
    per_event = {0: 2e-6, 2: 5e-5}.get(args.config)       # aggregate seconds per event on ~16 cores x 3 (margin)
    if per_event is None:
        per_event = {4: 1.5e-7, 5: 4e-7, 6: 1.2e-6, 7: 4e-6, 8: 1.2e-5, 9: 4e-5, 10: 1.3e-4, 11: 4e-4, 12: 1.3e-3}[n]
    return int(max(64, min(N, 15.0 / per_event)))


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, on the host cores, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    n, N, flop, name = workload_desc(args)
    S = cpu_sample_size(args, n, N)
    S = max(64, S // max(1, args.steps + args.warmup) * 2) if args.steps + args.warmup > 4 else S
    ev = make_events(args, n, S, 0)
    # torchrun exports OMP_NUM_THREADS=1 to every rank; here rank 0 works alone, so it takes the host cores it may
    # run on (the same count the N=1 launch gets from OpenMP's default)
    threads = len(os.sched_getaffinity(0)) if int(os.environ.get("WORLD_SIZE", "1")) > 1 else 0
    cores = threads or oracle.max_threads()
    for _ in range(max(1, min(args.warmup, 3))):
        oracle_eval(args, ev.head(max(64, S // 8)), threads)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_eval(args, ev, threads)
    dt = time.perf_counter() - t0
    value = S * args.steps / dt
    line = {"impl": "reference", "metric": "n-gluon |M|^2 events/sec", "value": value, "unit": "events/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": name, "n": n, "events_per_step": S, "note": "CPU oracle (oracle/bg_oracle.cpp, "
                       "double, OpenMP), bounded sample of the workload per step"},
            "cpu_baseline": {"value": value, "unit": "events/s", "cores": cores, "kind": "oracle",
                             "sample": f"{S} events per step x {args.steps} steps of {name}"},
            "e2e": {"value": value, "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_b200(args):
    import torch
    import torch.distributed as dist
    import paper_2106_06507_b200 as bg
    from paper_2106_06507_b200 import workload as wl

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the B200 path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    n, N, flop_per_event, name = workload_desc(args)
    ev = make_events(args, n, N, rank)
    mode = mode_for(args.config, args.lc)
    d_phi = d_eta = None
    if args.continuous:
        if args.config in (0, 2):
            raise SystemExit("--continuous applies to the colour-dressed configs (1, 3, 4)")
        mode = bg.BG_CDBG_CONTINUOUS
        phi, eta = wl.continuous_states(n, N, seed=1, stream=rank)
        sphi, seta = wl.continuous_to_soa(phi, eta)
        d_phi, d_eta = torch.from_numpy(sphi).to(dev), torch.from_numpy(seta).to(dev)
        # dense colour: 3^(n-1) - 2^n + 1 ordered splits x 27 colour terms x ~446 flop with complex currents (SURVEY 8d
        # "dense-colour bound"); real polarisations make every number real: half of that
        flop_per_event = (3 ** (n - 1) - 2 ** n + 1) * 27 * 223.0
        args.no_e2e = True
        name += " - continuous colour/polarisation states (Eq. 5-14)"
    if args.comc:
        if args.config in (0, 2) or args.continuous:
            raise SystemExit("--comc applies to the colour-dressed configs (1, 3, 4) with discrete colours")
        mode = bg.BG_COMC_GIVEN          # same events, same |M|^2, same algorithmic flop: another recursion
        name += " - CO_MC (Eq. 19, colour-ordered currents)"
    mom = wl.to_soa(mom=ev.mom)
    hel = None if ev.hel is None else wl.to_soa(hel=ev.hel)
    col = None if ev.col is None else wl.to_soa(col=ev.col)
    # pinned host copies (end-to-end path) and device-resident copies (kernel path)
    h_mom = torch.from_numpy(mom).pin_memory()
    h_hel = None if hel is None else torch.from_numpy(hel).pin_memory()
    h_col = None if col is None else torch.from_numpy(col).pin_memory()
    h_out = torch.empty(N, dtype=torch.float64).pin_memory()
    d_mom = h_mom.to(dev)
    d_hel = None if h_hel is None else h_hel.to(dev)
    d_col = None if h_col is None else h_col.to(dev)
    d_out = torch.empty(N, dtype=torch.float64, device=dev)

    ctx = bg.bg_init(n, mode)
    if args.kernel:
        bg.bg_set_option(ctx, bg.BG_OPT_KERNEL, args.kernel)
    if args.lanes is not None:
        bg.bg_set_option(ctx, bg.BG_OPT_LANES, args.lanes)
    if args.precision is not None:
        bg.bg_set_option(ctx, bg.BG_OPT_PRECISION, args.precision)
    if args.smem_limit is not None:
        bg.bg_set_option(ctx, bg.BG_OPT_SMEM_LIMIT, args.smem_limit)
    bg.bg_reserve(ctx, N)
    stream = torch.cuda.current_stream()
    sh = stream.cuda_stream

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        if args.continuous:
            bg.bg_eval_continuous(ctx, sh, N, d_mom, d_phi, d_eta, d_out)
        else:
            bg.bg_eval(ctx, sh, N, d_mom, d_hel, d_col, d_out)

    peak_tf = bg.bg_fp64_peak_probe(1 << 14) if rank == 0 else None

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        torch.cuda.nvtx.range_push("bg_timed_step")      # (for `ncu --nvtx --nvtx-include "bg_timed_step/"`: profiles/*.md)
        step()
        torch.cuda.nvtx.range_pop()
    e1.record(stream)
    barrier()
    # same steps again with the library's CUDA events around the dominant (recursion) kernel, on the launching
    # stream; these launches are part of the same hot loop (clock sampler still running)
    bg.bg_set_option(ctx, bg.BG_OPT_TIMING, 1)
    kms = []
    for _ in range(args.steps):
        step()
        kms.append(bg.bg_last_kernel_ms(ctx))
    bg.bg_set_option(ctx, bg.BG_OPT_TIMING, 0)
    barrier()
    clocks = sampler.stop()
    total_ms = e0.elapsed_time(e1)
    launches_per_step = bg.bg_last_launch_count(ctx)
    kernel_name = bg.bg_last_kernel_name(ctx)
    kernel_ms = float(np.mean(kms))      # per step: all launches of the recursion kernels (FP64 + re-evaluation)
    flagged, refine_ms, second = (0, 0.0, 0)
    if not args.continuous:
        bg.bg_set_option(ctx, bg.BG_OPT_TIMING, 1)
        step()
        flagged, refine_ms = bg.bg_last_refined(ctx)
        second = bg.bg_last_twin(ctx)
        bg.bg_set_option(ctx, bg.BG_OPT_TIMING, 0)
    auto_default = args.precision is None and flagged > 0
    total_ms = max_over_ranks(total_ms, world, dev)
    value = N * world * args.steps / (total_ms * 1e-3)

    # generation on the device inside the timed region (the paper's timings include phase-space generation, L259):
    # nothing crosses PCIe but the seed
    devgen = None
    default_line = (world == 1 and args.config == 1 and args.events is None and args.precision is None and not args.kernel
                    and args.lanes is None and not (args.continuous or args.comc or args.lc))
    if (args.device_gen or default_line) and not args.continuous:
        g_mom = torch.empty_like(d_mom)
        g_hel = None if d_hel is None or (mode & bg.BG_HEL_SUM) else torch.empty_like(d_hel)
        g_col = None if d_col is None or not (mode & bg.BG_COL_GIVEN) else torch.empty_like(d_col)
        cuts = (0.0, 0.0) if args.config == 0 else (wl.PT_MIN, wl.DR_MIN)

        def gen_step(i):
            bg.bg_generate(sh, n, N, 1, 9000 + args.config, i * N, wl.SQRT_S, cuts[0], cuts[1], True, g_mom, g_hel, g_col)
            bg.bg_eval(ctx, sh, N, g_mom, g_hel, g_col, d_out)
        for i in range(3):
            gen_step(i)
        barrier()
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g0.record(stream)
        for i in range(args.steps):
            torch.cuda.nvtx.range_push("bg_gen_step")
            gen_step(3 + i)
            torch.cuda.nvtx.range_pop()
        g1.record(stream)
        barrier()
        gms = max_over_ranks(g0.elapsed_time(g1), world, dev)
        devgen = {"value": N * world * args.steps / (gms * 1e-3), "unit": "events/s", "ms_per_step": gms / args.steps,
                  "note": "bg_generate (RAMBO + cuts + helicity/colour draws on the device) + bg_eval per step; fresh events every step"}
        step()      # restore d_out of the resident workload for the checks below
        barrier()   # (bg_eval_host runs on the context's own streams and shares its scratch)

    # end-to-end: host buffers through bg_eval_host (H2D of inputs + D2H of results inside the timed region)
    e2e = None
    if not args.no_e2e:
        k2 = max(3, min(args.steps, 10))
        for _ in range(2):
            bg.bg_eval_host(ctx, N, h_mom, h_hel, h_col, h_out)
        barrier()
        t0 = time.perf_counter()
        for _ in range(k2):
            bg.bg_eval_host(ctx, N, h_mom, h_hel, h_col, h_out)
        barrier()
        dt = max_over_ranks(time.perf_counter() - t0, world, dev)
        h2d = mom.nbytes + (0 if hel is None or mode & bg.BG_HEL_SUM else hel.nbytes) + \
            (0 if col is None or not (mode & bg.BG_COL_GIVEN) else col.nbytes)
        e2e = {"value": N * world * k2 / dt, "unit": "events/s", "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(N * 8), "steps": k2}
        if rank == 0 and not np.allclose(h_out.numpy(), d_out.cpu().numpy(), rtol=0, atol=0, equal_nan=True):
            raise SystemExit("bench.py: host path and device path disagree")

    if rank == 0:
        out_host = d_out.cpu().numpy()
        if not np.all(np.isfinite(out_host)):
            raise SystemExit("bench.py: non-finite |M|^2 in the output")
        # dominant kernel = the FP64 recursion kernel, which evaluates every event; the double-double re-evaluation of
        # the flagged events is reported beside it (precision_auto) and counted in ms_per_step / value
        fp64_kernel_ms = kernel_ms - refine_ms
        achieved_tf = flop_per_event * N / (fp64_kernel_ms * 1e-3) * 1e-12
        traffic, traffic_src = ncu_traffic(kernel_name, n, N)
        roofline = {"bound": "alu", "achieved": achieved_tf, "peak": peak_tf, "unit": "TFLOP/s",
                    "frac": achieved_tf / peak_tf, "traffic": traffic, "traffic_source": traffic_src,
                    "kernel": kernel_name,
                    "peak_source": "bg_fp64_peak_probe (DFMA chains, this run); nominal 148 SM x 64 lanes x 2 x 1.965 GHz = 37.2",
                    "flop_per_event": flop_per_event, "kernel_ms": fp64_kernel_ms,
                    "kernel_share_of_step": fp64_kernel_ms / (total_ms / args.steps),
                    "frac_of_whole_step": flop_per_event * N / (total_ms / args.steps * 1e-3) * 1e-12 / peak_tf}
        cpu = None
        parity = None
        if not args.no_cpu_baseline and not args.lc and not args.continuous and not args.comc:    # no batched oracle entry for these
            import oracle
            S = cpu_sample_size(args, n, N)
            sample = ev.head(S)
            oracle_eval(args, sample.head(max(64, S // 16)))
            reps, dt = 0, 0.0
            t0 = time.perf_counter()
            while reps < 1 or (dt < 2.0 and reps < 2000):      # small workloads are repeated up to ~2 s of wall time
                ref = oracle_eval(args, sample)
                reps += 1
                dt = time.perf_counter() - t0
            err = np.abs(out_host[:S] - ref) / np.abs(ref)
            cpu = {"value": S * reps / dt, "unit": "events/s", "cores": oracle.max_threads(), "kind": "oracle",
                   "sample": f"first {S} events of the workload x {reps} pass(es), {dt:.2f} s wall",
                   "median_rel_diff_gpu_vs_oracle": float(np.median(err))}
            S1 = max(64, S // (4 * oracle.max_threads()))
            t0 = time.perf_counter()
            oracle_eval(args, ev.head(S1), threads=1)
            cpu["one_core"] = {"value": S1 / (time.perf_counter() - t0), "unit": "events/s", "sample": f"first {S1} events"}
            # parity of the default path against the extended-precision oracle on a stated sample
            St = truth_sample_size(n, N) * 4 if args.config != 2 else 1024
            St = min(St, N)
            sub = ev.head(St)
            if args.config == 0:
                truth = oracle.cobg_full_colour(sub.mom, None, prec="long double")
            elif args.config == 2:
                truth = oracle.cobg_full_colour(sub.mom, sub.hel, prec="long double")
            else:
                truth = oracle.cdbg(sub.mom, sub.hel, sub.col, prec="long double")
            terr = np.abs(out_host[:St] - truth) / np.abs(truth)
            parity = {"max_rel_err_vs_long_double": float(terr.max()), "median": float(np.median(terr)),
                      "n_over_1e-11": int(np.sum(terr > 1e-11)), "sample": f"first {St} events"}
        line = {"metric": "n-gluon |M|^2 events/sec", "value": value, "unit": "events/s",
                "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
                "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": name, "n": n, "events_per_step_per_gpu": N, "mode": hex(mode),
                           "l2": "inputs larger than L2" if mom.nbytes > 126e6 else "inputs fit L2 (no flush; "
                           "compute-bound kernel, compulsory traffic 35n+8 B/event)",
                           "kernel": kernel_name, "current_bytes_per_event": bg.bg_current_bytes_per_event(ctx)},
                "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_step * args.steps,
                "roofline": roofline, "cpu_baseline": cpu}
        if devgen is not None:
            line["generate_on_device"] = devgen
        line["parity"] = parity
        prec_now = 2 if auto_default else (args.precision if args.precision is not None else 0)
        line["config"]["precision"] = {0: "FP64", 1: "double-double (all events)", 2: "FP64 + conditioning flag + "
                                       "double-double re-evaluation of the flagged events (default)"}.get(prec_now, str(prec_now))
        if auto_default:
            # the FP64-only path (BG_OPT_PRECISION = 0) timed beside the default one, same events
            bg.bg_set_option(ctx, bg.BG_OPT_PRECISION, 0)
            for _ in range(3):
                step()
            torch.cuda.synchronize()
            f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            f0.record(stream)
            for _ in range(args.steps):
                step()
            f1.record(stream)
            torch.cuda.synchronize()
            ms0 = f0.elapsed_time(f1) / args.steps
            bg.bg_set_option(ctx, bg.BG_OPT_PRECISION, 2)
            line["precision_auto"] = {"flagged_frac": flagged / N, "second_fp64_frac": second / N, "reevaluation_ms": refine_ms,
                                      "overhead_pct": 100.0 * (total_ms / args.steps / ms0 - 1.0),
                                      "fp64_only_events_per_s": N / (ms0 * 1e-3), "fp64_only_ms_per_step": ms0}
        if default_line and not args.no_configs:
            # every BASELINE.json config in the same record: C1, C3, C4 and the C5 sweep n = 4..12 ("events/s vs n")
            import oracle as oracle_mod
            ksteps = max(3, min(args.steps, 10))
            cfgs = {}
            with_cpu = not args.no_cpu_baseline
            cfgs["C1"] = measure_config(bg, wl, oracle_mod, dev, 0, 4, max(ksteps, 20), peak_tf, with_cpu)
            cfgs["C3"] = measure_config(bg, wl, oracle_mod, dev, 2, 7, ksteps, peak_tf, with_cpu)
            cfgs["C4"] = measure_config(bg, wl, oracle_mod, dev, 3, 9, ksteps, peak_tf, with_cpu)
            cfgs["COBG_n8"] = measure_config(bg, wl, oracle_mod, dev, 2, 8, 3, peak_tf, with_cpu)
            cfgs["C5"] = {str(k): measure_config(bg, wl, oracle_mod, dev, 4, k, ksteps, peak_tf, with_cpu) for k in range(4, 13)}
            line["configs"] = cfgs
            line["next_rows"] = measure_next_rows(bg, wl, dev)
        print(json.dumps(line), flush=True)
    bg.bg_destroy(ctx)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
