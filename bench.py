#!/usr/bin/env python
"""bench.py — site-updates/s of the fused Abelian-Higgs leapfrog step on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--size 1024] [--impl ours|reference]
                    [--diag-every M] [--pre-steps P] [--sustained-steps S]

One "step" = one pass of the whole hot path over the lattice.  Workload at
N=1: BASELINE.json configs[3] — 1024^3 periodic lattice, dx=0.5, dt=0.1, fp32 SoA with ping-pong
buffers (85.9 GB), lambda=2, e=1, sigma=1, radiation era, s=1, seeded random-phase IC, no
diagnostics.  The path does not shard: with --gpus N each
rank evolves its own replica of the same lattice (a different seed), value = all ranks' site-updates
divided by the slowest rank's device time, scaling "weak".  Started without a torchrun environment,
`--gpus N` (N > 1) re-executes itself under `python -m torch.distributed.run` with N ranks on 127.0.0.1.

Order of the device-timed windows (all CUDA events on the launching stream, max over ranks):
  W warm-up steps -> one K-step window straight after the warm-up (`roofline.burst`: the board has not reached
  its power cap yet) -> one S-step window (`roofline.sustained`, S = 200: BASELINE configs[3]'s "steady-state
  throughput timed over 200 steps") -> R = 3 repetitions of the K-step window with the board in that steady state.
  The top-level `value` / `ms_per_step` / `roofline` are the MEDIAN repetition ("3 repetitions, report
  median and best"); `repetitions` lists all three and the best.  `clocks` spans the sustained window and the
  repetitions (continuous load), so it holds enough samples to mean something.

Prints ONE JSON line on rank 0.  `--impl reference` times the fp64 CPU oracle (oracle/) on the host
cores on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import socket
import subprocess
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "site-updates/sec at 1024^3 fp32 on 1 B200; % of HBM roofline (80 B/site)"
UNIT = "site-updates/s"
BYTES_PER_SITE = 80.0          # 10 fp32 read + 10 fp32 written
DX, DT, TAU0 = 0.5, 0.1, 1.0
NOMINAL_HBM_GBS = 8000.0       # the metric's own denominator (8 TB/s)
REPS = 3                       # repetitions of the K-step timed window ("report median and best")
FALLBACK_HBM_GBS = 6650.0      # B200_PROFILING.md fallback


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--size", type=int, default=1024, help="lattice extent N (N^3 sites)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--kernel", default="auto", choices=["auto", "site", "tiled"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--diag-every", type=int, default=0, help="fused diagnostics every n steps (0 = none)")
    ap.add_argument("--diag-sums-only", action="store_true",
                    help="with --diag-every: ah_step_diag_sums (xi_L, <v^2>, Gauss; no winding), the paper's timed set")
    ap.add_argument("--pre-steps", type=int, default=0,
                    help="untimed steps before the warm-up (starts the timed window at a later epoch tau)")
    ap.add_argument("--sustained-steps", type=int, default=200,
                    help="after the K timed steps, time a further window of this many steps (0 = skip) and report it "
                         "as roofline.sustained: the number the board holds under its power cap")
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "slabs"],
                    help="N > 1: independent replicas (default; BASELINE north_star keeps one lattice on one GPU) or ONE "
                         "lattice of size x size x (N size) cut into z slabs with a per-step exchange of boundary planes "
                         "over NCCL (SURVEY 8(f)2; untimed on this 1-GPU pool)")
    ap.add_argument("--seed", type=int, default=1,
                    help="seed of the random-phase initial condition (SURVEY 8(d): seeds 1-3 for run-to-run variance)")
    ap.add_argument("--oracle-leg", default="", help=argparse.SUPPRESS)   # "n,steps": one oracle timing (cpu_baseline's child)
    ap.add_argument("--selftest-launcher", action="store_true",
                    help="CPU-only check of the multi-rank launch path (gloo): no kernels, synthetic per-rank timings")
    return ap.parse_args()


TAU_REF = TAU0 + DT * (20 + 200)   # a(tau) = 1 after its 20 warm-up + 200 timed steps (reading #6)


def workload_params(n):
    # configs[3]: radiation era (p=1), s=1.  tau_ref is a constant of the workload: it does not move with --steps,
    # --warmup, --pre-steps or --sustained-steps, so every invocation times the same physical configuration.
    return dict(dx=DX, lambda0=2.0, e0=1.0, sigma=1.0, s=1.0, p=1.0, tau_ref=TAU_REF, alpha=2.0, compact=1)


def measured_peak():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return float(json.loads(p.read_text())["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def recorded_traffic(n, kernel_name):
    """(DRAM bytes per launch, source) of the dominant kernel from the committed ncu --set full captures, or (None, None).

    The figure is NOT measured in this run (a number taken under a profiler is never a bench value, and the bench
    does not run under one): it is read from profiles/traffic.csv, which names the capture each row came from."""
    p = ROOT / "profiles" / "traffic.csv"
    if not p.exists():
        return None, None
    try:
        import csv
        with open(p, newline="") as fh:
            for rec in csv.DictReader(fh):
                if int(rec["size"]) == n and rec["kernel"] == kernel_name:
                    return float(rec["dram_bytes_per_launch"]), f"profiles/traffic.csv (ncu --set full, builder-run): {rec['source']}"
    except Exception:
        return None, None
    return None, None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            parts = [x.strip() for x in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
                power.append(float(parts[2]))
            except ValueError:
                continue
            for name, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# --------------------------------------------------------------------------- oracle (CPU) legs

def oracle_rate(params, n_sample, steps, seed=1):
    """Time the oracle, as it stands, for `steps` steps on an n_sample^3 lattice of the same workload."""
    from oracle import ah_oracle as o
    P = o.make_params(n_sample, **params)
    f = o.init_fields(P, seed)
    t0 = time.perf_counter()
    o.step(P, f, steps, TAU0, DT)
    el = time.perf_counter() - t0
    return n_sample ** 3 * steps / el, el, o.num_threads()


def cpu_model():
    try:
        for ln in Path("/proc/cpuinfo").read_text().splitlines():
            if ln.lower().startswith("model name"):
                return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_leg_single_thread(n_sample, steps):
    """The same oracle timing in a child process whose OpenMP runtime is limited to ONE thread (the oracle has no
    thread-count call of its own and is not given one for this: OMP_NUM_THREADS must be set before it loads)."""
    env = dict(os.environ, OMP_NUM_THREADS="1")
    res = subprocess.run([sys.executable, str(Path(__file__).resolve()), "--oracle-leg", f"{n_sample},{steps}"], env=env,
                         capture_output=True, text=True, timeout=600)
    if res.returncode != 0:
        return {"error": (res.stderr or res.stdout)[-300:]}
    return json.loads(res.stdout.strip().splitlines()[-1])


def run_oracle_leg(spec):
    n_sample, steps = (int(v) for v in spec.split(","))
    rate, el, threads = oracle_rate(workload_params(n_sample), n_sample, steps)
    print(json.dumps({"lattice": f"{n_sample}^3", "steps": steps, "threads": threads, "value": rate, "unit": UNIT,
                      "seconds": el}), flush=True)
    return 0


def cpu_baseline(params):
    """SURVEY 8(d) "oracle timing beside it": the fp64 oracle, as it stands, on 64^3 x 160 steps and 256^3 x 10 steps,
    with OpenMP on all host cores (in this process) and single-threaded (child process); step counts of the slower
    legs are cut so that the whole baseline stays within ~30 s of CPU work, and each leg says what it ran."""
    legs = []

    def leg(n_s, steps, rate, el, threads):
        legs.append({"lattice": f"{n_s}^3", "steps": steps, "threads": threads, "value": rate, "unit": UNIT, "seconds": el})

    cal, _, _ = oracle_rate(params, 64, 2)                         # calibration: sizes the legs below
    steps64 = max(1, min(160, int(6.0 * cal / 64 ** 3)))           # 160 steps (BASELINE configs[0]) on any recent host
    rate64, el, threads = oracle_rate(params, 64, steps64)
    leg(64, steps64, rate64, el, threads)
    steps256 = max(1, min(10, int(8.0 * rate64 * 3 / 256 ** 3)))   # larger lattices run ~3x the 64^3 rate
    rate, el256, threads = oracle_rate(params, 256, steps256)
    leg(256, steps256, rate, el256, threads)
    # single thread: assume at best perfect scaling to size the legs (~10 s and ~6 s)
    one = max(rate / max(threads, 1), 1.0)
    s64 = max(1, min(160, int(10.0 * one / 64 ** 3)))
    s256 = max(1, min(10, int(6.0 * one / 256 ** 3)))
    for n_s, st in ((64, s64), (256, s256)):
        r = oracle_leg_single_thread(n_s, st)
        legs.append(r if "error" in r else {k: r[k] for k in ("lattice", "steps", "threads", "value", "unit", "seconds")})
    return {"value": rate, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": f"256^3 sub-lattice of the same workload (same parameters, seeded random-phase IC), "
                      f"{steps256} leapfrog steps, fp64, {threads} OpenMP threads, {el256:.1f} s; the other legs "
                      f"(64^3 up to 160 steps, single-threaded runs) are under 'legs'",
            "legs": legs, "host_cpus": os.cpu_count(), "cpu_model": cpu_model(),
            "compiler": "gcc -O2 -std=c99 -fopenmp -ffp-contract=off (oracle/ah_oracle.py build())"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    n = args.size
    params = workload_params(n)
    from oracle import ah_oracle as o
    rate64, _, threads = oracle_rate(params, 64, 2)
    budget_s = 150.0
    n_s = 64
    for cand in (96, 128, 192, 256):
        if (args.steps + args.warmup) * cand ** 3 / (rate64 * 3) <= budget_s:
            n_s = cand
    P = o.make_params(n_s, **params)
    f = o.init_fields(P, 1)
    o.step(P, f, args.warmup, TAU0, DT)
    t0 = time.perf_counter()
    o.step(P, f, args.steps, TAU0 + args.warmup * DT, DT)
    el = time.perf_counter() - t0
    value = n_s ** 3 * args.steps / el
    sample = (f"each step = one oracle leapfrog step on a {n_s}^3 sub-lattice of the {n}^3 workload "
              f"(same parameters and IC recipe), fp64, {threads} OpenMP threads")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{n}^3 periodic lattice, dx=0.5, dt=0.1, lambda=2, e=1, sigma=1, radiation era, s=1, "
                               f"seeded random-phase IC, no diagnostics (BASELINE configs[3])", "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------- CUDA arm

def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_2005_14454_b200 import replicas
    rank, local, world = replicas.rank_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    from paper_2005_14454_b200 import build, binding
    build.build()

    n, K, W = args.size, args.steps, max(args.warmup, 3)
    params = workload_params(n)
    if args.decomp == "slabs":
        return run_slabs(args, torch, dist, binding, replicas, params, rank, local, world)
    sim = binding.Simulation(params=binding.make_params(n, **params), device=f"cuda:{local}")
    if args.kernel != "auto":
        sim.set_kernel({"site": binding.KERNEL_SITE, "tiled": binding.KERNEL_TILED}[args.kernel])
    kernel_used = {binding.KERNEL_SITE: "site_step_kernel", binding.KERNEL_TILED: "tiled_step_kernel"}[sim.get_kernel()]
    sites = float(n) ** 3
    stream = sim.stream

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def advance(nsteps, tau):
        if args.diag_every > 0:
            return len(sim.step_diag(nsteps, tau, DT, args.diag_every, winding=not args.diag_sums_only))
        sim.step(nsteps, tau, DT)
        return 0

    def timed_window(nsteps, tau, sample_clocks=True):
        """(max-over-ranks ms, whole-job units, launches, clocks) of nsteps steps from tau, device-timed."""
        barrier()
        sampler = ClockSampler(local) if (sample_clocks and rank == 0) else None
        if sampler:
            sampler.start()
        l0 = sim.launch_count()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(stream)
        advance(nsteps, tau)
        ev1.record(stream)
        barrier()
        ms_local = ev0.elapsed_time(ev1)
        launches = sim.launch_count() - l0
        clocks = sampler.stop() if sampler else None
        ms, units = replicas.aggregate(ms_local, sites * nsteps, dist if world > 1 else None, device="cuda")
        return ms, units, launches, clocks

    def window_record(nsteps, ms_w, units_w, clocks_w):
        return {"steps": nsteps, "ms_per_step": ms_w / nsteps, "value": replicas.throughput(ms_w, units_w), "unit": UNIT,
                "clocks": clocks_w}

    # ---- device-resident throughput
    sim.init_fields(replicas.replica_seed(args.seed, rank))
    tau = TAU0
    if args.pre_steps > 0:
        sim.step(args.pre_steps, tau, DT)
        tau += args.pre_steps * DT
    advance(W, tau)
    tau += W * DT

    # (1) K steps straight after the warm-up: the board is still below its power cap
    ms_b, units_b, _, clocks_b = timed_window(K, tau)
    tau += K * DT
    burst = window_record(K, ms_b, units_b, clocks_b)

    # (2) the longer window (BASELINE configs[3]: "steady-state throughput timed over 200 steps"), which also brings
    # the board to the clocks it holds under its power cap; the clock sampler of the top-level record starts here
    span_sampler = ClockSampler(local) if rank == 0 else None
    if span_sampler:
        span_sampler.start()
    sustained = None
    if args.sustained_steps > 0:
        ms_s, units_s, _, clocks_s = timed_window(args.sustained_steps, tau)
        tau += args.sustained_steps * DT
        sustained = window_record(args.sustained_steps, ms_s, units_s, clocks_s)

    # (3) the K timed steps, REPS times, in that steady state; the median repetition is the line's value
    tau_timed = tau
    reps = []
    for _ in range(REPS):
        ms_r, units_r, launches_r, _ = timed_window(K, tau, sample_clocks=False)
        tau += K * DT
        reps.append((ms_r, units_r, launches_r))
    clocks = span_sampler.stop() if span_sampler else None
    ms, units, launches = sorted(reps)[len(reps) // 2]
    value = replicas.throughput(ms, units)
    repetitions = {"n": REPS, "steps_each": K, "ms_per_step": [r[0] / K for r in reps],
                   "values": [replicas.throughput(r[0], r[1]) for r in reps],
                   "median_value": value, "best_value": max(replicas.throughput(r[0], r[1]) for r in reps),
                   "what": "back-to-back K-step windows after the sustained window; the line's value is the median"}

    # ---- end to end through the C ABI with HOST buffers: upload, K steps, download
    e2e = None
    if not args.no_e2e:
        nbytes = int(sites) * 10 * 4
        try:
            host = torch.empty(int(sites) * 10, dtype=torch.float32, pin_memory=True)
            pinned = True
        except Exception:
            host = torch.empty(int(sites) * 10, dtype=torch.float32)
            pinned = False
        sim.get_fields_ptr(host.data_ptr())          # a real state as the host-side input
        barrier()
        t0 = time.perf_counter()
        sim.set_fields_ptr(host.data_ptr())          # H2D inside the timed region
        sim.step(K, tau_timed, DT)
        sim.get_fields_ptr(host.data_ptr())          # D2H (synchronises)
        torch.cuda.synchronize()
        el = time.perf_counter() - t0
        el_ms, units_e = replicas.aggregate(el * 1e3, sites * K, dist if world > 1 else None, device="cuda")
        el = el_ms * 1e-3
        e2e = {"value": units_e / el, "unit": UNIT, "h2d_bytes_per_step": nbytes / K,
               "d2h_bytes_per_step": nbytes / K, "pinned_host": pinned, "seconds": el,
               "what": f"ah_set_fields(host) + ah_step({K}) + ah_get_fields(host), wall clock"}
        del host

    if rank == 0:
        peak, peak_src = measured_peak()
        diag = args.diag_every > 0
        kernel_name = kernel_used
        # one step-kernel launch per step; on diagnostic steps the launch is the DIAG instantiation of the same kernel
        avg_launch_ms = ms / K
        achieved = BYTES_PER_SITE * sites / (avg_launch_ms * 1e-3) / 1e9
        traffic, traffic_src = recorded_traffic(n, kernel_name + ("<DIAG>" if diag else ""))
        roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                    "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src, "kernel": kernel_name,
                    "algorithmic_bytes_per_launch": BYTES_PER_SITE * sites,
                    "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS,
                    "timing": "CUDA events on the launching stream around the K timed steps of the median repetition "
                              "(the board already at the clocks it sustains: see the module docstring); avg = elapsed/K "
                              "(each step = 1 tiled_step_kernel launch + 1 conditional-redo launch that exits "
                              "at once, ~2 us; see profiles/ launch list)"
                              + (f" (every {args.diag_every}th step is the DIAG instantiation + 2 small launches; "
                                 "the average is over all steps)" if diag else "")}
        for name, rec in (("sustained", sustained), ("burst", burst)):
            if rec is not None:
                ach = BYTES_PER_SITE * sites / (rec["ms_per_step"] * 1e-3) / 1e9
                rec.update(achieved=ach, frac=ach / peak, frac_of_nominal_8TBs=ach / NOMINAL_HBM_GBS)
                roofline[name] = rec
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"{n}^3 periodic lattice, dx=0.5, dt=0.1, fp32 SoA ping-pong ({20 * 4 * sites / 1e9:.1f} GB), "
                                   f"lambda=2, e=1, sigma=1, radiation era, s=1, seeded random-phase IC, "
                                   f"{'no diagnostics' if not diag else 'fused diagnostics every %d steps' % args.diag_every}"
                                   f"{' (sums only: xi_L, <v^2>, Gauss; no winding)' if diag and args.diag_sums_only else ''}"
                                   f"{' (BASELINE configs[3])' if n == 1024 and not diag else ''}"
                                   f"{' (BASELINE configs[4] row)' if diag and args.diag_every == 10 else ''}",
                       "kernel": kernel_name, "parallelism": "replicas only" if world > 1 else "single GPU",
                       "tau_at_timed_window": tau_timed, "tau_ref": TAU_REF, "seed": args.seed,
                       "windows": f"warm-up {W} -> burst {K} -> sustained {args.sustained_steps} -> {REPS} x {K} timed "
                                  "(value = median repetition)",
                       "l2": "working set (80 B/site x N^3) exceeds the 126 MB L2 for N >= 128; no flush needed"
                             if n >= 128 else "working set fits in L2 (small-lattice case)"},
            "pct_of_8TBs_roofline": 100.0 * value / world * BYTES_PER_SITE / (NOMINAL_HBM_GBS * 1e9),
            "roofline": roofline, "gpu_launches": int(launches), "clocks": clocks, "repetitions": repetitions,
        }
        if e2e is not None:
            line["e2e"] = e2e
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(params)
        print(json.dumps(line), flush=True)
    sim.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_slabs(args, torch, dist, binding, replicas, params, rank, local, world):
    """--decomp slabs: ONE periodic lattice of size x size x (world * size) sites, one z slab per rank, boundary planes
    exchanged over torch.distributed (NCCL) every step, overlapped with the update of the interior (weak scaling in z)."""
    n, K, W = args.size, args.steps, max(args.warmup, 3)
    if world == 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", str(free_port()))
        dist.init_process_group("gloo", rank=0, world_size=1)
    P = binding.make_params(n, n, n * world, **params)
    ds = binding.DistributedSlab(P, dist, device=f"cuda:{local}")
    ds.slab.init_fields(1)
    ds.step(W, TAU0, DT)
    torch.cuda.synchronize()
    dist.barrier()
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = ds.slab.launch_count()
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
    ev0.record(ds.slab.stream)
    ds.step(K, TAU0 + W * DT, DT)
    ev1.record(ds.slab.stream)
    torch.cuda.synchronize()
    dist.barrier()
    clocks = sampler.stop() if sampler else None
    ms, units = replicas.aggregate(ev0.elapsed_time(ev1), float(n) ** 3 * K, dist if world > 1 else None,
                                   device="cuda" if dist.get_backend() == "nccl" else "cpu")
    if rank == 0:
        value = replicas.throughput(ms, units)
        peak, peak_src = measured_peak()
        # per GPU: one slab of n^3 sites per step = 3 step-kernel launches (two boundary planes, then the interior)
        achieved = BYTES_PER_SITE * float(n) ** 3 / (ms / K * 1e-3) / 1e9
        roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                    "traffic": None, "peak_source": peak_src, "kernel": "tiled_step_kernel (per slab: 2 boundary launches "
                    "+ 1 interior launch per step)", "algorithmic_bytes_per_launch": BYTES_PER_SITE * float(n) ** 3,
                    "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS,
                    "timing": "CUDA events on the slab's compute stream around the K timed steps, max over ranks; "
                              "per-GPU bytes = 80 B x the slab's own sites per step"}
        print(json.dumps({
            "roofline": roofline, "clocks": clocks, "e2e": None, "cpu_baseline": None,
            "note": "z-slab decomposition (SURVEY 8(f)2), outside BASELINE's single-GPU north_star: no host-buffer (e2e) "
                    "leg and no oracle leg are run for it; the replica line (default --decomp) carries both",
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms / K,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"ONE {n}x{n}x{n * world} periodic lattice in {world} z slab(s), radiation era, s=1, "
                                   "seeded random-phase IC, no diagnostics", "parallelism": f"z slabs x{world}, halo exchange "
                                   "of 6 planes per direction and step on a communication stream"},
            "pct_of_8TBs_roofline": 100.0 * value / world * BYTES_PER_SITE / (NOMINAL_HBM_GBS * 1e9),
            "gpu_launches": int(ds.slab.launch_count() - l0)}), flush=True)
    ds.slab.close()
    dist.destroy_process_group()
    return 0


# ------------------------------------------------------------------------------- launcher

def free_port():
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        return sk.getsockname()[1]


def relaunch_under_torchrun(args):
    """`python bench.py --gpus N` without a torchrun environment: start N ranks (one per GPU) of this same command."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()), str(Path(__file__).resolve())] + sys.argv[1:]
    return subprocess.call(cmd)


def run_selftest_launcher(args):
    """The multi-rank path without a GPU (tests/test_replicas_gloo.py): every rank reports a synthetic device time and
    unit count through the same replicas.aggregate / JSON code as the CUDA arm, over gloo."""
    import torch.distributed as dist
    from paper_2005_14454_b200 import replicas
    rank, local, world = replicas.rank_world()
    if world > 1:
        dist.init_process_group("gloo")
    ms_local, units_local = 10.0 * (rank + 1), 1000.0 * args.steps
    ms, units = replicas.aggregate(ms_local, units_local, dist if world > 1 else None, device="cpu")
    if rank == 0:
        print(json.dumps({"selftest": "launcher", "n_gpus": world, "steps": args.steps, "ms": ms, "units": units,
                          "value": replicas.throughput(ms, units), "seed_of_last_rank": replicas.replica_seed(1, world - 1)}),
              flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    args = parse()
    if args.oracle_leg:
        return run_oracle_leg(args.oracle_leg)
    if args.gpus < 1:
        raise SystemExit("--gpus must be >= 1")
    in_torchrun = "WORLD_SIZE" in os.environ and "RANK" in os.environ
    if in_torchrun and int(os.environ["WORLD_SIZE"]) != args.gpus:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={os.environ['WORLD_SIZE']}")
    if args.gpus > 1 and not in_torchrun and (args.impl == "ours" or args.selftest_launcher):
        return relaunch_under_torchrun(args)
    if args.selftest_launcher:
        return run_selftest_launcher(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
