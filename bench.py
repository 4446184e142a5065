#!/usr/bin/env python
"""bench.py -- QFT time / DFT-equivalent GFLOP/s / HBM roofline on B200 (BASELINE.json's metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--n 30] [--k K] [--impl ours|reference]

A "step" is one pass of the whole hot path: one qft_execute (every fused pass, the folded bit
reversal and the normalisation) over one synthetic 2^n complex64 state that is already resident in
HBM.  Default workload: n = 30 exact QFT (BASELINE config 4 with k = 30: 8 GiB state, the largest
configuration whose full parity check also runs in the test suite; n = 33 is reachable with --n 33).
The state is far larger than the 126 MB L2, so no L2 flush is needed between iterations.

With N > 1 (torchrun) every rank transforms its own state (replicas only: the path does not shard,
DESIGN.md section "multi-GPU"); value = all ranks' work / max-over-ranks time, "scaling": "weak".

The default run also times, briefly, n = 26 and n = 33 and one batched shape ("sweep" / "batched" in the
JSON line, each with its own fraction of the HBM roofline), and the CPU oracle on whole circuits at
n = 22 and n = 26 ("cpu_baseline").

--impl reference times the CPU oracle (oracle/, as it stands) on the host cores: every step is one WHOLE
gate-by-gate circuit at the largest n <= 26 for which steps + warmup circuits fit the time budget (a bounded
sample of the n = 30 workload: same circuit family, smaller state); see DESIGN.md "measurement".
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--n", type=int, default=30, help="qubits (state = 2^n complex64)")
    ap.add_argument("--k", type=int, default=None, help="AQFT cutoff (default: exact)")
    ap.add_argument("--max-fused", type=int, default=13)
    ap.add_argument("--tile-bits", type=int, default=0)
    ap.add_argument("--hub-bits", type=int, default=0)
    ap.add_argument("--flags", type=int, default=0)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-variants", action="store_true")
    ap.add_argument("--extrapolate-cpu", action="store_true",
                    help="also estimate the oracle's time at the bench n from a few gates (labelled as extrapolated)")
    ap.add_argument("--sweep", default="26,33", help="comma list of extra n to time briefly ('' = none)")
    ap.add_argument("--sweep-fused", default="26:2,26:4,26:6",
                    help="comma list of n:max_fused_qubits timed briefly (BASELINE config 3; '' = none)")
    ap.add_argument("--small-n", default="20,22", help="comma list of launch-bound sizes to time over 1000 back-to-back "
                                                       "transforms ('' = none)")
    ap.add_argument("--batched", default="12:16,16:12,22:6", help="comma list of n:log2_batch pairs to time briefly (batched "
                                                       "plans; '' = none), e.g. 10:18,16:12")
    return ap.parse_args()


def measured_peak_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [l for (t, l) in self.lines if t0 - 0.05 <= t <= t1 + 0.15] or [l for (_, l) in self.lines]
        for l in rows:
            p = [x.strip() for x in l.split(",")]
            try:
                sm.append(float(p[0]))
                smax = float(p[1])
                for nm, v in zip(names, p[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                continue
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": smax, "reasons": sorted(reasons),
                "samples": len(sm)}


def dist_setup(args):
    import torch

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist

        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        backend = "nccl" if torch.cuda.is_available() else "gloo"
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return world, rank, local


def barrier(world):
    if world > 1:
        import torch.distributed as dist

        dist.barrier()


def max_over_ranks(x: float, world: int, device) -> float:
    if world == 1:
        return x
    import torch
    import torch.distributed as dist

    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def time_config(qft, torch, n, k, args, steps, warmup, per_pass=True, log2_batch=0, max_fused=None):
    """Device-resident timing of qft_execute on a fresh synthetic state; returns a dict."""
    import qft_inputs as qi

    dev = torch.device("cuda", torch.cuda.current_device())
    plan = qft.Plan(n, n if k is None else k, args.max_fused if max_fused is None else max_fused, -1,
                    qft.QFT_NORM_UNITARY, args.tile_bits,
                    args.hub_bits, args.flags, log2_batch)
    n = n + log2_batch  # address bits of the state
    state = torch.empty(1 << n, dtype=torch.complex64, device=dev)
    if n <= 27:
        state.copy_(torch.from_numpy(qi.gaussian(n, 1)))
    else:
        qi.gaussian_device(n, 2, device=dev, out=state)
    stream = torch.cuda.current_stream(dev)
    sptr = stream.cuda_stream
    for _ in range(warmup):
        qft.qft_execute(plan.handle, state.data_ptr(), sptr)
    torch.cuda.synchronize()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    ev[0].record(stream)
    for i in range(steps):
        qft.qft_execute(plan.handle, state.data_ptr(), sptr)
        ev[i + 1].record(stream)
    torch.cuda.synchronize()
    total_ms = ev[0].elapsed_time(ev[steps])
    per_step = sorted(ev[i].elapsed_time(ev[i + 1]) for i in range(steps))
    res = {"plan": plan, "state": state, "total_ms": total_ms, "median_ms": per_step[len(per_step) // 2],
           "min_ms": per_step[0], "passes": plan.num_passes, "launches": plan.num_launches}
    if per_pass:
        # per-pass CUDA-event timing (same stream), cycling through the passes in order so that the
        # state keeps going through whole transforms
        npass = plan.num_passes
        reps = max(3, min(steps, 10))
        acc = [0.0] * npass
        for _ in range(reps):
            evs = [torch.cuda.Event(enable_timing=True) for _ in range(npass + 1)]
            evs[0].record(stream)
            for p in range(npass):
                qft.qft_execute_pass(plan.handle, p, state.data_ptr(), sptr)
                evs[p + 1].record(stream)
            torch.cuda.synchronize()
            for p in range(npass):
                acc[p] += evs[p].elapsed_time(evs[p + 1])
        res["pass_ms"] = [a / reps for a in acc]
    return res


def oracle_full(n, k, warmup=1, trials=3):
    """Time the oracle's WHOLE gate-by-gate circuit (every H, controlled-R_m and swap, fp64) on a seeded
    Gaussian state of 2^n amplitudes: `warmup` untimed runs, then `trials` timed ones.  Returns (times, cores)."""
    import oracle
    import qft_inputs as qi

    x = qi.gaussian(n, 1)
    for _ in range(warmup):
        oracle.qft(x, n if k is None else k)
    times = []
    for _ in range(trials):
        t0 = time.perf_counter()
        oracle.qft(x, n if k is None else k)
        times.append(time.perf_counter() - t0)
    return times, oracle.max_threads()


def oracle_sample(n, k, reps=1):
    """EXTRAPOLATION, reported only as a labelled extra: time a few gates of the n-qubit circuit on the full 2^n fp64
    state (H, controlled-R_m and SWAP at low, middle and high qubit positions) and scale by gate type:
    t = n_H t_H + n_CR t_CR + n_SWAP t_SWAP."""
    import numpy as np

    import oracle

    gates = oracle.gate_list(n, n if k is None else k)
    n_h = int((gates[:, 0] == oracle.GATE_H).sum())
    n_cr = int((gates[:, 0] == oracle.GATE_CR).sum())
    n_sw = int((gates[:, 0] == oracle.GATE_SWAP).sum())
    s = np.zeros(1 << n, dtype=np.complex128)
    s[:] = 1.0 / math.sqrt(1 << n)
    hs = [g for g in gates if g[0] == oracle.GATE_H]
    crs = [g for g in gates if g[0] == oracle.GATE_CR]
    sws = [g for g in gates if g[0] == oracle.GATE_SWAP]
    pick = lambda v: [v[0], v[len(v) // 2], v[-1]] if len(v) >= 3 else list(v)
    sample = pick(hs) + pick(crs) + pick(sws)[:2]
    t = {0: [], 1: [], 2: []}
    for _ in range(reps):
        for g in sample:
            t0 = time.perf_counter()
            oracle.apply_gate_inplace(s, g)
            t[int(g[0])].append(time.perf_counter() - t0)
    mean = lambda v: sum(v) / len(v) if v else 0.0
    est = n_h * mean(t[0]) + n_cr * mean(t[1]) + n_sw * mean(t[2])
    spent = sum(sum(v) for v in t.values())
    desc = (f"EXTRAPOLATED from {len(sample)} of the {len(gates)} gates of the n={n} circuit on the full 2^{n} fp64 "
            f"state as n_H*t_H + n_CR*t_CR + n_SWAP*t_SWAP = {est:.1f} s ({spent:.1f} s measured)")
    return est, spent, desc, oracle.max_threads()


def workload_text(n, k):
    """The workload both arms report (config.workload)."""
    return (f"n={n} {'exact QFT' if k is None else 'AQFT k=%d' % k}: 2^{n} complex64 amplitudes "
            f"({8 * (1 << n) / 2 ** 30:.3g} GiB) per GPU, in place, forward sign, unitary scaling, "
            f"natural order in and out")


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    n = args.n
    steps, warmup = max(1, args.steps), max(0, args.warmup)
    # Every step = one whole oracle circuit.  The n = 30 workload itself (16 GiB of fp64 state, minutes per circuit)
    # does not fit `steps + warmup` circuits into a few minutes, so the step is a bounded sample of it: the same
    # circuit on a 2^n_eff state, n_eff the largest of 26, 24, 22, 20 whose projected total stays under the budget.
    budget_s = 200.0
    n_eff, probe = None, None
    for cand in (26, 24, 22, 20):
        if cand > n:
            continue
        tt, cores = oracle_full(cand, args.k, warmup=0, trials=1)
        n_eff, probe = cand, tt[0]
        if probe * (steps + warmup) <= budget_s:
            break
    if n_eff is None:
        n_eff = n
    warm_left = max(0, warmup - 1)  # the probe was the first warm-up
    times, cores = oracle_full(n_eff, args.k, warmup=warm_left, trials=steps)
    t_step = sum(times) / len(times)
    flops = 5.0 * (1 << n_eff) * n_eff
    gf = flops / t_step / 1e9
    med = sorted(times)[len(times) // 2]
    sample = (f"{steps} timed + {warmup} warm-up WHOLE gate-by-gate oracle circuits (fp64, OpenMP) at n={n_eff} instead of "
              f"n={n}: the largest state for which that many circuits fit {budget_s:.0f} s; mean {t_step:.3f} s, "
              f"median {med:.3f} s per circuit; GFLOP/s = 5 N log2 N / t at n={n_eff}")
    line = {
        "impl": "reference", "metric": "dft_equiv_gflops", "value": gf, "unit": "GFLOP/s", "n_gpus": args.gpus,
        "steps": steps, "warmup": warmup, "ms_per_step": t_step * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_text(n, args.k) if n_eff == n else
                   (workload_text(n, args.k) + f"; THIS ARM's steps are whole circuits at n={n_eff} "
                    f"({8 * (1 << n_eff) / 2 ** 20:.0f} MiB states in complex64 terms, fp64 on the host): a bounded "
                    f"sample of that workload, see cpu_baseline.sample"),
                   "n_qubits": n,
                   "aqft_cutoff_k": n if args.k is None else min(args.k, n),
                   "implementation": "CPU oracle (gate-by-gate fp64, OpenMP)", "sample_n_qubits": n_eff},
        "cpu_baseline": {"value": gf, "unit": "GFLOP/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": gf, "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch

    import paper_2606_18981_b200 as qft

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback for the QFT path)")
    qft.load()
    world, rank, local = dist_setup(args)
    torch.cuda.set_device(local % torch.cuda.device_count())
    dev = torch.device("cuda", torch.cuda.current_device())
    n, steps, warmup = args.n, max(1, args.steps), max(3, args.warmup)
    N = 1 << n
    flops = 5.0 * N * n
    peak, peak_src = measured_peak_gbs()

    # ---- device-resident timing: W warm-ups, then exactly K steps between barriers ----
    import qft_inputs as qi

    plan = qft.Plan(n, n if args.k is None else args.k, args.max_fused, -1, qft.QFT_NORM_UNITARY, args.tile_bits,
                    args.hub_bits, args.flags)
    state = torch.empty(N, dtype=torch.complex64, device=dev)
    if n <= 27:
        state.copy_(torch.from_numpy(qi.gaussian(n, 1)))
    else:
        qi.gaussian_device(n, 2, device=dev, out=state)
    stream = torch.cuda.current_stream(dev)
    sptr = stream.cuda_stream
    for _ in range(warmup):
        qft.qft_execute(plan.handle, state.data_ptr(), sptr)
    torch.cuda.synchronize()
    barrier(world)
    sampler = ClockSampler(torch.cuda.current_device())
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.time()
    e0.record(stream)
    for _ in range(steps):
        qft.qft_execute(plan.handle, state.data_ptr(), sptr)
    e1.record(stream)
    torch.cuda.synchronize()
    t1 = time.time()
    barrier(world)
    total_ms = max_over_ranks(e0.elapsed_time(e1), world, dev)
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    ms_per_step = total_ms / steps
    value = world * flops / (ms_per_step * 1e-3) / 1e9

    # ---- per-pass timing for the roofline of the dominant kernel ----
    npass = plan.num_passes
    nlaunch = plan.num_launches  # kernels one qft_execute enqueues (1 when the plan runs as a single cooperative launch)
    reps = max(3, min(steps, 10))
    acc = [0.0] * npass
    for _ in range(reps):
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(npass + 1)]
        evs[0].record(stream)
        for p in range(npass):
            qft.qft_execute_pass(plan.handle, p, state.data_ptr(), sptr)
            evs[p + 1].record(stream)
        torch.cuda.synchronize()
        for p in range(npass):
            acc[p] += evs[p].elapsed_time(evs[p + 1])
    pass_ms = [a / reps for a in acc]
    desc = plan.describe()
    kernels = [p["kernel"] for p in desc["passes"]]
    # dominant kernel = the kernel kind with the largest share of the step
    share = {}
    for kname, ms in zip(kernels, pass_ms):
        share.setdefault(kname, []).append(ms)
    dom = max(share, key=lambda kk: sum(share[kk]))
    dom_ms = sum(share[dom]) / len(share[dom])
    bytes_per_launch = 16.0 * N  # 8 B read + 8 B written per amplitude per pass
    achieved = bytes_per_launch / (dom_ms * 1e-3) / 1e9
    # measured DRAM bytes per launch of the dominant kernel: a COPY of the figure in the committed ncu --set full
    # capture (profiles/r03_traffic.csv: n, kernel, bytes), null when that file has no row for this (n, kernel)
    traffic, traffic_source = None, None
    try:
        with open(os.path.join(ROOT, "profiles", "r03_traffic.csv")) as fh:
            for row in fh:
                f = [v.strip() for v in row.split(",")]
                if len(f) >= 3 and f[0] == str(n) and f[1] == dom:
                    traffic = float(f[2])
                    traffic_source = ("profiles/r03_traffic.csv (dram__bytes_read.sum + dram__bytes_write.sum of one "
                                      "ncu --set full capture of this kernel at this n; not re-measured in this run)")
    except Exception:
        pass
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_source, "peak_source": peak_src,
                "bytes_per_launch": bytes_per_launch, "launch_ms": dom_ms,
                "pass_ms": pass_ms, "pass_kernels": kernels,
                "step_gbs": npass * bytes_per_launch / (ms_per_step * 1e-3) / 1e9,
                "step_frac": npass * bytes_per_launch / (ms_per_step * 1e-3) / 1e9 / peak}

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region ----
    e2e = None
    if not args.no_e2e:
        try:
            host = torch.empty(N, dtype=torch.complex64).pin_memory()
            host.copy_(state.cpu() if n <= 27 else state.to("cpu", non_blocking=False))
            e2e_steps = max(1, min(steps, 3 if n >= 28 else 10))
            qft.qft_execute_host(plan.handle, host.data_ptr(), sptr)  # warm-up (allocates the plan's device buffer)
            torch.cuda.synchronize()
            barrier(world)
            ta = time.perf_counter()
            for _ in range(e2e_steps):
                qft.qft_execute_host(plan.handle, host.data_ptr(), sptr)
            torch.cuda.synchronize()
            tb = time.perf_counter()
            e2e_ms = max_over_ranks((tb - ta) * 1e3 / e2e_steps, world, dev)
            e2e = {"value": world * flops / (e2e_ms * 1e-3) / 1e9, "unit": "GFLOP/s", "h2d_bytes_per_step": 8 * N,
                   "d2h_bytes_per_step": 8 * N, "ms_per_step": e2e_ms, "steps": e2e_steps,
                   "host_memory": "pinned"}
            del host
        except Exception as exc:  # e.g. not enough pinned host memory
            e2e = {"value": None, "unit": "GFLOP/s", "h2d_bytes_per_step": 8 * N, "d2h_bytes_per_step": 8 * N,
                   "error": str(exc)}

    # ---- the variants of SURVEY.md section 8 (f2) at the same n, briefly: swaps deferred (the paper's own timed mode,
    # PAPER.md:137) and out-of-place execute; reported beside the headline, not part of it ----
    variants = None
    if rank == 0 and world == 1 and not args.no_variants:
        try:
            vsteps = max(3, min(steps, 5))

            def timed(fn):
                for _ in range(2):
                    fn()
                torch.cuda.synchronize()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                for _ in range(vsteps):
                    fn()
                b.record(stream)
                torch.cuda.synchronize()
                return a.elapsed_time(b) / vsteps

            dplan = qft.Plan(n, n if args.k is None else args.k, args.max_fused, -1, qft.QFT_NORM_UNITARY, args.tile_bits,
                             args.hub_bits, args.flags | qft.QFT_FLAG_DEFER_SWAPS)
            d_ms = timed(lambda: qft.qft_execute(dplan.handle, state.data_ptr(), sptr))
            variants = {"steps": vsteps, "defer_swaps": {"ms": d_ms, "passes": dplan.num_passes,
                                                         "gbs": dplan.num_passes * 16.0 * N / (d_ms * 1e-3) / 1e9,
                                                         "roofline_frac": dplan.num_passes * 16.0 * N / (d_ms * 1e-3) / 1e9 / peak}}
            dplan.close()
            free, _ = torch.cuda.mem_get_info()
            if 8 * N * 1.05 < free:
                out = torch.empty_like(state)
                o_ms = timed(lambda: qft.qft_execute_oop(plan.handle, state.data_ptr(), out.data_ptr(), sptr))
                variants["out_of_place"] = {"ms": o_ms, "passes": npass, "gbs": npass * 16.0 * N / (o_ms * 1e-3) / 1e9,
                                            "roofline_frac": npass * 16.0 * N / (o_ms * 1e-3) / 1e9 / peak}
                del out
        except Exception as exc:
            variants = {"error": str(exc)}

    # ---- optional brief sweep over other n (reported, not the headline) ----
    sweep = []
    if args.sweep and rank == 0 and world == 1:
        del state
        plan.close()
        torch.cuda.empty_cache()
        for sn in [int(v) for v in args.sweep.split(",") if v]:
            if sn == n:
                continue
            free, _ = torch.cuda.mem_get_info()
            if 8 * (1 << sn) * 1.05 > free:
                sweep.append({"n": sn, "skipped": "not enough free device memory"})
                continue
            st = 5 if sn >= 32 else 10
            r = time_config(qft, torch, sn, None, args, st, 3, per_pass=True)
            gbs = r["passes"] * 16.0 * (1 << sn) / (r["median_ms"] * 1e-3) / 1e9
            kinds = [p["kernel"] for p in r["plan"].describe()["passes"]]
            slow = max(r["pass_ms"])
            sweep.append({"n": sn, "passes": r["passes"], "ideal_passes": math.ceil(sn / 13), "steps": st,
                          "median_ms": r["median_ms"],
                          "gflops": 5.0 * (1 << sn) * sn / (r["median_ms"] * 1e-3) / 1e9,
                          "gbs": gbs, "roofline_frac": gbs / peak,
                          "slowest_pass_frac": 16.0 * (1 << sn) / (slow * 1e-3) / 1e9 / peak,
                          "pass_ms": r["pass_ms"], "pass_kernels": kinds})
            r["plan"].close()
            del r
            torch.cuda.empty_cache()

    # ---- BASELINE config 3: the fused-window cap (the paper's max_fused_size) swept at n = 26 ----
    fused_sweep = []
    if args.sweep_fused and rank == 0 and world == 1:
        try:
            del state
            plan.close()
        except Exception:  # already released by the sweep
            pass
        torch.cuda.empty_cache()
        for pair in [v for v in args.sweep_fused.split(",") if v]:
            fn, fw = (int(v) for v in pair.split(":"))
            r = time_config(qft, torch, fn, None, args, 10, 3, per_pass=True, max_fused=fw)
            slow = max(r["pass_ms"])
            gbs = r["passes"] * 16.0 * (1 << fn) / (r["median_ms"] * 1e-3) / 1e9
            fused_sweep.append({"n": fn, "max_fused_qubits": fw, "passes": r["passes"], "steps": 10,
                                "median_ms": r["median_ms"],
                                "gflops": 5.0 * (1 << fn) * fn / (r["median_ms"] * 1e-3) / 1e9,
                                "gbs": gbs, "roofline_frac": gbs / peak,
                                "slowest_pass_frac": 16.0 * (1 << fn) / (slow * 1e-3) / 1e9 / peak,
                                "pass_kernels": sorted({p["kernel"] for p in r["plan"].describe()["passes"]})})
            r["plan"].close()
            del r
            torch.cuda.empty_cache()

    batched = []
    if args.batched and rank == 0 and world == 1:
        try:
            del state
        except Exception:  # already released by the sweep
            pass
        torch.cuda.empty_cache()
        for pair in [v for v in args.batched.split(",") if v]:
            bn, bb = (int(v) for v in pair.split(":"))
            r = time_config(qft, torch, bn, None, args, 10, 3, per_pass=True, log2_batch=bb)
            tot = 1 << (bn + bb)
            gbs = r["passes"] * 16.0 * tot / (r["median_ms"] * 1e-3) / 1e9
            batched.append({"n": bn, "log2_batch": bb, "passes": r["passes"], "median_ms": r["median_ms"],
                            "gflops": 5.0 * tot * bn / (r["median_ms"] * 1e-3) / 1e9,
                            "gbs": gbs, "roofline_frac": gbs / peak, "pass_ms": r["pass_ms"]})
            r["plan"].close()
            del r
            torch.cuda.empty_cache()

    # ---- the launch-bound regime (PAPER.md:197's sizes): microseconds per transform over 1000 back-to-back executes ----
    small = []
    if args.small_n and rank == 0 and world == 1:
        torch.cuda.empty_cache()
        for sn in [int(v) for v in args.small_n.split(",") if v]:
            pl = qft.Plan(sn, sn if args.k is None else args.k, args.max_fused, -1, qft.QFT_NORM_UNITARY, args.tile_bits,
                          args.hub_bits, args.flags)
            stt = torch.empty(1 << sn, dtype=torch.complex64, device="cuda")
            torch.view_as_real(stt).normal_()
            stt.mul_(2.0 ** (-(sn + 1) / 2))
            strm = torch.cuda.current_stream()
            for _ in range(20):
                qft.qft_execute(pl.handle, stt.data_ptr(), strm.cuda_stream)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(strm)
            for _ in range(1000):
                qft.qft_execute(pl.handle, stt.data_ptr(), strm.cuda_stream)
            e1.record(strm)
            torch.cuda.synchronize()
            us = e0.elapsed_time(e1)  # ms for 1000 transforms = microseconds per transform
            row = {"n": sn, "transforms": 1000, "us_per_transform": us, "launches_per_transform": pl.num_launches,
                   "gflops": 5.0 * (1 << sn) * sn / (us * 1e-6) / 1e9}
            pl.close()
            del stt
            small.append(row)

    # ---- CPU baseline: the oracle as it stands, WHOLE circuits, rank 0 at N = 1 only ----
    # 1 warm-up + 3 trials, median, at n = 22 (to sit beside PAPER.md:185's 3.86 s / 0.064 s)
    # and n = 26 (the largest size whose whole circuit takes seconds); a bounded sample of the n = 30 workload
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        try:
            torch.cuda.empty_cache()
            t20, cores = oracle_full(20, args.k)
            t22, cores = oracle_full(22, args.k)
            t22k4, cores = oracle_full(22, 4)  # AQFT k = 4 at the paper's size (Fig. 5)
            t26, cores = oracle_full(26, args.k)
            m20, m22, m22k4, m26 = sorted(t20)[1], sorted(t22)[1], sorted(t22k4)[1], sorted(t26)[1]
            cpu_baseline = {"value": 5.0 * (1 << 26) * 26 / m26 / 1e9, "unit": "GFLOP/s", "cores": cores, "kind": "oracle",
                            "sample": ("whole gate-by-gate oracle circuit (fp64, OpenMP), 1 warm-up + 3 trials, median, at "
                                       f"n=26: {m26:.3f} s (value = 5 N log2 N / t there), n=22: {m22:.4f} s (k=4: {m22k4:.4f} s) and n=20: "
                                       f"{m20:.4f} s; bounded "
                                       f"sample of the n={n} workload: same circuit, smaller states"),
                            "seconds_n26": m26, "seconds_n22": m22, "seconds_n20": m20, "seconds_n22_k4": m22k4,
                            "trials_n26": t26, "trials_n22": t22,
                            "gflops_n22": 5.0 * (1 << 22) * 22 / m22 / 1e9}
            if n >= 28 and args.extrapolate_cpu:
                est, spent, sdesc, _ = oracle_sample(n, args.k)
                cpu_baseline["extrapolated_not_measured"] = {"n": n, "seconds": est, "how": sdesc}
        except Exception as exc:
            cpu_baseline = {"value": None, "unit": "GFLOP/s", "cores": os.cpu_count(), "kind": "oracle",
                            "sample": f"failed: {exc}"}

    if rank == 0:
        line = {
            "metric": "dft_equiv_gflops", "value": value, "unit": "GFLOP/s", "n_gpus": world, "steps": steps,
            "warmup": warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_text(n, args.k),
                       "n_qubits": n, "aqft_cutoff_k": desc["k"], "passes": npass, "ideal_passes": math.ceil(n / 13),
                       "tile_bits": desc["tile_bits"], "hub_bits": desc["hub_bits"], "folded_bit_reversal": desc["folded"],
                       "tensor_memory_extended_tile": desc["ext_tile"],
                       "l2": "state larger than L2, no flush needed" if 8 * N > 2 * 126e6 else
                             "state fits L2: HBM fraction not meaningful",
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "time_ms": ms_per_step, "hbm_gbs": roofline["step_gbs"], "hbm_frac_of_measured_peak": roofline["step_frac"],
            "roofline": roofline, "e2e": e2e, "cpu_baseline": cpu_baseline, "gpu_launches": steps * nlaunch,
            "clocks": clocks,
        }
        if variants:
            line["variants"] = variants
        line["tensor_map_fallbacks"] = qft.qft_tensor_map_fallbacks()  # launches that took the slow generic path: 0
        if sweep:
            line["sweep"] = sweep
        if fused_sweep:
            line["max_fused_sweep"] = fused_sweep
        if batched:
            line["batched"] = batched
        if small:
            line["small_n"] = small
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist

        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
