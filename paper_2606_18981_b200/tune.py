"""Per-pass timing of one plan configuration (a tuning aid for the layout knobs of qft_plan_create_tuned).

    python -m paper_2606_18981_b200.tune --n 30 [--k K] [--tile-bits T] [--hub-bits L] [--flags F] [--max-fused W]

Prints one JSON line: the pass list (kernel kind, register steps) and the CUDA-event time of every pass.
With --reps R --no-time it only runs R transforms, which is the command to wrap in ncu.
"""
from __future__ import annotations

import argparse
import json


def main() -> int:
    import torch

    import paper_2606_18981_b200 as qft

    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=30)
    ap.add_argument("--k", type=int, default=None)
    ap.add_argument("--tile-bits", type=int, default=0)
    ap.add_argument("--hub-bits", type=int, default=0)
    ap.add_argument("--flags", type=int, default=0)
    ap.add_argument("--max-fused", type=int, default=13)
    ap.add_argument("--log2-batch", type=int, default=0, help="2^b independent transforms back to back")
    ap.add_argument("--reps", type=int, default=2)
    ap.add_argument("--no-time", action="store_true")
    ap.add_argument("--phase-lib", default=None,
                    help="a library built with `python -m paper_2606_18981_b200.build --define QFT_PHASE_TIMING --lib PATH`: "
                         "print, per pass, the clocks thread 0 of CTA 0 spends in each phase of the TMA kernel per tile")
    ap.add_argument("--loop", type=int, default=0, help="also time this many back-to-back qft_execute calls (launch-bound sizes)")
    a = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("needs a CUDA device")
    if a.phase_lib:
        qft.LIB_PATH = a.phase_lib  # before the first call loads the library
    n = a.n
    plan = qft.Plan(n, n if a.k is None else a.k, a.max_fused, -1, qft.QFT_NORM_UNITARY, a.tile_bits, a.hub_bits, a.flags,
                    a.log2_batch)
    n = a.n + a.log2_batch  # address bits from here on
    st = torch.empty(1 << n, dtype=torch.complex64, device="cuda")
    torch.view_as_real(st).normal_()
    st.mul_(2.0 ** (-(n + 1) / 2))
    s = torch.cuda.current_stream().cuda_stream
    for _ in range(a.reps):
        qft.qft_execute(plan.handle, st.data_ptr(), s)
    torch.cuda.synchronize()
    if a.phase_lib:
        import ctypes

        lib = qft.load()
        lib.qft_debug_set_phase_buffer.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p]
        names = ["bookkeeping", "wait for the tile's load", "step 1 reads + barrier", "step 1 arithmetic + exchange writes + barrier",
                 "step 2 reads + barrier + next load + next end table", "step 2 arithmetic", "park first half in tensor memory",
                 "extension butterfly + stores"]
        for p in range(plan.num_passes):
            buf = torch.zeros(16, dtype=torch.int64, device="cuda")
            lib.qft_debug_set_phase_buffer(plan.handle, p, buf.data_ptr())
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            qft.qft_execute_pass(plan.handle, p, st.data_ptr(), s)
            e1.record()
            torch.cuda.synchronize()
            lib.qft_debug_set_phase_buffer(plan.handle, p, None)
            c = buf.cpu().tolist()
            tiles = max(c[8], 1)
            print(json.dumps({"n": a.n, "pass": p, "ms": round(e0.elapsed_time(e1), 3), "tiles_of_cta0": c[8],
                              "clocks_per_tile": {names[i]: round(c[i] / tiles) for i in range(8)},
                              "total_clocks_per_tile": round(sum(c[:8]) / tiles)}))
        return 0
    if a.no_time:
        return 0
    npass = plan.num_passes
    acc = [0.0] * npass
    reps = 5
    for _ in range(reps):
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(npass + 1)]
        ev[0].record()
        for p in range(npass):
            qft.qft_execute_pass(plan.handle, p, st.data_ptr(), s)
            ev[p + 1].record()
        torch.cuda.synchronize()
        for p in range(npass):
            acc[p] += ev[p].elapsed_time(ev[p + 1]) / reps
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        qft.qft_execute(plan.handle, st.data_ptr(), s)
    e1.record()
    torch.cuda.synchronize()
    execute_ms = round(e0.elapsed_time(e1) / reps, 3)
    loop_us = None
    if a.loop:
        for _ in range(20):
            qft.qft_execute(plan.handle, st.data_ptr(), s)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(a.loop):
            qft.qft_execute(plan.handle, st.data_ptr(), s)
        e1.record()
        torch.cuda.synchronize()
        loop_us = round(1000.0 * e0.elapsed_time(e1) / a.loop, 2)
    d = plan.describe()
    print(json.dumps({"launches": plan.num_launches, "loop_us_per_execute": loop_us, "n": d["n"], "batch_bits": d["batch_bits"], "k": d["k"], "tile_bits": d["tile_bits"], "hub_bits": d["hub_bits"], "passes": npass,
                      "kernels": [p["kernel"] for p in d["passes"]], "steps": [p["steps"] for p in d["passes"]],
                      "pass_ms": [round(v, 3) for v in acc], "execute_ms": execute_ms,
                      "gbs_per_pass": [round(16.0 * (1 << n) / v / 1e6) for v in acc]}))
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
