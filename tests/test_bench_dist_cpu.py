"""The N > 1 plumbing of bench.py (rendezvous, barrier, max over ranks) on the CPU: world size 2, gloo.

The QFT path itself does not shard (replicas only), so bench.py --gpus N runs N
independent replicas and the only cross-rank steps are the barrier around the timed region and the
MAX reduction of the device time.  Also: under torchrun the reference arm runs on rank 0 alone.
"""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import sys, types
sys.path.insert(0, %r)
import torch
import bench
args = types.SimpleNamespace(gpus=2)
world, rank, local = bench.dist_setup(args)
assert world == 2 and rank in (0, 1) and local == rank
bench.barrier(world)
m = bench.max_over_ranks(10.0 + 5.0 * rank, world, torch.device("cpu"))
bench.barrier(world)
print("RESULT", rank, m)
import torch.distributed as dist
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_world_size_2_gloo_barrier_and_max():
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, WORLD_SIZE="2", RANK=str(rank), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER % ROOT], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=180) for p in procs]
    for p, (so, se) in zip(procs, outs):
        assert p.returncode == 0, se[-2000:]
    vals = sorted(float(line.split()[2]) for so, _ in outs for line in so.splitlines() if line.startswith("RESULT"))
    assert vals == [15.0, 15.0]  # both ranks see the maximum


def test_reference_arm_runs_on_rank_0_only():
    env = dict(os.environ, WORLD_SIZE="2", RANK="1", LOCAL_RANK="1", CUDA_VISIBLE_DEVICES="")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--n", "12", "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True,
                       timeout=180)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"] = "0"
    env["LOCAL_RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--n", "12", "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True,
                       timeout=180)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0


def test_reference_arm_times_whole_oracle_circuits():
    """bench.py --impl reference: every step is one whole oracle circuit (here n = 20: seconds on any host)."""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--n", "20", "--steps", "2",
                        "--warmup", "1"], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["steps"] == 2 and d["warmup"] == 1 and d["metric"] == "dft_equiv_gflops"
    assert d["config"]["sample_n_qubits"] == 20 and d["cpu_baseline"]["kind"] == "oracle"
    assert abs(d["value"] - 5.0 * (1 << 20) * 20 / (d["ms_per_step"] * 1e-3) / 1e9) < 1e-6 * d["value"]
    assert d["e2e"]["value"] == d["value"] and d["e2e"]["h2d_bytes_per_step"] == 0
