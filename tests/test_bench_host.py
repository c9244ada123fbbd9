"""Host logic of bench.py and the N > 1 path ("replicas only"), on CPU: gloo, world_size 2, 127.0.0.1."""
import json
import os
import socket
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))
import bench  # noqa: E402


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def golden():
    out = {}
    for line in (ROOT / "tests" / "golden" / "paper_values.txt").read_text().splitlines():
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            out[k.strip()] = float(v)
    return out


def test_algorithmic_bytes_per_lup():
    """27 populations read + 27 written (x 8 or 4 bytes), two-phase adds phi read + phi written."""
    assert bench.lb_bytes_per_lup(False) == 432 and bench.lb_bytes_per_lup(True) == 216
    assert bench.step_bytes_per_lup(False, True) == 448 and bench.step_bytes_per_lup(True, True) == 232
    assert bench.step_bytes_per_lup(False, False) == 432


def test_paper_throughput_context():
    """BASELINE.md's derived figures follow from the numbers PAPER.md:L149 prints."""
    g = golden()
    assert abs(g["glups_a100_single"] / g["n_gpus"] - 2.42) < 0.005
    assert abs(g["glups_a100_two"] / g["n_gpus"] - 1.65) < 0.005
    assert abs(g["glups_a100_single"] / g["glups_a100_two"] - 1.47) < 0.005
    assert abs(g["glups_mi250x_single"] / g["glups_mi250x_two"] - 1.41) < 0.005
    # nu = cs2 (tau - 1/2): the paper's benchmark viscosity corresponds to tau = 0.515
    assert abs(g["nu_benchmark"] / g["cs2"] + 0.5 - 0.515) < 1e-12


def test_roofline_object_from_kernel_times():
    """The headline `achieved` / `frac` are the whole step's (448 B/LUP two-phase over the event-timed region); the
    dominant kernel is reported beside it with its own algorithmic bytes: the fused k_lb_tp moves the step's 448 B/LUP."""
    meas = {"n": 512, "two_phase": True, "ms": 20 * 12.0,
            "kernels": {"k_lb_tp": (20 * 11.2, 20), "k_seam": (20 * 0.8, 60), "k_normal": (0.0, 0)}}
    r = bench.roofline_of(meas, 20, False)
    assert r["kernel"] == "k_lb_tp" and r["bound"] == "hbm" and r["unit"] == "GB/s"
    assert abs(r["achieved"] - 448 * 512 ** 3 / 12.0e-3 / 1e9) < 1e-6
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and r["step_frac"] == r["frac"]
    assert abs(r["kernel_achieved"] - 448 * 512 ** 3 / 11.2e-3 / 1e9) < 1e-6
    assert abs(r["kernel_share_of_step"] - 11.2 / 12.0) < 1e-12
    assert r["traffic"] is None or r["traffic_source"]
    # the two-kernel variant: k_lb_tp then moves only the 54 populations
    meas["kernels"] = {"k_lb_tp": (20 * 10.8, 20), "k_advect": (20 * 2.6, 20)}
    assert bench.roofline_of(meas, 20, False)["kernel_bytes_per_lup"] == 432
    # single-phase
    sp = {"n": 512, "two_phase": False, "ms": 20 * 8.8, "kernels": {"k_lb": (20 * 8.8, 20)}}
    r1 = bench.roofline_of(sp, 20, False)
    assert r1["bytes_per_lup"] == 432 and abs(r1["frac"] - 432 * 512 ** 3 / 8.8e-3 / 1e9 / r1["peak"]) < 1e-12


WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=2)
rank = dist.get_rank()
out = bench.max_over_ranks([10.0 + rank, 5.0 - rank])
assert out == [11.0, 5.0], out
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
"""


def test_max_over_ranks_gloo_world2():
    port = free_port()
    code = WORKER.format(root=str(ROOT), port=port)
    procs = [subprocess.Popen([sys.executable, "-c", code, str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(2)]
    for p in procs:
        out, err = p.communicate(timeout=180)
        assert p.returncode == 0 and out.startswith("ok"), err[-2000:]
    assert bench.max_over_ranks([3.0, 4.0]) == [3.0, 4.0]  # no process group: identity


def test_reference_arm_under_torchrun_world2():
    """`bench.py --impl reference` under torchrun with 2 ranks: rank 0 alone prints ONE JSON line, rank 1 exits 0."""
    env = dict(os.environ, OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(free_port()), str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--workload", "sweep2",
           "--grid", "32", "--steps", "1", "--warmup", "1"]
    p = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env, cwd=str(ROOT))
    assert p.returncode == 0, p.stderr[-3000:]
    lines = [json.loads(l) for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = lines[0]
    assert d["impl"] == "reference" and d["unit"] == "GLUPS" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0 and d["gpu_launches"] == 0
    assert d["config"]["two_phase"] is True
