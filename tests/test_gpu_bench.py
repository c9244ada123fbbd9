"""bench.py end to end on a small grid: the JSON line of the CUDA arm carries every key the contract and DESIGN.md section 8
name (roofline, e2e, cpu_baseline, clocks, gpu_launches and the extra legs), and the --slabs line its own."""
import json
import subprocess
import sys
from pathlib import Path

import pytest

pytestmark = pytest.mark.gpu
ROOT = Path(__file__).resolve().parents[1]


def run(*flags):
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), *flags], capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout[-2000:]
    return json.loads(lines[0])


def test_default_line_small_grid():
    d = run("--n", "64", "--steps", "4", "--warmup", "3")
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "clocks", "gpu_launches", "roofline", "e2e", "cpu_baseline", "single_phase",
              "single_phase_moment_storage", "two_phase_rk3", "z_slab"):
        assert k in d, k
    assert d["unit"] == "GLUPS" and d["dtype"] == "f64" and d["n_gpus"] == 1 and d["steps"] == 4 and d["vs_baseline"] is None
    assert d["gpu_launches"] == 2 * 4                       # k_lb_tp + k_seam per step
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["kernel"] == "k_lb_tp" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    assert abs(d["value"] - 64 ** 3 * 4 / (d["ms_per_step"] * 4e-3) / 1e9) < 1e-9 * d["value"]
    e = d["e2e"]
    assert e["h2d_bytes_per_step"] == 5 * 64 ** 3 * 8 / 4 and e["d2h_bytes_per_step"] > e["h2d_bytes_per_step"] and e["value"] < d["value"]
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] > 0
    assert d["two_phase_rk3"]["gpu_launches"] == 6 * 4      # (k_lb_tp | stage) + k_seam, three stages per step
    assert set(d["two_phase_rk3"]["kernels_ms_per_step"]) == {"k_lb_tp", "k_seam", "k_lb_tp_stage"}
    assert d["z_slab"]["halo_bytes_sent_per_step"] == 2 * (27 + 3) * 64 * 64 * 8 and d["z_slab"]["gpu_launches"] == 2 * 4
    assert d["single_phase"]["gpu_launches"] == 4 and d["single_phase_moment_storage"]["gpu_launches"] == 4
    # conserved sums before / after the timed region
    a, b = d["diagnostics"]["before"], d["diagnostics"]["after"]
    assert abs(a["sum_phi"] - b["sum_phi"]) <= 1e-12 * a["sum_phi"] and abs(a["sum_pstar"] - b["sum_pstar"]) <= 1e-12 * a["sum_pstar"]


def test_slabs_line_small_grid():
    d = run("--slabs", "--n", "64", "--steps", "4", "--warmup", "3", "--workload", "hit")
    assert d["n_gpus"] == 1 and d["scaling"] == "weak" and d["gpu_launches"] == 4
    assert d["config"]["halo_bytes_sent_per_rank_and_step"] == 2 * 9 * 64 * 64 * 8
    assert d["config"]["planes_computed_per_rank"] == 66 and d["exchange_ms_per_step"] > 0
    a, b = d["diagnostics"]["before"], d["diagnostics"]["after"]
    assert abs(a["sum_pstar"] - b["sum_pstar"]) <= 1e-12 * a["sum_pstar"]
