#!/usr/bin/env python
"""bench.py -- GLUPS of the accLB hot path on B200 (BASELINE.json metric) + roofline + CPU-oracle baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W]              # this repo's CUDA path, ONE JSON line
    python bench.py --impl reference [--steps K] [--warmup W]        # the CPU oracle as it stands, ONE JSON line
    torchrun --nproc-per-node N ... bench.py --gpus N ...            # N independent replicas ("replicas only")
    python bench.py --sweep [--sweep-out FILE]                       # BASELINE config 5 table (several JSON lines)
    [torchrun ...] bench.py --slabs --gpus N ...                     # one domain in N z-slabs with halo exchange (8(f) #3)

A "step" is one pass of the whole hot path (rows a1-a8: pull-stream, moments, phase geometry,
forces, velocity, Hermite coefficient, regularized reconstruction, conservative Allen-Cahn update) over one lattice.
Workload at N = 1: BASELINE config 4 (bubble-laden forced turbulence, 512^3, fp64, two-phase), the configuration the
north-star bar (>= 80 % of the HBM roofline at 512^3 fp64) is quoted on; inputs are seeded and synthetic
(paper_2505_01126_b200/workloads.py).  `value` times accLB_step with the state resident in HBM; `e2e` times
accLB_run_host (host buffers in, host buffers out, copies inside the timed region).  The state (66 GB) is far larger
than L2 (126 MB), so no L2 flush is needed between iterations.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "GLUPS on 1 B200 (fp64) and achieved HBM GB/s as fraction of roofline"
UNIT = "GLUPS"
# Algorithmic bytes per lattice update (DESIGN.md section 7 / SURVEY.md 8(d)):
#   fused LB kernel: 27 populations read + 27 written, 8 B (fp64) or 4 B (fp32 storage) each;
#   whole two-phase step: + phi read + phi written (8 B each).
def lb_bytes_per_lup(fp32, moment=False):
    return 20 * 8 if moment else 54 * (4 if fp32 else 8)  # moment representation: 10 fields read + 10 written (8(f) #2)


def step_bytes_per_lup(fp32, two_phase):
    return lb_bytes_per_lup(fp32) + (16 if two_phase else 0)


def hbm_peak():
    """(GB/s, 'measured'|'fallback'): MEASURED_PEAKS.json hbm_gbs, else the profiling guide's fallback 6650."""
    p = ROOT / "MEASURED_PEAKS.json"
    try:
        return float(json.loads(p.read_text())["hbm_gbs"]), "measured"
    except Exception:
        return 6650.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line)

    def __exit__(self, *exc):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()
            self.thread.join(timeout=2)

    def summary(self):
        sm, smax, power, reasons = [], 0.0, [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.lines:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                smax = max(smax, float(f[1]))
                power.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": smax, "reasons": sorted(reasons), "samples": len(sm),
                "power_w_max": max(power) if power else None}


# ------------------------------------------------------------------------------------------------------ workload
WORKLOADS = {  # bench name -> (workloads.make_config name, description)
    "bubbly": ("bubbly", "BASELINE config 4: bubble-laden forced turbulence, two-phase, tau=0.505, 60 bubbles R=16 at 512^3"),
    "hit": ("hit", "BASELINE config 2 setup: single-phase forced isotropic turbulence, tau=0.51"),
    "sweep1": ("sweep1", "BASELINE config 5 single-phase (config 2 setup)"),
    "sweep2": ("sweep2", "BASELINE config 5 two-phase (config 4 setup at 3 % void fraction)"),
}


def make_workload(name, n):
    from paper_2505_01126_b200 import workloads as wl

    return wl.make_config(WORKLOADS[name][0], n=n)


# ------------------------------------------------------------------------------------------------------ oracle leg
def oracle_threads():
    return int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))


def oracle_sample(cfg, s):
    """Periodic s^3 sub-box at the origin of the workload's fields, and the oracle set up on it (forcing keeps the
    period of the full box).  A bounded sample of the same workload: same parameters, same value distributions."""
    import oracle
    from paper_2505_01126_b200 import workloads as wl

    n = cfg["n"]
    s = min(s, n)
    rho = wl.subbox(cfg["rho"], (0, 0, 0), s)
    u = wl.subbox(cfg["u"], (0, 0, 0), s)
    phi = wl.subbox(cfg["phi"], (0, 0, 0), s) if cfg["phi"] is not None else None
    o = oracle.Oracle(s, s, s, **cfg["params"], force_period=(n, n, n), force_origin=(0, 0, 0))
    o.init(rho, u, phi)
    return o, s


def time_oracle(cfg, steps, warmup, budget_s):
    """Time the oracle as it stands on a sub-box sized so that (steps + warmup) steps take about budget_s.
    Returns (GLUPS, seconds per step, sub-box edge, cores)."""
    o, s0 = oracle_sample(cfg, 32)
    o.step(1)
    t = time.perf_counter()
    o.step(2)
    rate = 2 * s0 ** 3 / (time.perf_counter() - t)  # LUP/s, calibration only
    o.close()
    s = 32
    for cand in (48, 64, 96, 128, 192, 256):
        if cand <= cfg["n"] and (steps + warmup) * cand ** 3 / rate <= budget_s:
            s = cand
    o, s = oracle_sample(cfg, s)
    o.step(warmup)
    t = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t
    d = o.diagnostics()
    o.close()
    assert d["step"] == steps + warmup
    return s ** 3 * steps / dt / 1e9, dt / steps, s, oracle_threads()


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on this arm's config/metric/unit (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle

    oracle.build()
    cfg = make_workload(args.workload, args.n)
    glups, sec, s, cores = time_oracle(cfg, args.steps, args.warmup, budget_s=150.0)
    two_phase = bool(cfg["params"]["two_phase"])
    sample = (f"{s}^3 periodic sub-box at the origin of the {args.n}^3 {args.workload} fields, {args.warmup} warm-up + "
              f"{args.steps} timed oracle steps, gcc -O2 -fopenmp, {cores} threads")
    line = {
        "impl": "reference", "metric": METRIC, "value": glups, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{args.workload} {args.n}^3 {'two' if two_phase else 'single'}-phase fp64 "
                               f"(timed on a {s}^3 sub-box sample)", "n": args.n, "sample_n": s,
                   "two_phase": two_phase},
        "cpu_baseline": {"value": glups, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": glups, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------------ CUDA arm
def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def measure_cuda(cfg, steps, warmup, *, local_rank=0, world=1, fp32=False, e2e=True, variant=None, barrier=None,
                 sample_clocks=True, moment=False):
    """Time `steps` steps of the CUDA path on one GPU.  Returns a dict of raw measurements (this rank's)."""
    import numpy as np
    import torch
    from paper_2505_01126_b200 import binding

    n = cfg["n"]
    two_phase = bool(cfg["params"]["two_phase"])
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    stream = torch.cuda.current_stream(dev)
    sim = binding.AccLB(n, n, n, device=local_rank, stream=stream, store_fp32=int(fp32), host_staging=int(e2e),
                        moment_storage=int(moment), **cfg["params"])
    if variant is not None:
        sim.set_variant(variant)
    h = {k: torch.from_numpy(np.ascontiguousarray(cfg[k])) for k in ("rho", "u", "phi") if cfg[k] is not None}
    d = {k: v.to(dev) for k, v in h.items()}
    sim.init(d["rho"], d["u"], d.get("phi"))
    sim.step(warmup)
    torch.cuda.synchronize(dev)
    diag0 = sim.diagnostics()
    sync = barrier or (lambda: None)

    # ---- timed region: `steps` steps, state resident in HBM; per-kernel events on the launching stream
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sim.profile(True)
    launches0 = sim.launch_count
    sync()
    torch.cuda.synchronize(dev)
    with ClockSampler(local_rank) as clk:
        ev0.record(stream)
        sim.step(steps)
        ev1.record(stream)
        torch.cuda.synchronize(dev)
        if not sample_clocks:
            clk.lines.clear()
    sync()
    ms = ev0.elapsed_time(ev1)
    launches = sim.launch_count - launches0
    kernels = sim.profile_read()
    sim.profile(False)
    diag1 = sim.diagnostics()

    out = {"ms": ms, "launches": launches, "kernels": kernels, "clocks": clk.summary(), "diag0": diag0, "diag1": diag1,
           "workspace_bytes": sim.workspace_bytes, "n": n, "two_phase": two_phase}

    # ---- end to end: HOST buffers in, HOST buffers out, through accLB_run_host (copies inside the timed region)
    if e2e:
        pin = {k: v.pin_memory() for k, v in h.items()}
        res = {k: torch.empty_like(v).pin_memory() for k, v in h.items()}
        sim.run_host(pin["rho"], pin["u"], pin.get("phi"), 1, res["rho"], res["u"], res.get("phi"), diag=True)  # warm-up
        sync()
        torch.cuda.synchronize(dev)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record(stream)
        dg = sim.run_host(pin["rho"], pin["u"], pin.get("phi"), steps, res["rho"], res["u"], res.get("phi"), diag=True)
        e1.record(stream)
        torch.cuda.synchronize(dev)
        wall = time.perf_counter() - t0
        sync()
        nbytes = sum(v.numel() * 8 for v in h.values())
        out["e2e"] = {"ms": e0.elapsed_time(e1), "wall_ms": wall * 1e3, "h2d": nbytes, "d2h": nbytes + 9 * 8,
                      "diag": dg}
    sim.close()
    del d
    torch.cuda.empty_cache()
    return out


# DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) of ONE launch of a kernel at 512^3, from the `ncu --set full`
# captures whose summaries are committed under profiles/ (bench.py does not read that folder).  A capture describes the
# kernel as it was at the commit named; when a kernel changes, its entry is re-measured or removed (then `traffic` is null).
NCU_TRAFFIC = {
    ("k_lb_tp", "two", "fp64", 512): (62_318_549_000, "ncu --set full capture of k_lb_tp at commit 25120c8, profiles/r02_ncu_full.txt"),
    ("k_mr_step", "single", "fp64", 512): (22_290_332_000, "ncu --set full capture of k_mr_step at commit f434175, profiles/r02_ncu_full.txt (last block)"),
    ("k_lb", "single", "fp64", 512): (57_937_901_000, "ncu --set full capture of k_lb at commit f434175, profiles/r02_ncu_full.txt"),
}


def roofline_of(meas, steps, fp32, moment=False):
    """Roofline object.  `achieved`/`frac` are for the WHOLE step (the north-star's figure of merit): algorithmic bytes of a
    step (54 populations, + phi read + phi written when two-phase) x nodes / the CUDA-event time of the timed region.  The
    dominant kernel (largest summed CUDA-event time inside the timed region; events bracket every launch on the launching
    stream) is reported beside it with its own algorithmic bytes: the fused two-phase kernel k_lb_tp moves all of the
    step's algorithmic bytes (the seam kernels only patch phi), the single-phase k_lb the 54 populations."""
    n3 = meas["n"] ** 3
    kernels = {k: v for k, v in meas["kernels"].items() if v[1]}
    name = max(kernels, key=lambda k: kernels[k][0])
    ms_k, cnt_k = kernels[name]
    step_bpl = lb_bytes_per_lup(fp32, True) if moment else step_bytes_per_lup(fp32, meas["two_phase"])
    bpl = step_bpl if moment or (name == "k_lb_tp" and "k_advect" not in kernels) else lb_bytes_per_lup(fp32)
    peak, how = hbm_peak()
    per_launch_ms = ms_k / max(cnt_k, 1)
    k_achieved = bpl * n3 / (per_launch_ms * 1e-3) / 1e9
    total_ms = sum(v[0] for v in kernels.values())
    achieved = step_bpl * n3 * steps / (meas["ms"] * 1e-3) / 1e9
    key = (name, "two" if meas["two_phase"] else "single", "fp32" if fp32 else "fp64", meas["n"])
    traffic, source = NCU_TRAFFIC.get(key, (None, None))
    return {"bound": "hbm", "scope": "whole step (all kernels of the timed region)", "achieved": achieved, "peak": peak,
            "peak_source": how, "unit": "GB/s", "frac": achieved / peak, "bytes_per_lup": step_bpl,
            "bytes_per_step": step_bpl * n3, "traffic": traffic, "traffic_source": source, "traffic_kernel": name,
            "kernel": name, "kernel_bytes_per_lup": bpl, "kernel_bytes_per_launch": bpl * n3,
            "kernel_ms_per_launch": per_launch_ms, "kernel_achieved": k_achieved, "kernel_frac": k_achieved / peak,
            "kernel_share_of_step": ms_k / total_ms if total_ms else None,
            "kernels_ms_per_step": {k: v[0] / steps for k, v in kernels.items()},
            "step_achieved": achieved, "step_frac": achieved / peak, "step_bytes_per_lup": step_bpl}


def max_over_ranks(values, device=None):
    """Element-wise maximum of `values` over all ranks of the default process group (the values themselves when
    torch.distributed is not initialised).  The N > 1 path of this repo is "replicas only": no data-path collective,
    this reduction of the device-timed milliseconds is the only exchange."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return list(values)
    t = torch.tensor(list(values), dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def run_cuda(args):
    import torch

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the CUDA arm has no CPU fallback)")
    barrier = None
    if world > 1:
        import torch.distributed as dist

        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

        def barrier():
            dist.barrier()

    from paper_2505_01126_b200 import build as _build

    if rank == 0:
        _build.build()
    if barrier:
        barrier()
    cfg = make_workload(args.workload, args.n)
    if args.rk3:
        cfg["params"]["phi_rk3"] = 1
    meas = measure_cuda(cfg, args.steps, args.warmup, local_rank=local_rank, world=world, fp32=bool(args.fp32),
                        e2e=not args.no_e2e, variant=args.variant, barrier=barrier, moment=bool(args.moment_storage))
    # replicas only: every rank ran the same-sized independent problem; time = max over ranks
    ms, e2e_ms = max_over_ranks([meas["ms"], meas.get("e2e", {}).get("ms", 0.0)], f"cuda:{local_rank}" if world > 1 else None)
    if rank != 0:
        if world > 1:
            torch.distributed.destroy_process_group()
        return
    n3 = args.n ** 3
    value = world * n3 * args.steps / (ms * 1e-3) / 1e9
    two_phase = meas["two_phase"]
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{args.workload} {args.n}^3 {'two' if two_phase else 'single'}-phase, "
                               f"{'fp32' if args.fp32 else 'fp64'} population storage, fp64 arithmetic; "
                               + WORKLOADS[args.workload][1],
                   "n": args.n, "two_phase": two_phase, "population_storage": "fp32" if args.fp32 else "fp64",
                   "phi_integrator": "ssp-rk3" if args.rk3 else "forward euler",
                   "state": "ten macroscopic fields (p*, u, a) per node" if args.moment_storage else "27 populations per node",
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": f"state of {meas['workspace_bytes'] / 1e9:.1f} GB streams through a 126 MB L2 every step; no flush needed",
                   "lups_per_step": world * n3},
        "clocks": meas["clocks"],
        "gpu_launches": meas["launches"],
        "roofline": roofline_of(meas, args.steps, bool(args.fp32), moment=bool(args.moment_storage)),
        "diagnostics": {"before": meas["diag0"], "after": meas["diag1"]},
    }
    if "e2e" in meas:
        e = meas["e2e"]
        line["e2e"] = {"value": world * n3 * args.steps / (e2e_ms * 1e-3) / 1e9, "unit": UNIT,
                       "h2d_bytes_per_step": e["h2d"] / args.steps, "d2h_bytes_per_step": e["d2h"] / args.steps,
                       "h2d_bytes_per_call": e["h2d"], "d2h_bytes_per_call": e["d2h"], "ms_per_call": e2e_ms,
                       "wall_ms_per_call": e["wall_ms"],
                       "call": f"accLB_run_host(nsteps={args.steps}): pinned host p*,u,phi -> init -> steps -> moments + "
                               "diagnostics -> pinned host"}
    if world == 1 and two_phase and not args.no_single:
        # the other half of the north-star bar: the fused single-phase step (config-2 set-up at the same size), timed in
        # this process with the same steps / warm-up
        sp_cfg = make_workload("hit", args.n)
        sp = measure_cuda(sp_cfg, args.steps, args.warmup, local_rank=local_rank, fp32=bool(args.fp32), e2e=False)
        mr = measure_cuda(sp_cfg, args.steps, args.warmup, local_rank=local_rank, e2e=False, moment=True) if not args.fp32 else None
        if mr:  # the same step on the paper's ten macroscopic fields instead of 27 populations
            g = n3 * args.steps / (mr["ms"] * 1e-3) / 1e9
            line["single_phase_moment_storage"] = {
                "workload": f"hit {args.n}^3 single-phase, state = (p*, u, a) per node (160 B/LUP moved, PAPER.md:L88, L118)",
                "value": g, "unit": UNIT, "ms_per_step": mr["ms"] / args.steps, "gpu_launches": mr["launches"], "clocks": mr["clocks"],
                "workspace_bytes": mr["workspace_bytes"],
                "of_population_roofline": g * lb_bytes_per_lup(False) / hbm_peak()[0],
                "of_own_roofline": g * lb_bytes_per_lup(False, True) / hbm_peak()[0],
                "note": "SM-latency-bound (two barriers per plane, 16 warps per SM), not HBM-bound"}
        if not args.fp32 and not args.rk3:
            # SURVEY 8(f) #1 and #3 on the same inputs: the SSP-RK3 integrator of phi, and the step as one z-slab with its halo
            # exchange (this GPU as its own neighbour)
            rk_cfg = dict(cfg, params=dict(cfg["params"], phi_rk3=1))
            rk = measure_cuda(rk_cfg, args.steps, args.warmup, local_rank=local_rank, e2e=False)
            line["two_phase_rk3"] = {"workload": f"{args.workload} {args.n}^3 two-phase, SSP-RK3 integrator of phi (three stages per step)",
                                     "value": n3 * args.steps / (rk["ms"] * 1e-3) / 1e9, "unit": UNIT, "ms_per_step": rk["ms"] / args.steps,
                                     "gpu_launches": rk["launches"], "clocks": rk["clocks"],
                                     "kernels_ms_per_step": {k: v[0] / args.steps for k, v in rk["kernels"].items() if v[1]}}
            sl = measure_slab(cfg, args.n, args.steps, args.warmup, local_rank=local_rank)
            line["z_slab"] = {"workload": f"{args.workload} {args.n}^3 two-phase as ONE z-slab of {args.n} own planes + {sl['halo']} halo planes "
                                          "per side, halo exchange after every step (the rank is its own neighbour: device copies)",
                              "value": n3 * args.steps / (sl["ms"] * 1e-3) / 1e9, "unit": UNIT, "ms_per_step": sl["ms"] / args.steps,
                              "exchange_ms_per_step": sl["exchange_ms"] / args.steps, "halo_bytes_sent_per_step": sl["halo_bytes"],
                              "gpu_launches": sl["launches"], "clocks": sl["clocks"]}
        line["single_phase"] = {"workload": f"hit {args.n}^3 single-phase; " + WORKLOADS["hit"][1],
                                "value": n3 * args.steps / (sp["ms"] * 1e-3) / 1e9, "unit": UNIT,
                                "ms_per_step": sp["ms"] / args.steps, "gpu_launches": sp["launches"], "clocks": sp["clocks"],
                                "roofline": roofline_of(sp, args.steps, bool(args.fp32))}
    if world == 1 and not args.no_cpu:
        import oracle

        oracle.build()
        glups, sec, s, cores = time_oracle(cfg, 5, 1, budget_s=20.0)
        line["cpu_baseline"] = {"value": glups, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"{s}^3 periodic sub-box at the origin of the same {args.n}^3 fields, 1 warm-up + "
                                          f"5 timed oracle steps ({sec:.2f} s/step), gcc -O2 -fopenmp"}
    print(json.dumps(line), flush=True)
    if world > 1:
        torch.distributed.destroy_process_group()


# ------------------------------------------------------------------------------------------------------ z-slabs (8(f) #3)
def measure_slab(cfg, n, steps, warmup, *, rank=0, world=1, local_rank=0, fp32=False, barrier=None):
    """Time `steps` steps of this rank's z-slab (n own planes + halos) of an n x n x (n * world) domain, the halo exchange
    after every step inside the timed region.  The n^3 fields of `cfg` repeat along z."""
    import numpy as np
    import torch

    from paper_2505_01126_b200 import slabs

    dev = torch.device("cuda", local_rank)
    sync = barrier or (lambda: None)
    part = slabs.SlabAccLB(n, n, n * world, rank=rank, world=world, device=local_rank, store_fp32=int(fp32), **cfg["params"])
    sl = part.slab
    planes = np.arange(sl.z_origin, sl.z_origin + sl.nz_local) % n
    loc = {k: torch.from_numpy(np.ascontiguousarray(np.take(cfg[k], planes, axis=1 if k == "u" else 0))).to(dev)
           for k in ("rho", "u", "phi") if cfg[k] is not None}
    part.init(loc["rho"], loc["u"], loc.get("phi"))
    part.step(warmup)
    torch.cuda.synchronize(dev)
    d0 = part.diagnostics()
    stream = torch.cuda.current_stream(dev)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * steps + 1)]
    launches0 = part.sim.launch_count
    sync()
    torch.cuda.synchronize(dev)
    with ClockSampler(local_rank) as clk:
        ev[0].record(stream)
        for t in range(steps):
            part.sim.step(1)
            ev[2 * t + 1].record(stream)
            part.exchange()
            ev[2 * t + 2].record(stream)
        torch.cuda.synchronize(dev)
    sync()
    out = {"ms": ev[0].elapsed_time(ev[-1]),
           "exchange_ms": sum(ev[2 * t + 1].elapsed_time(ev[2 * t + 2]) for t in range(steps)),
           "launches": part.sim.launch_count - launches0,  # the copies / NCCL kernels of the exchange are not counted
           "clocks": clk.summary(), "halo_bytes": part.halo_bytes_per_step(), "halo": sl.halo, "nz_local": sl.nz_local,
           "diag0": d0, "diag1": part.diagnostics()}
    part.close()
    del loc
    torch.cuda.empty_cache()
    return out


def run_slabs(args):
    """`--slabs`: ONE periodic domain n x n x (n * N) cut into N z-slabs, one per rank / GPU (the shape of the paper's weak
    scaling), halo exchange after every step inside the timed region (NCCL send / recv between the ranks;
    with N = 1 the rank is its own neighbour and the exchange is device copies).  The fields are the n^3 workload repeated
    along z.  Not the driver's line: `python bench.py --gpus N` without --slabs stays "replicas only"."""
    import torch

    from paper_2505_01126_b200 import build as _build

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the CUDA arm has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    barrier = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        barrier = dist.barrier
    if rank == 0:
        _build.build()
    if barrier:
        barrier()
    n = args.n
    cfg = make_workload(args.workload, n)
    two_phase = bool(cfg["params"]["two_phase"])
    m = measure_slab(cfg, n, args.steps, args.warmup, rank=rank, world=world, local_rank=local_rank, fp32=bool(args.fp32),
                     barrier=barrier)
    ms, ms_x = max_over_ranks([m["ms"], m["exchange_ms"]], f"cuda:{local_rank}" if world > 1 else None)
    if rank == 0:
        own = n ** 3
        bpl = step_bytes_per_lup(bool(args.fp32), two_phase)
        peak, how = hbm_peak()
        value = world * own * args.steps / (ms * 1e-3) / 1e9
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": f"{args.workload} {n} x {n} x {n * world} {'two' if two_phase else 'single'}-phase, one periodic "
                                   f"domain in {world} z-slab(s) of {n} planes + {m['halo']} halo planes per side; the {n}^3 fields "
                                   "repeated along z; " + WORKLOADS[args.workload][1],
                       "parallelism": f"z-slabs x{world}, one halo exchange per step ("
                                      + ("NCCL send/recv" if world > 1 else "the rank is its own neighbour: device copies") + ")",
                       "halo_bytes_sent_per_rank_and_step": m["halo_bytes"],
                       "lups_per_step": world * own, "planes_computed_per_rank": m["nz_local"]},
            "exchange_ms_per_step": ms_x / args.steps, "clocks": m["clocks"], "gpu_launches": m["launches"],
            "roofline": {"bound": "hbm", "scope": "whole step incl. halo exchange, own planes only", "unit": "GB/s", "peak": peak * world,
                         "peak_source": how, "achieved": value * bpl, "frac": value * bpl / (peak * world), "traffic": None},
            "diagnostics": {"before": m["diag0"], "after": m["diag1"]}}), flush=True)
    if world > 1:
        torch.distributed.destroy_process_group()


# ------------------------------------------------------------------------------------------------------ config 5 sweep
def run_sweep(args):
    """BASELINE config 5: N in {64,...,512}, single- and two-phase, fp64 and fp32 population storage; 200 timed steps
    after 20 warm-up steps unless --steps/--warmup say otherwise.  One JSON line per case (not the driver's line)."""
    peak, how = hbm_peak()
    sizes = [int(s) for s in args.sweep_sizes.split(",")]
    rows = []
    for name in ("sweep1", "sweep2"):
        for n in sizes:
            cfg = make_workload(name, n)
            for fp32 in (False, True):
                m = measure_cuda(cfg, args.steps, args.warmup, fp32=fp32, e2e=False, variant=args.variant,
                                 sample_clocks=False)
                glups = n ** 3 * args.steps / (m["ms"] * 1e-3) / 1e9
                bpl = step_bytes_per_lup(fp32, m["two_phase"])
                row = {"case": name, "n": n, "two_phase": m["two_phase"], "storage": "fp32" if fp32 else "fp64",
                       "glups": glups, "ms_per_step": m["ms"] / args.steps, "bytes_per_lup": bpl,
                       "gbs": glups * bpl, "frac_of_hbm_peak": glups * bpl / peak, "peak": peak, "peak_source": how,
                       "kernels_ms_per_step": {k: v[0] / args.steps for k, v in m["kernels"].items() if v[1]}}
                rows.append(row)
                print(json.dumps(row), flush=True)
    if args.sweep_out:
        Path(args.sweep_out).parent.mkdir(parents=True, exist_ok=True)
        Path(args.sweep_out).write_text("\n".join(json.dumps(r) for r in rows) + "\n")


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", choices=("cuda", "reference"), default="cuda")
    ap.add_argument("--workload", choices=sorted(WORKLOADS), default="bubbly")
    ap.add_argument("--n", "--grid", dest="n", type=int, default=512, help="grid edge (default: the 512^3 the metric is quoted on)")
    ap.add_argument("--fp32", type=int, default=0, help="1: fp32 population storage (arithmetic stays fp64)")
    ap.add_argument("--variant", type=int, default=None, help="kernel variant (accLB_set_variant), default = best")
    ap.add_argument("--rk3", type=int, default=0, help="1: SSP-RK3 integrator for phi (SURVEY 8(f) #1) instead of forward Euler")
    ap.add_argument("--moment-storage", type=int, default=0, help="1: single-phase state = the ten fields (p*, u, a) per node (SURVEY 8(f) #2); use with --workload hit")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-single", action="store_true", help="skip the extra legs of a two-phase run (single_phase, "
                                                             "single_phase_moment_storage, two_phase_rk3, z_slab)")
    ap.add_argument("--slabs", action="store_true", help="one domain n x n x (n N) in N z-slabs with halo exchange (SURVEY 8(f) #3) "
                                                         "instead of N independent replicas")
    ap.add_argument("--sweep", action="store_true")
    ap.add_argument("--sweep-sizes", default="64,128,256,384,512")
    ap.add_argument("--sweep-out", default=None)
    args = ap.parse_args()
    if args.steps < 1 or args.warmup < 0:
        raise SystemExit("bench.py: --steps >= 1 and --warmup >= 0")
    if args.impl == "reference":
        return run_reference(args)
    if args.sweep:
        return run_sweep(args)
    if args.slabs:
        return run_slabs(args)
    return run_cuda(args)


if __name__ == "__main__":
    main()
