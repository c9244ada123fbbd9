"""Laplace-jump study of the static droplet with the ORACLE only (test infrastructure; calls nothing but oracle/).

    python oracle/laplace_study.py [--radii 12,16,24] [--out tests/golden/laplace_oracle.txt]

For every radius R (box edge 4 R, tau = 0.8, D = 0.05, delta = 4, gamma = 0.01: BASELINE config 3 scaled) and density
ratio 1 and 10 (zero gauge, R26) the droplet is run to 1.5 R^2 / nu steps (nu = 0.1) and the pressure jump
Delta p / (2 gamma / R_eff), R_eff = (3 sum phi / 4 pi)^(1/3) (reading R8), is recorded, averaged over the
last fifth of the run, in two ways:
  A  centre node minus corner node (R26, what the GPU test of config 3 uses);
  B  mean over the ball r < R / 2 minus mean over the far region r > 1.6 R (insensitive to acoustic ringing at a point).
The table goes to tests/golden/laplace_oracle.txt and is quoted in DESIGN.md section 8.
"""
import argparse
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))
import oracle  # noqa: E402


def droplet(n, R, W=4.0):
    c = (n - 1) / 2.0
    ax = np.arange(n, dtype=np.float64)
    Z, Y, X = np.meshgrid(ax, ax, ax, indexing="ij")
    r = np.sqrt((X - c) ** 2 + (Y - c) ** 2 + (Z - c) ** 2)
    return 0.5 * (1.0 + np.tanh(2.0 * (R - r) / W)), r


def run(R, ratio, sigma=0.01, tau=0.8):
    n = int(4 * R)
    phi, r = droplet(n, R)
    rho = np.ones((n, n, n)) if ratio == 1.0 else np.zeros((n, n, n))
    o = oracle.Oracle(n, n, n, tau=tau, two_phase=1, rho_l=ratio, rho_g=1.0, sigma=sigma, mobility=0.05, width=4.0)
    o.init(rho, np.zeros((3, n, n, n)), phi)
    nu = (tau - 0.5) / 3.0
    steps = int(1.5 * R * R / nu)
    ball, far = r < 0.5 * R, r > 1.6 * R
    c = n // 2
    a, b, t0 = [], [], time.time()
    every = 20
    for it in range(steps // every):
        o.step(every)
        if it * every >= 0.8 * steps:
            ps, _, ph = o.moments()
            p = ps * (1.0 + (ratio - 1.0) * ph) / 3.0            # p = p* rho(phi) c_s^2
            R_eff = (3.0 * ph.sum() / (4.0 * np.pi)) ** (1.0 / 3.0)
            ref = 2.0 * sigma / R_eff
            a.append((p[c, c, c] - p[0, 0, 0]) / ref)
            b.append((p[ball].mean() - p[far].mean()) / ref)
    d = o.diagnostics()
    o.close()
    return dict(R=R, n=n, ratio=ratio, steps=steps, A=float(np.mean(a)), B=float(np.mean(b)), A_std=float(np.std(a)),
                umax=d["umax"], R_eff=float(R_eff), seconds=time.time() - t0)


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--radii", default="12,16,24")
    ap.add_argument("--out", default=str(ROOT / "tests" / "golden" / "laplace_oracle.txt"))
    args = ap.parse_args()
    oracle.build()
    lines = ["# written by oracle/laplace_study.py (oracle only); columns: R n ratio steps A(centre-corner) B(ball-far) std(A) umax R_eff",
             "# Delta p / (2 gamma / R_eff), mean over the last fifth of 1.5 R^2/nu steps; PAPER.md:L55, L102; readings R8, R26"]
    for R in [float(x) for x in args.radii.split(",")]:
        for ratio in (1.0, 10.0):
            res = run(R, ratio)
            line = f"{res['R']:g} {res['n']} {res['ratio']:g} {res['steps']} {res['A']:.4f} {res['B']:.4f} {res['A_std']:.4f} {res['umax']:.2e} {res['R_eff']:.3f}"
            print(line, f"({res['seconds']:.0f} s)", flush=True)
            lines.append(line)
            Path(args.out).write_text("\n".join(lines) + "\n")
