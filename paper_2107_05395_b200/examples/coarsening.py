"""The paper's coarsening study (Fig. 9): 2^20 independent periodic 1-D Cahn-Hilliard
runs (gamma = 0.01, dx = 2 pi / 256, dt = 0.1 dx, C(x, 0) uniform in [-0.1, 0.1]) advanced to T = 100 on
one GPU, recording lbar(t) = mean over the runs of 1 / (1 - <C^2>) at every step (eq. 30), then a linear
regression of lbar against log t (the paper reports r = 0.9989 for L = 2 pi and r = 0.9996 for L = 4 pi).

    python -m paper_2107_05395_b200.examples.coarsening [--runs 1048576] [--length-factor 1] [--T 100] [--out file.csv]

Everything on the path runs in the library's kernels (ch_step_batched_stat); torch only holds the memory.
"""
from __future__ import annotations

import argparse
import math
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--runs", type=int, default=1 << 20)
    ap.add_argument("--length-factor", type=int, default=1, help="L = factor * 2 pi, N = factor * 256")
    ap.add_argument("--T", type=float, default=100.0)
    ap.add_argument("--gamma", type=float, default=0.01)
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--fit-from", type=float, default=1.0, help="regression window starts at this t")
    ap.add_argument("--out", default="")
    args = ap.parse_args()

    import numpy as np
    import torch
    import inputs
    import paper_2107_05395_b200 as b

    n = 256 * args.length_factor
    dx = 2.0 * math.pi / 256
    dt = 0.1 * dx
    steps = int(round(args.T / dt))
    sigma, alpha = args.gamma * dt / dx ** 4, dt / dx ** 2
    h = b.penta_factor_periodic([sigma] * n, [-4 * sigma] * n, [1 + 6 * sigma] * n, [-4 * sigma] * n, [sigma] * n)
    c = torch.empty(n, args.runs, dtype=torch.float64, device="cuda")
    inputs.fill_uniform_device(c, n, seed=args.seed, scale=0.1)
    mass0 = c.sum(dim=0)
    lbar = torch.zeros(steps, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    b.ch_step_batched_stat(h, c, alpha, steps, lbar)
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    drift = float((c.sum(dim=0) - mass0).abs().max())
    l = lbar.cpu().numpy()
    t = dt * np.arange(1, steps + 1)
    sel = t >= args.fit_from
    if int(sel.sum()) >= 3:
        r = float(np.corrcoef(np.log(t[sel]), l[sel])[0, 1])
        slope, icpt = np.polyfit(np.log(t[sel]), l[sel], 1)
    else:  # a run shorter than the regression window: no fit
        r = slope = icpt = float("nan")
    print(f"N={n} runs={args.runs} steps={steps} dt={dt:.6g} sigma={sigma:.6g} alpha={alpha:.6g}")
    print(f"wall {wall:.2f} s  ({wall / steps * 1e3:.4f} ms/step, {args.runs * steps / wall:.3e} run-steps/s)")
    print(f"max |mass drift| over the runs: {drift:.3e}   max |C|: {float(c.abs().max()):.4f}")
    print(f"lbar(T) = {l[-1]:.6f};  lbar vs log t on t >= {args.fit_from}: r = {r:.4f}, slope {slope:.5f}, intercept {icpt:.5f}")
    if args.out:
        np.savetxt(args.out, np.stack([t, l], axis=1)[:: max(1, steps // 4000)], delimiter=",", header="t,lbar", comments="")


if __name__ == "__main__":
    main()
