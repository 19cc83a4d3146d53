"""Time loops of the paper's schemes on one GPU ("1000 time steps", RHS = previous solution):
backward-Euler diffusion / hyperdiffusion (BASELINE.json configs 2, 3), the Cahn-Hilliard step (config 5) and the
periodic Crank-Nicolson steps of Tables 1 and 2, advanced `--steps` steps by ONE library call; the library keeps
a tile on chip for up to 64 steps per launch (btps_tune "fuse_steps").

    python -m paper_2107_05395_b200.examples.time_loop --scheme tri --n 512 --log2-batch 16 --steps 64

Prints the plan and the time per step.  Also the command behind profiles/r01e_fused_time_loop.md.
"""
from __future__ import annotations

import argparse
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

SCHEMES = ("tri", "penta", "ch", "ch_periodic", "tri_cn_periodic", "penta_cn_periodic")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--scheme", choices=SCHEMES, default="tri")
    ap.add_argument("--n", type=int, default=512)
    ap.add_argument("--log2-batch", type=int, default=16)
    ap.add_argument("--steps", type=int, default=64)
    ap.add_argument("--calls", type=int, default=4, help="timed calls (after one warm-up call)")
    ap.add_argument("--fuse-steps", type=int, default=-1, help="steps per launch (default: the library's)")
    args = ap.parse_args()

    import torch
    import inputs
    import paper_2107_05395_b200 as b

    n, batch, steps = args.n, 1 << args.log2_batch, args.steps
    if args.fuse_steps > 0:
        b.btps_tune("fuse_steps", args.fuse_steps)
    u = torch.empty(n, batch, dtype=torch.float64, device="cuda")
    inputs.fill_uniform_device(u, n, seed=1, scale=0.1)
    sigma = 0.5
    if args.scheme == "tri":
        h = b.tri_factor(*inputs.tri_lhs(n, sigma))
        call = lambda: b.tri_solve_steps(h, u, steps)
    elif args.scheme == "penta":
        h = b.penta_factor(*inputs.penta_lhs(n, sigma))
        call = lambda: b.penta_solve_steps(h, u, steps)
    elif args.scheme in ("ch", "ch_periodic"):
        lhs = inputs.ch_lhs(n)
        h = b.penta_factor(*lhs) if args.scheme == "ch" else b.penta_factor_periodic(*lhs)
        _, alpha = inputs.ch_params(n)
        call = lambda: b.ch_step_batched(h, u, alpha, steps)
    elif args.scheme == "tri_cn_periodic":  # eq. 9-11: (I - s/2 D2) u+ = (I + s/2 D2) u
        s = sigma / 2
        h = b.tri_factor_periodic([-s] * n, [1 + 2 * s] * n, [-s] * n)
        call = lambda: b.tri_cn_step_batched(h, u, s, 1 - 2 * s, s, steps)
    else:  # eq. 17-19: (I + s/2 D4) u+ = (I - s/2 D4) u
        s = sigma / 2
        h = b.penta_factor_periodic([s] * n, [-4 * s] * n, [1 + 6 * s] * n, [-4 * s] * n, [s] * n)
        call = lambda: b.penta_cn_step_batched(h, u, [-s, 4 * s, 1 - 6 * s, 4 * s, -s], steps)

    call()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = b.btps_launch_count()
    e0.record()
    for _ in range(args.calls):
        call()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / (args.calls * steps)
    launches = (b.btps_launch_count() - n0) // args.calls
    plan = h.plan(8) if args.scheme in ("tri", "penta") else (h.ch_plan(8) if args.scheme.startswith("ch") else h.cn_plan(8))
    print(f"{args.scheme}: N={n} batch=2^{args.log2_batch} steps={steps} launches/call={launches} plan={plan}")
    print(f"{ms * 1e3:.2f} us per step, {batch / ms * 1e3:.4g} system-steps/s, "
          f"effective {2.0 * n * batch * 8 / ms / 1e6:.0f} GB/s of per-step algorithmic bytes; max |u| = {u.abs().max().item():.3e}")


if __name__ == "__main__":
    main()
