"""Time one shared-LHS solve ("single A, multiple b") under different `btps_tune` settings: the
measurement behind the library's launch defaults (cluster split, held stores).

    python -m paper_2107_05395_b200.examples.tune_sweep --kind tri --dtype f64 --n 1024 --log2-batch 19 20 22 \
        --key cluster -1 0 --key hold_stores -1 0 1

Every combination of the given keys' values is applied (-1 = library default); the fraction printed is
2*N*M*sizeof(T) / time over --peak-gbs.  Also the command behind profiles/r01f_cluster_default.md.
"""
from __future__ import annotations

import argparse
import itertools
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--kind", choices=("tri", "penta"), default="tri")
    ap.add_argument("--dtype", choices=("f64", "f32"), default="f64")
    ap.add_argument("--n", type=int, default=1024)
    ap.add_argument("--log2-batch", type=int, nargs="+", default=[19])
    ap.add_argument("--batch", type=int, nargs="+", default=[], help="batch sizes that are not powers of two")
    ap.add_argument("--key", action="append", nargs="+", default=[], metavar=("NAME", "VALUE"))
    ap.add_argument("--plan-key", action="append", nargs=2, default=[], metavar=("NAME", "VALUE"),
                    help="tune key read when a handle is built (rows, lanes, vec, tiles_per_cta, ...): set once, before the factor call")
    ap.add_argument("--reps", type=int, default=8)
    ap.add_argument("--peak-gbs", type=float, default=6549.8)
    args = ap.parse_args()

    import numpy as np
    import torch
    import paper_2107_05395_b200.binding as b

    n, r = args.n, 0.5
    for k, v in args.plan_key:
        b.btps_tune(k, int(v))
    dt = torch.float64 if args.dtype == "f64" else torch.float32
    if args.kind == "tri":
        h = b.tri_factor(np.full(n, -r), np.full(n, 1 + 2 * r), np.full(n, -r))
        solve = b.tri_solve_batched if args.dtype == "f64" else b.tri_solve_batched_f32
    else:
        h = b.penta_factor(np.full(n, r), np.full(n, -4 * r), np.full(n, 1 + 6 * r), np.full(n, -4 * r), np.full(n, r))
        solve = b.penta_solve_batched if args.dtype == "f64" else b.penta_solve_batched_f32
    print("plan:", h.plan(8 if args.dtype == "f64" else 4), flush=True)
    keys = [k[0] for k in args.key]
    values = [[int(v) for v in k[1:]] for k in args.key]
    for m in [1 << lm for lm in args.log2_batch] + list(args.batch):
        x = torch.rand(n, m, device="cuda", dtype=dt) * 1e-3
        for combo in itertools.product(*values):
            for k, v in zip(keys, combo):
                b.btps_tune(k, v)
            for _ in range(3):
                solve(h, x)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(args.reps):
                solve(h, x)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / args.reps
            gbs = 2.0 * n * m * x.element_size() / ms / 1e6
            print(f"{args.kind} {args.dtype} n={n} batch={m} {dict(zip(keys, combo))}: {ms:.4f} ms  "
                  f"{gbs:.1f} GB/s  {gbs / args.peak_gbs:.4f} of peak", flush=True)
        for k in keys:
            b.btps_tune(k, -1)
        del x


if __name__ == "__main__":
    main()
