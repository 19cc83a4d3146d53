#!/usr/bin/env python
"""bench.py -- throughput of the shared-LHS batched tri / penta / fused Cahn-Hilliard path on B200.

Contract (driver): ``python bench.py --gpus N --steps K --warmup W`` prints ONE compact JSON line (the LAST line of
stdout) on rank 0.  The per-config table (BASELINE.json configs 1-5) goes to the side file named in the line
(``bench_configs.json``, git-ignored), never to stdout.

Workload: BASELINE.json configs[1] shape -- N=512 unknowns, batch=65536 systems per GPU,
fp64, interleaved.  One *step* is one pass of the whole hot path over that batch:
  (a2) one tridiagonal sweep   (LHS of config 2: tridiag(-r, 1+2r, -r), r = 0.5; u0 = 4 sine modes)
  (a4) one pentadiagonal sweep (LHS of config 3: I + r*[1,-4,6,-4,1];    rhs uniform[-1,1))
  (a5) one fused Cahn-Hilliard step (LHS I + sigma*D4, RHS built in the kernel; c0 = 0.1*uniform)
each on its own 256 MiB buffer (768 MiB rotate through the 126 MB L2: every launch is cold), advanced in place step
after step (RHS = previous solution, the (a6) driver).  The factorisations (a1)/(a3) are done once before the loop, as
the paper does; their host time is reported as ``factor_ms``.

value = system-solves per second, whole job (3 * batch * n_gpus per step).

Other modes (measurement tools, all through the C-ABI binding):
  --cell kind,n,log2batch,dtype [--tune key=value ...]   time single cells under btps_tune settings
  --paper-tables                                         the paper's Table 1 / 2 workloads into the side file (context)
"""
from __future__ import annotations

import argparse
import csv
import json
import math
import os
import re
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

N_ROWS = 512
BATCH = 65536
METRIC = "systems solved/s (tri + penta + fused CH step, shared LHS)"
UNIT = "systems/s"
L2_BYTES = 126 * 1024 * 1024
SIDE_FILE = "bench_configs.json"
# dram__bytes_read.sum + dram__bytes_write.sum per launch come from this committed ncu capture of
# `bench.py --steps 2 --warmup 3 --no-cpu-baseline --no-e2e --no-extra` (profiles/r02_traffic.md names the command and
# the library build it was taken with); bench.py reports them only for the kernels and the build it has just timed.
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r02_traffic.csv")
TRAFFIC_MD = os.path.join(ROOT, "profiles", "r02_traffic.md")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--batch", type=int, default=BATCH, help="systems per GPU (default: config 2's 65536)")
    ap.add_argument("--n", type=int, default=N_ROWS)
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the per-config table (configs 1-5)")
    ap.add_argument("--paper-tables", action="store_true", help="also time the paper's Table 1 / 2 workloads (context only)")
    ap.add_argument("--side-file", default=os.path.join(ROOT, SIDE_FILE))
    ap.add_argument("--cell", action="append", default=[], metavar="KIND,N,LOG2BATCH,DTYPE",
                    help="time one cell instead of the headline step, e.g. tri,1024,19,f64 (kinds: tri, penta, ch, "
                         "tri_periodic, penta_periodic, ch_periodic, tri_f32s, penta_f32s, tri_cn[_periodic], penta_cn[_periodic]); "
                         "may be repeated")
    ap.add_argument("--tune", action="append", default=[], metavar="KEY=VALUE", help="btps_tune setting applied first")
    ap.add_argument("--cell-steps", type=int, default=1, help="--cell: time steps per call (tri/penta_solve_steps, ch_step_batched)")
    ap.add_argument("--rotate", type=int, default=0, help="--cell: rotate over this many buffers (default: as many as keep the cell cold)")
    return ap.parse_args()


def peaks():
    """Measured HBM copy bandwidth (driver-written), else the profiling guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ---------------------------------------------------------------------------------------------------
# inputs (host, seeded; inputs/ holds no solver arithmetic)
# ---------------------------------------------------------------------------------------------------
def make_host_inputs(n, batch, seed, rank):
    import numpy as np
    import inputs
    from paper_2107_05395_b200 import sharding
    j0, j1 = sharding.weak_shard(batch, rank)  # each rank: its own systems, no exchange
    sys_ids = np.arange(j0, j1, dtype=np.uint64)
    u_tri, _, _ = inputs.sine_modes_u0(n, batch, seed=seed, systems=sys_ids)
    u_penta = inputs.uniform_rhs(n, batch, seed=seed, systems=sys_ids)
    c_ch = inputs.uniform_rhs(n, batch, seed=seed + 1, scale=0.1, systems=sys_ids)
    return u_tri, u_penta, c_ch


# ---------------------------------------------------------------------------------------------------
# clocks sampler (nvidia-smi in the background during the timed region)
# ---------------------------------------------------------------------------------------------------
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(prefix="btps_clocks_", suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.FIELDS}",
                 "--format=csv,noheader,nounits", "-lms", "50"],
                stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        try:
            self.proc.terminate()
            self.proc.wait(timeout=5)
        except Exception:
            pass
        try:
            rows = [r.strip().split(",") for r in open(self.path) if r.strip()]
            os.unlink(self.path)
        except Exception:
            return out
        sm, reasons = [], set()
        for r in rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0]))
                out["sm_max_mhz"] = float(r[1])
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.strip().lower().startswith("active"):
                    reasons.add(name)
        if sm:
            sm.sort()
            out["sm_mhz"] = sm[len(sm) // 2]
        out["reasons"] = sorted(reasons)
        out["samples"] = len(sm)
        return out


# ---------------------------------------------------------------------------------------------------
# oracle arm: one step = tri sweep + penta sweep + CH step on `sample` systems, on the host cores
# ---------------------------------------------------------------------------------------------------
def oracle_step_fn(n, sample, seed, nthreads=0):
    import numpy as np
    import inputs
    import oracle
    ft = oracle.tri_factor(*inputs.tri_lhs(n, 0.5))
    fp = oracle.penta_factor(*inputs.penta_lhs(n, 0.5))
    sigma, alpha = inputs.ch_params(n)
    fc = oracle.penta_factor(*inputs.ch_lhs(n))
    ids = np.arange(sample, dtype=np.uint64)
    u_tri, _, _ = inputs.sine_modes_u0(n, sample, seed=seed, systems=ids)
    u_penta = inputs.uniform_rhs(n, sample, seed=seed, systems=ids)
    c_ch = inputs.uniform_rhs(n, sample, seed=seed + 1, scale=0.1, systems=ids)
    state = {"cores": 0}

    def step():
        c = oracle.tri_solve_interleaved(ft, u_tri, nthreads=nthreads)
        oracle.penta_solve_interleaved(fp, u_penta, nthreads=nthreads)
        oracle.ch_step_interleaved(fc, c_ch, alpha, nsteps=1, nthreads=nthreads)
        state["cores"] = c
    return step, state


def workload_config(n, batch):
    """The workload both arms name in `config` (the reference arm times a bounded sample of it)."""
    return {"workload": f"BASELINE.json configs[1] shape: N={n}, batch={batch}/GPU, fp64, interleaved; "
                        "step = tri sweep + penta sweep + fused CH step",
            "n": n, "batch_per_gpu": batch}


def run_reference(args):
    """--impl reference: the oracle as it stands, on this box's host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    oracle.build()
    n, sample = args.n, min(args.batch, 16384)
    step, state = oracle_step_fn(n, sample, args.seed)
    for _ in range(max(args.warmup, 1)):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    value = 3.0 * sample * args.steps / dt
    desc = f"first {sample} systems of the N={n} batch per step (tri + penta + CH step)"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic (seeded; DESIGN.md input recipe)",
        "config": {**workload_config(n, args.batch), "parallelism": "host cores (rank 0 only)",
                   "sample_systems_per_step": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": state["cores"], "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def cpu_baseline(n, batch, seed, budget_s=10.0, budget_1core_s=5.0):
    """The oracle timed on this box's host cores on a bounded sample of the same workload: all cores, then one."""
    import oracle
    oracle.build()

    def timed(sample, nthreads, budget):
        step, state = oracle_step_fn(n, sample, seed, nthreads=nthreads)
        step()  # warm-up (page faults, OpenMP team start)
        t0 = time.perf_counter()
        step()
        t1 = time.perf_counter() - t0
        reps = int(max(1, min(50, math.ceil(budget / max(t1, 1e-3)))))
        t0 = time.perf_counter()
        for _ in range(reps):
            step()
        dt = time.perf_counter() - t0
        return 3.0 * sample * reps / dt, state["cores"], reps, dt

    sample = min(batch, 65536)
    v, cores, reps, dt = timed(sample, 0, budget_s)
    s1 = min(batch, 8192)
    v1, _, reps1, dt1 = timed(s1, 1, budget_1core_s)
    return {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "value_1core": v1,
            "sample": f"{reps} steps x {sample} systems on {cores} cores ({dt:.1f} s); 1 core: {reps1} x {s1} systems "
                      f"({dt1:.1f} s); N={n}, tri + penta + CH step per step"}


# ---------------------------------------------------------------------------------------------------
# ncu traffic of the dominant kernel, from the committed capture (never a pasted constant)
# ---------------------------------------------------------------------------------------------------
def ncu_traffic(tag, build_id):
    """Mean dram__bytes_read.sum + dram__bytes_write.sum per launch of sweep_kernel<tag> in profiles/r02_traffic.csv,
    or None when the capture is missing, is of another build of the library, or does not hold that kernel."""
    try:
        md = open(TRAFFIC_MD).read()
        m = re.search(r"build_id:\s*`?([0-9a-f]+)`?", md)
        if not m or m.group(1) != build_id:
            return None
        per_launch = {}
        with open(TRAFFIC_CSV, newline="") as f:
            rows = [r for r in f if r.startswith('"')]
        for r in csv.DictReader(rows):
            if f"sweep_kernel<{tag}>" not in r["Kernel Name"]:
                continue
            if r["Metric Name"] not in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                continue
            v = float(r["Metric Value"].replace(",", ""))
            scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(r["Metric Unit"], None)
            if scale is None:
                return None
            per_launch[r["ID"]] = per_launch.get(r["ID"], 0.0) + v * scale
        if not per_launch:
            return None
        return sum(per_launch.values()) / len(per_launch)
    except Exception:
        return None


# ---------------------------------------------------------------------------------------------------
# per-config table (BASELINE.json configs 1-5) -> side file; not the headline
# ---------------------------------------------------------------------------------------------------
def time_launches(torch, fn_of_buf, bufs, launches, repeats=3):
    """Median over `repeats` of the mean CUDA-event time (ms) of `launches` back-to-back calls,
    rotating over `bufs` (so small working sets do not stay in L2)."""
    ts = []
    for _ in range(repeats):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for i in range(launches):
            fn_of_buf(bufs[i % len(bufs)])
        e1.record()
        torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1) / launches)
    ts.sort()
    return ts[len(ts) // 2]


def time_in_graph(torch, fn_of_buf, bufs, launches, repeats=3):
    """The same launches captured once in a CUDA graph and replayed: device-side cost without the host launch path."""
    s = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        for i in range(len(bufs)):
            fn_of_buf(bufs[i], s.cuda_stream)
        torch.cuda.synchronize()
        with torch.cuda.graph(g, stream=s):
            for i in range(launches):
                fn_of_buf(bufs[i % len(bufs)], s.cuda_stream)
    ts = []
    for _ in range(repeats):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        g.replay()
        e1.record()
        torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1) / launches)
    ts.sort()
    return ts[len(ts) // 2]


KIND_INDEX = {"tri": 0, "tri_periodic": 0, "tri_f32s": 0, "penta": 1, "penta_periodic": 1, "penta_f32s": 1, "ch": 2,
              "ch_periodic": 2, "tri_cn": 3, "tri_cn_periodic": 3, "penta_cn": 4, "penta_cn_periodic": 4}


def make_cell(torch, b, inputs, kind, n, batch, elem, steps_per_call=1, rotate=0):
    """(handle, fn(buf, stream=None), buffers) of one cell; buffers rotate when one would stay in L2."""
    dt = torch.float64 if elem == 8 else torch.float32
    size = n * batch * elem
    nbuf = 1 if size > 2 * L2_BYTES else int(min(64, math.ceil(4 * L2_BYTES / size)))
    nbuf = rotate if rotate > 0 else nbuf
    bufs = []
    for k in range(nbuf):
        t = torch.empty(n, batch, dtype=dt, device="cuda")
        inputs.fill_uniform_device(t, n, seed=100 + k, scale=0.1 if kind.startswith("ch") else 1.0)
        bufs.append(t)
    if kind == "tri_f32s":
        h = b.tri_factor(*inputs.tri_lhs(n, 0.5))
        fn = lambda t, s=None: b.tri_solve_batched_f32s(h, t, s)
    elif kind == "penta_f32s":
        h = b.penta_factor(*inputs.penta_lhs(n, 0.5))
        fn = lambda t, s=None: b.penta_solve_batched_f32s(h, t, s)
    elif kind in ("tri", "tri_periodic"):
        h = b.tri_factor(*inputs.tri_lhs(n, 0.5)) if kind == "tri" else b.tri_factor_periodic(*inputs.tri_lhs(n, 0.5))
        one = b.tri_solve_batched if elem == 8 else b.tri_solve_batched_f32
        fn = (lambda t, s=None: one(h, t, s)) if steps_per_call == 1 else \
            (lambda t, s=None: b.tri_solve_steps(h, t, steps_per_call, s))
    elif kind in ("penta", "penta_periodic"):
        h = b.penta_factor(*inputs.penta_lhs(n, 0.5)) if kind == "penta" else \
            b.penta_factor_periodic(*inputs.penta_lhs(n, 0.5))
        one = b.penta_solve_batched if elem == 8 else b.penta_solve_batched_f32
        fn = (lambda t, s=None: one(h, t, s)) if steps_per_call == 1 else \
            (lambda t, s=None: b.penta_solve_steps(h, t, steps_per_call, s))
    elif kind in ("tri_cn", "tri_cn_periodic"):
        # Crank-Nicolson diffusion step (eq. 9-11; periodic: the scheme of the paper's Table 1), sigma = 0.5
        h = (b.tri_factor if kind == "tri_cn" else b.tri_factor_periodic)(*inputs.tri_lhs(n, 0.5))
        fn = lambda t, s=None: b.tri_cn_step_batched(h, t, 0.5, 0.0, 0.5, steps_per_call, s)
    elif kind in ("penta_cn", "penta_cn_periodic"):
        # Crank-Nicolson hyperdiffusion step (eq. 17-19; periodic: Table 2's scheme), sigma = 0.5
        h = (b.penta_factor if kind == "penta_cn" else b.penta_factor_periodic)(*inputs.penta_lhs(n, 0.5))
        x5 = [-0.5, 2.0, -2.0, 2.0, -0.5]
        fn = lambda t, s=None: b.penta_cn_step_batched(h, t, x5, steps_per_call, s)
    else:
        h = b.penta_factor(*inputs.ch_lhs(n)) if kind == "ch" else b.penta_factor_periodic(*inputs.ch_lhs(n))
        _, alpha = inputs.ch_params(n)
        fn = lambda t, s=None: b.ch_step_batched(h, t, alpha, steps_per_call, s)
    return h, fn, bufs


def extra_table(torch, b, inputs, peak):
    """Throughput at the other BASELINE.json configs: single launches, cold (rotating over
    buffers whose total exceeds 4x L2 when one buffer would fit in L2)."""
    out = []

    def entry(name, kind, n, batch, elem, steps_per_call=1, launches=10, graph=False):
        h, fn, bufs = make_cell(torch, b, inputs, kind, n, batch, elem, steps_per_call)
        size = n * batch * elem
        fn(bufs[0])
        ms = time_launches(torch, fn, bufs, launches) / steps_per_call
        gbs = 2.0 * size / ms / 1e6
        extra = {}
        if graph:
            msg = time_in_graph(torch, fn, bufs, max(launches, len(bufs)))
            extra["ms_per_solve_in_cuda_graph"] = round(msg, 5)
            extra["frac_in_cuda_graph"] = round(2.0 * size / msg / 1e6 / peak, 4)
        if steps_per_call > 1:
            # time loops advance up to 64 steps per launch while a tile is on chip (btps_tune "fuse_steps"):
            # HBM then moves 2*N*M*sizeof(T) per launch, so the per-step figure below is an EFFECTIVE rate
            # (it may exceed the HBM peak); the same loop with one launch per step is timed beside it.
            b.btps_tune("fuse_steps", 1)
            try:
                ms1 = time_launches(torch, fn, bufs, launches) / steps_per_call
            finally:
                b.btps_tune("fuse_steps", -1)
            extra.update({"fused_steps_per_launch": min(64, steps_per_call), "ms_per_solve_one_step_per_launch": round(ms1, 5),
                          "frac_one_step_per_launch": round(2.0 * size / ms1 / 1e6 / peak, 4),
                          "note": "frac is effective (per-step algorithmic bytes / time)"})
        kidx = KIND_INDEX[kind]
        out.append({"config": name, "kind": kind, "n": n, "batch": batch, "dtype": "f64" if elem == 8 else "f32",
                    **extra, "ms_per_solve": round(ms, 5), "systems_per_s": batch / ms * 1e3,
                    "hbm_gbs": round(gbs, 1), "frac": round(gbs / peak, 4),
                    "cold": "rotating %d buffers" % len(bufs) if len(bufs) > 1 else "buffer > 2x L2",
                    "kernel": b.btps_kernel_tag(h, 12 if kind.endswith("f32s") else elem, batch, steps_per_call, kind=kidx)})
        del bufs
        torch.cuda.empty_cache()

    entry("1 (latency-bound: 512 KiB)", "tri", 64, 1024, 8, launches=64, graph=True)
    # periodic BCs, the form the paper's own benchmarks solve
    for n in (512, 1024):
        entry("f1 periodic (single solve)", "tri_periodic", n, 65536, 8)
        entry("f1 periodic (single solve)", "penta_periodic", n, 65536, 8)
        entry("f1 periodic (single step)", "ch_periodic", n, 65536, 8)
    # fp32 in HBM, fp64 arithmetic (algorithmic bytes = 2 * N * M * 4)
    for kind in ("tri_f32s", "penta_f32s"):
        for n, lb in ((512, 16), (64, 20), (256, 20), (1024, 19)):
            entry("f4 fp32 storage, fp64 sweeps", kind, n, 1 << lb, 4)
    # systems longer than 1024 rows
    for kind in ("tri", "penta"):
        for n in (2048, 4096):
            entry("f4 long systems", kind, n, 65536, 8, launches=4)
    for kind in ("tri", "penta"):
        for elem in (8, 4):
            for n in (64, 256, 1024):
                for lb in (10, 13, 16, 19, 22):  # 2^22 x 1024 x 8 B = 32 GiB, under 60 % of HBM
                    # cells of a few microseconds are bound by the host's launch path: also replayed from a CUDA graph
                    entry("4 sweep", kind, n, 1 << lb, elem, launches=10 if lb < 22 else 4,
                          graph=(n * (1 << lb) * elem <= (32 << 20)))
    # The time loops last: seconds of fp64-pipe-bound work at the board's power cap, after which the SM clock stays low for
    # a while -- single-solve cells timed right behind them read 8-20 % low (seen on the periodic cells when they followed
    # config 5).  Listed in the side file right after config 1, as BASELINE.json numbers them.
    head = len(out)
    entry("2 (100 steps per call)", "tri", 512, 65536, 8, steps_per_call=100, launches=2)
    entry("3 (100 steps per call)", "penta", 512, 65536, 8, steps_per_call=100, launches=2)
    entry("5 (1000 steps per call)", "ch", 256, 1 << 20, 8, steps_per_call=1000, launches=1)
    entry("f1 periodic CH, 2^20 runs (1000 steps per call)", "ch_periodic", 256, 1 << 20, 8, steps_per_call=1000,
          launches=1)
    return out[:1] + out[head:] + out[1:head]


# The paper's own benchmarks (Table 1; 302-335 Table 2): periodic Crank-Nicolson diffusion /
# hyperdiffusion, 1000 time steps; its numbers are a V100's for the whole step including a separate stencil pass (and
# Table 2's units are unresolved): context, not a target.  Only with --paper-tables.
PAPER_TABLE1_V100_S = {(6, 64): 0.097, (6, 256): 0.161, (6, 1024): 0.510, (12, 64): 0.101, (12, 256): 0.255,
                       (12, 1024): 1.020, (16, 64): 1.278, (16, 256): 5.015, (16, 1024): 20.268}
PAPER_TABLE2_V100 = {(6, 64): 369.902, (6, 256): 461.727, (6, 1024): 658.475, (12, 64): 460.857, (12, 256): 429.127,
                     (12, 1024): 1344.377, (16, 64): 1786.018, (16, 256): 6535.750, (16, 1024): 25893.904}


def paper_tables(torch, b, inputs, sigma=0.5, steps=1000):
    t1, t2 = [], []
    for (lb, n), paper_s in sorted(PAPER_TABLE1_V100_S.items()):
        batch = 1 << lb
        h = b.tri_factor_periodic([-sigma] * n, [1 + 2 * sigma] * n, [-sigma] * n)
        u = torch.empty(n, batch, dtype=torch.float64, device="cuda")
        inputs.fill_uniform_device(u, n, seed=7)
        fn = lambda t: b.tri_cn_step_batched(h, t, sigma, 1 - 2 * sigma, sigma, steps)
        fn(u)
        ms = time_launches(torch, fn, [u], 1)
        t1.append({"batch": batch, "n": n, "seconds_1000_steps": round(ms * 1e-3, 6), "paper_v100_seconds": paper_s})
        del u
    x5 = [-sigma, 4 * sigma, 1 - 6 * sigma, 4 * sigma, -sigma]
    for (lb, n), paper_v in sorted(PAPER_TABLE2_V100.items()):
        batch = 1 << lb
        h = b.penta_factor_periodic([sigma] * n, [-4 * sigma] * n, [1 + 6 * sigma] * n, [-4 * sigma] * n, [sigma] * n)
        u = torch.empty(n, batch, dtype=torch.float64, device="cuda")
        inputs.fill_uniform_device(u, n, seed=8)
        fn = lambda t: b.penta_cn_step_batched(h, t, x5, steps)
        fn(u)
        ms = time_launches(torch, fn, [u], 1)
        t2.append({"batch": batch, "n": n, "seconds_1000_steps": round(ms * 1e-3, 6),
                   "paper_v100_value_units_unresolved": paper_v})
        del u
    return {"table1_periodic_cn_diffusion_1000_steps": t1, "table2_periodic_cn_hyperdiffusion_1000_steps": t2,
            "note": "paper's numbers: Tesla V100, whole step incl. a separate stencil pass; context only"}


def run_cells(args):
    """--cell: time single cells (cold, CUDA events) under the given btps_tune settings; one JSON line per cell."""
    import torch
    import inputs
    import paper_2107_05395_b200 as b
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    peak, _ = peaks()
    for kv in args.tune:
        k, v = kv.split("=")
        b.btps_tune(k, int(v))
    for cell in args.cell:
        kind, n, lb, dt = cell.split(",")
        n, batch, elem = int(n), 1 << int(lb), 8 if dt == "f64" else 4
        ks = max(1, args.cell_steps)
        h, fn, bufs = make_cell(torch, b, inputs, kind, n, batch, elem, steps_per_call=ks, rotate=args.rotate)
        fn(bufs[0])
        ms = time_launches(torch, fn, bufs, (max(4, min(20, len(bufs))) if not args.rotate else 12) if ks == 1 else 2, repeats=5) / ks
        gbs = 2.0 * n * batch * elem / ms / 1e6
        kidx = KIND_INDEX[kind]
        print(json.dumps({"cell": cell, "tune": args.tune, "steps_per_call": ks, "ms": round(ms, 5), "hbm_gbs": round(gbs, 1),
                          "frac": round(gbs / peak, 4),
                          "kernel": b.btps_kernel_tag(h, 12 if kind.endswith("f32s") else elem, batch, ks, kind=kidx),
                          "plan": h.ch_plan(elem) if kind.startswith("ch") else (h.cn_plan(elem) if kind.startswith("penta_cn") else h.plan(elem))}),
              flush=True)
        del bufs
        torch.cuda.empty_cache()


# ---------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------
def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the library has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    import inputs
    import paper_2107_05395_b200 as b  # raises if libbtps.so is missing

    for kv in args.tune:
        k, v = kv.split("=")
        b.btps_tune(k, int(v))
    n, batch, K, W = args.n, args.batch, args.steps, max(args.warmup, 3)
    peak, peak_src = peaks()

    # ---- set-up: factor once (a1, a3), inputs on the host (pinned), resident copies in HBM -------
    t0 = time.perf_counter()
    h_tri = b.tri_factor(*inputs.tri_lhs(n, 0.5))
    h_pen = b.penta_factor(*inputs.penta_lhs(n, 0.5))
    h_ch = b.penta_factor(*inputs.ch_lhs(n))
    factor_ms = 1e3 * (time.perf_counter() - t0)
    _, alpha = inputs.ch_params(n)
    host = [torch.from_numpy(x).pin_memory() for x in make_host_inputs(n, batch, args.seed, rank)]
    dev = [x.cuda(non_blocking=True) for x in host]
    torch.cuda.synchronize()
    stream = torch.cuda.current_stream().cuda_stream

    def step(ev=None):
        if ev is not None:
            ev[0].record()
        b.tri_solve_batched(h_tri, dev[0], stream)
        if ev is not None:
            ev[1].record()
        b.penta_solve_batched(h_pen, dev[1], stream)
        if ev is not None:
            ev[2].record()
        b.ch_step_batched(h_ch, dev[2], alpha, 1, stream)
        if ev is not None:
            ev[3].record()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(W):
        step()
    barrier()

    # ---- timed region: exactly K steps, nothing but the library's launches on the stream ------------
    # (an event recorded between two launches would break their programmatic dependent launch pairing, so the
    #  per-kernel events are taken in a second pass of K steps below; `value` comes from this clean pass)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.15)
    launches0 = b.btps_launch_count()
    barrier()
    e0.record()
    for k in range(K):
        step()
    e1.record()
    barrier()
    launches = b.btps_launch_count() - launches0
    total_ms = e0.elapsed_time(e1)
    # ---- the same K steps captured once in a CUDA graph and replayed: what the host's launch gaps cost (context) ------
    graph_ms = None
    try:
        gs = torch.cuda.Stream()
        gstream = gs.cuda_stream
        with torch.cuda.stream(gs):
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=gs):
                for k in range(K):
                    b.tri_solve_batched(h_tri, dev[0], gstream)
                    b.penta_solve_batched(h_pen, dev[1], gstream)
                    b.ch_step_batched(h_ch, dev[2], alpha, 1, gstream)
            g.replay()
            torch.cuda.synchronize()
            g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            g0.record(gs)
            g.replay()
            g1.record(gs)
            torch.cuda.synchronize()
            graph_ms = g0.elapsed_time(g1) / K
    except Exception:
        graph_ms = None
    # ---- the same K steps again with an event between the kernels: per-kernel durations for the roofline object ----
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(K)]
    for k in range(K):
        step(evs[k])
    torch.cuda.synchronize()
    # keep the GPU busy a little longer so that nvidia-smi catches clocks under load
    t_end = time.perf_counter() + 0.6
    while time.perf_counter() < t_end:
        step()
    torch.cuda.synchronize()
    clocks = sampler.stop()

    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    ms_per_step = total_ms / K
    value = 3.0 * batch * world / (ms_per_step * 1e-3)

    kern_ms = {name: float(np.mean([evs[k][i].elapsed_time(evs[k][i + 1]) for k in range(K)]))
               for i, name in enumerate(("tri", "penta", "ch"))}
    alg_bytes = 2.0 * n * batch * 8  # one read + one write of every element
    tags = {"tri": b.btps_kernel_tag(h_tri, 8, batch, 1), "penta": b.btps_kernel_tag(h_pen, 8, batch, 1),
            "ch": b.btps_kernel_tag(h_ch, 8, batch, 1, kind=2)}
    kernels = {name: {"ms": round(ms, 5), "frac": round(alg_bytes / ms / 1e6 / peak, 4)} for name, ms in kern_ms.items()}
    # context: what a plain in-place streaming pass (torch x.mul_(1.0): one read + one write of the
    # same 256 MiB buffer) reaches on this box, next to the driver's out-of-place copy peak
    stream_ms = time_launches(torch, lambda t: t.mul_(1.0), [dev[0]], 10)
    dom = max(kern_ms, key=kern_ms.get)
    traffic = ncu_traffic(tags[dom], b.btps_build_id())
    roofline = {"bound": "hbm", "kernel": f"{dom}: sweep_kernel<{tags[dom]}>", "achieved": round(alg_bytes / kern_ms[dom] / 1e6, 1),
                "peak": peak, "unit": "GB/s", "frac": kernels[dom]["frac"], "traffic": traffic,
                "frac_of_nominal_7700": round(alg_bytes / kern_ms[dom] / 1e6 / 7700.0, 4),
                "algorithmic_bytes_per_launch": alg_bytes, "peak_source": peak_src,
                "share_of_step": round(kern_ms[dom] / sum(kern_ms.values()), 4),
                "timing": "CUDA events around each launch, mean over a second pass of the same K steps"}

    # ---- end to end through the host-buffer C-ABI calls (pinned host in, host out) ---------------
    e2e = None
    if not args.no_e2e:
        Ke = min(K, 5)
        b.tri_solve_batched_host(h_tri, host[0], 1)  # warm-up: allocates the staging buffers
        barrier()
        t0 = time.perf_counter()
        for _ in range(Ke):
            b.tri_solve_batched_host(h_tri, host[0], 1)
            b.penta_solve_batched_host(h_pen, host[1], 1)
            b.ch_step_batched_host(h_ch, host[2], alpha, 1)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([dt], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        e2e = {"value": 3.0 * batch * world * Ke / dt, "unit": UNIT, "h2d_bytes_per_step": int(3 * n * batch * 8),
               "d2h_bytes_per_step": int(3 * n * batch * 8), "steps": Ke,
               "api": "tri/penta_solve_batched_host + ch_step_batched_host (pinned host buffers)"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic (seeded; DESIGN.md input recipe)",
        "config": {**workload_config(n, batch), "l2": "inputs larger than L2 (3 x 256 MiB buffers per step)",
                   "parallelism": f"dp{world} (independent shards, no collective)"},
        "frac_of_peak_step": round(3 * alg_bytes / ms_per_step / 1e6 / peak, 4),
        "ms_per_step_in_cuda_graph": None if graph_ms is None else round(graph_ms, 5),
        "roofline": roofline, "kernels": kernels, "inplace_stream_gbs": round(alg_bytes / stream_ms / 1e6, 1),
        "factor_ms": round(factor_ms, 3), "build_id": b.btps_build_id(),
        "gpu_launches": int(launches), "clocks": clocks, "e2e": e2e,
    }
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(n, batch, args.seed)
    if rank == 0 and world == 1 and not args.no_extra:
        del dev
        torch.cuda.empty_cache()
        side = {"build_id": b.btps_build_id(), "peak_gbs": peak, "peak_source": peak_src,
                "configs": extra_table(torch, b, inputs, peak)}
        if args.paper_tables:
            side["paper_tables"] = paper_tables(torch, b, inputs)
        try:
            with open(args.side_file, "w") as f:
                json.dump(side, f, indent=1)
            line["configs_file"] = os.path.relpath(args.side_file, ROOT)
        except OSError:
            line["configs_file"] = None
        # the target cells of north_star: plain tri / penta solves at batch >= 2^16
        tgt = [c for c in side["configs"] if c["config"] == "4 sweep" and c["batch"] >= 65536]
        worst = min(tgt, key=lambda c: c["frac"])
        line["config4_cells_ge_2p16"] = {"n": len(tgt), "below_0.70": sum(c["frac"] < 0.70 for c in tgt),
                                         "min_frac": worst["frac"],
                                         "min_cell": f'{worst["kind"]} N={worst["n"]} 2^{int(math.log2(worst["batch"]))} {worst["dtype"]}'}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.cell:
        run_cells(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
