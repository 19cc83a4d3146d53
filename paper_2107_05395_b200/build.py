"""Build the CUDA library (libbtps.so) and the device-side input generator (libbtps_inputs.so)
in-tree with nvcc for sm_100a.  ``python -m paper_2107_05395_b200.build`` or ``build()``.

nvcc cross-compiles without a GPU; the resulting .so files are git-ignored but travel to the
GPU box with the repo snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libbtps.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC,-fvisibility=hidden"]
# BTPS_TUNING_VARIANTS=1: also compile the partitioned kernels with 8 / 16 rows per thread (btps_tune("rows", 8 | 16)),
# which only A/B measurements use; the default library leaves them out (a third of its size)
if os.environ.get("BTPS_TUNING_VARIANTS", "") not in ("", "0"):
    NVCC_FLAGS = NVCC_FLAGS + ["-DBTPS_TUNING_VARIANTS"]
UNITS = ["btps.cu"] + [f"inst_{k}_{t}.cu" for k in ("tri", "penta", "ch", "trip", "pentap", "chp") for t in ("f64", "f32")] + \
        ["inst_tricn_f64.cu", "inst_tricnp_f64.cu", "inst_pentacn_f64.cu", "inst_pentacnp_f64.cu",
         "inst_pentapf_f64.cu", "inst_pentapf_f32.cu", "inst_chpf_f64.cu", "inst_pentacnpf_f64.cu",
         "inst_tripf_f64.cu", "inst_tripf_f32.cu", "inst_tricnpf_f64.cu", "inst_f32s.cu"]
HEADERS = ["sweep.cuh", "inst_common.cuh", os.path.join(ROOT, "include", "btps.h")]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _newest(paths) -> float:
    return max(os.path.getmtime(p if os.path.isabs(p) else os.path.join(CSRC, p)) for p in paths)


def _run(cmd):
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("command failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
    return r.stdout + r.stderr


def build_id() -> str:
    """Hash of the kernel sources (csrc/*.cu, *.cuh) and the compile flags: what btps_build_id() returns."""
    import hashlib
    h = hashlib.sha1()
    for name in sorted(UNITS) + [x for x in HEADERS if not os.path.isabs(x)]:
        with open(name if os.path.isabs(name) else os.path.join(CSRC, name), "rb") as f:
            h.update(f.read())
    h.update(" ".join(NVCC_FLAGS).encode())
    return h.hexdigest()[:12]


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/*.cu -> libbtps.so.  Returns the library path."""
    os.makedirs(OBJ, exist_ok=True)
    src_time = _newest(UNITS + HEADERS + [os.path.abspath(__file__)])
    bid = build_id()
    stamp = os.path.join(OBJ, "build_id.txt")
    same_flags = os.path.exists(stamp) and open(stamp).read().strip() == bid
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= src_time and same_flags:
        return LIB
    nvcc = _nvcc()

    def compile_one(unit):
        obj = os.path.join(OBJ, unit.replace(".cu", ".o"))
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
              ([f'-DBTPS_BUILD_ID="{bid}"'] if unit == "btps.cu" else []) + \
              ["-c", os.path.join(CSRC, unit), "-o", obj]
        out = _run(cmd)
        if verbose:
            sys.stderr.write(out)
        return obj

    with ThreadPoolExecutor(max_workers=len(UNITS)) as ex:
        objs = list(ex.map(compile_one, UNITS))
    tmp = LIB + f".tmp{os.getpid()}"
    _run([nvcc, "-shared", "-o", tmp] + objs + ["-gencode", "arch=compute_100a,code=sm_100a",
                                                  "-Xcompiler", "-fPIC", "-cudart", "static"])
    os.replace(tmp, LIB)
    with open(stamp, "w") as f:
        f.write(bid + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
