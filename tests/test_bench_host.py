"""Host-side logic of bench.py that needs no GPU: the ncu traffic lookup (roofline.traffic is read from a committed capture,
matched by kernel tag and library build id, never a pasted constant) and the shape of the reference arm's line."""
import json
import os
import re
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402


def _capture_build_id():
    m = re.search(r"build_id:\s*`?([0-9a-f]+)`?", open(bench.TRAFFIC_MD).read())
    assert m, "profiles/r02_traffic.md must name the build it was captured with"
    return m.group(1)


def test_traffic_lookup_matches_kernel_and_build():
    bid = _capture_build_id()
    ch = bench.ncu_traffic("double, 2, 32, 0, 2, 1, 1, 0, 0, double", bid)
    tri = bench.ncu_traffic("double, 2, 32, 0, 0, 1, 1, 0, 0, double", bid)
    alg = 2.0 * 512 * 65536 * 8
    # one read of the buffer plus most of one write inside the launch (the rest is still dirty in L2): no re-reads
    assert ch is not None and 0.80 * alg <= ch <= 1.02 * alg
    assert tri is not None and 0.80 * alg <= tri <= 1.02 * alg
    # another build of the library, or a kernel the capture does not hold: no number rather than a stale one
    assert bench.ncu_traffic("double, 2, 32, 0, 2, 1, 1, 0, 0, double", "0" * 12) is None
    assert bench.ncu_traffic("double, 2, 32, 0, 9, 1, 1, 0, 0, double", bid) is None


def test_traffic_capture_is_of_the_committed_sources():
    """The capture's build id equals the hash of the kernel sources in the tree (default build flags): a kernel change
    without a new capture makes bench.py print traffic = null, and this test says so here first (as a skip: a stale
    capture is reported as no number, never as a wrong one)."""
    import pytest
    from paper_2107_05395_b200 import build
    if os.environ.get("BTPS_TUNING_VARIANTS", "") not in ("", "0"):
        pytest.skip("tuning build: another build id by construction")
    if build.build_id() != _capture_build_id():
        pytest.skip(f"profiles/r02_traffic.csv is of build {_capture_build_id()}, the sources are {build.build_id()}: "
                    "bench.py will print roofline.traffic = null until the capture is taken again")


def test_reference_arm_prints_one_compact_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "1",
                        "--batch", "512", "--n", "64"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr
    line = r.stdout.strip().splitlines()[-1]
    d = json.loads(line)
    assert len(line) < 2500
    assert d["impl"] == "reference" and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["gpu_launches"] == 0
