"""The example scripts under paper_2107_05395_b200/examples are commands that profiles/*.md name: they must keep
running.  CPU: every script parses its arguments without touching CUDA.  GPU: a small run of each through the C-ABI."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
EXAMPLES = ("coarsening",)


def _run(args, timeout=300):
    return subprocess.run([sys.executable, "-m"] + args, cwd=ROOT, capture_output=True, text=True, timeout=timeout)


@pytest.mark.parametrize("name", EXAMPLES)
def test_example_help(name):
    r = _run([f"paper_2107_05395_b200.examples.{name}", "--help"])
    assert r.returncode == 0, r.stderr
    assert "usage" in r.stdout


@pytest.mark.gpu
def test_coarsening_runs_small():
    r = _run(["paper_2107_05395_b200.examples.coarsening", "--runs", "4096", "--T", "0.05"])
    assert r.returncode == 0, r.stderr  # shorter than the regression window: statistic printed, no fit
    r = _run(["paper_2107_05395_b200.examples.coarsening", "--runs", "4096", "--T", "0.05", "--fit-from", "0.01"])
    assert r.returncode == 0, r.stderr
    assert "lbar(T)" in r.stdout
