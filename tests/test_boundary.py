"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/btps.h declares (no compute call is made: there is no GPU here), and the binding lists
the same names.  Also pins the seeded input generator (host side) that both arms draw from."""
import ctypes
import os
import re

import numpy as np

import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "btps.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"BTPS_API\s+[\w\s\*]+?\b(\w+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = _declared_symbols()
    for must in ("tri_factor", "penta_factor", "tri_solve_batched", "penta_solve_batched",
                 "ch_step_batched", "tri_destroy", "penta_destroy", "btps_last_error"):
        assert must in names


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2107_05395_b200 import build as b
    path = b.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    for name in _declared_symbols():
        assert hasattr(lib, name), f"libbtps.so does not export {name}"


def test_binding_lists_the_same_names():
    import paper_2107_05395_b200 as pkg
    assert sorted(pkg.EXPORTS) == _declared_symbols()
    for name in pkg.EXPORTS:
        if name not in ("tri_destroy", "penta_destroy", "btps_error_string"):
            assert callable(getattr(pkg, name)), name


def test_error_string_and_argument_errors_need_no_gpu():
    lib = ctypes.CDLL(os.path.join(ROOT, "paper_2107_05395_b200", "libbtps.so"))
    lib.btps_error_string.restype = ctypes.c_char_p
    assert lib.btps_error_string(0) == b"ok"
    lib.tri_factor.restype = ctypes.c_void_p
    lib.tri_factor.argtypes = [ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    assert lib.tri_factor(0, None, None, None) is None      # n < 1 -> NULL, BTPS_E_ARG
    row = ctypes.c_int(-1)
    assert lib.btps_last_error(ctypes.byref(row)) == -1
    # zero pivot is detected on the host before any device work
    z = (ctypes.c_double * 3)(0.0, 0.0, 0.0)
    assert lib.tri_factor(3, z, z, z) is None
    assert lib.btps_last_error(ctypes.byref(row)) == -2 and row.value == 1


def test_oracle_and_product_share_no_code():
    """oracle/ imports nothing from the package and the package nothing from oracle/."""
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2107_05395_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "oracle.c" not in text and "liboracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2107_05395_b200" not in text.replace("paper_2107_05395_b200/", ""), f
            assert "btps.h" not in text and "libbtps" not in text, f


# ---- input generator (host) ----------------------------------------------------------------------

def test_generator_is_keyed_on_system_and_row_not_on_batch():
    full = inputs.uniform_rhs(16, 100, seed=3)
    sub = inputs.uniform_rhs(16, 7, seed=3, systems=np.arange(40, 47))
    assert np.array_equal(full[:, 40:47], sub)
    assert not np.array_equal(full, inputs.uniform_rhs(16, 100, seed=4))


def test_generator_range_and_moments():
    x = inputs.uniform_rhs(64, 4096, seed=0)
    assert x.min() >= -1.0 and x.max() < 1.0
    assert abs(x.mean()) < 5e-3 and abs(x.var() - 1.0 / 3.0) < 5e-3
    # fp32 inputs are the fp64 values rounded
    assert np.array_equal(inputs.uniform_rhs(8, 8, seed=1, dtype=np.float32),
                          inputs.uniform_rhs(8, 8, seed=1).astype(np.float32))


def test_splitmix_finaliser_known_value():
    """mix(0) of the SplitMix64 finaliser is 0; mix is a bijection (spot check: no collisions)."""
    z = inputs._mix(np.arange(0, 4096, dtype=np.uint64))
    assert z[0] == 0 and np.unique(z).size == 4096


def test_config_recipes():
    a, b, c = inputs.tri_lhs(5, 0.5)
    assert (a == -0.5).all() and (b == 2.0).all() and (c == -0.5).all()
    e, a, d, c, f = inputs.penta_lhs(5, 0.5)
    assert (e == 0.5).all() and (a == -2.0).all() and (d == 4.0).all() and (c == -2.0).all() and (f == 0.5).all()
    sigma, alpha = inputs.ch_params(256)
    assert abs(sigma - 1.3778768139120494) < 1e-12 and abs(alpha - 0.08300231363980311) < 1e-14
    u0, k, A = inputs.sine_modes_u0(32, 10, seed=0)
    assert k.min() >= 1 and k.max() <= 16 and u0.shape == (32, 10)
