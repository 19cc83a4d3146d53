"""paper_2107_05395_b200 -- B200-native batched shared-LHS tridiagonal / pentadiagonal solves
and the fused Cahn-Hilliard step (hot path of arxiv/paper_2107_05395).

Thin ctypes binding over the C-ABI in ``include/btps.h`` (same names, argument marshalling
only; every step of the path runs in the CUDA kernels of ``csrc/``).  PyTorch is used by callers
for device memory and streams only.  There is no CPU fallback: if ``libbtps.so`` has not been
built (``python -m paper_2107_05395_b200.build``) importing the binding raises.
"""
from .binding import (  # noqa: F401
    BtpsError,
    TriHandle,
    PentaHandle,
    tri_factor,
    penta_factor,
    tri_solve_batched,
    tri_solve_batched_f32,
    penta_solve_batched,
    penta_solve_batched_f32,
    tri_solve_steps,
    penta_solve_steps,
    ch_step_batched,
    tri_solve_batched_host,
    penta_solve_batched_host,
    ch_step_batched_host,
    btps_last_error,
    btps_plan_info,
    btps_tune,
    btps_launch_count,
    lib_path,
    EXPORTS,
)
