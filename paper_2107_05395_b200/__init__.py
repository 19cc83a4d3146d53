"""paper_2107_05395_b200 -- B200-native batched shared-LHS tridiagonal / pentadiagonal solves
and the fused Cahn-Hilliard step (hot path of arxiv/paper_2107_05395).

Thin ctypes binding over the C-ABI in ``include/btps.h`` (same names, argument marshalling
only; every step of the path runs in the CUDA kernels of ``csrc/``).  PyTorch is used by callers
for device memory and streams only.  There is no CPU fallback: if ``libbtps.so`` has not been
built (``python -m paper_2107_05395_b200.build``) the first use of any binding name raises
ImportError.  (The binding is resolved on first attribute access so that the build module of
this package can be run before the library exists.)
"""
_NAMES = (
    "BtpsError", "TriHandle", "PentaHandle", "tri_factor", "tri_factor_periodic", "penta_factor", "penta_factor_periodic",
    "tri_solve_batched", "tri_solve_batched_f32", "penta_solve_batched", "penta_solve_batched_f32",
    "tri_solve_batched_f32s", "penta_solve_batched_f32s",
    "tri_solve_steps", "penta_solve_steps", "ch_step_batched", "ch_step_batched_stat", "tri_cn_step_batched", "penta_cn_step_batched",
    "tri_solve_batched_host", "penta_solve_batched_host", "ch_step_batched_host", "tri_solve_batched_host_static",
    "STATIC_SCRATCH_BYTES",
    "btps_last_error", "btps_plan_info", "btps_tune", "btps_launch_count", "btps_kernel_tag", "btps_build_id", "lib_path",
    "EXPORTS",
)
__all__ = list(_NAMES)


def __getattr__(name):
    if name in _NAMES:
        from . import binding  # raises ImportError when libbtps.so is missing
        return getattr(binding, name)
    raise AttributeError(f"module {__name__!r} has no attribute {name!r}")
