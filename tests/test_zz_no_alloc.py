"""tri_solve_batched_host_static (include/btps.h): the host-buffer solve that allocates nothing -- its device staging is
a fixed `static __device__` array of BTPS_STATIC_SCRATCH_BYTES inside the library instead of cudaMalloc'd buffers.

Checked against the existing paths (tri_solve_steps on a device buffer, tri_solve_batched_host) and the oracle, on two
calls in a row that share the array (the second smaller and of another shape, so anything the first call left behind
would show), plus the size limit.  Collected last on purpose (file name): the run is `pytest -x`.
"""
import numpy as np
import pytest

import inputs
import oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_STEPS = 1e-10   # BASELINE.json: fp64 after time steps
LIMIT = 32 << 20    # btps.h BTPS_STATIC_SCRATCH_BYTES


@pytest.fixture(scope="module")
def lib():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    import paper_2107_05395_b200 as b
    return b


def rel_err(got, ref):
    return float(np.max(np.abs(got - ref)) / max(np.max(np.abs(ref)), 1e-300))


def existing_path(lib, h, rhs, nsteps):
    d = torch.from_numpy(rhs).cuda()
    lib.tri_solve_steps(h, d, nsteps)
    return d.cpu().numpy()


def test_static_scratch_matches_existing_path_on_two_calls_in_a_row(lib):
    assert lib.STATIC_SCRATCH_BYTES == LIMIT
    # call 1 fills the whole array (512 * 8192 * 8 = 32 MiB, the limit exactly); call 2 is smaller, ragged in n and batch
    # and periodic, so it runs other kernels on the front of the same array while the rest still holds call 1's state
    cases = [(512, 8192, 1, False, 7), (100, 1003, 3, True, 8)]
    handles, rhs0, want = [], [], []
    for n, batch, nsteps, periodic, seed in cases:
        lhs = inputs.tri_lhs(n, 0.5)
        h = (lib.tri_factor_periodic if periodic else lib.tri_factor)(*lhs)
        r = inputs.uniform_rhs(n, batch, seed=seed)
        handles.append(h)
        rhs0.append(r)
        want.append(existing_path(lib, h, r.copy(), nsteps))
    torch.cuda.synchronize()
    got = [r.copy() for r in rhs0]
    for (n, batch, nsteps, periodic, seed), h, g in zip(cases, handles, got):   # the two calls, back to back
        lib.tri_solve_batched_host_static(h, g, nsteps)
    for (n, batch, nsteps, periodic, seed), h, g, w, r in zip(cases, handles, got, want, rhs0):
        assert rel_err(g, w) <= TOL_STEPS, (n, batch)
        ref = r.copy()
        if periodic:
            oracle.tri_periodic_solve_interleaved(oracle.tri_periodic_factor(*inputs.tri_lhs(n, 0.5)), ref, nsteps=nsteps)
        else:
            oracle.tri_solve_interleaved(oracle.tri_factor(*inputs.tri_lhs(n, 0.5)), ref, nsteps=nsteps)
        assert rel_err(g, ref) <= TOL_STEPS, (n, batch)
    # the other existing host path, and a pinned torch tensor as the buffer, on a caller's stream
    n, batch, nsteps = cases[0][:3]
    a = rhs0[0].copy()
    lib.tri_solve_batched_host(handles[0], a, nsteps)
    b = torch.from_numpy(rhs0[0].copy()).pin_memory()
    s = torch.cuda.Stream()
    lib.tri_solve_batched_host_static(handles[0], b, nsteps, stream=s.cuda_stream)
    assert rel_err(b.numpy(), a) <= TOL_STEPS


def test_static_scratch_allocates_no_device_memory(lib):
    n, batch = 256, 4096
    h = lib.tri_factor(*inputs.tri_lhs(n, 0.5))
    r = inputs.uniform_rhs(n, batch, seed=3)
    lib.tri_solve_batched_host_static(h, r, 2)      # first use of these kernels may load their module
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(2):
        lib.tri_solve_batched_host_static(h, r, 2)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0


def test_static_scratch_rejects_sizes_beyond_the_limit(lib):
    n = 512
    h = lib.tri_factor(*inputs.tri_lhs(n, 0.5))
    batch = LIMIT // (8 * n) + 1
    r = np.ones((n, batch))
    with pytest.raises(lib.BtpsError) as ei:
        lib.tri_solve_batched_host_static(h, r, 1)
    assert ei.value.code == -6 and "BTPS_STATIC_SCRATCH_BYTES" in str(ei.value)
    assert np.all(r == 1.0)                          # rejected before anything was issued
    ok = np.ones((n, batch - 1))
    lib.tri_solve_batched_host_static(h, ok, 1)      # the limit itself is accepted
    assert np.all(np.isfinite(ok)) and not np.all(ok == 1.0)
