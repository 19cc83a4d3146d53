"""GPU parity: the CUDA path (through the C-ABI binding) against the CPU oracle, element by element,
on the same seeded inputs.  Tolerances are BASELINE.json's: max|gpu-oracle| / max|oracle| <= 1e-12
(fp64 single solve), 1e-10 (fp64 after all time steps), 1e-5 (fp32 GPU vs fp64 oracle).
"""
import numpy as np
import pytest

import inputs
import oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_SINGLE = 1e-12
TOL_STEPS = 1e-10
TOL_F32 = 1e-5


@pytest.fixture(scope="module")
def lib():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    import paper_2107_05395_b200 as b
    return b


def rel_err(got, ref):
    return float(np.max(np.abs(got - ref)) / max(np.max(np.abs(ref)), 1e-300))


def dev(x):
    return torch.from_numpy(x).cuda()


def rand_tri(n, seed):
    rng = np.random.default_rng(seed)
    a = rng.uniform(-1, 1, n)
    c = rng.uniform(-1, 1, n)
    b = np.abs(a) + np.abs(c) + rng.uniform(0.5, 1.5, n)
    b *= rng.choice([-1.0, 1.0], n)
    return a, b, c


def rand_penta(n, seed):
    rng = np.random.default_rng(seed)
    e, a, c, f = (rng.uniform(-1, 1, n) for _ in range(4))
    d = np.abs(e) + np.abs(a) + np.abs(c) + np.abs(f) + rng.uniform(0.5, 1.5, n)
    d *= rng.choice([-1.0, 1.0], n)
    return e, a, d, c, f


# ---- config 1 ----------------------------------------------------------------------------------

def test_config1_tri_single_solve(lib):
    n, batch = 64, 1024
    a, b, c = inputs.tri_lhs(n, 0.5)
    rhs = inputs.uniform_rhs(n, batch, seed=0)
    ref = rhs.copy()
    oracle.tri_solve_interleaved(oracle.tri_factor(a, b, c), ref)
    h = lib.tri_factor(a, b, c)
    d = dev(rhs)
    lib.tri_solve_batched(h, d)
    torch.cuda.synchronize()
    assert rel_err(d.cpu().numpy(), ref) <= TOL_SINGLE


# ---- general LHS, edge sizes, ragged batches ----------------------------------------------------

SIZES = [1, 2, 3, 4, 5, 7, 8, 9, 16, 17, 31, 32, 33, 64, 100, 255, 256, 512, 777, 1024, 1500, 2048, 4096,
         5000]


@pytest.mark.parametrize("n", SIZES)
def test_tri_general_lhs_sizes(lib, n):
    a, b, c = rand_tri(n, 100 + n)
    fac = oracle.tri_factor(a, b, c)
    h = lib.tri_factor(a, b, c)
    for batch in (1, 33, 257 if n > 1024 else 1000):
        rhs = inputs.uniform_rhs(n, batch, seed=n)
        ref = rhs.copy()
        oracle.tri_solve_interleaved(fac, ref)
        d = dev(rhs)
        lib.tri_solve_batched(h, d)
        assert rel_err(d.cpu().numpy(), ref) <= TOL_SINGLE, (n, batch, h.plan())


@pytest.mark.parametrize("n", SIZES)
def test_penta_general_lhs_sizes(lib, n):
    e, a, d_, c, f = rand_penta(n, 200 + n)
    fac = oracle.penta_factor(e, a, d_, c, f)
    h = lib.penta_factor(e, a, d_, c, f)
    for batch in (1, 33, 257 if n > 1024 else 1000):
        rhs = inputs.uniform_rhs(n, batch, seed=n + 1)
        ref = rhs.copy()
        oracle.penta_solve_interleaved(fac, ref)
        d = dev(rhs)
        lib.penta_solve_batched(h, d)
        assert rel_err(d.cpu().numpy(), ref) <= TOL_SINGLE, (n, batch, h.plan())


@pytest.mark.parametrize("n", [1, 5, 33, 64, 256, 1024, 5000])
def test_fp32_tri_and_penta(lib, n):
    for kind in ("tri", "penta"):
        if kind == "tri":
            lhs = inputs.tri_lhs(n, 0.5)
            fac, h = oracle.tri_factor(*lhs), lib.tri_factor(*lhs)
        else:
            lhs = inputs.penta_lhs(n, 0.5)
            fac, h = oracle.penta_factor(*lhs), lib.penta_factor(*lhs)
        for batch in (1, 31, 1000, 1001):   # odd batches take the scalar (unvectorised) kernel
            rhs32 = inputs.uniform_rhs(n, batch, seed=3, dtype=np.float32)
            ref = rhs32.astype(np.float64)
            (oracle.tri_solve_interleaved if kind == "tri" else oracle.penta_solve_interleaved)(fac, ref)
            d = dev(rhs32)
            (lib.tri_solve_batched_f32 if kind == "tri" else lib.penta_solve_batched_f32)(h, d)
            assert rel_err(d.cpu().numpy().astype(np.float64), ref) <= TOL_F32, (kind, n, batch)


def test_unaligned_base_pointer_fp32(lib):
    """A float buffer that starts 4 bytes off 8-byte alignment must take the scalar path."""
    n, batch = 64, 512
    lhs = inputs.tri_lhs(n, 0.5)
    fac, h = oracle.tri_factor(*lhs), lib.tri_factor(*lhs)
    rhs32 = inputs.uniform_rhs(n, batch, seed=5, dtype=np.float32)
    ref = rhs32.astype(np.float64)
    oracle.tri_solve_interleaved(fac, ref)
    big = torch.empty(n * batch + 1, dtype=torch.float32, device="cuda")
    view = big[1:]
    view.copy_(torch.from_numpy(rhs32).reshape(-1))
    lib.tri_solve_batched_f32(h, view)
    assert rel_err(view.cpu().numpy().reshape(n, batch).astype(np.float64), ref) <= TOL_F32


# ---- properties ----------------------------------------------------------------------------------

def test_result_independent_of_batch_position(lib):
    """A system's solution must not depend on where it sits in the batch or on the batch size
    (bitwise: one code path per plan)."""
    n = 512
    lhs = inputs.penta_lhs(n, 0.5)
    h = lib.penta_factor(*lhs)
    full = inputs.uniform_rhs(n, 4096, seed=9)
    d_full = dev(full)
    lib.penta_solve_batched(h, d_full)
    sub = np.ascontiguousarray(full[:, 1000:1777])
    d_sub = dev(sub)
    lib.penta_solve_batched(h, d_sub)
    assert np.array_equal(d_full.cpu().numpy()[:, 1000:1777], d_sub.cpu().numpy())


def test_handle_shared_by_two_streams(lib):
    n, batch = 256, 8192
    lhs = inputs.tri_lhs(n, 0.5)
    h = lib.tri_factor(*lhs)
    x1, x2 = dev(inputs.uniform_rhs(n, batch, seed=1)), dev(inputs.uniform_rhs(n, batch, seed=2))
    ref1, ref2 = x1.clone(), x2.clone()
    lib.tri_solve_batched(h, ref1)
    lib.tri_solve_batched(h, ref2)
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    for _ in range(3):
        y1, y2 = x1.clone(), x2.clone()
        torch.cuda.synchronize()
        lib.tri_solve_batched(h, y1, stream=s1.cuda_stream)
        lib.tri_solve_batched(h, y2, stream=s2.cuda_stream)
        torch.cuda.synchronize()
        assert torch.equal(y1, ref1) and torch.equal(y2, ref2)


def test_linearity(lib):
    n, batch = 100, 64
    lhs = rand_penta(n, 5)
    h = lib.penta_factor(*lhs)
    x, y = inputs.uniform_rhs(n, batch, seed=1), inputs.uniform_rhs(n, batch, seed=2)
    dx, dy, dz = dev(x), dev(y), dev(2.0 * x - 3.0 * y)
    for t in (dx, dy, dz):
        lib.penta_solve_batched(h, t)
    z = (2.0 * dx - 3.0 * dy).cpu().numpy()
    assert rel_err(dz.cpu().numpy(), z) <= 1e-13


def test_two_pass_kernel_matches(lib):
    """The paper-form two-pass kernel (used beyond the on-chip limit) against the oracle at a size
    the register-resident plan also covers."""
    n, batch = 256, 1000
    try:
        lib.btps_tune("force_two_pass", 1)
        lt, lp = inputs.tri_lhs(n), inputs.penta_lhs(n)
        ht, hp = lib.tri_factor(*lt), lib.penta_factor(*lp)
    finally:
        lib.btps_tune("force_two_pass", -1)
    assert ht.plan()["rows_per_thread"] == 0
    rhs = inputs.uniform_rhs(n, batch, seed=4)
    for h, fac, solve, osolve in ((ht, oracle.tri_factor(*lt), lib.tri_solve_batched, oracle.tri_solve_interleaved),
                                  (hp, oracle.penta_factor(*lp), lib.penta_solve_batched,
                                   oracle.penta_solve_interleaved)):
        ref = rhs.copy()
        osolve(fac, ref)
        d = dev(rhs)
        solve(h, d)
        assert rel_err(d.cpu().numpy(), ref) <= TOL_SINGLE
    sigma, alpha = inputs.ch_params(n)
    c0 = 0.1 * inputs.uniform_rhs(n, batch, seed=6)
    ref = c0.copy()
    oracle.ch_step_interleaved(oracle.penta_factor(*inputs.ch_lhs(n)), ref, alpha, nsteps=20)
    try:
        lib.btps_tune("force_two_pass", 1)
        hc = lib.penta_factor(*inputs.ch_lhs(n))
    finally:
        lib.btps_tune("force_two_pass", -1)
    d = dev(c0)
    lib.ch_step_batched(hc, d, alpha, 20)
    assert rel_err(d.cpu().numpy(), ref) <= TOL_STEPS


@pytest.mark.parametrize("rows,lanes,vec", [(8, 32, 1), (16, 32, 1), (16, 16, 2), (32, 16, 1), (32, 8, 1), (16, 4, 2)])
def test_plan_variants(lib, rows, lanes, vec):
    """Every (rows per thread, lanes, vector width) variant the tuner can pick gives the same answer."""
    n, batch = 200, 600
    lt, lp = rand_tri(n, 1), rand_penta(n, 2)
    try:
        try:
            lib.btps_tune("rows", rows)
        except lib.BtpsError:
            pytest.skip("8 / 16 rows per thread with several partitions: tuning build only (BTPS_TUNING_VARIANTS=1)")
        lib.btps_tune("lanes", lanes)
        lib.btps_tune("vec", vec)
        ht, hp = lib.tri_factor(*lt), lib.penta_factor(*lp)
    finally:
        for k in ("rows", "lanes", "vec"):
            lib.btps_tune(k, -1)
    assert ht.plan()["rows_per_thread"] == rows
    rhs = inputs.uniform_rhs(n, batch, seed=8)
    ref = rhs.copy()
    oracle.tri_solve_interleaved(oracle.tri_factor(*lt), ref)
    d = dev(rhs)
    lib.tri_solve_batched(h=ht, rhs=d)
    assert rel_err(d.cpu().numpy(), ref) <= TOL_SINGLE
    ref = rhs.copy()
    oracle.penta_solve_interleaved(oracle.penta_factor(*lp), ref)
    d = dev(rhs)
    lib.penta_solve_batched(hp, d)
    assert rel_err(d.cpu().numpy(), ref) <= TOL_SINGLE


# ---- time stepping (configs 2, 3, 5) at reduced batch --------------------------------------------

def test_config2_diffusion_100_steps(lib):
    n, batch, steps = 512, 3000, 100
    lhs = inputs.tri_lhs(n, 0.5)
    u0, k, A = inputs.sine_modes_u0(n, batch, seed=0)
    ref = u0.copy()
    oracle.tri_solve_interleaved(oracle.tri_factor(*lhs), ref, nsteps=steps)
    h = lib.tri_factor(*lhs)
    d = dev(u0)
    lib.tri_solve_steps(h, d, steps)
    got = d.cpu().numpy()
    assert rel_err(got, ref) <= TOL_STEPS
    # exact modal decay (closed form, independent of both implementations)
    x = np.arange(1, n + 1) / (n + 1)
    lam = 1.0 + 4 * 0.5 * np.sin(k * np.pi / (2 * (n + 1))) ** 2
    exact = sum((A[m] * lam[m] ** -steps)[None, :] * np.sin(np.pi * k[m][None, :] * x[:, None]) for m in range(4))
    assert rel_err(got, exact) <= 1e-10


def test_config3_hyperdiffusion_100_steps(lib):
    n, batch, steps = 512, 3000, 100
    lhs = inputs.penta_lhs(n, 0.5)
    rhs = inputs.uniform_rhs(n, batch, seed=0)
    ref = rhs.copy()
    oracle.penta_solve_interleaved(oracle.penta_factor(*lhs), ref, nsteps=steps)
    h = lib.penta_factor(*lhs)
    d = dev(rhs)
    lib.penta_solve_steps(h, d, steps)
    assert rel_err(d.cpu().numpy(), ref) <= TOL_STEPS


def test_config5_cahn_hilliard_1000_steps(lib):
    n, batch, steps = 256, 1536, 1000
    sigma, alpha = inputs.ch_params(n)
    lhs = inputs.ch_lhs(n)
    c0 = 0.1 * inputs.uniform_rhs(n, batch, seed=0)
    ref = c0.copy()
    oracle.ch_step_interleaved(oracle.penta_factor(*lhs), ref, alpha, nsteps=steps)
    h = lib.penta_factor(*lhs)
    d = dev(c0)
    lib.ch_step_batched(h, d, alpha, steps)
    assert rel_err(d.cpu().numpy(), ref) <= TOL_STEPS


@pytest.mark.parametrize("n", [2, 3, 31, 33, 100, 777])
def test_ch_step_edge_sizes(lib, n):
    sigma, alpha = 0.7, 0.05
    lhs = inputs.penta_lhs(n, sigma)
    for batch in (1, 45, 600):
        c0 = 0.5 * inputs.uniform_rhs(n, batch, seed=n)
        ref = c0.copy()
        oracle.ch_step_interleaved(oracle.penta_factor(*lhs), ref, alpha, nsteps=3)
        h = lib.penta_factor(*lhs)
        d = dev(c0)
        lib.ch_step_batched(h, d, alpha, 3)
        assert rel_err(d.cpu().numpy(), ref) <= 1e-12, (n, batch)


def test_reverse_tile_order_same_result(lib):
    n, batch, steps = 256, 5000, 6
    lhs = inputs.penta_lhs(n, 0.5)
    h = lib.penta_factor(*lhs)
    rhs = inputs.uniform_rhs(n, batch, seed=11)
    d0, d1 = dev(rhs), dev(rhs)
    lib.penta_solve_steps(h, d0, steps)
    try:
        lib.btps_tune("reverse", 1)
        lib.penta_solve_steps(h, d1, steps)
    finally:
        lib.btps_tune("reverse", -1)
    assert torch.equal(d0, d1)


# ---- host-buffer (end-to-end) calls ---------------------------------------------------------------

def test_host_buffer_calls(lib):
    n, batch = 256, 40000   # several chunks plus a ragged last one
    lt, lp = inputs.tri_lhs(n), inputs.penta_lhs(n)
    ht, hp = lib.tri_factor(*lt), lib.penta_factor(*lp)
    rhs = inputs.uniform_rhs(n, batch, seed=12)
    pinned = torch.from_numpy(rhs.copy()).pin_memory()
    d = dev(rhs)
    lib.tri_solve_steps(ht, d, 3)
    lib.tri_solve_batched_host(ht, pinned, 3)
    assert np.array_equal(pinned.numpy(), d.cpu().numpy())
    pageable = rhs.copy()
    d = dev(rhs)
    lib.penta_solve_batched(hp, d)
    lib.penta_solve_batched_host(hp, pageable, 1)
    assert np.array_equal(pageable, d.cpu().numpy())
    sigma, alpha = inputs.ch_params(n)
    hc = lib.penta_factor(*inputs.ch_lhs(n))
    c0 = 0.1 * rhs
    d = dev(c0)
    lib.ch_step_batched(hc, d, alpha, 5)
    host = c0.copy()
    lib.ch_step_batched_host(hc, host, alpha, 5)
    assert np.array_equal(host, d.cpu().numpy())


# ---- errors ---------------------------------------------------------------------------------------

def test_error_paths(lib):
    with pytest.raises(lib.BtpsError) as ei:
        lib.tri_factor([0.0, 1.0, 1.0], [1.0, 1.0, 1.0], [1.0, 1.0, 0.0])   # b^_2 = 1 - 1*1 = 0
    assert ei.value.code == -2 and ei.value.row == 2
    with pytest.raises(lib.BtpsError):
        lib.penta_factor([0.0] * 3, [0.0] * 3, [1.0, 0.0, 1.0], [0.0] * 3, [0.0] * 3)
    h = lib.tri_factor(*inputs.tri_lhs(8))
    with pytest.raises(ValueError):
        lib.tri_solve_batched(h, torch.zeros(9, dtype=torch.float64, device="cuda"))
    with pytest.raises(ValueError):
        lib.tri_solve_batched(h, torch.zeros(8, dtype=torch.float32, device="cuda"))


def test_inputs_device_generator_bitwise(lib):
    for dtype, tdt in ((np.float64, torch.float64), (np.float32, torch.float32)):
        n, batch = 37, 1001
        host = inputs.uniform_rhs(n, batch, seed=42, scale=0.1, dtype=dtype)
        t = torch.empty(n, batch, dtype=tdt, device="cuda")
        inputs.fill_uniform_device(t, n, seed=42, scale=0.1)
        assert np.array_equal(t.cpu().numpy(), host)


# ---- kernel variants: TMA prefetch / direct loads, warp scan / serial carry walk, vector widths --------

def _solve_all(lib, n, batch, seed, f32=False):
    """tri + penta + 2 CH steps through the current tune settings; returns [(got, ref, tol, tag)]."""
    lt, lp = rand_tri(n, seed), rand_penta(n, seed + 1)
    ht, hp = lib.tri_factor(*lt), lib.penta_factor(*lp)
    dt = np.float32 if f32 else np.float64
    rhs = inputs.uniform_rhs(n, batch, seed=seed).astype(dt)
    out = []
    ref = rhs.astype(np.float64)
    oracle.tri_solve_interleaved(oracle.tri_factor(*lt), ref)
    d = dev(rhs)
    (lib.tri_solve_batched_f32 if f32 else lib.tri_solve_batched)(ht, d)
    out.append((d.cpu().numpy(), ref, TOL_F32 if f32 else TOL_SINGLE, "tri"))
    ref = rhs.astype(np.float64)
    oracle.penta_solve_interleaved(oracle.penta_factor(*lp), ref)
    d = dev(rhs)
    (lib.penta_solve_batched_f32 if f32 else lib.penta_solve_batched)(hp, d)
    out.append((d.cpu().numpy(), ref, TOL_F32 if f32 else TOL_SINGLE, "penta"))
    if not f32:
        lc = inputs.penta_lhs(n, 0.7)
        hc = lib.penta_factor(*lc)
        c0 = 0.5 * rhs
        ref = c0.copy()
        oracle.ch_step_interleaved(oracle.penta_factor(*lc), ref, 0.05, nsteps=2)
        d = dev(c0)
        lib.ch_step_batched(hc, d, 0.05, 2)
        out.append((d.cpu().numpy(), ref, TOL_SINGLE, "ch"))
    return out, ht.plan(4 if f32 else 8)


@pytest.mark.parametrize("tune", [
    dict(prefetch=0), dict(warp_scan=0), dict(prefetch=0, warp_scan=0), dict(vec=1), dict(vec=2), dict(vec=1, lanes=32),
    dict(vec=2, lanes=32), dict(lanes=8), dict(tiles_per_cta=1), dict(rows=16), dict(rows=16, vec=2), dict(pdl=0), dict(pdl=1),
])
@pytest.mark.parametrize("batch", [4096 + 64, 1001])  # 16-byte aligned pitch (TMA) / odd (direct loads, scalar tail)
def test_kernel_variants_fp64(lib, tune, batch):
    n = 300  # 10 partitions of 32 rows (padded), ragged last partition
    try:
        for k, v in tune.items():
            try:
                lib.btps_tune(k, v)
            except lib.BtpsError:
                pytest.skip("8 / 16 rows per thread with several partitions: tuning build only (BTPS_TUNING_VARIANTS=1)")
        res, plan = _solve_all(lib, n, batch, seed=21)
    finally:
        for k in tune:
            lib.btps_tune(k, -1)
    for got, ref, tol, tag in res:
        assert rel_err(got, ref) <= tol, (tag, tune, batch, plan)


@pytest.mark.parametrize("tune", [dict(), dict(vec=4), dict(vec=2), dict(vec=1), dict(prefetch=0), dict(warp_scan=0)])
@pytest.mark.parametrize("batch", [2048 + 128, 999])
def test_kernel_variants_fp32(lib, tune, batch):
    n = 300
    try:
        for k, v in tune.items():
            lib.btps_tune(k, v)
        res, plan = _solve_all(lib, n, batch, seed=22, f32=True)
    finally:
        for k in tune:
            lib.btps_tune(k, -1)
    for got, ref, tol, tag in res:
        assert rel_err(got, ref) <= tol, (tag, tune, batch, plan)


@pytest.mark.parametrize("n", [530, 545, 1000, 1024, 1500, 2500])
def test_partition_padding_and_serial_walk(lib, n):
    """n = 530/545: odd partition counts are padded so groups are whole warps; 1000/1024: 32 partitions
    (5-step scan, merged step-4 table slot); 1500/2500: more than 32 partitions -> serial carry walk."""
    for batch in (515, 2048):
        res, plan = _solve_all(lib, n, batch, seed=n)
        for got, ref, tol, tag in res:
            assert rel_err(got, ref) <= tol, (tag, n, batch, plan)
    if n <= 1024:
        assert plan["warp_scan"] == 1
    else:
        assert plan["warp_scan"] == 0   # the single-CTA fallback plan (unaligned batches); aligned ones run the cluster chain


def test_plan_reports_tma_and_ch_shape(lib):
    h = lib.penta_factor(*inputs.penta_lhs(512, 0.5))
    p, c = h.plan(8), h.ch_plan(8)
    assert p["tma_prefetch"] == 1 and c["tma_prefetch"] == 1
    assert p["partitions"] == c["partitions"] == 16
    assert p["smem_bytes"] <= 227 * 1024 and c["smem_bytes"] <= 227 * 1024
    big = lib.penta_factor(*inputs.penta_lhs(1024, 0.5))
    assert big.plan(8)["tma_prefetch"] == 1 and big.plan(8)["smem_bytes"] <= 227 * 1024


# ---- BASELINE.json's full sizes, in the launch configuration bench.py times: sampled systems ---------

def _sample_ids(batch):
    ids = np.concatenate([np.arange(0, 96), np.arange(batch - 96, batch),
                          np.arange(97, batch - 96, max(1, batch // 257))])
    return np.unique(ids).astype(np.int64)


@pytest.mark.parametrize("kind,n,lb,f32", [("tri", 512, 16, False), ("penta", 512, 16, False), ("ch", 256, 20, False),
                                           ("tri", 64, 20, False), ("penta", 1024, 18, False), ("tri", 1024, 18, True),
                                           ("penta", 256, 20, True)])
def test_full_size_sampled(lib, kind, n, lb, f32):
    batch = 1 << lb
    dtype = torch.float32 if f32 else torch.float64
    scale = 0.1 if kind == "ch" else 1.0
    d = torch.empty(n, batch, dtype=dtype, device="cuda")
    inputs.fill_uniform_device(d, n, seed=5, scale=scale)
    ids = _sample_ids(batch)
    # the oracle regenerates its subset on the host (generator keyed on (system, row), bit-identical)
    ref = inputs.uniform_rhs(n, len(ids), seed=5, scale=scale, systems=ids.astype(np.uint64))
    if f32:
        ref = ref.astype(np.float32).astype(np.float64)
    assert np.array_equal(d[:, torch.from_numpy(ids).cuda()].cpu().numpy().astype(np.float64), ref)
    if kind == "tri":
        lhs = inputs.tri_lhs(n, 0.5)
        h = lib.tri_factor(*lhs)
        (lib.tri_solve_batched_f32 if f32 else lib.tri_solve_batched)(h, d)
        oracle.tri_solve_interleaved(oracle.tri_factor(*lhs), ref)
    elif kind == "penta":
        lhs = inputs.penta_lhs(n, 0.5)
        h = lib.penta_factor(*lhs)
        (lib.penta_solve_batched_f32 if f32 else lib.penta_solve_batched)(h, d)
        oracle.penta_solve_interleaved(oracle.penta_factor(*lhs), ref)
    else:
        lhs = inputs.ch_lhs(n)
        _, alpha = inputs.ch_params(n)
        h = lib.penta_factor(*lhs)
        lib.ch_step_batched(h, d, alpha, 3)
        oracle.ch_step_interleaved(oracle.penta_factor(*lhs), ref, alpha, nsteps=3)
    got = d[:, torch.from_numpy(ids).cuda()].cpu().numpy().astype(np.float64)
    assert rel_err(got, ref) <= (TOL_F32 if f32 else TOL_SINGLE), (kind, n, batch, h.plan(4 if f32 else 8))
    assert bool(torch.isfinite(d).all())


# ---- fused time steps (several steps per launch while the tile is on chip) ---------------------------

@pytest.mark.parametrize("n,batch", [(300, 2048 + 32), (20, 640), (512, 1024), (1000, 512)])
def test_fused_steps_equal_single_step_launches(lib, n, batch):
    """tri/penta_solve_steps and ch_step_batched advance up to 64 steps per launch; the arithmetic per
    step is the same as one launch per step, so the results must be bitwise equal -- and both must
    match the oracle's step-by-step loop."""
    steps = 11  # one launch by default, 8 + 3 with fuse_steps = 8
    lt, lp, lc = inputs.tri_lhs(n, 0.5), inputs.penta_lhs(n, 0.5), inputs.penta_lhs(n, 0.7)
    rhs = inputs.uniform_rhs(n, batch, seed=31)
    c0 = 0.5 * rhs
    outs = {}
    for fuse in (1, -1, 3, 8):
        try:
            lib.btps_tune("fuse_steps", fuse)
            ht, hp, hc = lib.tri_factor(*lt), lib.penta_factor(*lp), lib.penta_factor(*lc)
            n0 = lib.btps_launch_count()
            dt_, dp_, dc_ = dev(rhs), dev(rhs), dev(c0)
            lib.tri_solve_steps(ht, dt_, steps)
            lib.penta_solve_steps(hp, dp_, steps)
            lib.ch_step_batched(hc, dc_, 0.05, steps)
            outs[fuse] = (dt_.cpu().numpy(), dp_.cpu().numpy(), dc_.cpu().numpy(), lib.btps_launch_count() - n0)
        finally:
            lib.btps_tune("fuse_steps", -1)
    # 11 steps: 11 launches unfused, 1 by default, 2 (8 + 3) with fuse_steps = 8, 4 with fuse_steps = 3; a variant
    # without a fused form (CH at n = 1000: no room for the halo exchange rows) falls back to one launch per step
    assert outs[1][3] == 3 * steps and 3 <= outs[-1][3] <= outs[8][3] <= outs[3][3] < 3 * steps
    if n <= 512:
        assert outs[-1][3] == 3 and outs[8][3] == 3 * 2 and outs[3][3] == 3 * 4
    for k in (-1, 3, 8):
        for a, b_ in zip(outs[1][:3], outs[k][:3]):
            assert np.array_equal(a, b_)
    ref = rhs.copy()
    oracle.tri_solve_interleaved(oracle.tri_factor(*lt), ref, nsteps=steps)
    assert rel_err(outs[-1][0], ref) <= TOL_STEPS
    ref = rhs.copy()
    oracle.penta_solve_interleaved(oracle.penta_factor(*lp), ref, nsteps=steps)
    assert rel_err(outs[-1][1], ref) <= TOL_STEPS
    ref = c0.copy()
    oracle.ch_step_interleaved(oracle.penta_factor(*lc), ref, 0.05, nsteps=steps)
    assert rel_err(outs[-1][2], ref) <= TOL_STEPS


@pytest.mark.parametrize("n,batch", [(512, 148 * 16 * 3 + 48), (256, 9000), (384, 4100)])
def test_long_fused_loops_on_half_width_tiles(lib, n, batch):
    """Launches of 4 or more fused steps of the plain tridiagonal loop, of the Cahn-Hilliard step and of the Crank-Nicolson
    steps run on half-width
    tiles (8 lanes, two or four tile groups per CTA) when the partitions share their coefficient blocks
    (btps_tune narrow_loops = 0 keeps the full-width tiles).  Same arithmetic per system: bitwise equal results, several
    tiles per group, a ragged last tile; and both match the oracle's loop.  40 steps: one launch; 70 steps: 64 + 6, both
    on half-width tiles; 3 steps: full-width tiles either way."""
    lt, lc, lp = inputs.tri_lhs(n, 0.5), inputs.ch_lhs(n), inputs.penta_lhs(n, 0.5)
    x5 = np.array([-0.5, 2.0, -2.0, 2.0, -0.5])
    _, al = inputs.ch_params(n)
    rhs = inputs.uniform_rhs(n, batch, seed=91)
    c0 = 0.1 * rhs
    for steps in (40, 70, 3):
        outs = {}
        for narrow in (-1, 0):
            try:
                lib.btps_tune("narrow_loops", narrow)
                ht, hc, hcp = lib.tri_factor(*lt), lib.penta_factor(*lc), lib.penta_factor_periodic(*lc)
                a, b_, c = dev(rhs), dev(c0), dev(c0)
                lib.tri_solve_steps(ht, a, steps)
                lib.ch_step_batched(hc, b_, al, steps)
                lib.ch_step_batched(hcp, c, al, steps)
                # the same loop with the coarsening statistic of eq. 30 recorded inside the kernel
                e, lb = dev(c0), torch.zeros(steps, dtype=torch.float64, device="cuda")
                lib.ch_step_batched_stat(hcp, e, al, steps, lb)
                # Crank-Nicolson diffusion / hyperdiffusion steps (eq. 9-11, 17-19), truncated and periodic
                cn = []
                for per in (False, True):
                    f, g = dev(rhs), dev(rhs)
                    lib.tri_cn_step_batched((lib.tri_factor_periodic if per else lib.tri_factor)(*lt), f, 0.5, 0.0, 0.5, steps)
                    lib.penta_cn_step_batched((lib.penta_factor_periodic if per else lib.penta_factor)(*lp), g, x5, steps)
                    cn += [f.cpu().numpy(), g.cpu().numpy()]
                outs[narrow] = [x.cpu().numpy() for x in (a, b_, c, e, lb)] + cn
            finally:
                lib.btps_tune("narrow_loops", -1)
        for x, y in zip(outs[-1][:4] + outs[-1][5:], outs[0][:4] + outs[0][5:]):
            assert np.array_equal(x, y)
        if steps == 40:
            for per in (False, True):
                ref = rhs.copy()
                oracle.tri_cn_step_interleaved((oracle.tri_periodic_factor if per else oracle.tri_factor)(*lt), ref, 0.5, 0.0, 0.5, nsteps=steps)
                assert rel_err(outs[-1][5 + 2 * per], ref) <= TOL_STEPS
                ref = rhs.copy()
                oracle.penta_cn_step_interleaved((oracle.penta_periodic_factor if per else oracle.penta_factor)(*lp), ref, x5, nsteps=steps)
                assert rel_err(outs[-1][6 + 2 * per], ref) <= TOL_STEPS
        assert np.array_equal(outs[-1][2], outs[-1][3])
        assert rel_err(outs[-1][4], outs[0][4]) <= 1e-12  # (the order of the sum over the runs is not fixed)
        if steps == 40:
            want = oracle.ch_steps_with_lbar(oracle.penta_periodic_factor(*lc), c0.copy(), al, steps, periodic=True)
            assert rel_err(outs[-1][4], np.asarray(want)) <= TOL_STEPS
        if steps == 40:
            ref = rhs.copy()
            oracle.tri_solve_interleaved(oracle.tri_factor(*lt), ref, nsteps=steps)
            assert rel_err(outs[-1][0], ref) <= TOL_STEPS
            ref = c0.copy()
            oracle.ch_step_interleaved(oracle.penta_factor(*lc), ref, al, nsteps=steps)
            assert rel_err(outs[-1][1], ref) <= TOL_STEPS
            ref = c0.copy()
            oracle.ch_periodic_step_interleaved(oracle.penta_periodic_factor(*lc), ref, al, nsteps=steps)
            assert rel_err(outs[-1][2], ref) <= TOL_STEPS


# ---- periodic tridiagonal (Sherman-Morrison) ---------------------------------------

def rand_cyclic(n, seed):
    rng = np.random.default_rng(seed)
    a, c = rng.uniform(-1, 1, n), rng.uniform(-1, 1, n)
    b = np.abs(a) + np.abs(c) + rng.uniform(0.5, 1.5, n)
    return a, b, c


@pytest.mark.parametrize("n", [3, 4, 31, 32, 33, 64, 300, 512, 1000, 1024, 1500, 5000])
def test_tri_periodic_sizes(lib, n):
    lhs = rand_cyclic(n, n)
    fo = oracle.tri_periodic_factor(*lhs)
    h = lib.tri_factor_periodic(*lhs)
    for batch in (1, 33, 1024 + 32, 1001):
        rhs = inputs.uniform_rhs(n, batch, seed=n + batch)
        ref = rhs.copy()
        oracle.tri_periodic_solve_interleaved(fo, ref)
        d = dev(rhs)
        lib.tri_solve_batched(h, d)
        assert rel_err(d.cpu().numpy(), ref) <= TOL_SINGLE, (n, batch, h.plan())
    rhs = inputs.uniform_rhs(n, 512, seed=3).astype(np.float32)
    ref = rhs.astype(np.float64)
    oracle.tri_periodic_solve_interleaved(fo, ref)
    d = dev(rhs)
    lib.tri_solve_batched_f32(h, d)
    assert rel_err(d.cpu().numpy(), ref) <= TOL_F32, (n, h.plan(4))


@pytest.mark.parametrize("tune", [dict(), dict(prefetch=0), dict(warp_scan=0), dict(vec=1), dict(force_two_pass=1),
                                  dict(fuse_steps=1)])
def test_tri_periodic_diffusion_steps_and_mass(lib, tune):
    """Periodic implicit diffusion (the paper's own benchmark form, PAPER.md:120-136 in BASELINE.json's
    backward-Euler reading): 20 steps against the oracle, conservation of each system's sum
    (PAPER.md:339-348 holds for periodic BCs) and the exact decay of a cosine mode."""
    n, batch, r, steps = 256, 2048 + 64, 0.5, 20
    lhs = ([-r] * n, [1 + 2 * r] * n, [-r] * n)
    try:
        for k, v in tune.items():
            lib.btps_tune(k, v)
        h = lib.tri_factor_periodic(*lhs)
    finally:
        for k in tune:
            lib.btps_tune(k, -1)
    rhs = inputs.uniform_rhs(n, batch, seed=17)
    rhs[:, 0] = np.cos(2 * np.pi * 3 * np.arange(n) / n)
    ref = rhs.copy()
    oracle.tri_periodic_solve_interleaved(oracle.tri_periodic_factor(*lhs), ref, nsteps=steps)
    d = dev(rhs)
    try:
        for k, v in tune.items():
            lib.btps_tune(k, v)
        lib.tri_solve_steps(h, d, steps)
    finally:
        for k in tune:
            lib.btps_tune(k, -1)
    got = d.cpu().numpy()
    assert rel_err(got, ref) <= TOL_STEPS, (tune, h.plan())
    assert np.max(np.abs(got.sum(axis=0) - rhs.sum(axis=0))) <= 1e-11
    lam = 1 + 4 * r * np.sin(np.pi * 3 / n) ** 2
    assert np.max(np.abs(got[:, 0] - rhs[:, 0] * lam ** -steps)) <= 1e-12


def test_tri_periodic_errors(lib):
    with pytest.raises(lib.BtpsError):
        lib.tri_factor_periodic([1.0, 1.0], [2.0, 2.0], [1.0, 1.0])          # n < 3
    with pytest.raises(lib.BtpsError):
        lib.tri_factor_periodic([1.0] * 4, [0.0, 2.0, 2.0, 2.0], [1.0] * 4)  # b_0 = 0


# ---- periodic pentadiagonal (Woodbury, C-31) and periodic Cahn-Hilliard --------------------

def rand_cyclic_penta(n, seed):
    rng = np.random.default_rng(seed)
    e, a, c, f = (rng.uniform(-1, 1, n) for _ in range(4))
    d = np.abs(e) + np.abs(a) + np.abs(c) + np.abs(f) + rng.uniform(0.5, 1.5, n)
    return e, a, d, c, f


@pytest.mark.parametrize("n", [5, 6, 31, 32, 33, 64, 300, 512, 1000, 1024, 1500, 5000])
def test_penta_periodic_sizes(lib, n):
    lhs = rand_cyclic_penta(n, n)
    fo = oracle.penta_periodic_factor(*lhs)   # paper naming (a,b,c,d,e) = API (e,a,d,c,f)
    h = lib.penta_factor_periodic(*lhs)
    for batch in (1, 33, 1024 + 32, 1001):
        rhs = inputs.uniform_rhs(n, batch, seed=n + batch)
        ref = rhs.copy()
        oracle.penta_periodic_solve_interleaved(fo, ref)
        d = dev(rhs)
        lib.penta_solve_batched(h, d)
        assert rel_err(d.cpu().numpy(), ref) <= TOL_SINGLE, (n, batch, h.plan())
    rhs = inputs.uniform_rhs(n, 512, seed=3).astype(np.float32)
    ref = rhs.astype(np.float64)
    oracle.penta_periodic_solve_interleaved(fo, ref)
    d = dev(rhs)
    lib.penta_solve_batched_f32(h, d)
    assert rel_err(d.cpu().numpy(), ref) <= TOL_F32, (n, h.plan(4))


@pytest.mark.parametrize("tune", [dict(), dict(prefetch=0), dict(warp_scan=0), dict(vec=1), dict(force_two_pass=1),
                                  dict(fuse_steps=1)])
@pytest.mark.parametrize("n", [256, 200])  # 200: not a multiple of the rows per thread -> two-pass form
def test_periodic_cahn_hilliard_steps_and_mass(lib, tune, n):
    """The paper's own Cahn-Hilliard setting (periodic): 40 steps against the oracle,
    exact conservation of every run's mass (eq. 21-22), and the periodic penta time loop."""
    batch, steps = 2048 + 64, 40
    sigma, alpha = inputs.ch_params(256)
    st = ([sigma] * n, [-4 * sigma] * n, [1 + 6 * sigma] * n, [-4 * sigma] * n, [sigma] * n)
    try:
        for k, v in tune.items():
            lib.btps_tune(k, v)
        h = lib.penta_factor_periodic(*st)
        c0 = 0.1 * inputs.uniform_rhs(n, batch, seed=23)
        d, d2 = dev(c0), dev(c0)
        lib.ch_step_batched(h, d, alpha, steps)
        lib.penta_solve_steps(h, d2, 11)
    finally:
        for k in tune:
            lib.btps_tune(k, -1)
    fo = oracle.penta_periodic_factor(*st)
    ref = c0.copy()
    oracle.ch_periodic_step_interleaved(fo, ref, alpha, nsteps=steps)
    got = d.cpu().numpy()
    assert rel_err(got, ref) <= TOL_STEPS, (tune, n, h.ch_plan())
    assert np.max(np.abs(got.sum(axis=0) - c0.sum(axis=0))) <= 1e-13
    ref = c0.copy()
    oracle.penta_periodic_solve_interleaved(fo, ref, nsteps=11)
    assert rel_err(d2.cpu().numpy(), ref) <= TOL_STEPS, (tune, n, h.plan())


def test_penta_periodic_errors(lib):
    with pytest.raises(lib.BtpsError):
        lib.penta_factor_periodic(*([[1.0] * 4] * 5))  # n < 5


# ---- coarsening statistic (eq. 30) ---------------------------------------------------

@pytest.mark.parametrize("periodic,n,batch,tune", [
    (True, 256, 4096 + 32, {}), (True, 256, 1001, {}), (True, 200, 2048, {}), (False, 256, 4096, {}),
    (True, 64, 8192, {}), (True, 256, 2048, dict(force_two_pass=1)), (True, 32, 640, {}),
])
def test_coarsening_statistic(lib, periodic, n, batch, tune):
    steps = 13
    sigma, alpha = inputs.ch_params(256)
    st = ([sigma] * n, [-4 * sigma] * n, [1 + 6 * sigma] * n, [-4 * sigma] * n, [sigma] * n)
    c0 = 0.3 * inputs.uniform_rhs(n, batch, seed=29)
    try:
        for k, v in tune.items():
            lib.btps_tune(k, v)
        h = lib.penta_factor_periodic(*st) if periodic else lib.penta_factor(*st)
        d = dev(c0)
        lbar = torch.full((steps,), -1.0, dtype=torch.float64, device="cuda")
        lib.ch_step_batched_stat(h, d, alpha, steps, lbar)
        d_plain = dev(c0)
        lib.ch_step_batched(h, d_plain, alpha, steps)
    finally:
        for k in tune:
            lib.btps_tune(k, -1)
    fo = oracle.penta_periodic_factor(*st) if periodic else oracle.penta_factor(*st)
    ref = c0.copy()
    ref_l = oracle.ch_steps_with_lbar(fo, ref, alpha, steps, periodic=periodic)
    assert torch.equal(d, d_plain)                      # recording the statistic does not change the state
    assert rel_err(d.cpu().numpy(), ref) <= TOL_STEPS
    got_l = lbar.cpu().numpy()
    assert np.max(np.abs(got_l - ref_l) / ref_l) <= TOL_STEPS, (got_l, ref_l)
    assert np.all(got_l > 1.0)


# ---- fused Crank-Nicolson diffusion step (eq. 9-11) -----------------------------------

@pytest.mark.parametrize("periodic", [True, False])
@pytest.mark.parametrize("n,batch", [(64, 4096 + 64), (256, 2048), (200, 1001), (512, 1024), (1024, 512), (20, 333), (1500, 256)])
def test_tri_cn_step(lib, periodic, n, batch):
    """The paper's diffusion benchmark scheme: explicit three-point half fused with the (periodic) solve;
    11 steps against the oracle, sum conservation and the von Neumann factor in the periodic case."""
    s, steps = 0.7, 11
    lhs = ([-s] * n, [1 + 2 * s] * n, [-s] * n)
    u0 = inputs.uniform_rhs(n, batch, seed=41)
    u0[:, 0] = np.cos(2 * np.pi * 2 * np.arange(n) / n)
    h = (lib.tri_factor_periodic if periodic else lib.tri_factor)(*lhs)
    fo = (oracle.tri_periodic_factor if periodic else oracle.tri_factor)(*lhs)
    ref = u0.copy()
    oracle.tri_cn_step_interleaved(fo, ref, s, 1 - 2 * s, s, nsteps=steps)
    outs = []
    for fuse in (-1, 1):
        try:
            lib.btps_tune("fuse_steps", fuse)
            d = dev(u0)
            lib.tri_cn_step_batched(h, d, s, 1 - 2 * s, s, steps)
        finally:
            lib.btps_tune("fuse_steps", -1)
        outs.append(d.cpu().numpy())
    assert np.array_equal(outs[0], outs[1])
    assert rel_err(outs[0], ref) <= TOL_STEPS, (n, batch, h.cn_plan())
    if periodic:
        assert np.max(np.abs(outs[0].sum(axis=0) - u0.sum(axis=0))) <= 1e-11
        q = 4 * s * np.sin(np.pi * 2 / n) ** 2
        assert np.max(np.abs(outs[0][:, 0] - u0[:, 0] * ((1 - q) / (1 + q)) ** steps)) <= 1e-12


# ---- run-to-run determinism (a shared-memory race or a missing barrier would show up as a bitwise difference) --

@pytest.mark.parametrize("n,batch", [(512, 8192), (1024, 4096), (64, 32768), (300, 5000)])
def test_repeated_launches_are_bitwise_identical(lib, n, batch):
    s = 0.5
    sg, al = inputs.ch_params(256)
    st = ([sg] * n, [-4 * sg] * n, [1 + 6 * sg] * n, [-4 * sg] * n, [sg] * n)
    tl = ([-s] * n, [1 + 2 * s] * n, [-s] * n)
    u = torch.from_numpy(inputs.uniform_rhs(n, batch, seed=77)).cuda()
    cases = []
    for h in (lib.tri_factor(*tl), lib.tri_factor_periodic(*tl)):
        cases += [lambda x, h=h: lib.tri_solve_batched(h, x), lambda x, h=h: lib.tri_solve_steps(h, x, 9),
                  lambda x, h=h: lib.tri_cn_step_batched(h, x, s, 1 - 2 * s, s, 9)]
    for h in (lib.penta_factor(*st), lib.penta_factor_periodic(*st)):
        cases += [lambda x, h=h: lib.penta_solve_batched(h, x), lambda x, h=h: lib.penta_solve_steps(h, x, 9),
                  lambda x, h=h: lib.ch_step_batched(h, x, al, 9)]
    for i, fn in enumerate(cases):
        first = None
        for rep in range(12):
            x = (0.1 * u).clone()
            fn(x)
            if first is None:
                first = x
            else:
                assert torch.equal(x, first), (i, rep, n, batch)


# ---- fused Crank-Nicolson hyperdiffusion step (eq. 17-19) -----------------------------

@pytest.mark.parametrize("periodic", [True, False])
@pytest.mark.parametrize("n,batch", [(64, 4096 + 64), (256, 2048), (200, 1001), (512, 1024), (1024, 512), (20, 333), (1500, 256)])
def test_penta_cn_step(lib, periodic, n, batch):
    s, steps = 0.3, 11
    st = ([s] * n, [-4 * s] * n, [1 + 6 * s] * n, [-4 * s] * n, [s] * n)
    x5 = [-s, 4 * s, 1 - 6 * s, 4 * s, -s]
    u0 = inputs.uniform_rhs(n, batch, seed=43)
    u0[:, 0] = np.cos(2 * np.pi * 2 * np.arange(n) / n)
    h = (lib.penta_factor_periodic if periodic else lib.penta_factor)(*st)
    fo = (oracle.penta_periodic_factor if periodic else oracle.penta_factor)(*st)
    ref = u0.copy()
    oracle.penta_cn_step_interleaved(fo, ref, x5, nsteps=steps)
    outs = []
    for fuse in (-1, 1):
        try:
            lib.btps_tune("fuse_steps", fuse)
            d = dev(u0)
            lib.penta_cn_step_batched(h, d, x5, steps)
        finally:
            lib.btps_tune("fuse_steps", -1)
        outs.append(d.cpu().numpy())
    assert np.array_equal(outs[0], outs[1])
    assert rel_err(outs[0], ref) <= TOL_STEPS, (n, batch, h.cn_plan())
    if periodic:
        assert np.max(np.abs(outs[0].sum(axis=0) - u0.sum(axis=0))) <= 1e-11
        q = 16 * s * np.sin(np.pi * 2 / n) ** 4
        assert np.max(np.abs(outs[0][:, 0] - u0[:, 0] * ((1 - q) / (1 + q)) ** steps)) <= 1e-12


# ---- cluster-chain kernels (rows of a tile over 2 / 4 / 8 CTAs, carries through distributed shared memory) ----

@pytest.mark.parametrize("n", [1024, 1000, 600, 544, 1500, 2048, 2500, 4096, 3000])
@pytest.mark.parametrize("batch", [4096 + 32, 64, 2048 * 9])
def test_cluster_chain_against_oracle(lib, n, batch):
    """More than 16 partitions: plain solves can run on a thread-block cluster whose CTAs each keep a block of the rows
    (two CTAs up to N = 1024, four up to 2048, eight up to 4096); carries cross the CTAs as a chain through distributed
    shared memory.  btps_tune cluster = 1 forces the chain for every eligible plan (0 forbids it).  Single solves, fused
    steps and fp32 against the oracle, and against the library's other plan for the same system."""
    if n * batch > 40_000_000:
        batch = 2048 * 3
    lt, lp = rand_tri(n, n), rand_penta(n, n + 1)
    rhs = inputs.uniform_rhs(n, batch, seed=51)
    outs = {}
    for cl in (1, 0):
        try:
            lib.btps_tune("cluster", cl)
            ht, hp = lib.tri_factor(*lt), lib.penta_factor(*lp)
            tags = (lib.btps_kernel_tag(ht, 8, batch), lib.btps_kernel_tag(hp, 8, batch), lib.btps_kernel_tag(hp, 4, batch))
            # ninth template argument: cluster split ("two_pass_kernel" has none)
            assert all(len(t.split(", ")) > 8 and t.split(", ")[8] == "1" for t in tags) == (cl == 1), tags
            a, b_, c, d = dev(rhs), dev(rhs), dev(rhs), dev(rhs)
            lib.tri_solve_batched(ht, a)
            lib.penta_solve_batched(hp, b_)
            lib.tri_solve_steps(ht, c, 11)
            lib.penta_solve_steps(hp, d, 11)
            f32 = dev(rhs.astype(np.float32))
            lib.penta_solve_batched_f32(hp, f32)
            g32 = dev(rhs.astype(np.float32))
            lib.tri_solve_batched_f32(ht, g32)
            outs[cl] = [x.cpu().numpy() for x in (a, b_, c, d, f32, g32)]
        finally:
            lib.btps_tune("cluster", -1)
    r32 = rhs.astype(np.float32).astype(np.float64)
    for cl in (1, 0):
        ref = rhs.copy()
        oracle.tri_solve_interleaved(oracle.tri_factor(*lt), ref)
        assert rel_err(outs[cl][0], ref) <= TOL_SINGLE, cl
        ref = rhs.copy()
        oracle.penta_solve_interleaved(oracle.penta_factor(*lp), ref)
        assert rel_err(outs[cl][1], ref) <= TOL_SINGLE, cl
        ref = rhs.copy()
        oracle.tri_solve_interleaved(oracle.tri_factor(*lt), ref, nsteps=11)
        assert rel_err(outs[cl][2], ref) <= TOL_STEPS, cl
        ref = rhs.copy()
        oracle.penta_solve_interleaved(oracle.penta_factor(*lp), ref, nsteps=11)
        assert rel_err(outs[cl][3], ref) <= TOL_STEPS, cl
        ref = r32.copy()
        oracle.penta_solve_interleaved(oracle.penta_factor(*lp), ref)
        assert rel_err(outs[cl][4].astype(np.float64), ref) <= TOL_F32, cl
        ref = r32.copy()
        oracle.tri_solve_interleaved(oracle.tri_factor(*lt), ref)
        assert rel_err(outs[cl][5].astype(np.float64), ref) <= TOL_F32, cl


@pytest.mark.parametrize("n", [1024, 2048, 4096])
def test_cluster_chain_repeats_bitwise_and_many_tiles(lib, n):
    """The chain hands carries from CTA to CTA through mbarrier-signalled inboxes that are reused tile after tile and
    step after step: many tiles per cluster (grid capped) with fused steps, run 6 times, must give the same bits and
    match the oracle."""
    batch = 32 * 37
    lt, lp = inputs.tri_lhs(n, 0.5), inputs.penta_lhs(n, 0.5)
    rhs = inputs.uniform_rhs(n, batch, seed=52)
    rt, rp = rhs.copy(), rhs.copy()
    oracle.tri_solve_interleaved(oracle.tri_factor(*lt), rt, nsteps=5)
    oracle.penta_solve_interleaved(oracle.penta_factor(*lp), rp, nsteps=5)
    try:
        lib.btps_tune("cluster", 1)
        lib.btps_tune("grid", 16)
        ht, hp = lib.tri_factor(*lt), lib.penta_factor(*lp)
        first = None
        for rep in range(6):
            a, b_ = dev(rhs), dev(rhs)
            lib.tri_solve_steps(ht, a, 5)
            lib.penta_solve_steps(hp, b_, 5)
            got = (a.cpu().numpy(), b_.cpu().numpy())
            if first is None:
                first = got
                assert rel_err(got[0], rt) <= TOL_STEPS and rel_err(got[1], rp) <= TOL_STEPS
            else:
                assert np.array_equal(first[0], got[0]) and np.array_equal(first[1], got[1])
    finally:
        lib.btps_tune("cluster", -1)
        lib.btps_tune("grid", -1)


# ---- CUDA graph capture of a time-step loop ------------------------------------------------------------

def test_time_loop_in_a_cuda_graph(lib):
    """The calls only enqueue kernels on the caller's stream (no allocation, no host sync), so a whole
    time-stepping loop can be captured once and replayed (launch-bound small problems)."""
    n, batch, steps = 64, 1024, 24
    sg, al = inputs.ch_params(256)
    st = ([sg] * n, [-4 * sg] * n, [1 + 6 * sg] * n, [-4 * sg] * n, [sg] * n)
    ht = lib.tri_factor(*inputs.tri_lhs(n, 0.5))
    hp = lib.penta_factor_periodic(*st)
    u0 = torch.from_numpy(inputs.uniform_rhs(n, batch, seed=61)).cuda()
    c0 = 0.1 * u0
    # eager reference (also warms up: first launches resolve occupancy outside the capture)
    ue, ce = u0.clone(), c0.clone()
    lib.tri_solve_steps(ht, ue, steps)
    lib.ch_step_batched(hp, ce, al, steps)
    ug, cg = u0.clone(), c0.clone()
    g = torch.cuda.CUDAGraph()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        with torch.cuda.graph(g, stream=s):
            lib.tri_solve_steps(ht, ug, steps, stream=s.cuda_stream)
            lib.ch_step_batched(hp, cg, al, steps, stream=s.cuda_stream)
    torch.cuda.current_stream().wait_stream(s)
    ug.copy_(u0)
    cg.copy_(c0)
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(ug, ue) and torch.equal(cg, ce)
    g.replay()   # second replay advances the state by another `steps`
    torch.cuda.synchronize()
    lib.tri_solve_steps(ht, ue, steps)
    assert torch.equal(ug, ue)


# ---- cyclic correction folded into the carry scan vs applied row by row ---------------------------------

@pytest.mark.parametrize("n", [64, 256, 512, 1024])
def test_cyclic_correction_in_scan_matches_rowwise(lib, n):
    """Periodic penta handles with whole partitions fold x = y - Z H V^T y into the carries (KIND_*F kernels);
    btps_tune('cyclic_in_scan', 0) applies it row by row.  Both must match the oracle; general (non-Toeplitz) LHS."""
    batch = 2048 + 32
    lhs = rand_cyclic_penta(n, n + 3)
    sg, al = inputs.ch_params(256)
    st = ([sg] * n, [-4 * sg] * n, [1 + 6 * sg] * n, [-4 * sg] * n, [sg] * n)
    x5 = [-0.3, 1.2, 1 - 1.8, 1.2, -0.3]
    rhs = inputs.uniform_rhs(n, batch, seed=71)
    fo, fs = oracle.penta_periodic_factor(*lhs), oracle.penta_periodic_factor(*st)
    r1 = rhs.copy(); oracle.penta_periodic_solve_interleaved(fo, r1)
    r2 = 0.1 * rhs; oracle.ch_periodic_step_interleaved(fs, r2, al, nsteps=9)
    r3 = rhs.copy(); oracle.penta_cn_step_interleaved(fs, r3, x5, nsteps=9)
    for mode in (-1, 0):
        try:
            lib.btps_tune("cyclic_in_scan", mode)
            h, hs = lib.penta_factor_periodic(*lhs), lib.penta_factor_periodic(*st)
        finally:
            lib.btps_tune("cyclic_in_scan", -1)
        d1, d2, d3, d4 = dev(rhs), dev(0.1 * rhs), dev(rhs), dev(rhs.astype(np.float32))
        lib.penta_solve_batched(h, d1)
        lib.ch_step_batched(hs, d2, al, 9)
        lib.penta_cn_step_batched(hs, d3, x5, 9)
        lib.penta_solve_batched_f32(h, d4)
        assert rel_err(d1.cpu().numpy(), r1) <= TOL_SINGLE, (mode, n)
        assert rel_err(d2.cpu().numpy(), r2) <= TOL_STEPS, (mode, n)
        assert rel_err(d3.cpu().numpy(), r3) <= TOL_STEPS, (mode, n)
        assert rel_err(d4.cpu().numpy().astype(np.float64), r1) <= TOL_F32, (mode, n)
        assert np.max(np.abs(d2.cpu().numpy().sum(axis=0) - (0.1 * rhs).sum(axis=0))) <= 1e-13


@pytest.mark.parametrize("n", [64, 256, 512, 1024])
def test_sherman_morrison_in_scan_matches_rowwise(lib, n):
    """Periodic tri handles with whole partitions fold x = y - (v.y)/(1+v.z) z into the carries (KIND_TRIPF / TRICNPF)."""
    batch = 2048 + 32
    lhs = rand_cyclic(n, n + 5)
    s = 0.7
    tl = ([-s] * n, [1 + 2 * s] * n, [-s] * n)
    rhs = inputs.uniform_rhs(n, batch, seed=73)
    fo, fs = oracle.tri_periodic_factor(*lhs), oracle.tri_periodic_factor(*tl)
    r1 = rhs.copy(); oracle.tri_periodic_solve_interleaved(fo, r1)
    r2 = rhs.copy(); oracle.tri_cn_step_interleaved(fs, r2, s, 1 - 2 * s, s, nsteps=9)
    r3 = rhs.copy(); oracle.tri_periodic_solve_interleaved(fo, r3, nsteps=9)
    for mode in (-1, 0):
        try:
            lib.btps_tune("cyclic_in_scan", mode)
            h, hs = lib.tri_factor_periodic(*lhs), lib.tri_factor_periodic(*tl)
        finally:
            lib.btps_tune("cyclic_in_scan", -1)
        d1, d2, d3, d4 = dev(rhs), dev(rhs), dev(rhs), dev(rhs.astype(np.float32))
        lib.tri_solve_batched(h, d1)
        lib.tri_cn_step_batched(hs, d2, s, 1 - 2 * s, s, 9)
        lib.tri_solve_steps(h, d3, 9)
        lib.tri_solve_batched_f32(h, d4)
        assert rel_err(d1.cpu().numpy(), r1) <= TOL_SINGLE, (mode, n)
        assert rel_err(d2.cpu().numpy(), r2) <= TOL_STEPS, (mode, n)
        assert rel_err(d3.cpu().numpy(), r3) <= TOL_STEPS, (mode, n)
        assert rel_err(d4.cpu().numpy().astype(np.float64), r1) <= TOL_F32, (mode, n)
        assert np.max(np.abs(d2.cpu().numpy().sum(axis=0) - rhs.sum(axis=0))) <= 1e-11


# ---- one-step calls through either instantiation of a kernel ---------------------------------------------

@pytest.mark.parametrize("n", [64, 512])
def test_one_step_through_fused_instantiation_is_bitwise_equal(lib, n):
    """btps_tune('one_step_fused', 0/1) picks the single-step or the multi-step instantiation for a one-step call
    (default: the one with the smaller local-memory frame); the arithmetic is the same, so the results are too."""
    batch = 4096 + 64
    rhs = inputs.uniform_rhs(n, batch, seed=81)
    _, al = inputs.ch_params(n)
    ht, hp, hc = lib.tri_factor(*rand_tri(n, n + 1)), lib.penta_factor(*rand_penta(n, n + 2)), lib.penta_factor(*inputs.ch_lhs(n))
    hpp, htp = lib.penta_factor_periodic(*rand_cyclic_penta(n, n + 3)), lib.tri_factor_periodic(*rand_cyclic(n, n + 5))
    got = {}
    for mode in (0, 1):
        try:
            lib.btps_tune("one_step_fused", mode)
            d = [dev(rhs), dev(rhs), dev(0.1 * rhs), dev(rhs), dev(rhs)]
            lib.tri_solve_batched(ht, d[0])
            lib.penta_solve_batched(hp, d[1])
            lib.ch_step_batched(hc, d[2], al, 1)
            lib.penta_solve_batched(hpp, d[3])
            lib.tri_solve_batched(htp, d[4])
            torch.cuda.synchronize()
        finally:
            lib.btps_tune("one_step_fused", -1)
        got[mode] = d
    for a, c in zip(got[0], got[1]):
        assert torch.equal(a, c)


@pytest.mark.parametrize("n", [5, 9, 17, 37, 131])
def test_two_pass_kernel_ragged_row_blocks(lib, n):
    """The two-pass form streams rows in blocks of 8 (16 in fp32): sizes around the block edges, general LHS,
    plain and periodic, fp64 and fp32, a batch that is not a multiple of the thread block."""
    batch = 300
    lt, lp, ltp, lpp = rand_tri(n, n), rand_penta(n, n + 1), rand_cyclic(n, n + 2), rand_cyclic_penta(n, n + 3)
    try:
        lib.btps_tune("force_two_pass", 1)
        ht, hp = lib.tri_factor(*lt), lib.penta_factor(*lp)
        htp, hpp = lib.tri_factor_periodic(*ltp), lib.penta_factor_periodic(*lpp)
    finally:
        lib.btps_tune("force_two_pass", -1)
    assert ht.plan()["rows_per_thread"] == 0 and hpp.plan()["rows_per_thread"] == 0
    rhs = inputs.uniform_rhs(n, batch, seed=90 + n)
    cases = ((ht, oracle.tri_factor(*lt), lib.tri_solve_batched, lib.tri_solve_batched_f32, oracle.tri_solve_interleaved),
             (hp, oracle.penta_factor(*lp), lib.penta_solve_batched, lib.penta_solve_batched_f32, oracle.penta_solve_interleaved),
             (htp, oracle.tri_periodic_factor(*ltp), lib.tri_solve_batched, lib.tri_solve_batched_f32,
              oracle.tri_periodic_solve_interleaved),
             (hpp, oracle.penta_periodic_factor(*lpp), lib.penta_solve_batched, lib.penta_solve_batched_f32,
              oracle.penta_periodic_solve_interleaved))
    for h, fac, solve, solve32, osolve in cases:
        r32 = rhs.astype(np.float32)
        ref = rhs.copy(); osolve(fac, ref)
        ref32 = r32.astype(np.float64); osolve(fac, ref32)
        d, d32 = dev(rhs), dev(r32)
        solve(h, d); solve32(h, d32)
        assert rel_err(d.cpu().numpy(), ref) <= TOL_SINGLE, n
        assert rel_err(d32.cpu().numpy().astype(np.float64), ref32) <= TOL_F32, n


def test_held_stores_are_bitwise_equal(lib):
    """btps_tune('hold_stores', 1) makes a tile's stores wait for the next tile's prefetch (a scheduling change only):
    same results as with 0, on a batch of many tiles per CTA, for every kernel family."""
    n, batch = 512, 32 * 148 * 3 + 64
    rhs = inputs.uniform_rhs(n, batch, seed=97)
    _, al = inputs.ch_params(n)
    ht, hp, hc = lib.tri_factor(*rand_tri(n, 3)), lib.penta_factor(*rand_penta(n, 4)), lib.penta_factor(*inputs.ch_lhs(n))
    htp = lib.tri_factor_periodic(*rand_cyclic(n, 5))
    got = {}
    for mode in (0, 1):
        try:
            lib.btps_tune("hold_stores", mode)
            d = [dev(rhs), dev(rhs), dev(0.1 * rhs), dev(rhs), dev(rhs.astype(np.float32)), dev(rhs)]
            lib.tri_solve_batched(ht, d[0])
            lib.penta_solve_batched(hp, d[1])
            lib.ch_step_batched(hc, d[2], al, 3)
            lib.tri_solve_batched(htp, d[3])
            lib.tri_solve_batched_f32(ht, d[4])
            lib.tri_cn_step_batched(ht, d[5], 0.3, 0.4, 0.3, 2)
            torch.cuda.synchronize()
        finally:
            lib.btps_tune("hold_stores", -1)
        got[mode] = d
    for a, c in zip(got[0], got[1]):
        assert torch.equal(a, c)
    ref = rhs.copy()
    oracle.tri_solve_interleaved(oracle.tri_factor(*rand_tri(n, 3)), ref)
    assert rel_err(got[1][0].cpu().numpy(), ref) <= TOL_SINGLE


@pytest.mark.parametrize("n", [64, 500, 512, 768, 1024, 2048, 3000])
def test_shared_coefficient_blocks_are_bitwise_equal(lib, n):
    """btps_tune('dedupe', 1): partitions whose coefficient blocks are bitwise equal read one shared block (constant-
    coefficient LHS: all interior partitions).  A storage change only: same bits as with every partition's own block,
    for every kernel family, on single-CTA and cluster plans; and a general LHS (no equal blocks) is left alone."""
    batch = 1024 + 32
    rhs = inputs.uniform_rhs(n, batch, seed=101)
    _, al = inputs.ch_params(n)
    x5 = np.array([0.02, -0.08, 0.88, -0.08, 0.02])
    got, info = {}, {}
    for mode in (0, 1):
        try:
            lib.btps_tune("dedupe", mode)
            ht, hp, hc = lib.tri_factor(*inputs.tri_lhs(n, 0.5)), lib.penta_factor(*inputs.penta_lhs(n, 0.5)), lib.penta_factor(*inputs.ch_lhs(n))
            htp = lib.tri_factor_periodic(*inputs.tri_lhs(n, 0.5))
            hpp, hcp = lib.penta_factor_periodic(*inputs.penta_lhs(n, 0.5)), lib.penta_factor_periodic(*inputs.ch_lhs(n))
            hg = lib.penta_factor(*rand_penta(n, 4))
            d = [dev(rhs), dev(rhs), dev(0.1 * rhs), dev(rhs), dev(rhs), dev(0.1 * rhs), dev(rhs.astype(np.float32)),
                 dev(rhs.astype(np.float32)), dev(rhs), dev(rhs), dev(rhs), dev(rhs)]
            lib.tri_solve_batched(ht, d[0])
            lib.penta_solve_batched(hp, d[1])
            lib.ch_step_batched(hc, d[2], al, 3)
            lib.tri_solve_batched(htp, d[3])
            lib.penta_solve_batched(hpp, d[4])
            lib.ch_step_batched(hcp, d[5], al, 3)
            lib.tri_solve_batched_f32(ht, d[6])
            lib.penta_solve_batched_f32(hp, d[7])
            lib.tri_cn_step_batched(ht, d[8], 0.3, 0.4, 0.3, 2)
            lib.penta_cn_step_batched(hpp, d[9], x5, 2)
            lib.penta_solve_steps(hp, d[10], 5)
            lib.penta_solve_batched(hg, d[11])
            torch.cuda.synchronize()
            info[mode] = (lib.btps_plan_info(hp, 8), lib.btps_plan_info(hg, 8))
        finally:
            lib.btps_tune("dedupe", -1)
        got[mode] = d
    for k, (a, c) in enumerate(zip(got[0], got[1])):
        assert torch.equal(a, c), k
    ref = rhs.copy()
    oracle.penta_solve_interleaved(oracle.penta_factor(*inputs.penta_lhs(n, 0.5)), ref)
    assert rel_err(got[1][1].cpu().numpy(), ref) <= TOL_SINGLE
    if info[0][0]["rows_per_thread"] and info[0][0]["partitions"] >= 4:   # on-chip plan, four or more partitions: the image shrank
        assert info[1][0]["table_bytes"] < info[0][0]["table_bytes"]
    assert info[1][1]["table_bytes"] == info[0][1]["table_bytes"]         # random LHS: no two blocks are equal


def two_regime_lhs(n, seed, penta):
    """Strongly dominant LHS whose coefficients repeat with a period of 32 rows (the rows of one partition), with one
    random pattern on the first half of the rows and another on the second half.  The factor recurrences contract by
    more than 10 per row, so they reach their 32-periodic limit bitwise within a partition or two: the partitions of each
    half then have equal coefficient blocks -- partial sharing, neither the constant-coefficient case nor the general one."""
    rng = np.random.default_rng(seed)
    pats = rng.uniform(-1, 1, (2, 4, 32))
    half = (n // 64) * 32
    def rows(k):
        return np.concatenate([np.resize(pats[0, k], half), np.resize(pats[1, k], n - half)])
    e, a, c, f = (rows(k) for k in range(4))
    d = 12.0 + np.concatenate([np.zeros(half), np.ones(n - half)])
    if penta:
        return e, a, d, c, f
    return a, d, c


@pytest.mark.parametrize("n", [512, 1024, 2048])
def test_partially_shared_coefficient_blocks_against_oracle(lib, n):
    batch = 512 + 32
    rhs = inputs.uniform_rhs(n, batch, seed=103)
    lt, lp = two_regime_lhs(n, 1, False), two_regime_lhs(n, 2, True)
    ht, hp = lib.tri_factor(*lt), lib.penta_factor(*lp)
    full = lib.btps_plan_info(lib.penta_factor(*rand_penta(n, 4)), 8)["table_bytes"]
    const = lib.btps_plan_info(lib.penta_factor(*inputs.penta_lhs(n, 0.5)), 8)["table_bytes"]
    part = lib.btps_plan_info(hp, 8)["table_bytes"]
    assert const < part < full, (const, part, full)   # some blocks shared, more distinct ones than a constant LHS has
    for h, lhs, solve, steps, fac, osolve in ((ht, lt, lib.tri_solve_batched, lib.tri_solve_steps, oracle.tri_factor, oracle.tri_solve_interleaved),
                                              (hp, lp, lib.penta_solve_batched, lib.penta_solve_steps, oracle.penta_factor, oracle.penta_solve_interleaved)):
        d = dev(rhs)
        solve(h, d)
        ref = rhs.copy()
        osolve(fac(*lhs), ref)
        assert rel_err(d.cpu().numpy(), ref) <= TOL_SINGLE
        d = dev(rhs)
        steps(h, d, 3)
        ref = rhs.copy()
        osolve(fac(*lhs), ref, nsteps=3)
        assert rel_err(d.cpu().numpy(), ref) <= TOL_STEPS
        d32 = dev(rhs.astype(np.float32))
        (lib.tri_solve_batched_f32 if h is ht else lib.penta_solve_batched_f32)(h, d32)
        ref = rhs.astype(np.float32).astype(np.float64)
        osolve(fac(*lhs), ref)
        assert rel_err(d32.cpu().numpy().astype(np.float64), ref) <= TOL_F32


def test_default_cluster_policy_by_row_pitch(lib):
    """Which kernel a call launches by default (btps_kernel_tag, nothing is launched): the cluster pair where a row of the
    batch is long enough for 256-byte segments to pay, one CTA per tile below that, clusters
    always above 1024 rows."""
    def cl(h, elem, batch):
        return lib.btps_kernel_tag(h, elem, batch).split(", ")[8] == "1"
    ht, hp = lib.tri_factor(*inputs.tri_lhs(1024, 0.5)), lib.penta_factor(*inputs.penta_lhs(1024, 0.5))
    assert not cl(ht, 8, 1 << 13) and cl(ht, 8, 1 << 16) and cl(ht, 8, 1 << 22)       # tri, 32 partitions: from 512 KiB rows
    assert not cl(ht, 4, 1 << 16) and cl(ht, 4, 1 << 17)
    assert not cl(hp, 8, 1 << 19) and cl(hp, 8, 1 << 20) and cl(hp, 4, 1 << 21)       # penta, 32 partitions: from 8 MiB rows
    h768, h640 = lib.tri_factor(*inputs.tri_lhs(768, 0.5)), lib.tri_factor(*inputs.tri_lhs(640, 0.5))
    assert not cl(h768, 8, 1 << 18) and cl(h768, 8, 1 << 19)                          # 24 partitions: from 4 MiB rows
    assert not cl(h640, 8, 1 << 21) and cl(h640, 8, 1 << 22)                          # 20 partitions: from 32 MiB rows
    assert not cl(lib.penta_factor(*inputs.penta_lhs(768, 0.5)), 8, 1 << 22)
    assert not cl(lib.tri_factor(*inputs.tri_lhs(512, 0.5)), 8, 1 << 22)              # 16 partitions: never
    for n in (1100, 2048, 4096):
        assert cl(lib.tri_factor(*inputs.tri_lhs(n, 0.5)), 8, 1 << 10) and cl(lib.penta_factor(*inputs.penta_lhs(n, 0.5)), 4, 1 << 10)
    assert not cl(ht, 8, (1 << 16) + 1)                                               # unaligned pitch: no TMA, no cluster
    # time loops (calls of 3 or more steps) keep up to 32 partitions on one CTA; above 1024 rows there is only the cluster plan
    def cl_steps(h, batch, nsteps):
        return lib.btps_kernel_tag(h, 8, batch, nsteps).split(", ")[8] == "1"
    assert cl_steps(ht, 1 << 22, 2) and not cl_steps(ht, 1 << 22, 3) and not cl_steps(ht, 1 << 16, 100)
    assert cl_steps(hp, 1 << 20, 2) and not cl_steps(hp, 1 << 20, 64)
    assert cl_steps(lib.tri_factor(*inputs.tri_lhs(2048, 0.5)), 1 << 12, 100)


def test_time_loops_of_long_rows_stay_on_one_cta(lib):
    """N = 1024 at 2^16 systems: a single solve runs on the cluster pair (256-byte row segments), a time loop on one CTA per
    tile (faster per step once the tile stays on chip).  The choice is made per call: every launch of one loop runs the same
    kernel, so fused and per-step launches stay bitwise equal, and the loop matches the oracle's."""
    n, batch, steps = 1024, 1 << 16, 5
    lt = inputs.tri_lhs(n, 0.5)
    rhs = inputs.uniform_rhs(n, batch, seed=77)
    h = lib.tri_factor(*lt)
    assert lib.btps_kernel_tag(h, 8, batch, 1).split(", ")[8] == "1"
    assert lib.btps_kernel_tag(h, 8, batch, steps).split(", ")[8] == "0"
    outs = []
    for fuse in (-1, 1):
        try:
            lib.btps_tune("fuse_steps", fuse)
            d = dev(rhs)
            lib.tri_solve_steps(h, d, steps)
            outs.append(d.cpu().numpy())
            del d
        finally:
            lib.btps_tune("fuse_steps", -1)
    assert np.array_equal(outs[0], outs[1])
    ref = rhs.copy()
    oracle.tri_solve_interleaved(oracle.tri_factor(*lt), ref, nsteps=steps)
    assert rel_err(outs[0], ref) <= TOL_STEPS


def test_cluster_pair_held_stores_bitwise_equal_and_against_oracle(lib):
    """The tridiagonal pair at 32 partitions holds its stores by default once a cluster has 8 tiles to walk: same bits as
    with free-running stores, equal to the oracle, over enough tiles for the default to be on (148 / 2 clusters x 8 x 32)."""
    n, batch = 1024, 32 * 74 * 9 + 64
    lhs = inputs.tri_lhs(n, 0.5)
    rhs = inputs.uniform_rhs(n, batch, seed=107)
    got = {}
    for mode in (-1, 0, 1):
        try:
            lib.btps_tune("hold_stores", mode)
            lib.btps_tune("cluster", 1)       # (the default takes the pair from 512 KiB rows; this batch has 167 KiB ones)
            h = lib.tri_factor(*lhs)
            assert lib.btps_kernel_tag(h, 8, batch).split(", ")[8] == "1"
            d, d32 = dev(rhs), dev(rhs.astype(np.float32))
            lib.tri_solve_batched(h, d)
            lib.tri_solve_steps(h, d, 3)
            lib.tri_solve_batched_f32(h, d32)
            torch.cuda.synchronize()
        finally:
            lib.btps_tune("hold_stores", -1)
            lib.btps_tune("cluster", -1)
        got[mode] = (d, d32)
    for mode in (0, 1):
        assert torch.equal(got[-1][0], got[mode][0]) and torch.equal(got[-1][1], got[mode][1])
    ids = np.unique(np.concatenate([np.arange(0, 128), np.arange(batch - 128, batch), np.arange(128, batch - 128, 97)]))
    ref = rhs[:, ids].copy()
    oracle.tri_solve_interleaved(oracle.tri_factor(*lhs), ref, nsteps=4)
    assert rel_err(got[-1][0].cpu().numpy()[:, ids], ref) <= TOL_STEPS


@pytest.mark.parametrize("n,batch", [(1056, 2344), (1835, 2276), (2048, 1027), (4000, 515)])
def test_explicit_halves_on_plans_padded_to_whole_cluster_ctas(lib, n, batch):
    """Above 1024 rows the partition count is padded to whole cluster CTAs (N = 1056: 33 -> 36 partitions).  The kinds with
    an explicit half have no cluster form there and walk the carries serially with direct loads; their halo loads must not
    reach for row r0 - 1 of a partition that lies wholly beyond row N (an out-of-bounds read that faulted at these sizes:
    found by a randomised sweep of sizes against the oracle, fixed in sweep.cuh)."""
    rhs = inputs.uniform_rhs(n, batch, seed=109)
    _, al = inputs.ch_params(n)
    x5 = np.array([-0.5, 2.0, -2.0, 2.0, -0.5])
    lt, lp, lc = inputs.tri_lhs(n, 0.5), inputs.penta_lhs(n, 0.5), inputs.ch_lhs(n)
    d = dev(0.1 * rhs)
    lib.ch_step_batched(lib.penta_factor(*lc), d, al, 2)
    ref = 0.1 * rhs
    oracle.ch_step_interleaved(oracle.penta_factor(*lc), ref, al, nsteps=2)
    assert rel_err(d.cpu().numpy(), ref) <= TOL_STEPS
    d = dev(rhs)
    lib.tri_cn_step_batched(lib.tri_factor(*lt), d, 0.5, 0.0, 0.5, 2)
    ref = rhs.copy()
    oracle.tri_cn_step_interleaved(oracle.tri_factor(*lt), ref, 0.5, 0.0, 0.5, nsteps=2)
    assert rel_err(d.cpu().numpy(), ref) <= TOL_STEPS
    d = dev(rhs)
    lib.penta_cn_step_batched(lib.penta_factor(*lp), d, x5, 2)
    ref = rhs.copy()
    oracle.penta_cn_step_interleaved(oracle.penta_factor(*lp), ref, x5, nsteps=2)
    assert rel_err(d.cpu().numpy(), ref) <= TOL_STEPS


@pytest.mark.parametrize("n", [64, 58, 40])
def test_one_warp_groups_reuse_their_ring_on_an_l2_resident_batch(lib, n):
    """N <= 64 runs eight one-warp tile groups per CTA, each with its own one-tile TMA ring.  On few CTAs every group walks
    many tiles, and on a batch that stays in L2 the next tile can arrive within a microsecond of being asked for -- while
    this tile's shared-memory loads (generic proxy) are still queued behind the other groups'.  The kernels order those
    reads before the TMA write with fence.proxy.async; without it this test failed in nearly every repetition (wrong
    tiles now and then, found by a randomised sweep against the oracle)."""
    batch, steps = 13632, 40
    lhs = inputs.tri_lhs(n, 0.5)
    rhs = inputs.uniform_rhs(n, batch, seed=383)
    ref = rhs.copy()
    oracle.tri_solve_interleaved(oracle.tri_factor(*lhs), ref, nsteps=steps)
    try:
        lib.btps_tune("grid", 3)
        lib.btps_tune("fuse_steps", 1)      # one launch per step: 40 launches over the same 7 MB
        h = lib.tri_factor(*lhs)
        assert lib.btps_plan_info(h, 8)["tma_prefetch"] == 1 and lib.btps_plan_info(h, 8)["tiles_per_cta"] >= 4
        for rep in range(4):
            d = dev(rhs)
            lib.tri_solve_steps(h, d, steps)
            assert rel_err(d.cpu().numpy(), ref) <= TOL_STEPS, rep
    finally:
        lib.btps_tune("grid", -1)
        lib.btps_tune("fuse_steps", -1)
