"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (default tune keys): the
time loops of configs 2 / 3 / 5 with their fused multi-step launches on a batch that gives every persistent CTA many
tiles (ring phase flips, next-tile prefetch, held stores, reverse order all active), and the 2^22-system cells whose
element offsets exceed 32 bits.  SURVEY 8(d): "Parity for configs 1-3 is on the full batch"; PAPER.md:172 (time loops),
PAPER.md:431-445 (2^20 runs).  Tolerances are BASELINE.json's.
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


def sample_ids(batch, want=4096):
    """>= `want` systems: the first and last 256 (first / last tiles and the tail), a stride through the rest."""
    ids = np.concatenate([np.arange(0, 256), np.arange(batch - 256, batch),
                          np.arange(257, batch - 256, max(1, (batch - 512) // (want - 512)))])
    return np.unique(ids).astype(np.int64)


# ---- configs 2 and 3: the FULL batch of 65536 systems, 100 steps, every element against the oracle --------------------

def test_config2_full_batch_100_steps(lib):
    n, batch, steps = 512, 65536, 100
    lhs = inputs.tri_lhs(n, 0.5)
    u0, k, A = inputs.sine_modes_u0(n, batch, seed=0)
    h = lib.tri_factor(*lhs)
    d = torch.from_numpy(u0).cuda()
    n0 = lib.btps_launch_count()
    lib.tri_solve_steps(h, d, steps)
    assert lib.btps_launch_count() - n0 == 2  # 64 + 36 fused steps: the launch configuration bench.py times
    got = d.cpu().numpy()
    ref = u0  # advanced in place by the oracle, all 65536 systems
    oracle.tri_solve_interleaved(oracle.tri_factor(*lhs), ref, nsteps=steps)
    assert rel_err(got, ref) <= TOL_STEPS
    # exact modal decay (closed form, independent of both implementations): u^100 = sum_m A_m lam_m^-100 sin(k_m pi x)
    x = np.arange(1, n + 1) / (n + 1)
    lam = 1.0 + 4 * 0.5 * np.sin(k * np.pi / (2 * (n + 1))) ** 2
    exact = np.zeros_like(got)
    for m in range(4):
        exact += (A[m] * lam[m] ** -steps)[None, :] * np.sin(np.pi * k[m][None, :] * x[:, None])
    assert rel_err(got, exact) <= TOL_STEPS


def test_config3_full_batch_100_steps(lib):
    n, batch, steps = 512, 65536, 100
    lhs = inputs.penta_lhs(n, 0.5)
    rhs = inputs.uniform_rhs(n, batch, seed=0)
    h = lib.penta_factor(*lhs)
    d = torch.from_numpy(rhs).cuda()
    n0 = lib.btps_launch_count()
    lib.penta_solve_steps(h, d, steps)
    assert lib.btps_launch_count() - n0 == 2
    got = d.cpu().numpy()
    oracle.penta_solve_interleaved(oracle.penta_factor(*lhs), rhs, nsteps=steps)
    assert rel_err(got, rhs) <= TOL_STEPS
    # SPD with spectrum in [1, 9]: the 2-norm of every system has not grown (SURVEY 8(c) config 3 invariant)
    assert np.all(np.linalg.norm(got, axis=0) <= np.sqrt(n) + 1e-9)


def test_configs_2_3_one_launch_per_step_full_batch(lib):
    """The same full-batch loops with one launch per step (btps_tune fuse_steps = 1): 100 back-to-back single-step
    launches with ~14 tiles per CTA, held stores on by default -- compared with the oracle on sampled systems."""
    n, batch, steps = 512, 65536, 100
    ids = sample_ids(batch, 2048)
    gi = torch.from_numpy(ids).cuda()
    try:
        lib.btps_tune("fuse_steps", 1)
        for kind in ("tri", "penta"):
            lhs = inputs.tri_lhs(n, 0.5) if kind == "tri" else inputs.penta_lhs(n, 0.5)
            d = torch.empty(n, batch, dtype=torch.float64, device="cuda")
            inputs.fill_uniform_device(d, n, seed=11)
            ref = inputs.uniform_rhs(n, len(ids), seed=11, systems=ids.astype(np.uint64))
            n0 = lib.btps_launch_count()
            if kind == "tri":
                lib.tri_solve_steps(lib.tri_factor(*lhs), d, steps)
                oracle.tri_solve_interleaved(oracle.tri_factor(*lhs), ref, nsteps=steps)
            else:
                lib.penta_solve_steps(lib.penta_factor(*lhs), d, steps)
                oracle.penta_solve_interleaved(oracle.penta_factor(*lhs), ref, nsteps=steps)
            assert lib.btps_launch_count() - n0 == steps
            assert rel_err(d[:, gi].cpu().numpy(), ref) <= TOL_STEPS, kind
    finally:
        lib.btps_tune("fuse_steps", -1)


# ---- the same path in seconds: few CTAs, so each walks many tiles with fused steps -------------------------------------

@pytest.mark.parametrize("grid", [8, 3])
@pytest.mark.parametrize("hold", [-1, 1])
def test_many_tiles_per_cta_with_fused_steps(lib, grid, hold):
    n, batch, steps = 512, 6144 + 32, 70   # 193 tiles of 32 systems on `grid` CTAs; 64 + 6 fused steps
    lt, lp, lc = inputs.tri_lhs(n, 0.5), inputs.penta_lhs(n, 0.5), inputs.ch_lhs(n)
    _, alpha = inputs.ch_params(n)
    rhs = inputs.uniform_rhs(n, batch, seed=41)
    c0 = 0.1 * rhs
    try:
        lib.btps_tune("grid", grid)
        lib.btps_tune("hold_stores", hold)
        for rev in (0, 1):
            lib.btps_tune("reverse", rev)
            dt_, dp_, dc_ = (torch.from_numpy(x).cuda() for x in (rhs, rhs, c0))
            lib.tri_solve_steps(lib.tri_factor(*lt), dt_, steps)
            lib.penta_solve_steps(lib.penta_factor(*lp), dp_, steps)
            lib.ch_step_batched(lib.penta_factor(*lc), dc_, alpha, steps)
            ref = rhs.copy()
            oracle.tri_solve_interleaved(oracle.tri_factor(*lt), ref, nsteps=steps)
            assert rel_err(dt_.cpu().numpy(), ref) <= TOL_STEPS
            ref = rhs.copy()
            oracle.penta_solve_interleaved(oracle.penta_factor(*lp), ref, nsteps=steps)
            assert rel_err(dp_.cpu().numpy(), ref) <= TOL_STEPS
            ref = c0.copy()
            oracle.ch_step_interleaved(oracle.penta_factor(*lc), ref, alpha, nsteps=steps)
            assert rel_err(dc_.cpu().numpy(), ref) <= TOL_STEPS
    finally:
        for key in ("grid", "hold_stores", "reverse"):
            lib.btps_tune(key, -1)


@pytest.mark.parametrize("grid", [8, 5])
def test_many_tiles_per_cta_single_solves(lib, grid):
    """Single-step launches, several tiles per CTA, held stores forced on and off, every default kernel family
    (fp64 / fp32, N = 64 / 512 / 1024 and a ragged N) against the oracle."""
    try:
        lib.btps_tune("grid", grid)
        for hold in (0, 1):
            lib.btps_tune("hold_stores", hold)
            for n, batch in ((512, 4096 + 64), (1024, 2048 + 16), (64, 16384 + 256), (777, 3000)):
                lt, lp = inputs.tri_lhs(n, 0.5), inputs.penta_lhs(n, 0.5)
                rhs = inputs.uniform_rhs(n, batch, seed=43)
                rt, rp = rhs.copy(), rhs.copy()
                oracle.tri_solve_interleaved(oracle.tri_factor(*lt), rt)
                oracle.penta_solve_interleaved(oracle.penta_factor(*lp), rp)
                ht, hp = lib.tri_factor(*lt), lib.penta_factor(*lp)
                d = torch.from_numpy(rhs).cuda()
                lib.tri_solve_batched(ht, d)
                assert rel_err(d.cpu().numpy(), rt) <= TOL_SINGLE, (n, hold)
                d = torch.from_numpy(rhs).cuda()
                lib.penta_solve_batched(hp, d)
                assert rel_err(d.cpu().numpy(), rp) <= TOL_SINGLE, (n, hold)
                r32 = rhs.astype(np.float32)
                rt, rp = r32.astype(np.float64), r32.astype(np.float64)
                oracle.tri_solve_interleaved(oracle.tri_factor(*lt), rt)
                oracle.penta_solve_interleaved(oracle.penta_factor(*lp), rp)
                d = torch.from_numpy(r32).cuda()
                lib.tri_solve_batched_f32(ht, d)
                assert rel_err(d.cpu().numpy().astype(np.float64), rt) <= TOL_F32, (n, hold)
                d = torch.from_numpy(r32).cuda()
                lib.penta_solve_batched_f32(hp, d)
                assert rel_err(d.cpu().numpy().astype(np.float64), rp) <= TOL_F32, (n, hold)
    finally:
        lib.btps_tune("grid", -1)
        lib.btps_tune("hold_stores", -1)


# ---- config 5: 2^20 independent runs, all 1000 steps --------------------------------------------------

def test_config5_full_2p20_runs_1000_steps(lib):
    n, batch, steps = 256, 1 << 20, 1000
    _, alpha = inputs.ch_params(n)
    lhs = inputs.ch_lhs(n)
    d = torch.empty(n, batch, dtype=torch.float64, device="cuda")
    inputs.fill_uniform_device(d, n, seed=0, scale=0.1)
    ids = sample_ids(batch)
    gi = torch.from_numpy(ids).cuda()
    ref = inputs.uniform_rhs(n, len(ids), seed=0, scale=0.1, systems=ids.astype(np.uint64))
    assert np.array_equal(d[:, gi].cpu().numpy(), ref)
    h = lib.penta_factor(*lhs)
    n0 = lib.btps_launch_count()
    lib.ch_step_batched(h, d, alpha, steps)
    assert lib.btps_launch_count() - n0 == 16  # 15 x 64 + 40 fused steps
    oracle.ch_step_interleaved(oracle.penta_factor(*lhs), ref, alpha, nsteps=steps)
    assert rel_err(d[:, gi].cpu().numpy(), ref) <= TOL_STEPS
    # properties that hold for every run at any size: finite, and inside the physical range of the order parameter
    # (c = +-1 are the two phases; after 1000 steps of dt = 5e-5 the largest |c| over the 2^20 runs
    # is ~0.2: spinodal growth has only begun)
    assert bool(torch.isfinite(d).all())
    assert float(d.abs().max()) < 1.0


# ---- N = 1024 at 2^22 systems: 2^32 elements (32 GiB fp64), the default cluster-pair launch for tri fp64 ---------------

@pytest.mark.parametrize("kind,f32", [("tri", False), ("penta", False), ("tri", True), ("penta", True)])
def test_n1024_batch_2p22_sampled(lib, kind, f32):
    n, batch = 1024, 1 << 22
    free, _ = torch.cuda.mem_get_info()
    if free < (n * batch * (4 if f32 else 8)) * 1.3:
        pytest.skip("not enough free device memory for the 2^22 x 1024 cell")
    dtype = torch.float32 if f32 else torch.float64
    d = torch.empty(n, batch, dtype=dtype, device="cuda")
    inputs.fill_uniform_device(d, n, seed=9)
    ids = sample_ids(batch)
    gi = torch.from_numpy(ids).cuda()
    ref = inputs.uniform_rhs(n, len(ids), seed=9, systems=ids.astype(np.uint64))
    if f32:
        ref = ref.astype(np.float32).astype(np.float64)
    assert np.array_equal(d[:, gi].cpu().numpy().astype(np.float64), ref)
    if kind == "tri":
        lhs = inputs.tri_lhs(n, 0.5)
        h = lib.tri_factor(*lhs)
        (lib.tri_solve_batched_f32 if f32 else lib.tri_solve_batched)(h, d)
        oracle.tri_solve_interleaved(oracle.tri_factor(*lhs), ref)
    else:
        lhs = inputs.penta_lhs(n, 0.5)
        h = lib.penta_factor(*lhs)
        (lib.penta_solve_batched_f32 if f32 else lib.penta_solve_batched)(h, d)
        oracle.penta_solve_interleaved(oracle.penta_factor(*lhs), ref)
    got = d[:, gi].cpu().numpy().astype(np.float64)
    assert rel_err(got, ref) <= (TOL_F32 if f32 else TOL_SINGLE), (kind, f32, lib.btps_kernel_tag(h, 4 if f32 else 8, batch))
    # every element, not only the sampled systems: finite and bounded by max|rhs| * ||A^-1||_inf (tri: an M-matrix with
    # row sums >= 1, so ||A^-1||_inf <= 1; the penta LHS is I + r*D4 with D4 positive semi-definite
    # -- bounded by 1 in the 2-norm and, computed densely for N = 1024, by 1.118 in the max-norm)
    assert bool(torch.isfinite(d).all())
    assert float(d.abs().max()) <= 1.2
    del d
    torch.cuda.empty_cache()


# ---- fp32 at full size: more config-4 cells (the oracle runs in fp64 on the same fp32-representable inputs) ------------

@pytest.mark.parametrize("kind,n,lb", [("tri", 64, 22), ("penta", 64, 22), ("tri", 256, 19), ("penta", 1024, 19),
                                       ("tri", 1024, 16), ("penta", 256, 16), ("tri", 64, 16), ("penta", 64, 16)])
def test_fp32_cells_sampled(lib, kind, n, lb):
    batch = 1 << lb
    d = torch.empty(n, batch, dtype=torch.float32, device="cuda")
    inputs.fill_uniform_device(d, n, seed=21)
    ids = sample_ids(batch, 2048)
    gi = torch.from_numpy(ids).cuda()
    ref = inputs.uniform_rhs(n, len(ids), seed=21, systems=ids.astype(np.uint64)).astype(np.float32).astype(np.float64)
    if kind == "tri":
        lhs = inputs.tri_lhs(n, 0.5)
        lib.tri_solve_batched_f32(lib.tri_factor(*lhs), d)
        oracle.tri_solve_interleaved(oracle.tri_factor(*lhs), ref)
    else:
        lhs = inputs.penta_lhs(n, 0.5)
        lib.penta_solve_batched_f32(lib.penta_factor(*lhs), d)
        oracle.penta_solve_interleaved(oracle.penta_factor(*lhs), ref)
    assert rel_err(d[:, gi].cpu().numpy().astype(np.float64), ref) <= TOL_F32
    assert bool(torch.isfinite(d).all())


# ---- two live handles of different n used in turn (the shared-memory attribute belongs to the kernel function) ---------

@pytest.mark.parametrize("f32", [False, True])
def test_alternating_handles_of_different_n(lib, f32):
    batch = 2048
    sizes = (1024, 512, 1024, 64, 1000, 512)
    dt = np.float32 if f32 else np.float64
    tol = TOL_F32 if f32 else TOL_SINGLE
    hs = {}
    for n in set(sizes):
        hs[n] = (lib.tri_factor(*inputs.tri_lhs(n, 0.5)), lib.penta_factor(*inputs.penta_lhs(n, 0.5)))
    for rnd, n in enumerate(sizes):
        rhs = inputs.uniform_rhs(n, batch, seed=50 + rnd).astype(dt)
        rt, rp = rhs.astype(np.float64), rhs.astype(np.float64)
        oracle.tri_solve_interleaved(oracle.tri_factor(*inputs.tri_lhs(n, 0.5)), rt)
        oracle.penta_solve_interleaved(oracle.penta_factor(*inputs.penta_lhs(n, 0.5)), rp)
        d = torch.from_numpy(rhs).cuda()
        (lib.tri_solve_batched_f32 if f32 else lib.tri_solve_batched)(hs[n][0], d)
        assert rel_err(d.cpu().numpy().astype(np.float64), rt) <= tol, (rnd, n)
        d = torch.from_numpy(rhs).cuda()
        (lib.penta_solve_batched_f32 if f32 else lib.penta_solve_batched)(hs[n][1], d)
        assert rel_err(d.cpu().numpy().astype(np.float64), rp) <= tol, (rnd, n)
        if not f32:
            # the fused multi-step instantiation and the CH step of the same handles
            rt = rhs.copy()
            oracle.tri_solve_interleaved(oracle.tri_factor(*inputs.tri_lhs(n, 0.5)), rt, nsteps=3)
            d = torch.from_numpy(rhs).cuda()
            lib.tri_solve_steps(hs[n][0], d, 3)
            assert rel_err(d.cpu().numpy(), rt) <= TOL_STEPS, (rnd, n)
            rc = 0.1 * rhs
            dc = torch.from_numpy(rc).cuda()
            oracle.ch_step_interleaved(oracle.penta_factor(*inputs.penta_lhs(n, 0.5)), rc, 0.05, nsteps=2)
            lib.ch_step_batched(hs[n][1], dc, 0.05, 2)
            assert rel_err(dc.cpu().numpy(), rc) <= TOL_STEPS, (rnd, n)
    # and the cluster-pair slot of the long handle after a short one has launched
    try:
        lib.btps_tune("cluster", 1)
        if not f32:
            n = 1024
            rhs = inputs.uniform_rhs(n, batch, seed=77)
            rt = rhs.copy()
            oracle.tri_solve_interleaved(oracle.tri_factor(*inputs.tri_lhs(n, 0.5)), rt)
            h = lib.tri_factor(*inputs.tri_lhs(n, 0.5))
            d = torch.from_numpy(rhs).cuda()
            lib.tri_solve_batched(h, d)
            d2 = torch.from_numpy(inputs.uniform_rhs(512, batch, seed=78)).cuda()
            lib.tri_solve_batched(hs[512][0], d2)
            d = torch.from_numpy(rhs).cuda()
            lib.tri_solve_batched(h, d)
            assert rel_err(d.cpu().numpy(), rt) <= TOL_SINGLE
    finally:
        lib.btps_tune("cluster", -1)


# ---- LHS that are valid for the paper's algorithm but not diagonally dominant ------------------------------------------

def spd_not_dominant_tri(n, seed, hi, nhi, lo, nlo):
    """Symmetric positive-definite tridiagonal matrix A = L L^T of a unit-diagonal bidiagonal L whose sub-diagonal
    alternates stretches of `nhi` entries near `hi` and `nlo` entries near `lo`: the LU pivots exist (they are 1), the
    elimination multipliers a_i / b^_i equal the sub-diagonal of L -- above 1 on the `hi` stretches -- and most rows are
    not diagonally dominant, yet the matrix stays well conditioned (cond 70 ... 1e4, checked in the test).  Rows are
    then scaled by random signs (mixed-sign diagonals; the solution is unchanged)."""
    rng = np.random.default_rng(seed)
    l = np.resize(np.concatenate([np.full(nhi, hi), np.full(nlo, lo)]), n) * rng.uniform(0.95, 1.05, n)
    b = 1.0 + np.concatenate([[0.0], l[1:] ** 2])
    a = np.concatenate([[0.0], l[1:]])
    c = np.concatenate([a[1:], [0.0]])
    sign = rng.choice([-1.0, 1.0], n)
    return a * sign, b * sign, c * sign


@pytest.mark.parametrize("n", [64, 512, 1024])
@pytest.mark.parametrize("pattern", [(0.9, 1, 0.9, 1), (1.25, 8, 0.4, 8), (1.0, 4, 0.5, 4), (1.5, 3, 0.3, 5), (1.1, 20, 0.5, 12)])
def test_tri_not_diagonally_dominant(lib, n, pattern):
    """The CUDA path evaluates the paper's LU solve partition-wise (carries = products of up to 32 multipliers); for
    LHS whose multipliers exceed 1 on stretches those products grow (here up to ~9x per partition).  Both sides are
    the same LU without pivoting in a different order of operations, so they agree to rounding times the conditioning
    of the matrix: tolerance = max(BASELINE tolerance, 16 eps cond(A))."""
    a, b, c = spd_not_dominant_tri(n, n, *pattern)
    A = np.diag(b) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)
    cond = np.linalg.cond(A)
    assert cond < 2e4 and np.mean(np.abs(b) >= np.abs(a) + np.abs(c)) < 0.95
    batch = 1500
    rhs = inputs.uniform_rhs(n, batch, seed=61)
    ref = rhs.copy()
    oracle.tri_solve_interleaved(oracle.tri_factor(a, b, c), ref)
    h = lib.tri_factor(a, b, c)
    d = torch.from_numpy(rhs).cuda()
    lib.tri_solve_batched(h, d)
    assert rel_err(d.cpu().numpy(), ref) <= max(TOL_SINGLE, 16 * 2.2e-16 * cond), (n, pattern, cond)
    r32 = rhs.astype(np.float32)
    ref = r32.astype(np.float64)
    oracle.tri_solve_interleaved(oracle.tri_factor(a, b, c), ref)
    d = torch.from_numpy(r32).cuda()
    lib.tri_solve_batched_f32(h, d)
    assert rel_err(d.cpu().numpy().astype(np.float64), ref) <= max(TOL_F32, 16 * 1.2e-7 * cond), (n, pattern, cond)


@pytest.mark.parametrize("n", [64, 512, 1024])
def test_penta_not_diagonally_dominant(lib, n):
    """I + r*T^2 with r = 50: diagonal 301 against an off-diagonal row sum of 500; SPD, cond ~ 800."""
    r = 50.0
    e, a, d_, c, f = inputs.penta_lhs(n, r)
    batch = 1500
    rhs = inputs.uniform_rhs(n, batch, seed=62)
    ref = rhs.copy()
    oracle.penta_solve_interleaved(oracle.penta_factor(e, a, d_, c, f), ref)
    h = lib.penta_factor(e, a, d_, c, f)
    d = torch.from_numpy(rhs).cuda()
    lib.penta_solve_batched(h, d)
    cond = 1.0 + 16.0 * r
    assert rel_err(d.cpu().numpy(), ref) <= max(TOL_SINGLE, 16 * 2.2e-16 * cond)
    r32 = rhs.astype(np.float32)
    ref = r32.astype(np.float64)
    oracle.penta_solve_interleaved(oracle.penta_factor(e, a, d_, c, f), ref)
    d = torch.from_numpy(r32).cuda()
    lib.penta_solve_batched_f32(h, d)
    assert rel_err(d.cpu().numpy().astype(np.float64), ref) <= max(TOL_F32, 16 * 1.2e-7 * cond)


# ---- fp32 storage, fp64 arithmetic ------------------------------------------------------------------------

TOL_F32S = 1.0e-7   # rounding of the stored result to float: 2^-24 = 6e-8 relative per entry (+ fp64 arithmetic)


@pytest.mark.parametrize("n", [1, 2, 5, 31, 32, 33, 64, 100, 256, 512, 777, 1000, 1024])
def test_f32_storage_f64_arithmetic(lib, n):
    """*_f32s: the batch lives in HBM as floats, the sweeps run in fp64.  Oracle = the fp64 oracle on the same
    (float-representable) inputs, rounded to float as the store does; tolerance = the output rounding.  The all-fp32
    path on the same inputs is checked to be the less accurate one (that is the point of the variant)."""
    lt, lp = inputs.tri_lhs(n, 0.5), inputs.penta_lhs(n, 0.5)
    ht, hp = lib.tri_factor(*lt), lib.penta_factor(*lp)
    for batch in (1, 333, 2048 + 64):
        r32 = inputs.uniform_rhs(n, batch, seed=70 + n).astype(np.float32)
        for kind in ("tri", "penta"):
            ref = r32.astype(np.float64)
            if kind == "tri":
                oracle.tri_solve_interleaved(oracle.tri_factor(*lt), ref)
            else:
                oracle.penta_solve_interleaved(oracle.penta_factor(*lp), ref)
            ref32 = ref.astype(np.float32).astype(np.float64)
            d = torch.from_numpy(r32).cuda()
            (lib.tri_solve_batched_f32s(ht, d) if kind == "tri" else lib.penta_solve_batched_f32s(hp, d))
            got = d.cpu().numpy().astype(np.float64)
            # at most one float ulp from the correctly rounded fp64 solution, entry by entry
            ulp = np.spacing(np.abs(ref32).astype(np.float32)).astype(np.float64)
            assert np.all(np.abs(got - ref32) <= ulp + 1e-300), (n, batch, kind)
            assert rel_err(got, ref) <= TOL_F32S, (n, batch, kind)
            if n >= 64 and batch > 1000:
                d2 = torch.from_numpy(r32).cuda()
                (lib.tri_solve_batched_f32(ht, d2) if kind == "tri" else lib.penta_solve_batched_f32(hp, d2))
                assert rel_err(got, ref) < rel_err(d2.cpu().numpy().astype(np.float64), ref), (n, kind)


@pytest.mark.parametrize("kind,n,lb", [("tri", 512, 16), ("penta", 512, 16), ("tri", 1024, 19), ("penta", 64, 20)])
def test_f32_storage_full_size_sampled(lib, kind, n, lb):
    batch = 1 << lb
    d = torch.empty(n, batch, dtype=torch.float32, device="cuda")
    inputs.fill_uniform_device(d, n, seed=23)
    ids = sample_ids(batch, 2048)
    gi = torch.from_numpy(ids).cuda()
    ref = inputs.uniform_rhs(n, len(ids), seed=23, systems=ids.astype(np.uint64)).astype(np.float32).astype(np.float64)
    if kind == "tri":
        lhs = inputs.tri_lhs(n, 0.5)
        h = lib.tri_factor(*lhs)
        lib.tri_solve_batched_f32s(h, d)
        oracle.tri_solve_interleaved(oracle.tri_factor(*lhs), ref)
    else:
        lhs = inputs.penta_lhs(n, 0.5)
        h = lib.penta_factor(*lhs)
        lib.penta_solve_batched_f32s(h, d)
        oracle.penta_solve_interleaved(oracle.penta_factor(*lhs), ref)
    assert lib.btps_kernel_tag(h, 12, batch).endswith("float") and lib.btps_kernel_tag(h, 12, batch).startswith("double")
    assert rel_err(d[:, gi].cpu().numpy().astype(np.float64), ref) <= TOL_F32S
    assert bool(torch.isfinite(d).all())


@pytest.mark.parametrize("n", [1024, 1100, 1536, 2048, 3000, 4096])
def test_f32_storage_on_clusters(lib, n):
    """*_f32s on the cluster kernels: N > 1024 (default) and the pair at N = 1024 (forced), a ring of floats, fp64 sweeps and
    fp64 carries across the CTAs.  Same bar as the single-CTA form: within one float ulp of the rounded fp64 solution."""
    batch = 1024 + 32
    lt, lp = inputs.tri_lhs(n, 0.5), inputs.penta_lhs(n, 0.5)
    r32 = inputs.uniform_rhs(n, batch, seed=80 + n).astype(np.float32)
    try:
        if n <= 1024:
            lib.btps_tune("cluster", 1)
        ht, hp = lib.tri_factor(*lt), lib.penta_factor(*lp)
        for kind in ("tri", "penta"):
            ref = r32.astype(np.float64)
            if kind == "tri":
                oracle.tri_solve_interleaved(oracle.tri_factor(*lt), ref)
            else:
                oracle.penta_solve_interleaved(oracle.penta_factor(*lp), ref)
            ref32 = ref.astype(np.float32).astype(np.float64)
            h = ht if kind == "tri" else hp
            tag = lib.btps_kernel_tag(h, 12, batch).split(", ")
            assert tag[0] == "double" and tag[8] == "1" and tag[9] == "float", tag
            d = torch.from_numpy(r32).cuda()
            (lib.tri_solve_batched_f32s if kind == "tri" else lib.penta_solve_batched_f32s)(h, d)
            got = d.cpu().numpy().astype(np.float64)
            ulp = np.spacing(np.abs(ref32).astype(np.float32)).astype(np.float64)
            assert np.all(np.abs(got - ref32) <= ulp + 1e-300), (n, kind)
            assert rel_err(got, ref) <= TOL_F32S, (n, kind)
    finally:
        lib.btps_tune("cluster", -1)


def test_f32_storage_rejects_what_it_does_not_cover(lib):
    # beyond the on-chip plans (N > 4096), and long systems whose row pitch TMA cannot take (not a multiple of 16 bytes)
    for n, batch in ((5000, 64), (2048, 63)):
        h = lib.tri_factor(*inputs.tri_lhs(n, 0.5))
        d = torch.zeros(n, batch, dtype=torch.float32, device="cuda")
        with pytest.raises(lib.BtpsError):
            lib.tri_solve_batched_f32s(h, d)
    hp = lib.tri_factor_periodic(*inputs.tri_lhs(64, 0.5))
    d = torch.zeros(64, 64, dtype=torch.float32, device="cuda")
    with pytest.raises(lib.BtpsError):
        lib.tri_solve_batched_f32s(hp, d)


# ---- long systems on thread-block clusters, at the batch bench.py times them on ---------------------------------------------

@pytest.mark.parametrize("kind,n,lb,f32", [("tri", 2048, 16, False), ("penta", 2048, 16, False), ("tri", 4096, 16, False),
                                           ("penta", 4096, 16, False), ("tri", 1536, 16, False), ("penta", 3072, 15, False),
                                           ("tri", 4096, 16, True), ("penta", 2048, 17, True)])
def test_long_systems_full_size_sampled(lib, kind, n, lb, f32):
    """N > 1024: the rows of a tile are spread over a cluster of 3-8 CTAs (default plan).  Sampled systems (first / last
    tiles, a stride through the rest) against the oracle, finiteness and the max-norm bound over every element, and the
    same launch twice gives the same bits (the carry inboxes are reused tile after tile)."""
    batch = 1 << lb
    dtype = torch.float32 if f32 else torch.float64
    elem = 4 if f32 else 8
    d = torch.empty(n, batch, dtype=dtype, device="cuda")
    inputs.fill_uniform_device(d, n, seed=31)
    ids = sample_ids(batch, 1024)
    gi = torch.from_numpy(ids).cuda()
    ref = inputs.uniform_rhs(n, len(ids), seed=31, systems=ids.astype(np.uint64))
    if f32:
        ref = ref.astype(np.float32).astype(np.float64)
    if kind == "tri":
        lhs = inputs.tri_lhs(n, 0.5)
        h = lib.tri_factor(*lhs)
        solve = lib.tri_solve_batched_f32 if f32 else lib.tri_solve_batched
        oracle.tri_solve_interleaved(oracle.tri_factor(*lhs), ref)
    else:
        lhs = inputs.penta_lhs(n, 0.5)
        h = lib.penta_factor(*lhs)
        solve = lib.penta_solve_batched_f32 if f32 else lib.penta_solve_batched
        oracle.penta_solve_interleaved(oracle.penta_factor(*lhs), ref)
    tag = lib.btps_kernel_tag(h, elem, batch)
    assert tag.split(", ")[8] == "1", tag   # the cluster kernel is the default plan for these sizes
    d2 = d.clone()
    solve(h, d)
    solve(h, d2)
    assert torch.equal(d, d2)
    got = d[:, gi].cpu().numpy().astype(np.float64)
    assert rel_err(got, ref) <= (TOL_F32 if f32 else TOL_SINGLE), (kind, n, batch, tag)
    assert bool(torch.isfinite(d).all())
    assert float(d.abs().max()) <= 1.2


def test_ragged_batch_at_full_size(lib):
    """A batch that is neither a multiple of the tile width nor 16-byte aligned in its pitch, at bench size: the direct-load
    scalar kernels on 2^20 + 17 systems (tail tile with 17 live columns), sampled against the oracle."""
    n, batch = 256, (1 << 20) + 17
    d = torch.empty(n, batch, dtype=torch.float64, device="cuda")
    inputs.fill_uniform_device(d, n, seed=33)
    ids = sample_ids(batch, 2048)
    gi = torch.from_numpy(ids).cuda()
    for kind in ("tri", "penta"):
        inputs.fill_uniform_device(d, n, seed=33)
        ref = inputs.uniform_rhs(n, len(ids), seed=33, systems=ids.astype(np.uint64))
        if kind == "tri":
            lhs = inputs.tri_lhs(n, 0.5)
            h = lib.tri_factor(*lhs)
            lib.tri_solve_batched(h, d)
            oracle.tri_solve_interleaved(oracle.tri_factor(*lhs), ref)
        else:
            lhs = inputs.penta_lhs(n, 0.5)
            h = lib.penta_factor(*lhs)
            lib.penta_solve_batched(h, d)
            oracle.penta_solve_interleaved(oracle.penta_factor(*lhs), ref)
        assert lib.btps_kernel_tag(h, 8, batch).split(", ")[5] == "0"   # no TMA prefetch: the pitch is not 16-byte aligned
        assert rel_err(d[:, gi].cpu().numpy(), ref) <= TOL_SINGLE, kind
        assert bool(torch.isfinite(d).all())
