"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on
the same seeded inputs.  Tolerance (BASELINE.json north_star; reading R): per species
block max|x_gpu - x_ref| / max|x_ref| <= 1e-10 for Jacobian values and C(f); conservation
residuals of the GPU's C(f) < 1e-12 relative; integer work (pattern) bit-exact.

Step a3 has two paths (include/landau.h): PER (every problem evaluates the pair tensor itself, k_pair_sym) and
SHARED (tensor once per call, fp64 tensor-core contraction, k_pair_tensor + k_apply_dmma).  The parity cases run
on both; the sizes are chosen so that every instantiation the launchers can select is compared with the oracle:
k_pair_split<4>, <2> (N < 1536, < 2560), k_pair_sym<64,2>, <128,2>, each with and without the all-pairs coincidence
test, k_apply_dmma<1,2>, <2,2>, <4,2>, k_band_factor / k_band_solve with 8-, 16- and 32-column blocks."""
import numpy as np
import pytest

from paper_2104_10000_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = 1e-10
PER, SHARED = 1, 2          # LANDAU_PAIR_PER_PROBLEM, LANDAU_PAIR_SHARED
PER_BATCH = 3               # (tests only) LANDAU_PAIR_PER_PROBLEM in a context made for >= 4 problems: the per-problem pair
                            # kernel then runs with its throughput tiling (k_pair_sym<64,2> / <128,2> from N = 2,560 / 4,096),
                            # in a context for fewer with the latency tiling (k_pair_split up to N = 8,192)
PATHS = [pytest.param(PER, id="per-problem"), pytest.param(PER_BATCH, id="per-problem-batch-tiles"), pytest.param(SHARED, id="shared")]


PATHS_BATCH = [pytest.param(PER, id="per-problem"), pytest.param(SHARED, id="shared")]      # contexts for >= 4 problems anyway


def ctx_args(path, nb):
    """(max_batch, pair_path) of a context that builds nb problems on `path`."""
    return (max(nb, 4), PER) if path == PER_BATCH else (nb, path)


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2104_10000_b200 import binding
    binding.lib()   # raises if the extension is missing: no silent fallback
    return binding


def block_err(x, ref):
    return np.abs(x - ref).max() / np.abs(ref).max()


def entry_err(x, ref):
    big = np.abs(ref) > 1e-8 * np.abs(ref).max()
    return (np.abs(x - ref)[big] / np.abs(ref)[big]).max()


def conservation_residuals(dof_r, dof_z, mass, Cf):
    S = Cf.shape[0]
    out = [abs(Cf[a].sum()) / np.abs(Cf[a]).sum() for a in range(S)]
    for psi in (dof_z, 0.5 * (dof_r ** 2 + dof_z ** 2)):
        num = abs(sum(mass[a] * (psi @ Cf[a]) for a in range(S)))
        den = sum(mass[a] * np.abs(psi * Cf[a]).sum() for a in range(S))
        out.append(num / den)
    return max(out)


def run_gpu(gpu, wl, problems, max_batch=None, batched=True, path=0):
    import torch
    mb, path = ctx_args(path, max_batch or len(problems))
    ctx = gpu.LandauContext(wl.mesh, wl.order, wl.species, mb, pair_path=path)
    if path:
        assert ctx.pair_path()[0] == path
    r, z = ctx.dof_coords()
    f = np.stack([inputs.nodal_f(wl, r, z, b) for b in problems])
    fd = torch.from_numpy(f).cuda()
    vals = torch.full((len(problems), ctx.S, ctx.nnz), float("nan"), dtype=torch.float64, device="cuda")
    Cf = torch.full((len(problems), ctx.S, ctx.n), float("nan"), dtype=torch.float64, device="cuda")
    if batched:
        ctx.jacobian_batched(fd, vals, Cf)
    else:
        for k in range(len(problems)):
            ctx.jacobian(fd[k], vals[k], Cf[k])
    mv = torch.zeros(ctx.nnz, dtype=torch.float64, device="cuda")
    ctx.mass(1.7, mv)
    torch.cuda.synchronize()
    return ctx, f, vals.cpu().numpy(), Cf.cpu().numpy(), mv.cpu().numpy()


def check_against_oracle(oracle, wl, ctx, f, vals, Cf, mv, problems):
    sp = oracle.build_space(wl.mesh, wl.order)
    rowptr, colidx = ctx.csr_pattern_host()
    assert np.array_equal(rowptr, sp.rowptr) and np.array_equal(colidx, sp.colidx)
    r, z = ctx.dof_coords()
    assert np.abs(r - sp.dof_r).max() < 1e-14 and np.abs(z - sp.dof_z).max() < 1e-14
    worst = 0.0
    for k in range(len(problems)):
        _, ovals, oCf, omv = oracle.build_all(wl.mesh, wl.order, wl.species, f[k], 1.7)
        for a in range(wl.species.S):
            ev, ec = block_err(vals[k, a], ovals[a]), block_err(Cf[k, a], oCf[a])
            assert ev <= TOL and ec <= TOL, (wl.name, k, a, ev, ec)
            assert entry_err(vals[k, a], ovals[a]) <= 1e-7
            worst = max(worst, ev, ec)
        assert block_err(mv, omv) <= 1e-13
        assert conservation_residuals(sp.dof_r, sp.dof_z, wl.species.mass, Cf[k]) < 1e-12
    return worst


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("cfg", [0, 1, 2])
def test_small_configs_full_parity(gpu, oracle, cfg, path):
    wl = inputs.config(cfg)
    ctx, f, vals, Cf, mv = run_gpu(gpu, wl, [0], path=path)
    worst = check_against_oracle(oracle, wl, ctx, f, vals, Cf, mv, [0])
    print(f"{wl.name}: worst block error {worst:.2e}")


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("cfg,variant", [(3, "A"), (3, "B"), (4, "B")])
def test_refined_configs_full_parity(gpu, oracle, cfg, variant, path):
    wl = inputs.config(cfg, variant=variant)
    ctx, f, vals, Cf, mv = run_gpu(gpu, wl, [0], path=path)
    worst = check_against_oracle(oracle, wl, ctx, f, vals, Cf, mv, [0])
    print(f"{wl.name}: worst block error {worst:.2e}")


@pytest.mark.parametrize("path", PATHS)
def test_table1_single_grid_mesh_parity_uses_the_64_point_tiles(gpu, oracle, path):
    """A uniform 10 x 20 Q3 mesh -- the single-grid case of the paper's Table I (3,200 integration points, L195-199;
    tests/golden/table1_counts.txt) -- has 2,560 <= N < 4,096, the range in which the per-problem pair kernel runs
    as k_pair_sym<64,2>: the whole path against the oracle, element by element."""
    mesh = inputs.mesh_uniform(0.0, 5.0, -5.0, 5.0, 10, 20)
    spc = inputs._sp([(1, -1, 1, 1), (3670, 1, 1, 1)])
    wl = inputs.Workload("table1-10x20-q3", 3, mesh, spc, [[inputs.Component(0, 1, 1), inputs.Component(1, 1, 1)]], 1e-3, 21)
    ctx, f, vals, Cf, mv = run_gpu(gpu, wl, [0], path=path)
    assert ctx.N == 3200
    worst = check_against_oracle(oracle, wl, ctx, f, vals, Cf, mv, [0])
    print(f"{wl.name}: worst block error {worst:.2e}")


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("cfg", [6, 7])
def test_paper_shaped_ten_species_context_parity(gpu, oracle, cfg, path):
    """e + D + 8 heavy-ion charge states on the 80- and 320-cell Q3 meshes."""
    wl = inputs.config(cfg)
    ctx, f, vals, Cf, mv = run_gpu(gpu, wl, [0], path=path)
    worst = check_against_oracle(oracle, wl, ctx, f, vals, Cf, mv, [0])
    print(f"{wl.name}: worst block error {worst:.2e}")


@pytest.mark.parametrize("cfg,variant", [(0, "B"), (3, "A"), (4, "B")])
def test_implicit_operator_parity(gpu, oracle, cfg, variant):
    """shift M + A(E_z) - J and A f - C(f) in one pass, against the oracle; two problems
    with different fields in one batched call; E_z = 0, shift = 0 reproduces -J and -C(f) bitwise."""
    import torch
    wl = inputs.config(cfg, variant=variant)
    ctx = gpu.LandauContext(wl.mesh, wl.order, wl.species, 2)
    r, z = ctx.dof_coords()
    f1 = inputs.nodal_f(wl, r, z)
    f = np.stack([f1, 1.25 * f1])
    Ez = np.array([0.37, -2.0])
    shift = 2.5
    fd = torch.from_numpy(f).cuda()
    vals = torch.full((2, ctx.S, ctx.nnz), float("nan"), dtype=torch.float64, device="cuda")
    F = torch.full((2, ctx.S, ctx.n), float("nan"), dtype=torch.float64, device="cuda")
    ctx.implicit_operator_batched(fd, torch.from_numpy(Ez).cuda(), shift, vals, F)
    sp = oracle.build_space(wl.mesh, wl.order)
    for k in range(2):
        ov, oF = oracle.implicit_operator(sp, wl.species, f[k], float(Ez[k]), shift)
        for a in range(ctx.S):
            assert block_err(vals[k, a].cpu().numpy(), ov[a]) <= TOL, (k, a)
            assert block_err(F[k, a].cpu().numpy(), oF[a]) <= TOL, (k, a)
    v0 = torch.zeros_like(vals); F0 = torch.zeros_like(F)
    ctx.implicit_operator_batched(fd, torch.zeros(2, dtype=torch.float64, device="cuda"), 0.0, v0, F0)
    vj = torch.zeros_like(vals); cj = torch.zeros_like(F)
    ctx.jacobian_batched(fd, vj, cj)
    assert torch.equal(v0, -vj) and torch.equal(F0, -cj)


def _multigrid_case(which):
    """inputs.multigrid_case, plus two cases with IDENTICAL Q3 grids (every point coincides with one of the other
    grid, so every pair is tested for coincidence) whose point totals select the 64- and 128-point tiles of the
    per-problem pair kernel: 'same2-q3-80' = 2 x 1,280 = 2,560 points, 'same2-q3-128' = 2 x 2,048 = 4,096 points;
    'same2-q3-60' = 2 x 960 = 1,920 points runs the 32-point tiles shared by two warps (the small Q2 'same2', 360
    points, those shared by four)."""
    if which in ("same2-q3-60", "same2-q3-80", "same2-q3-128"):
        m = {"same2-q3-60": inputs.mesh_uniform(0.0, 5.0, -5.0, 5.0, 6, 10), "same2-q3-80": inputs.config(6).mesh,
             "same2-q3-128": inputs.mesh_uniform(0.0, 5.0, -5.0, 5.0, 8, 16)}[which]
        spc = inputs._sp([(1, -1, 1, 1), (4, 1, 1, 1)])
        return which, 3, [m, m], spc, [0, 1], [inputs.Component(0, 1, 1), inputs.Component(1, 1, 1)]
    return inputs.multigrid_case(which)


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("which", ["same2", "scaled", "paper3", "same2-q3-60", "same2-q3-80", "same2-q3-128"])
def test_multigrid_parity(gpu, oracle, which, path):
    """SURVEY 8(f) NEXT-2 (section III-C): species on several grids, pair loop over the union of
    points.  'same2*' have every point of grid 1 on top of one of grid 0 (coincident pairs skipped across
    grids); 'paper3' is Table I's three 20-cell grids with ten species (960 points, 1,930 equations)."""
    import torch
    name, order, meshes, spc, sgrid, comps = _multigrid_case(which)
    mb, path = ctx_args(path, 2)
    ctx = gpu.LandauMultigridContext(meshes, sgrid, order, spc, mb)
    ctx.set_pair_path(path)
    assert ctx.pair_path()[0] == path
    if which == "same2-q3-80":
        assert ctx.N == 2560
    if which == "same2-q3-128":
        assert ctx.N == 4096
    if which == "paper3":
        assert ctx.N == 960 and ctx.f_stride == 1930
    fl = []
    for a, c in enumerate(comps):
        r, z = ctx.grid_dof_coords(sgrid[a])
        fa = inputs.maxwellian(float(spc.mass[a]), c.n, c.T, c.zs, r, z)
        fl.append(fa * (1.0 + 1e-3 * np.cos(7.0 * np.arange(r.shape[0]) + a)))
    f = np.concatenate(fl)
    fb = np.stack([f, 0.5 * f])
    vals = torch.full((2, ctx.vals_stride), float("nan"), dtype=torch.float64, device="cuda")
    Cf = torch.full((2, ctx.f_stride), float("nan"), dtype=torch.float64, device="cuda")
    mv = torch.full((ctx.mvals_size,), float("nan"), dtype=torch.float64, device="cuda")
    ctx.jacobian_batched(torch.from_numpy(fb).cuda(), vals, Cf)
    ctx.mass(1.7, mv)
    vals, Cf, mv = vals.cpu().numpy(), Cf.cpu().numpy(), mv.cpu().numpy()
    spaces, ov, oC, om = oracle.build_all_multigrid(meshes, order, spc, sgrid, fl, 1.7)
    for g, sp_ in enumerate(spaces):
        rowptr, colidx = ctx.grid_csr_pattern_host(g)
        assert np.array_equal(rowptr, sp_.rowptr) and np.array_equal(colidx, sp_.colidx)
    assert block_err(mv, np.concatenate(om)) <= 1e-13
    fs, vs = ctx.species_slices(), ctx.vals_slices()
    for a in range(ctx.S):
        assert block_err(vals[0, vs[a]], ov[a]) <= TOL, (which, a)
        assert block_err(Cf[0, fs[a]], oC[a]) <= TOL, (which, a)
        # the operator is quadratic in f: problem 1 (f/2) is a quarter of problem 0 (exact in binary)
        assert np.array_equal(Cf[1, fs[a]], 0.25 * Cf[0, fs[a]]) and np.array_equal(vals[1, vs[a]], 0.5 * vals[0, vs[a]])
    # conservation across grids: density per species, total z-momentum and energy
    psi_z = [spaces[sgrid[a]].dof_z for a in range(ctx.S)]
    psi_e = [0.5 * (spaces[sgrid[a]].dof_r ** 2 + spaces[sgrid[a]].dof_z ** 2) for a in range(ctx.S)]
    for a in range(ctx.S):
        assert abs(Cf[0, fs[a]].sum()) <= 1e-12 * np.abs(Cf[0, fs[a]]).sum()
    for psi in (psi_z, psi_e):
        num = abs(sum(spc.mass[a] * (psi[a] @ Cf[0, fs[a]]) for a in range(ctx.S)))
        den = sum(spc.mass[a] * np.abs(psi[a] * Cf[0, fs[a]]).sum() for a in range(ctx.S))
        assert num <= 1e-12 * den


HULL, FRONT = 1, 2          # LANDAU_BAND_HULL, LANDAU_BAND_FRONT


@pytest.mark.parametrize("method", [pytest.param(HULL, id="hull"), pytest.param(FRONT, id="front")])
@pytest.mark.parametrize("cfg,variant", [(0, "B"), (1, "B"), (3, "A"), (3, "B")])
def test_band_lu_solve_parity(gpu, oracle, cfg, variant, method):
    """SURVEY 8(f) NEXT-4 (section III-G): the matrices shift M + A - J of two problems factored and
    solved on the device (RCM order, no pivoting) against the library solve of the oracle's dense blocks, with both
    factorisation kernels: the front (envelope) kernel -- 16-column blocks for configs 0, 1, 3A, 32-column blocks for
    3B -- and the hull kernel.  The band workspace is NaN-filled first: neither kernel may read what the fill did not
    write.  Tolerance: 50 cond(A) eps on max|x| (forward error of a backward-stable solve), and the residual."""
    import torch
    wl = inputs.config(cfg, variant=variant)
    ctx = gpu.LandauContext(wl.mesh, wl.order, wl.species, 2)
    ctx.band_set_method(method)
    assert ctx.band_method()[0] == method
    r, z = ctx.dof_coords()
    f1 = inputs.nodal_f(wl, r, z)
    f = np.stack([f1, 0.8 * f1])
    Ez = np.array([0.1, -0.3]); shift = 4.0
    fd = torch.from_numpy(f).cuda()
    vals = torch.zeros((2, ctx.S, ctx.nnz), dtype=torch.float64, device="cuda")
    F = torch.zeros((2, ctx.S, ctx.n), dtype=torch.float64, device="cuda")
    ctx.implicit_operator_batched(fd, torch.from_numpy(Ez).cuda(), shift, vals, F)
    bw, md, ws = ctx.band_sizes()
    band = torch.full((2 * ws,), float("nan"), dtype=torch.float64, device="cuda")
    ctx.band_factor_batched(vals, band)
    rhs = torch.from_numpy(np.cos(0.37 * np.arange(2 * ctx.S * ctx.n)).reshape(2, ctx.S, ctx.n) + 2.0).cuda()
    x = torch.zeros_like(rhs)
    ctx.band_solve_batched(band, rhs, x)
    x2 = rhs.clone()
    ctx.band_solve_batched(band, x2, x2)                       # in place
    assert torch.equal(x, x2)
    sp = oracle.build_space(wl.mesh, wl.order)
    vals_h, x_h, rhs_h = vals.cpu().numpy(), x.cpu().numpy(), rhs.cpu().numpy()
    for k in range(2):
        for a in range(ctx.S):
            A = oracle.dense_from_csr(sp, vals_h[k, a])
            xo = oracle.solve_species(sp, vals_h[k, a], rhs_h[k, a])
            cond = np.linalg.cond(A)
            assert np.abs(x_h[k, a] - xo).max() <= 50 * cond * 2.2e-16 * np.abs(xo).max(), (k, a, cond)
            res = np.abs(A @ x_h[k, a] - rhs_h[k, a]).max() / (np.abs(A).sum(axis=1).max() * np.abs(x_h[k, a]).max())
            assert res <= 1e-13, (k, a, res)
    print(f"{wl.name}: n = {ctx.n}, half-bandwidth after RCM {bw}")


def test_band_lu_front_and_hull_kernels_agree_and_auto_chooses(gpu):
    """The two factorisation kernels give the same solution up to rounding (they eliminate the same entries; only
    the order inside a rank-KB update differs); LANDAU_BAND_AUTO takes the front family on the refined meshes (its
    flops are a sixth of the hull's) and, since the slot kernel needs neither fill nor gather nor scatter, also on the
    uniform Q3 mesh (front = hull there); the hull kernel where the largest front cannot fit shared memory, and forcing
    the front kernel there is refused; both are bitwise reproducible."""
    import torch
    for cfg, variant, want in ((3, "B", FRONT), (6, "B", FRONT), (2, "B", FRONT)):
        wl = inputs.config(cfg, variant=variant)
        ctx = gpu.LandauContext(wl.mesh, wl.order, wl.species, 2)
        assert ctx.band_method()[0] == want, (wl.name, ctx.band_method())
        r, z = ctx.dof_coords()
        f1 = inputs.nodal_f(wl, r, z)
        fd = torch.from_numpy(np.stack([f1, 0.9 * f1])).cuda()
        vals = torch.zeros((2, ctx.S, ctx.nnz), dtype=torch.float64, device="cuda")
        ctx.implicit_operator_batched(fd, torch.tensor([0.2, -0.1], dtype=torch.float64, device="cuda"), 3.0, vals, None)
        bw, md, ws = ctx.band_sizes()
        rhs = torch.from_numpy(np.sin(0.11 * np.arange(2 * ctx.S * ctx.n)).reshape(2, ctx.S, ctx.n) + 1.5).cuda()
        sols = {}
        for method in (HULL, FRONT, FRONT):
            ctx.band_set_method(method)
            band = torch.full((2 * ws,), float("nan"), dtype=torch.float64, device="cuda")
            piv = torch.zeros((2, ctx.S, 2), dtype=torch.float64, device="cuda")
            x = torch.empty_like(rhs)
            ctx.band_factor_batched(vals, band, piv)
            ctx.band_solve_batched(band, rhs, x)
            sols.setdefault(method, []).append((x.clone(), piv.clone()))
        (xh, ph), (xf, pf), (xf2, pf2) = sols[HULL][0], sols[FRONT][0], sols[FRONT][1]
        assert torch.equal(xf, xf2) and torch.equal(pf, pf2)
        assert bool(torch.isfinite(xf).all())
        assert float((xf - xh).abs().max() / xh.abs().max()) <= 1e-12
        assert float(((pf - ph).abs() / ph.abs()).max()) <= 1e-10          # the same pivots
        ctx.band_set_method(0)
        assert ctx.band_method()[0] == want
        ctx.destroy()
    mesh = inputs.mesh_uniform(0.0, 5.0, -5.0, 5.0, 46, 46)                # fronts of 420 rows: no shared memory for them
    ctx = gpu.LandauContext(mesh, 3, inputs._sp([(1, -1, 1, 1)]), 1)
    assert ctx.band_method()[0] == HULL
    with pytest.raises(gpu.LandauError) as ei:
        ctx.band_set_method(FRONT)
    assert ei.value.code == gpu.LANDAU_EINVAL


def test_one_implicit_step_through_the_whole_path_conserves(gpu):
    """Operator -> band LU -> solve chained on the device: one quasi-Newton iteration of backward Euler for
    Eq. 4 (E_z = 0), (M/dt - J(f0)) delta = C(f0), f1 = f0 + delta.  Because 1^T J_a = 0 and
    1^T C_a = 0 hold discretely, the step conserves every species' density to the accuracy of the linear
    solve (residual ~ eps |A| |delta|) -- the density part of the paper's conservation claim (L17) carried
    through the solver.  (Momentum and energy are conserved by C(f), i.e. at convergence of the iteration,
    not by one frozen-coefficient step.)"""
    import torch
    wl = inputs.config(3, variant="A")
    ctx = gpu.LandauContext(wl.mesh, wl.order, wl.species, 1)
    r, z = ctx.dof_coords()
    f0 = inputs.nodal_f(wl, r, z)[None]
    dt = 0.5
    fd = torch.from_numpy(f0).cuda()
    vals = torch.zeros((1, ctx.S, ctx.nnz), dtype=torch.float64, device="cuda")
    F = torch.zeros((1, ctx.S, ctx.n), dtype=torch.float64, device="cuda")
    ctx.implicit_operator_batched(fd, torch.zeros(1, dtype=torch.float64, device="cuda"), 1.0 / dt, vals, F)
    band = torch.empty(ctx.band_sizes()[2], dtype=torch.float64, device="cuda")
    ctx.band_factor_batched(vals, band)
    delta = torch.empty_like(F)
    ctx.band_solve_batched(band, -F, delta)           # F = -C(f0) here
    mv = torch.zeros(ctx.nnz, dtype=torch.float64, device="cuda")
    ctx.mass(1.0, mv)
    rowptr, colidx = ctx.csr_pattern_host()
    import scipy.sparse as sps
    M = sps.csr_matrix((mv.cpu().numpy(), colidx, rowptr), shape=(ctx.n, ctx.n))
    d = delta.cpu().numpy()[0]
    assert np.abs(d).max() > 1e-6 * np.abs(f0).max()                      # the step does something
    for a in range(ctx.S):
        Md = M @ d[a]
        assert abs(Md.sum()) <= 1e-9 * np.abs(Md).sum()                   # density of every species (solver accuracy)


def test_band_lu_wide_band_uses_the_16_column_blocks(gpu):
    """A 46 x 46 Q3 mesh (n = 19,321; the best order is the row sweep, half-bandwidth 3 x 139 + 3 = 420 > 416): the
    panels no longer fit shared memory with 32-column blocks, so the 16-column, 512-thread instantiation runs.
    Reference: scipy's sparse direct solve of the same CSR matrix (too large for the oracle's dense solve);
    tolerance through the residual."""
    import torch
    import scipy.sparse as sps
    import scipy.sparse.linalg as spla
    mesh = inputs.mesh_uniform(0.0, 5.0, -5.0, 5.0, 46, 46)
    spc = inputs._sp([(1, -1, 1, 1)])
    wl = inputs.Workload("q3-46x46", 3, mesh, spc, [[inputs.Component(0, 1, 1)]], 1e-3, 11)
    ctx = gpu.LandauContext(mesh, 3, spc, 1)
    bw, md, ws = ctx.band_sizes()
    assert 416 < bw <= 832 and ctx.n == 139 * 139, bw
    assert gpu.landau_band_order_host(mesh, 3)["block_columns"] == 16
    r, z = ctx.dof_coords()
    fd = torch.from_numpy(inputs.nodal_f(wl, r, z)[None]).cuda()
    vals = torch.zeros((1, 1, ctx.nnz), dtype=torch.float64, device="cuda")
    ctx.implicit_operator_batched(fd, torch.zeros(1, dtype=torch.float64, device="cuda"), 2.0, vals, None)
    band = torch.empty(ws, dtype=torch.float64, device="cuda")
    ctx.band_factor_batched(vals, band)
    rhs = torch.from_numpy(np.cos(0.01 * np.arange(ctx.n))[None, None] + 2.0).cuda()
    x = torch.empty_like(rhs)
    ctx.band_solve_batched(band, rhs, x)
    rowptr, colidx = ctx.csr_pattern_host()
    A = sps.csr_matrix((vals.cpu().numpy()[0, 0], colidx, rowptr), shape=(ctx.n, ctx.n))
    xg, b = x.cpu().numpy()[0, 0], rhs.cpu().numpy()[0, 0]
    res = np.abs(A @ xg - b).max() / (abs(A).sum(axis=1).max() * np.abs(xg).max())
    assert res <= 1e-13, res
    xs = spla.spsolve(A.tocsc(), b)
    assert np.abs(xg - xs).max() <= 1e-8 * np.abs(xs).max()


def test_deeply_refined_mesh_parity(gpu, oracle):
    """Six refinement levels toward the origin (cells from 2 down to 0.03, Gauss points 2e-3 from the axis, cell size
    ratios 64:1 across hanging-node chains): near pairs with k' = d/sqrt(s) ~ 1e-3 need the most AGM passes, far /
    near-axis pairs the small-m accuracy.  Cold electrons + ions resolved only by the finest cells."""
    mesh = inputs.mesh_quadtree(0.0, 8.0, -8.0, 8.0, 4, 8, 0.3, 6, 1.5, 3)
    spc = inputs._sp([(1, -1, 1, 0.01), (3670, 1, 1, 0.01)])
    comps = [[inputs.Component(0, 0.98, 0.01), inputs.Component(0, 0.02, 1.0, 0.5), inputs.Component(1, 1.0, 20.0)]]
    wl = inputs.Workload("deep-refined-q3", 3, mesh, spc, comps, 1e-3, 13)
    ctx, f, vals, Cf, mv = run_gpu(gpu, wl, [0])
    assert ctx.Ne == 332
    worst = check_against_oracle(oracle, wl, ctx, f, vals, Cf, mv, [0])
    print(f"{wl.name}: worst block error {worst:.2e}")


def test_edge_cases_of_the_next_rows(gpu, oracle):
    """One-cell mesh through the implicit operator and the band LU (n = 9 < one elimination block); NULL outputs;
    argument errors of the multigrid constructor."""
    import torch
    mesh = inputs.mesh_uniform(0.0, 2.0, -1.0, 1.0, 1, 1)
    spc = inputs._sp([(1, -1, 1, 1), (2, 1, 1, 1)])
    wl = inputs.Workload("one-cell-2sp", 2, mesh, spc, [[inputs.Component(0, 1, 1), inputs.Component(1, 1, 1)]], 1e-3, 7)
    ctx = gpu.LandauContext(mesh, 2, spc, 1)
    r, z = ctx.dof_coords()
    f = inputs.nodal_f(wl, r, z)[None]
    fd = torch.from_numpy(f).cuda()
    Ez = torch.tensor([0.5], dtype=torch.float64, device="cuda")
    vals = torch.zeros((1, ctx.S, ctx.nnz), dtype=torch.float64, device="cuda")
    ctx.implicit_operator_batched(fd, Ez, 3.0, vals, None)          # F skipped
    ctx.implicit_operator_batched(fd, Ez, 3.0, None, None)          # both skipped
    sp = oracle.build_space(mesh, 2)
    ov, _ = oracle.implicit_operator(sp, spc, f[0], 0.5, 3.0)
    bw, md, ws = ctx.band_sizes()
    assert ctx.n == 9 and bw == 8
    band = torch.empty(ws, dtype=torch.float64, device="cuda")
    ctx.band_factor_batched(vals, band)
    rhs = torch.arange(1.0, 1.0 + ctx.S * ctx.n, dtype=torch.float64, device="cuda").reshape(1, ctx.S, ctx.n)
    x = torch.empty_like(rhs)
    ctx.band_solve_batched(band, rhs, x)
    for a in range(ctx.S):
        assert block_err(vals[0, a].cpu().numpy(), ov[a]) <= TOL
        xo = oracle.solve_species(sp, ov[a], rhs[0, a].cpu().numpy())
        assert np.abs(x[0, a].cpu().numpy() - xo).max() <= 1e-10 * np.abs(xo).max()
    with pytest.raises(gpu.LandauError):
        ctx.band_solve_batched(band, torch.zeros((2, ctx.S, ctx.n), dtype=torch.float64, device="cuda"),
                               torch.zeros((2, ctx.S, ctx.n), dtype=torch.float64, device="cuda"))       # nb > max_batch
    g = inputs.config(0).mesh
    sp3 = inputs._sp([(1, -1, 1, 1), (4, 1, 1, 1), (8, 1, 1, 1)])
    for bad in ([1, 0, 1], [0, 0, 0], [0, 2, 2], [0, 1, 5]):         # not grouped / grid unused / out of range
        with pytest.raises(gpu.LandauError) as ei:
            gpu.LandauMultigridContext([g, inputs.mesh_scaled(g, 0.5)], bad, 2, sp3, 1)
        assert ei.value.code == gpu.LANDAU_EINVAL


def _inner_case(which):
    if which == "q2-180":         # 5 tiles of 32 + a tail of 20, four warps per tile pair
        return inputs.config(0)
    if which == "q3-2048":        # 64 whole tiles of 32, two warps per tile pair
        return inputs.config(2)
    if which == "q3-2992":        # 46 tiles of 64 + a tail of 48
        mesh = inputs.mesh_uniform(0.0, 5.0, -5.0, 5.0, 11, 17)
        spc = inputs._sp([(1, -1, 1, 1), (25, 1, 1, 1)])
        return inputs.Workload("q3-11x17", 3, mesh, spc, [[inputs.Component(0, 1, 1), inputs.Component(1, 1, 1, 0.2)]], 1e-3, 31)
    return inputs.config(3)       # 'q3-4928': 38 tiles of 128 + a tail of 64


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("which", ["q2-180", "q3-2048", "q3-2992", "q3-4928"])
def test_inner_integral_parity(gpu, oracle, which, path):
    """Steps a1-a3 alone: G_D, G_K at every integration point, one case per launch shape of the per-problem pair
    kernel (32-point tiles shared by 4 / 2 warps, 64- and 128-point tiles), with ragged last tiles, and the same cases through the shared path
    (ragged last chunk of 16 source points, ragged target tile, 1 / 2 / 4 splits of the source range)."""
    import torch
    wl = _inner_case(which)
    mb, path = ctx_args(path, 1)
    ctx = gpu.LandauContext(wl.mesh, wl.order, wl.species, mb, pair_path=path)
    r, z = ctx.dof_coords()
    f = inputs.nodal_f(wl, r, z)
    G = torch.zeros((1, 5, ctx.N), dtype=torch.float64, device="cuda")
    ctx.inner_integral(torch.from_numpy(f[None]).cuda(), G)
    G = G.cpu().numpy()[0]
    sp = oracle.build_space(wl.mesh, wl.order)
    pr, pz, pw = ctx.points()
    assert np.abs(pr - sp.r).max() < 1e-14 and np.abs(pz - sp.z).max() < 1e-14 and np.abs(pw - sp.w_in).max() <= 1e-15 * sp.w_in.max()
    _, _, (GD, GK) = oracle.coefficients(sp, wl.species, f)
    ref = np.concatenate([GD.T, GK.T])
    for c in range(5):
        assert block_err(G[c], ref[c]) <= 1e-12, c


@pytest.mark.parametrize("path", PATHS_BATCH)
def test_config5_batched_full_size(gpu, oracle, path):
    """BASELINE config 5 at full size (512 problems, the launch shape bench.py times): sampled
    problems against the oracle one by one; conservation (holds at any size) on all 512."""
    wl = inputs.config(5)
    problems = list(range(wl.nbatch))
    ctx, f, vals, Cf, mv = run_gpu(gpu, wl, problems, path=path)
    assert np.isfinite(vals).all() and np.isfinite(Cf).all()
    # scratch of step a3 does not grow with the batch beyond ~1 GB on either path (per-problem: the batch goes
    # through the pair kernel in groups of 139 problems, so this call is 139 + 139 + 139 + 95)
    assert ctx.pair_path()[1] <= 1.6e9
    sp = oracle.build_space(wl.mesh, wl.order)
    for k in problems:
        assert conservation_residuals(sp.dof_r, sp.dof_z, wl.species.mass, Cf[k]) < 1e-12, k
    # first, last, and the extremes of bulk temperature, tail fraction and z-shift, filled up to 8
    Tb = [wl.components[b][0].T for b in problems]
    tail = [wl.components[b][1].n for b in problems]
    zs = [wl.components[b][1].zs for b in problems]
    sample = {0, wl.nbatch - 1}
    for q in (Tb, tail, zs):
        sample |= {int(np.argmin(q)), int(np.argmax(q))}
    sample = sorted(sample | set(range(101, 101 + 8 - len(sample))))
    assert len(sample) >= 8
    for k in sample:
        _, ovals, oCf, _ = oracle.build_all(wl.mesh, wl.order, wl.species, f[k], 1.0)
        for a in range(2):
            assert block_err(vals[k, a], ovals[a]) <= TOL, (k, a)
            assert block_err(Cf[k, a], oCf[a]) <= TOL, (k, a)


@pytest.mark.parametrize("path", PATHS_BATCH)
@pytest.mark.parametrize("cfg,variant,nb", [(1, "B", 8192), (2, "B", 512), (3, "A", 1024)])
def test_per_config_batches_of_the_bench_at_full_size(gpu, oracle, cfg, variant, nb, path):
    """The batched launches bench.py times for configs 1, 2 and 3A (`per_config[*].batched`: 8,192 / 512 / 1,024 problems,
    both paths through step a3) at full size: every problem gets its own f (the config's f, each species scaled by
    a problem-dependent factor), all outputs finite, conservation on a spread of problems, and sampled problems
    against the oracle one by one."""
    import torch
    wl = inputs.config(cfg, variant=variant)
    mb, path = ctx_args(path, nb)
    ctx = gpu.LandauContext(wl.mesh, wl.order, wl.species, mb, pair_path=path)
    r, z = ctx.dof_coords()
    f0 = inputs.nodal_f(wl, r, z)
    S = wl.species.S
    scale = 1.0 + 0.3 * np.sin(0.37 * np.arange(nb)[:, None] + 1.3 * np.arange(S)[None, :])       # [nb][S], in [0.7, 1.3]
    f = f0[None] * scale[:, :, None]
    fd = torch.from_numpy(f).cuda()
    vals = torch.full((nb, ctx.S, ctx.nnz), float("nan"), dtype=torch.float64, device="cuda")
    Cf = torch.full((nb, ctx.S, ctx.n), float("nan"), dtype=torch.float64, device="cuda")
    ctx.jacobian_batched(fd, vals, Cf)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(vals).all()) and bool(torch.isfinite(Cf).all())
    sp = oracle.build_space(wl.mesh, wl.order)
    Cf_h = Cf.cpu().numpy()
    for k in range(0, nb, max(1, nb // 64)):
        assert conservation_residuals(sp.dof_r, sp.dof_z, wl.species.mass, Cf_h[k]) < 1e-12, k
    for k in (0, nb // 2 + 1, nb - 1):
        _, ovals, oCf, _ = oracle.build_all(wl.mesh, wl.order, wl.species, f[k], 1.0)
        vk = vals[k].cpu().numpy()
        for a in range(S):
            assert block_err(vk[a], ovals[a]) <= TOL, (k, a)
            assert block_err(Cf_h[k, a], oCf[a]) <= TOL, (k, a)


@pytest.mark.parametrize("path", PATHS_BATCH)
def test_batched_equals_loop_of_singles_bitwise_and_is_deterministic(gpu, path):
    """Inside one path a problem's result does not depend on the batch it is built in: 24 problems in one call,
    again, one by one, and (other tile shapes of the shared path's contraction) in calls of 17 + 7."""
    import torch
    wl = inputs.config(5, nbatch=24, variant="A")
    problems = list(range(24))
    _, _, v1, c1, _ = run_gpu(gpu, wl, problems, batched=True, path=path)
    _, _, v2, c2, _ = run_gpu(gpu, wl, problems, batched=True, path=path)
    _, _, v3, c3, _ = run_gpu(gpu, wl, problems, batched=False, path=path)
    assert np.array_equal(v1, v2) and np.array_equal(c1, c2)      # run-to-run determinism
    assert np.array_equal(v1, v3) and np.array_equal(c1, c3)      # batch shape == split shape, bitwise
    ctx = gpu.LandauContext(wl.mesh, wl.order, wl.species, 24, pair_path=ctx_args(path, 24)[1])
    r, z = ctx.dof_coords()
    fd = torch.from_numpy(np.stack([inputs.nodal_f(wl, r, z, b) for b in problems])).cuda()
    v4 = torch.zeros((24, ctx.S, ctx.nnz), dtype=torch.float64, device="cuda")
    c4 = torch.zeros((24, ctx.S, ctx.n), dtype=torch.float64, device="cuda")
    ctx.jacobian_batched(fd[:17], v4[:17], c4[:17])
    ctx.jacobian_batched(fd[17:], v4[17:], c4[17:])
    assert np.array_equal(v4.cpu().numpy(), v1) and np.array_equal(c4.cpu().numpy(), c1)


@pytest.mark.parametrize("path", PATHS_BATCH)
def test_calls_of_64_and_more_problems_equal_smaller_calls_bitwise(gpu, path):
    """From 64 problems per call on, a warp of `k_element_q3` takes four cells one after the other and prefetches the
    next cell's inputs (cp.async, two shared-memory buffers); below, one cell per warp.  Same values, bitwise: mesh 3A
    (98 cells: the last block and the last rounds are ragged), Jacobian and implicit-step operator, 70 problems in one
    call against 35 + 35; and Table I's three 20-cell grids with ten species, 64 problems against 32 + 32."""
    import torch
    wl = inputs.config(3, variant="A")
    nb = 70
    mb, pth = ctx_args(path, nb)
    ctx = gpu.LandauContext(wl.mesh, wl.order, wl.species, mb, pair_path=pth)
    r, z = ctx.dof_coords()
    f0 = inputs.nodal_f(wl, r, z)
    scale = 1.0 + 0.3 * np.sin(0.41 * np.arange(nb)[:, None] + 1.1 * np.arange(ctx.S)[None, :])
    fd = torch.from_numpy(f0[None] * scale[:, :, None]).cuda()
    Ez = torch.from_numpy(0.1 + 0.01 * np.arange(nb)).cuda()
    out = []
    for split in ((nb,), (35, 35)):
        v = torch.full((nb, ctx.S, ctx.nnz), float("nan"), dtype=torch.float64, device="cuda")
        c = torch.full((nb, ctx.S, ctx.n), float("nan"), dtype=torch.float64, device="cuda")
        vi, ci = torch.full_like(v, float("nan")), torch.full_like(c, float("nan"))
        b0 = 0
        for m in split:
            ctx.jacobian_batched(fd[b0:b0 + m], v[b0:b0 + m], c[b0:b0 + m])
            ctx.implicit_operator_batched(fd[b0:b0 + m], Ez[b0:b0 + m], 2.0, vi[b0:b0 + m], ci[b0:b0 + m])
            b0 += m
        out.append([t.cpu().numpy() for t in (v, c, vi, ci)])
    for a, b in zip(*out):
        assert np.isfinite(a).all() and np.array_equal(a, b)
    ctx.destroy()
    name, order, meshes, spc, sgrid, comps = inputs.multigrid_case("paper3")
    nb = 64
    mb, pth = ctx_args(path, nb)
    ctx = gpu.LandauMultigridContext(meshes, sgrid, order, spc, mb)
    ctx.set_pair_path(pth)
    fl = []
    for a, c in enumerate(comps):
        r, z = ctx.grid_dof_coords(sgrid[a])
        fl.append(inputs.maxwellian(float(spc.mass[a]), c.n, c.T, c.zs, r, z))
    f = np.concatenate(fl)
    fd = torch.from_numpy(f[None] * (1.0 + 0.2 * np.cos(0.3 * np.arange(nb)))[:, None]).cuda()
    out = []
    for split in ((nb,), (32, 32)):
        v = torch.full((nb, ctx.vals_stride), float("nan"), dtype=torch.float64, device="cuda")
        c = torch.full((nb, ctx.f_stride), float("nan"), dtype=torch.float64, device="cuda")
        b0 = 0
        for m in split:
            ctx.jacobian_batched(fd[b0:b0 + m], v[b0:b0 + m], c[b0:b0 + m])
            b0 += m
        out.append([v.cpu().numpy(), c.cpu().numpy()])
    for a, b in zip(*out):
        assert np.isfinite(a).all() and np.array_equal(a, b)
    ctx.destroy()


def test_no_state_carried_between_calls(gpu):
    """A, then a different problem and a different batch size, then A again in the same context: bitwise the
    same A (nothing is read from scratch that the call itself did not write); also through the implicit
    operator and the band LU, whose workspace is poisoned with NaN in between."""
    import torch
    wl = inputs.config(5, nbatch=6, variant="A")
    ctx = gpu.LandauContext(wl.mesh, wl.order, wl.species, 6)
    r, z = ctx.dof_coords()
    f = torch.from_numpy(np.stack([inputs.nodal_f(wl, r, z, b) for b in range(6)])).cuda()

    def build(fb):
        nb = fb.shape[0]
        v = torch.full((nb, ctx.S, ctx.nnz), float("nan"), dtype=torch.float64, device="cuda")
        c = torch.full((nb, ctx.S, ctx.n), float("nan"), dtype=torch.float64, device="cuda")
        ctx.implicit_operator_batched(fb, torch.full((nb,), 0.2, dtype=torch.float64, device="cuda"), 3.0, v, c)
        band = torch.full((nb * ctx.band_sizes()[2],), float("nan"), dtype=torch.float64, device="cuda")
        ctx.band_factor_batched(v, band)
        x = torch.full_like(c, float("nan"))
        ctx.band_solve_batched(band, c, x)
        return v, c, x
    a1 = build(f[:2])
    build(7.0 * f[1:6])
    a2 = build(f[:2])
    for p, q in zip(a1, a2):
        assert torch.isfinite(p).all() and torch.equal(p, q)


def test_host_entry_point_equals_device_entry_point(gpu):
    import torch
    wl = inputs.config(5, nbatch=3, variant="A")
    ctx, f, vals, Cf, _ = run_gpu(gpu, wl, [0, 1, 2])
    fh = torch.from_numpy(f).pin_memory()
    vh = torch.zeros((3, ctx.S, ctx.nnz), dtype=torch.float64).pin_memory()
    ch = torch.zeros((3, ctx.S, ctx.n), dtype=torch.float64).pin_memory()
    ctx.jacobian_host(fh, vh, ch)
    assert np.array_equal(vh.numpy(), vals) and np.array_equal(ch.numpy(), Cf)
    v2 = np.zeros_like(vals)
    ctx.jacobian_host(f, v2, None)                                  # pageable numpy buffers
    assert np.array_equal(v2, vals)


def test_edge_cases(gpu, oracle):
    import torch
    # single cell, Q2: 9 points, one ragged tile
    mesh = inputs.mesh_uniform(0.0, 2.0, -1.0, 1.0, 1, 1)
    spc = inputs._sp([(1, -1, 1, 1)])
    wl = inputs.Workload("one-cell", 2, mesh, spc, [[inputs.Component(0, 1, 1)]], 1e-3, 5)
    ctx, f, vals, Cf, mv = run_gpu(gpu, wl, [0])
    check_against_oracle(oracle, wl, ctx, f, vals, Cf, mv, [0])
    # f = 0 -> J = 0, C = 0 exactly
    z = torch.zeros((1, ctx.n), dtype=torch.float64, device="cuda")
    v = torch.ones((1, ctx.nnz), dtype=torch.float64, device="cuda")
    c = torch.ones((1, ctx.n), dtype=torch.float64, device="cuda")
    ctx.jacobian(z, v, c)
    assert float(v.abs().max()) == 0.0 and float(c.abs().max()) == 0.0
    # nb > max_batch is refused; NULL outputs are skipped
    with pytest.raises(gpu.LandauError):
        ctx.jacobian_batched(torch.zeros((2, 1, ctx.n), dtype=torch.float64, device="cuda"), None, None)
    ctx.jacobian(z, None, None)
    torch.cuda.synchronize()
    # maximum species count (16) on a refined mesh
    m16 = inputs.config(0).mesh
    rows = [(1.0 + 3.0 * s, (-1) ** s * (1 + s % 3), 1.0, 1.0) for s in range(16)]
    sp16 = inputs._sp(rows)
    wl16 = inputs.Workload("16sp", 2, m16, sp16, [[inputs.Component(s, 1.0, 1.0 + 0.1 * s, 0.05 * s) for s in range(16)]], 1e-3, 6)
    ctx, f, vals, Cf, mv = run_gpu(gpu, wl16, [0])
    check_against_oracle(oracle, wl16, ctx, f, vals, Cf, mv, [0])
    with pytest.raises(gpu.LandauError):
        gpu.LandauContext(m16, 2, inputs._sp(rows + [(2.0, 1, 1, 1)]))   # S = 17 > 16


def test_band_lu_widest_band_uses_the_8_column_blocks(gpu):
    """A 92 x 92 Q3 mesh (n = 76,729, N = 135,424 points; half-bandwidth of the row sweep 3 x 277 + 3 = 834 > 832):
    the panels only fit shared memory with 8-column blocks, so k_band_factor<8,512> / k_band_solve<8,512> run.
    Reference: scipy's sparse direct solve of the same CSR matrix; the pivot report must show a healthy elimination."""
    import torch
    import scipy.sparse as sps
    import scipy.sparse.linalg as spla
    mesh = inputs.mesh_uniform(0.0, 5.0, -5.0, 5.0, 92, 92)
    spc = inputs._sp([(1, -1, 1, 1)])
    wl = inputs.Workload("q3-92x92", 3, mesh, spc, [[inputs.Component(0, 1, 1)]], 1e-3, 12)
    ctx = gpu.LandauContext(mesh, 3, spc, 1)
    bw, md, ws = ctx.band_sizes()
    assert bw > 832 and ctx.n == 277 * 277, bw
    assert gpu.landau_band_order_host(mesh, 3)["block_columns"] == 8
    r, z = ctx.dof_coords()
    fd = torch.from_numpy(inputs.nodal_f(wl, r, z)[None]).cuda()
    vals = torch.zeros((1, 1, ctx.nnz), dtype=torch.float64, device="cuda")
    ctx.implicit_operator_batched(fd, torch.zeros(1, dtype=torch.float64, device="cuda"), 2.0, vals, None)
    band = torch.empty(ws, dtype=torch.float64, device="cuda")
    piv = torch.full((1, 1, 2), float("nan"), dtype=torch.float64, device="cuda")
    ctx.band_factor_batched(vals, band, piv)
    rhs = torch.from_numpy(np.cos(0.01 * np.arange(ctx.n))[None, None] + 2.0).cuda()
    x = torch.empty_like(rhs)
    ctx.band_solve_batched(band, rhs, x)
    pmin, pmax = piv.cpu().numpy()[0, 0]
    assert 0.0 < pmin <= pmax and pmin > 1e-8 * pmax
    rowptr, colidx = ctx.csr_pattern_host()
    A = sps.csr_matrix((vals.cpu().numpy()[0, 0], colidx, rowptr), shape=(ctx.n, ctx.n))
    xg, b = x.cpu().numpy()[0, 0], rhs.cpu().numpy()[0, 0]
    res = np.abs(A @ xg - b).max() / (abs(A).sum(axis=1).max() * np.abs(xg).max())
    assert res <= 1e-13, res
    xs = spla.spsolve(A.tocsc(), b)
    assert np.abs(xg - xs).max() <= 1e-8 * np.abs(xs).max()


def test_band_lu_reports_breakdown_instead_of_returning_nan_silently(gpu, oracle):
    """landau_band_factor_batched's pivot report: for sound matrices the smallest and largest |pivot| equal those of
    Alg. 4.3.1 (Golub & Van Loan) run by the oracle on the RCM-ordered dense block; a matrix with
    a zero pivot is flagged by smallest = 0 while its neighbours in the batch are untouched."""
    import torch
    wl = inputs.config(0)
    ctx = gpu.LandauContext(wl.mesh, wl.order, wl.species, 3)
    r, z = ctx.dof_coords()
    f = np.stack([inputs.nodal_f(wl, r, z)] * 3)
    fd = torch.from_numpy(f).cuda()
    vals = torch.zeros((3, ctx.S, ctx.nnz), dtype=torch.float64, device="cuda")
    ctx.implicit_operator_batched(fd, torch.zeros(3, dtype=torch.float64, device="cuda"), 3.0, vals, None)
    vals[1, 0].zero_()                                   # problem 1, species 0: the zero matrix
    bw, md, ws = ctx.band_sizes()
    band = torch.empty(3 * ws, dtype=torch.float64, device="cuda")
    piv = torch.full((3, ctx.S, 2), float("nan"), dtype=torch.float64, device="cuda")
    ctx.band_factor_batched(vals, band, piv)
    piv = piv.cpu().numpy()
    assert piv[1, 0, 0] == 0.0                           # breakdown reported
    sp = oracle.build_space(wl.mesh, wl.order)
    perm = gpu.landau_band_order_host(wl.mesh, wl.order)["perm"]
    for (k, a) in [(0, 0), (0, 1), (1, 1), (2, 0), (2, 1)]:
        A = oracle.dense_from_csr(sp, vals[k, a].cpu().numpy())[np.ix_(perm, perm)]
        LU = oracle.band_lu_outer_product(A, bw, bw)
        d = np.abs(np.diag(LU))
        assert abs(piv[k, a, 0] - d.min()) <= 1e-10 * d.min() and abs(piv[k, a, 1] - d.max()) <= 1e-10 * d.max(), (k, a)
    rhs = torch.ones((3, ctx.S, ctx.n), dtype=torch.float64, device="cuda")
    x = torch.empty_like(rhs)
    ctx.band_solve_batched(band, rhs, x)
    assert torch.isfinite(x[0]).all() and torch.isfinite(x[2]).all() and torch.isfinite(x[1, 1]).all()
    assert torch.equal(x[0], x[2])


def test_multigrid_implicit_operator_band_lu_and_partial_solve(gpu, oracle):
    """Several grids through NEXT-3 and NEXT-4 together: the implicit-step operator of the 'scaled' two-grid case
    (blocks = each grid's mass + advection - its Jacobian block), band LU of every species block, solves; then a
    solve of the FIRST problem only against the workspace factored for two (problem-major workspace)."""
    import torch
    name, order, meshes, spc, sgrid, comps = inputs.multigrid_case("scaled")
    ctx = gpu.LandauMultigridContext(meshes, sgrid, order, spc, 2)
    fl = []
    for a, c in enumerate(comps):
        r, z = ctx.grid_dof_coords(sgrid[a])
        fl.append(inputs.maxwellian(float(spc.mass[a]), c.n, c.T, c.zs, r, z))
    f = np.concatenate(fl)
    fb = torch.from_numpy(np.stack([f, 0.7 * f])).cuda()
    Ez, shift = np.array([0.2, -0.1]), 5.0
    vals = torch.full((2, ctx.vals_stride), float("nan"), dtype=torch.float64, device="cuda")
    F = torch.full((2, ctx.f_stride), float("nan"), dtype=torch.float64, device="cuda")
    ctx.implicit_operator_batched(fb, torch.from_numpy(Ez).cuda(), shift, vals, F)
    vj = torch.zeros_like(vals); cj = torch.zeros_like(F); mv = torch.zeros(ctx.mvals_size, dtype=torch.float64, device="cuda")
    ctx.jacobian_batched(fb, vj, cj)
    ctx.mass(shift, mv)
    spaces = [oracle.build_space(m, order) for m in meshes]
    fs, vs = ctx.species_slices(), ctx.vals_slices()
    moff = np.concatenate([[0], np.cumsum([g["nnz"] for g in ctx.grids])])
    vals_h, F_h, vj_h, cj_h, mv_h = (t.cpu().numpy() for t in (vals, F, vj, cj, mv))
    one = inputs._sp([(1, 1, 1, 1)])
    for k in range(2):
        for a in range(ctx.S):
            g = sgrid[a]
            qm = float(spc.charge[a] * spc.m0 / spc.mass[a])
            Aadv = qm * oracle.csr_values(spaces[g], oracle.advection(spaces[g], one, float(Ez[k]))[0])   # unit species, scaled
            ref = mv_h[moff[g]:moff[g + 1]] + Aadv - vj_h[k, vs[a]]
            assert block_err(vals_h[k, vs[a]], ref) <= 1e-12, (k, a)
    bw, md, ws = ctx.band_sizes()
    band = torch.empty(2 * ws, dtype=torch.float64, device="cuda")
    piv = torch.zeros((2, ctx.S, 2), dtype=torch.float64, device="cuda")
    ctx.band_factor_batched(vals, band, piv)
    assert (piv[:, :, 0] > 0).all()
    rhs = torch.from_numpy(np.cos(0.3 * np.arange(2 * ctx.f_stride)).reshape(2, ctx.f_stride) + 2.0).cuda()
    x = torch.empty_like(rhs)
    ctx.band_solve_batched(band, rhs, x)
    x_h, rhs_h = x.cpu().numpy(), rhs.cpu().numpy()
    for k in range(2):
        for a in range(ctx.S):
            A = oracle.dense_from_csr(spaces[sgrid[a]], vals_h[k, vs[a]])
            xo = np.linalg.solve(A, rhs_h[k, fs[a]])
            assert np.abs(x_h[k, fs[a]] - xo).max() <= 50 * np.linalg.cond(A) * 2.2e-16 * np.abs(xo).max(), (k, a)
    x1 = torch.empty((1, ctx.f_stride), dtype=torch.float64, device="cuda")
    ctx.band_solve_batched(band, rhs[:1].contiguous(), x1)       # nb = 1 against the workspace factored with nb = 2
    assert torch.equal(x1[0], x[0])


def test_pair_paths_can_be_switched_and_the_tensor_cache_changes_nothing(gpu):
    """landau_set_pair_path replaces the scratch of step a3 inside a live ctx; both paths give the same sums up to
    rounding; with the tensor cache on, calls skip k_pair_tensor (one launch fewer) and are bitwise equal to a
    call that evaluates it again."""
    import torch
    wl = inputs.config(5, nbatch=5, variant="A")
    ctx = gpu.LandauContext(wl.mesh, wl.order, wl.species, 5)
    assert ctx.pair_path()[0] == gpu.LANDAU_PAIR_SHARED           # max_batch >= LANDAU_SHARED_MIN_BATCH
    assert gpu.LandauContext(wl.mesh, wl.order, wl.species, 3).pair_path()[0] == gpu.LANDAU_PAIR_PER_PROBLEM
    r, z = ctx.dof_coords()
    fd = torch.from_numpy(np.stack([inputs.nodal_f(wl, r, z, b) for b in range(5)])).cuda()

    def build():
        v = torch.full((5, ctx.S, ctx.nnz), float("nan"), dtype=torch.float64, device="cuda")
        c = torch.full((5, ctx.S, ctx.n), float("nan"), dtype=torch.float64, device="cuda")
        l0 = ctx.launch_count()
        ctx.jacobian_batched(fd, v, c)
        torch.cuda.synchronize()
        return v, c, ctx.launch_count() - l0
    vs, cs, ls = build()
    ctx.set_tensor_cache(True)
    v1, c1, l1 = build()
    v2, c2, l2 = build()
    assert l1 == ls - 1 and l2 == ls - 1        # the tensor of the call before the switch is still valid
    assert torch.equal(v1, vs) and torch.equal(v2, vs) and torch.equal(c2, cs)
    ctx.set_tensor_cache(False)
    assert build()[2] == ls
    ctx.set_pair_path(gpu.LANDAU_PAIR_PER_PROBLEM)
    path, nbytes = ctx.pair_path()
    assert path == gpu.LANDAU_PAIR_PER_PROBLEM and nbytes > 0
    vp, cp, _ = build()
    for a in range(ctx.S):
        assert block_err(vp[:, a].cpu().numpy(), vs[:, a].cpu().numpy()) <= 1e-12
        assert block_err(cp[:, a].cpu().numpy(), cs[:, a].cpu().numpy()) <= 1e-12
    ctx.set_pair_path(gpu.LANDAU_PAIR_AUTO)
    assert ctx.pair_path()[0] == gpu.LANDAU_PAIR_SHARED
    v3, c3, _ = build()
    assert torch.equal(v3, vs) and torch.equal(c3, cs)


def test_a_batch_that_cannot_fit_fails_cleanly_with_enomem(gpu):
    """max_batch = 65,535 with 16 species on mesh 3B asks for 660 GB of element matrices: landau_create returns
    LANDAU_ENOMEM (nothing is left allocated: a normal ctx can be created and used right after)."""
    import torch
    mesh = inputs.mesh_config3("B")
    rows = [(1.0 + 3.0 * s, (-1) ** s * (1 + s % 3), 1.0, 1.0) for s in range(16)]
    free0 = torch.cuda.mem_get_info()[0]
    with pytest.raises(gpu.LandauError) as ei:
        gpu.LandauContext(mesh, 3, inputs._sp(rows), 65535)
    assert ei.value.code == gpu.LANDAU_ENOMEM
    with pytest.raises(gpu.LandauError) as ei:
        gpu.LandauContext(mesh, 3, inputs._sp(rows), 65536)        # beyond the documented range of max_batch
    assert ei.value.code == gpu.LANDAU_EINVAL
    assert abs(torch.cuda.mem_get_info()[0] - free0) < (64 << 20)
    wl = inputs.config(0)
    ctx, f, vals, Cf, mv = run_gpu(gpu, wl, [0])
    assert np.isfinite(vals).all()
