"""landau_band_solve_static (include/landau.h): the band solve of PAPER.md section III-G with its permuted vectors in
a file-scope __device__ scratch of the library instead of shared memory / a cudaMalloc'ed scratch -- the entry point
for callers that cannot allocate.  Compared with the existing path, landau_band_solve_batched, on the same factors.

Collected last on purpose (file name): the suite runs with `pytest -x`, a failure here must not hide other tests.
The tests pass alone in a fresh process and after the other GPU tests (the scratch is shared by every ctx of the
process and keeps the last call's contents; nothing in it has to start at zero)."""
import numpy as np
import pytest

from paper_2104_10000_b200 import inputs

pytestmark = pytest.mark.gpu
RTOL = 1e-12        # both paths run the same substitutions in the same order; the parity tests' TOL is 1e-10


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2104_10000_b200 import binding
    binding.lib()   # raises if the extension is missing: no silent fallback
    return binding


def _rel(a, b):
    return float((a - b).abs().max() / b.abs().max())


def _factored(gpu, torch, ctx, f, nb):
    """The matrices shift M + A(E_z) - J of nb problems, factored: (band workspace, ws doubles per problem)."""
    multigrid = hasattr(ctx, "f_stride")         # the two context classes name their layouts differently
    fshape = (nb, ctx.f_stride) if multigrid else (nb, ctx.S, ctx.n)
    vshape = (nb, ctx.vals_stride) if multigrid else (nb, ctx.S, ctx.nnz)
    fd = torch.from_numpy(np.ascontiguousarray(f).reshape(fshape)).cuda()
    Ez = torch.from_numpy(0.1 - 0.05 * np.arange(nb)).cuda()
    vals = torch.zeros(vshape, dtype=torch.float64, device="cuda")
    F = torch.zeros(fshape, dtype=torch.float64, device="cuda")
    ctx.implicit_operator_batched(fd, Ez, 4.0, vals, F)
    ws = ctx.band_sizes()[2]
    band = torch.full((nb * ws,), float("nan"), dtype=torch.float64, device="cuda")
    ctx.band_factor_batched(vals, band)
    return band


def test_static_scratch_solve_equals_existing_solve_on_two_calls_in_a_row(gpu):
    """Mesh 3A (n = 901, two species): three problems solved by the existing path and by the static-scratch entry point,
    twice in a row with different right-hand sides and batch sizes (the second call finds the first one's vectors in
    the scratch), out of place and in place; then a second ctx on the ten-species 80-cell mesh, which shares the array."""
    import torch
    wl = inputs.config(3, variant="A")
    nb = 3
    ctx = gpu.LandauContext(wl.mesh, wl.order, wl.species, nb)
    r, z = ctx.dof_coords()
    f1 = inputs.nodal_f(wl, r, z)
    f = np.stack([f1 * (1.0 - 0.1 * b) for b in range(nb)]).reshape(nb, -1)
    band = _factored(gpu, torch, ctx, f, nb)
    rhs_a = torch.from_numpy(np.cos(0.37 * np.arange(nb * ctx.S * ctx.n)).reshape(nb, ctx.S * ctx.n) + 2.0).cuda()
    rhs_b = torch.from_numpy(np.sin(0.11 * np.arange(2 * ctx.S * ctx.n)).reshape(2, ctx.S * ctx.n) - 0.5).cuda()
    ref_a, ref_b = torch.zeros_like(rhs_a), torch.zeros_like(rhs_b)
    ctx.band_solve_batched(band, rhs_a, ref_a)
    ctx.band_solve_batched(band, rhs_b, ref_b)
    x_a = torch.full_like(rhs_a, float("nan"))
    x_b = rhs_b.clone()
    ctx.band_solve_static(band, rhs_a, x_a)            # first call: three problems, out of place
    ctx.band_solve_static(band, x_b, x_b)              # second call, straight after: two problems, in place
    torch.cuda.synchronize()
    assert bool(torch.isfinite(x_a).all()) and bool(torch.isfinite(x_b).all())
    assert _rel(x_a, ref_a) <= RTOL and _rel(x_b, ref_b) <= RTOL
    x_a2 = torch.full_like(rhs_a, float("nan"))
    ctx.band_solve_static(band, rhs_a, x_a2)           # and again the first: bitwise what it gave before
    assert torch.equal(x_a2, x_a)
    ctx.destroy()

    wl = inputs.config(6)                               # ten species, 80 Q3 cells (n = 745): 20 matrices
    nb = 2
    ctx = gpu.LandauContext(wl.mesh, wl.order, wl.species, nb)
    r, z = ctx.dof_coords()
    f1 = inputs.nodal_f(wl, r, z)
    f = np.stack([f1, 0.9 * f1]).reshape(nb, -1)
    band = _factored(gpu, torch, ctx, f, nb)
    rhs = torch.from_numpy(np.cos(0.23 * np.arange(nb * ctx.S * ctx.n)).reshape(nb, ctx.S * ctx.n) + 1.5).cuda()
    ref, x = torch.zeros_like(rhs), torch.full_like(rhs, float("nan"))
    ctx.band_solve_batched(band, rhs, ref)
    ctx.band_solve_static(band, rhs, x)
    assert _rel(x, ref) <= RTOL
    ctx.destroy()


def test_static_scratch_solve_on_several_grids(gpu):
    """Two grids (species on grids of different extent): each grid's solve uses the scratch from its start, one after
    the other on the stream; equal to the existing path, on two calls in a row."""
    import torch
    name, order, meshes, spc, sgrid, comps = inputs.multigrid_case("scaled")
    nb = 2
    ctx = gpu.LandauMultigridContext(meshes, sgrid, order, spc, nb)
    fl = []
    for a, c in enumerate(comps):
        r, z = ctx.grid_dof_coords(sgrid[a])
        fl.append(inputs.maxwellian(float(spc.mass[a]), c.n, c.T, c.zs, r, z))
    f1 = np.concatenate(fl)
    f = np.stack([f1, 0.7 * f1])
    band = _factored(gpu, torch, ctx, f, nb)
    for seed in (0.31, 0.53):
        rhs = torch.from_numpy(np.cos(seed * np.arange(nb * ctx.f_stride)).reshape(nb, ctx.f_stride) + 2.0).cuda()
        ref, x = torch.zeros_like(rhs), torch.full_like(rhs, float("nan"))
        ctx.band_solve_batched(band, rhs, ref)
        ctx.band_solve_static(band, rhs, x)
        assert bool(torch.isfinite(x).all()) and _rel(x, ref) <= RTOL
    ctx.destroy()


def test_static_scratch_limit_is_an_error_not_an_overrun(gpu):
    """nb * S * n beyond LANDAU_STATIC_SCRATCH_DOUBLES (4 Mi doubles = 32 MiB) is refused with LANDAU_EINVAL and the sizes
    in the message, before anything is launched (x stays untouched); the largest batch that fits is accepted."""
    import torch
    wl = inputs.config(3, variant="A")
    cap = gpu.LANDAU_STATIC_SCRATCH_DOUBLES
    assert cap == 4 << 20
    ctx0 = gpu.LandauContext(wl.mesh, wl.order, wl.species, 1)
    per = ctx0.S * ctx0.n
    ctx0.destroy()
    nb_fit = cap // per
    ctx = gpu.LandauContext(wl.mesh, wl.order, wl.species, nb_fit + 1)
    assert ctx.S * ctx.n == per
    ws = ctx.band_sizes()[2]
    rhs = torch.ones((nb_fit + 1, per), dtype=torch.float64, device="cuda")
    x = torch.full_like(rhs, -7.0)
    dummy = torch.zeros(16, dtype=torch.float64, device="cuda")       # never read: the call is refused first
    with pytest.raises(gpu.LandauError) as ei:
        ctx.band_solve_static(dummy, rhs, x)
    assert ei.value.code == gpu.LANDAU_EINVAL
    assert "exceed the static scratch" in str(ei.value) and str((nb_fit + 1) * per) in str(ei.value)
    torch.cuda.synchronize()
    assert bool((x == -7.0).all())
    # exactly nb_fit problems are accepted (one factored problem's workspace repeated: ~12 GB), through both paths
    f = inputs.nodal_f(wl, *ctx.dof_coords()).reshape(1, -1)
    band1 = _factored(gpu, torch, ctx, f, 1)
    nbs = nb_fit
    assert nbs * per <= cap < (nbs + 1) * per
    band = band1.repeat(nbs)
    assert band.numel() == nbs * ws
    ref, xs = torch.zeros_like(rhs[:nbs]), torch.zeros_like(rhs[:nbs])
    ctx.band_solve_batched(band, rhs[:nbs], ref)
    ctx.band_solve_static(band, rhs[:nbs], xs)
    assert _rel(xs, ref) <= RTOL
    ctx.destroy()
