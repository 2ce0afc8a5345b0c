"""Operator-level pins of the CPU oracle: invariants the paper states (exact conservation, L17;
species-uncoupled Jacobian, L75; N = Ne*Nq, Table I) and those the mathematics fixes."""
import math
import os

import numpy as np
import pytest

from paper_2104_10000_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    return [ln.split("#")[0].split() for ln in open(os.path.join(GOLD, name)) if ln.split("#")[0].split()]


@pytest.fixture(scope="module")
def built(oracle):
    """cfg0 (refined Q2, hanging nodes, 2 species) and a refined Q3 3-species case, built once."""
    out = {}
    wl = inputs.config(0)
    sp = oracle.build_space(wl.mesh, wl.order)
    f = inputs.nodal_f(wl, sp.dof_r, sp.dof_z)
    out["q2"] = (wl, sp, f) + tuple(oracle.build_all(wl.mesh, wl.order, wl.species, f, 1.0)[1:])
    mesh = inputs.mesh_quadtree(0.0, 4.0, -4.0, 4.0, 2, 4, 1.0, 2, 2.0, 1)
    spc = inputs._sp([(1, -1, 1, 1), (3670, 1, 0.5, 1), (7344, 2, 0.25, 1)])
    comps = [[inputs.Component(0, 1, 1), inputs.Component(0, 0.05, 2.0, 0.7), inputs.Component(1, 0.5, 400.0),
              inputs.Component(2, 0.25, 900.0, -0.2)]]
    wl3 = inputs.Workload("q3-3sp", 3, mesh, spc, comps, 1e-3, 99)
    sp3 = oracle.build_space(mesh, 3)
    f3 = inputs.nodal_f(wl3, sp3.dof_r, sp3.dof_z)
    out["q3"] = (wl3, sp3, f3) + tuple(oracle.build_all(mesh, 3, spc, f3, 1.0)[1:])
    return out


@pytest.mark.parametrize("key", ["q2", "q3"])
def test_discrete_conservation_of_density_momentum_energy(built, key):
    """the discretisation conserves density, momentum and energy exactly:
    1^T C_a = 0 for every a;  sum_a m_a z^T C_a = 0;  sum_a m_a (v^2/2)^T C_a = 0
    (nodal interpolants of 1, z, r^2+z^2 lie in Q2/Q3 and survive the constraints)."""
    wl, sp, f, vals, Cf, mv = built[key]
    m = wl.species.mass
    S = wl.species.S
    for a in range(S):
        assert abs(Cf[a].sum()) <= 1e-13 * np.abs(Cf[a]).sum()
    for psi in (sp.dof_z, 0.5 * (sp.dof_r ** 2 + sp.dof_z ** 2)):
        num = abs(sum(m[a] * (psi @ Cf[a]) for a in range(S)))
        den = sum(m[a] * np.abs(psi * Cf[a]).sum() for a in range(S))
        assert num <= 1e-13 * den
    # a single species alone does NOT conserve momentum/energy when others are present: the pin bites
    assert abs(sp.dof_z @ Cf[0]) > 1e-6 * np.abs(sp.dof_z * Cf[0]).sum()


@pytest.mark.parametrize("key", ["q2", "q3"])
def test_jacobian_column_sums_vanish_and_Jf_equals_Cf(built, oracle, key):
    wl, sp, f, vals, Cf, mv = built[key]
    rows = np.repeat(np.arange(sp.n), np.diff(sp.rowptr))
    for a in range(wl.species.S):
        colsum = np.zeros(sp.n)
        np.add.at(colsum, sp.colidx, vals[a])
        assert np.abs(colsum).max() <= 1e-12 * np.abs(vals[a]).max()      # sum_a grad psi_a = 0
        Jf = np.zeros(sp.n)
        np.add.at(Jf, rows, vals[a] * f[a, sp.colidx])
        # frozen-coefficient Jacobian applied to f reproduces C(f) (computed independently)
        assert np.abs(Jf - Cf[a]).max() <= 1e-11 * np.abs(Cf[a]).max()


def test_mass_matrix(built, oracle):
    wl, sp, f, vals, Cf, mv = built["q3"]
    # sum of all entries = shift * 2 pi int r dr dz = shift * pi R^2 Lz
    assert abs(mv.sum() - math.pi * 4.0 ** 2 * 8.0) < 1e-12 * mv.sum()
    assert abs(oracle.mass(sp, 2.5).sum() - 2.5 * mv.sum()) < 1e-12 * mv.sum()
    rows = np.repeat(np.arange(sp.n), np.diff(sp.rowptr))
    M = np.zeros((sp.n, sp.n)); M[rows, sp.colidx] = mv
    assert np.abs(M - M.T).max() < 1e-14 * np.abs(M).max()
    # 1^T M f = density of the interpolated Maxwellian (electrons: n = 1.05), to discretisation error
    assert abs(np.ones(sp.n) @ M @ f[0] - 1.05) < 2e-2
    wl1 = inputs.config(1)
    sp1 = oracle.build_space(wl1.mesh, 2)
    assert abs(oracle.mass(sp1, 1.0).sum() - 785.3981633974483) < 1e-10   # pi * 25 * 10


@pytest.mark.parametrize("p", [2, 3])
def test_constraints_reproduce_polynomials(oracle, p):
    """A global polynomial of degree <= p in each variable set on the free DOFs is reproduced
    exactly at every integration point (including through chained hanging nodes)."""
    mesh = inputs.mesh_config3("A") if p == 3 else inputs.config(0).mesh
    sp = oracle.build_space(mesh, p)
    assert sp.n_constrained > 0
    poly = lambda r, z: 1 + 0.3 * r - 0.7 * z + 0.2 * r ** p * z ** p - 0.11 * r ** (p - 1) * z + 0.05 * z ** p
    dpr = lambda r, z: 0.3 + 0.2 * p * r ** (p - 1) * z ** p - 0.11 * (p - 1) * r ** (p - 2) * z
    dpz = lambda r, z: -0.7 + 0.2 * p * r ** p * z ** (p - 1) - 0.11 * r ** (p - 1) + 0.05 * p * z ** (p - 1)
    fq, dfr, dfz = oracle.fields_at_points(sp, poly(sp.dof_r, sp.dof_z)[None, :])
    sc = np.abs(fq).max()
    assert np.abs(fq[0] - poly(sp.r, sp.z)).max() < 1e-12 * sc
    assert np.abs(dfr[0] - dpr(sp.r, sp.z)).max() < 1e-11 * sc
    assert np.abs(dfz[0] - dpz(sp.r, sp.z)).max() < 1e-11 * sc


def test_hanging_weights_golden(oracle):
    for row in _rows("hanging_weights.txt"):
        p, xi, w = int(row[0]), float(row[1]), np.array(row[2:], dtype=float)
        val, _ = oracle.lagrange_1d(p, [xi])
        assert np.allclose(val[0], w, atol=1e-15)


def test_sizes_and_patterns(oracle):
    """n = prod(p n_d + 1), nnz(A1) = prod[2(p+1) + (n_d-1)(2p+1) + n_d (p-1)(p+1)] on uniform
    tensor meshes (1-D Lagrange connectivity counted by hand); N = Ne*Nq (Table I)."""
    for k, n, nnz, N in ((1, 231, 3321, 450), (2, 1225, 29161, 2048)):
        wl = inputs.config(k)
        sp = oracle.build_space(wl.mesh, wl.order)
        assert (sp.n, sp.nnz, sp.N) == (n, nnz, N)
        assert sp.n_constrained == 0
        assert np.all(np.diff(sp.dof_z) >= 0)
    for grids, cells, Npaper in _rows("table1_counts.txt"):
        assert int(grids) * int(cells) * 16 == int(Npaper)
    sp = oracle.build_space(inputs.mesh_config3("B"), 3)
    assert (sp.Ne, sp.N) == (308, 4928)
    for i in range(sp.n):   # columns ascending, diagonal present
        cols = sp.colidx[sp.rowptr[i]:sp.rowptr[i + 1]]
        assert np.all(np.diff(cols) > 0) and i in cols


def test_linearity_scaling_and_species_permutation(oracle):
    wl = inputs.config(0)
    sp = oracle.build_space(wl.mesh, wl.order)
    f = inputs.nodal_f(wl, sp.dof_r, sp.dof_z)
    spc = wl.species
    v1 = oracle.jacobian(sp, spc, f)
    # J is linear in f (frozen coefficients are linear functionals of f)
    v2 = oracle.jacobian(sp, spc, 3.0 * f)
    assert np.abs(v2 - 3.0 * v1).max() <= 1e-13 * np.abs(v2).max()
    # J scales with nu
    spn = inputs.Species(spc.mass, spc.charge, spc.density, spc.temperature, spc.m0, 2.0)
    assert np.abs(oracle.jacobian(sp, spn, f) - 2.0 * v1).max() <= 1e-13 * np.abs(v1).max()
    # permuting species permutes the diagonal blocks
    spp = inputs.Species(spc.mass[::-1].copy(), spc.charge[::-1].copy(), spc.density[::-1].copy(), spc.temperature[::-1].copy())
    vp = oracle.jacobian(sp, spp, f[::-1].copy())
    for a in range(2):
        assert np.abs(vp[1 - a] - v1[a]).max() <= 1e-13 * np.abs(v1[a]).max()
    # m0 is arbitrary (L42) only up to the overall nu normalisation: doubling m0 scales K by 2*2, D by 4
    # -> J scales by 4 (nu_ab carries 1/m0^2 in physical units; here nu is held fixed)
    sp2 = inputs.Species(spc.mass, spc.charge, spc.density, spc.temperature, 2.0, 1.0)
    assert np.abs(oracle.jacobian(sp, sp2, f) - 4.0 * v1).max() <= 1e-13 * 4 * np.abs(v1).max()


def test_double_and_long_double_instantiations_agree(oracle):
    wl = inputs.config(1)
    sp = oracle.build_space(wl.mesh, wl.order)
    f = inputs.nodal_f(wl, sp.dof_r, sp.dof_z)
    a = oracle.jacobian(sp, wl.species, f, "ld")
    b = oracle.jacobian(sp, wl.species, f, "d")
    assert np.abs(a - b).max() <= 1e-12 * np.abs(a).max()


def test_advection_term_and_implicit_operator_pins(built, oracle):
    """E-field term of Eq. 4 (L52) and the implicit-step operator shift M + A - J.
    Pins: d(const)/dz = 0 (row sums); psi = 1 against f = z gives the exact integral
    (e/m) E_z 2 pi int r dr dz; integration by parts against z for a distribution that vanishes on
    the z boundaries gives minus the density moment (the force on the species); the residual from
    the weak form equals the matrix applied to f; the operator is affine in shift and E_z."""
    wl, sp, f, vals, Cf, mv = built["q3"]
    spc = wl.species
    Ez, shift = 0.37, 2.5
    A = oracle.advection(sp, spc, Ez)
    S = spc.S
    R, L = wl.mesh.rmax, wl.mesh.zmax - wl.mesh.zmin
    M1 = oracle.mass(sp, 1.0)
    rows = np.repeat(np.arange(sp.n), np.diff(sp.rowptr))
    Md = np.zeros((sp.n, sp.n)); Md[rows, sp.colidx] = M1
    for a in range(S):
        fac = spc.charge[a] * spc.m0 / spc.mass[a] * Ez
        assert np.abs(A[a].sum(axis=1)).max() <= 1e-12 * np.abs(A[a]).max()            # A 1 = 0
        assert abs(np.ones(sp.n) @ A[a] @ sp.dof_z - fac * math.pi * R * R * L) <= 1e-11 * abs(fac) * math.pi * R * R * L
        # z in the FE space: A z = fac * M 1 exactly
        assert np.abs(A[a] @ sp.dof_z - fac * (Md @ np.ones(sp.n))).max() <= 1e-11 * abs(fac) * np.abs(Md).max() * 10
    # integration by parts with the electron distribution (e^{-16} at the z boundary, 4 thermal speeds)
    fe = inputs.maxwellian(1.0, 1.0, 1.0, 0.0, sp.dof_r, sp.dof_z)
    dens = np.ones(sp.n) @ Md @ fe
    assert abs(dens - 1.0) < 1e-2                      # int f d^3v = n (coarse Q3 interpolant, cut at 4 v_th)
    force = sp.dof_z @ A[0] @ fe
    assert abs(force + spc.charge[0] * Ez * dens) < 1e-5 * abs(Ez)    # exact for f_h up to the boundary term
    assert abs(np.ones(sp.n) @ A[0] @ fe) < 1e-5 * abs(Ez)                            # no density change
    # the operator: residual from the weak form == matrix applied to f; affine in (shift, Ez)
    ov, F = oracle.implicit_operator(sp, spc, f, Ez, shift)
    for a in range(S):
        V = np.zeros((sp.n, sp.n)); V[rows, sp.colidx] = ov[a]
        lhs = V @ f[a]
        rhs = shift * (Md @ f[a]) + F[a]
        assert np.abs(lhs - rhs).max() <= 1e-11 * np.abs(lhs).max()
        assert np.abs(ov[a] - (shift * M1 + A[a][rows, sp.colidx] - vals[a])).max() <= 1e-13 * np.abs(ov[a]).max()
    ov0, F0 = oracle.implicit_operator(sp, spc, f, 0.0, 0.0)
    assert np.abs(ov0 + vals).max() <= 1e-13 * np.abs(vals).max() and np.abs(F0 + Cf).max() <= 1e-13 * np.abs(Cf).max()


def _grid20():
    return inputs.mesh_quadtree(0.0, 5.0, -5.0, 5.0, 2, 4, 1.0, 2, 2.5, 1)


def test_paper_vertex_count_of_the_20_cell_grid(oracle):
    """the 20-cell Q3 grid of Fig. 3 has 193 unconstrained vertices (pins the hanging-node
    constraint counting); Table I: three such grids give N = 960 points and 10 x 193 = 1,930 equations."""
    (cells, order, n), = _rows("vertex_counts.txt")
    sp = oracle.build_space(_grid20(), int(order))
    assert (sp.Ne, sp.n) == (int(cells), int(n))
    assert 3 * sp.N == 960 and 10 * sp.n == 1930


def _scaled(mesh, k):
    return inputs.Mesh(mesh.rmin * k, mesh.rmax * k, mesh.zmin * k, mesh.zmax * k, mesh.nbr, mesh.nbz, mesh.level, mesh.ir, mesh.iz)


def test_multigrid_equals_single_grid_on_identical_meshes_and_conserves(oracle):
    """Section III-C (L179-206).  (1) Two species on two IDENTICAL grids give the single-grid result (every
    cross-grid coincident pair is skipped exactly like j = i).  (2) Species on grids of different extent:
    density per species, total z-momentum and total energy are conserved exactly (z and r^2+z^2 lie in
    every grid's space)."""
    wl = inputs.config(0)
    sp = oracle.build_space(wl.mesh, wl.order)
    f = inputs.nodal_f(wl, sp.dof_r, sp.dof_z)
    _, vals, Cf, mv = oracle.build_all(wl.mesh, wl.order, wl.species, f, 1.3)
    _, mvals, mCf, mm = oracle.build_all_multigrid([wl.mesh, wl.mesh], wl.order, wl.species, [0, 1], [f[0], f[1]], 1.3)
    for a in range(2):
        assert np.abs(mvals[a] - vals[a]).max() <= 1e-13 * np.abs(vals[a]).max()
        assert np.abs(mCf[a] - Cf[a]).max() <= 1e-13 * np.abs(Cf[a]).max()
        assert np.array_equal(mm[a], mv)
    # three species, two grids of different extent (electron grid, ion grid 8x smaller: v_th ratio)
    spc = inputs._sp([(1, -1, 1, 1), (64, 1, 0.6, 1), (128, 2, 0.2, 1)])
    g0 = inputs.mesh_quadtree(0.0, 4.0, -4.0, 4.0, 2, 4, 1.0, 2, 2.0, 1)
    g1 = _scaled(g0, 0.125)
    grids = [0, 1, 1]
    spaces = [oracle.build_space(g, 2) for g in (g0, g1)]
    fl = []
    for a in range(3):
        s_ = spaces[grids[a]]
        fa = inputs.maxwellian(spc.mass[a], spc.density[a], 1.0, 0.02 * a, s_.dof_r, s_.dof_z)
        fl.append(fa * (1.0 + 1e-3 * np.cos(7.0 * np.arange(s_.n))))
    _, v, C, _ = oracle.build_all_multigrid([g0, g1], 2, spc, grids, fl, 1.0)
    for a in range(3):
        assert abs(C[a].sum()) <= 1e-13 * np.abs(C[a]).sum()
    for psi in (lambda s_: s_.dof_z, lambda s_: 0.5 * (s_.dof_r ** 2 + s_.dof_z ** 2)):
        num = abs(sum(spc.mass[a] * (psi(spaces[grids[a]]) @ C[a]) for a in range(3)))
        den = sum(spc.mass[a] * np.abs(psi(spaces[grids[a]]) * C[a]).sum() for a in range(3))
        assert num <= 1e-12 * den
    assert abs(spaces[0].dof_z @ C[0]) > 1e-6 * np.abs(spaces[0].dof_z * C[0]).sum()   # the pin bites


def test_linear_solve_pins(built, oracle):
    """Section III-G (L169-175): per-species solve of the implicit step.  Pins: M x = M 1 gives x = 1;
    the outer-product band LU (Alg. 4.3.1) reproduces A = L U with no fill outside the band and its
    triangular solves agree with the library solve and with scipy's banded solver; a manufactured solution."""
    import scipy.linalg
    wl, sp, f, vals, Cf, mv = built["q2"]
    ov, F = oracle.implicit_operator(sp, wl.species, f, 0.2, 3.0)
    M = oracle.dense_from_csr(sp, oracle.mass(sp, 1.0))
    assert np.abs(oracle.solve_species(sp, oracle.mass(sp, 1.0), M @ np.ones(sp.n)) - 1.0).max() < 1e-12
    for a in range(wl.species.S):
        A = oracle.dense_from_csr(sp, ov[a])
        rows, cols = np.nonzero(A)
        p = int((rows - cols).max()); q = int((cols - rows).max())
        LU = oracle.band_lu_outer_product(A, p, q)
        L = np.tril(LU, -1) + np.eye(sp.n); U = np.triu(LU)
        assert np.abs(L @ U - A).max() <= 1e-13 * np.abs(A).max()
        ii, jj = np.nonzero(LU)
        assert (ii - jj).max() <= p and (jj - ii).max() <= q                # no fill outside the band
        xs = np.cos(np.arange(sp.n) * 0.37) + 2.0                            # manufactured solution
        b = A @ xs
        x = oracle.solve_species(sp, ov[a], b)
        cond = np.linalg.cond(A)
        assert np.abs(x - xs).max() <= 50 * cond * 2.2e-16 * np.abs(xs).max()
        y = scipy.linalg.solve_triangular(L, b, lower=True, unit_diagonal=True)
        x2 = scipy.linalg.solve_triangular(U, y)
        assert np.abs(x2 - x).max() <= 50 * cond * 2.2e-16 * np.abs(x).max()
        ab = np.zeros((p + q + 1, sp.n))
        for i, j in zip(rows, cols):
            ab[q + i - j, j] = A[i, j]
        x3 = scipy.linalg.solve_banded((p, q), ab, b)
        assert np.abs(x3 - x).max() <= 50 * cond * 2.2e-16 * np.abs(x).max()
