"""CPU ORACLE for the Landau Jacobian hot path -- test infrastructure, NOT the product path.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module.  It shares no code with
``paper_2104_10000_b200/csrc`` or its Python binding and imports neither.

What it computes (PAPER.md = /root/reference/PAPER.md, arxiv 2104.10000):

* the conservative finite-element Landau operator in axisymmetric (r,z) velocity space,
  weak form Eqs. 4-8 (L52-67), with the frozen-coefficient Jacobian of L75, following
  Algorithm 1 (L109-131) step by step: inner integral (lines 3-12, in ``landau_pair.c``),
  species scaling (13-16), transform to the reference basis (18-20), element matrix
  (Transform&Assemble, line 23), assembly with hanging-node interpolation (L101, L297);
* C(f), the weak-form residual (right-hand side of Eq. 4 without E-field and source),
  evaluated DIRECTLY from Eqs. 5-6 at f -- not as J f, so that J f = C(f) is a test;
* the scaled mass matrix (L280);
* the E-field advection term on the left of Eq. 4 (L52) and the operator of a fully implicit step,
  shift M + A_a - J_a with its residual A_a f_a - C_a(f);
* the same operator with species clustered on several grids (section III-C, Table I; NEXT-2);
* the per-species linear solve of the implicit step (section III-G; NEXT-4).

Everything outside the O(N^2) pair loop is plain numpy in fp64 with dense matrices (no
blocking, no gather lists).  The pair loop is plain C in long double (``_ld``) for parity and
double (``_d``) for the timed CPU baseline.

Readings of the paper where it is silent or garbled are DESIGN.md's Q1-Q13; each is marked
where it is used.  Conventions shared with include/landau.h (they are part of the problem
statement, not code): cell/point/DOF/CSR orderings described in ``Space``.

Parity pins: tests/test_oracle_pins.py (elliptic closed forms, Legendre relation, brute-force
azimuthal quadrature of Eq. 3, Rosenbluth potentials of a Maxwellian, exact discrete
conservation, column sums, J f = C(f), mass integrals, constraint polynomial reproduction,
Table I counting; for the advection term: zero row sums, exact integral of d(z)/dz, integration by
parts against z for a distribution that vanishes on the boundary, vals f = shift M f + F).  Numerical values of individual Jacobian entries are "parity unpinned" by
the paper (it prints none); they are pinned only through those invariants.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBS: dict = {}


def build(force: bool = False) -> None:
    """Compile landau_pair.c twice with gcc: long double (parity) and double (timing)."""
    src = os.path.join(_HERE, "landau_pair.c")
    for tag, flag in (("ld", "-DREAL_LD"), ("d", "")):
        out = os.path.join(_HERE, f"liboracle_pair_{tag}.so")
        if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
            cmd = ["gcc", "-O2", "-fPIC", "-shared", "-fopenmp", "-std=c99", src, "-o", out, "-lm"]
            if flag:
                cmd.insert(1, flag)
            subprocess.check_call(cmd)


def _lib(tag: str):
    if tag not in _LIBS:
        build()
        lib = ctypes.CDLL(os.path.join(_HERE, f"liboracle_pair_{tag}.so"))
        dp = ctypes.POINTER(ctypes.c_double)
        getattr(lib, f"oracle_ellip_{tag}").argtypes = [ctypes.c_double, dp]
        getattr(lib, f"oracle_tensor2d_{tag}").argtypes = [ctypes.c_double] * 4 + [dp, dp]
        getattr(lib, f"oracle_inner_integral_{tag}").argtypes = (
            [ctypes.c_int, ctypes.c_int] + [dp] * 8 + [ctypes.c_int, ctypes.c_int] + [dp, dp])
        for n in ("ellip", "tensor2d", "inner_integral"):
            getattr(lib, f"oracle_{n}_{tag}").restype = None
        _LIBS[tag] = lib
    return _LIBS[tag]


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def ellip_KEDS(m: float, precision: str = "ld"):
    """(K, E, D, S)(m), parameter convention; D=(K-E)/m, S=int sin^2 cos^2 (1-m sin^2)^(-3/2)."""
    out = np.zeros(4)
    getattr(_lib(precision), f"oracle_ellip_{precision}")(float(m), _p(out))
    return tuple(out)


def tensor2d(r, z, rb, zb, precision: str = "ld"):
    """U^D = (rr, rz, zz) and U^K = [[r rb, r zb], [z rb, z zb]] (reading Q1)."""
    ud, uk = np.zeros(3), np.zeros(4)
    getattr(_lib(precision), f"oracle_tensor2d_{precision}")(float(r), float(z), float(rb), float(zb), _p(ud), _p(uk))
    return ud, uk.reshape(2, 2)


def inner_integral(r, z, w, f, dfr, dfz, e2, m0m, rows=None, precision: str = "ld"):
    """Alg. 1 lines 3-12 (L114-121) for rows [rows[0], rows[1]) (default all).

    Returns GD[N][3] = (rr,rz,zz), GK[N][2]; rows outside the range are left zero.
    """
    N, S = r.shape[0], f.shape[0]
    arrs = [np.ascontiguousarray(a, dtype=np.float64) for a in (r, z, w, f, dfr, dfz, e2, m0m)]
    GD, GK = np.zeros((N, 3)), np.zeros((N, 2))
    i0, i1 = (0, N) if rows is None else rows
    getattr(_lib(precision), f"oracle_inner_integral_{precision}")(
        N, S, *[_p(a) for a in arrs], int(i0), int(i1), _p(GD), _p(GK))
    return GD, GK


# --------------------------------------------------------------------------------------------
# Finite-element space on a 2:1 face-balanced quadtree forest
# --------------------------------------------------------------------------------------------

def lagrange_1d(p: int, x):
    """Values and derivatives of the p+1 Lagrange polynomials on EQUISPACED nodes of [-1,1]
    (reading Q7) at the points x.  Returns (val[len(x)][p+1], der[len(x)][p+1])."""
    x = np.atleast_1d(np.asarray(x, dtype=np.float64))
    nodes = np.linspace(-1.0, 1.0, p + 1)
    val = np.ones((x.shape[0], p + 1))
    der = np.zeros((x.shape[0], p + 1))
    for a in range(p + 1):
        for b in range(p + 1):
            if b != a:
                val[:, a] *= (x - nodes[b]) / (nodes[a] - nodes[b])
        for c in range(p + 1):
            if c == a:
                continue
            term = np.full(x.shape[0], 1.0 / (nodes[a] - nodes[c]))
            for b in range(p + 1):
                if b != a and b != c:
                    term *= (x - nodes[b]) / (nodes[a] - nodes[b])
            der[:, a] += term
    return val, der


@dataclass
class Space:
    """Discrete space + quadrature for one mesh and one order p (2 or 3).

    Orderings (the problem statement shared with include/landau.h):
      * cells in the order of the mesh's leaf list;
      * integration point gi = e*Nq + qz*(p+1) + qr, tensor Gauss-Legendre, abscissae ascending;
      * local basis a = az*(p+1) + ar on equispaced nodes;
      * unconstrained DOFs numbered by ascending (z, r) lattice coordinate of their node;
      * CSR pattern A1: rows in DOF order, columns ascending; entry (a,b) present iff some cell
        has both a and b among the free DOFs its (constrained) local nodes depend on.
    """

    p: int
    Ne: int
    Nq: int
    Nb: int
    N: int
    n: int
    r: np.ndarray          # [N]
    z: np.ndarray          # [N]
    w_in: np.ndarray       # [N]  omega * detJ * r               (Eqs. 7-8, no 2 pi)   reading Q2
    w_out: np.ndarray      # [N]  2 pi * omega * detJ * r        (Eq. 4)               reading Q2
    invJ: np.ndarray       # [Ne][2] diagonal of J^{-1} = (2/hr, 2/hz)
    B: np.ndarray          # [Nq][Nb]   psi_a(x_q)
    E: np.ndarray          # [Nq][Nb][2] reference gradient of psi_a at x_q
    cell_dofs: list        # per cell: int array of the distinct free DOFs it touches (ascending)
    cell_P: list           # per cell: dense [Nb][len(cell_dofs)] interpolation matrix P_e
    dof_r: np.ndarray      # [n]
    dof_z: np.ndarray      # [n]
    rowptr: np.ndarray     # [n+1] int32
    colidx: np.ndarray     # [nnz] int32
    n_constrained: int

    @property
    def nnz(self) -> int:
        return int(self.colidx.shape[0])


def build_space(mesh, p: int) -> Space:
    """mesh: any object with rmin,rmax,zmin,zmax,nbr,nbz,level,ir,iz (the landau_mesh fields)."""
    assert p in (2, 3)
    level = np.asarray(mesh.level, dtype=np.int64)
    ir = np.asarray(mesh.ir, dtype=np.int64)
    iz = np.asarray(mesh.iz, dtype=np.int64)
    Ne = level.shape[0]
    Lmax = int(level.max())
    leaves = {(int(level[e]), int(ir[e]), int(iz[e])): e for e in range(Ne)}
    hr0 = (mesh.rmax - mesh.rmin) / mesh.nbr
    hz0 = (mesh.zmax - mesh.zmin) / mesh.nbz
    npl = p + 1

    # --- node lattice: unit = node spacing of a level-Lmax cell -----------------------------
    def cell_nodes(e):
        """lattice coords (R,Z) of the local nodes a = az*(p+1)+ar of cell e."""
        H = 1 << (Lmax - int(level[e]))
        out = []
        for az in range(npl):
            for ar in range(npl):
                out.append((int(ir[e]) * p * H + ar * H, int(iz[e]) * p * H + az * H))
        return out

    # --- hanging nodes (reading Q8): nodes of a fine edge whose face neighbour is one level
    # coarser take the coarse edge's 1-D Lagrange interpolant; coincident nodes are shared.
    nodes1d = np.arange(npl, dtype=np.float64)

    def lag_weights(t):
        wts = np.ones(npl)
        for a in range(npl):
            for b in range(npl):
                if b != a:
                    wts[a] *= (t - nodes1d[b]) / (nodes1d[a] - nodes1d[b])
        return wts

    constraint = {}  # node -> list of (parent node, weight)
    for e in range(Ne):
        l, i, j = int(level[e]), int(ir[e]), int(iz[e])
        if l == 0:
            continue
        H = 1 << (Lmax - l)
        Hc = 2 * H
        for (di, dj) in ((-1, 0), (1, 0), (0, -1), (0, 1)):
            ni, nj = i + di, j + dj
            if ni < 0 or nj < 0 or ni >= (mesh.nbr << l) or nj >= (mesh.nbz << l):
                continue
            if (l, ni, nj) in leaves:
                continue
            par = (l - 1, ni >> 1, nj >> 1)
            if par not in leaves:
                continue  # neighbour is finer (or same-level subdivided): not our constraint
            I, J = par[1], par[2]
            for a in range(npl):
                if di != 0:   # edge of constant R; runs along z
                    R = (i + (1 if di > 0 else 0)) * p * H
                    Z = j * p * H + a * H
                    t = (Z - J * p * Hc) / Hc
                    parents = [(R, J * p * Hc + b * Hc) for b in range(npl)]
                else:         # edge of constant Z; runs along r
                    Z = (j + (1 if dj > 0 else 0)) * p * H
                    R = i * p * H + a * H
                    t = (R - I * p * Hc) / Hc
                    parents = [(I * p * Hc + b * Hc, Z) for b in range(npl)]
                if abs(t - round(t)) < 1e-12:
                    continue  # coincides with a coarse node
                wts = lag_weights(t)
                constraint[(R, Z)] = [(parents[b], float(wts[b])) for b in range(npl)]

    # --- closure of chained constraints ------------------------------------------------------
    def resolve(node, depth=0):
        assert depth < 64
        if node not in constraint:
            return {node: 1.0}
        acc = {}
        for (par, wt) in constraint[node]:
            for (nd, w2) in resolve(par, depth + 1).items():
                acc[nd] = acc.get(nd, 0.0) + wt * w2
        return acc

    all_nodes = set()
    for e in range(Ne):
        all_nodes.update(cell_nodes(e))
    free = sorted((nd for nd in all_nodes if nd not in constraint), key=lambda t: (t[1], t[0]))
    dof_of = {nd: k for k, nd in enumerate(free)}
    n = len(free)
    unit_r = hr0 / (p * (1 << Lmax))
    unit_z = hz0 / (p * (1 << Lmax))
    dof_r = np.array([mesh.rmin + nd[0] * unit_r for nd in free])
    dof_z = np.array([mesh.zmin + nd[1] * unit_z for nd in free])

    cell_dofs, cell_P = [], []
    for e in range(Ne):
        rows = [resolve(nd) for nd in cell_nodes(e)]
        dofs = sorted({dof_of[nd] for row in rows for nd in row})
        pos = {d: c for c, d in enumerate(dofs)}
        P = np.zeros((npl * npl, len(dofs)))
        for a, row in enumerate(rows):
            for nd, wt in row.items():
                P[a, pos[dof_of[nd]]] += wt
        cell_dofs.append(np.array(dofs, dtype=np.int64))
        cell_P.append(P)

    # --- quadrature points -----------------------------------------------------------------
    xg, wg = np.polynomial.legendre.leggauss(npl)
    Nq = npl * npl
    N = Ne * Nq
    r = np.zeros(N); z = np.zeros(N); w_in = np.zeros(N); invJ = np.zeros((Ne, 2))
    for e in range(Ne):
        hr, hz = hr0 / (1 << int(level[e])), hz0 / (1 << int(level[e]))
        r0, z0 = mesh.rmin + int(ir[e]) * hr, mesh.zmin + int(iz[e]) * hz
        invJ[e] = (2.0 / hr, 2.0 / hz)
        detJ = hr * hz / 4.0
        for qz in range(npl):
            for qr in range(npl):
                gi = e * Nq + qz * npl + qr
                r[gi] = r0 + 0.5 * (xg[qr] + 1.0) * hr
                z[gi] = z0 + 0.5 * (xg[qz] + 1.0) * hz
                w_in[gi] = wg[qr] * wg[qz] * detJ * r[gi]
    w_out = 2.0 * np.pi * w_in

    # --- tabulations -----------------------------------------------------------------------
    val, der = lagrange_1d(p, xg)
    B = np.zeros((Nq, Nq)); E = np.zeros((Nq, Nq, 2))
    for qz in range(npl):
        for qr in range(npl):
            for az in range(npl):
                for ar in range(npl):
                    q, a = qz * npl + qr, az * npl + ar
                    B[q, a] = val[qr, ar] * val[qz, az]
                    E[q, a, 0] = der[qr, ar] * val[qz, az]
                    E[q, a, 1] = val[qr, ar] * der[qz, az]

    # --- CSR pattern -------------------------------------------------------------------------
    pat = np.zeros((n, n), dtype=bool)
    for dofs in cell_dofs:
        pat[np.ix_(dofs, dofs)] = True
    rows_idx, cols_idx = np.nonzero(pat)
    rowptr = np.zeros(n + 1, dtype=np.int32)
    np.add.at(rowptr, rows_idx + 1, 1)
    rowptr = np.cumsum(rowptr).astype(np.int32)
    return Space(p, Ne, Nq, Nq, N, n, r, z, w_in, w_out, invJ, B, E, cell_dofs, cell_P,
                 dof_r, dof_z, rowptr, cols_idx.astype(np.int32), len(constraint))


# --------------------------------------------------------------------------------------------
# The operator (Algorithm 1; weak form Eqs. 4-8)
# --------------------------------------------------------------------------------------------

def fields_at_points(sp: Space, f: np.ndarray):
    """f_b(q), grad f_b(q) at all integration points (L101): u = P_e f_b, f = B u,
    grad f = J^{-T} (E u).  f: [S][n] -> fq, dfr, dfz: [S][N]."""
    S = f.shape[0]
    fq = np.zeros((S, sp.N)); dfr = np.zeros((S, sp.N)); dfz = np.zeros((S, sp.N))
    for e in range(sp.Ne):
        sl = slice(e * sp.Nq, (e + 1) * sp.Nq)
        for b in range(S):
            u = sp.cell_P[e] @ f[b, sp.cell_dofs[e]]
            fq[b, sl] = sp.B @ u
            dfr[b, sl] = sp.invJ[e, 0] * (sp.E[:, :, 0] @ u)
            dfz[b, sl] = sp.invJ[e, 1] * (sp.E[:, :, 1] @ u)
    return fq, dfr, dfz


def coefficients(sp: Space, species, f: np.ndarray, rows=None, precision: str = "ld"):
    """Alg. 1 lines 3-16: G_D, G_K by the pair loop, then per species (reading Q6: nu_ab =
    nu e_a^2 e_b^2, L83)  K_a = nu e_a^2 (m0/m_a) G_K,  D_a = -nu e_a^2 (m0/m_a)^2 G_D.
    Returns K[S][N][2], D[S][N][2][2], and the raw (GD, GK)."""
    fq, dfr, dfz = fields_at_points(sp, f)
    e2 = np.asarray(species.charge, dtype=np.float64) ** 2
    m0m = species.m0 / np.asarray(species.mass, dtype=np.float64)
    GD, GK = inner_integral(sp.r, sp.z, sp.w_in, fq, dfr, dfz, e2, m0m, rows, precision)
    S = f.shape[0]
    K = np.zeros((S, sp.N, 2)); D = np.zeros((S, sp.N, 2, 2))
    for a in range(S):
        K[a] = species.nu * e2[a] * m0m[a] * GK
        D[a, :, 0, 0] = -species.nu * e2[a] * m0m[a] ** 2 * GD[:, 0]
        D[a, :, 0, 1] = -species.nu * e2[a] * m0m[a] ** 2 * GD[:, 1]
        D[a, :, 1, 0] = D[a, :, 0, 1]
        D[a, :, 1, 1] = -species.nu * e2[a] * m0m[a] ** 2 * GD[:, 2]
    return K, D, (GD, GK)


def element_matrices(sp: Space, K: np.ndarray, D: np.ndarray):
    """Alg. 1 lines 18-23: KK = J^{-1} K w, DD = J^{-1} D J^{-T} w (reading Q5; w = w_out, Q2),
    C_e[a][b] = sum_q ( Ehat_qa . DD_q . Ehat_qb + Ehat_qa . KK_q B_qb ).  -> Ce[S][Ne][Nb][Nb]"""
    S = K.shape[0]
    Ce = np.zeros((S, sp.Ne, sp.Nb, sp.Nb))
    for a in range(S):
        for e in range(sp.Ne):
            Jinv = np.diag(sp.invJ[e])
            for q in range(sp.Nq):
                gi = e * sp.Nq + q
                KK = Jinv @ K[a, gi] * sp.w_out[gi]
                DD = Jinv @ D[a, gi] @ Jinv.T * sp.w_out[gi]
                Eq = sp.E[q]                      # [Nb][2]
                Ce[a, e] += Eq @ DD @ Eq.T + np.outer(Eq @ KK, sp.B[q])
    return Ce


def assemble_dense(sp: Space, Ce_one: np.ndarray) -> np.ndarray:
    """J = sum_e P_e^T C_e P_e (hanging-node interpolation, L101/L297), dense n x n."""
    J = np.zeros((sp.n, sp.n))
    for e in range(sp.Ne):
        P = sp.cell_P[e]
        J[np.ix_(sp.cell_dofs[e], sp.cell_dofs[e])] += P.T @ Ce_one[e] @ P
    return J


def csr_values(sp: Space, Jd: np.ndarray) -> np.ndarray:
    rows = np.repeat(np.arange(sp.n), np.diff(sp.rowptr))
    return Jd[rows, sp.colidx]


def jacobian(sp: Space, species, f: np.ndarray, precision: str = "ld", dense: bool = False):
    """Frozen-coefficient Jacobian (L75): returns vals[S][nnz] on the pattern A1 (block
    diagonal I_S (x) A1) and, if dense, also the dense blocks."""
    K, D, _ = coefficients(sp, species, f, None, precision)
    Ce = element_matrices(sp, K, D)
    S = f.shape[0]
    vals = np.zeros((S, sp.nnz)); dens = []
    for a in range(S):
        Jd = assemble_dense(sp, Ce[a])
        vals[a] = csr_values(sp, Jd)
        if dense:
            dens.append(Jd)
    return (vals, dens) if dense else vals


def collision(sp: Space, species, f: np.ndarray, precision: str = "ld", KD=None):
    """C(f)_a[i] = sum_q w_out grad psi_i . ( K_a f_a + D_a grad f_a ), Eqs. 4-6 with PHYSICAL
    gradients (reading Q10) -- independent of element_matrices()."""
    if KD is None:
        K, D, _ = coefficients(sp, species, f, None, precision)
    else:
        K, D = KD
    fq, dfr, dfz = fields_at_points(sp, f)
    S = f.shape[0]
    Cf = np.zeros((S, sp.n))
    for a in range(S):
        for e in range(sp.Ne):
            ce = np.zeros(sp.Nb)
            for q in range(sp.Nq):
                gi = e * sp.Nq + q
                flux = K[a, gi] * fq[a, gi] + D[a, gi] @ np.array([dfr[a, gi], dfz[a, gi]])
                gradpsi = sp.E[q] * sp.invJ[e][None, :]        # [Nb][2], physical
                ce += sp.w_out[gi] * (gradpsi @ flux)
            Cf[a, sp.cell_dofs[e]] += sp.cell_P[e].T @ ce
    return Cf


def mass(sp: Space, shift: float) -> np.ndarray:
    """Scaled mass matrix (L280): M[a][b] = shift * sum_q w_out psi_a psi_b -> mvals[nnz]."""
    M = np.zeros((sp.n, sp.n))
    for e in range(sp.Ne):
        Me = np.zeros((sp.Nb, sp.Nb))
        for q in range(sp.Nq):
            Me += shift * sp.w_out[e * sp.Nq + q] * np.outer(sp.B[q], sp.B[q])
        P = sp.cell_P[e]
        M[np.ix_(sp.cell_dofs[e], sp.cell_dofs[e])] += P.T @ Me @ P
    return csr_values(sp, M)


def advection(sp: Space, species, Ez: float):
    """E-field term on the left of Eq. 4 (L52): 2 pi int r psi (0, (e_a/m_a) E_z) . grad f, i.e.
    A_a[i][j] = (e_a m0/m_a) E_z sum_q w_out psi_i d(psi_j)/dz  (charges in e, masses in m0, E in the
    units of Appendix A: DESIGN.md reading Q14).  Dense blocks [S][n][n]."""
    S = len(species.mass)
    A1 = np.zeros((sp.n, sp.n))
    for e in range(sp.Ne):
        Ae = np.zeros((sp.Nb, sp.Nb))
        for q in range(sp.Nq):
            dpsi_dz = sp.invJ[e, 1] * sp.E[q, :, 1]
            Ae += sp.w_out[e * sp.Nq + q] * np.outer(sp.B[q], dpsi_dz)
        P = sp.cell_P[e]
        A1[np.ix_(sp.cell_dofs[e], sp.cell_dofs[e])] += P.T @ Ae @ P
    return [float(species.charge[a]) * species.m0 / float(species.mass[a]) * Ez * A1 for a in range(S)]


def implicit_operator(sp: Space, species, f: np.ndarray, Ez: float, shift: float, precision: str = "ld"):
    """What a fully implicit step of Eq. 4 needs about the state f (L75, L280; no source term):
        vals_a = shift M + A_a - J_a(f)        on the pattern A1, [S][nnz]
        F_a    = A_a f_a - C_a(f)              [S][n]  (the residual without the d/dt term)
    F is evaluated from the weak form with physical gradients at the integration points (not as a
    matrix-vector product), so vals f = shift M f + F is a test of both."""
    S = f.shape[0]
    K, D, _ = coefficients(sp, species, f, None, precision)
    Ce = element_matrices(sp, K, D)
    A = advection(sp, species, Ez)
    M1 = mass(sp, shift)
    vals = np.stack([M1 + csr_values(sp, A[a]) - csr_values(sp, assemble_dense(sp, Ce[a])) for a in range(S)])
    Cf = collision(sp, species, f, precision, (K, D))
    _, _, dfz = fields_at_points(sp, f)
    F = np.zeros((S, sp.n))
    for a in range(S):
        fac = float(species.charge[a]) * species.m0 / float(species.mass[a]) * Ez
        for e in range(sp.Ne):
            sl = slice(e * sp.Nq, (e + 1) * sp.Nq)
            fe = sp.B.T @ (sp.w_out[sl] * fac * dfz[a, sl])          # sum_q w psi_i (e/m) E_z df/dz
            F[a, sp.cell_dofs[e]] += sp.cell_P[e].T @ fe
    return vals, F - Cf


def build_all(mesh, order: int, species, f: np.ndarray, shift: float = 1.0, precision: str = "ld"):
    """One full pass of the hot path on the CPU (what bench.py's cpu_baseline times)."""
    sp = build_space(mesh, order)
    K, D, _ = coefficients(sp, species, f, None, precision)
    Ce = element_matrices(sp, K, D)
    vals = np.stack([csr_values(sp, assemble_dense(sp, Ce[a])) for a in range(f.shape[0])])
    Cf = collision(sp, species, f, precision, (K, D))
    return sp, vals, Cf, mass(sp, shift)


# --------------------------------------------------------------------------------------------
# Multiple grids (section III-C, Table I): species clustered by thermal speed
# live on separate meshes; the inner integral of Eqs. 7-8 runs over the UNION of all grids'
# integration points ("overbar terms are evaluated on the grid for the domain of species beta",
# L42), each species contributing only at the points of its own grid.
# --------------------------------------------------------------------------------------------

def build_all_multigrid(meshes, order: int, species, species_grid, f_list, shift: float = 1.0, precision: str = "ld"):
    """species_grid[a] = grid of species a; f_list[a] = nodal values of species a on ITS grid.
    Returns (spaces, vals_list, Cf_list, mass_list): per species CSR values / C(f) on its grid's
    pattern, per grid the scaled mass matrix.  A coincident pair (same location, also when the
    two points belong to different grids) contributes nothing (reading Q3)."""
    spaces = [build_space(m, order) for m in meshes]
    S = len(f_list)
    off = np.concatenate([[0], np.cumsum([sp.N for sp in spaces])])
    Ntot = int(off[-1])
    r = np.concatenate([sp.r for sp in spaces]); z = np.concatenate([sp.z for sp in spaces])
    w = np.concatenate([sp.w_in for sp in spaces])
    fq = np.zeros((S, Ntot)); dfr = np.zeros((S, Ntot)); dfz = np.zeros((S, Ntot))
    for a in range(S):
        g = int(species_grid[a]); sp = spaces[g]
        q, dr_, dz_ = fields_at_points(sp, np.asarray(f_list[a])[None, :])
        sl = slice(off[g], off[g + 1])
        fq[a, sl], dfr[a, sl], dfz[a, sl] = q[0], dr_[0], dz_[0]
    e2 = np.asarray(species.charge, dtype=np.float64) ** 2
    m0m = species.m0 / np.asarray(species.mass, dtype=np.float64)
    GD, GK = inner_integral(r, z, w, fq, dfr, dfz, e2, m0m, None, precision)
    vals_list, Cf_list = [], []
    for a in range(S):
        g = int(species_grid[a]); sp = spaces[g]
        sl = slice(off[g], off[g + 1])
        K = (species.nu * e2[a] * m0m[a] * GK[sl])[None]
        D = np.zeros((1, sp.N, 2, 2))
        c = -species.nu * e2[a] * m0m[a] ** 2
        D[0, :, 0, 0] = c * GD[sl, 0]; D[0, :, 0, 1] = c * GD[sl, 1]; D[0, :, 1, 0] = c * GD[sl, 1]; D[0, :, 1, 1] = c * GD[sl, 2]
        Ce = element_matrices(sp, K, D)
        vals_list.append(csr_values(sp, assemble_dense(sp, Ce[0])))
        # C(f) from the weak form with physical gradients, as in collision()
        Cf = np.zeros(sp.n)
        for e in range(sp.Ne):
            ce = np.zeros(sp.Nb)
            for q in range(sp.Nq):
                gi = e * sp.Nq + q
                flux = K[0, gi] * fq[a, off[g] + gi] + D[0, gi] @ np.array([dfr[a, off[g] + gi], dfz[a, off[g] + gi]])
                ce += sp.w_out[gi] * ((sp.E[q] * sp.invJ[e][None, :]) @ flux)
            Cf[sp.cell_dofs[e]] += sp.cell_P[e].T @ ce
        Cf_list.append(Cf)
    return spaces, vals_list, Cf_list, [mass(sp, shift) for sp in spaces]


# --------------------------------------------------------------------------------------------
# Linear solve of the implicit step (section III-G).
# The paper's band solver is Gaussian elimination WITHOUT pivoting in outer-product form
# (Golub & Van Loan Alg. 4.3.1) on the RCM-ordered matrix, one independent solve per species.
# The result it reaches has a plain definition -- x with A x = b -- so the oracle is that
# definition through a library routine (LAPACK, partial pivoting); the ordering is internal to
# the device path and does not appear here.  band_lu_outer_product() restates Alg. 4.3.1 itself
# on a dense array for the pins (L U = A, no fill outside the band).
# --------------------------------------------------------------------------------------------

def dense_from_csr(sp: Space, vals_one: np.ndarray) -> np.ndarray:
    rows = np.repeat(np.arange(sp.n), np.diff(sp.rowptr))
    A = np.zeros((sp.n, sp.n))
    A[rows, sp.colidx] = vals_one
    return A


def solve_species(sp: Space, vals_one: np.ndarray, rhs_one: np.ndarray) -> np.ndarray:
    """x = A^-1 b for one species block given its CSR values on the pattern A1."""
    return np.linalg.solve(dense_from_csr(sp, vals_one), rhs_one)


def band_lu_outer_product(A: np.ndarray, p: int, q: int) -> np.ndarray:
    """Golub & Van Loan Alg. 4.3.1 (L173): for k = 1..n-1: A(k+1:k+p, k) /= A(k,k);
    A(k+1:k+p, k+1:k+q) -= A(k+1:k+p, k) A(k, k+1:k+q).  Lower bandwidth p, upper q, no pivoting.
    Returns the factors in one array (unit lower L below the diagonal, U on and above)."""
    A = np.array(A, dtype=np.float64)
    n = A.shape[0]
    for k in range(n - 1):
        i1 = min(k + p, n - 1)
        j1 = min(k + q, n - 1)
        A[k + 1:i1 + 1, k] /= A[k, k]
        A[k + 1:i1 + 1, k + 1:j1 + 1] -= np.outer(A[k + 1:i1 + 1, k], A[k, k + 1:j1 + 1])
    return A
