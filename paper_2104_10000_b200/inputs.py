"""Seeded synthetic inputs for the Landau Jacobian hot path (meshes, species, distributions).

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2104_10000_b200/csrc``): it holds input recipes only -- quadtree leaf lists, species tables
and Maxwellian nodal values -- and none of the method's arithmetic (no tensor, no quadrature,
no finite-element code).  It imports neither the oracle nor the CUDA binding.

Recipes follow SURVEY.md section 8(d) / DESIGN.md "Input recipe"; they stand in for the paper's
own PETSc example (e + D + impurity charge states on p4est-refined Q3
meshes), which is not available.  Random numbers: splitmix64, seed = 20210410 + 1000*config +
problem index.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SEED0 = 20210410
MASK64 = (1 << 64) - 1


class SplitMix64:
    """Counter-based splitmix64 stream -> uniform doubles in [0,1)."""

    def __init__(self, seed: int):
        self.state = seed & MASK64

    def next_u64(self) -> int:
        self.state = (self.state + 0x9E3779B97F4A7C15) & MASK64
        z = self.state
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK64
        return z ^ (z >> 31)

    def uniform(self, lo: float = 0.0, hi: float = 1.0) -> float:
        return lo + (hi - lo) * ((self.next_u64() >> 11) * (1.0 / (1 << 53)))

    def uniform_array(self, n: int, lo: float = 0.0, hi: float = 1.0) -> np.ndarray:
        return np.array([self.uniform(lo, hi) for _ in range(n)], dtype=np.float64)


@dataclass
class Mesh:
    """Quadtree-forest leaves on a rectangle (the ``landau_mesh`` struct of include/landau.h).

    Leaf k at level l covers r in rmin + hr0/2^l * [ir, ir+1], z in zmin + hz0/2^l * [iz, iz+1]
    with hr0 = (rmax-rmin)/nbr, hz0 = (zmax-zmin)/nbz.
    """

    rmin: float
    rmax: float
    zmin: float
    zmax: float
    nbr: int
    nbz: int
    level: np.ndarray
    ir: np.ndarray
    iz: np.ndarray

    @property
    def ncells(self) -> int:
        return int(self.level.shape[0])


def mesh_uniform(rmin, rmax, zmin, zmax, nbr, nbz) -> Mesh:
    """Uniform nbr x nbz mesh, leaves in row-major (z outer, r inner) order."""
    iz, ir = np.meshgrid(np.arange(nbz, dtype=np.int32), np.arange(nbr, dtype=np.int32), indexing="ij")
    n = nbr * nbz
    return Mesh(rmin, rmax, zmin, zmax, nbr, nbz, np.zeros(n, np.int32), ir.ravel().copy(), iz.ravel().copy())


def mesh_quadtree(rmin, rmax, zmin, zmax, nbr, nbz, R_in, L_in, R_out, L_out) -> Mesh:
    """p4est-style refinement toward the origin, then 2:1 face balance.

    A leaf is split while (level < L_in and dist < R_in) or (level < L_out and dist < R_out),
    dist = distance from the origin (r,z)=(0,0) to the closed cell.  Leaves are emitted in
    depth-first (Morton-like) order: base cells row-major, children in (iz,ir) order.
    """
    hr0 = (rmax - rmin) / nbr
    hz0 = (zmax - zmin) / nbz

    def dist(l, i, j):
        hr, hz = hr0 / (1 << l), hz0 / (1 << l)
        r0, r1 = rmin + i * hr, rmin + (i + 1) * hr
        z0, z1 = zmin + j * hz, zmin + (j + 1) * hz
        dr = 0.0 if r0 <= 0.0 <= r1 else min(abs(r0), abs(r1))
        dz = 0.0 if z0 <= 0.0 <= z1 else min(abs(z0), abs(z1))
        return math.hypot(dr, dz)

    leaves = set()

    def refine(l, i, j):
        d = dist(l, i, j)
        if (l < L_in and d < R_in) or (l < L_out and d < R_out):
            for cj in (0, 1):
                for ci in (0, 1):
                    refine(l + 1, 2 * i + ci, 2 * j + cj)
        else:
            leaves.add((l, i, j))

    for j in range(nbz):
        for i in range(nbr):
            refine(0, i, j)

    # 2:1 face balance: split any leaf with a face neighbour more than one level finer.
    def covering_leaf(l, i, j):
        """Leaf (at level <= l) covering the level-l cell (i,j), or None if it is subdivided."""
        while l >= 0:
            if (l, i, j) in leaves:
                return (l, i, j)
            l, i, j = l - 1, i >> 1, j >> 1
        return None

    changed = True
    while changed:
        changed = False
        for (l, i, j) in sorted(leaves):
            if (l, i, j) not in leaves:
                continue
            for di, dj in ((-1, 0), (1, 0), (0, -1), (0, 1)):
                ni, nj = i + di, j + dj
                if ni < 0 or nj < 0 or ni >= nbr << l or nj >= nbz << l:
                    continue
                nb = covering_leaf(l, ni, nj)
                while nb is not None and nb[0] < l - 1:
                    leaves.discard(nb)
                    L, I, J = nb
                    for cj in (0, 1):
                        for ci in (0, 1):
                            leaves.add((L + 1, 2 * I + ci, 2 * J + cj))
                    changed = True
                    nb = covering_leaf(l, ni, nj)

    # depth-first order
    def key(leaf):
        l, i, j = leaf
        path = []
        for lev in range(l, 0, -1):
            path.append(((j >> (l - lev)) & 1) * 2 + ((i >> (l - lev)) & 1))
        bi, bj = i >> l, j >> l
        return (bj * nbr + bi, tuple(reversed(path)))

    out = sorted(leaves, key=key)
    lev = np.array([t[0] for t in out], np.int32)
    ir = np.array([t[1] for t in out], np.int32)
    iz = np.array([t[2] for t in out], np.int32)
    return Mesh(rmin, rmax, zmin, zmax, nbr, nbz, lev, ir, iz)


def mesh_refine_uniform(m: Mesh) -> Mesh:
    """Every leaf split into its four children (children in (iz,ir) order, parents in place)."""
    lev, ir, iz = [], [], []
    for l, i, j in zip(m.level, m.ir, m.iz):
        for cj in (0, 1):
            for ci in (0, 1):
                lev.append(l + 1); ir.append(2 * i + ci); iz.append(2 * j + cj)
    return Mesh(m.rmin, m.rmax, m.zmin, m.zmax, m.nbr, m.nbz, np.array(lev, np.int32), np.array(ir, np.int32),
                np.array(iz, np.int32))


def mesh_scaled(m: Mesh, k: float) -> Mesh:
    """The same leaves on a domain scaled by k (a grid for a species cluster with thermal speed k)."""
    return Mesh(m.rmin * k, m.rmax * k, m.zmin * k, m.zmax * k, m.nbr, m.nbz, m.level, m.ir, m.iz)


def multigrid_case(which: str = "paper3"):
    """Multiple-grid workloads (section III-C, Table I).  Returns
    (name, order, meshes, species, species_grid, components) with one Component per species.
      'paper3': ten species on three 20-cell Q3 grids (the 20-cell / 193-vertex grid of Fig. 3, domain
                5 v_th of its cluster): e | D+ | eight heavy-ion charge states -- 960 points, 1,930 equations;
      'same2' : two species on two IDENTICAL refined Q2 grids (every point coincides with one of the other grid);
      'scaled': three species on two refined Q2 grids of different extent."""
    g20 = mesh_quadtree(0.0, 5.0, -5.0, 5.0, 2, 4, 1.0, 2, 2.5, 1)
    if which == "paper3":
        mw = 184.0 * 1836.0
        rows = [(1.0, -1.0, 1.0, 1.0), (3670.0, 1.0, 0.64, 1.0)] + [(mw, float(q), 0.01, 1.0) for q in range(1, 9)]
        sp = _sp(rows)
        meshes = [g20, mesh_scaled(g20, 1.0 / math.sqrt(3670.0)), mesh_scaled(g20, 1.0 / math.sqrt(mw))]
        grid = [0, 1] + [2] * 8
        return "mg-paper3-10sp-q3", 3, meshes, sp, grid, [Component(s, rows[s][2], 1.0) for s in range(10)]
    g = mesh_quadtree(0.0, 4.0, -4.0, 4.0, 2, 4, 1.0, 2, 2.0, 1)
    if which == "same2":
        sp = _sp([(1, -1, 1, 1), (4, 1, 1, 1)])
        return "mg-same2-q2", 2, [g, g], sp, [0, 1], [Component(0, 1, 1), Component(1, 1, 1)]
    if which == "scaled":
        sp = _sp([(1, -1, 1, 1), (64, 1, 0.6, 1), (128, 2, 0.2, 1)])
        return "mg-scaled-q2", 2, [g, mesh_scaled(g, 0.125)], sp, [0, 1, 1], [Component(0, 1, 1), Component(1, 0.6, 1, 0.02), Component(2, 0.2, 1, 0.04)]
    raise ValueError(which)


@dataclass
class Species:
    """The ``landau_species`` struct: masses in m_e, charges in e, nu = 1, m0 = m_e (Appendix A)."""

    mass: np.ndarray
    charge: np.ndarray
    density: np.ndarray
    temperature: np.ndarray
    m0: float = 1.0
    nu: float = 1.0

    @property
    def S(self) -> int:
        return int(self.mass.shape[0])


@dataclass
class Component:
    """One Maxwellian component n (m/(pi T))^{3/2} exp(-m (r^2 + (z - zs)^2)/T) of a species."""

    species: int
    n: float
    T: float
    zs: float = 0.0


@dataclass
class Workload:
    name: str
    order: int
    mesh: Mesh
    species: Species
    # components[b] = list of Component for problem b of the batch
    components: list = field(default_factory=list)
    noise: float = 0.0
    seed: int = SEED0

    @property
    def nbatch(self) -> int:
        return len(self.components)


def maxwellian(mass: float, n: float, T: float, zs: float, r: np.ndarray, z: np.ndarray) -> np.ndarray:
    """f = n (m/(pi T))^{3/2} exp(-m (r^2+(z-zs)^2)/T), units v_th,e = sqrt(2 T_ref/m_e) = 1."""
    return n * (mass / (math.pi * T)) ** 1.5 * np.exp(-mass * (r * r + (z - zs) ** 2) / T)


def nodal_f(wl: Workload, r: np.ndarray, z: np.ndarray, problem: int = 0) -> np.ndarray:
    """Nodal values f[S][n] at the DOF coordinates (r,z) for one problem of the workload.

    The multiplicative noise (1 + noise*U(-1,1)) is drawn per species, per node, in DOF order from
    splitmix64(seed + problem) -- after all Maxwellian components are summed.
    """
    S, n = wl.species.S, r.shape[0]
    f = np.zeros((S, n))
    for c in wl.components[problem]:
        f[c.species] += maxwellian(float(wl.species.mass[c.species]), c.n, c.T, c.zs, r, z)
    if wl.noise:
        rng = SplitMix64(wl.seed + problem)
        for s in range(S):
            f[s] *= 1.0 + wl.noise * rng.uniform_array(n, -1.0, 1.0)
    return f


def _sp(rows) -> Species:
    a = np.array(rows, dtype=np.float64)
    return Species(a[:, 0].copy(), a[:, 1].copy(), a[:, 2].copy(), a[:, 3].copy())


def mesh_config3(variant: str = "B") -> Mesh:
    """Config-3 mesh.  'B' = size-matched (R_in,L_in,R_out,L_out) = (1,4,4,2): 308 cells;
    'A' = literal reading (1,3,3,1): 98 cells.  See DESIGN.md reading Q13."""
    p = (1.0, 4, 4.0, 2) if variant == "B" else (1.0, 3, 3.0, 1)
    return mesh_quadtree(0.0, 8.0, -8.0, 8.0, 4, 8, *p)


def config(k: int, nbatch: int | None = None, variant: str = "B") -> Workload:
    """The five BASELINE.json configs (k = 1..5), k = 0, a tiny refined Q2 case for tests, and
    k = 6, 7, the paper-shaped ten-species context runs."""
    seed = SEED0 + 1000 * k
    if k == 0:
        mesh = mesh_quadtree(0.0, 4.0, -4.0, 4.0, 2, 4, 1.0, 2, 2.0, 1)
        sp = _sp([(1, -1, 1, 1), (4, 1, 1, 1)])
        comps = [[Component(0, 1, 1), Component(1, 1, 1)]]
        return Workload("cfg0-tiny-refined-q2", 2, mesh, sp, comps, 1e-3, seed)
    if k == 1:
        mesh = mesh_uniform(0.0, 5.0, -5.0, 5.0, 5, 10)
        sp = _sp([(1, -1, 1, 1)])
        return Workload("cfg1-e-q2-5x10", 2, mesh, sp, [[Component(0, 1, 1)]], 1e-3, seed)
    if k == 2:
        mesh = mesh_uniform(0.0, 5.0, -5.0, 5.0, 8, 16)
        sp = _sp([(1, -1, 1, 1), (3670, 1, 1, 1)])
        return Workload("cfg2-eD-q3-8x16", 3, mesh, sp, [[Component(0, 1, 1), Component(1, 1, 1)]], 1e-3, seed)
    if k == 3:
        mesh = mesh_config3(variant)
        sp = _sp([(1, -1, 1, 0.05), (3670, 1, 1, 0.05)])
        comps = [[Component(0, 0.99, 0.05), Component(0, 0.01, 1.0, 0.5), Component(1, 1.0, 0.05)]]
        return Workload(f"cfg3{variant}-eD-q3-quench", 3, mesh, sp, comps, 0.0, seed)
    if k == 4:
        mesh = mesh_config3(variant)
        rng = SplitMix64(seed)
        mi = 40.0 * 1836.0
        dens = [1.0, 0.7, 0.1, 0.05, 1.0 / 30.0]  # sum q n over ions = 0.7+0.1+0.1+0.1 = 1 = n_e
        mass = [1.0, 3670.0, mi, mi, mi]
        chg = [-1.0, 1.0, 1.0, 2.0, 3.0]
        T = [rng.uniform(0.05, 1.0) for _ in range(5)]
        sp = _sp(list(zip(mass, chg, dens, T)))
        comps = []
        for s in range(5):
            comps.append(Component(s, 0.9 * dens[s], T[s]))
            comps.append(Component(s, 0.1 * dens[s], rng.uniform(0.05, 1.0)))
        return Workload(f"cfg4{variant}-5sp-q3-quench", 3, mesh, sp, [comps], 0.0, seed)
    if k == 5:
        mesh = mesh_config3(variant)
        nb = 512 if nbatch is None else nbatch
        sp = _sp([(1, -1, 1, 0.05), (3670, 1, 1, 0.05)])
        comps = []
        for b in range(nb):
            rng = SplitMix64(seed + b)
            Tb = rng.uniform(0.02, 1.0)
            tail = rng.uniform(0.0, 0.02)
            zs = rng.uniform(0.0, 1.0)
            comps.append([Component(0, 1.0 - tail, Tb), Component(0, tail, 1.0, zs), Component(1, 1.0, Tb)])
        return Workload(f"cfg5{variant}-batch{nb}-eD-q3-quench", 3, mesh, sp, comps, 0.0, seed)
    if k in (6, 7):
        # Paper-shaped context runs: ten species -- e, D+ and
        # eight effective ionisation states of a heavy ion (m = 184 x 1836), all at the same temperature --
        # on an 80-cell Q3 mesh (k = 6) and its uniform refinement to 320 cells (k = 7).
        mesh = mesh_quadtree(0.0, 5.0, -5.0, 5.0, 4, 8, 1.0, 2, 2.5, 1)
        if k == 7:
            mesh = mesh_refine_uniform(mesh)
        mw = 184.0 * 1836.0
        rows = [(1.0, -1.0, 1.0, 1.0), (3670.0, 1.0, 0.64, 1.0)] + [(mw, float(q), 0.01, 1.0) for q in range(1, 9)]
        sp = _sp(rows)   # sum q n over ions = 0.64 + 0.01 * 36 = 1 = n_e
        nb = 1 if nbatch is None else nbatch
        comps = [[Component(s, rows[s][2], 1.0) for s in range(10)] for _ in range(nb)]
        return Workload(f"ctx{mesh.ncells}-10sp-q3", 3, mesh, sp, comps, 1e-3, seed)
    raise ValueError(f"unknown config {k}")
