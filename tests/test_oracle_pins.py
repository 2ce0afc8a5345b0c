"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only).

Every check here compares the oracle with something OTHER than itself: closed forms, an
independent library (scipy / mpmath), brute-force azimuthal quadrature of the 3-D tensor of
Eq. 3, Rosenbluth potentials of a Maxwellian, or exact invariants of the weak
form (conservation).
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest
import scipy.special as ss

from paper_2104_10000_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    out = []
    for line in open(os.path.join(GOLD, name)):
        line = line.split("#")[0].split()
        if line:
            out.append(line)
    return out


# ---------------------------------------------------------------------------- elliptic integrals
def test_elliptic_closed_forms(oracle):
    idx = {"K": 0, "E": 1, "D": 2, "S": 3}
    for name, m, val in _rows("elliptic_values.txt"):
        got = oracle.ellip_KEDS(float(m))[idx[name]]
        assert abs(got - float(val)) <= 2e-16 * abs(float(val)), (name, m, got)
    # the golden K(1/2) really is Gamma(1/4)^2/(4 sqrt(pi))
    assert abs(math.gamma(0.25) ** 2 / (4 * math.sqrt(math.pi)) - 1.8540746773013719) < 1e-15


def test_elliptic_vs_scipy_and_legendre(oracle):
    rng = np.random.default_rng(7)
    ms = np.concatenate([rng.uniform(0, 1, 200), 1 - 10.0 ** rng.uniform(-7, -1, 50), 10.0 ** rng.uniform(-8, -1, 50)])
    for m in ms:
        K, E, D, S = oracle.ellip_KEDS(m)
        assert abs(K - ss.ellipk(m)) <= 4e-16 * K
        assert abs(E - ss.ellipe(m)) <= 4e-16 * E
        K1, E1, _, _ = oracle.ellip_KEDS(1 - m)
        # Legendre relation E K' + E' K - K K' = pi/2
        assert abs(E * K1 + E1 * K - K * K1 - math.pi / 2) <= 1e-14 * max(1.0, K * K1)


@pytest.mark.parametrize("m", [1e-7, 1e-4, 3e-3, 0.049, 0.051, 0.3, 0.77, 0.99, 1 - 1e-5])
def test_D_and_S_against_their_integral_definitions(oracle, m):
    mp.mp.dps = 40
    mm = mp.mpf(m)
    Dq = mp.quad(lambda t: mp.cos(t) ** 2 / (1 - mm * mp.sin(t) ** 2) ** mp.mpf(1.5), [0, mp.pi / 4, mp.pi / 2])
    Sq = mp.quad(lambda t: (mp.sin(t) * mp.cos(t)) ** 2 / (1 - mm * mp.sin(t) ** 2) ** mp.mpf(1.5), [0, mp.pi / 4, mp.pi / 2])
    K, E, D, S = oracle.ellip_KEDS(m)
    assert abs(D - float(Dq)) <= 4e-16 * D
    assert abs(S - float(Sq)) <= 6e-16 * S
    # double-precision instantiation (timed baseline) agrees to its own rounding amplification
    Kd, Ed, Dd, Sd = oracle.ellip_KEDS(m, "d")
    assert abs(Dd - D) <= 1e-13 * D and abs(Kd - K) <= 1e-14 * K and abs(Ed - E) <= 1e-14 * E


# ---------------------------------------------------------------------------- Eq. 3 and its azimuth integral
def landau_tensor_3d(u):
    """Eq. 3 (L44): U = (|u|^2 I - u u)/|u|^3 -- the test's own transcription."""
    n2 = u @ u
    return (n2 * np.eye(3) - np.outer(u, u)) / n2 ** 1.5


def test_eq3_properties():
    rng = np.random.default_rng(1)
    for _ in range(20):
        u = rng.normal(size=3)
        U = landau_tensor_3d(u)
        assert np.allclose(U @ u, 0, atol=1e-14)
        assert np.allclose(U, U.T)
        assert abs(np.trace(U) - 2 / np.linalg.norm(u)) < 1e-13


def brute_force_UD_UK(r, z, rb, zb, nphi):
    """Periodic trapezoid rule in phi of Eq. 3 with v at azimuth 0 and vbar at azimuth phi.
    U^D = (x,z) block; U^K columns = U . (d vbar/d rbar direction, zhat)."""
    UD = np.zeros((2, 2)); UK = np.zeros((2, 2))
    for k in range(nphi):
        phi = 2 * math.pi * (k + 0.5) / nphi
        u = np.array([r - rb * math.cos(phi), -rb * math.sin(phi), z - zb])
        U = landau_tensor_3d(u)
        erb = np.array([math.cos(phi), math.sin(phi), 0.0])
        ez = np.array([0.0, 0.0, 1.0])
        UD += U[np.ix_([0, 2], [0, 2])]
        UK[:, 0] += (U @ erb)[[0, 2]]
        UK[:, 1] += (U @ ez)[[0, 2]]
    return UD * 2 * math.pi / nphi, UK * 2 * math.pi / nphi


PAIRS = [(0.7, 0.4, 1.3, -0.6), (0.0087, 3.0, 7.9, -7.5), (2.0, 0.1, 0.3, 0.2), (1.0, 0.0, 1.0, 0.5),
         (0.05, -0.02, 0.06, 0.03), (4.0, 1.0, 0.01, 1.0), (0.5, 0.5, 0.55, 0.5)]


@pytest.mark.parametrize("pair", PAIRS)
def test_tensor2d_vs_brute_force_azimuth_quadrature(oracle, pair):
    r, z, rb, zb = pair
    UD, UK = oracle.tensor2d(r, z, rb, zb)
    bd, bk = brute_force_UD_UK(r, z, rb, zb, 4096)
    scale = np.abs(bd).max()
    assert np.allclose([UD[0], UD[1], UD[2]], [bd[0, 0], bd[0, 1], bd[1, 1]], rtol=0, atol=2e-12 * scale)
    assert abs(bd[0, 1] - bd[1, 0]) < 1e-12 * scale
    assert np.allclose(UK, bk, rtol=0, atol=2e-12 * max(scale, np.abs(bk).max()))


def test_tensor2d_near_coincident_vs_mpmath(oracle):
    """Near-neighbour pair (m -> 1): the trapezoid rule converges slowly, use adaptive mp quad."""
    mp.mp.dps = 30
    r, z, rb, zb = 1.0, 0.2, 1.004, 0.197

    def comp(fn):
        return float(mp.quad(fn, [0, mp.mpf("0.01"), mp.mpf("0.1"), 1, mp.pi, 2 * mp.pi - 1, 2 * mp.pi - mp.mpf("0.1"),
                                  2 * mp.pi - mp.mpf("0.01"), 2 * mp.pi]))
    dz = z - zb
    n3 = lambda p: (r * r + rb * rb - 2 * r * rb * mp.cos(p) + dz * dz) ** mp.mpf(1.5)
    P0 = comp(lambda p: 1 / n3(p)); Pc = comp(lambda p: (1 - mp.cos(p)) / n3(p)); Pss = comp(lambda p: mp.sin(p) ** 2 / n3(p))
    UD, UK = oracle.tensor2d(r, z, rb, zb)
    ref = [rb * rb * Pss + dz * dz * P0, -dz * ((r - rb) * P0 + rb * Pc), (r - rb) ** 2 * P0 + 2 * r * rb * Pc]
    assert np.allclose(UD, ref, rtol=1e-12)
    assert abs(UK[0, 0] - (dz * dz * (P0 - Pc) + r * rb * Pss)) < 1e-12 * abs(UK[0, 0])
    assert abs(UK[1, 0] - dz * ((rb - r) * P0 + r * Pc)) < 1e-12 * abs(ref[2])


def test_tensor2d_structure(oracle):
    rng = np.random.default_rng(3)
    for _ in range(50):
        r, rb = rng.uniform(0.01, 5, 2); z, zb = rng.uniform(-5, 5, 2)
        UD, UK = oracle.tensor2d(r, z, rb, zb)
        UDx, UKx = oracle.tensor2d(rb, zb, r, z)
        sc = np.abs(UK).max()
        # exchange symmetry U^K(v,vb)^T = U^K(vb,v)
        assert np.allclose(UK.T, UKx, rtol=0, atol=1e-13 * sc)
        # axisymmetric image of U.u = 0:  U^D (r,z)^T = U^K (rb,zb)^T
        UDm = np.array([[UD[0], UD[1]], [UD[1], UD[2]]])
        lhs, rhs = UDm @ np.array([r, z]), UK @ np.array([rb, zb])
        assert np.allclose(lhs, rhs, rtol=0, atol=1e-12 * sc * max(r, rb, abs(z), abs(zb), 1))


# ---------------------------------------------------------------------------- Rosenbluth potentials
def _rosenbluth_error(oracle, mesh, probes):
    sp = oracle.build_space(mesh, 3)
    fq = (math.pi ** -1.5 * np.exp(-(sp.r ** 2 + sp.z ** 2)))[None, :]
    dfr, dfz = -2 * sp.r * fq, -2 * sp.z * fq
    errs = []
    for a, b in probes:
        i = int(np.argmin((sp.r - a) ** 2 + (sp.z - b) ** 2))
        GD, GK = oracle.inner_integral(sp.r, sp.z, sp.w_in, fq, dfr, dfz, np.ones(1), np.ones(1), rows=(i, i + 1))
        r, z = sp.r[i], sp.z[i]
        v = math.hypot(r, z); e = math.erf(v); ex = math.exp(-v * v) / math.sqrt(math.pi)
        g1 = (1 - 1 / (2 * v * v)) * e + ex / v                      # g'
        g2 = e / v ** 3 - 2 * ex / (v * v)                           # g''
        h1 = 2 * ex / v - e / (v * v)                                # h'
        vr, vz = r / v, z / v
        gg = np.array([g2 * vr * vr + g1 / v * (1 - vr * vr), (g2 - g1 / v) * vr * vz, g2 * vz * vz + g1 / v * (1 - vz * vz)])
        kk = np.array([2 * h1 * vr, 2 * h1 * vz])
        errs.append(max(np.abs(GD[i] - gg).max() / np.abs(gg).max(), np.abs(GK[i] - kk).max() / np.abs(kk).max()))
    return max(errs)


def test_inner_integral_reproduces_rosenbluth_potentials_of_a_maxwellian(oracle):
    """For f = pi^{-3/2} exp(-v^2):  int d^3vb U f = grad grad g,  int d^3vb U.grad f = 2 grad h,
    g = (v + 1/(2v)) erf v + exp(-v^2)/sqrt(pi),  h = erf(v)/v  (U = grad grad |u|, so
    div_vb U = -2 grad(1/|u|)).  Pins scale, sign, component order, the r-bar weight and the
    placement of 2 pi (reading Q2).  The quadrature skips a log-singular self cell, so the match is
    to discretisation error, which must shrink ~h^2 under refinement toward the probes."""
    probes = [(0.3, 0.2), (0.1, -0.4), (0.6, 0.1)]
    e4 = _rosenbluth_error(oracle, inputs.mesh_quadtree(0, 5, -5, 5, 5, 10, 1.0, 4, 2.5, 2), probes)
    e5 = _rosenbluth_error(oracle, inputs.mesh_quadtree(0, 5, -5, 5, 5, 10, 1.0, 5, 2.5, 3), probes)
    assert e4 < 1.2e-3 and e5 < 3.5e-4 and e5 < e4 / 3
