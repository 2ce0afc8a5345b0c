"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/landau.h
declares, its host set-up agrees BIT-EXACTLY with the oracle's independent DOF numbering and CSR
pattern, and its error paths return codes instead of crashing.  No compute calls (no GPU)."""
import os
import re

import numpy as np
import pytest

from paper_2104_10000_b200 import inputs


@pytest.fixture(scope="module")
def binding():
    from paper_2104_10000_b200 import build
    build.build()
    from paper_2104_10000_b200 import binding as b
    b.lib()
    return b


def test_exports_every_declared_symbol(binding):
    hdr = open(os.path.join(os.path.dirname(__file__), "..", "include", "landau.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(landau_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(binding.SIGNATURES), declared ^ set(binding.SIGNATURES)
    L = binding.lib()
    for name in declared:
        assert hasattr(L, name)


@pytest.mark.parametrize("cfg", [0, 1, 2, 3, "3A", 6, 7])
def test_setup_matches_oracle_numbering_and_pattern(binding, oracle, cfg):
    if cfg == "3A":
        wl = inputs.config(3, variant="A")
    else:
        wl = inputs.config(cfg)
    hs = binding.landau_setup_host(wl.mesh, wl.order)
    sp = oracle.build_space(wl.mesh, wl.order)
    assert (hs["n"], hs["nnz"], hs["N"]) == (sp.n, sp.nnz, sp.N)
    assert np.array_equal(hs["rowptr"], sp.rowptr)          # integer work: bit-exact
    assert np.array_equal(hs["colidx"], sp.colidx)
    assert np.abs(hs["dof_r"] - sp.dof_r).max() < 1e-14 and np.abs(hs["dof_z"] - sp.dof_z).max() < 1e-14


def test_setup_rejects_bad_meshes(binding):
    m = inputs.mesh_uniform(0.0, 1.0, -1.0, 1.0, 2, 2)
    L = binding.lib()

    def code(mesh, order=3):
        try:
            binding.landau_setup_host(mesh, order)
            return 0
        except binding.LandauError as e:
            return e.code
    assert code(m) == 0
    assert code(m, order=4) == binding.LANDAU_EINVAL
    bad = inputs.Mesh(-1.0, 1.0, -1.0, 1.0, 2, 2, m.level, m.ir, m.iz)           # rmin < 0
    assert code(bad) == binding.LANDAU_EINVAL
    hole = inputs.Mesh(0.0, 1.0, -1.0, 1.0, 2, 2, m.level[:3], m.ir[:3], m.iz[:3])  # does not tile
    assert code(hole) == binding.LANDAU_EINVAL
    dup = inputs.Mesh(0.0, 1.0, -1.0, 1.0, 2, 2, m.level, np.array([0, 0, 0, 1], np.int32), m.iz)
    assert code(dup) == binding.LANDAU_EINVAL
    # not 2:1 balanced: one level-0 cell next to level-2 cells
    lev, ir, iz = [0], [1], [0]
    for cj in range(2):
        for ci in range(2):
            if (ci, cj) == (1, 0):
                for dj in range(2):
                    for di in range(2):
                        lev.append(2); ir.append(2 + di); iz.append(0 + dj)
            else:
                lev.append(1); ir.append(ci); iz.append(cj)
    unb = inputs.Mesh(0.0, 2.0, 0.0, 1.0, 2, 1, np.array(lev, np.int32), np.array(ir, np.int32), np.array(iz, np.int32))
    assert code(unb) == binding.LANDAU_EINVAL
    assert L.landau_strerror(binding.LANDAU_EINVAL).decode() == "invalid argument"


def test_create_without_gpu_fails_loudly(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    wl = inputs.config(1)
    with pytest.raises(binding.LandauError) as ei:
        binding.LandauContext(wl.mesh, wl.order, wl.species)
    assert ei.value.code == binding.LANDAU_ECUDA


def _envelope_work(rowptr, colidx, perm, KB):
    """2 KB sum m_s^2 over the block steps: m_s = rows below block s that elimination without pivoting can reach,
    i.e. the monotone hull of the envelope (no fill left of a row's first entry).  Written out here from that
    definition, independently of the library."""
    n = len(perm)
    pos = np.empty(n, int); pos[perm] = np.arange(n)
    rows = np.repeat(np.arange(n), np.diff(rowptr))
    first = np.arange(n)
    np.minimum.at(first, pos[rows], pos[colidx])
    work = 0.0
    for k0 in range(0, n, KB):
        ke = min(k0 + KB, n) - 1
        reach = max([i for i in range(n) if first[i] <= ke] or [ke])       # last row whose envelope starts at or before ke
        work += 2.0 * (ke - k0 + 1) * max(0, reach - ke) ** 2
    return work


@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 6])
def test_band_order_is_a_valid_bandwidth_reducing_permutation(binding, cfg):
    """Host logic of the band LU (RCM ordering, band storage): the order is a permutation, the
    reported half-bandwidth is the one it gives on the pattern and the reported flop its envelope work; both are no
    worse than those of scipy's RCM (the library tries several RCM starting nodes and the row sweep and keeps the
    cheapest of the narrow ones); on the refined meshes the band is far below the natural order's, on the uniform
    Q3 mesh it is the row sweep's 3 (3 nr + 1) + 3; the envelope work is at most the uniform-band work."""
    import scipy.sparse as sps
    from scipy.sparse.csgraph import reverse_cuthill_mckee
    wl = inputs.config(cfg)
    hs = binding.landau_setup_host(wl.mesh, wl.order)
    bo = binding.landau_band_order_host(wl.mesh, wl.order)
    n = hs["n"]
    assert sorted(bo["perm"].tolist()) == list(range(n))
    pos = np.empty(n, int); pos[bo["perm"]] = np.arange(n)
    rows = np.repeat(np.arange(n), np.diff(hs["rowptr"]))
    assert int(np.abs(pos[rows] - pos[hs["colidx"]]).max()) == bo["bw"]
    A = sps.csr_matrix((np.ones(hs["nnz"]), hs["colidx"], hs["rowptr"]), shape=(n, n))
    p = reverse_cuthill_mckee(A, symmetric_mode=True)
    ps = np.empty(n, int); ps[p] = np.arange(n)
    bw_scipy = int(np.abs(ps[rows] - ps[hs["colidx"]]).max())
    bw_natural = int(np.abs(rows - hs["colidx"]).max())
    assert bo["bw"] <= bw_scipy
    if cfg == 3:
        assert bo["bw"] < 0.5 * bw_natural
    if cfg == 2:
        assert bo["bw"] == 3 * (3 * 8 + 1) + 3
    assert bo["block_columns"] in (8, 16, 32)
    assert 0 < bo["flop"] <= 2.0 * n * bo["bw"] ** 2
    assert bo["flop"] == _envelope_work(hs["rowptr"], hs["colidx"], bo["perm"], bo["block_columns"])
    assert bo["flop"] <= _envelope_work(hs["rowptr"], hs["colidx"], np.asarray(p), bo["block_columns"])


@pytest.mark.parametrize("cfg", [0, 2, 3, 6])
def test_front_lists_of_the_envelope_factorisation(binding, cfg):
    """Host logic of the front kernel: LU without pivoting keeps the envelope, so block step s involves, beside its
    own block, the next block's rows and every later row whose first entry lies at or before the block.  Recomputed
    here from that definition: the longest list and the flop 2 KB sum na_s^2 must match; on the refined meshes the
    front does a fraction of the hull's flops, on the uniform mesh about the same."""
    wl = inputs.config(cfg)
    hs = binding.landau_setup_host(wl.mesh, wl.order)
    bo = binding.landau_band_order_host(wl.mesh, wl.order)
    fr = binding.landau_band_front_host(wl.mesh, wl.order)
    n, KB = hs["n"], bo["block_columns"]
    pos = np.empty(n, int); pos[bo["perm"]] = np.arange(n)
    rows = np.repeat(np.arange(n), np.diff(hs["rowptr"]))
    first = np.arange(n)
    np.minimum.at(first, pos[rows], pos[hs["colidx"]])
    rows_max, flop = 0, 0.0
    for k0 in range(0, n, KB):
        ke = min(k0 + KB, n) - 1
        act = {i for i in range(ke + 1, n) if i <= ke + KB or first[i] <= ke}
        rows_max = max(rows_max, len(act))
        flop += 2.0 * (ke - k0 + 1) * len(act) ** 2
    assert fr["rows_max"] == rows_max and fr["flop"] == flop and fr["fits"]
    if cfg in (3, 6):
        assert fr["flop"] < 0.3 * bo["flop"]
    if cfg == 2:
        assert fr["flop"] > 0.6 * bo["flop"]


def test_factor_block_width_in_the_32_column_range(binding):
    """Half-bandwidths in (256, 384] mean 32-column blocks for the solves; the factorisation takes 16-column blocks (slot
    kernel) there when the envelope is jagged and the window of its largest front fits an SM: mesh 3B of config 5 (96
    rows beside the block: two windows per SM) and the ten-species 320-cell mesh (99 rows: one).  Flop and front sizes
    are reported for the width chosen."""
    for cfg, rows in ((5, 96), (7, 99)):
        wl = inputs.config(cfg)
        hs = binding.landau_setup_host(wl.mesh, wl.order)
        bo = binding.landau_band_order_host(wl.mesh, wl.order)
        fr = binding.landau_band_front_host(wl.mesh, wl.order)
        assert 256 < bo["bw"] <= 384 and bo["block_columns"] == 16
        assert bo["flop"] == _envelope_work(hs["rowptr"], hs["colidx"], bo["perm"], 16)
        assert fr["fits"] and fr["flop"] < 0.3 * bo["flop"] and fr["rows_max"] == rows


def test_multigrid_argument_checks_need_no_gpu(binding):
    """landau_create_multigrid validates its species -> grid map before it looks for a device: bad maps give
    LANDAU_EINVAL everywhere; a good one gives LANDAU_ECUDA on a machine without a GPU."""
    import torch
    g = inputs.config(0).mesh
    sp3 = inputs._sp([(1, -1, 1, 1), (4, 1, 1, 1), (8, 1, 1, 1)])
    for bad in ([1, 0, 1], [0, 0, 0], [0, 2, 2], [0, 1, 5], [-1, 0, 1]):
        with pytest.raises(binding.LandauError) as ei:
            binding.LandauMultigridContext([g, inputs.mesh_scaled(g, 0.5)], bad, 2, sp3, 1)
        assert ei.value.code == binding.LANDAU_EINVAL, bad
    with pytest.raises(binding.LandauError) as ei:
        binding.LandauMultigridContext([g, inputs.mesh_scaled(g, 0.5)], [0, 1, 1], 2, sp3, 0)      # max_batch < 1
    assert ei.value.code == binding.LANDAU_EINVAL
    if not torch.cuda.is_available():
        with pytest.raises(binding.LandauError) as ei:
            binding.LandauMultigridContext([g, inputs.mesh_scaled(g, 0.5)], [0, 1, 1], 2, sp3, 1)
        assert ei.value.code == binding.LANDAU_ECUDA


def test_new_entry_points_check_their_arguments_without_a_gpu(binding):
    """Path selection, tensor cache, issue probe and the max_batch range: bad arguments give LANDAU_EINVAL before any
    device is looked for."""
    import ctypes
    L = binding.lib()
    assert L.landau_set_pair_path(None, binding.LANDAU_PAIR_SHARED) == binding.LANDAU_EINVAL
    assert L.landau_pair_path(None, None, None) == binding.LANDAU_EINVAL
    assert L.landau_set_tensor_cache(None, 1) == binding.LANDAU_EINVAL
    cyc = ctypes.c_double()
    assert L.landau_fp64_issue_probe(8, 16, ctypes.byref(cyc), None) == binding.LANDAU_EINVAL       # unknown mode
    assert L.landau_fp64_issue_probe(0, 0, ctypes.byref(cyc), None) == binding.LANDAU_EINVAL        # iters < 1
    assert L.landau_fp64_issue_probe(0, 16, None, None) == binding.LANDAU_EINVAL
    wl = inputs.config(1)
    for bad_batch in (0, 65536):
        with pytest.raises(binding.LandauError) as ei:
            binding.LandauContext(wl.mesh, wl.order, wl.species, bad_batch)
        assert ei.value.code == binding.LANDAU_EINVAL
    assert (binding.LANDAU_PAIR_AUTO, binding.LANDAU_PAIR_PER_PROBLEM, binding.LANDAU_PAIR_SHARED) == (0, 1, 2)
    hdr = open(os.path.join(os.path.dirname(__file__), "..", "include", "landau.h")).read()
    for name, val in (("LANDAU_PAIR_AUTO", 0), ("LANDAU_PAIR_PER_PROBLEM", 1), ("LANDAU_PAIR_SHARED", 2),
                      ("LANDAU_SHARED_MIN_BATCH", binding.LANDAU_SHARED_MIN_BATCH)):
        assert re.search(rf"#define {name} {val}\b", hdr), name
