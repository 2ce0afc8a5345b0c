"""Thin ctypes binding of include/landau.h -- argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; torch is used here only for
device memory and streams.  There is no fallback: if the shared library is missing or fails to
load, importing names from it raises.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, c_double, c_int, c_int32, c_int64, c_void_p

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblandau_b200.so")

LANDAU_OK, LANDAU_EINVAL, LANDAU_ENOMEM, LANDAU_ECUDA = 0, -1, -2, -3
LANDAU_PAIR_AUTO, LANDAU_PAIR_PER_PROBLEM, LANDAU_PAIR_SHARED = 0, 1, 2
LANDAU_BAND_AUTO, LANDAU_BAND_HULL, LANDAU_BAND_FRONT = 0, 1, 2
LANDAU_STATIC_SCRATCH_DOUBLES = 4 << 20      # landau_band_solve_static: doubles of the library's static device scratch
LANDAU_SHARED_MIN_BATCH = 4


class landau_mesh(ctypes.Structure):
    _fields_ = [("rmin", c_double), ("rmax", c_double), ("zmin", c_double), ("zmax", c_double),
                ("nbr", c_int32), ("nbz", c_int32), ("ncells", c_int32),
                ("level", POINTER(c_int32)), ("ir", POINTER(c_int32)), ("iz", POINTER(c_int32))]


class landau_species(ctypes.Structure):
    _fields_ = [("S", c_int32), ("mass", POINTER(c_double)), ("charge", POINTER(c_double)),
                ("density", POINTER(c_double)), ("temperature", POINTER(c_double)),
                ("m0", c_double), ("nu", c_double)]


_lib = None

# every symbol include/landau.h declares: name -> (restype, argtypes)
SIGNATURES = {
    "landau_create": (c_int, [POINTER(landau_mesh), c_int, POINTER(landau_species), c_int, POINTER(c_void_p)]),
    "landau_destroy": (c_int, [c_void_p]),
    "landau_create_multigrid": (c_int, [POINTER(landau_mesh), c_int, POINTER(c_int32), c_int, POINTER(landau_species), c_int,
                                        POINTER(c_void_p)]),
    "landau_grid_count": (c_int, [c_void_p, POINTER(c_int32)]),
    "landau_grid_sizes": (c_int, [c_void_p, c_int, POINTER(c_int32), POINTER(c_int32), POINTER(c_int64), POINTER(c_int64),
                                  POINTER(c_int64), POINTER(c_int64)]),
    "landau_strides": (c_int, [c_void_p, POINTER(c_int32), POINTER(c_int64), POINTER(c_int64), POINTER(c_int64), POINTER(c_int64)]),
    "landau_grid_csr_pattern": (c_int, [c_void_p, c_int, POINTER(c_void_p), POINTER(c_void_p)]),
    "landau_grid_csr_pattern_host": (c_int, [c_void_p, c_int, POINTER(c_int32), POINTER(c_int32)]),
    "landau_grid_dof_coords": (c_int, [c_void_p, c_int, POINTER(c_double), POINTER(c_double)]),
    "landau_setup_host": (c_int, [POINTER(landau_mesh), c_int, POINTER(c_int64), POINTER(c_int64), POINTER(c_int64),
                                  POINTER(c_int32), POINTER(c_int32), POINTER(c_double), POINTER(c_double)]),
    "landau_sizes": (c_int, [c_void_p, POINTER(c_int32), POINTER(c_int64), POINTER(c_int64), POINTER(c_int64), POINTER(c_int64)]),
    "landau_csr_pattern": (c_int, [c_void_p, POINTER(c_void_p), POINTER(c_void_p)]),
    "landau_csr_pattern_host": (c_int, [c_void_p, POINTER(c_int32), POINTER(c_int32)]),
    "landau_dof_coords": (c_int, [c_void_p, POINTER(c_double), POINTER(c_double)]),
    "landau_points": (c_int, [c_void_p, POINTER(c_double), POINTER(c_double), POINTER(c_double)]),
    "landau_inner_integral": (c_int, [c_void_p, c_int, c_void_p, c_void_p, c_void_p]),
    "landau_jacobian": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]),
    "landau_jacobian_batched": (c_int, [c_void_p, c_int, c_void_p, c_void_p, c_void_p, c_void_p]),
    "landau_mass": (c_int, [c_void_p, c_double, c_void_p, c_void_p]),
    "landau_implicit_operator_batched": (c_int, [c_void_p, c_int, c_void_p, c_void_p, c_double, c_void_p, c_void_p, c_void_p]),
    "landau_band_order_host": (c_int, [POINTER(landau_mesh), c_int, POINTER(c_int32), POINTER(c_int32), POINTER(c_int32), POINTER(c_double)]),
    "landau_band_sizes": (c_int, [c_void_p, c_int, POINTER(c_int32), POINTER(c_int64), POINTER(c_int64), POINTER(c_double)]),
    "landau_band_factor_batched": (c_int, [c_void_p, c_int, c_void_p, c_void_p, c_void_p, c_void_p]),
    "landau_band_solve_batched": (c_int, [c_void_p, c_int, c_void_p, c_void_p, c_void_p, c_void_p]),
    "landau_band_solve_static": (c_int, [c_void_p, c_int, c_void_p, c_void_p, c_void_p, c_void_p]),
    "landau_band_front_host": (c_int, [POINTER(landau_mesh), c_int, POINTER(c_int32), POINTER(c_double), POINTER(c_int32)]),
    "landau_band_set_method": (c_int, [c_void_p, c_int]),
    "landau_band_method": (c_int, [c_void_p, c_int, POINTER(c_int32), POINTER(c_int32), POINTER(c_double)]),
    "landau_jacobian_host": (c_int, [c_void_p, c_int, c_void_p, c_void_p, c_void_p]),
    "landau_launch_count": (c_int, [c_void_p, POINTER(c_int64)]),
    "landau_profile_enable": (c_int, [c_void_p, c_int]),
    "landau_profile_read": (c_int, [c_void_p, POINTER(c_double), POINTER(c_int64)]),
    "landau_fp64_peak_probe": (c_int, [c_int, POINTER(c_double), POINTER(c_double)]),
    "landau_fp64_issue_probe": (c_int, [c_int, c_int, POINTER(c_double), POINTER(c_double)]),
    "landau_set_pair_path": (c_int, [c_void_p, c_int]),
    "landau_pair_path": (c_int, [c_void_p, POINTER(c_int32), POINTER(c_int64)]),
    "landau_set_tensor_cache": (c_int, [c_void_p, c_int]),
    "landau_strerror": (ctypes.c_char_p, [c_int]),
    "landau_last_cuda_error": (ctypes.c_char_p, []),
}


def lib():
    """Loads liblandau_b200.so (built in-tree by paper_2104_10000_b200.build); raises if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2104_10000_b200.build` "
                               "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


class LandauError(RuntimeError):
    def __init__(self, code: int):
        L = lib()
        msg = L.landau_strerror(code).decode()
        detail = L.landau_last_cuda_error().decode()
        super().__init__(f"landau error {code}: {msg}" + (f" ({detail})" if detail else ""))
        self.code = code


def _check(code: int) -> None:
    if code != LANDAU_OK:
        raise LandauError(code)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _mesh_struct(mesh):
    lev, ir, iz = _i32(mesh.level), _i32(mesh.ir), _i32(mesh.iz)
    m = landau_mesh(float(mesh.rmin), float(mesh.rmax), float(mesh.zmin), float(mesh.zmax), int(mesh.nbr), int(mesh.nbz),
                    int(lev.shape[0]), lev.ctypes.data_as(POINTER(c_int32)), ir.ctypes.data_as(POINTER(c_int32)),
                    iz.ctypes.data_as(POINTER(c_int32)))
    return m, (lev, ir, iz)


def _dp(a):
    return a.ctypes.data_as(POINTER(c_double))


def landau_setup_host(mesh, order: int):
    """Host-only set-up: returns dict(n, nnz, N, rowptr, colidx, dof_r, dof_z).  No GPU needed."""
    L = lib()
    m, keep = _mesh_struct(mesh)
    n, nnz, N = c_int64(), c_int64(), c_int64()
    _check(L.landau_setup_host(ctypes.byref(m), order, ctypes.byref(n), ctypes.byref(nnz), ctypes.byref(N), None, None, None, None))
    rowptr, colidx = np.zeros(n.value + 1, np.int32), np.zeros(nnz.value, np.int32)
    dr, dz = np.zeros(n.value), np.zeros(n.value)
    _check(L.landau_setup_host(ctypes.byref(m), order, None, None, None, rowptr.ctypes.data_as(POINTER(c_int32)),
                               colidx.ctypes.data_as(POINTER(c_int32)), _dp(dr), _dp(dz)))
    return dict(n=n.value, nnz=nnz.value, N=N.value, rowptr=rowptr, colidx=colidx, dof_r=dr, dof_z=dz)


def landau_band_order_host(mesh, order: int):
    """Host-only: dict(perm, bw, block_columns, flop) of the band LU's order (best RCM start or sweep) for this mesh."""
    L = lib()
    m, keep = _mesh_struct(mesh)
    n = landau_setup_host(mesh, order)["n"]
    perm = np.zeros(n, np.int32)
    bw, kb, fl = c_int32(), c_int32(), c_double()
    _check(L.landau_band_order_host(ctypes.byref(m), order, perm.ctypes.data_as(POINTER(c_int32)), ctypes.byref(bw), ctypes.byref(kb),
                                    ctypes.byref(fl)))
    return dict(perm=perm, bw=bw.value, block_columns=kb.value, flop=fl.value)


def landau_band_front_host(mesh, order: int):
    """Host-only: dict(rows_max, flop, fits) of the front (envelope) factorisation for this mesh's band order."""
    L = lib()
    m, keep = _mesh_struct(mesh)
    r, fl, fits = c_int32(), c_double(), c_int32()
    _check(L.landau_band_front_host(ctypes.byref(m), order, ctypes.byref(r), ctypes.byref(fl), ctypes.byref(fits)))
    return dict(rows_max=r.value, flop=fl.value, fits=bool(fits.value))


def landau_fp64_peak_probe(iters: int = 1 << 16):
    L = lib()
    fl, mhz = c_double(), c_double()
    _check(L.landau_fp64_peak_probe(iters, ctypes.byref(fl), ctypes.byref(mhz)))
    return fl.value, mhz.value


def landau_fp64_issue_probe(mode: int, iters: int = 1 << 14):
    """(SM cycles per warp instruction and sub-partition, whole-GPU flop/s) of issue-rate probe `mode`."""
    L = lib()
    cyc, fl = c_double(), c_double()
    _check(L.landau_fp64_issue_probe(mode, iters, ctypes.byref(cyc), ctypes.byref(fl)))
    return cyc.value, fl.value


def _stream_ptr(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return c_void_p(s.cuda_stream)


class LandauContext:
    """Owns a landau_ctx.  Methods mirror the C entry points one to one (same names without the
    prefix); tensors are torch CUDA float64, contiguous."""

    def __init__(self, mesh, order: int, species, max_batch: int = 1, pair_path: int = LANDAU_PAIR_AUTO):
        L = lib()
        m, keep = _mesh_struct(mesh)
        mass, charge = _f64(species.mass), _f64(species.charge)
        dens, temp = _f64(species.density), _f64(species.temperature)
        sp = landau_species(int(mass.shape[0]), _dp(mass), _dp(charge), _dp(dens), _dp(temp), float(species.m0), float(species.nu))
        h = c_void_p()
        _check(L.landau_create(ctypes.byref(m), order, ctypes.byref(sp), int(max_batch), ctypes.byref(h)))
        self._h = h
        if pair_path != LANDAU_PAIR_AUTO:
            self.set_pair_path(pair_path)
        S, n, nnz, N, Ne = c_int32(), c_int64(), c_int64(), c_int64(), c_int64()
        _check(L.landau_sizes(h, ctypes.byref(S), ctypes.byref(n), ctypes.byref(nnz), ctypes.byref(N), ctypes.byref(Ne)))
        self.S, self.n, self.nnz, self.N, self.Ne = S.value, n.value, nnz.value, N.value, Ne.value
        self.max_batch = int(max_batch)

    def destroy(self):
        if getattr(self, "_h", None):
            lib().landau_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def set_pair_path(self, path: int):
        _check(lib().landau_set_pair_path(self._h, int(path)))

    def pair_path(self):
        """(path in use: LANDAU_PAIR_PER_PROBLEM or LANDAU_PAIR_SHARED, bytes of its scratch)."""
        p, b = c_int32(), c_int64()
        _check(lib().landau_pair_path(self._h, ctypes.byref(p), ctypes.byref(b)))
        return p.value, b.value

    def set_tensor_cache(self, on: bool):
        _check(lib().landau_set_tensor_cache(self._h, int(bool(on))))

    def csr_pattern_host(self):
        rowptr, colidx = np.zeros(self.n + 1, np.int32), np.zeros(self.nnz, np.int32)
        _check(lib().landau_csr_pattern_host(self._h, rowptr.ctypes.data_as(POINTER(c_int32)), colidx.ctypes.data_as(POINTER(c_int32))))
        return rowptr, colidx

    def csr_pattern(self):
        """Device pointers (ints) of rowptr/colidx owned by the ctx."""
        a, b = c_void_p(), c_void_p()
        _check(lib().landau_csr_pattern(self._h, ctypes.byref(a), ctypes.byref(b)))
        return a.value, b.value

    def dof_coords(self):
        r, z = np.zeros(self.n), np.zeros(self.n)
        _check(lib().landau_dof_coords(self._h, _dp(r), _dp(z)))
        return r, z

    def points(self):
        r, z, w = np.zeros(self.N), np.zeros(self.N), np.zeros(self.N)
        _check(lib().landau_points(self._h, _dp(r), _dp(z), _dp(w)))
        return r, z, w

    @staticmethod
    def _ptr(t, shape):
        import torch
        assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == tuple(shape), (t.shape, shape)
        return c_void_p(t.data_ptr())

    def inner_integral(self, f, G, stream=None):
        nb = f.shape[0]
        _check(lib().landau_inner_integral(self._h, nb, self._ptr(f, (nb, self.S, self.n)), self._ptr(G, (nb, 5, self.N)), _stream_ptr(stream)))

    def jacobian(self, f, vals=None, Cf=None, stream=None):
        pv = self._ptr(vals, (self.S, self.nnz)) if vals is not None else None
        pc = self._ptr(Cf, (self.S, self.n)) if Cf is not None else None
        _check(lib().landau_jacobian(self._h, self._ptr(f, (self.S, self.n)), pv, pc, _stream_ptr(stream)))

    def jacobian_batched(self, f, vals=None, Cf=None, stream=None):
        nb = f.shape[0]
        pv = self._ptr(vals, (nb, self.S, self.nnz)) if vals is not None else None
        pc = self._ptr(Cf, (nb, self.S, self.n)) if Cf is not None else None
        _check(lib().landau_jacobian_batched(self._h, nb, self._ptr(f, (nb, self.S, self.n)), pv, pc, _stream_ptr(stream)))

    def mass(self, shift, mvals, stream=None):
        _check(lib().landau_mass(self._h, float(shift), self._ptr(mvals, (self.nnz,)), _stream_ptr(stream)))

    def implicit_operator_batched(self, f, Ez, shift, vals=None, F=None, stream=None):
        nb = f.shape[0]
        pv = self._ptr(vals, (nb, self.S, self.nnz)) if vals is not None else None
        pf = self._ptr(F, (nb, self.S, self.n)) if F is not None else None
        _check(lib().landau_implicit_operator_batched(self._h, nb, self._ptr(f, (nb, self.S, self.n)), self._ptr(Ez, (nb,)),
                                                      float(shift), pv, pf, _stream_ptr(stream)))

    def band_sizes(self, grid=0):
        """(half-bandwidth of the band order, doubles per matrix, workspace doubles per problem)."""
        bw, md, ws, fl = c_int32(), c_int64(), c_int64(), c_double()
        _check(lib().landau_band_sizes(self._h, grid, ctypes.byref(bw), ctypes.byref(md), ctypes.byref(ws), ctypes.byref(fl)))
        self.band_flop_per_factorization = fl.value
        return bw.value, md.value, ws.value

    def band_set_method(self, method):
        """LANDAU_BAND_AUTO / _HULL / _FRONT: which kernel factors the band (include/landau.h)."""
        _check(lib().landau_band_set_method(self._h, int(method)))

    def band_method(self, grid=0):
        """(kernel in use for the grid: LANDAU_BAND_HULL or _FRONT, rows of the largest front beside its block)."""
        m, r, fl = c_int32(), c_int32(), c_double()
        _check(lib().landau_band_method(self._h, grid, ctypes.byref(m), ctypes.byref(r), ctypes.byref(fl)))
        self.band_flop_in_use = fl.value
        return m.value, r.value

    def band_factor_batched(self, vals, band, pivots=None, stream=None):
        """pivots: None or a CUDA float64 tensor [nb][S][2] receiving (min |pivot|, max |pivot|) per matrix."""
        nb = vals.shape[0]
        assert band.is_cuda and band.is_contiguous() and band.numel() >= nb * self.band_sizes()[2]
        pp = self._ptr(pivots, (nb, self.S, 2)) if pivots is not None else None
        _check(lib().landau_band_factor_batched(self._h, nb, c_void_p(vals.data_ptr()), c_void_p(band.data_ptr()), pp, _stream_ptr(stream)))

    def band_solve_batched(self, band, rhs, x, stream=None):
        nb = rhs.shape[0]
        _check(lib().landau_band_solve_batched(self._h, nb, c_void_p(band.data_ptr()), c_void_p(rhs.data_ptr()),
                                               c_void_p(x.data_ptr()), _stream_ptr(stream)))

    def band_solve_static(self, band, rhs, x, stream=None):
        """landau_band_solve_static: the solve with its vectors in the library's static device scratch (no allocation)."""
        nb = rhs.shape[0]
        _check(lib().landau_band_solve_static(self._h, nb, c_void_p(band.data_ptr()), c_void_p(rhs.data_ptr()),
                                              c_void_p(x.data_ptr()), _stream_ptr(stream)))

    def jacobian_host(self, f_host, vals_host=None, Cf_host=None):
        """Host buffers: numpy arrays or pinned CPU torch tensors (float64, contiguous)."""
        def hp(a):
            if a is None:
                return None
            return c_void_p(a.ctypes.data if isinstance(a, np.ndarray) else a.data_ptr())
        nb = f_host.shape[0]
        _check(lib().landau_jacobian_host(self._h, nb, hp(f_host), hp(vals_host), hp(Cf_host)))

    def profile_enable(self, on: bool = True):
        _check(lib().landau_profile_enable(self._h, int(bool(on))))

    def profile_read(self):
        """([ms of the tensor evaluation, ms of the batch-shared contraction], [launches of each]) since the last read."""
        ms, cnt = (c_double * 2)(), (c_int64 * 2)()
        _check(lib().landau_profile_read(self._h, ms, cnt))
        return [ms[0], ms[1]], [cnt[0], cnt[1]]

    def launch_count(self) -> int:
        c = c_int64()
        _check(lib().landau_launch_count(self._h, ctypes.byref(c)))
        return c.value


class LandauMultigridContext:
    """landau_create_multigrid: species clustered on several grids.  Per-problem layouts are flat:
    f, Cf, F: [nb][f_stride] (species after species, each with the n of its grid), vals: [nb][vals_stride],
    mvals: [mvals_size]; `species_slices()` / `vals_slices()` give each species' range."""

    def __init__(self, meshes, species_grid, order: int, species, max_batch: int = 1):
        L = lib()
        structs, keep = [], []
        for m in meshes:
            st, k = _mesh_struct(m)
            structs.append(st); keep.append(k)
        arr = (landau_mesh * len(meshes))(*structs)
        sg = _i32(species_grid)
        mass, charge = _f64(species.mass), _f64(species.charge)
        dens, temp = _f64(species.density), _f64(species.temperature)
        sp = landau_species(int(mass.shape[0]), _dp(mass), _dp(charge), _dp(dens), _dp(temp), float(species.m0), float(species.nu))
        h = c_void_p()
        _check(L.landau_create_multigrid(arr, len(meshes), sg.ctypes.data_as(POINTER(c_int32)), order, ctypes.byref(sp),
                                         int(max_batch), ctypes.byref(h)))
        self._h = h
        S, fs, vs, ms, Nt = c_int32(), c_int64(), c_int64(), c_int64(), c_int64()
        _check(L.landau_strides(h, ctypes.byref(S), ctypes.byref(fs), ctypes.byref(vs), ctypes.byref(ms), ctypes.byref(Nt)))
        self.S, self.f_stride, self.vals_stride, self.mvals_size, self.N = S.value, fs.value, vs.value, ms.value, Nt.value
        ng = c_int32()
        _check(L.landau_grid_count(h, ctypes.byref(ng)))
        self.grids = []
        for g in range(ng.value):
            Sg, s0, n, nnz, N, Ne = c_int32(), c_int32(), c_int64(), c_int64(), c_int64(), c_int64()
            _check(L.landau_grid_sizes(h, g, ctypes.byref(Sg), ctypes.byref(s0), ctypes.byref(n), ctypes.byref(nnz), ctypes.byref(N), ctypes.byref(Ne)))
            self.grids.append(dict(S=Sg.value, first_species=s0.value, n=n.value, nnz=nnz.value, N=N.value, Ne=Ne.value))
        self.species_grid = [int(g) for g in sg]
        self.max_batch = int(max_batch)

    destroy = LandauContext.destroy
    __del__ = LandauContext.__del__
    _ptr = staticmethod(LandauContext._ptr)
    launch_count = LandauContext.launch_count
    set_pair_path = LandauContext.set_pair_path
    pair_path = LandauContext.pair_path
    set_tensor_cache = LandauContext.set_tensor_cache
    band_sizes = LandauContext.band_sizes
    band_factor_batched = LandauContext.band_factor_batched
    band_solve_batched = LandauContext.band_solve_batched
    band_solve_static = LandauContext.band_solve_static

    def species_slices(self):
        out, o = [], 0
        for a in range(self.S):
            n = self.grids[self.species_grid[a]]["n"]
            out.append(slice(o, o + n)); o += n
        return out

    def vals_slices(self):
        out, o = [], 0
        for a in range(self.S):
            n = self.grids[self.species_grid[a]]["nnz"]
            out.append(slice(o, o + n)); o += n
        return out

    def grid_dof_coords(self, g):
        n = self.grids[g]["n"]
        r, z = np.zeros(n), np.zeros(n)
        _check(lib().landau_grid_dof_coords(self._h, g, _dp(r), _dp(z)))
        return r, z

    def grid_csr_pattern_host(self, g):
        rowptr, colidx = np.zeros(self.grids[g]["n"] + 1, np.int32), np.zeros(self.grids[g]["nnz"], np.int32)
        _check(lib().landau_grid_csr_pattern_host(self._h, g, rowptr.ctypes.data_as(POINTER(c_int32)), colidx.ctypes.data_as(POINTER(c_int32))))
        return rowptr, colidx

    def jacobian_batched(self, f, vals=None, Cf=None, stream=None):
        nb = f.shape[0]
        pv = self._ptr(vals, (nb, self.vals_stride)) if vals is not None else None
        pc = self._ptr(Cf, (nb, self.f_stride)) if Cf is not None else None
        _check(lib().landau_jacobian_batched(self._h, nb, self._ptr(f, (nb, self.f_stride)), pv, pc, _stream_ptr(stream)))

    def implicit_operator_batched(self, f, Ez, shift, vals=None, F=None, stream=None):
        nb = f.shape[0]
        pv = self._ptr(vals, (nb, self.vals_stride)) if vals is not None else None
        pf = self._ptr(F, (nb, self.f_stride)) if F is not None else None
        _check(lib().landau_implicit_operator_batched(self._h, nb, self._ptr(f, (nb, self.f_stride)), self._ptr(Ez, (nb,)),
                                                      float(shift), pv, pf, _stream_ptr(stream)))

    def mass(self, shift, mvals, stream=None):
        _check(lib().landau_mass(self._h, float(shift), self._ptr(mvals, (self.mvals_size,)), _stream_ptr(stream)))
