"""CPU oracle for the GSPM hot path (TEST INFRASTRUCTURE ONLY).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
may import this package.  It never imports the CUDA binding (paper_2510_09812_b200.binding)
and shares no code with it; `cm_oracle.c` is the implementation, this file only compiles
it with gcc and marshals numpy arrays through ctypes.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "cm_oracle.c"

ORC_E_BREAKDOWN = -6
ORC_W_MAXITER = -7

MAT_K_MS, MAT_K_GS1, MAT_K_GS2, MAT_MASS, MAT_K_MECH, MAT_K_FREE, MAT_K_M, MAT_K_MECH_FREE = range(8)


def lib_path(dtype: str) -> Path:
    return _HERE / f"liboracle_{dtype}.so"


def build(force: bool = False) -> None:
    """gcc -O2 -fopenmp, once per precision.  No -ffast-math, no -march (no FMA contraction)."""
    for dtype, flag in (("f64", []), ("f32", ["-DORC_F32"])):
        out = lib_path(dtype)
        if not force and out.exists() and out.stat().st_mtime >= _SRC.stat().st_mtime:
            continue
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-ffp-contract=off", *flag,
               str(_SRC), "-o", str(out), "-lm"]
        subprocess.run(cmd, check=True)


class _Material(C.Structure):
    _fields_ = [("Ms", C.c_double), ("Aex", C.c_double), ("K1", C.c_double), ("lambda100", C.c_double),
                ("lambda111", C.c_double), ("alpha", C.c_double), ("gamma", C.c_double),
                ("length_scale", C.c_double), ("Nd", C.c_double * 9), ("n_elastic", C.c_int),
                ("C_voigt", C.POINTER(C.c_double)), ("R", C.c_double * 9), ("sigma_ext", C.c_double * 6)]


class _StepParams(C.Structure):
    _fields_ = [("dt", C.c_double), ("Hext", C.c_double * 3), ("terms", C.c_uint), ("gspm_variant", C.c_int),
                ("cg_tol", C.c_double), ("cg_maxiter", C.c_int), ("cg_fixed_iters", C.c_int), ("cg_precond", C.c_int)]


class StepInfo(C.Structure):
    _fields_ = [("it_ms", C.c_int), ("it_mech", C.c_int), ("it_gs", C.c_int * 8), ("res_ms", C.c_double),
                ("res_mech", C.c_double), ("res_gs", C.c_double * 8), ("mbar", C.c_double * 3),
                ("mean_dm", C.c_double), ("energy", C.c_double)]


class _HystParams(C.Structure):
    _fields_ = [("H0", C.c_double * 3), ("dH", C.c_double * 3), ("conv_tol", C.c_double), ("max_fields", C.c_int),
                ("max_steps", C.c_int)]


class HystResult(C.Structure):
    _fields_ = [("n_fields", C.c_int), ("reversed", C.c_int), ("total_steps", C.c_long)]


_libs = {}


def _lib(dtype: str):
    if dtype not in _libs:
        build()
        L = C.CDLL(str(lib_path(dtype)))
        L.orc_scalar.restype = C.c_double
        L.orc_energy.restype = C.c_double
        L.orc_nnz.restype = C.c_long
        for name in ("orc_scalar", "orc_nnz", "orc_get", "orc_get_values", "orc_spmv", "orc_cg", "orc_volume_average",
                     "orc_rhs_ms", "orc_demag_field", "orc_rhs_mech", "orc_stress_recover", "orc_field", "orc_energy",
                     "orc_gspm_step", "orc_rhs_gs", "orc_destroy", "orc_create_wrapped", "orc_periodic_wrap", "orc_hysteresis_run", "orc_voigt_rotation", "orc_create_hex", "orc_cg_pc", "orc_set_cg_history"):
            getattr(L, name).argtypes = None
        _libs[dtype] = L
    return _libs[dtype]


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def reorder(xyz, tets, method: int):
    """(order[new]=old, iperm[old]=new, relabelled+sorted tets, tet_order[new]=old)"""
    L = _lib("f64")
    xyz = np.ascontiguousarray(xyz, np.float64)
    tets = np.ascontiguousarray(tets, np.int32)
    n, ne = xyz.shape[0], tets.shape[0]
    order = np.empty(n, np.int32); iperm = np.empty(n, np.int32)
    tnew = np.empty((ne, 4), np.int32); torder = np.empty(ne, np.int32)
    rc = L.orc_reorder(_p(xyz), C.c_long(n), _p(tets), C.c_long(ne), C.c_int(method), _p(order), _p(iperm), _p(tnew), _p(torder))
    if rc:
        raise RuntimeError(f"orc_reorder rc={rc}")
    return order, iperm, tnew, torder


def periodic_wrap(xyz, axes: int, rel_tol: float = 1e-9):
    """dof_of_node (int32, n_nodes) and n_dof for the periodic directions in the bit mask `axes`."""
    L = _lib("f64")
    xyz = np.ascontiguousarray(xyz, np.float64)
    n = xyz.shape[0]
    dof = np.empty(n, np.int32)
    nd = C.c_long()
    rc = L.orc_periodic_wrap(_p(xyz), C.c_long(n), C.c_uint(axes), C.c_double(rel_tol), _p(dof), C.byref(nd))
    if rc:
        raise RuntimeError(f"orc_periodic_wrap rc={rc}")
    return dof, int(nd.value)


def voigt_rotation(R):
    """Eq. D.3: 6x6 M with sigma_sim = M sigma_crystal."""
    L = _lib("f64")
    R = np.ascontiguousarray(R, np.float64).reshape(9)
    M = np.zeros(36)
    L.orc_voigt_rotation(_p(R), _p(M))
    return M.reshape(6, 6)


class Oracle:
    """One mesh + material + dt, in the node order it is given (no reordering)."""

    def __init__(self, mesh, material, dt, clamp_dof=None, pin_node=0, dtype="f64", dof_of_node=None, n_dof=None):
        """mesh: inputs.Mesh (linear tetrahedra) or inputs.HexMesh (linear hexahedra, R26); dof_of_node / n_dof: periodic wrap (R23)."""
        self.dtype = dtype
        self.real = np.float64 if dtype == "f64" else np.float32
        self.L = _lib(dtype)
        assert self.L.orc_sizeof_real() == np.dtype(self.real).itemsize
        self.Ng, self.Ne = mesh.n_nodes, mesh.n_tets
        self.N = self.Ng if dof_of_node is None else int(n_dof)       # degrees of freedom
        dof = None if dof_of_node is None else np.ascontiguousarray(dof_of_node, np.int32)
        xyz = np.ascontiguousarray(mesh.xyz, np.float64)
        tets = None if hasattr(mesh, "hexes") else np.ascontiguousarray(mesh.tets, np.int32)
        mag = np.ascontiguousarray(mesh.magnetic, np.uint8)
        eid = np.ascontiguousarray(mesh.elastic_id, np.int32)
        self._Cv = np.ascontiguousarray(material.C_voigt, np.float64).reshape(-1, 36) if material.C_voigt is not None else None
        m = _Material(material.Ms, material.Aex, material.K1, material.lambda100, material.lambda111, material.alpha,
                      material.gamma, material.length_scale, (C.c_double * 9)(*material.Nd),
                      0 if self._Cv is None else self._Cv.shape[0],
                      None if self._Cv is None else self._Cv.ctypes.data_as(C.POINTER(C.c_double)),
                      (C.c_double * 9)(*(np.zeros(9) if getattr(material, "R", None) is None else np.asarray(material.R, float).ravel())),
                      (C.c_double * 6)(*(np.zeros(6) if getattr(material, "sigma_ext", None) is None else np.asarray(material.sigma_ext, float).ravel())))
        clamp = None if clamp_dof is None else np.ascontiguousarray(clamp_dof, np.uint8)
        h = C.c_void_p()
        self.is_hex = hasattr(mesh, "hexes")
        if self.is_hex:
            hexes = np.ascontiguousarray(mesh.hexes, np.int32)
            rc = self.L.orc_create_hex(_p(xyz), C.c_long(self.Ng), _p(hexes), C.c_long(self.Ne), _p(mag), _p(eid), _p(dof),
                                       C.c_long(self.N), C.byref(m), C.c_double(dt), _p(clamp), C.c_long(pin_node), C.byref(h))
        else:
            rc = self.L.orc_create_wrapped(_p(xyz), C.c_long(self.Ng), _p(tets), C.c_long(self.Ne), _p(mag), _p(eid), _p(dof),
                                           C.c_long(self.N), C.byref(m), C.c_double(dt), _p(clamp), C.c_long(pin_node), C.byref(h))
        if rc:
            raise RuntimeError(f"orc_create rc={rc}")
        self.h = h
        self.nnz = self.L.orc_nnz(self.h)
        self.Ms = material.Ms

    def __del__(self):
        if getattr(self, "h", None):
            self.L.orc_destroy(self.h)
            self.h = None

    # ---- accessors -------------------------------------------------------------------
    def scalar(self, what):
        return self.L.orc_scalar(self.h, C.c_int(what))

    @property
    def Vtot(self): return self.scalar(0)
    @property
    def Vmag(self): return self.scalar(1)
    @property
    def Astar(self): return self.scalar(2)
    @property
    def Kstar(self): return self.scalar(3)
    @property
    def dtau(self): return self.scalar(4)

    def _get(self, what, shape, dt):
        a = np.empty(shape, dt)
        rc = self.L.orc_get(self.h, C.c_int(what), _p(a))
        assert rc == 0
        return a

    def rowptr(self): return self._get(0, self.N + 1, np.int32)
    def colidx(self): return self._get(1, self.nnz, np.int32)
    def n2e_ptr(self): return self._get(2, self.N + 1, np.int32)
    def n2e(self): return self._get(3, self.Ne * (8 if self.is_hex else 4), np.int32)
    def V(self): return self._get(4, self.Ne, self.real)
    def G(self): return self._get(5, (self.Ne, 4, 3), self.real)
    def mL(self): return self._get(6, self.N, self.real)
    def mLm(self): return self._get(7, self.N, self.real)
    def live(self): return self._get(8, self.N, np.uint8)

    def values(self, mat):
        shape = (self.nnz, 3, 3) if mat in (MAT_K_MECH, MAT_K_MECH_FREE) else (self.nnz,)
        a = np.empty(shape, self.real)
        rc = self.L.orc_get_values(self.h, C.c_int(mat), _p(a))
        assert rc == 0
        return a

    def csr(self, mat):
        """scipy matrix of a scalar (CSR) or block (BSR) matrix -- for tests."""
        import scipy.sparse as sp
        v = self.values(mat).astype(np.float64)
        if v.ndim == 1:
            return sp.csr_matrix((v, self.colidx(), self.rowptr()), shape=(self.N, self.N))
        return sp.bsr_matrix((v, self.colidx(), self.rowptr()), shape=(3 * self.N, 3 * self.N)).tocsr()

    # ---- operations ------------------------------------------------------------------
    def _r(self, a):
        return np.ascontiguousarray(a, self.real)

    def spmv(self, mat, x):
        x = self._r(x); y = np.empty_like(x)
        rc = self.L.orc_spmv(self.h, C.c_int(mat), _p(x), _p(y)); assert rc == 0
        return y

    def cg(self, mat, b, x0=None, tol=1e-7, maxiter=100000, fixed=-1):
        b = self._r(b)
        x = np.zeros_like(b) if x0 is None else self._r(x0).copy()
        it = C.c_int(); res = C.c_double()
        rc = self.L.orc_cg(self.h, C.c_int(mat), _p(b), _p(x), C.c_double(tol), C.c_int(maxiter), C.c_int(fixed),
                           C.byref(it), C.byref(res))
        return x, it.value, res.value, rc

    def cg_pc(self, mat, b, x0=None, tol=1e-7, maxiter=100000, fixed=-1, precond=1):
        """Jacobi-preconditioned CG (precond = 1; 0 = plain CG through the same routine)."""
        b = self._r(b)
        x = np.zeros_like(b) if x0 is None else self._r(x0).copy()
        it = C.c_int(); res = C.c_double()
        rc = self.L.orc_cg_pc(self.h, C.c_int(mat), _p(b), _p(x), C.c_double(tol), C.c_int(maxiter), C.c_int(fixed),
                              C.c_int(precond), C.byref(it), C.byref(res))
        return x, it.value, res.value, rc

    def cg_history(self, mat, b, x0=None, tol=1e-7, maxiter=100000, precond=0, cap=1 << 16):
        """(x, iters, history): history[k] = ||r_k|| / ||b|| before iteration k, k = 0 .. iters."""
        hist = np.zeros(cap); n = C.c_int()
        self.L.orc_set_cg_history(_p(hist), C.c_int(cap), C.byref(n))
        try:
            x, it, res, rc = self.cg_pc(mat, b, x0, tol, maxiter, -1, precond)
        finally:
            self.L.orc_set_cg_history(None, C.c_int(0), None)
        return x, it, hist[:n.value].copy()

    def volume_average(self, g):
        g = self._r(g)
        nc = 1 if g.ndim == 1 else g.shape[1]
        out = np.empty(nc, np.float64)
        rc = self.L.orc_volume_average(self.h, _p(g), C.c_int(nc), _p(out)); assert rc == 0
        return out

    def rhs_ms(self, m, mbar=None):
        m = self._r(m)
        mbar = self.volume_average(m) if mbar is None else np.ascontiguousarray(mbar, np.float64)
        b = np.empty(self.N, self.real)
        rc = self.L.orc_rhs_ms(self.h, _p(m), _p(mbar), _p(b)); assert rc == 0
        return b

    def demag_field(self, U, mbar, terms):
        U = self._r(U); mbar = np.ascontiguousarray(mbar, np.float64)
        hd = np.empty((self.N, 3), self.real); gm = np.empty(3, np.float64)
        rc = self.L.orc_demag_field(self.h, _p(U), _p(mbar), C.c_uint(terms), _p(hd), _p(gm)); assert rc == 0
        return hd, gm

    def rhs_mech(self, m):
        m = self._r(m); b = np.empty((self.N, 3), self.real)
        rc = self.L.orc_rhs_mech(self.h, _p(m), _p(b)); assert rc == 0
        return b

    def stress_recover(self, u, w):
        u = self._r(u); w = self._r(w); s = np.empty((self.N, 6), self.real)
        rc = self.L.orc_stress_recover(self.h, _p(u), _p(w), _p(s)); assert rc == 0
        return s

    def field(self, w, hd, sig, hext_nd, terms):
        w = self._r(w)
        hd = self._r(np.zeros((self.N, 3)) if hd is None else hd)
        sig = self._r(np.zeros((self.N, 6)) if sig is None else sig)
        hext = np.ascontiguousarray(hext_nd, np.float64)
        h = np.empty((self.N, 3), self.real)
        rc = self.L.orc_field(self.h, _p(w), _p(hd), _p(sig), _p(hext), C.c_uint(terms), _p(h)); assert rc == 0
        return h

    def rhs_gs(self, f):
        f = self._r(f); b = np.empty_like(f)
        rc = self.L.orc_rhs_gs(self.h, _p(f), _p(b)); assert rc == 0
        return b

    def energy(self, m, U, u, hext_nd, terms):
        m = self._r(m)
        U = self._r(np.zeros(self.N) if U is None else U)
        u = self._r(np.zeros((self.N, 3)) if u is None else u)
        hext = np.ascontiguousarray(hext_nd, np.float64)
        return self.L.orc_energy(self.h, _p(m), _p(U), _p(u), _p(hext), C.c_uint(terms))

    def gspm_step(self, m, U, u, dt, Hext, terms, variant=0, cg_tol=1e-7, cg_maxiter=100000, cg_fixed_iters=-1, cg_precond=0):
        """In-place on m (N,3), U (N,), u (N,3) arrays of self.real dtype.  Returns (StepInfo, rc)."""
        for a in (m, U, u):
            assert a.dtype == self.real and a.flags.c_contiguous
        p = _StepParams(dt, (C.c_double * 3)(*Hext), terms, variant, cg_tol, cg_maxiter, cg_fixed_iters, cg_precond)
        info = StepInfo()
        rc = self.L.orc_gspm_step(self.h, C.byref(p), _p(m), _p(U), _p(u), C.byref(info))
        return info, rc

    def hysteresis_run(self, m, U, u, dt, H0, dH, terms, conv_tol=5e-10, max_fields=100, max_steps=100000, variant=0,
                       cg_tol=1e-7, cg_maxiter=100000, cg_fixed_iters=-1):
        """in place on m, U, u.  Returns (H_log, mbar_log, steps_log, HystResult, rc), logs cut to n_fields."""
        for a in (m, U, u):
            assert a.dtype == self.real and a.flags.c_contiguous
        p = _StepParams(dt, (C.c_double * 3)(0, 0, 0), terms, variant, cg_tol, cg_maxiter, cg_fixed_iters, 0)
        hp = _HystParams((C.c_double * 3)(*H0), (C.c_double * 3)(*dH), conv_tol, max_fields, max_steps)
        Hl = np.zeros((max_fields, 3)); ml = np.zeros((max_fields, 3)); sl = np.zeros(max_fields, np.int32)
        res = HystResult()
        rc = self.L.orc_hysteresis_run(self.h, C.byref(p), C.byref(hp), _p(m), _p(U), _p(u), _p(Hl), _p(ml), _p(sl), C.byref(res))
        n = res.n_fields
        return Hl[:n], ml[:n], sl[:n], res, rc
