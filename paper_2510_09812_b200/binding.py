"""Thin ctypes binding of the C ABI in include/cupymag_b200.h (argument marshalling only).

Every step of the hot path runs inside libcupymag_b200.so; PyTorch is used for device memory
(`tensor.data_ptr()`) and streams only.  There is no CPU fallback: if the shared library is missing or
no CUDA device is present, the calls fail loudly.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path
from typing import Optional

import numpy as np

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libcupymag_b200.so"

CM_F64, CM_F32 = 0, 1
CM_REORDER_NONE, CM_REORDER_MORTON, CM_REORDER_RCM, CM_REORDER_MORTON_SORTED = 0, 1, 2, 3
CM_MAT_K_MS, CM_MAT_K_GS1, CM_MAT_K_GS2, CM_MAT_MASS, CM_MAT_K_MECH = range(5)
CM_RHS_MS, CM_RHS_MECH, CM_RHS_GS, CM_OUT_HD, CM_OUT_SIGMA, CM_OUT_FIELD = range(6)
CM_TERM_ANIS, CM_TERM_ZEEMAN, CM_TERM_DEMAG, CM_TERM_FARFIELD, CM_TERM_MAGEL = 1, 2, 4, 8, 16
CM_OK, CM_E_BADARG, CM_E_DEGENERATE_TET, CM_E_INDEX_RANGE, CM_E_ALLOC, CM_E_CUDA, CM_E_CG_BREAKDOWN, CM_E_CG_MAXITER = \
    0, -1, -2, -3, -4, -5, -6, -7
(CM_GET_COUNTS, CM_GET_ORDER, CM_GET_IPERM, CM_GET_TETS, CM_GET_TET_ORDER, CM_GET_ROWPTR, CM_GET_COLIDX, CM_GET_N2E_PTR,
 CM_GET_N2E) = range(9)
CM_GET_LAYOUT = 9
CM_PC_NONE, CM_PC_JACOBI = 0, 1
CM_NOALLOC_MAX_NODES = 16777216
CM_OPT_STORED_GEOMETRY, CM_OPT_NO_FUSED_S5S8 = 0, 1
CM_PROF_CG_MS, CM_PROF_CG_MECH, CM_PROF_CG_GS, CM_PROF_SPMV, CM_PROF_ELEMENT, CM_PROF_POINTWISE, CM_PROF_NCLASS = range(7)
PROF_NAMES = ("cg_ms", "cg_mech", "cg_gs", "spmv", "element", "pointwise")

EXPORTS = ("cm_mesh_create", "cm_mesh_create_hex", "cm_mesh_create_hex_wrapped", "cm_mesh_create_wrapped", "cm_periodic_wrap", "cm_mesh_destroy", "cm_mesh_get", "cm_assemble_csr", "cm_system_destroy", "cm_system_get_values",
           "cm_system_get_geometry", "cm_spmv", "cm_spmv3", "cm_cg_solve", "cm_cg_solve3", "cm_cg_solve_pc", "cm_cg_solve3_pc", "cm_cg_history_enable", "cm_cg_history", "cm_spmv_matfree", "cm_cg_solve_matfree", "cm_field_rhs", "cm_volume_average", "cm_volume_average_noalloc",
           "cm_gspm_step", "cm_gspm_step_host", "cm_hysteresis_run", "cm_system_set_option", "cm_profile_enable", "cm_profile_get", "cm_profile_reset", "cm_last_error",
           "cm_version")


class CmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"cupymag_b200 error {code}: {msg}")
        self.code = code


class cm_material(C.Structure):
    _fields_ = [("Ms", C.c_double), ("Aex", C.c_double), ("K1", C.c_double), ("lambda100", C.c_double),
                ("lambda111", C.c_double), ("alpha", C.c_double), ("gamma", C.c_double), ("length_scale", C.c_double),
                ("Nd", C.c_double * 9), ("n_elastic", C.c_int), ("C_voigt", C.POINTER(C.c_double)), ("R", C.c_double * 9),
                ("sigma_ext", C.c_double * 6)]


class cm_step_params(C.Structure):
    _fields_ = [("dt", C.c_double), ("Hext", C.c_double * 3), ("terms", C.c_uint), ("gspm_variant", C.c_int),
                ("cg_tol", C.c_double), ("cg_maxiter", C.c_int), ("cg_fixed_iters", C.c_int), ("cg_precond", C.c_int),
                ("mech_matfree", C.c_int)]


class cm_step_info(C.Structure):
    _fields_ = [("it_ms", C.c_int), ("it_mech", C.c_int), ("it_gs", C.c_int * 8), ("res_ms", C.c_double),
                ("res_mech", C.c_double), ("res_gs", C.c_double * 8), ("mbar", C.c_double * 3), ("mean_dm", C.c_double),
                ("energy", C.c_double)]


class cm_hyst_params(C.Structure):
    _fields_ = [("H0", C.c_double * 3), ("dH", C.c_double * 3), ("conv_tol", C.c_double), ("max_fields", C.c_int),
                ("max_steps", C.c_int)]


class cm_hyst_result(C.Structure):
    _fields_ = [("n_fields", C.c_int), ("reversed", C.c_int), ("total_steps", C.c_long), ("cg_iters_ms", C.c_long),
                ("cg_iters_mech", C.c_long), ("cg_passes_gs", C.c_long), ("worst_cg_status", C.c_int), ("device_ms", C.c_double)]


class cm_profile(C.Structure):
    _fields_ = [("ms", C.c_double * CM_PROF_NCLASS), ("launches", C.c_long * CM_PROF_NCLASS),
                ("cg_iters", C.c_long * CM_PROF_NCLASS), ("cg_matrix_passes", C.c_long * CM_PROF_NCLASS)]


_lib = None


def lib():
    """Loads the shared library (building it first if the sources are newer and nvcc is available)."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise CmError(CM_E_CUDA, f"{LIB_PATH} is missing: run `python -m paper_2510_09812_b200.build` "
                                     "(there is no CPU fallback)")
        L = C.CDLL(str(LIB_PATH))
        vp, lg, it, db = C.c_void_p, C.c_long, C.c_int, C.c_double
        L.cm_mesh_create.argtypes = [vp, lg, vp, lg, vp, vp, it, vp, C.POINTER(vp)]
        L.cm_mesh_create_wrapped.argtypes = [vp, lg, vp, lg, vp, vp, vp, lg, it, vp, C.POINTER(vp)]
        L.cm_mesh_create_hex.argtypes = [vp, lg, vp, lg, vp, vp, it, vp, C.POINTER(vp)]
        L.cm_mesh_create_hex_wrapped.argtypes = [vp, lg, vp, lg, vp, vp, vp, lg, it, vp, C.POINTER(vp)]
        L.cm_periodic_wrap.argtypes = [vp, lg, C.c_uint, db, vp, C.POINTER(lg)]
        L.cm_mesh_destroy.argtypes = [vp]
        L.cm_mesh_get.argtypes = [vp, it, vp, lg]
        L.cm_assemble_csr.argtypes = [vp, C.POINTER(cm_material), it, db, vp, lg, vp, C.POINTER(vp)]
        L.cm_system_destroy.argtypes = [vp]
        L.cm_system_get_values.argtypes = [vp, it, vp, lg]
        L.cm_system_get_geometry.argtypes = [vp, it, vp, lg]
        L.cm_spmv.argtypes = [vp, it, vp, vp, vp]
        L.cm_spmv3.argtypes = [vp, it, vp, vp, vp]
        L.cm_cg_solve.argtypes = [vp, it, vp, vp, db, it, it, C.POINTER(it), C.POINTER(db), vp]
        L.cm_cg_solve3.argtypes = [vp, it, vp, vp, db, it, it, C.POINTER(it), C.POINTER(db), vp]
        L.cm_cg_solve_pc.argtypes = [vp, it, vp, vp, db, it, it, it, C.POINTER(it), C.POINTER(db), vp]
        L.cm_cg_solve3_pc.argtypes = [vp, it, vp, vp, db, it, it, it, C.POINTER(it), C.POINTER(db), vp]
        L.cm_cg_history_enable.argtypes = [vp, it]
        L.cm_cg_history.argtypes = [vp, vp, lg, C.POINTER(lg)]
        L.cm_spmv_matfree.argtypes = [vp, vp, vp, vp]
        L.cm_cg_solve_matfree.argtypes = [vp, vp, vp, db, it, it, it, C.POINTER(it), C.POINTER(db), vp]
        L.cm_field_rhs.argtypes = [vp, it, vp, vp, vp, C.POINTER(cm_step_params), db, vp, vp]
        L.cm_volume_average.argtypes = [vp, it, vp, it, C.POINTER(db), vp]
        L.cm_volume_average_noalloc.argtypes = [vp, it, vp, it, vp, vp]
        L.cm_gspm_step.argtypes = [vp, C.POINTER(cm_step_params), vp, vp, vp, C.POINTER(cm_step_info), vp]
        L.cm_gspm_step_host.argtypes = [vp, C.POINTER(cm_step_params), vp, vp, vp, C.POINTER(cm_step_info), vp]
        L.cm_hysteresis_run.argtypes = [vp, C.POINTER(cm_step_params), C.POINTER(cm_hyst_params), vp, vp, vp, vp, vp, vp,
                                        C.POINTER(cm_hyst_result), vp]
        L.cm_system_set_option.argtypes = [vp, it, it]
        L.cm_profile_enable.argtypes = [vp, it]
        L.cm_profile_get.argtypes = [vp, C.POINTER(cm_profile)]
        L.cm_profile_reset.argtypes = [vp]
        L.cm_last_error.restype = C.c_char_p
        L.cm_version.restype = C.c_char_p
        for name in EXPORTS:
            if name not in ("cm_last_error", "cm_version"):
                getattr(L, name).restype = it
        _lib = L
    return _lib


def _check(rc, allow=()):
    if rc < 0 and rc not in allow:
        raise CmError(rc, lib().cm_last_error().decode())
    return rc


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _np(a, dt):
    return None if a is None else np.ascontiguousarray(a, dt)


def _hp(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _dp(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def make_params(dt, Hext=(0, 0, 0), terms=0, variant=0, cg_tol=1e-7, cg_maxiter=100000, cg_fixed_iters=-1, cg_precond=CM_PC_NONE,
                mech_matfree=0):
    return cm_step_params(dt, (C.c_double * 3)(*[float(h) for h in Hext]), int(terms), int(variant), cg_tol, int(cg_maxiter),
                          int(cg_fixed_iters), int(cg_precond), int(mech_matfree))


def periodic_wrap(xyz, axes: int, rel_tol: float = 1e-9):
    """cm_periodic_wrap: (dof_of_node int32[n_nodes], n_dof) for the periodic directions in the bit mask `axes`."""
    xyz = _np(xyz, np.float64)
    dof = np.empty(xyz.shape[0], np.int32)
    nd = C.c_long()
    _check(lib().cm_periodic_wrap(_hp(xyz), xyz.shape[0], int(axes), float(rel_tol), _hp(dof), C.byref(nd)))
    return dof, int(nd.value)


class Mesh:
    """cm_mesh_create: S0 preprocessing (reordering, node->element lists, CSR pattern)."""

    def __init__(self, xyz, tets, magnetic=None, elastic_id=None, reorder=CM_REORDER_MORTON, dof_of_node=None, n_dof=None):
        """dof_of_node / n_dof (from periodic_wrap): cm_mesh_create_wrapped, the mesh then has n_dof "nodes"."""
        L = lib()
        xyz = _np(xyz, np.float64); tets = _np(tets, np.int32)
        mag = _np(magnetic, np.uint8); eid = _np(elastic_id, np.int32)
        self.h = C.c_void_p()
        self.nen = 8 if tets.shape[1] == 8 else 4            # (Ne, 8): linear hexahedra, local node a = i + 2 j + 4 k
        if self.nen == 8 and dof_of_node is not None:
            dof = _np(dof_of_node, np.int32)
            assert dof.shape[0] == xyz.shape[0]
            _check(L.cm_mesh_create_hex_wrapped(_hp(xyz), xyz.shape[0], _hp(tets), tets.shape[0], _hp(mag), _hp(eid), _hp(dof), int(n_dof),
                                                reorder, _stream(), C.byref(self.h)))
        elif self.nen == 8:
            _check(L.cm_mesh_create_hex(_hp(xyz), xyz.shape[0], _hp(tets), tets.shape[0], _hp(mag), _hp(eid), reorder, _stream(),
                                        C.byref(self.h)))
        elif dof_of_node is None:
            _check(L.cm_mesh_create(_hp(xyz), xyz.shape[0], _hp(tets), tets.shape[0], _hp(mag), _hp(eid), reorder, _stream(),
                                    C.byref(self.h)))
        else:
            dof = _np(dof_of_node, np.int32)
            assert dof.shape[0] == xyz.shape[0]
            _check(L.cm_mesh_create_wrapped(_hp(xyz), xyz.shape[0], _hp(tets), tets.shape[0], _hp(mag), _hp(eid), _hp(dof), int(n_dof),
                                            reorder, _stream(), C.byref(self.h)))
        cnt = np.zeros(3, np.int64)
        _check(L.cm_mesh_get(self.h, CM_GET_COUNTS, _hp(cnt), 3))
        self.n_nodes, self.n_tets, self.nnz = (int(c) for c in cnt)

    def get(self, what):
        n = {CM_GET_ORDER: self.n_nodes, CM_GET_IPERM: self.n_nodes, CM_GET_TETS: self.nen * self.n_tets, CM_GET_TET_ORDER: self.n_tets,
             CM_GET_ROWPTR: self.n_nodes + 1, CM_GET_COLIDX: self.nnz, CM_GET_N2E_PTR: self.n_nodes + 1,
             CM_GET_N2E: self.nen * self.n_tets}[what]
        a = np.empty(n, np.int32)
        _check(lib().cm_mesh_get(self.h, what, _hp(a), n))
        return a.reshape(-1, self.nen) if what == CM_GET_TETS else a

    def layout(self):
        """CM_GET_LAYOUT: padding of the sliced matrix layouts and occupancy of the element chunks."""
        a = np.zeros(6, np.int64)
        _check(lib().cm_mesh_get(self.h, CM_GET_LAYOUT, _hp(a), 6))
        e16, e8, nch, nsl, cap_e, cap_n = (int(v) for v in a)
        return {"sell16_padding": e16 / self.nnz - 1.0, "sell8_padding": e8 / self.nnz - 1.0, "chunks": nch, "slots": nsl,
                "slots_per_node": nsl / self.n_nodes, "elements_per_chunk": self.n_tets / max(1, nch), "chunk_capacity": (cap_e, cap_n),
                "nodes_per_chunk": nsl / max(1, nch)}

    def volume_average(self, g):
        """cm_volume_average of a torch CUDA tensor (N,) or (N, ncomp), float64 / float32."""
        import torch
        assert g.is_cuda and g.is_contiguous()
        nc = 1 if g.dim() == 1 else g.shape[1]
        out = (C.c_double * nc)()
        dt = CM_F64 if g.dtype == torch.float64 else CM_F32
        _check(lib().cm_volume_average(self.h, dt, _dp(g), nc, out, _stream()))
        return np.array(out[:])

    def volume_average_noalloc(self, g, out):
        """cm_volume_average_noalloc: the same average for callers that must not allocate device memory (their own pool
        owns the device, or a cudaMalloc would stall their other streams).  `g`: CUDA tensor (N,) or (N, ncomp);
        `out`: the CALLER's float64 CUDA tensor of ncomp elements, written asynchronously on the current stream
        (read it after that stream has been waited for).  Nothing is allocated here or in the library; the scratch is
        a fixed array inside the library shared by every call on this GPU, so calls that may overlap on the GPU race.
        At most binding.CM_NOALLOC_MAX_NODES nodes, ncomp 1, 3 or 6 (else CmError)."""
        import torch
        assert g.is_cuda and g.is_contiguous() and out.is_cuda and out.is_contiguous() and out.dtype == torch.float64
        nc = 1 if g.dim() == 1 else g.shape[1]
        assert out.numel() == nc
        dt = CM_F64 if g.dtype == torch.float64 else CM_F32
        _check(lib().cm_volume_average_noalloc(self.h, dt, _dp(g), nc, _dp(out), _stream()))
        return out

    def close(self):
        if self.h:
            lib().cm_mesh_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class System:
    """cm_assemble_csr: geometry + matrices for one dtype and one dt; the cm_* compute calls."""

    def __init__(self, mesh: Mesh, material, dt, dtype="f64", clamp_dof=None, pin_node=0):
        import torch
        L = lib()
        self.mesh = mesh
        self.dtype = dtype
        self.cm_dtype = CM_F64 if dtype == "f64" else CM_F32
        self.torch_dtype = torch.float64 if dtype == "f64" else torch.float32
        self.np_dtype = np.float64 if dtype == "f64" else np.float32
        self.dt = dt
        Cv = None if material.C_voigt is None else np.ascontiguousarray(material.C_voigt, np.float64).reshape(-1, 36)
        self._Cv = Cv
        m = cm_material(material.Ms, material.Aex, material.K1, material.lambda100, material.lambda111, material.alpha,
                        material.gamma, material.length_scale, (C.c_double * 9)(*material.Nd),
                        0 if Cv is None else Cv.shape[0], None if Cv is None else Cv.ctypes.data_as(C.POINTER(C.c_double)),
                        (C.c_double * 9)(*(np.zeros(9) if getattr(material, "R", None) is None else np.asarray(material.R, float).ravel())),
                        (C.c_double * 6)(*(np.zeros(6) if getattr(material, "sigma_ext", None) is None
                                           else np.asarray(material.sigma_ext, float).ravel())))
        clamp = _np(clamp_dof, np.uint8)
        self.h = C.c_void_p()
        _check(L.cm_assemble_csr(mesh.h, C.byref(m), self.cm_dtype, dt, _hp(clamp), pin_node, _stream(), C.byref(self.h)))
        self.N = mesh.n_nodes

    # ---- getters (host numpy, library order)
    def values(self, mat):
        n = self.mesh.nnz * (9 if mat == CM_MAT_K_MECH else 1)
        a = np.empty(n, self.np_dtype)
        _check(lib().cm_system_get_values(self.h, mat, _hp(a), n))
        return a.reshape(-1, 3, 3) if mat == CM_MAT_K_MECH else a

    def geometry(self, what):
        n = {0: self.mesh.n_tets, 1: 12 * self.mesh.n_tets, 2: self.N, 3: self.N}[what]
        a = np.empty(n, self.np_dtype)
        _check(lib().cm_system_get_geometry(self.h, what, _hp(a), n))
        return a.reshape(-1, 4, 3) if what == 1 else a

    # ---- compute calls on torch CUDA tensors (user order)
    def _chk(self, t):
        assert t.is_cuda and t.is_contiguous() and t.dtype == self.torch_dtype
        return t

    def spmv(self, mat, x):
        import torch
        y = torch.empty_like(self._chk(x))
        _check(lib().cm_spmv(self.h, mat, _dp(x), _dp(y), _stream()))
        return y

    def spmv3(self, mat, x):
        import torch
        y = torch.empty_like(self._chk(x))
        _check(lib().cm_spmv3(self.h, mat, _dp(x), _dp(y), _stream()))
        return y

    def cg_solve(self, mat, b, x, tol=1e-7, maxiter=100000, fixed_iters=-1, precond=None):
        """In place on x.  Returns (iters, relres, status).  precond: None = cm_cg_solve, else cm_cg_solve_pc."""
        it = C.c_int(); res = C.c_double()
        if precond is None:
            rc = lib().cm_cg_solve(self.h, mat, _dp(self._chk(b)), _dp(self._chk(x)), tol, maxiter, fixed_iters, C.byref(it),
                                   C.byref(res), _stream())
        else:
            rc = lib().cm_cg_solve_pc(self.h, mat, _dp(self._chk(b)), _dp(self._chk(x)), tol, maxiter, fixed_iters, int(precond),
                                      C.byref(it), C.byref(res), _stream())
        return it.value, res.value, _check(rc, allow=(CM_E_CG_BREAKDOWN, CM_E_CG_MAXITER))

    def cg_solve3(self, mat, b, x, tol=1e-7, maxiter=100000, fixed_iters=-1, precond=None):
        it = (C.c_int * 3)(); res = (C.c_double * 3)()
        if precond is None:
            rc = lib().cm_cg_solve3(self.h, mat, _dp(self._chk(b)), _dp(self._chk(x)), tol, maxiter, fixed_iters, it, res, _stream())
        else:
            rc = lib().cm_cg_solve3_pc(self.h, mat, _dp(self._chk(b)), _dp(self._chk(x)), tol, maxiter, fixed_iters, int(precond), it,
                                       res, _stream())
        return list(it), list(res), _check(rc, allow=(CM_E_CG_BREAKDOWN, CM_E_CG_MAXITER))

    def spmv_matfree(self, x):
        import torch
        y = torch.empty_like(self._chk(x))
        _check(lib().cm_spmv_matfree(self.h, _dp(x), _dp(y), _stream()))
        return y

    def cg_solve_matfree(self, b, x, tol=1e-7, maxiter=100000, fixed_iters=-1, precond=CM_PC_NONE):
        it = C.c_int(); res = C.c_double()
        rc = lib().cm_cg_solve_matfree(self.h, _dp(self._chk(b)), _dp(self._chk(x)), tol, maxiter, fixed_iters, int(precond),
                                       C.byref(it), C.byref(res), _stream())
        return it.value, res.value, _check(rc, allow=(CM_E_CG_BREAKDOWN, CM_E_CG_MAXITER))

    def cg_history_enable(self, on=True):
        _check(lib().cm_cg_history_enable(self.h, int(on)))

    def cg_history(self, n_rhs=1, cap=3 << 16):
        """Residual history of the last cg_solve* call: array [k] (n_rhs = 1) or [k][3]."""
        a = np.zeros(cap); n = C.c_long()
        _check(lib().cm_cg_history(self.h, _hp(a), cap, C.byref(n)))
        a = a[:n.value]
        return a if n_rhs == 1 else a.reshape(-1, n_rhs)

    def field_rhs(self, rhs_id, m, U=None, u=None, params: Optional[cm_step_params] = None, coeff=0.0):
        import torch
        shape = {CM_RHS_MS: (self.N,), CM_RHS_MECH: (self.N, 3), CM_RHS_GS: (self.N, 3), CM_OUT_HD: (self.N, 3),
                 CM_OUT_SIGMA: (self.N, 6), CM_OUT_FIELD: (self.N, 3)}[rhs_id]
        b = torch.empty(shape, dtype=self.torch_dtype, device=m.device)
        _check(lib().cm_field_rhs(self.h, rhs_id, _dp(self._chk(m)), _dp(U), _dp(u), None if params is None else C.byref(params),
                                  coeff, _dp(b), _stream()))
        return b

    def gspm_step(self, params: cm_step_params, m, U, u, want_info=True):
        """One GSPM step in place on CUDA tensors m (N,3), U (N,), u (N,3).  Returns (cm_step_info | None, status)."""
        info = cm_step_info() if want_info else None
        rc = _check(lib().cm_gspm_step(self.h, C.byref(params), _dp(self._chk(m)), _dp(U), _dp(u),
                                       None if info is None else C.byref(info), _stream()),
                    allow=(CM_E_CG_BREAKDOWN, CM_E_CG_MAXITER))
        return info, rc

    def gspm_step_host(self, params: cm_step_params, m, U, u):
        """Same through HOST buffers (numpy arrays or pinned torch CPU tensors), copies inside the call."""
        info = cm_step_info()

        def hp(a):
            if a is None:
                return None
            return C.c_void_p(a.data_ptr()) if hasattr(a, "data_ptr") else a.ctypes.data_as(C.c_void_p)

        rc = _check(lib().cm_gspm_step_host(self.h, C.byref(params), hp(m), hp(U), hp(u), C.byref(info), _stream()),
                    allow=(CM_E_CG_BREAKDOWN, CM_E_CG_MAXITER))
        return info, rc

    def hysteresis_run(self, params: cm_step_params, m, U, u, H0, dH, conv_tol=5e-10, max_fields=100, max_steps=100000):
        """cm_hysteresis_run: the whole field loop on the device (one CUDA graph launch).
        Returns (H_log, mbar_log, steps_log, cm_hyst_result, rc) with the logs cut to n_fields."""
        for t in (m, U, u):
            if t is not None:
                self._chk(t)
        hp = cm_hyst_params((C.c_double * 3)(*[float(x) for x in H0]), (C.c_double * 3)(*[float(x) for x in dH]), conv_tol,
                            int(max_fields), int(max_steps))
        Hl = np.zeros((max_fields, 3)); ml = np.zeros((max_fields, 3)); sl = np.zeros(max_fields, np.int32)
        res = cm_hyst_result()
        rc = _check(lib().cm_hysteresis_run(self.h, C.byref(params), C.byref(hp), _dp(m), _dp(U), _dp(u), _hp(Hl), _hp(ml), _hp(sl),
                                            C.byref(res), _stream()), allow=(CM_E_CG_MAXITER, CM_E_CG_BREAKDOWN))
        n = res.n_fields
        return Hl[:n], ml[:n], sl[:n], res, rc

    def set_option(self, option, value):
        _check(lib().cm_system_set_option(self.h, int(option), int(value)))

    def profile_enable(self, on=True):
        _check(lib().cm_profile_enable(self.h, int(on)))

    def profile_reset(self):
        _check(lib().cm_profile_reset(self.h))

    def profile(self):
        p = cm_profile()
        _check(lib().cm_profile_get(self.h, C.byref(p)))
        return {n: {"ms": p.ms[i], "launches": p.launches[i], "cg_iters": p.cg_iters[i],
                    "cg_matrix_passes": p.cg_matrix_passes[i]} for i, n in enumerate(PROF_NAMES)}

    def close(self):
        if self.h:
            lib().cm_system_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
