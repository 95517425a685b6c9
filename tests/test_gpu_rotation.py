"""GPU parity of the rotated crystal frame (Appendix D; R25) against the oracle:
K^mech with C_sim = M C M^T, mechanical right-hand side, recovered stress, fields <= 1e-12 (fp64) / 1e-5 (fp32); ten GSPM steps
with all terms <= 1e-9 / 1e-4."""
import numpy as np
import pytest

from paper_2510_09812_b200 import inputs
from paper_2510_09812_b200.inputs import TERM_ANIS, TERM_DEMAG, TERM_FARFIELD, TERM_MAGEL, TERM_ZEEMAN

pytestmark = pytest.mark.gpu
NM = 1e-9
ALL = TERM_ANIS | TERM_ZEEMAN | TERM_DEMAG | TERM_FARFIELD | TERM_MAGEL


@pytest.fixture(scope="module")
def torch():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    return torch


@pytest.fixture(scope="module")
def cm():
    from paper_2510_09812_b200 import binding
    binding.lib()
    return binding


def rel(a, b):
    a = np.asarray(a, np.float64); b = np.asarray(b, np.float64)
    return np.abs(a - b).max() / max(np.abs(b).max(), 1e-300)


def material(R):
    Cc = inputs.cubic_voigt(2.4e11, 1.5e11, 1.2e11)
    return inputs.Material(C_voigt=np.stack([Cc, 2 * Cc]), R=R)


def _to_user(gm, vals_lib):
    import scipy.sparse as sp
    rp, ci, iperm, N = gm.get(5), gm.get(6), gm.get(2), gm.n_nodes
    A = sp.bsr_matrix((vals_lib.astype(np.float64), ci, rp), shape=(3 * N, 3 * N)).tocsr()
    idx = (3 * iperm[:, None] + np.arange(3)[None, :]).ravel()
    return A[idx][:, idx].tocsr()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("which", ["R111", "random"])
def test_rotated_matrices_rhs_fields(cm, oracle_mod, torch, dtype, which):
    R = inputs.R_111 if which == "R111" else inputs.random_rotation(11)
    mesh = inputs.kuhn_box((23, 19, 17), (66 * NM, 54 * NM, 48 * NM), seed_mesh=51, seed_perm=52)
    mesh = inputs.flag_inclusion(mesh, np.array(mesh.box) / 2, (14 * NM, 12 * NM, 10 * NM))
    mat = material(R)
    clamp = inputs.clamp_bottom(mesh)
    gm = cm.Mesh(mesh.xyz, mesh.tets, mesh.magnetic, mesh.elastic_id, cm.CM_REORDER_MORTON)
    gs = cm.System(gm, mat, 2e-12, dtype, clamp, 5)
    o = oracle_mod.Oracle(mesh, mat, 2e-12, clamp_dof=clamp, pin_node=5)
    f64 = dtype == "f64"
    tol = 1e-12 if f64 else 1e-5
    td = torch.float64 if f64 else torch.float32
    dev = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=td, device="cuda")
    A = _to_user(gm, gs.values(cm.CM_MAT_K_MECH))
    B = o.csr(oracle_mod.MAT_K_MECH)
    assert abs(A - B).max() < (1e-12 if f64 else 2e-7) * abs(B).max()
    rng = np.random.default_rng(8)
    N = o.N
    m = inputs.init_m_random(mesh, 9).astype(gs.np_dtype); m64 = m.astype(np.float64)
    U = rng.normal(size=N).astype(gs.np_dtype); u = (1e-3 * rng.normal(size=(N, 3))).astype(gs.np_dtype)
    md, Ud, ud = dev(m), dev(U), dev(u)
    Hext = np.array([3e4, -1e4, 2e4])
    p = cm.make_params(2e-12, Hext, ALL)
    assert rel(gs.field_rhs(cm.CM_RHS_MECH, md).cpu().numpy(), o.rhs_mech(m64)) < tol
    sig_o = o.stress_recover(u.astype(np.float64), m64)
    assert rel(gs.field_rhs(cm.CM_OUT_SIGMA, md, None, ud, p).cpu().numpy(), sig_o) < tol
    hd_o, _ = o.demag_field(U.astype(np.float64), o.volume_average(m64), TERM_DEMAG | TERM_FARFIELD)
    h_o = o.field(m64, hd_o, sig_o, Hext / mat.Ms, ALL)
    assert rel(gs.field_rhs(cm.CM_OUT_FIELD, md, Ud, ud, p).cpu().numpy(), h_o) < tol
    for terms in (TERM_ANIS, TERM_MAGEL):
        h_t = o.field(m64, hd_o, sig_o, Hext / mat.Ms, terms)
        assert rel(gs.field_rhs(cm.CM_OUT_FIELD, md, Ud, ud, cm.make_params(2e-12, Hext, terms)).cpu().numpy(), h_t) < tol
    # the rotation matters: the unrotated system gives a different field
    gsI = cm.System(gm, material(None), 2e-12, dtype, clamp, 5)
    assert rel(gsI.field_rhs(cm.CM_OUT_FIELD, md, Ud, ud, p).cpu().numpy(), h_o) > 1e-3


@pytest.mark.parametrize("dtype,tol,bar", [("f64", 1e-12, 1e-9), ("f32", 1e-6, 1e-4)])
def test_rotated_gspm_10_steps(cm, oracle_mod, torch, dtype, tol, bar):
    """Reduced config 2 (all terms, x2-stiff non-magnetic inclusion, clamped bottom) in the paper's <111> frame (Eq. D.1)."""
    mesh = inputs.kuhn_box((13, 13, 7), (40 * NM, 40 * NM, 20 * NM), seed_mesh=21, seed_perm=22)
    mesh = inputs.flag_inclusion(mesh, np.array(mesh.box) / 2, (8 * NM,) * 3)
    mat = material(inputs.R_111)
    clamp = inputs.clamp_bottom(mesh)
    gm = cm.Mesh(mesh.xyz, mesh.tets, mesh.magnetic, mesh.elastic_id, cm.CM_REORDER_MORTON)
    gs = cm.System(gm, mat, 1e-12, dtype, clamp)
    o = oracle_mod.Oracle(mesh, mat, 1e-12, clamp_dof=clamp)
    td = torch.float64 if dtype == "f64" else torch.float32
    N = o.N
    m0 = inputs.init_m_noisy_x(mesh, 23)
    m = m0.copy(); U = np.zeros(N); u = np.zeros((N, 3))
    mg = torch.as_tensor(m0, dtype=td, device="cuda").contiguous()
    Ug = torch.zeros(N, dtype=td, device="cuda"); ug = torch.zeros((N, 3), dtype=td, device="cuda")
    H = [2e4, 0, 0]
    for k in range(10):
        io, rco = o.gspm_step(m, U, u, 1e-12, H, ALL, cg_tol=tol)
        ig, rcg = gs.gspm_step(cm.make_params(1e-12, H, ALL, 0, tol), mg, Ug, ug)
        assert rco == 0 and rcg == 0
        if dtype == "f64" and k == 0:
            assert abs(io.it_ms - ig.it_ms) <= 1 and abs(io.it_mech - ig.it_mech) <= 1
    assert np.abs(mg.cpu().numpy().astype(np.float64) - m).max() <= bar
    if dtype == "f64":
        assert np.abs(ug.cpu().numpy() - u).max() <= 1e-9 * max(1.0, np.abs(u).max())


def test_bad_rotation_rejected(cm, torch):
    mesh = inputs.kuhn_box((4, 4, 4), (9 * NM,) * 3)
    gm = cm.Mesh(mesh.xyz, mesh.tets)
    for R in (np.diag([1.0, 1.0, 2.0]), np.diag([1.0, 1.0, -1.0])):
        with pytest.raises(cm.CmError) as e:
            cm.System(gm, inputs.Material(R=R), 1e-12)
        assert e.value.code == cm.CM_E_BADARG


@pytest.mark.parametrize("dtype,tol,bar", [("f64", 1e-12, 1e-9), ("f32", 1e-6, 1e-4)])
def test_rotated_hexahedra(cm, oracle_mod, torch, dtype, tol, bar):
    """Appendix D on linear hexahedra (R25 x R26): both sides honour cm_material.R on a hexahedral mesh -- K^mech with
    C_sim, mechanical right-hand side, recovered stress, field, and five GSPM steps in the <111> frame."""
    mesh = inputs.hex_box((12, 11, 7), (33 * NM, 30 * NM, 18 * NM), seed_mesh=81, seed_perm=82)
    mesh = inputs.flag_inclusion(mesh, np.array(mesh.box) / 2, (8 * NM, 7 * NM, 5 * NM))
    mat = material(inputs.R_111)
    clamp = inputs.clamp_bottom(mesh)
    gm = cm.Mesh(mesh.xyz, mesh.hexes, mesh.magnetic, mesh.elastic_id, cm.CM_REORDER_MORTON)
    gs = cm.System(gm, mat, 1e-12, dtype, clamp, 5)
    o = oracle_mod.Oracle(mesh, mat, 1e-12, clamp_dof=clamp, pin_node=5)
    f64 = dtype == "f64"
    ftol = 1e-12 if f64 else 1e-5
    td = torch.float64 if f64 else torch.float32
    dev = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=td, device="cuda")
    A = _to_user(gm, gs.values(cm.CM_MAT_K_MECH))
    B = o.csr(oracle_mod.MAT_K_MECH)
    assert abs(A - B).max() < (1e-12 if f64 else 2e-7) * abs(B).max()
    rng = np.random.default_rng(83)
    N = o.N
    live = o.live().astype(bool)
    m = rng.normal(size=(N, 3)); m /= np.linalg.norm(m, axis=1, keepdims=True); m[~live] = 0
    m = m.astype(gs.np_dtype); m64 = m.astype(np.float64)
    u = (1e-3 * rng.normal(size=(N, 3))).astype(gs.np_dtype)
    p = cm.make_params(1e-12, [3e4, -1e4, 2e4], TERM_ANIS | TERM_ZEEMAN | TERM_MAGEL)
    assert rel(gs.field_rhs(cm.CM_RHS_MECH, dev(m)).cpu().numpy(), o.rhs_mech(m64)) < ftol
    sig_o = o.stress_recover(u.astype(np.float64), m64)
    assert rel(gs.field_rhs(cm.CM_OUT_SIGMA, dev(m), None, dev(u), p).cpu().numpy(), sig_o) < ftol
    h_o = o.field(m64, None, sig_o, np.array([3e4, -1e4, 2e4]) / mat.Ms, TERM_ANIS | TERM_ZEEMAN | TERM_MAGEL)
    assert rel(gs.field_rhs(cm.CM_OUT_FIELD, dev(m), None, dev(u), p).cpu().numpy(), h_o) < ftol
    # the rotation matters on hexahedra too
    gsI = cm.System(gm, material(None), 1e-12, dtype, clamp, 5)
    assert rel(gsI.field_rhs(cm.CM_RHS_MECH, dev(m)).cpu().numpy(), o.rhs_mech(m64)) > 1e-3
    mo = m64.copy(); U = np.zeros(N); uo = np.zeros((N, 3))
    mg = dev(m64); Ug = torch.zeros(N, dtype=td, device="cuda"); ug = torch.zeros((N, 3), dtype=td, device="cuda")
    H = [2e4, 0, 0]
    for k in range(5):
        io, rco = o.gspm_step(mo, U, uo, 1e-12, H, ALL, cg_tol=tol)
        ig, rcg = gs.gspm_step(cm.make_params(1e-12, H, ALL, 0, tol), mg, Ug, ug)
        assert rco == 0 and rcg == 0
        if f64 and k == 0:
            assert abs(io.it_ms - ig.it_ms) <= 1 and abs(io.it_mech - ig.it_mech) <= 1
    assert np.abs(mg.cpu().numpy().astype(np.float64) - mo).max() <= bar
