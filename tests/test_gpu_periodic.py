"""GPU parity of the periodic (node-wrapped) path against the oracle: structure bit-exact, matrices / SpMV /
right-hand sides / fields <= 1e-12 (fp64) and 1e-5 (fp32), ten GSPM steps <= 1e-9 / 1e-4.  All vectors are in DOF
numbering (R23)."""
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


def mat2():
    C = inputs.isotropic_voigt(200e9, 0.3)
    return inputs.Material(C_voigt=np.stack([C, 2 * C]))


def periodic_case(cm, orc, grid, box, axes, reorder, dtype="f64", inclusion=None, seeds=(81, 82), dt=1e-12, pin=0):
    mesh = inputs.kuhn_box(grid, box, seed_mesh=seeds[0], seed_perm=seeds[1])
    if inclusion is not None:
        mesh = inputs.flag_inclusion(mesh, np.array(mesh.box) / 2, inclusion)
    dof, nd = cm.periodic_wrap(mesh.xyz, axes)
    dof_o, nd_o = orc.periodic_wrap(mesh.xyz, axes)
    assert nd == nd_o and np.array_equal(dof, dof_o)
    clamp = np.zeros((nd, 3), np.uint8); clamp[7] = 1; clamp = clamp.ravel()      # pin d = 3 displacement DOFs
    gm = cm.Mesh(mesh.xyz, mesh.tets, mesh.magnetic, mesh.elastic_id, reorder, dof_of_node=dof, n_dof=nd)
    gs = cm.System(gm, mat2(), dt, dtype, clamp, pin)
    o = orc.Oracle(mesh, mat2(), dt, clamp_dof=clamp, pin_node=pin, dof_of_node=dof, n_dof=nd)
    return mesh, dof, nd, clamp, gm, gs, o


@pytest.mark.parametrize("reorder", [0, 1, 2])
@pytest.mark.parametrize("axes", [7, 3, 4])
def test_periodic_structure_bit_exact(cm, oracle_mod, torch, reorder, axes):
    mesh = inputs.kuhn_box((9, 8, 7), (20 * NM, 18 * NM, 15 * NM), seed_mesh=61, seed_perm=62)
    dof, nd = cm.periodic_wrap(mesh.xyz, axes)
    gm = cm.Mesh(mesh.xyz, mesh.tets, reorder=reorder, dof_of_node=dof, n_dof=nd)
    assert gm.n_nodes == nd
    # the oracle's reordering of the DOF mesh: DOF coordinates = those of the representative (componentwise minimum)
    dxyz = np.full((nd, 3), np.inf); np.minimum.at(dxyz, dof, mesh.xyz)
    dtets = dof[mesh.tets].astype(np.int32)
    order, iperm, tnew, torder = oracle_mod.reorder(dxyz, dtets, reorder)
    assert np.array_equal(gm.get(cm.CM_GET_ORDER), order)
    assert np.array_equal(gm.get(cm.CM_GET_IPERM), iperm)
    assert np.array_equal(gm.get(cm.CM_GET_TETS), tnew)
    assert np.array_equal(gm.get(cm.CM_GET_TET_ORDER), torder)
    o = oracle_mod.Oracle(mesh, inputs.Material(), 1e-12, dof_of_node=iperm[dof], n_dof=nd)     # oracle in library numbering
    # (its tets are in user order, so n2e differs; the pattern does not depend on the tet order)
    assert gm.nnz == o.nnz
    assert np.array_equal(gm.get(cm.CM_GET_ROWPTR), o.rowptr())
    assert np.array_equal(gm.get(cm.CM_GET_COLIDX), o.colidx())


def test_periodic_errors(cm, torch):
    mesh = inputs.kuhn_box((2, 4, 4), (5 * NM, 12 * NM, 12 * NM))
    dof, nd = cm.periodic_wrap(mesh.xyz, 1)
    with pytest.raises(cm.CmError) as e:                      # one cell wide along x: tets collapse
        cm.Mesh(mesh.xyz, mesh.tets, dof_of_node=dof, n_dof=nd)
    assert e.value.code == cm.CM_E_BADARG
    mesh = inputs.kuhn_box((4, 4, 4), (9 * NM,) * 3)
    dof, nd = cm.periodic_wrap(mesh.xyz, 7)
    bad = dof.copy(); bad[0] = nd
    with pytest.raises(cm.CmError) as e:
        cm.Mesh(mesh.xyz, mesh.tets, dof_of_node=bad, n_dof=nd)
    assert e.value.code == cm.CM_E_INDEX_RANGE


def _to_user(gm, vals_lib, block):
    import scipy.sparse as sp
    rp, ci, iperm, N = gm.get(5), gm.get(6), gm.get(2), gm.n_nodes
    if not block:
        A = sp.csr_matrix((vals_lib.astype(np.float64), ci, rp), shape=(N, N))
        return A[iperm][:, iperm].tocsr()
    A = sp.bsr_matrix((vals_lib.astype(np.float64), ci, rp), shape=(3 * N, 3 * N)).tocsr()
    idx = (3 * iperm[:, None] + np.arange(3)[None, :]).ravel()
    return A[idx][:, idx].tocsr()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_periodic_matrices_spmv_rhs_fields(cm, oracle_mod, torch, dtype):
    """7 x 10^3-DOF fully periodic box with a x2-stiff non-magnetic inclusion (several SELL slices / element chunks,
    ragged tail), Morton order."""
    mesh, dof, nd, clamp, gm, gs, o = periodic_case(cm, oracle_mod, (23, 19, 17), (66 * NM, 54 * NM, 48 * NM), 7, 1, dtype,
                                                    inclusion=(14 * NM, 12 * NM, 10 * NM), dt=2e-12, pin=5)
    f64 = dtype == "f64"
    tol = 1e-12 if f64 else 1e-5
    vtol = tol if f64 else 2e-7
    td = torch.float64 if f64 else torch.float32
    dev = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=td, device="cuda")
    torder, order = gm.get(cm.CM_GET_TET_ORDER), gm.get(cm.CM_GET_ORDER)
    assert rel(gs.geometry(0), o.V()[torder]) < vtol
    assert rel(gs.geometry(1), o.G()[torder]) < vtol
    assert rel(gs.geometry(2), o.mL()[order]) < vtol
    for mg, mo in ((cm.CM_MAT_K_MS, oracle_mod.MAT_K_MS), (cm.CM_MAT_K_GS1, oracle_mod.MAT_K_GS1),
                   (cm.CM_MAT_MASS, oracle_mod.MAT_MASS), (cm.CM_MAT_K_MECH, oracle_mod.MAT_K_MECH)):
        A = _to_user(gm, gs.values(mg), mg == cm.CM_MAT_K_MECH)
        B = o.csr(mo)
        assert abs(A - B).max() < vtol * abs(B).max(), mg
    rng = np.random.default_rng(7)
    x = rng.normal(size=nd).astype(gs.np_dtype)
    assert rel(gs.spmv(cm.CM_MAT_K_MS, dev(x)).cpu().numpy(), o.spmv(oracle_mod.MAT_K_MS, x.astype(np.float64))) < tol
    x3 = rng.normal(size=(nd, 3)).astype(gs.np_dtype)
    y3 = gs.spmv(cm.CM_MAT_K_MECH, dev(x3)).cpu().numpy()
    assert rel(y3.ravel(), o.spmv(oracle_mod.MAT_K_MECH, x3.astype(np.float64).ravel())) < tol

    m = rng.normal(size=(nd, 3)); m /= np.linalg.norm(m, axis=1, keepdims=True)
    m[~o.live().astype(bool)] = 0
    m = m.astype(gs.np_dtype); m64 = m.astype(np.float64)
    U = rng.normal(size=nd).astype(gs.np_dtype); u = (1e-3 * rng.normal(size=(nd, 3))).astype(gs.np_dtype)
    md, Ud, ud = dev(m), dev(U), dev(u)
    Hext = np.array([3e4, -1e4, 2e4])
    p = cm.make_params(2e-12, Hext, ALL)
    assert np.abs(gm.volume_average(md) - o.volume_average(m64)).max() < (1e-13 if f64 else 1e-7)
    assert rel(gs.field_rhs(cm.CM_RHS_MS, md).cpu().numpy(), o.rhs_ms(m64)) < tol
    assert rel(gs.field_rhs(cm.CM_RHS_MECH, md).cpu().numpy(), o.rhs_mech(m64)) < tol
    hd_o, _ = o.demag_field(U.astype(np.float64), o.volume_average(m64), TERM_DEMAG | TERM_FARFIELD)
    assert rel(gs.field_rhs(cm.CM_OUT_HD, md, Ud, None, p).cpu().numpy(), hd_o) < tol
    sig_o = o.stress_recover(u.astype(np.float64), m64)
    assert rel(gs.field_rhs(cm.CM_OUT_SIGMA, md, None, ud, p).cpu().numpy(), sig_o) < tol
    h_o = o.field(m64, hd_o, sig_o, Hext / 1.2e6, ALL)
    assert rel(gs.field_rhs(cm.CM_OUT_FIELD, md, Ud, ud, p).cpu().numpy(), h_o) < tol


def _steps(cm, torch, gs, o, nd, m0, terms, H, nsteps, dtype, tol, dt=1e-12):
    td = torch.float64 if dtype == "f64" else torch.float32
    m = m0.copy(); U = np.zeros(nd); u = np.zeros((nd, 3))
    mg = torch.as_tensor(m0, dtype=td, device="cuda").contiguous()
    Ug = torch.zeros(nd, dtype=td, device="cuda"); ug = torch.zeros((nd, 3), dtype=td, device="cuda")
    infos = []
    for k in range(nsteps):
        io, rco = o.gspm_step(m, U, u, dt, H, terms, cg_tol=tol)
        ig, rcg = gs.gspm_step(cm.make_params(dt, H, terms, 0, tol), mg, Ug, ug)
        assert rco == 0 and rcg == 0
        infos.append((io, ig))
    return m, U, u, mg.cpu().numpy().astype(np.float64), Ug.cpu().numpy(), ug.cpu().numpy(), infos


@pytest.mark.parametrize("axes,reorder", [(7, 1), (7, 2), (3, 1)])
def test_periodic_gspm_10_steps_f64(cm, oracle_mod, torch, axes, reorder):
    """Config-0 physics (anisotropy + demag + far field) on a periodic box: max |dm| <= 1e-9 after 10 steps."""
    mesh, dof, nd, clamp, gm, gs, o = periodic_case(cm, oracle_mod, (9, 9, 8), (20 * NM, 20 * NM, 18 * NM), axes, reorder)
    rng = np.random.default_rng(83)
    m0 = rng.normal(size=(nd, 3)); m0 /= np.linalg.norm(m0, axis=1, keepdims=True)
    terms = TERM_ANIS | TERM_DEMAG | TERM_FARFIELD
    m, U, u, mg, Ug, ug, infos = _steps(cm, torch, gs, o, nd, m0, terms, [0, 0, 0], 10, "f64", 1e-12)
    assert np.abs(mg - m).max() <= 1e-9
    assert np.abs(Ug - U).max() <= 1e-9 * max(1.0, np.abs(U).max())
    assert np.abs(np.linalg.norm(mg, axis=1) - 1).max() <= 4 * np.finfo(float).eps
    for io, ig in infos:
        assert abs(io.it_ms - ig.it_ms) <= 1
        assert all(abs(io.it_gs[a] - ig.it_gs[a]) <= 1 for a in range(8))


def test_periodic_magnetoelastic_inclusion_steps(cm, oracle_mod, torch):
    """All terms, fully periodic array of x2-stiff non-magnetic inclusions (the paper's setting), d = 3
    displacement DOFs pinned: fp64 1e-9 after 10 steps, fp32 1e-4."""
    for dtype, tol, bar in (("f64", 1e-12, 1e-9), ("f32", 1e-6, 1e-4)):
        mesh, dof, nd, clamp, gm, gs, o = periodic_case(cm, oracle_mod, (13, 13, 9), (40 * NM, 40 * NM, 26 * NM), 7, 1, dtype,
                                                        inclusion=(8 * NM,) * 3)
        rng = np.random.default_rng(84)
        m0 = np.array([1.0, 0, 0]) + 0.1 * rng.normal(size=(nd, 3)); m0 /= np.linalg.norm(m0, axis=1, keepdims=True)
        m0[~o.live().astype(bool)] = 0
        m, U, u, mg, Ug, ug, infos = _steps(cm, torch, gs, o, nd, m0, ALL, [2e4, 0, 0], 10, dtype, tol)
        assert np.abs(mg - m).max() <= bar
        if dtype == "f64":
            assert np.abs(ug - u).max() <= 1e-9 * max(1.0, np.abs(u).max())
            io, ig = infos[0]
            assert abs(io.it_ms - ig.it_ms) <= 1 and abs(io.it_mech - ig.it_mech) <= 1
            assert io.it_mech > 10
