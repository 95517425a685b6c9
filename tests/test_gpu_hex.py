"""GPU parity of the linear-hexahedral (Q1) matrices and of SpMV / CG on them (DESIGN.md
R26) against the oracle: structure bit-exact, matrix values / lumped masses / SpMV <= 1e-12 (fp64) and 1e-5 (fp32), CG
iteration counts +-1, volume averages; the tetrahedral-only entry points refuse hexahedral meshes."""
import numpy as np
import pytest

from paper_2510_09812_b200 import inputs

pytestmark = pytest.mark.gpu
NM = 1e-9


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


@pytest.mark.parametrize("reorder", [0, 1, 2])
def test_hex_structure_bit_exact(cm, oracle_mod, torch, reorder):
    mesh = inputs.hex_box((9, 8, 7), (20 * NM, 18 * NM, 15 * NM), seed_mesh=61, seed_perm=62)
    gm = cm.Mesh(mesh.xyz, mesh.hexes, reorder=reorder)
    assert gm.nen == 8 and gm.n_tets == 8 * 7 * 6
    # node order from the oracle (Morton needs coordinates only; RCM the node graph, the same for any element type that
    # connects the same node sets -- here the graph is taken from the oracle's own hexahedral pattern)
    if reorder == 2:
        o_user = oracle_mod.Oracle(mesh, inputs.Material(), 1e-12)
        rp, ci = o_user.rowptr(), o_user.colidx()
        deg = np.diff(rp) - 1
        N = o_user.N
        seen = np.zeros(N, bool); cmo = []
        bydeg = sorted(range(N), key=lambda i: (deg[i], i))
        for s in bydeg:
            if seen[s]:
                continue
            seen[s] = True; queue = [s]; cmo.append(s); head = len(cmo) - 1
            while head < len(cmo):
                v = cmo[head]; head += 1
                nb = [j for j in ci[rp[v]:rp[v + 1]] if j != v and not seen[j]]
                for j in nb:
                    seen[j] = True
                cmo.extend(sorted(nb, key=lambda j: (deg[j], j)))
        order = np.array(cmo[::-1], np.int32)
    else:
        order = oracle_mod.reorder(mesh.xyz, mesh.hexes[:, :4].copy(), reorder)[0]
    iperm = np.empty_like(order); iperm[order] = np.arange(len(order), dtype=np.int32)
    assert np.array_equal(gm.get(cm.CM_GET_ORDER), order)
    assert np.array_equal(gm.get(cm.CM_GET_IPERM), iperm)
    rel_h = iperm[mesh.hexes]
    key = np.lexsort((np.arange(len(rel_h)), rel_h.min(1)))                 # by (min new id, user index)
    assert np.array_equal(gm.get(cm.CM_GET_TET_ORDER), key.astype(np.int32))
    assert np.array_equal(gm.get(cm.CM_GET_TETS), rel_h[key])
    relab = inputs.replace(mesh, xyz=mesh.xyz[order], hexes=rel_h[key].astype(np.int32))
    o = oracle_mod.Oracle(relab, inputs.Material(), 1e-12)
    assert gm.nnz == o.nnz
    assert np.array_equal(gm.get(cm.CM_GET_ROWPTR), o.rowptr())
    assert np.array_equal(gm.get(cm.CM_GET_COLIDX), o.colidx())
    assert np.array_equal(gm.get(cm.CM_GET_N2E_PTR), o.n2e_ptr())
    assert np.array_equal(gm.get(cm.CM_GET_N2E), o.n2e())


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
def test_hex_matrices_spmv_cg_average(cm, oracle_mod, torch, dtype):
    """8 x 10^3-node jittered hexahedral box with a x2-stiff non-magnetic inclusion, clamped bottom face, Morton order."""
    mesh = inputs.hex_box((24, 20, 17), (69 * NM, 57 * NM, 48 * NM), seed_mesh=51, seed_perm=52)
    mesh = inputs.flag_inclusion(mesh, np.array(mesh.box) / 2, (14 * NM, 12 * NM, 10 * NM))
    clamp = inputs.clamp_bottom(mesh)
    gm = cm.Mesh(mesh.xyz, mesh.hexes, mesh.magnetic, mesh.elastic_id, cm.CM_REORDER_MORTON)
    gs = cm.System(gm, mat2(), 2e-12, dtype, clamp, 5)
    o = oracle_mod.Oracle(mesh, mat2(), 2e-12, clamp_dof=clamp, pin_node=5)
    f64 = dtype == "f64"
    tol = 1e-12 if f64 else 1e-5
    vtol = 1e-12 if f64 else 2e-7
    td = torch.float64 if f64 else torch.float32
    dev = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=td, device="cuda")
    order = gm.get(cm.CM_GET_ORDER)
    assert rel(gs.geometry(2), o.mL()[order]) < vtol and rel(gs.geometry(3), o.mLm()[order]) < vtol
    for mg, mo in ((cm.CM_MAT_K_MS, oracle_mod.MAT_K_MS), (cm.CM_MAT_K_GS1, oracle_mod.MAT_K_GS1), (cm.CM_MAT_K_GS2, oracle_mod.MAT_K_GS2),
                   (cm.CM_MAT_MASS, oracle_mod.MAT_MASS), (cm.CM_MAT_K_MECH, oracle_mod.MAT_K_MECH)):
        A = _to_user(gm, gs.values(mg), mg == cm.CM_MAT_K_MECH)
        B = o.csr(mo)
        assert abs(A - B).max() < vtol * abs(B).max(), mg
    rng = np.random.default_rng(7)
    N = o.N
    x = rng.normal(size=N).astype(gs.np_dtype)
    for mg, mo in ((cm.CM_MAT_K_MS, oracle_mod.MAT_K_MS), (cm.CM_MAT_K_GS1, oracle_mod.MAT_K_GS1)):
        assert rel(gs.spmv(mg, dev(x)).cpu().numpy(), o.spmv(mo, x.astype(np.float64))) < tol
    x3 = rng.normal(size=(N, 3)).astype(gs.np_dtype)
    assert rel(gs.spmv(cm.CM_MAT_K_MECH, dev(x3)).cpu().numpy().ravel(), o.spmv(oracle_mod.MAT_K_MECH, x3.astype(np.float64).ravel())) < tol
    assert rel(gs.spmv3(cm.CM_MAT_MASS, dev(x3)).cpu().numpy(), o.rhs_gs(x3.astype(np.float64))) < tol
    g = np.stack([mesh.xyz[:, 0] / NM, rng.normal(size=N), np.ones(N)], axis=1).astype(gs.np_dtype)
    assert np.abs(gm.volume_average(dev(g)) - o.volume_average(g.astype(np.float64))).max() < (1e-12 if f64 else 1e-5)
    # CG to convergence: iteration counts +-1 (fp64), solution against a tight oracle solve
    tol_cg = 1e-10 if f64 else 1e-5
    for mg, mo, shape in ((cm.CM_MAT_K_MS, oracle_mod.MAT_K_MS, (N,)), (cm.CM_MAT_K_MECH, oracle_mod.MAT_K_MECH, (N, 3))):
        b = rng.normal(size=shape).astype(gs.np_dtype)
        if mg == cm.CM_MAT_K_MS:
            b[5] = 0
        else:
            b[clamp.reshape(N, 3).astype(bool)] = 0
        xg = torch.zeros(shape, dtype=td, device="cuda")
        it, res, rc = gs.cg_solve(mg, dev(b), xg, tol=tol_cg)
        xo, ito, reso, rco = o.cg(mo, b.astype(np.float64).ravel(), tol=tol_cg)
        assert rc == 0 and rco == 0 and res < tol_cg
        # (fp32 against the fp64 oracle at the fp32 rounding floor of a ~300-iteration recurrence: 3 %)
        # fp64: +-1; the ~460-iteration mechanical solve gets 1 % (two runs of the ORACLE differ by +-2 there: DESIGN.md section 8)
        assert abs(it - ito) <= (1 if f64 else max(2, ito // 33)), (mg, it, ito)
        x64 = o.cg(mo, b.astype(np.float64).ravel(), tol=1e-13)[0]
        assert rel(xg.cpu().numpy().ravel(), x64) < (1e-7 if f64 else 2e-3)
        xg.zero_()
        it, res, rc = gs.cg_solve(mg, dev(b), xg, fixed_iters=3)
        x3o = o.cg(mo, b.astype(np.float64).ravel(), fixed=3)[0]
        assert it == 3 and rel(xg.cpu().numpy().ravel(), x3o) < (1e-11 if f64 else 1e-4)


def test_hex_rhs_fields_and_steps(cm, oracle_mod, torch):
    """Element-wise right-hand sides, recovered fields and ten GSPM steps (all terms, x2-stiff non-magnetic inclusion, clamped
    bottom) on hexahedra: <= 1e-12 / 1e-5 on every pass, max |dm| <= 1e-9 (fp64) / 1e-4 (fp32) after ten steps."""
    from paper_2510_09812_b200.inputs import TERM_ANIS, TERM_DEMAG, TERM_FARFIELD, TERM_MAGEL, TERM_ZEEMAN
    ALL = TERM_ANIS | TERM_ZEEMAN | TERM_DEMAG | TERM_FARFIELD | TERM_MAGEL
    mesh = inputs.hex_box((13, 12, 8), (40 * NM, 36 * NM, 22 * NM), seed_mesh=21, seed_perm=22)
    mesh = inputs.flag_inclusion(mesh, np.array(mesh.box) / 2, (9 * NM, 8 * NM, 6 * NM))
    clamp = inputs.clamp_bottom(mesh)
    for dtype, tol, cgt, bar in (("f64", 1e-12, 1e-12, 1e-9), ("f32", 1e-5, 1e-6, 1e-4)):
        gm = cm.Mesh(mesh.xyz, mesh.hexes, mesh.magnetic, mesh.elastic_id, cm.CM_REORDER_MORTON)
        gs = cm.System(gm, mat2(), 1e-12, dtype, clamp, 3)
        o = oracle_mod.Oracle(mesh, mat2(), 1e-12, clamp_dof=clamp, pin_node=3)
        td = torch.float64 if dtype == "f64" else torch.float32
        dev = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=td, device="cuda")
        N = o.N
        rng = np.random.default_rng(8)
        live = o.live().astype(bool)
        assert 0 < (~live).sum() < N
        m = rng.normal(size=(N, 3)); m /= np.linalg.norm(m, axis=1, keepdims=True); m[~live] = 0
        m = m.astype(gs.np_dtype); m64 = m.astype(np.float64)
        U = rng.normal(size=N).astype(gs.np_dtype); u = (1e-3 * rng.normal(size=(N, 3))).astype(gs.np_dtype)
        md, Ud, ud = dev(m), dev(U), dev(u)
        Hext = np.array([3e4, -1e4, 2e4])
        p = cm.make_params(1e-12, Hext, ALL)
        assert rel(gs.field_rhs(cm.CM_RHS_MS, md).cpu().numpy(), o.rhs_ms(m64)) < tol
        assert rel(gs.field_rhs(cm.CM_RHS_MECH, md).cpu().numpy(), o.rhs_mech(m64)) < tol
        hd_o, _ = o.demag_field(U.astype(np.float64), o.volume_average(m64), TERM_DEMAG | TERM_FARFIELD)
        assert rel(gs.field_rhs(cm.CM_OUT_HD, md, Ud, None, p).cpu().numpy(), hd_o) < tol
        sig_o = o.stress_recover(u.astype(np.float64), m64)
        assert rel(gs.field_rhs(cm.CM_OUT_SIGMA, md, None, ud, p).cpu().numpy(), sig_o) < tol
        h_o = o.field(m64, hd_o, sig_o, Hext / 1.2e6, ALL)
        assert rel(gs.field_rhs(cm.CM_OUT_FIELD, md, Ud, ud, p).cpu().numpy(), h_o) < tol
        assert rel(gs.field_rhs(cm.CM_RHS_GS, md, Ud, ud, p, coeff=0.37).cpu().numpy(), o.rhs_gs(m64 + 0.37 * h_o)) < tol
        # ten steps
        m0 = np.array([1.0, 0, 0]) + 0.1 * rng.normal(size=(N, 3)); m0 /= np.linalg.norm(m0, axis=1, keepdims=True); m0[~live] = 0
        mo = m0.copy(); Uo = np.zeros(N); uo = np.zeros((N, 3))
        mg = torch.as_tensor(m0, dtype=td, device="cuda").contiguous()
        Ug = torch.zeros(N, dtype=td, device="cuda"); ug = torch.zeros((N, 3), dtype=td, device="cuda")
        for k in range(10):
            io, rco = o.gspm_step(mo, Uo, uo, 1e-12, [2e4, 0, 0], ALL, cg_tol=cgt)
            ig, rcg = gs.gspm_step(cm.make_params(1e-12, [2e4, 0, 0], ALL, 0, cgt), mg, Ug, ug)
            assert rco == 0 and rcg == 0
            if dtype == "f64" and k == 0:
                assert abs(io.it_ms - ig.it_ms) <= 1 and abs(io.it_mech - ig.it_mech) <= 1
                assert all(abs(io.it_gs[a] - ig.it_gs[a]) <= 1 for a in range(8)) and io.it_mech > 10
        mgh = mg.cpu().numpy().astype(np.float64)
        assert np.abs(mgh - mo).max() <= bar
        assert np.abs(mgh[~live]).max() == 0
        if dtype == "f64":
            assert np.abs(ug.cpu().numpy() - uo).max() <= 1e-9 * max(1.0, np.abs(uo).max())
            assert np.abs(np.linalg.norm(mgh[live], axis=1) - 1).max() <= 4 * np.finfo(float).eps


def test_hex_hysteresis_loop_and_errors(cm, oracle_mod, torch):
    """The device-resident hysteresis loop runs on hexahedra too (two fields of three steps each against the oracle's loop)."""
    from paper_2510_09812_b200.inputs import TERM_ANIS, TERM_DEMAG, TERM_FARFIELD, TERM_ZEEMAN
    terms = TERM_ANIS | TERM_ZEEMAN | TERM_DEMAG | TERM_FARFIELD
    mesh = inputs.hex_box((8, 8, 8), (20 * NM,) * 3, seed_mesh=1, seed_perm=2)
    gm = cm.Mesh(mesh.xyz, mesh.hexes)
    gs = cm.System(gm, inputs.Material(), 1e-12)
    o = oracle_mod.Oracle(mesh, inputs.Material(), 1e-12)
    N = o.N
    rng = np.random.default_rng(5)
    m0 = np.array([1.0, 0, 0]) + 0.1 * rng.normal(size=(N, 3)); m0 /= np.linalg.norm(m0, axis=1, keepdims=True)
    m = m0.copy(); U = np.zeros(N); u = np.zeros((N, 3))
    Hl, ml, sl, res, rc = o.hysteresis_run(m, U, u, 1e-12, [4e4, 0, 0], [-3e4, 0, 0], terms, conv_tol=0.0, max_fields=2, max_steps=3, cg_tol=1e-12)
    mg = torch.as_tensor(m0, dtype=torch.float64, device="cuda").contiguous()
    Ug = torch.zeros(N, dtype=torch.float64, device="cuda")
    Hg, mlg, slg, resg, rcg = gs.hysteresis_run(cm.make_params(1e-12, (0, 0, 0), terms, 0, 1e-12), mg, Ug, None, [4e4, 0, 0], [-3e4, 0, 0],
                                                conv_tol=0.0, max_fields=2, max_steps=3)
    assert rc == 0 and rcg == 0 and resg.n_fields == 2 and list(slg) == [3, 3]
    assert np.array_equal(Hg, Hl) and np.abs(mlg - ml).max() < 1e-11
    assert np.abs(mg.cpu().numpy() - m).max() <= 1e-9
    with pytest.raises(cm.CmError) as e:
        gs.geometry(0)                                            # chunk-blocked element geometry exists for tetrahedra only
    assert e.value.code == cm.CM_E_BADARG
    bad = mesh.hexes.copy(); bad[3] = bad[3][[1, 0, 2, 3, 4, 5, 6, 7]]
    with pytest.raises(cm.CmError) as e:
        cm.Mesh(mesh.xyz, bad)
    assert e.value.code == cm.CM_E_DEGENERATE_TET
    bad = mesh.hexes.copy(); bad[0, 7] = N
    with pytest.raises(cm.CmError) as e:
        cm.Mesh(mesh.xyz, bad)
    assert e.value.code == cm.CM_E_INDEX_RANGE


def test_periodic_hexahedra_parity(cm, oracle_mod, torch):
    """Node-wrapped (fully periodic) hexahedral box with a x2-stiff non-magnetic inclusion, d = 3 displacement DOFs pinned --
    the paper's own setting: structure, matrices, right-hand sides, ten GSPM steps (1e-9 fp64 / 1e-4 fp32)."""
    from paper_2510_09812_b200.inputs import TERM_ANIS, TERM_DEMAG, TERM_FARFIELD, TERM_MAGEL, TERM_ZEEMAN
    ALL = TERM_ANIS | TERM_ZEEMAN | TERM_DEMAG | TERM_FARFIELD | TERM_MAGEL
    mesh = inputs.hex_box((13, 12, 9), (40 * NM, 36 * NM, 26 * NM), seed_mesh=21, seed_perm=22)
    mesh = inputs.flag_inclusion(mesh, np.array(mesh.box) / 2, (9 * NM, 8 * NM, 6 * NM))
    dof, nd = cm.periodic_wrap(mesh.xyz, 7)
    dof_o, nd_o = oracle_mod.periodic_wrap(mesh.xyz, 7)
    assert nd == nd_o == 12 * 11 * 8 and np.array_equal(dof, dof_o)
    clamp = np.zeros((nd, 3), np.uint8); clamp[7] = 1; clamp = clamp.ravel()
    for dtype, tol, cgt, bar in (("f64", 1e-12, 1e-12, 1e-9), ("f32", 1e-5, 1e-6, 1e-4)):
        gm = cm.Mesh(mesh.xyz, mesh.hexes, mesh.magnetic, mesh.elastic_id, cm.CM_REORDER_MORTON, dof_of_node=dof, n_dof=nd)
        assert gm.n_nodes == nd and gm.nnz == 27 * nd
        gs = cm.System(gm, mat2(), 1e-12, dtype, clamp, 3)
        o = oracle_mod.Oracle(mesh, mat2(), 1e-12, clamp_dof=clamp, pin_node=3, dof_of_node=dof, n_dof=nd)
        td = torch.float64 if dtype == "f64" else torch.float32
        dev = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=td, device="cuda")
        vtol = 1e-12 if dtype == "f64" else 2e-7
        order = gm.get(cm.CM_GET_ORDER)
        assert rel(gs.geometry(2), o.mL()[order]) < vtol
        for mg, mo in ((cm.CM_MAT_K_MS, oracle_mod.MAT_K_MS), (cm.CM_MAT_K_GS1, oracle_mod.MAT_K_GS1), (cm.CM_MAT_K_MECH, oracle_mod.MAT_K_MECH)):
            A = _to_user(gm, gs.values(mg), mg == cm.CM_MAT_K_MECH)
            B = o.csr(mo)
            assert abs(A - B).max() < vtol * abs(B).max(), mg
        rng = np.random.default_rng(9)
        live = o.live().astype(bool)
        m = rng.normal(size=(nd, 3)); m /= np.linalg.norm(m, axis=1, keepdims=True); m[~live] = 0
        m = m.astype(gs.np_dtype); m64 = m.astype(np.float64)
        u = (1e-3 * rng.normal(size=(nd, 3))).astype(gs.np_dtype)
        p = cm.make_params(1e-12, [3e4, -1e4, 2e4], ALL)
        assert rel(gs.field_rhs(cm.CM_RHS_MS, dev(m)).cpu().numpy(), o.rhs_ms(m64)) < tol
        assert rel(gs.field_rhs(cm.CM_RHS_MECH, dev(m)).cpu().numpy(), o.rhs_mech(m64)) < tol
        assert rel(gs.field_rhs(cm.CM_OUT_SIGMA, dev(m), None, dev(u), p).cpu().numpy(), o.stress_recover(u.astype(np.float64), m64)) < tol
        assert np.abs(gm.volume_average(dev(m)) - o.volume_average(m64)).max() < (1e-13 if dtype == "f64" else 1e-6)
        m0 = np.array([1.0, 0, 0]) + 0.1 * rng.normal(size=(nd, 3)); m0 /= np.linalg.norm(m0, axis=1, keepdims=True); m0[~live] = 0
        mo_ = m0.copy(); Uo = np.zeros(nd); uo = np.zeros((nd, 3))
        mg_ = torch.as_tensor(m0, dtype=td, device="cuda").contiguous()
        Ug = torch.zeros(nd, dtype=td, device="cuda"); ug = torch.zeros((nd, 3), dtype=td, device="cuda")
        for k in range(10):
            io, rco = o.gspm_step(mo_, Uo, uo, 1e-12, [2e4, 0, 0], ALL, cg_tol=cgt)
            ig, rcg = gs.gspm_step(cm.make_params(1e-12, [2e4, 0, 0], ALL, 0, cgt), mg_, Ug, ug)
            assert rco == 0 and rcg == 0
        assert np.abs(mg_.cpu().numpy().astype(np.float64) - mo_).max() <= bar
    thin = inputs.hex_box((2, 4, 4), (5 * NM, 12 * NM, 12 * NM))
    dof, nd = cm.periodic_wrap(thin.xyz, 1)
    with pytest.raises(cm.CmError) as e:
        cm.Mesh(thin.xyz, thin.hexes, dof_of_node=dof, n_dof=nd)
    assert e.value.code == cm.CM_E_BADARG
