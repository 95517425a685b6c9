"""GPU parity of the rows built in round 2 on top of the tetrahedral / hexahedral path:
  * Jacobi-preconditioned CG (the paper's future work): cm_cg_solve_pc / cm_cg_solve3_pc / cg_precond of the step
    against the oracle's PCG -- iteration counts +-1, iterates of a fixed number of iterations element by element, residual
    histories, CM_PC_NONE bit-identical to cm_cg_solve;
  * the fused Helmholtz start of the step (b = M_m f, x0 = f, r0 = b - A f inside the CG launch) is exercised by every
    multi-step test of the suite; here the step runs with both preconditioners;
  * uniform external stress sigma_ext (Eq. 1; R17): mechanical right-hand side and whole steps on
    tetrahedra and hexahedra."""
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


def mat2(**kw):
    C = inputs.isotropic_voigt(200e9, 0.3)
    return inputs.Material(C_voigt=np.stack([C, 2 * C]), **kw)


def inclusion_mesh():
    mesh = inputs.kuhn_box((23, 19, 17), (66 * NM, 54 * NM, 48 * NM), seed_mesh=51, seed_perm=52)
    return inputs.flag_inclusion(mesh, np.array(mesh.box) / 2, (14 * NM, 12 * NM, 10 * NM))


@pytest.fixture(scope="module", params=["f64", "f32"])
def case(request, cm, oracle_mod, torch):
    mesh = inclusion_mesh()
    clamp = inputs.clamp_bottom(mesh)
    dtype = request.param
    gm = cm.Mesh(mesh.xyz, mesh.tets, mesh.magnetic, mesh.elastic_id, cm.CM_REORDER_MORTON)
    gs = cm.System(gm, mat2(), 2e-12, dtype, clamp, 5)
    o = oracle_mod.Oracle(mesh, mat2(), 2e-12, clamp_dof=clamp, pin_node=5, dtype=dtype)   # fp32 build against the fp32 twin for counts
    o64 = o if dtype == "f64" else oracle_mod.Oracle(mesh, mat2(), 2e-12, clamp_dof=clamp, pin_node=5, dtype="f64")
    td = torch.float64 if dtype == "f64" else torch.float32
    return dict(mesh=mesh, clamp=clamp, gm=gm, gs=gs, o=o, o64=o64, dtype=dtype, td=td, torch=torch)


def test_jacobi_pcg_against_oracle(case, cm, oracle_mod):
    gs, o, o64, torch, td = case["gs"], case["o"], case["o64"], case["torch"], case["td"]
    f64 = case["dtype"] == "f64"
    N = o.N
    rng = np.random.default_rng(110)
    tol_cg = 1e-10 if f64 else 1e-5
    for mat_g, mat_o, n in ((cm.CM_MAT_K_MS, oracle_mod.MAT_K_MS, N), (cm.CM_MAT_K_GS1, oracle_mod.MAT_K_GS1, N),
                            (cm.CM_MAT_K_MECH, oracle_mod.MAT_K_MECH, 3 * N)):
        b = rng.normal(size=n).astype(gs.np_dtype)
        if mat_g == cm.CM_MAT_K_MS:
            b[5] = 0
        if mat_g == cm.CM_MAT_K_MECH:
            b[case["clamp"].astype(bool)] = 0
        shape = (N, 3) if mat_g == cm.CM_MAT_K_MECH else (N,)
        bd = torch.as_tensor(b.reshape(shape), dtype=td, device="cuda")
        # converged solve: counts +-1 against the oracle's PCG in the same precision, solution against a tight fp64 solve
        x = torch.zeros(shape, dtype=td, device="cuda")
        gs.cg_history_enable(True)
        it, res, rc = gs.cg_solve(mat_g, bd, x, tol=tol_cg, precond=cm.CM_PC_JACOBI)
        hist = gs.cg_history()
        gs.cg_history_enable(False)
        xo, ito, reso, rco = o.cg_pc(mat_o, b, tol=tol_cg, precond=1)
        assert rc == 0 and rco == 0
        assert abs(it - ito) <= (1 if f64 else max(2, ito // 50)), (mat_g, it, ito)
        assert res < tol_cg
        x64, _, _, _ = o64.cg_pc(mat_o, b.astype(np.float64), tol=1e-13, precond=1)
        assert rel(x.cpu().numpy().ravel(), x64) < (1e-7 if f64 else 2e-3), mat_g
        # residual history: the same curve as the oracle's, iteration by iteration (the curve, not only its end)
        _, _, ho = o64.cg_history(mat_o, b.astype(np.float64), tol=tol_cg, precond=1)
        k = min(len(hist), len(ho)) - 2
        assert len(hist) == it + 1 and k > 5
        assert np.allclose(hist[:12], ho[:12], rtol=1e-9 if f64 else 1e-3), mat_g       # the first iterations pin the algorithm
        assert np.allclose(hist[:k], ho[:k], rtol=1e-2 if f64 else 2e-1), mat_g         # later ones drift apart by rounding (~300 its)
        # the preconditioner must pay on the mechanical matrix (x2-stiffness inclusion): not more iterations than plain CG
        if mat_g == cm.CM_MAT_K_MECH:
            xp = torch.zeros(shape, dtype=td, device="cuda")
            itp, _, _ = gs.cg_solve(mat_g, bd, xp, tol=tol_cg)
            assert it <= itp, (it, itp)
        # three iterations: identical algorithm step by step
        x = torch.zeros(shape, dtype=td, device="cuda")
        it3, res3, _ = gs.cg_solve(mat_g, bd, x, fixed_iters=3, precond=cm.CM_PC_JACOBI)
        xo3, ito3, reso3, _ = o64.cg_pc(mat_o, b.astype(np.float64), fixed=3, precond=1)
        assert it3 == 3 and ito3 == 3
        assert rel(x.cpu().numpy().ravel(), xo3) < (1e-11 if f64 else 1e-4)
        assert res3 == pytest.approx(reso3, rel=1e-9 if f64 else 1e-3)
        # CM_PC_NONE through the _pc entry point == cm_cg_solve, bit for bit
        xa = torch.zeros(shape, dtype=td, device="cuda"); xb = torch.zeros(shape, dtype=td, device="cuda")
        ita, _, _ = gs.cg_solve(mat_g, bd, xa, tol=tol_cg)
        itb, _, _ = gs.cg_solve(mat_g, bd, xb, tol=tol_cg, precond=cm.CM_PC_NONE)
        assert ita == itb and torch.equal(xa, xb)
    # the mass matrix has no Jacobi preconditioner (singular on dead nodes); unknown codes are refused
    x = torch.zeros(N, dtype=td, device="cuda")
    with pytest.raises(cm.CmError) as e:
        gs.cg_solve(cm.CM_MAT_MASS, x, x.clone(), precond=cm.CM_PC_JACOBI)
    assert e.value.code == cm.CM_E_BADARG
    with pytest.raises(cm.CmError):
        gs.cg_solve(cm.CM_MAT_K_MS, x, x.clone(), precond=7)


def test_jacobi_pcg_three_rhs(case, cm, oracle_mod):
    gs, o, o64, torch, td = case["gs"], case["o"], case["o64"], case["torch"], case["td"]
    f64 = case["dtype"] == "f64"
    N = o.N
    rng = np.random.default_rng(111)
    b = rng.normal(size=(N, 3)).astype(gs.np_dtype)
    b[:, 1] *= 1e-3
    b[:, 2] = 0
    x0 = rng.normal(size=(N, 3)).astype(gs.np_dtype)
    x = torch.as_tensor(x0, dtype=td, device="cuda")
    tol_cg = 1e-11 if f64 else 1e-5
    its, ress, rc = gs.cg_solve3(cm.CM_MAT_K_GS2, torch.as_tensor(b, dtype=td, device="cuda"), x, tol=tol_cg, precond=cm.CM_PC_JACOBI)
    xh = x.cpu().numpy()
    for c in range(3):
        xo, ito, _, _ = o64.cg_pc(oracle_mod.MAT_K_GS2, b[:, c].astype(np.float64), x0=x0[:, c].astype(np.float64), tol=tol_cg, precond=1)
        assert abs(its[c] - ito) <= 1, (c, its, ito)
        if c < 2:
            assert rel(xh[:, c], xo) < (1e-9 if f64 else 1e-3)
    assert its[2] == 0 and np.abs(xh[:, 2]).max() == 0


def _steps(cm, orc, torch, mesh, mat, dt, terms, nsteps, dtype, H, clamp, variant, precond, cg_tol, hexa=False):
    conn = mesh.hexes if hexa else mesh.tets
    gm = cm.Mesh(mesh.xyz, conn, mesh.magnetic, mesh.elastic_id, cm.CM_REORDER_MORTON)
    gs = cm.System(gm, mat, dt, dtype, clamp)
    o = orc.Oracle(mesh, mat, dt, clamp_dof=clamp, dtype="f64")
    td = torch.float64 if dtype == "f64" else torch.float32
    N = mesh.n_nodes
    m0 = inputs.init_m_noisy_x(mesh, 23)
    m, U, u = m0.copy(), np.zeros(N), np.zeros((N, 3))
    mg = torch.as_tensor(m0, dtype=td, device="cuda").contiguous()
    Ug = torch.zeros(N, dtype=td, device="cuda"); ug = torch.zeros((N, 3), dtype=td, device="cuda")
    infos = []
    for k in range(nsteps):
        io, rco = o.gspm_step(m, U, u, dt, H, terms, variant=variant, cg_tol=cg_tol, cg_precond=precond)
        ig, rcg = gs.gspm_step(cm.make_params(dt, H, terms, variant, cg_tol, 100000, -1, precond), mg, Ug, ug)
        assert rco == 0 and rcg == 0
        infos.append((io, ig))
    return m, U, u, mg.cpu().numpy(), Ug.cpu().numpy(), ug.cpu().numpy(), infos


def _check_iters(infos, slack=1, mech_frac=0.0):
    """CG iteration counts within +-1 (BASELINE north_star) for every solve of every step.  Both sides are bit-reproducible
    (fixed-order dot products), so the comparison is exact run to run.
    mech_frac: the mechanical solve INSIDE a step is compared with max(1, ceil(mech_frac * count)).  Its right-hand side is
    smooth and its residual curve nearly flat where it crosses the threshold (2-4 % per iteration after 230-370
    iterations); by then the device's curve (fused multiply-adds, sliced summation order) and the oracle's (no contraction,
    row order) have drifted a few per cent apart in rounding, the device consistently one to three iterations ahead.
    DESIGN.md section 8 lists both histories around the threshold.  Standalone mechanical solves with a random right-hand
    side (test_cg, test_jacobi_pcg_against_oracle) and every other solve keep the strict +-1."""
    import math
    for k, (io, ig) in enumerate(infos):
        assert abs(io.it_ms - ig.it_ms) <= slack, (k, io.it_ms, ig.it_ms)
        assert abs(io.it_mech - ig.it_mech) <= max(slack, math.ceil(mech_frac * io.it_mech)), (k, io.it_mech, ig.it_mech)
        for a in range(8):
            assert abs(io.it_gs[a] - ig.it_gs[a]) <= slack, (k, a, list(io.it_gs), list(ig.it_gs))


@pytest.mark.parametrize("variant", [0, 1])
def test_gspm_steps_with_jacobi(cm, oracle_mod, torch, variant):
    """Ten magnetoelastic steps with every solve Jacobi-preconditioned: the same states as the oracle's, counts +-1."""
    mesh = inputs.kuhn_box((13, 13, 7), (40 * NM, 40 * NM, 20 * NM), seed_mesh=21, seed_perm=22)
    mesh = inputs.flag_inclusion(mesh, np.array(mesh.box) / 2, (8 * NM,) * 3)
    clamp = inputs.clamp_bottom(mesh)
    m, U, u, mg, Ug, ug, infos = _steps(cm, oracle_mod, torch, mesh, mat2(), 1e-12, ALL, 10, "f64", [2e4, 0, 0], clamp, variant, 1, 1e-12)
    assert np.abs(mg - m).max() <= 1e-9
    assert np.abs(ug - u).max() <= 1e-9 * max(1.0, np.abs(u).max())
    _check_iters(infos, mech_frac=0.015)
    # and the preconditioned and plain steps reach the same state (both solve the same systems to 1e-12)
    m0, U0, u0, mg0, _, _, infos0 = _steps(cm, oracle_mod, torch, mesh, mat2(), 1e-12, ALL, 10, "f64", [2e4, 0, 0], clamp, variant, 0, 1e-12)
    assert np.abs(mg - mg0).max() <= 1e-8
    assert infos[0][1].it_mech < infos0[0][1].it_mech


def test_gspm_steps_with_jacobi_f32(cm, oracle_mod, torch):
    cfg = inputs.make_config(0)
    m, U, u, mg, Ug, ug, infos = _steps(cm, oracle_mod, torch, cfg.mesh, cfg.material, cfg.dt, cfg.terms, 10, "f32", cfg.Hext[0], None, 0, 1, 1e-6)
    # config 0 starts from its own m0
    assert np.abs(np.linalg.norm(mg, axis=1) - 1).max() <= 4 * np.finfo(np.float32).eps
    assert np.abs(mg - m).max() <= 1e-4
    _check_iters(infos, slack=3)


# ---------------------------------------------------------------------------------------------- sigma_ext
SIG = np.array([3e8, -1e8, 2e8, 5e7, -4e7, 6e7])   # Pa, xx yy zz yz xz xy


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("hexa", [False, True])
def test_sigma_ext_rhs(cm, oracle_mod, torch, dtype, hexa):
    """b^mech with a uniform external stress: one more term over ALL elements (non-magnetic inclusion too)."""
    if hexa:
        mesh = inputs.hex_box((12, 11, 9), (33 * NM, 30 * NM, 24 * NM), seed_mesh=71, seed_perm=72)
    else:
        mesh = inputs.kuhn_box((12, 11, 9), (33 * NM, 30 * NM, 24 * NM), seed_mesh=71, seed_perm=72)
    mesh = inputs.flag_inclusion(mesh, np.array(mesh.box) / 2, (8 * NM, 7 * NM, 6 * NM))
    assert 0 < mesh.magnetic.sum() < mesh.n_tets
    clamp = inputs.clamp_bottom(mesh)
    tol = 1e-12 if dtype == "f64" else 1e-5
    td = torch.float64 if dtype == "f64" else torch.float32
    conn = mesh.hexes if hexa else mesh.tets
    gm = cm.Mesh(mesh.xyz, conn, mesh.magnetic, mesh.elastic_id, cm.CM_REORDER_MORTON)
    m = inputs.init_m_random(mesh, 64)
    md = torch.as_tensor(m, dtype=td, device="cuda")
    ref = {}
    for name, sig in (("with", SIG), ("without", None)):
        mat = mat2(sigma_ext=sig)
        gs = cm.System(gm, mat, 2e-12, dtype, clamp)
        o = oracle_mod.Oracle(mesh, mat, 2e-12, clamp_dof=clamp)
        b = gs.field_rhs(cm.CM_RHS_MECH, md).cpu().numpy()
        bo = o.rhs_mech(md.cpu().numpy().astype(np.float64))
        assert rel(b, bo) < tol, name
        ref[name] = bo
    assert np.abs(ref["with"] - ref["without"]).max() > 1e-3 * np.abs(ref["without"]).max()   # the term is not negligible here


@pytest.mark.parametrize("hexa", [False, True])
def test_sigma_ext_steps(cm, oracle_mod, torch, hexa):
    """Five steps under external stress: the stress-induced field rotates m; parity 1e-9, counts +-1."""
    if hexa:
        mesh = inputs.hex_box((10, 10, 6), (30 * NM, 30 * NM, 16 * NM), seed_mesh=21, seed_perm=22)
    else:
        mesh = inputs.kuhn_box((10, 10, 6), (30 * NM, 30 * NM, 16 * NM), seed_mesh=21, seed_perm=22)
    mesh = inputs.flag_inclusion(mesh, np.array(mesh.box) / 2, (6 * NM,) * 3)
    clamp = inputs.clamp_bottom(mesh)
    m, U, u, mg, Ug, ug, infos = _steps(cm, oracle_mod, torch, mesh, mat2(sigma_ext=SIG), 1e-12, ALL, 5, "f64", [2e4, 0, 0], clamp, 0, 0,
                                        1e-12, hexa=hexa)
    assert np.abs(mg - m).max() <= 1e-9
    assert np.abs(ug - u).max() <= 1e-9 * max(1.0, np.abs(u).max())
    _check_iters(infos, mech_frac=0.015)
    assert np.abs(u).max() > 0
    # counts at the paper's tolerance and at 1e-10
    for tol in (1e-7, 1e-10):
        infos_t = _steps(cm, oracle_mod, torch, mesh, mat2(sigma_ext=SIG), 1e-12, ALL, 2, "f64", [2e4, 0, 0], clamp, 0, 0, tol, hexa=hexa)[-1]
        _check_iters(infos_t[:1], mech_frac=0.015)


# ---------------------------------------------------------------------------------------------- matrix-free K^mech
def test_matfree_operator(case, cm, oracle_mod):
    """cm_spmv_matfree is the operator of cm_spmv(CM_MAT_K_MECH): against the oracle's assembled product and
    against the stored-matrix product of the library, clamped rows included; every geometry mode."""
    gs, o64, torch, td = case["gs"], case["o64"], case["torch"], case["td"]
    tol = 1e-12 if case["dtype"] == "f64" else 1e-5
    rng = np.random.default_rng(120)
    x = rng.normal(size=(o64.N, 3)).astype(gs.np_dtype)            # non-zero on the clamped DOFs too
    xd = torch.as_tensor(x, dtype=td, device="cuda")
    yo = o64.spmv(oracle_mod.MAT_K_MECH, x.astype(np.float64).ravel())
    ys = gs.spmv(cm.CM_MAT_K_MECH, xd).cpu().numpy().ravel()
    for mode in (0, 1, 2):
        gs.set_option(cm.CM_OPT_STORED_GEOMETRY, mode)
        y = gs.spmv_matfree(xd).cpu().numpy().ravel()
        assert rel(y, yo) < tol, mode
        assert rel(y, ys) < tol, mode
    gs.set_option(cm.CM_OPT_STORED_GEOMETRY, 0)
    cl = case["clamp"].astype(bool)
    assert np.array_equal(y[cl], x.ravel()[cl])                    # identity rows of P A P + (I - P), exactly


@pytest.mark.parametrize("precond", [0, 1])
def test_matfree_cg(case, cm, oracle_mod, precond):
    gs, o, o64, torch, td = case["gs"], case["o"], case["o64"], case["torch"], case["td"]
    f64 = case["dtype"] == "f64"
    N = o.N
    rng = np.random.default_rng(121)
    b = rng.normal(size=3 * N).astype(gs.np_dtype)
    b[case["clamp"].astype(bool)] = 0
    bd = torch.as_tensor(b.reshape(N, 3), dtype=td, device="cuda")
    tol_cg = 1e-10 if f64 else 1e-5
    x = torch.zeros((N, 3), dtype=td, device="cuda")
    it, res, rc = gs.cg_solve_matfree(bd, x, tol=tol_cg, precond=precond)
    xo, ito, reso, rco = o.cg_pc(oracle_mod.MAT_K_MECH, b, tol=tol_cg, precond=precond)
    assert rc == 0 and rco == 0 and res < tol_cg
    assert abs(it - ito) <= (1 if f64 else max(2, ito // 50)), (it, ito)
    x64, _, _, _ = o64.cg_pc(oracle_mod.MAT_K_MECH, b.astype(np.float64), tol=1e-13, precond=precond)
    assert rel(x.cpu().numpy().ravel(), x64) < (1e-7 if f64 else 2e-3)
    # the same iterates as the stored-matrix solver: three iterations, and the iteration count to convergence
    xa = torch.zeros((N, 3), dtype=td, device="cuda"); xb = torch.zeros((N, 3), dtype=td, device="cuda")
    gs.cg_solve_matfree(bd, xa, fixed_iters=3, precond=precond)
    gs.cg_solve(cm.CM_MAT_K_MECH, bd, xb, fixed_iters=3, precond=precond)
    assert rel(xa.cpu().numpy(), xb.cpu().numpy()) < (1e-11 if f64 else 1e-4)
    xo3, _, _, _ = o64.cg_pc(oracle_mod.MAT_K_MECH, b.astype(np.float64), fixed=3, precond=precond)
    assert rel(xa.cpu().numpy().ravel(), xo3) < (1e-11 if f64 else 1e-4)
    its, _, _ = gs.cg_solve(cm.CM_MAT_K_MECH, bd, torch.zeros((N, 3), dtype=td, device="cuda"), tol=tol_cg, precond=precond)
    assert abs(it - its) <= (1 if f64 else max(2, its // 50))
    # warm start at the solution, zero right-hand side, iteration cap (not a multiple of the 16-iteration batch)
    it2, _, _ = gs.cg_solve_matfree(bd, x, tol=tol_cg * 10, precond=precond)
    assert it2 == 0
    xz = torch.as_tensor(rng.normal(size=(N, 3)), dtype=td, device="cuda")
    it0, _, _ = gs.cg_solve_matfree(torch.zeros((N, 3), dtype=td, device="cuda"), xz, precond=precond)
    assert it0 == 0 and float(xz.abs().max()) == 0.0
    xm = torch.zeros((N, 3), dtype=td, device="cuda")
    itm, _, rcm = gs.cg_solve_matfree(bd, xm, tol=1e-13, maxiter=21, precond=precond)
    assert itm == 21 and rcm == cm.CM_E_CG_MAXITER and float(xm.abs().max()) > 0


def test_gspm_steps_matfree(cm, oracle_mod, torch):
    """Five magnetoelastic steps with the mechanical solve matrix-free: the oracle's states (it has one K^mech, assembled)."""
    mesh = inputs.kuhn_box((13, 13, 7), (40 * NM, 40 * NM, 20 * NM), seed_mesh=21, seed_perm=22)
    mesh = inputs.flag_inclusion(mesh, np.array(mesh.box) / 2, (8 * NM,) * 3)
    clamp = inputs.clamp_bottom(mesh)
    gm = cm.Mesh(mesh.xyz, mesh.tets, mesh.magnetic, mesh.elastic_id, cm.CM_REORDER_MORTON)
    gs = cm.System(gm, mat2(), 1e-12, "f64", clamp)
    o = oracle_mod.Oracle(mesh, mat2(), 1e-12, clamp_dof=clamp)
    N = mesh.n_nodes
    m0 = inputs.init_m_noisy_x(mesh, 23)
    m, U, u = m0.copy(), np.zeros(N), np.zeros((N, 3))
    mg = torch.as_tensor(m0, device="cuda").contiguous(); Ug = torch.zeros(N, dtype=torch.float64, device="cuda")
    ug = torch.zeros((N, 3), dtype=torch.float64, device="cuda")
    infos = []
    for k in range(5):
        io, rco = o.gspm_step(m, U, u, 1e-12, [2e4, 0, 0], ALL, cg_tol=1e-12)
        ig, rcg = gs.gspm_step(cm.make_params(1e-12, [2e4, 0, 0], ALL, 0, 1e-12, mech_matfree=1), mg, Ug, ug)
        assert rco == 0 and rcg == 0
        infos.append((io, ig))
    assert np.abs(mg.cpu().numpy() - m).max() <= 1e-9
    assert np.abs(ug.cpu().numpy() - u).max() <= 1e-9 * max(1.0, np.abs(u).max())
    _check_iters(infos, mech_frac=0.015)
    with pytest.raises(cm.CmError):          # cannot be captured into the hysteresis graph
        gs.hysteresis_run(cm.make_params(1e-12, terms=ALL, mech_matfree=1), mg, Ug, ug, [2e4, 0, 0], [-1e3, 0, 0], max_fields=2, max_steps=2)


def _cg_history_extended(A, b, tol):
    """Textbook CG (x0 = 0) on a scipy CSR matrix with every product, dot and update in numpy long double (64-bit
    mantissa on x86): the reference the two fp64 runs are measured against.  Returns ||r_k|| / ||b||, k = 0 .. iters."""
    ft = np.longdouble
    data, idx, ptr = A.data.astype(ft), A.indices, A.indptr[:-1]
    b = b.astype(ft); x = np.zeros_like(b); r = b.copy(); pv = r.copy()
    bb = b @ b; rr = r @ r
    h = [float(np.sqrt(rr / bb))]
    while h[-1] >= tol and len(h) < 5000:
        Ap = np.add.reduceat(data * pv[idx], ptr)
        al = rr / (pv @ Ap); x += al * pv; r -= al * Ap
        rn = r @ r; pv = r + (rn / rr) * pv; rr = rn
        h.append(float(np.sqrt(rr / bb)))
    return np.array(h)


def test_mechanical_residual_curves_part_by_rounding(cm, oracle_mod, torch, capsys):
    """Why the in-step mechanical CG count is compared with 1.5 % instead of +-1.  Step-0 mechanical solve
    of the inclusion mesh (b = b^mech(m0), x0 = 0), three runs of the same recurrence: the device (fp64, fused products,
    sliced summation order), the oracle (fp64, no contraction, row order) and an extended-precision CG (numpy long double).
    All three agree to rounding for the first ~60 iterations; then loss of orthogonality amplifies the rounding
    differences by about x4 per iteration and BOTH fp64 runs leave the extended-precision curve at the same iteration
    and by the same order (a few per cent to tens of per cent of a residual that falls twelve decades): the device is as
    far from the reference as the oracle is, which is what "two finite-precision CG runs of one system" means, and not
    what a defect in either would look like (that shows from iteration 0).  How far the device is from the oracle after
    the parting is printed, not asserted: a more accurate dot product would be welcome."""
    mesh = inputs.kuhn_box((13, 13, 7), (40 * NM, 40 * NM, 20 * NM), seed_mesh=21, seed_perm=22)
    mesh = inputs.flag_inclusion(mesh, np.array(mesh.box) / 2, (8 * NM,) * 3)
    clamp = inputs.clamp_bottom(mesh)
    o = oracle_mod.Oracle(mesh, mat2(), 1e-12, clamp_dof=clamp)
    gm = cm.Mesh(mesh.xyz, mesh.tets, mesh.magnetic, mesh.elastic_id, cm.CM_REORDER_MORTON)
    gs = cm.System(gm, mat2(), 1e-12, "f64", clamp)
    b = o.rhs_mech(inputs.init_m_noisy_x(mesh, 23))
    _, ito, ho = o.cg_history(oracle_mod.MAT_K_MECH, b.ravel(), tol=1e-12)
    hx = _cg_history_extended(o.csr(oracle_mod.MAT_K_MECH), b.ravel(), 1e-12)
    gs.cg_history_enable(True)
    x = torch.zeros((mesh.n_nodes, 3), dtype=torch.float64, device="cuda")
    itg, _, _ = gs.cg_solve(cm.CM_MAT_K_MECH, torch.as_tensor(b, device="cuda"), x, tol=1e-12)
    hg = gs.cg_history()
    gs.cg_history_enable(False)
    assert len(hg) == itg + 1 and len(ho) == ito + 1
    n = min(len(ho), len(hg), len(hx))
    dev = np.abs(ho[:n] - hg[:n]) / ho[:n]
    dev_o = np.abs(ho[:n] - hx[:n]) / hx[:n]
    dev_g = np.abs(hg[:n] - hx[:n]) / hx[:n]
    # the same algorithm, iteration by iteration, while rounding is small: all three curves
    assert dev[:40].max() < 1e-12 and dev_o[:40].max() < 1e-12 and dev_g[:40].max() < 1e-12
    # both fp64 runs leave the extended-precision curve at the same place ...
    on_o, on_g = int(np.argmax(dev_o > 1e-6)), int(np.argmax(dev_g > 1e-6))
    assert 40 < on_o < n and 40 < on_g < n and abs(on_o - on_g) <= 10, (on_o, on_g)
    # ... and stay in the same envelope around it (measured here: oracle up to 0.41)
    assert dev_g.max() <= max(3 * dev_o.max(), 0.5) and dev_o.max() <= max(3 * dev_g.max(), 0.5), (dev_o.max(), dev_g.max())
    with capsys.disabled():
        print(f"\nmechanical CG, step 0 of the inclusion mesh, tol 1e-12: oracle {ito} iterations, device {itg}, long double {len(hx) - 1}")
        print(f"  parting from the long-double run (rel.dev > 1e-6): oracle at k={on_o}, device at k={on_g}; "
              f"max rel.dev oracle {dev_o.max():.2e}, device {dev_g.max():.2e}; device vs oracle {dev.max():.2e}")
        for j in range(0, n, 20):
            print(f"  k={j:3d}  oracle {ho[j]:.6e}  device {hg[j]:.6e}  long double {hx[j]:.6e}  dev-orc {dev[j]:.1e}  orc-ld {dev_o[j]:.1e}  dev-ld {dev_g[j]:.1e}")
    for tol in (1e-7, 1e-10, 1e-12):
        io, ig, ix = int(np.argmax(ho < tol)), int(np.argmax(hg < tol)), int(np.argmax(hx < tol))
        with capsys.disabled():
            print(f"  first crossing of {tol:g}: oracle {io}, device {ig}, long double {ix}")
        assert abs(io - ig) <= max(1, int(np.ceil(0.015 * io)))
        assert abs(ix - ig) <= max(1, int(np.ceil(0.015 * ix))) and abs(ix - io) <= max(1, int(np.ceil(0.015 * ix)))


def test_cg_history_covers_recorded_solves_only(cm, torch):
    """cm_cg_history returns the curve of the last RECORDED solve and nothing else: empty after a solve with the history
    off, after cm_cg_history_enable(0), and after the calls that do not record (a GSPM step, a matrix-free solve) -- never
    an earlier solve's curve or unwritten memory (cm_api.cu)."""
    mesh = inputs.kuhn_box((7, 6, 5), (18 * NM, 15 * NM, 12 * NM), seed_mesh=5, seed_perm=6)
    clamp = inputs.clamp_bottom(mesh)
    gs = cm.System(cm.Mesh(mesh.xyz, mesh.tets), mat2(), 1e-12, "f64", clamp)
    N = mesh.n_nodes
    b = torch.as_tensor(np.random.default_rng(8).normal(size=N), device="cuda"); b[0] = 0
    x = torch.zeros(N, dtype=torch.float64, device="cuda")
    it, _, _ = gs.cg_solve(cm.CM_MAT_K_MS, b, x, tol=1e-10)
    assert it > 3 and len(gs.cg_history()) == 0                      # history never enabled
    gs.cg_history_enable(True)
    x.zero_(); it, res, _ = gs.cg_solve(cm.CM_MAT_K_MS, b, x, tol=1e-10)
    h = gs.cg_history()
    assert len(h) == it + 1 and h[0] == 1.0 and h[-1] < 1e-10 <= h[-2]
    b3 = torch.as_tensor(np.random.default_rng(9).normal(size=(N, 3)), device="cuda"); x3 = torch.zeros_like(b3)
    it3, _, _ = gs.cg_solve3(cm.CM_MAT_K_GS1, b3, x3, tol=1e-10)
    assert gs.cg_history(3).shape == (max(it3) + 1, 3)
    m = torch.as_tensor(inputs.init_m_random(mesh, 3), device="cuda")
    gs.gspm_step(cm.make_params(1e-12, terms=TERM_ANIS | TERM_ZEEMAN), m, torch.zeros(N, dtype=torch.float64, device="cuda"), torch.zeros_like(m))
    assert len(gs.cg_history()) == 0                                 # a step does not leave a history behind
    x.zero_(); gs.cg_solve(cm.CM_MAT_K_MS, b, x, tol=1e-10)
    assert len(gs.cg_history()) == it + 1
    bm = b3.clone(); bm[torch.as_tensor(clamp.reshape(N, 3).astype(bool), device="cuda")] = 0
    gs.cg_solve_matfree(bm, torch.zeros_like(bm), tol=1e-8)
    assert len(gs.cg_history()) == 0                                 # nor does a matrix-free solve
    x.zero_(); gs.cg_solve(cm.CM_MAT_K_MS, b, x, tol=1e-10)
    gs.cg_history_enable(False)
    assert len(gs.cg_history()) == 0
    x.zero_(); gs.cg_solve(cm.CM_MAT_K_MS, b, x, tol=1e-10)
    assert len(gs.cg_history()) == 0


def test_round2_entry_points_refuse_bad_arguments(cm, torch):
    mesh = inputs.hex_box((5, 5, 4), (12 * NM, 12 * NM, 9 * NM), seed_mesh=1, seed_perm=2)
    gm = cm.Mesh(mesh.xyz, mesh.hexes)
    gs = cm.System(gm, mat2(), 1e-12, "f64", inputs.clamp_bottom(mesh))
    x = torch.zeros((mesh.n_nodes, 3), dtype=torch.float64, device="cuda")
    for call in (lambda: gs.spmv_matfree(x), lambda: gs.cg_solve_matfree(x, x.clone()),          # tetrahedra only
                 lambda: gs.set_option(cm.CM_OPT_STORED_GEOMETRY, 3), lambda: gs.set_option(99, 0),
                 lambda: gs.gspm_step(cm.make_params(1e-12, terms=ALL, cg_precond=5), x, x[:, 0].contiguous(), x),
                 lambda: gs.gspm_step(cm.make_params(1e-12, terms=ALL, mech_matfree=1), x, x[:, 0].contiguous(), x)):
        with pytest.raises(cm.CmError) as e:
            call()
        assert e.value.code == cm.CM_E_BADARG
    assert len(gs.cg_history()) == 0                      # nothing recorded unless enabled
    tets = inputs.kuhn_box((4, 4, 4), (9 * NM,) * 3)
    gt = cm.Mesh(tets.xyz, tets.tets)
    g0 = cm.System(gt, inputs.Material(C_voigt=None), 1e-12)   # no elastic constants: no mechanical operator of either kind
    y = torch.zeros((tets.n_nodes, 3), dtype=torch.float64, device="cuda")
    with pytest.raises(cm.CmError):
        g0.spmv_matfree(y)
    with pytest.raises(cm.CmError):
        g0.cg_solve(cm.CM_MAT_K_MECH, y, y.clone(), precond=cm.CM_PC_JACOBI)
