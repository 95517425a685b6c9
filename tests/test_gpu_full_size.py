"""GPU parity at BASELINE.json's FULL size: config 3 (245x245x50 = 3,001,250 nodes, 17.5 M tets, 44.3 M nonzeros), fp64,
Morton order -- the launch configuration `bench.py` times.  The oracle is fast enough per operation to compute every
output of a single pass at this size (SpMV, right-hand sides, fields, a few CG iterations, one step with fixed
iteration counts), so outputs are compared element by element, not sampled; what it cannot afford is the ~2000
iterations per solve of a converged step, which the mid-size tests cover.  Tolerances: DESIGN.md section 8."""
import os

import numpy as np
import pytest

from paper_2510_09812_b200 import inputs

pytestmark = pytest.mark.gpu


def rel(a, b):
    a = np.asarray(a, np.float64); b = np.asarray(b, np.float64)
    return np.abs(a - b).max() / max(np.abs(b).max(), 1e-300)


@pytest.fixture(scope="module")
def full(oracle_mod):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    from paper_2510_09812_b200 import binding as cm
    cfg = inputs.make_config(3)
    gm = cm.Mesh(cfg.mesh.xyz, cfg.mesh.tets, cfg.mesh.magnetic, cfg.mesh.elastic_id, cm.CM_REORDER_MORTON)
    gs = cm.System(gm, cfg.material, cfg.dt, "f64", cfg.clamp_dof, cfg.pin_node)
    o = oracle_mod.Oracle(cfg.mesh, cfg.material, cfg.dt, clamp_dof=cfg.clamp_dof, pin_node=cfg.pin_node)
    return cfg, cm, gm, gs, o, torch


def _dev(torch, a):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device="cuda")


def test_full_size_structure(full, oracle_mod):
    cfg, cm, gm, gs, o, torch = full
    assert cfg.mesh.n_nodes == 3001250 and cfg.mesh.n_tets == 17503584
    assert gm.nnz == o.nnz == 44344708
    order = gm.get(cm.CM_GET_ORDER)
    order_o, _ = oracle_mod.reorder(cfg.mesh.xyz, cfg.mesh.tets, 1)[:2]
    assert np.array_equal(order, order_o)                       # Morton order, bit-exact (R21)
    # pattern: row i of the library = row order[i] of the oracle with columns relabelled, ascending
    iperm = gm.get(cm.CM_GET_IPERM)
    rp, ci = gm.get(cm.CM_GET_ROWPTR), gm.get(cm.CM_GET_COLIDX)
    rpo, cio = o.rowptr(), o.colidx()
    assert np.array_equal(np.diff(rp), np.diff(rpo)[order])
    rng = np.random.default_rng(0)
    for i in rng.integers(0, o.N, 2000):                        # sampled rows: column sets
        a = ci[rp[i]:rp[i + 1]]
        b = np.sort(iperm[cio[rpo[order[i]]:rpo[order[i] + 1]]])
        assert np.array_equal(a, b)
    # volumes sum to the box volume (closed form) in the library's own geometry
    V = gs.geometry(0)
    box = np.array(cfg.mesh.box) / cfg.material.length_scale
    assert abs(V.sum() - box.prod()) <= 1e-12 * box.prod()


def test_full_size_spmv_and_rhs(full, oracle_mod):
    cfg, cm, gm, gs, o, torch = full
    rng = np.random.default_rng(41)
    N = o.N
    for mg, mo in ((cm.CM_MAT_K_MS, oracle_mod.MAT_K_MS), (cm.CM_MAT_K_GS1, oracle_mod.MAT_K_GS1),
                   (cm.CM_MAT_K_GS2, oracle_mod.MAT_K_GS2), (cm.CM_MAT_MASS, oracle_mod.MAT_MASS)):
        x = rng.normal(size=N)
        assert rel(gs.spmv(mg, _dev(torch, x)).cpu().numpy(), o.spmv(mo, x)) < 1e-12, mg
    x = rng.normal(size=(N, 3))
    y = gs.spmv(cm.CM_MAT_K_MECH, _dev(torch, x)).cpu().numpy()
    assert rel(y.ravel(), o.spmv(oracle_mod.MAT_K_MECH, x.ravel())) < 1e-12
    assert rel(gs.spmv3(cm.CM_MAT_MASS, _dev(torch, x)).cpu().numpy(), o.rhs_gs(x)) < 1e-12

    m = cfg.m0
    md = _dev(torch, m)
    mbar = gm.volume_average(md)
    assert np.abs(mbar - o.volume_average(m)).max() < 1e-12        # 17.5 M-term sums in different orders
    assert rel(gs.field_rhs(cm.CM_RHS_MS, md).cpu().numpy(), o.rhs_ms(m)) < 1e-12
    assert rel(gs.field_rhs(cm.CM_RHS_MECH, md).cpu().numpy(), o.rhs_mech(m)) < 1e-12
    U = rng.normal(size=N); u = 1e-3 * rng.normal(size=(N, 3))
    p = cm.make_params(cfg.dt, cfg.Hext[3], cfg.terms)
    hd_o, _ = o.demag_field(U, o.volume_average(m), cfg.terms)
    assert rel(gs.field_rhs(cm.CM_OUT_HD, md, _dev(torch, U), None, p).cpu().numpy(), hd_o) < 1e-12
    sig_o = o.stress_recover(u, m)
    assert rel(gs.field_rhs(cm.CM_OUT_SIGMA, md, None, _dev(torch, u), p).cpu().numpy(), sig_o) < 1e-12
    h_o = o.field(m, hd_o, sig_o, np.asarray(cfg.Hext[3]) / cfg.material.Ms, cfg.terms)
    assert rel(gs.field_rhs(cm.CM_OUT_FIELD, md, _dev(torch, U), _dev(torch, u), p).cpu().numpy(), h_o) < 1e-12


def test_full_size_cg_fixed_iterations(full, oracle_mod):
    """The persistent CG kernels in the bench's launch shape (296 CTAs over 3 M rows): three textbook iterations
    against the oracle's, element by element; then the CG invariants at a size the oracle cannot iterate to
    convergence: the true residual of the returned iterate equals the reported recurrence residual."""
    cfg, cm, gm, gs, o, torch = full
    rng = np.random.default_rng(42)
    N = o.N
    b = rng.normal(size=N); b[cfg.pin_node] = 0
    x = torch.zeros(N, dtype=torch.float64, device="cuda")
    it, res, rc = gs.cg_solve(cm.CM_MAT_K_MS, _dev(torch, b), x, fixed_iters=3)
    xo, ito, reso, _ = o.cg(oracle_mod.MAT_K_MS, b, fixed=3)
    assert it == ito == 3 and rel(x.cpu().numpy(), xo) < 1e-11 and res == pytest.approx(reso, rel=1e-9)

    b3 = rng.normal(size=(N, 3)); b3[cfg.clamp_dof.reshape(N, 3).astype(bool)] = 0
    x3 = torch.zeros((N, 3), dtype=torch.float64, device="cuda")
    it, res, rc = gs.cg_solve(cm.CM_MAT_K_MECH, _dev(torch, b3), x3, fixed_iters=3)
    xo, ito, reso, _ = o.cg(oracle_mod.MAT_K_MECH, b3.ravel(), fixed=3)
    assert it == ito == 3 and rel(x3.cpu().numpy().ravel(), xo) < 1e-11 and res == pytest.approx(reso, rel=1e-9)

    # 200 iterations on the device; true residual from the ORACLE's SpMV of the device iterate
    x3.zero_()
    it, res, rc = gs.cg_solve(cm.CM_MAT_K_MECH, _dev(torch, b3), x3, fixed_iters=200)
    r_true = b3.ravel() - o.spmv(oracle_mod.MAT_K_MECH, x3.cpu().numpy().ravel())
    assert np.linalg.norm(r_true) / np.linalg.norm(b3) == pytest.approx(res, rel=1e-6)

    f = rng.normal(size=(N, 3))
    bg = o.rhs_gs(f)
    xg = _dev(torch, f).clone()
    its, ress, rc = gs.cg_solve3(cm.CM_MAT_K_GS1, _dev(torch, bg), xg, fixed_iters=3)
    for a in range(3):
        xo, ito, reso, _ = o.cg(oracle_mod.MAT_K_GS1, bg[:, a].copy(), x0=f[:, a].copy(), fixed=3)
        assert its[a] == 3 and rel(xg[:, a].cpu().numpy(), xo) < 1e-11


def test_full_size_gspm_step_fixed_iterations(full, oracle_mod):
    """Two whole GSPM steps of config 3 (all physics, field sweep) with every CG solve cut at 4 iterations: identical
    arithmetic on both sides, so max |dm| must meet the 1e-9 bar of the converged runs."""
    cfg, cm, gm, gs, o, torch = full
    N = o.N
    m = cfg.m0.copy(); U = np.zeros(N); u = np.zeros((N, 3))
    mg = _dev(torch, m); Ug = torch.zeros(N, dtype=torch.float64, device="cuda")
    ug = torch.zeros((N, 3), dtype=torch.float64, device="cuda")
    for k in range(2):
        p = cm.make_params(cfg.dt, cfg.Hext[k], cfg.terms, 0, 1e-7, 100000, 4)
        io, rco = o.gspm_step(m, U, u, cfg.dt, cfg.Hext[k], cfg.terms, cg_tol=1e-7, cg_fixed_iters=4)
        ig, rcg = gs.gspm_step(p, mg, Ug, ug)
        assert rco == 0 and rcg == 0
        assert np.allclose(ig.mbar[:], io.mbar[:], atol=1e-12)
        assert ig.mean_dm == pytest.approx(io.mean_dm, rel=1e-9)
    mgh = mg.cpu().numpy()
    assert np.abs(mgh - m).max() <= 1e-9
    assert rel(Ug.cpu().numpy(), U) <= 1e-9 and rel(ug.cpu().numpy(), u) <= 1e-9
    live = o.live().astype(bool)
    assert np.abs(np.linalg.norm(mgh[live], axis=1) - 1).max() <= 4 * np.finfo(float).eps
    assert np.abs(mgh[~live]).max() == 0.0


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config1_full_size_10_steps(oracle_mod, dtype):
    """BASELINE config 1 at its own size (81x81x21 = 137,781 nodes, anisotropy + Zeeman at -50 mT, dt = 5 ps): ten steps,
    every solve iterated to convergence on both sides.  fp64: tol 1e-12, max |dm| <= 1e-9, counts +-1;  fp32 against the
    fp64 oracle: tol 1e-6, max |dm| <= 1e-4."""
    import torch
    from paper_2510_09812_b200 import binding as cm
    cfg = inputs.make_config(1)
    assert cfg.mesh.n_nodes == 137781
    f64 = dtype == "f64"
    tol = 1e-12 if f64 else 1e-6
    td = torch.float64 if f64 else torch.float32
    gm = cm.Mesh(cfg.mesh.xyz, cfg.mesh.tets, cfg.mesh.magnetic, cfg.mesh.elastic_id, cm.CM_REORDER_MORTON)
    gs = cm.System(gm, cfg.material, cfg.dt, dtype, cfg.clamp_dof, cfg.pin_node)
    o = oracle_mod.Oracle(cfg.mesh, cfg.material, cfg.dt, clamp_dof=cfg.clamp_dof, pin_node=cfg.pin_node)
    N = o.N
    m = cfg.m0.copy(); U = np.zeros(N); u = np.zeros((N, 3))
    mg = torch.as_tensor(cfg.m0, dtype=td, device="cuda").contiguous()
    Ug = torch.zeros(N, dtype=td, device="cuda"); ug = torch.zeros((N, 3), dtype=td, device="cuda")
    for k in range(10):
        p = cm.make_params(cfg.dt, cfg.Hext[k], cfg.terms, 0, tol)
        io, rco = o.gspm_step(m, U, u, cfg.dt, cfg.Hext[k], cfg.terms, cg_tol=tol)
        ig, rcg = gs.gspm_step(p, mg, Ug, ug)
        assert rco == 0 and rcg == 0
        for a in range(8):
            assert abs(io.it_gs[a] - ig.it_gs[a]) <= (1 if f64 else 3), (k, a, list(io.it_gs), list(ig.it_gs))
    err = np.abs(mg.cpu().numpy().astype(np.float64) - m).max()
    assert err <= (1e-9 if f64 else 1e-4), err


def test_full_size_fp32_build_against_fp64_oracle(full, oracle_mod):
    """The fp32 library build at config 3's size (what `bench.py --dtype f32` times) against the fp64 oracle already set up:
    SpMV, right-hand sides and fields <= 1e-5 over all 3 M outputs; three CG iterations <= 1e-4."""
    cfg, cm, gm, gs64, o, torch = full
    gs = cm.System(gm, cfg.material, cfg.dt, "f32", cfg.clamp_dof, cfg.pin_node)
    dev = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float32, device="cuda")
    rng = np.random.default_rng(43)
    N = o.N
    x = rng.normal(size=N).astype(np.float32)
    assert rel(gs.spmv(cm.CM_MAT_K_MS, dev(x)).cpu().numpy(), o.spmv(oracle_mod.MAT_K_MS, x.astype(np.float64))) < 1e-5
    x3 = rng.normal(size=(N, 3)).astype(np.float32)
    y3 = gs.spmv(cm.CM_MAT_K_MECH, dev(x3)).cpu().numpy()
    assert rel(y3.ravel(), o.spmv(oracle_mod.MAT_K_MECH, x3.astype(np.float64).ravel())) < 1e-5
    m = cfg.m0.astype(np.float32); m64 = m.astype(np.float64)
    md = dev(m)
    assert rel(gs.field_rhs(cm.CM_RHS_MS, md).cpu().numpy(), o.rhs_ms(m64)) < 1e-5
    assert rel(gs.field_rhs(cm.CM_RHS_MECH, md).cpu().numpy(), o.rhs_mech(m64)) < 1e-5
    U = rng.normal(size=N).astype(np.float32); u = (1e-3 * rng.normal(size=(N, 3))).astype(np.float32)
    p = cm.make_params(cfg.dt, cfg.Hext[3], cfg.terms)
    hd_o, _ = o.demag_field(U.astype(np.float64), o.volume_average(m64), cfg.terms)
    sig_o = o.stress_recover(u.astype(np.float64), m64)
    h_o = o.field(m64, hd_o, sig_o, np.asarray(cfg.Hext[3]) / cfg.material.Ms, cfg.terms)
    assert rel(gs.field_rhs(cm.CM_OUT_FIELD, md, dev(U), dev(u), p).cpu().numpy(), h_o) < 1e-5
    b3 = rng.normal(size=(N, 3)).astype(np.float32); b3[cfg.clamp_dof.reshape(N, 3).astype(bool)] = 0
    xg = torch.zeros((N, 3), dtype=torch.float32, device="cuda")
    it, res, rc = gs.cg_solve(cm.CM_MAT_K_MECH, dev(b3), xg, fixed_iters=3)
    xo, ito, reso, _ = o.cg(oracle_mod.MAT_K_MECH, b3.astype(np.float64).ravel(), fixed=3)
    assert it == 3 and rel(xg.cpu().numpy().ravel(), xo) < 1e-4 and res == pytest.approx(reso, rel=1e-3)


def test_config3_one_converged_step(full, oracle_mod):
    """ONE whole GSPM step of config 3 with every solve iterated to the paper's tolerance 1e-7 on both sides -- the
    ~1800-iteration persistent launches `bench.py` times (about 2.5 minutes of oracle time on the GPU box's host cores).
    Counts: magnetostatic and Helmholtz solves +-1, mechanical solve 1.5 % (tests/test_gpu_parity.py::_check_iters); the
    device's U and u satisfy the ORACLE's operator to the reported residual; m agrees to the accuracy two tol-1e-7 solves
    of the same systems can (each side's U, u carry an O(tol x condition) error of their own)."""
    cfg, cm, gm, gs, o, torch = full
    N = o.N
    m = cfg.m0.copy(); U = np.zeros(N); u = np.zeros((N, 3))
    mg = _dev(torch, m); Ug = torch.zeros(N, dtype=torch.float64, device="cuda")
    ug = torch.zeros((N, 3), dtype=torch.float64, device="cuda")
    ig, rcg = gs.gspm_step(cm.make_params(cfg.dt, cfg.Hext[0], cfg.terms, 0, 1e-7), mg, Ug, ug)
    io, rco = o.gspm_step(m, U, u, cfg.dt, cfg.Hext[0], cfg.terms, cg_tol=1e-7)
    assert rco == 0 and rcg == 0
    print(f"\nconfig 3, one converged step: CG its oracle ms/mech/gs {io.it_ms}/{io.it_mech}/{list(io.it_gs)}  "
          f"device {ig.it_ms}/{ig.it_mech}/{list(ig.it_gs)}")
    assert abs(io.it_ms - ig.it_ms) <= 1, (io.it_ms, ig.it_ms)
    assert abs(io.it_mech - ig.it_mech) <= int(np.ceil(0.015 * io.it_mech)), (io.it_mech, ig.it_mech)
    for a in range(8):
        assert abs(io.it_gs[a] - ig.it_gs[a]) <= 1, (a, list(io.it_gs), list(ig.it_gs))
    assert ig.it_ms > 1000 and ig.it_mech > 1000
    # true residuals of the device's solutions under the oracle's operators and right-hand sides
    b_ms = o.rhs_ms(cfg.m0)
    r = b_ms - o.spmv(oracle_mod.MAT_K_MS, Ug.cpu().numpy())
    assert np.linalg.norm(r) / np.linalg.norm(b_ms) < 1.05e-7
    b_me = o.rhs_mech(cfg.m0)
    r = b_me.ravel() - o.spmv(oracle_mod.MAT_K_MECH, ug.cpu().numpy().ravel())
    assert np.linalg.norm(r) / np.linalg.norm(b_me) < 1.05e-7
    assert ig.res_ms < 1e-7 and ig.res_mech < 1e-7
    dm = np.abs(mg.cpu().numpy() - m).max()
    print(f"config 3, one converged step at tol 1e-7: max |dm| = {dm:.2e}, max |dU| / max |U| = {rel(Ug.cpu().numpy(), U):.2e}, "
          f"max |du| / max |u| = {rel(ug.cpu().numpy(), u):.2e}")
    assert dm <= 1e-7                                  # measured 6.1e-9 (profiles/r02_fullsize_converged.txt); two tol-1e-7 solves
    assert np.allclose(ig.mbar[:], io.mbar[:], atol=1e-12) and ig.mean_dm == pytest.approx(io.mean_dm, rel=1e-7)
    # the fp32 build on the same step (BASELINE config 3 lists fp64 AND fp32), same tolerance as `bench.py --dtype f32` runs it with,
    # against the fp64 oracle's step: north_star's 1e-4 (measured 6.95e-5), counts within 0.5 % of the fp64 oracle's (measured 1625 / 1969
    # against 1623 / 1964, the eight Helmholtz counts identical)
    gs32 = cm.System(gm, cfg.material, cfg.dt, "f32", cfg.clamp_dof, cfg.pin_node)
    m32 = torch.as_tensor(cfg.m0, dtype=torch.float32, device="cuda").contiguous()
    U32 = torch.zeros(N, dtype=torch.float32, device="cuda"); u32 = torch.zeros((N, 3), dtype=torch.float32, device="cuda")
    i32, rc32 = gs32.gspm_step(cm.make_params(cfg.dt, cfg.Hext[0], cfg.terms, 0, 1e-7), m32, U32, u32)
    dm32 = np.abs(m32.cpu().numpy().astype(np.float64) - m).max()
    print(f"config 3, one converged step, fp32 device against the fp64 oracle: max |dm| = {dm32:.2e}, CG its ms/mech/gs "
          f"{i32.it_ms}/{i32.it_mech}/{list(i32.it_gs)} (rc {rc32}), <|dm|> {i32.mean_dm:.6f} against {io.mean_dm:.6f}")
    gs32.close()
    assert rc32 == 0
    assert abs(i32.it_ms - io.it_ms) <= 0.005 * io.it_ms and abs(i32.it_mech - io.it_mech) <= 0.005 * io.it_mech
    assert all(abs(i32.it_gs[a] - io.it_gs[a]) <= 1 for a in range(8))
    assert dm32 <= 1e-4


SLOW = pytest.mark.skipif(os.environ.get("CM_SLOW_TESTS", "0") != "1",
                          reason="about 7 minutes of oracle time: set CM_SLOW_TESTS=1 (log of the last run: profiles/r02_fullsize_converged.txt)")


def test_config2_full_size_3_steps_f64(oracle_mod):
    """BASELINE config 2 at its own 515,871 nodes in the DEFAULT suite: three converged steps, fp64, tol 1e-12, max |dm| <= 1e-9,
    counts +-1 (mechanical 1.5 %).  The ten-step fp64 / fp32 runs of the same configuration stay behind CM_SLOW_TESTS=1."""
    _config2_full_size(oracle_mod, "f64", 3)


@SLOW
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config2_full_size_10_steps(oracle_mod, dtype):
    """Ten steps of the same (see _config2_full_size)."""
    _config2_full_size(oracle_mod, dtype, 10)


def _config2_full_size(oracle_mod, dtype, nsteps):
    """BASELINE config 2 at its own size (129x129x31 = 515,871 nodes, all physics, spherical inclusion with x2 stiffness,
    clamped bottom face, dt = 10 ps): ten steps, every solve iterated to convergence on both sides.
    fp64: tol 1e-12, max |dm| <= 1e-9, counts +-1 (mechanical 1.5 %).
    fp32 against the fp64 oracle, tol 1e-6: <= 1e-4 after the FIRST step (the rounding level of an fp32 step).  Over ten steps
    the difference grows by a factor ~2 per step -- config 2 runs at dtau = 2.65, where m changes by O(1) per step (R5) and
    any perturbation, an fp32 rounding included, is amplified; north_star's 1e-4 after ten steps holds on the stable
    configurations (0 and 1, tests/test_gpu_parity.py, test_config1_full_size_10_steps) and is reported, not met, here."""
    import torch
    from paper_2510_09812_b200 import binding as cm
    cfg = inputs.make_config(2)
    assert cfg.mesh.n_nodes == 515871
    f64 = dtype == "f64"
    tol = 1e-12 if f64 else 1e-6
    td = torch.float64 if f64 else torch.float32
    gm = cm.Mesh(cfg.mesh.xyz, cfg.mesh.tets, cfg.mesh.magnetic, cfg.mesh.elastic_id, cm.CM_REORDER_MORTON)
    gs = cm.System(gm, cfg.material, cfg.dt, dtype, cfg.clamp_dof, cfg.pin_node)
    o = oracle_mod.Oracle(cfg.mesh, cfg.material, cfg.dt, clamp_dof=cfg.clamp_dof, pin_node=cfg.pin_node)
    N = o.N
    m = cfg.m0.copy(); U = np.zeros(N); u = np.zeros((N, 3))
    mg = torch.as_tensor(cfg.m0, dtype=td, device="cuda").contiguous()
    Ug = torch.zeros(N, dtype=td, device="cuda"); ug = torch.zeros((N, 3), dtype=td, device="cuda")
    errs = []
    for k in range(nsteps):
        io, rco = o.gspm_step(m, U, u, cfg.dt, cfg.Hext[k], cfg.terms, cg_tol=tol)
        ig, rcg = gs.gspm_step(cm.make_params(cfg.dt, cfg.Hext[k], cfg.terms, 0, tol), mg, Ug, ug)
        assert rco == 0 and rcg == 0
        errs.append(float(np.abs(mg.cpu().numpy().astype(np.float64) - m).max()))
        if f64:
            assert abs(io.it_ms - ig.it_ms) <= 1, (k, io.it_ms, ig.it_ms)
            assert abs(io.it_mech - ig.it_mech) <= int(np.ceil(0.015 * io.it_mech)), (k, io.it_mech, ig.it_mech)
            for a in range(8):
                assert abs(io.it_gs[a] - ig.it_gs[a]) <= 1, (k, a, list(io.it_gs), list(ig.it_gs))
    print(f"\nconfig 2 full size, {dtype}: max |dm| after steps 1..{nsteps} = {['%.1e' % e for e in errs]}; last-step CG its ms/mech "
          f"{ig.it_ms}/{ig.it_mech}, <|dm|> per step {io.mean_dm:.2f}")
    if f64:
        assert errs[-1] <= 1e-9, errs
    else:
        # ten steps: reported, not met (1e-4 is north_star's) -- first-step accuracy times the amplification of the dynamics,
        # pinned at reduced size in tests/test_gpu_parity.py::test_config2_fp32_error_is_first_step_accuracy_times_...
        assert errs[0] <= 1e-4 and errs[-1] <= 5e-2, errs
