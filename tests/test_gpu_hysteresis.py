"""GPU parity of the device-resident hysteresis driver (cm_hysteresis_run: one CUDA graph with a conditional WHILE node,
P:96 / P:284 / P:304) against the oracle's plain loop.  What is unique is compared exactly or to tolerance: the number of
fields, the field log, the reversal flag, the logged averages and the final state.  The step count at a field is an
integer decided by `mean_dm < conv_tol` in fp64 on both sides; it can differ by one step only when mean_dm lands within
rounding of the threshold, so it is compared exactly where the margin is large (stated per test)."""
import numpy as np
import pytest

from paper_2510_09812_b200 import inputs
from paper_2510_09812_b200.inputs import TERM_ANIS, TERM_DEMAG, TERM_FARFIELD, TERM_MAGEL, TERM_ZEEMAN

pytestmark = pytest.mark.gpu
NM = 1e-9
MU0 = 4e-7 * np.pi


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


def _pair(cm, orc, torch, mesh, mat, dt, clamp=None, dtype="f64"):
    gm = cm.Mesh(mesh.xyz, mesh.tets, mesh.magnetic, mesh.elastic_id, cm.CM_REORDER_MORTON)
    gs = cm.System(gm, mat, dt, dtype, clamp)
    o = orc.Oracle(mesh, mat, dt, clamp_dof=clamp)
    return gm, gs, o


def _run_both(cm, torch, gs, o, m0, dt, H0, dH, terms, dtype="f64", **kw):
    td = torch.float64 if dtype == "f64" else torch.float32
    N = o.N
    m = m0.copy(); U = np.zeros(N); u = np.zeros((N, 3))
    ref = o.hysteresis_run(m, U, u, dt, H0, dH, terms, **kw)
    mg = torch.as_tensor(m0, dtype=td, device="cuda").contiguous()
    Ug = torch.zeros(N, dtype=td, device="cuda"); ug = torch.zeros((N, 3), dtype=td, device="cuda")
    p = cm.make_params(dt, (0, 0, 0), terms, 0, kw.get("cg_tol", 1e-7))
    dev = gs.hysteresis_run(p, mg, Ug, ug, H0, dH, conv_tol=kw.get("conv_tol", 5e-10), max_fields=kw.get("max_fields", 100),
                            max_steps=kw.get("max_steps", 100000))
    return ref, dev, (m, U, u), (mg.cpu().numpy().astype(np.float64), Ug.cpu().numpy(), ug.cpu().numpy())


def test_macrospin_loop_matches_oracle_and_switching_field(cm, oracle_mod, torch):
    """The macrospin hysteresis of tests/test_oracle_hysteresis.py (anisotropy + Zeeman, field 2 degrees off the easy axis):
    ~3 x 10^4 steps inside ONE graph launch.  Same number of fields and the same reversal field as the oracle; the averages
    logged at every converged field agree to 1e-8 (each is the end of a ~10^3-step relaxation to 5e-10)."""
    mat = inputs.Material()
    Kstar = mat.K1 / (MU0 * mat.Ms ** 2)
    psi = np.deg2rad(2.0)
    e = np.array([np.cos(psi), np.sin(psi), 0.0])
    Hk = 2 * Kstar * mat.Ms
    mesh = inputs.kuhn_box((4, 4, 4), (10 * NM,) * 3, seed_mesh=5, seed_perm=6)
    dt = 5e-12
    gm, gs, o = _pair(cm, oracle_mod, torch, mesh, mat, dt)
    m0 = np.tile([1.0, 0.0, 0.0], (o.N, 1))
    ref, dev, so, sg = _run_both(cm, torch, gs, o, m0, dt, 0.10 * Hk * e, -0.05 * Hk * e, TERM_ANIS | TERM_ZEEMAN,
                                 conv_tol=5e-10, max_fields=40, max_steps=200000, cg_tol=1e-12)
    Hl, ml, sl, res, rc = ref
    Hg, mlg, slg, resg, rcg = dev
    assert rc == 0 and rcg == 0
    assert resg.n_fields == res.n_fields and resg.reversed == res.reversed == 1
    assert np.array_equal(Hg, Hl)
    assert np.abs(mlg - ml).max() < 1e-8
    assert resg.total_steps == slg.sum()
    assert np.abs(slg.astype(int) - sl).max() <= np.maximum(2, sl // 200).max()      # ~1e3-step relaxations to a 5e-10 threshold
    assert np.abs(sg[0] - so[0]).max() < 1e-6                                        # state right after the switch
    assert -2 * Kstar < (Hg[-1] @ e) / mat.Ms < -1.5 * Kstar                         # macrospin switching field at 2 degrees: -1.56 K*


def test_micromagnetic_loop_parity(cm, oracle_mod, torch):
    """Config-0 body (exchange + anisotropy + demag + far field + Zeeman), three fields with a loose convergence threshold:
    short enough for the oracle, long enough to exercise convergence at a field, the decrement and the caps.  The
    threshold (2e-4) is crossed with a wide margin, so step counts must agree exactly; state within 1e-9."""
    cfg = inputs.make_config(0)
    terms = TERM_ANIS | TERM_ZEEMAN | TERM_DEMAG | TERM_FARFIELD
    gm, gs, o = _pair(cm, oracle_mod, torch, cfg.mesh, cfg.material, cfg.dt)
    m0 = inputs.init_m_noisy_x(cfg.mesh, 9)
    ref, dev, so, sg = _run_both(cm, torch, gs, o, m0, cfg.dt, [4e4, 0, 0], [-3e4, 0, 0], terms, conv_tol=2e-4, max_fields=3,
                                 max_steps=25, cg_tol=1e-12)
    Hl, ml, sl, res, rc = ref
    Hg, mlg, slg, resg, rcg = dev
    assert rc == 0 and rcg == 0
    assert resg.n_fields == res.n_fields == 3 and resg.reversed == res.reversed
    assert np.array_equal(Hg, Hl) and list(slg) == list(sl)
    assert resg.total_steps == res.total_steps
    assert np.abs(mlg - ml).max() < 1e-10
    assert np.abs(sg[0] - so[0]).max() <= 1e-9
    assert np.abs(sg[1] - so[1]).max() <= 1e-9 * max(1.0, np.abs(so[1]).max())
    assert resg.cg_iters_ms > 0 and resg.cg_passes_gs > 0 and resg.device_ms > 0


def test_magnetoelastic_loop_and_caps(cm, oracle_mod, torch):
    """All terms with an inclusion and a clamped face; convergence never reached (conv_tol = 0), so every field runs
    exactly max_steps steps: the caps and the field schedule, and parity of the state after 2 x 3 steps."""
    mesh = inputs.kuhn_box((11, 10, 6), (33 * NM, 30 * NM, 16 * NM), seed_mesh=71, seed_perm=72)
    mesh = inputs.flag_inclusion(mesh, np.array(mesh.box) / 2, (7 * NM, 6 * NM, 5 * NM))
    C = inputs.isotropic_voigt(200e9, 0.3)
    mat = inputs.Material(C_voigt=np.stack([C, 2 * C]))
    clamp = inputs.clamp_bottom(mesh)
    terms = TERM_ANIS | TERM_ZEEMAN | TERM_DEMAG | TERM_FARFIELD | TERM_MAGEL
    gm, gs, o = _pair(cm, oracle_mod, torch, mesh, mat, 1e-12, clamp)
    m0 = inputs.init_m_noisy_x(mesh, 73)
    ref, dev, so, sg = _run_both(cm, torch, gs, o, m0, 1e-12, [2e4, 1e4, 0], [-1e4, -5e3, 0], terms, conv_tol=0.0, max_fields=2,
                                 max_steps=3, cg_tol=1e-12)
    Hl, ml, sl, res, rc = ref
    Hg, mlg, slg, resg, rcg = dev
    assert rc == 0 and rcg == 0
    assert resg.n_fields == 2 and list(slg) == [3, 3] == list(sl) and resg.total_steps == 6 and resg.reversed == 0
    assert np.array_equal(Hg, Hl) and np.array_equal(Hg[1], [1e4, 5e3, 0])
    assert np.abs(mlg - ml).max() < 1e-11
    assert np.abs(sg[0] - so[0]).max() <= 1e-9
    assert np.abs(sg[2] - so[2]).max() <= 1e-9 * max(1.0, np.abs(so[2]).max())
    assert resg.cg_iters_mech > 30


def test_hysteresis_bad_arguments_and_reuse(cm, oracle_mod, torch):
    cfg = inputs.make_config(0)
    gm = cm.Mesh(cfg.mesh.xyz, cfg.mesh.tets)
    gs = cm.System(gm, cfg.material, cfg.dt)
    N = gm.n_nodes
    m = torch.as_tensor(inputs.init_m_noisy_x(cfg.mesh, 9), dtype=torch.float64, device="cuda").contiguous()
    p = cm.make_params(cfg.dt, (0, 0, 0), TERM_ANIS | TERM_ZEEMAN)
    with pytest.raises(cm.CmError) as e:
        gs.hysteresis_run(p, m, None, None, [0, 0, 0], [-1, 0, 0], max_fields=2, max_steps=2)
    assert e.value.code == cm.CM_E_BADARG
    with pytest.raises(cm.CmError):
        gs.hysteresis_run(p, m, None, None, [1e4, 0, 0], [-1, 0, 0], max_fields=0, max_steps=2)
    with pytest.raises(cm.CmError):                               # DEMAG without U
        gs.hysteresis_run(cm.make_params(cfg.dt, (0, 0, 0), TERM_DEMAG), m, None, None, [1e4, 0, 0], [-1, 0, 0], max_fields=2, max_steps=2)
    # the system is reusable: a plain step after a hysteresis run, and a second run with a larger log
    Hl, ml, sl, res, rc = gs.hysteresis_run(p, m, None, None, [1e4, 0, 0], [-1e3, 0, 0], conv_tol=1e-30, max_fields=2, max_steps=2)
    assert res.n_fields == 2 and res.total_steps == 4
    info, rc = gs.gspm_step(cm.make_params(cfg.dt, (1e4, 0, 0), TERM_ANIS | TERM_ZEEMAN), m, None, None)
    assert rc == 0 and np.isfinite(info.mean_dm)
    Hl, ml, sl, res, rc = gs.hysteresis_run(p, m, None, None, [1e4, 0, 0], [-1e3, 0, 0], conv_tol=1e-30, max_fields=5, max_steps=1)
    assert res.n_fields == 5 and list(sl) == [1] * 5
    assert float((m.norm(dim=1) - 1).abs().max()) <= 4 * np.finfo(float).eps
