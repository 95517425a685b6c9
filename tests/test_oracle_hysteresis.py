"""Pins for the oracle's hysteresis driver (R24).  CPU only.
The switching field the driver reports for a uniformly magnetised body is pinned to the static macrospin analysis of the
same energy (Eq. 1 with cubic anisotropy + Zeeman): the metastable branch of e(theta) is followed by Newton continuation
and loses stability where e'' = 0 -- a computation that shares nothing with the time stepper."""
import numpy as np
import pytest

from paper_2510_09812_b200 import inputs
from paper_2510_09812_b200.inputs import TERM_ANIS, TERM_DEMAG, TERM_FARFIELD, TERM_ZEEMAN

NM = 1e-9
MU0 = 4e-7 * np.pi


@pytest.fixture(scope="module")
def orc(oracle_mod):
    return oracle_mod


def macrospin_switching_field(Kstar, psi):
    """Cubic anisotropy, m = (cos t, sin t, 0), field h (signed) along (cos psi, sin psi, 0):
    e(t) = K* sin^2 t cos^2 t - h cos(t - psi).  Follow the minimum that starts at t = psi for h > 0 while h decreases;
    return the (negative) h at which e'' reaches 0.  In-plane is the softest direction (e_phiphi - e_tt = 12 K* s^2 c^2 >= 0)."""
    de = lambda t, h: 0.5 * Kstar * np.sin(4 * t) + h * np.sin(t - psi)
    d2e = lambda t, h: 2 * Kstar * np.cos(4 * t) + h * np.cos(t - psi)
    h, dh = 2 * Kstar, 2 * Kstar * 1e-5
    t = psi
    for _ in range(100):                                        # the minimum at the starting field (between 0 and psi)
        t -= de(t, h) / d2e(t, h)
    assert abs(de(t, h)) < 1e-14 * Kstar and d2e(t, h) > 0 and -1e-12 <= t <= psi
    while True:
        h_new = h - dh
        tn = t
        for _ in range(50):
            c = d2e(tn, h_new)
            if c <= 0:
                return h
            step = de(tn, h_new) / c
            tn -= step
            if abs(step) < 1e-15:
                break
        if d2e(tn, h_new) <= 1e-9 * Kstar or abs(tn - t) > 0.05:
            return h
        t, h = tn, h_new
        assert h > -4 * Kstar


def test_macrospin_reference_limits():
    # aligned field: the textbook nucleation field -2 K1 / (mu0 Ms), i.e. h = -2 K*
    assert macrospin_switching_field(0.01, 1e-7) == pytest.approx(-0.02, rel=2e-3)
    # misalignment lowers the barrier
    assert -0.02 < macrospin_switching_field(0.01, np.deg2rad(5)) < -0.01


@pytest.mark.parametrize("psi_deg", [2.0, 10.0])
def test_driver_switching_field_matches_macrospin(orc, psi_deg):
    mat = inputs.Material()                                      # Ms 1.2e6, K1 2e4, alpha 0.5
    Kstar = mat.K1 / (MU0 * mat.Ms ** 2)
    psi = np.deg2rad(psi_deg)
    h_sw = macrospin_switching_field(Kstar, psi)                  # negative, units of Ms
    mesh = inputs.kuhn_box((4, 4, 4), (10 * NM,) * 3, seed_mesh=5, seed_perm=6)
    dt = 5e-12
    o = orc.Oracle(mesh, mat, dt)
    e = np.array([np.cos(psi), np.sin(psi), 0.0])
    Hk = 2 * Kstar * mat.Ms
    H0, dH = 0.10 * Hk * e, -0.05 * Hk * e
    m = np.tile([1.0, 0.0, 0.0], (o.N, 1)); U = np.zeros(o.N); u = np.zeros((o.N, 3))
    Hl, ml, sl, res, rc = o.hysteresis_run(m, U, u, dt, H0, dH, TERM_ANIS | TERM_ZEEMAN, conv_tol=5e-10, max_fields=40,
                                           max_steps=200000, cg_tol=1e-12)
    assert rc == 0 and res.reversed == 1 and res.n_fields == len(Hl) < 40
    assert res.total_steps == sl.sum()
    assert np.allclose(Hl, H0 + np.arange(len(Hl))[:, None] * dH, rtol=0, atol=1e-9)
    proj = ml @ e
    assert np.all(proj[:-1] > 0) and proj[-1] < 0                # reversal is logged once, at the last field
    h_rev = (Hl[-1] @ e) / mat.Ms
    # the branch is stable down to h_sw, so the body cannot switch before; and it must have switched by the field after
    assert h_rev <= h_sw * (1 - 1e-6)
    assert h_rev > h_sw - 2 * 0.05 * 2 * Kstar
    # the body stays uniform; before switching it sits in the macrospin minimum of each field, in plane
    assert np.abs(m - m[0]).max() < 1e-12 and np.abs(ml[:-1, 2]).max() < 1e-7
    k = len(Hl) - 2
    h_k = (Hl[k] @ e) / mat.Ms
    t_k = np.arctan2(ml[k, 1], ml[k, 0])
    assert abs(0.5 * Kstar * np.sin(4 * t_k) + h_k * np.sin(t_k - psi)) < 1e-7 * Kstar      # e'(theta) = 0


def test_driver_is_the_plain_loop_over_gspm_step(orc):
    """The same loop written out here around o.gspm_step gives identical logs and state (control flow only)."""
    cfg = inputs.make_config(0)
    terms = TERM_ANIS | TERM_ZEEMAN | TERM_DEMAG | TERM_FARFIELD
    o = orc.Oracle(cfg.mesh, cfg.material, cfg.dt)
    H0, dH = np.array([4e4, 0, 0]), np.array([-3e4, 0, 0])
    args = dict(conv_tol=2e-4, max_fields=4, max_steps=25, cg_tol=1e-10)
    m = cfg.m0.copy(); U = np.zeros(o.N); u = np.zeros((o.N, 3))
    Hl, ml, sl, res, rc = o.hysteresis_run(m, U, u, cfg.dt, H0, dH, terms, **args)
    m2 = cfg.m0.copy(); U2 = np.zeros(o.N); u2 = np.zeros((o.N, 3))
    logs = []
    for k in range(4):
        H = H0 + k * dH
        steps = 0
        while True:
            info, rc2 = o.gspm_step(m2, U2, u2, cfg.dt, H, terms, cg_tol=1e-10)
            steps += 1
            if info.mean_dm < 2e-4 or steps >= 25:
                break
        mb = o.volume_average(m2)
        logs.append((H, mb, steps))
        if mb @ (H0 / np.linalg.norm(H0)) < 0:
            break
    assert res.n_fields == len(logs) and list(sl) == [l[2] for l in logs]
    assert np.array_equal(Hl, np.array([l[0] for l in logs]))
    # (two runs of the oracle differ at rounding level: its OpenMP dot products are not order-deterministic)
    assert np.abs(ml - np.array([l[1] for l in logs])).max() < 1e-10
    assert np.abs(m - m2).max() < 1e-9
    assert any(s == 25 for s in sl) or any(s < 25 for s in sl)


def test_driver_caps_and_bad_arguments(orc):
    cfg = inputs.make_config(0)
    o = orc.Oracle(cfg.mesh, cfg.material, cfg.dt)
    m = inputs.init_m_noisy_x(cfg.mesh, 9); U = np.zeros(o.N); u = np.zeros((o.N, 3))      # mbar . e0 > 0: no reversal
    Hl, ml, sl, res, rc = o.hysteresis_run(m, U, u, cfg.dt, [1e4, 0, 0], [-1e3, 0, 0], TERM_ANIS | TERM_ZEEMAN,
                                           conv_tol=1e-30, max_fields=3, max_steps=2, cg_tol=1e-10)
    assert res.n_fields == 3 and list(sl) == [2, 2, 2] and res.total_steps == 6 and res.reversed == 0
    assert np.abs(np.linalg.norm(m, axis=1) - 1).max() <= 4 * np.finfo(float).eps
    *_, rc = o.hysteresis_run(m, U, u, cfg.dt, [0, 0, 0], [-1e3, 0, 0], TERM_ANIS, max_fields=3, max_steps=2)
    assert rc == -1                                              # H0 = 0 has no direction to measure reversal along
