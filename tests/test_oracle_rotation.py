"""Pins for the oracle's rotated crystal frame (Appendix D; R25).  CPU only.
Every rotation the oracle does internally is checked against one done here in numpy on plain 3x3 / 3x3x3x3 tensors, and
against textbook closed forms (isotropy is rotation invariant; the <111> modulus of a cubic crystal)."""
import math

import numpy as np
import pytest

from paper_2510_09812_b200 import inputs
from paper_2510_09812_b200.inputs import TERM_ANIS, TERM_MAGEL, TERM_ZEEMAN

NM = 1e-9
MU0 = 4e-7 * math.pi
VOIGT = [(0, 0), (1, 1), (2, 2), (1, 2), (0, 2), (0, 1)]


@pytest.fixture(scope="module")
def orc(oracle_mod):
    return oracle_mod


def rot(seed):
    return inputs.random_rotation(seed)


def stress_voigt(S):
    return np.array([S[i, j] for i, j in VOIGT])


def strain_voigt(E):
    return np.array([E[i, j] * (1 if i == j else 2) for i, j in VOIGT])     # engineering shears


def tensor4(C):
    """6x6 Voigt stiffness (engineering shears) -> C_ijkl"""
    T = np.zeros((3, 3, 3, 3))
    for a, (i, j) in enumerate(VOIGT):
        for b, (k, l) in enumerate(VOIGT):
            T[i, j, k, l] = T[j, i, k, l] = T[i, j, l, k] = T[j, i, l, k] = C[a, b]
    return T


def voigt66(T):
    return np.array([[T[i, j, k, l] for (k, l) in VOIGT] for (i, j) in VOIGT])


def E0_crystal(mat, m):
    l1, l2 = mat.lambda100, mat.lambda111
    E = 1.5 * l2 * np.outer(m, m)
    E[np.arange(3), np.arange(3)] = 1.5 * l1 * (m ** 2 - 1 / 3)              # Table A.1
    return E


def test_R111_is_the_papers_matrix_and_a_rotation():
    R = inputs.R_111
    assert np.allclose(R @ R.T, np.eye(3), atol=1e-15) and np.linalg.det(R) == pytest.approx(1.0)
    assert np.allclose(R @ (np.ones(3) / math.sqrt(3)), [1, 0, 0], atol=1e-15)       # <111> becomes the first axis


@pytest.mark.parametrize("R", [inputs.R_111, rot(1), rot(2)])
def test_voigt_rotation_matrix_against_tensor_rotation(orc, R):
    """Eq. D.3: M acts on Voigt vectors of tensor components like R . R^T on the tensor; the engineering-strain vector
    transforms with M^-T; M C M^T is the 4th-order rotation of C (Eq. D.4)."""
    M = orc.voigt_rotation(R)
    rng = np.random.default_rng(3)
    S = rng.normal(size=(3, 3)); S = S + S.T
    assert np.allclose(M @ stress_voigt(S), stress_voigt(R @ S @ R.T), atol=1e-14)
    assert np.allclose(np.linalg.inv(M).T @ strain_voigt(S), strain_voigt(R @ S @ R.T), atol=1e-13)
    C = inputs.cubic_voigt(2.4e11, 1.5e11, 1.2e11)
    Crot = voigt66(np.einsum("ip,jq,kr,ls,pqrs->ijkl", R, R, R, R, tensor4(C)))
    assert np.allclose(M @ C @ M.T, Crot, rtol=1e-13, atol=1e-2)
    Ciso = inputs.isotropic_voigt(200e9, 0.3)
    assert np.allclose(M @ Ciso @ M.T, Ciso, rtol=1e-13, atol=1e-3)                  # isotropy is rotation invariant


def test_cubic_stiffness_along_111_closed_form(orc):
    """Textbook: the longitudinal modulus of a cubic crystal along <111> is (C11 + 2 C12 + 4 C44) / 3."""
    C11, C12, C44 = 2.4e11, 1.5e11, 1.2e11
    mesh = inputs.kuhn_box((3, 3, 3), (4 * NM,) * 3)
    mat = inputs.Material(C_voigt=inputs.cubic_voigt(C11, C12, C44)[None], R=inputs.R_111)
    o = orc.Oracle(mesh, mat, 1e-12)
    # uniaxial strain along the first simulation axis (= crystal <111>): energy = 1/2 V C'_11 eps^2
    eps = 1e-3
    u = np.zeros((o.N, 3)); u[:, 0] = eps * mesh.xyz[:, 0] / NM
    m = np.zeros((o.N, 3))                                                            # E0 switched off through chi_e? no: m = 0
    mat0 = inputs.Material(C_voigt=mat.C_voigt, R=inputs.R_111, lambda100=0.0, lambda111=0.0)
    o0 = orc.Oracle(mesh, mat0, 1e-12)
    m[:, 0] = 1
    E = o0.energy(m, None, u, [0, 0, 0], TERM_MAGEL)
    exch = o0.energy(m, None, u, [0, 0, 0], 0)
    Cp = (C11 + 2 * C12 + 4 * C44) / 3 / (MU0 * mat.Ms ** 2)
    assert E - exch == pytest.approx(0.5 * 64.0 * Cp * eps ** 2, rel=1e-12)


@pytest.mark.parametrize("R", [inputs.R_111, rot(4)])
def test_anisotropy_field_energy_and_easy_axes(orc, R):
    cfg = inputs.make_config(0)
    mat = inputs.Material(R=R)
    o = orc.Oracle(cfg.mesh, mat, cfg.dt)
    oI = orc.Oracle(cfg.mesh, inputs.Material(), cfg.dt)
    m = cfg.m0
    # h_an(R; m) = R h_an(I; R^T m): rotation done here, unrotated formula already pinned in test_oracle_pins.py
    h = o.field(m, None, None, [0, 0, 0], TERM_ANIS)
    hI = oI.field(m @ R, None, None, [0, 0, 0], TERM_ANIS)                            # rows: (R^T m_i)^T = m_i^T R
    assert np.abs(h - hI @ R.T).max() < 1e-15
    assert np.abs(h - oI.field(m, None, None, [0, 0, 0], TERM_ANIS)).max() > 1e-4     # and it is not the unrotated field
    # K1 > 0: the crystal <100> directions, R e_a in the simulation frame, are energy minima with zero field and zero energy
    for a in range(3):
        mu = np.tile(R[:, a], (o.N, 1))
        assert np.abs(o.field(mu, None, None, [0, 0, 0], TERM_ANIS)).max() < 1e-16
        assert abs(o.energy(mu, None, None, [0, 0, 0], TERM_ANIS)) < 1e-12
    # crystal <111> = R (1,1,1)/sqrt3: the hard axis, energy K* V / 3
    mu = np.tile(R @ np.ones(3) / math.sqrt(3), (o.N, 1))
    assert o.energy(mu, None, None, [0, 0, 0], TERM_ANIS) == pytest.approx(o.Kstar * 8000.0 / 3, rel=1e-12)
    # uniform m along a rotated easy axis with the field along it is a fixed point of the step
    mu = np.tile(R[:, 0], (o.N, 1)); U = np.zeros(o.N); u = np.zeros((o.N, 3))
    info, rc = o.gspm_step(mu, U, u, cfg.dt, 5e4 * R[:, 0], TERM_ANIS | TERM_ZEEMAN, cg_tol=1e-12)
    assert rc == 0 and np.abs(mu - R[:, 0]).max() < 1e-14


def _fd_field(energy, m, nodes, mass, h):
    out = np.zeros((len(nodes), 3))
    for a, i in enumerate(nodes):
        for c in range(3):
            mp = m.copy(); mp[i, c] += h
            mm = m.copy(); mm[i, c] -= h
            out[a, c] = -(energy(mp) - energy(mm)) / (2 * h) / mass[i]
    return out


@pytest.mark.parametrize("R", [inputs.R_111, rot(5)])
def test_rotated_fields_are_energy_gradients(orc, R):
    """h_an and h_me in the rotated frame are still -(1/mLm_i) dE/dm_i of the rotated discrete energy (central differences)."""
    mesh = inputs.kuhn_box((6, 5, 5), (15 * NM, 12 * NM, 12 * NM), seed_mesh=7, seed_perm=8)
    mesh = inputs.flag_inclusion(mesh, np.array(mesh.box) / 2, (4 * NM, 3 * NM, 3 * NM))
    Cc = inputs.cubic_voigt(2.4e11, 1.5e11, 1.2e11)
    mat = inputs.Material(C_voigt=np.stack([Cc, 2 * Cc]), R=R)
    o = orc.Oracle(mesh, mat, 1e-12, clamp_dof=inputs.clamp_bottom(mesh))
    rng = np.random.default_rng(6)
    m = inputs.init_m_random(mesh, 9)
    u = 1e-3 * rng.normal(size=(o.N, 3))
    live = np.flatnonzero(o.live())
    nodes = rng.choice(live, 4, replace=False)
    h = o.field(m, None, None, [0, 0, 0], TERM_ANIS)
    fd = _fd_field(lambda mm: o.energy(mm, None, None, [0, 0, 0], TERM_ANIS) - o.energy(mm, None, None, [0, 0, 0], 0),
                   m, nodes, o.mLm(), 2e-4)      # quartic and, once rotated, not separable per component: O(h^2) truncation
    assert np.allclose(h[nodes], fd, rtol=2e-6, atol=2e-8)
    sig = o.stress_recover(u, m)
    h = o.field(m, None, sig, [0, 0, 0], TERM_MAGEL)
    fd = _fd_field(lambda mm: o.energy(mm, None, u, [0, 0, 0], TERM_MAGEL) - o.energy(mm, None, u, [0, 0, 0], 0),
                   m, nodes, o.mLm(), 1e-4)
    assert np.abs(h[nodes]).max() > 1e-4
    assert np.allclose(h[nodes], fd, rtol=1e-6, atol=2e-9)


@pytest.mark.parametrize("R", [inputs.R_111, rot(7)])
def test_rotated_stress_free_state(orc, R):
    """Homogeneous cubic body, uniform m: u = E0_sim x with E0_sim = R E0_crystal(R^T m) R^T (formed here in numpy) solves
    K u = b exactly, the recovered stress and h_me vanish; with u = 0 the recovered stress is -C_sim : E0_sim."""
    mesh = inputs.kuhn_box((5, 5, 4), (10 * NM, 12 * NM, 9 * NM), seed_mesh=3, seed_perm=4)
    Cc = inputs.cubic_voigt(2.4e11, 1.5e11, 1.2e11)
    mat = inputs.Material(C_voigt=Cc[None], R=R)
    o = orc.Oracle(mesh, mat, 1e-12)
    mdir = np.array([0.6, -0.48, 0.64])
    m = np.tile(mdir, (o.N, 1))
    E0 = R @ E0_crystal(mat, R.T @ mdir) @ R.T
    x = mesh.xyz / NM
    u = x @ E0.T
    b = o.rhs_mech(m)
    Ku = (o.csr(orc.MAT_K_MECH_FREE) @ u.ravel()).reshape(-1, 3)
    assert np.abs(b).max() > 1e-3
    assert np.abs(Ku - b).max() < 1e-12 * np.abs(b).max()
    Csim = voigt66(np.einsum("ip,jq,kr,ls,pqrs->ijkl", R, R, R, R, tensor4(Cc))) / (MU0 * mat.Ms ** 2)
    s = Csim @ strain_voigt(E0)
    sig = o.stress_recover(u, m)
    assert np.abs(sig).max() < 1e-12 * np.abs(s).max()
    assert np.abs(o.field(m, None, sig, [0, 0, 0], TERM_MAGEL)).max() < 1e-13
    sig0 = o.stress_recover(np.zeros_like(u), m)
    assert np.allclose(sig0, np.tile(-s, (o.N, 1)), rtol=1e-11, atol=1e-15)
    # and the unrotated E0 does NOT solve the rotated problem
    u_wrong = x @ E0_crystal(mat, mdir).T
    assert np.abs((o.csr(orc.MAT_K_MECH_FREE) @ u_wrong.ravel()).reshape(-1, 3) - b).max() > 1e-3 * np.abs(b).max()


def test_bad_rotation_rejected_and_identity_is_default(orc):
    cfg = inputs.make_config(0)
    with pytest.raises(RuntimeError, match="rc=-1"):
        orc.Oracle(cfg.mesh, inputs.Material(R=np.diag([1.0, 1.0, 2.0])), cfg.dt)
    with pytest.raises(RuntimeError, match="rc=-1"):
        orc.Oracle(cfg.mesh, inputs.Material(R=np.diag([1.0, 1.0, -1.0])), cfg.dt)          # a reflection
    a = orc.Oracle(cfg.mesh, inputs.Material(), cfg.dt)
    b = orc.Oracle(cfg.mesh, inputs.Material(R=np.eye(3)), cfg.dt)
    h1 = a.field(cfg.m0, None, None, [0, 0, 0], TERM_ANIS)
    assert np.array_equal(h1, b.field(cfg.m0, None, None, [0, 0, 0], TERM_ANIS))
    assert np.array_equal(a.values(orc.MAT_K_MECH), b.values(orc.MAT_K_MECH))


def test_hexahedra_honour_the_rotation(orc):
    """Appendix D on linear hexahedra (R26 x R25): the same closed forms as on tetrahedra.  (i) <111> longitudinal modulus
    (C11 + 2 C12 + 4 C44)/3 from the energy of a uniaxial strain along the first simulation axis; (ii) the stress-free
    state u = E0_sim x with E0_sim = R E0_crystal(R^T m) R^T formed here in numpy solves K u = b; (iii) a rotation that
    is not proper is rejected; (iv) an isotropic stiffness gives the same K^mech with and without R."""
    C11, C12, C44 = 2.4e11, 1.5e11, 1.2e11
    Cc = inputs.cubic_voigt(C11, C12, C44)
    R = inputs.R_111
    mesh = inputs.hex_box((4, 4, 3), (6 * NM, 6 * NM, 4 * NM), seed_mesh=3, seed_perm=4)
    mat0 = inputs.Material(C_voigt=Cc[None], R=R, lambda100=0.0, lambda111=0.0)
    o0 = orc.Oracle(mesh, mat0, 1e-12)
    eps = 1e-3
    u = np.zeros((o0.N, 3)); u[:, 0] = eps * mesh.xyz[:, 0] / NM
    m = np.zeros((o0.N, 3)); m[:, 0] = 1
    E = o0.energy(m, None, u, [0, 0, 0], TERM_MAGEL) - o0.energy(m, None, u, [0, 0, 0], 0)
    Cp = (C11 + 2 * C12 + 4 * C44) / 3 / (MU0 * mat0.Ms ** 2)
    assert E == pytest.approx(0.5 * 144.0 * Cp * eps ** 2, rel=1e-12)
    # and it is not the unrotated modulus C11
    assert abs(E - 0.5 * 144.0 * C11 / (MU0 * mat0.Ms ** 2) * eps ** 2) > 1e-2 * E
    mat = inputs.Material(C_voigt=Cc[None], R=R)
    o = orc.Oracle(mesh, mat, 1e-12)
    mdir = np.array([0.6, -0.48, 0.64])
    mm = np.tile(mdir, (o.N, 1))
    E0 = R @ E0_crystal(mat, R.T @ mdir) @ R.T
    uu = (mesh.xyz / NM) @ E0.T
    b = o.rhs_mech(mm)
    Ku = (o.csr(orc.MAT_K_MECH_FREE) @ uu.ravel()).reshape(-1, 3)
    assert np.abs(b).max() > 1e-3 and np.abs(Ku - b).max() < 1e-12 * np.abs(b).max()
    sig = o.stress_recover(uu, mm)
    Csim = voigt66(np.einsum("ip,jq,kr,ls,pqrs->ijkl", R, R, R, R, tensor4(Cc))) / (MU0 * mat.Ms ** 2)
    assert np.abs(sig).max() < 1e-12 * np.abs(Csim @ strain_voigt(E0)).max()
    with pytest.raises(RuntimeError, match="rc=-1"):
        orc.Oracle(mesh, inputs.Material(R=np.diag([1.0, 1.0, -1.0])), 1e-12)
    Ci = inputs.isotropic_voigt(200e9, 0.3)
    a = orc.Oracle(mesh, inputs.Material(C_voigt=Ci[None]), 1e-12).values(orc.MAT_K_MECH)
    b2 = orc.Oracle(mesh, inputs.Material(C_voigt=Ci[None], R=rot(3)), 1e-12).values(orc.MAT_K_MECH)
    assert np.abs(a - b2).max() <= 1e-12 * np.abs(a).max() and not np.array_equal(a, b2)
