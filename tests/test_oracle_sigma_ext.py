"""Pins for the uniform external stress sigma_ext of Eq. 1 (term -sigma_ext : E, second half;
DESIGN.md R17).  CPU only.  Under R17's reading (E = sym grad u, no homogeneous-strain unknown) sigma_ext is one more term of
the mechanical right-hand side, b_(i,a) += sum_e V_e sigma_ext,ab d_b phi_i over ALL elements.  Checked against: the closed-form
homogeneous state u = (C^-1 sigma_ext + E0) x (Hooke's law written out here in numpy), the energy with the -sigma_ext : E term
(first variation by central differences), the traction interpretation (sum of nodal forces on a face = sigma_ext n Area),
linearity, and the response of the magnetoelastic field (stress-induced anisotropy, the mechanism of the paper's Fig. 6)."""
import math

import numpy as np
import pytest

from paper_2510_09812_b200 import inputs
from paper_2510_09812_b200.inputs import TERM_MAGEL

NM = 1e-9
MU0 = 4e-7 * math.pi
SIG = np.array([3.0e8, -1.0e8, 0.5e8, 0.8e8, -0.6e8, 1.2e8])           # Pa, xx yy zz yz xz xy


def E0_tensor(mat, m):
    l1, l2 = mat.lambda100, mat.lambda111
    E = 1.5 * l2 * np.outer(m, m)
    E[np.arange(3), np.arange(3)] = 1.5 * l1 * (m ** 2 - 1 / 3)          # Table A.1
    return E


def tensor(v):
    return np.array([[v[0], v[5], v[4]], [v[5], v[1], v[3]], [v[4], v[3], v[2]]])


@pytest.fixture(scope="module")
def orc(oracle_mod):
    return oracle_mod


@pytest.mark.parametrize("kind", ["tet", "hex"])
def test_homogeneous_state_under_external_stress(orc, kind):
    """Homogeneous body, uniform m, no constraints: u = (S : sigma_ext + E0(m)) x solves K u = b exactly (linear u is in the
    P1 / Q1 space), the recovered stress C : (E - E0) equals sigma_ext at every node."""
    C = inputs.cubic_voigt(2.4e11, 1.5e11, 1.2e11)
    if kind == "tet":
        mesh = inputs.kuhn_box((5, 5, 4), (10 * NM, 12 * NM, 9 * NM), seed_mesh=3, seed_perm=4)
    else:
        mesh = inputs.hex_box((5, 5, 4), (10 * NM, 12 * NM, 9 * NM), seed_mesh=3, seed_perm=4)
    mat = inputs.Material(C_voigt=C[None], sigma_ext=SIG)
    o = orc.Oracle(mesh, mat, 1e-12)
    mdir = np.array([0.6, -0.48, 0.64])
    m = np.tile(mdir, (o.N, 1))
    eps_eng = np.linalg.solve(C, SIG)                                   # Hooke: engineering-shear Voigt strain
    Eel = tensor(eps_eng * np.array([1, 1, 1, 0.5, 0.5, 0.5]))
    Etot = Eel + E0_tensor(mat, mdir)
    u = (mesh.xyz / NM) @ Etot.T
    b = o.rhs_mech(m)
    Ku = (o.csr(orc.MAT_K_MECH_FREE) @ u.ravel()).reshape(-1, 3)
    assert np.abs(b).max() > 1e-3 and np.abs(Ku - b).max() < 1e-12 * np.abs(b).max()
    sig = o.stress_recover(u, m)
    s_nd = SIG / (MU0 * mat.Ms ** 2)
    assert np.abs(sig - s_nd).max() < 1e-11 * np.abs(s_nd).max()
    # without sigma_ext the same u is NOT an equilibrium
    o0 = orc.Oracle(mesh, inputs.Material(C_voigt=C[None]), 1e-12)
    assert np.abs(Ku - o0.rhs_mech(m)).max() > 1e-2 * np.abs(b).max()


@pytest.mark.parametrize("kind", ["tet", "hex"])
def test_equilibrium_is_the_minimum_of_the_energy_with_the_stress_term(orc, kind):
    """Clamped bottom, x2-stiff non-magnetic inclusion: the CG solution of K u = b(m, sigma_ext) makes the energy
    1/2 (E - E0):C:(E - E0) - sigma_ext : E stationary (central differences) and minimal."""
    C = inputs.isotropic_voigt(200e9, 0.3)
    box = (18 * NM, 15 * NM, 10 * NM)
    mesh = (inputs.kuhn_box if kind == "tet" else inputs.hex_box)((7, 6, 5), box, seed_mesh=3, seed_perm=4)
    mesh = inputs.flag_inclusion(mesh, np.array(box) / 2, (5 * NM, 4 * NM, 3 * NM))
    clamp = inputs.clamp_bottom(mesh)
    mat = inputs.Material(C_voigt=np.stack([C, 2 * C]), sigma_ext=SIG)
    o = orc.Oracle(mesh, mat, 1e-12, clamp_dof=clamp)
    rng = np.random.default_rng(5)
    live = o.live().astype(bool)
    m = rng.normal(size=(o.N, 3)); m /= np.linalg.norm(m, axis=1, keepdims=True); m[~live] = 0
    b = o.rhs_mech(m)
    u, it, res, rc = o.cg(orc.MAT_K_MECH, b.ravel(), tol=1e-13)
    assert rc == 0
    u = u.reshape(-1, 3)
    cl = clamp.astype(bool).reshape(-1, 3)
    E0 = o.energy(m, None, u, [0, 0, 0], TERM_MAGEL)
    for _ in range(3):
        du = 1e-4 * rng.normal(size=u.shape); du[cl] = 0
        Ep, Em = o.energy(m, None, u + du, [0, 0, 0], TERM_MAGEL), o.energy(m, None, u - du, [0, 0, 0], TERM_MAGEL)
        assert Ep > E0 and Em > E0
        assert abs(Ep - Em) < 1e-6 * (Ep + Em - 2 * E0)
    # sigma_ext moved the equilibrium: the solution without it is not stationary for this energy
    o0 = orc.Oracle(mesh, inputs.Material(C_voigt=np.stack([C, 2 * C])), 1e-12, clamp_dof=clamp)
    u0, _, _, _ = o0.cg(orc.MAT_K_MECH, o0.rhs_mech(m).ravel(), tol=1e-13)
    u0 = u0.reshape(-1, 3)
    du = 1e-4 * rng.normal(size=u.shape); du[cl] = 0
    Ep, Em = o.energy(m, None, u0 + du, [0, 0, 0], TERM_MAGEL), o.energy(m, None, u0 - du, [0, 0, 0], TERM_MAGEL)
    assert abs(Ep - Em) > 1e-3 * abs(Ep + Em - 2 * o.energy(m, None, u0, [0, 0, 0], TERM_MAGEL))


def test_rhs_is_the_boundary_traction_and_is_linear(orc):
    """b(sigma_ext) - b(0) = int grad phi_i . sigma_ext = surface traction sigma_ext n: zero at interior nodes of a box, and
    the nodal forces of the face x = L sum to sigma_ext e_x times the face area; b is affine in sigma_ext."""
    mesh = inputs.kuhn_box((6, 5, 5), (15 * NM, 12 * NM, 8 * NM), seed_mesh=7, seed_perm=8)
    C = inputs.isotropic_voigt(200e9, 0.3)
    m = inputs.init_m_random(mesh, 9)
    o0 = orc.Oracle(mesh, inputs.Material(C_voigt=C[None]), 1e-12)
    o1 = orc.Oracle(mesh, inputs.Material(C_voigt=C[None], sigma_ext=SIG), 1e-12)
    o2 = orc.Oracle(mesh, inputs.Material(C_voigt=C[None], sigma_ext=2 * SIG), 1e-12)
    db = o1.rhs_mech(m) - o0.rhs_mech(m)
    x = mesh.xyz / NM
    L = np.array(mesh.box) / NM
    interior = ((x > 1e-9) & (x < L - 1e-9)).all(axis=1)
    scale = np.abs(db).max()
    assert np.abs(db[interior]).max() < 1e-12 * scale
    s = tensor(SIG / (MU0 * 1.2e6 ** 2))
    face = (x[:, 0] > L[0] - 1e-9)
    # nodes of the face x = L, minus what the adjacent faces contribute at shared edges: sum over ALL nodes of the
    # x-max half is cleaner -- total force on the body is zero, and the first moment gives the stress: sum_i x_i (x) b_i = V sigma
    assert np.abs(db.sum(axis=0)).max() < 1e-12 * scale * len(db)
    assert np.allclose(x.T @ db, np.prod(L) * s, rtol=1e-12, atol=1e-12 * np.abs(s).max() * np.prod(L))
    assert face.any()
    assert np.allclose(o2.rhs_mech(m) - o0.rhs_mech(m), 2 * db, rtol=1e-12, atol=1e-13 * scale)


def test_external_stress_changes_the_magnetoelastic_field_through_the_strain(orc):
    """Stress-induced anisotropy (the paper's Fig. 6 mechanism): on the homogeneous body the equilibrium stress is
    sigma_ext, so h_me = 3 [lam100 m_a s_aa + lam111 sum_{b != a} m_b s_ab] with s = sigma_ext / (mu0 Ms^2) (R14)."""
    C = inputs.cubic_voigt(2.4e11, 1.5e11, 1.2e11)
    mesh = inputs.kuhn_box((4, 4, 4), (9 * NM,) * 3, seed_mesh=3, seed_perm=4)
    mat = inputs.Material(C_voigt=C[None], sigma_ext=SIG)
    o = orc.Oracle(mesh, mat, 1e-12)
    mdir = np.array([0.36, 0.48, 0.8])
    m = np.tile(mdir, (o.N, 1))
    Etot = tensor(np.linalg.solve(C, SIG) * np.array([1, 1, 1, 0.5, 0.5, 0.5])) + E0_tensor(mat, mdir)
    u = (mesh.xyz / NM) @ Etot.T
    h = o.field(m, None, o.stress_recover(u, m), [0, 0, 0], TERM_MAGEL)
    s = tensor(SIG / (MU0 * mat.Ms ** 2))
    l1, l2 = mat.lambda100, mat.lambda111
    expect = np.array([3 * (l1 * mdir[a] * s[a, a] + l2 * sum(mdir[b] * s[a, b] for b in range(3) if b != a)) for a in range(3)])
    assert np.abs(expect).max() > 1e-5
    assert np.abs(h - expect).max() < 1e-11 * np.abs(expect).max()
