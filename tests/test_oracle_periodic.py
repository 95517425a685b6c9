"""Pins for the oracle's periodic boundary conditions (node wrapping; R23).
CPU only.  Every check is against something other than the oracle: a brute-force wrap written from the definition,
counting arguments, the closed-form Fourier symbol of the P1 stiffness on a uniform Kuhn grid (= the 7-point
difference operator), Eq. 20's null-space dimension, and the equality of the paper's literal right-hand
side (Eq. 14) with the adjoint form the build uses (R9) once the domain is periodic."""
import numpy as np
import pytest

from paper_2510_09812_b200 import inputs
from paper_2510_09812_b200.inputs import TERM_ANIS, TERM_DEMAG, TERM_FARFIELD, TERM_ZEEMAN

NM = 1e-9


@pytest.fixture(scope="module")
def orc(oracle_mod):
    return oracle_mod


def brute_wrap(xyz, axes, rel_tol=1e-9):
    """The definition, O(n^2): representatives = nodes on no periodic max face, numbered in ascending node index;
    a wrapped node takes the number of the representative at its image x - span_d e_d."""
    lo, hi = xyz.min(0), xyz.max(0)
    span = hi - lo
    tol = rel_tol * span
    per = np.array([(axes >> d) & 1 for d in range(3)], bool)
    onmax = (xyz >= hi - tol) & per
    wrapped = onmax.any(1)
    dof = -np.ones(len(xyz), np.int64)
    reps = np.flatnonzero(~wrapped)
    dof[reps] = np.arange(len(reps))
    for i in np.flatnonzero(wrapped):
        w = xyz[i] - span * onmax[i]
        hit = reps[(np.abs(xyz[reps] - w) <= tol).all(1)]
        assert len(hit) == 1
        dof[i] = dof[hit[0]]
    return dof.astype(np.int32), len(reps)


@pytest.mark.parametrize("axes", range(8))
def test_wrap_matches_bruteforce(orc, axes):
    mesh = inputs.kuhn_box((5, 4, 6), (20 * NM, 12 * NM, 25 * NM), seed_mesh=3, seed_perm=4)
    dof, nd = orc.periodic_wrap(mesh.xyz, axes)
    dof_b, nd_b = brute_wrap(mesh.xyz, axes)
    assert nd == nd_b == np.prod([n - ((axes >> d) & 1) for d, n in enumerate((5, 4, 6))])
    assert np.array_equal(dof, dof_b)
    assert np.array_equal(np.unique(dof), np.arange(nd))


def test_wrap_rejects_mismatched_faces(orc):
    mesh = inputs.kuhn_box((5, 4, 6), (20 * NM, 12 * NM, 25 * NM), seed_mesh=3, seed_perm=4)
    xyz = mesh.xyz.copy()
    i = np.flatnonzero((xyz[:, 0] == xyz[:, 0].max()) & (xyz[:, 1] > 0) & (xyz[:, 1] < xyz[:, 1].max()))[0]
    xyz[i, 1] += 0.3 * NM                                        # this max-face node has no partner any more
    with pytest.raises(RuntimeError, match="rc=-1"):
        orc.periodic_wrap(xyz, 1)


def test_single_cell_periodic_direction_rejected(orc):
    mesh = inputs.kuhn_box((2, 4, 4), (5 * NM, 12 * NM, 12 * NM), seed_mesh=3, seed_perm=4)
    dof, nd = orc.periodic_wrap(mesh.xyz, 1)
    with pytest.raises(RuntimeError, match="rc=-1"):             # both x-faces are the same DOFs: tets collapse
        orc.Oracle(mesh, inputs.Material(), 1e-12, dof_of_node=dof, n_dof=nd)


def test_identity_map_is_the_unwrapped_oracle(orc):
    cfg = inputs.make_config(0)
    dof, nd = orc.periodic_wrap(cfg.mesh.xyz, 0)
    assert nd == cfg.mesh.n_nodes and np.array_equal(dof, np.arange(nd))
    a = orc.Oracle(cfg.mesh, cfg.material, cfg.dt)
    b = orc.Oracle(cfg.mesh, cfg.material, cfg.dt, dof_of_node=dof, n_dof=nd)
    for mat in (orc.MAT_K_MS, orc.MAT_K_GS1, orc.MAT_MASS):
        assert np.array_equal(a.values(mat), b.values(mat))


def _periodic(orc, grid, box, axes, jitter=0.15, mat=None, clamp_node=None, **kw):
    mesh = inputs.kuhn_box(grid, box, jitter=jitter, seed_mesh=5, seed_perm=6)
    dof, nd = orc.periodic_wrap(mesh.xyz, axes)
    clamp = None
    if clamp_node is not None:
        clamp = np.zeros((nd, 3), np.uint8); clamp[clamp_node] = 1; clamp = clamp.ravel()
    o = orc.Oracle(mesh, mat or inputs.Material(), 1e-12, clamp_dof=clamp, dof_of_node=dof, n_dof=nd, **kw)
    return mesh, dof, nd, o


def test_counts_symmetry_rowsums_volume(orc):
    grid, box = (6, 5, 7), (25 * NM, 16 * NM, 30 * NM)
    mesh, dof, nd, o = _periodic(orc, grid, box, 7)
    assert nd == 5 * 4 * 6
    rp = o.rowptr()
    assert np.all(np.diff(rp) == 15) and o.nnz == 15 * nd        # every node of a periodic Kuhn grid is an interior node
    K = o.csr(orc.MAT_K_FREE).toarray()
    assert np.abs(K - K.T).max() <= 1e-14 * np.abs(K).max()
    assert np.abs(K.sum(1)).max() <= 1e-13 * np.abs(K).sum(1).max()
    vol = np.prod(np.array(box) / 1e-9)
    assert o.Vtot == pytest.approx(vol, rel=1e-13)
    assert o.mL().sum() == pytest.approx(vol, rel=1e-13)
    M = o.csr(orc.MAT_MASS).toarray()
    assert np.allclose(M.sum(1), o.mLm(), rtol=1e-13)


def test_uniform_grid_stiffness_is_the_periodic_7_point_operator(orc):
    """On the un-jittered Kuhn grid the P1 stiffness is the 7-point difference operator; with the wrap it is circulant, so
    cos(2 pi x / L) is an eigenvector with the closed-form symbol -- at every DOF, including those across the seam."""
    grid, box = (7, 6, 5), (24 * NM, 15 * NM, 10 * NM)
    mesh, dof, nd, o = _periodic(orc, grid, box, 7, jitter=0.0)
    h = np.array(box) / 1e-9 / (np.array(grid) - 1)
    L = np.array(box) / 1e-9
    x = np.zeros((nd, 3)); x[dof] = np.where(mesh.xyz / 1e-9 >= L - 1e-9, 0.0, mesh.xyz / 1e-9)   # DOF coordinates
    mL = o.mL()
    assert np.allclose(mL, h.prod(), rtol=1e-13)                 # translation invariance of the lumped mass
    for d in range(3):
        u = np.cos(2 * np.pi * x[:, d] / L[d])
        lam = h.prod() / h[d] ** 2 * (2 - 2 * np.cos(2 * np.pi * h[d] / L[d]))
        assert np.abs(o.spmv(orc.MAT_K_FREE, u) - lam * u).max() <= 1e-12 * lam
    # partial periodicity (x only): the same function is still an eigenvector along x, natural faces in y, z
    mesh, dof, nd, o = _periodic(orc, grid, box, 1, jitter=0.0)
    x = np.zeros((nd, 3)); x[dof] = mesh.xyz / 1e-9
    x[:, 0] = np.where(x[:, 0] >= L[0] - 1e-9, 0.0, x[:, 0])
    u = np.cos(2 * np.pi * x[:, 0] / L[0])
    r = o.spmv(orc.MAT_K_FREE, u) / o.mL() - (2 - 2 * np.cos(2 * np.pi * h[0] / L[0])) / h[0] ** 2 * u
    assert np.abs(r).max() <= 1e-12


def test_nullspace_dimension_is_d(orc):
    """Eq. 20: under periodic boundary conditions ker K = constants, dim = d (1 for the scalar problems, 3 for
    K^mech: translations only -- infinitesimal rotations are not periodic)."""
    C = inputs.isotropic_voigt(200e9, 0.3)
    mesh, dof, nd, o = _periodic(orc, (5, 5, 4), (16 * NM, 16 * NM, 12 * NM), 7, mat=inputs.Material(C_voigt=C[None]))
    w = np.linalg.eigvalsh(o.csr(orc.MAT_K_FREE).toarray())
    assert np.sum(np.abs(w) < 1e-10 * w.max()) == 1 and w.min() > -1e-10 * w.max()
    A = o.csr(orc.MAT_K_MECH_FREE).toarray()
    assert np.abs(A - A.T).max() <= 1e-13 * np.abs(A).max()
    w = np.linalg.eigvalsh(A)
    assert np.sum(np.abs(w) < 1e-10 * w.max()) == 3 and w.min() > -1e-10 * w.max()
    for a in range(3):                                           # translations
        t = np.zeros((nd, 3)); t[:, a] = 1
        assert np.abs(o.spmv(orc.MAT_K_MECH_FREE, t.ravel())).max() <= 1e-12 * np.abs(A).max()
    # the non-periodic box of the same mesh has the six rigid-body modes
    o2 = orc.Oracle(mesh, inputs.Material(C_voigt=C[None]), 1e-12)
    w2 = np.linalg.eigvalsh(o2.csr(orc.MAT_K_MECH_FREE).toarray())
    assert np.sum(np.abs(w2) < 1e-10 * w2.max()) == 6


def test_literal_rhs_equals_adjoint_rhs_when_periodic(orc):
    """R9: the paper's Eq. 14 right-hand side -int phi_i div(m~) and the adjoint form int grad phi_i . m~ differ
    by a boundary term that vanishes on a fully periodic domain.  Literal form written out here from the oracle's
    element volumes and gradients: -sum_{e contains i} V_e/4 sum_k grad phi_k . m_k."""
    mesh, dof, nd, o = _periodic(orc, (6, 5, 5), (20 * NM, 16 * NM, 16 * NM), 7, pin_node=3)
    rng = np.random.default_rng(7)
    m = rng.normal(size=(nd, 3)); m /= np.linalg.norm(m, axis=1, keepdims=True)
    V, G = o.V(), o.G()
    t = dof[mesh.tets]
    div = np.einsum("ekd,ekd->e", G, m[t])
    lit = np.zeros(nd)
    np.add.at(lit, t.ravel(), np.repeat(-V * div / 4, 4))
    b = o.rhs_ms(m)
    assert b[3] == 0.0
    keep = np.arange(nd) != 3
    assert np.abs(b[keep] - lit[keep]).max() <= 1e-12 * np.abs(lit).max()
    assert abs(lit.sum()) <= 1e-12 * np.abs(lit).sum()
    # on the natural-boundary box the two forms differ (that is why R9 is needed there)
    o2 = orc.Oracle(mesh, inputs.Material(), 1e-12, pin_node=3)
    m2 = rng.normal(size=(mesh.n_nodes, 3))
    lit2 = np.zeros(mesh.n_nodes)
    np.add.at(lit2, mesh.tets.ravel(), np.repeat(-o2.V() * np.einsum("ekd,ekd->e", o2.G(), m2[mesh.tets]) / 4, 4))
    assert np.abs(o2.rhs_ms(m2) - lit2).max() > 1e-3 * np.abs(lit2).max()


def test_periodic_gspm_fixed_point_energy_decay_unit_length(orc):
    terms = TERM_ANIS | TERM_DEMAG | TERM_FARFIELD | TERM_ZEEMAN
    mesh, dof, nd, o = _periodic(orc, (7, 7, 6), (18 * NM, 18 * NM, 15 * NM), 7)
    dt = 1e-12
    # uniform m along an easy axis, field along it: fixed point (no exchange, no demag charge, h || m)
    m = np.zeros((nd, 3)); m[:, 2] = 1
    U = np.zeros(nd); u = np.zeros((nd, 3))
    info, rc = o.gspm_step(m, U, u, dt, [0, 0, 5e4], terms, cg_tol=1e-12)
    assert rc == 0 and np.abs(m - [0, 0, 1]).max() <= 1e-14
    # random start: |m| = 1 after every step, discrete energy decays
    rng = np.random.default_rng(8)
    m = rng.normal(size=(nd, 3)); m /= np.linalg.norm(m, axis=1, keepdims=True)
    hext = np.zeros(3)
    E = [o.energy(m, U, u, hext, terms)]
    for _ in range(8):
        info, rc = o.gspm_step(m, U, u, dt, [0, 0, 0], terms, cg_tol=1e-12)
        assert rc == 0
        assert np.abs(np.linalg.norm(m, axis=1) - 1).max() <= 4 * np.finfo(float).eps
        E.append(o.energy(m, U, u, hext, terms))
    assert all(b < a for a, b in zip(E, E[1:])), E


@pytest.mark.parametrize("d", [0, 1, 2])
def test_plane_wave_demag_chain_closed_form(orc, d):
    """The SOLVED magnetostatic chain (right-hand side -> CG on the pinned K^ms -> gradient recovery, O-3 items 2-3)
    against a closed form.  Fully periodic un-jittered Kuhn grid, m~ = a cos(k x_d) with k = 2 pi n / L_d.  Then m_h
    depends on x_d only, the nodal basis functions of a lattice plane sum to the 1-D hat function, and every node's
    support is point-symmetric, so all three steps collapse to 1-D central differences:
        b_i = a_d (V_cell / h_d) sin(k h_d) sin(k x_i),   K U = (V_cell / h_d^2)(2 - 2 cos k h_d) U,
        recovered dU/dx_d = (U_{+} - U_{-}) / (2 h_d)
    =>  h_d = -e_d a_d cos^2(k h_d / 2) cos(k x_d)   (continuum: -k (k.a)/|k|^2 cos(k.x); mbar = 0)."""
    grid, box = (9, 7, 6), (24 * NM, 15 * NM, 10 * NM)
    mesh, dof, nd, o = _periodic(orc, grid, box, 7, jitter=0.0, pin_node=11)
    L = np.array(box) / 1e-9
    h = L / (np.array(grid) - 1)
    x = np.zeros((nd, 3)); x[dof] = np.where(mesh.xyz / 1e-9 >= L - 1e-9, 0.0, mesh.xyz / 1e-9)
    a = np.array([0.7, -0.4, 0.55])
    n = 2 if d == 0 else 1
    k = 2 * np.pi * n / L[d]
    m = np.outer(np.cos(k * x[:, d]), a)
    mbar = o.volume_average(m)
    assert np.abs(mbar).max() < 1e-14
    b = o.rhs_ms(m, mbar)
    b_exact = a[d] * h.prod() / h[d] * np.sin(k * h[d]) * np.sin(k * x[:, d])
    keep = np.arange(nd) != 11
    assert b[11] == 0.0 and np.abs(b[keep] - b_exact[keep]).max() <= 1e-13 * np.abs(b_exact).max()
    U, it, res, rc = o.cg(orc.MAT_K_MS, b, tol=1e-14)
    assert rc == 0 and it > 0
    A = a[d] * h[d] / 2 / np.tan(k * h[d] / 2)
    U_exact = A * (np.sin(k * x[:, d]) - np.sin(k * x[11, d]))
    assert np.abs(U - U_exact).max() <= 1e-11 * abs(A)
    hd, gm = o.demag_field(U, mbar, TERM_DEMAG | TERM_FARFIELD)
    assert np.abs(gm).max() <= 1e-13
    hd_exact = np.zeros((nd, 3)); hd_exact[:, d] = -a[d] * np.cos(k * h[d] / 2) ** 2 * np.cos(k * x[:, d])
    assert np.abs(hd - hd_exact).max() <= 1e-11 * abs(a[d])
