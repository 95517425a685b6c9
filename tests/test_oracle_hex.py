"""Pins for the oracle's linear hexahedral (Q1) matrices (R26).  CPU only.
Closed forms of the trilinear element on a uniform grid (the classical 27-point stiffness and the tensor-product mass),
exactness properties of the 2 x 2 x 2 Gauss rule on distorted cells (volume, patch test, rigid-body modes, linear-field
energies and averages), and dense solves."""
import numpy as np
import pytest

from paper_2510_09812_b200 import inputs

NM = 1e-9
MU0 = 4e-7 * np.pi


@pytest.fixture(scope="module")
def orc(oracle_mod):
    return oracle_mod


def mat2():
    C = inputs.isotropic_voigt(200e9, 0.3)
    return inputs.Material(C_voigt=np.stack([C, 2 * C]))


@pytest.fixture(scope="module")
def jit(orc):
    mesh = inputs.hex_box((7, 6, 5), (18 * NM, 15 * NM, 10 * NM), seed_mesh=3, seed_perm=4)
    mesh = inputs.flag_inclusion(mesh, np.array(mesh.box) / 2, (5 * NM, 4 * NM, 3 * NM))
    clamp = inputs.clamp_bottom(mesh)
    return mesh, orc.Oracle(mesh, mat2(), 1e-12, clamp_dof=clamp, pin_node=2), clamp


def test_hex_generator_local_node_order():
    mesh = inputs.hex_box((3, 4, 5), (2 * NM, 3 * NM, 4 * NM), jitter=0.0)
    x = mesh.xyz[mesh.hexes] / NM                     # (Ne, 8, 3)
    assert np.allclose(x[:, 1] - x[:, 0], [1, 0, 0]) and np.allclose(x[:, 2] - x[:, 0], [0, 1, 0])
    assert np.allclose(x[:, 4] - x[:, 0], [0, 0, 1]) and np.allclose(x[:, 7] - x[:, 0], [1, 1, 1])
    assert mesh.n_tets == 2 * 3 * 4


def test_uniform_grid_closed_forms(orc):
    """Cubic cells of side h: K = 27-point stencil (8h/3 centre, 0 faces, -h/6 edges, -h/12 corners);
    M = tensor product of the 1D consistent mass h/6 [1 4 1]."""
    n, h = 6, 2.0
    mesh = inputs.hex_box((n, n, n), ((n - 1) * h * NM,) * 3, jitter=0.0, permute=False)
    o = orc.Oracle(mesh, inputs.Material(), 1e-12)
    assert o.nnz == (3 * n - 2) ** 3                               # (sum over a line of 2,3,...,3,2)^3
    K = o.csr(orc.MAT_K_FREE).toarray(); M = o.csr(orc.MAT_MASS).toarray()
    nid = lambda a, b, c: (c * n + b) * n + a
    i = nid(2, 3, 2)
    kexp = {0: 8 * h / 3, 1: 0.0, 2: -h / 6, 3: -h / 12}
    m1 = {0: 4 * h / 6, 1: h / 6}
    for da in (-1, 0, 1):
        for db in (-1, 0, 1):
            for dc in (-1, 0, 1):
                j = nid(2 + da, 3 + db, 2 + dc)
                assert K[i, j] == pytest.approx(kexp[abs(da) + abs(db) + abs(dc)], abs=1e-13)
                assert M[i, j] == pytest.approx(m1[abs(da)] * m1[abs(db)] * m1[abs(dc)], rel=1e-13)
    assert np.count_nonzero(np.abs(K[i]) > 1e-12) == 1 + 12 + 8
    assert np.allclose(o.mL().reshape(n, n, n)[1:-1, 1:-1, 1:-1], h ** 3, rtol=1e-13)


def test_symmetry_rowsums_volume_patch(orc, jit):
    mesh, o, clamp = jit
    K = o.csr(orc.MAT_K_FREE); Km = o.csr(orc.MAT_K_M); M = o.csr(orc.MAT_MASS)
    for A in (K, Km, M):
        assert abs(A - A.T).max() <= 1e-14 * abs(A).max()
    assert np.abs(K.sum(1)).max() <= 1e-13 * abs(K).sum(1).max()
    vol = np.prod(np.array(mesh.box) / NM)
    assert o.Vtot == pytest.approx(vol, rel=1e-13) and o.V().sum() == pytest.approx(vol, rel=1e-13)
    assert o.mL().sum() == pytest.approx(vol, rel=1e-13)
    assert np.allclose(np.asarray(M.sum(1)).ravel(), o.mLm(), rtol=1e-12, atol=1e-13)
    assert M.sum() == pytest.approx(o.Vmag, rel=1e-13) and 0 < o.Vmag < vol
    # patch test: a linear field gives zero at every node off the outer boundary (2 x 2 x 2 Gauss is exact for it)
    x = mesh.xyz / NM
    u = x @ np.array([0.3, -0.7, 0.2]) + 1.5
    r = K @ u
    L = np.array(mesh.box) / NM
    interior = ((x > 1e-9) & (x < L - 1e-9)).all(1)
    assert interior.sum() > 20 and np.abs(r[interior]).max() <= 1e-12 * np.abs(K).max() * np.abs(u).max()
    assert u @ r == pytest.approx(vol * (0.09 + 0.49 + 0.04), rel=1e-12)          # int |grad u|^2
    w = np.linalg.eigvalsh(K.toarray())
    assert np.sum(np.abs(w) < 1e-10 * w.max()) == 1 and w.min() > -1e-10 * w.max()
    # consistent mass: u^T M u = int_{Omega_m} u^2 is NOT exact on distorted cells (degree 4 per variable), but 1^T M u is
    assert np.ones(o.N) @ (M @ u) == pytest.approx((o.mLm() * u).sum(), rel=1e-13)


def test_mech_matrix_rigid_modes_and_linear_energy(orc, jit):
    mesh, o, clamp = jit
    A = o.csr(orc.MAT_K_MECH_FREE)
    assert abs(A - A.T).max() <= 1e-13 * abs(A).max()
    x = mesh.xyz / NM
    for a in range(3):
        t = np.zeros((o.N, 3)); t[:, a] = 1
        assert np.abs(A @ t.ravel()).max() <= 1e-12 * abs(A).max()
        rot = np.cross(np.eye(3)[a], x)
        assert np.abs(A @ rot.ravel()).max() <= 1e-11 * abs(A).max() * np.abs(x).max()
    w = np.linalg.eigvalsh(A.toarray())
    assert np.sum(np.abs(w) < 1e-9 * w.max()) == 6
    # homogeneous body: u = G x has energy vol * symG : C* : symG
    mesh1 = inputs.hex_box((5, 5, 4), (10 * NM, 12 * NM, 9 * NM), seed_mesh=5, seed_perm=6)
    m1 = inputs.Material()
    o1 = orc.Oracle(mesh1, m1, 1e-12)
    G = np.array([[1e-3, 2e-3, 0.0], [-1e-3, 5e-4, 3e-3], [2e-3, 0.0, -1e-3]])
    u = (mesh1.xyz / NM) @ G.T
    E = 0.5 * (G + G.T)
    ev = np.array([E[0, 0], E[1, 1], E[2, 2], 2 * E[1, 2], 2 * E[0, 2], 2 * E[0, 1]])
    Cs = m1.C_voigt[0] / (MU0 * m1.Ms ** 2)
    A1 = o1.csr(orc.MAT_K_MECH_FREE)
    assert u.ravel() @ (A1 @ u.ravel()) == pytest.approx(10 * 12 * 9 * ev @ Cs @ ev, rel=1e-12)
    # constrained matrix: identity rows / columns at clamped DOFs
    Ac = o.csr(orc.MAT_K_MECH).toarray()
    c = np.flatnonzero(clamp)
    assert np.array_equal(Ac[c][:, c], np.eye(len(c))) and np.abs(Ac[c]).sum() == len(c)


def test_constraints_dead_nodes_and_helmholtz(orc, jit):
    mesh, o, clamp = jit
    live = o.live().astype(bool)
    assert 0 < (~live).sum() < o.N
    Kms = o.csr(orc.MAT_K_MS).toarray()
    assert Kms[2, 2] == 1 and np.abs(Kms[2]).sum() == 1 and np.abs(Kms[:, 2]).sum() == 1
    G1 = o.csr(orc.MAT_K_GS1).toarray()
    d = np.flatnonzero(~live)
    assert np.array_equal(G1[d][:, d], np.eye(len(d))) and np.abs(G1[d]).sum() == len(d)
    M = o.csr(orc.MAT_MASS).toarray(); Km = o.csr(orc.MAT_K_M).toarray()
    eps1 = o.Astar * o.dtau
    assert np.allclose(G1[live][:, live], (M + eps1 * Km)[live][:, live], rtol=1e-13, atol=1e-15)
    assert np.linalg.eigvalsh(G1).min() > 0


def test_volume_average_and_cg(orc, jit):
    mesh, o, clamp = jit
    x = mesh.xyz / NM
    g = np.stack([x @ [0.2, 0.1, -0.4] + 3.0, np.ones(o.N), x[:, 2]], axis=1)
    L = np.array(mesh.box) / NM
    assert np.allclose(o.volume_average(g), [L @ [0.2, 0.1, -0.4] / 2 + 3.0, 1.0, L[2] / 2], rtol=1e-13)
    rng = np.random.default_rng(1)
    for mat, n in ((orc.MAT_K_MS, o.N), (orc.MAT_K_GS1, o.N), (orc.MAT_K_MECH, 3 * o.N)):
        b = rng.normal(size=n)
        if mat == orc.MAT_K_MS:
            b[2] = 0
        if mat == orc.MAT_K_MECH:
            b[clamp.astype(bool)] = 0
        xs, it, res, rc = o.cg(mat, b, tol=1e-12)
        assert rc == 0 and it > 3
        assert np.abs(xs - np.linalg.solve(o.csr(mat).toarray(), b)).max() <= 1e-9 * np.abs(xs).max()


def test_hex_rhs_identities(orc, jit):
    """The tetrahedral pins of S3 / S5 / S6 / S8 carry over: uniform m gives b^ms = 0 and h_d = -N_d mbar; sum_i b_i = 0; the
    recovered gradient of a linear potential is exact; u = E0 x is stress free on a homogeneous body."""
    mesh, o, clamp = jit
    from paper_2510_09812_b200.inputs import TERM_DEMAG, TERM_FARFIELD, TERM_MAGEL
    mu = np.tile([0.6, 0.0, 0.8], (o.N, 1))
    mbar = o.volume_average(mu)
    assert np.allclose(mbar, [0.6, 0.0, 0.8], rtol=1e-14)
    assert np.abs(o.rhs_ms(mu)).max() < 1e-12
    hd, gm = o.demag_field(np.zeros(o.N), mbar, TERM_DEMAG | TERM_FARFIELD)
    assert np.allclose(hd, -mbar / 3, rtol=1e-13)
    rng = np.random.default_rng(3)
    m = rng.normal(size=(o.N, 3)); m /= np.linalg.norm(m, axis=1, keepdims=True)
    b = o.rhs_ms(m)
    o3 = orc.Oracle(mesh, mat2(), 1e-12, clamp_dof=clamp, pin_node=3)          # same body, other pin: gives the entry zeroed above
    b_full = b.copy(); b_full[2] = o3.rhs_ms(m)[2]
    assert b[2] == 0 and abs(b_full.sum()) < 1e-12 * np.abs(b_full).sum()      # sum_i grad phi_i = 0 pointwise
    x = mesh.xyz / NM
    a = np.array([0.3, -0.2, 0.5])
    hd, gm = o.demag_field(x @ a, np.zeros(3), TERM_DEMAG)
    assert np.allclose(gm, a, rtol=1e-13) and np.abs(hd).max() < 1e-12       # -grad U + <grad U> = 0 for linear U
    hd, gm = o.demag_field(x[:, 0] ** 2, np.zeros(3), TERM_DEMAG)
    assert np.abs(hd[:, 1:]).max() < 0.3 and np.abs(hd[:, 0]).max() > 1   # quadratic U: x-gradient only
    # stress-free state on a homogeneous, unclamped body
    mesh1 = inputs.hex_box((5, 5, 4), (10 * NM, 12 * NM, 9 * NM), seed_mesh=5, seed_perm=6)
    mat = inputs.Material()
    o1 = orc.Oracle(mesh1, mat, 1e-12)
    mdir = np.array([0.6, -0.48, 0.64])
    m1 = np.tile(mdir, (o1.N, 1))
    l1, l2 = mat.lambda100, mat.lambda111
    E0 = 1.5 * l2 * np.outer(mdir, mdir); E0[np.arange(3), np.arange(3)] = 1.5 * l1 * (mdir ** 2 - 1 / 3)
    u = (mesh1.xyz / NM) @ E0.T
    bm = o1.rhs_mech(m1)
    Ku = (o1.csr(orc.MAT_K_MECH_FREE) @ u.ravel()).reshape(-1, 3)
    assert np.abs(bm).max() > 1e-3 and np.abs(Ku - bm).max() < 1e-12 * np.abs(bm).max()
    sig = o1.stress_recover(u, m1)
    Cs = mat.C_voigt[0] / (MU0 * mat.Ms ** 2)
    e0v = np.array([E0[0, 0], E0[1, 1], E0[2, 2], 2 * E0[1, 2], 2 * E0[0, 2], 2 * E0[0, 1]])
    assert np.abs(sig).max() < 1e-12 * np.abs(Cs @ e0v).max()
    assert np.abs(o1.field(m1, None, sig, [0, 0, 0], TERM_MAGEL)).max() < 1e-13
    assert np.allclose(o1.stress_recover(np.zeros_like(u), m1), np.tile(-(Cs @ e0v), (o1.N, 1)), rtol=1e-12, atol=1e-16)


def _fd_field(energy, m, nodes, mass, h):
    out = np.zeros((len(nodes), 3))
    for a, i in enumerate(nodes):
        for c in range(3):
            mp = m.copy(); mp[i, c] += h
            mm = m.copy(); mm[i, c] -= h
            out[a, c] = -(energy(mp) - energy(mm)) / (2 * h) / mass[i]
    return out


def test_hex_fields_are_energy_gradients(orc, jit):
    """h_me = -(1/mLm_i) dE_el/dm_i at fixed u, and h_d = -(1/mLm_i) d/dm_i [1/2 U^T K U + far field] with U re-solved
    (central differences of the hexahedral discrete energy)."""
    mesh, o, clamp = jit
    from paper_2510_09812_b200.inputs import TERM_DEMAG, TERM_FARFIELD, TERM_MAGEL
    rng = np.random.default_rng(4)
    live = np.flatnonzero(o.live())
    m = rng.normal(size=(o.N, 3)); m /= np.linalg.norm(m, axis=1, keepdims=True); m[o.live() == 0] = 0
    u = 1e-3 * rng.normal(size=(o.N, 3))
    nodes = rng.choice(live, 4, replace=False)
    sig = o.stress_recover(u, m)
    h = o.field(m, None, sig, [0, 0, 0], TERM_MAGEL)
    fd = _fd_field(lambda mm: o.energy(mm, None, u, [0, 0, 0], TERM_MAGEL) - o.energy(mm, None, u, [0, 0, 0], 0), m, nodes, o.mLm(), 1e-4)
    assert np.abs(h[nodes]).max() > 1e-4 and np.allclose(h[nodes], fd, rtol=2e-6, atol=2e-8)
    assert np.abs(sig[o.live() == 0]).max() == 0

    def demag_energy(mm):
        b = o.rhs_ms(mm)
        U = o.cg(orc.MAT_K_MS, b, tol=1e-13)[0]
        return o.energy(mm, U, None, [0, 0, 0], TERM_DEMAG | TERM_FARFIELD) - o.energy(mm, U, None, [0, 0, 0], 0)
    U = o.cg(orc.MAT_K_MS, o.rhs_ms(m), tol=1e-13)[0]
    hd, _ = o.demag_field(U, o.volume_average(m), TERM_DEMAG | TERM_FARFIELD)
    interior_live = [i for i in live if o.mL()[i] == pytest.approx(o.mLm()[i], rel=1e-12)][:3]
    fd = _fd_field(demag_energy, m, interior_live, o.mL(), 1e-4)
    assert np.allclose(hd[interior_live], fd, rtol=1e-5, atol=1e-7)


def test_hex_gspm_step_invariants(orc):
    """|m| = 1 after every step, dead nodes stay zero, the discrete energy decays (config-0 physics on a hexahedral mesh),
    and uniform m along an easy axis with the field along it is a fixed point."""
    from paper_2510_09812_b200.inputs import TERM_ANIS, TERM_DEMAG, TERM_FARFIELD, TERM_ZEEMAN
    mesh = inputs.hex_box((8, 8, 8), (20 * NM,) * 3, seed_mesh=1, seed_perm=2)
    o = orc.Oracle(mesh, inputs.Material(), 1e-12)
    terms = TERM_ANIS | TERM_DEMAG | TERM_FARFIELD
    m = np.tile([0.0, 0.0, 1.0], (o.N, 1)); U = np.zeros(o.N); u = np.zeros((o.N, 3))
    info, rc = o.gspm_step(m, U, u, 1e-12, [0, 0, 5e4], TERM_ANIS | TERM_ZEEMAN | TERM_FARFIELD, cg_tol=1e-12)
    assert rc == 0 and np.abs(m - [0, 0, 1]).max() < 1e-14
    rng = np.random.default_rng(3)
    m = rng.normal(size=(o.N, 3)); m /= np.linalg.norm(m, axis=1, keepdims=True)
    E = [o.energy(m, U, u, np.zeros(3), terms)]
    for _ in range(8):
        info, rc = o.gspm_step(m, U, u, 1e-12, [0, 0, 0], terms, cg_tol=1e-12)
        assert rc == 0 and info.it_ms > 5
        assert np.abs(np.linalg.norm(m, axis=1) - 1).max() <= 4 * np.finfo(float).eps
        E.append(o.energy(m, U, u, np.zeros(3), terms))
    assert all(b < a for a, b in zip(E, E[1:])), E


def test_hex_degenerate_cell_rejected(orc, jit):
    mesh, o, clamp = jit
    bad = inputs.replace(mesh, hexes=mesh.hexes[:, [1, 0, 2, 3, 4, 5, 6, 7]].copy())     # inverted cells
    with pytest.raises(RuntimeError, match="rc=-2"):
        orc.Oracle(bad, mat2(), 1e-12)


def test_periodic_hexahedra(orc):
    """Node wrapping on hexahedra -- the paper's own setting (structured hexahedral meshes, periodic): 27 entries
    in every row; on the uniform grid the stiffness is circulant with the closed-form symbol of the trilinear element;
    ker K = constants, ker K^mech = the three translations (Eq. 20: d = 3); the literal Eq. 14 right-hand side equals the
    adjoint one (R9); uniform m along an easy axis is a fixed point and the energy decays."""
    from paper_2510_09812_b200.inputs import TERM_ANIS, TERM_DEMAG, TERM_FARFIELD
    grid, box = (7, 6, 5), (24 * NM, 15 * NM, 10 * NM)
    mesh = inputs.hex_box(grid, box, jitter=0.0, seed_mesh=5, seed_perm=6)
    dof, nd = orc.periodic_wrap(mesh.xyz, 7)
    assert nd == 6 * 5 * 4
    o = orc.Oracle(mesh, inputs.Material(), 1e-12, dof_of_node=dof, n_dof=nd)
    assert o.N == nd and np.all(np.diff(o.rowptr()) == 27)
    h = np.array(box) / NM / (np.array(grid) - 1)
    L = np.array(box) / NM
    x = np.zeros((nd, 3)); x[dof] = np.where(mesh.xyz / NM >= L - 1e-9, 0.0, mesh.xyz / NM)
    assert np.allclose(o.mL(), h.prod(), rtol=1e-13)
    for d in range(3):
        u = np.cos(2 * np.pi * x[:, d] / L[d])
        th = 2 * np.pi * h[d] / L[d]
        lam = h.prod() / h[d] ** 2 * (2 - 2 * np.cos(th))        # k1(theta) m1(0) m1(0): 1D stiffness symbol x full 1D masses
        assert np.abs(o.spmv(orc.MAT_K_FREE, u) - lam * u).max() <= 1e-12 * lam
        mu = h.prod() * (4 + 2 * np.cos(th)) / 6                 # 1D consistent-mass symbol h (4 + 2 cos theta) / 6
        assert np.abs(o.spmv(orc.MAT_MASS, u) - mu * u).max() <= 1e-12 * mu
    # jittered periodic cells with mechanics
    C = inputs.isotropic_voigt(200e9, 0.3)
    mesh = inputs.hex_box((6, 5, 5), (20 * NM, 16 * NM, 16 * NM), seed_mesh=5, seed_perm=6)
    dof, nd = orc.periodic_wrap(mesh.xyz, 7)
    clamp = np.zeros((nd, 3), np.uint8); clamp[4] = 1
    o = orc.Oracle(mesh, inputs.Material(C_voigt=C[None]), 1e-12, clamp_dof=clamp.ravel(), pin_node=3, dof_of_node=dof, n_dof=nd)
    assert o.Vtot == pytest.approx(20 * 16 * 16, rel=1e-13)
    w = np.linalg.eigvalsh(o.csr(orc.MAT_K_FREE).toarray())
    assert np.sum(np.abs(w) < 1e-10 * w.max()) == 1
    w = np.linalg.eigvalsh(o.csr(orc.MAT_K_MECH_FREE).toarray())
    assert np.sum(np.abs(w) < 1e-10 * w.max()) == 3
    rng = np.random.default_rng(7)
    m = rng.normal(size=(nd, 3)); m /= np.linalg.norm(m, axis=1, keepdims=True)
    # literal Eq. 14: -sum_e sum_p |J| phi_i div m_h, written out here with numpy from the trilinear shape functions
    g = 1 / np.sqrt(3)
    lit = np.zeros(nd)
    sgn = np.array([[(a >> d & 1) * 2 - 1 for d in range(3)] for a in range(8)], float)
    for e in range(mesh.n_tets):
        X = mesh.xyz[mesh.hexes[e]] / NM
        t = dof[mesh.hexes[e]]
        for p in range(8):
            xi = np.array([(p >> d & 1) * 2 - 1 for d in range(3)], float) * g
            f = 1 + sgn * xi
            phi = f.prod(1) / 8
            dN = np.stack([sgn[:, 0] * f[:, 1] * f[:, 2], f[:, 0] * sgn[:, 1] * f[:, 2], f[:, 0] * f[:, 1] * sgn[:, 2]], 1) / 8
            J = X.T @ dN
            G = dN @ np.linalg.inv(J)
            lit[t] += -np.linalg.det(J) * phi * np.einsum("ad,ad->", G, m[t])
    b = o.rhs_ms(m)
    keep = np.arange(nd) != 3
    assert b[3] == 0 and np.abs(b[keep] - lit[keep]).max() <= 1e-11 * np.abs(lit).max()
    terms = TERM_ANIS | TERM_DEMAG | TERM_FARFIELD
    mz = np.tile([0.0, 0.0, 1.0], (nd, 1)); U = np.zeros(nd); u = np.zeros((nd, 3))
    info, rc = o.gspm_step(mz, U, u, 1e-12, [0, 0, 0], terms, cg_tol=1e-12)
    assert rc == 0 and np.abs(mz - [0, 0, 1]).max() < 1e-14
    E = [o.energy(m, U, u, np.zeros(3), terms)]
    for _ in range(6):
        info, rc = o.gspm_step(m, U, u, 1e-12, [0, 0, 0], terms, cg_tol=1e-12)
        assert rc == 0 and np.abs(np.linalg.norm(m, axis=1) - 1).max() <= 4 * np.finfo(float).eps
        E.append(o.energy(m, U, u, np.zeros(3), terms))
    assert all(b2 < a2 for a2, b2 in zip(E, E[1:])), E
    # one cell across a periodic direction collapses the cell
    thin = inputs.hex_box((2, 4, 4), (5 * NM, 12 * NM, 12 * NM))
    dof, nd = orc.periodic_wrap(thin.xyz, 1)
    with pytest.raises(RuntimeError, match="rc=-1"):
        orc.Oracle(thin, inputs.Material(), 1e-12, dof_of_node=dof, n_dof=nd)
