"""Pins for the oracle's Jacobi-preconditioned CG (SURVEY 8f unranked row; the paper's future work: "no
preconditioner by choice").  CPU only.  Checked against things other than the oracle: dense solves, the textbook identity
PCG(A, D) == CG(D^-1/2 A D^-1/2) iterate by iterate (plain CG written out here in numpy), and the iteration counts of plain CG."""
import numpy as np
import pytest

from paper_2510_09812_b200 import inputs

NM = 1e-9


@pytest.fixture(scope="module")
def orc(oracle_mod):
    return oracle_mod


@pytest.fixture(scope="module")
def case(orc):
    mesh = inputs.kuhn_box((9, 8, 7), (27 * NM, 24 * NM, 21 * NM), seed_mesh=61, seed_perm=62)
    mesh = inputs.flag_inclusion(mesh, np.array(mesh.box) / 2, (6 * NM, 5 * NM, 5 * NM))
    C = inputs.isotropic_voigt(200e9, 0.3)
    clamp = inputs.clamp_bottom(mesh)
    o = orc.Oracle(mesh, inputs.Material(C_voigt=np.stack([C, 2 * C])), 5e-12, clamp_dof=clamp, pin_node=4)
    return mesh, clamp, o


def numpy_cg(A, b, k):
    """k iterations of textbook CG from x0 = 0, plain numpy."""
    x = np.zeros_like(b); r = b.copy(); p = r.copy(); rr = r @ r
    for _ in range(k):
        Ap = A @ p
        al = rr / (p @ Ap)
        x += al * p; r -= al * Ap
        rn = r @ r
        p = r + (rn / rr) * p
        rr = rn
    return x


def rhs(o, orc, mat, clamp, seed):
    rng = np.random.default_rng(seed)
    n = 3 * o.N if mat == orc.MAT_K_MECH else o.N
    b = rng.normal(size=n)
    if mat == orc.MAT_K_MS:
        b[4] = 0
    if mat == orc.MAT_K_MECH:
        b[clamp.astype(bool)] = 0
    return b


@pytest.mark.parametrize("which", ["ms", "gs1", "mech"])
def test_pcg_is_cg_on_the_symmetrically_scaled_system(orc, case, which):
    mesh, clamp, o = case
    mat = {"ms": orc.MAT_K_MS, "gs1": orc.MAT_K_GS1, "mech": orc.MAT_K_MECH}[which]
    A = o.csr(mat)
    d = A.diagonal()
    assert np.all(d > 0)
    s = 1 / np.sqrt(d)
    import scipy.sparse as sp
    Ah = sp.diags(s) @ A @ sp.diags(s)
    b = rhs(o, orc, mat, clamp, 5)
    for k in (1, 2, 5, 9):
        x, it, res, rc = o.cg_pc(mat, b, fixed=k, precond=1)
        assert it == k and rc == 0
        xs = s * numpy_cg(Ah, s * b, k)
        assert np.abs(x - xs).max() <= 1e-11 * np.abs(xs).max(), (which, k)
        # and it is NOT plain CG: the preconditioner changes the iterates (the diagonal is not constant)
        x0, _, _, _ = o.cg(mat, b, fixed=k)
        assert np.abs(x - x0).max() > 1e-6 * np.abs(x0).max()


@pytest.mark.parametrize("which", ["ms", "gs2", "mech"])
def test_pcg_dense_solution_and_stopping_rule(orc, case, which):
    mesh, clamp, o = case
    mat = {"ms": orc.MAT_K_MS, "gs2": orc.MAT_K_GS2, "mech": orc.MAT_K_MECH}[which]
    A = o.csr(mat).toarray()
    b = rhs(o, orc, mat, clamp, 6)
    x, it, res, rc = o.cg_pc(mat, b, tol=1e-12, precond=1)
    xd = np.linalg.solve(A, b)
    assert rc == 0 and np.abs(x - xd).max() <= 1e-9 * np.abs(xd).max()
    # the stopping rule is the 2-norm of the residual in both variants: reported = true residual
    assert res < 1e-12 and np.linalg.norm(b - A @ x) / np.linalg.norm(b) == pytest.approx(res, rel=1e-2, abs=1e-13)
    # zero right-hand side, warm start at the solution, maxiter
    x0, it0, _, _ = o.cg_pc(mat, np.zeros_like(b), x0=b, precond=1)
    assert it0 == 0 and np.abs(x0).max() == 0
    _, it1, _, _ = o.cg_pc(mat, b, x0=x, tol=1e-9, precond=1)
    assert it1 == 0
    _, it2, _, rc2 = o.cg_pc(mat, b, tol=1e-14, maxiter=3, precond=1)
    assert it2 == 3 and rc2 == orc.ORC_W_MAXITER


def test_precond_zero_is_plain_cg_bit_for_bit(orc, case):
    mesh, clamp, o = case
    for mat, seed in ((orc.MAT_K_MS, 7), (orc.MAT_K_MECH, 8)):
        b = rhs(o, orc, mat, clamp, seed)
        xa, ita, resa, _ = o.cg(mat, b, tol=1e-9)
        xb, itb, resb, _ = o.cg_pc(mat, b, tol=1e-9, precond=0)
        assert ita == itb and resa == resb and np.array_equal(xa, xb)


def test_jacobi_does_not_need_more_iterations_on_the_stiff_inclusion(orc, case):
    """x2 stiffness in the inclusion and short rows on the boundary make diag(K^mech) non-uniform: Jacobi scaling
    helps a little; on the (nearly uniform) Laplacian it is neutral.  Counts printed for DESIGN.md."""
    mesh, clamp, o = case
    out = {}
    for name, mat, seed in (("ms", orc.MAT_K_MS, 9), ("mech", orc.MAT_K_MECH, 10), ("gs1", orc.MAT_K_GS1, 11)):
        b = rhs(o, orc, mat, clamp, seed)
        _, it_plain, _, _ = o.cg(mat, b, tol=1e-8)
        _, it_pc, _, _ = o.cg_pc(mat, b, tol=1e-8, precond=1)
        out[name] = (it_plain, it_pc)
        assert it_pc <= it_plain + 1, out
    print(out)


def test_history_is_the_recurrence_residual(orc, case):
    mesh, clamp, o = case
    b = rhs(o, orc, orc.MAT_K_MECH, clamp, 12)
    x, it, hist = o.cg_history(orc.MAT_K_MECH, b, tol=1e-8)
    assert len(hist) == it + 1 and hist[0] == pytest.approx(1.0) and hist[-1] < 1e-8 <= hist[-2]
    A = o.csr(orc.MAT_K_MECH)
    for k in (3, 10):
        xk, _, resk, _ = o.cg(orc.MAT_K_MECH, b, fixed=k)
        assert hist[k] == resk
        assert np.linalg.norm(b - A @ xk) / np.linalg.norm(b) == pytest.approx(hist[k], rel=1e-9)


def test_fp64_cg_parts_from_an_extended_precision_cg_by_rounding():
    """The fact behind the 1.5 % allowance on in-step mechanical CG counts, on the CPU side: the
    oracle's fp64 CG and a numpy long-double CG of the same system (step-0 mechanical solve of the inclusion mesh of
    tests/test_gpu_pcg_sigma.py::test_mechanical_residual_curves_part_by_rounding) agree to rounding for the first 40
    iterations, part between iterations 40 and 100 (loss of orthogonality amplifies rounding by about x4 per iteration)
    and from there on differ by per cent to tens of per cent while crossing 1e-7 / 1e-10 / 1e-12 within 1.5 % of each
    other.  Any second fp64 run with another rounding (plain numpy here; the device in the GPU test) does the same."""
    import oracle as orc
    orc.build()
    mesh = inputs.kuhn_box((13, 13, 7), (40 * NM, 40 * NM, 20 * NM), seed_mesh=21, seed_perm=22)
    mesh = inputs.flag_inclusion(mesh, np.array(mesh.box) / 2, (8 * NM,) * 3)
    C = inputs.isotropic_voigt(200e9, 0.3)
    o = orc.Oracle(mesh, inputs.Material(C_voigt=np.stack([C, 2 * C])), 1e-12, clamp_dof=inputs.clamp_bottom(mesh))
    b = o.rhs_mech(inputs.init_m_noisy_x(mesh, 23)).ravel()
    _, ito, ho = o.cg_history(orc.MAT_K_MECH, b, tol=1e-12)
    A = o.csr(orc.MAT_K_MECH)

    def history(ft):
        data, idx, ptr = A.data.astype(ft), A.indices, A.indptr[:-1]
        bb_ = b.astype(ft); x = np.zeros_like(bb_); r = bb_.copy(); p = r.copy()
        bb = bb_ @ bb_; rr = r @ r
        h = [float(np.sqrt(rr / bb))]
        while h[-1] >= 1e-12 and len(h) < 5000:
            Ap = np.add.reduceat(data * p[idx], ptr)
            al = rr / (p @ Ap); x += al * p; r -= al * Ap
            rn = r @ r; p = r + (rn / rr) * p; rr = rn
            h.append(float(np.sqrt(rr / bb)))
        return np.array(h)

    hx, hn = history(np.longdouble), history(np.float64)
    if np.finfo(np.longdouble).nmant <= 52:
        pytest.skip("long double is not wider than double on this platform")
    n = min(len(ho), len(hx), len(hn))
    for h in (ho, hn):
        dev = np.abs(h[:n] - hx[:n]) / hx[:n]
        onset = int(np.argmax(dev > 1e-6))
        assert dev[:40].max() < 1e-12 and 40 < onset < 100 and 1e-3 < dev.max() < 1.5, (onset, dev.max())
    for tol in (1e-7, 1e-10, 1e-12):
        io, ix = int(np.argmax(ho < tol)), int(np.argmax(hx < tol))
        assert abs(io - ix) <= max(1, int(np.ceil(0.015 * ix)))
