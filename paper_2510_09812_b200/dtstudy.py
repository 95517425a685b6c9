"""Time-step study in the paper's own setting (Fig. 3): structured linear-hexahedral mesh, periodic boundaries, a
non-magnetic cuboid defect with doubled stiffness, uniform initial magnetisation under a fixed field of 200 A/m, all physics.
For each dt the state is relaxed for a fixed number of GSPM steps and the CG iteration counts of the last steps are reported
(the paper quotes 1-3 per Helmholtz solve, 40-90 magnetostatic, 150-200 mechanical near equilibrium on its 550 k-node mesh and
material; BASELINE's material is used here, so the counts are context, not a reproduction).

  python -m paper_2510_09812_b200.dtstudy [--side 82] [--steps 150] [--dts 2,4,8,11]
"""
from __future__ import annotations

import argparse

import numpy as np

from . import inputs


def main(argv=None):
    import torch
    from . import binding as cm
    ap = argparse.ArgumentParser()
    ap.add_argument("--side", type=int, default=82, help="nodes per edge before wrapping (82 -> 531,441 DOFs)")
    ap.add_argument("--steps", type=int, default=150)
    ap.add_argument("--dts", default="2,4,8,11", help="time steps in ps")
    ap.add_argument("--alpha", type=float, default=0.15, help="Gilbert damping (P:284)")
    a = ap.parse_args(argv)
    n = a.side
    L = (n - 1) * 2.5e-9
    mesh = inputs.hex_box((n, n, n), (L, L, L), seed_mesh=91, seed_perm=92)
    c = mesh.xyz[mesh.hexes].mean(axis=1) - L / 2
    inside = (np.abs(c) <= np.array([0.15, 0.10, 0.10]) * L).all(axis=1)          # cuboid defect at the centre
    mag = mesh.magnetic.copy(); eid = mesh.elastic_id.copy()
    mag[inside] = 0; eid[inside] = 1
    dof, nd = cm.periodic_wrap(mesh.xyz, 7)
    C = inputs.isotropic_voigt(200e9, 0.3)
    mat = inputs.Material(alpha=a.alpha, C_voigt=np.stack([C, 2 * C]))
    clamp = np.zeros((nd, 3), np.uint8); clamp[0] = 1                              # pin d = 3 displacement DOFs
    terms = inputs.TERM_ANIS | inputs.TERM_ZEEMAN | inputs.TERM_DEMAG | inputs.TERM_FARFIELD | inputs.TERM_MAGEL
    gm = cm.Mesh(mesh.xyz, mesh.hexes, mag, eid, cm.CM_REORDER_MORTON, dof_of_node=dof, n_dof=nd)
    print(f"periodic hexahedral mesh: {nd} DOFs, {gm.n_tets} cells ({int(inside.sum())} in the defect), {gm.nnz} nonzeros; "
          f"alpha = {a.alpha}, H = 200 A/m e1, CG tol 1e-7, {a.steps} steps per dt")
    print(f"{'dt/ps':>6} {'dtau':>7} {'ms/step':>8} {'it_ms':>6} {'it_mech':>8} {'it_gs (8 solves)':>28} {'<|dm|>':>10}")
    for dt_ps in [float(x) for x in a.dts.split(",")]:
        dt = dt_ps * 1e-12
        gs = cm.System(gm, mat, dt, "f64", clamp.ravel(), 0)
        rng = np.random.default_rng(93)
        m0 = np.array([1.0, 0.0, 0.0]) + 1e-3 * rng.normal(size=(nd, 3))
        m0 /= np.linalg.norm(m0, axis=1, keepdims=True)
        m = torch.as_tensor(m0, dtype=torch.float64, device="cuda").contiguous()
        live = torch.as_tensor(gs.geometry(3) > 0, device="cuda")                    # mLm > 0 <=> magnetic node (library order)
        order = torch.as_tensor(gm.get(cm.CM_GET_ORDER).astype(np.int64), device="cuda")
        mask = torch.zeros(nd, dtype=torch.bool, device="cuda"); mask[order] = live
        m[~mask] = 0
        U = torch.zeros(nd, dtype=torch.float64, device="cuda"); u = torch.zeros((nd, 3), dtype=torch.float64, device="cuda")
        p = cm.make_params(dt, [200.0, 0.0, 0.0], terms, 0, 1e-7)
        last = []
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        for k in range(a.steps):
            info, rc = gs.gspm_step(p, m, U, u)
            if k >= a.steps - 10:
                last.append((info.it_ms, info.it_mech, list(info.it_gs), info.mean_dm))
        ev1.record(); torch.cuda.synchronize()
        ms = ev0.elapsed_time(ev1) / a.steps
        it_ms = np.mean([l[0] for l in last]); it_me = np.mean([l[1] for l in last])
        it_gs = np.mean([l[2] for l in last], axis=0)
        finite = bool(torch.isfinite(m).all())
        print(f"{dt_ps:6.1f} {gs_dtau(mat, dt):7.3f} {ms:8.2f} {it_ms:6.1f} {it_me:8.1f} {np.array2string(it_gs, precision=1, floatmode='fixed'):>28} "
              f"{last[-1][3]:10.2e}{'' if finite else '  (diverged)'}")
        gs.close()
    gm.close()


def gs_dtau(mat, dt):
    return mat.gamma * mat.Ms * dt


if __name__ == "__main__":
    main()
