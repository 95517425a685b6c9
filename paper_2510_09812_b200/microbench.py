"""BASELINE.json config 4: SpMV / CG microbenchmark sweep.

Scalar P1 Laplacian (CSR) and 3x3-block linear-elasticity stiffness (BSR) assembled from jittered Kuhn-tet cubes of
n^3 nodes (2.5 nm spacing, seeded node permutation), before (CM_REORDER_NONE) and after (Morton / RCM) locality
reordering, fp32 and fp64; right-hand side = seeded Gaussian; unpreconditioned CG for a fixed 3 iterations and to
relative residual 1e-8.  Reports time, algorithmic GB/s (SURVEY 8d byte model) and the fraction of the measured
HBM copy bandwidth.  Sizes <= 80^3 are L2-resident on B200 (126 MB L2) and are labelled so.

  python -m paper_2510_09812_b200.microbench [--sides 47,80,100,144] [--dtypes f64,f32] [--reorders none,morton]
                                             [--only spmv_bsr3] [--reps 20] [--json out.json]
"""
from __future__ import annotations

import argparse
import json
import sys
from pathlib import Path

import numpy as np

from . import inputs

ROOT = Path(__file__).resolve().parent.parent


def peak_gbs():
    p = ROOT / "MEASURED_PEAKS.json"
    return float(json.loads(p.read_text())["hbm_gbs"]) if p.exists() else 6650.0


def model_bytes(N, nnz, s):
    return {"spmv_csr1": nnz * (s + 4) + N * (4 + 2 * s), "spmv_csr3": nnz * (s + 4) + N * 4 + 6 * N * s,
            "spmv_bsr3": nnz * (9 * s + 4) + N * 4 + 6 * N * s,
            "cg_csr1": nnz * (s + 4) + N * (4 + 2 * s) + 10 * N * s, "cg_csr3": nnz * (s + 4) + N * 4 + 36 * N * s,
            "cg_bsr3": nnz * (9 * s + 4) + N * 4 + 36 * N * s}


def elem_bytes(N, Ne, s):
    """Element passes, stored gradients: 16 B connectivity + 13 words per tet, nodal input and output once."""
    tet = Ne * (16 + 13 * s)
    return {"elem_rhs_ms": tet + N * 4 * s, "elem_hd": tet + N * 4 * s, "elem_rhs_mech": tet + N * 6 * s,
            "elem_sigma": tet + N * 12 * s}


def hex_elem_bytes(N, Ne, s):
    """Hexahedral passes: 32 B connectivity per cell, coordinates (fp64) and nodal input / output once (not their bound: they are
    fp64-ALU-bound)."""
    cell = Ne * 32 + N * 24
    return {"elem_rhs_ms": cell + N * 4 * s, "elem_hd": cell + N * 4 * s, "elem_rhs_mech": cell + N * 6 * s,
            "elem_sigma": cell + N * 12 * s}


def run(sides, dtypes, reorders, only, reps, tol=1e-8, skip_tol=False, hex_mesh=False, delaunay=False):
    import torch
    from . import binding as cm
    peak = peak_gbs()
    L2 = 126e6
    rows = []
    names = {"none": cm.CM_REORDER_NONE, "morton": cm.CM_REORDER_MORTON, "rcm": cm.CM_REORDER_RCM, "sorted": cm.CM_REORDER_MORTON_SORTED}

    def timeit(fn, n):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        ts = []
        for _ in range(n):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); fn(); e1.record(); torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        return float(np.median(ts))

    for side in sides:
        if delaunay:      # irregular valence: Delaunay tetrahedralisation of a strongly jittered lattice
            L = 2.5e-9 * (side - 1)
            mesh = inputs.delaunay_box((side,) * 3, (L,) * 3, seed_mesh=41, seed_perm=42)
        else:
            mesh = inputs.make_config4_hex_mesh(side) if hex_mesh else inputs.make_config4_mesh(side)
        clamp = inputs.clamp_face_x0(mesh)
        mat = inputs.Material()
        for ro in reorders:
            gm = cm.Mesh(mesh.xyz, mesh.hexes if hex_mesh else mesh.tets, reorder=names[ro])
            lay = gm.layout()
            rp = gm.get(cm.CM_GET_ROWPTR)
            deg = np.diff(rp)
            print(f"{side:4d}^3 N={gm.n_nodes:8d} {ro:7s} layout: nnz/row {deg.mean():.2f} (min {deg.min()}, max {deg.max()}), SELL-16 padding "
                  f"{100 * lay['sell16_padding']:.1f} %, SELL-8 padding {100 * lay['sell8_padding']:.1f} %, "
                  f"{lay['elements_per_chunk']:.0f} elements and {lay['nodes_per_chunk']:.0f} nodes per chunk (capacity {lay['chunk_capacity']}), "
                  f"{lay['slots_per_node']:.2f} slots per node", flush=True)
            for dtype in dtypes:
                gs = cm.System(gm, mat, 1e-12, dtype, clamp, 0)
                td = torch.float64 if dtype == "f64" else torch.float32
                s = 8 if dtype == "f64" else 4
                N, nnz = gm.n_nodes, gm.nnz
                mb = model_bytes(N, nnz, s)
                rng = np.random.default_rng(43)
                b1 = torch.as_tensor(rng.normal(size=N), dtype=td, device="cuda")
                b1[0] = 0
                b3 = torch.as_tensor(rng.normal(size=(N, 3)), dtype=td, device="cuda")
                b3c = b3.clone(); b3c[torch.as_tensor(clamp.reshape(-1, 3).astype(bool), device="cuda")] = 0
                x1, x3 = torch.zeros_like(b1), torch.zeros_like(b3)
                gs.profile_enable(True)

                def kernel_ms(fn, cls, n):
                    """median-free mean of the library's own event timers around the kernel (excludes permutation)"""
                    for _ in range(3):
                        fn()
                    gs.profile_reset()
                    for _ in range(n):
                        fn()
                    p = gs.profile()[cls]
                    return p["ms"] / max(1, p["launches"]), p

                cases = []
                if not only or "spmv_csr1" in only:
                    t, _ = kernel_ms(lambda: gs.spmv(cm.CM_MAT_K_MS, b1), "spmv", reps)
                    cases.append(("spmv_csr1", t, mb["spmv_csr1"], None))
                if not only or "spmv_csr3" in only:
                    t, _ = kernel_ms(lambda: gs.spmv3(cm.CM_MAT_MASS, b3), "spmv", reps)
                    cases.append(("spmv_csr3", t, mb["spmv_csr3"], None))
                if not only or "spmv_bsr3" in only:
                    t, _ = kernel_ms(lambda: gs.spmv(cm.CM_MAT_K_MECH, b3), "spmv", reps)
                    cases.append(("spmv_bsr3", t, mb["spmv_bsr3"], None))
                for name, matid, cls, b, x, key in (("cg_csr1", cm.CM_MAT_K_MS, "cg_ms", b1, x1, "cg_csr1"),
                                                    ("cg_bsr3", cm.CM_MAT_K_MECH, "cg_mech", b3c, x3, "cg_bsr3")):
                    if only and name not in only:
                        continue
                    def f3():
                        x.zero_(); gs.cg_solve(matid, b, x, fixed_iters=3)
                    t, p = kernel_ms(f3, cls, max(3, reps // 2))
                    cases.append((name + "_fixed3", t, 3 * mb[key], 3))
                    if skip_tol:
                        continue
                    its = []
                    def ft():
                        x.zero_(); its.append(gs.cg_solve(matid, b, x, tol=tol, maxiter=200000)[0])
                    t, p = kernel_ms(ft, cls, 2)
                    cases.append((name + "_tol1e-8", t, its[-1] * mb[key], its[-1]))
                eb = elem_bytes(N, gm.n_tets, s) if not hex_mesh else hex_elem_bytes(N, gm.n_tets, s)
                rng44 = np.random.default_rng(44)
                m0 = np.array([1.0, 0.0, 0.0]) + 0.1 * rng44.normal(size=(N, 3))
                m3 = torch.as_tensor(m0 / np.linalg.norm(m0, axis=1, keepdims=True), dtype=td, device="cuda").contiguous()
                # tetrahedra: the default per-pass choice, every pass streaming the stored gradients, every pass recomputing them
                for stored in ((0,) if hex_mesh else (0, 1, 2)):
                    gs.set_option(cm.CM_OPT_STORED_GEOMETRY, stored)
                    for name, rid, kw in (("elem_rhs_ms", cm.CM_RHS_MS, {}), ("elem_hd", cm.CM_OUT_HD, {"U": b1}),
                                          ("elem_rhs_mech", cm.CM_RHS_MECH, {}), ("elem_sigma", cm.CM_OUT_SIGMA, {"u": b3})):
                        if only and name not in only and "elem" not in only:
                            continue
                        t, p = kernel_ms(lambda: gs.field_rhs(rid, m3, **kw), "element", reps)
                        # kernel_ms divides by launches; a pass is 2-3 launches, so take the class total per call
                        cases.append((name + ("", "_stored", "_recomputed")[stored], p["ms"] / reps, eb[name], None))
                gs.set_option(cm.CM_OPT_STORED_GEOMETRY, 0)
                if not only or "cg_csr3" in only:
                    def f33():
                        x3.zero_(); gs.cg_solve3(cm.CM_MAT_K_GS1, b3, x3, fixed_iters=3)
                    t, p = kernel_ms(f33, "cg_gs", max(3, reps // 2))
                    cases.append(("cg_csr3_fixed3", t, 3 * mb["cg_csr3"], 3))
                for name, t, byts, its in cases:
                    gbs = byts / (t * 1e-3) / 1e9
                    resident = (mb["spmv_bsr3" if "bsr" in name else "spmv_csr1"] < L2) and not name.startswith("elem")
                    rows.append({"side": side, "n_nodes": N, "nnz": nnz, "reorder": ro, "dtype": dtype, "kernel": name, "ms": t,
                                 "iters": its, "algorithmic_GBps": gbs, "frac_of_measured_hbm": gbs / peak,
                                 "l2_resident": bool(resident)})
                    print(f"{side:4d}^3 N={N:8d} {ro:7s} {dtype} {name:18s} {t:10.4f} ms  its={its}  {gbs:8.1f} GB/s  "
                          f"{100 * gbs / peak:5.1f}% of {peak:.0f}{'  (L2-resident)' if resident else ''}", flush=True)
                gs.close()
            gm.close()
    return rows


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--sides", default="47,80,100,144")
    ap.add_argument("--dtypes", default="f64,f32")
    ap.add_argument("--reorders", default="none,morton")
    ap.add_argument("--only", default="")
    ap.add_argument("--reps", type=int, default=20)
    ap.add_argument("--json", default="")
    ap.add_argument("--hex", action="store_true", help="linear hexahedral meshes (27 nnz/row; the paper's Fig. 2 workload) instead of tetrahedra")
    ap.add_argument("--delaunay", action="store_true", help="irregular-valence Delaunay meshes (rows of 5-30 entries) instead of Kuhn grids")
    ap.add_argument("--skip-tol", action="store_true", help="skip the CG-to-1e-8 solves (fixed 3 iterations only)")
    a = ap.parse_args(argv)
    rows = run([int(s) for s in a.sides.split(",")], a.dtypes.split(","), a.reorders.split(","),
               set(a.only.split(",")) if a.only else set(), a.reps, skip_tol=a.skip_tol, hex_mesh=a.hex, delaunay=a.delaunay)
    if a.json:
        Path(a.json).write_text(json.dumps(rows, indent=1))


if __name__ == "__main__":
    main(sys.argv[1:])
