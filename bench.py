#!/usr/bin/env python
"""bench.py -- GSPM time steps/s at the 3M-node mesh (BASELINE.json config 3), one replica per GPU.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--dtype f64|f32] [--impl ours|reference]

A "step" is one cm_gspm_step: the whole hot path (volume average, magnetostatic RHS + CG, gradient recovery,
mechanical RHS + CG, stress recovery, field, 8 Helmholtz CG solves, Gauss-Seidel update, projection) on the
synthetic 245x245x50-node magnetoelastic mesh with an ellipsoidal inclusion, fp64, CG tolerance 1e-7,
field sweep of config 3.  The path does not shard ("replicas only"): with N > 1 every rank steps its own
replica, no collective on the data path; value = replicas * steps / max-over-ranks time.

Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle (oracle/) on a bounded sample instead.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

from paper_2510_09812_b200 import inputs  # noqa: E402

NM = 1e-9
METRIC = "gspm_time_steps_per_s_3M_nodes"
UNIT = "steps/s"
CG_TOL = 1e-7           # the paper's CG tolerance
FULL_GRID = (245, 245, 50)
SAMPLE_GRID, SAMPLE_BOX = (62, 62, 50), (250 * NM, 250 * NM, 200 * NM)   # same spacing, 1/16 of the area


def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, index: int):
        self.index, self.rows, self.stop = index, [], threading.Event()
        self.t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        while not self.stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-i", str(self.index)],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([c.strip() for c in out.split(",")])
            except Exception:
                pass
            self.stop.wait(0.2)

    def __enter__(self):
        self.t.start()
        return self

    def __exit__(self, *a):
        self.stop.set()
        self.t.join(timeout=6)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        sm = sorted(int(r[0]) for r in self.rows if r[0].isdigit())
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(len(r) > 2 + k and r[2 + k].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": int(self.rows[0][1]) if self.rows[0][1].isdigit() else None,
                "reasons": reasons, "samples": len(self.rows)}


def sample_config():
    return inputs.make_config(3, grid=SAMPLE_GRID, box=SAMPLE_BOX)


def time_oracle(steps: int, warmup: int, variant: int = 0, full_mesh: bool = False, maxiter: int = 100000):
    """The oracle as it stands, on the box's host cores, on a bounded sample of config 3.  Default sample: a sub-box at
    the same spacing / physics / tolerance, `warmup` untimed steps first (warm starts of U and u as on the GPU side),
    steps/s scaled to the 3M-node mesh by node count.  full_mesh: config 3 ITSELF with every solve capped at `maxiter`
    iterations (the truncation is part of the sample's description).  Returns a dict."""
    import oracle
    cfg = inputs.make_config(3) if full_mesh else sample_config()
    t_setup = time.perf_counter()
    o = oracle.Oracle(cfg.mesh, cfg.material, cfg.dt, clamp_dof=cfg.clamp_dof)
    t_setup = time.perf_counter() - t_setup
    m = cfg.m0.copy(); U = np.zeros(o.N); u = np.zeros((o.N, 3))
    its = []
    t0 = time.perf_counter()
    for k in range(warmup + steps):
        if k == warmup:
            t0 = time.perf_counter()
        info, rc = o.gspm_step(m, U, u, cfg.dt, cfg.Hext[k % cfg.steps], cfg.terms, variant=variant, cg_tol=CG_TOL, cg_maxiter=maxiter)
        its.append((info.it_ms, info.it_mech, int(sum(info.it_gs))))
    dt = time.perf_counter() - t0
    n_full = FULL_GRID[0] * FULL_GRID[1] * FULL_GRID[2]
    scale = o.N / n_full
    cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    cpu_model = "unknown"
    try:
        for ln in Path("/proc/cpuinfo").read_text().splitlines():
            if ln.startswith("model name"):
                cpu_model = ln.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    timed = its[warmup:]
    n_it = sum(a + b + c for a, b, c in timed)
    where = (f"config 3 itself ({o.N} nodes), every CG solve capped at {maxiter} iterations" if full_mesh else
             f"a {SAMPLE_GRID[0]}x{SAMPLE_GRID[1]}x{SAMPLE_GRID[2]}-node sub-box of config 3 ({o.N} nodes, same spacing/physics); "
             f"steps/s multiplied by {o.N}/{n_full} (node count)")
    desc = (f"{steps} GSPM step(s) after {warmup} warm-up step(s), gspm_variant {variant}, tol {CG_TOL:g}, on {where}; "
            f"CG its per timed step (ms, mech, sum gs) {timed}")
    return {"value": steps / dt * scale, "sec_per_step": dt / steps, "desc": desc, "cores": cores, "cg_iters_per_step": timed,
            "ms_per_cg_iteration_all_solves": 1e3 * dt / max(1, n_it), "nodes": o.N, "setup_s": t_setup, "cpu_model": cpu_model,
            "omp_num_threads": os.environ.get("OMP_NUM_THREADS", f"unset (OpenMP default: {os.cpu_count()} logical CPUs)")}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    r = time_oracle(args.steps, args.warmup, args.variant, args.full_mesh, args.oracle_maxiter)
    cb = {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["desc"],
          "cg_iters_per_step": r["cg_iters_per_step"], "ms_per_cg_iteration_all_solves": r["ms_per_cg_iteration_all_solves"],
          "setup_s": r["setup_s"], "cpu_model": r["cpu_model"], "omp_num_threads": r["omp_num_threads"]}
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": r["sec_per_step"] * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "config3_paper_scale (bounded CPU sample)", "sample": r["desc"], "gspm_variant": args.variant},
            "cpu_baseline": cb,
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def algorithmic_bytes(N, nnz, s):
    """Bytes per matrix pass, s = bytes per value.  `*_iter_*`: SURVEY 8(d)'s per-unit figures for one CG iteration
    (SpMV with its x read and y write + 10 vector words per DOF; the figure `roofline.achieved` uses).  `*_streams_*`: what
    the kernel actually streams per iteration -- p, Ap of the product are among the 10 words, so 8 more on top of the
    SpMV (x, r, p_old read, x, p written in phase C'; Ap, r read, r written in phase B; p gathered, Ap written by the
    product) -- reported beside it.  `*_r0_*`: the r0 = b - A x0 pass of a launch (product + b, Ap read, r written).
    The three-right-hand-side solver keeps p padded to four words per node (one 32 B / 16 B gather per nonzero)."""
    spmv_csr = nnz * (s + 4) + N * (4 + s + s)
    spmv_bsr = nnz * (9 * s + 4) + N * (4 + 3 * s + 3 * s)
    spmv_csr3 = nnz * (s + 4) + N * 4 + 2 * 3 * N * s
    return {
        "cg_iter_csr1": spmv_csr + 10 * N * s,                  # SURVEY: 277 B/row fp64
        "cg_iter_bsr3": spmv_bsr + 10 * 3 * N * s,              # SURVEY: 1415 B/node fp64
        "cg_iter_csr3": spmv_csr3 + 10 * 3 * N * s,             # 3-RHS: matrix read once per iteration
        "cg_streams_csr1": spmv_csr + 8 * N * s,
        "cg_streams_bsr3": spmv_bsr + 8 * 3 * N * s,
        "cg_streams_csr3": nnz * (s + 4) + N * 4 + N * s * (4 + 3) + N * s * (3 + 3 + 4 + 3 + 4 + 3 + 3 + 3),
        "cg_r0_csr1": spmv_csr + 3 * N * s,
        "cg_r0_bsr3": spmv_bsr + 3 * 3 * N * s,
        "cg_r0_csr3": nnz * (2 * s + 4) + N * 4 + N * s * (4 + 4 + 3 + 3),   # Helmholtz start: K^GS and M_m streamed together, f4 gathered and read, r0 and x0 written
        "spmv_csr3": spmv_csr3,
    }


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2510_09812_b200 import binding as cm, replicas

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    dtype = args.dtype

    grid = tuple(int(g) for g in args.grid.split("x")) if args.grid else None
    cfg = inputs.make_config(3, grid=grid)
    t_setup = time.perf_counter()
    mesh = cm.Mesh(cfg.mesh.xyz, cfg.mesh.tets, cfg.mesh.magnetic, cfg.mesh.elastic_id, cm.CM_REORDER_MORTON)
    sysm = cm.System(mesh, cfg.material, cfg.dt, dtype, cfg.clamp_dof, cfg.pin_node)
    if args.no_fuse_s5s8:
        sysm.set_option(cm.CM_OPT_NO_FUSED_S5S8, 1)
    torch.cuda.synchronize()
    t_setup = time.perf_counter() - t_setup
    N, nnz = mesh.n_nodes, mesh.nnz
    peak, peak_src = measured_peaks()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def timed_run(system, dt_name, steps, warmup, variant, fixed, precond, matfree=0):
        """W untimed + K timed cm_gspm_step calls from the config's initial state; CUDA events on the launching stream."""
        td = torch.float64 if dt_name == "f64" else torch.float32
        m = torch.as_tensor(cfg.m0, dtype=td, device=dev).contiguous()
        U = torch.zeros(N, dtype=td, device=dev)
        u = torch.zeros((N, 3), dtype=td, device=dev)

        def params(k):
            return cm.make_params(cfg.dt, cfg.Hext[k % cfg.steps], cfg.terms, variant, CG_TOL, 100000, fixed, precond, matfree)

        k = 0
        for _ in range(warmup):
            system.gspm_step(params(k), m, U, u); k += 1
        system.profile_enable(True)
        system.profile_reset()
        infos = []
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        with ClockSampler(local) as clocks:
            ev0.record()
            for _ in range(steps):
                info, rc = system.gspm_step(params(k), m, U, u); k += 1
                infos.append(info)
            ev1.record()
            barrier()
        ms = ev0.elapsed_time(ev1)
        prof = system.profile()
        system.profile_enable(False)
        _, ms, value = replicas.aggregate(steps, ms, dist if world > 1 else None, dev)
        return {"value": value, "ms_total": ms, "prof": prof, "infos": infos, "clocks": clocks.summary(), "state": (m, U, u),
                "params": params, "k": k}

    def kernel_table(prof, steps, s):
        """Per kernel class: device time, launches, algorithmic GB/s (SURVEY 8d figures) and fraction of the measured peak."""
        ab = algorithmic_bytes(N, nnz, s)
        out = {}
        for name, key in (("cg_mech", "bsr3"), ("cg_ms", "csr1"), ("cg_gs", "csr3")):
            p = prof[name]
            if p["ms"] > 0 and p["cg_matrix_passes"] > 0:
                iters = p["cg_matrix_passes"] - p["launches"]        # every launch makes one r0 pass
                byts = ab["cg_iter_" + key] * iters + ab["cg_r0_" + key] * p["launches"]
                streamed = ab["cg_streams_" + key] * iters + ab["cg_r0_" + key] * p["launches"]
                gbs = byts / (p["ms"] * 1e-3) / 1e9
                out[name] = {"ms": p["ms"], "launches": p["launches"], "matrix_passes": p["cg_matrix_passes"], "iterations": iters,
                             "algorithmic_GBps": gbs, "frac_of_measured_peak": gbs / peak, "frac_of_spec_8000": gbs / 8000.0,
                             "streamed_GBps": streamed / (p["ms"] * 1e-3) / 1e9}
        for name in ("spmv", "element", "pointwise"):
            out[name] = {"ms": prof[name]["ms"], "launches": prof[name]["launches"]}
        # assembly.  The step launches FOUR chunk passes when S5 shares S8's pass (demag + mechanics on tetrahedra, the default):
        # S3, S6, S5+S8 at m^n, S8 at m*; five otherwise.  Two numerators, both printed ("report which numerator is used"):
        #  algorithmic_GBps -- SURVEY 8(d)'s stored-gradient figure for the passes that RAN: per tetrahedron 16 B connectivity +
        #                      13 words, nodal inputs and outputs once (38 words per node and step);
        #  streamed_GBps    -- the bytes of the variant that ran: a pass that recomputes its geometry (fp64 S3; fp64 S5 only when it
        #                      runs unfused) reads 3 words per tetrahedron plus its chunk's slot coordinates (24 B per slot)
        #                      instead of the ten stored geometry words.
        fused = mesh.nen == 4 and not args.no_fuse_s5s8
        n_pass = 4 if fused else 5
        n_recompute = (1 if fused else 2) if s == 8 else 0
        nodal = N * s * (4 + 4 + 6 + 2 * 12)
        elem_step = n_pass * mesh.n_tets * (16 + 13 * s) + nodal
        elem_streamed = ((n_pass - n_recompute) * mesh.n_tets * (16 + 13 * s) + n_recompute * (mesh.n_tets * (16 + 3 * s) + n_slots * 24)
                         + nodal)
        if out["element"]["ms"] > 0:
            gbs = elem_step * steps / (out["element"]["ms"] * 1e-3) / 1e9
            gbs_s = elem_streamed * steps / (out["element"]["ms"] * 1e-3) / 1e9
            out["element"].update({"algorithmic_GBps": gbs, "frac_of_measured_peak": gbs / peak, "frac_of_spec_8000": gbs / 8000.0,
                                   "streamed_GBps": gbs_s, "streamed_frac_of_measured_peak": gbs_s / peak,
                                   "chunk_passes_per_step": n_pass, "passes_recomputing_geometry": n_recompute,
                                   "numerator": "frac_of_measured_peak: SURVEY 8(d) stored-gradient bytes of the chunk passes that ran "
                                                "(S5 fused into S8's pass counts once); streamed_*: bytes of the variant that ran "
                                                "(recomputed-geometry passes read coordinates, not gradients); the class time also "
                                                "holds the node passes"})
        return out, ab

    s = 8 if dtype == "f64" else 4
    n_slots = int(round(mesh.layout()["slots_per_node"] * N))
    main = timed_run(sysm, dtype, args.steps, args.warmup, args.variant, args.fixed_iters, args.precond)
    ms_total, value, prof, infos = main["ms_total"], main["value"], main["prof"], main["infos"]

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region, all --steps
    m, U, u = main["state"]
    mh = m.cpu().pin_memory(); Uh = U.cpu().pin_memory(); uh = u.cpu().pin_memory()
    k = main["k"]
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        sysm.gspm_step_host(main["params"](k), mh, Uh, uh); k += 1
    torch.cuda.synchronize()
    _, _, e2e_value = replicas.aggregate(args.steps, (time.perf_counter() - t0) * 1e3, dist if world > 1 else None, dev)
    io_bytes = 7 * N * s
    del m, U, u, mh, Uh, uh

    # ---- variants SURVEY 8(d) asks for beside steps/s (each its own W + K steps from the initial state, same mesh):
    # every solve cut at 3 iterations (the paper's regime for the Helmholtz solves), fp32 (north_star (4)),
    # Jacobi-preconditioned CG and the matrix-free mechanical operator (the paper's future work), and the other
    # reading of Alg. B.1 Step 2 (R1)
    variants = {}
    if not args.no_variants:
        vs = max(1, min(args.steps, args.variant_steps))

        def brief(r, extra=None):
            d = {"value": r["value"], "unit": UNIT, "ms_per_step": r["ms_total"] / len(r["infos"]), "steps": len(r["infos"]),
                 "cg_iters_per_step": [[i.it_ms, i.it_mech, int(sum(i.it_gs))] for i in r["infos"]],
                 "mean_dm_last_step": float(r["infos"][-1].mean_dm)}
            d.update(extra or {})
            return d

        r = timed_run(sysm, dtype, vs, args.warmup, args.variant, 3, args.precond)
        kt, _ = kernel_table(r["prof"], vs, s)
        variants["fixed3"] = brief(r, {"kernels": {n: {q: v[q] for q in ("ms", "frac_of_measured_peak") if q in v} for n, v in kt.items()}})
        r = timed_run(sysm, dtype, vs, args.warmup, args.variant, args.fixed_iters, 1 - args.precond)
        variants["jacobi" if args.precond == 0 else "plain_cg"] = brief(r)
        r = timed_run(sysm, dtype, vs, args.warmup, args.variant, args.fixed_iters, args.precond, matfree=1)
        pm = r["prof"]["cg_mech"]
        variants["mech_matfree"] = brief(r, {"cg_mech_ms_per_matrix_pass": pm["ms"] / max(1, pm["cg_matrix_passes"]),
                                            "stored_matrix_ms_per_matrix_pass": prof["cg_mech"]["ms"] / max(1, prof["cg_mech"]["cg_matrix_passes"])})
        r = timed_run(sysm, dtype, vs, args.warmup, 1 - args.variant, args.fixed_iters, args.precond)
        variants[f"gspm_variant{1 - args.variant}"] = brief(r)
        other = "f32" if dtype == "f64" else "f64"
        sys2 = cm.System(mesh, cfg.material, cfg.dt, other, cfg.clamp_dof, cfg.pin_node)
        r = timed_run(sys2, other, vs, args.warmup, args.variant, args.fixed_iters, args.precond)
        kt, _ = kernel_table(r["prof"], vs, 12 - s)
        variants[other] = brief(r, {"kernels": {n: {q: v[q] for q in ("ms", "frac_of_measured_peak") if q in v} for n, v in kt.items()}})
        sys2.close()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (by accumulated device time)
    per_class, ab = kernel_table(prof, args.steps, s)
    dom = max(("cg_mech", "cg_ms", "cg_gs"), key=lambda n: prof[n]["ms"])
    key = {"cg_mech": "bsr3", "cg_ms": "csr1", "cg_gs": "csr3"}[dom]
    # DRAM bytes per matrix pass measured by `ncu --set full` on config 3 (21 passes per launch), read from the committed
    # profiles/ncu_constants.json (each entry names the capture it comes from), EXTRAPOLATED to the average launch of this run,
    # like `achieved`.  Only known for the captured workload.
    ncu_const = json.loads((ROOT / "profiles" / "ncu_constants.json").read_text())
    ncu_bytes_per_pass = {(k.split("/")[0], k.split("/")[1]): v["dram_bytes"] / v["matrix_passes"] for k, v in ncu_const["cg"].items()}
    ncu_source = {(k.split("/")[0], k.split("/")[1]): v["source"] for k, v in ncu_const["cg"].items()}
    traffic = None
    passes_per_launch = prof[dom]["cg_matrix_passes"] / max(1, prof[dom]["launches"])
    if (dom, dtype) in ncu_bytes_per_pass and not args.grid:
        traffic = ncu_bytes_per_pass[(dom, dtype)] * passes_per_launch
    roof = {"bound": "hbm", "kernel": f"cg_kernel<{dtype},{dom}> (persistent cooperative CG solve)",
            "achieved": per_class.get(dom, {}).get("algorithmic_GBps"), "peak": peak, "unit": "GB/s",
            "frac": per_class.get(dom, {}).get("frac_of_measured_peak"), "traffic": traffic, "peak_source": peak_src,
            "share_of_step": prof[dom]["ms"] / ms_total,
            "algorithmic_bytes_per_iteration": ab["cg_iter_" + key], "streamed_bytes_per_iteration": ab["cg_streams_" + key],
            "bytes_r0_pass": ab["cg_r0_" + key], "matrix_passes_per_launch": passes_per_launch,
            "achieved_streamed": per_class.get(dom, {}).get("streamed_GBps"),
            "traffic_source": ("extrapolated: ncu --set full dram__bytes_read+write per matrix pass of a 21-pass capture ("
                               + ncu_source.get((dom, dtype), "none") + ") x matrix passes per launch of this run")}

    launches = sum(p["launches"] for p in prof.values())
    last = infos[-1]
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": dtype, "data": "synthetic",
            "config": {"workload": "config3_paper_scale", "grid": "x".join(map(str, cfg.mesh.grid)), "n_nodes": N,
                       "n_tets": mesh.n_tets, "nnz": nnz, "dt_ps": cfg.dt * 1e12, "cg_tol": CG_TOL, "cg_fixed_iters": args.fixed_iters,
                       "cg_precond": args.precond,
                       "terms": "exchange+anis+zeeman+demag+farfield+magel", "parallelism": f"replicas x{world}",
                       "l2": "inputs larger than L2 (matrices 3.2 GB fp64 per solve)", "setup_s": t_setup,
                       "gspm_variant": args.variant,
                       "cg_iters_last_step": {"ms": last.it_ms, "mech": last.it_mech, "gs": list(last.it_gs)},
                       "cg_iters_per_step": [[i.it_ms, i.it_mech, int(sum(i.it_gs))] for i in infos],
                       "mean_dm_per_step": [float(i.mean_dm) for i in infos]},
            "clocks": main["clocks"],
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": io_bytes, "d2h_bytes_per_step": io_bytes,
                    "steps": args.steps},
            "gpu_launches": launches, "roofline": roof, "kernels": per_class, "variants": variants}
    if world == 1 and not args.no_cpu_baseline:
        r = time_oracle(2, 1, args.variant)
        line["cpu_baseline"] = {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["desc"],
                                "cg_iters_per_step": r["cg_iters_per_step"],
                                "ms_per_cg_iteration_all_solves": r["ms_per_cg_iteration_all_solves"],
                                "cpu_model": r["cpu_model"], "omp_num_threads": r["omp_num_threads"]}
        if not args.no_cpu_full_mesh and not args.grid:
            # like for like: the oracle on config 3 ITSELF, one step with every solve capped at 40 iterations (a bounded sample:
            # ~1 min of set-up + ~20 s of solves), against the GPU's time per matrix pass of the dominant solve on the same mesh
            rf = time_oracle(1, 0, args.variant, full_mesh=True, maxiter=40)
            gpu_ms_pass = prof["cg_mech"]["ms"] / max(1, prof["cg_mech"]["cg_matrix_passes"])
            line["cpu_baseline"].update({"full_mesh_ms_per_cg_iteration": rf["ms_per_cg_iteration_all_solves"],
                                         "full_mesh_sample": rf["desc"], "full_mesh_setup_s": rf["setup_s"],
                                         "gpu_ms_per_matrix_pass_cg_mech": gpu_ms_pass,
                                         "gpu_ms_per_cg_iteration_all_solves": (prof["cg_mech"]["ms"] + prof["cg_ms"]["ms"] + prof["cg_gs"]["ms"])
                                                                               / max(1, sum(a + b + c for a, b, c in line["config"]["cg_iters_per_step"]))})
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=4)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--fixed-iters", type=int, default=-1, help="run every CG solve for exactly this many iterations")
    ap.add_argument("--variant", type=int, default=0, choices=[0, 1], help="Alg. B.1 Step 2: 0 as printed (P:438), 1 fully Gauss-Seidel (R1)")
    ap.add_argument("--precond", type=int, default=0, choices=[0, 1], help="CG preconditioner: 0 none (the paper's), 1 Jacobi (P:355)")
    ap.add_argument("--no-variants", action="store_true", help="skip the fixed3 / f32 / jacobi / other-variant re-runs")
    ap.add_argument("--variant-steps", type=int, default=4, help="timed steps of each variant re-run")
    ap.add_argument("--full-mesh", action="store_true", help="--impl reference: time the oracle on config 3 itself (capped solves)")
    ap.add_argument("--oracle-maxiter", type=int, default=100000, help="--impl reference: cap of every CG solve")
    ap.add_argument("--grid", default="", help="override the node grid, e.g. 81x81x21 (not the headline workload)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-fuse-s5s8", action="store_true", help="run S5 and S8 as separate element passes (CM_OPT_NO_FUSED_S5S8)")
    ap.add_argument("--no-cpu-full-mesh", action="store_true", help="skip the like-for-like oracle leg on config 3 itself (about 80 s)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
