"""Device-resident hysteresis loop (cm_hysteresis_run, one CUDA graph launch) against the same steps driven from the host
through cm_gspm_step, on BASELINE config 1 (81x81x21, anisotropy + Zeeman) and config 0.  Prints steps/s of each.

  python -m paper_2510_09812_b200.hystbench [--steps 200]
"""
from __future__ import annotations

import argparse
import time

import numpy as np

from . import inputs


def main(argv=None):
    import torch
    from . import binding as cm
    ap = argparse.ArgumentParser()
    ap.add_argument("--steps", type=int, default=200)
    a = ap.parse_args(argv)
    for idx in (0, 1):
        cfg = inputs.make_config(idx)
        gm = cm.Mesh(cfg.mesh.xyz, cfg.mesh.tets, cfg.mesh.magnetic, cfg.mesh.elastic_id)
        gs = cm.System(gm, cfg.material, cfg.dt, "f64", cfg.clamp_dof, cfg.pin_node)
        N = gm.n_nodes
        H = [float(h) for h in cfg.Hext[0]]
        if not any(H):
            H = [1e4, 0.0, 0.0]
        terms = cfg.terms | inputs.TERM_ZEEMAN

        def fresh():
            return (torch.as_tensor(cfg.m0, dtype=torch.float64, device="cuda").contiguous(),
                    torch.zeros(N, dtype=torch.float64, device="cuda"), torch.zeros((N, 3), dtype=torch.float64, device="cuda"))

        p = cm.make_params(cfg.dt, H, terms, 0, 1e-7)
        rows = []
        for name in ("host loop, info read back every step", "host loop, no read-back", "device loop (CUDA graph, WHILE node)"):
            m, U, u = fresh()
            for _ in range(3):
                gs.gspm_step(p, m, U, u)
            m, U, u = fresh()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            if name.startswith("device"):
                _, _, sl, res, _ = gs.hysteresis_run(p, m, U, u, H, [0, 0, 0], conv_tol=0.0, max_fields=1, max_steps=a.steps)
                assert res.total_steps == a.steps
            else:
                for _ in range(a.steps):
                    gs.gspm_step(p, m, U, u, want_info=name.endswith("every step"))
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            rows.append((name, a.steps / dt, float(m.double().sum())))
        print(f"config {idx}: {N} nodes, {a.steps} steps at fixed field {H}")
        for name, sps, chk in rows:
            print(f"  {name:42s} {sps:10.1f} steps/s   checksum {chk:.12e}")
        gs.close(); gm.close()


if __name__ == "__main__":
    main()
