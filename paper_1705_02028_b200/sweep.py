"""Config 5 of BASELINE.json as a sweep (the table of BASELINE.md section 6):

    python -m paper_1705_02028_b200.sweep [--sizes 256 512 1024 2048 4096] [--steps 100] [--reps 5] [--out sweep.json]

For every size: Morton input numbering (reorder on) and a seeded random permutation of the numbering with the layout
stage's reordering off and on, each in fp64 and fp32; scheme B, RK2, CFL 0.5 on the isentropic vortex (the paper's
figure-of-merit workload, scaled; recipe in DESIGN.md section 4).  Prints one JSON line per run:
median over `reps` repetitions of `steps` steps (CUDA events on the launching stream, after 5 warm-up steps), the time
of the one-off layout stage (mrd_mesh_create, upload included) and the device memory of the mesh.
Needs a GPU and the built extension; there is no CPU fallback."""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

import numpy as np


def run(sizes, steps, reps, out):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("sweep: no CUDA device")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    if root not in sys.path:
        sys.path.insert(0, root)
    import workloads as wl
    import paper_1705_02028_b200 as mrd

    rows = []
    stream = torch.cuda.current_stream()
    for n in sizes:
        for numbering in ("morton", "permuted"):
            cfg = wl.make_config("sweep", n=n, numbering=numbering)
            for prec in ("fp64", "fp32"):
                for reorder in ((1,) if numbering == "morton" else (0, 1)):
                    t0 = time.perf_counter()
                    gm = mrd.Mesh(cfg.mesh.xy, cfg.mesh.tri, period=cfg.mesh.period, reorder=bool(reorder), gamma=cfg.gamma,
                                  cfl=cfg.cfl, scheme=cfg.scheme, time_order=cfg.time_order,
                                  precision=mrd.FP64 if prec == "fp64" else mrd.FP32)
                    layout_s = time.perf_counter() - t0
                    gm.set_state(torch.tensor(cfg.W0, device="cuda", dtype=torch.float64 if prec == "fp64" else torch.float32))
                    gm.step(5)
                    k = steps if n < 4096 else max(1, steps * 2 // 5)
                    ms = []
                    for _ in range(reps):
                        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        e0.record(stream)
                        gm.step_async(k)
                        e1.record(stream)
                        torch.cuda.synchronize()
                        ms.append(e0.elapsed_time(e1) / k)
                    gm.sync()
                    m = float(np.median(ms))
                    row = dict(N=n, triangles=cfg.mesh.nt, precision=prec, numbering=numbering, reorder=reorder, steps=k, reps=reps,
                               ms_per_step=m, g_triangle_updates_per_s=cfg.mesh.nt / m / 1e6, g_vertex_updates_per_s=cfg.mesh.nv / m / 1e6,
                               layout_s=layout_s, device_gb=gm.device_bytes() / 1e9)
                    rows.append(row)
                    print(json.dumps(row), flush=True)
                    del gm
                    torch.cuda.empty_cache()
    if out:
        with open(out, "w") as f:
            json.dump(rows, f, indent=1)
    return rows


def main():
    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("--sizes", type=int, nargs="+", default=[256, 512, 1024, 2048, 4096])
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--reps", type=int, default=5)
    ap.add_argument("--out", default=None)
    a = ap.parse_args()
    run(a.sizes, a.steps, a.reps, a.out)
    return 0


if __name__ == "__main__":
    sys.exit(main())
