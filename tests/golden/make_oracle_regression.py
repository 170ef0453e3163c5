"""Writes tests/golden/oracle_regression.txt: stage-1 residuals of three fixed triangles and a checksum of config 1 after
5 steps, computed by the ORACLE ONLY (never by the CUDA path).  It guards the oracle against accidental edits of its
arithmetic; regenerate only together with a commit that names the paper passage justifying the change.

    python tests/golden/make_oracle_regression.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
import workloads as wl  # noqa: E402

TRIANGLES = [  # (primitive states rho,u,v,p of the 3 vertices, CCW coordinates)
    ([[1.0, 0.3, -0.2, 1.0], [1.1, 0.35, -0.1, 1.2], [0.9, 0.2, -0.25, 0.9]], [[0, 0], [1, 0.1], [0.3, 0.8]]),
    ([[1.0, 2.5, 0.5, 0.4], [0.8, 2.2, 0.7, 0.3], [1.3, 2.8, 0.2, 0.6]], [[0, 0], [0.02, 0.0], [0.0, 0.03]]),       # supersonic
    ([[1.0, 0.0, 0.0, 1.0], [0.125, 0.0, 0.0, 0.1], [1.0, 0.0, 0.0, 1.0]], [[0, 0], [0.1, 0], [0.1, 0.1]]),        # at rest (C8)
]


def main():
    lines = ["# written by tests/golden/make_oracle_regression.py from oracle/ only; %.17g round-trips doubles"]
    for k, (prim, xy) in enumerate(TRIANGLES):
        W = np.array([wl.primitive_to_conserved(*p)[:, None][:, 0] if False else
                      [p[0], p[0] * p[1], p[0] * p[2], 0.5 * p[0] * (p[1] ** 2 + p[2] ** 2) + p[3] / 0.4] for p in prim])
        o = oracle.triangle_stage1(1.4, W, np.array(xy, dtype=float))
        for key in ("phiT", "phiN", "phiLDA", "phiB", "theta"):
            lines.append(f"tri{k}.{key} = " + " ".join("%.17g" % v for v in np.ravel(o[key])))
        lines.append(f"tri{k}.sT = %.17g" % o["sT"])
    cfg = wl.make_config("vortex")
    om = oracle.OracleMesh(cfg.mesh.xy, cfg.mesh.tri, period=cfg.mesh.period)
    om.set_state(cfg.W0)
    n, t, dt = om.step(5)
    W = om.get_state()
    lines.append("vortex32.t5 = %.17g" % t)
    lines.append("vortex32.sum5 = " + " ".join("%.17g" % v for v in W.sum(axis=1)))
    lines.append("vortex32.sumsq5 = " + " ".join("%.17g" % v for v in (W * W).sum(axis=1)))
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_regression.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
