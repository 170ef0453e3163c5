"""Timing of the mesh-generation kernels (section 4.1.6: a mesh of 1.3 million vertices):

    python -m paper_1705_02028_b200.meshgen_bench [--cells 1140] [--reps 5] [--out meshgen.json]

Workload: `workloads.scrambled_triangulation(cells, cells)` -- (cells + 1)^2 jittered vertices in a rectangle, 2 cells^2
triangles, a seeded third of the edges flipped away from Delaunay.  Timed, each as the median of
`reps` calls through the C-ABI with CUDA events on the launching stream (the calls allocate their work space and read their
counters back, which is inside the time):

* build_edges       triangleEdges / edgeTriangles from triangleVertices (section 4.1.2)
* delaunay_flip     flips to the Delaunay triangulation (section 2.4.6 / 4.1.5), from the scrambled input every time
* check_only        the same call on the finished triangulation: one pass of the exact INCIRCLE2D over all edges
* test_quality      eq. 2 for every triangle
* find_triangle     the containing triangle of every triangle's circumcentre, walking from that triangle (section 2.4.2)
* refine            Delaunay refinement (section 2.4, 4.1.1) of a 40 x 40-cell start mesh of the same square down to the
                    circumradius bound that gives about as many vertices as the mesh above (B = sqrt 2): the paper's own test of
                    section 4.1.6, "the generation of a uniform unstructured mesh ... with 1.3 million vertices"
* --only fig8       the experiment of Fig. 8: insertion iterations against L / s for random and regular priorities

Prints one JSON line per item with the algorithmic bytes per unit (stated in DESIGN.md section 9c) and the GB/s they amount
to.  Needs a GPU and the built extension; there is no CPU fallback."""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np

# algorithmic bytes per unit: what one pass must read and write at least, gathers counted once per use
BYTES = {
    "build_edges": 12 + 12 + 8,            # per triangle: tv read, te written, 1.5 edges x 8 B of et written (sort traffic not counted)
    "check_only": 8 + 12 + 12 + 4 * 16,    # per edge: et, te of t2, tv of t1, four vertex coordinates
    "test_quality": 12 + 3 * 16 + 8 + 8 + 16 + 1,   # per triangle: tv, three coordinates, r, beta, circumcentre, flag
    "find_triangle": 16 + 4 + 4 + 1,       # per point, plus (12 + 48 + 12 + 8) per triangle visited
}
BYTES_PER_VISIT = 12 + 3 * 16 + 12 + 8


def timed(fn, reps, torch, setup=None):
    ms = []
    out = None
    s = torch.cuda.current_stream()
    for _ in range(reps + 1):                                     # the first call is the warm-up
        if setup:
            setup()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(s)
        out = fn()
        e1.record(s)
        torch.cuda.synchronize()
        ms.append(e0.elapsed_time(e1))
    return float(np.median(ms[1:])), out


def run(cells, reps, out_path, only=None):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("meshgen_bench: no CUDA device")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    if root not in sys.path:
        sys.path.insert(0, root)
    import workloads as wl
    from paper_1705_02028_b200 import binding as b

    m = wl.scrambled_triangulation(cells, cells, seed=1, Lx=2.0, Ly=2.0)
    nt, nv = m.nt, m.nv
    xy = torch.tensor(m.xy, dtype=torch.float64, device="cuda")
    tv0 = torch.tensor(m.tri, dtype=torch.int32, device="cuda")
    rows = []

    def emit(name, ms, units, unit_name, extra=None, bytes_total=None):
        bt = BYTES[name] * units if bytes_total is None else bytes_total
        row = dict(kernel=name, ms=ms, units=units, unit=unit_name, g_units_per_s=units / ms / 1e6,
                   alg_bytes=bt, alg_gbs=bt / ms / 1e6, n_vertices=nv, n_triangles=nt)
        row.update(extra or {})
        rows.append(row)
        print(json.dumps(row), flush=True)

    if only == "refine":
        return refine_part(wl, b, torch, nv, reps, rows, out_path)
    if only == "fig8":
        return fig8_part(wl, b, torch, out_path)
    ms, (te0, et0) = timed(lambda: b.meshgen_build_edges(tv0), reps, torch)
    ne = et0.shape[0]
    emit("build_edges", ms, nt, "triangles", dict(n_edges=ne))

    state = {}

    def fresh():
        state["tv"], state["te"], state["et"] = tv0.clone(), te0.clone(), et0.clone()

    ms, info = timed(lambda: b.meshgen_delaunay_flip(xy, state["tv"], state["te"], state["et"]), reps, torch, setup=fresh)
    row = dict(kernel="delaunay_flip", ms=ms, units=info["flips"], unit="flips", g_units_per_s=info["flips"] / ms / 1e6,
               n_vertices=nv, n_triangles=nt, n_edges=ne, **info)
    rows.append(row)
    print(json.dumps(row), flush=True)
    tv, te, et = state["tv"], state["te"], state["et"]

    ms, info = timed(lambda: b.meshgen_delaunay_flip(xy, tv, te, et), reps, torch)
    assert info["flips"] == 0
    emit("check_only", ms, ne, "edges", dict(exact=info["exact"]))

    ms, q = timed(lambda: b.meshgen_test_quality(xy, tv, 1e9, 1.0), reps, torch)
    emit("test_quality", ms, nt, "triangles", dict(n_bad=q["n_bad"]))

    t0 = torch.arange(nt, dtype=torch.int32, device="cuda")
    ms, (t, code) = timed(lambda: b.meshgen_find_triangle(xy, tv, te, et, q["cc"], t0), reps, torch)
    found = int((t >= 0).sum().item())
    moved = int(((t != t0) & (t >= 0)).sum().item())
    emit("find_triangle", ms, nt, "points", dict(found=found, left_the_mesh=nt - found, not_in_start_triangle=moved),
         bytes_total=BYTES["find_triangle"] * nt + BYTES_PER_VISIT * nt)   # at least the start triangle is visited
    return refine_part(wl, b, torch, nv, reps, rows, out_path)


def fig8_part(wl, b, torch, out_path):
    """Fig. 8 of the paper (L654): the number of insertion iterations against the mesh size L / s (s: the circumradius bound), for
    random priorities and for the regular assignment i(v_n) = n, on a mesh that is Morton-ordered after every insertion step;
    beside the O(log^2(L / s)) of Spielman et al.  Unit square, B = sqrt 2, from a 21 x 21-vertex start mesh."""
    m = wl.scrambled_triangulation(20, 20, seed=1, Lx=1.0, Ly=1.0)
    xy = torch.tensor(m.xy, dtype=torch.float64, device="cuda")
    tv = torch.tensor(m.tri, dtype=torch.int32, device="cuda")
    te, et = b.meshgen_build_edges(tv)
    b.meshgen_delaunay_flip(xy, tv, te, et)
    rows = []
    for R in (0.02, 0.01, 0.005, 0.0025, 0.00125, 0.000625):
        row = dict(R=R, L_over_s=1.0 / R, log2_squared=float(np.log2(1.0 / R) ** 2))
        for name, seed, box in (("random", 7, (0, 0, 1, 1)), ("regular", b.MESHGEN_PRIORITY_REGULAR, (0, 0, 1, 1)), ("random_in_place", 7, None)):
            g = b.meshgen_refine(xy, tv, te, et, R, float(np.sqrt(2.0)), seed=seed, box=box, cap_vertex=4000000, max_iterations=3000)
            row["iterations_" + name], row["vertices_" + name], row["bad_left_" + name] = g[4]["iterations"], int(g[0].shape[0]), g[4]["bad_left"]
        rows.append(row)
        print(json.dumps(row), flush=True)
    if out_path:
        with open(out_path, "w") as f:
            json.dump(rows, f, indent=1)
    return rows


def refine_part(wl, b, torch, nv, reps, rows, out_path):
    # refinement from a coarse mesh of the same square to about nv vertices: vertices ~ 0.69 area / R^2 at B = sqrt 2 (measured)
    c = wl.scrambled_triangulation(40, 40, seed=2, Lx=2.0, Ly=2.0)
    cxy = torch.tensor(c.xy, dtype=torch.float64, device="cuda")
    ctv = torch.tensor(c.tri, dtype=torch.int32, device="cuda")
    cte, cet = b.meshgen_build_edges(ctv)
    b.meshgen_delaunay_flip(cxy, ctv, cte, cet)
    R = float(np.sqrt(0.69 * 4.0 / nv))
    for name, box in (("refine", None), ("refine_morton", (0.0, 0.0, 2.0, 2.0))):
        ms, g = timed(lambda: b.meshgen_refine(cxy, ctv, cte, cet, R, np.sqrt(2.0), seed=1, cap_vertex=int(1.6 * nv), box=box), min(reps, 3), torch)
        row = dict(kernel=name, ms=ms, units=int(g[0].shape[0]) - c.nv, unit="vertices inserted",
                   g_units_per_s=(int(g[0].shape[0]) - c.nv) / ms / 1e6, n_vertices=int(g[0].shape[0]), n_triangles=int(g[1].shape[0]),
                   n_edges=int(g[3].shape[0]), R=R, B=float(np.sqrt(2.0)), start_vertices=c.nv, **g[4])
        rows.append(row)
        print(json.dumps(row), flush=True)
    if out_path:
        with open(out_path, "w") as f:
            json.dump(rows, f, indent=1)
    return rows


def main():
    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("--cells", type=int, default=1140)
    ap.add_argument("--reps", type=int, default=5)
    ap.add_argument("--out", default=None)
    ap.add_argument("--only", default=None, choices=["refine", "fig8"],
                    help="refine: time the refinement alone; fig8: iterations against mesh size for random and regular priorities")
    a = ap.parse_args()
    run(a.cells, a.reps, a.out, a.only)
    return 0


if __name__ == "__main__":
    sys.exit(main())
