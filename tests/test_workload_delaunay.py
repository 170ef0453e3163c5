"""The second, genuinely unstructured workload (shape: the paper's Delaunay mesh of L685): a seeded Delaunay
triangulation with valence 3...12 and a >= 100:1 area ratio, the Triangle-format ingest path for externally generated
meshes, and the oracle's pins on it (uniform flow, conservation)."""
import numpy as np

import oracle
import workloads as wl


def areas(m):
    a, b, c = m.xy[m.tri[:, 0]], m.xy[m.tri[:, 1]], m.xy[m.tri[:, 2]]
    return 0.5 * ((b[:, 0] - a[:, 0]) * (c[:, 1] - a[:, 1]) - (b[:, 1] - a[:, 1]) * (c[:, 0] - a[:, 0]))


def test_delaunay_mesh_is_unstructured_graded_and_seeded():
    m = wl.delaunay_mesh(6000, seed=3)
    a = areas(m)
    assert np.all(a > 0)                                             # counter-clockwise, no degenerate triangle
    val = np.bincount(m.tri.ravel(), minlength=m.nv)
    interior = m.boundary == 0
    assert val[interior].min() >= 3 and 9 <= val[interior].max() <= 14 and np.std(val[interior]) > 0.9
    assert np.percentile(a, 99) / np.percentile(a, 1) > 100.0        # graded: non-uniform V_i
    # the flagged ring is exactly the boundary: edges that belong to one triangle only join flagged vertices
    e = np.sort(np.concatenate([m.tri[:, [0, 1]], m.tri[:, [1, 2]], m.tri[:, [2, 0]]]), axis=1)
    ue, cnt = np.unique(e, axis=0, return_counts=True)
    assert set(np.unique(ue[cnt == 1])) == set(np.nonzero(m.boundary)[0])
    # area of the annular sector r in [1, 10], angle ln(10): (100 - 1) ln(10) / 2, up to the chords of the boundary ring
    assert abs(a.sum() - 0.5 * 99.0 * np.log(10.0)) < 0.02 * a.sum()
    m2 = wl.delaunay_mesh(6000, seed=3)
    assert np.array_equal(m.xy, m2.xy) and np.array_equal(m.tri, m2.tri)
    assert not np.array_equal(wl.delaunay_mesh(6000, seed=4).xy, m.xy)


def test_triangle_file_round_trip(tmp_path):
    m = wl.delaunay_mesh(800, seed=5)
    stem = str(tmp_path / "ext")
    wl.write_triangle_files(m, stem, vertex_flag=m.boundary)
    r, flag = wl.read_triangle_files(stem)
    assert np.array_equal(r.xy, m.xy) and np.array_equal(r.tri, m.tri) and np.array_equal(flag, m.boundary)   # repr() keeps every bit
    # 0-based numbering, comments and a vertex attribute are accepted too
    with open(stem + "0.node", "w") as f:
        f.write("# three points\n3 2 1 1\n0 0.0 0.0 7.5 1\n1 1.0 0.0 7.5 1\n2 0.0 1.0 7.5 0\n")
    with open(stem + "0.ele", "w") as f:
        f.write("1 3 0\n0 0 1 2\n")
    r0, f0 = wl.read_triangle_files(stem + "0")
    assert r0.tri.tolist() == [[0, 1, 2]] and f0.tolist() == [1, 1, 0] and r0.xy[1].tolist() == [1.0, 0.0]


def test_oracle_pins_on_the_delaunay_mesh():
    m = wl.delaunay_mesh(3000, seed=2)
    # uniform flow: every residual exactly zero, state bitwise unchanged (L237) -- any valence, any triangle shape
    for prim in [(1.3, 0.4, -0.7, 2.1), (1.0, 0.0, 0.0, 1.0)]:
        W = wl.uniform_state(m, *prim)
        for scheme, order in [(oracle.SCHEME_B, 2), (oracle.SCHEME_N, 1), (oracle.SCHEME_LDA, 2)]:
            om = oracle.OracleMesh(m.xy, m.tri, vertex_flag=m.boundary, scheme=scheme, time_order=order)
            om.set_state(W)
            om.step(3)
            assert np.array_equal(om.get_state(), W)
    # conservation (L455): a perturbation with compact support in the interior; until it reaches the frozen boundary the
    # totals sum_i V_i W_i do not change, with variable V_i and valence 3...12
    x, y = m.xy[:, 0], m.xy[:, 1]
    xc, yc = x[m.boundary == 0].mean(), y[m.boundary == 0].mean()
    r2 = ((x - xc) ** 2 + (y - yc) ** 2) / 0.6 ** 2
    bump = np.where(r2 < 1.0, np.exp(-1.0 / np.maximum(1.0 - r2, 1e-300)), 0.0)
    W = wl.primitive_to_conserved(1.0 + 0.5 * bump, 0.3 * bump, -0.2 * bump, 1.0 + 0.5 * bump)
    om = oracle.OracleMesh(m.xy, m.tri, vertex_flag=m.boundary)
    om.set_state(W)
    tot0, _, _ = om.diagnostics()
    om.step(2)
    # a step moves information by one ring of triangles per stage: 4 rings of the longest edge in 2 steps
    e = np.concatenate([m.xy[m.tri[:, 1]] - m.xy[m.tri[:, 0]], m.xy[m.tri[:, 2]] - m.xy[m.tri[:, 1]], m.xy[m.tri[:, 0]] - m.xy[m.tri[:, 2]]])
    reach = 0.6 + 4 * np.hypot(e[:, 0], e[:, 1]).max()
    d = np.sqrt((x - xc) ** 2 + (y - yc) ** 2)
    assert (d > reach).sum() > 100 and np.array_equal(om.get_state()[:, d > reach], W[:, d > reach])   # the far field has not moved at all
    om.step(3)
    tot1, mr, mp = om.diagnostics()
    assert np.abs(om.get_state() - W).max() > 1e-3 and mr > 0 and mp > 0
    assert np.abs(tot1 - tot0).max() <= 1e-13 * np.abs(tot0).max()
