"""Pins of the oracle's mesh data structure (section 4.1.2), Delaunay triangulator (section 2.4.6 / 4.1.5) and point location
(section 2.4.2) -- oracle/meshgen.py -- against what the paper and elementary geometry fix: the Delaunay triangulation of points
in general position is unique (L96), so a library triangulation of the same points must be the same set of triangles; empty
circumcircles by brute force; Lawson's angle criterion; every flip raises the smallest angle of its quadrilateral (L108);
cocircular points are left alone; the containing triangle of a point by exhaustive search."""
import numpy as np
import pytest

import workloads as wl
from oracle import meshgen as mg


def scrambled(nx, ny, seed):
    m = wl.scrambled_triangulation(nx, ny, seed)
    return m.xy, m.tri.astype(np.int32)


def angles(xy, tri):
    p = xy[tri]
    out = []
    for k in range(3):
        u, v = p[:, (k + 1) % 3] - p[:, k], p[:, (k + 2) % 3] - p[:, k]
        out.append(np.arccos(np.clip((u * v).sum(1) / np.hypot(*u.T) / np.hypot(*v.T), -1, 1)))
    return np.stack(out, axis=1)


def assert_structure(xy, tv, te, et):
    """te / et describe tv: edge k of a triangle joins its vertices k+1 and k+2, both neighbours of an edge hold its endpoints,
    every triangle is counter-clockwise."""
    for t in range(tv.shape[0]):
        assert mg.orient2d(*xy[tv[t]]) == 1
        for k in range(3):
            e = te[t, k]
            assert t in et[e]
            ends = {int(tv[t, (k + 1) % 3]), int(tv[t, (k + 2) % 3])}
            for t2 in et[e]:
                if t2 >= 0:
                    assert ends <= set(int(v) for v in tv[t2]) and e in te[t2]
    assert (et[:, 0] >= 0).all()


@pytest.mark.parametrize("shape,Lx,Ly,seed", [((36, 48), 100.0, 64.0, 778), ((3, 59), 1.0, 64.0, 5), ((200, 200), 2.0, 2.0, 3)])
def test_the_workload_is_a_valid_triangulation_at_the_largest_allowed_jitter(shape, Lx, Ly, seed):
    # the input recipe of DESIGN.md 9c: every triangle counter-clockwise (exact test), the areas add up to the rectangle; the first
    # case is one that a jitter of 0.3 cell widths turns over, which is why the generator stops at 0.25
    m = wl.scrambled_triangulation(*shape, seed=seed, amplitude=0.25, Lx=Lx, Ly=Ly)
    p = m.xy[m.tri]
    area = 0.5 * ((p[:, 1, 0] - p[:, 0, 0]) * (p[:, 2, 1] - p[:, 0, 1]) - (p[:, 1, 1] - p[:, 0, 1]) * (p[:, 2, 0] - p[:, 0, 0]))
    assert (area > 0).all() and abs(area.sum() - Lx * Ly) < 1e-9 * Lx * Ly
    worst = np.argsort(area)[:50]
    assert all(mg.orient2d(*m.xy[m.tri[t]]) == 1 for t in worst)
    with pytest.raises(ValueError, match="0.25"):
        wl.scrambled_triangulation(*shape, seed=seed, amplitude=0.3, Lx=Lx, Ly=Ly)


def test_build_edges_follows_the_stated_conventions():
    m = wl.uniform_mesh(7, 5, 1.0, 1.0, periodic=False)
    tv = m.tri.astype(np.int32)
    te, et = mg.build_edges(tv)
    assert et.shape[0] == m.nt + m.nv - 1                         # Euler: V - E + T = 1 for a triangulated disc
    assert (et[:, 1] < 0).sum() == 2 * 7 + 2 * 5                  # the boundary edges of the rectangle of 7 x 5 cells
    assert_structure(m.xy, tv, te, et)
    ends = np.array([sorted((tv[t, (k + 1) % 3], tv[t, (k + 2) % 3])) for e in range(et.shape[0])
                     for t in [et[e, 0]] for k in [list(te[t]).index(e)]])
    assert (np.lexsort((ends[:, 1], ends[:, 0])) == np.arange(len(ends))).all()    # numbered by (smaller, larger) vertex
    assert ((et[:, 1] < 0) | (et[:, 0] < et[:, 1])).all()
    with pytest.raises(ValueError):
        mg.build_edges(np.array([[0, 1, 2], [0, 1, 3], [1, 0, 4]], dtype=np.int32))   # an edge with three triangles


def test_check_edge_is_lawsons_angle_criterion():
    """An edge is locally Delaunay iff the two angles opposite to it add up to at most pi (textbook form of the empty circle)."""
    rng = np.random.default_rng(3)
    n = 0
    while n < 300:
        p = rng.random((4, 2))
        a, b, c, d = p
        if mg.orient2d(a, b, c) <= 0 or mg.orient2d(d, c, b) <= 0:
            continue
        tv = np.array([[0, 1, 2], [3, 2, 1]], dtype=np.int32)    # share the edge (b, c)
        te, et = mg.build_edges(tv)
        e = int(te[0, 0])
        ang = angles(p, tv)
        s = ang[0, 0] + ang[1, 0]
        if abs(s - np.pi) < 1e-9:
            continue
        assert mg.check_edge(p, tv, te, et, e) == (s > np.pi)
        n += 1


def test_flip_edge_of_the_quadrilateral_of_fig_4():
    xy = np.array([[0.0, 0.0], [1.0, -0.2], [1.0, 1.2], [1.3, 0.5]])  # a, b, c, d with a long shared edge (b, c)
    tv = np.array([[0, 1, 2], [3, 2, 1]], dtype=np.int32)
    te, et = mg.build_edges(tv)
    e = int(te[0, 0])
    assert mg.check_edge(xy, tv, te, et, e)                       # circle through a, b, c: centre (0.62, 0.5), radius 0.797; d is 0.68 from it
    mg.flip_edge(tv, te, et, e)
    assert mg.triangle_set(tv) == {(0, 1, 3), (0, 3, 2)}          # E' joins a and d (L102)
    assert_structure(xy, tv, te, et)
    assert not mg.check_edge(xy, tv, te, et, e)                   # "if E is not locally Delaunay, E' would be" (L102)
    assert sorted(et[e]) == [0, 1]


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_delaunay_flip_reaches_the_unique_delaunay_triangulation(seed):
    from scipy.spatial import Delaunay
    xy, tv = scrambled(14, 11, seed)
    for t in tv:
        assert mg.orient2d(*xy[t]) == 1                           # the input is a valid triangulation
    out, te, et, flips = mg.delaunay_flip(xy, tv)
    assert flips > 50
    lib = Delaunay(xy).simplices
    cw = np.array([mg.orient2d(*xy[s]) for s in lib]) < 0
    lib[cw] = lib[cw][:, [0, 2, 1]]
    assert mg.triangle_set(out) == mg.triangle_set(lib)
    assert mg.triangle_set(out) != mg.triangle_set(tv)
    assert_structure(xy, out, te, et)
    te0, et0 = mg.build_edges(tv)
    assert et.shape == et0.shape and (et[:, 1] < 0).sum() == (et0[:, 1] < 0).sum()


def test_result_has_empty_circumcircles_by_brute_force():
    xy, tv = scrambled(7, 6, 9)
    out, te, et, _ = mg.delaunay_flip(xy, tv)
    for t in out:
        for v in range(xy.shape[0]):
            if v not in t:
                assert mg.incircle2d(*xy[t], xy[v]) <= 0


def test_every_flip_raises_the_smallest_angle_of_its_quadrilateral():
    xy, tv = scrambled(9, 8, 5)
    te, et = mg.build_edges(tv)
    tv = tv.copy()
    flips = 0
    for sweep in range(100):
        todo = [e for e in range(et.shape[0]) if mg.check_edge(xy, tv, te, et, e)]
        if not todo:
            break
        for e in todo:
            if not mg.check_edge(xy, tv, te, et, e):              # (an earlier flip of this sweep changed its quadrilateral)
                continue
            pair = et[e].copy()
            before = angles(xy, tv[pair]).min()
            mg.flip_edge(tv, te, et, e)
            assert angles(xy, tv[pair]).min() > before - 1e-12
            flips += 1
    assert flips > 20 and sweep < 99


def test_cocircular_points_are_left_alone():
    m = wl.uniform_mesh(6, 6, 1.0, 1.0, periodic=False)            # every interior edge has four cocircular points: INCIRCLE2D = 0
    out, te, et, flips = mg.delaunay_flip(m.xy, m.tri)
    assert flips == 0 and np.array_equal(out, m.tri)


def test_find_triangle_against_exhaustive_search():
    xy, tv = scrambled(10, 9, 4)
    tv, te, et, _ = mg.delaunay_flip(xy, tv)
    rng = np.random.default_rng(8)
    pts = rng.random((150, 2)) * np.array([2.0, 1.5])
    for p in pts:
        inside = [t for t in range(tv.shape[0]) if all(mg.orient2d(xy[tv[t, k]], xy[tv[t, (k + 1) % 3]], p) > 0 for k in range(3))]
        assert len(inside) == 1                                   # random points are strictly inside exactly one triangle
        for t0 in (0, tv.shape[0] // 2, tv.shape[0] - 1):
            assert mg.find_triangle(xy, tv, te, et, p, t0) == (inside[0], 0)


def test_find_triangle_on_edges_vertices_and_outside():
    xy = np.array([[0.0, 0.0], [1.0, 0.0], [0.0, 1.0], [1.0, 1.0]])
    tv = np.array([[0, 1, 2], [1, 3, 2]], dtype=np.int32)
    te, et = mg.build_edges(tv)
    t, code = mg.find_triangle(xy, tv, te, et, (0.5, 0.5), 0)     # on the shared diagonal: edge (1, 2), opposite local vertex 0 of t = 0
    assert (t, code) == (0, 1 + 0) and set(tv[t][[1, 2]]) == {1, 2}
    t, code = mg.find_triangle(xy, tv, te, et, (0.5, 0.5), 1)     # started on the other side it stays there: either is right (L168)
    assert t == 1 and 1 <= code <= 3 and int(te[t, code - 1]) == int(te[0, 0])
    assert mg.find_triangle(xy, tv, te, et, (0.25, 0.0), 1) == (0, 1 + 2)          # on the boundary edge (0, 1) of triangle 0
    assert mg.find_triangle(xy, tv, te, et, (1.0, 1.0), 0) == (1, 4 + 1)           # on vertex 3 = local vertex 1 of triangle 1
    assert mg.find_triangle(xy, tv, te, et, (0.0, 0.0), 1) == (0, 4 + 0)
    assert mg.find_triangle(xy, tv, te, et, (0.3, -0.1), 1) == (-1 - 0, 0)         # leaves through the boundary edge of triangle 0
    assert mg.find_triangle(xy, tv, te, et, (2.0, 2.0), 0) == (-1 - 1, 0)
