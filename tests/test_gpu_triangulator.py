"""GPU parity of the second mesh-generation slice: mesh data structure (section 4.1.2), Delaunay triangulator
(section 2.4.6 / 4.1.5) and point location (section 2.4.2) against oracle/meshgen.py.  Integer work: bit-exact where the
result is unique (edge numbering, containing triangle, the Delaunay triangulation as a SET of triangles -- the numbering of
triangles and the rotation of their vertices depend on the order of the flips, which the parallel independent sets change),
and validity of the rest (te / et describe tv; every triangle counter-clockwise)."""
import numpy as np
import pytest

import workloads as wl
from oracle import meshgen as mg

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mrdb():
    import torch
    assert torch.cuda.is_available()
    import paper_1705_02028_b200.binding as b
    return b


def dev(a, dtype):
    import torch
    return torch.tensor(np.ascontiguousarray(a), dtype=dtype, device="cuda")


def structure_ok(tv, te, et):
    """te / et describe tv (vectorised form of the oracle tests' assert_structure): edge k of t joins vertices k+1 and k+2 of t,
    t is one of the two neighbours of each of its edges, both neighbours agree on the edge's end points."""
    nt = tv.shape[0]
    ends = np.sort(np.stack([tv[:, [1, 2]], tv[:, [2, 0]], tv[:, [0, 1]]], axis=1), axis=2)      # [nt][3][2]
    e = te.astype(np.int64)
    first = np.full((et.shape[0], 2), -1, dtype=np.int64)
    for k in range(3):
        first[e[:, k]] = ends[:, k]
    same = (first[e] == ends).all()
    t_idx = np.repeat(np.arange(nt), 3).reshape(nt, 3)
    member = ((et[e, 0] == t_idx) | (et[e, 1] == t_idx)).all()
    uses = np.bincount(e.ravel(), minlength=et.shape[0])
    count = (uses == (et >= 0).sum(axis=1)).all()
    return bool(same and member and count)


def ccw_all(mrdb, xy, tv):
    import torch
    s, _ = mrdb.meshgen_orient2d(dev(xy, torch.float64), dev(tv, torch.int32))
    return bool((s == 1).all().item())


@pytest.mark.parametrize("shape", [(14, 11), (61, 47), (200, 150)])
def test_build_edges_is_bitwise_the_oracle(mrdb, shape):
    import torch
    m = wl.scrambled_triangulation(*shape, seed=2)
    te, et = mrdb.meshgen_build_edges(dev(m.tri, torch.int32))
    te, et = te.cpu().numpy(), et.cpu().numpy()
    assert et.shape[0] == m.nt + m.nv - 1
    if m.nt <= 6000:
        ote, oet = mg.build_edges(m.tri)
        assert np.array_equal(te, ote) and np.array_equal(et, oet)
    assert structure_ok(m.tri, te, et) and (et[:, 1] < 0).sum() == 2 * (shape[0] + shape[1])
    # numbered by (smaller, larger) vertex; neighbours in ascending triangle order
    ends = np.sort(np.stack([m.tri[:, [1, 2]], m.tri[:, [2, 0]], m.tri[:, [0, 1]]], axis=1), axis=2)
    key = np.zeros((et.shape[0], 2), dtype=np.int64)
    for k in range(3):
        key[te[:, k]] = ends[:, k]
    assert (np.lexsort((key[:, 1], key[:, 0])) == np.arange(et.shape[0])).all()
    assert ((et[:, 1] < 0) | (et[:, 0] < et[:, 1])).all()


def test_build_edges_rejects_an_edge_with_three_triangles(mrdb):
    import torch
    with pytest.raises(mrdb.MrdError):
        mrdb.meshgen_build_edges(dev(np.array([[0, 1, 2], [0, 1, 3], [1, 0, 4]]), torch.int32))
    te, et = mrdb.meshgen_build_edges(torch.empty((0, 3), dtype=torch.int32, device="cuda"))
    assert te.shape == (0, 3) and et.shape == (0, 2)


@pytest.mark.parametrize("shape,seed", [((14, 11), 1), ((40, 31), 2), ((61, 47), 3)])
def test_delaunay_flip_reaches_the_oracles_triangulation(mrdb, shape, seed):
    """Sizes the sequential oracle finishes in seconds; the largest is 5734 triangles = 23 blocks of 256 edges' worth of work
    with a ragged tail, and needs several iterations of independent sets."""
    import torch
    m = wl.scrambled_triangulation(*shape, seed=seed)
    xy, tv = dev(m.xy, torch.float64), dev(m.tri, torch.int32)
    te, et = mrdb.meshgen_build_edges(tv)
    info = mrdb.meshgen_delaunay_flip(xy, tv, te, et)
    otv, ote, oet, oflips = mg.delaunay_flip(m.xy, m.tri)
    gtv, gte, get = tv.cpu().numpy(), te.cpu().numpy(), et.cpu().numpy()
    assert mg.triangle_set(gtv) == mg.triangle_set(otv)           # the Delaunay triangulation is unique (L96)
    assert structure_ok(gtv, gte, get) and ccw_all(mrdb, m.xy, gtv)
    assert info["flips"] >= 0.5 * oflips and info["iterations"] >= 3
    # boundary edges (segments) are untouched: same vertex pairs as before
    def boundary(tvv, tee, ett):
        b = np.nonzero(ett[:, 1] < 0)[0]
        out = set()
        for e in b:
            t = ett[e, 0]
            k = list(tee[t]).index(e)
            out.add(tuple(sorted((int(tvv[t, (k + 1) % 3]), int(tvv[t, (k + 2) % 3])))))
        return out
    te0, et0 = mg.build_edges(m.tri)
    assert boundary(gtv, gte, get) == boundary(m.tri, te0, et0)
    # a second call finds nothing to do; a rerun from the same input gives bitwise the same arrays (deterministic)
    again = mrdb.meshgen_delaunay_flip(xy, tv, te, et)
    assert again["flips"] == 0 and again["iterations"] == 1 and np.array_equal(tv.cpu().numpy(), gtv)
    tv2 = dev(m.tri, torch.int32)
    te2, et2 = mrdb.meshgen_build_edges(tv2)
    mrdb.meshgen_delaunay_flip(xy, tv2, te2, et2)
    assert np.array_equal(tv2.cpu().numpy(), gtv) and np.array_equal(te2.cpu().numpy(), gte) and np.array_equal(et2.cpu().numpy(), get)


def test_delaunay_flip_at_size_against_the_library_triangulation(mrdb):
    """360 000 triangles (beyond the sequential oracle): the result must be THE Delaunay triangulation of the points -- compared
    with scipy's (Qhull) as a set of triangles -- and every interior edge must pass the exact INCIRCLE2D test (the oracle's
    rational arithmetic on a sample, the library's own exact predicate on all of them)."""
    import torch
    from scipy.spatial import Delaunay
    m = wl.scrambled_triangulation(600, 300, seed=5, Lx=4.0, Ly=2.0)
    xy, tv = dev(m.xy, torch.float64), dev(m.tri, torch.int32)
    te, et = mrdb.meshgen_build_edges(tv)
    info = mrdb.meshgen_delaunay_flip(xy, tv, te, et)
    gtv, gte, get = tv.cpu().numpy(), te.cpu().numpy(), et.cpu().numpy()
    assert info["flips"] > 50000 and structure_ok(gtv, gte, get) and ccw_all(mrdb, m.xy, gtv)
    lib = Delaunay(m.xy).simplices.astype(np.int32)
    p = m.xy[lib]
    cw = (p[:, 0, 0] - p[:, 2, 0]) * (p[:, 1, 1] - p[:, 2, 1]) - (p[:, 0, 1] - p[:, 2, 1]) * (p[:, 1, 0] - p[:, 2, 0]) < 0
    lib[cw] = lib[cw][:, [0, 2, 1]]

    def canon(t):
        r = np.argmin(t, axis=1)
        t = np.stack([t[np.arange(len(t)), (r + j) % 3] for j in range(3)], axis=1)
        return t[np.lexsort((t[:, 2], t[:, 1], t[:, 0]))]
    assert np.array_equal(canon(gtv), canon(lib))
    inner = np.nonzero(get[:, 1] >= 0)[0]
    t1, t2 = get[inner, 0], get[inner, 1]
    k2 = (gte[t2] == inner[:, None]).argmax(axis=1)
    quads = np.concatenate([gtv[t1], gtv[t2, k2][:, None]], axis=1).astype(np.int32)
    s, _ = mrdb.meshgen_incircle2d(xy, dev(quads, torch.int32))
    s = s.cpu().numpy()
    assert (s <= 0).all()
    rng = np.random.default_rng(0)
    for q in quads[rng.choice(len(quads), 300, replace=False)]:
        assert mg.incircle2d(*m.xy[q]) <= 0


@pytest.mark.parametrize("dist,n", [("uniform", 20000), ("ring", 20000), ("aniso", 20000), ("cluster", 3000)])
def test_delaunay_flip_on_scrambled_triangulations_of_random_point_sets(mrdb, dist, n):
    """Point sets that are nothing like a grid: uniform, a thin ring (every point near one circle), anisotropic (10^5 : 1) and
    clustered (distances from 1e-9 to 0.5).  A library triangulation of the points, scrambled by seeded flips of convex
    quadrilaterals, goes back to a triangulation in which every interior edge passes the exact INCIRCLE2D with no zero -- the
    unique Delaunay triangulation, whatever the library made of the same points (it is off by a few triangles on the last two)."""
    import torch
    from scipy.spatial import Delaunay
    rng = np.random.default_rng(17)
    P = rng.random((n, 2))
    if dist == "ring":
        a, r = rng.random(n) * 2 * np.pi, 1 + 1e-3 * rng.random(n)
        P = np.stack([r * np.cos(a), r * np.sin(a)], axis=1)
    elif dist == "aniso":
        P = P * np.array([1000.0, 0.01])
    elif dist == "cluster":
        P = 0.5 + 0.2 * rng.standard_normal((n, 2)) * rng.random((n, 1)) ** 3
    lib = Delaunay(P).simplices.astype(np.int64)
    used = np.unique(lib)                                          # the library drops points it takes for duplicates
    new = -np.ones(n, dtype=np.int64)
    new[used] = np.arange(len(used))
    P, lib = P[used], new[lib]
    pl = P[lib]
    cw = (pl[:, 1, 0] - pl[:, 0, 0]) * (pl[:, 2, 1] - pl[:, 0, 1]) - (pl[:, 1, 1] - pl[:, 0, 1]) * (pl[:, 2, 0] - pl[:, 0, 0]) < 0
    lib[cw] = lib[cw][:, [0, 2, 1]]
    m = wl.flip_edges(wl.UniformMesh(P, lib.astype(np.int32), (0.0, 0.0), None, None, None, (1.0, 1.0)), fraction=0.7, seed=3, rounds=3)
    xy, tv = dev(P, torch.float64), dev(m.tri, torch.int32)
    te, et = mrdb.meshgen_build_edges(tv)
    try:
        info = mrdb.meshgen_delaunay_flip(xy, tv, te, et)
    except mrdb.MrdError as ex:                                    # a library result that is not a triangulation is refused, not flipped
        assert dist == "cluster" and "do not describe a triangulation" in str(ex)
        return
    assert info["flips"] > 50                                      # (the scrambler only flips quadrilaterals that stay well-shaped: few on the ring)
    gtv, gte, get = tv.cpu().numpy(), te.cpu().numpy(), et.cpu().numpy()
    te2, et2 = mrdb.meshgen_build_edges(tv)                        # still a triangulation: the tables can be rebuilt, same edges
    assert len(gtv) == len(lib) and et2.shape == et.shape and ccw_all(mrdb, P, gtv)
    inner = np.nonzero(get[:, 1] >= 0)[0]
    t1, t2 = get[inner, 0], get[inner, 1]
    k2 = (gte[t2] == inner[:, None]).argmax(axis=1)
    quads = np.concatenate([gtv[t1], gtv[t2, k2][:, None]], axis=1).astype(np.int32)
    s, _ = mrdb.meshgen_incircle2d(xy, dev(quads, torch.int32))
    assert (s < 0).all().item()
    for q in quads[np.random.default_rng(0).choice(len(quads), 200, replace=False)]:
        assert mg.incircle2d(*P[q]) < 0


def test_delaunay_flip_leaves_cocircular_points_alone_and_handles_degenerate_sizes(mrdb):
    import torch
    m = wl.uniform_mesh(40, 30, 1.0, 1.0, periodic=False)          # INCIRCLE2D = 0 on every interior edge: all take the exact path
    xy, tv = dev(m.xy, torch.float64), dev(m.tri, torch.int32)
    te, et = mrdb.meshgen_build_edges(tv)
    info = mrdb.meshgen_delaunay_flip(xy, tv, te, et)
    assert info["flips"] == 0 and info["iterations"] == 1 and info["exact"] > 1000
    assert np.array_equal(tv.cpu().numpy(), m.tri)
    one = dev(np.array([[0, 1, 2]]), torch.int32)                  # a single triangle: three boundary edges
    te1, et1 = mrdb.meshgen_build_edges(one)
    assert mrdb.meshgen_delaunay_flip(dev(np.array([[0.0, 0.0], [1.0, 0.0], [0.0, 1.0]]), torch.float64), one, te1, et1)["flips"] == 0
    empty = torch.empty((0, 3), dtype=torch.int32, device="cuda")
    assert mrdb.meshgen_delaunay_flip(xy, empty, empty.clone(), torch.empty((0, 2), dtype=torch.int32, device="cuda"))["flips"] == 0
    mrdb.meshgen_release()                                         # the kept work space comes back on the next call
    te, et = mrdb.meshgen_build_edges(tv)
    assert mrdb.meshgen_delaunay_flip(xy, tv, te, et)["flips"] == 0


def test_overlapping_triangles_and_inconsistent_edge_tables_are_refused(mrdb):
    """Input validation of the triangulator and the refinement: two counter-clockwise triangles on the SAME side of their shared
    edge pass every local check (orientation, at most two triangles per edge) and still overlap -- flips on such an input
    produce edges with three triangles (found by a soak run on library triangulations of clustered points, which drop
    near-duplicate points); edge tables that belong to another numbering are refused as well."""
    import torch
    xy = dev(np.array([[0.0, 0.0], [1.0, 0.0], [0.5, 1.0], [0.5, 0.4]]), torch.float64)
    tv = dev(np.array([[0, 1, 2], [0, 1, 3]]), torch.int32)
    te, et = mrdb.meshgen_build_edges(tv)
    with pytest.raises(mrdb.MrdError, match="same side"):
        mrdb.meshgen_delaunay_flip(xy, tv, te, et)
    with pytest.raises(mrdb.MrdError, match="same side"):
        mrdb.meshgen_refine(xy, tv, te, et, 0.1, 1.5)
    m = wl.scrambled_triangulation(6, 5, seed=3)
    xy, tv = dev(m.xy, torch.float64), dev(m.tri, torch.int32)
    te, et = mrdb.meshgen_build_edges(tv)
    for k in range(3):
        te2, et2 = te.clone(), et.clone()
        if k == 0:
            et2[[4, 9]] = et2[[9, 4]]                              # edgeTriangles of two edges exchanged
        elif k == 1:
            te2[7] = te2[7].roll(1)                                # a triangle's edges in the wrong local places
        else:
            inner = int((et[:, 1] >= 0).nonzero()[0])
            et2[inner, 1] = et2[inner, 0]                          # an edge with the same triangle twice
        with pytest.raises(mrdb.MrdError, match="do not describe a triangulation"):
            mrdb.meshgen_delaunay_flip(xy, tv.clone(), te2, et2)
        with pytest.raises(mrdb.MrdError, match="do not describe a triangulation"):
            mrdb.meshgen_refine(xy, tv, te2, et2, 0.1, 1.5)
    assert mrdb.meshgen_delaunay_flip(xy, tv, te, et)["flips"] > 0     # the unchanged tables are accepted


def test_find_triangle_matches_the_oracle(mrdb):
    import torch
    m = wl.scrambled_triangulation(40, 31, seed=7)
    xy, tv = dev(m.xy, torch.float64), dev(m.tri, torch.int32)
    te, et = mrdb.meshgen_build_edges(tv)
    mrdb.meshgen_delaunay_flip(xy, tv, te, et)
    htv, hte, het = tv.cpu().numpy(), te.cpu().numpy(), et.cpu().numpy()
    rng = np.random.default_rng(12)
    inside = rng.random((3000, 2)) * np.array([2.0, 1.5])
    outside = rng.random((200, 2)) * np.array([3.0, 2.5]) - 0.5
    # degenerate positions (L168): vertices of the mesh, midpoints of edges with exactly representable halves, boundary points
    verts = m.xy[rng.choice(m.nv, 200, replace=False)]
    grid = wl.uniform_mesh(40, 31, 2.0, 1.5, periodic=False).xy[:300]
    pts = np.concatenate([inside, outside, verts, grid])
    t0 = rng.integers(0, m.nt, size=len(pts)).astype(np.int32)
    t, code = mrdb.meshgen_find_triangle(xy, tv, te, et, dev(pts, torch.float64), dev(t0, torch.int32))
    t, code = t.cpu().numpy(), code.cpu().numpy()
    for i in rng.choice(len(pts), 700, replace=False):
        assert (int(t[i]), int(code[i])) == mg.find_triangle(m.xy, htv, hte, het, pts[i], t0[i]), i
    assert (code[:3000] == 0).all() and (t[:3000] >= 0).all() and (t[3000:3200] < 0).any() and (code[3200:3400] >= 4).all()
    # strictly inside: the start triangle does not matter
    t_b, _ = mrdb.meshgen_find_triangle(xy, tv, te, et, dev(inside, torch.float64), dev(np.zeros(3000), torch.int32))
    assert np.array_equal(t_b.cpu().numpy(), t[:3000])


def test_flip_loop_hands_tests_that_need_long_expansions_back_to_the_host_path(mrdb):
    """The late iterations of a flip loop run in one cooperative launch that can evaluate INCIRCLE2D exactly only when the six
    translations are exact.  Here: the fan triangulation of 40 points on the unit circle (as doubles: cocircular to within
    rounding, so every INCIRCLE2D test is beyond the filter and decided by the last bits; coordinates of every magnitude, so
    translations are rarely exact).  Neighbouring diagonals share triangles, so many edges lose their triangle and come back
    in the next iteration with the same test: those iterations go back to the kernels with the long expansions.
    Result: the oracle's triangles (exact rational arithmetic), every edge locally Delaunay."""
    import torch
    from fractions import Fraction
    n = 40
    ang = 2.0 * np.pi * np.arange(n) / n + 0.1
    xy = np.stack([np.cos(ang), np.sin(ang)], axis=1)
    tri = np.array([[0, i, i + 1] for i in range(1, n - 1)], dtype=np.int32)
    te0, et0 = mg.build_edges(tri)                                  # how many INCIRCLE2D tests of the input have an inexact translation?
    inexact = 0
    for e in np.nonzero(et0[:, 1] >= 0)[0]:
        t1, t2 = et0[e]
        d = xy[tri[t2, list(te0[t2]).index(e)]]
        inexact += any(Fraction(float(p[k])) - Fraction(float(d[k])) != Fraction(float(p[k] - d[k])) for p in xy[tri[t1]] for k in (0, 1))
    assert inexact > 10
    dxy, tv = dev(xy, torch.float64), dev(tri, torch.int32)
    te, et = mrdb.meshgen_build_edges(tv)
    mrdb.meshgen_flip_stats(reset=True)
    info = mrdb.meshgen_delaunay_flip(dxy, tv, te, et)
    stats = mrdb.meshgen_flip_stats()
    otv, ote, oet, oflips = mg.delaunay_flip(xy, tri)
    gtv, gte, get = tv.cpu().numpy(), te.cpu().numpy(), et.cpu().numpy()
    assert oflips > 5 and info["flips"] > 5 and info["iterations"] >= 3 and info["exact"] > 20
    assert stats["cooperative_launches"] >= 1 and stats["handed_back"] >= 1, stats
    assert stats["cooperative_iterations"] + stats["launched_iterations"] == info["iterations"]
    assert mg.triangle_set(gtv) == mg.triangle_set(otv) and structure_ok(gtv, gte, get)
    for e in range(get.shape[0]):
        assert not mg.check_edge(xy, gtv, gte, get, e)
