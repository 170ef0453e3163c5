"""GPU parity of the Delaunay refinement (section 2.3-2.4, 4.1.1) against oracle/meshgen.py: refine.
Integer and index work with IEEE-exact coordinates: the refined mesh must be the oracle's ARRAY FOR ARRAY (vertex coordinates
bit for bit, triangleVertices, triangleEdges, edgeTriangles) -- iteration by iteration, after k in-place iterations and for the
whole run -- because every
decision is exact (ORIENT2D, INCIRCLE2D), prescribed (eq. 2 and eq. 4 one IEEE operation at a time) or an integer rule
(priorities, numbering, canonical order).  At sizes beyond the oracle: the guarantees of section 2.3 and the library
triangulation of the final vertex set."""
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


def start(seed, shape):
    m = wl.scrambled_triangulation(*shape, seed=seed)
    tv = mg.canonical_order(mg.delaunay_flip(m.xy, m.tri)[0])
    te, et = mg.build_edges(tv)
    return m.xy, tv, te, et


def to_dev(xy, tv, te, et):
    import torch
    return dev(xy, torch.float64), dev(tv, torch.int32), dev(te, torch.int32), dev(et, torch.int32)


def same(g, o):
    return all(np.array_equal(a.cpu().numpy(), b) for a, b in zip(g, o))


@pytest.mark.parametrize("B,R,seed,shape", [(1.0, 0.09, 1, (6, 5)), (np.sqrt(2.0), 0.05, 2, (6, 5)), (1.2, 0.04, 3, (9, 7))])
def test_every_iteration_and_the_whole_run_match_the_oracle(mrdb, B, R, seed, shape):
    xy, tv, te, et = start(seed, shape)
    state = (xy, tv, te, et)
    kinds = np.zeros(4, dtype=int)
    for it in range(100):                                          # iteration by iteration, from the oracle's state
        o = mg.refine_iteration(*state, R, B, seed, it)
        g = mrdb.meshgen_refine(*to_dev(*state), R, B, seed=seed, first_iteration=it, max_iterations=1)
        assert same(g[:4], o[:4]), it
        assert g[4]["iterations"] == (1 if o[4]["n_bad"] else 0)
        kinds += np.bincount(o[4]["kinds"], minlength=4)
        if o[4]["n_bad"] == 0:
            assert g[4]["bad_left"] == 0
            break
        state = o[:4]
    assert it >= 4 and kinds[mg.KIND_TRI] > 20 and kinds[mg.KIND_SEG] > 5     # both common kinds of insertion were exercised
    # free-running: the iterations renumber in place (reading M15), one re-sort at the end -- after 2, 3, 5 iterations and for
    # the whole run the oracle's arrays
    for k in (2, 3, 5):
        o = mg.refine(xy, tv, R, B, seed=seed, max_iterations=k)
        g = mrdb.meshgen_refine(*to_dev(xy, tv, te, et), R, B, seed=seed, max_iterations=k)
        assert same(g[:4], o[:4]) and g[4]["iterations"] == k and g[4]["bad_left"] > 0, k
    o = mg.refine(xy, tv, R, B, seed=seed)
    g = mrdb.meshgen_refine(*to_dev(xy, tv, te, et), R, B, seed=seed)
    assert same(g[:4], o[:4]) and g[4] == dict(iterations=o[4], bad_left=0)
    assert g[0].shape[0] > 3 * xy.shape[0] and o[4] >= 5
    q = mg.test_quality(o[0], o[1], R, B)
    assert q["bad"].sum() == 0


@pytest.mark.parametrize("jitter,cells,height,R,whole", [(0.25, 34, 8.0, 1.0, True), (0.0, 40, 6.0, 0.8, True), (0.2, 90, 20.0, 3.0, False)])
def test_cavities_beyond_the_per_thread_list_match_the_oracle(mrdb, jitter, cells, height, R, whole):
    """Reading M11 / L638: a cavity is the whole set, however large.  A start mesh of slivers (two rows of boundary vertices: a coarse
    outline) has first cavities of most of its triangles -- more than the 64 a thread keeps in its list, so the kernels walk the
    outline of the cavity instead (cavity_walk).  Every iteration from the oracle's state and the whole run, array for array;
    jitter 0 makes every cell's four vertices cocircular (INCIRCLE2D exactly zero: the exact path)."""
    m = wl.uniform_mesh(cells, 1, 1.0, height, periodic=False)
    if jitter:
        m = wl.jitter_mesh(m, jitter, seed=4)
    tv = mg.canonical_order(mg.delaunay_flip(m.xy, m.tri)[0])
    te, et = mg.build_edges(tv)
    xy, B, seed = m.xy, float(np.sqrt(2.0)), 2
    q0 = mg.test_quality(xy, tv, R, B)
    sizes = [len(mg.cavity(xy, tv, te, et, q0["cc"][t], [loc[0]])) for t in np.nonzero(q0["bad"])[0]
             for loc in [mg.find_triangle(xy, tv, te, et, q0["cc"][t], int(t))] if loc[1] == 0]
    assert max(sizes) > (64 if whole else 150)
    state = (xy, tv, te, et)
    for it in range(100 if whole else 6):                          # the third case: the first iterations only (the oracle's time)
        o = mg.refine_iteration(*state, R, B, seed, it)
        g = mrdb.meshgen_refine(*to_dev(*state), R, B, seed=seed, first_iteration=it, max_iterations=1)
        assert same(g[:4], o[:4]), it
        if o[4]["n_bad"] == 0:
            break
        state = o[:4]
    assert it >= 3
    if not whole:
        return
    o = mg.refine(xy, tv, R, B, seed=seed)
    g = mrdb.meshgen_refine(*to_dev(xy, tv, te, et), R, B, seed=seed)
    assert same(g[:4], o[:4]) and g[4] == dict(iterations=o[4], bad_left=0)
    box = (0.0, 0.0, 1.0, height)
    o = mg.refine(xy, tv, R, B, seed=seed, box=box)
    g = mrdb.meshgen_refine(*to_dev(xy, tv, te, et), R, B, seed=seed, box=box)
    assert same(g[:4], o[:4]) and g[4]["bad_left"] == 0


@pytest.mark.parametrize("B,R,seed,shape", [(1.0, 0.07, 4, (6, 5)), (np.sqrt(2.0), 0.045, 5, (8, 6))])
def test_refinement_with_morton_reordering_matches_the_oracle(mrdb, B, R, seed, shape):
    """Section 4.1.4: vertices renumbered along the Morton curve after every insertion step -- every iteration and the whole
    run array for array the oracle's, keys in ascending order at the end."""
    xy, tv, te, et = start(seed, shape)
    box = (0.0, 0.0, 2.0, 1.5)
    state = (xy, tv, te, et)
    for it in range(100):
        o = mg.refine_iteration(*state, R, B, seed, it, box)
        g = mrdb.meshgen_refine(*to_dev(*state), R, B, seed=seed, first_iteration=it, max_iterations=1, box=box)
        assert same(g[:4], o[:4]), it
        if o[4]["n_bad"] == 0:
            break
        state = o[:4]
    g = mrdb.meshgen_refine(*to_dev(xy, tv, te, et), R, B, seed=seed, box=box)
    assert same(g[:4], state) and g[4]["iterations"] == it and it >= 4
    X = g[0].cpu().numpy()
    keys = [mg.morton_key(x, y, box) for x, y in X]
    assert keys == sorted(keys) and len(X) > 3 * len(xy)
    with pytest.raises(mrdb.MrdError):
        mrdb.meshgen_refine(*to_dev(xy, tv, te, et), R, B, box=(0.0, 0.0, 0.0, 1.0))


def test_graded_refinement_matches_the_oracle(mrdb):
    """Section 2.3.1: the size bound as a function of space (reading M16) -- iteration by iteration and whole runs the oracle's
    arrays, in both numbering modes; the refined mesh is finer where the factor is small."""
    import torch
    xy, tv, te, et = start(6, (7, 5))
    dom = (0.0, 0.0, 2.0, 1.5)
    grid = np.array([[0.2, 0.5, 1.0, 1.0], [0.3, 0.6, 1.0, 1.3], [0.2, 0.5, 1.0, 1.0]])
    dgrid = dev(grid, torch.float64)
    R, B, seed = 0.25, 1.1, 6
    state = (xy, tv, te, et)
    for it in range(100):
        o = mg.refine_iteration(*state, R, B, seed, it, size=(grid, dom))
        g = mrdb.meshgen_refine(*to_dev(*state), R, B, seed=seed, first_iteration=it, max_iterations=1, size=(dgrid, dom))
        assert same(g[:4], o[:4]), it
        if o[4]["n_bad"] == 0:
            break
        state = o[:4]
    assert it >= 5
    for box in (None, dom):
        o = mg.refine(xy, tv, R, B, seed=seed, box=box, size=(grid, dom))
        g = mrdb.meshgen_refine(*to_dev(xy, tv, te, et), R, B, seed=seed, box=box, size=(dgrid, dom))
        assert same(g[:4], o[:4]) and g[4] == dict(iterations=o[4], bad_left=0)
    X = g[0].cpu().numpy()
    assert (X[:, 0] < 0.4).sum() / 0.4 > 4 * (X[:, 0] > 1.4).sum() / 0.6
    q = mg.test_quality(o[0], o[1], R, B, size=(grid, dom))
    assert q["bad"].sum() == 0
    with pytest.raises(mrdb.MrdError):
        mrdb.meshgen_refine(*to_dev(xy, tv, te, et), R, B, size=(dev(np.ones((1, 4)), torch.float64), dom))


def test_regular_priorities_match_the_oracle_and_need_more_iterations(mrdb):
    """L654 / Fig. 8: regular integer assignment i(v_n) = n against random integers, on a Morton-ordered mesh."""
    xy, tv, te, et = start(3, (6, 5))
    box = (0.0, 0.0, 2.0, 1.5)
    o = mg.refine(xy, tv, 0.09, np.sqrt(2.0), seed=mg.PRIORITY_REGULAR, box=box)
    g = mrdb.meshgen_refine(*to_dev(xy, tv, te, et), 0.09, np.sqrt(2.0), seed=mrdb.MESHGEN_PRIORITY_REGULAR, box=box)
    assert same(g[:4], o[:4]) and g[4] == dict(iterations=o[4], bad_left=0)
    r = mrdb.meshgen_refine(*to_dev(xy, tv, te, et), 0.09, np.sqrt(2.0), seed=7, box=box)
    assert g[4]["iterations"] > 1.3 * r[4]["iterations"]
    # at a size beyond the oracle the gap widens
    m = wl.scrambled_triangulation(30, 30, seed=1, Lx=2.0, Ly=2.0)
    import torch
    dxy, dtv = dev(m.xy, torch.float64), dev(m.tri, torch.int32)
    dte, det = mrdb.meshgen_build_edges(dtv)
    mrdb.meshgen_delaunay_flip(dxy, dtv, dte, det)
    its = [mrdb.meshgen_refine(dxy, dtv, dte, det, 0.01, np.sqrt(2.0), seed=sd, box=(0, 0, 2, 2), cap_vertex=200000)[4]["iterations"]
           for sd in (7, mrdb.MESHGEN_PRIORITY_REGULAR)]
    assert its[1] > 2 * its[0]


def test_edge_insertions_on_a_uniform_mesh(mrdb):
    """Right isosceles triangles: every circumcentre is the midpoint of a hypotenuse -- on an interior edge (KIND_EDGE) or on a
    segment -- and every interior edge has four cocircular vertices (all INCIRCLE2D tests take the exact path)."""
    m = wl.uniform_mesh(5, 4, 2.0, 1.5, periodic=False)
    tv = mg.canonical_order(m.tri)
    te, et = mg.build_edges(tv)
    state = (m.xy, tv, te, et)
    seen = np.zeros(4, dtype=int)
    for it in range(3):
        o = mg.refine_iteration(*state, 0.12, 0.6, 5, it)
        g = mrdb.meshgen_refine(*to_dev(*state), 0.12, 0.6, seed=5, first_iteration=it, max_iterations=1)
        assert same(g[:4], o[:4]), it
        seen += np.bincount(o[4]["kinds"], minlength=4)
        state = o[:4]
    assert seen[mg.KIND_EDGE] > 5
    # ... and free-running (in-place renumbering between the iterations) on the same degenerate mesh
    for k in (2, 4):
        o = mg.refine(m.xy, m.tri, 0.12, 0.6, seed=5, max_iterations=k)
        g = mrdb.meshgen_refine(*to_dev(m.xy, tv, te, et), 0.12, 0.6, seed=5, max_iterations=k)
        assert same(g[:4], o[:4]) and g[4]["iterations"] == k, k


def test_refinement_at_size_keeps_the_guarantees_of_section_2_3(mrdb):
    """40 x 30 cells refined to ~10^5 vertices (beyond the sequential oracle): no bad triangle, no angle below arcsin(1 / 2B),
    THE Delaunay triangulation of its vertices (library), same domain, input vertices kept, no encroached segment."""
    import torch
    from scipy.spatial import Delaunay
    m = wl.scrambled_triangulation(40, 30, seed=4)
    xy, tv = dev(m.xy, torch.float64), dev(m.tri, torch.int32)
    te, et = mrdb.meshgen_build_edges(tv)
    mrdb.meshgen_delaunay_flip(xy, tv, te, et)
    B, R = np.sqrt(2.0), 0.004
    gx, gt, gte, get, info = mrdb.meshgen_refine(xy, tv, te, et, R, B, seed=9, cap_vertex=400000)
    assert info["bad_left"] == 0 and 10 < info["iterations"] < 200
    X, T, TE, ET = gx.cpu().numpy(), gt.cpu().numpy(), gte.cpu().numpy(), get.cpu().numpy()
    assert X.shape[0] > 50000 and np.array_equal(X[:m.nv], m.xy)
    q = mg.test_quality(X, T, R, B)
    assert q["bad"].sum() == 0
    p = X[T]
    ang = []
    for k in range(3):
        u, v = p[:, (k + 1) % 3] - p[:, k], p[:, (k + 2) % 3] - p[:, k]
        ang.append(np.arccos(np.clip((u * v).sum(1) / np.hypot(*u.T) / np.hypot(*v.T), -1, 1)))
    assert np.min(ang) >= np.arcsin(1 / (2 * B)) - 1e-9
    area = 0.5 * ((p[:, 1, 0] - p[:, 0, 0]) * (p[:, 2, 1] - p[:, 0, 1]) - (p[:, 1, 1] - p[:, 0, 1]) * (p[:, 2, 0] - p[:, 0, 0]))
    assert (area > 0).all() and abs(area.sum() - 3.0) < 1e-10
    lib = Delaunay(X).simplices.astype(np.int32)
    pl = X[lib]
    cw = (pl[:, 0, 0] - pl[:, 2, 0]) * (pl[:, 1, 1] - pl[:, 2, 1]) - (pl[:, 0, 1] - pl[:, 2, 1]) * (pl[:, 1, 0] - pl[:, 2, 0]) < 0
    lib[cw] = lib[cw][:, [0, 2, 1]]
    r = np.argmin(lib, axis=1)
    lib = np.stack([lib[np.arange(len(lib)), (r + j) % 3] for j in range(3)], axis=1)
    lib = lib[np.lexsort((lib[:, 2], lib[:, 1], lib[:, 0]))]
    # All edges locally Delaunay <=> Delaunay (L100): the exact INCIRCLE2D of every interior edge (the predicate kernel, itself
    # under parity in test_gpu_meshgen.py; a sample again through the oracle's rational arithmetic).  The library triangulation
    # (Qhull: floating-point with tolerances, and this vertex set has exactly cocircular quadruples and thousands of collinear
    # boundary points, where the Delaunay triangulation is not unique, L96) must agree on all but a few triangles.
    lib_set = set(map(tuple, lib.tolist()))
    extra = [t for t, row in enumerate(T.tolist()) if tuple(row) not in lib_set]
    assert len(lib) == len(T) and len(extra) < 0.005 * len(T)
    inner = np.nonzero(ET[:, 1] >= 0)[0]
    t1, t2 = ET[inner, 0], ET[inner, 1]
    k2 = (TE[t2] == inner[:, None]).argmax(axis=1)
    quads = np.concatenate([T[t1], T[t2, k2][:, None]], axis=1).astype(np.int32)
    sgn, _ = mrdb.meshgen_incircle2d(gx, dev(quads, torch.int32))
    assert (sgn <= 0).all().item()
    rng = np.random.default_rng(3)
    for qd in quads[rng.choice(len(quads), 300, replace=False)]:
        assert mg.incircle2d(*X[qd]) <= 0
    seg = np.nonzero(ET[:, 1] < 0)[0]
    tri_of = ET[seg, 0]
    k = (TE[tri_of] == seg[:, None]).argmax(axis=1)
    u, w = T[tri_of, (k + 1) % 3], T[tri_of, (k + 2) % 3]
    on = np.unique(np.concatenate([u, w]))
    assert (np.isin(X[on, 0], [0.0, 2.0]) | np.isin(X[on, 1], [0.0, 1.5])).all()
    mid, rad = 0.5 * (X[u] + X[w]), 0.5 * np.hypot(*(X[u] - X[w]).T)
    near = X[(X[:, 0] < 0.05) | (X[:, 0] > 1.95) | (X[:, 1] < 0.05) | (X[:, 1] > 1.45)]     # only vertices near the sides can encroach
    d = np.hypot(near[:, None, 0] - mid[None, :, 0], near[:, None, 1] - mid[None, :, 1])
    assert (d >= rad[None, :] * (1 - 1e-12)).all()
    # deterministic
    g2 = mrdb.meshgen_refine(xy, tv, te, et, R, B, seed=9, cap_vertex=400000)
    assert all(torch.equal(a, b) for a, b in zip((gx, gt, gte, get), g2[:4]))


def refined_and_checked(mrdb, X0, T0, R, B, seed, cap, area0):
    """Start mesh (X0, T0) made Delaunay and refined on the device; asserts what section 2.3 guarantees and what must hold of any
    refinement -- no bad triangle left, every triangle counter-clockwise, the domain covered exactly once, the input vertices kept,
    every interior edge locally Delaunay by the exact test (the kernel's, a sample again by the oracle's rational arithmetic), the
    same arrays on a second call -- and returns the refined mesh on the host."""
    import torch
    xy, tv = dev(X0, torch.float64), dev(T0, torch.int32)
    te, et = mrdb.meshgen_build_edges(tv)
    mrdb.meshgen_delaunay_flip(xy, tv, te, et)
    gx, gt, gte, get, info = mrdb.meshgen_refine(xy, tv, te, et, R, B, seed=seed, cap_vertex=cap)
    assert info["bad_left"] == 0 and info["iterations"] >= 3
    X, T, TE, ET = gx.cpu().numpy(), gt.cpu().numpy(), gte.cpu().numpy(), get.cpu().numpy()
    assert np.array_equal(X[:len(X0)], X0)
    assert mg.test_quality(X, T, R, B)["bad"].sum() == 0
    p = X[T]
    area = 0.5 * ((p[:, 1, 0] - p[:, 0, 0]) * (p[:, 2, 1] - p[:, 0, 1]) - (p[:, 1, 1] - p[:, 0, 1]) * (p[:, 2, 0] - p[:, 0, 0]))
    assert (area > 0).all() and abs(area.sum() - area0) < 1e-10 * area0
    inner = np.nonzero(ET[:, 1] >= 0)[0]
    t1, t2 = ET[inner, 0], ET[inner, 1]
    k2 = (TE[t2] == inner[:, None]).argmax(axis=1)
    quads = np.concatenate([T[t1], T[t2, k2][:, None]], axis=1).astype(np.int32)
    sgn, _ = mrdb.meshgen_incircle2d(gx, dev(quads, torch.int32))
    assert (sgn <= 0).all().item()
    for qd in quads[np.random.default_rng(1).choice(len(quads), min(100, len(quads)), replace=False)]:
        assert mg.incircle2d(*X[qd]) <= 0
    g2 = mrdb.meshgen_refine(xy, tv, te, et, R, B, seed=seed, cap_vertex=cap)
    assert all(torch.equal(u, w) for u, w in zip((gx, gt, gte, get), g2[:4]))
    return X, T, TE, ET


@pytest.mark.parametrize("n,ax,ay,B,target", [(400, 3.0, 2.0, np.sqrt(2.0), 20000), (2000, 1.0, 1.0, 1.0, 200000), (30, 3.0, 1.0, 1.2, 2000)])
def test_refinement_of_an_outline_keeps_the_guarantees(mrdb, n, ax, ay, B, target):
    """The way a user starts (section 2.4: "starting from the boundary"): the domain given by its boundary vertices only -- a convex
    polygon inscribed in an ellipse, triangulated as a fan, made Delaunay by flips (slivers: the first cavities hold most of
    the mesh, reading M11), then refined.  No bad triangle left, every edge locally Delaunay by the exact test, the polygon
    covered exactly once, boundary vertices only on the polygon's sides, the same result on a second call."""
    import torch
    rng = np.random.default_rng(n)
    ang = np.unique(np.sort(rng.random(n)) * 2 * np.pi)
    n = len(ang)
    X0 = np.stack([ax * np.cos(ang), ay * np.sin(ang)], axis=1)
    T0 = np.stack([np.zeros(n - 2, dtype=np.int32), np.arange(1, n - 1, dtype=np.int32), np.arange(2, n, dtype=np.int32)], axis=1)
    area0 = 0.5 * np.abs(np.sum(X0[:, 0] * np.roll(X0[:, 1], -1) - np.roll(X0[:, 0], -1) * X0[:, 1]))
    R = float(np.sqrt(0.69 * area0 / target))
    X, T, TE, ET = refined_and_checked(mrdb, X0, T0, R, B, 3, 20 * target, area0)
    assert X.shape[0] > 0.3 * target
    # the boundary vertices of the result lie on the sides of the polygon (midpoints of midpoints ... of its sides, up to rounding)
    seg = np.nonzero(ET[:, 1] < 0)[0]
    k = (TE[ET[seg, 0]] == seg[:, None]).argmax(axis=1)
    on = np.unique(np.concatenate([T[ET[seg, 0], (k + 1) % 3], T[ET[seg, 0], (k + 2) % 3]]))
    side = np.clip(np.searchsorted(ang, np.arctan2(X[on, 1] / ay, X[on, 0] / ax) % (2 * np.pi), side="right") - 1, -1, n - 1)
    a, c = X0[side], X0[(side + 1) % n]
    dist = np.abs((c[:, 0] - a[:, 0]) * (X[on, 1] - a[:, 1]) - (c[:, 1] - a[:, 1]) * (X[on, 0] - a[:, 0])) / np.hypot(*(c - a).T)
    assert dist.max() < 1e-12 * max(ax, ay)


@pytest.mark.parametrize("domain,shape,Lx,Ly,B,target", [("L", (8, 6), 2.0, 1.5, 1.2, 300), ("hole", (7, 7), 1.0, 1.0, np.sqrt(2.0), 300),
                                                          ("notch", (9, 6), 2.0, 1.0, 1.0, 300), ("hole", (40, 3), 30.0, 1.0, 1.2, 20000),
                                                          ("L", (33, 47), 2.0, 20.0, np.sqrt(2.0), 200000), ("notch", (5, 44), 30.0, 1.5, 2.0, 20000)])
def test_domains_with_reentrant_corners_notches_and_holes(mrdb, domain, shape, Lx, Ly, B, target):
    """Bounded domains that are not convex: a grid with its upper right quarter ("L"), a block of cells in the middle ("hole") or
    most of one column of cells ("notch") taken out.  A circumcentre beyond a reentrant corner or across a notch is outside the
    triangulation as far as the walk of section 2.4.2 can tell: the segment the walk left through is split (reading M8).  The
    small cases whole runs against the oracle, array for array; all cases the guarantees."""
    m = wl.uniform_mesh(*shape, Lx, Ly, periodic=False)
    c = m.xy[m.tri].mean(axis=1)
    ci, cj = np.floor(c[:, 0] / Lx * shape[0]).astype(int), np.floor(c[:, 1] / Ly * shape[1]).astype(int)
    drop = {"L": (ci >= shape[0] // 2) & (cj >= shape[1] // 2),
            "hole": (ci >= shape[0] // 2) & (ci < shape[0] // 2 + 2) & (cj == shape[1] // 2),
            "notch": (ci == shape[0] // 2) & (cj >= shape[1] // 3)}[domain]
    tri = m.tri[~drop]
    used = np.unique(tri)
    new = -np.ones(m.nv, dtype=np.int64)
    new[used] = np.arange(len(used))
    X0, T0 = m.xy[used], mg.canonical_order(new[tri].astype(np.int32))      # a grid: Delaunay as it stands (cocircular cells)
    area0 = Lx * Ly * (1.0 - drop.sum() / len(drop))
    R = float(np.sqrt(0.69 * area0 / target))
    X, T, TE, ET = refined_and_checked(mrdb, X0, T0, R, B, 5, 3000000, area0)
    assert X.shape[0] > 0.3 * target
    if target <= 300:
        o = mg.refine(X0, T0, R, B, seed=5)
        assert np.array_equal(o[0], X) and np.array_equal(o[1], T) and np.array_equal(o[2], TE) and np.array_equal(o[3], ET)


def test_capacity_and_bad_input_are_reported(mrdb):
    import torch
    xy, tv, te, et = start(1, (6, 5))
    d = to_dev(xy, tv, te, et)
    with pytest.raises(mrdb.MrdError) as ex:
        mrdb.meshgen_refine(*d, 0.02, 1.0, cap_vertex=xy.shape[0] + 20)
    assert ex.value.code == mrdb.MRD_ENOMEM
    # "the arrays then hold a valid Delaunay mesh, partly refined" (include/mrd.h): with a Morton box, going on from it with more room
    # and the iteration count carried over gives the arrays of an uninterrupted run
    box = (0.0, 0.0, 2.0, 1.5)
    whole = mrdb.meshgen_refine(*d, 0.03, 1.2, seed=3, box=box, cap_vertex=20000)
    with pytest.raises(mrdb.MrdError) as ex:
        mrdb.meshgen_refine(*d, 0.03, 1.2, seed=3, box=box, cap_vertex=whole[0].shape[0] // 3)
    part = ex.value.partial
    assert ex.value.code == mrdb.MRD_ENOMEM and 0 < part[4]["iterations"] < whole[4]["iterations"] and part[4]["bad_left"] > 0
    assert xy.shape[0] < part[0].shape[0] <= whole[0].shape[0] // 3
    P, PT = part[0].cpu().numpy(), part[1].cpu().numpy()
    pe, pet = mg.build_edges(PT)
    assert np.array_equal(pe, part[2].cpu().numpy()) and np.array_equal(pet, part[3].cpu().numpy())
    assert all(not mg.check_edge(P, PT, pe, pet, e) for e in range(pet.shape[0]))             # Delaunay
    rest = mrdb.meshgen_refine(*part[:4], 0.03, 1.2, seed=3, box=box, first_iteration=part[4]["iterations"], cap_vertex=20000)
    assert all(torch.equal(a, b) for a, b in zip(rest[:4], whole[:4]))
    assert rest[4]["iterations"] + part[4]["iterations"] == whole[4]["iterations"] and rest[4]["bad_left"] == 0
    g = mrdb.meshgen_refine(*d, 0.5, 10.0)                         # nothing is bad: nothing happens
    assert g[4] == dict(iterations=0, bad_left=0) and same(g[:4], (xy, tv, te, et))
    g = mrdb.meshgen_refine(*d, 0.05, 1.0, max_iterations=2)       # stopped early: still a valid mesh, and says what is left
    assert g[4]["iterations"] == 2 and g[4]["bad_left"] > 0
    with pytest.raises(mrdb.MrdError):
        mrdb.meshgen_refine(*d, -1.0, 1.0)
    # an input that is not a valid triangulation (one triangle turned over) is refused by the refinement and by the triangulator
    import torch
    bad_tv = tv.copy()
    bad_tv[5] = bad_tv[5][[0, 2, 1]]
    db = to_dev(xy, bad_tv, te, et)
    for call in (lambda: mrdb.meshgen_refine(*db, 0.05, 1.0), lambda: mrdb.meshgen_delaunay_flip(*db)):
        with pytest.raises(mrdb.MrdError) as ex:
            call()
        assert ex.value.code == mrdb.MRD_EINVAL and "clockwise" in str(ex.value)


def test_generated_mesh_runs_in_the_solver(mrdb):
    """The point of the generator (section 4): the refined mesh goes straight into the solver.  A mesh refined on the GPU
    (bounded rectangle, boundary vertices frozen) carries 20 RK2 steps of scheme B to the oracle's result, and a uniform
    flow on it has residuals that are exactly zero."""
    import torch
    from types import SimpleNamespace
    import oracle
    import paper_1705_02028_b200 as mrd
    from helpers import field_errors
    xy, tv, te, et = start(2, (9, 7))
    gx, gt, gte, get, info = mrdb.meshgen_refine(*to_dev(xy, tv, te, et), 0.02, np.sqrt(2.0), seed=4, cap_vertex=40000)
    X, T, TE, ET = gx.cpu().numpy(), gt.cpu().numpy(), gte.cpu().numpy(), get.cpu().numpy()
    assert info["bad_left"] == 0 and 3000 < X.shape[0] < 40000
    seg = np.nonzero(ET[:, 1] < 0)[0]
    k = (TE[ET[seg, 0]] == seg[:, None]).argmax(axis=1)
    flag = np.zeros(X.shape[0], dtype=np.uint8)
    flag[T[ET[seg, 0], (k + 1) % 3]] = 1
    flag[T[ET[seg, 0], (k + 2) % 3]] = 1
    val = np.bincount(T.ravel(), minlength=X.shape[0])
    assert val.max() >= 8 and val[flag == 0].min() >= 4             # an unstructured mesh: variable valence
    mesh = SimpleNamespace(xy=X, nv=X.shape[0], lengths=(2.0, 1.5))
    W = wl.random_smooth_state(mesh, mach=0.7, seed=2)
    gm = mrd.Mesh(X, T, vertex_flag=flag, scheme=mrd.SCHEME_B, time_order=2)
    om = oracle.OracleMesh(X, T, vertex_flag=flag, scheme=oracle.SCHEME_B, time_order=2, threads=4)
    gm.set_state(torch.tensor(W, device="cuda"))
    om.set_state(W)
    gm.step(1)
    om.step(1)
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= 1e-12
    gm.step(19)
    om.step(19)
    Wg = gm.get_state().cpu().numpy()
    assert field_errors(Wg, om.get_state()) <= 1e-9
    assert np.array_equal(Wg[:, flag == 1], W[:, flag == 1]) and Wg[0].min() > 0
    U = wl.uniform_state(mesh)
    gm.set_state(torch.tensor(U, device="cuda"))
    gm.step(3)
    assert np.array_equal(gm.get_state().cpu().numpy(), U)          # zero residuals, bit for bit (reading C3)
