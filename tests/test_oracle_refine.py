"""Pins of the oracle's Delaunay refinement (oracle/meshgen.py; section 2.3-2.4, 4.1.1): what the paper and geometry
fix -- the three ways of inserting a vertex keep a valid structure and add 2 / 2 / 1 triangles (L180-L184); a cavity is exactly
the set of triangles whose circumcircles contain the new vertex (L640); eq. 4 is the diametric-circle test (L136); selected
cavities do not overlap (L642) and inserting the selected vertices gives THE Delaunay triangulation of the enlarged vertex set
(checked against the library triangulation); the finished mesh has no triangle with r > R or beta > B, hence no angle below
arcsin(1 / 2B) (L120), is Delaunay, covers the same rectangle, keeps the input vertices, and has no encroached segment."""
import numpy as np
import pytest

import workloads as wl
from oracle import meshgen as mg
from test_oracle_triangulator import angles, assert_structure


def start_mesh(seed=3, shape=(6, 5)):
    m = wl.scrambled_triangulation(*shape, seed=seed)
    tv, te, et, _ = mg.delaunay_flip(m.xy, m.tri)
    return m.xy, tv, te, et


def area(xy, tv):
    p = xy[tv]
    return 0.5 * ((p[:, 1, 0] - p[:, 0, 0]) * (p[:, 2, 1] - p[:, 0, 1]) - (p[:, 1, 1] - p[:, 0, 1]) * (p[:, 2, 0] - p[:, 0, 0]))


def grown(tv, te, et, dt, de):
    return (np.concatenate([tv, np.full((dt, 3), -1, np.int32)]), np.concatenate([te, np.full((dt, 3), -1, np.int32)]),
            np.concatenate([et, np.full((de, 2), -1, np.int32)]))


def library_triangulation(xy):
    from scipy.spatial import Delaunay
    lib = Delaunay(xy).simplices
    cw = np.array([mg.orient2d(*xy[s]) for s in lib]) < 0
    lib[cw] = lib[cw][:, [0, 2, 1]]
    return mg.triangle_set(lib)


def test_the_three_insertions_keep_a_valid_structure_and_add_2_2_1_triangles():
    xy, tv, te, et = start_mesh()
    nv, nt, ne = xy.shape[0], tv.shape[0], et.shape[0]
    total = area(xy, tv).sum()
    # inside a triangle: its centroid
    t = 7
    p = xy[tv[t]].mean(axis=0)
    tv2, te2, et2 = grown(tv, te, et, 2, 3)
    assert mg.insert_vertex(tv2, te2, et2, mg.KIND_TRI, t, -1, nv, nt, ne) == (2, 3)
    xy2 = np.vstack([xy, p])
    assert_structure(xy2, tv2, te2, et2)
    assert abs(area(xy2, tv2).sum() - total) < 1e-13 and (tv2 == nv).sum() == 3
    # on an interior edge: its midpoint (exactly representable halves are not needed: orientation of the four pieces is what counts)
    e = int(np.nonzero(et[:, 1] >= 0)[0][5])
    t1 = int(et[e, 0])
    u, w = mg._edge_ends(tv, te, t1, e)
    xyg = xy.copy()
    xyg[[u, w]] = np.round(xyg[[u, w]] * 1024) / 1024                # make the midpoint exact, so that it IS on the edge
    p = 0.5 * (xyg[u] + xyg[w])
    assert mg.orient2d(xyg[u], xyg[w], p) == 0
    tv2, te2, et2 = grown(tv, te, et, 2, 3)
    assert mg.insert_vertex(tv2, te2, et2, mg.KIND_EDGE, t1, e, nv, nt, ne) == (2, 3)
    xy2 = np.vstack([xyg, p])
    assert_structure(xy2, tv2, te2, et2)
    assert (tv2 == nv).sum() == 4 and abs(area(xy2, tv2).sum() - area(xyg, tv).sum()) < 1e-13
    # on a segment: "the single triangle of which the segment is part is split into two"
    s = int(np.nonzero(et[:, 1] < 0)[0][3])
    t1 = int(et[s, 0])
    p = np.array(mg._midpoint(xy, *mg._edge_ends(tv, te, t1, s)))
    tv2, te2, et2 = grown(tv, te, et, 1, 2)
    assert mg.insert_vertex(tv2, te2, et2, mg.KIND_SEG, t1, s, nv, nt, ne) == (1, 2)
    xy2 = np.vstack([xy, p])
    assert_structure(xy2, tv2, te2, et2)
    assert (tv2 == nv).sum() == 2 and (et2[:, 1] < 0).sum() == (et[:, 1] < 0).sum() + 1
    assert abs(area(xy2, tv2).sum() - total) < 1e-13


def test_cavity_is_every_triangle_whose_circumcircle_contains_the_point():
    xy, tv, te, et = start_mesh(seed=5, shape=(9, 7))
    rng = np.random.default_rng(1)
    for p in rng.random((40, 2)) * np.array([2.0, 1.5]):
        t, code = mg.find_triangle(xy, tv, te, et, p, 0)
        assert code == 0
        brute = [k for k in range(tv.shape[0]) if mg.incircle2d(*xy[tv[k]], p) > 0]
        cav = mg.cavity(xy, tv, te, et, p, [t])
        assert cav == brute and t in cav and len(cav) >= 1        # connected: the walk from t finds them all (L644)


def sliver_mesh(cells=34, height=8.0, seed=4):
    """A Delaunay start mesh made of slivers: two rows of `cells` + 1 boundary vertices, `height` apart, seeded spacing along the rows
    (a coarse outline, as a user would give it): the circumcircles are as large as the strip, so the first cavities hold most
    of the mesh."""
    m = wl.jitter_mesh(wl.uniform_mesh(cells, 1, 1.0, height, periodic=False), 0.25, seed=seed)
    tv, te, et, _ = mg.delaunay_flip(m.xy, m.tri)
    return m.xy, tv, te, et


def test_a_cavity_has_no_vertex_inside_so_its_triangles_form_a_tree():
    # what lets a walk without a list of visited triangles find a cavity (L640-L646; reading M11): a vertex with every one of its
    # triangles in the cavity would vanish from the new triangulation, so there is none, and a triangulated polygon without inner
    # vertices has one shared edge less than it has triangles
    for xy, tv, te, et in (start_mesh(seed=5, shape=(9, 7)), sliver_mesh()):
        rng = np.random.default_rng(3)
        lo, hi = xy.min(axis=0), xy.max(axis=0)
        sizes = []
        for p in lo + rng.random((40, 2)) * (hi - lo):
            t, code = mg.find_triangle(xy, tv, te, et, p, 0)
            if code != 0:
                continue
            cav = set(mg.cavity(xy, tv, te, et, p, [t]))
            inner = [e for e in range(et.shape[0]) if int(et[e, 0]) in cav and int(et[e, 1]) in cav]
            assert len(inner) == len(cav) - 1
            rim = {int(v) for e in np.nonzero(et[:, 1] < 0)[0] for v in mg._edge_ends(tv, te, int(et[e, 0]), int(e))}
            used = {int(v) for c in cav for v in tv[c]} - rim      # vertices inside the domain
            assert not any(all(k in cav for k in np.nonzero((tv == v).any(axis=1))[0]) for v in used)
            sizes.append(len(cav))
        assert len(sizes) > 20
    assert max(sizes) > 40                                        # the sliver mesh: most of its 68 triangles in one cavity


def test_refinement_from_a_mesh_of_slivers_with_cavities_of_most_of_the_mesh():
    # L638 defines the cavity as the whole set: no bound on its size (reading M11)
    xy0, tv0, te0, et0 = sliver_mesh()
    q0 = mg.test_quality(xy0, tv0, 1.0, np.sqrt(2.0))
    first = [len(mg.cavity(xy0, tv0, te0, et0, q0["cc"][t], [mg.find_triangle(xy0, tv0, te0, et0, q0["cc"][t], int(t))[0]]))
             for t in np.nonzero(q0["bad"])[0] if mg.find_triangle(xy0, tv0, te0, et0, q0["cc"][t], int(t))[1] == 0]
    assert max(first) > 64
    xy, tv, te, et, it = mg.refine(xy0, tv0, 1.0, np.sqrt(2.0), seed=2)
    assert mg.test_quality(xy, tv, 1.0, np.sqrt(2.0))["bad"].sum() == 0 and xy.shape[0] > 2 * xy0.shape[0]
    assert_structure(xy, tv, te, et)
    assert all(not mg.check_edge(xy, tv, te, et, e) for e in range(et.shape[0]))
    # the library's triangulation of the same points, up to the diagonals of cocircular quadrilaterals (midpoints of a strip's sides)
    assert len(mg.triangle_set(tv) ^ library_triangulation(xy)) <= 0.05 * tv.shape[0]
    assert abs(area(xy, tv).sum() - 8.0) < 1e-12 and np.array_equal(xy[:xy0.shape[0]], xy0)


def test_eq_4_is_the_diametric_circle():
    rng = np.random.default_rng(2)
    xy = rng.random((2, 2))
    m, r = xy.mean(axis=0), 0.5 * np.hypot(*(xy[0] - xy[1]))
    n = 0
    for p in rng.random((2000, 2)) * 2 - 0.5:
        d = np.hypot(*(p - m))
        if abs(d - r) > 1e-9:
            assert mg._encroaches(xy, 0, 1, p) == (d < r)         # L136: "if any vertex lies inside the diametric circle"
            n += d < r
    assert n > 50


def test_candidates_of_constructed_cases():
    # two right isosceles triangles: both circumcentres are the midpoint of the shared diagonal -> on the interior edge
    xy = np.array([[0.0, 0.0], [1.0, 0.0], [0.0, 1.0], [1.0, 1.0]])
    tv = np.array([[0, 1, 2], [1, 3, 2]], dtype=np.int32)
    te, et = mg.build_edges(tv)
    q = mg.test_quality(xy, tv, 1.0, 0.5)
    kind, p, t, e = mg.candidate(xy, tv, te, et, 0, q["cc"][0])
    assert kind == mg.KIND_EDGE and p == (0.5, 0.5) and int(et[e, 1]) >= 0
    # an obtuse triangle at the boundary: the circumcentre is outside the domain -> the walk leaves through a segment,
    # which is split at its midpoint
    xy = np.array([[0.0, 0.0], [4.0, 0.0], [2.0, 0.5], [2.0, 3.0]])
    tv = np.array([[0, 1, 2], [1, 3, 2], [3, 0, 2]], dtype=np.int32)
    te, et = mg.build_edges(tv)
    q = mg.test_quality(xy, tv, 10.0, 1.0)
    assert q["cc"][0][1] < 0                                       # below the edge (0, 1)
    kind, p, t, e = mg.candidate(xy, tv, te, et, 0, q["cc"][0])
    assert kind == mg.KIND_SEG and p == (2.0, 0.0) and t == 0 and set(mg._edge_ends(tv, te, t, e)) == {0, 1}
    # a point inside the domain but inside the diametric circle of a segment: the segment is split, not the triangle
    cc = np.array([2.0, 0.2])
    assert mg.find_triangle(xy, tv, te, et, cc, 1) == (0, 0)
    kind, p, t, e = mg.candidate(xy, tv, te, et, 1, cc)
    assert kind == mg.KIND_SEG and p == (2.0, 0.0)
    # well inside a larger domain, far from every segment: into the triangle that contains it
    xyb, tvb, teb, etb = start_mesh()
    cc = np.array([1.03, 0.77])
    kind, p, t, e = mg.candidate(xyb, tvb, teb, etb, 0, cc)
    assert kind == mg.KIND_TRI and p == (1.03, 0.77) and e == -1 and mg.find_triangle(xyb, tvb, teb, etb, cc, 5) == (t, 0)
    # exactly on a vertex: nothing to insert
    assert mg.candidate(xy, tv, te, et, 0, xy[2])[0] == mg.KIND_NONE


def test_priority_is_unique_reproducible_and_mixes():
    pr = [mg.priority(7, 2, t) for t in range(4000)]
    assert len(set(pr)) == 4000 and all(p & 0xFFFFFFFF == t for t, p in enumerate(pr))
    hi = np.array([p >> 32 for p in pr], dtype=np.float64)
    assert 0.45 < hi.mean() / 2 ** 32 < 0.55 and abs(np.corrcoef(hi[:-1], hi[1:])[0, 1]) < 0.1
    assert mg.priority(7, 2, 5) != mg.priority(7, 3, 5) != mg.priority(8, 3, 5) and mg.priority(7, 2, 5) == pr[5]
    assert mg.priority(0, 0, 0) == 0                              # the mix maps 0 to 0


def test_one_iteration_inserts_an_independent_set_and_stays_delaunay():
    xy, tv, te, et = start_mesh()
    xy2, tv2, te2, et2, info = mg.refine_iteration(xy, tv, te, et, 0.06, 1.0, seed=3, iteration=0)
    assert 0 < info["n_selected"] < info["n_candidates"] <= info["n_bad"]
    cavs = [set(c[3]) for c in info["selected"]]
    for i in range(len(cavs)):
        for j in range(i):
            assert not (cavs[i] & cavs[j])                        # L642: "their cavities do not overlap"
    assert [c[0] for c in info["selected"]] == sorted(c[0] for c in info["selected"])
    assert np.array_equal(xy2[:xy.shape[0]], xy) and xy2.shape[0] == xy.shape[0] + info["n_selected"]
    assert np.array_equal(xy2[xy.shape[0]:], np.array([c[2] for c in info["selected"]]))
    kinds = np.bincount(info["kinds"], minlength=4)
    assert tv2.shape[0] == tv.shape[0] + 2 * (kinds[1] + kinds[2]) + kinds[3] and kinds[1] > 0 and kinds[3] > 0
    assert_structure(xy2, tv2, te2, et2)
    assert mg.triangle_set(tv2) == library_triangulation(xy2)     # THE Delaunay triangulation of the enlarged vertex set
    # a loser of this iteration is a candidate again in the next one, and another seed picks another set
    other = mg.refine_iteration(xy, tv, te, et, 0.06, 1.0, seed=4, iteration=0)[4]
    assert [c[0] for c in other["selected"]] != [c[0] for c in info["selected"]]


@pytest.mark.parametrize("B,R,seed", [(1.0, 0.09, 1), (np.sqrt(2.0), 0.07, 2)])
def test_refinement_ends_with_the_guarantees_of_section_2_3(B, R, seed):
    xy0, tv0, te0, et0 = start_mesh(seed=seed)
    xy, tv, te, et, it = mg.refine(xy0, tv0, R, B, seed=seed)
    assert 3 <= it < 60 and xy.shape[0] > 3 * xy0.shape[0]
    q = mg.test_quality(xy, tv, R, B)
    assert q["bad"].sum() == 0 and q["r"].max() <= R and q["beta"].max() <= B
    assert angles(xy, tv).min() >= np.arcsin(1.0 / (2.0 * B)) - 1e-12          # L120: 2 beta = 1 / sin(alpha)
    assert_structure(xy, tv, te, et)
    assert all(not mg.check_edge(xy, tv, te, et, e) for e in range(et.shape[0]))
    assert mg.triangle_set(tv) == library_triangulation(xy)
    assert np.array_equal(xy[:xy0.shape[0]], xy0)
    assert abs(area(xy, tv).sum() - 2.0 * 1.5) < 1e-12            # the rectangle of the workload, no more, no less
    seg = np.nonzero(et[:, 1] < 0)[0]
    ends = np.array([mg._edge_ends(tv, te, int(et[s, 0]), int(s)) for s in seg])
    on_boundary = np.unique(ends)
    b = xy[on_boundary]
    assert (np.isin(b[:, 0], [0.0, 2.0]) | np.isin(b[:, 1], [0.0, 1.5])).all()   # segments stay on the sides (midpoints are exact there)
    mid, rad = 0.5 * (xy[ends[:, 0]] + xy[ends[:, 1]]), 0.5 * np.hypot(*(xy[ends[:, 0]] - xy[ends[:, 1]]).T)
    d = np.hypot(xy[:, None, 0] - mid[None, :, 0], xy[:, None, 1] - mid[None, :, 1])
    assert (d >= rad[None, :] * (1 - 1e-12)).all()               # L136: no vertex inside a diametric circle -- no encroached segment
    # "the resulting mesh ... is not unique ... the locations of the vertices depend on the order" (L144), the guarantees do not
    xy_b, tv_b, _, _, _ = mg.refine(xy0, tv0, R, B, seed=seed + 10)
    assert xy_b.shape != xy.shape or not np.array_equal(xy_b, xy)
    assert mg.test_quality(xy_b, tv_b, R, B)["bad"].sum() == 0
    xy_c, tv_c, _, _, _ = mg.refine(xy0, tv0, R, B, seed=seed)
    assert np.array_equal(xy_c, xy) and np.array_equal(tv_c, tv)


def test_canonical_order_renumbers_without_changing_the_triangulation():
    xy, tv, te, et = start_mesh(seed=8)
    rng = np.random.default_rng(0)
    shuffled = tv[rng.permutation(tv.shape[0])]
    rot = rng.integers(0, 3, size=tv.shape[0])
    shuffled = np.stack([shuffled[np.arange(len(rot)), (rot + j) % 3] for j in range(3)], axis=1).astype(np.int32)
    c = mg.canonical_order(shuffled)
    assert mg.triangle_set(c) == mg.triangle_set(tv) and np.array_equal(c, mg.canonical_order(tv))
    assert (c[:, 0] < c[:, 1]).all() and (c[:, 0] < c[:, 2]).all()
    assert (np.lexsort((c[:, 2], c[:, 1], c[:, 0])) == np.arange(len(c))).all()
    assert all(mg.orient2d(*xy[t]) == 1 for t in c)               # rotation only: every triangle stays counter-clockwise
    assert np.array_equal(mg.canonical_order(c), c)


def test_morton_order_follows_the_z_curve_and_changes_numbers_only():
    """Section 4.1.4: 'assigning a Morton value to each vertex, and then sorting'.  On a 4 x 4 grid of cell centres the order is
    the textbook Z curve; on a mesh it is a renumbering (same points, same triangles) with neighbours in number close in space."""
    c = (np.arange(4) + 0.5) / 4
    pts = np.array([(x, y) for y in c for x in c])                # row-major
    keys = [mg.morton_key(x, y, (0.0, 0.0, 1.0, 1.0)) for x, y in pts]
    z = [0, 1, 4, 5, 2, 3, 6, 7, 8, 9, 12, 13, 10, 11, 14, 15]     # Z order of a 4 x 4 block, row-major index
    assert [int(np.argsort(keys)[i]) for i in range(16)] == z
    assert mg.morton_key(0.0, 0.0, (0, 0, 1, 1)) == 0 and mg.morton_key(1.0, 1.0, (0, 0, 1, 1)) == 2 ** 42 - 1   # the far corner is clamped
    assert mg.morton_key(1.0, 0.0, (0, 0, 1, 1)) == int("01" * 21, 2) and mg.morton_key(0.0, 1.0, (0, 0, 1, 1)) == int("10" * 21, 2)
    xy, tv, te, et = start_mesh(seed=6, shape=(12, 9))
    box = (0.0, 0.0, 2.0, 1.5)
    xy2, tv2, new = mg.morton_order(xy, tv, box)
    assert sorted(new) == list(range(len(new))) and np.array_equal(xy2[new], xy)
    assert mg.triangle_set(tv2) == mg.triangle_set(new[tv]) and np.array_equal(tv2, mg.canonical_order(tv2))
    k2 = [mg.morton_key(x, y, box) for x, y in xy2]
    assert k2 == sorted(k2)
    step = np.hypot(*(xy2[1:] - xy2[:-1]).T)
    step0 = np.hypot(*(xy[1:] - xy[:-1]).T)
    assert np.median(step) < 1.5 * np.median(step0) and step.max() <= 2.5   # consecutive numbers are neighbours; the curve's jumps stay in the box
    # refinement with the reordering gives the same kind of mesh (another vertex order changes the insertion order, L144)
    xa, ta, _, _, ita = mg.refine(xy, tv, 0.08, 1.0, seed=2, box=box)
    q = mg.test_quality(xa, ta, 0.08, 1.0)
    assert q["bad"].sum() == 0 and mg.triangle_set(ta) == library_triangulation(xa)
    ka = [mg.morton_key(x, y, box) for x, y in xa]
    assert ka == sorted(ka)


def test_in_place_renumbering_keeps_survivors_and_does_not_depend_on_the_flip_order():
    """Reading M15 (renumber_in_place): what an iteration without re-sort leaves behind."""
    xy, tv, te, et = start_mesh(seed=7, shape=(10, 8))
    tv = mg.canonical_order(tv)
    te, et = mg.build_edges(tv)
    xy2, tvr, ter, etr, info = mg.refine_iteration(xy, tv, te, et, 0.3, 0.9, seed=5, iteration=0)
    xy3, tvp, tep, etp, _ = mg.refine_iteration_in_place(xy, tv, te, et, 0.3, 0.9, seed=5, iteration=0)
    assert np.array_equal(xy2, xy3) and 0 < info["n_selected"]
    assert_structure(xy3, tvp, tep, etp)
    assert mg.triangle_set(tvp) == mg.triangle_set(tvr)           # the same mesh ...
    tvs = mg.canonical_order(tvp)
    assert np.array_equal(tvs, tvr) and all(np.array_equal(a, b) for a, b in zip(mg.build_edges(tvs), (ter, etr)))   # ... and the same after a re-sort
    nt0, ne0 = tv.shape[0], et.shape[0]
    final = mg.triangle_set(tvp)
    survives = np.array([mg._canon(r) in final for r in tv])
    assert 0.2 < survives.mean() < 1.0
    assert np.array_equal(tvp[:nt0][survives], tv[survives])      # survivors: same number, same rotation
    assert np.array_equal(tep[:nt0][survives], te[survives])      # ... and so the same edges
    free = np.concatenate([np.nonzero(~survives)[0], np.arange(nt0, tvp.shape[0])])
    rows = tvp[free]
    assert (rows[:, 0] < rows[:, 1]).all() and (rows[:, 0] < rows[:, 2]).all()
    assert (np.lexsort((rows[:, 2], rows[:, 1], rows[:, 0])) == np.arange(len(rows))).all()    # created triangles: ascending triples into ascending slots
    assert ((etp[:, 1] < 0) | (etp[:, 0] < etp[:, 1])).all()
    old_pairs = {tuple(sorted(mg._edge_ends(tv, te, int(et[e, 0]), e))): e for e in range(ne0)}
    new_pairs = {tuple(sorted(mg._edge_ends(tvp, tep, int(etp[e, 0]), e))): e for e in range(etp.shape[0])}
    same = [k for k in old_pairs if k in new_pairs]
    assert len(same) > 0.2 * ne0 and all(old_pairs[k] == new_pairs[k] for k in same)            # surviving edges keep their numbers
    created = sorted(k for k in new_pairs if k not in old_pairs)
    assert [new_pairs[k] for k in created] == sorted(new_pairs[k] for k in created)
    # any numbering and rotation of the triangles after the flips gives the same result
    rng = np.random.default_rng(1)
    sh = tvr[rng.permutation(tvr.shape[0])]
    rot = rng.integers(0, 3, size=sh.shape[0])
    sh = np.stack([sh[np.arange(len(rot)), (rot + j) % 3] for j in range(3)], axis=1).astype(np.int32)
    again = mg.renumber_in_place(tv, te, et, sh)
    assert all(np.array_equal(a, b) for a, b in zip(again, (tvp, tep, etp)))


def test_refine_without_box_is_in_place_iterations_and_one_final_sort():
    xy0, tv0, te0, et0 = start_mesh(seed=2)
    xy, tv, te, et, it = mg.refine(xy0, tv0, 0.09, 1.0, seed=6)
    sx, st = xy0, mg.canonical_order(tv0)
    ste, set_ = mg.build_edges(st)
    for k in range(it):
        sx, st, ste, set_, info = mg.refine_iteration_in_place(sx, st, ste, set_, 0.09, 1.0, 6, k)
        assert info["n_selected"] > 0
    assert mg.refine_iteration_in_place(sx, st, ste, set_, 0.09, 1.0, 6, it)[4]["n_bad"] == 0
    assert np.array_equal(xy, sx) and np.array_equal(tv, mg.canonical_order(st))
    assert np.array_equal(mg.refine(xy0, tv0, 0.09, 1.0, seed=6, max_iterations=1)[1],
                          mg.refine_iteration(xy0, mg.canonical_order(tv0), *mg.build_edges(mg.canonical_order(tv0)), 0.09, 1.0, 6, 0)[1])


def test_size_function_is_bilinear_and_grades_the_mesh():
    """Reading M16 (section 2.3.1: the size bound as a function of space)."""
    grid = np.array([[1.0, 2.0, 4.0], [3.0, 5.0, 9.0]])             # ny = 2, nx = 3 on the rectangle [0, 2] x [10, 11]
    box = (0.0, 10.0, 2.0, 11.0)
    f = lambda x, y: float(mg.size_factor([[x, y]], grid, box)[0])
    assert [f(0, 10), f(1, 10), f(2, 10), f(0, 11), f(1, 11), f(2, 11)] == [1.0, 2.0, 4.0, 3.0, 5.0, 9.0]   # the grid points themselves
    assert f(0.5, 10) == 1.5 and f(1.5, 11) == 7.0 and f(0, 10.5) == 2.0 and f(1.5, 10.5) == 5.0            # midpoints of edges and of a cell
    assert f(0.25, 10.25) == (1.0 * 0.75 + 2.0 * 0.25) * 0.75 + (3.0 * 0.75 + 5.0 * 0.25) * 0.25
    assert f(-3, 9) == 1.0 and f(5, 12) == 9.0 and f(1, 99) == 5.0                                           # outside: the nearest point of the rim
    rng = np.random.default_rng(0)
    a, b, c = 0.7, -0.3, 1.9                                        # bilinear interpolation reproduces a + b x + c y + d x y
    gx, gy = np.meshgrid(np.linspace(0, 2, 5), np.linspace(10, 11, 4))
    lin = a + b * gx + c * gy + 0.5 * gx * gy
    pts = rng.random((50, 2)) * np.array([2.0, 1.0]) + np.array([0.0, 10.0])
    assert np.allclose(mg.size_factor(pts, lin, box), a + b * pts[:, 0] + c * pts[:, 1] + 0.5 * pts[:, 0] * pts[:, 1], rtol=1e-13)
    # a constant function changes nothing; a graded one grades the mesh and keeps the guarantees
    xy0, tv0, te0, et0 = start_mesh(seed=4)
    dom = (0.0, 0.0, 2.0, 1.5)
    plain = mg.refine(xy0, tv0, 0.1, 1.0, seed=1)
    const = mg.refine(xy0, tv0, 0.05, 1.0, seed=1, size=(np.full((3, 4), 2.0), dom))
    assert np.array_equal(plain[0], const[0]) and np.array_equal(plain[1], const[1])
    g = np.array([[0.25, 1.0, 1.0], [0.25, 1.0, 1.0]])              # a quarter of the size at the left side
    xy, tv, te, et, it = mg.refine(xy0, tv0, 0.2, 1.0, seed=1, size=(g, dom))
    q = mg.test_quality(xy, tv, 0.2, 1.0, size=(g, dom))
    assert q["bad"].sum() == 0 and (q["r"] <= 0.2 * mg.size_factor(q["cc"], g, dom)).all() and q["beta"].max() <= 1.0
    assert mg.triangle_set(tv) == library_triangulation(xy)
    left, right = (xy[:, 0] < 0.3).sum() / 0.3, (xy[:, 0] > 1.2).sum() / 0.8
    assert left > 4 * right                                         # ~16 times the vertex density where the bound is a quarter
    assert mg.test_quality(xy, tv, 0.2, 1.0)["bad"].sum() == 0 and mg.test_quality(xy, tv, 0.05, 1.0)["bad"].sum() > 0


def test_regular_priorities_need_more_iterations_than_random_ones_on_a_morton_ordered_mesh():
    """L654 / Fig. 8: "because of Morton ordering, vertices with large values of i are located very close to each other, making
    the parallel selection method very inefficient.  However, for random integer assignment, the number of iterations necessary
    follows the theoretical limit rather nicely."  Same guarantees either way."""
    assert mg.priority(mg.PRIORITY_REGULAR, 3, 41) == (41 << 32) | 41 and mg.priority(mg.PRIORITY_REGULAR, 0, 7) < mg.priority(mg.PRIORITY_REGULAR, 9, 8)
    xy0, tv0, te0, et0 = start_mesh(seed=3)
    box = (0.0, 0.0, 2.0, 1.5)
    xr, tr, _, _, it_random = mg.refine(xy0, tv0, 0.09, np.sqrt(2.0), seed=7, box=box)
    xg, tg, _, _, it_regular = mg.refine(xy0, tv0, 0.09, np.sqrt(2.0), seed=mg.PRIORITY_REGULAR, box=box)
    assert it_regular > 1.3 * it_random
    for x, t in ((xr, tr), (xg, tg)):
        assert mg.test_quality(x, t, 0.09, np.sqrt(2.0))["bad"].sum() == 0 and mg.triangle_set(t) == library_triangulation(x)
    # in one iteration the regular assignment selects fewer vertices from the same candidates
    tvc = mg.canonical_order(tv0)
    tec, etc = mg.build_edges(tvc)
    xm, tm, _ = mg.morton_order(xy0, tvc, box)
    tem, etm = mg.build_edges(tm)
    a = mg.refine_iteration(xm, tm, tem, etm, 0.05, np.sqrt(2.0), 7, 0, box)[4]
    b = mg.refine_iteration(xm, tm, tem, etm, 0.05, np.sqrt(2.0), mg.PRIORITY_REGULAR, 0, box)[4]
    assert a["n_candidates"] == b["n_candidates"] and b["n_selected"] < a["n_selected"]
