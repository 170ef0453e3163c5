"""CPU ORACLE of the mesh-generation layer -- test infrastructure, NOT the product.

Only tests/ may import it.  Written from PAPER.md sections 2.2-2.4 (L84-L208) and 4.1 (L624-L681), step by step in the paper's
order; shares nothing with paper_1705_02028_b200/.  Plain Python and numpy fp64; pure-Python loops: small cases only.

* TestQuality (eq. 2), eq. 4 and the size function: one IEEE operation at a time in the order the formulas are written (numpy
  never contracts to FMA), so that the kernels can be compared bit for bit;
* ORIENT2D (eq. 3) and INCIRCLE2D (eq. 5): EXACTLY, in rational arithmetic (`fractions.Fraction` represents every double
  exactly), the sign of the determinant as the paper demands it (L162-L166, L206);
* the mesh data structure (section 4.1.2), the Delaunay triangulator by sequential edge flips (2.4.6), the walk to the containing
  triangle (2.4.2), candidates with encroachment (2.4.3), cavities and the independent insertion set (4.1.1), the three vertex
  insertions (2.4.4), the re-sorts (4.1.4) and the refinement loop (2.4).

Readings where the paper is silent (M1-M16) are listed in DESIGN.md section 9c.  Pins (tests/test_oracle_meshgen.py,
test_oracle_triangulator.py, test_oracle_refine.py): textbook triangles, the library Delaunay triangulation of the same points,
brute-force empty circumcircles and cavities, Lawson's angle criterion, exhaustive containment search, the diametric circle of
eq. 4, disjoint selected cavities, the guarantees of section 2.3 on finished meshes, the Z curve of a 4 x 4 grid, bilinear
functions, Fig. 8's ordering of random against regular priorities.  No function here is "parity unpinned".
"""
from __future__ import annotations

from fractions import Fraction

import numpy as np


def size_factor(p, grid, box):
    """Section 2.3.1 (L126): "the maximum size can be a function of space, allowing for non-uniform meshes".  Reading M16: the
    function is given on a grid -- grid[j][i] > 0 at the points (x0 + i (x1 - x0) / (nx - 1), y0 + j (y1 - y0) / (ny - 1)) of the
    rectangle box = (x0, y0, x1, y1) -- and interpolated bilinearly (points outside the rectangle take the value of the nearest
    point of its rim); a triangle is too big when r > R * size_factor(circumcentre).  One IEEE operation at a time, in this order."""
    grid = np.asarray(grid, dtype=np.float64)
    p = np.asarray(p, dtype=np.float64).reshape(-1, 2)
    ny, nx = grid.shape
    x0, y0, x1, y1 = (float(v) for v in box)
    sx, sy = (nx - 1.0) / (x1 - x0), (ny - 1.0) / (y1 - y0)
    fx = np.minimum(np.maximum((p[:, 0] - x0) * sx, 0.0), nx - 1.0)
    fy = np.minimum(np.maximum((p[:, 1] - y0) * sy, 0.0), ny - 1.0)
    fi, fj = np.minimum(np.floor(fx), nx - 2.0), np.minimum(np.floor(fy), ny - 2.0)
    i, j = fi.astype(np.int64), fj.astype(np.int64)
    tx, ty = fx - fi, fy - fj
    ux, uy = 1.0 - tx, 1.0 - ty
    g0 = grid[j, i] * ux + grid[j, i + 1] * tx
    g1 = grid[j + 1, i] * ux + grid[j + 1, i + 1] * tx
    return g0 * uy + g1 * ty


def test_quality(xy, tri, R, B, size=None):
    """eq. 2 (L146): r = l_a l_b l_c / (2 det), det = |a_x - c_x, a_y - c_y; b_x - c_x, b_y - c_y| (eq. 3; footnote 5);
    beta = r / shortest edge (L120); bad = r > R or beta > B (L150), or det <= 0 (the mesh is counter-clockwise);
    cc = circumcentre, where the new vertex goes (L150): c + (|A|^2 (B_y, -B_x) - |B|^2 (A_y, -A_x)) / (2 det), A = a - c, B = b - c.
    size = (grid, box): the size bound is R * size_factor(cc, grid, box) instead of R (reading M16)."""
    xy = np.asarray(xy, dtype=np.float64)
    a, b, c = xy[tri[:, 0]], xy[tri[:, 1]], xy[tri[:, 2]]
    Ax, Ay, Bx, By = a[:, 0] - c[:, 0], a[:, 1] - c[:, 1], b[:, 0] - c[:, 0], b[:, 1] - c[:, 1]
    det = Ax * By - Ay * Bx
    Cx, Cy = a[:, 0] - b[:, 0], a[:, 1] - b[:, 1]
    la2, lb2, lc2 = Bx * Bx + By * By, Ax * Ax + Ay * Ay, Cx * Cx + Cy * Cy
    la, lb, lc = np.sqrt(la2), np.sqrt(lb2), np.sqrt(lc2)
    with np.errstate(divide="ignore", invalid="ignore"):
        r = ((la * lb) * lc) / (2.0 * det)
        beta = r / np.minimum(la, np.minimum(lb, lc))
        d2 = 2.0 * det
        ux = (lb2 * By - la2 * Ay) / d2
        uy = (la2 * Ax - lb2 * Bx) / d2
    cc = np.stack([c[:, 0] + ux, c[:, 1] + uy], axis=1)
    Rloc = R if size is None else R * size_factor(cc, size[0], size[1])
    bad = ((r > Rloc) | (beta > B) | ~(det > 0.0)).astype(np.uint8)
    return dict(r=r, beta=beta, cc=cc, bad=bad)


def _sign(x) -> int:
    return (x > 0) - (x < 0)


def orient2d(a, b, c) -> int:
    """Sign of eq. 3 (L160): +1 if (a, b, c) are in counter-clockwise order, -1 if clockwise, 0 if collinear.  Exact."""
    ax, ay, bx, by, cx, cy = (Fraction(float(v)) for v in (*a, *b, *c))
    return _sign((ax - cx) * (by - cy) - (ay - cy) * (bx - cx))


def incircle2d(a, b, c, d) -> int:
    """Sign of eq. 5 (L198): +1 if d lies inside the circle through the counter-clockwise (a, b, c), -1 outside, 0 on it.  Exact."""
    ax, ay, bx, by, cx, cy, dx, dy = (Fraction(float(v)) for v in (*a, *b, *c, *d))
    rows = []
    for px, py in ((ax, ay), (bx, by), (cx, cy)):
        x, y = px - dx, py - dy
        rows.append((x, y, x * x + y * y))
    (a1, a2, a3), (b1, b2, b3), (c1, c2, c3) = rows
    det = a1 * (b2 * c3 - b3 * c2) - a2 * (b1 * c3 - b3 * c1) + a3 * (b1 * c2 - b2 * c1)
    return _sign(det)


# ----------------------------------------------------------------------------------------------------------------------
# Mesh data structure (section 4.1.2) and the Delaunay triangulator (section 2.4.6, section 4.1.5)
# ----------------------------------------------------------------------------------------------------------------------
def build_edges(tv):
    """triangleEdges and edgeTriangles of section 4.1.2 from triangleVertices.  Conventions the paper leaves open (DESIGN.md 9c,
    reading M4): edge k of a triangle is the one OPPOSITE its local vertex k (it joins vertices k+1 and k+2); edges are numbered
    in ascending order of (smaller vertex, larger vertex); edgeTriangles lists the two neighbours in ascending triangle order,
    -1 in the second place for a boundary edge (a segment, L663).  Returns (te [nt][3], et [ne][2])."""
    tv = np.asarray(tv)
    keys = {}
    for t in range(tv.shape[0]):
        for k in range(3):
            a, b = int(tv[t, (k + 1) % 3]), int(tv[t, (k + 2) % 3])
            keys.setdefault((min(a, b), max(a, b)), []).append((t, k))
    te = np.full(tv.shape, -1, dtype=np.int32)
    et = np.full((len(keys), 2), -1, dtype=np.int32)
    for e, key in enumerate(sorted(keys)):
        uses = sorted(keys[key])
        if len(uses) > 2:
            raise ValueError(f"edge {key} belongs to {len(uses)} triangles")
        for j, (t, k) in enumerate(uses):
            te[t, k] = e
            et[e, j] = t
    return te, et


def _opposite(te, t, e):
    k = [int(x) for x in te[t]].index(e)
    return k


def check_edge(xy, tv, te, et, e) -> bool:
    """section 2.4.6 (L190-L196): with T = (a, b, c) one neighbour of E and d the vertex of the other neighbour T' that is not
    part of T, E is NOT Delaunay when INCIRCLE2D(a, b, c, d) > 0, exactly.  Boundary edges are Delaunay by definition."""
    t1, t2 = int(et[e, 0]), int(et[e, 1])
    if t2 < 0:
        return False
    d = int(tv[t2, _opposite(te, t2, e)])
    a, b, c = (int(v) for v in tv[t1])
    return incircle2d(xy[a], xy[b], xy[c], xy[d]) > 0


def flip_edge(tv, te, et, e):
    """Replace E by E' (L102): with a opposite E in t1 = (a, b, c) and d opposite E in t2 = (d, c, b), the quadrilateral a-b-d-c
    becomes t1 = (a, b, d) and t2 = (a, d, c); E keeps its index and its two neighbours, the edges (b, d) and (c, a) change
    sides (the repair of section 4.1.5, done in place)."""
    t1, t2 = int(et[e, 0]), int(et[e, 1])
    i1, i2 = _opposite(te, t1, e), _opposite(te, t2, e)
    a, b, c = (int(tv[t1, (i1 + j) % 3]) for j in range(3))
    d = int(tv[t2, i2])
    assert int(tv[t2, (i2 + 1) % 3]) == c and int(tv[t2, (i2 + 2) % 3]) == b
    e_ca, e_ab = int(te[t1, (i1 + 1) % 3]), int(te[t1, (i1 + 2) % 3])
    e_bd, e_dc = int(te[t2, (i2 + 1) % 3]), int(te[t2, (i2 + 2) % 3])
    tv[t1] = (a, b, d)
    te[t1] = (e_bd, e, e_ab)
    tv[t2] = (a, d, c)
    te[t2] = (e_dc, e_ca, e)
    for f, old, new in ((e_bd, t2, t1), (e_ca, t1, t2)):
        j = 0 if int(et[f, 0]) == old else 1
        assert int(et[f, j]) == old
        et[f, j] = new
    return e_ca, e_ab, e_bd, e_dc


def delaunay_flip(xy, tv, max_sweeps=10 ** 6):
    """"Start with any valid triangulation, and perform edge flips until all edges are locally Delaunay" (L112).  One edge at a
    time, in ascending edge order, sweep after sweep, with the exact INCIRCLE2D.  Returns (tv, te, et, number of flips)."""
    xy = np.asarray(xy, dtype=np.float64)
    tv = np.array(tv, dtype=np.int32)
    te, et = build_edges(tv)
    flips = 0
    for _ in range(max_sweeps):
        done = True
        for e in range(et.shape[0]):
            if check_edge(xy, tv, te, et, e):
                flip_edge(tv, te, et, e)
                flips += 1
                done = False
        if done:
            return tv, te, et, flips
    raise RuntimeError("delaunay_flip did not terminate")


def triangle_set(tv):
    """A triangulation as a set: every triangle rotated so that its smallest vertex comes first (orientation kept)."""
    out = set()
    for a, b, c in np.asarray(tv).tolist():
        m = min(a, b, c)
        out.add((a, b, c) if a == m else (b, c, a) if b == m else (c, a, b))
    return out


# ----------------------------------------------------------------------------------------------------------------------
# Finding the triangle that contains a new vertex (section 2.4.2)
# ----------------------------------------------------------------------------------------------------------------------
def find_triangle(xy, tv, te, et, p, t0, max_steps=10 ** 7):
    """Walk from t0 "to a neighbouring triangle in the direction of v until we have found a triangle containing v" (L168).
    T = (a, b, c) contains v when ORIENT2D(a, b, v), (b, c, v), (c, a, v) are all >= 0 (L156; exact).  Rule where the paper is
    silent (reading M5): the edges are tried in the order (a, b), (b, c), (c, a) and the walk crosses the FIRST one that has v
    strictly on its outer side.  Returns (t, code): code 0 = strictly inside, 1 + k = on edge k of t (opposite local vertex k;
    "located exactly on an edge", L168), 4 + k = on local vertex k; t = -1 - t_last when the walk leaves the triangulation
    through a boundary edge of t_last."""
    t = int(t0)
    for _ in range(max_steps):
        a, b, c = (int(v) for v in tv[t])
        s = (orient2d(xy[a], xy[b], p), orient2d(xy[b], xy[c], p), orient2d(xy[c], xy[a], p))
        # the edge (a, b) is opposite local vertex 2, (b, c) opposite 0, (c, a) opposite 1
        opp = (2, 0, 1)
        out = [j for j in range(3) if s[j] < 0]
        if not out:
            zeros = [j for j in range(3) if s[j] == 0]
            if len(zeros) == 0:
                return t, 0
            if len(zeros) == 1:
                return t, 1 + opp[zeros[0]]
            # on two edge lines at once: on the vertex they share
            shared = {(0, 1): 1, (1, 2): 2, (0, 2): 0}[tuple(zeros[:2])]
            return t, 4 + shared
        e = int(te[t, opp[out[0]]])
        nxt = int(et[e, 0]) if int(et[e, 0]) != t else int(et[e, 1])
        if nxt < 0:
            return -1 - t, 0
        t = nxt
    raise RuntimeError("find_triangle did not terminate")


# ----------------------------------------------------------------------------------------------------------------------
# Delaunay refinement (section 2.4) with the parallel insertion set of section 4.1.1 (L634-L654), bounded domains
# ----------------------------------------------------------------------------------------------------------------------
KIND_NONE, KIND_TRI, KIND_EDGE, KIND_SEG = 0, 1, 2, 3
PRIORITY_REGULAR = 0xFFFFFFFF   # this value of `seed` selects the regular assignment i(v) = number of the bad triangle (Fig. 8)


def priority(seed: int, iteration: int, t: int) -> int:
    """The "unique random integer" i(v) of L648 for the candidate of bad triangle t (reading M10): a 32-bit mix of (seed,
    iteration, t) in the upper half, t itself in the lower half (which makes it unique).  Integer arithmetic modulo 2^32."""
    m = 0xFFFFFFFF
    if seed == PRIORITY_REGULAR:                                  # "regular integer assignment (i.e. i(v_n) = n)", L654 / Fig. 8
        return (t << 32) | t
    x = (t * 2654435761 + iteration * 40503 + seed) & m
    x ^= x >> 15
    x = (x * 2246822519) & m
    x ^= x >> 13
    x = (x * 3266489917) & m
    x ^= x >> 16
    return (x << 32) | t


def _encroaches(xy, u, w, p) -> bool:
    """eq. 4 (L172), one IEEE operation at a time: (r_u - p) . (r_w - p) < 0  -- "no need for exact predicates" (L174)."""
    ux, uy, wx, wy = xy[u][0] - p[0], xy[u][1] - p[1], xy[w][0] - p[0], xy[w][1] - p[1]
    return ux * wx + uy * wy < 0.0


def _edge_ends(tv, te, t, e):
    k = _opposite(te, t, e)
    return int(tv[t, (k + 1) % 3]), int(tv[t, (k + 2) % 3])


def _midpoint(xy, u, w):
    return (0.5 * (xy[u][0] + xy[w][0]), 0.5 * (xy[u][1] + xy[w][1]))


def candidate(xy, tv, te, et, t_bad, cc):
    """Sections 2.4.2-2.4.3 for the circumcentre cc of the bad triangle t_bad: where, and as what, a vertex would go in.
    Returns (kind, p, t_ins, e): KIND_TRI inside triangle t_ins; KIND_EDGE on the interior edge e (t_ins = et[e][0]);
    KIND_SEG: the midpoint of segment e (boundary edge of t_ins) -- because the walk left the triangulation through e
    (reading M8: "if the circumcentre happens to be outside the triangulation ... somewhere a segment is encroached", L140),
    because cc lies on e, or because cc encroaches upon e (eq. 4; of several encroached segments the one with the lowest edge
    number, reading M9); KIND_NONE when cc coincides with an existing vertex."""
    t, code = find_triangle(xy, tv, te, et, cc, t_bad)
    if t < 0:
        t_last = -1 - t
        a, b, c = (int(v) for v in tv[t_last])
        # the walk crosses the first edge with cc strictly outside; at a boundary edge that is where it left
        s = (orient2d(xy[a], xy[b], cc), orient2d(xy[b], xy[c], cc), orient2d(xy[c], xy[a], cc))
        k = (2, 0, 1)[[j for j in range(3) if s[j] < 0][0]]
        e = int(te[t_last, k])
        return KIND_SEG, _midpoint(xy, *_edge_ends(tv, te, t_last, e)), t_last, e
    if code >= 4:
        return KIND_NONE, (float(cc[0]), float(cc[1])), t, -1
    if code >= 1:
        e = int(te[t, code - 1])
        if int(et[e, 1]) < 0:
            return KIND_SEG, _midpoint(xy, *_edge_ends(tv, te, t, e)), t, e
        kind, tris = KIND_EDGE, [int(et[e, 0]), int(et[e, 1])]
    else:
        e, kind, tris = -1, KIND_TRI, [t]
    # eq. 4 against every segment of "all triangles that have either a, b or c as a vertex" (L176-L178)
    verts = set(int(v) for tt in tris for v in tv[tt])
    hit = []
    for tt in range(tv.shape[0]):
        if verts & set(int(v) for v in tv[tt]):
            for k in range(3):
                s = int(te[tt, k])
                if int(et[s, 1]) < 0 and _encroaches(xy, *_edge_ends(tv, te, tt, s), cc):
                    hit.append((s, tt))
    if hit:
        s, tt = min(hit)
        return KIND_SEG, _midpoint(xy, *_edge_ends(tv, te, tt, s)), tt, s
    return kind, (float(cc[0]), float(cc[1])), tris[0], e


def cavity(xy, tv, te, et, p, start):
    """Section 4.1.1 (L640-L644): the triangles whose circumcircles contain p (exact INCIRCLE2D > 0), reached from the insertion
    triangle(s) through shared edges.  Returns a sorted list."""
    seen, todo = set(start), list(start)
    while todo:
        t = todo.pop()
        for k in range(3):
            e = int(te[t, k])
            n = int(et[e, 0]) if int(et[e, 0]) != t else int(et[e, 1])
            if n >= 0 and n not in seen and incircle2d(*(xy[int(v)] for v in tv[n]), p) > 0:
                seen.add(n)
                todo.append(n)
    return sorted(seen)


def _replace(et, e, old, new):
    j = 0 if int(et[e, 0]) == old else 1
    assert int(et[e, j]) == old
    et[e, j] = new


def insert_vertex(tv, te, et, kind, t, e, v, nt, ne):
    """Section 2.4.4 (L180-L184) for new vertex v, with the new triangles numbered from nt and the new edges from ne.
    KIND_TRI: T = (a, b, c) becomes (a, b, v), (b, c, v), (c, a, v): "adds two triangles".  KIND_EDGE: the two triangles
    sharing E are each split into two.  KIND_SEG: "the single triangle of which the segment is part is split into two".
    tv, te, et must have room.  Returns (triangles added, edges added)."""
    if kind == KIND_TRI:
        a, b, c = (int(x) for x in tv[t])
        e0, e1, e2 = (int(x) for x in te[t])
        t1, t2, f0, f1, f2 = nt, nt + 1, ne, ne + 1, ne + 2       # f0 = (v, a), f1 = (v, b), f2 = (v, c)
        tv[t], te[t] = (a, b, v), (f1, f0, e2)
        tv[t1], te[t1] = (b, c, v), (f2, f1, e0)
        tv[t2], te[t2] = (c, a, v), (f0, f2, e1)
        et[f0], et[f1], et[f2] = (t, t2), (t, t1), (t1, t2)
        _replace(et, e0, t, t1)
        _replace(et, e1, t, t2)
        return 2, 3
    t1 = t
    i1 = _opposite(te, t1, e)
    a, b, c = (int(tv[t1, (i1 + j) % 3]) for j in range(3))      # E = (b, c), a opposite
    e_ca, e_ab = int(te[t1, (i1 + 1) % 3]), int(te[t1, (i1 + 2) % 3])
    if kind == KIND_SEG:
        n1, g0, g1 = nt, ne, ne + 1                               # E becomes (b, v); g0 = (v, c) is the other half; g1 = (a, v)
        tv[t1], te[t1] = (a, b, v), (e, g1, e_ab)
        tv[n1], te[n1] = (a, v, c), (g0, e_ca, g1)
        et[g0], et[g1] = (n1, -1), (t1, n1)
        _replace(et, e_ca, t1, n1)
        return 1, 2
    t2 = int(et[e, 0]) if int(et[e, 0]) != t1 else int(et[e, 1])
    i2 = _opposite(te, t2, e)
    d = int(tv[t2, i2])
    e_bd, e_dc = int(te[t2, (i2 + 1) % 3]), int(te[t2, (i2 + 2) % 3])
    n1, n2, g0, g1, g2 = nt, nt + 1, ne, ne + 1, ne + 2           # E becomes (b, v); g0 = (v, c), g1 = (a, v), g2 = (v, d)
    tv[t1], te[t1] = (a, b, v), (e, g1, e_ab)
    tv[n1], te[n1] = (a, v, c), (g0, e_ca, g1)
    tv[t2], te[t2] = (d, v, b), (e, e_bd, g2)
    tv[n2], te[n2] = (d, c, v), (g0, g2, e_dc)
    et[g0], et[g1], et[g2] = (n1, n2), (t1, n1), (t2, n2)
    _replace(et, e_ca, t1, n1)
    _replace(et, e_dc, t2, n2)
    return 2, 3


def flip_to_delaunay(xy, tv, te, et):
    """delaunay_flip on an existing structure, in place; returns the number of flips."""
    flips = 0
    while True:
        done = True
        for e in range(et.shape[0]):
            if check_edge(xy, tv, te, et, e):
                flip_edge(tv, te, et, e)
                flips += 1
                done = False
        if done:
            return flips


def canonical_order(tv):
    """Reading M12: every iteration ends with the triangles renumbered -- each rotated so that its smallest vertex comes first,
    all sorted by (first, second, third) vertex -- and the edge arrays rebuilt (build_edges numbers edges by their end points).
    The paper re-sorts vertices, edges and triangles after every insertion step too (section 4.1.4, by Morton value); this
    order has no ties, which makes the numbering, and with it the priorities of the next iteration, independent of the order
    in which the flips happened."""
    rows = sorted(triangle_set(tv))
    return np.array(rows, dtype=np.int32).reshape(-1, 3)


def morton_key(x, y, box):
    """Morton value of a vertex (section 4.1.4; reading M14): 21 bits per coordinate, i = min(2^21 - 1,
    floor((x - x0) * (2^21 / (x1 - x0)))) with one IEEE operation at a time, the bits of i_x in the even places."""
    x0, y0, x1, y1 = (float(v) for v in box)
    sx, sy = 2097152.0 / (x1 - x0), 2097152.0 / (y1 - y0)
    ix = min(2097151, max(0, int(np.floor((float(x) - x0) * sx))))
    iy = min(2097151, max(0, int(np.floor((float(y) - y0) * sy))))
    key = 0
    for b in range(21):
        key |= ((ix >> b) & 1) << (2 * b) | ((iy >> b) & 1) << (2 * b + 1)
    return key


def morton_order(xy, tv, box):
    """Renumber the vertices in ascending Morton value (ties keep their order) and the triangles' entries with them; the
    triangle order is then made canonical, which follows the vertices' curve.  Returns (xy, tv, new number of every old vertex)."""
    keys = [morton_key(x, y, box) for x, y in np.asarray(xy)]
    order = sorted(range(len(keys)), key=lambda i: (keys[i], i))
    new = np.empty(len(keys), dtype=np.int32)
    new[order] = np.arange(len(keys), dtype=np.int32)
    return np.asarray(xy)[order].copy(), canonical_order(new[np.asarray(tv)]), new


def _insert_and_flip(xy, tv, te, et, R, B, seed, iteration, size=None):
    """Steps 2.4.1-2.4.6 of one iteration (everything but the re-sort): returns the enlarged arrays, Delaunay again, numbered as
    the insertions and flips left them (which depends on the order of the flips), and the info record."""
    xy = np.asarray(xy, dtype=np.float64)
    q = test_quality(xy, tv, R, B, size)
    bad = np.nonzero(q["bad"])[0]
    cands = []
    for t in bad:
        kind, p, t_ins, e = candidate(xy, tv, te, et, int(t), q["cc"][t])
        if kind == KIND_NONE:
            continue
        start = [int(et[e, 0]), int(et[e, 1])] if kind == KIND_EDGE else [t_ins]
        cav = cavity(xy, tv, te, et, p, start)        # the whole set of L638, however large (reading M11)
        cands.append((int(t), kind, p, t_ins, e, cav))
    lock = {}
    for t, kind, p, t_ins, e, cav in cands:
        pr = priority(seed, iteration, t)
        for c in cav:
            lock[c] = max(lock.get(c, 0), pr)
    sel = [cd for cd in cands if all(lock[c] == priority(seed, iteration, cd[0]) for c in cd[5])]
    nv, nt, ne = xy.shape[0], tv.shape[0], et.shape[0]
    add_t = sum(1 if cd[1] == KIND_SEG else 2 for cd in sel)
    add_e = sum(2 if cd[1] == KIND_SEG else 3 for cd in sel)
    xy2 = np.concatenate([xy, np.array([cd[2] for cd in sel], dtype=np.float64).reshape(-1, 2)])
    tv2 = np.concatenate([np.array(tv, dtype=np.int32), np.full((add_t, 3), -1, np.int32)])
    te2 = np.concatenate([np.array(te, dtype=np.int32), np.full((add_t, 3), -1, np.int32)])
    et2 = np.concatenate([np.array(et, dtype=np.int32), np.full((add_e, 2), -1, np.int32)])
    for j, (t, kind, p, t_ins, e, cav) in enumerate(sel):
        dt, de = insert_vertex(tv2, te2, et2, kind, t_ins, e, nv + j, nt, ne)
        nt, ne = nt + dt, ne + de
    flips = flip_to_delaunay(xy2, tv2, te2, et2)
    info = dict(n_bad=len(bad), n_candidates=len(cands), n_selected=len(sel), kinds=[cd[1] for cd in sel], flips=flips,
                selected=[(cd[0], cd[1], cd[2], cd[5]) for cd in sel])
    return xy2, tv2, te2, et2, info


def refine_iteration(xy, tv, te, et, R, B, seed, iteration, box=None, size=None):
    """One iteration of section 2.4 on a Delaunay triangulation: TestQuality; for every bad triangle, in ascending order, its
    candidate; cavities and the independent set of section 4.1.1 (a triangle claimed by several cavities goes to the highest
    priority; a candidate is selected when it holds every triangle of its cavity); the selected vertices are numbered, and
    their triangles and edges appended, in ascending order of their bad triangle; flips restore the Delaunay property; the
    triangles are put in canonical order (reading M12) -- after the vertices have been renumbered along the Morton curve of
    the rectangle `box` = (x0, y0, x1, y1), when one is given (section 4.1.4, reading M14).
    Returns (xy, tv, te, et, info) as new arrays; info: n_bad, n_selected, kinds of the selected, flips."""
    xy2, tv2, te2, et2, info = _insert_and_flip(xy, tv, te, et, R, B, seed, iteration, size)
    if box is not None:                                           # section 4.1.4: Morton order after every insertion step
        xy2, tv2, _ = morton_order(xy2, tv2, box)
    else:
        tv2 = canonical_order(tv2)
    te2, et2 = build_edges(tv2)
    return xy2, tv2, te2, et2, info


def _canon(row):
    a, b, c = (int(v) for v in row)
    m = min(a, b, c)
    return (a, b, c) if a == m else (b, c, a) if b == m else (c, a, b)


def renumber_in_place(tv0, te0, et0, tv2):
    """Reading M15: the numbering an iteration leaves behind when it is NOT followed by a re-sort.  tv0, te0, et0: the mesh
    before the iteration; tv2: the triangles after it, in any order and rotation.  A triangle that survives the iteration keeps
    its number and its rotation; the numbers of the triangles that did not survive, and the new numbers at the end, go to the
    triangles the iteration created, in ascending order of their vertex triple (each rotated to its smallest vertex).  Edges
    likewise, by their pair of end points (smaller, larger).  te and et then follow from the triangles (edge k opposite local
    vertex k; neighbours in ascending order, -1 for the missing one).  Nothing here depends on the order in which the flips
    happened.  Returns (tv, te, et)."""
    nt0, nt2 = np.asarray(tv0).shape[0], np.asarray(tv2).shape[0]
    final = triangle_set(tv2)
    kept = [s for s in range(nt0) if _canon(tv0[s]) in final]
    kept_set = set(kept)
    free = [s for s in range(nt0) if s not in kept_set] + list(range(nt0, nt2))
    added = sorted(final - {_canon(tv0[s]) for s in kept})
    assert len(free) == len(added)
    tv = np.full((nt2, 3), -1, dtype=np.int32)
    for s in kept:
        tv[s] = tv0[s]
    for s, row in zip(free, added):
        tv[s] = row
    # edges: end points of the old slots, the edge set of the new triangulation
    def sides(rows):
        out = {}
        for t, (a, b, c) in enumerate(np.asarray(rows).tolist()):
            for k, (u, w) in enumerate(((b, c), (c, a), (a, b))):
                out.setdefault((min(u, w), max(u, w)), []).append((t, k))
        return out
    ne0 = np.asarray(et0).shape[0]
    old_ends = {}
    for (u, w), uses in sides(tv0).items():
        t, k = uses[0]
        old_ends[int(te0[t, k])] = (u, w)
    new_sides = sides(tv)
    ne2 = len(new_sides)
    slot = {}
    for e in range(ne0):
        if old_ends[e] in new_sides:
            slot[old_ends[e]] = e
    free_e = [e for e in range(ne0) if old_ends[e] not in new_sides] + list(range(ne0, ne2))
    added_e = sorted(k for k in new_sides if k not in slot)
    assert len(free_e) == len(added_e)
    for e, key in zip(free_e, added_e):
        slot[key] = e
    te = np.full((nt2, 3), -1, dtype=np.int32)
    et = np.full((ne2, 2), -1, dtype=np.int32)
    for key, uses in new_sides.items():
        e = slot[key]
        for j, (t, k) in enumerate(sorted(uses)):
            te[t, k] = e
            et[e, j] = t
    return tv, te, et


def refine_iteration_in_place(xy, tv, te, et, R, B, seed, iteration, size=None):
    """One iteration as refine_iteration, but WITHOUT the re-sort: the mesh keeps its numbering where it did not change
    (renumber_in_place, reading M15).  This is what the iterations of refine() do when no Morton box is given."""
    xy2, tv2, te2, et2, info = _insert_and_flip(xy, tv, te, et, R, B, seed, iteration, size)
    tv3, te3, et3 = renumber_in_place(tv, te, et, tv2)
    return xy2, tv3, te3, et3, info


def refine(xy, tv, R, B, seed=0, max_iterations=10 ** 6, box=None, size=None):
    """Section 2.4: iterate "until no more vertices need to be inserted".  The input is made Delaunay and put in canonical
    order first.  With a Morton `box` every iteration ends with the re-sort of section 4.1.4 (readings M12, M14); without one
    the iterations renumber in place (reading M15) and ONE canonical re-sort follows the last of them (so a run of a single
    iteration is refine_iteration either way).  size = (grid, box of the grid): a size bound that varies in space (reading M16).  Returns (xy, tv, te, et, number of iterations that inserted something)."""
    xy = np.asarray(xy, dtype=np.float64)
    tv = canonical_order(delaunay_flip(xy, tv)[0])
    te, et = build_edges(tv)
    it = 0
    while it < max_iterations:
        if box is not None:
            xy, tv, te, et, info = refine_iteration(xy, tv, te, et, R, B, seed, it, box, size)
        else:
            xy, tv, te, et, info = refine_iteration_in_place(xy, tv, te, et, R, B, seed, it, size)
        if info["n_bad"] == 0:
            break
        it += 1
    if box is None and it > 0:
        tv = canonical_order(tv)
        te, et = build_edges(tv)
    return xy, tv, te, et, it
