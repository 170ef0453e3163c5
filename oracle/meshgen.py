"""CPU ORACLE of the mesh-generation slice -- test infrastructure, NOT the product.

Written from PAPER.md section 2.4 (L142-L208): TestQuality (eq. 2) in numpy fp64, one IEEE operation at a time in the order
the formulas are written (numpy never contracts to FMA), and the two geometric predicates ORIENT2D (eq. 3) and INCIRCLE2D
(eq. 5) EXACTLY, in rational arithmetic (`fractions.Fraction` represents every double exactly): the sign of the determinant
as the paper demands it (L162-L166, L206), with no floating-point rounding anywhere.  Pure-Python loops: small cases only.
Shares nothing with paper_1705_02028_b200/.
"""
from __future__ import annotations

from fractions import Fraction

import numpy as np


def test_quality(xy, tri, R, B):
    """eq. 2 (L146): r = l_a l_b l_c / (2 det), det = |a_x - c_x, a_y - c_y; b_x - c_x, b_y - c_y| (eq. 3; footnote 5);
    beta = r / shortest edge (L120); bad = r > R or beta > B (L150), or det <= 0 (the mesh is counter-clockwise);
    cc = circumcentre, where the new vertex goes (L150): c + (|A|^2 (B_y, -B_x) - |B|^2 (A_y, -A_x)) / (2 det), A = a - c, B = b - c."""
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
    bad = ((r > R) | (beta > B) | ~(det > 0.0)).astype(np.uint8)
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
