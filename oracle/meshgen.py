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
