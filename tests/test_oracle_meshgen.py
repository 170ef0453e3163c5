"""Pins of the mesh-generation oracle (oracle/meshgen.py): what the paper and elementary geometry fix about
TestQuality (eq. 2), ORIENT2D (eq. 3) and INCIRCLE2D (eq. 5)."""
import numpy as np

from oracle import meshgen as mg


def test_circumradius_and_quality_of_textbook_triangles():
    s3 = np.sqrt(3.0)
    xy = np.array([[0.0, 0.0], [1.0, 0.0], [0.5, s3 / 2], [0.0, 1.0], [2.0, 0.0], [1.0, 1e-3]])
    tri = np.array([[0, 1, 2], [0, 1, 3], [0, 4, 5]], dtype=np.int32)
    q = mg.test_quality(xy, tri, R=0.6, B=1.0)
    # equilateral: r = side / sqrt(3), 2 beta = 1 / sin(60 deg);  right isosceles: r = hypotenuse / 2, 2 beta = 1 / sin(45 deg)
    assert abs(q["r"][0] - 1 / s3) < 1e-15 and abs(2 * q["beta"][0] - 1 / np.sin(np.pi / 3)) < 1e-15
    assert abs(q["r"][1] - np.sqrt(2.0) / 2) < 1e-15 and abs(2 * q["beta"][1] - np.sqrt(2.0)) < 1e-15
    assert np.allclose(q["cc"][0], [0.5, s3 / 6]) and np.allclose(q["cc"][1], [0.5, 0.5])
    # a sliver: huge circumradius, beta >> B
    assert q["r"][2] > 100 and q["beta"][2] > 100
    assert q["bad"].tolist() == [0, 1, 1]                        # r = 0.707 > R = 0.6;  the sliver fails both
    assert mg.test_quality(xy, tri, R=10.0, B=0.5)["bad"].tolist() == [1, 1, 1]     # beta = 0.577 > B = 0.5
    assert mg.test_quality(xy, tri[:, [0, 2, 1]], R=1e9, B=1e9)["bad"].tolist() == [1, 1, 1]   # clockwise: flagged


def test_circumcentre_is_equidistant_and_two_beta_is_one_over_sin_of_the_smallest_angle():
    rng = np.random.default_rng(4)
    xy = rng.random((600, 2)) * 3.0 - 1.0
    tri = rng.permutation(600).reshape(-1, 3).astype(np.int32)
    a, b, c = xy[tri[:, 0]], xy[tri[:, 1]], xy[tri[:, 2]]
    ccw = (a[:, 0] - c[:, 0]) * (b[:, 1] - c[:, 1]) - (a[:, 1] - c[:, 1]) * (b[:, 0] - c[:, 0]) > 0
    tri[~ccw] = tri[~ccw][:, [0, 2, 1]]
    a, b, c = xy[tri[:, 0]], xy[tri[:, 1]], xy[tri[:, 2]]
    q = mg.test_quality(xy, tri, R=1.0, B=1.0)
    ok = q["beta"] < 50                                           # (away from the slivers, where everything is ill-conditioned)
    for p in (a, b, c):
        assert np.allclose(np.hypot(*(q["cc"] - p).T)[ok], q["r"][ok], rtol=1e-9)
    # L120: 2 beta = 1 / sin(alpha), alpha the smallest angle, here from the law of cosines
    la, lb, lc = np.hypot(*(b - c).T), np.hypot(*(a - c).T), np.hypot(*(a - b).T)
    s = np.sort(np.stack([la, lb, lc]), axis=0)
    alpha = np.arccos((s[1] ** 2 + s[2] ** 2 - s[0] ** 2) / (2 * s[1] * s[2]))   # opposite the shortest edge
    assert np.allclose(2 * q["beta"][ok], 1 / np.sin(alpha[ok]), rtol=1e-8)
    assert np.array_equal(q["bad"], ((q["r"] > 1.0) | (q["beta"] > 1.0)).astype(np.uint8))


def test_orient2d_is_exact():
    assert mg.orient2d((0, 0), (1, 0), (0, 1)) == 1 and mg.orient2d((0, 0), (0, 1), (1, 0)) == -1
    assert mg.orient2d((0, 0), (1, 1), (2, 2)) == 0 and mg.orient2d((0.1, 0.2), (0.2, 0.4), (0.3, 0.6)) == 0     # doubling is exact
    assert mg.orient2d((0.1, 0.3), (0.2, 0.6), (0.3, 0.9)) != 0   # the doubles nearest to 0.3, 0.6, 0.9 are not three times those nearest to 0.1, 0.2, 0.3
    # c one ulp above the diagonal through a and b: the determinant is 2^-53, far below the rounding error of a naive evaluation
    c = (0.5, 0.5 * (1 + 2.0 ** -52))
    assert mg.orient2d((0, 0), (1, 1), c) == 1 and mg.orient2d((0, 0), (1, 1), (c[1], c[0])) == -1
    big = 2.0 ** 40                                               # ... and with coordinates far from the origin
    assert mg.orient2d((big, big), (big + 1, big + 1), (big + 0.5, big + 0.5 + 2.0 ** -12)) == 1
    rng = np.random.default_rng(1)
    for _ in range(200):                                          # the symmetries of a determinant
        a, b, c = rng.random((3, 2))
        s = mg.orient2d(a, b, c)
        assert s == mg.orient2d(b, c, a) == mg.orient2d(c, a, b) == -mg.orient2d(b, a, c)
        assert s == np.sign((a[0] - c[0]) * (b[1] - c[1]) - (a[1] - c[1]) * (b[0] - c[0]))   # generic position: plain arithmetic agrees


def test_incircle2d_is_exact():
    a, b, c = (1.0, 0.0), (0.0, 1.0), (-1.0, 0.0)                 # counter-clockwise on the unit circle
    assert mg.incircle2d(a, b, c, (0.0, 0.0)) == 1 and mg.incircle2d(a, b, c, (2.0, 0.0)) == -1
    assert mg.incircle2d(a, b, c, (0.0, -1.0)) == 0               # four points of the unit circle
    assert mg.incircle2d((0, 0), (1, 0), (1, 1), (0, 1)) == 0     # the corners of a square (every cell of a uniform mesh)
    assert mg.incircle2d(a, b, c, (0.0, -1.0 + 2.0 ** -53)) == 1 and mg.incircle2d(a, b, c, (0.0, -1.0 - 2.0 ** -52)) == -1
    assert mg.incircle2d(a, c, b, (0.0, 0.0)) == -1               # clockwise (a, c, b): the sign flips
    rng = np.random.default_rng(2)
    for _ in range(200):
        p = rng.random((4, 2))
        if mg.orient2d(*p[:3]) < 0:
            p[[1, 2]] = p[[2, 1]]
        q = mg.test_quality(p, np.array([[0, 1, 2]], dtype=np.int32), 1.0, 1.0)
        inside = np.hypot(*(p[3] - q["cc"][0])) < q["r"][0]
        if abs(np.hypot(*(p[3] - q["cc"][0])) - q["r"][0]) > 1e-9 * q["r"][0]:
            assert mg.incircle2d(*p) == (1 if inside else -1)     # generic position: "inside the circumcircle" by distance
        assert mg.incircle2d(p[1], p[2], p[0], p[3]) == mg.incircle2d(*p) == -mg.incircle2d(p[1], p[0], p[2], p[3])
