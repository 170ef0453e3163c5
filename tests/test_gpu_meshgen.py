"""GPU parity of the mesh-generation slice: TestQuality bit for bit against the oracle, and
the exact predicates ORIENT2D / INCIRCLE2D sign for sign against the oracle's rational arithmetic -- on seeded point sets:
a Delaunay mesh, random index tuples, and the degenerate inputs the paper warns about (L162-L166: exactly collinear and
cocircular points of a uniform grid, points one ulp off a line or circle, coordinates far from the origin)."""
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


def test_test_quality_is_bitwise_the_oracle(mrdb):
    import torch
    mesh = wl.delaunay_mesh(20000, seed=6)
    for R, B in [(0.05, 1.0), (1e9, np.sqrt(2.0)), (0.02, 0.8)]:
        g = mrdb.meshgen_test_quality(dev(mesh.xy, torch.float64), dev(mesh.tri, torch.int32), R, B)
        o = mg.test_quality(mesh.xy, mesh.tri, R, B)
        assert np.array_equal(g["r"].cpu().numpy(), o["r"]) and np.array_equal(g["beta"].cpu().numpy(), o["beta"])
        assert np.array_equal(g["cc"].cpu().numpy(), o["cc"]) and np.array_equal(g["bad"].cpu().numpy(), o["bad"])
        assert g["n_bad"] == int(o["bad"].sum()) and 0 < g["n_bad"] < mesh.nt
    # a clockwise triangle and a zero-area one are flagged
    xy = np.array([[0.0, 0.0], [1.0, 0.0], [0.0, 1.0], [2.0, 0.0]])
    tri = np.array([[0, 2, 1], [0, 1, 3], [0, 1, 2]], dtype=np.int32)
    g = mrdb.meshgen_test_quality(dev(xy, torch.float64), dev(tri, torch.int32), 10.0, 10.0)
    assert g["bad"].cpu().numpy().tolist() == [1, 1, 0] and g["n_bad"] == 2


def point_sets():
    rng = np.random.default_rng(11)
    out = {}
    out["random"] = rng.random((400, 2)) * 4.0 - 2.0
    gi, gj = np.meshgrid(np.arange(12), np.arange(12))
    grid = np.stack([gi.ravel(), gj.ravel()], axis=1) / 8.0       # exactly representable: collinear / cocircular tuples abound
    out["grid"] = grid
    near = grid.copy()                                             # every point one or two ulps off its grid position
    near += np.spacing(np.abs(near) + 0.125) * rng.integers(-2, 3, size=near.shape)
    out["near_grid"] = near
    out["far"] = near + 2.0 ** 30                                  # the same configuration far from the origin
    out["delaunay"] = wl.delaunay_mesh(300, seed=3).xy
    return out


@pytest.mark.parametrize("name", ["random", "grid", "near_grid", "far", "delaunay"])
def test_orient2d_and_incircle2d_are_exact(mrdb, name):
    import torch
    xy = point_sets()[name]
    rng = np.random.default_rng(5)
    n = 1500
    i3 = rng.integers(0, len(xy), size=(n, 3)).astype(np.int32)
    i4 = rng.integers(0, len(xy), size=(n, 4)).astype(np.int32)
    i3[:50, 2] = i3[:50, 0]                                        # repeated points: exactly zero
    i4[:50, 3] = i4[:50, 1]
    if name in ("grid", "near_grid", "far"):                       # three points of one grid row, four corners of a grid rectangle
        row = rng.integers(0, 12, size=300)
        cols = np.stack([rng.permutation(12)[:3] for _ in range(300)])
        i3[50:350] = (row[:, None] * 12 + cols).astype(np.int32)
        r0, c0 = rng.integers(0, 8, size=300), rng.integers(0, 8, size=300)
        dr, dc = rng.integers(1, 4, size=300), rng.integers(1, 4, size=300)
        i4[50:350] = np.stack([r0 * 12 + c0, r0 * 12 + c0 + dc, (r0 + dr) * 12 + c0 + dc, (r0 + dr) * 12 + c0], axis=1).astype(np.int32)
    s3, e3 = mrdb.meshgen_orient2d(dev(xy, torch.float64), dev(i3, torch.int32))
    s4, e4 = mrdb.meshgen_incircle2d(dev(xy, torch.float64), dev(i4, torch.int32))
    s3, s4 = s3.cpu().numpy(), s4.cpu().numpy()
    o3 = np.array([mg.orient2d(xy[a], xy[b], xy[c]) for a, b, c in i3], dtype=np.int8)
    o4 = np.array([mg.incircle2d(xy[a], xy[b], xy[c], xy[d]) for a, b, c, d in i4], dtype=np.int8)
    assert np.array_equal(s3, o3) and np.array_equal(s4, o4)
    assert set(np.unique(s3)) <= {-1, 0, 1} and set(np.unique(s4)) <= {-1, 0, 1}
    if name in ("grid", "near_grid", "far"):
        assert e3 > 50 and e4 > 50                                 # the filter gave up on the degenerate tuples: the exact path ran
        assert (o3 == 0).sum() >= 50 and (o4 == 0).sum() >= 50
    if name == "random":
        assert e3 <= 100 and e4 <= 100                             # ... and on little else than the 50 repeated points in general position


def test_predicates_on_the_edges_of_a_mesh(mrdb):
    """The use the refinement makes of them (L170, L194-L200): every triangle of the Delaunay mesh is counter-clockwise, and no
    vertex opposite an interior edge lies inside the circumcircle of the triangle on the other side (the mesh IS Delaunay)."""
    import torch
    mesh = wl.delaunay_mesh(4000, seed=8)
    # (the mesh is Delaunay in the PARAMETER square; the conformal map to physical space keeps circles only infinitesimally)
    tri = mesh.tri
    s3, _ = mrdb.meshgen_orient2d(dev(mesh.xy, torch.float64), dev(tri, torch.int32))
    assert (s3.cpu().numpy() == 1).all()
    e = np.concatenate([tri[:, [0, 1, 2]], tri[:, [1, 2, 0]], tri[:, [2, 0, 1]]])          # directed edge (a, b), opposite vertex c
    key = e[:, 0].astype(np.int64) * mesh.nv + e[:, 1]
    rkey = e[:, 1].astype(np.int64) * mesh.nv + e[:, 0]
    order = np.argsort(key)
    pos = np.minimum(np.searchsorted(key[order], rkey), len(key) - 1)
    mate = order[pos]
    has = key[mate] == rkey
    quads = np.stack([e[has, 0], e[has, 1], e[has, 2], e[mate[has], 2]], axis=1).astype(np.int32)   # (a, b, c) ccw, d across edge ab
    s4, _ = mrdb.meshgen_incircle2d(dev(mesh.xy, torch.float64), dev(quads, torch.int32))
    s4 = s4.cpu().numpy()
    o4 = np.array([mg.incircle2d(*mesh.xy[q]) for q in quads[:600]], dtype=np.int8)
    assert np.array_equal(s4[:600], o4)
    assert (s4 > 0).mean() < 0.05        # locally Delaunay almost everywhere (exactly so before the conformal map bends the circles)
