"""Synthetic meshes: uniform vertex grids with every square split along the same diagonal
(eq. 1 / Fig. 1), periodic or bounded, plus seeded renumberings.

Mesh format = the paper's first two mesh arrays:
`xy` float64 [nv][2] (vertexCoordinates) and `tri` int32 [nt][3] (triangleVertices, CCW).
Periodic meshes hold each unique vertex once, coordinates in [0, period).
No arithmetic of the hydrodynamics method lives here.
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import numpy as np


@dataclass
class UniformMesh:
    xy: np.ndarray          # [nv][2] float64
    tri: np.ndarray         # [nt][3] int32, counter-clockwise
    period: tuple           # (px, py); 0.0 = bounded in that direction
    grid_ij: np.ndarray     # [nv][2] int64: grid index (i, j) of each vertex (keys PRNG / BC helpers)
    shape: tuple            # (nvx, nvy) unique vertices per direction
    cells: tuple            # (ncx, ncy)
    lengths: tuple          # (Lx, Ly)

    @property
    def nv(self) -> int:
        return int(self.xy.shape[0])

    @property
    def nt(self) -> int:
        return int(self.tri.shape[0])


def uniform_mesh(ncx: int, ncy: int, Lx: float = 1.0, Ly: float = 1.0, periodic: bool = True) -> UniformMesh:
    """ncx x ncy squares on [0,Lx] x [0,Ly], each split along its SW-NE diagonal into two CCW
    triangles; natural (row-major) vertex numbering, triangles numbered cell by cell.

    periodic=True : ncx*ncy unique vertices (the last row/column are periodic images).
    periodic=False: (ncx+1)*(ncy+1) vertices.
    """
    nvx, nvy = (ncx, ncy) if periodic else (ncx + 1, ncy + 1)
    hx, hy = Lx / ncx, Ly / ncy
    jj, ii = np.meshgrid(np.arange(nvy, dtype=np.int64), np.arange(nvx, dtype=np.int64), indexing="ij")
    ii = ii.ravel()
    jj = jj.ravel()
    xy = np.stack([ii * hx, jj * hy], axis=1).astype(np.float64)
    grid_ij = np.stack([ii, jj], axis=1)

    cj, ci = np.meshgrid(np.arange(ncy, dtype=np.int64), np.arange(ncx, dtype=np.int64), indexing="ij")
    ci = ci.ravel()
    cj = cj.ravel()
    if periodic:
        ip, jp = (ci + 1) % ncx, (cj + 1) % ncy
    else:
        ip, jp = ci + 1, cj + 1
    v00 = cj * nvx + ci
    v10 = cj * nvx + ip
    v01 = jp * nvx + ci
    v11 = jp * nvx + ip
    tri = np.empty((2 * ncx * ncy, 3), dtype=np.int32)
    tri[0::2] = np.stack([v00, v10, v11], axis=1)   # lower-right triangle, CCW
    tri[1::2] = np.stack([v00, v11, v01], axis=1)   # upper-left triangle, CCW
    period = (float(Lx), float(Ly)) if periodic else (0.0, 0.0)
    return UniformMesh(xy, tri, period, grid_ij, (nvx, nvy), (ncx, ncy), (float(Lx), float(Ly)))


def _renumber(mesh: UniformMesh, vorder: np.ndarray, torder: np.ndarray, rot: np.ndarray | None):
    """new vertex k = old vertex vorder[k]; new triangle k = old triangle torder[k]."""
    rank = np.empty(mesh.nv, dtype=np.int64)
    rank[vorder] = np.arange(mesh.nv, dtype=np.int64)
    tri = rank[mesh.tri.astype(np.int64)][torder]
    if rot is not None:
        cols = (np.arange(3)[None, :] + rot[:, None]) % 3     # cyclic shift keeps CCW
        tri = np.take_along_axis(tri, cols, axis=1)
    new = replace(mesh, xy=np.ascontiguousarray(mesh.xy[vorder]), tri=np.ascontiguousarray(tri.astype(np.int32)),
                  grid_ij=np.ascontiguousarray(mesh.grid_ij[vorder]))
    return new, vorder, torder


def permute_mesh(mesh: UniformMesh, seed: int = 12345):
    """Seeded random renumbering of vertices and triangles plus a seeded cyclic rotation of
    each triangle's local node order (config 3 / config 5b). Returns (mesh, vorder, torder):
    new vertex k is old vertex vorder[k] (so a per-vertex field f becomes f[..., vorder])."""
    rng = np.random.default_rng(seed)
    vorder = rng.permutation(mesh.nv)
    torder = rng.permutation(mesh.nt)
    rot = rng.integers(0, 3, size=mesh.nt)
    return _renumber(mesh, vorder, torder, rot)


def _interleave16(a: np.ndarray) -> np.ndarray:
    a = a.astype(np.uint64) & np.uint64(0xFFFF)
    a = (a | (a << np.uint64(8))) & np.uint64(0x00FF00FF)
    a = (a | (a << np.uint64(4))) & np.uint64(0x0F0F0F0F)
    a = (a | (a << np.uint64(2))) & np.uint64(0x33333333)
    a = (a | (a << np.uint64(1))) & np.uint64(0x55555555)
    return a


def morton_order_mesh(mesh: UniformMesh):
    """Input numbering along a Z-order curve of the grid index (config 5a "Morton-ordered input").
    This is an INPUT ordering; the library's own layout stage is separate and independent."""
    gi, gj = mesh.grid_ij[:, 0], mesh.grid_ij[:, 1]
    vkey = _interleave16(gi) | (_interleave16(gj) << np.uint64(1))
    vorder = np.argsort(vkey, kind="stable")
    # triangle key: Morton key of the owning cell, then parity (uniform_mesh numbers the two
    # triangles of cell c as 2c and 2c+1, so this needs the mesh in its creation order)
    ncx = mesh.cells[0]
    cell = np.arange(mesh.nt, dtype=np.int64) // 2
    ci, cj = cell % ncx, cell // ncx
    tkey = ((_interleave16(ci) | (_interleave16(cj) << np.uint64(1))) << np.uint64(1)) | (
        np.arange(mesh.nt, dtype=np.uint64) & np.uint64(1))
    torder = np.argsort(tkey, kind="stable")
    return _renumber(mesh, vorder, torder, None)


def jitter_mesh(mesh: UniformMesh, amplitude: float = 0.25, seed: int = 7) -> UniformMesh:
    """Move every vertex by a seeded uniform offset of at most `amplitude` cell widths in x and y
    (amplitude <= 0.25 keeps every triangle of the SW-NE split positively oriented: a corner and the opposite side
    can each move 0.25 sqrt 2 cell widths towards each other, together the 0.707 between them; 0.3 already turns about one
    triangle in 10^4 over).
    Gives non-uniform triangle shapes/areas for pins and parity on "genuinely unstructured" geometry.
    Boundary vertices of bounded meshes are only moved along their boundary."""
    rng = np.random.default_rng(seed)
    hx, hy = mesh.lengths[0] / mesh.cells[0], mesh.lengths[1] / mesh.cells[1]
    d = (rng.random((mesh.shape[1], mesh.shape[0], 2)) * 2.0 - 1.0) * amplitude
    gi, gj = mesh.grid_ij[:, 0], mesh.grid_ij[:, 1]
    off = d[gj, gi] * np.array([hx, hy])
    if mesh.period[0] == 0.0:
        on_x = (gi == 0) | (gi == mesh.shape[0] - 1)
        off[on_x, 0] = 0.0
    if mesh.period[1] == 0.0:
        on_y = (gj == 0) | (gj == mesh.shape[1] - 1)
        off[on_y, 1] = 0.0
    xy = mesh.xy + off
    if mesh.period[0] > 0.0:
        xy[:, 0] = np.mod(xy[:, 0], mesh.period[0])
    if mesh.period[1] > 0.0:
        xy[:, 1] = np.mod(xy[:, 1], mesh.period[1])
    return replace(mesh, xy=np.ascontiguousarray(xy))


def flip_edges(mesh: UniformMesh, fraction: float = 0.35, seed: int = 11, rounds: int = 2) -> UniformMesh:
    """Variable-valence triangulation (stand-in for the paper's Delaunay-refined meshes, L685, which are not in
    the container): flip a seeded random set of interior edges.  Edge ab shared by the CCW triangles (a,b,c) and
    (b,a,d) becomes edge cd, giving (a,d,c) and (d,b,c); it is flipped only if both new triangles keep a
    positive area of at least 15 % of the mean (strictly convex quadrilateral).  Per round every edge is a
    candidate with probability `fraction`, and a candidate is taken when it has the highest random priority among
    the candidates of both its triangles (so no triangle is flipped twice in a round).  Vertices a, b lose one
    incident triangle, c, d gain one: valences spread from 6 to about 4...9.  Vertex numbering, coordinates and
    boundary edges are unchanged (bounded meshes keep their wall edges and frozen vertices)."""
    rng = np.random.default_rng(seed)
    tri = mesh.tri.astype(np.int64).copy()
    nt = tri.shape[0]
    px, py = mesh.period

    def unwrap(d, period):
        return d - period * np.round(d / period) if period > 0.0 else d

    def area2(a, b, c):
        abx, aby = unwrap(mesh.xy[b, 0] - mesh.xy[a, 0], px), unwrap(mesh.xy[b, 1] - mesh.xy[a, 1], py)
        acx, acy = unwrap(mesh.xy[c, 0] - mesh.xy[a, 0], px), unwrap(mesh.xy[c, 1] - mesh.xy[a, 1], py)
        return abx * acy - aby * acx

    amin = 0.15 * float(np.mean(area2(tri[:, 0], tri[:, 1], tri[:, 2])))
    for _ in range(rounds):
        # directed edges (a -> b) of every triangle with the opposite vertex; pair a->b with b->a
        t_id = np.repeat(np.arange(nt), 3)
        k = np.tile(np.arange(3), nt)
        a, b, c = tri[t_id, k], tri[t_id, (k + 1) % 3], tri[t_id, (k + 2) % 3]
        key = a * mesh.nv + b
        rkey = b * mesh.nv + a
        order = np.argsort(key)
        pos = np.searchsorted(key[order], rkey)
        pos = np.minimum(pos, len(key) - 1)
        mate = order[pos]
        has = (key[mate] == rkey) & (a < b)               # interior edge, counted once
        e1 = np.nonzero(has)[0]
        e2 = mate[e1]
        A, B, Cc, D = a[e1], b[e1], c[e1], c[e2]
        T1, T2 = t_id[e1], t_id[e2]
        ok = (area2(A, D, Cc) > amin) & (area2(D, B, Cc) > amin) & (rng.random(len(e1)) < fraction)
        prio = rng.random(len(e1)) + 1.0
        prio[~ok] = 0.0
        best = np.zeros(nt)
        np.maximum.at(best, T1, prio)
        np.maximum.at(best, T2, prio)
        take = ok & (prio == best[T1]) & (prio == best[T2])
        tri[T1[take]] = np.stack([A[take], D[take], Cc[take]], axis=1)
        tri[T2[take]] = np.stack([D[take], B[take], Cc[take]], axis=1)
    return replace(mesh, tri=np.ascontiguousarray(tri.astype(np.int32)))


def scrambled_triangulation(ncx: int, ncy: int, seed: int = 1, amplitude: float = 0.25, rounds: int = 3, Lx: float = 2.0,
                            Ly: float = 1.5) -> UniformMesh:
    """Input of the Delaunay triangulator (section 2.4.6): a VALID but far-from-Delaunay triangulation of points in
    general position inside a rectangle -- a jittered ncx x ncy-cell grid (boundary vertices slide along the boundary, so the
    hull stays the rectangle and the Delaunay triangulation of the points is the triangulation of the domain), then `rounds`
    rounds of seeded flips of strictly convex quadrilaterals (every second edge a candidate)."""
    if not 0.0 <= amplitude <= 0.25:
        raise ValueError("scrambled_triangulation: amplitude beyond 0.25 cell widths can turn triangles over (not a valid triangulation)")
    m = jitter_mesh(uniform_mesh(ncx, ncy, Lx, Ly, periodic=False), amplitude, seed=seed)
    return flip_edges(m, fraction=0.5, seed=seed + 1, rounds=rounds)


def boundary_vertices(mesh: UniformMesh, x_ends: bool = True, y_ends: bool = True) -> np.ndarray:
    """uint8 [nv] flag: 1 on the requested boundary rows/columns of a bounded mesh (PAPER.md L582:
    boundary vertices promoted to ghost vertices that keep the initial condition)."""
    gi, gj = mesh.grid_ij[:, 0], mesh.grid_ij[:, 1]
    f = np.zeros(mesh.nv, dtype=np.uint8)
    if x_ends and mesh.period[0] == 0.0:
        f |= ((gi == 0) | (gi == mesh.shape[0] - 1)).astype(np.uint8)
    if y_ends and mesh.period[1] == 0.0:
        f |= ((gj == 0) | (gj == mesh.shape[1] - 1)).astype(np.uint8)
    return f


def wall_edges_y(mesh: UniformMesh) -> np.ndarray:
    """int32 [ne][2]: vertex pairs of the mesh edges lying on the bottom (j=0) and top
    (j=nvy-1) rows of a mesh bounded in y (reflecting walls of the 2D Sod tube, config 2)."""
    assert mesh.period[1] == 0.0
    nvx, nvy = mesh.shape
    rank = np.full((nvy, nvx), -1, dtype=np.int64)
    rank[mesh.grid_ij[:, 1], mesh.grid_ij[:, 0]] = np.arange(mesh.nv)
    nseg = mesh.cells[0]
    i0 = np.arange(nseg)
    i1 = (i0 + 1) % nvx if mesh.period[0] > 0.0 else i0 + 1
    bot = np.stack([rank[0, i0], rank[0, i1]], axis=1)
    top = np.stack([rank[nvy - 1, i0], rank[nvy - 1, i1]], axis=1)
    return np.ascontiguousarray(np.concatenate([bot, top], axis=0).astype(np.int32))


def delaunay_mesh(n_points: int = 20000, seed: int = 1, grading: float = 10.0) -> UniformMesh:
    """A genuinely unstructured, bounded triangulation (stand-in for the paper's Delaunay meshes, which are
    not in the container): the Delaunay triangulation (scipy.spatial.Delaunay, i.e. Qhull) of seeded random points.

    Points: one uniformly random point in every cell of an m x m stratification of the parameter square (m^2 ~ n_points;
    valences 3...12, no two triangles alike), plus a ring of points ON the four sides (the boundary vertices, returned as
    flag 1 by `boundary_vertices`).  The triangulation is made in the parameter square and then carried to physical space
    by the conformal map w = exp(c (u + i v)), c = ln(grading): angles are kept, lengths grow by e^{c u}, so that the
    largest triangles have ~grading^2 times the area of the smallest (100:1 by default) -- non-uniform V_i, an annular-
    sector domain.  `grid_ij`, `shape`, `cells` are None: nothing here is a grid."""
    rng = np.random.default_rng(seed)
    m = max(4, int(round(np.sqrt(n_points))))
    jj, ii = np.meshgrid(np.arange(m), np.arange(m), indexing="ij")
    u = (ii + rng.random((m, m))) / m
    v = (jj + rng.random((m, m))) / m
    # keep the interior points a quarter of a cell away from the sides, so that the ring below IS the boundary
    pad = 0.25 / m
    u, v = np.clip(u, pad, 1.0 - pad).ravel(), np.clip(v, pad, 1.0 - pad).ravel()
    s = (np.arange(m) + 0.5) / m
    ring = np.concatenate([
        np.stack([s, np.zeros(m)], axis=1), np.stack([s, np.ones(m)], axis=1),
        np.stack([np.zeros(m), s], axis=1), np.stack([np.ones(m), s], axis=1),
        np.array([[0.0, 0.0], [1.0, 0.0], [0.0, 1.0], [1.0, 1.0]])])
    uv = np.concatenate([np.stack([u, v], axis=1), ring], axis=0)
    from scipy.spatial import Delaunay
    tri = Delaunay(uv).simplices.astype(np.int64)
    # drop the slivers Qhull makes of (nearly) collinear boundary points
    a, b, c = uv[tri[:, 0]], uv[tri[:, 1]], uv[tri[:, 2]]
    area = 0.5 * ((b[:, 0] - a[:, 0]) * (c[:, 1] - a[:, 1]) - (b[:, 1] - a[:, 1]) * (c[:, 0] - a[:, 0]))
    tri = tri[np.abs(area) > 1e-12 / (m * m)]
    area = area[np.abs(area) > 1e-12 / (m * m)]
    tri[area < 0] = tri[area < 0][:, [0, 2, 1]]                      # counter-clockwise
    cgr = np.log(grading)
    w = np.exp(cgr * (uv[:, 0] + 1j * uv[:, 1]))
    xy = np.ascontiguousarray(np.stack([w.real, w.imag], axis=1))
    xy -= xy.min(axis=0)
    lengths = tuple(float(x) for x in xy.max(axis=0))
    mesh = UniformMesh(xy, np.ascontiguousarray(tri.astype(np.int32)), (0.0, 0.0), None, None, None, lengths)
    mesh.boundary = np.zeros(len(xy), dtype=np.uint8)
    mesh.boundary[len(u):] = 1
    return mesh


def write_triangle_files(mesh: UniformMesh, stem: str, vertex_flag=None) -> None:
    """Write `stem.node` / `stem.ele` in the ASCII format of the mesh generator Triangle (vertices with one boundary
    marker, triangles by 1-based vertex number): the ingest format for externally generated meshes."""
    flag = np.zeros(mesh.nv, dtype=np.int64) if vertex_flag is None else np.asarray(vertex_flag, dtype=np.int64)
    with open(stem + ".node", "w") as f:
        f.write(f"{mesh.nv} 2 0 1\n")
        for k in range(mesh.nv):
            f.write(f"{k + 1} {float(mesh.xy[k, 0])!r} {float(mesh.xy[k, 1])!r} {flag[k]}\n")
    with open(stem + ".ele", "w") as f:
        f.write(f"{mesh.nt} 3 0\n")
        for k in range(mesh.nt):
            f.write(f"{k + 1} {mesh.tri[k, 0] + 1} {mesh.tri[k, 1] + 1} {mesh.tri[k, 2] + 1}\n")


def read_triangle_files(stem: str):
    """Read a mesh written by an external generator in Triangle's `.node` / `.ele` format (comments `#`, 0- or 1-based
    numbering, optional attributes; 3-node triangles).  Returns (mesh, vertex_flag) with the boundary markers as flags
    (non-zero marker -> 1), ready for `Mesh(mesh.xy, mesh.tri, vertex_flag=...)`."""
    def rows(path):
        with open(path) as f:
            for line in f:
                line = line.split("#", 1)[0].split()
                if line:
                    yield line
    it = rows(stem + ".node")
    nv, dim, nattr, nmark = (int(x) for x in next(it))
    assert dim == 2
    ids, xy, flag = np.empty(nv, dtype=np.int64), np.empty((nv, 2)), np.zeros(nv, dtype=np.uint8)
    for k in range(nv):
        r = next(it)
        ids[k] = int(r[0])
        xy[k] = float(r[1]), float(r[2])
        if nmark:
            flag[k] = 1 if int(r[3 + nattr]) != 0 else 0
    base = int(ids.min())
    assert np.array_equal(ids, np.arange(base, base + nv)), "vertices must be numbered consecutively"
    it = rows(stem + ".ele")
    nt, nodes = (int(x) for x in next(it)[:2])
    assert nodes == 3, "3-node triangles only"
    tri = np.empty((nt, 3), dtype=np.int32)
    for k in range(nt):
        r = next(it)
        tri[k] = int(r[1]) - base, int(r[2]) - base, int(r[3]) - base
    xy = np.ascontiguousarray(xy)
    lo = xy.min(axis=0)
    lengths = tuple(float(x) for x in (xy.max(axis=0) - lo))
    mesh = UniformMesh(xy, np.ascontiguousarray(tri), (0.0, 0.0), None, None, None, lengths)
    mesh.boundary = flag
    return mesh, flag


def uniform_strip_part(n: int, world: int, rank: int, L: float = 10.0):
    """The pieces of ONE part of the N-GPU bench workload, made without the whole mesh: the periodic strip of `world` squares
    of n x n cells stacked in y (`uniform_mesh(n, n * world, L, L * world, periodic=True)`, natural numbering), cut into
    the `world` row bands of n vertex rows.  Returns a dict with what `Partition.from_local` takes: the band's n rows plus the
    row below and the row above (the vertices of every triangle that touches the band), their global ids and owners, and the
    n + 1 rows of cells between them -- (n + 2) n vertices and 2 (n + 1) n triangles however large `world` is."""
    assert world >= 2 and n >= 3
    nvy = n * world
    h = L / n
    j0 = rank * n
    rows = (np.arange(j0 - 1, j0 + n + 1, dtype=np.int64)) % nvy            # global vertex row of each local row
    ii = np.arange(n, dtype=np.int64)
    gid = (rows[:, None] * n + ii[None, :]).ravel()
    owner = np.repeat(rows // n, n)
    xy = np.stack([np.tile(ii * h, n + 2), np.repeat(rows * h, n)], axis=1).astype(np.float64)
    lc, ci = np.meshgrid(np.arange(n + 1, dtype=np.int64), ii, indexing="ij")  # local cell row, column
    lc, ci = lc.ravel(), ci.ravel()
    ip = (ci + 1) % n
    v00, v10, v01, v11 = lc * n + ci, lc * n + ip, (lc + 1) * n + ci, (lc + 1) * n + ip
    tri = np.empty((2 * (n + 1) * n, 3), dtype=np.int32)
    tri[0::2] = np.stack([v00, v10, v11], axis=1)
    tri[1::2] = np.stack([v00, v11, v01], axis=1)
    cell = rows[lc] * n + ci                                                  # global cell = global row of its lower vertices
    tri_global = np.empty(2 * (n + 1) * n, dtype=np.int64)
    tri_global[0::2], tri_global[1::2] = 2 * cell, 2 * cell + 1
    return dict(n_vertex_global=n * nvy, n_triangle_global=2 * n * nvy, vertex_global=gid.astype(np.int32), owner=owner.astype(np.int32),
                xy=np.ascontiguousarray(xy), tri=tri, tri_global=tri_global.astype(np.int32), period=(float(L), float(L * world)),
                domain_size=float(L * world), local_rows=rows % n)
