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
    (amplitude < 0.5 keeps all triangles positively oriented for the SW-NE split when < ~0.3).
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
