"""Parity of the tile kernels WITHOUT the geometry table (`tile_kernel<..., GTAB = false>`: every jittered or flipped
mesh) at a size where the persistent loop iterates: 512^2 vertices = 524 288 triangles = 2048 tiles of 256 (the default;
4096 of 128, 8192 of 64) on a grid of 148 x 1024 / tile blocks, so every block refills its buffers several times, uses the second buffer and
flips the mbarrier phase (mrd_tile.cuh: the "last warp out refills" branch and the parity `(k >> 1) & 1`).  The small
meshes of tests/test_gpu_parity.py give every block exactly one tile and never reach those branches.
Shape: the paper's unstructured periodic mesh, scaled down; SURVEY 8(f2).
Tolerances: north_star / DESIGN.md section 6 (1e-12 of the largest nodal residual per triangle -- see the note in the
test --, 1e-12 after one step, 1e-9 after 50 free-running steps; fp32 1e-5 after 10 steps against the fp64 oracle)."""
import os

import numpy as np
import pytest

import oracle
import workloads as wl
from helpers import field_errors

pytestmark = pytest.mark.gpu

N = 512
THREADS = os.cpu_count() or 1


@pytest.fixture(scope="module")
def mrd():
    import torch
    assert torch.cuda.is_available()
    import paper_1705_02028_b200 as m
    return m


_cache = {}


def big_mesh(kind):
    """jitter: every triangle has its own shape; flip: also variable valence (3...12); bounded: non-periodic with a
    frozen boundary ring (the frozen flag and ragged boundary tiles inside an iterating block)."""
    if kind not in _cache:
        if kind == "bounded":
            mesh = wl.jitter_mesh(wl.uniform_mesh(N, N - 37, 3.0, 2.7, periodic=False), 0.2, seed=5)
            mesh = wl.flip_edges(mesh, seed=13)
            flag = wl.boundary_vertices(mesh)
        else:
            mesh = wl.jitter_mesh(wl.uniform_mesh(N, N, 2.0, 2.0, periodic=True), 0.2, seed=7)
            if kind == "flip":
                mesh = wl.flip_edges(mesh, seed=11)
            flag = None
        W = wl.random_smooth_state(mesh, mach=0.8, seed=6)
        _cache[kind] = (mesh, flag, W)
    return _cache[kind]


def make_pair(mrd, kind, **kw):
    import torch
    mesh, flag, W = big_mesh(kind)
    okw = {k: v for k, v in kw.items() if k in ("scheme", "time_order")}
    gm = mrd.Mesh(mesh.xy, mesh.tri, vertex_flag=flag, period=mesh.period, **kw)
    dt = torch.float64 if kw.get("precision", 0) == 0 else torch.float32
    gm.set_state(torch.tensor(W, dtype=dt, device="cuda"))
    om = oracle.OracleMesh(mesh.xy, mesh.tri, vertex_flag=flag, period=mesh.period, threads=THREADS, **okw)
    om.set_state(W)
    return mesh, flag, W, gm, om


@pytest.mark.parametrize("scheme", [2, 5])             # B, Bx
@pytest.mark.parametrize("tile", [0, 64, 128])
@pytest.mark.parametrize("kind", ["jitter", "flip", "bounded"])
def test_non_table_tile_path_where_the_persistent_loop_iterates(mrd, kind, tile, scheme):
    import torch
    mesh, flag, W, gm, om = make_pair(mrd, kind, tile=tile, scheme=scheme)
    lay = mrd.Layout(mesh.xy, mesh.tri, vertex_flag=flag, period=mesh.period, tile=tile)
    assert lay.ntile >= 1850                            # >= 3 tiles per block on any grid the launcher can pick (<= 148 x 1024 / tile blocks)
    if kind != "jitter":
        val = np.bincount(mesh.tri.ravel(), minlength=mesh.nv)
        assert val.max() >= 9 and val.min() <= 4
    g, o = gm.dump_stage1(), om.dump_stage1()
    scale = np.abs(o["phiN"]).max()
    # Tolerance: the kernels compute the geometry from coordinates in the TILE's frame (exact differences), the oracle from
    # absolute coordinates after re-adding the first vertex (reading C19), which costs it up to ulp(L) per coordinate for
    # triangles across a periodic seam -- a relative difference of ulp(L)/l_min ~ 2e-13 in edge vectors at this resolution
    # (reading D2; measured 1e-13 in s_T, 9e-14 in the residuals).  Hence 1e-12 where the small meshes use 2e-13 / 1e-14.
    for key in ("phiT", "phiN", "phiLDA", "phiB"):
        assert np.abs(g[key] - o[key]).max() <= 1e-12 * scale, key
    assert np.allclose(g["sT"], o["sT"], rtol=1e-12, atol=0)
    n, t, dt = gm.step(1)
    no, to, dto = om.step(1)
    assert n == 1 and abs(dt - dto) <= 1e-14 * dto
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= 1e-12
    gm.step(49)
    om.step(49)
    Wg = gm.get_state().cpu().numpy()
    assert field_errors(Wg, om.get_state()) <= 1e-9
    if flag is not None:
        fr = flag.astype(bool)
        assert np.array_equal(Wg[:, fr], W[:, fr])
    else:
        _, vol = om.geometry()
        tot0 = (W * vol[None, :]).sum(axis=1)
        tot = gm.diagnostics()[0]
        assert np.abs(tot - tot0).max() <= 1e-12 * np.abs(tot0).max()
    # bitwise rerun determinism of the iterating path (C20)
    g2 = mrd.Mesh(mesh.xy, mesh.tri, vertex_flag=flag, period=mesh.period, tile=tile, scheme=scheme)
    g2.set_state(torch.tensor(W, device="cuda"))
    g2.step(50)
    assert np.array_equal(g2.get_state().cpu().numpy(), Wg)


@pytest.mark.parametrize("tile", [0, 64])
@pytest.mark.parametrize("kind", ["jitter", "flip", "bounded"])
def test_non_table_tile_path_fp32(mrd, kind, tile):
    mesh, flag, W, g32, om = make_pair(mrd, kind, tile=tile, precision=1)
    g32.step(10)
    om.step(10)
    assert field_errors(g32.get_state().cpu().numpy().astype(np.float64), om.get_state()) <= 1e-5


@pytest.mark.parametrize("scheme,order", [(0, 1), (1, 2), (3, 2)])       # N1, LDA2, Bmax2 on the flipped mesh
def test_non_table_tile_path_other_schemes(mrd, scheme, order):
    mesh, flag, W, gm, om = make_pair(mrd, "flip", scheme=scheme, time_order=order)
    gm.step(1)
    om.step(1)
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= 1e-12
    gm.step(29)
    om.step(29)
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= 1e-9
