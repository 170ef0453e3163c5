"""GPU parity on the seeded Delaunay workload: valence 3...12, 100:1 area ratio, frozen
boundary ring, ingested through the Triangle-format reader the way an externally generated mesh would be.
Tolerances as tests/test_gpu_parity.py."""
import os

import numpy as np
import pytest

import oracle
import workloads as wl
from helpers import field_errors

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mrd():
    import torch
    assert torch.cuda.is_available()
    import paper_1705_02028_b200 as m
    return m


@pytest.fixture(scope="module")
def ingested(tmp_path_factory):
    src = wl.delaunay_mesh(60000, seed=9)                            # ~120 k triangles: ~950 tiles, several per block
    stem = str(tmp_path_factory.mktemp("ext") / "sector")
    wl.write_triangle_files(src, stem, vertex_flag=src.boundary)
    mesh, flag = wl.read_triangle_files(stem)
    assert np.array_equal(mesh.xy, src.xy) and np.array_equal(mesh.tri, src.tri)
    return mesh, flag


@pytest.mark.parametrize("scheme,order,tile", [(2, 2, 0), (2, 2, 64), (2, 2, -1), (5, 2, 0), (0, 1, 0), (1, 2, 0)])
def test_delaunay_mesh_matches_oracle(mrd, ingested, scheme, order, tile):
    import torch
    mesh, flag = ingested
    W = wl.random_smooth_state(mesh, mach=0.5 if scheme == 1 else 0.8, seed=12)
    gm = mrd.Mesh(mesh.xy, mesh.tri, vertex_flag=flag, scheme=scheme, time_order=order, tile=tile)
    gm.set_state(torch.tensor(W, device="cuda"))
    om = oracle.OracleMesh(mesh.xy, mesh.tri, vertex_flag=flag, scheme=scheme, time_order=order, threads=os.cpu_count() or 1)
    om.set_state(W)
    g, o = gm.dump_stage1(), om.dump_stage1()
    scale = np.abs(o["phiN"]).max()
    for key in ("phiT", "phiN", "phiLDA", "phiB"):
        assert np.abs(g[key] - o[key]).max() <= 2e-13 * scale, key
    # (reading D2: a tile whose 128 Morton-consecutive triangles straddle a jump of the curve holds vertices far from its anchor,
    #  whose tile-frame coordinates are rounded to ulp(distance) -- up to ulp(L) / l_min ~ 2e-12 relative in an edge vector here)
    assert np.allclose(g["sT"], o["sT"], rtol=4e-12, atol=0)
    n, t, dt = gm.step(1)
    no, to, dto = om.step(1)
    assert n == 1 and abs(dt - dto) <= 1e-14 * dto
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= 1e-12
    gm.step(49)
    om.step(49)
    Wg = gm.get_state().cpu().numpy()
    assert field_errors(Wg, om.get_state()) <= 1e-9
    fr = flag.astype(bool)
    assert np.array_equal(Wg[:, fr], W[:, fr])


def test_delaunay_mesh_fp32_and_determinism(mrd, ingested):
    import torch
    mesh, flag = ingested
    W = wl.random_smooth_state(mesh, mach=0.8, seed=12)
    om = oracle.OracleMesh(mesh.xy, mesh.tri, vertex_flag=flag, threads=os.cpu_count() or 1)
    om.set_state(W)
    om.step(10)
    g32 = mrd.Mesh(mesh.xy, mesh.tri, vertex_flag=flag, precision=mrd.FP32)
    g32.set_state(torch.tensor(W, device="cuda", dtype=torch.float32))
    g32.step(10)
    assert field_errors(g32.get_state().cpu().numpy().astype(np.float64), om.get_state()) <= 1e-5
    runs = []
    for _ in range(2):
        gm = mrd.Mesh(mesh.xy, mesh.tri, vertex_flag=flag)
        gm.set_state(torch.tensor(W, device="cuda"))
        gm.step(25)
        runs.append(gm.get_state().cpu().numpy())
    assert np.array_equal(runs[0], runs[1])
