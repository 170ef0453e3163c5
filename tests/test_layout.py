"""Host logic of the CUDA path that needs no GPU: the C-ABI library loads and exports every symbol
of include/mrd.h, and the mesh-layout stage is a pure relabelling with a correct
vertex->triangle CSR, geometry equal to the oracle's, and a consistent tile plan."""
import ctypes as C

import numpy as np
import pytest

import oracle
import paper_1705_02028_b200 as mrd
import workloads as wl


def test_library_exports_every_declared_symbol():
    L = mrd.lib()
    names = mrd.exported_symbols()
    assert {"mrd_mesh_create", "mrd_set_state", "mrd_step", "mrd_get_state"} <= set(names)
    assert len(names) >= 20
    for n in names:
        assert hasattr(L, n), n
    assert "sm_100a" in mrd.version()


def test_params_struct_matches_header_size():
    # 2 doubles + 4 int32 + 2 doubles + 2 int32 + 1 double (domain_size)
    assert C.sizeof(mrd.Params) == 16 + 16 + 16 + 8 + 8


MESHES = {
    "periodic_natural": lambda: wl.uniform_mesh(16, 12, 4.0, 3.0, periodic=True),
    "periodic_permuted": lambda: wl.permute_mesh(wl.uniform_mesh(16, 16, 1.0, 1.0, periodic=True), 3)[0],
    "periodic_jitter": lambda: wl.jitter_mesh(wl.uniform_mesh(20, 10, 2.0, 1.0, periodic=True), 0.2, seed=2),
    "bounded": lambda: wl.uniform_mesh(9, 7, 1.0, 0.5, periodic=False),
    "bounded_permuted": lambda: wl.permute_mesh(wl.uniform_mesh(13, 5, 1.0, 0.5, periodic=False), 9)[0],
}


@pytest.mark.parametrize("name", sorted(MESHES))
@pytest.mark.parametrize("reorder", [True, False])
def test_layout_is_a_relabelling_with_correct_csr_and_geometry(name, reorder):
    mesh = MESHES[name]()
    lay = mrd.Layout(mesh.xy, mesh.tri, period=mesh.period, reorder=reorder, tile=64)
    g = lay.get()
    nv, nt = mesh.nv, mesh.nt
    assert (lay.nv, lay.nt) == (nv, nt)
    # permutations are permutations; identity when reorder is off
    assert np.array_equal(np.sort(g["vperm"]), np.arange(nv))
    assert np.array_equal(np.sort(g["tperm"]), np.arange(nt))
    if not reorder:
        assert np.array_equal(g["vperm"], np.arange(nv)) and np.array_equal(g["tperm"], np.arange(nt))
    # internal connectivity maps back to the user's triangles (as vertex sets, same cyclic order: all CCW already)
    back = g["vperm"][g["tri"]]
    user = mesh.tri[g["tperm"]]
    for r in range(3):
        ok = np.all(back == np.roll(user, -r, axis=1), axis=1) if r else np.all(back == user, axis=1)
        if r == 0:
            same = ok
    assert same.all()
    # CSR: entry e = tri*3+node lists exactly the incidences of each vertex, ascending
    off, ent = g["csr_off"], g["csr_ent"]
    assert off[0] == 0 and off[-1] == 3 * nt
    flat = g["tri"].ravel()
    for i in range(nv):
        seg = ent[off[i]:off[i + 1]]
        assert np.all(flat[seg] == i)
        assert np.all(np.diff(seg) > 0)
    assert np.array_equal(np.sort(ent), np.arange(3 * nt))
    # geometry equals the oracle's (computed independently), relabelled
    om = oracle.OracleMesh(mesh.xy, mesh.tri, period=mesh.period)
    area_o, vol_o = om.geometry()
    assert np.allclose(g["area"], area_o[g["tperm"]], rtol=1e-14, atol=0)
    assert np.allclose(g["vol"], vol_o[g["vperm"]], rtol=1e-14, atol=0)
    assert lay.ntile == (nt + 63) // 64 and lay.nslot >= nv


def test_morton_order_is_local():
    # consecutive internal vertices of a Morton-ordered uniform grid are close in space (L669-L675)
    mesh = wl.permute_mesh(wl.uniform_mesh(64, 64, 1.0, 1.0, periodic=True), 1)[0]
    lay = mrd.Layout(mesh.xy, mesh.tri, period=mesh.period, reorder=True)
    g = lay.get()
    xy = mesh.xy[g["vperm"]]
    d = np.abs(np.diff(xy, axis=0)).max(axis=1)
    assert np.median(d) <= 1.0 / 64 + 1e-12
    # a 256-triangle run touches few distinct vertices (what the fused tile kernel relies on)
    tri = g["tri"]
    touched = [len(np.unique(tri[k:k + 256])) for k in range(0, len(tri), 256)]
    assert np.mean(touched) < 200


def test_orientation_fix_and_errors():
    mesh = wl.uniform_mesh(6, 6, 1.0, 1.0, periodic=False)
    tri = mesh.tri.copy()
    tri[::3] = tri[::3][:, [0, 2, 1]]                       # make every third triangle clockwise
    lay = mrd.Layout(mesh.xy, tri, period=mesh.period)
    assert np.all(lay.get()["area"] > 0)
    bad = mesh.tri.copy()
    bad[0, 0] = mesh.nv
    with pytest.raises(mrd.MrdError) as e:
        mrd.Layout(mesh.xy, bad)
    assert e.value.code == mrd.MRD_EINVAL
    bad = mesh.tri.copy()
    bad[0, 1] = bad[0, 0]
    with pytest.raises(mrd.MrdError):
        mrd.Layout(mesh.xy, bad)
    with pytest.raises(mrd.MrdError):
        mrd.Layout(mesh.xy, mesh.tri, gamma=1.0)
    with pytest.raises(mrd.MrdError):                       # interior edge is not a wall edge
        mrd.Layout(mesh.xy, mesh.tri, wall_edge=np.array([[8, 9]], dtype=np.int32))
    walls = wl.wall_edges_y(mesh)
    lay = mrd.Layout(mesh.xy, mesh.tri, wall_edge=walls, vertex_flag=wl.boundary_vertices(mesh, True, False))
    assert lay.ne == len(walls) and lay.nf == 2 * 7


def test_mesh_create_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    mesh = wl.uniform_mesh(4, 4, 1.0, 1.0, periodic=True)
    with pytest.raises(mrd.MrdError) as e:
        mrd.Mesh(mesh.xy, mesh.tri, period=mesh.period)
    assert e.value.code == mrd.MRD_ECUDA
    # and the C entry point itself refuses too
    h = C.c_void_p()
    p = mrd.binding.make_params(period=mesh.period)
    xy = np.ascontiguousarray(mesh.xy)
    tri = np.ascontiguousarray(mesh.tri)
    rc = mrd.lib().mrd_mesh_create(C.byref(h), C.byref(p), mesh.nv, xy.ctypes.data_as(C.POINTER(C.c_double)), mesh.nt,
                                   tri.ctypes.data_as(C.POINTER(C.c_int32)), None, 0, None)
    assert rc == mrd.MRD_ECUDA and b"no CPU fallback" in mrd.lib().mrd_last_error()


def test_maximum_size_is_checked_before_anything_is_read():
    """Indices are 32-bit (int32 suffices up to 3 nt < 2^31): larger counts are refused up front, for the layout
    stage and for the partitioner alike (the arrays passed here are tiny: nothing may be read before the check)."""
    import ctypes as C
    L = mrd.lib()
    xy = np.zeros((3, 2))
    tri = np.zeros((1, 3), np.int32)
    p = mrd.binding.make_params()
    dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int32)
    for nv, nt in ((2 ** 31, 1), (3, 2 ** 30)):            # nv too large; 3 nt too large
        h = C.c_void_p()
        rc = L.mrd_layout_create(C.byref(h), C.byref(p), nv, xy.ctypes.data_as(dp), nt, tri.ctypes.data_as(ip), None, 0, None)
        assert rc == mrd.MRD_EINVAL and b"32-bit" in L.mrd_last_error()
        rc = L.mrd_partition_create(C.byref(h), nv, xy.ctypes.data_as(dp), nt, tri.ctypes.data_as(ip), None, 0, None, 0.0, 0.0, 2, 0)
        assert rc == mrd.MRD_EINVAL and b"32-bit" in L.mrd_last_error()
