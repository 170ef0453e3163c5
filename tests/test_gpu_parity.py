"""GPU parity: the CUDA path (through the C-ABI binding) against the CPU oracle, element by element on
the same seeded inputs.  Tolerances (BASELINE.json north_star, reading C17):
fp64 max relative field error <= 1e-12 after 1 step and <= 1e-9 after 100 steps; fp32 <= 1e-5 after
10 steps against the fp64 oracle."""
import numpy as np
import pytest

import oracle
import workloads as wl
from helpers import field_errors

pytestmark = pytest.mark.gpu

TOL_1 = 1e-12
TOL_100 = 1e-9
TOL_F32 = 1e-5


@pytest.fixture(scope="module")
def mrd():
    import torch
    assert torch.cuda.is_available()
    import paper_1705_02028_b200 as m
    return m


def gpu_mesh(mrd, cfg_or_mesh, W, **kw):
    import torch
    mesh = cfg_or_mesh
    gm = mrd.Mesh(mesh.xy, mesh.tri, period=mesh.period, **kw)
    dt = torch.float64 if kw.get("precision", 0) == 0 else torch.float32
    gm.set_state(torch.tensor(np.ascontiguousarray(W), dtype=dt, device="cuda").contiguous())
    return gm


def orc_mesh(mesh, W, **kw):
    om = oracle.OracleMesh(mesh.xy, mesh.tri, period=mesh.period, **kw)
    om.set_state(W)
    return om


def rel(a, b):
    s = np.abs(b).max()
    return np.abs(a - b).max() / (s if s > 0 else 1.0)


# ------------------------------------------------------------------------------------------------
# per-triangle quantities
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("case", ["smooth_jitter", "vortex", "kh_permuted", "supersonic"])
@pytest.mark.parametrize("tile", [-1, 0, 64, 128])
def test_stage1_per_triangle_matches_oracle(mrd, case, tile):
    if case == "smooth_jitter":
        mesh = wl.jitter_mesh(wl.uniform_mesh(37, 29, 2.0, 1.5, periodic=True), 0.22, seed=3)
        W = wl.random_smooth_state(mesh, mach=0.7, seed=1)
    elif case == "vortex":
        mesh = wl.uniform_mesh(48, 48, 10.0, 10.0, periodic=True)
        W = wl.vortex_state(mesh)
    elif case == "kh_permuted":
        mesh = wl.permute_mesh(wl.uniform_mesh(40, 40, 1.0, 1.0, periodic=True), 12345)[0]
        W = wl.kelvin_helmholtz_state(mesh)
    else:
        mesh = wl.jitter_mesh(wl.uniform_mesh(30, 31, 1.0, 1.0, periodic=True), 0.15, seed=8)
        W = wl.random_smooth_state(mesh, mach=2.5, seed=5)
    g = gpu_mesh(mrd, mesh, W, tile=tile).dump_stage1()
    o = orc_mesh(mesh, W).dump_stage1()
    scale = np.abs(o["phiN"]).max()
    for key in ("phiT", "phiN", "phiLDA", "phiB"):
        assert np.abs(g[key] - o[key]).max() <= 2e-13 * scale, key
    assert np.allclose(g["sT"], o["sT"], rtol=1e-14, atol=0)


def test_uniform_flow_has_exactly_zero_residual_and_state_is_bitwise_kept(mrd):
    mesh = wl.jitter_mesh(wl.uniform_mesh(24, 20, 3.0, 2.0, periodic=True), 0.25, seed=5)
    for prim in [(1.3, 0.4, -0.7, 2.1), (1.0, 0.0, 0.0, 1.0), (0.2, 2.5, 1.0, 0.1)]:
        W = wl.uniform_state(mesh, *prim)
        for scheme, order in [(2, 2), (0, 1), (1, 2)]:
            gm = gpu_mesh(mrd, mesh, W, scheme=scheme, time_order=order)
            d = gm.dump_stage1()
            assert np.all(d["phiB"] == 0.0) and np.all(d["phiN"] == 0.0) and np.all(d["phiT"] == 0.0)
            gm.step(5)
            assert np.array_equal(gm.get_state().cpu().numpy(), W)


# ------------------------------------------------------------------------------------------------
# whole steps
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("scheme,order", [(2, 2), (0, 1), (1, 2), (0, 2), (2, 1)])
@pytest.mark.parametrize("reorder", [True, False])
@pytest.mark.parametrize("tile", [-1, 0, 64, 128])
def test_one_step_and_many_steps_match_oracle(mrd, scheme, order, reorder, tile):
    mesh = wl.jitter_mesh(wl.uniform_mesh(33, 27, 1.0, 1.0, periodic=True), 0.2, seed=11)
    # LDA is not monotone (L457): at Mach 1.2 the steepening waves drive p <= 0 in the oracle too, so it gets Mach 0.5
    W = wl.random_smooth_state(mesh, mach=0.5 if scheme == 1 else 1.2, seed=4)
    gm = gpu_mesh(mrd, mesh, W, scheme=scheme, time_order=order, reorder=reorder, tile=tile)
    om = orc_mesh(mesh, W, scheme=scheme, time_order=order)
    n, t, dt = gm.step(1)
    no, to, dto = om.step(1)
    assert n == 1 and abs(dt - dto) <= 1e-14 * dto
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_1
    gm.step(99)
    om.step(99)
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_100
    assert abs(gm.sync()[1] - om.step(0)[1]) <= 1e-11


def test_config1_vortex_10_steps(mrd):
    cfg = wl.make_config("vortex")
    gm = gpu_mesh(mrd, cfg.mesh, cfg.W0)
    om = orc_mesh(cfg.mesh, cfg.W0)
    for _ in range(10):
        gm.step(1)
        om.step(1)
        assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= 10 * TOL_1
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= 1e-11


def test_config2_sod_walls_frozen_and_t_end(mrd):
    # Grid-aligned shocks amplify rounding-level differences exponentially IN THE ORACLE ITSELF
    # (tests/test_oracle_sensitivity.py): 1e-9 holds for ~50 steps, not for a whole run.
    cfg = wl.make_config("sod", n=256)
    kw = dict(vertex_flag=cfg.vertex_flag, wall_edge=cfg.wall_edge)
    gm = gpu_mesh(mrd, cfg.mesh, cfg.W0, **kw)
    om = orc_mesh(cfg.mesh, cfg.W0, **kw)
    gm.step(1)
    om.step(1)
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_1
    gm.step(49)
    om.step(49)
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_100
    n, t, _ = gm.step(100000, t_end=0.05)
    no, to, _ = om.step(100000, t_end=0.05)
    assert abs(n - no) <= 1 and t == 0.05 and abs(to - 0.05) < 1e-15
    Wg, Wo = gm.get_state().cpu().numpy(), om.get_state()
    assert field_errors(Wg, Wo) <= 2e-2                       # same solution up to the amplified round-off
    frozen = cfg.vertex_flag.astype(bool)
    assert np.array_equal(Wg[:, frozen], cfg.W0[:, frozen])


def test_oblique_wall_terms_match_oracle(mrd):
    # flow not aligned with the walls: the correction of eq. 68-71 is non-zero
    mesh = wl.uniform_mesh(24, 12, 2.0, 1.0, periodic=False)
    W = wl.random_smooth_state(mesh, mach=0.6, seed=9)
    kw = dict(vertex_flag=wl.boundary_vertices(mesh, True, False), wall_edge=wl.wall_edges_y(mesh))
    for reorder in (True, False):
        gm = gpu_mesh(mrd, mesh, W, reorder=reorder, **kw)
        om = orc_mesh(mesh, W, **kw)
        gm.step(1)
        om.step(1)
        assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_1
        gm.step(30)
        om.step(30)
        assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_100


def test_config3_kh_permuted_fp64_and_fp32(mrd):
    cfg = wl.make_config("kh", n=128)
    om = orc_mesh(cfg.mesh, cfg.W0)
    for reorder in (True, False):
        gm = gpu_mesh(mrd, cfg.mesh, cfg.W0, reorder=reorder)
        om.set_state(cfg.W0)
        gm.step(1)
        om.step(1)
        assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_1
        gm.step(99)
        om.step(99)
        assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_100
    om.set_state(cfg.W0)
    g32 = gpu_mesh(mrd, cfg.mesh, cfg.W0, precision=1)
    g32.step(10)
    om.step(10)
    assert field_errors(g32.get_state().cpu().numpy().astype(np.float64), om.get_state()) <= TOL_F32


def test_config4_riemann_frozen_boundary_and_stagnation(mrd):
    # see the note in test_config2: the oracle amplifies 1-ulp perturbations ~7x per step on this problem
    cfg = wl.make_config("riemann4", n=127)
    kw = dict(vertex_flag=cfg.vertex_flag)
    gm = gpu_mesh(mrd, cfg.mesh, cfg.W0, **kw)
    om = orc_mesh(cfg.mesh, cfg.W0, **kw)
    gm.step(1)
    om.step(1)
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_1
    gm.step(4)
    om.step(4)
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_100
    gm.step(15)
    om.step(15)
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= 1e-6
    _, mr, mp = gm.diagnostics()
    assert mr > 0 and mp > 0
    Wg = gm.get_state().cpu().numpy()
    frozen = cfg.vertex_flag.astype(bool)
    assert np.array_equal(Wg[:, frozen], cfg.W0[:, frozen])


def test_conservation_determinism_and_permutation_invariance(mrd):
    base = wl.uniform_mesh(48, 48, 1.0, 1.0, periodic=True)
    W = wl.kelvin_helmholtz_state(base)
    gm = gpu_mesh(mrd, base, W)
    tot0, _, _ = gm.diagnostics()
    gm.step(25)
    tot1, mr, mp = gm.diagnostics()
    scale = np.array([tot0[0], 1.0, 1.0, tot0[3]])
    assert np.all(np.abs(tot1 - tot0) <= 5e-13 * scale) and mr > 0 and mp > 0
    W1 = gm.get_state().cpu().numpy()
    gm2 = gpu_mesh(mrd, base, W)
    gm2.step(25)
    assert np.array_equal(gm2.get_state().cpu().numpy(), W1)          # run-to-run bitwise determinism (C20)
    perm, vorder, _ = wl.permute_mesh(base, 77)
    gp = gpu_mesh(mrd, perm, W[:, vorder])
    gp.step(25)
    assert field_errors(gp.get_state().cpu().numpy(), W1[:, vorder]) <= 1e-10


def test_host_buffer_calls_and_async_stepping(mrd):
    mesh = wl.uniform_mesh(32, 32, 10.0, 10.0, periodic=True)
    W = wl.vortex_state(mesh)
    gm = gpu_mesh(mrd, mesh, W)
    g2 = mrd.Mesh(mesh.xy, mesh.tri, period=mesh.period)
    g2.set_state_host(W)
    assert np.array_equal(g2.get_state_host(), W)
    gm.step(7)
    g2.step_async(3)
    g2.step_async(4)
    n, t, dt = g2.sync()
    assert n == 7
    assert np.array_equal(g2.get_state_host(), gm.get_state().cpu().numpy())
    assert g2.launch_count() > 7 * 3


def test_nonphysical_state_is_reported_and_state_kept(mrd):
    import torch
    mesh = wl.uniform_mesh(16, 16, 1.0, 1.0, periodic=True)
    W = wl.uniform_state(mesh)
    bad = W.copy()
    bad[0, 5] = -1.0
    gm = mrd.Mesh(mesh.xy, mesh.tri, period=mesh.period)
    with pytest.raises(mrd.MrdError) as e:
        gm.set_state(torch.tensor(bad, device="cuda"))
    assert e.value.code == mrd.MRD_ENONPHYSICAL
    # a state that turns non-physical during a step: huge momentum spike next to near-vacuum
    W2 = wl.primitive_to_conserved(np.where(np.arange(mesh.nv) % 7 == 0, 1e-6, 1.0), 0.0, 0.0,
                                   np.where(np.arange(mesh.nv) % 5 == 0, 1e3, 1e-6))
    gm.set_state(torch.tensor(W2, device="cuda"))
    om = orc_mesh(mesh, W2)
    try:
        om.step(50)
        oracle_failed = False
    except oracle.OracleError:
        oracle_failed = True
    try:
        gm.step(50)
        gpu_failed = False
    except mrd.MrdError as err:
        gpu_failed = err.code == mrd.MRD_ENONPHYSICAL
    assert gpu_failed == oracle_failed
    if gpu_failed:                                          # state left at the last good step, still usable
        Wg = gm.get_state().cpu().numpy()
        assert np.isfinite(Wg).all() and (Wg[0] > 0).all()
        assert field_errors(Wg, om.get_state()) <= 1e-6


@pytest.mark.parametrize("scheme", [3, 4])          # Bmax, Bmin
@pytest.mark.parametrize("tile", [-1, 0])
def test_bmax_bmin_variants_match_oracle(mrd, scheme, tile):
    mesh = wl.jitter_mesh(wl.uniform_mesh(31, 26, 1.0, 1.0, periodic=True), 0.2, seed=21)
    W = wl.random_smooth_state(mesh, mach=1.1, seed=6)
    gm = gpu_mesh(mrd, mesh, W, scheme=scheme, tile=tile)
    om = orc_mesh(mesh, W, scheme=scheme)
    g, o = gm.dump_stage1(), om.dump_stage1()
    assert np.abs(g["phiB"] - o["phiB"]).max() <= 2e-13 * np.abs(o["phiN"]).max()
    gm.step(1)
    om.step(1)
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_1
    gm.step(49)
    om.step(49)
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_100
    # the variant is not the diagonal blend
    gb = gpu_mesh(mrd, mesh, W, scheme=2, tile=tile)
    gb.step(50)
    assert field_errors(gb.get_state().cpu().numpy(), om.get_state()) > 1e-6


@pytest.mark.parametrize("scheme", [2, 1, 0])
@pytest.mark.parametrize("tile", [-1, 0])
def test_selective_lumping_matches_oracle(mrd, scheme, tile):
    # eq. 66-67 (L563-L570): advected vortex, so that dW/dt and with it the anti-diffusive term is O(1)
    mesh = wl.uniform_mesh(40, 36, 10.0, 10.0, periodic=True)
    W = wl.vortex_state(mesh, advect=(1.0, 0.5))
    gm = gpu_mesh(mrd, mesh, W, scheme=scheme, tile=tile, lumping=1)
    om = oracle.OracleMesh(mesh.xy, mesh.tri, period=mesh.period, scheme=scheme, lumping=1)
    om.set_state(W)
    gm.step(1)
    om.step(1)
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_1
    gm.step(49)
    om.step(49)
    Wo = om.get_state()
    assert field_errors(gm.get_state().cpu().numpy(), Wo) <= TOL_100
    g0 = gpu_mesh(mrd, mesh, W, scheme=scheme, tile=tile)            # global lumping is a different scheme
    g0.step(50)
    assert field_errors(g0.get_state().cpu().numpy(), Wo) > 1e-6


def test_api_edge_cases(mrd):
    import torch
    cfg = wl.make_config("sod", n=64)
    kw = dict(vertex_flag=cfg.vertex_flag, wall_edge=cfg.wall_edge)
    gm = mrd.Mesh(cfg.mesh.xy, cfg.mesh.tri, period=cfg.mesh.period, **kw)
    with pytest.raises(mrd.MrdError) as e:                       # no state yet
        gm.step(1)
    assert e.value.code == mrd.MRD_EINVAL
    with pytest.raises(mrd.MrdError):
        gm.get_state()
    W0 = torch.tensor(cfg.W0, device="cuda")
    gm.set_state(W0)
    assert gm.step(0) == (0, 0.0, 0.0)                           # nothing to do
    n, t, dt = gm.step(5)
    assert n == 5 and t > 0 and dt > 0
    n2, t2, _ = gm.step(1000, t_end=t)                           # already there
    assert n2 == 0 and t2 == t
    n3, t3, _ = gm.step(3, t_end=1.0)                            # max_steps binds before t_end
    assert n3 == 3 and t < t3 < 1.0
    gm.set_state(W0)                                             # restart: clock and counters reset
    assert gm.sync()[0] == 0 and gm.sync()[1] == 0.0
    a = mrd.Mesh(cfg.mesh.xy, cfg.mesh.tri, period=cfg.mesh.period, **kw)   # two meshes alive at once, interleaved
    a.set_state(W0)
    a.step_async(4); gm.step_async(4); a.step_async(3); gm.step_async(3)
    assert np.array_equal(a.get_state().cpu().numpy(), gm.get_state().cpu().numpy())
    s = torch.cuda.Stream()                                      # a non-default stream
    with torch.cuda.stream(s):
        b = mrd.Mesh(cfg.mesh.xy, cfg.mesh.tri, period=cfg.mesh.period, **kw)
        b.set_state(W0, stream=s)
        b.step(7, stream=s)
        Wb = b.get_state(stream=s)
    s.synchronize()
    assert np.array_equal(Wb.cpu().numpy(), gm.get_state().cpu().numpy())


@pytest.mark.parametrize("scheme,order", [(2, 2), (0, 1)])
def test_walls_and_frozen_vertices_in_fp32_and_first_order(mrd, scheme, order):
    cfg = wl.make_config("sod", n=128)
    kw = dict(vertex_flag=cfg.vertex_flag, wall_edge=cfg.wall_edge, scheme=scheme, time_order=order)
    om = orc_mesh(cfg.mesh, cfg.W0, **kw)
    gm = gpu_mesh(mrd, cfg.mesh, cfg.W0, **kw)
    g32 = gpu_mesh(mrd, cfg.mesh, cfg.W0, precision=1, **kw)
    gm.step(1); om.step(1)
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_1
    gm.step(9); om.step(9); g32.step(10)
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_100
    assert field_errors(g32.get_state().cpu().numpy().astype(np.float64), om.get_state()) <= TOL_F32


@pytest.mark.parametrize("scheme,order", [(2, 2), (1, 2), (0, 1)])
def test_linear_sound_wave_strip(mrd, scheme, order):
    # PAPER.md 5.1.1 (L766): amplitude 1e-4 on a quasi-1D periodic strip; tiny residuals on an O(1) background
    mesh = wl.uniform_mesh(64, 4, 1.0, 4.0 / 64, periodic=True)
    W = wl.sound_wave_state(mesh)
    gm = gpu_mesh(mrd, mesh, W, scheme=scheme, time_order=order)
    om = orc_mesh(mesh, W, scheme=scheme, time_order=order)
    n, t, _ = gm.step(10 ** 6, t_end=0.25)
    no, to, _ = om.step(10 ** 6, t_end=0.25)
    assert abs(n - no) <= 1 and t == 0.25
    Wg, Wo = gm.get_state().cpu().numpy(), om.get_state()
    if scheme == 2:
        # eq. 53 is 0/0 for the transverse momentum (its exact residual vanishes, the nodal N residuals do not): Theta_y is
        # decided by round-off and two ORACLE runs differing by 1 ulp drift by 2e-4 of the amplitude in rho
        # (tests/test_oracle_sensitivity.py); the GPU must stay within that band
        assert np.abs(Wg[0] - Wo[0]).max() <= 1e-3 * 1e-4
        assert np.abs(Wg[3] - Wo[3]).max() <= 1e-3 * 1e-4 * 2.5
    else:
        assert field_errors(Wg, Wo) <= TOL_100
        # the perturbation itself (1e-4 of the background) agrees to 1e-9 of its amplitude
        assert np.abs((Wg[0] - 1.0) - (Wo[0] - 1.0)).max() <= 1e-9 * 1e-4


def test_noh_infinite_mach_shock_first_order(mrd):
    # PAPER.md 5.2.2 (L901-L913): p = 1e-6, Mach ~ 800 inflow towards the centre; scheme N, first order (the paper:
    # "less diffusive blended schemes either fail on this problem", L917).  Boundary vertices keep the initial state.
    mesh = wl.uniform_mesh(48, 48, 2.0, 2.0, periodic=False)
    W = wl.noh_state(mesh)
    kw = dict(gamma=5.0 / 3.0, scheme=0, time_order=1, vertex_flag=wl.boundary_vertices(mesh, True, True))
    gm = gpu_mesh(mrd, mesh, W, **kw)
    om = orc_mesh(mesh, W, **kw)
    gm.step(1); om.step(1)
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_1
    gm.step(29); om.step(29)
    Wg, Wo = gm.get_state().cpu().numpy(), om.get_state()
    assert field_errors(Wg, Wo) <= TOL_100
    _, mr, mp = gm.diagnostics()
    assert mr > 0 and mp > 0 and Wg[0].max() > 2.0               # the central compression has started


# ------------------------------------------------------------------------------------------------
# variable-valence triangulation (stand-in for the paper's Delaunay-refined meshes, L685)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("tile", [-1, 0, 64])
@pytest.mark.parametrize("periodic", [True, False])
def test_variable_valence_mesh_matches_oracle(mrd, tile, periodic):
    mesh = wl.flip_edges(wl.jitter_mesh(wl.uniform_mesh(40, 36, 2.0, 1.8, periodic=periodic), 0.2, seed=3), seed=11)
    val = np.bincount(mesh.tri.ravel(), minlength=mesh.nv)
    assert val.max() >= 8 and val.min() <= 4
    W = wl.random_smooth_state(mesh, mach=0.8, seed=6)
    flag = None if periodic else wl.boundary_vertices(mesh)
    import torch
    gm = mrd.Mesh(mesh.xy, mesh.tri, vertex_flag=flag, period=mesh.period, tile=tile)
    gm.set_state(torch.tensor(W, device="cuda"))
    om = oracle.OracleMesh(mesh.xy, mesh.tri, period=mesh.period, vertex_flag=flag)
    om.set_state(W)
    g, o = gm.dump_stage1(), om.dump_stage1()
    scale = np.abs(o["phiN"]).max()
    for key in ("phiT", "phiN", "phiLDA", "phiB"):
        assert np.abs(g[key] - o[key]).max() <= 2e-13 * scale, key
    assert np.allclose(g["sT"], o["sT"], rtol=1e-14, atol=0)
    n, t, dt = gm.step(1)
    no, to, dto = om.step(1)
    assert abs(dt - dto) <= 1e-14 * dto
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_1
    gm.step(49)
    om.step(49)
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_100
    if periodic:
        tot0 = (W * om.geometry()[1][None, :]).sum(axis=1)
        tot = gm.diagnostics()[0]
        assert np.abs(tot - tot0).max() <= 1e-12 * np.abs(tot0).max()        # conservation with variable V_i and valence


# ------------------------------------------------------------------------------------------------
# Bx shock-sensor blend (eq. 54-56; readings C23-C26)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("tile", [-1, 0, 64])
@pytest.mark.parametrize("order", [2, 1])
def test_bx_blend_matches_oracle(mrd, tile, order):
    mesh = wl.flip_edges(wl.jitter_mesh(wl.uniform_mesh(33, 27, 1.0, 1.0, periodic=True), 0.2, seed=11), seed=4)
    W = wl.random_smooth_state(mesh, mach=1.1, seed=4)
    gm = gpu_mesh(mrd, mesh, W, scheme=mrd.SCHEME_BX, time_order=order, tile=tile)
    om = orc_mesh(mesh, W, scheme=oracle.SCHEME_BX, time_order=order)
    g, o = gm.dump_stage1(), om.dump_stage1()
    scale = np.abs(o["phiN"]).max()
    assert np.abs(o["phiB"] - o["phiLDA"]).max() > 1e-3 * scale and np.abs(o["phiB"] - o["phiN"]).max() > 1e-3 * scale
    for key in ("phiT", "phiN", "phiLDA", "phiB"):
        assert np.abs(g[key] - o[key]).max() <= 2e-13 * scale, key
    n, t, dt = gm.step(1)
    no, to, dto = om.step(1)
    assert n == 1 and abs(dt - dto) <= 1e-14 * dto
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_1
    gm.step(49)
    om.step(49)
    assert field_errors(gm.get_state().cpu().numpy(), om.get_state()) <= TOL_100
    # replayed (CUDA graph) and eager steps agree bit for bit; the scheme is deterministic
    gm2 = gpu_mesh(mrd, mesh, W, scheme=mrd.SCHEME_BX, time_order=order, tile=tile)
    for _ in range(50):
        gm2.step(1)
    assert np.array_equal(gm2.get_state().cpu().numpy(), gm.get_state().cpu().numpy())


def test_bx_on_the_sod_tube_with_walls_and_frozen_ends(mrd):
    cfg = wl.make_config("sod", n=96)
    mesh = cfg.mesh
    import torch
    gm = mrd.Mesh(mesh.xy, mesh.tri, vertex_flag=cfg.vertex_flag, wall_edge=cfg.wall_edge, period=mesh.period, scheme=mrd.SCHEME_BX)
    gm.set_state(torch.tensor(cfg.W0, device="cuda"))
    om = oracle.OracleMesh(mesh.xy, mesh.tri, period=mesh.period, vertex_flag=cfg.vertex_flag, wall_edge=cfg.wall_edge,
                           scheme=oracle.SCHEME_BX)
    om.set_state(cfg.W0)
    # u = 0 everywhere at t = 0: |v|_max = |v|_min, sensor 0 (reading C24), the first step is an LDA step on both sides
    for k in range(4):
        n, t, dt = gm.step(1)
        no, to, dto = om.step(1)
        assert abs(dt - dto) <= 1e-14 * dto
        # the scheme amplifies round-off on this grid-aligned shock: resynchronise every step
        err = field_errors(gm.get_state().cpu().numpy(), om.get_state())
        assert err <= TOL_1, (k, err)
        gm.set_state(torch.tensor(om.get_state(), device="cuda"))


@pytest.mark.parametrize("scheme", [2, 5])
def test_fp32_on_the_variable_valence_mesh(mrd, scheme):
    mesh = wl.flip_edges(wl.jitter_mesh(wl.uniform_mesh(40, 36, 2.0, 1.8, periodic=True), 0.2, seed=3), seed=11)
    W = wl.random_smooth_state(mesh, mach=0.8, seed=6)
    gm = gpu_mesh(mrd, mesh, W, scheme=scheme, precision=1)
    om = orc_mesh(mesh, W, scheme=scheme)
    gm.step(10)
    om.step(10)
    assert field_errors(gm.get_state().cpu().numpy().astype(np.float64), om.get_state()) <= TOL_F32


@pytest.mark.parametrize("n,free_rim", [(3, False), (5, True), (300, False), (2000, True), (20000, False)])
@pytest.mark.parametrize("tile", [64, 256])
def test_extreme_valence_a_fan_and_a_wheel(mrd, n, free_rim, tile):
    """One vertex in every triangle of the mesh: a fan over a convex polygon (vertex 0, valence n - 2) and a wheel (a hub of
    valence n) -- incidence lists far longer than a tile, tiles whose triangles all share a vertex, and meshes of one to three
    triangles.  Five RK2 steps of scheme B against the oracle, rim frozen or free."""
    import torch
    from types import SimpleNamespace
    rng = np.random.default_rng(n)
    ang = np.sort(rng.random(n)) * 2 * np.pi if n > 5 else (np.arange(n) + 0.3) * 2 * np.pi / n
    rim = np.stack([2.0 * np.cos(ang), np.sin(ang)], axis=1)
    i = np.arange(n, dtype=np.int32)
    fan = (rim, np.stack([np.zeros(n - 2, dtype=np.int32), i[1:-1], i[2:]], axis=1), np.ones(n, dtype=np.uint8))
    wheel = (np.concatenate([rim, [[0.1, 0.05]]]), np.stack([np.full(n, n, dtype=np.int32), i, (i + 1) % n], axis=1),
             np.concatenate([np.zeros(n, dtype=np.uint8) if free_rim else np.ones(n, dtype=np.uint8), [0]]))
    for X, T, flag in (fan, wheel):
        W = wl.random_smooth_state(SimpleNamespace(xy=X, nv=X.shape[0], lengths=(4.0, 2.0)), mach=0.5, seed=2)
        gm = mrd.Mesh(X, T, vertex_flag=flag, scheme=mrd.SCHEME_B, time_order=2, tile=tile)
        gm.set_state(torch.tensor(W, device="cuda"))
        om = oracle.OracleMesh(X, T, vertex_flag=flag, scheme=oracle.SCHEME_B, time_order=2, threads=4)
        om.set_state(W)
        gm.step(5)
        om.step(5)
        Wg = gm.get_state().cpu().numpy()
        assert field_errors(Wg, om.get_state()) <= 1e-10
        assert np.array_equal(Wg[:, flag == 1], W[:, flag == 1])
