"""Mesh-level pins for the oracle's time stepper (eq. 43-45, 60-65, §3.5; SURVEY §8c "Whole step")."""
import numpy as np
import pytest

import oracle
import workloads as wl
from helpers import field_errors, prim_to_cons

GAMMA = 1.4


def make(mesh, W, **kw):
    om = oracle.OracleMesh(mesh.xy, mesh.tri, period=mesh.period, **kw)
    om.set_state(W)
    return om


@pytest.mark.parametrize("prim", [(1.3, 0.4, -0.7, 2.1), (1.0, 0.0, 0.0, 1.0), (0.2, 2.5, 1.0, 0.1)])
@pytest.mark.parametrize("jitter", [False, True])
def test_uniform_flow_is_preserved_bitwise(prim, jitter):
    mesh = wl.uniform_mesh(12, 10, 3.0, 2.0, periodic=True)
    if jitter:
        mesh = wl.jitter_mesh(mesh, 0.25, seed=5)
    W = wl.uniform_state(mesh, *prim)
    for scheme, order in [(oracle.SCHEME_B, 2), (oracle.SCHEME_N, 1), (oracle.SCHEME_LDA, 2)]:
        om = make(mesh, W, scheme=scheme, time_order=order)
        om.step(5)
        assert np.array_equal(om.get_state(), W)


@pytest.mark.parametrize("scheme,order", [(oracle.SCHEME_B, 2), (oracle.SCHEME_N, 1), (oracle.SCHEME_LDA, 2),
                                          (oracle.SCHEME_N, 2), (oracle.SCHEME_B, 1)])
def test_conservation_on_periodic_meshes(scheme, order):
    # all schemes are conservative (L455): sum_i V_i W_i is constant to round-off
    mesh = wl.jitter_mesh(wl.uniform_mesh(24, 24, 1.0, 1.0, periodic=True), 0.2, seed=11)
    W = wl.random_smooth_state(mesh, mach=1.2, seed=4)
    om = make(mesh, W, scheme=scheme, time_order=order)
    tot0, _, _ = om.diagnostics()
    om.step(20)
    tot1, mr, mp = om.diagnostics()
    scale = np.array([tot0[0], np.abs(W[1:3]).max() * 1.0, np.abs(W[1:3]).max() * 1.0, tot0[3]])
    assert np.all(np.abs(tot1 - tot0) < 2e-13 * scale)
    assert mr > 0 and mp > 0
    assert np.abs(om.get_state() - W).max() > 1e-3          # something did happen


def test_volumes_and_areas():
    mesh = wl.uniform_mesh(8, 6, 4.0, 3.0, periodic=True)
    om = make(mesh, wl.uniform_state(mesh))
    area, vol = om.geometry()
    assert np.allclose(area, 0.5 * 0.5 * 0.5)               # h = 0.5: |T| = h^2/2
    assert np.allclose(vol, 0.25)                           # V_i = 6 |T| / 3 = h^2 (reading C5)
    mesh = wl.uniform_mesh(4, 4, 1.0, 1.0, periodic=False)
    om = make(mesh, wl.uniform_state(mesh))
    area, vol = om.geometry()
    assert abs(area.sum() - 1.0) < 1e-14 and abs(vol.sum() - 1.0) < 1e-14


def test_time_step_formula():
    # eq. 44-45 on a uniform state / uniform periodic mesh: V_i = h^2, six triangles with l_max = sqrt(2) h
    mesh = wl.uniform_mesh(16, 16, 2.0, 2.0, periodic=True)
    rho, u, v, p = 1.3, 0.4, -0.7, 2.1
    om = make(mesh, wl.uniform_state(mesh, rho, u, v, p), cfl=0.5)
    _, t, dt = om.step(1)
    h = 2.0 / 16
    speed = np.hypot(u, v) + np.sqrt(GAMMA * p / rho)
    assert abs(dt - 0.5 * 2 * h * h / (6 * np.sqrt(2) * h * speed)) < 1e-15
    assert t == dt


def test_time_step_general_mesh_and_clip():
    mesh = wl.jitter_mesh(wl.uniform_mesh(10, 10, 1.0, 1.0, periodic=True), 0.2, seed=2)
    W = wl.random_smooth_state(mesh, seed=9)
    om = make(mesh, W, cfl=0.4)
    d = om.dump_stage1()
    _, vol = om.geometry()
    S = np.zeros(mesh.nv)
    np.add.at(S, mesh.tri.ravel(), np.repeat(d["sT"], 3))
    expect = 0.4 * np.min(2 * vol / S)
    _, t, dt = om.step(1)
    assert abs(dt - expect) < 1e-15
    # clipping lands exactly on t_end (reading C13)
    t_end = t + 0.37 * dt
    n, t2, dt2 = om.step(100, t_end=t_end)
    assert n == 1 and t2 == t_end and abs(dt2 - 0.37 * dt) < 1e-15
    n, t3, _ = om.step(100, t_end=t_end)
    assert n == 0 and t3 == t_end


def test_first_order_update_is_eq43():
    # W^{n+1} = W^n - dt/V_i sum_T phi_i^T with the dumped per-triangle residuals
    mesh = wl.jitter_mesh(wl.uniform_mesh(9, 7, 1.0, 1.0, periodic=True), 0.2, seed=3)
    W = wl.random_smooth_state(mesh, seed=1)
    for scheme, key in [(oracle.SCHEME_N, "phiN"), (oracle.SCHEME_LDA, "phiLDA"), (oracle.SCHEME_B, "phiB")]:
        om = make(mesh, W, scheme=scheme, time_order=1)
        d = om.dump_stage1()
        _, vol = om.geometry()
        acc = np.zeros((mesh.nv, 4))
        np.add.at(acc, mesh.tri.ravel(), d[key].reshape(-1, 4))
        _, _, dt = om.step(1)
        expect = W - dt / vol * acc.T
        assert np.allclose(om.get_state(), expect, rtol=0, atol=1e-14)


def test_rk2_with_scheme_N_is_heun():
    # SURVEY §8c "RK2": with V_i = sum |T|/3 and no blending, stage 2 reduces to
    # W^{n+1} = W^n - dt/(2 V_i) sum [phi_i^N(W^n) + phi_i^N(W*)]
    mesh = wl.jitter_mesh(wl.uniform_mesh(10, 8, 1.0, 1.0, periodic=True), 0.2, seed=8)
    W = wl.random_smooth_state(mesh, seed=6)
    om1 = make(mesh, W, scheme=oracle.SCHEME_N, time_order=1)
    d0 = om1.dump_stage1()
    _, vol = om1.geometry()
    _, _, dt = om1.step(1)
    Wstar = om1.get_state()
    om1.set_state(Wstar)
    d1 = om1.dump_stage1()
    acc = np.zeros((mesh.nv, 4))
    np.add.at(acc, mesh.tri.ravel(), (d0["phiN"] + d1["phiN"]).reshape(-1, 4))
    heun = W - 0.5 * dt / vol * acc.T
    om2 = make(mesh, W, scheme=oracle.SCHEME_N, time_order=2)
    _, _, dt2 = om2.step(1)
    assert dt2 == dt
    assert np.allclose(om2.get_state(), heun, rtol=0, atol=5e-14)


def _wall_sums(mesh, walls, W, gamma=GAMMA, alpha=0.75):
    """Per-vertex sum of the wall corrections of eq. 68-71 (L586-L602), retyped in numpy from the paper and independent of
    the oracle's code: F^c = (desired no-through-flow flux) - (computed flux) = -(rho, rho u, rho v, e + p) v_n with the
    OUTWARD unit normal n; Phi_a = l/2 (alpha F^c_a + (1 - alpha) F^c_b), Phi_b likewise with the weights swapped."""
    nvx, nvy = mesh.shape
    acc = np.zeros((mesh.nv, 4))
    for a, b in walls:
        ya = mesh.xy[a, 1]
        n = np.array([0.0, -1.0]) if ya < 0.5 * mesh.lengths[1] else np.array([0.0, 1.0])
        ln = np.hypot(*(mesh.xy[b] - mesh.xy[a]))
        Fc = []
        for i in (a, b):
            rho, m, nn, e = W[:, i]
            u, v = m / rho, nn / rho
            p = (gamma - 1.0) * (e - 0.5 * rho * (u * u + v * v))
            vn = u * n[0] + v * n[1]
            Fc.append(-np.array([rho, m, nn, e + p]) * vn)
        acc[a] += 0.5 * ln * (alpha * Fc[0] + (1.0 - alpha) * Fc[1])
        acc[b] += 0.5 * ln * ((1.0 - alpha) * Fc[0] + alpha * Fc[1])
    return acc


def test_rk2_with_scheme_N_and_walls_is_heun_with_the_wall_term_averaged():
    # Pin of reading C15 (stage 2 uses (Phi^c(W^n) + Phi^c(W*)) / 2).  Mathematics, not the oracle's formula: with scheme N
    # and V_i = sum |T|/3 the two stages of eq. 60-62 are Heun's method for dW_i/dt = -(1/V_i)(sum_T phi_i^N + Phi_i^c), i.e.
    #   W^{n+1} = W^n - dt/(2 V_i) [sum phi^N(W^n) + sum phi^N(W*) + Phi^c(W^n) + Phi^c(W*)],
    # which holds only if the stage-2 wall term is the plain average of the two evaluations.  Oblique flow (v_n != 0 on
    # both walls), no frozen vertices anywhere, so every wall vertex is updated with the term under test.
    mesh = wl.jitter_mesh(wl.uniform_mesh(12, 7, 2.0, 1.0, periodic=False), 0.15, seed=5)
    walls = wl.wall_edges_y(mesh)
    W = wl.random_smooth_state(mesh, mach=0.6, seed=12)
    on_wall = np.unique(walls.ravel())
    assert np.abs(W[2, on_wall] / W[0, on_wall]).min() > 1e-3          # v_n != 0 at every wall vertex
    om1 = oracle.OracleMesh(mesh.xy, mesh.tri, wall_edge=walls, scheme=oracle.SCHEME_N, time_order=1)
    om1.set_state(W)
    d0 = om1.dump_stage1()
    _, vol = om1.geometry()
    _, _, dt = om1.step(1)
    Wstar = om1.get_state()
    c0 = _wall_sums(mesh, walls, W)
    acc0 = np.zeros((mesh.nv, 4))
    np.add.at(acc0, mesh.tri.ravel(), d0["phiN"].reshape(-1, 4))
    assert np.allclose(Wstar, W - dt / vol * (acc0 + c0).T, rtol=0, atol=5e-14)     # eq. 60 with the wall term
    om1.set_state(Wstar)
    d1 = om1.dump_stage1()
    c1 = _wall_sums(mesh, walls, Wstar)
    acc1 = np.zeros((mesh.nv, 4))
    np.add.at(acc1, mesh.tri.ravel(), d1["phiN"].reshape(-1, 4))
    heun = W - 0.5 * dt / vol * (acc0 + acc1 + c0 + c1).T
    om2 = oracle.OracleMesh(mesh.xy, mesh.tri, wall_edge=walls, scheme=oracle.SCHEME_N, time_order=2)
    om2.set_state(W)
    _, _, dt2 = om2.step(1)
    assert dt2 == dt
    W2 = om2.get_state()
    assert np.abs(W2 - heun).max() <= 5e-14
    # the test has teeth: each plausible mistake (term of W^n dropped, term of W* dropped, no factor 1/2, wrong sign)
    # moves the wall vertices by far more than the tolerance
    for wrong in (c1, c0, 2.0 * (c0 + c1), -(c0 + c1), 0.5 * c0 + c1):
        bad = W - 0.5 * dt / vol * (acc0 + acc1 + wrong).T
        assert np.abs(W2 - bad)[:, on_wall].max() > 1e-6


def test_renumbering_invariance():
    # permuting vertex / triangle numbering and rotating local node order permutes the result
    base = wl.jitter_mesh(wl.uniform_mesh(16, 16, 1.0, 1.0, periodic=True), 0.2, seed=13)
    W = wl.random_smooth_state(base, seed=21, mach=1.5)
    perm, vorder, _ = wl.permute_mesh(base, seed=99)
    a = make(base, W)
    b = make(perm, W[:, vorder])
    a.step(10)
    b.step(10)
    assert field_errors(b.get_state(), a.get_state()[:, vorder]) < 1e-13


def test_diagonal_mirror_symmetry_of_the_four_quadrant_problem():
    # config 4 is symmetric under (x,y,u,v) -> (y,x,v,u) on a SW-NE diagonal split
    # The N scheme keeps the symmetry to round-off for many steps; the blended scheme only for a few:
    # where a component of the residual is pure rounding noise, Theta_kk (eq. 53) is an O(1) ratio of
    # noise and grid-aligned shocks amplify the resulting 1e-16 asymmetry step by step ("noise").
    cfg = wl.make_config("riemann4", n=24)
    m = cfg.mesh
    for scheme, order, steps, tol in [(oracle.SCHEME_N, 1, 24, 1e-13), (oracle.SCHEME_B, 2, 3, 1e-12)]:
        om = oracle.OracleMesh(m.xy, m.tri, vertex_flag=cfg.vertex_flag, scheme=scheme, time_order=order)
        om.set_state(cfg.W0)
        om.step(steps)
        W = om.get_state().reshape(4, m.shape[1], m.shape[0])
        Wt = W.transpose(0, 2, 1)[[0, 2, 1, 3]]
        assert np.abs(W - Wt).max() < tol
    # frozen boundary vertices keep the initial condition (L582)
    f = cfg.vertex_flag.astype(bool)
    assert np.array_equal(om.get_state()[:, f], cfg.W0[:, f])
    assert np.abs(om.get_state() - cfg.W0).max() > 1e-3


def test_wall_term_vanishes_for_tangential_flow_and_balances_mass_otherwise():
    mesh = wl.uniform_mesh(12, 6, 2.0, 1.0, periodic=False)
    walls = wl.wall_edges_y(mesh)
    frozen = wl.boundary_vertices(mesh, x_ends=True, y_ends=False)
    # (a) uniform flow along the walls stays uniform bitwise (v_n = 0 exactly)
    W = wl.uniform_state(mesh, 1.0, 0.8, 0.0, 1.0)
    om = oracle.OracleMesh(mesh.xy, mesh.tri, vertex_flag=frozen, wall_edge=walls)
    om.set_state(W)
    om.step(5)
    assert np.array_equal(om.get_state(), W)
    # (b) flow into the top wall: d(mass)/dt = -(boundary terms); no frozen vertices, walls top+bottom,
    # periodic-free x-ends are open edges whose flux the scheme computes "as if there was no wall"
    W = wl.uniform_state(mesh, 1.0, 0.0, 0.3, 1.0)
    free = oracle.OracleMesh(mesh.xy, mesh.tri, wall_edge=None, scheme=oracle.SCHEME_N, time_order=1)
    wall = oracle.OracleMesh(mesh.xy, mesh.tri, wall_edge=walls, scheme=oracle.SCHEME_N, time_order=1)
    free.set_state(W)
    wall.set_state(W)
    t0, _, _ = free.diagnostics()
    _, _, dt = free.step(1)
    _, _, dt2 = wall.step(1)
    assert dt == dt2
    tf, _, _ = free.diagnostics()
    tw, _, _ = wall.diagnostics()
    # uniform state: triangle residuals vanish, so without walls nothing changes at all
    assert np.allclose(tf, t0, rtol=1e-15)
    # with walls: sum of eq. 69 over the edges; top (n=+y): -rho v L, bottom (n=-y): +rho v L -> mass cancels,
    # y-momentum: top -rho v v L, bottom +rho v v L ... signs follow n; energy likewise cancels
    rho, v, L = 1.0, 0.3, 2.0
    h = (W[3, 0] + 1.0) / rho
    top = -np.array([rho * v, 0.0, rho * v * v, rho * h * v]) * L
    bot = +np.array([rho * v, 0.0, rho * v * v, rho * h * v]) * L
    assert np.allclose(tw - t0, -dt * (top + bot), atol=1e-14)
    # and locally: the top row loses momentum towards the wall, i.e. rho*v decreases there
    Wn = wall.get_state().reshape(4, mesh.shape[1], mesh.shape[0])
    assert np.all(Wn[0, -1, 1:-1] > 1.0) and np.all(Wn[0, 0, 1:-1] < 1.0)


def test_oblique_wall_keeps_parallel_uniform_flow():
    th = 0.4
    Rm = np.array([[np.cos(th), -np.sin(th)], [np.sin(th), np.cos(th)]])
    mesh = wl.uniform_mesh(10, 5, 2.0, 1.0, periodic=False)
    walls = wl.wall_edges_y(mesh)
    frozen = wl.boundary_vertices(mesh, x_ends=True, y_ends=False)
    xy = mesh.xy @ Rm.T
    vel = Rm @ np.array([0.9, 0.0])
    W = np.tile(prim_to_cons(1.1, vel[0], vel[1], 0.9, GAMMA)[:, None], (1, mesh.nv))
    om = oracle.OracleMesh(xy, mesh.tri, vertex_flag=frozen, wall_edge=walls)
    om.set_state(W)
    om.step(10)
    assert np.abs(om.get_state() - W).max() < 1e-14


def test_nonphysical_state_is_reported_and_state_kept():
    mesh = wl.uniform_mesh(8, 8, 1.0, 1.0, periodic=True)
    W = wl.uniform_state(mesh)
    W[3, 5] = 0.01                                         # negative pressure at one vertex
    om = make(mesh, W)
    with pytest.raises(oracle.OracleError) as ei:
        om.step(1)
    assert ei.value.code == oracle.ORC_ENONPHYSICAL
    assert np.array_equal(om.get_state(), W)


def test_bad_meshes_are_rejected():
    mesh = wl.uniform_mesh(4, 4, 1.0, 1.0, periodic=False)
    tri = mesh.tri.copy()
    tri[0, 0] = 9999
    with pytest.raises(oracle.OracleError):
        oracle.OracleMesh(mesh.xy, tri)
    tri = mesh.tri.copy()
    tri[0] = [0, 0, 1]
    with pytest.raises(oracle.OracleError):
        oracle.OracleMesh(mesh.xy, tri)
    # clockwise input is accepted and made counter-clockwise
    om = oracle.OracleMesh(mesh.xy, mesh.tri[:, [0, 2, 1]])
    area, _ = om.geometry()
    assert np.all(area > 0)
