"""Pins for the Bx shock-sensor blend of the oracle (eq. 54-56; readings C23-C26 of DESIGN.md).
What the paper and the algebra fix, each checked with code that shares nothing with the oracle:
  * eq. 54-56 retyped in numpy from the oracle's OWN N / LDA dumps and an independent divergence (least-squares /
    Green-Gauss on the unwrapped vertex coordinates), so a wrong normal, length, sign or normalisation shows up;
  * "non-zero only in regions of compression" (L517): expansion or divergence-free flow -> Bx is LDA, bit for bit;
  * strong compression -> theta = 1 -> Bx is N; theta in [0, 1]; a scalar theta keeps sum_i phi_i = phi^T;
  * theta = O(h) in smooth flow (L517): halving h halves the largest theta of a fixed smooth field;
  * stationary vortex: "the Bx scheme yields exactly the same results as the LDA scheme" (L885) to plotting accuracy;
  * sound wave: Bx and LDA indistinguishable (L778); Sod: N at the captured shock (L824), LDA in the rarefaction;
  * uniform flow preserved exactly, conservation on a periodic mesh."""
import numpy as np
import pytest

import oracle
import workloads as wl


def _om(mesh, W, scheme, **kw):
    om = oracle.OracleMesh(mesh.xy, mesh.tri, period=mesh.period, scheme=scheme, **kw)
    om.set_state(W)
    return om


def _unwrapped(mesh):
    """[nt][3][2] vertex coordinates of every triangle, 2nd and 3rd vertex by minimum image relative to the 1st."""
    x = mesh.xy[mesh.tri].copy()
    for d in range(2):
        p = mesh.period[d]
        if p > 0:
            for j in (1, 2):
                dd = x[:, j, d] - x[:, 0, d]
                x[:, j, d] = x[:, 0, d] + dd - p * np.round(dd / p)
    return x


def _theta_numpy(mesh, W):
    """eq. 55-56 from scratch: the divergence of the linear interpolant by solving for its gradient."""
    x = _unwrapped(mesh)
    vel = np.stack([W[1] / W[0], W[2] / W[0]], axis=1)           # [nv][2]
    speed = np.sqrt((vel ** 2).sum(axis=1))
    vrange = speed.max() - speed.min()
    v = vel[mesh.tri]                                            # [nt][3][2]
    # gradient of a linear function on a triangle: solve [x1-x0; x2-x0] g = [f1-f0; f2-f0]
    A = np.stack([x[:, 1] - x[:, 0], x[:, 2] - x[:, 0]], axis=1)  # [nt][2][2]
    du = np.stack([v[:, 1, 0] - v[:, 0, 0], v[:, 2, 0] - v[:, 0, 0]], axis=1)
    dv = np.stack([v[:, 1, 1] - v[:, 0, 1], v[:, 2, 1] - v[:, 0, 1]], axis=1)
    gu = np.linalg.solve(A, du[..., None])[..., 0]
    gv = np.linalg.solve(A, dv[..., None])[..., 0]
    div = gu[:, 0] + gv[:, 1]
    edges = np.stack([x[:, 2] - x[:, 1], x[:, 0] - x[:, 2], x[:, 1] - x[:, 0]], axis=1)
    lmax = np.sqrt((edges ** 2).sum(axis=2)).max(axis=1)
    lo, hi = mesh.xy.min(axis=0), mesh.xy.max(axis=0)
    L = max(mesh.period[0] if mesh.period[0] > 0 else hi[0] - lo[0], mesh.period[1] if mesh.period[1] > 0 else hi[1] - lo[1])
    if not vrange > 0:
        return np.zeros(len(div)), div
    s = np.maximum(0.0, -L * div / vrange)
    return np.minimum(1.0, s * s * lmax / L), div


@pytest.mark.parametrize("periodic", [True, False])
def test_bx_blend_is_eq_54_to_56_retyped(periodic):
    mesh = wl.flip_edges(wl.jitter_mesh(wl.uniform_mesh(18, 15, 2.0, 1.5, periodic=periodic), 0.2, seed=3), seed=5)
    W = wl.random_smooth_state(mesh, mach=1.1, seed=2)
    d = _om(mesh, W, oracle.SCHEME_BX).dump_stage1()
    N, L, T = d["phiN"], d["phiLDA"], d["phiT"]
    theta, div = _theta_numpy(mesh, W)
    assert (div < 0).mean() > 0.2 and (div > 0).mean() > 0.2 and theta.max() > 1e-3      # both regimes are present
    expect = theta[:, None, None] * N + (1.0 - theta[:, None, None]) * L
    scale = np.abs(N).max()
    assert np.abs(d["phiB"] - expect).max() <= 1e-13 * scale
    assert np.all(theta >= 0) and np.all(theta <= 1)
    assert np.array_equal(d["phiB"][div > 1e-12], L[div > 1e-12])                        # expansion: LDA exactly (L517)
    assert np.abs(d["phiB"].sum(axis=1) - T).max() <= 1e-13 * scale                      # conservative (L455)
    # the same N and LDA residuals as the other schemes: only the blend differs
    b = _om(mesh, W, oracle.SCHEME_B).dump_stage1()
    assert np.array_equal(b["phiN"], N) and np.array_equal(b["phiLDA"], L)


def test_expanding_flow_is_lda_and_strong_compression_is_n():
    for sign, same_as in ((+1.0, "phiLDA"), (-1.0, "phiN")):
        # v = sign * a * (x, y): div v = 2 sign a everywhere; |v| spans 0 ... a/sqrt(2), so s ~ 2.8 and theta ~ 8 l_max / L:
        # above 1 (clamped) on a mesh of 6 x 6 cells
        n = 16 if sign > 0 else 6
        mesh = wl.jitter_mesh(wl.uniform_mesh(n, n, 1.0, 1.0, periodic=False), 0.15, seed=4)
        x, y = mesh.xy[:, 0] - 0.5, mesh.xy[:, 1] - 0.5
        a = 1.0
        W = wl.primitive_to_conserved(1.0 + 0.1 * x, sign * a * x, sign * a * y, 1.0 + 0.05 * y)
        d = _om(mesh, W, oracle.SCHEME_BX).dump_stage1()
        if sign < 0:
            theta, _ = _theta_numpy(mesh, W)
            sel = theta >= 1.0
            assert sel.mean() > 0.02
            assert np.array_equal(d["phiB"][sel], d["phiN"][sel])
            assert np.all(theta > 0)
        else:
            assert np.array_equal(d["phiB"], d["phiLDA"])


def test_fluid_at_rest_has_zero_sensor():
    # |v|_max = |v|_min: the ratio of eq. 56 is 0/0; reading C24: s = 0 (no compression without motion)
    mesh = wl.uniform_mesh(12, 12, 1.0, 1.0, periodic=True)
    x = mesh.xy[:, 0]
    W = wl.primitive_to_conserved(1.0 + 0.2 * np.sin(2 * np.pi * x), 0 * x, 0 * x, 1.0 + 0.1 * np.cos(2 * np.pi * x))
    d = _om(mesh, W, oracle.SCHEME_BX).dump_stage1()
    assert np.array_equal(d["phiB"], d["phiLDA"]) and np.all(np.isfinite(d["phiB"]))


def test_theta_is_first_order_in_h_for_a_smooth_field():
    # "O(1) in regions of smooth flow, which makes theta O(h)" (L517)
    tmax = []
    for n in (24, 48, 96):
        mesh = wl.uniform_mesh(n, n, 10.0, 10.0, periodic=True)
        x, y = mesh.xy[:, 0], mesh.xy[:, 1]
        u = 0.5 + 0.2 * np.sin(2 * np.pi * x / 10.0) * np.cos(2 * np.pi * y / 10.0)    # smooth, compressive in places
        W = wl.primitive_to_conserved(1.0 + 0.1 * np.cos(2 * np.pi * x / 10.0), u, 0.3 + 0 * x, 1.0 + 0 * x)
        tmax.append(_theta_numpy(mesh, W)[0].max())
        d = _om(mesh, W, oracle.SCHEME_BX).dump_stage1()
        th = _theta_numpy(mesh, W)[0][:, None, None]
        assert np.abs(d["phiB"] - (th * d["phiN"] + (1 - th) * d["phiLDA"])).max() <= 1e-13 * np.abs(d["phiN"]).max()
    assert tmax[0] / tmax[1] == pytest.approx(2.0, rel=0.15) and tmax[1] / tmax[2] == pytest.approx(2.0, rel=0.1)


def _l1_density(mesh, om, exact):
    vol = om.geometry()[1]
    return float((vol * np.abs(om.get_state()[0] - exact)).sum() / vol.sum())


def test_stationary_vortex_bx_gives_the_lda_result():
    # L885: "since there are no shocks present, the Bx scheme yields exactly the same results as the LDA scheme" (Fig. 19,
    # a log-log plot): the density errors of Bx approach those of LDA as theta = O(h) vanishes, and beat B and N
    gap = []
    for n in (32, 64):
        mesh = wl.uniform_mesh(n, n, 10.0, 10.0, periodic=True)
        W = wl.vortex_state(mesh)
        exact = wl.vortex_exact_density(mesh)
        err = {}
        for name, sch in (("LDA", oracle.SCHEME_LDA), ("Bx", oracle.SCHEME_BX), ("B", oracle.SCHEME_B), ("N", oracle.SCHEME_N)):
            om = _om(mesh, W, sch, time_order=2, threads=4)
            om.step(10 ** 6, 1.0)
            err[name] = _l1_density(mesh, om, exact)
        assert err["LDA"] <= err["Bx"] < err["B"] < err["N"]
        gap.append(err["Bx"] / err["LDA"] - 1.0)
    assert gap[0] <= 0.25 and gap[1] <= 0.08 and gap[1] < 0.5 * gap[0]


def test_sound_wave_b_bx_lda_indistinguishable():
    # L778: "results obtained with the LDA scheme are indistinguishable from those obtained with both B and Bx"
    mesh = wl.uniform_mesh(64, 4, 1.0, 4.0 / 64.0, periodic=True)
    W = wl.sound_wave_state(mesh)
    out = {}
    for name, sch in (("LDA", oracle.SCHEME_LDA), ("Bx", oracle.SCHEME_BX)):
        om = _om(mesh, W, sch, time_order=2)
        om.step(30)
        out[name] = om.get_state()
    amp = np.abs(W[0] - W[0].mean()).max()
    # (in the compression half of the wave s = O(L k) = O(1) as L517 says, theta = s^2 h is not small at 64 cells per
    # wavelength, and still the two solutions differ by a few per cent of the amplitude: the same curve in Fig. 14)
    assert np.abs(out["Bx"][0] - out["LDA"][0]).max() <= 0.05 * amp


def test_sod_bx_is_n_at_the_shock_and_lda_like_in_the_rarefaction():
    # At a captured shock div v ~ -du/h, so s ~ L/h and theta = min(1, s^2 h) = 1: Bx IS the N scheme there (Noh, L824:
    # "results for the B and Bx schemes ... almost indistinguishable from the results with the N scheme").  In the
    # rarefaction (expansion, div v > 0) it IS the LDA scheme.  (The remark of L798 that Bx gives sharper shocks than
    # B is not reproduced by a sensor clamped at 1 -- DESIGN.md reading C26.)
    cfg = wl.make_config("sod", n=128)
    mesh = cfg.mesh
    row = mesh.grid_ij[:, 1] == mesh.shape[1] // 2
    order = np.argsort(mesh.xy[row, 0])
    x = mesh.xy[row, 0][order]
    t_end = 0.12
    rho = {}
    for name, sch in (("N", oracle.SCHEME_N), ("Bx", oracle.SCHEME_BX), ("B", oracle.SCHEME_B)):
        om = oracle.OracleMesh(mesh.xy, mesh.tri, period=mesh.period, vertex_flag=cfg.vertex_flag, wall_edge=cfg.wall_edge, scheme=sch)
        om.set_state(cfg.W0)
        om.step(10 ** 6, t_end)
        tot, mr, mp = om.diagnostics()
        assert mr > 0 and mp > 0
        rho[name] = om.get_state()[0][row][order]
        assert rho[name].max() <= 1.0 + 0.05 and rho[name].min() >= 0.125 - 0.02
    lo, hi = 0.125 + 0.1 * (0.265574 - 0.125), 0.125 + 0.9 * (0.265574 - 0.125)   # post-shock density of the exact solution
    width = {k: int(((x > 0.62) & (r > lo) & (r < hi)).sum()) for k, r in rho.items()}
    assert abs(width["Bx"] - width["N"]) <= 2 and width["B"] < width["N"]
    # exact rarefaction fan (textbook): u = 2/(g+1) (c_L + xi), c = c_L - (g-1)/2 u, rho = rho_L (c/c_L)^(2/(g-1)), xi = (x-x0)/t
    g = 1.4
    cL = np.sqrt(g)
    fan = (x > 0.5 - cL * t_end + 0.02) & (x < 0.5 - 0.0703 * t_end - 0.02)      # head speed -c_L, tail speed u* - c* = -0.0703
    xi = (x[fan] - 0.5) / t_end
    u = 2.0 / (g + 1.0) * (cL + xi)
    exact = (1.0 - (g - 1.0) / 2.0 * u / cL) ** (2.0 / (g - 1.0))
    err = {k: float(np.abs(r[fan] - exact).mean()) for k, r in rho.items()}
    assert fan.sum() >= 8 and err["Bx"] < 0.6 * err["N"]


def test_uniform_flow_and_conservation():
    mesh = wl.flip_edges(wl.jitter_mesh(wl.uniform_mesh(16, 16, 1.0, 1.0, periodic=True), 0.2, seed=11), seed=2)
    Wu = wl.uniform_state(mesh, 1.3, 0.4, -0.7, 2.1)
    om = _om(mesh, Wu, oracle.SCHEME_BX)
    om.step(3)
    assert np.array_equal(om.get_state(), Wu)
    W = wl.random_smooth_state(mesh, mach=0.9, seed=4)
    om.set_state(W)
    tot0, _, _ = om.diagnostics()
    om.step(15)
    tot1, mr, mp = om.diagnostics()
    scale = np.array([tot0[0], np.abs(W[1:3]).max(), np.abs(W[1:3]).max(), tot0[3]])
    assert np.all(np.abs(tot1 - tot0) < 2e-13 * scale) and mr > 0 and mp > 0
