"""Pins for selective lumping in the oracle (eq. 66-67).  The Galerkin mass matrix is pinned
against its definition m_ij = int_T N_i N_j dA (linear shape functions, quadrature exact for quadratics); the
anti-diffusive term must equal sum_j (|T| delta_ij/3 - m_ij) dW_j/dt with THAT matrix, vanish for equal nodal
increments, sum to zero over the nodes (total residual and conservation unchanged) and keep uniform flow exact."""
import numpy as np
import pytest

import oracle
import workloads as wl

GAMMA = 1.4


def galerkin_mass_by_quadrature(xy):
    # edge-midpoint rule: exact for polynomials of degree 2 on a triangle; N_i = barycentric coordinate i
    area = 0.5 * abs((xy[1, 0] - xy[0, 0]) * (xy[2, 1] - xy[0, 1]) - (xy[1, 1] - xy[0, 1]) * (xy[2, 0] - xy[0, 0]))
    pts = np.array([[0.5, 0.5, 0.0], [0.0, 0.5, 0.5], [0.5, 0.0, 0.5]])
    m = np.zeros((3, 3))
    for lam in pts:
        m += area / 3.0 * np.outer(lam, lam)
    return m, area


def test_selective_lumping_term_matches_the_galerkin_mass_matrix():
    rng = np.random.default_rng(3)
    xy = np.array([[0.0, 0.0], [1.0, 0.1], [0.3, 0.8]])
    mG, area = galerkin_mass_by_quadrature(xy)
    assert np.allclose(mG, area / 12.0 * (np.eye(3) + 1.0), rtol=1e-14)           # eq. 67
    assert np.allclose(mG.sum(axis=1), area / 3.0)                                 # rows sum to the lumped mass
    prim = np.array([[1.0, 0.3, -0.2, 1.0], [1.1, 0.35, -0.1, 1.2], [0.9, 0.2, -0.25, 0.9]])
    Wn = np.array([wl.primitive_to_conserved(*p)[:, None][:, 0] if False else
                   np.array([p[0], p[0] * p[1], p[0] * p[2], 0.5 * p[0] * (p[1] ** 2 + p[2] ** 2) + p[3] / (GAMMA - 1)]) for p in prim])
    Ws = Wn * (1.0 + 0.01 * rng.standard_normal(Wn.shape))
    dt = 0.013
    s1 = oracle.triangle_stage1(GAMMA, Wn, xy)
    a = oracle.triangle_stage2(GAMMA, Wn, Ws, xy, dt, s1["phiT"], s1["phiN"], lumping=0)
    b = oracle.triangle_stage2(GAMMA, Wn, Ws, xy, dt, s1["phiT"], s1["phiN"], lumping=1)
    dW = (Ws - Wn) / dt
    extra = (area / 3.0 * np.eye(3) - mG) @ dW                                     # eq. 66
    scale = np.abs(a["PhiN"]).max()
    assert np.abs((b["PhiN"] - a["PhiN"]) - extra).max() <= 1e-13 * scale
    assert np.abs((b["PhiLDA"] - a["PhiLDA"]) - extra).max() <= 1e-13 * scale
    assert np.abs(extra.sum(axis=0)).max() <= 1e-14 * np.abs(extra).max()          # sums to zero over the nodes
    assert np.abs(b["PhiT"] - a["PhiT"]).max() == 0.0                              # total residual untouched
    assert np.abs(b["PhiB"].sum(axis=0) - b["PhiT"]).max() <= 1e-13 * scale        # still conservative after blending
    assert np.abs(extra).max() > 1e-3 * scale                                      # and it is not a no-op
    # equal increments at the three nodes: the term vanishes (row sums of m^G equal the lumped mass)
    Ws2 = Wn + np.array([0.01, 0.002, -0.003, 0.02])
    c0 = oracle.triangle_stage2(GAMMA, Wn, Ws2, xy, dt, s1["phiT"], s1["phiN"], lumping=0)
    c1 = oracle.triangle_stage2(GAMMA, Wn, Ws2, xy, dt, s1["phiT"], s1["phiN"], lumping=1)
    assert np.abs(c1["PhiN"] - c0["PhiN"]).max() <= 1e-15 * np.abs(c0["PhiN"]).max()


@pytest.mark.parametrize("scheme", [oracle.SCHEME_B, oracle.SCHEME_LDA])
def test_selective_lumping_conserves_and_preserves_uniform_flow(scheme):
    mesh = wl.jitter_mesh(wl.uniform_mesh(18, 16, 1.0, 1.0, periodic=True), 0.2, seed=7)
    Wu = wl.uniform_state(mesh, 1.3, 0.4, -0.7, 2.1)
    om = oracle.OracleMesh(mesh.xy, mesh.tri, period=mesh.period, scheme=scheme, lumping=1)
    om.set_state(Wu)
    om.step(3)
    assert np.array_equal(om.get_state(), Wu)
    W = wl.random_smooth_state(mesh, mach=0.5, seed=4)
    om.set_state(W)
    ref = oracle.OracleMesh(mesh.xy, mesh.tri, period=mesh.period, scheme=scheme)
    ref.set_state(W)
    tot0, _, _ = om.diagnostics()
    om.step(20)
    ref.step(20)
    tot1, mr, mp = om.diagnostics()
    scale = np.array([tot0[0], np.abs(W[1:3]).max(), np.abs(W[1:3]).max(), tot0[3]])
    assert np.all(np.abs(tot1 - tot0) < 2e-13 * scale) and mr > 0 and mp > 0
    d = np.abs(om.get_state() - ref.get_state()).max()
    assert 1e-8 < d < 1.0                                                          # a different scheme, still bounded


@pytest.mark.slow
def test_selective_lumping_lowers_the_error_of_the_advected_vortex():
    # eq. 66 "adds an anti-diffusive term": on the smooth advected vortex (L887) the L1 density error (eq. 72) against
    # the translated exact solution must drop, for LDA and for B
    mesh = wl.uniform_mesh(32, 32, 10.0, 10.0, periodic=True)
    adv = (1.0, 0.5)
    W = wl.vortex_state(mesh, advect=adv)
    for scheme in (oracle.SCHEME_LDA, oracle.SCHEME_B):
        err = []
        for lump in (0, 1):
            om = oracle.OracleMesh(mesh.xy, mesh.tri, period=mesh.period, scheme=scheme, lumping=lump, threads=4)
            om.set_state(W)
            _, t, _ = om.step(100000, t_end=2.0)
            exact = wl.vortex_exact_density(mesh, centre=(5.0 + adv[0] * t, 5.0 + adv[1] * t))
            err.append(np.abs(om.get_state()[0] - exact).mean())
        assert err[1] < 0.95 * err[0], (scheme, err)
