"""Pins for the Bmax / Bmin blends of the oracle (all diagonal entries of Theta set to the maximum /
minimum over k of Theta_kk).  What the paper and the algebra fix: a scalar theta keeps the scheme conservative
(sum_i phi_i = phi^T), theta_min <= Theta_kk <= theta_max orders the three blends between LDA and N, the variants
coincide with B where all Theta_kk are equal, uniform flow stays exactly preserved."""
import numpy as np
import pytest

import oracle
import workloads as wl


def dumps(mesh, W):
    out = {}
    for name, sch in (("B", oracle.SCHEME_B), ("Bmax", oracle.SCHEME_BMAX), ("Bmin", oracle.SCHEME_BMIN)):
        om = oracle.OracleMesh(mesh.xy, mesh.tri, period=mesh.period, scheme=sch)
        om.set_state(W)
        out[name] = om.dump_stage1()
    return out


def test_scalar_theta_is_the_max_and_min_of_the_diagonal_blend():
    mesh = wl.jitter_mesh(wl.uniform_mesh(14, 11, 2.0, 1.5, periodic=True), 0.2, seed=3)
    W = wl.random_smooth_state(mesh, mach=1.1, seed=2)
    d = dumps(mesh, W)
    N, L, T = d["B"]["phiN"], d["B"]["phiLDA"], d["B"]["phiT"]
    den = np.abs(N).sum(axis=1)                                            # [nt][4]
    theta = np.where(den > 0, np.minimum(1.0, np.abs(T) / np.where(den > 0, den, 1.0)), 0.0)
    for name, red in (("Bmax", theta.max(axis=1)), ("Bmin", theta.min(axis=1))):
        th = red[:, None, None]
        expect = th * N + (1.0 - th) * L
        assert np.abs(d[name]["phiB"] - expect).max() <= 1e-15 * np.abs(N).max()
        # conservative for any scalar theta: the nodal residuals still sum to phi^T (L455)
        assert np.abs(d[name]["phiB"].sum(axis=1) - T).max() <= 1e-14 * np.abs(N).max()
    # the diagonal blend lies between the two scalar ones, component by component
    lo = np.minimum(d["Bmin"]["phiB"], d["Bmax"]["phiB"]) - 1e-15 * np.abs(N).max()
    hi = np.maximum(d["Bmin"]["phiB"], d["Bmax"]["phiB"]) + 1e-15 * np.abs(N).max()
    assert np.all(d["B"]["phiB"] >= lo) and np.all(d["B"]["phiB"] <= hi)
    assert np.abs(d["Bmax"]["phiB"] - d["Bmin"]["phiB"]).max() > 1e-3 * np.abs(N).max()   # and they do differ


@pytest.mark.parametrize("scheme", [oracle.SCHEME_BMAX, oracle.SCHEME_BMIN])
def test_variants_conserve_and_preserve_uniform_flow(scheme):
    mesh = wl.jitter_mesh(wl.uniform_mesh(16, 16, 1.0, 1.0, periodic=True), 0.2, seed=11)
    Wu = wl.uniform_state(mesh, 1.3, 0.4, -0.7, 2.1)
    om = oracle.OracleMesh(mesh.xy, mesh.tri, period=mesh.period, scheme=scheme)
    om.set_state(Wu)
    om.step(3)
    assert np.array_equal(om.get_state(), Wu)
    W = wl.random_smooth_state(mesh, mach=0.9, seed=4)
    om.set_state(W)
    tot0, _, _ = om.diagnostics()
    om.step(15)
    tot1, mr, mp = om.diagnostics()
    scale = np.array([tot0[0], np.abs(W[1:3]).max(), np.abs(W[1:3]).max(), tot0[3]])
    assert np.all(np.abs(tot1 - tot0) < 2e-13 * scale) and mr > 0 and mp > 0


def test_bmax_is_the_more_diffusive_variant_on_the_sod_tube():
    # "Bmax favours the N scheme when in doubt ... Bmin favours the LDA scheme" (L503): total variation of the density
    # along the tube after the same number of steps is ordered N <= Bmax <= Bmin (up to a small slack)
    cfg = wl.make_config("sod", n=128)
    tv = {}
    for name, sch, order in (("N", oracle.SCHEME_N, 1), ("Bmax", oracle.SCHEME_BMAX, 2), ("Bmin", oracle.SCHEME_BMIN, 2)):
        om = oracle.OracleMesh(cfg.mesh.xy, cfg.mesh.tri, period=cfg.mesh.period, scheme=sch, time_order=order,
                               vertex_flag=cfg.vertex_flag, wall_edge=cfg.wall_edge)
        om.set_state(cfg.W0)
        om.step(60)
        rho = om.get_state()[0].reshape(cfg.mesh.shape[1], cfg.mesh.shape[0])[cfg.mesh.shape[1] // 2]
        tv[name] = np.abs(np.diff(rho)).sum()
    assert tv["N"] <= tv["Bmax"] * (1 + 1e-3) and tv["Bmax"] <= tv["Bmin"] * (1 + 1e-3)
