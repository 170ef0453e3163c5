"""The variable-valence workload (stand-in for the paper's Delaunay-refined meshes, L685): the generator's
invariants, the layout stage on it, and the oracle's mesh-independent pins (uniform flow, conservation) there."""
import numpy as np
import pytest

import oracle
import paper_1705_02028_b200 as mrd
import workloads as wl


def _mesh(periodic, seed=11):
    return wl.flip_edges(wl.jitter_mesh(wl.uniform_mesh(40, 36, 2.0, 1.8, periodic=periodic), 0.2, seed=3), seed=seed)


@pytest.mark.parametrize("periodic", [True, False])
def test_flip_edges_keeps_a_valid_triangulation(periodic):
    base = wl.jitter_mesh(wl.uniform_mesh(40, 36, 2.0, 1.8, periodic=periodic), 0.2, seed=3)
    m = _mesh(periodic)
    assert m.tri.shape == base.tri.shape and np.array_equal(m.xy, base.xy)
    assert (m.tri != base.tri).any(axis=1).mean() > 0.2                      # a good part of the mesh was flipped
    e = np.concatenate([m.tri[:, [0, 1]], m.tri[:, [1, 2]], m.tri[:, [2, 0]]]).astype(np.int64)
    key = e[:, 0] * m.nv + e[:, 1]
    assert len(np.unique(key)) == len(key)                                   # manifold: every directed edge once
    mate = np.isin(e[:, 1] * m.nv + e[:, 0], key)
    b0 = np.concatenate([base.tri[:, [0, 1]], base.tri[:, [1, 2]], base.tri[:, [2, 0]]]).astype(np.int64)
    kb = b0[:, 0] * m.nv + b0[:, 1]
    bmate = np.isin(b0[:, 1] * m.nv + b0[:, 0], kb)
    assert set(key[~mate].tolist()) == set(kb[~bmate].tolist())              # boundary edges untouched (none if periodic)
    val = np.bincount(m.tri.ravel(), minlength=m.nv)
    assert val.min() >= (3 if periodic else 1) and val.max() >= 8 and (val != 6).mean() > 0.5   # variable valence
    L = mrd.Layout(m.xy, m.tri, period=m.period)
    g = L.get()
    assert g["area"].min() > 0 and g["area"].sum() == pytest.approx(2.0 * 1.8, rel=1e-13)   # still CCW, still tiles the domain
    assert np.array_equal(np.sort(np.diff(g["csr_off"])), np.sort(val))      # the CSR is general (variable degree)
    assert wl.flip_edges(base, seed=11).tri.tobytes() == m.tri.tobytes()     # seeded


def test_oracle_pins_hold_on_the_variable_valence_mesh():
    m = _mesh(True)
    W = wl.uniform_state(m, 1.3, 0.4, -0.7, 2.1)
    om = oracle.OracleMesh(m.xy, m.tri, period=m.period)
    om.set_state(W)
    om.step(3)
    assert np.array_equal(om.get_state(), W)                                 # uniform flow: residuals exactly zero
    W = wl.random_smooth_state(m, mach=0.8, seed=2)
    om.set_state(W)
    t0 = om.diagnostics()[0]
    om.step(10)
    t1 = om.diagnostics()[0]
    assert np.abs(t1 - t0).max() <= 1e-13 * np.abs(t0).max()                 # conservation (L455) on a periodic mesh
