"""Pin of the oracle against PAPER.md 5.1.1 (L766-L778): the linear sound wave of amplitude 1e-4 on a quasi-1D periodic
strip, evolved for one period.  "For high enough resolution, all [first-order] schemes show linear convergence" and
"second order convergence is obtained for all second order schemes around h ~ 0.01" (L778); LDA is second order."""
import numpy as np
import pytest

import oracle
import workloads as wl


def l1_error(n, scheme, order):
    mesh = wl.uniform_mesh(n, 4, 1.0, 4.0 / n, periodic=True)
    W = wl.sound_wave_state(mesh)
    om = oracle.OracleMesh(mesh.xy, mesh.tri, period=mesh.period, scheme=scheme, time_order=order, threads=4)
    om.set_state(W)
    _, t, _ = om.step(10 ** 6, t_end=1.0)
    assert t == pytest.approx(1.0, abs=1e-12)
    return np.abs(om.get_state()[0] - W[0]).mean()          # eq. 72 on equal dual cells; exact solution = initial state


@pytest.mark.slow
def test_sound_wave_convergence_orders():
    eN = [l1_error(n, oracle.SCHEME_N, 1) for n in (16, 32, 64)]
    eL = [l1_error(n, oracle.SCHEME_LDA, 2) for n in (16, 32, 64)]
    eB = [l1_error(n, oracle.SCHEME_B, 2) for n in (16, 32, 64)]
    oN = np.log2(eN[1] / eN[2])
    oL = np.log2(eL[1] / eL[2])
    oB = np.log2(eB[1] / eB[2])
    assert 0.7 < oN < 1.2                                   # first order, approached from below
    assert 1.9 < oL < 2.1                                   # LDA + RK2: second order
    assert 1.5 < oB < 2.1 and oB > np.log2(eB[0] / eB[1])   # B: tends to second order as h -> 0.01
    assert eL[2] < eB[2] < eN[2]                            # and the errors are ordered LDA < B < N
    assert eN[2] < 0.5 * 1e-4                               # all far below the wave amplitude
