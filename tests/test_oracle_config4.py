"""Reading D3, as a property of the ORACLE: on the four-quadrant Riemann problem (PAPER.md
L944-L969, split at the centre, frozen boundary) the blended scheme with the RK2 of eq. 60-65 loses positivity in the
interaction of the four shocks next to the low-pressure quadrant -- in the interior, a few cells from the centre on the
diagonal, after ~100 steps at ANY resolution and any CFL number (a self-similar start-up structure), whatever the last bits
of the initial state.  It is therefore neither the frozen boundary (reading C16) nor round-off in Theta (reading C10).
First-order time stepping (B1), the variant the paper recommends for strong shocks (Bmax2, L503), the shock-sensor blend
(Bx2) and the positive N scheme (N1) all run to t = 0.3."""
import numpy as np
import pytest

import oracle
import workloads as wl


def run(n, scheme, order, cfl=0.5, perturb=None, t_end=0.3):
    cfg = wl.make_config("riemann4", n=n)
    m = cfg.mesh
    om = oracle.OracleMesh(m.xy, m.tri, vertex_flag=cfg.vertex_flag, scheme=scheme, time_order=order, cfl=cfl, threads=4)
    W0 = cfg.W0 if perturb is None else cfg.W0 * (1.0 + 1e-15 * np.random.default_rng(perturb).standard_normal(cfg.W0.shape))
    om.set_state(W0)
    steps, t = 0, 0.0
    try:
        while True:
            k, t, _ = om.step(1, t_end=t_end)
            steps += k
            if k == 0:
                return m, om, steps, t, None
    except oracle.OracleError as e:
        assert e.code == oracle.ORC_ENONPHYSICAL
        return m, om, steps, t, steps + 1


@pytest.mark.slow
def test_b2_fails_at_the_four_shock_interaction_not_at_the_boundary_and_other_schemes_complete():
    where = {}
    for n in (63, 127):
        m, om, steps, t, failed = run(n, oracle.SCHEME_B, 2)
        assert failed is not None and 60 <= failed <= 200            # ~100 steps at either resolution
        p = wl.conserved_to_primitive(om.get_state())[3]
        i = int(np.argmin(p))
        where[n] = m.xy[i]
        assert np.abs(m.xy[i] - 0.5).max() < 8.0 / n                  # a few cells from the centre: the interior
        assert abs(m.xy[i, 0] - m.xy[i, 1]) < 1e-12                   # on the diagonal, in the SW (low-pressure) quadrant
        assert m.xy[i, 0] < 0.5
        assert t * n == pytest.approx(5.04, rel=0.1)                  # self-similar: the same time in units of cells
    # not round-off: a 1e-15 perturbation of the initial state moves the step a little, not the place
    m, om, steps, t, failed = run(63, oracle.SCHEME_B, 2, perturb=1)
    assert failed is not None and 60 <= failed <= 200
    i = int(np.argmin(wl.conserved_to_primitive(om.get_state())[3]))
    assert np.abs(m.xy[i] - where[63]).max() <= 2.0 / 63
    # not the time-step size: CFL 0.2 fails at the same TIME
    m, om, steps, t2, failed = run(63, oracle.SCHEME_B, 2, cfl=0.2)
    assert failed is not None and 0.07 < t2 < 0.12
    # the other schemes complete
    for scheme, order in [(oracle.SCHEME_B, 1), (oracle.SCHEME_BMAX, 2), (oracle.SCHEME_N, 1), (oracle.SCHEME_BX, 2)]:
        m, om, steps, t, failed = run(63, scheme, order)
        assert failed is None and t == pytest.approx(0.3, abs=1e-15), (scheme, order)
        rho, _, _, p = wl.conserved_to_primitive(om.get_state())
        assert rho.min() > 0.12 and p.min() > 0.02
