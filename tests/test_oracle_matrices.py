"""Pins for the oracle's Appendix-A matrices (SURVEY.md §8c "pins").

Everything the oracle is compared with here is built independently of it: the flux Jacobian by
complex-step differentiation of the Euler flux (eq. 6-9), eigen-decompositions by numpy.
"""
import numpy as np
import pytest

import oracle
from helpers import flux_normal, prim_to_cons, enthalpy

GAMMA = 1.4
RNG = np.random.default_rng(20170502)


def random_case(mach=None):
    rho = RNG.uniform(0.2, 3.0)
    p = RNG.uniform(0.2, 3.0)
    c = np.sqrt(GAMMA * p / rho)
    m = RNG.uniform(0.0, 3.0) if mach is None else mach
    ang = RNG.uniform(0, 2 * np.pi)
    u, v = m * c * np.cos(ang), m * c * np.sin(ang)
    th = RNG.uniform(0, 2 * np.pi)
    nx, ny = np.cos(th), np.sin(th)
    length = RNG.uniform(0.1, 2.0)
    W = prim_to_cons(rho, u, v, p, GAMMA)
    return W, u, v, enthalpy(W, GAMMA), c, nx, ny, length


def jacobian_complex_step(W, nx, ny):
    J = np.empty((4, 4))
    for k in range(4):
        Wc = W.astype(complex)
        Wc[k] += 1e-30j
        J[:, k] = flux_normal(Wc, nx, ny, GAMMA).imag / 1e-30
    return J


CASES = [random_case() for _ in range(40)] + [random_case(m) for m in (0.0, 1e-9, 0.5, 0.999999, 1.0, 1.000001, 5.0)]


@pytest.mark.parametrize("case", CASES)
def test_K_is_the_flux_jacobian(case):
    # eq. A2 == d(F nx + G ny)/dW (times l/2, eq. 37 with d = 2)
    W, u, v, h, c, nx, ny, length = case
    K, _, _ = oracle.euler_matrices(GAMMA, u, v, h, nx, ny, length)
    J = jacobian_complex_step(W, nx, ny) * length / 2.0
    assert np.allclose(K, J, rtol=1e-13, atol=1e-13 * np.abs(J).max())


@pytest.mark.parametrize("case", CASES)
def test_eigenvectors(case):
    # eq. A3-A7: K R = R Lambda with lambda = (w+c, w-c, w, w) (L1280); corrected eq. A8: R R^-1 = I
    W, u, v, h, c, nx, ny, length = case
    R, Ri, lam = oracle.eigenvectors(GAMMA, u, v, h, nx, ny)
    J = jacobian_complex_step(W, nx, ny)
    w = u * nx + v * ny
    assert np.allclose(lam, [w + c, w - c, w, w], rtol=1e-14, atol=1e-14)
    assert np.allclose(J @ R, R @ np.diag(lam), rtol=1e-12, atol=1e-12 * np.abs(J).max())
    assert np.allclose(R @ Ri, np.eye(4), atol=1e-12 * max(1.0, np.abs(R).max() * np.abs(Ri).max()))


@pytest.mark.parametrize("case", CASES)
def test_A10_A25_recover_K_for_l_equal_lambda(case):
    # L1350: "If we set l_k = lambda_k we recover K"
    W, u, v, h, c, nx, ny, length = case
    w = u * nx + v * ny
    K = oracle.euler_matrices_l(GAMMA, u, v, h, nx, ny, w + c, w - c, w)
    J = jacobian_complex_step(W, nx, ny)
    assert np.allclose(K, J, rtol=1e-12, atol=1e-12 * np.abs(J).max())


@pytest.mark.parametrize("case", CASES)
def test_split_matrices(case):
    # eq. 41-42: K+ + K- = K; K+/- = V Lambda+/- V^-1 with V, Lambda from numpy's eig of the
    # independently differentiated Jacobian; spectra have the right sign.
    W, u, v, h, c, nx, ny, length = case
    K, Kp, Km = oracle.euler_matrices(GAMMA, u, v, h, nx, ny, length)
    scale = np.abs(K).max() + 1e-300
    assert np.allclose(Kp + Km, K, rtol=0, atol=1e-13 * scale)
    J = jacobian_complex_step(W, nx, ny) * length / 2.0
    lam, V = np.linalg.eig(J)
    lam, V = lam.real, V.real
    if np.linalg.cond(V) < 1e8:       # eig of the repeated eigenvalue can be ill-conditioned: skip then
        Vi = np.linalg.inv(V)
        Jp = V @ np.diag(np.maximum(lam, 0.0)) @ Vi
        Jm = V @ np.diag(np.minimum(lam, 0.0)) @ Vi
        tol = 1e-9 * scale
        # eigenvalues within 1e-6 relative of zero make max(lambda,0) non-smooth: compare the sum only
        if np.min(np.abs(lam)) > 1e-5 * np.abs(lam).max():
            assert np.allclose(Kp, Jp, rtol=0, atol=tol)
            assert np.allclose(Km, Jm, rtol=0, atol=tol)
    ep = np.linalg.eigvals(Kp).real
    em = np.linalg.eigvals(Km).real
    assert ep.min() > -1e-7 * scale
    assert em.max() < 1e-7 * scale


def test_split_matrices_via_eigenvector_matrices():
    # K+/- == R diag(l+/-) R^-1 entry by entry, with R from eq. A7 and its inverse taken NUMERICALLY
    # (so that eq. A10-A25 are checked without trusting the corrected eq. A8)
    for case in CASES:
        W, u, v, h, c, nx, ny, length = case
        R, _, lam = oracle.eigenvectors(GAMMA, u, v, h, nx, ny)
        Ri = np.linalg.inv(R)
        _, Kp, Km = oracle.euler_matrices(GAMMA, u, v, h, nx, ny, length)
        lp = 0.5 * length * np.maximum(lam, 0.0)
        lm = 0.5 * length * np.minimum(lam, 0.0)
        scale = np.abs(Kp).max() + np.abs(Km).max()
        assert np.allclose(Kp, R @ np.diag(lp) @ Ri, rtol=0, atol=1e-11 * scale)
        assert np.allclose(Km, R @ np.diag(lm) @ Ri, rtol=0, atol=1e-11 * scale)


def test_printed_A8_fourth_column_is_wrong_and_corrected_one_is_right():
    # reading C7: eq. A8 as printed (L1299) has the sign of its 4th column flipped
    W, u, v, h, c, nx, ny, length = CASES[0]
    R, Ri, _ = oracle.eigenvectors(GAMMA, u, v, h, nx, ny)
    printed = Ri.copy()
    printed[:, 3] *= -1.0
    assert np.abs(R @ Ri - np.eye(4)).max() < 1e-12
    assert np.abs(R @ printed - np.eye(4)).max() > 1e-2


def test_sum_of_K_over_a_closed_triangle_vanishes():
    # sum_i K_i = 0 because sum_i l_i n_i = 0 (eq. 37)
    xy = np.array([[0.1, 0.2], [1.3, 0.1], [0.4, 0.9]])
    W, u, v, h, c, *_ = CASES[3]
    S = np.zeros((4, 4))
    for i in range(3):
        a, b = xy[(i + 1) % 3], xy[(i + 2) % 3]
        e = b - a
        length = np.hypot(*e)
        K, _, _ = oracle.euler_matrices(GAMMA, u, v, h, -e[1] / length, e[0] / length, length)
        S += K
    assert np.abs(S).max() < 1e-14 * np.abs(K).max()
