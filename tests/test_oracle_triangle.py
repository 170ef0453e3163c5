"""Pins for the oracle's single-triangle residual and distribution (§3.2-3.4).

Independent references built here with numpy only: the Simpson contour integral of the Euler flux
(eq. 12), a literal evaluation of eq. 36/48/50 with K from complex-step differentiation and K+/-
from numpy's eig, and the symmetrising-variable block form (reading C9).
"""
import numpy as np
import pytest

import oracle
from helpers import flux_normal, prim_to_cons

GAMMA = 1.4
G1 = GAMMA - 1.0
RNG = np.random.default_rng(1705_02028)


def cross2(a, b):
    return a[0] * b[1] - a[1] * b[0]


def random_triangle():
    while True:
        xy = RNG.uniform(-1, 1, size=(3, 2))
        cross = cross2(xy[1] - xy[0], xy[2] - xy[0])
        if abs(cross) > 0.2:
            return xy if cross > 0 else xy[[0, 2, 1]]


def random_states(mach=1.0, jitter=0.3):
    rho0, p0 = RNG.uniform(0.3, 2.0), RNG.uniform(0.3, 2.0)
    c0 = np.sqrt(GAMMA * p0 / rho0)
    ang = RNG.uniform(0, 2 * np.pi)
    W = np.empty((3, 4))
    for j in range(3):
        rho = rho0 * (1 + jitter * RNG.uniform(-1, 1))
        p = p0 * (1 + jitter * RNG.uniform(-1, 1))
        u = mach * c0 * (np.cos(ang) + jitter * RNG.uniform(-1, 1))
        v = mach * c0 * (np.sin(ang) + jitter * RNG.uniform(-1, 1))
        W[j] = prim_to_cons(rho, u, v, p, GAMMA)
    return W


CASES = [(random_triangle(), random_states(m)) for m in (0.01, 0.3, 0.8, 1.0, 1.5, 3.0, 8.0) for _ in range(6)]


# ---------------------------------------------------------------- independent numpy pieces
def Z_of_W(W):
    rho, m, n, e = W
    p = G1 * (e - 0.5 * (m * m + n * n) / rho)
    s = np.sqrt(rho)
    return np.array([s, m / s, n / s, (e + p) / s])


def W_of_Z(Z):
    # reading C1: W is quadratic in Z
    return np.array([Z[0] ** 2, Z[0] * Z[1], Z[0] * Z[2], Z[0] * Z[3] / GAMMA + G1 / (2 * GAMMA) * (Z[1] ** 2 + Z[2] ** 2)])


def contour_integral(W, xy):
    """phi = closed integral of F.n_out over the triangle boundary (eq. 12) for Z linear on each edge:
    Simpson's rule is exact because F is quadratic in Z (L411)."""
    Z = np.array([Z_of_W(w) for w in W])
    phi = np.zeros(4)
    for a in range(3):
        b = (a + 1) % 3
        e = xy[b] - xy[a]
        length = np.hypot(*e)
        nx, ny = e[1] / length, -e[0] / length        # outward for a counter-clockwise triangle
        fa = flux_normal(W_of_Z(Z[a]), nx, ny, GAMMA)
        fm = flux_normal(W_of_Z(0.5 * (Z[a] + Z[b])), nx, ny, GAMMA)
        fb = flux_normal(W_of_Z(Z[b]), nx, ny, GAMMA)
        phi += length / 6.0 * (fa + 4.0 * fm + fb)
    return phi


def split_by_spectral_projectors(J):
    """f(J) = sum_k f(mu_k) P_k with the Lagrange projectors P_k = prod_{m != k} (J - mu_m)/(mu_k - mu_m)
    over the DISTINCT eigenvalues (J is diagonalisable, eq. 40): needs no eigenvectors, so the
    repeated eigenvalue w causes no trouble. Eigenvalues from numpy; the closest pair is merged."""
    lam = np.sort(np.linalg.eigvals(J).real)
    gaps = np.diff(lam)
    k = int(np.argmin(gaps))
    mu = np.array([*lam[:k], 0.5 * (lam[k] + lam[k + 1]), *lam[k + 2:]])
    I = np.eye(4)
    Jp, Jm = np.zeros((4, 4)), np.zeros((4, 4))
    for a in range(3):
        P = I.copy()
        for b in range(3):
            if b != a:
                P = P @ (J - mu[b] * I) / (mu[a] - mu[b])
        Jp += max(mu[a], 0.0) * P
        Jm += min(mu[a], 0.0) * P
    return Jp, Jm


def literal_reference(W, xy):
    """eq. 36, 48-51 evaluated literally: K_i from the differentiated flux at the linearised state,
    K_i^+/- from spectral projectors, N-hat from numpy inv, hat-W_i = D(Zbar) Z_i (not differences)."""
    Z = np.array([Z_of_W(w) for w in W])
    Zb = Z.mean(axis=0)
    Wb = W_of_Z(Zb)
    D = np.array([[2 * Zb[0], 0, 0, 0], [Zb[1], Zb[0], 0, 0], [Zb[2], 0, Zb[0], 0],
                  [Zb[3] / GAMMA, G1 * Zb[1] / GAMMA, G1 * Zb[2] / GAMMA, Zb[0] / GAMMA]])
    What = Z @ D.T
    K, Kp, Km = [], [], []
    for i in range(3):
        a, b = xy[(i + 1) % 3], xy[(i + 2) % 3]
        e = b - a
        n = np.array([-e[1], e[0]])                   # inward, length-scaled (eq. 35)
        J = np.empty((4, 4))
        for k in range(4):
            Wc = Wb.astype(complex)
            Wc[k] += 1e-30j
            J[:, k] = flux_normal(Wc, n[0], n[1], GAMMA).imag / 1e-30
        J *= 0.5                                       # eq. 37, d = 2
        Jp, Jm = split_by_spectral_projectors(J)
        K.append(J)
        Kp.append(Jp)
        Km.append(Jm)
    Nhat = np.linalg.inv(sum(Km))
    phiT = sum(K[i] @ What[i] for i in range(3))
    inflow = Nhat @ sum(Km[j] @ What[j] for j in range(3))
    phiN = np.array([Kp[i] @ (What[i] - inflow) for i in range(3)])
    phiLDA = np.array([-Kp[i] @ Nhat @ phiT for i in range(3)])
    return phiT, phiN, phiLDA


def symmetrising_reference(W, xy):
    """Reading C9: in dQ = (dp/c, rho du, rho dv, dp - c^2 drho) the K_i are a symmetric 3x3 acoustic
    block plus a scalar entropy mode; N and LDA evaluated there, then mapped back to conserved."""
    Z = np.array([Z_of_W(w) for w in W])
    Zb = Z.mean(axis=0)
    u, v, h = Zb[1] / Zb[0], Zb[2] / Zb[0], Zb[3] / Zb[0]
    q2 = u * u + v * v
    c = np.sqrt(G1 * (h - 0.5 * q2))
    D = np.array([[2 * Zb[0], 0, 0, 0], [Zb[1], Zb[0], 0, 0], [Zb[2], 0, Zb[0], 0],
                  [Zb[3] / GAMMA, G1 * Zb[1] / GAMMA, G1 * Zb[2] / GAMMA, Zb[0] / GAMMA]])
    dW = (Z - Z[0]) @ D.T
    M = np.array([[1 / c, 0, 0, -1 / c ** 2], [u / c, 1, 0, -u / c ** 2], [v / c, 0, 1, -v / c ** 2],
                  [h / c, u, v, -0.5 * q2 / c ** 2]])
    Mi = np.linalg.inv(M)
    dQ = dW @ Mi.T
    Kp, Km = [], []
    for i in range(3):
        a, b = xy[(i + 1) % 3], xy[(i + 2) % 3]
        e = b - a
        length = np.hypot(*e)
        n = np.array([-e[1], e[0]]) / length
        w = u * n[0] + v * n[1]
        out = []
        for sgn in (+1, -1):
            part = (lambda x: 0.5 * (x + sgn * abs(x)))
            l1, l2, l3 = (0.5 * length * part(x) for x in (w + c, w - c, w))
            A = np.zeros((4, 4))
            A[0, 0] = 0.5 * (l1 + l2)
            A[0, 1:3] = A[1:3, 0] = 0.5 * (l1 - l2) * n
            A[1:3, 1:3] = l3 * np.eye(2) + (0.5 * (l1 + l2) - l3) * np.outer(n, n)
            A[3, 3] = l3
            out.append(A)
        Kp.append(out[0])
        Km.append(out[1])
    S = sum(Km)
    Sinv = np.zeros((4, 4))
    Sinv[:3, :3] = np.linalg.inv(S[:3, :3])
    Sinv[3, 3] = 1.0 / S[3, 3] if S[3, 3] != 0 else 0.0
    phiT = sum((Kp[i] + Km[i]) @ dQ[i] for i in range(3))
    inflow = Sinv @ sum(Km[j] @ dQ[j] for j in range(3))
    phiN = np.array([M @ (Kp[i] @ (dQ[i] - inflow)) for i in range(3)])
    phiLDA = np.array([-(M @ (Kp[i] @ (Sinv @ phiT))) for i in range(3)])
    return M @ phiT, phiN, phiLDA


def scale_of(o):
    return max(np.abs(o["phiN"]).max(), np.abs(o["phiLDA"]).max(), np.abs(o["phiT"]).max(), 1e-300)


# ---------------------------------------------------------------- pins
@pytest.mark.parametrize("xy,W", CASES)
def test_residual_is_the_contour_integral_of_the_flux(xy, W):
    o = oracle.triangle_stage1(GAMMA, W, xy)
    ref = contour_integral(W, xy)
    flux_scale = max(np.abs(flux_normal(w, 1.0, 1.0, GAMMA)).max() for w in W)
    assert np.allclose(o["phiT"], ref, rtol=0, atol=2e-14 * flux_scale * 3)


@pytest.mark.parametrize("xy,W", CASES)
def test_distribution_is_conservative(xy, W):
    # sum_i phi_i^N = phi^T, sum_i beta_i = I, blended scheme too (L455)
    o = oracle.triangle_stage1(GAMMA, W, xy)
    s = scale_of(o)
    for key in ("phiN", "phiLDA", "phiB"):
        assert np.allclose(o[key].sum(axis=0), o["phiT"], rtol=0, atol=1e-12 * s), key
    assert np.allclose(o["Nhat"] @ o["sumKm"], np.eye(4), atol=1e-9)


@pytest.mark.parametrize("xy,W", CASES)
def test_against_literal_evaluation(xy, W):
    o = oracle.triangle_stage1(GAMMA, W, xy)
    phiT, phiN, phiLDA = literal_reference(W, xy)
    s = scale_of(o)
    # the literal form (hat-W_i, not differences) carries cancellation noise ~ eps * |K| |W|
    noise = 1e-9 * max(s, np.abs(W).max())
    assert np.allclose(o["phiT"], phiT, rtol=0, atol=noise)
    assert np.allclose(o["phiN"], phiN, rtol=0, atol=noise)
    assert np.allclose(o["phiLDA"], phiLDA, rtol=0, atol=noise)


@pytest.mark.parametrize("xy,W", CASES)
def test_against_symmetrising_variable_form(xy, W):
    o = oracle.triangle_stage1(GAMMA, W, xy)
    phiT, phiN, phiLDA = symmetrising_reference(W, xy)
    s = scale_of(o)
    assert np.allclose(o["phiT"], phiT, rtol=0, atol=1e-11 * s)
    assert np.allclose(o["phiN"], phiN, rtol=0, atol=1e-11 * s)
    assert np.allclose(o["phiLDA"], phiLDA, rtol=0, atol=1e-11 * s)


@pytest.mark.parametrize("xy,W", CASES)
def test_blend(xy, W):
    # eq. 52-53: Theta in [0,1]; phi^B = Theta phi^N + (1-Theta) phi^LDA; Theta_k = 1 (B = N) when all
    # phi^N_{j,k} share a sign
    o = oracle.triangle_stage1(GAMMA, W, xy)
    th = o["theta"]
    assert np.all(th >= 0) and np.all(th <= 1)
    den = np.abs(o["phiN"]).sum(axis=0)
    assert np.allclose(th, np.minimum(1.0, np.abs(o["phiT"]) / den), rtol=1e-13)
    assert np.allclose(o["phiB"], th * o["phiN"] + (1 - th) * o["phiLDA"], rtol=1e-13, atol=1e-300)
    for k in range(4):
        col = o["phiN"][:, k]
        if np.all(col > 0) or np.all(col < 0):
            assert abs(th[k] - 1.0) < 1e-9
            assert np.allclose(o["phiB"][:, k], col, rtol=1e-8)


def test_uniform_state_gives_exactly_zero():
    # L237 / L891 and SURVEY §8c O3: all residuals exactly 0, including u = v = 0 (stagnation rule C8)
    for prim in [(1.3, 0.4, -0.7, 2.1), (1.0, 0.0, 0.0, 1.0), (0.125, 3.0, 0.0, 0.1)]:
        W = np.tile(prim_to_cons(*prim, GAMMA), (3, 1))
        o = oracle.triangle_stage1(GAMMA, W, random_triangle())
        for key in ("phiT", "phiN", "phiLDA", "phiB", "theta"):
            assert np.all(o[key] == 0.0), (prim, key)


def test_stagnation_rule_is_the_limit():
    # reading C8: at u = v = 0 exactly the generalised inverse reproduces the u -> 0 limit
    xy = random_triangle()
    prims = [(1.0, 1.0), (0.125, 0.1), (0.6, 0.4)]
    W0 = np.array([prim_to_cons(r, 0.0, 0.0, p, GAMMA) for r, p in prims])
    o0 = oracle.triangle_stage1(GAMMA, W0, xy)
    assert np.all(o0["Nhat"][0, :] == 0) and np.all(o0["Nhat"][:, 0] == 0)
    s = scale_of(o0)
    for eps, ang in [(1e-7, 0.3), (1e-7, 2.5), (1e-10, 4.0)]:
        We = np.array([prim_to_cons(r, eps * np.cos(ang), eps * np.sin(ang), p, GAMMA) for r, p in prims])
        oe = oracle.triangle_stage1(GAMMA, We, xy)
        for key in ("phiT", "phiN", "phiLDA", "phiB"):
            assert np.allclose(oe[key], o0[key], rtol=0, atol=50 * eps * s), (eps, key)


def test_sod_like_jump_at_rest_is_finite_and_conservative():
    xy = np.array([[0.0, 0.0], [1.0, 0.0], [1.0, 1.0]])
    W = np.array([prim_to_cons(1.0, 0, 0, 1.0, GAMMA), prim_to_cons(0.125, 0, 0, 0.1, GAMMA),
                  prim_to_cons(0.125, 0, 0, 0.1, GAMMA)])
    o = oracle.triangle_stage1(GAMMA, W, xy)
    assert np.all(np.isfinite(o["phiB"]))
    assert np.allclose(o["phiB"].sum(axis=0), o["phiT"], atol=1e-14)
    assert np.allclose(o["phiT"], contour_integral(W, xy), atol=1e-14)
    assert o["phiT"][0] == 0.0 and o["phiT"][3] == 0.0      # no mass / energy flux at rest


@pytest.mark.parametrize("xy,W", CASES[::3])
def test_rotation_covariance(xy, W):
    # rotating the triangle and the velocities rotates the momentum residuals and leaves mass/energy alone
    th = 0.7345
    Rm = np.array([[np.cos(th), -np.sin(th)], [np.sin(th), np.cos(th)]])
    xy2 = xy @ Rm.T
    W2 = W.copy()
    W2[:, 1:3] = W[:, 1:3] @ Rm.T
    o, o2 = oracle.triangle_stage1(GAMMA, W, xy), oracle.triangle_stage1(GAMMA, W2, xy2)
    s = scale_of(o)
    for key in ("phiN", "phiLDA"):
        a, b = o[key].copy(), o2[key]
        a[:, 1:3] = a[:, 1:3] @ Rm.T
        assert np.allclose(a, b, rtol=0, atol=1e-11 * s), key
    assert abs(o["sT"] - o2["sT"]) < 1e-13 * o["sT"]


@pytest.mark.parametrize("xy,W", CASES[1::3])
def test_cyclic_relabelling(xy, W):
    o = oracle.triangle_stage1(GAMMA, W, xy)
    perm = [1, 2, 0]
    o2 = oracle.triangle_stage1(GAMMA, W[perm], xy[perm])
    s = scale_of(o)
    for key in ("phiN", "phiLDA", "phiB"):
        assert np.allclose(o[key][perm], o2[key], rtol=0, atol=1e-11 * s), key
    assert np.allclose(o["phiT"], o2["phiT"], rtol=0, atol=1e-11 * s)


@pytest.mark.parametrize("xy,W", CASES[2::3])
def test_mirror_symmetry(xy, W):
    # reflection about x = y: (x,y,u,v) -> (y,x,v,u); orientation flips, so swap two nodes
    xy2 = xy[:, ::-1][[0, 2, 1]]
    W2 = W[:, [0, 2, 1, 3]][[0, 2, 1]]
    o, o2 = oracle.triangle_stage1(GAMMA, W, xy), oracle.triangle_stage1(GAMMA, W2, xy2)
    s = scale_of(o)
    for key in ("phiN", "phiLDA", "phiB"):
        a = o[key][:, [0, 2, 1, 3]][[0, 2, 1]]
        assert np.allclose(a, o2[key], rtol=0, atol=1e-11 * s), key


def test_signal_speed():
    # eq. 44-45 with vertex values (reading C14)
    xy, W = CASES[5]
    o = oracle.triangle_stage1(GAMMA, W, xy)
    lmax = max(np.hypot(*(xy[(i + 2) % 3] - xy[(i + 1) % 3])) for i in range(3))
    sp = []
    for w in W:
        rho, u, v = w[0], w[1] / w[0], w[2] / w[0]
        p = G1 * (w[3] - 0.5 * rho * (u * u + v * v))
        sp.append(np.hypot(u, v) + np.sqrt(GAMMA * p / rho))
    assert abs(o["sT"] - lmax * max(sp)) < 1e-14 * o["sT"]


@pytest.mark.parametrize("xy,W", CASES[::4])
def test_stage2_reduces_to_stage1_when_nothing_moved(xy, W):
    # eq. 57, 62-63 with W* = W^n: mass terms vanish and the averages return the stage-1 values
    o = oracle.triangle_stage1(GAMMA, W, xy)
    o2 = oracle.triangle_stage2(GAMMA, W, W, xy, 0.01, o["phiT"], o["phiN"])
    assert np.array_equal(o2["PhiT"], o["phiT"])
    assert np.array_equal(o2["PhiN"], o["phiN"])
    assert np.allclose(o2["PhiLDA"], o["phiLDA"], rtol=1e-14, atol=0)
    assert np.allclose(o2["PhiB"], o["phiB"], rtol=1e-13, atol=0)


@pytest.mark.parametrize("xy,W", CASES[1::4])
def test_stage2_definitions(xy, W):
    # eq. 57 + 61-65 re-evaluated with numpy from the oracle's own stage-1 pieces at W^n and W*
    Ws = W * (1 + 0.01 * RNG.uniform(-1, 1, size=W.shape))
    dt = 0.013
    area = 0.5 * cross2(xy[1] - xy[0], xy[2] - xy[0])
    on, os_ = oracle.triangle_stage1(GAMMA, W, xy), oracle.triangle_stage1(GAMMA, Ws, xy)
    o2 = oracle.triangle_stage2(GAMMA, W, Ws, xy, dt, on["phiT"], on["phiN"])
    dW = (Ws - W) / dt
    PhiT = area / 3 * dW.sum(axis=0) + 0.5 * (on["phiT"] + os_["phiT"])
    PhiN = area / 3 * dW + 0.5 * (on["phiN"] + os_["phiN"])
    s = max(np.abs(PhiN).max(), np.abs(PhiT).max())
    assert np.allclose(o2["PhiT"], PhiT, rtol=0, atol=1e-13 * s)
    assert np.allclose(o2["PhiN"], PhiN, rtol=0, atol=1e-13 * s)
    assert np.allclose(o2["PhiLDA"].sum(axis=0), o2["PhiT"], rtol=0, atol=1e-11 * s)     # sum beta_i = I
    # beta_i(W*) from the stage-1 LDA residual of W*: beta_i x is linear in x; check on x = phi^T(W*)
    th = np.minimum(1.0, np.abs(o2["PhiT"]) / np.abs(o2["PhiN"]).sum(axis=0))
    assert np.allclose(o2["PhiB"], th * o2["PhiN"] + (1 - th) * o2["PhiLDA"], rtol=1e-12, atol=1e-14 * s)


def test_wall_edge_term():
    # eq. 68-71: zero when v.n = 0; otherwise -(rho, rho u, rho v, rho h) v_n weights 3/4 : 1/4
    Wa = prim_to_cons(1.0, 0.3, 0.0, 1.0, GAMMA)
    Wb = prim_to_cons(0.5, -0.2, 0.0, 0.7, GAMMA)
    Pa, Pb = oracle.wall_edge(GAMMA, Wa, Wb, 0.0, 1.0, 0.5)
    assert np.all(Pa == 0) and np.all(Pb == 0)
    Wa = prim_to_cons(1.0, 0.3, 0.4, 1.0, GAMMA)
    Wb = prim_to_cons(0.5, -0.2, 0.1, 0.7, GAMMA)
    nx, ny, length = 0.6, 0.8, 0.5
    def corr(W):
        rho, u, v = W[0], W[1] / W[0], W[2] / W[0]
        p = G1 * (W[3] - 0.5 * rho * (u * u + v * v))
        vn = u * nx + v * ny
        return -np.array([rho, rho * u, rho * v, W[3] + p]) * vn
    Fa, Fb = corr(Wa), corr(Wb)
    Pa, Pb = oracle.wall_edge(GAMMA, Wa, Wb, nx, ny, length)
    assert np.allclose(Pa, length / 2 * (0.75 * Fa + 0.25 * Fb), rtol=1e-14)
    assert np.allclose(Pb, length / 2 * (0.25 * Fa + 0.75 * Fb), rtol=1e-14)
    assert np.allclose(Pa + Pb, length / 2 * (Fa + Fb), rtol=1e-14)       # eq. 69 (trapezium rule)
    # the corrected normal flux is the wall flux (0, p nx, p ny, 0): computed + correction
    full = flux_normal(Wa, nx, ny, GAMMA) + Fa
    rho, u, v = Wa[0], Wa[1] / Wa[0], Wa[2] / Wa[0]
    p = G1 * (Wa[3] - 0.5 * rho * (u * u + v * v))
    assert np.allclose(full, [0, p * nx, p * ny, 0], atol=1e-14)


def test_operation_count_is_reported():
    xy, W = CASES[8]
    c1 = oracle.count_ops(GAMMA, W, xy, stage=1)
    c2 = oracle.count_ops(GAMMA, W, xy, stage=2)
    flops1 = c1["add"] + c1["mul"] + c1["div"] + c1["sqrt"]
    flops2 = c2["add"] + c2["mul"] + c2["div"] + c2["sqrt"]
    assert 1000 < flops1 < 4000 and flops2 > flops1
