"""Shared test helpers: the error norm of DESIGN.md reading C17 and small independent numpy
restatements of textbook gas dynamics used to PIN the oracle (none of this is oracle code)."""
import numpy as np


def field_errors(W, Wref):
    """Per conserved field k: max_i |W_k,i - Wref_k,i| / max_i |Wref_k,i|; the two momentum fields
    are normalised by max_i |(rho u, rho v)| (reading C17). Returns the max over fields."""
    W, Wref = np.asarray(W, dtype=np.float64), np.asarray(Wref, dtype=np.float64)
    mom = np.sqrt(Wref[1] ** 2 + Wref[2] ** 2).max()
    scale = np.array([np.abs(Wref[0]).max(), mom, mom, np.abs(Wref[3]).max()])
    scale = np.where(scale > 0, scale, 1.0)
    err = np.abs(W - Wref).reshape(4, -1).max(axis=1) / scale
    return float(err.max())


def flux_normal(W, nx, ny, gamma=1.4):
    """F nx + G ny for conserved W (eq. 6-9 of PAPER.md), plain numpy."""
    rho, m, n, e = W
    u, v = m / rho, n / rho
    p = (gamma - 1.0) * (e - 0.5 * rho * (u * u + v * v))
    vn = u * nx + v * ny
    return np.array([rho * vn, m * vn + p * nx, n * vn + p * ny, (e + p) * vn])


def prim_to_cons(rho, u, v, p, gamma=1.4):
    return np.array([rho, rho * u, rho * v, 0.5 * rho * (u * u + v * v) + p / (gamma - 1.0)])


def enthalpy(W, gamma=1.4):
    rho, m, n, e = W
    p = (gamma - 1.0) * (e - 0.5 * (m * m + n * n) / rho)
    return (e + p) / rho


def exact_riemann(rl, ul, pl, rr, ur, pr, xi, g=1.4):
    """Exact solution of the 1D Riemann problem sampled at xi = (x - x0)/t."""
    cl, cr = np.sqrt(g * pl / rl), np.sqrt(g * pr / rr)

    def f(p, r, pk, c):
        if p > pk:   # shock
            A, B = 2 / ((g + 1) * r), (g - 1) / (g + 1) * pk
            return (p - pk) * np.sqrt(A / (p + B)), np.sqrt(A / (p + B)) * (1 - 0.5 * (p - pk) / (p + B))
        return 2 * c / (g - 1) * ((p / pk) ** ((g - 1) / (2 * g)) - 1), 1 / (r * c) * (p / pk) ** (-(g + 1) / (2 * g))

    p = 0.5 * (pl + pr)
    for _ in range(100):
        fl, dfl = f(p, rl, pl, cl)
        fr, dfr = f(p, rr, pr, cr)
        dp = (fl + fr + ur - ul) / (dfl + dfr)
        p = max(p - dp, 1e-12)
        if abs(dp) < 1e-15 * p:
            break
    us = 0.5 * (ul + ur) + 0.5 * (f(p, rr, pr, cr)[0] - f(p, rl, pl, cl)[0])
    rho = np.empty_like(xi)
    # left of the contact
    if p > pl:
        rsl = rl * ((p / pl + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * p / pl + 1))
        sl = ul - cl * np.sqrt((g + 1) / (2 * g) * p / pl + (g - 1) / (2 * g))
        left = np.where(xi < sl, rl, rsl)
    else:
        rsl = rl * (p / pl) ** (1 / g)
        csl = cl * (p / pl) ** ((g - 1) / (2 * g))
        head, tail = ul - cl, us - csl
        fan = rl * (2 / (g + 1) + (g - 1) / ((g + 1) * cl) * (ul - xi)) ** (2 / (g - 1))
        left = np.where(xi < head, rl, np.where(xi < tail, fan, rsl))
    if p > pr:
        rsr = rr * ((p / pr + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * p / pr + 1))
        sr = ur + cr * np.sqrt((g + 1) / (2 * g) * p / pr + (g - 1) / (2 * g))
        right = np.where(xi > sr, rr, rsr)
    else:
        rsr = rr * (p / pr) ** (1 / g)
        csr = cr * (p / pr) ** ((g - 1) / (2 * g))
        head, tail = ur + cr, us + csr
        fan = rr * (2 / (g + 1) - (g - 1) / ((g + 1) * cr) * (ur - xi)) ** (2 / (g - 1))
        right = np.where(xi > head, rr, np.where(xi > tail, fan, rsr))
    rho = np.where(xi < us, left, right)
    return rho, p, us


def sod_checks(x, W, t=0.2):
    """The physical checks of config 2 on a [4][ny][nx] state at time t (SURVEY 8c "Sod"):
    L1(rho) of eq. 72 against the exact Riemann solution over all rows, the shock position (steepest descent of the
    mid row right of the contact; exact: 0.5 + 1.752156 t), and the row-to-row spread of the density."""
    exact, _, _ = exact_riemann(1.0, 0.0, 1.0, 0.125, 0.0, 0.1, (x - 0.5) / t)
    l1 = float(np.mean(np.abs(W[0] - exact)))
    mid = W[0, W.shape[1] // 2]
    sel = x > 0.75
    k = int(np.argmin(np.diff(mid[sel])))
    spread = float(np.mean(np.abs(W[0] - mid)))
    return l1, float(x[sel][k]), spread
