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
