"""Initial conditions as conserved states W[4][nv] = (rho, rho*u, rho*v, e), SoA, float64.

Only the equation of state (eq. 10) is used to turn primitives into conserved
variables; nothing of the residual-distribution scheme is evaluated here. Each recipe cites the
paper passage that prints it.
"""
from __future__ import annotations

import numpy as np

from .meshes import UniformMesh


def primitive_to_conserved(rho, u, v, p, gamma: float = 1.4) -> np.ndarray:
    rho = np.asarray(rho, dtype=np.float64)
    u = np.broadcast_to(np.asarray(u, dtype=np.float64), rho.shape)
    v = np.broadcast_to(np.asarray(v, dtype=np.float64), rho.shape)
    p = np.broadcast_to(np.asarray(p, dtype=np.float64), rho.shape)
    e = 0.5 * rho * (u * u + v * v) + p / (gamma - 1.0)          # eq. 10
    return np.ascontiguousarray(np.stack([rho, rho * u, rho * v, e], axis=0))


def conserved_to_primitive(W: np.ndarray, gamma: float = 1.4):
    rho = W[0]
    u = W[1] / rho
    v = W[2] / rho
    p = (gamma - 1.0) * (W[3] - 0.5 * (W[1] * W[1] + W[2] * W[2]) / rho)
    return rho, u, v, p


def _min_image(d: np.ndarray, period: float) -> np.ndarray:
    if period > 0.0:
        return d - period * np.round(d / period)
    return d


def _vortex_profile(r2: np.ndarray, beta: float, gamma: float):
    # eq. 75, 78, 79-80 with p_inf = rho_inf = K = 1 (L875)
    omega = beta * np.exp(0.5 * (1.0 - r2)) / (2.0 * np.pi)
    T = 1.0 - (gamma - 1.0) / gamma * beta * beta / (8.0 * np.pi ** 2) * np.exp(1.0 - r2)
    rho = T ** (1.0 / (gamma - 1.0))
    p = rho ** gamma
    return omega, rho, p


def vortex_state(mesh: UniformMesh, gamma: float = 1.4, beta: float = 5.0, centre=None,
                 advect=(0.0, 0.0)) -> np.ndarray:
    """Isentropic (Yee) vortex, §5.2.1 eq. 74-80; default centre = domain centre,
    periodic min-image distance (reading C18: the paper's domain is [0,10)^2)."""
    Lx, Ly = mesh.lengths
    xc, yc = (0.5 * Lx, 0.5 * Ly) if centre is None else centre
    dx = _min_image(mesh.xy[:, 0] - xc, mesh.period[0])
    dy = _min_image(mesh.xy[:, 1] - yc, mesh.period[1])
    omega, rho, p = _vortex_profile(dx * dx + dy * dy, beta, gamma)
    u = -omega * dy + advect[0]                                   # eq. 74
    v = omega * dx + advect[1]
    return primitive_to_conserved(rho, u, v, p, gamma)


def vortex_exact_density(mesh: UniformMesh, gamma: float = 1.4, beta: float = 5.0, centre=None) -> np.ndarray:
    Lx, Ly = mesh.lengths
    xc, yc = (0.5 * Lx, 0.5 * Ly) if centre is None else centre
    dx = _min_image(mesh.xy[:, 0] - xc, mesh.period[0])
    dy = _min_image(mesh.xy[:, 1] - yc, mesh.period[1])
    return _vortex_profile(dx * dx + dy * dy, beta, gamma)[1]


def sod_state(mesh: UniformMesh, gamma: float = 1.4, x0: float = 0.5) -> np.ndarray:
    """Sod shock tube, §5.1.2: (rho,p) = (1,1) left, (0.125,0.1) right, u = v = 0.
    Vertices exactly at x0 take the left state."""
    left = mesh.xy[:, 0] <= x0
    rho = np.where(left, 1.0, 0.125)
    p = np.where(left, 1.0, 0.1)
    return primitive_to_conserved(rho, 0.0, 0.0, p, gamma)


def kelvin_helmholtz_state(mesh: UniformMesh, gamma: float = 1.4, seed: int = 2017,
                           amplitude: float = 0.01) -> np.ndarray:
    """Sharp Kelvin-Helmholtz shear layer, eq. 90-91 (L987-L996) with U0 = 1/2,
    rho_H = 2, rho_L = 1 (L1037), p0 = 2.5; v_y = amplitude*(2U-1), U ~ U(0,1) drawn once per
    GRID index so that renumbered meshes carry the same physical state."""
    y = mesh.xy[:, 1] / mesh.lengths[1]
    inner = (y > 0.25) & (y <= 0.75)
    rho = np.where(inner, 2.0, 1.0)
    u = np.where(inner, 0.5, -0.5)
    rng = np.random.default_rng(seed)
    noise = rng.random((mesh.shape[1], mesh.shape[0]))
    v = amplitude * (2.0 * noise[mesh.grid_ij[:, 1], mesh.grid_ij[:, 0]] - 1.0)
    return primitive_to_conserved(rho, u, v, 2.5, gamma)


def riemann4_state(mesh: UniformMesh, gamma: float = 1.4, x0: float = 0.5, y0: float = 0.5) -> np.ndarray:
    """Four-quadrant 2D Riemann problem, eq. 85-89 (L948-L959); split point (x0, y0)
    (paper: 0.8; BASELINE.json config 4 / DESIGN.md reading C16: 0.5)."""
    x, y = mesh.xy[:, 0], mesh.xy[:, 1]
    U1 = (0.5322581, 1.2060454, 0.0, 0.3)                     # x <= x0, y > y0   (NW)
    U2 = (1.5, 0.0, 0.0, 1.5)                                 # x >  x0, y > y0   (NE)
    U3 = (0.1379928, 1.2060454, 1.2060454, 0.0290323)         # x <= x0, y <= y0  (SW)
    U4 = (0.5322581, 0.0, 1.2060454, 0.3)                     # x >  x0, y <= y0  (SE)
    west, north = x <= x0, y > y0
    prim = np.empty((4, mesh.nv))
    for k in range(4):
        prim[k] = np.where(north, np.where(west, U1[k], U2[k]), np.where(west, U3[k], U4[k]))
    return primitive_to_conserved(prim[0], prim[1], prim[2], prim[3], gamma)


def uniform_state(mesh: UniformMesh, rho=1.3, u=0.4, v=-0.7, p=2.1, gamma: float = 1.4) -> np.ndarray:
    one = np.ones(mesh.nv)
    return primitive_to_conserved(rho * one, u * one, v * one, p * one, gamma)


def random_smooth_state(mesh: UniformMesh, gamma: float = 1.4, seed: int = 3, mach: float = 0.8,
                        contrast: float = 0.3) -> np.ndarray:
    """Seeded low-wavenumber periodic field with O(1) density/pressure contrast and the given
    typical Mach number: a generic state that exercises every term (used for pins and parity)."""
    rng = np.random.default_rng(seed)
    Lx, Ly = mesh.lengths
    x, y = mesh.xy[:, 0] / Lx, mesh.xy[:, 1] / Ly

    def field():
        f = np.zeros(mesh.nv)
        for _ in range(4):
            kx, ky = rng.integers(1, 4, size=2)
            ph = rng.random(2) * 2.0 * np.pi
            f += rng.normal() * np.sin(2 * np.pi * kx * x + ph[0]) * np.cos(2 * np.pi * ky * y + ph[1])
        return f / 2.0

    rho = 1.0 + contrast * np.tanh(field())
    p = 1.0 + contrast * np.tanh(field())
    c = np.sqrt(gamma * p / rho)
    u = mach * c * np.tanh(field())
    v = mach * c * np.tanh(field())
    return primitive_to_conserved(rho, u, v, p, gamma)


def sound_wave_state(mesh: UniformMesh, gamma: float = 1.4, amplitude: float = 1e-4) -> np.ndarray:
    """Linear right-moving sound wave, PAPER.md 5.1.1 (L766): rho = 1, v = 0, c = 1 background, wavelength = domain
    length in x, amplitude 1e-4.  Eigenvector of the linearised equations: d rho = A s, d u = c A s / rho, d p = c^2 A s."""
    s = np.sin(2.0 * np.pi * mesh.xy[:, 0] / mesh.lengths[0])
    rho = 1.0 + amplitude * s
    u = amplitude * s
    p = 1.0 / gamma + amplitude * s
    return primitive_to_conserved(rho, u, 0.0, p, gamma)


def noh_state(mesh: UniformMesh, gamma: float = 5.0 / 3.0, p0: float = 1e-6) -> np.ndarray:
    """Noh problem, PAPER.md 5.2.2 (L901-L913): rho = 1, unit velocity towards the centre of the domain, p = 1e-6."""
    x = mesh.xy[:, 0] - 0.5 * mesh.lengths[0]
    y = mesh.xy[:, 1] - 0.5 * mesh.lengths[1]
    r = np.sqrt(x * x + y * y)
    safe = np.where(r > 0, r, 1.0)
    u = np.where(r > 0, -x / safe, 0.0)
    v = np.where(r > 0, -y / safe, 0.0)
    return primitive_to_conserved(np.ones(mesh.nv), u, v, p0, gamma)
