"""The five BASELINE.json configurations as synthetic inputs, at full or
reduced size. Returns plain arrays + scalar parameters; no method arithmetic."""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from . import meshes, states

CONFIG_NAMES = ("vortex", "sod", "kh", "riemann4", "sweep")

SCHEME_N, SCHEME_LDA, SCHEME_B = 0, 1, 2


@dataclass
class Config:
    name: str
    mesh: meshes.UniformMesh
    W0: np.ndarray                      # [4][nv] float64 conserved, in the mesh's numbering
    vertex_flag: np.ndarray | None      # uint8 [nv] (1 = frozen) or None
    wall_edge: np.ndarray | None        # int32 [ne][2] or None
    gamma: float = 1.4
    cfl: float = 0.5
    scheme: int = SCHEME_B
    time_order: int = 2
    steps: int | None = None            # run for this many steps ...
    t_end: float | None = None          # ... or to this time
    notes: dict = field(default_factory=dict)

    @property
    def period(self):
        return self.mesh.period


def make_config(name: str, n: int | None = None, numbering: str = "natural", seed: int = 12345) -> Config:
    """name: vortex | sod | kh | riemann4 | sweep.  n: resolution override (cells along x);
    numbering: natural | morton | permuted (seeded)."""
    if name in ("vortex", "sweep"):
        n = n or (32 if name == "vortex" else 256)
        m = meshes.uniform_mesh(n, n, 10.0, 10.0, periodic=True)
        mk_state = lambda mm: states.vortex_state(mm)
        flags, walls = None, None
        run = dict(steps=10 if name == "vortex" else 100)
    elif name == "sod":
        n = n or 1024
        m = meshes.uniform_mesh(n, max(n // 8, 4), 1.0, 0.125 * max(n // 8, 4) / (n / 8.0), periodic=False)
        mk_state = lambda mm: states.sod_state(mm)
        flags = "x"
        walls = True
        run = dict(t_end=0.2)
    elif name == "kh":
        n = n or 1024
        m = meshes.uniform_mesh(n, n, 1.0, 1.0, periodic=True)
        mk_state = lambda mm: states.kelvin_helmholtz_state(mm)
        flags, walls = None, None
        run = dict(steps=200)
        if numbering == "natural":
            numbering = "permuted"          # config 3 is defined on the permuted numbering
    elif name == "riemann4":
        n = n or 2047
        m = meshes.uniform_mesh(n, n, 1.0, 1.0, periodic=False)
        mk_state = lambda mm: states.riemann4_state(mm)
        flags, walls = "xy", None
        run = dict(t_end=0.3)
    else:
        raise ValueError(f"unknown config {name!r}")

    if numbering == "morton":
        m, _, _ = meshes.morton_order_mesh(m)
    elif numbering == "permuted":
        m, _, _ = meshes.permute_mesh(m, seed)
    elif numbering != "natural":
        raise ValueError(numbering)

    W0 = mk_state(m)
    vflag = None
    if flags == "x":
        vflag = meshes.boundary_vertices(m, x_ends=True, y_ends=False)
    elif flags == "xy":
        vflag = meshes.boundary_vertices(m, x_ends=True, y_ends=True)
    wedge = meshes.wall_edges_y(m) if walls else None
    return Config(name=name, mesh=m, W0=W0, vertex_flag=vflag, wall_edge=wedge,
                  notes=dict(n=n, numbering=numbering, seed=seed), **run)
