"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no residuals, no K matrices, no time
stepping): it only builds meshes (vertex coordinates + triangle connectivity + boundary
lists) and initial conserved states W = (rho, rho*u, rho*v, e) as plain numpy arrays.
Both `oracle/` and `paper_1705_02028_b200/` consume the same arrays; neither is imported here.

Recipes follow SURVEY.md §8(d) / DESIGN.md "Input recipe"; paper citations are PAPER.md lines.
"""
from .meshes import (  # noqa: F401
    uniform_mesh,
    permute_mesh,
    morton_order_mesh,
    jitter_mesh,
    flip_edges,
    scrambled_triangulation,
    delaunay_mesh,
    uniform_strip_part,
    read_triangle_files,
    write_triangle_files,
    boundary_vertices,
    wall_edges_y,
    UniformMesh,
)
from .states import (  # noqa: F401
    primitive_to_conserved,
    conserved_to_primitive,
    vortex_state,
    vortex_exact_density,
    sod_state,
    kelvin_helmholtz_state,
    riemann4_state,
    uniform_state,
    random_smooth_state,
    sound_wave_state,
    noh_state,
)
from .configs import make_config, CONFIG_NAMES  # noqa: F401
