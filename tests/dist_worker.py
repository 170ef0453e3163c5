"""Worker of tests/test_gpu_distributed.py: one rank of a `DistributedMesh` run, launched by torch.distributed.run
with the gloo backend.  All ranks share cuda:0 (the box has one GPU; the halo rows are staged through host memory,
no kernel waits on another rank's kernel).  Rank 0 writes the gathered results to --out (npz)."""
import argparse
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402


def cases():
    """name -> (mesh, W0, vertex_flag, wall_edge, params, steps, t_end); the test rebuilds the same inputs."""
    out = {}
    m = wl.uniform_mesh(48, 48, 10.0, 10.0, periodic=True)
    out["vortex_b2"] = (m, wl.vortex_state(m), None, None, dict(scheme=2, time_order=2), 20, 0.0)
    out["vortex_b2_fp32"] = (m, wl.vortex_state(m), None, None, dict(scheme=2, time_order=2, precision=1), 10, 0.0)
    out["vortex_b2_unfused"] = (m, wl.vortex_state(m), None, None, dict(scheme=2, time_order=2, tile=-1), 5, 0.0)
    c = wl.make_config("sod", n=64)
    out["sod_walls_tend"] = (c.mesh, c.W0, c.vertex_flag, c.wall_edge, dict(scheme=2, time_order=2), 200, 0.02)
    k = wl.make_config("kh", n=40, numbering="permuted")
    out["kh_permuted_n1"] = (k.mesh, k.W0, None, None, dict(scheme=0, time_order=1), 8, 0.0)
    j = wl.jitter_mesh(wl.uniform_mesh(33, 27, 1.0, 1.0, periodic=True), 0.2, seed=11)
    out["jitter_lda2"] = (j, wl.random_smooth_state(j, mach=0.5, seed=4), None, None,
                          dict(scheme=1, time_order=2, reorder=False, tile=64), 10, 0.0)
    f = wl.flip_edges(wl.jitter_mesh(wl.uniform_mesh(40, 36, 2.0, 1.8, periodic=True), 0.2, seed=3), seed=11)
    out["variable_valence_b2"] = (f, wl.random_smooth_state(f, mach=0.8, seed=6), None, None, dict(scheme=2, time_order=2), 10, 0.0)
    out["variable_valence_bx"] = (f, wl.random_smooth_state(f, mach=1.1, seed=6), None, None, dict(scheme=5, time_order=2), 10, 0.0)
    out["vortex_bx_n1"] = (m, wl.vortex_state(m, advect=(0.3, 0.1)), None, None, dict(scheme=5, time_order=1), 6, 0.0)
    r = wl.make_config("riemann4", n=40)
    out["riemann4_frozen"] = (r.mesh, r.W0, r.vertex_flag, None, dict(scheme=2, time_order=2), 6, 0.0)
    # Bx on a BOUNDED domain: L of eq. 56 must be the whole tube's length on every part, not the part's bounding box
    out["sod_bx_walls"] = (c.mesh, c.W0, c.vertex_flag, c.wall_edge, dict(scheme=5, time_order=2), 8, 0.0)
    return out


def nonphysical_case():
    """A state that stays physical for one step and turns non-physical in STAGE 2 of the second one, at an interior vertex
    of the first Morton range only (a Mach-3 momentum spike at one vertex of a gas at rest): (mesh, W0, steps asked for)."""
    m = wl.uniform_mesh(32, 32, 1.0, 1.0, periodic=True)
    rho, u, v, p = np.ones(m.nv), np.zeros(m.nv), np.zeros(m.nv), np.ones(m.nv)
    i0 = 5 * 32 + 6
    u[i0], p[i0] = 4.0, 0.2
    return m, wl.primitive_to_conserved(rho, u, v, p), 5


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", required=True)
    args = ap.parse_args()
    import torch
    import torch.distributed as dist
    from paper_1705_02028_b200.distributed import DistributedMesh
    torch.cuda.set_device(0)
    dist.init_process_group("gloo")
    rank = dist.get_rank()
    res = {}
    for name, (mesh, W0, flag, wall, params, steps, t_end) in cases().items():
        dm = DistributedMesh(mesh.xy, mesh.tri, vertex_flag=flag, wall_edge=wall, period=mesh.period, **params)
        dm.set_state(W0)
        n1, t1, dt1 = dm.step(1)
        W1 = dm.get_state()
        n, t, dt = dm.step(steps - 1, t_end)
        W = dm.get_state()
        tot, mr, mp = dm.diagnostics()
        res[name + "/W1"] = W1
        res[name + "/W"] = W
        res[name + "/scalars"] = np.array([n1, t1, dt1, n, t, dt, mr, mp, dm.part.n_owned, dm.part.n_recv, dm.launch_count()], dtype=np.float64)
        res[name + "/totals"] = tot
        dm.close()
    # a step that fails on ONE part must be discarded by ALL of them: same (error, steps, t) everywhere, state still usable
    from paper_1705_02028_b200 import MrdError
    mesh, W0, steps = nonphysical_case()
    dm = DistributedMesh(mesh.xy, mesh.tri, period=mesh.period, scheme=2, time_order=2)
    dm.set_state(W0)
    code = 0
    try:
        dm.step(steps)
    except MrdError as e:
        code = e.code
    n_tot, t_tot, _ = dm.mesh.sync()
    mine = [float(code), float(n_tot), float(t_tot)]
    everyone = [None] * dist.get_world_size()
    dist.all_gather_object(everyone, mine)
    res["nonphysical/ranks"] = np.array(everyone, dtype=np.float64)
    res["nonphysical/W"] = dm.get_state()                       # collective: hangs if the ranks disagree about the step
    n_more = dm.step(1) if code == 0 else None                  # (not reached in the failing case)
    dm.close()
    dist.barrier()
    if rank == 0:
        np.savez(args.out, **res)
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
