"""Host logic of bench.py that needs no GPU: the N > 1 path (one process per GPU, max-over-ranks timing, whole-job
rate, rank 0 alone prints) on world_size 2 with the gloo backend, and the reference arm's JSON contract."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, "cpu")          # rank 1 is the slow one
    rate = bench.whole_job_rate(world, 1000, 4, ms * 1e-3)
    dist.barrier()
    out.put((rank, ms, rate))
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_rate_world_size_2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, rate in res:
        assert ms == 15.0                                   # the max, on every rank
        assert rate == pytest.approx(2 * 1000 * 4 / 15e-3)  # all ranks' units / slowest rank's time


def test_single_process_helpers():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, None, "cpu") == 3.5
    assert bench.whole_job_rate(1, 10, 2, 0.5) == 40.0
    assert bench.fp64_peak_nominal(1965.0, "fp64") == pytest.approx(37.2, rel=1e-2)


def test_roofline_figures_come_from_the_committed_capture_of_the_same_configuration():
    """`roofline.traffic` is the committed ncu capture's dram bytes per triangle only when precision, kind of mesh and tile size
    are those of the capture; any other run gets null and a `traffic_source` that says why."""
    from types import SimpleNamespace
    sys.path.insert(0, ROOT)
    import bench
    rows, src = bench.kernel_metrics("fp64", "uniform", 0)             # tile 0 = the default, 256
    assert set(rows) == set(bench.STEP_KERNELS) and "r02_kernel_metrics.csv" in src
    for prec in ("fp64", "fp32"):                                      # the built-in fall-back is the same capture
        r, _ = bench.kernel_metrics(prec, "uniform", 256)
        for k in bench.STEP_KERNELS:
            assert float(r[k]["flops_per_triangle"]) == bench.FLOPS_BUILTIN[prec][k]
    total = sum(float(rows[k]["dram_bytes_per_triangle"]) for k in bench.STEP_KERNELS)
    assert 480 < total < 500                                           # 491.6 B per triangle-update (profiles/r02_kernels_full.md)
    assert bench.kernel_metrics("fp64", "delaunay", 0)[0]["tri_stage1"]["size"] == "1140"
    for prec, mesh, tile in (("fp64", "uniform", 64), ("fp32", "flip", 0)):
        rows, src = bench.kernel_metrics(prec, mesh, tile)
        assert rows == {} and src.startswith("none:")
    a = SimpleNamespace(mesh="delaunay", n=1140, numbering="morton")
    assert "Delaunay" in bench.workload_text(a, 7) and "periodic uniform" not in bench.workload_text(a, 7)
    a.mesh = "uniform"
    assert "periodic uniform triangulation 1140^2" in bench.workload_text(a, 7)


@pytest.mark.slow
def test_reference_arm_prints_one_json_line_under_torchrun():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(29600 + os.getpid() % 300), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--size", "64", "--steps", "1", "--warmup", "3"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                  # rank 0 alone prints; the other rank exits 0 without work
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "triangle_updates_per_s_rk2_step" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"] and d["higher_is_better"] is True


def test_n_gpu_setup_builds_only_the_local_part():
    """bench.py --gpus N: the host side of one rank's set-up (no GPU needed) touches (n + 2) n vertices whatever N is."""
    import bench
    n, world = 256, 8
    sizes = []
    for rank in (0, 3, 7):
        part, W, stats = bench.setup_part(n, world, rank)
        assert part.n_part == world and part.part == rank and part.n_owned == n * n and part.n_local == (n + 2) * n
        assert part.n_tri == 2 * (n + 1) * n and part.n_neighbour == 2 and part.n_send == part.n_recv == 2 * n
        assert sorted(part.neighbour.tolist()) == sorted({(rank - 1) % world, (rank + 1) % world})
        assert W.shape == (4, part.n_local) and np.isfinite(W).all() and W[0].min() > 0.4
        assert stats["n_vertex_global"] == n * n * world and stats["n_triangle_global"] == 2 * n * n * world
        sizes.append(part.n_local)
        # every square carries the same vortex: the owned block of rank r equals that of rank 0
        if rank == 0:
            W_first = W[:, :part.n_owned].copy()
        else:
            assert np.abs(W[:, :part.n_owned] - W_first).max() < 1e-12
    assert len(set(sizes)) == 1
