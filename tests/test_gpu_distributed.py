"""The N > 1 path on the GPU: a `DistributedMesh` over 2, 3 and 4 ranks (separate processes, gloo backend, all
on the one GPU of the box, halo rows staged through host memory) against the CPU oracle on the WHOLE mesh, element
by element, and against the single-mesh run of the same library (they differ by summation order only).
Tolerances as tests/test_gpu_parity.py."""
import os
import subprocess
import sys

import numpy as np
import pytest

import oracle
from dist_worker import cases, nonphysical_case
from helpers import field_errors

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(world, tmp_path):
    out = str(tmp_path / f"dist_{world}.npz")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world), "--master-addr", "127.0.0.1",
           "--master-port", str(29700 + os.getpid() % 200 + world), os.path.join(ROOT, "tests", "dist_worker.py"), "--out", out]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=1500, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-3000:]
    return np.load(out)


@pytest.fixture(scope="module")
def single():
    """The same cases on one mesh: oracle and single-GPU library results."""
    import torch
    import paper_1705_02028_b200 as mrd
    ref = {}
    for name, (mesh, W0, flag, wall, params, steps, t_end) in cases().items():
        fp32 = params.get("precision", 0) == 1
        gm = mrd.Mesh(mesh.xy, mesh.tri, vertex_flag=flag, wall_edge=wall, period=mesh.period, **params)
        gm.set_state(torch.tensor(np.ascontiguousarray(W0), dtype=torch.float32 if fp32 else torch.float64, device="cuda"))
        g1 = gm.step(1)
        G1 = gm.get_state().cpu().numpy()
        g = gm.step(steps - 1, t_end)
        G = gm.get_state().cpu().numpy()
        gtot = gm.diagnostics()
        om = oracle.OracleMesh(mesh.xy, mesh.tri, period=mesh.period, vertex_flag=flag, wall_edge=wall,
                               scheme=params["scheme"], time_order=params["time_order"])
        om.set_state(W0)
        o1 = om.step(1)
        O1 = om.get_state().copy()
        o = om.step(steps - 1, t_end)
        O = om.get_state().copy()
        ref[name] = dict(g1=g1, G1=G1, g=g, G=G, gtot=gtot, o1=o1, O1=O1, o=o, O=O, fp32=fp32, nv=mesh.nv)
    return ref


@pytest.mark.parametrize("world", [1, 2, 3, 4])
def test_distributed_mesh_matches_oracle_and_single_mesh(world, single, tmp_path):
    res = _run(world, tmp_path)
    for name, ref in single.items():
        W1, W, sc, tot = res[name + "/W1"], res[name + "/W"], res[name + "/scalars"], res[name + "/totals"]
        n1, t1, dt1, n, t, dt, mr, mp, n_owned, n_recv, launches = sc
        tol1, toln = (1e-5, 1e-5) if ref["fp32"] else (1e-12, 1e-9)
        # the oracle on the whole mesh
        assert n1 == 1 and n == ref["o"][0], name
        assert abs(dt1 - ref["o1"][2]) <= (1e-6 if ref["fp32"] else 1e-14) * ref["o1"][2], name
        assert field_errors(W1, ref["O1"]) <= tol1, name
        assert field_errors(W, ref["O"]) <= toln, name
        assert abs(t - ref["o"][1]) <= (1e-5 if ref["fp32"] else 1e-11) * max(1.0, abs(t)), name
        # the single-mesh run of the library: same step count, time step and state up to summation order
        assert n == ref["g"][0] and abs(dt - ref["g"][2]) <= (1e-5 if ref["fp32"] else 1e-12) * dt, name
        assert field_errors(W1, ref["G1"]) <= (1e-6 if ref["fp32"] else 1e-13), name
        gt, gmr, gmp = ref["gtot"]
        scale = np.abs(gt).max()
        assert np.abs(tot - gt).max() <= (1e-5 if ref["fp32"] else 1e-11) * scale, name   # halo vertices are not double counted
        assert abs(mr - gmr) <= 1e-5 * abs(gmr) and abs(mp - gmp) <= 1e-4 * abs(gmp), name
        # the work really was split and exchanged, and ran in this library's kernels
        assert launches > 0 and ((0 < n_owned < ref["nv"] and n_recv > 0) if world > 1 else (n_owned == ref["nv"] and n_recv == 0)), name


@pytest.mark.parametrize("world", [2, 3])
def test_a_step_that_fails_on_one_part_is_discarded_by_all(world, tmp_path):
    import torch
    import paper_1705_02028_b200 as mrd
    mesh, W0, steps = nonphysical_case()
    gm = mrd.Mesh(mesh.xy, mesh.tri, period=mesh.period)
    gm.set_state(torch.tensor(W0, device="cuda"))
    with pytest.raises(mrd.MrdError) as e:
        gm.step(steps)
    assert e.value.code == mrd.MRD_ENONPHYSICAL
    n_ref, t_ref, _ = gm.sync()
    assert n_ref == 1                                              # one good step, the second one is discarded
    Wref = gm.get_state().cpu().numpy()
    res = _run(world, tmp_path)
    ranks = res["nonphysical/ranks"]
    assert ranks.shape == (world, 3)
    assert np.all(ranks[:, 0] == mrd.MRD_ENONPHYSICAL)             # every rank raised the same error ...
    assert np.all(ranks[:, 1] == n_ref) and np.all(np.abs(ranks[:, 2] - t_ref) <= 1e-14)   # ... at the same step and time
    assert field_errors(res["nonphysical/W"], Wref) <= 1e-13       # and holds the last good state


def test_bench_n2_runs_one_mesh_over_two_ranks():
    """bench.py --gpus 2 as the driver launches it, except for the backend (two ranks on the one GPU need gloo)."""
    import json
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(29950 + os.getpid() % 40), os.path.join(ROOT, "bench.py"), "--gpus", "2", "--size", "256", "--steps", "4",
           "--warmup", "3", "--backend", "gloo"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["scaling"] == "weak" and d["value"] > 0 and d["gpu_launches"] > 0
    assert d["config"]["n_triangles"] == 2 * 2 * 256 * 256 and "one mesh over 2 GPUs" in d["config"]["parallelism"]
    assert d["config"]["n_triangles_rank0"] > 2 * 256 * 256          # its square plus the cut triangles of both cut lines
    assert d["e2e"]["h2d_bytes_per_step"] > 0 and d["roofline"]["kernel"].startswith("tri_stage")


def test_bench_line_carries_every_key_of_the_contract():
    """python bench.py (N = 1) at a small size: one JSON line with the contract's keys, the roofline and the CPU baseline."""
    import json
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--size", "256", "--steps", "4", "--warmup", "3"],
                       capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
                "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert key in d, key
    assert d["metric"] == "triangle_updates_per_s_rk2_step" and d["n_gpus"] == 1 and d["steps"] == 4 and d["warmup"] == 3
    assert d["dtype"] == "f64" and d["data"] == "synthetic" and d["higher_is_better"] is True and d["vs_baseline"] is None
    assert "workload" in d["config"] and d["value"] == pytest.approx(d["config"]["n_triangles"] * 1e3 / d["ms_per_step"], rel=1e-6)
    assert d["gpu_launches"] >= 4 * 4                                   # four kernels per RK2 step
    for key in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"):
        assert key in d["e2e"], key
    assert d["e2e"]["h2d_bytes_per_step"] == 4 * 256 * 256 * 8 and 0 < d["e2e"]["value"] < d["value"]
    for key in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert key in d["roofline"], key
    assert d["roofline"]["bound"] in ("alu", "hbm") and d["roofline"]["frac"] == pytest.approx(d["roofline"]["achieved"] / d["roofline"]["peak"])
    for key in ("sm_mhz", "sm_max_mhz", "reasons"):
        assert key in d["clocks"], key
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["unit"] == d["unit"] and c["sample"]


def test_bench_on_a_mesh_generated_by_the_library():
    """python bench.py --mesh refined: the paper's pipeline (generate the mesh on the GPU, then solve on it) at a small size."""
    import json
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--mesh", "refined", "--size", "160", "--steps", "4", "--warmup", "3",
                        "--no-cpu-baseline"], capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-3000:]
    d = json.loads([l for l in r.stdout.splitlines() if l.startswith("{")][-1])
    gen = d["config"]["mesh_generation"]
    assert gen["iterations"] >= 5 and 0.7 * 160 * 160 < gen["n_vertices"] == d["config"]["n_vertices"] < 1.4 * 160 * 160
    assert 1.9 < d["config"]["n_triangles"] / d["config"]["n_vertices"] < 2.0 and d["value"] > 0
    assert "GENERATED on the GPU" in d["config"]["workload"] and d["roofline"]["traffic"] is None


def test_measurement_modules_run_at_a_small_size():
    """python -m paper_1705_02028_b200.sweep and .meshgen_bench (the commands behind BASELINE.md section 6 and profiles/r02_meshgen.md)."""
    import json
    r = subprocess.run([sys.executable, "-m", "paper_1705_02028_b200.sweep", "--sizes", "64", "--steps", "5", "--reps", "2"],
                       capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    rows = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(rows) == 6 and all(row["ms_per_step"] > 0 and row["triangles"] == 2 * 64 * 64 for row in rows)
    r = subprocess.run([sys.executable, "-m", "paper_1705_02028_b200.meshgen_bench", "--cells", "60", "--reps", "1"],
                       capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    rows = {row["kernel"]: row for row in (json.loads(l) for l in r.stdout.splitlines() if l.startswith("{"))}
    assert set(rows) == {"build_edges", "delaunay_flip", "check_only", "test_quality", "find_triangle", "refine", "refine_morton"}
    assert rows["delaunay_flip"]["flips"] > 1000 and rows["refine"]["bad_left"] == 0 and rows["refine_morton"]["bad_left"] == 0
    assert rows["find_triangle"]["found"] == rows["find_triangle"]["units"]
