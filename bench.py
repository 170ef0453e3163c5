#!/usr/bin/env python
"""bench.py -- triangle-updates/s of the residual-distribution sweep (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl mrd|reference] [--size 4096]
                    [--precision fp64|fp32] [--numbering morton|natural|permuted] [--reorder 0|1]

A "step" is one RK2 time step of scheme B (both stages, dt reduction included) over the whole mesh:
config 5 of BASELINE.json at its largest size (isentropic vortex on a periodic uniform triangulation of
4096^2 vertices, 33.5M triangles, Morton-ordered input).  Prints ONE JSON line (rank 0).
N > 1 (launched by torchrun, one process per GPU): ONE mesh -- N copies of that workload stacked in y -- spread over
the N GPUs by the domain decomposition of DESIGN.md section 9 (halo exchange per stage + one min-reduction per step over
NCCL); `--decomposition replicas` runs N independent replicas instead.
`--impl reference` times the CPU oracle (oracle/), as it stands, on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "triangle_updates_per_s_rk2_step"
UNIT = "triangle-updates/s"

# ---- per-unit algorithmic figures --------------------------------
# FLOPs per triangle and launch = min(oracle operation count, FLOPs the kernel executes).  The kernel's count
# (2*FMA + ADD + MUL thread instructions, predicated on, of the profiled launch) is the smaller one; it comes, with the
# measured dram bytes per triangle, from the committed capture profiles/r02_kernel_metrics.csv (+ .md: the command).
# The built-in figures below are that file's fp64 / fp32 rows for the uniform mesh and tiles of 256 triangles: they
# serve when no row of the file matches the run (then `flops_source` says so and `traffic` is null).
METRICS_CSV = os.path.join(ROOT, "profiles", "r02_kernel_metrics.csv")
FLOPS_BUILTIN = {"fp64": {"tri_stage1": 635.2, "gather_dt": 11.0, "update": 71.4, "tri_stage2": 718.1, "gather_update": 63.4},
                 "fp32": {"tri_stage1": 598.2, "gather_dt": 9.6, "update": 38.4, "tri_stage2": 684.2, "gather_update": 31.9}}
STEP_KERNELS = ("tri_stage1", "gather_dt", "update", "tri_stage2", "gather_update")
ORACLE_FLOPS_TRI = (2098.0, 2194.0)    # oracle.count_ops(stage 1 / stage 2): add+mul+div+sqrt
# compulsory HBM bytes per triangle of one launch (shares of SURVEY 8d's 130 B per triangle-update):
# tile kernels: state read once (32 B per vertex / 2), connectivity 12 B, coordinates 8 B; stage 2 also reads dW/dt;
# vertex kernels (what is left of the 130 B): one state written per stage (32 B per vertex / 2) and V_i read (8 B / 2)
BYTES_ALG = {"fp64": {"tri_stage1": 36.0, "tri_stage2": 52.0, "gather_dt": 2.0, "update": 20.0, "gather_update": 20.0},
             "fp32": {"tri_stage1": 24.0, "tri_stage2": 32.0, "gather_dt": 1.0, "update": 9.5, "gather_update": 9.5}}
# bytes the fused kernels move BY DESIGN per triangle (slot copies, stored stage-1 cells, partials),
# for comparison with ncu's dram__bytes (the roofline object's `traffic`)
DESIGN_BYTES_TRI = {"tri_stage1": {"fp64": 144.0, "fp32": 72.0}, "tri_stage2": {"fp64": 155.0, "fp32": 77.0}}
B_ALG_STEP = {"fp64": 130.0, "fp32": 76.0}


def kernel_metrics(precision: str, mesh: str, tile: int):
    """Rows of the committed ncu capture that describe THIS run: same precision, same kind of mesh (the geometry-table
    kernels of the uniform mesh and the coordinate kernels of every other mesh are different instantiations) and same tile
    size.  Returns ({kernel: row}, source text) -- ({}, reason) when nothing matches."""
    import csv
    tile = 256 if tile == 0 else tile
    try:
        with open(METRICS_CSV) as f:
            rows = [r for r in csv.DictReader(f)]
    except OSError:
        return {}, "none: profiles/r02_kernel_metrics.csv not found"
    hit = {r["kernel"]: r for r in rows if r["precision"] == precision and r["mesh"] == mesh and int(r["tile"]) == tile}
    if not hit:
        return {}, f"none: no ncu capture of precision {precision}, mesh '{mesh}', tile {tile} in profiles/r02_kernel_metrics.csv"
    size = next(iter(hit.values()))["size"]
    return hit, f"profiles/r02_kernel_metrics.csv ({precision}, mesh '{mesh}' --size {size}, tile {tile}): ncu dram bytes per triangle x triangles of this run"


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """SM clock and throttle reasons sampled DURING the timed region (B200_PROFILING.md), through NVML
    (nvidia_ml_py; the same counters nvidia-smi prints) every 5 ms from a background thread, started before the warm-up steps."""
    REASONS = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}

    def __init__(self, index: int):
        self.index, self.sm, self.mask, self.max_mhz, self.power = index, [], 0, None, []
        self._stop = threading.Event()
        self._thread = None

    def __enter__(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            visible = os.environ.get("CUDA_VISIBLE_DEVICES")
            idx = self.index
            if visible:
                try:
                    idx = int(visible.split(",")[self.index])
                except Exception:
                    pass
            self._nvml = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        except Exception:
            self._thread = None
        return self

    def _run(self):
        n = self._nvml
        while not self._stop.is_set():
            try:
                self.sm.append(float(n.nvmlDeviceGetClockInfo(self._h, n.NVML_CLOCK_SM)))
                self.mask |= int(n.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                self.power.append(n.nvmlDeviceGetPowerUsage(self._h) / 1000.0)
            except Exception:
                pass
            self._stop.wait(0.005)

    def __exit__(self, *a):
        self._stop.set()
        if self._thread:
            self._thread.join(timeout=2)

    def summary(self):
        if not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(self.sm)), "sm_min_mhz": float(min(self.sm)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(k for k, bit in self.REASONS.items() if self.mask & bit), "samples": len(self.sm),
                "power_w_max": max(self.power) if self.power else None}


def max_over_ranks(value: float, dist, device) -> float:
    """Multi-rank timings are the MAX over ranks (one process per GPU); identity for a single process."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([value], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(world: int, units_per_rank: int, steps: int, seconds: float) -> float:
    """Weak scaling: value = the units all ranks processed / the max-over-ranks time."""
    return world * units_per_rank * steps / seconds


def build_workload(n: int, numbering: str, kind: str = "uniform"):
    """config 5; kind 'jitter' moves every vertex by up to 0.2 cell widths (no two triangles alike), 'flip' also flips a seeded
    third of the edges (valence 4...10): the second, genuinely unstructured workload of SURVEY 8f-2."""
    import workloads as wl
    if kind == "delaunay":
        # the paper's unstructured mesh shape (L685: 1.3 M vertices): seeded Delaunay triangulation, graded 100:1, frozen ring
        cfg = wl.make_config("sweep", n=32, numbering="natural")
        cfg.mesh = wl.delaunay_mesh(n * n, seed=1)
        cfg.vertex_flag = cfg.mesh.boundary
        cfg.W0 = wl.vortex_state(cfg.mesh)
        return cfg
    if kind == "refined":
        # the paper's own pipeline (section 4): the mesh is GENERATED on the GPU by the library's Delaunay refinement (about n^2
        # vertices in [0, 10]^2, B = sqrt 2, vertices along the Morton curve), its boundary vertices frozen, then solved on
        import torch
        from paper_1705_02028_b200 import binding as b
        from workloads.meshes import UniformMesh
        cfg = wl.make_config("sweep", n=32, numbering="natural")
        c = wl.scrambled_triangulation(40, 40, seed=2, Lx=10.0, Ly=10.0)
        xy = torch.tensor(c.xy, dtype=torch.float64, device="cuda")
        tv = torch.tensor(c.tri, dtype=torch.int32, device="cuda")
        te, et = b.meshgen_build_edges(tv)
        b.meshgen_delaunay_flip(xy, tv, te, et)
        t0 = time.perf_counter()
        xy, tv, te, et, info = b.meshgen_refine(xy, tv, te, et, float(np.sqrt(0.69 * 100.0 / (n * n))), float(np.sqrt(2.0)), seed=1,
                                                cap_vertex=int(1.6 * n * n) + 4096, box=(0.0, 0.0, 10.0, 10.0))
        torch.cuda.synchronize()
        gen_s = time.perf_counter() - t0
        assert info["bad_left"] == 0
        X, T, TE, ET = xy.cpu().numpy(), tv.cpu().numpy(), te.cpu().numpy(), et.cpu().numpy()
        seg = np.nonzero(ET[:, 1] < 0)[0]
        k = (TE[ET[seg, 0]] == seg[:, None]).argmax(axis=1)
        flag = np.zeros(X.shape[0], dtype=np.uint8)
        flag[T[ET[seg, 0], (k + 1) % 3]] = 1
        flag[T[ET[seg, 0], (k + 2) % 3]] = 1
        cfg.mesh = UniformMesh(X, T, (0.0, 0.0), None, None, None, (10.0, 10.0))
        cfg.vertex_flag = flag
        cfg.W0 = wl.vortex_state(cfg.mesh)
        cfg.generated = dict(seconds=gen_s, iterations=info["iterations"], n_vertices=int(X.shape[0]))
        return cfg
    cfg = wl.make_config("sweep", n=n, numbering=numbering)
    if kind in ("jitter", "flip"):
        cfg.mesh = wl.jitter_mesh(cfg.mesh, 0.2, seed=7)
    if kind == "flip":
        cfg.mesh = wl.flip_edges(cfg.mesh, seed=11)
    if kind != "uniform":
        cfg.W0 = wl.vortex_state(cfg.mesh)     # the same vortex, sampled at the moved vertices
    return cfg


def workload_text(args, nt: int) -> str:
    """config.workload of the single-GPU line: what was actually built (build_workload)."""
    tail = f"{nt} triangles, scheme B, RK2, CFL 0.5"
    if args.mesh == "delaunay":
        return (f"isentropic vortex on a seeded graded Delaunay triangulation ({args.n}^2 points, cell size 100:1, frozen boundary ring; the "
                f"shape of the paper's unstructured mesh, PAPER.md L685), Morton-ordered by the layout stage, {tail}")
    if args.mesh == "refined":
        return (f"isentropic vortex on a mesh GENERATED on the GPU by the library's Delaunay refinement (section 2.4 / 4.1 of the paper: about "
                f"{args.n}^2 vertices in [0, 10]^2, B = sqrt 2, Morton-ordered, frozen boundary; the paper's test mesh has 1.3 M vertices, "
                f"L685), {tail}")
    head = f"BASELINE.json config 5: isentropic vortex, periodic uniform triangulation {args.n}^2 vertices"
    if args.mesh == "jitter":
        head += ", every vertex moved by up to 0.2 cell widths (seed 7: no two triangles alike)"
    if args.mesh == "flip":
        head += ", every vertex moved by up to 0.2 cell widths and a seeded third of the edges flipped (variable valence)"
    return f"{head}, {args.numbering} input numbering, {tail}"


def setup_part(n: int, world: int, rank: int):
    """Host-side set-up of ONE rank of the N-GPU run, from local pieces only (needs no GPU): the part of the periodic strip of
    `world` vortex squares (workloads.uniform_strip_part -> mrd_partition_create_local) and its initial state.
    Returns (Partition, W_local [4][n_local] in the part's vertex order, stats)."""
    import resource
    from types import SimpleNamespace
    import workloads as wl
    import paper_1705_02028_b200 as mrd
    t0 = time.perf_counter()
    pc = wl.uniform_strip_part(n, world, rank)
    part = mrd.Partition.from_local(pc["n_vertex_global"], pc["vertex_global"], pc["owner"], pc["xy"], pc["tri"], pc["tri_global"],
                                    world, rank, period=pc["period"], domain_size=pc["domain_size"])
    L = pc["period"][0]
    # the vortex of every square: the state at (x, y mod L) of the single-square workload
    sq = SimpleNamespace(xy=np.stack([part.xy[:, 0], np.mod(part.xy[:, 1], L)], axis=1), lengths=(L, L), period=(L, L),
                         nv=part.n_local)
    W_local = wl.vortex_state(sq)
    stats = dict(n_vertex_global=pc["n_vertex_global"], n_triangle_global=pc["n_triangle_global"],
                 setup_s=time.perf_counter() - t0, host_rss_gb=resource.getrusage(resource.RUSAGE_SELF).ru_maxrss / 1e6)
    return part, W_local, stats


# ------------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle, as it stands, on the host cores, on a bounded sample
# ------------------------------------------------------------------------------------------------------
def oracle_rate(n_sample: int, steps: int, warmup: int, numbering: str):
    import oracle
    cfg = build_workload(n_sample, numbering)
    cores = os.cpu_count() or 1
    om = oracle.OracleMesh(cfg.mesh.xy, cfg.mesh.tri, period=cfg.mesh.period, gamma=cfg.gamma, cfl=cfg.cfl,
                           scheme=cfg.scheme, time_order=cfg.time_order, threads=cores)
    om.set_state(cfg.W0)
    if warmup:
        om.step(warmup)
    t0 = time.perf_counter()
    om.step(steps)
    dt = time.perf_counter() - t0
    return cfg.mesh.nt * steps / dt, dt / steps, cores, cfg.mesh.nt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    n_s = min(args.n, 1024)
    steps = max(1, min(args.steps, 3))
    rate, spstep, cores, nt = oracle_rate(n_s, steps, min(args.warmup, 1), args.numbering)
    sample = (f"isentropic vortex, periodic {n_s}^2 vertices ({nt} triangles = 1/{(args.n // n_s) ** 2} of the "
              f"{args.n}^2 workload), {steps} RK2 steps of scheme B, OpenMP triangle loops on {cores} threads")
    line = {"impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": min(args.warmup, 1), "ms_per_step": spstep * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"sweep vortex {args.n}^2 periodic, {args.numbering} numbering, B2 (oracle sample)"},
            "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------------
# the CUDA arm
# ------------------------------------------------------------------------------------------------------
def fp64_peak_nominal(sm_max_mhz: float, precision: str) -> float:
    """Plain-ALU peak in TFLOP/s: 148 SMs x 4 sub-partitions x 16 DFMA lanes (fp64)
    or 32 FFMA lanes (fp32) x 2 flops x the maximum SM clock."""
    lanes = 64 if precision == "fp64" else 128
    return 148 * lanes * 2 * sm_max_mhz * 1e6 * 1e-12


def run_mrd(args):
    import torch
    import paper_1705_02028_b200 as mrd

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the mrd path has no CPU fallback")
    local %= torch.cuda.device_count()    # (more ranks than GPUs only happens with --backend gloo, a functional test)
    torch.cuda.set_device(local)
    dist = None
    rdev = "cuda"                          # where the max-over-ranks reduction lives
    if world > 1:
        import torch.distributed as dist
        if args.backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group("gloo")
            rdev = "cpu"

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    prec = args.precision
    tile_eff = 256 if args.tile == 0 else args.tile      # 0 = the library's default
    tdtype = torch.float64 if prec == "fp64" else torch.float32
    halo = world > 1 and args.decomposition == "halo"
    params = dict(gamma=1.4, cfl=0.5, scheme=mrd.SCHEME_B, time_order=2, precision=mrd.FP64 if prec == "fp64" else mrd.FP32,
                  reorder=bool(args.reorder), tile=args.tile)
    t0 = time.perf_counter()
    setup = None
    if not halo:
        # one GPU, or N independent replicas of the single-GPU workload
        cfg = build_workload(args.n, args.numbering, args.mesh)
        mesh = cfg.mesh
        nt, nv = mesh.nt, mesh.nv                 # units per rank
        nt_job, nv_job = world * nt, world * nv
        t0 = time.perf_counter()                  # layout_s: the library's one-off stage alone (mrd_mesh_create, upload included)
        gm = sim = mrd.Mesh(mesh.xy, mesh.tri, vertex_flag=cfg.vertex_flag, period=mesh.period, **params)
        layout_s = time.perf_counter() - t0
        gm.set_state(torch.tensor(cfg.W0, dtype=tdtype, device="cuda"))
        parallelism = "1 GPU" if world == 1 else f"{world} independent replicas"
    else:
        # ONE mesh over N GPUs (weak scaling): a periodic strip of N copies of the single-GPU workload stacked in y, cut into
        # its N squares; one halo exchange per stage and two scalar reductions per step over NCCL.  Every rank builds ITS part
        # only (setup_part): no array of the whole mesh exists anywhere, so start-up time and host memory do not grow with N.
        from paper_1705_02028_b200.distributed import DistributedMesh
        part, W_local, setup = setup_part(args.n, world, rank)
        sim = DistributedMesh(None, None, part=part, period=part.period, **params)
        gm = sim.mesh                             # this rank's part (owned + halo vertices, cut triangles on both sides)
        nt_job, nv_job = setup["n_triangle_global"], setup["n_vertex_global"]   # unique triangles / vertices of the whole mesh
        nt, nv = gm.nt, gm.nv                     # this rank's share (kernel-level numbers)
        layout_s = time.perf_counter() - t0
        sim.set_state_local(W_local)
        parallelism = (f"one mesh over {world} GPUs: row-band domain decomposition built locally per rank, {sim.part.n_send} halo vertices "
                       f"sent per rank per stage to {sim.part.n_neighbour} neighbours, 2 scalar all-reduces per step")
        del W_local
    stream = torch.cuda.current_stream()

    # ---- device-resident throughput: W warm-up steps, then exactly K timed steps -------------------------
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clk:
        sim.step(args.warmup)
        barrier()
        l0 = sim.launch_count()
        e0.record(stream)
        sim.step_async(args.steps)
        e1.record(stream)
        torch.cuda.synchronize()
        barrier()
    n_done, t_sim, _ = sim.sync()
    launches = sim.launch_count() - l0
    ms_total = max_over_ranks(e0.elapsed_time(e1), dist, rdev)
    assert n_done == (args.steps if halo else args.warmup + args.steps), (n_done, args.warmup, args.steps)
    ms_step = ms_total / args.steps
    value = whole_job_rate(1, nt_job, args.steps, ms_total * 1e-3)

    _, mr, mp = sim.diagnostics()
    assert mr > 0 and mp > 0

    # ---- end to end through the host-buffer C-ABI calls: H2D of the state, one step, D2H of the result ----
    # (N > 1, one mesh: every rank moves its own part, halo copies included, and the step runs with its exchanges)
    ke = max(1, min(args.steps, args.e2e_steps))
    h_in = torch.empty((4, nv), dtype=tdtype).pin_memory()
    h_out = torch.empty((4, nv), dtype=tdtype).pin_memory()
    h_in.copy_(gm.get_state().cpu())
    gm.set_state_host(h_in.numpy()); sim.step(1); gm.get_state_host(h_out.numpy())      # warm-up
    barrier()
    t0 = time.perf_counter()
    for _ in range(ke):
        gm.set_state_host(h_in.numpy())
        sim.step(1)
        gm.get_state_host(h_out.numpy())
        h_in, h_out = h_out, h_in
    torch.cuda.synchronize()
    e2e_s = max_over_ranks(time.perf_counter() - t0, dist, rdev)
    state_bytes = 4 * nv * (8 if prec == "fp64" else 4)
    e2e = {"value": whole_job_rate(1, nt_job, ke, e2e_s), "unit": UNIT, "h2d_bytes_per_step": state_bytes,
           "d2h_bytes_per_step": state_bytes, "steps": ke, "ms_per_step": e2e_s / ke * 1e3,
           "api": "mrd_set_state_host + mrd_step(1) + mrd_get_state_host, pinned host buffers"
                  + (" (bytes per rank; the step is the phase sequence with its halo exchanges)" if halo else "")}

    # ---- live per-kernel durations (CUDA events on the launching stream), averaged over 5 steps ------------
    # (last: on a partitioned mesh these local steps run without exchanges, which is all a kernel timing needs)
    prof = {}
    nprof = 5
    for _ in range(nprof):
        for k, v in gm.step_profile().items():
            prof[k] = prof.get(k, 0.0) + v / nprof

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel -------------------------------------------------------------------
    hbm_gbs, hbm_src = measured_peaks()
    clocks = clk.summary()
    sm_max = clocks["sm_max_mhz"] or 1965.0
    main = {k: v for k, v in prof.items() if k in STEP_KERNELS}
    dom = max(main, key=main.get)
    dom_ms = main[dom]
    ncu, ncu_src = kernel_metrics(prec, args.mesh, args.tile)
    if not args.reorder and args.numbering != "morton":
        ncu, ncu_src = {}, "none: the ncu captures are of Morton-ordered layouts (--reorder 0 on a non-Morton numbering moves other bytes)"
    if ncu:
        flops = {k: float(ncu[k]["flops_per_triangle"]) for k in STEP_KERNELS}
        flops_src = ncu_src.split(":")[0] + ": executed 2*FMA + MUL + ADD per triangle"
    else:
        flops = dict(FLOPS_BUILTIN[prec])
        flops_src = f"built-in ({prec}, uniform mesh, tile 256, of profiles/r02_kernel_metrics.csv): {ncu_src[6:]}"
    flops_unit, bytes_unit = flops[dom], BYTES_ALG[prec][dom]
    flops_step = sum(flops.values())
    alu_peak = fp64_peak_nominal(sm_max, prec)
    t_alu = flops_unit * nt / (alu_peak * 1e12)
    t_hbm = bytes_unit * nt / (hbm_gbs * 1e9)
    try:
        dfma_tf, ffma_tf, copy_gbs = mrd.measure_peaks()
    except Exception:
        dfma_tf = ffma_tf = copy_gbs = None
    if t_alu >= t_hbm:
        ach = flops_unit * nt / (dom_ms * 1e-3) * 1e-12
        roof = {"bound": "alu", "achieved": ach, "peak": alu_peak, "unit": "TFLOP/s", "frac": ach / alu_peak}
    else:
        ach = bytes_unit * nt / (dom_ms * 1e-3) * 1e-9
        roof = {"bound": "hbm", "achieved": ach, "peak": hbm_gbs, "unit": "GB/s", "frac": ach / hbm_gbs}
    if args.traffic is not None:
        traffic, traffic_src = args.traffic, "--traffic (bytes per launch given on the command line)"
    elif ncu and 0.5 <= nt / float(ncu[dom]["triangles"]) <= 4.0:
        traffic, traffic_src = float(ncu[dom]["dram_bytes_per_triangle"]) * nt, ncu_src    # per launch, like `achieved`
    elif ncu:
        # (bytes per triangle depend on how much of the mesh the 126 MB L2 holds: only a capture of a comparable size counts)
        traffic, traffic_src = None, f"none: the ncu capture of this configuration has {ncu[dom]['triangles']} triangles, this run {nt}"
    else:
        traffic, traffic_src = None, ncu_src
    roof.update({"traffic": traffic, "traffic_source": traffic_src, "kernel": dom, "kernel_ms": dom_ms,
                 "peak_source": hbm_src if roof["bound"] == "hbm"
                 else "derived: 148 SM x %d lanes x 2 x %.0f MHz" % (64 if prec == "fp64" else 128, sm_max),
                 "alg_flops_per_triangle": flops_unit, "alg_bytes_per_triangle": bytes_unit, "flops_source": flops_src,
                 "oracle_flops_per_triangle": {"tri_stage1": ORACLE_FLOPS_TRI[0], "tri_stage2": ORACLE_FLOPS_TRI[1]}.get(dom),
                 "alu_frac": flops_unit * nt / (dom_ms * 1e-3) * 1e-12 / alu_peak,
                 "hbm_frac": bytes_unit * nt / (dom_ms * 1e-3) * 1e-9 / hbm_gbs,
                 "measured_fma_tflops": dfma_tf if prec == "fp64" else ffma_tf, "measured_copy_gbs": copy_gbs,
                 "design_bytes_per_triangle": DESIGN_BYTES_TRI.get(dom, {}).get(prec) if tile_eff == 256 else None,
                 "kernels_ms": prof,
                 "step_alg": {"flops_per_triangle_update": flops_step,
                              "bytes_per_triangle_update": B_ALG_STEP[prec],
                              "roofline_ms": max(flops_step * nt / (alu_peak * 1e12), B_ALG_STEP[prec] * nt / (hbm_gbs * 1e9)) * 1e3}})
    roof["step_alg"]["frac"] = roof["step_alg"]["roofline_ms"] / ms_step

    # ---- the oracle beside it (rank 0, N = 1 only): bounded sample of the same workload --------------------
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        n_s = min(args.n, 1024)
        rate, spstep, cores, nts = oracle_rate(n_s, 2, 0, args.numbering)
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"isentropic vortex, periodic {n_s}^2 vertices ({nts} triangles), 2 RK2 steps, "
                         f"{spstep:.2f} s/step, OpenMP triangle loops on {cores} threads"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64" if prec == "fp64" else "f32", "data": "synthetic",
            "config": {"workload": workload_text(args, nt) if not halo else
                                   (f"BASELINE.json config 5 stacked {world} times in y: row of {world} isentropic vortices, periodic uniform "
                                    f"triangulation {args.n} x {args.n * world} vertices, {nt_job} triangles, natural input numbering, "
                                    f"scheme B, RK2, CFL 0.5"),
                       "n_triangles": nt_job, "n_vertices": nv_job, "n_triangles_rank0": nt, "reorder": int(args.reorder), "tile": tile_eff,
                       "l2": "inputs larger than L2 (state %.0f MB, per-triangle arrays %.1f GB)" % (
                           state_bytes / 1e6, gm.device_bytes() / 1e9),
                       "parallelism": parallelism,
                       "layout_s": layout_s, "device_gb": gm.device_bytes() / 1e9, "t_sim": t_sim,
                       "host_rss_gb": __import__("resource").getrusage(__import__("resource").RUSAGE_SELF).ru_maxrss / 1e6,
                       "part_setup_s": None if setup is None else setup["setup_s"],
                       "mesh_generation": getattr(cfg, "generated", None) if not halo else None},
            "vertex_updates_per_s": nv_job * args.steps / (ms_total * 1e-3),
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roof, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="mrd", choices=["mrd", "reference"])
    ap.add_argument("--size", dest="n", type=int, default=4096, help="vertices per side of the periodic mesh")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32"])
    ap.add_argument("--numbering", default="morton", choices=["morton", "natural", "permuted"])
    ap.add_argument("--reorder", type=int, default=1)
    ap.add_argument("--tile", type=int, default=0)
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--traffic", type=float, default=None, help="dram bytes per launch of the dominant kernel (ncu)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--mesh", default="uniform", choices=["uniform", "jitter", "flip", "delaunay", "refined"],
                    help="uniform triangulation (config 5), jittered vertices, jittered + flipped edges (variable valence), or a seeded "
                         "graded Delaunay triangulation of --size^2 points with a frozen boundary ring (--size 1140: the paper's 1.3 M vertices), or "
                         "(refined) a mesh of about --size^2 vertices generated on the GPU by mrd_meshgen_refine")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"],
                    help="N > 1: torch.distributed backend (gloo stages the halo rows through host memory; functional tests only)")
    ap.add_argument("--decomposition", default="halo", choices=["halo", "replicas"],
                    help="N > 1: one mesh over the N GPUs with halo exchanges (default), or N independent replicas")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)
    return run_mrd(args)


if __name__ == "__main__":
    sys.exit(main())
