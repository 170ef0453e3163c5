"""Host side of the multi-GPU path (include/mrd.h "Domain decomposition"), no GPU needed:
the partitioner's invariants on the paper's mesh kinds, the layout stage on the local meshes, and the halo
exchange plumbing over torch.distributed with the gloo backend on world size 2 (payload = global vertex ids,
so that a wrong list, offset or peer shows up as a wrong id)."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import paper_1705_02028_b200 as mrd  # noqa: E402
import workloads as wl  # noqa: E402


def _mesh(kind):
    if kind == "vortex":          # periodic, natural numbering
        return wl.make_config("vortex")
    if kind == "kh":              # periodic, seeded-permuted numbering and node order
        return wl.make_config("kh", n=48, numbering="permuted")
    if kind == "sod":             # wall edges in y, frozen vertices at the x ends
        return wl.make_config("sod", n=64)
    if kind == "riemann4":        # bounded, frozen boundary
        return wl.make_config("riemann4", n=33)
    raise ValueError(kind)


def _parts(cfg, P):
    m = cfg.mesh
    return [mrd.Partition(m.xy, m.tri, P, r, vertex_flag=cfg.vertex_flag, wall_edge=cfg.wall_edge, period=m.period) for r in range(P)]


@pytest.mark.parametrize("kind", ["vortex", "kh", "sod", "riemann4"])
@pytest.mark.parametrize("P", [1, 2, 3, 5])
def test_partition_invariants(kind, P):
    cfg = _mesh(kind)
    m = cfg.mesh
    parts = _parts(cfg, P)
    owner = parts[0].owner
    counts = np.bincount(owner, minlength=P)
    assert counts.sum() == m.nv and counts.max() - counts.min() <= 1          # balanced ranges of the Morton order
    gflag = np.zeros(m.nv, np.uint8) if cfg.vertex_flag is None else np.asarray(cfg.vertex_flag, np.uint8)
    gwall = np.zeros((0, 2), np.int32) if cfg.wall_edge is None else np.asarray(cfg.wall_edge, np.int32)
    seen = np.zeros(m.nv, int)
    for r, p in enumerate(parts):
        assert np.array_equal(p.owner, owner) and p.n_global == m.nv
        vg = p.vertex_global
        own, halo = vg[:p.n_owned], vg[p.n_owned:]
        assert np.array_equal(own, np.nonzero(owner == r)[0])                  # owned first, ascending global id
        assert np.all(np.diff(halo) > 0) and np.all(owner[halo] != r)
        seen[own] += 1
        # local triangles: exactly those with an owned vertex, ascending, same node order
        touch = np.nonzero((owner[m.tri] == r).any(axis=1))[0]
        assert np.array_equal(p.tri_global, touch)
        assert np.array_equal(vg[p.tri], m.tri[touch])
        assert set(np.unique(m.tri[touch])) == set(vg.tolist())               # halo = the other vertices of those triangles
        assert np.array_equal(p.xy, m.xy[vg])
        # flags: halo -> 2, otherwise the global flag
        assert np.all(p.vertex_flag[p.n_owned:] == 2) and np.array_equal(p.vertex_flag[:p.n_owned], gflag[own])
        # wall edges with an owned end, both ends local
        keep = (owner[gwall] == r).any(axis=1) if len(gwall) else np.zeros(0, bool)
        assert np.array_equal(vg[p.wall_edge].reshape(-1, 2), gwall[keep])
        # exchange lists: sends are owned, receives are halo, every halo vertex is received exactly once
        assert np.all(p.send_idx < p.n_owned) and np.array_equal(np.sort(p.recv_idx), np.arange(p.n_owned, p.n_local))
        assert p.send_off[0] == 0 and p.send_off[-1] == p.n_send and p.recv_off[-1] == p.n_recv
        assert r not in p.neighbour and np.all(np.diff(p.neighbour) > 0)
        for k, q in enumerate(p.neighbour):
            rcv = vg[p.recv_idx[p.recv_off[k]:p.recv_off[k + 1]]]
            assert np.all(owner[rcv] == q) and np.all(np.diff(rcv) > 0)
    assert np.all(seen == 1)
    # what a sends to b is what b expects from a, in the same order
    for a, pa in enumerate(parts):
        for k, b in enumerate(pa.neighbour):
            pb = parts[b]
            kb = list(pb.neighbour).index(a)
            sent = pa.vertex_global[pa.send_idx[pa.send_off[k]:pa.send_off[k + 1]]]
            want = pb.vertex_global[pb.recv_idx[pb.recv_off[kb]:pb.recv_off[kb + 1]]]
            assert len(sent) > 0 and np.array_equal(sent, want)
    if P == 1:
        assert parts[0].n_neighbour == 0 and parts[0].n_local == m.nv and parts[0].n_tri == m.nt


@pytest.mark.parametrize("kind", ["vortex", "sod"])
def test_local_layout_has_the_global_volumes_on_owned_vertices(kind):
    """The update of an owned vertex needs its full fan: V_i of the local layout == V_i of the global one there."""
    cfg = _mesh(kind)
    m = cfg.mesh
    G = mrd.Layout(m.xy, m.tri, vertex_flag=cfg.vertex_flag, wall_edge=cfg.wall_edge, period=m.period)
    g = G.get()
    vol_g = np.empty(m.nv)
    vol_g[g["vperm"]] = g["vol"]
    for p in _parts(cfg, 3):
        L = mrd.Layout(p.xy, p.tri, vertex_flag=p.vertex_flag, wall_edge=p.wall_edge if p.n_wall else None, period=m.period)
        l = L.get()
        vol_l = np.empty(p.n_local)
        vol_l[l["vperm"]] = l["vol"]
        own = p.vertex_global[:p.n_owned]
        assert np.allclose(vol_l[:p.n_owned], vol_g[own], rtol=1e-14, atol=0)
        vh = vol_g[p.vertex_global[p.n_owned:]]
        assert np.all(vol_l[p.n_owned:] <= vh * (1 + 1e-14)) and np.any(vol_l[p.n_owned:] < 0.9 * vh)  # halo fans are cut
        assert L.nf == int((p.vertex_flag != 0).sum())


def test_partition_errors():
    cfg = _mesh("vortex")
    m = cfg.mesh
    with pytest.raises(mrd.MrdError):
        mrd.Partition(m.xy, m.tri, 0, 0, period=m.period)
    with pytest.raises(mrd.MrdError):
        mrd.Partition(m.xy, m.tri, 2, 2, period=m.period)
    with pytest.raises(mrd.MrdError):
        mrd.Partition(m.xy, m.tri, m.nv + 1, 0, period=m.period)
    bad = m.tri.copy()
    bad[0, 0] = m.nv
    with pytest.raises(mrd.MrdError):
        mrd.Partition(m.xy, bad, 2, 0, period=m.period)
    with pytest.raises(mrd.MrdError):
        mrd.Partition(m.xy, m.tri, 2, 0, vertex_flag=np.full(m.nv, 2, np.uint8), period=m.period)
    with pytest.raises(mrd.MrdError):   # layout stage: flag values above 2
        mrd.Layout(m.xy, m.tri, vertex_flag=np.full(m.nv, 3, np.uint8), period=m.period)


def _exchange_worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    from paper_1705_02028_b200.distributed import HaloExchange
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = _mesh("kh")
    m = cfg.mesh
    p = mrd.Partition(m.xy, m.tri, world, rank, period=m.period)
    comm = HaloExchange(p.neighbour, p.send_off, p.recv_off, 4)
    gid = torch.as_tensor(p.vertex_global, dtype=torch.float64)
    comp = torch.arange(4, dtype=torch.float64) * 0.25
    send = (gid[torch.as_tensor(p.send_idx, dtype=torch.long)][:, None] + comp[None, :]).reshape(-1).contiguous()
    recv = torch.full((4 * p.n_recv,), -1.0, dtype=torch.float64)
    comm.exchange(send, recv)
    want = (gid[torch.as_tensor(p.recv_idx, dtype=torch.long)][:, None] + comp[None, :]).reshape(-1)
    d = torch.tensor([3.0 + rank, -1.0 if rank == 1 else 0.0], dtype=torch.float64)
    comm.allreduce_min(d)
    dist.barrier()
    out.put((rank, bool(torch.equal(recv, want)), d.tolist(), p.n_recv))
    dist.destroy_process_group()


def test_halo_exchange_gloo_world_size_2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29100 + os.getpid() % 300
    procs = [ctx.Process(target=_exchange_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ok, d, nrecv in res:
        assert nrecv > 0 and ok          # every halo row arrived from the right peer at the right offset
        assert d == [3.0, -1.0]          # the minimum over ranks of both doubles (dt bound, non-physical flag)


@pytest.mark.parametrize("world", [2, 3, 8])
def test_part_made_from_local_pieces_equals_the_part_of_the_whole_mesh(world):
    """N > 1 start-up without any whole-mesh array: `uniform_strip_part` + `Partition.from_local` give exactly what
    the partitioner gives for the whole strip with the same owners -- local numbering, triangles, flags and exchange lists."""
    n = 16
    whole = wl.uniform_mesh(n, n * world, 10.0, 10.0 * world, periodic=True)
    owner = (np.arange(whole.nv) // n // n).astype(np.int32)               # row bands of n vertex rows
    for rank in range(world):
        pc = wl.uniform_strip_part(n, world, rank)
        assert pc["n_vertex_global"] == whole.nv and len(pc["vertex_global"]) == (n + 2) * n and len(pc["tri"]) == 2 * (n + 1) * n
        assert np.array_equal(whole.xy[pc["vertex_global"]], pc["xy"])
        assert np.array_equal(whole.tri[pc["tri_global"]], pc["vertex_global"][pc["tri"]])
        loc = mrd.Partition.from_local(pc["n_vertex_global"], pc["vertex_global"], pc["owner"], pc["xy"], pc["tri"], pc["tri_global"],
                                       world, rank, period=pc["period"], domain_size=pc["domain_size"])
        ref = mrd.Partition(whole.xy, whole.tri, world, rank, period=whole.period, owner=owner)
        for name in ("vertex_global", "xy", "tri", "tri_global", "vertex_flag", "wall_edge", "neighbour", "send_off", "send_idx",
                     "recv_off", "recv_idx"):
            assert np.array_equal(getattr(loc, name), getattr(ref, name)), (name, rank)
        assert (loc.n_owned, loc.n_send, loc.n_recv, loc.n_global) == (ref.n_owned, ref.n_send, ref.n_recv, ref.n_global)
        assert loc.owner is None and loc.domain_size == ref.domain_size == 10.0 * world


def test_local_part_rejects_bad_input():
    pc = wl.uniform_strip_part(6, 2, 0)
    args = (pc["n_vertex_global"], pc["vertex_global"], pc["owner"], pc["xy"], pc["tri"], pc["tri_global"], 2, 0)
    bad = pc["tri"].copy()
    bad[0, 0] = 10 ** 6
    with pytest.raises(mrd.MrdError):
        mrd.Partition.from_local(args[0], args[1], args[2], args[3], bad, args[5], 2, 0)
    dup = pc["vertex_global"].copy()
    dup[1] = dup[0]
    with pytest.raises(mrd.MrdError):
        mrd.Partition.from_local(args[0], dup, *args[2:])
    with pytest.raises(mrd.MrdError):                                      # a part that owns nothing of what it was given
        mrd.Partition.from_local(args[0], args[1], np.ones_like(pc["owner"]), *args[3:])
