"""One mesh over several GPUs: one process per GPU, `torch.distributed` for the plumbing.

Each rank holds one part of the domain decomposition of include/mrd.h ("Domain decomposition": owner-computes
over contiguous Morton ranges, cut triangles recomputed on both sides) as an ordinary `Mesh` and steps it in
phases; between the phases this module moves bytes and nothing else:

  * after RESIDUAL1: all-reduce(min) of two doubles (eq. 44: the global minimum of 2 V_i / sum s_T; the
    non-physical flag rides along),
  * after UPDATE1 and after STAGE2: neighbour exchange of the conserved state of the vertices on the cut
    (`mrd_halo_pack` -> send/recv -> `mrd_halo_unpack`),
  * before END: all-reduce(max) of one double, the non-physical flag of the whole step, so that every rank commits
    or discards the same step (and `step` returns the same (steps, t) or raises the same error everywhere).

With the `nccl` backend the packed buffers go device to device over NVLink; with `gloo` (tests on a box with
one GPU, or none for the host logic) they are staged through host memory.  No arithmetic of the method lives
here: every value is produced by the kernels behind `mrd_phase` / `mrd_halo_unpack`.
"""
from __future__ import annotations

import numpy as np

from .binding import Mesh, Partition


class HaloExchange:
    """Neighbour exchange of packed rows and the min-reduction, over a torch.distributed process group."""

    def __init__(self, neighbour, send_off, recv_off, width=4, group=None):
        import torch
        import torch.distributed as dist
        self._torch, self._dist, self.group = torch, dist, group
        self.neighbour = [int(q) for q in neighbour]
        self.send_off = [int(x) * width for x in send_off]
        self.recv_off = [int(x) * width for x in recv_off]
        self.staged = dist.get_backend(group) != "nccl"  # gloo moves host memory only
        self.rank = dist.get_rank(group)

    def _peer(self, q):
        return self._dist.get_global_rank(self.group, q) if self.group is not None else q

    def exchange(self, send, recv):
        """send / recv: flat tensors holding the rows for / from each neighbour back to back (list order)."""
        t, dist = self._torch, self._dist
        if not self.neighbour:
            return
        src = send.cpu() if self.staged else send
        dst = t.empty(recv.shape, dtype=recv.dtype) if self.staged else recv
        ops = []
        for k, q in enumerate(self.neighbour):
            s0, s1, r0, r1 = self.send_off[k], self.send_off[k + 1], self.recv_off[k], self.recv_off[k + 1]
            if s1 > s0:
                ops.append(dist.P2POp(dist.isend, src[s0:s1], self._peer(q), self.group))
            if r1 > r0:
                ops.append(dist.P2POp(dist.irecv, dst[r0:r1], self._peer(q), self.group))
        for w in dist.batch_isend_irecv(ops):
            w.wait()
        if self.staged:
            recv.copy_(dst)

    def allreduce_min(self, d):
        self._allreduce(d, self._dist.ReduceOp.MIN)

    def allreduce_max(self, d):
        self._allreduce(d, self._dist.ReduceOp.MAX)

    def _allreduce(self, d, op):
        dist = self._dist
        if self.staged:
            h = d.cpu()
            dist.all_reduce(h, op=op, group=self.group)
            d.copy_(h)
        else:
            dist.all_reduce(d, op=op, group=self.group)


class DistributedMesh:
    """The `Mesh` interface for one global mesh spread over the ranks of a process group.

    Every rank passes the same global arrays (`xy`, `tri`, `vertex_flag`, `wall_edge`) and parameters; the state
    crosses this interface in GLOBAL user numbering.  Call from every rank in the same order."""

    def __init__(self, xy, tri, vertex_flag=None, wall_edge=None, group=None, part=None, **params):
        """Either the whole mesh (every rank passes the same global arrays; fine up to a few 10^7 triangles), or `part`, a
        `Partition` each rank made for itself (`Partition.from_local`: no whole-mesh array anywhere; xy and tri are ignored)."""
        import torch
        import torch.distributed as dist
        self._torch, self._dist, self.group = torch, dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        period = params.get("period", (0.0, 0.0))
        if part is None:
            part = Partition(xy, tri, self.world, self.rank, vertex_flag=vertex_flag, wall_edge=wall_edge, period=period)
        assert part.n_part == self.world and part.part == self.rank
        P = self.part = part
        params = dict(params, domain_size=P.domain_size)     # Bx: L of eq. 56 is the WHOLE mesh's, not the part's
        self.mesh = Mesh(P.xy, P.tri, vertex_flag=P.vertex_flag, wall_edge=P.wall_edge if P.n_wall else None, **params)
        self.mesh.halo_set(P.send_idx, P.recv_idx)
        self.nv, self.dtype, self.np_dtype = P.n_global, self.mesh.dtype, self.mesh.np_dtype
        self.nt_local = P.n_tri
        self.comm = HaloExchange(P.neighbour, P.send_off, P.recv_off, 4, group)
        self._send = torch.empty(4 * P.n_send, dtype=self.dtype, device="cuda")
        self._recv = torch.empty(4 * P.n_recv, dtype=self.dtype, device="cuda")
        self._d = torch.empty(2, dtype=torch.float64, device="cuda")
        self._rk2 = self.mesh.params.time_order == 2
        self._bx = self.mesh.params.scheme == 5   # Bx: the speed range of eq. 56 is reduced over all parts
        self._r = torch.empty(2, dtype=torch.float64, device="cuda")
        self._f = torch.empty(1, dtype=torch.float64, device="cuda")
        self._open = False

    def close(self):
        self.mesh.close()

    # ---- state ----
    def set_state(self, W):
        """W: [4][nv_global] numpy array or torch tensor (any device); each rank keeps its part."""
        t = self._torch
        idx = self.part.vertex_global
        if isinstance(W, t.Tensor):
            loc = W.to("cuda", self.dtype)[:, t.as_tensor(idx, device="cuda", dtype=t.long)].contiguous()
        else:
            loc = t.as_tensor(np.ascontiguousarray(np.asarray(W)[:, idx], dtype=self.np_dtype), device="cuda")
        self.mesh.set_state(loc)

    def owned_state(self):
        """(global ids [n_owned], W [4][n_owned]) of the vertices this rank owns."""
        no = self.part.n_owned
        return self.part.vertex_global[:no], self.mesh.get_state()[:, :no].contiguous()

    def set_state_local(self, W_local):
        """W_local: [4][n_local] in the part's own vertex order (`part.vertex_global`): nothing global is touched."""
        t = self._torch
        loc = t.as_tensor(np.ascontiguousarray(W_local, dtype=self.np_dtype), device="cuda") if not isinstance(W_local, t.Tensor) \
            else W_local.to("cuda", self.dtype).contiguous()
        self.mesh.set_state(loc)

    def get_state(self):
        """The whole state [4][nv_global] (host, numpy) on every rank (small meshes: tests, output)."""
        t, dist = self._torch, self._dist
        ids, W = self.owned_state()
        counts = [None] * self.world
        dist.all_gather_object(counts, int(len(ids)), group=self.group)
        width = max(counts)
        pad = t.zeros((4, width), dtype=self.dtype, device="cuda")
        pad[:, :W.shape[1]] = W
        pid = t.zeros(width, dtype=t.int32, device="cuda")
        pid[:len(ids)] = t.as_tensor(ids, device="cuda")
        if self.comm.staged:
            pad, pid = pad.cpu(), pid.cpu()
        parts = [t.empty_like(pad) for _ in range(self.world)]
        pids = [t.empty_like(pid) for _ in range(self.world)]
        dist.all_gather(parts, pad, group=self.group)
        dist.all_gather(pids, pid, group=self.group)
        out = np.empty((4, self.nv), dtype=self.np_dtype)
        for q in range(self.world):
            out[:, pids[q][:counts[q]].cpu().numpy()] = parts[q][:, :counts[q]].cpu().numpy()
        return out

    # ---- stepping ----
    def _exchange(self):
        m = self.mesh
        m.halo_pack(self._send)
        self.comm.exchange(self._send, self._recv)
        m.halo_unpack(self._recv)

    def _range(self, stage):
        m = self.mesh
        m.range_get(stage, self._r)
        self.comm.allreduce_max(self._r)
        m.range_set(stage, self._r)

    def _one_step(self):
        m = self.mesh
        m.phase(m.PHASE_RESIDUAL1)
        m.dt_get(self._d)
        self.comm.allreduce_min(self._d)
        m.dt_set(self._d)
        m.phase(m.PHASE_UPDATE1)
        self._exchange()
        if self._rk2:
            if self._bx:
                self._range(2)
            m.phase(m.PHASE_STAGE2)
            self._exchange()
        m.status_get(self._f)                 # a rank that met rho <= 0, p <= 0 or c^2 <= 0 anywhere in this step ...
        self.comm.allreduce_max(self._f)
        m.status_set(self._f)                 # ... makes every rank discard it
        m.phase(m.PHASE_END)
        if self._bx:
            self._range(1)

    def step_async(self, n_steps):
        """Enqueue n steps without the final synchronisation (timing loops); follow with sync()."""
        if not self._open:
            self.mesh.phase_begin(0.0)
            if self._bx:
                self._range(1)
            self._open = True
        for _ in range(int(n_steps)):
            self._one_step()

    def sync(self):
        if self._open:
            self._open = False
            return self.mesh.phase_end()
        return self.mesh.sync()

    def step(self, max_steps=1, t_end=0.0):
        """As Mesh.step: (steps done, t, dt of the last step); the same values on every rank."""
        assert not self._open, "sync() first"
        done, t, dt = 0, 0.0, 0.0
        left = int(max_steps)
        while left > 0:
            chunk = min(left, 32) if t_end > 0.0 else left
            self.mesh.phase_begin(t_end)
            if self._bx:
                self._range(1)
            for _ in range(chunk):
                self._one_step()
            n, t, dt = self.mesh.phase_end()
            done += n
            left -= chunk
            if n < chunk or (t_end > 0.0 and t >= t_end):
                break
        return done, t, dt

    def diagnostics(self):
        """(totals[4] = sum_i V_i W_i over the whole mesh, min rho, min p) on every rank."""
        t, dist = self._torch, self._dist
        tot, mr, mp = self.mesh.diagnostics()
        a = t.tensor(list(tot), dtype=t.float64)
        b = t.tensor([mr, mp], dtype=t.float64)
        if not self.comm.staged:
            a, b = a.cuda(), b.cuda()
        dist.all_reduce(a, op=dist.ReduceOp.SUM, group=self.group)
        dist.all_reduce(b, op=dist.ReduceOp.MIN, group=self.group)
        a, b = a.cpu().numpy(), b.cpu().numpy()
        return a, float(b[0]), float(b[1])

    def launch_count(self) -> int:
        return self.mesh.launch_count()
