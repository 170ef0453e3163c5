"""ctypes binding of include/mrd.h.  Marshalling only; no arithmetic of the method lives here."""
from __future__ import annotations

import ctypes as C
import os
import re

import numpy as np

from . import build as _build

MRD_OK, MRD_EINVAL, MRD_ENOMEM, MRD_ECUDA, MRD_ENONPHYSICAL = 0, -1, -2, -3, -4
SCHEME_N, SCHEME_LDA, SCHEME_B, SCHEME_BMAX, SCHEME_BMIN, SCHEME_BX = 0, 1, 2, 3, 4, 5
FP64, FP32 = 0, 1


class Params(C.Structure):
    """mrd_params of include/mrd.h."""
    _fields_ = [("gamma", C.c_double), ("cfl", C.c_double), ("scheme", C.c_int32), ("time_order", C.c_int32),
                ("precision", C.c_int32), ("reorder", C.c_int32), ("period_x", C.c_double), ("period_y", C.c_double),
                ("tile", C.c_int32), ("lumping", C.c_int32), ("domain_size", C.c_double)]


class MrdError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"mrd error {code}: {msg}")
        self.code = code


_lib = None
_dp, _ip, _lp, _bp = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_int64), C.POINTER(C.c_uint8)


def lib():
    """Load (building it first when missing or stale) paper_1705_02028_b200/libmrd.so. Fails loudly."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        vp, pp = C.c_void_p, C.POINTER(Params)
        mesh_args = [pp, C.c_int64, _dp, C.c_int64, _ip, _bp, C.c_int64, _ip]
        L.mrd_layout_create.argtypes = [C.POINTER(vp)] + mesh_args
        L.mrd_layout_destroy.argtypes = [vp]
        L.mrd_layout_destroy.restype = None
        L.mrd_layout_sizes.argtypes = [vp, _lp]
        L.mrd_layout_get.argtypes = [vp, _ip, _ip, _ip, _ip, _ip, _dp, _dp]
        L.mrd_mesh_create.argtypes = [C.POINTER(vp)] + mesh_args
        L.mrd_mesh_destroy.argtypes = [vp]
        L.mrd_mesh_destroy.restype = None
        L.mrd_mesh_device_bytes.argtypes = [vp, _lp]
        L.mrd_set_state.argtypes = [vp, vp, vp]
        L.mrd_set_state_host.argtypes = [vp, vp, vp]
        L.mrd_get_state.argtypes = [vp, vp, vp]
        L.mrd_get_state_host.argtypes = [vp, vp, vp]
        L.mrd_step.argtypes = [vp, C.c_int64, C.c_double, vp, _lp, _dp, _dp]
        L.mrd_step_async.argtypes = [vp, C.c_int64, vp]
        L.mrd_sync.argtypes = [vp, vp, _lp, _dp, _dp]
        L.mrd_get_diagnostics.argtypes = [vp, _dp, _dp, _dp, vp]
        L.mrd_dump_stage1.argtypes = [vp, _dp, _dp, _dp, _dp, _dp, vp]
        L.mrd_dump_stage1_sample.argtypes = [vp, C.c_int64, _lp, _dp, _dp, _dp, _dp, _dp, vp]
        L.mrd_measure_peaks.argtypes = [_dp, _dp, _dp, vp]
        L.mrd_launch_count.argtypes = [vp, _lp]
        L.mrd_step_profile.argtypes = [vp, vp, C.POINTER(C.c_float)]
        L.mrd_partition_create.argtypes = [C.POINTER(vp), C.c_int64, _dp, C.c_int64, _ip, _bp, C.c_int64, _ip, C.c_double,
                                           C.c_double, C.c_int32, C.c_int32]
        L.mrd_partition_create_owned.argtypes = [C.POINTER(vp), C.c_int64, _dp, C.c_int64, _ip, _bp, C.c_int64, _ip, C.c_double,
                                                 C.c_double, C.c_int32, C.c_int32, _ip]
        L.mrd_partition_create_local.argtypes = [C.POINTER(vp), C.c_int64, C.c_double, C.c_int64, _ip, _ip, _dp, _bp, C.c_int64, _ip,
                                                 _ip, C.c_int64, _ip, C.c_int32, C.c_int32]
        L.mrd_partition_destroy.argtypes = [vp]
        L.mrd_partition_destroy.restype = None
        L.mrd_partition_sizes.argtypes = [vp, _lp]
        L.mrd_partition_get.argtypes = [vp, C.c_char_p, vp, C.c_int64]
        L.mrd_halo_set.argtypes = [vp, C.c_int64, _ip, C.c_int64, _ip]
        L.mrd_phase_begin.argtypes = [vp, C.c_double, vp]
        L.mrd_phase.argtypes = [vp, C.c_int32, vp]
        L.mrd_phase_end.argtypes = [vp, vp, _lp, _dp, _dp]
        L.mrd_dt_get.argtypes = [vp, vp, vp]
        L.mrd_dt_set.argtypes = [vp, vp, vp]
        L.mrd_status_get.argtypes = [vp, vp, vp]
        L.mrd_status_set.argtypes = [vp, vp, vp]
        L.mrd_partition_domain_size.argtypes = [vp, _dp]
        L.mrd_halo_pack.argtypes = [vp, vp, vp]
        L.mrd_range_get.argtypes = [vp, C.c_int32, vp, vp]
        L.mrd_range_set.argtypes = [vp, C.c_int32, vp, vp]
        L.mrd_halo_unpack.argtypes = [vp, vp, vp]
        L.mrd_meshgen_test_quality.argtypes = [C.c_int64, vp, vp, C.c_double, C.c_double, vp, vp, vp, vp, _lp, vp]
        L.mrd_meshgen_orient2d.argtypes = [C.c_int64, vp, vp, vp, _lp, vp]
        L.mrd_meshgen_incircle2d.argtypes = [C.c_int64, vp, vp, vp, _lp, vp]
        L.mrd_meshgen_orient2d_static.argtypes = [C.c_int64, vp, vp, vp, vp, vp]
        L.mrd_meshgen_release.argtypes = []
        L.mrd_meshgen_flip_stats.argtypes = [_lp, C.c_int]
        L.mrd_meshgen_build_edges.argtypes = [C.c_int64, vp, vp, vp, _lp, vp]
        L.mrd_meshgen_delaunay_flip.argtypes = [C.c_int64, C.c_int64, vp, vp, vp, vp, _lp, _lp, _lp, vp]
        L.mrd_meshgen_refine.argtypes = [C.c_double, C.c_double, C.c_uint32, C.c_int64, C.c_int64, _dp, vp, _dp, C.c_int64, C.c_int64,
                                         C.c_int64, C.c_int64, C.c_int64,
                                         _lp, _lp, _lp, vp, vp, vp, vp, _lp, _lp, vp]
        L.mrd_meshgen_find_triangle.argtypes = [C.c_int64, vp, vp, C.c_int64, vp, vp, vp, vp, vp, vp, vp]
        L.mrd_last_error.restype = C.c_char_p
        L.mrd_version.restype = C.c_char_p
        L._path = path
        _lib = L
    return _lib


def exported_symbols():
    """Names declared in include/mrd.h (functions `mrd_*(`), for the symbol-export test."""
    hdr = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "mrd.h")
    text = open(hdr).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mrd_[a-z0-9_]+)\s*\(", text)))


def version() -> str:
    return lib().mrd_version().decode()


def _check(rc):
    if rc != 0:
        raise MrdError(rc, lib().mrd_last_error().decode())


def _np_ptr(a, ctype):
    return None if a is None else a.ctypes.data_as(C.POINTER(ctype))


def _mesh_args(xy, tri, vertex_flag, wall_edge):
    xy = np.ascontiguousarray(xy, dtype=np.float64)
    tri = np.ascontiguousarray(tri, dtype=np.int32)
    assert xy.ndim == 2 and xy.shape[1] == 2 and tri.ndim == 2 and tri.shape[1] == 3
    flag = None if vertex_flag is None else np.ascontiguousarray(vertex_flag, dtype=np.uint8)
    wedge = None if wall_edge is None else np.ascontiguousarray(wall_edge, dtype=np.int32)
    ne = 0 if wedge is None else int(wedge.shape[0])
    keep = (xy, tri, flag, wedge)
    args = (xy.shape[0], _np_ptr(xy, C.c_double), tri.shape[0], _np_ptr(tri, C.c_int32), _np_ptr(flag, C.c_uint8), ne,
            _np_ptr(wedge, C.c_int32))
    return keep, args


def make_params(gamma=1.4, cfl=0.5, scheme=SCHEME_B, time_order=2, precision=FP64, reorder=True,
                period=(0.0, 0.0), tile=0, lumping=0, domain_size=0.0) -> Params:
    return Params(float(gamma), float(cfl), int(scheme), int(time_order), int(precision), int(bool(reorder)),
                  float(period[0]), float(period[1]), int(tile), int(lumping), float(domain_size))


class Layout:
    """mrd_layout_*: the host-only mesh-layout stage (no CUDA needed)."""

    def __init__(self, xy, tri, vertex_flag=None, wall_edge=None, **params):
        self.params = make_params(**params)
        keep, args = _mesh_args(xy, tri, vertex_flag, wall_edge)
        h = C.c_void_p()
        _check(lib().mrd_layout_create(C.byref(h), C.byref(self.params), *args))
        self._h = h
        n = (C.c_int64 * 6)()
        _check(lib().mrd_layout_sizes(h, n))
        self.nv, self.nt, self.ne, self.nf, self.ntile, self.nslot = [int(x) for x in n]

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h and lib is not None:                                  # module globals are gone when the interpreter shuts down
            lib().mrd_layout_destroy(h)

    def get(self):
        nv, nt = self.nv, self.nt
        o = dict(vperm=np.empty(nv, np.int32), tperm=np.empty(nt, np.int32), tri=np.empty((nt, 3), np.int32),
                 csr_off=np.empty(nv + 1, np.int32), csr_ent=np.empty(3 * nt, np.int32), area=np.empty(nt),
                 vol=np.empty(nv))
        _check(lib().mrd_layout_get(self._h, _np_ptr(o["vperm"], C.c_int32), _np_ptr(o["tperm"], C.c_int32),
                                    _np_ptr(o["tri"], C.c_int32), _np_ptr(o["csr_off"], C.c_int32),
                                    _np_ptr(o["csr_ent"], C.c_int32), _np_ptr(o["area"], C.c_double),
                                    _np_ptr(o["vol"], C.c_double)))
        return o


def _stream_ptr(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return C.c_void_p(int(stream.cuda_stream))


class Partition:
    """mrd_partition_*: one part of the domain decomposition of a global mesh (host only, no CUDA needed)."""

    _ARRAYS = (("vertex_global", np.int32, lambda n: (n[0],)), ("xy", np.float64, lambda n: (n[0], 2)),
               ("tri", np.int32, lambda n: (n[2], 3)), ("tri_global", np.int32, lambda n: (n[2],)),
               ("vertex_flag", np.uint8, lambda n: (n[0],)), ("wall_edge", np.int32, lambda n: (n[3], 2)),
               ("neighbour", np.int32, lambda n: (n[4],)), ("send_off", np.int32, lambda n: (n[4] + 1,)),
               ("send_idx", np.int32, lambda n: (n[5],)), ("recv_off", np.int32, lambda n: (n[4] + 1,)),
               ("recv_idx", np.int32, lambda n: (n[6],)), ("owner", np.int32, lambda n: (n[7],)))

    def __init__(self, xy, tri, n_part, part, vertex_flag=None, wall_edge=None, period=(0.0, 0.0), owner=None):
        """Part `part` of `n_part` of the WHOLE mesh (xy, tri, ...): owners = contiguous ranges of the vertices' Morton order,
        or the `owner` array (int32 [nv]) when given."""
        keep, args = _mesh_args(xy, tri, vertex_flag, wall_edge)
        h = C.c_void_p()
        if owner is None:
            _check(lib().mrd_partition_create(C.byref(h), *args, float(period[0]), float(period[1]), int(n_part), int(part)))
        else:
            own = np.ascontiguousarray(owner, dtype=np.int32)
            assert own.shape == (args[0],)
            _check(lib().mrd_partition_create_owned(C.byref(h), *args, float(period[0]), float(period[1]), int(n_part), int(part),
                                                    _np_ptr(own, C.c_int32)))
        self._load(h, n_part, part, period, has_owner=True)

    @classmethod
    def from_local(cls, n_vertex_global, vertex_global, owner, xy, tri, tri_global, n_part, part, vertex_flag=None, wall_edge=None,
                   period=(0.0, 0.0), domain_size=0.0):
        """mrd_partition_create_local: the part assembled from local pieces (no whole-mesh array); `tri` / `wall_edge` index the
        local arrays.  `self.owner` is None."""
        vg = np.ascontiguousarray(vertex_global, dtype=np.int32)
        own = np.ascontiguousarray(owner, dtype=np.int32)
        xy = np.ascontiguousarray(xy, dtype=np.float64)
        tri = np.ascontiguousarray(tri, dtype=np.int32)
        tg = np.ascontiguousarray(tri_global, dtype=np.int32)
        flag = None if vertex_flag is None else np.ascontiguousarray(vertex_flag, dtype=np.uint8)
        wedge = None if wall_edge is None else np.ascontiguousarray(wall_edge, dtype=np.int32)
        assert vg.shape == own.shape == (xy.shape[0],) and tri.shape == (tg.shape[0], 3)
        self = cls.__new__(cls)
        h = C.c_void_p()
        _check(lib().mrd_partition_create_local(C.byref(h), int(n_vertex_global), float(domain_size), xy.shape[0], _np_ptr(vg, C.c_int32),
                                                _np_ptr(own, C.c_int32), _np_ptr(xy, C.c_double), _np_ptr(flag, C.c_uint8),
                                                tri.shape[0], _np_ptr(tri, C.c_int32), _np_ptr(tg, C.c_int32),
                                                0 if wedge is None else wedge.shape[0], _np_ptr(wedge, C.c_int32), int(n_part), int(part)))
        self._load(h, n_part, part, period, has_owner=False)
        return self

    def _load(self, h, n_part, part, period, has_owner):
        try:
            n = (C.c_int64 * 8)()
            _check(lib().mrd_partition_sizes(h, n))
            n = [int(x) for x in n]
            (self.n_local, self.n_owned, self.n_tri, self.n_wall, self.n_neighbour, self.n_send, self.n_recv,
             self.n_global) = n
            ds = C.c_double()
            _check(lib().mrd_partition_domain_size(h, C.byref(ds)))
            self.domain_size = ds.value
            for name, dt, shape in self._ARRAYS:
                if name == "owner" and not has_owner:
                    self.owner = None
                    continue
                a = np.empty(shape(n), dtype=dt)
                _check(lib().mrd_partition_get(h, name.encode(), C.c_void_p(a.ctypes.data), a.nbytes))
                setattr(self, name, a)
        finally:
            lib().mrd_partition_destroy(h)
        self.n_part, self.part, self.period = int(n_part), int(part), (float(period[0]), float(period[1]))


class Mesh:
    """mrd_mesh_*: mesh + device state + stepper.  State tensors are torch CUDA tensors [4][nv]
    (float64 or float32 per `precision`) in USER numbering, or numpy arrays for the *_host calls."""

    def __init__(self, xy, tri, vertex_flag=None, wall_edge=None, **params):
        import torch
        if not torch.cuda.is_available():
            raise MrdError(MRD_ECUDA, "no CUDA device: the mrd path has no CPU fallback")
        self._torch = torch
        self.params = make_params(**params)
        self.dtype = torch.float64 if self.params.precision == FP64 else torch.float32
        self.np_dtype = np.float64 if self.params.precision == FP64 else np.float32
        keep, args = _mesh_args(xy, tri, vertex_flag, wall_edge)
        self.nv, self.nt = int(args[0]), int(args[2])
        h = C.c_void_p()
        _check(lib().mrd_mesh_create(C.byref(h), C.byref(self.params), *args))
        self._h = h

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h and lib is not None:                                  # module globals are gone when the interpreter shuts down
            lib().mrd_mesh_destroy(h)

    close = __del__

    def device_bytes(self) -> int:
        n = C.c_int64()
        _check(lib().mrd_mesh_device_bytes(self._h, C.byref(n)))
        return n.value

    def _check_tensor(self, W):
        t = self._torch
        assert isinstance(W, t.Tensor) and W.is_cuda and W.dtype == self.dtype and W.is_contiguous()
        assert tuple(W.shape) == (4, self.nv), (tuple(W.shape), self.nv)

    def set_state(self, W, stream=None):
        self._check_tensor(W)
        _check(lib().mrd_set_state(self._h, C.c_void_p(W.data_ptr()), _stream_ptr(stream)))

    def set_state_host(self, W, stream=None):
        W = np.ascontiguousarray(W, dtype=self.np_dtype)
        assert W.shape == (4, self.nv)
        _check(lib().mrd_set_state_host(self._h, C.c_void_p(W.ctypes.data), _stream_ptr(stream)))

    def get_state(self, out=None, stream=None):
        if out is None:
            out = self._torch.empty((4, self.nv), dtype=self.dtype, device="cuda")
        self._check_tensor(out)
        _check(lib().mrd_get_state(self._h, C.c_void_p(out.data_ptr()), _stream_ptr(stream)))
        return out

    def get_state_host(self, out=None, stream=None):
        if out is None:
            out = np.empty((4, self.nv), dtype=self.np_dtype)
        assert out.dtype == self.np_dtype and out.shape == (4, self.nv) and out.flags.c_contiguous
        _check(lib().mrd_get_state_host(self._h, C.c_void_p(out.ctypes.data), _stream_ptr(stream)))
        return out

    def step(self, max_steps=1, t_end=0.0, stream=None):
        n, t, dt = C.c_int64(0), C.c_double(0.0), C.c_double(0.0)
        _check(lib().mrd_step(self._h, int(max_steps), float(t_end), _stream_ptr(stream), C.byref(n), C.byref(t),
                              C.byref(dt)))
        return n.value, t.value, dt.value

    def step_async(self, n_steps, stream=None):
        _check(lib().mrd_step_async(self._h, int(n_steps), _stream_ptr(stream)))

    def sync(self, stream=None):
        n, t, dt = C.c_int64(0), C.c_double(0.0), C.c_double(0.0)
        _check(lib().mrd_sync(self._h, _stream_ptr(stream), C.byref(n), C.byref(t), C.byref(dt)))
        return n.value, t.value, dt.value

    def diagnostics(self, stream=None):
        tot = np.empty(4)
        mr, mp = C.c_double(), C.c_double()
        _check(lib().mrd_get_diagnostics(self._h, _np_ptr(tot, C.c_double), C.byref(mr), C.byref(mp),
                                         _stream_ptr(stream)))
        return tot, mr.value, mp.value

    def dump_stage1(self, stream=None):
        nt = self.nt
        o = dict(phiT=np.empty((nt, 4)), phiN=np.empty((nt, 3, 4)), phiLDA=np.empty((nt, 3, 4)),
                 phiB=np.empty((nt, 3, 4)), sT=np.empty(nt))
        _check(lib().mrd_dump_stage1(self._h, _np_ptr(o["phiT"], C.c_double), _np_ptr(o["phiN"], C.c_double),
                                     _np_ptr(o["phiLDA"], C.c_double), _np_ptr(o["phiB"], C.c_double),
                                     _np_ptr(o["sT"], C.c_double), _stream_ptr(stream)))
        return o

    def dump_stage1_sample(self, tri_ids, stream=None):
        ids = np.ascontiguousarray(tri_ids, dtype=np.int64)
        n = len(ids)
        o = dict(phiT=np.empty((n, 4)), phiN=np.empty((n, 3, 4)), phiLDA=np.empty((n, 3, 4)), phiB=np.empty((n, 3, 4)),
                 sT=np.empty(n))
        _check(lib().mrd_dump_stage1_sample(self._h, n, _np_ptr(ids, C.c_int64), _np_ptr(o["phiT"], C.c_double),
                                            _np_ptr(o["phiN"], C.c_double), _np_ptr(o["phiLDA"], C.c_double),
                                            _np_ptr(o["phiB"], C.c_double), _np_ptr(o["sT"], C.c_double),
                                            _stream_ptr(stream)))
        return o

    # ---- domain decomposition: halo lists and the step in phases (include/mrd.h "Domain decomposition") ----
    PHASE_RESIDUAL1, PHASE_UPDATE1, PHASE_STAGE2, PHASE_END = 0, 1, 2, 3

    def halo_set(self, send_idx, recv_idx):
        si = np.ascontiguousarray(send_idx, dtype=np.int32)
        ri = np.ascontiguousarray(recv_idx, dtype=np.int32)
        _check(lib().mrd_halo_set(self._h, len(si), _np_ptr(si, C.c_int32), len(ri), _np_ptr(ri, C.c_int32)))
        self.n_send, self.n_recv = len(si), len(ri)

    def phase_begin(self, t_end=0.0, stream=None):
        _check(lib().mrd_phase_begin(self._h, float(t_end), _stream_ptr(stream)))

    def phase(self, k, stream=None):
        _check(lib().mrd_phase(self._h, int(k), _stream_ptr(stream)))

    def phase_end(self, stream=None):
        n, t, dt = C.c_int64(0), C.c_double(0.0), C.c_double(0.0)
        _check(lib().mrd_phase_end(self._h, _stream_ptr(stream), C.byref(n), C.byref(t), C.byref(dt)))
        return n.value, t.value, dt.value

    def _check_buf(self, buf, rows, dtype):
        t = self._torch
        assert isinstance(buf, t.Tensor) and buf.is_cuda and buf.dtype == dtype and buf.is_contiguous()
        assert buf.numel() == rows, (buf.numel(), rows)

    def dt_get(self, d, stream=None):
        self._check_buf(d, 2, self._torch.float64)
        _check(lib().mrd_dt_get(self._h, C.c_void_p(d.data_ptr()), _stream_ptr(stream)))

    def dt_set(self, d, stream=None):
        self._check_buf(d, 2, self._torch.float64)
        _check(lib().mrd_dt_set(self._h, C.c_void_p(d.data_ptr()), _stream_ptr(stream)))

    def status_get(self, d, stream=None):
        self._check_buf(d, 1, self._torch.float64)
        _check(lib().mrd_status_get(self._h, C.c_void_p(d.data_ptr()), _stream_ptr(stream)))

    def status_set(self, d, stream=None):
        self._check_buf(d, 1, self._torch.float64)
        _check(lib().mrd_status_set(self._h, C.c_void_p(d.data_ptr()), _stream_ptr(stream)))

    def range_get(self, stage, d, stream=None):
        self._check_buf(d, 2, self._torch.float64)
        _check(lib().mrd_range_get(self._h, int(stage), C.c_void_p(d.data_ptr()), _stream_ptr(stream)))

    def range_set(self, stage, d, stream=None):
        self._check_buf(d, 2, self._torch.float64)
        _check(lib().mrd_range_set(self._h, int(stage), C.c_void_p(d.data_ptr()), _stream_ptr(stream)))

    def halo_pack(self, buf, stream=None):
        self._check_buf(buf, 4 * self.n_send, self.dtype)
        _check(lib().mrd_halo_pack(self._h, C.c_void_p(buf.data_ptr()), _stream_ptr(stream)))

    def halo_unpack(self, buf, stream=None):
        self._check_buf(buf, 4 * self.n_recv, self.dtype)
        _check(lib().mrd_halo_unpack(self._h, C.c_void_p(buf.data_ptr()), _stream_ptr(stream)))

    PROFILE_SLOTS = ("tri_stage1", "gather_dt", "wall1", "update", "tri_stage2", "wall2", "gather_update", "ctl")

    def step_profile(self, stream=None):
        """One step with per-kernel CUDA-event timing: dict slot name -> ms."""
        ms = (C.c_float * 8)()
        _check(lib().mrd_step_profile(self._h, _stream_ptr(stream), ms))
        return dict(zip(self.PROFILE_SLOTS, [float(x) for x in ms]))

    def launch_count(self) -> int:
        n = C.c_int64()
        _check(lib().mrd_launch_count(self._h, C.byref(n)))
        return n.value


def measure_peaks(stream=None):
    """(fp64 TFLOP/s, fp32 TFLOP/s, copy GB/s) micro-benchmarks of the current device."""
    a, b, c = C.c_double(), C.c_double(), C.c_double()
    _check(lib().mrd_measure_peaks(C.byref(a), C.byref(b), C.byref(c), _stream_ptr(stream)))
    return a.value, b.value, c.value


# ---- mesh generation, first slice (include/mrd.h "Mesh generation"): torch CUDA tensors in, torch CUDA tensors out ----
def meshgen_test_quality(xy, tri, R, B, stream=None):
    """xy float64 [nv][2], tri int32 [nt][3] (CUDA tensors) -> dict(r, beta, cc, bad, n_bad)."""
    import torch
    assert xy.is_cuda and xy.dtype == torch.float64 and xy.is_contiguous() and tri.is_cuda and tri.dtype == torch.int32 and tri.is_contiguous()
    nt = tri.shape[0]
    r = torch.empty(nt, dtype=torch.float64, device="cuda")
    beta = torch.empty(nt, dtype=torch.float64, device="cuda")
    cc = torch.empty((nt, 2), dtype=torch.float64, device="cuda")
    bad = torch.empty(nt, dtype=torch.uint8, device="cuda")
    n_bad = C.c_int64(0)
    _check(lib().mrd_meshgen_test_quality(nt, C.c_void_p(xy.data_ptr()), C.c_void_p(tri.data_ptr()), float(R), float(B),
                                          C.c_void_p(r.data_ptr()), C.c_void_p(beta.data_ptr()), C.c_void_p(cc.data_ptr()),
                                          C.c_void_p(bad.data_ptr()), C.byref(n_bad), _stream_ptr(stream)))
    return dict(r=r, beta=beta, cc=cc, bad=bad, n_bad=n_bad.value)


def _meshgen_predicate(fn, width, xy, idx, stream):
    import torch
    assert xy.is_cuda and xy.dtype == torch.float64 and xy.is_contiguous()
    assert idx.is_cuda and idx.dtype == torch.int32 and idx.is_contiguous() and idx.shape[1] == width
    sign = torch.empty(idx.shape[0], dtype=torch.int8, device="cuda")
    n_exact = C.c_int64(0)
    _check(fn(idx.shape[0], C.c_void_p(xy.data_ptr()), C.c_void_p(idx.data_ptr()), C.c_void_p(sign.data_ptr()), C.byref(n_exact),
              _stream_ptr(stream)))
    return sign, n_exact.value


def meshgen_orient2d(xy, idx, stream=None):
    """Exact sign of eq. 3 for every row (a, b, c) of idx: (int8 tensor, number of tests that took the exact path)."""
    return _meshgen_predicate(lib().mrd_meshgen_orient2d, 3, xy, idx, stream)


def meshgen_incircle2d(xy, idx, stream=None):
    """Exact sign of eq. 5 for every row (a, b, c, d) of idx."""
    return _meshgen_predicate(lib().mrd_meshgen_incircle2d, 4, xy, idx, stream)


def _dev(t, dtype, cols):
    import torch
    assert t.is_cuda and t.dtype == dtype and t.is_contiguous() and t.ndim == 2 and t.shape[1] == cols, (t.dtype, t.shape)
    return C.c_void_p(t.data_ptr())


def meshgen_build_edges(tv, stream=None):
    """triangleEdges te int32 [nt][3] and edgeTriangles et int32 [ne][2] (section 4.1.2) from triangleVertices tv (CUDA tensor)."""
    import torch
    nt = tv.shape[0]
    te = torch.empty((nt, 3), dtype=torch.int32, device="cuda")
    et = torch.empty((3 * nt, 2), dtype=torch.int32, device="cuda")
    ne = C.c_int64(0)
    _check(lib().mrd_meshgen_build_edges(nt, _dev(tv, torch.int32, 3), C.c_void_p(te.data_ptr()), C.c_void_p(et.data_ptr()),
                                         C.byref(ne), _stream_ptr(stream)))
    return te, et[:ne.value].clone()


def meshgen_delaunay_flip(xy, tv, te, et, stream=None):
    """Flip (tv, te, et) IN PLACE to the Delaunay triangulation of xy; returns dict(flips, iterations, exact)."""
    import torch
    f, it, ex = C.c_int64(0), C.c_int64(0), C.c_int64(0)
    _check(lib().mrd_meshgen_delaunay_flip(tv.shape[0], et.shape[0], _dev(xy, torch.float64, 2), _dev(tv, torch.int32, 3),
                                           _dev(te, torch.int32, 3), _dev(et, torch.int32, 2), C.byref(f), C.byref(it), C.byref(ex),
                                           _stream_ptr(stream)))
    return dict(flips=f.value, iterations=it.value, exact=ex.value)


def meshgen_find_triangle(xy, tv, te, et, p, t0, stream=None):
    """For every point p[i] the containing triangle, walking from t0[i]: (t int32 [n], code int8 [n]); see include/mrd.h."""
    import torch
    n = p.shape[0]
    assert t0.is_cuda and t0.dtype == torch.int32 and t0.is_contiguous() and t0.shape == (n,)
    t = torch.empty(n, dtype=torch.int32, device="cuda")
    code = torch.empty(n, dtype=torch.int8, device="cuda")
    _check(lib().mrd_meshgen_find_triangle(n, _dev(p, torch.float64, 2), C.c_void_p(t0.data_ptr()), tv.shape[0], _dev(xy, torch.float64, 2),
                                           _dev(tv, torch.int32, 3), _dev(te, torch.int32, 3), _dev(et, torch.int32, 2),
                                           C.c_void_p(t.data_ptr()), C.c_void_p(code.data_ptr()), _stream_ptr(stream)))
    return t, code


def meshgen_release():
    """Free the work space the mrd_meshgen_* calls keep between calls."""
    _check(lib().mrd_meshgen_release())


def meshgen_refine(xy, tv, te, et, R, B, seed=0, first_iteration=0, max_iterations=10 ** 6, cap_vertex=None, box=None, size=None,
                   stream=None):
    """Delaunay refinement (include/mrd.h: mrd_meshgen_refine) of the Delaunay triangulation (xy, tv, te, et) (CUDA tensors).
    Returns (xy, tv, te, et, info) as new tensors trimmed to the refined mesh; info: iterations, bad_left.  cap_vertex bounds
    the refined mesh (default 8 x the input + 1024); MrdError(MRD_ENOMEM) when it does not suffice -- its attribute `partial` is
    the valid, partly refined mesh (same tuple as the return value), to go on from with a larger cap_vertex (and, with box,
    first_iteration = first_iteration + partial[4]["iterations"] for the same mesh as an uninterrupted run).  box = (x0, y0, x1, y1):
    renumber the vertices along the Morton curve of that rectangle after every insertion step.  size = (grid, rectangle): the
    size bound is R times the bilinear interpolant of grid (float64 CUDA tensor [ny][nx], > 0) over rectangle = (x0, y0, x1, y1)."""
    import torch
    nv, nt, ne = xy.shape[0], tv.shape[0], et.shape[0]
    cv = int(cap_vertex) if cap_vertex else 8 * nv + 1024
    ct = 2 * cv                                       # a triangulated disc has fewer than 2 V triangles and 3 V edges
    ce = 3 * ct
    big = [torch.empty((cv, 2), dtype=torch.float64, device="cuda"), torch.empty((ct, 3), dtype=torch.int32, device="cuda"),
           torch.empty((ct, 3), dtype=torch.int32, device="cuda"), torch.empty((ce, 2), dtype=torch.int32, device="cuda")]
    for dst, src in zip(big, (xy, tv, te, et)):
        dst[:src.shape[0]].copy_(src)
    n = [C.c_int64(nv), C.c_int64(nt), C.c_int64(ne)]
    it, left = C.c_int64(0), C.c_int64(0)
    hbox = None if box is None else (C.c_double * 4)(*[float(v) for v in box])
    sgrid, sbox, snx, sny = None, None, 0, 0
    if size is not None:
        g = size[0]
        assert g.is_cuda and g.dtype == torch.float64 and g.is_contiguous() and g.ndim == 2
        sgrid, sbox, sny, snx = C.c_void_p(g.data_ptr()), (C.c_double * 4)(*[float(v) for v in size[1]]), g.shape[0], g.shape[1]
    rc = lib().mrd_meshgen_refine(float(R), float(B), int(seed) & 0xFFFFFFFF, int(first_iteration), int(max_iterations), hbox,
                                  sgrid, sbox, snx, sny, cv, ct, ce,
                                  C.byref(n[0]), C.byref(n[1]), C.byref(n[2]), *[C.c_void_p(t.data_ptr()) for t in big],
                                  C.byref(it), C.byref(left), _stream_ptr(stream))
    if rc == MRD_ENOMEM:                              # the arrays hold a valid, partly refined Delaunay mesh: hand it to the caller
        err = MrdError(rc, lib().mrd_last_error().decode())
        out = [t[:k.value].clone() for t, k in zip(big, (n[0], n[1], n[1], n[2]))]
        err.partial = (*out, dict(iterations=it.value, bad_left=left.value))
        raise err
    _check(rc)
    out = [t[:k.value].clone() for t, k in zip(big, (n[0], n[1], n[1], n[2]))]
    return (*out, dict(iterations=it.value, bad_left=left.value))


MESHGEN_STATIC_MAX_TESTS = 1 << 20
MESHGEN_PRIORITY_REGULAR = 0xFFFFFFFF    # seed value of meshgen_refine: regular instead of random priorities (Fig. 8 of the paper)


def meshgen_orient2d_static(xy, idx, sign, n_exact=None, stream=None):
    """mrd_meshgen_orient2d_static: the exact sign of eq. 3 for every row (a, b, c) of idx into the caller's `sign` (int8 CUDA
    tensor [n]) -- no allocation anywhere (the scratch is a static device array of the library; at most 2^20 tests per call),
    no synchronisation.  n_exact: optional int64 CUDA tensor [1] that receives the number of tests that took the exact path.
    Calls that overlap on the GPU race (include/mrd.h)."""
    import torch
    n = idx.shape[0]
    assert xy.is_cuda and xy.dtype == torch.float64 and xy.is_contiguous()
    assert idx.is_cuda and idx.dtype == torch.int32 and idx.is_contiguous() and idx.ndim == 2 and idx.shape[1] == 3
    assert sign.is_cuda and sign.dtype == torch.int8 and sign.is_contiguous() and sign.shape == (n,)
    assert n_exact is None or (n_exact.is_cuda and n_exact.dtype == torch.int64 and n_exact.numel() == 1)
    _check(lib().mrd_meshgen_orient2d_static(n, C.c_void_p(xy.data_ptr()), C.c_void_p(idx.data_ptr()), C.c_void_p(sign.data_ptr()),
                                             None if n_exact is None else C.c_void_p(n_exact.data_ptr()), _stream_ptr(stream)))


def meshgen_flip_stats(reset=False):
    """dict(cooperative_launches, cooperative_iterations, handed_back, launched_iterations) of the flip loops since the last reset."""
    out = (C.c_int64 * 4)()
    _check(lib().mrd_meshgen_flip_stats(out, 1 if reset else 0))
    return dict(zip(("cooperative_launches", "cooperative_iterations", "handed_back", "launched_iterations"), [int(v) for v in out]))
