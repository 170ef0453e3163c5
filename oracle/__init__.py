"""Python (ctypes) face of the CPU ORACLE -- test infrastructure, NOT the product.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this package.  It loads `oracle/libmrd_oracle.so` (built by `oracle/build.py`
from `mrd_oracle.cpp`) and never touches the CUDA path.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

ORC_OK, ORC_EINVAL, ORC_ENOMEM, ORC_ENONPHYSICAL = 0, -1, -2, -4
SCHEME_N, SCHEME_LDA, SCHEME_B, SCHEME_BMAX, SCHEME_BMIN, SCHEME_BX = 0, 1, 2, 3, 4, 5

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int32)
        L.orc_mesh_create.argtypes = [C.POINTER(C.c_void_p), C.c_double, C.c_double, C.c_int, C.c_int, C.c_double,
                                      C.c_double, C.c_int64, dp, C.c_int64, ip, C.POINTER(C.c_uint8), C.c_int64, ip]
        L.orc_mesh_destroy.argtypes = [C.c_void_p]
        L.orc_mesh_destroy.restype = None
        L.orc_set_num_threads.argtypes = [C.c_void_p, C.c_int]
        L.orc_set_lumping.argtypes = [C.c_void_p, C.c_int]
        L.orc_triangle_stage2_lumping.argtypes = [C.c_int]
        L.orc_triangle_stage2_lumping.restype = None
        L.orc_set_state.argtypes = [C.c_void_p, dp]
        L.orc_get_state.argtypes = [C.c_void_p, dp]
        L.orc_step.argtypes = [C.c_void_p, C.c_int64, C.c_double, C.POINTER(C.c_int64), dp, dp]
        L.orc_get_diagnostics.argtypes = [C.c_void_p, dp, dp, dp]
        L.orc_get_geometry.argtypes = [C.c_void_p, dp, dp]
        L.orc_dump_stage1.argtypes = [C.c_void_p, dp, dp, dp, dp, dp]
        L.orc_euler_matrices.argtypes = [C.c_double] * 7 + [dp, dp, dp]
        L.orc_euler_matrices.restype = None
        L.orc_euler_matrices_l.argtypes = [C.c_double] * 9 + [dp]
        L.orc_euler_matrices_l.restype = None
        L.orc_eigenvectors.argtypes = [C.c_double] * 6 + [dp, dp, dp]
        L.orc_eigenvectors.restype = None
        L.orc_triangle_stage1.argtypes = [C.c_double] + [dp] * 10
        L.orc_triangle_stage2.argtypes = [C.c_double, dp, dp, dp, C.c_double] + [dp] * 6
        L.orc_wall_edge.argtypes = [C.c_double, dp, dp, C.c_double, C.c_double, C.c_double, dp, dp]
        L.orc_wall_edge.restype = None
        L.orc_count_ops.argtypes = [C.c_double, dp, dp, C.c_int, C.c_int, C.POINTER(C.c_int64)]
        L.orc_last_error.restype = C.c_char_p
        _lib = L
    return _lib


class OracleError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"oracle error {code}: {msg}")
        self.code = code


def _check(rc):
    if rc != 0:
        raise OracleError(rc, lib().orc_last_error().decode())


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def _f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        assert a.shape == shape, (a.shape, shape)
    return a


class OracleMesh:
    """The oracle's mesh + stepper."""

    def __init__(self, xy, tri, gamma=1.4, cfl=0.5, scheme=SCHEME_B, time_order=2, period=(0.0, 0.0),
                 vertex_flag=None, wall_edge=None, threads=1, lumping=0):
        L = lib()
        self._xy = _f64(xy)
        self._tri = np.ascontiguousarray(tri, dtype=np.int32)
        self.nv, self.nt = self._xy.shape[0], self._tri.shape[0]
        flag = None if vertex_flag is None else np.ascontiguousarray(vertex_flag, dtype=np.uint8)
        wedge = None if wall_edge is None else np.ascontiguousarray(wall_edge, dtype=np.int32)
        ne = 0 if wedge is None else wedge.shape[0]
        h = C.c_void_p()
        _check(L.orc_mesh_create(C.byref(h), gamma, cfl, scheme, time_order, period[0], period[1], self.nv,
                                 _dp(self._xy), self.nt, self._tri.ctypes.data_as(C.POINTER(C.c_int32)),
                                 None if flag is None else flag.ctypes.data_as(C.POINTER(C.c_uint8)), ne,
                                 None if wedge is None else wedge.ctypes.data_as(C.POINTER(C.c_int32))))
        self._h = h
        self.gamma = gamma
        if threads != 1:
            self.set_threads(threads)
        if lumping:
            _check(L.orc_set_lumping(self._h, int(lumping)))

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h and lib is not None:      # (module globals are already gone at interpreter shutdown)
            lib().orc_mesh_destroy(h)

    def set_threads(self, n):
        _check(lib().orc_set_num_threads(self._h, int(n)))

    def set_state(self, W):
        W = _f64(W, (4, self.nv))
        _check(lib().orc_set_state(self._h, _dp(W)))

    def get_state(self):
        W = np.empty((4, self.nv))
        _check(lib().orc_get_state(self._h, _dp(W)))
        return W

    def step(self, max_steps=1, t_end=0.0):
        n, t, dt = C.c_int64(0), C.c_double(0.0), C.c_double(0.0)
        _check(lib().orc_step(self._h, int(max_steps), float(t_end), C.byref(n), C.byref(t), C.byref(dt)))
        return n.value, t.value, dt.value

    def diagnostics(self):
        tot = np.empty(4)
        mr, mp = C.c_double(), C.c_double()
        _check(lib().orc_get_diagnostics(self._h, _dp(tot), C.byref(mr), C.byref(mp)))
        return tot, mr.value, mp.value

    def geometry(self):
        area, vol = np.empty(self.nt), np.empty(self.nv)
        _check(lib().orc_get_geometry(self._h, _dp(area), _dp(vol)))
        return area, vol

    def dump_stage1(self):
        nt = self.nt
        out = dict(phiT=np.empty((nt, 4)), phiN=np.empty((nt, 3, 4)), phiLDA=np.empty((nt, 3, 4)),
                   phiB=np.empty((nt, 3, 4)), sT=np.empty(nt))
        _check(lib().orc_dump_stage1(self._h, _dp(out["phiT"]), _dp(out["phiN"]), _dp(out["phiLDA"]),
                                     _dp(out["phiB"]), _dp(out["sT"])))
        return out


def euler_matrices(gamma, u, v, h, nx, ny, length):
    K, Kp, Km = np.empty((4, 4)), np.empty((4, 4)), np.empty((4, 4))
    lib().orc_euler_matrices(gamma, u, v, h, nx, ny, length, _dp(K), _dp(Kp), _dp(Km))
    return K, Kp, Km


def euler_matrices_l(gamma, u, v, h, nx, ny, l1, l2, l3):
    K = np.empty((4, 4))
    lib().orc_euler_matrices_l(gamma, u, v, h, nx, ny, l1, l2, l3, _dp(K))
    return K


def eigenvectors(gamma, u, v, h, nx, ny):
    R, Ri, lam = np.empty((4, 4)), np.empty((4, 4)), np.empty(4)
    lib().orc_eigenvectors(gamma, u, v, h, nx, ny, _dp(R), _dp(Ri), _dp(lam))
    return R, Ri, lam


def triangle_stage1(gamma, W, xy):
    W, xy = _f64(W, (3, 4)), _f64(xy, (3, 2))
    o = dict(phiT=np.empty(4), phiN=np.empty((3, 4)), phiLDA=np.empty((3, 4)), phiB=np.empty((3, 4)),
             theta=np.empty(4), sT=np.empty(1), Nhat=np.empty((4, 4)), sumKm=np.empty((4, 4)))
    _check(lib().orc_triangle_stage1(gamma, _dp(W), _dp(xy), _dp(o["phiT"]), _dp(o["phiN"]), _dp(o["phiLDA"]),
                                     _dp(o["phiB"]), _dp(o["theta"]), _dp(o["sT"]), _dp(o["Nhat"]), _dp(o["sumKm"])))
    o["sT"] = float(o["sT"][0])
    return o


def triangle_stage2(gamma, Wn, Ws, xy, dt, phiT_n, phiN_n, lumping=0):
    lib().orc_triangle_stage2_lumping(int(lumping))
    Wn, Ws, xy = _f64(Wn, (3, 4)), _f64(Ws, (3, 4)), _f64(xy, (3, 2))
    pT, pN = _f64(phiT_n, (4,)), _f64(phiN_n, (3, 4))
    o = dict(PhiT=np.empty(4), PhiN=np.empty((3, 4)), PhiLDA=np.empty((3, 4)), PhiB=np.empty((3, 4)))
    _check(lib().orc_triangle_stage2(gamma, _dp(Wn), _dp(Ws), _dp(xy), float(dt), _dp(pT), _dp(pN), _dp(o["PhiT"]),
                                     _dp(o["PhiN"]), _dp(o["PhiLDA"]), _dp(o["PhiB"])))
    return o


def wall_edge(gamma, Wa, Wb, nx, ny, length):
    Wa, Wb = _f64(Wa, (4,)), _f64(Wb, (4,))
    Pa, Pb = np.empty(4), np.empty(4)
    lib().orc_wall_edge(gamma, _dp(Wa), _dp(Wb), nx, ny, length, _dp(Pa), _dp(Pb))
    return Pa, Pb


def count_ops(gamma, W, xy, stage=1, scheme=SCHEME_B):
    W, xy = _f64(W, (3, 4)), _f64(xy, (3, 2))
    c = (C.c_int64 * 6)()
    _check(lib().orc_count_ops(gamma, _dp(W), _dp(xy), stage, scheme, c))
    return dict(zip(("add", "mul", "div", "sqrt", "abs", "cmp"), [int(x) for x in c]))
