"""fp32 build of the oracle's own source -- TEST INFRASTRUCTURE, control experiment only.

oracle/libjenga_oracle32.so is jenga_oracle.c compiled with every floating-point variable in fp32 (same file, same
order of operations; see the ORC_REAL_FLOAT note in the source).  It is never a parity reference and the CUDA package
never loads it.  Its one use: the rollout-agreement study (tests/test_gpu_parity.py) asks whether the
collapse / no-collapse flips between the fp64 oracle and the fp32 CUDA path are what fp32 arithmetic alone produces, in
rate and in direction.  Only the rollout entry is exposed.
"""
from __future__ import annotations

import ctypes as C
import os
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, _HERE)
import build as _build  # noqa: E402

_lib = None
c_fp = C.POINTER(C.c_float)
c_ip = C.POINTER(C.c_int32)


class OrcParams32(C.Structure):
    _fields_ = [("dt", C.c_float), ("g", C.c_float * 3), ("restitution", C.c_float),
                ("aabb_margin", C.c_float), ("beta", C.c_float), ("slop", C.c_float),
                ("edge_bias_rel", C.c_float), ("edge_bias_abs", C.c_float), ("par_eps", C.c_float),
                ("tie_eps", C.c_float), ("match_tol", C.c_float),
                ("n_substeps", C.c_int32), ("pgs_iters", C.c_int32), ("warm_start", C.c_int32),
                ("gyroscopic", C.c_int32), ("max_pairs", C.c_int32), ("max_contacts", C.c_int32)]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build(bits=32))
    return _lib


def make_params(wp) -> OrcParams32:
    p = OrcParams32()
    p.dt = wp.dt
    p.g[:] = list(wp.gravity)
    p.restitution, p.aabb_margin = wp.restitution, wp.aabb_margin
    p.beta, p.slop = wp.baumgarte_beta, wp.slop
    p.edge_bias_rel, p.edge_bias_abs, p.par_eps, p.tie_eps = wp.edge_bias_rel, wp.edge_bias_abs, wp.par_eps, wp.tie_eps
    p.match_tol = wp.match_tol
    p.n_substeps, p.pgs_iters, p.warm_start, p.gyroscopic = wp.n_substeps, wp.pgs_iters, wp.warm_start, wp.gyroscopic
    p.max_pairs, p.max_contacts = wp.max_pairs, wp.max_contacts
    return p


def _fp(a):
    assert a.dtype == np.float32 and a.flags.c_contiguous
    return a.ctypes.data_as(c_fp)


def _ip(a):
    assert a.dtype == np.int32 and a.flags.c_contiguous
    return a.ctypes.data_as(c_ip)


class World32:
    """fp32 AoS copy of [E][13][S] / [E][8][S] tiles (the same fp32 inputs both other sides get) plus the warm-start cache."""

    def __init__(self, wp, state, props, mu):
        B = wp.n_bodies
        s, p = np.asarray(state, np.float32), np.asarray(props, np.float32)
        tr = lambda a: np.ascontiguousarray(np.transpose(a, (0, 2, 1)))
        self.wp, self.E, self.B = wp, s.shape[0], B
        self.x, self.q, self.v, self.w = tr(s[:, 0:3, :B]), tr(s[:, 3:7, :B]), tr(s[:, 7:10, :B]), tr(s[:, 10:13, :B])
        self.inv_m, self.inv_I, self.he = np.ascontiguousarray(p[:, 0, :B]), tr(p[:, 1:4, :B]), tr(p[:, 4:7, :B])
        self.active = np.ascontiguousarray(p[:, 7, :B] != 0).astype(np.int32)
        self.mu = np.ascontiguousarray(mu, np.float32)
        self.x0, self.q0 = self.x.copy(), self.q.copy()
        pc = max(1, wp.max_contacts // 4)
        self.key_pair = np.zeros((self.E, pc), np.int32); self.key_meta = np.zeros((self.E, pc), np.int32)
        self.n_keys = np.zeros(self.E, np.int32)
        self.lam = np.zeros((self.E, pc, 4, 3), np.float32); self.pt = np.zeros((self.E, pc, 4, 3), np.float32)
        self.status = np.zeros(self.E, np.uint32)
        self.collapsed = np.zeros(self.E, np.int32)
        self.P = make_params(wp)

    def rollout(self, n_steps, fext_tiles=None, length=0.075):
        """n_steps dt advances of every env (OpenMP over envs); Eq. 18 OR-latched into self.collapsed every step."""
        f = None
        if fext_tiles is not None:
            f = np.ascontiguousarray(np.transpose(np.asarray(fext_tiles, np.float32)[:, :, :self.B], (0, 2, 1)))
        lib().orc_rollout(C.byref(self.P), C.c_int32(self.E), C.c_int32(self.B), C.c_int32(int(n_steps)),
                          _fp(self.x), _fp(self.q), _fp(self.v), _fp(self.w), _fp(self.inv_m), _fp(self.inv_I), _fp(self.he),
                          _ip(self.active), _fp(self.mu), _fp(f) if f is not None else None,
                          _ip(self.key_pair), _ip(self.key_meta), _ip(self.n_keys), _fp(self.lam), _fp(self.pt),
                          self.status.ctypes.data_as(C.POINTER(C.c_uint32)), _fp(self.x0), _fp(self.q0), C.c_float(length),
                          _ip(self.collapsed), None)
