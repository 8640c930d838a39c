"""ctypes front-end of oracle/libjenga_oracle.so -- TEST INFRASTRUCTURE (see jenga_oracle.c).

Only tests/, bench.py's cpu_baseline / --impl reference legs and
__graft_entry__.smoke() may import this.  It never imports the CUDA package's binding.
Arrays cross as fp64 AoS; `unpack_tiles` widens the fp32 SoA tiles of include/jenga.h.
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

c_dp = C.POINTER(C.c_double)
c_ip = C.POINTER(C.c_int32)
c_up = C.POINTER(C.c_uint32)


class OrcParams(C.Structure):
    _fields_ = [("dt", C.c_double), ("g", C.c_double * 3), ("restitution", C.c_double),
                ("aabb_margin", C.c_double), ("beta", C.c_double), ("slop", C.c_double),
                ("edge_bias_rel", C.c_double), ("edge_bias_abs", C.c_double), ("par_eps", C.c_double),
                ("tie_eps", C.c_double), ("match_tol", C.c_double),
                ("n_substeps", C.c_int32), ("pgs_iters", C.c_int32), ("warm_start", C.c_int32),
                ("gyroscopic", C.c_int32), ("max_pairs", C.c_int32), ("max_contacts", C.c_int32)]


class OrcContacts(C.Structure):
    _fields_ = [("n", C.c_int32), ("pair", c_ip), ("slot", c_ip), ("axis", c_ip),
                ("nrm", c_dp), ("pt", c_dp), ("depth", c_dp)]


class OrcCache(C.Structure):
    _fields_ = [("n_pairs", C.c_int32), ("key_pair", c_ip), ("key_meta", c_ip), ("lam", c_dp), ("pt", c_dp)]


class OrcMargins(C.Structure):
    _fields_ = [("aabb", C.c_double), ("sat_sign", C.c_double), ("axis_choice", C.c_double),
                ("incident", C.c_double), ("clip", C.c_double), ("reduce", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}

    def reset(self):
        for k, _ in self._fields_:
            setattr(self, k, 1e300)


class OrcTrace(C.Structure):
    _fields_ = [("pairs", c_ip), ("n_pairs", c_ip), ("contacts", C.POINTER(OrcContacts)),
                ("lam", c_dp), ("colour", c_ip), ("v_pre", c_dp), ("w_pre", c_dp),
                ("margins", C.POINTER(OrcMargins))]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_ziglar_force.restype = C.c_double
        _lib.orc_ziglar_force.argtypes = [C.c_double] * 4
        _lib.orc_pair_index.restype = C.c_int32
        _lib.orc_broadphase.restype = C.c_int32
        _lib.orc_collide_boxes.restype = C.c_int32
        _lib.orc_collide_ground.restype = C.c_int32
        _lib.orc_narrowphase.restype = C.c_int32
        _lib.orc_colour_pairs.restype = C.c_int32
        _lib.orc_step_env.restype = C.c_uint32
        _lib.orc_collapse_test.restype = C.c_int32
        _lib.orc_max_threads.restype = C.c_int32
        _lib.orc_support_margin.restype = C.c_double
        _lib.orc_ziglar_block_analysis.restype = C.c_int32
    return _lib


def dp(a):
    return a.ctypes.data_as(c_dp)


def ip(a):
    return a.ctypes.data_as(c_ip)


def make_params(wp) -> OrcParams:
    """wp: workloads.WorldParams (floats already fp32-representable)."""
    p = OrcParams()
    p.dt = wp.dt
    p.g[:] = list(wp.gravity)
    p.restitution = wp.restitution
    p.aabb_margin = wp.aabb_margin
    p.beta, p.slop = wp.baumgarte_beta, wp.slop
    p.edge_bias_rel, p.edge_bias_abs, p.par_eps, p.tie_eps = wp.edge_bias_rel, wp.edge_bias_abs, wp.par_eps, wp.tie_eps
    p.match_tol = wp.match_tol
    p.n_substeps, p.pgs_iters, p.warm_start, p.gyroscopic = wp.n_substeps, wp.pgs_iters, wp.warm_start, wp.gyroscopic
    p.max_pairs, p.max_contacts = wp.max_pairs, wp.max_contacts
    return p


class Bodies:
    """fp64 AoS view of E envs x B bodies."""

    def __init__(self, x, q, v, w, inv_m, inv_I, he, active):
        self.x, self.q, self.v, self.w = x, q, v, w
        self.inv_m, self.inv_I, self.he, self.active = inv_m, inv_I, he, active
        self.E, self.B = x.shape[0], x.shape[1]

    def copy(self):
        return Bodies(*(a.copy() for a in (self.x, self.q, self.v, self.w, self.inv_m, self.inv_I, self.he, self.active)))

    def env(self, e):
        return Bodies(*(a[e:e + 1] for a in (self.x, self.q, self.v, self.w, self.inv_m, self.inv_I, self.he, self.active)))


def unpack_tiles(state, props, n_bodies) -> Bodies:
    """[E][13][S], [E][8][S] fp32 tiles -> contiguous fp64 AoS arrays (exact widening)."""
    B = n_bodies
    s = np.asarray(state, dtype=np.float64)
    p = np.asarray(props, dtype=np.float64)
    tr = lambda a: np.ascontiguousarray(np.transpose(a, (0, 2, 1)))
    return Bodies(tr(s[:, 0:3, :B]), tr(s[:, 3:7, :B]), tr(s[:, 7:10, :B]), tr(s[:, 10:13, :B]),
                  np.ascontiguousarray(p[:, 0, :B]), tr(p[:, 1:4, :B]), tr(p[:, 4:7, :B]),
                  np.ascontiguousarray(p[:, 7, :B] != 0).astype(np.int32))


def pack_state(bod: Bodies, stride: int) -> np.ndarray:
    """fp64 [E][13][S] tile from the AoS arrays (for comparing with the GPU state)."""
    E, B = bod.E, bod.B
    s = np.zeros((E, 13, stride))
    s[:, 3, :] = 1.0
    s[:, 0:3, :B] = np.transpose(bod.x, (0, 2, 1))
    s[:, 3:7, :B] = np.transpose(bod.q, (0, 2, 1))
    s[:, 7:10, :B] = np.transpose(bod.v, (0, 2, 1))
    s[:, 10:13, :B] = np.transpose(bod.w, (0, 2, 1))
    return s


def unpack_fext(fext, n_bodies):
    if fext is None:
        return None
    f = np.asarray(fext, dtype=np.float64)
    return np.ascontiguousarray(np.transpose(f[:, :, :n_bodies], (0, 2, 1)))


class Contacts:
    def __init__(self, cap):
        self.cap = cap
        self.pair = np.zeros(cap, np.int32); self.slot = np.zeros(cap, np.int32); self.axis = np.zeros(cap, np.int32)
        self.nrm = np.zeros((cap, 3)); self.pt = np.zeros((cap, 3)); self.depth = np.zeros(cap)
        self.c = OrcContacts(0, ip(self.pair), ip(self.slot), ip(self.axis), dp(self.nrm), dp(self.pt), dp(self.depth))

    @property
    def n(self):
        return self.c.n

    def trimmed(self):
        n = self.n
        return dict(pair=self.pair[:n].copy(), slot=self.slot[:n].copy(), axis=self.axis[:n].copy(),
                    nrm=self.nrm[:n].copy(), pt=self.pt[:n].copy(), depth=self.depth[:n].copy())

    @staticmethod
    def from_arrays(pair, slot, axis, nrm, pt, depth):
        c = Contacts(max(1, len(pair)))
        n = len(pair)
        c.pair[:n], c.slot[:n], c.axis[:n] = pair, slot, axis
        c.nrm[:n], c.pt[:n], c.depth[:n] = nrm, pt, depth
        c.c.n = n
        return c


class Cache:
    """warm-start cache of E envs (persisting between step calls)."""

    def __init__(self, E, max_contacts):
        self.pc = max(1, max_contacts // 4)
        self.key_pair = np.zeros((E, self.pc), np.int32)
        self.key_meta = np.zeros((E, self.pc), np.int32)
        self.n_keys = np.zeros(E, np.int32)
        self.lam = np.zeros((E, self.pc, 4, 3))
        self.pt = np.zeros((E, self.pc, 4, 3))

    def env_struct(self, e):
        return OrcCache(int(self.n_keys[e]), ip(self.key_pair[e]), ip(self.key_meta[e]), dp(self.lam[e]), dp(self.pt[e]))


def inertia_box(m, l, w, h):
    out = np.zeros(3)
    lib().orc_inertia_box(C.c_double(m), C.c_double(l), C.c_double(w), C.c_double(h), dp(out))
    return out


def quat_to_R(q):
    q = np.ascontiguousarray(q, dtype=np.float64); R = np.zeros(9)
    lib().orc_quat_to_R(dp(q), dp(R))
    return R.reshape(3, 3)


def ziglar_force(k, mu, m, g=9.81):
    return lib().orc_ziglar_force(k, mu, m, g)


def pair_index(B, i, j):
    return lib().orc_pair_index(C.c_int32(B), C.c_int32(i), C.c_int32(j))


def pair_bodies(B, idx):
    i, j = C.c_int32(), C.c_int32()
    lib().orc_pair_bodies(C.c_int32(B), C.c_int32(int(idx)), C.byref(i), C.byref(j))
    return i.value, j.value


def broadphase(P: OrcParams, bod: Bodies, e=0, margins=None):
    pairs = np.zeros(max(1, P.max_pairs), np.int32)
    status = C.c_uint32(0)
    n = lib().orc_broadphase(C.byref(P), C.c_int32(bod.B), dp(bod.x[e]), dp(bod.q[e]), dp(bod.he[e]), dp(bod.inv_m[e]),
                             ip(bod.active[e]), ip(pairs), C.byref(status), C.byref(margins) if margins is not None else None)
    return pairs[:n].copy(), status.value


def collide_boxes(P, xA, qA, hA, xB, qB, hB, margins=None):
    arr = [np.ascontiguousarray(a, dtype=np.float64) for a in (xA, qA, hA, xB, qB, hB)]
    axis = C.c_int32(-1); n = np.zeros(3); sd = C.c_double(0); pts = np.zeros((4, 3)); dep = np.zeros(4)
    k = lib().orc_collide_boxes(C.byref(P), *[dp(a) for a in arr], C.byref(axis), dp(n), C.byref(sd), dp(pts), dp(dep),
                                C.byref(margins) if margins is not None else None)
    return dict(npts=k, axis=axis.value, n=n, sat_depth=sd.value, pts=pts[:k].copy(), depths=dep[:k].copy())


def collide_ground(x, q, he, margins=None):
    arr = [np.ascontiguousarray(a, dtype=np.float64) for a in (x, q, he)]
    pts = np.zeros((4, 3)); dep = np.zeros(4)
    k = lib().orc_collide_ground(*[dp(a) for a in arr], dp(pts), dp(dep), C.byref(margins) if margins is not None else None)
    return dict(npts=k, pts=pts[:k].copy(), depths=dep[:k].copy())


def narrowphase(P, bod: Bodies, pairs, e=0, margins=None):
    pairs = np.ascontiguousarray(pairs, np.int32)
    cont = Contacts(max(4, P.max_contacts))
    status = C.c_uint32(0)
    lib().orc_narrowphase(C.byref(P), C.c_int32(bod.B), dp(bod.x[e]), dp(bod.q[e]), dp(bod.he[e]), ip(pairs),
                          C.c_int32(len(pairs)), C.byref(cont.c), C.byref(status),
                          C.byref(margins) if margins is not None else None)
    return cont, status.value


def colour_pairs(B, pair_idx, inv_m):
    pair_idx = np.ascontiguousarray(pair_idx, np.int32)
    col = np.zeros(max(1, len(pair_idx)), np.int32); status = C.c_uint32(0)
    inv_m = np.ascontiguousarray(inv_m, np.float64)
    nc = lib().orc_colour_pairs(C.c_int32(B), ip(pair_idx), C.c_int32(len(pair_idx)), dp(inv_m), ip(col), C.byref(status))
    return col[:len(pair_idx)], nc, status.value


def world_inv_inertia(bod: Bodies, e=0):
    Iw = np.zeros((bod.B, 9))
    lib().orc_world_inv_inertia(C.c_int32(bod.B), dp(bod.q[e]), dp(bod.inv_I[e]), dp(Iw))
    # inactive / static bodies contribute nothing
    Iw[(bod.active[e] == 0) | (bod.inv_m[e] == 0)] = 0.0
    return Iw


def solve(P, bod: Bodies, cont: Contacts, mu, e=0, cache: Cache = None, iters=None, perm=None):
    """S4+S5 on a given contact list; updates bod.v[e], bod.w[e] in place."""
    n = cont.n
    lam = np.zeros((max(1, n), 3)); col = np.zeros(max(1, n), np.int32); status = C.c_uint32(0)
    Iw = world_inv_inertia(bod, e)
    cs = cache.env_struct(e) if cache is not None else None
    pp = np.ascontiguousarray(perm, np.int32) if perm is not None else None
    lib().orc_solve(C.byref(P), C.c_int32(bod.B), dp(bod.x[e]), dp(bod.v[e]), dp(bod.w[e]), dp(bod.inv_m[e]), dp(Iw),
                    C.c_double(float(mu)), C.byref(cont.c), C.byref(cs) if cs is not None else None,
                    C.c_int32(P.pgs_iters if iters is None else iters), dp(lam), ip(col),
                    ip(pp) if pp is not None else None, C.byref(status))
    return lam[:n], col[:n], status.value


def step_env(P, bod: Bodies, mu, e=0, fext=None, cache: Cache = None, trace=False):
    """One dt advance of env e in place.  trace=True returns the last substep's stage outputs."""
    tr = None; keep = None
    if trace:
        pairs = np.zeros(max(1, P.max_pairs), np.int32); npairs = C.c_int32(0)
        cont = Contacts(max(4, P.max_contacts))
        lam = np.zeros((max(4, P.max_contacts), 3)); col = np.zeros(max(4, P.max_contacts), np.int32)
        v_pre = np.zeros((bod.B, 3)); w_pre = np.zeros((bod.B, 3)); mg = OrcMargins()
        tr = OrcTrace(ip(pairs), C.pointer(npairs), C.pointer(cont.c), dp(lam), ip(col), dp(v_pre), dp(w_pre), C.pointer(mg))
        keep = (pairs, npairs, cont, lam, col, v_pre, w_pre, mg)
    cs = cache.env_struct(e) if cache is not None else None
    f = dp(fext[e]) if fext is not None else None
    st = lib().orc_step_env(C.byref(P), C.c_int32(bod.B), dp(bod.x[e]), dp(bod.q[e]), dp(bod.v[e]), dp(bod.w[e]),
                            dp(bod.inv_m[e]), dp(bod.inv_I[e]), dp(bod.he[e]), ip(bod.active[e]), C.c_double(float(mu)),
                            f, C.byref(cs) if cs is not None else None, C.byref(tr) if tr is not None else None)
    if cache is not None:
        cache.n_keys[e] = cs.n_pairs
    if not trace:
        return st
    pairs, npairs, cont, lam, col, v_pre, w_pre, mg = keep
    n = cont.n
    return dict(status=st, pairs=pairs[:npairs.value].copy(), contacts=cont, lam=lam[:n].copy(), colour=col[:n].copy(),
                v_pre=v_pre, w_pre=w_pre, margins=mg.as_dict())


def rollout(P, bod: Bodies, mu, n_steps, fext=None, cache: Cache = None, x0=None, q0=None, length=0.075,
            collapsed=None, contact_count=None):
    """n_steps dt advances of every env in place (OpenMP over envs).  Returns status [E]."""
    E, B = bod.E, bod.B
    if cache is None:
        cache = Cache(E, P.max_contacts)
    status = np.zeros(E, np.uint32)
    mu = np.ascontiguousarray(mu, np.float64)
    lib().orc_rollout(C.byref(P), C.c_int32(E), C.c_int32(B), C.c_int32(n_steps), dp(bod.x), dp(bod.q), dp(bod.v), dp(bod.w),
                      dp(bod.inv_m), dp(bod.inv_I), dp(bod.he), ip(bod.active), dp(mu),
                      dp(fext) if fext is not None else None,
                      ip(cache.key_pair), ip(cache.key_meta), ip(cache.n_keys), dp(cache.lam), dp(cache.pt),
                      status.ctypes.data_as(c_up),
                      dp(x0) if x0 is not None else None, dp(q0) if q0 is not None else None, C.c_double(length),
                      ip(collapsed) if collapsed is not None else None,
                      contact_count.ctypes.data_as(C.POINTER(C.c_int64)) if contact_count is not None else None)
    return status


def rollout_until_rest(P, bod: Bodies, mu, max_steps=400, ek_rest=1e-7, cache: Cache = None):
    """per env, steps until E_k < ek_rest (checked after every step), at most max_steps.
    Returns (steps [E], E_k at exit [E], status [E])."""
    E, B = bod.E, bod.B
    if cache is None:
        cache = Cache(E, P.max_contacts)
    status = np.zeros(E, np.uint32); steps = np.zeros(E, np.int32); ek = np.zeros(E)
    mu = np.ascontiguousarray(mu, np.float64)
    lib().orc_rollout_until_rest(C.byref(P), C.c_int32(E), C.c_int32(B), C.c_int32(max_steps), C.c_double(ek_rest),
                                 dp(bod.x), dp(bod.q), dp(bod.v), dp(bod.w), dp(bod.inv_m), dp(bod.inv_I), dp(bod.he),
                                 ip(bod.active), dp(mu), ip(cache.key_pair), ip(cache.key_meta), ip(cache.n_keys),
                                 dp(cache.lam), dp(cache.pt), status.ctypes.data_as(c_up), ip(steps), dp(ek))
    return steps, ek, status


def collapse_test(bod: Bodies, x0, q0, e=0, length=0.075):
    out = np.zeros(3)
    r = lib().orc_collapse_test(C.c_int32(bod.B), dp(bod.x[e]), dp(bod.q[e]), dp(bod.v[e]), dp(bod.w[e]), dp(x0), dp(q0),
                                dp(bod.inv_m[e]), dp(bod.inv_I[e]), ip(bod.active[e]), C.c_double(length), dp(out))
    return bool(r), out


def support_margin(bod: Bodies, e=0, eps=0.002):
    """Eq. 17: (margin d, COM_xy, number of hull vertices) of env e."""
    com = np.zeros(2); nh = C.c_int32(0)
    d = lib().orc_support_margin(C.c_int32(bod.B), dp(bod.x[e]), dp(bod.q[e]), dp(bod.he[e]), dp(bod.inv_m[e]), ip(bod.active[e]),
                                 C.c_double(eps), dp(com), C.byref(nh))
    return d, com, nh.value


def ziglar_block_analysis(slot, axis, mu_s, m, g=9.81):
    """Table 1: (class 0 center_xaxis / 1 side_yaxis / 2 side_xaxis, F_min [N], torque flag)."""
    f = C.c_double(0); t = C.c_int32(0)
    c = lib().orc_ziglar_block_analysis(C.c_int32(slot), C.c_int32(axis), C.c_double(mu_s), C.c_double(m), C.c_double(g),
                                        C.byref(f), C.byref(t))
    return c, f.value, bool(t.value)


def n_threads():
    return lib().orc_max_threads()
