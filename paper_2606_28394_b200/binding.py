"""Thin Python binding of csrc/libjenga.so (include/jenga.h): argument marshalling only.

PyTorch allocates the device buffers and supplies the stream; every step of the method
runs inside the library's CUDA kernels.  There is no CPU fallback: if the library is
missing or the device is not a B200-class (sm_100) GPU the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "csrc", "libjenga.so")
_lib = None

N_COUNTERS = 12
COUNTER_NAMES = ("env_steps", "body_steps", "candidates", "colliding", "contacts", "contact_iters", "colours", "ground_contacts",
                 "max_candidates", "max_colliding", "max_colours", "reserved")
ST_PAIR_OVERFLOW, ST_CONTACT_OVERFLOW, ST_COLOUR_OVERFLOW, ST_NONFINITE = 1, 2, 4, 8
AXIS_GROUND = 15


class JengaError(RuntimeError):
    pass


class WorldDesc(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_envs", C.c_int32), ("n_bodies", C.c_int32), ("body_stride", C.c_int32),
                ("dt", C.c_float), ("n_substeps", C.c_int32), ("pgs_iters", C.c_int32), ("gravity", C.c_float * 3),
                ("restitution", C.c_float), ("aabb_margin", C.c_float), ("baumgarte_beta", C.c_float), ("slop", C.c_float),
                ("edge_bias_rel", C.c_float), ("edge_bias_abs", C.c_float), ("par_eps", C.c_float), ("tie_eps", C.c_float),
                ("match_tol", C.c_float), ("warm_start", C.c_int32), ("gyroscopic", C.c_int32), ("max_pairs", C.c_int32),
                ("max_contacts", C.c_int32), ("materialise", C.c_int32), ("device", C.c_int32),
                ("collapse_length", C.c_float), ("collapse_fd", C.c_float), ("collapse_ek", C.c_float), ("collapse_theta", C.c_float),
                ("solver_tier", C.c_int32), ("env_group", C.c_int32)]


class Buffers(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("state", "props", "mu", "f_ext", "pairs", "n_pairs", "contacts", "n_contacts",
                                          "lambda_", "cache_key", "cache_lam", "cache_pt", "n_cache", "status", "counters",
                                          "ref_pose", "collapsed", "collapse_stats", "rest_steps", "scratch")] + [("scratch_bytes", C.c_size_t)]


TIERS = {"auto": 0, "smem": 1, "tmem256": 2, "tmem512": 3, "tmem160": 4, "tmem128": 5}


def lib():
    """Load csrc/libjenga.so; build it first if it is absent and nvcc is here.  Raises if neither works."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            from . import build as _build
            try:
                _build.build()
            except Exception as exc:  # no silent fallback
                raise JengaError(f"libjenga.so is missing and could not be built: {exc}") from exc
        L = C.CDLL(_LIB_PATH)
        L.jenga_world_create.argtypes = [C.POINTER(WorldDesc), C.POINTER(Buffers), C.POINTER(C.c_void_p)]
        L.jenga_world_destroy.argtypes = [C.c_void_p]
        L.jenga_broadphase.argtypes = [C.c_void_p, C.c_void_p]
        L.jenga_narrowphase.argtypes = [C.c_void_p, C.c_void_p]
        L.jenga_pgs_solve.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.jenga_step.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.jenga_simulate_until_rest.argtypes = [C.c_void_p, C.c_int, C.c_float, C.c_void_p]
        L.jenga_set_f_ext.argtypes = [C.c_void_p, C.c_void_p]
        L.jenga_step_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        L.jenga_smem_bytes.argtypes = [C.POINTER(WorldDesc)]
        L.jenga_smem_bytes.restype = C.c_size_t
        L.jenga_block_threads.argtypes = [C.POINTER(WorldDesc)]
        L.jenga_env_group.argtypes = [C.POINTER(WorldDesc)]
        L.jenga_support_margin.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.jenga_ziglar_block_analysis.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.jenga_profile_enable.argtypes = [C.c_void_p, C.c_int]
        L.jenga_profile_read.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.jenga_scratch_bytes.argtypes = [C.POINTER(WorldDesc)]
        L.jenga_scratch_bytes.restype = C.c_size_t
        L.jenga_strerror.argtypes = [C.c_int]
        L.jenga_measure_peaks.argtypes = [C.POINTER(C.c_double), C.c_void_p, C.c_void_p]
        L.jenga_measure_peaks.restype = C.c_int
        L.jenga_peaks_scratch_bytes.restype = C.c_size_t
        L.jenga_strerror.restype = C.c_char_p
        L.jenga_narrowphase_static.argtypes = [C.POINTER(WorldDesc)] + [C.c_void_p] * 8
        L.jenga_narrowphase_static.restype = C.c_int
        L.jenga_narrowphase_static_env_bytes.argtypes = [C.POINTER(WorldDesc)]
        L.jenga_narrowphase_static_env_bytes.restype = C.c_size_t
        for f in ("jenga_world_create", "jenga_world_destroy", "jenga_broadphase", "jenga_narrowphase", "jenga_pgs_solve",
                  "jenga_step", "jenga_step_host", "jenga_simulate_until_rest", "jenga_set_f_ext", "jenga_block_threads", "jenga_env_group",
                  "jenga_profile_enable", "jenga_profile_read", "jenga_support_margin", "jenga_ziglar_block_analysis"):
            getattr(L, f).restype = C.c_int
        _lib = L
    return _lib


def _check(code: int, what: str):
    if code != 0:
        raise JengaError(f"{what} failed ({code}): {lib().jenga_strerror(code).decode()}")


def make_desc(wp, materialise: bool = False, device: int = 0, tier: str = "auto", group: int = 0) -> WorldDesc:
    """wp: any object with the fields of workloads.WorldParams."""
    d = WorldDesc()
    d.struct_size = C.sizeof(WorldDesc)
    d.n_envs, d.n_bodies, d.body_stride = wp.n_envs, wp.n_bodies, wp.body_stride
    d.dt, d.n_substeps, d.pgs_iters = wp.dt, wp.n_substeps, wp.pgs_iters
    d.gravity[:] = list(wp.gravity)
    d.restitution, d.aabb_margin = wp.restitution, wp.aabb_margin
    d.baumgarte_beta, d.slop = wp.baumgarte_beta, wp.slop
    d.edge_bias_rel, d.edge_bias_abs, d.par_eps, d.tie_eps = wp.edge_bias_rel, wp.edge_bias_abs, wp.par_eps, wp.tie_eps
    d.match_tol, d.warm_start, d.gyroscopic = wp.match_tol, wp.warm_start, wp.gyroscopic
    d.max_pairs, d.max_contacts = wp.max_pairs, wp.max_contacts
    d.materialise, d.device = int(materialise), device
    d.collapse_length = getattr(wp, "collapse_length", 0.0)
    d.collapse_fd, d.collapse_ek, d.collapse_theta = 0.5, 5.0e-5, 0.5235987755982988      # Eq. 18: f_d, eps_k [J], 30 deg
    d.solver_tier = TIERS[tier]
    d.env_group = int(group)
    return d


def jenga_measure_peaks(device: int = 0) -> dict:
    """FP32 issue rate and shared-memory bandwidth of the device, measured by the library's micro-benchmarks."""
    if not torch.cuda.is_available():
        raise JengaError("no CUDA device")
    L = lib()
    dev = torch.device("cuda", device)
    scratch = torch.empty(L.jenga_peaks_scratch_bytes(), dtype=torch.uint8, device=dev)
    out = (C.c_double * 8)()
    with torch.cuda.device(dev):
        _check(L.jenga_measure_peaks(out, C.c_void_p(scratch.data_ptr()), C.c_void_p(torch.cuda.current_stream(dev).cuda_stream)),
               "jenga_measure_peaks")
    return dict(fp32_instr_per_s=out[0], smem_bytes_per_s=out[1], n_sm=int(out[2]), ffma_s=out[3], lds_s=out[4], fp32_instr_per_s_3reg=out[5], fp32_instr_per_s_noreuse=out[6], fp32_fma_per_s_packed_noreuse=out[7])


STATIC_SCRATCH_BYTES = 8 << 20
E_STATIC_CAPACITY = -4


def jenga_narrowphase_static(desc: WorldDesc, state, props, pairs, n_pairs, contacts, n_contacts, status):
    """jenga_narrowphase for a caller that has no device memory to give the library as scratch (include/jenga.h).

    Every argument after `desc` is a CUDA tensor the caller already owns (inputs state, props, pairs, n_pairs; outputs
    contacts, n_contacts, status); this function only passes their addresses and torch's current stream on.  Neither it
    nor the library allocates: the kernel's hand-off area is an 8 MiB array inside libjenga.so (STATIC_SCRATCH_BYTES),
    one per device, shared by all calls -- so a batch must fit it (JengaError with code E_STATIC_CAPACITY otherwise;
    jenga_narrowphase_static_env_bytes(desc) is the share of one env) and calls on one device must not overlap in time.
    The first call on a device does a one-off set-up and belongs outside stream capture."""
    dev = state.device
    for t in (state, props, pairs, n_pairs, contacts, n_contacts, status):
        assert t.is_cuda and t.device == dev and t.is_contiguous()
    p = lambda t: C.c_void_p(t.data_ptr())
    with torch.cuda.device(dev):
        _check(lib().jenga_narrowphase_static(C.byref(desc), p(state), p(props), p(pairs), p(n_pairs), p(contacts), p(n_contacts),
                                              p(status), C.c_void_p(torch.cuda.current_stream(dev).cuda_stream)),
               "jenga_narrowphase_static")


def jenga_narrowphase_static_env_bytes(desc: WorldDesc) -> int:
    return int(lib().jenga_narrowphase_static_env_bytes(C.byref(desc)))


class World:
    """Device buffers of one batch of envs plus the library handle.

    state/props/mu are host arrays (numpy or torch, fp32) in the tile layout of include/jenga.h;
    they are copied to the device once here.  All methods enqueue on torch's current stream.
    """

    def __init__(self, wp, state, props, mu, materialise: bool = False, device: int = 0, collapse_length: float = 0.0,
                 tier: str = "auto", ref_state=None, group: int = 0, stage_buffers: bool = True):
        """stage_buffers=False: pairs / contacts / lambda are not allocated (2.3 GB at 65,536 envs); such a world steps
        (materialise must be off) but refuses jenga_broadphase / jenga_narrowphase / jenga_pgs_solve."""
        if not torch.cuda.is_available():
            raise JengaError("no CUDA device: the Jenga step has no CPU path")
        self.wp = wp
        self.dev = torch.device("cuda", device)
        E, S = wp.n_envs, wp.body_stride
        pc = wp.max_contacts // 4
        t = lambda a, dt: torch.as_tensor(a, dtype=dt).contiguous().to(self.dev)
        self.state = t(state, torch.float32)
        self.props = t(props, torch.float32)
        self.mu = t(mu, torch.float32)
        assert self.state.shape == (E, 13, S) and self.props.shape == (E, 8, S) and self.mu.shape == (E,)
        z = lambda shape, dt: torch.zeros(shape, dtype=dt, device=self.dev)
        self.f_ext = None
        if stage_buffers:
            self.pairs = z((E, wp.max_pairs), torch.int32)
            self.n_pairs = z((E,), torch.int32)
            self.contacts = z((E, wp.max_contacts, 8), torch.float32)
            self.n_contacts = z((E,), torch.int32)
            self.lam = z((E, wp.max_contacts, 3), torch.float32)
        else:
            self.pairs = self.n_pairs = self.contacts = self.n_contacts = self.lam = None
        self.cache_key = z((E, pc, 2), torch.int32)
        self.cache_lam = z((E, pc, 4, 3), torch.float32)
        self.cache_pt = z((E, pc, 4, 3), torch.float32)
        self.n_cache = z((E,), torch.int32)
        self.status = z((E,), torch.int32)
        self.counters = z((N_COUNTERS,), torch.int64)
        self.desc = make_desc(wp, materialise, device, tier, group)
        self.desc.collapse_length = float(collapse_length)
        n_scr = lib().jenga_scratch_bytes(C.byref(self.desc))
        if n_scr == 0:
            raise JengaError("jenga_scratch_bytes: the world descriptor is out of range")
        self.scratch = z((n_scr,), torch.uint8)
        b = Buffers()
        b.state, b.props, b.mu, b.f_ext = self.state.data_ptr(), self.props.data_ptr(), self.mu.data_ptr(), None
        if stage_buffers:
            b.pairs, b.n_pairs = self.pairs.data_ptr(), self.n_pairs.data_ptr()
            b.contacts, b.n_contacts, b.lambda_ = self.contacts.data_ptr(), self.n_contacts.data_ptr(), self.lam.data_ptr()
        b.cache_key, b.cache_lam, b.cache_pt = self.cache_key.data_ptr(), self.cache_lam.data_ptr(), self.cache_pt.data_ptr()
        b.n_cache, b.status, b.counters = self.n_cache.data_ptr(), self.status.data_ptr(), self.counters.data_ptr()
        self.ref_pose = self.collapsed = self.collapse_stats = None
        self.rest_steps = z((E,), torch.int32)
        b.rest_steps = self.rest_steps.data_ptr()
        b.scratch, b.scratch_bytes = self.scratch.data_ptr(), n_scr
        if collapse_length > 0.0:                      # Eq. 18 latch against the pose the world starts from
            src = self.state if ref_state is None else t(ref_state, torch.float32)      # Eq. 18's reference pose
            self.ref_pose = src[:, 0:7, :].clone()             # a copy also when E = 1 (contiguous() would alias the live state)
            self.collapsed = z((E,), torch.int32)
            self.collapse_stats = z((E, 4), torch.float32)
            b.ref_pose, b.collapsed, b.collapse_stats = self.ref_pose.data_ptr(), self.collapsed.data_ptr(), self.collapse_stats.data_ptr()
        self.bufs = b
        self.handle = C.c_void_p()
        _check(lib().jenga_world_create(C.byref(self.desc), C.byref(b), C.byref(self.handle)), "jenga_world_create")

    # -- the C-ABI calls, same names ------------------------------------------------------
    def _stream(self):
        return C.c_void_p(torch.cuda.current_stream(self.dev).cuda_stream)

    def jenga_broadphase(self):
        _check(lib().jenga_broadphase(self.handle, self._stream()), "jenga_broadphase")

    def jenga_narrowphase(self):
        _check(lib().jenga_narrowphase(self.handle, self._stream()), "jenga_narrowphase")

    def jenga_pgs_solve(self, iters: int = 0):
        _check(lib().jenga_pgs_solve(self.handle, int(iters), self._stream()), "jenga_pgs_solve")

    def jenga_step(self, n_steps: int = 1):
        _check(lib().jenga_step(self.handle, int(n_steps), self._stream()), "jenga_step")

    def jenga_simulate_until_rest(self, max_steps: int = 400, ek_rest: float = 1.0e-7):
        _check(lib().jenga_simulate_until_rest(self.handle, int(max_steps), C.c_float(ek_rest), self._stream()), "jenga_simulate_until_rest")

    def jenga_step_host(self, h_state_in, h_state_out, n_steps: int = 1):
        """h_state_in / h_state_out: None or contiguous fp32 CPU tensors [E][13][S] (pinned for async copies)."""
        for t in (h_state_in, h_state_out):
            if t is not None:
                assert t.device.type == "cpu" and t.dtype == torch.float32 and t.is_contiguous() and t.shape == self.state.shape
        pi = C.c_void_p(h_state_in.data_ptr()) if h_state_in is not None else None
        po = C.c_void_p(h_state_out.data_ptr()) if h_state_out is not None else None
        _check(lib().jenga_step_host(self.handle, pi, po, int(n_steps), self._stream()), "jenga_step_host")

    def jenga_set_f_ext(self, f_ext):
        """f_ext: None or an [E][6][S] fp32 array/tensor (copied to the device, kept alive here)."""
        if f_ext is None:
            self.f_ext = None
            _check(lib().jenga_set_f_ext(self.handle, None), "jenga_set_f_ext")
        else:
            self.f_ext = torch.as_tensor(f_ext, dtype=torch.float32).contiguous().to(self.dev)
            assert self.f_ext.shape == (self.wp.n_envs, 6, self.wp.body_stride)
            _check(lib().jenga_set_f_ext(self.handle, C.c_void_p(self.f_ext.data_ptr())), "jenga_set_f_ext")

    def jenga_support_margin(self):
        """Eq. 17 per env: tensor [E][4] = margin, COM_x, COM_y, hull vertices (device)."""
        out = torch.empty((self.wp.n_envs, 4), dtype=torch.float32, device=self.dev)
        _check(lib().jenga_support_margin(self.handle, C.c_void_p(out.data_ptr()), self._stream()), "jenga_support_margin")
        return out

    def jenga_ziglar_block_analysis(self, block, axis):
        """Table 1 per env: block, axis int arrays [E]; tensor [E][4] = class, F_min [N], torque flag, k (device)."""
        tb = torch.as_tensor(block, dtype=torch.int32).contiguous().to(self.dev)
        ta = torch.as_tensor(axis, dtype=torch.int32).contiguous().to(self.dev)
        assert tb.shape == (self.wp.n_envs,) and ta.shape == (self.wp.n_envs,)
        out = torch.empty((self.wp.n_envs, 4), dtype=torch.float32, device=self.dev)
        _check(lib().jenga_ziglar_block_analysis(self.handle, C.c_void_p(tb.data_ptr()), C.c_void_p(ta.data_ptr()),
                                                 C.c_void_p(out.data_ptr()), self._stream()), "jenga_ziglar_block_analysis")
        return out

    def jenga_profile_enable(self, on: bool = True):
        _check(lib().jenga_profile_enable(self.handle, int(on)), "jenga_profile_enable")

    def jenga_profile_read(self) -> dict:
        out = (C.c_double * 5)()
        _check(lib().jenga_profile_read(self.handle, out), "jenga_profile_read")
        return dict(detect_ms=out[0], manifold_ms=out[1], slot_ms=out[2], collide_ms=out[0] + out[1] + out[2], solve_ms=out[3],
                    substeps=int(out[4]))

    def jenga_world_destroy(self):
        if self.handle:
            _check(lib().jenga_world_destroy(self.handle), "jenga_world_destroy")
            self.handle = C.c_void_p()

    broadphase, narrowphase, pgs_solve, step, step_host, simulate_until_rest, set_f_ext, destroy = (
        jenga_broadphase, jenga_narrowphase, jenga_pgs_solve, jenga_step, jenga_step_host, jenga_simulate_until_rest,
        jenga_set_f_ext, jenga_world_destroy)

    def __del__(self):
        try:
            self.jenga_world_destroy()
        except Exception:
            pass

    # -- helpers ---------------------------------------------------------------------------
    def reset_cache(self):
        self.n_cache.zero_()

    def counters_dict(self):
        return dict(zip(COUNTER_NAMES, self.counters.tolist()))

    def launch_info(self):
        return dict(threads=lib().jenga_block_threads(C.byref(self.desc)), smem_bytes=lib().jenga_smem_bytes(C.byref(self.desc)),
                    env_group=lib().jenga_env_group(C.byref(self.desc)))
