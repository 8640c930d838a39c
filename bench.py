#!/usr/bin/env python
"""bench.py -- env-steps/s of the batched Jenga step (BASELINE.json metric) on N B200s of one node.

    python bench.py [--gpus N] [--steps K] [--warmup W]            # the CUDA path (libjenga.so)
    python bench.py --impl reference [--steps K] [--warmup W]       # the fp64 oracle on the host cores

Workload: BASELINE.json configs[4] ("cfg5", the throughput headline): 65,536 envs of 18-level, 54-block
towers per GPU, mu_s round-robin, 0-12 removals, Ziglar push sweep, dt = 1/240, 20 PGS iterations, fp32;
seeded synthetic inputs from paper_2606_28394_b200/workloads.py.  A "step" is one dt
advance of every env of the batch through the whole hot path (S1..S7, six kernels per substep).  With no --steps the
timed region is the whole 480-step rollout (cold warm-start cache, settle window, push at steps 60-83, collapse);
with --steps K below that, the K timed steps are spread evenly over the rollout and the steps in between run untimed
(config.window says which), so a short run still measures the rollout's mix and not only its standing towers.
Weak scaling: each rank owns its own 65,536 envs (env ids rank*E ..), no collective on the data path.

One JSON line on stdout (rank 0).  See DESIGN.md §7 for the work model behind "roofline".
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
sys.path.insert(0, ROOT)

METRIC = "env-steps/s"
CFG = 5
N_SM, FP32_LANES_PER_SM = 148, 128          # B200: 148 SMs x 4 SMSPs x 32 FP32 lanes (guide: B200_PROFILING.md table)

# Algorithmic FP32 thread-instructions (FMA = 1), SURVEY.md §8(d) / DESIGN.md §7
W_ROW, W_ROW_GROUND = 87, 51                # per contact-iteration: 3 rows x (J.v 12 + clamp 5 + apply 12); ground rows touch one body
W_SETUP = 190                               # per contact: r, basis, 3 x (2 cross + 2 I^-1 mul + k)
W_MANIFOLD, W_MANIFOLD_GROUND = 600, 100    # per colliding pair
W_SAT = 250                                 # per candidate pair
W_AABB_TEST, W_AABB_BODY, W_INTEGRATE = 15, 30, 100


def work_model(cnt: dict, n_bodies: int, iters: int) -> dict:
    """Algorithmic FP32 thread-instructions of the launches that produced the counters `cnt`."""
    gc, c = cnt["ground_contacts"], cnt["contacts"]
    ground_pairs = gc / 4.0                                   # a resting block has 4 ground corners
    tests = n_bodies * (n_bodies - 1) // 2 + n_bodies
    parts = {
        "pgs_rows": iters * ((c - gc) * W_ROW + gc * W_ROW_GROUND),
        "setup": c * W_SETUP,
        "manifold": (cnt["colliding"] - ground_pairs) * W_MANIFOLD + ground_pairs * W_MANIFOLD_GROUND,
        "sat": cnt["candidates"] * W_SAT,
        "broadphase": cnt["env_steps"] * (tests * W_AABB_TEST + n_bodies * W_AABB_BODY),
        "integrate": cnt["body_steps"] * W_INTEGRATE,
    }
    parts["total"] = float(sum(parts.values()))
    return parts


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU through NVML while the timed region runs."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, cuda_index: int, period: float = 0.1):
        super().__init__(daemon=True)
        self.period, self.samples, self.mask, self.sm_max, self.power = period, [], 0, None, 0.0
        self._halt = threading.Event()
        self.h = None
        try:
            import pynvml as N
            import torch
            N.nvmlInit()
            self.N = N
            try:
                uuid = "GPU-" + str(torch.cuda.get_device_properties(cuda_index).uuid)
                self.h = N.nvmlDeviceGetHandleByUUID(uuid.encode() if isinstance(uuid, str) else uuid)
            except Exception:
                self.h = N.nvmlDeviceGetHandleByIndex(cuda_index)
            self.sm_max = int(N.nvmlDeviceGetMaxClockInfo(self.h, N.NVML_CLOCK_SM))
        except Exception as exc:                 # NVML missing: report that, never fake a clock
            self.err = repr(exc)

    def run(self):
        if self.h is None:
            return
        N = self.N
        while not self._halt.is_set():
            try:
                self.samples.append(int(N.nvmlDeviceGetClockInfo(self.h, N.NVML_CLOCK_SM)))
                self.mask |= int(N.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                self.power = max(self.power, N.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            self._halt.wait(self.period)

    def stop(self) -> dict:
        self._halt.set()
        if self.is_alive():
            self.join()
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": ["nvml_unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.sm_max,
                "reasons": [n for b, n in self.REASONS.items() if self.mask & b],
                "samples": len(self.samples), "power_w_max": round(self.power, 1)}


def schedule(wl, n_steps: int, chunk: int):
    """Split steps [0, n_steps) into launches: boundaries where the push switches on/off and every `chunk` steps.
    Yields (first_step, n, push_active)."""
    s = 0
    while s < n_steps:
        active = wl.push_fext is not None and wl.push_start <= s < wl.push_end
        nxt = n_steps
        for b in (wl.push_start, wl.push_end):
            if s < b < nxt:
                nxt = b
        n = min(chunk, nxt - s)
        yield s, n, active
        s += n


def timed_plan(wl, K: int, chunk: int):
    """The launches of the timed pass: (first_step, n, push_active, timed).  K = the whole rollout: every launch is timed
    (chunks of `chunk` steps).  K below the rollout length (the driver's --steps 20): the K timed steps are spread evenly
    over the WHOLE rollout -- step round(i N / K), one step per call -- and the steps in between run untimed, so that the
    figure is the rollout's (settle window, push, collapse, debris), not that of its first K steps of standing towers."""
    N = wl.n_steps
    if K >= N:
        return [(s, n, a, True) for s, n, a in schedule(wl, N, chunk)]
    picked = sorted({int(i * N / K) for i in range(K)})
    assert len(picked) == K
    pset = set(picked)
    return [(s, 1, a, s in pset) for s, _, a in schedule(wl, picked[-1] + 1, 1)]


# ------------------------------------------------------------------------------- oracle arm (CPU)
# the oracle is timed on cfg1 and cfg2 in full, the first 256 envs of cfg3 / cfg4, the first 1024 of cfg5
ORACLE_SUBSET = {1: 1, 2: 450, 3: 256, 4: 256, 5: 1024, 6: 450}
CFG_ENVS = {1: 1, 2: 450, 3: 4096, 4: 4096, 5: 65536, 6: 450}      # BASELINE.json configs[0..4]; 6 = the paper's Table 6 set
CFG_NAMES = {1: "cfg1 (BASELINE.json configs[0]): 1 env, 3-level tower, 10 PGS iters, 240 steps",
             2: "cfg2 (BASELINE.json configs[1]): 450 envs of 18-level 54-block towers, removals + push k ~ U(2,5), 20 PGS iters, 480 steps",
             3: "cfg3 (BASELINE.json configs[2]): 4096 envs of 54-block collapse debris, 20 PGS iters, 720 steps",
             4: "cfg4 (BASELINE.json configs[3]): 4096 envs of 30-level 90-block towers, 0-20 removals, 50 PGS iters, 480 steps",
             6: "cfg6 (SURVEY §8(f) NEXT-3): 450 envs of 54-block towers with the paper's Table 6 parameters (81x26x18 mm, 19.6 g, e = 0.10, 3 substeps, 14 PGS iters)"}


def oracle_sample(n_envs: int, env_offset: int = 0, cfg: int = CFG):
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import oracle as O                                     # test infrastructure; allowed here (cpu_baseline / --impl reference)
    from paper_2606_28394_b200 import workloads as W
    wl = W.make_config(cfg, n_envs=n_envs, env_offset=env_offset)
    P = O.make_params(wl.params)
    bod = O.unpack_tiles(wl.state, wl.props, wl.params.n_bodies)
    cache = O.Cache(bod.E, wl.params.max_contacts)
    fext = O.unpack_fext(wl.push_fext, wl.params.n_bodies)
    return O, wl, P, bod, cache, fext


def oracle_advance(O, wl, P, bod, cache, fext, first: int, n: int):
    """Steps [first, first+n) of the rollout with the push schedule; returns seconds."""
    t0 = time.perf_counter()
    mu = wl.mu.astype(np.float64)
    for s, k, active in schedule(wl, first + n, 1 << 30):
        if s + k <= first:
            continue
        lo = max(s, first)
        O.rollout(P, bod, mu, s + k - lo, fext=fext if active else None, cache=cache)
    return time.perf_counter() - t0


def cpu_baseline(budget_s: float = 15.0, cfg: int = CFG) -> dict:
    """The oracle as it stands on the host cores, on a bounded sample of the same workload: the whole rollout of the
    first n envs of the config, n sized from a probe so that the run takes ~budget_s, at most SURVEY §8(d)'s subset."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import oracle as O
    cores = int(O.n_threads())
    cap = ORACLE_SUBSET.get(cfg, 1024)
    n_probe = min(2 * cores, cap)
    O, wl, P, bod, cache, fext = oracle_sample(n_probe, cfg=cfg)
    oracle_advance(O, wl, P, bod, cache, fext, 0, 2)                      # page in, spin up the OpenMP team
    t_probe = oracle_advance(O, wl, P, bod, cache, fext, 2, 10)
    rate = n_probe * 10 / t_probe                                          # env-steps/s
    n_envs = int(min(cap, max(min(cores, cap), round(budget_s * rate / wl.n_steps / cores) * cores)))
    O, wl, P, bod, cache, fext = oracle_sample(n_envs, cfg=cfg)
    t = oracle_advance(O, wl, P, bod, cache, fext, 0, wl.n_steps)
    return {"value": n_envs * wl.n_steps / t, "unit": METRIC, "cores": cores, "kind": "oracle",
            "sample": f"first {n_envs} envs of cfg{cfg}, all {wl.n_steps} steps of the rollout (fp64, OpenMP over envs), {t:.1f} s"}


def run_reference(args) -> dict:
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        sys.exit(0)
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import oracle as O
    cores = int(O.n_threads())
    n_envs = max(32, 2 * cores)
    O, wl, P, bod, cache, fext = oracle_sample(n_envs)
    steps = min(args.steps, wl.n_steps - args.warmup)
    oracle_advance(O, wl, P, bod, cache, fext, 0, args.warmup)
    t = oracle_advance(O, wl, P, bod, cache, fext, args.warmup, steps)
    v = n_envs * steps / t
    sample = f"first {n_envs} envs of cfg5 per step, steps {args.warmup}..{args.warmup + steps} of the rollout (fp64 oracle, OpenMP over envs)"
    return {"impl": "reference", "metric": METRIC, "value": v, "unit": METRIC, "n_gpus": args.gpus, "steps": steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t / steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "cfg5: 18-level 54-block towers, 20 PGS iters, dt=1/240 (bounded sample)", "envs_per_step": n_envs},
            "cpu_baseline": {"value": v, "unit": METRIC, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": METRIC, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def run_dry(args):
    """The multi-rank plumbing of the CUDA arm without a GPU: process group, env ranges, max-over-ranks timing."""
    import torch.distributed as dist
    from paper_2606_28394_b200 import shard
    rank, world_size = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    if world_size > 1:
        dist.init_process_group(args.backend)
    lo, hi = shard.env_range(rank, world_size, args.envs or CFG_ENVS[args.cfg])
    ms = shard.max_over_ranks(100.0 + rank)                       # stands in for the device time of this rank
    total = shard.sum_over_ranks(hi - lo)
    if world_size > 1:
        dist.destroy_process_group()
    if rank != 0:
        return None
    return {"dry_run": True, "n_gpus": world_size, "env_ranges_rank0": [lo, hi], "total_envs": total, "ms_max_over_ranks": ms,
            "scaling": "weak"}


# ------------------------------------------------------------------------------- CUDA arm
def run_cuda(args) -> dict:
    import torch
    import torch.distributed as dist
    from paper_2606_28394_b200 import binding, shard, workloads as W

    rank, world_size = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the Jenga step has no CPU path")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world_size > 1:
        dist.init_process_group(args.backend, device_id=dev)
    binding.lib()                                            # fail loudly if libjenga.so is missing

    E = args.envs or CFG_ENVS[args.cfg]
    wl = W.make_config(args.cfg, n_envs=E, env_offset=shard.env_range(rank, world_size, E)[0])
    if wl.push_fext is None:
        wl.push_fext = np.zeros((E, 6, wl.params.body_stride), np.float32); wl.push_start = wl.push_end = 0   # weak scaling: every rank has its own E envs
    wp = wl.params
    if args.max_contacts:
        wp.max_contacts = args.max_contacts
    if args.max_pairs:
        wp.max_pairs = args.max_pairs
    K = min(args.steps, wl.n_steps) if args.steps > 0 else wl.n_steps
    # a world that only steps: no pairs / contacts / lambda buffers (2.3 GB at 65,536 envs that nothing would write)
    world = binding.World(wp, wl.state, wl.props, wl.mu, device=local, tier=args.tier, group=args.group, stage_buffers=False)
    state0 = world.state.clone()
    fext_dev = torch.as_tensor(wl.push_fext).to(dev)
    fext_ptr = binding.C.c_void_p(fext_dev.data_ptr())
    L = binding.lib()
    stream = torch.cuda.current_stream(dev)

    def set_push(active: bool):
        binding._check(L.jenga_set_f_ext(world.handle, fext_ptr if active else None), "jenga_set_f_ext")

    def reset():
        world.state.copy_(state0)
        world.n_cache.zero_(); world.status.zero_(); world.counters.zero_()
        set_push(False)

    def barrier():
        if world_size > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # warm-up: W untimed steps of the same launch shape, then back to step 0
    for _ in range(max(args.warmup, 0)):
        world.jenga_step(min(args.chunk, K))
    reset()

    # ---- roofline denominators measured on this device now (FP32 FFMA issue rate, LDS.128 bandwidth)
    peaks = binding.jenga_measure_peaks(local)

    # ---- device-resident timing: inputs already in HBM, CUDA events on the launching stream.  Two passes over the same
    # launches: pass 1 is the headline (no per-kernel events, the shipping configuration); pass 2 repeats it with
    # jenga_profile_* on and gives the per-kernel split for the roofline (its own total is reported as "profiled_ms").
    launches = timed_plan(wl, K, args.chunk)
    n_timed = sum(1 for l in launches if l[3])
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for l in launches if l[3]]
    # inputs far larger than L2 (cfg3-5) need no flush; the small configs rewrite a 256 MB buffer between the timed calls
    scratch_per_env = world.scratch.numel() // E
    small = E * (scratch_per_env + 13 * wp.body_stride * 4) < 2 * 126e6
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if small else None
    ACC = ("env_steps", "body_steps", "candidates", "colliding", "contacts", "contact_iters", "colours", "ground_contacts")
    sampler = ClockSampler(local); sampler.start()
    barrier()
    snaps, k = [], 0
    for s, n, active, timed in launches:
        set_push(active)
        if not timed:
            world.jenga_step(n)
            continue
        if flush is not None:
            flush.zero_()
        c0 = world.counters.clone()                          # counters of the timed launches only (device-side copies, no sync)
        ev[k][0].record(stream)
        world.jenga_step(n)
        ev[k][1].record(stream)
        snaps.append((c0, world.counters.clone())); k += 1
    barrier()
    clocks = sampler.stop()
    launch_ms = [a.elapsed_time(b) for a, b in ev]
    ms = sum(launch_ms)                                      # the timed region = the timed jenga_step calls
    cnt = world.counters_dict()                              # running maxima: of the whole pass
    acc = sum((b - a for a, b in snaps), torch.zeros_like(world.counters)).tolist()
    for name in ACC:
        cnt[name] = int(acc[binding.COUNTER_NAMES.index(name)])
    status_or = int(np.bitwise_or.reduce(world.status.cpu().numpy()))
    n_flagged = int((world.status != 0).sum().item())
    assert cnt["env_steps"] == E * K, (cnt, E, K)
    # pass 2: the same launches with events around every kernel of the timed ones
    reset()
    prof = dict(detect_ms=0.0, manifold_ms=0.0, slot_ms=0.0, collide_ms=0.0, solve_ms=0.0, substeps=0)
    barrier()
    for s, n, active, timed in launches:
        set_push(active)
        if not timed:
            world.jenga_step(n)
            continue
        if flush is not None:
            flush.zero_()
        world.jenga_profile_enable(True)
        world.jenga_step(n)
        for key, v in world.jenga_profile_read().items():    # synchronises on this launch's events
            prof[key] += v
        world.jenga_profile_enable(False)
    barrier()
    del flush
    first_timed, last_timed = min(l[0] for l in launches if l[3]), max(l[0] + l[1] - 1 for l in launches if l[3])
    window = (f"all {K} steps of the rollout, {args.chunk} per call" if K >= wl.n_steps else
              f"{K} timed steps spread over rollout steps {first_timed}..{last_timed} of {wl.n_steps} (every {wl.n_steps / K:.0f}th step, one per call; "
              f"the steps in between run untimed)")

    # ---- end to end through the C-ABI with HOST buffers: every step, for every env, H2D of the state tile (pinned
    # memory), the step, D2H of the result (jenga_step_host).  The batch is served as `--e2e-split` worlds of E/split
    # envs on their own streams, so that one part's copies overlap the other part's kernel (what a user of the
    # library would do with a PCIe-bound call); the result of step s is the host input of step s+1.
    linfo = world.launch_info()
    linfo_scratch = world.scratch.numel() // E
    world.destroy(); del world
    torch.cuda.empty_cache()
    n_split = max(1, min(args.e2e_split, E))
    bounds = [(i * E // n_split, (i + 1) * E // n_split) for i in range(n_split)]
    parts = []
    for lo, hi in bounds:
        wpi = W.WorldParams(**{**wp.__dict__, "n_envs": hi - lo})
        wi = binding.World(wpi, wl.state[lo:hi], wl.props[lo:hi], wl.mu[lo:hi], device=local, tier=args.tier, group=args.group, stage_buffers=False)
        h_a = torch.empty(wi.state.shape, dtype=torch.float32, pin_memory=True)
        h_b = torch.empty_like(h_a, pin_memory=True)
        h_a.copy_(torch.as_tensor(wl.state[lo:hi]))
        parts.append(dict(w=wi, st=torch.cuda.Stream(dev), h_a=h_a, h_b=h_b, h_fext=torch.as_tensor(wl.push_fext[lo:hi]).pin_memory(),
                          fdev=torch.zeros((hi - lo, 6, wp.body_stride), dtype=torch.float32, device=dev)))
    Ke = min(K, args.e2e_steps) if args.e2e_steps > 0 else K
    h2d = d2h = 0
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for p in parts:
        p["st"].wait_event(e0)
    pushing = False
    for s in range(Ke):
        active = wl.push_start <= s < wl.push_end
        for p in parts:
            with torch.cuda.stream(p["st"]):
                if active and not pushing:
                    p["fdev"].copy_(p["h_fext"], non_blocking=True); h2d += p["h_fext"].numel() * 4
                if active != pushing:
                    binding._check(L.jenga_set_f_ext(p["w"].handle, binding.C.c_void_p(p["fdev"].data_ptr()) if active else None), "jenga_set_f_ext")
                p["w"].jenga_step_host(p["h_a"], p["h_b"], 1)
                p["h_a"], p["h_b"] = p["h_b"], p["h_a"]
                h2d += p["h_a"].numel() * 4; d2h += p["h_a"].numel() * 4
        pushing = active
    for p in parts:
        ev = torch.cuda.Event(); ev.record(p["st"]); stream.wait_event(ev)
    e1.record(stream)
    barrier()
    ms_e2e = e0.elapsed_time(e1)
    e2e_launches = Ke * n_split

    ms, ms_e2e = shard.max_over_ranks(ms, dev), shard.max_over_ranks(ms_e2e, dev)
    total_env_steps = E * K * world_size
    value = total_env_steps / (ms * 1e-3)
    e2e_value = E * Ke * world_size / (ms_e2e * 1e-3)

    # ---- roofline.  Six kernels per substep: k_detect, k_walk, k_plan (timed together), k_manifold, k_slot (S1-S4) and k_solve (S4 warm
    # start, S5, S6, S7), timed with CUDA events on the launching stream (jenga_profile_*).  `roofline` is the dominant kernel
    # (k_solve): its algorithmic FP32 thread-instructions / its summed launch time vs the FP32 issue rate measured by
    # jenga_measure_peaks on this device; "step" carries the same ratio for the whole step (both kernels).
    wm = work_model(cnt, wp.n_bodies, wp.pgs_iters)
    solve_s, collide_s = prof["solve_ms"] * 1e-3, prof["collide_ms"] * 1e-3
    peak = peaks["fp32_instr_per_s"] / 1e12
    w_solve = wm["pgs_rows"] + wm["integrate"]
    w_collide = wm["total"] - w_solve
    achieved = w_solve / solve_s / 1e12
    n_sub = prof["substeps"]
    smem_model = (cnt["contact_iters"] * 96.0) / solve_s / 1e12       # 96 B of body traffic per contact-iteration
    # traffic is NOT measured by this run: it is the committed ncu figure (dram__bytes_read + write per env-step of one
    # --set full capture of k_solve at cfg5, profiles/k_solve_traffic.csv) scaled to the env-steps of one launch
    traffic = traffic_src = step_dram = None
    tpath = os.path.join(ROOT, "profiles", "k_solve_traffic.csv")
    if os.path.exists(tpath):
        import csv
        row = next(csv.DictReader(open(tpath)))
        traffic = float(row["dram_bytes_per_env_step"]) * cnt["env_steps"] / max(n_sub, 1)
        traffic_src = "profiles/k_solve_traffic.csv (ncu --set full of k_solve at cfg5, not this run) x env-steps per launch"
        step_dram = float(row["step_dram_bytes_per_env_step"]) if row.get("step_dram_bytes_per_env_step") else None
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "Tinstr/s (FP32 thread-instructions, FMA=1)",
                "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src,
                "step_dram_bytes_per_env_step": step_dram,            # all six kernels, ncu (profiles/), cfg5
                "algorithmic_bytes_per_env_step": 25e3,               # state in + out, props, warm-start cache <= 25 KB
                "kernel": "k_solve", "launch_ms_avg": prof["solve_ms"] / max(n_sub, 1),
                "launches": n_sub, "share_of_step_time": solve_s / (solve_s + collide_s),
                "peak_source": f"measured now by jenga_measure_peaks: dependent-free FFMA streams on {peaks['n_sm']} SMs "
                               f"({peaks['fp32_instr_per_s_noreuse'] / 1e12:.2f} T/s when no source register is reused, {peaks['fp32_fma_per_s_packed_noreuse'] / 1e12:.2f} T FMA/s packed f32x2); "
                               f"LDS.128 {peaks['smem_bytes_per_s'] / 1e12:.2f} TB/s; nominal 148 x 128 x {clocks.get('sm_max_mhz') or 1965} MHz = "
                               f"{N_SM * FP32_LANES_PER_SM * (clocks.get('sm_max_mhz') or 1965) * 1e6 / 1e12:.2f} T/s",
                "smem_model_frac": smem_model / (peaks["smem_bytes_per_s"] / 1e12),
                # the solver's FFMAs read three registers that change from one instruction to the next; a dependent-free stream
                # of that shape is register-file bound below the FFMA peak (jenga_measure_peaks, csrc/peaks.cu)
                "peak_noreuse": peaks["fp32_instr_per_s_noreuse"] / 1e12, "frac_of_noreuse_peak": achieved / (peaks["fp32_instr_per_s_noreuse"] / 1e12),
                "algorithmic_instr_per_env_step": wm["total"] / cnt["env_steps"],
                "shares": {k: round(v / wm["total"], 4) for k, v in wm.items() if k != "total"},
                "collision_kernels": {"achieved": w_collide / collide_s / 1e12, "frac": w_collide / collide_s / 1e12 / peak,
                                      "k_detect_ms_avg": prof["detect_ms"] / max(n_sub, 1), "k_manifold_ms_avg": prof["manifold_ms"] / max(n_sub, 1),
                                      "k_slot_ms_avg": prof["slot_ms"] / max(n_sub, 1)},
                "step": {"achieved": wm["total"] / (solve_s + collide_s) / 1e12, "frac": wm["total"] / (solve_s + collide_s) / 1e12 / peak,
                         "kernel_ms": prof["solve_ms"] + prof["collide_ms"], "wall_ms": sum(launch_ms)},
                "timing": "value / ms_per_step: pass 1, CUDA events around the timed jenga_step calls, no per-kernel events; "
                          "kernel times and fractions: pass 2 over the same steps with jenga_profile_* events around every kernel"}
    out = {
        "metric": METRIC, "value": value, "unit": METRIC, "n_gpus": world_size, "steps": K, "warmup": args.warmup,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": "cfg5 (BASELINE.json configs[4]): 18-level 54-block towers, mu_s {0.25,0.40,0.60} round-robin, 0-12 removals, "
                               "Ziglar push sweep, dt=1/240, 20 PGS iters" if args.cfg == CFG else CFG_NAMES[args.cfg] + " (not the headline workload)",
                   "window": window,
                   "envs_per_gpu": E, "n_bodies": wp.n_bodies, "pgs_iters": wp.pgs_iters, "steps_per_call": args.chunk, "kernels_per_substep": 6,
                   "parallelism": f"env-sharded x{world_size}, no data-path collective",
                   "l2": (f"inputs larger than L2: state {E * 13 * wp.body_stride * 4 / 1e6:.0f} MB + scratch {E * linfo_scratch / 1e6:.0f} MB + warm-start cache "
                          f"{E * (wp.max_contacts // 4) * 104 / 1e6:.0f} MB per step vs 126 MB L2") if not small else
                         "working set smaller than L2 (small config): an 8 x 32 MB buffer is rewritten between the timed launches"},
        "body_steps_per_s": cnt["body_steps"] * world_size / (ms * 1e-3),
        "contacts_per_s": cnt["contacts"] * world_size / (ms * 1e-3),
        "contact_iters_per_s": cnt["contact_iters"] * world_size / (ms * 1e-3),
        "contacts_per_env_step": cnt["contacts"] / cnt["env_steps"],
        "colours_per_env_step": cnt["colours"] / cnt["env_steps"],
        "status": {"or": status_or, "envs_flagged": n_flagged},
        "maxima": {k: cnt[k] for k in ("max_candidates", "max_colliding", "max_colours")},
        "capacity": {"max_pairs": wp.max_pairs, "max_contacts": wp.max_contacts, "smem_bytes_per_cta": linfo["smem_bytes"],
                     "threads_per_cta": linfo["threads"], "envs_per_warp": linfo["env_group"],
                     "envs_in_flight_per_sm": linfo["threads"] // 32 * linfo["env_group"]},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": METRIC, "h2d_bytes_per_step": h2d // Ke, "d2h_bytes_per_step": d2h // Ke, "steps": Ke,
                "split": n_split, "launches": e2e_launches, "window": f"rollout steps 0..{Ke - 1}, contiguous (every step's state goes through the host)"},
        "gpu_launches": 6 * n_sub,
        "roofline": roofline,
    }
    if rank == 0 and world_size == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(cfg=args.cfg)
    if world_size > 1:
        dist.destroy_process_group()
    return out if rank == 0 else None


def spawn_ranks(n: int, argv) -> int:
    """`python bench.py --gpus N` without a launcher: re-exec this script under torch.distributed.run, one rank per GPU
    (envs are independent episodes: each rank owns its own env range)."""
    import socket
    import subprocess
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + list(argv)
    env = dict(os.environ, NCCL_DEBUG=os.environ.get("NCCL_DEBUG", "WARN"))
    return subprocess.call(cmd, env=env)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=0, help="dt advances timed (default 0: the config's full rollout, 480 steps for cfg5)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["cuda", "reference"], default="cuda")
    ap.add_argument("--envs", type=int, default=0, help="envs per GPU (default: the config's own count; cfg5: 65,536)")
    ap.add_argument("--chunk", type=int, default=12, help="dt advances per jenga_step launch")
    ap.add_argument("--e2e-steps", type=int, default=96, help="steps of the end-to-end (host buffers) leg; 0 = K")
    ap.add_argument("--e2e-split", type=int, default=2, help="worlds (streams) the e2e leg serves the batch with")
    ap.add_argument("--cfg", type=int, default=CFG, help="BASELINE.json config number (5 = the bench workload; others: manual runs)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--group", type=int, default=0, choices=[0, 1, 2], help="envs per k_solve warp (0 = auto)")
    ap.add_argument("--tier", default="auto", choices=["auto", "smem", "tmem128", "tmem160", "tmem256", "tmem512"], help="where k_solve keeps the contact constants")
    ap.add_argument("--max-contacts", type=int, default=0, help="override the workload's contact capacity per env")
    ap.add_argument("--max-pairs", type=int, default=0, help="override the workload's candidate capacity per env")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"], help="torch.distributed backend (gloo: the CPU test of the launch path)")
    ap.add_argument("--dry-run", action="store_true", help="rendezvous, shard bookkeeping and the timing reduction only (no GPU work): the CPU test of --gpus N")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "cuda":
        sys.exit(spawn_ranks(args.gpus, sys.argv[1:]))
    if args.dry_run:
        out = run_dry(args)
        if out is not None:
            print(json.dumps(out), flush=True)
        return
    if args.impl == "reference":
        args.steps = min(args.steps, 60) if args.steps > 0 else 20      # bounded: the oracle is slow by design
        out = run_reference(args)
    else:
        out = run_cuda(args)
    if out is not None:
        print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
