"""Seeded synthetic inputs for the batched Jenga step (shared by the oracle tests,
the GPU parity tests and bench.py).

This module holds NO arithmetic of the method (no collision, solver or integrator
code): it only lays out blocks, draws jitter / removals / pushes and packs the
result into the SoA tile layout of include/jenga.h.  Everything is generated in
NumPy fp64 and rounded ONCE to fp32; the oracle gets the same fp32 values widened.

Workload recipe: SURVEY.md §8(d) "Synthetic inputs"; tower shape from
PAPER.md:126 (§3: 3 blocks per layer, alternating perpendicular layers, 18 layers),
friction levels from PAPER.md:17 (abstract: 0.25 / 0.40 / 0.60), push magnitudes
F = k*mu_s*m*g from PAPER.md:209,224 (Eq. 8-9).  The paper's own 450 episode files
are not available; these inputs stand in for them.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np

# ---- block geometry of BASELINE.json's configs -------------
BLOCK_L, BLOCK_W, BLOCK_H = 0.075, 0.025, 0.015      # full sizes along body x, y, z [m]
DENSITY = 600.0                                       # kg/m^3
G_LAT = 0.0025                                        # lateral play between blocks of a level [m]
DELTA0 = 1.0e-4                                       # initial vertical overlap per interface [m] (A18)
GRAV = 9.81

STATE_ROWS = 13   # px py pz qw qx qy qz vx vy vz wx wy wz
PROP_ROWS = 8     # inv_m invIx invIy invIz hx hy hz active
FEXT_ROWS = 6     # fx fy fz tx ty tz


def f32(x: float) -> float:
    """Round a Python float to the nearest fp32 and return it as a Python float."""
    return float(np.float32(x))


@dataclasses.dataclass
class WorldParams:
    """World descriptor; every float is already fp32-representable so that the
    CUDA path (float) and the oracle (double) see bit-identical parameters."""
    n_envs: int
    n_bodies: int
    body_stride: int
    dt: float = f32(1.0 / 240.0)
    n_substeps: int = 1
    pgs_iters: int = 20
    gravity: tuple = (0.0, 0.0, f32(-GRAV))
    restitution: float = 0.0
    aabb_margin: float = f32(0.002)
    baumgarte_beta: float = f32(0.35)
    slop: float = f32(4.0e-4)
    edge_bias_rel: float = f32(0.95)
    edge_bias_abs: float = f32(1.0e-4)
    par_eps: float = f32(1.0e-6)
    tie_eps: float = f32(1.0e-6)
    match_tol: float = f32(2.0e-3)
    warm_start: int = 1
    gyroscopic: int = 0
    max_pairs: int = 512       # candidate-pair capacity per env
    max_contacts: int = 1024   # contact capacity per env (4 slots per colliding pair)


def stride_for(n_bodies: int) -> int:
    return (n_bodies + 3) // 4 * 4


def box_mass_props(l: float, w: float, h: float, mass: float):
    """inv_m and the inverse principal moments of a uniform box; the formula is the
    input recipe's (Eq. 3), the oracle has its own pinned copy."""
    ixx = mass / 12.0 * (w * w + h * h)
    iyy = mass / 12.0 * (l * l + h * h)
    izz = mass / 12.0 * (l * l + w * w)
    return 1.0 / mass, (1.0 / ixx, 1.0 / iyy, 1.0 / izz)


BLOCK_MASS = DENSITY * BLOCK_L * BLOCK_W * BLOCK_H   # 0.016875 kg


@dataclasses.dataclass
class Workload:
    name: str
    params: WorldParams
    state: np.ndarray            # [E][13][S] float32
    props: np.ndarray            # [E][8][S]  float32
    mu: np.ndarray               # [E] float32
    n_steps: int
    push_fext: Optional[np.ndarray] = None   # [E][6][S] float32, applied for steps [push_start, push_end)
    push_start: int = 0
    push_end: int = 0
    push_body: Optional[np.ndarray] = None   # [E] int32 (-1 = none)
    push_k: Optional[np.ndarray] = None      # [E] float64 multiple of mu*m*g
    push_kthr: Optional[np.ndarray] = None   # [E] 3 (along) or 4 (across)
    meta: dict = dataclasses.field(default_factory=dict)

    def fext_at(self, step: int):
        if self.push_fext is not None and self.push_start <= step < self.push_end:
            return self.push_fext
        return None


def empty_tiles(E: int, B: int):
    S = stride_for(B)
    state = np.zeros((E, STATE_ROWS, S), dtype=np.float64)
    state[:, 3, :] = 1.0           # identity quaternion in padding lanes too
    props = np.zeros((E, PROP_ROWS, S), dtype=np.float64)
    props[:, 4:7, :] = 1.0e-3      # harmless half-extents for padding (inactive)
    return state, props, S


def set_body(state, props, e, b, pos, quat, half, inv_m, inv_I, vel=(0, 0, 0), omg=(0, 0, 0), active=1.0):
    state[e, 0:3, b] = pos
    state[e, 3:7, b] = quat
    state[e, 7:10, b] = vel
    state[e, 10:13, b] = omg
    props[e, 0, b] = inv_m
    props[e, 1:4, b] = inv_I
    props[e, 4:7, b] = half
    props[e, 7, b] = active


def tower_nominal(levels: int, width: float = BLOCK_W, height: float = BLOCK_H, g_lat: float = G_LAT):
    """Nominal (unjittered) block centres and yaw of an L-level tower.
    body id = 3*level + slot; even levels have the length along world x."""
    n = 3 * levels
    pos = np.zeros((n, 3))
    yaw = np.zeros(n)
    for lv in range(levels):
        psi = 0.0 if lv % 2 == 0 else math.pi / 2
        ybody = np.array([-math.sin(psi), math.cos(psi), 0.0])
        for s in range(3):
            b = 3 * lv + s
            pos[b] = (s - 1) * (width + g_lat) * ybody
            pos[b, 2] = height / 2 - DELTA0 + lv * (height - DELTA0)
            yaw[b] = psi
    return pos, yaw


_TOWER_CFG = {
    # cfg: (E, levels, iters, steps, jitter, max_removals, removal_levels, push k range, friction rule)
    1: dict(E=1, levels=3, iters=10, steps=240, max_rem=0, rem_levels=0, push=None, mu="fixed"),
    2: dict(E=450, levels=18, iters=20, steps=480, max_rem=12, rem_levels=15, push=(2.0, 5.0), mu="block150"),
    4: dict(E=4096, levels=30, iters=50, steps=480, max_rem=20, rem_levels=27, push=None, mu="draw"),
    5: dict(E=65536, levels=18, iters=20, steps=480, max_rem=12, rem_levels=15, push=(2.5, 4.5), mu="roundrobin"),
    # cfg6: the paper's own parameter set, App. A Table 6: 81 x 26 x 18 mm blocks of
    # 19.6 g, e = 0.10, three substeps, 14 PGS iterations; 450 episodes = 150 per friction level, the
    # removal / push recipe of cfg2.  Lateral play 1.5 mm (81 mm vs 3 x 26 mm); the jitter is halved
    # (+-0.25 mm, +-0.5 deg) so that neighbours cannot interpenetrate at t = 0 with that play.
    6: dict(E=450, levels=18, iters=14, steps=480, max_rem=12, rem_levels=15, push=(2.0, 5.0), mu="block150",
            size=(0.081, 0.026, 0.018), mass=0.0196, g_lat=0.0015, jitter_mm=0.25, jitter_deg=0.5, restitution=0.10, n_substeps=3),
}
MU_LEVELS = (0.25, 0.40, 0.60)
SETTLE_STEPS = 60
PUSH_STEPS = 24


def make_tower(cfg: int, n_envs: Optional[int] = None, env_offset: int = 0, jitter: bool = True) -> Workload:
    """Configs 1, 2, 4, 5 of BASELINE.json.  `n_envs`/`env_offset` select a slice of
    the config's envs (every env has its own RNG stream, so slices reproduce)."""
    c = _TOWER_CFG[cfg]
    E = c["E"] if n_envs is None else n_envs
    levels = c["levels"]
    B = 3 * levels
    state, props, S = empty_tiles(E, B)
    bl, bw, bh = c.get("size", (BLOCK_L, BLOCK_W, BLOCK_H))
    mass = c.get("mass", BLOCK_MASS)
    jit_pos, jit_yaw = 1.0e-3 * c.get("jitter_mm", 0.5), math.radians(c.get("jitter_deg", 1.0))
    nom_pos, nom_yaw = tower_nominal(levels, bw, bh, c.get("g_lat", G_LAT))
    inv_m, inv_I = box_mass_props(bl, bw, bh, mass)
    half = (bl / 2, bw / 2, bh / 2)
    mu = np.zeros(E)
    fext = np.zeros((E, FEXT_ROWS, S)) if c["push"] else None
    push_body = np.full(E, -1, dtype=np.int32)
    push_k = np.zeros(E)
    push_kthr = np.zeros(E)
    n_removed = np.zeros(E, dtype=np.int32)
    for e in range(E):
        env = e + env_offset
        rng = np.random.default_rng([283940 + cfg, env])
        # 1. jitter, body order
        jit = rng.uniform(-1.0, 1.0, size=(B, 3))
        if not jitter:
            jit[:] = 0.0
        px = nom_pos[:, 0] + jit_pos * jit[:, 0]
        py = nom_pos[:, 1] + jit_pos * jit[:, 1]
        yaw = nom_yaw + jit_yaw * jit[:, 2]
        state[e, 0, :B] = px
        state[e, 1, :B] = py
        state[e, 2, :B] = nom_pos[:, 2]
        state[e, 3, :B] = np.cos(yaw / 2)
        state[e, 6, :B] = np.sin(yaw / 2)
        props[e, 0, :B] = inv_m
        props[e, 1, :B], props[e, 2, :B], props[e, 3, :B] = inv_I
        props[e, 4, :B], props[e, 5, :B], props[e, 6, :B] = half
        props[e, 7, :B] = 1.0
        # 2. friction
        u_mu = rng.integers(0, 3)
        if c["mu"] == "fixed":
            mu[e] = 0.40
        elif c["mu"] == "block150":
            mu[e] = MU_LEVELS[min(env // 150, 2)]
        elif c["mu"] == "roundrobin":
            mu[e] = MU_LEVELS[env % 3]
        else:
            mu[e] = MU_LEVELS[int(u_mu)]
        # 3. removals
        removed = np.zeros(0, dtype=np.int64)
        if c["max_rem"] > 0:
            n_rem = int(rng.integers(0, c["max_rem"] + 1))
            removed = rng.choice(3 * c["rem_levels"], size=n_rem, replace=False)
            props[e, 7, removed] = 0.0
            n_removed[e] = n_rem
        # 4. push
        if c["push"]:
            cells = np.setdiff1d(np.arange(3 * c["rem_levels"]), removed)
            b = int(cells[rng.integers(0, len(cells))])
            u_kind, u_sign = rng.random(), rng.random()
            k = rng.uniform(*c["push"])
            slot = b % 3
            psi = yaw[b]
            along = np.array([math.cos(psi), math.sin(psi), 0.0])
            across = np.array([-math.sin(psi), math.cos(psi), 0.0])
            if slot == 1 or u_kind < 0.5:
                d = along * (1.0 if u_sign < 0.5 else -1.0)
                kthr = 3.0
            else:
                d = across * float(slot - 1)
                kthr = 4.0
            F = k * mu[e] * mass * GRAV
            fext[e, 0:3, b] = F * d
            push_body[e], push_k[e], push_kthr[e] = b, k, kthr
    params = WorldParams(n_envs=E, n_bodies=B, body_stride=S, pgs_iters=c["iters"],
                         restitution=f32(c.get("restitution", 0.0)), n_substeps=c.get("n_substeps", 1),
                         max_pairs=768 if B <= 54 else 1536,       # 54 blocks: <= 570 candidates / 171 colliding pairs seen in
                         max_contacts=704 if B <= 54 else 1216)    # collapses (156 standing); 90 blocks: > 768 / 269 (264 standing)
    return Workload(
        name=f"cfg{cfg}", params=params,
        state=state.astype(np.float32), props=props.astype(np.float32), mu=mu.astype(np.float32),
        n_steps=c["steps"],
        push_fext=None if fext is None else fext.astype(np.float32),
        push_start=SETTLE_STEPS, push_end=SETTLE_STEPS + PUSH_STEPS,
        push_body=push_body, push_k=push_k, push_kthr=push_kthr,
        meta=dict(cfg=cfg, levels=levels, n_removed=n_removed, env_offset=env_offset, block_length=bl, block_mass=mass))


def make_debris(n_envs: int = 4096, env_offset: int = 0, n_bodies: int = 54) -> Workload:
    """Config 3: blocks dropped from uniform positions in a 0.3x0.3x0.4 m box,
    uniform random quaternions, v ~ N(0, 0.2 m/s) per axis, no overlap rejection."""
    E, B = n_envs, n_bodies
    state, props, S = empty_tiles(E, B)
    inv_m, inv_I = box_mass_props(BLOCK_L, BLOCK_W, BLOCK_H, BLOCK_MASS)
    for e in range(E):
        rng = np.random.default_rng([283940 + 3, e + env_offset])
        state[e, 0, :B] = rng.uniform(-0.15, 0.15, B)
        state[e, 1, :B] = rng.uniform(-0.15, 0.15, B)
        state[e, 2, :B] = rng.uniform(0.05, 0.45, B)
        q = rng.standard_normal((B, 4))
        q /= np.linalg.norm(q, axis=1, keepdims=True)
        state[e, 3:7, :B] = q.T
        state[e, 7:10, :B] = 0.2 * rng.standard_normal((3, B))
        props[e, 0, :B] = inv_m
        props[e, 1, :B], props[e, 2, :B], props[e, 3, :B] = inv_I
        props[e, 4, :B], props[e, 5, :B], props[e, 6, :B] = BLOCK_L / 2, BLOCK_W / 2, BLOCK_H / 2
        props[e, 7, :B] = 1.0
    params = WorldParams(n_envs=E, n_bodies=B, body_stride=S, pgs_iters=20, max_pairs=512, max_contacts=704)   # seen: 235 candidates, 111 colliding pairs
    mu = np.full(E, 0.40)
    return Workload(name="cfg3", params=params, state=state.astype(np.float32), props=props.astype(np.float32),
                    mu=mu.astype(np.float32), n_steps=720, meta=dict(cfg=3, env_offset=env_offset))


def make_config(cfg: int, n_envs: Optional[int] = None, env_offset: int = 0) -> Workload:
    if cfg == 3:
        return make_debris(4096 if n_envs is None else n_envs, env_offset)
    return make_tower(cfg, n_envs, env_offset)


def make_custom(bodies, mu: float = 0.4, **param_overrides) -> Workload:
    """One env from an explicit body list (closed-form rigs in the tests).
    Each body: dict(pos, quat, size(l,w,h full), mass [or inv_m/inv_I], vel, omg, active)."""
    B = len(bodies)
    state, props, S = empty_tiles(1, B)
    for b, d in enumerate(bodies):
        l, w, h = d["size"]
        if "mass" in d:
            inv_m, inv_I = box_mass_props(l, w, h, d["mass"])
        else:
            inv_m, inv_I = d["inv_m"], d["inv_I"]
        set_body(state, props, 0, b, d["pos"], d.get("quat", (1, 0, 0, 0)), (l / 2, w / 2, h / 2),
                 inv_m, inv_I, d.get("vel", (0, 0, 0)), d.get("omg", (0, 0, 0)), d.get("active", 1.0))
    kw = dict(n_envs=1, n_bodies=B, body_stride=S, max_pairs=max(64, 2 * B * B), max_contacts=max(64, 4 * B * B))
    kw.update({k: (f32(v) if isinstance(v, float) else v) for k, v in param_overrides.items()})
    if "gravity" in kw:
        kw["gravity"] = tuple(f32(g) for g in kw["gravity"])
    params = WorldParams(**kw)
    return Workload(name="custom", params=params, state=state.astype(np.float32), props=props.astype(np.float32),
                    mu=np.array([mu], dtype=np.float32), n_steps=0)


def random_box_pairs(n: int, seed: int = 2839406):
    """Stage-test soup for the narrowphase: n box pairs (A at the origin region, B near it)
    with ~50 % overlapping.  Returns fp32 arrays xA,qA,hA,xB,qB,hB."""
    rng = np.random.default_rng(seed)
    half = np.array([BLOCK_L / 2, BLOCK_W / 2, BLOCK_H / 2])
    hA = np.tile(half, (n, 1)) * rng.uniform(0.6, 1.6, (n, 3))
    hB = np.tile(half, (n, 1)) * rng.uniform(0.6, 1.6, (n, 3))
    qA = rng.standard_normal((n, 4)); qA /= np.linalg.norm(qA, axis=1, keepdims=True)
    qB = rng.standard_normal((n, 4)); qB /= np.linalg.norm(qB, axis=1, keepdims=True)
    # a third of the pairs are near-aligned (tower-like), the rest fully random
    al = rng.random(n) < 0.33
    yawA = rng.uniform(-0.05, 0.05, n); yawB = rng.uniform(-0.05, 0.05, n) + (rng.random(n) < 0.5) * math.pi / 2
    qA[al] = np.stack([np.cos(yawA / 2), 0 * yawA, 0 * yawA, np.sin(yawA / 2)], 1)[al]
    qB[al] = np.stack([np.cos(yawB / 2), 0 * yawB, 0 * yawB, np.sin(yawB / 2)], 1)[al]
    xA = rng.uniform(-0.1, 0.1, (n, 3))
    dirn = rng.standard_normal((n, 3)); dirn /= np.linalg.norm(dirn, axis=1, keepdims=True)
    dist = rng.uniform(0.0, 0.07, (n, 1))
    xB = xA + dirn * dist
    return tuple(a.astype(np.float32) for a in (xA, qA, hA, xB, qB, hB))
