"""Pins P7-P10 of the oracle: PGS closed forms / LCP enumeration / order invariance, incline,
Ziglar rigs, resting tower, energy.  CPU only."""
import itertools
import math

import numpy as np
import pytest

from paper_2606_28394_b200 import workloads as W

L, Wd, H, M = W.BLOCK_L, W.BLOCK_W, W.BLOCK_H, W.BLOCK_MASS
G = W.GRAV
SLAB = 20.0      # ballast slab mass in block masses (P9 rig; 1e4 as SURVEY proposed does not converge in PGS)
SLAB_W = 2 * (W.G_LAT + Wd / 2) + 2.0e-3   # slab overlaps each side block on a 1 mm strip only: with wide patches the
                                            # P/Q load split is statically indeterminate (+-10 % seen) and moves the threshold


def block(pos, yaw=0.0, **kw):
    d = dict(pos=pos, quat=(math.cos(yaw / 2), 0, 0, math.sin(yaw / 2)), size=(L, Wd, H), mass=M)
    d.update(kw)
    return d


def kinetic_energy(orc, bod, e=0):
    ke = 0.0
    for b in range(bod.B):
        if not bod.active[e, b] or bod.inv_m[e, b] == 0:
            continue
        R = orc.quat_to_R(bod.q[e, b]); wb = R.T @ bod.w[e, b]
        ke += 0.5 / bod.inv_m[e, b] * bod.v[e, b] @ bod.v[e, b] + 0.5 * np.sum(wb * wb / bod.inv_I[e, b])
    return ke


def test_P7i_single_contact_one_iteration(orc):
    """one frictionless contact under the COM: one iteration gives jn = -vn/k_n = m |vn| and v -> 0 (Eq. 13-14)."""
    wl = W.make_custom([block((0, 0, H / 2))], mu=0.0, warm_start=0)
    P = orc.make_params(wl.params)
    bod = orc.unpack_tiles(wl.state, wl.props, 1)
    bod.v[0, 0] = [0, 0, -0.3]
    c = orc.Contacts.from_arrays([0], [0], [15], [[0, 0, 1.0]], [[0, 0, 0.0]], [1e-4])
    lam, col, st = orc.solve(P, bod, c, 0.0, iters=1)
    m = 1.0 / bod.inv_m[0, 0]                    # the fp32-rounded inverse mass the step sees
    assert abs(lam[0, 0] - m * 0.3) < 1e-15 and abs(bod.v[0, 0, 2]) < 1e-15 and np.all(bod.w == 0)
    # off-centre contact: k_n = 1/m + (r x n) . I^-1 (r x n)   (Eq. 13)
    bod.v[0, 0] = [0, 0, -0.3]; bod.w[:] = 0
    r = np.array([0.03, 0.0, -H / 2])
    c = orc.Contacts.from_arrays([0], [0], [15], [[0, 0, 1.0]], [r + bod.x[0, 0]], [1e-4])
    lam, _, _ = orc.solve(P, bod, c, 0.0, iters=1)
    rxn = np.cross(r, [0, 0, 1.0])
    kn = bod.inv_m[0, 0] + rxn @ (bod.inv_I[0, 0] * rxn)
    assert abs(lam[0, 0] - 0.3 / kn) < 1e-15
    vp = bod.v[0, 0] + np.cross(bod.w[0, 0], r)
    assert abs(vp[2]) < 1e-15                           # the contact point stopped approaching


def test_P7ii_box_on_ground_supports_its_weight(orc):
    for mu in (0.25, 0.6):
        wl = W.make_custom([block((0, 0, H / 2 - 1e-4))], mu=mu)
        P = orc.make_params(wl.params)
        bod = orc.unpack_tiles(wl.state, wl.props, 1)
        cache = orc.Cache(1, P.max_contacts)
        for s in range(30):
            tr = orc.step_env(P, bod, mu, cache=cache, trace=True)
            lam = tr["lam"]
            assert np.all(lam[:, 0] >= 0) and np.all(np.abs(lam[:, 1:]) <= mu * lam[:, :1] + 1e-18)   # Eq. 14-15
        assert tr["contacts"].n == 4
        assert abs(lam[:, 0].sum() + P.g[2] * P.dt / bod.inv_m[0, 0]) < 1e-9 and np.abs(bod.v).max() < 1e-9


def _lcp_velocities(Minv, J, v0):
    """frictionless contact LCP by active-set enumeration: find S with lam_S = -(A_SS)^-1 b_S >= 0 and
    (A lam + b)_notS >= 0; return v0 + Minv J^T lam (unique even if lam is not)."""
    A = J @ Minv @ J.T; b = J @ v0; n = len(b)
    for k in range(n + 1):
        for S in itertools.combinations(range(n), k):
            S = list(S); lam = np.zeros(n)
            if S:
                try:
                    lam[S] = np.linalg.lstsq(A[np.ix_(S, S)], -b[S], rcond=None)[0]
                except np.linalg.LinAlgError:
                    continue
            w = A @ lam + b
            if np.all(lam >= -1e-12) and np.all(w >= -1e-10) and np.all(np.abs(w[S]) < 1e-10 if S else True):
                return v0 + Minv @ J.T @ lam
    raise AssertionError("no active set found")


def test_P7iii_frictionless_pgs_converges_to_the_lcp_solution(orc):
    """two stacked boxes, 8 contacts, mu = 0, e = 0: 1e5 sweeps reach the LCP velocities found by
    enumerating active sets (velocities are unique; impulses need not be)."""
    rng = np.random.default_rng(3)
    for trial in range(4):
        wl = W.make_custom([block((0, 0, H / 2 - 1e-4)), block((0.004, 0.003, 1.5 * H - 2e-4), yaw=math.pi / 2 + 0.1)],
                           mu=0.0, warm_start=0)
        P = orc.make_params(wl.params)
        bod = orc.unpack_tiles(wl.state, wl.props, 2)
        pairs, _ = orc.broadphase(P, bod)
        cont, _ = orc.narrowphase(P, bod, pairs)
        assert cont.n == 8
        bod.v[0] = rng.normal(0, 0.3, (2, 3)) + [0, 0, -0.5]; bod.w[0] = rng.normal(0, 3.0, (2, 3))
        v0 = np.concatenate([bod.v[0, 0], bod.w[0, 0], bod.v[0, 1], bod.w[0, 1]])
        Iw = orc.world_inv_inertia(bod)
        Minv = np.zeros((12, 12))
        for b in range(2):
            Minv[6 * b:6 * b + 3, 6 * b:6 * b + 3] = np.eye(3) * bod.inv_m[0, b]
            Minv[6 * b + 3:6 * b + 6, 6 * b + 3:6 * b + 6] = Iw[b].reshape(3, 3)
        d = cont.trimmed(); J = np.zeros((8, 12))
        for c in range(8):
            i, j = orc.pair_bodies(2, d["pair"][c]); n = d["nrm"][c]
            J[c, 6 * j:6 * j + 3] = n; J[c, 6 * j + 3:6 * j + 6] = np.cross(d["pt"][c] - bod.x[0, j], n)
            if i >= 0:
                J[c, 6 * i:6 * i + 3] = -n; J[c, 6 * i + 3:6 * i + 6] = -np.cross(d["pt"][c] - bod.x[0, i], n)
        want = _lcp_velocities(Minv, J, v0)
        orc.solve(P, bod, cont, 0.0, iters=100000)
        got = np.concatenate([bod.v[0, 0], bod.w[0, 0], bod.v[0, 1], bod.w[0, 1]])
        assert np.allclose(got, want, atol=1e-8), trial


def _tower_contacts(orc, levels_cfg=2, n_env=1):
    wl = W.make_tower(levels_cfg, n_env)
    P = orc.make_params(wl.params)
    bod = orc.unpack_tiles(wl.state, wl.props, wl.params.n_bodies)
    pairs, _ = orc.broadphase(P, bod)
    cont, _ = orc.narrowphase(P, bod, pairs)
    bod.v[0, :, 2] += P.dt * P.g[2] * (bod.active[0] != 0)
    return wl, P, bod, cont


def test_colouring_is_greedy_and_proper(orc):
    wl, P, bod, cont = _tower_contacts(orc)
    d = cont.trimmed()
    pidx = np.unique(d["pair"])
    col, ncol, st = orc.colour_pairs(54, pidx, bod.inv_m[0])
    assert st == 0 and ncol == col.max() + 1 and ncol <= 12
    used = {}
    for p, c in zip(pidx, col):
        i, j = orc.pair_bodies(54, p)
        nb = [b for b in (i, j) if b >= 0]
        taken = set().union(*[used.get(b, set()) for b in nb])
        assert c not in taken                                   # proper
        assert all(k in taken for k in range(c))                # greedy: the lowest free colour
        for b in nb:
            used.setdefault(b, set()).add(int(c))


def test_P7iv_order_inside_a_colour_does_not_matter(orc):
    """pairs of one colour share no dynamic body, so any visiting order inside the colour gives
    bit-identical results (this is what lets the GPU solve a colour in parallel)."""
    wl, P, bod, cont = _tower_contacts(orc)
    npairs = len(np.unique(cont.trimmed()["pair"]))
    b1, b2 = bod.copy(), bod.copy()
    lam1, col1, _ = orc.solve(P, b1, cont, wl.mu[0], iters=5)
    perm = np.random.default_rng(0).permutation(npairs).astype(np.int32)
    lam2, col2, _ = orc.solve(P, b2, cont, wl.mu[0], iters=5, perm=perm)
    assert np.array_equal(lam1, lam2) and np.array_equal(b1.v, b2.v) and np.array_equal(b1.w, b2.w)
    assert np.array_equal(col1, col2) and lam1[:, 0].max() > 0


def test_P7vi_small_stack_converges_within_14_iterations(orc):
    """Fig. 3a: 14 iterations give < 1 % error on the normal impulse (2-body stack,
    cold start; a 3-body stack is at 4 % after 14 sweeps and needs the warm start of A12)."""
    bodies = [block((0, 0, H / 2 - 1e-4)), block((0, 0, 1.5 * H - 2e-4), yaw=math.pi / 2)]
    wl = W.make_custom(bodies, mu=0.4, warm_start=0)
    P = orc.make_params(wl.params)
    bod = orc.unpack_tiles(wl.state, wl.props, 2)
    pairs, _ = orc.broadphase(P, bod); cont, _ = orc.narrowphase(P, bod, pairs)
    bod.v[0, :, 2] = P.dt * P.g[2]
    ref = bod.copy(); lam_ref, _, _ = orc.solve(P, ref, cont, 0.4, iters=2000)
    b14 = bod.copy(); lam14, _, _ = orc.solve(P, b14, cont, 0.4, iters=14)
    pr = cont.trimmed()["pair"]
    for p in np.unique(pr):                                    # per-interface normal impulse
        a, b = lam14[pr == p, 0].sum(), lam_ref[pr == p, 0].sum()
        assert abs(a - b) <= 0.01 * b
    assert abs(lam_ref[pr < 2, 0].sum() + 2 * P.g[2] * P.dt / bod.inv_m[0, 0]) < 1e-9


def test_P10_kinetic_energy_non_increasing_without_push(orc):
    """zero gravity, e = 0: a collision never raises KE (each row update minimises KE along its row)."""
    rng = np.random.default_rng(11)
    for trial in range(5):
        bodies = [block((0, 0, 0.2), vel=tuple(rng.normal(0, 0.3, 3)), omg=tuple(rng.normal(0, 4, 3))),
                  block((0.01, 0.005, 0.2 + H - 3e-4), yaw=1.0, vel=tuple(rng.normal(0, 0.3, 3) - [0, 0, 0.4]),
                        omg=tuple(rng.normal(0, 4, 3)))]
        wl = W.make_custom(bodies, mu=0.5, gravity=(0.0, 0.0, 0.0), baumgarte_beta=0.0)
        P = orc.make_params(wl.params)
        bod = orc.unpack_tiles(wl.state, wl.props, 2)
        cache = orc.Cache(1, P.max_contacts)
        ke = kinetic_energy(orc, bod)
        hit = False
        for s in range(12):
            tr = orc.step_env(P, bod, 0.5, cache=cache, trace=True)
            hit |= tr["contacts"].n > 0
            ke2 = kinetic_energy(orc, bod)
            if s == 0:
                assert ke2 <= ke * (1 + 1e-12)          # first step has no warm start: strictly a projection
                ke_first = ke2
            ke = ke2
        assert hit and ke <= ke_first * 1.02             # later steps: warm-start re-application may wiggle by <2 %


def test_P8_incline_stick_slip(orc):
    """north_star: a block on an incline stays at rest iff tan(theta) <= mu_s; tilt gravity instead of the
    ground.  Along t1 (x) and t2 (y)."""
    for mu in (0.25, 0.4, 0.6):
        for ax in (0, 1):
            for fac, slides in ((0.95, False), (1.05, True)):
                th = math.atan(fac * mu)
                g = [0.0, 0.0, -G * math.cos(th)]; g[ax] = G * math.sin(th)
                wl = W.make_custom([block((0, 0, H / 2 - 1e-4))], mu=mu, gravity=tuple(g))
                P = orc.make_params(wl.params)
                bod = orc.unpack_tiles(wl.state, wl.props, 1)
                cache = orc.Cache(1, P.max_contacts)
                orc.rollout(P, bod, [mu], 240, cache=cache)
                disp = bod.x[0, 0, ax]
                if not slides:
                    assert abs(disp) < 1e-4, (mu, ax, fac, disp)
                else:
                    a = G * (math.sin(th) - mu * math.cos(th))
                    want = 0.5 * a * 1.0 ** 2
                    assert abs(disp - want) < 0.05 * want + 2e-4, (mu, ax, fac, disp, want)


def _rig(mu, Wfac, axis, kfac):
    """SURVEY P9 determinate rig: side blocks P, Q on the ground, ballast slab T (mass 1e4 m) on top with an
    upward force so that its net weight is W = Wfac m g; P is pushed with k mu (W + m g)."""
    off = Wd + W.G_LAT
    slab = dict(pos=(0, 0, 1.5 * H - 2e-4), quat=(1, 0, 0, 0), size=(L, SLAB_W, H), mass=SLAB * M)
    bodies = [block((0, -off, H / 2 - 1e-4)), block((0, +off, H / 2 - 1e-4)), slab]
    wl = W.make_custom(bodies, mu=mu, pgs_iters=60)
    f = np.zeros((1, 3, 6))
    f[0, 2, 2] = SLAB * M * G - Wfac * M * G
    push = np.zeros((1, 3, 6))
    F = kfac * mu * (Wfac + 1.0) * M * G
    push[0, 0, 0 if axis == "along" else 1] = F if axis == "along" else -F      # across: outward (-y for P)
    return wl, f, f + push


@pytest.mark.parametrize("mu", [0.25, 0.40, 0.60])
@pytest.mark.parametrize("Wfac,axis", [(2.0, "along"), (3.0, "across")])
def test_P9_ziglar_rigs(orc, mu, Wfac, axis):
    """north_star: a side push at 0.9x the Ziglar force (3 mu m g along the length = the paper's Y,
    4 mu m g across = the paper's X) leaves the block static, 1.1x slides it."""
    kz = Wfac + 1.0
    assert abs(orc.ziglar_force(kz, mu, M, G) - mu * (Wfac + 1) * M * G) < 1e-15
    for kfac, slides in ((0.9, False), (1.1, True)):
        wl, f_hold, f_push = _rig(mu, Wfac, axis, kfac)
        P = orc.make_params(wl.params)
        bod = orc.unpack_tiles(wl.state, wl.props, 3)
        cache = orc.Cache(1, P.max_contacts)
        orc.rollout(P, bod, [mu], 60, fext=f_hold, cache=cache)
        x0 = bod.x.copy()
        orc.rollout(P, bod, [mu], 24, fext=f_push, cache=cache)
        orc.rollout(P, bod, [mu], 120, fext=f_hold, cache=cache)
        moved = np.linalg.norm(bod.x[0, 0] - x0[0, 0])
        if slides:
            assert moved > 1e-3, (mu, axis, moved)
        else:
            assert moved < 1e-4, (mu, axis, moved)
        assert np.linalg.norm(bod.x[0, 1] - x0[0, 1]) < 1e-4          # the other side block stays


def test_P10_resting_tower_drift(orc):
    """north_star: a resting 18-level tower drifts < 0.5 mm over 2 s (after the 60-step warm-start
    transient), 20 iterations, n_sub = 1; and the paper's own n_sub = 3 / 14 iterations."""
    for kw, lim in ((dict(), 0.5e-3), (dict(n_substeps=3, pgs_iters=14), 0.2e-3)):
        wl = W.make_tower(2, 1, jitter=False)
        wl.props[:, 7, :54] = 1.0
        for k, v in kw.items():
            setattr(wl.params, k, v)
        P = orc.make_params(wl.params)
        bod = orc.unpack_tiles(wl.state, wl.props, 54)
        cache = orc.Cache(1, P.max_contacts)
        orc.rollout(P, bod, wl.mu, 60, cache=cache)
        x60 = bod.x.copy()
        st = orc.rollout(P, bod, wl.mu, 480, cache=cache)
        assert st[0] == 0
        assert np.linalg.norm(bod.x - x60, axis=2).max() < lim


def test_until_rest_sliding_block_closed_form(orc):
    """simulate_until_rest: a block sliding on the ground with speed v0 decelerates with mu g, so
    it is at rest (E_k < 1e-7 J) after ceil(v0 / (mu g h)) steps up to the E_k threshold; a block already at rest
    takes exactly one step; an airborne block runs into the step limit."""
    mu, v0 = 0.4, 0.30
    h = W.f32(1.0 / 240.0)
    wl = W.make_custom([dict(pos=(0, 0, W.BLOCK_H / 2 - 1e-4), size=(W.BLOCK_L, W.BLOCK_W, W.BLOCK_H), mass=W.BLOCK_MASS, vel=(v0, 0, 0))], mu=mu)
    P = orc.make_params(wl.params); bod = orc.unpack_tiles(wl.state, wl.props, 1)
    steps, ek, _ = orc.rollout_until_rest(P, bod, wl.mu, max_steps=400, ek_rest=1e-7)
    n_stop = v0 / (mu * 9.81 * h)                      # steps until Coulomb friction has removed v0
    assert abs(steps[0] - n_stop) <= 3 and ek[0] < 1e-7, (steps, n_stop, ek)
    assert abs(bod.x[0, 0, 0] - v0 * v0 / (2 * mu * 9.81)) < 2e-3       # stopping distance v0^2 / (2 mu g)
    steps2, ek2, _ = orc.rollout_until_rest(P, bod, wl.mu, max_steps=400, ek_rest=1e-7)   # now at rest
    assert steps2[0] == 1 and ek2[0] < 1e-7
    air = W.make_custom([dict(pos=(0, 0, 5.0), size=(W.BLOCK_L, W.BLOCK_W, W.BLOCK_H), mass=W.BLOCK_MASS)])
    b3 = orc.unpack_tiles(air.state, air.props, 1)
    steps3, ek3, _ = orc.rollout_until_rest(orc.make_params(air.params), b3, air.mu, max_steps=50, ek_rest=1e-7)
    assert steps3[0] == 50 and abs(ek3[0] - 0.5 * W.BLOCK_MASS * (9.81 * 50 * h) ** 2) < 1e-4 * ek3[0] + 1e-9
