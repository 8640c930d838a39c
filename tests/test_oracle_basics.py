"""Pins P1-P4 of the oracle: closed forms and definitions.  CPU only."""
import math

import numpy as np
import pytest

from paper_2606_28394_b200 import workloads as W

L, Wd, H, M = W.BLOCK_L, W.BLOCK_W, W.BLOCK_H, W.BLOCK_MASS


def one_box(pos, quat=(1, 0, 0, 0), vel=(0, 0, 0), omg=(0, 0, 0), **kw):
    return W.make_custom([dict(pos=pos, quat=quat, size=(L, Wd, H), mass=M, vel=vel, omg=omg)], **kw)


def test_golden_ziglar_forces(orc):
    """F = k mu_s m g for m = 19.6 g (printed values, mN)."""
    rows = [l.split() for l in open(__file__.replace("test_oracle_basics.py", "golden/ziglar_forces.txt")) if l[0] != "#"]
    assert len(rows) == 6
    for k, mu, want_mN, tol in rows:
        got = orc.ziglar_force(float(k), float(mu), 0.0196, 9.81) * 1e3
        assert abs(got - float(want_mN)) <= float(tol), (k, mu, got)


def test_P3_inertia_closed_form_vs_volume_integration(orc):
    """Eq. 3 against a midpoint-rule integral of rho (r^2 d_ij - r_i r_j)."""
    m, l, w, h = 0.0196, 0.081, 0.026, 0.018       # paper's block
    I = orc.inertia_box(m, l, w, h)
    n = 60
    xs = (np.arange(n) + 0.5) / n - 0.5
    X, Y, Z = np.meshgrid(xs * l, xs * w, xs * h, indexing="ij")
    dm = m / n ** 3
    brute = np.array([np.sum(Y ** 2 + Z ** 2), np.sum(X ** 2 + Z ** 2), np.sum(X ** 2 + Y ** 2)]) * dm
    assert np.allclose(I, brute, rtol=1e-3)
    # distinguishes a swapped l/w/h: I_xx < I_yy < I_zz for l > w > h
    assert I[0] < I[1] < I[2]
    assert np.allclose(I, [1.633e-6, 1.1246e-5, 1.1820e-5], rtol=1e-3)   # SURVEY A1 (Eq. 3 evaluated)
    # the generator's props for the config block agree with the oracle's Eq. 3
    inv_m, inv_I = W.box_mass_props(L, Wd, H, M)
    assert np.allclose(1.0 / np.array(inv_I), orc.inertia_box(M, L, Wd, H), rtol=1e-14)


def test_quat_to_R_is_rotation_and_matches_axis_angle(orc):
    """Eq. 1 against Rodrigues' formula."""
    rng = np.random.default_rng(1)
    for _ in range(20):
        ax = rng.standard_normal(3); ax /= np.linalg.norm(ax)
        th = rng.uniform(-3, 3)
        q = np.concatenate([[math.cos(th / 2)], math.sin(th / 2) * ax])
        K = np.array([[0, -ax[2], ax[1]], [ax[2], 0, -ax[0]], [-ax[1], ax[0], 0]])
        Rr = np.eye(3) + math.sin(th) * K + (1 - math.cos(th)) * K @ K
        assert np.allclose(orc.quat_to_R(q), Rr, atol=1e-14)


def test_P1_free_fall_closed_form(orc):
    """Semi-implicit Euler (Eq. 5-6): v_n = -g n h, z_n = z0 - g h^2 n(n+1)/2."""
    wl = one_box((0.0, 0.0, 5.0))
    P = orc.make_params(wl.params)
    bod = orc.unpack_tiles(wl.state, wl.props, 1)
    h, g = P.dt, -P.g[2]
    for n in range(1, 241):
        orc.step_env(P, bod, 0.4)
        assert abs(bod.v[0, 0, 2] + g * n * h) < 1e-12
        assert abs(bod.x[0, 0, 2] - (5.0 - g * h * h * n * (n + 1) / 2)) < 1e-12
    assert np.all(bod.x[0, 0, :2] == 0) and np.all(bod.w == 0)


def test_P2_constant_omega_world_frame(orc):
    """Eq. 2 in the world-frame reading A3: each step rotates by
    2 atan(|w| h / 2) about the WORLD axis w/|w|; body pre-tilted so frames differ."""
    tilt = math.radians(30)
    q0 = np.array([math.cos(tilt / 2), math.sin(tilt / 2), 0, 0])     # 30 deg about x
    omg = np.array([0.0, 0.0, 3.0])                                    # about world z
    wl = one_box((0, 0, 5.0), quat=q0, omg=omg, gravity=(0.0, 0.0, 0.0))
    P = orc.make_params(wl.params)
    bod = orc.unpack_tiles(wl.state, wl.props, 1)
    q0 = bod.q[0, 0].copy(); R0 = orc.quat_to_R(q0)
    n = 100
    for _ in range(n):
        orc.step_env(P, bod, 0.4)
        assert abs(np.linalg.norm(bod.q[0, 0]) - 1) < 1e-14
    ang = n * 2 * math.atan(np.linalg.norm(omg) * P.dt / 2)
    Rz = np.array([[math.cos(ang), -math.sin(ang), 0], [math.sin(ang), math.cos(ang), 0], [0, 0, 1]])
    assert np.allclose(orc.quat_to_R(bod.q[0, 0]), Rz @ R0, atol=1e-7)
    # the body-frame reading would give R0 @ Rz instead; make sure the pin separates them
    assert not np.allclose(R0 @ Rz, Rz @ R0, atol=1e-3)
    assert np.allclose(bod.w[0, 0], omg)                                # no torque, no gyroscopic term (A4)


def _aabb(orc, x, q, he):
    R = orc.quat_to_R(q)
    ext = np.abs(R) @ he
    return x - ext, x + ext


def test_P4_broadphase_is_eq10_and_eq11(orc):
    """Eq. 10 vs the min/max form of Eq. 11 with boxes inflated by eps/2;
    ascending canonical order; translation invariance; superset of SAT-colliding pairs."""
    wl = W.make_debris(2)
    B = wl.params.n_bodies
    wl.params.max_pairs = 4000
    P = orc.make_params(wl.params)
    bod = orc.unpack_tiles(wl.state, wl.props, B)
    for e in range(2):
        pairs, st = orc.broadphase(P, bod, e)
        assert st == 0 and np.all(np.diff(pairs) > 0)
        want = []
        lo, hi = zip(*[_aabb(orc, bod.x[e, b], bod.q[e, b], bod.he[e, b]) for b in range(B)])
        lo, hi = np.array(lo) - P.aabb_margin / 2, np.array(hi) + P.aabb_margin / 2
        for b in range(B):
            if lo[b, 2] - P.aabb_margin / 2 <= 0:
                want.append(b)
        for i in range(B):
            for j in range(i + 1, B):
                if not (np.any(lo[i] > hi[j]) or np.any(hi[i] < lo[j])):          # Eq. 11
                    want.append(orc.pair_index(B, i, j))
        assert list(pairs) == want
        for p in pairs[:50]:
            i, j = orc.pair_bodies(B, p)
            assert orc.pair_index(B, i, j) == p and i < j
        # translation invariance (x, y only: the ground is at z = 0)
        b2 = bod.copy(); b2.x[e, :, :2] += np.array([0.37, -1.2])
        p2, _ = orc.broadphase(P, b2, e)
        assert list(p2) == list(pairs)
        # superset of SAT
        cset = set(pairs.tolist())
        for i in range(0, B, 3):
            for j in range(i + 1, B):
                r = orc.collide_boxes(P, bod.x[e, i], bod.q[e, i], bod.he[e, i], bod.x[e, j], bod.q[e, j], bod.he[e, j])
                if r["npts"] > 0:
                    assert orc.pair_index(B, i, j) in cset


def test_pair_index_is_dense_and_ascending(orc):
    B = 9
    seen = [orc.pair_index(B, -1, b) for b in range(B)]
    for i in range(B):
        for j in range(i + 1, B):
            seen.append(orc.pair_index(B, i, j))
    assert seen == list(range(B + B * (B - 1) // 2))


def test_inactive_bodies_never_appear(orc):
    wl = W.make_tower(2, 2)
    P = orc.make_params(wl.params)
    bod = orc.unpack_tiles(wl.state, wl.props, 54)
    for e in range(2):
        pairs, _ = orc.broadphase(P, bod, e)
        dead = set(np.nonzero(bod.active[e] == 0)[0].tolist())
        assert dead, "the seeded envs 0,1 of cfg 2 have removals"
        for p in pairs:
            i, j = orc.pair_bodies(54, p)
            assert i not in dead and j not in dead
