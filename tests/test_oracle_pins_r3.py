"""Pins for four parts of the oracle's step that no test reached before: Eq. 16 with a penetration above
the slop, restitution e > 0 in Eq. 14, the external-torque half of Eq. 5, and the gyroscopic term of Eq. 4; plus
SURVEY P7(v), kinetic energy never rises in a PGS row update with e = 0.  Every expectation below is a closed form or a
conservation law evaluated on the fp32-rounded inputs the oracle sees -- none re-types the oracle's code path.  CPU only.
"""
import math

import numpy as np
import pytest

from paper_2606_28394_b200 import workloads as W

L, Wd, H, M = W.BLOCK_L, W.BLOCK_W, W.BLOCK_H, W.BLOCK_MASS
ZERO_G = (0.0, 0.0, 0.0)


def block(pos, quat=(1, 0, 0, 0), **kw):
    d = dict(pos=pos, quat=quat, size=(L, Wd, H), mass=M)
    d.update(kw)
    return d


def world(orc, bodies, **kw):
    wl = W.make_custom(bodies, **kw)
    return orc.make_params(wl.params), orc.unpack_tiles(wl.state, wl.props, len(bodies))


# ----------------------------------------------------------------------------- Eq. 16, reading A14
@pytest.mark.parametrize("sink_mm", [1.0, 2.5])
def test_eq16_block_sunk_into_the_ground_rises_by_beta_times_excess(orc, sink_mm):
    """g = 0, v = 0: nothing but the position correction acts.  A block whose bottom face is delta below z = 0 moves up by
    beta (delta - slop) in one step (static ground: the whole correction goes to the block), x and y untouched."""
    P, bod = world(orc, [block((0, 0, H / 2 - sink_mm * 1e-3))], gravity=ZERO_G, mu=0.4)
    delta = bod.he[0, 0, 2] - bod.x[0, 0, 2]                     # depth of the four bottom corners, from the rounded inputs
    z0 = bod.x[0, 0].copy()
    orc.step_env(P, bod, 0.4)
    rise = bod.x[0, 0, 2] - z0[2]
    assert delta > P.slop and abs(rise - P.beta * (delta - P.slop)) < 1e-15
    assert abs(rise - 0.35 * (sink_mm * 1e-3 - 4e-4)) < 1e-8     # the paper's beta = 0.35, slop = 0.4 mm
    assert np.all(bod.x[0, 0, :2] == z0[:2]) and np.all(bod.v == 0) and np.all(bod.w == 0)
    assert np.allclose(bod.q[0, 0], [1, 0, 0, 0], atol=0)


def test_eq16_no_correction_at_or_below_the_slop(orc):
    for sink in (0.1e-3, 0.39e-3):
        P, bod = world(orc, [block((0, 0, H / 2 - sink))], gravity=ZERO_G)
        z0 = bod.x[0, 0, 2]
        orc.step_env(P, bod, 0.4)
        assert bod.x[0, 0, 2] == z0


def test_eq16_two_free_boxes_split_by_inverse_mass_once_per_pair(orc):
    """Masses m (below) and 3 m (above), faces overlapping by delta = 1 mm, no gravity, at rest.  The pair has a four-point
    face manifold; the correction is applied ONCE per pair (four times would be 4x too far), along -n for A and +n for B
    (n from A to B = +z), in the ratio of the inverse masses 3/4 : 1/4."""
    delta = 1.0e-3
    P, bod = world(orc, [block((0, 0, 1.0)), block((0, 0, 1.0 + H - delta), mass=3 * M)], gravity=ZERO_G)
    x0 = bod.x[0].copy()
    gap = (bod.he[0, 0, 2] + bod.he[0, 1, 2]) - (bod.x[0, 1, 2] - bod.x[0, 0, 2])      # the overlap the oracle sees
    tr = orc.step_env(P, bod, 0.4, trace=True)
    assert tr["contacts"].n == 4                                  # face-face: four points on the one pair
    s = P.beta * (gap - P.slop)
    ima, imb = bod.inv_m[0, 0], bod.inv_m[0, 1]
    dA, dB = bod.x[0, 0] - x0[0], bod.x[0, 1] - x0[1]
    assert abs(dA[2] + s * ima / (ima + imb)) < 1e-15 and abs(dB[2] - s * imb / (ima + imb)) < 1e-15
    assert abs(dA[2] / dB[2] + 3.0) < 1e-6                        # the light box moves three times as far, the other way
    assert abs((dB[2] - dA[2]) - 0.35 * (delta - 4e-4)) < 1e-7    # total separation gained = beta (delta - slop)
    assert np.all(dA[:2] == 0) and np.all(dB[:2] == 0)


# ----------------------------------------------------------------------------- Eq. 14 with e > 0, reading A11
@pytest.mark.parametrize("e_rest", [0.1, 0.5])
def test_eq14_restitution_reverses_the_current_normal_velocity_every_iteration(orc, e_rest):
    """One frictionless contact under the COM of a block approaching at v_n.  Eq. 14 as read (A11): every iteration applies
    -(1 + e) v_n / k_n on the CURRENT v_n, so after one iteration v_n' = -e v_n exactly and after k iterations (-e)^k v_n:
    the bounce is damped away by the sweeps (e = 0.1, 14 iterations: 1e-14 of v_n), which DESIGN §3 records."""
    vn = -0.3
    for iters in (1, 2, 3, 14):
        P, bod = world(orc, [block((0, 0, H / 2))], mu=0.0, warm_start=0, restitution=float(np.float32(e_rest)))
        bod.v[0, 0] = [0, 0, vn]
        c = orc.Contacts.from_arrays([0], [0], [15], [[0, 0, 1.0]], [[0, 0, 0.0]], [1e-4])
        lam, _, _ = orc.solve(P, bod, c, 0.0, iters=iters)
        e = P.restitution
        assert abs(e - e_rest) < 1e-7
        assert abs(bod.v[0, 0, 2] - (-e) ** iters * vn) < 1e-15, iters
        m = 1.0 / bod.inv_m[0, 0]
        assert abs(lam[0, 0] - m * (bod.v[0, 0, 2] - vn)) < 1e-15          # accumulated impulse = momentum change
        assert np.all(bod.w == 0) and np.all(bod.v[0, 0, :2] == 0)


# ----------------------------------------------------------------------------- external torque in S1 (Eq. 5)
def tilt():
    ax = np.array([1.0, 2.0, -0.5]); ax /= np.linalg.norm(ax)
    a = 0.9
    return (math.cos(a / 2), *(math.sin(a / 2) * ax))


def free_body(orc, **kw):
    """a tilted block far above the ground, no gravity: only what the test applies acts on it"""
    return world(orc, [block((0, 0, 5.0), quat=tilt())], gravity=ZERO_G, **kw)


def test_torque_about_a_principal_axis_spins_up_linearly(orc):
    """tau = tau0 a with a = the body's x axis in the world.  I_w^-1 a = a / I_xx (Eq. 3 + I_w^-1 = R I_b^-1 R^T), and a
    rotation about a leaves a where it is, so w(n) = n h tau0 / I_xx a for every n -- with the gyroscopic term on as well
    (w parallel to a principal axis: w x I w = 0)."""
    for gyro in (0, 1):
        P, bod = free_body(orc, gyroscopic=gyro)
        R = orc.quat_to_R(bod.q[0, 0]); a = R[:, 0].copy()
        tau0, n = 2.0e-4, 25
        f = np.zeros((1, 1, 6)); f[0, 0, 3:6] = tau0 * a
        for k in range(1, n + 1):
            orc.step_env(P, bod, 0.4, fext=f)
            expect = k * P.dt * tau0 * bod.inv_I[0, 0, 0] * a
            # 2e-7: the tilt quaternion is an fp32 input, unit to 6e-8 only, so R is orthogonal to that order
            assert np.max(np.abs(bod.w[0, 0] - expect)) < 2e-7 * np.linalg.norm(expect), (gyro, k)
        assert np.all(bod.v == 0) and np.all(bod.x[0, 0] == [0, 0, 5.0])   # a pure torque moves nothing
        # and the body has turned about a by the sum of the semi-implicit angles (Eq. 2: q from the NEW w)
        Rn = orc.quat_to_R(bod.q[0, 0])
        assert np.allclose(Rn[:, 0], a, atol=2e-7) and not np.allclose(Rn[:, 1], R[:, 1], atol=1e-2)


def test_general_torque_uses_the_world_inertia_of_the_tilted_body(orc):
    """first step from rest: w = h R diag(1/I) R^T tau.  With R transposed, or the body-frame inverse inertia used in the
    world frame, the result differs by tens of percent for this tilt."""
    P, bod = free_body(orc)
    R = orc.quat_to_R(bod.q[0, 0])
    tau = np.array([1.0e-4, -2.0e-4, 1.5e-4])
    f = np.zeros((1, 1, 6)); f[0, 0, 3:6] = tau
    orc.step_env(P, bod, 0.4, fext=f)
    expect = P.dt * R @ (bod.inv_I[0, 0] * (R.T @ tau))
    assert np.max(np.abs(bod.w[0, 0] - expect)) < 1e-13 * np.linalg.norm(expect)
    wrong = (P.dt * R.T @ (bod.inv_I[0, 0] * (R @ tau)), P.dt * bod.inv_I[0, 0] * tau)
    assert all(np.linalg.norm(w_ - expect) > 0.1 * np.linalg.norm(expect) for w_ in wrong)


# ----------------------------------------------------------------------------- gyroscopic term (Eq. 4), reading A4
def angular_momentum(orc, bod):
    R = orc.quat_to_R(bod.q[0, 0])
    return R @ ((R.T @ bod.w[0, 0]) / bod.inv_I[0, 0])            # L = R I_b R^T w


def test_gyroscopic_term_conserves_angular_momentum_of_a_free_body(orc):
    """Torque-free tumbling about a non-principal axis.  With gyroscopic = 1 (Eq. 4: I dw/dt = tau - w x I w) the world
    angular momentum L = I_w w is conserved up to the integrator's O(h) error; with the default gyroscopic = 0 (w is
    simply held, reading A4) L swings with the body's orientation.  Also: the first step's change of w is the closed form
    -h I_w^-1 (w x I_w w)."""
    w0 = np.array([6.0, 2.0, -3.0])
    drift = {}
    for gyro in (1, 0):
        P, bod = free_body(orc, gyroscopic=gyro)
        bod.w[0, 0] = w0
        L0 = angular_momentum(orc, bod)
        if gyro:
            R = orc.quat_to_R(bod.q[0, 0])
            dw = -P.dt * R @ (bod.inv_I[0, 0] * (R.T @ np.cross(w0, L0)))
        worst = 0.0
        for k in range(100):
            orc.step_env(P, bod, 0.4)
            if gyro and k == 0:
                assert np.max(np.abs(bod.w[0, 0] - (w0 + dw))) < 1e-13 * np.linalg.norm(w0)
                assert np.linalg.norm(dw) > 1e-3 * np.linalg.norm(w0)        # the term is not negligible here
            worst = max(worst, np.linalg.norm(angular_momentum(orc, bod) - L0) / np.linalg.norm(L0))
        drift[gyro] = worst
        if not gyro:
            assert np.all(bod.w[0, 0] == w0)                      # A4: without the term w is untouched by S1
    assert drift[1] < 0.05 and drift[0] > 0.5 and drift[0] > 10 * drift[1], drift


# ----------------------------------------------------------------------------- KE never rises in a row update (e = 0)
def kinetic_energy(orc, bod):
    ke = 0.0
    for b in range(bod.B):
        if bod.inv_m[0, b] == 0:
            continue
        R = orc.quat_to_R(bod.q[0, b]); wb = R.T @ bod.w[0, b]
        ke += 0.5 / bod.inv_m[0, b] * bod.v[0, b] @ bod.v[0, b] + 0.5 * np.sum(wb * wb / bod.inv_I[0, b])
    return ke


def test_P7v_kinetic_energy_never_rises_in_a_row_update(orc):
    """Eq. 14-15 with e = 0: each row update moves the impulse to the minimiser of the kinetic energy along that row's
    direction, or to the nearest admissible value -- never uphill.  Checked on 200 random two-body contacts from
    lambda = 0: with mu = 0 one sweep is the normal row alone; with mu > 0 it is the three rows of the contact in
    Listing 1's order (n, t1, t2); several sweeps keep going downhill."""
    rng = np.random.default_rng(28394)
    for trial in range(200):
        qa, qb = rng.standard_normal(4), rng.standard_normal(4)
        bodies = [block(tuple(rng.uniform(-0.02, 0.02, 3) + [0, 0, 1.0]), quat=tuple(qa / np.linalg.norm(qa))),
                  block(tuple(rng.uniform(-0.02, 0.02, 3) + [0, 0, 1.03]), quat=tuple(qb / np.linalg.norm(qb)), mass=M * rng.uniform(0.3, 3))]
        mu = 0.0 if trial % 2 == 0 else float(rng.uniform(0.2, 0.8))
        P, bod = world(orc, bodies, gravity=ZERO_G, warm_start=0)
        bod.v[0] = rng.standard_normal((2, 3)); bod.w[0] = 5 * rng.standard_normal((2, 3))
        n = rng.standard_normal(3); n /= np.linalg.norm(n)
        pt = 0.5 * (bod.x[0, 0] + bod.x[0, 1]) + rng.uniform(-0.02, 0.02, 3)
        pair = orc.pair_index(2, 0, 1)
        c = orc.Contacts.from_arrays([pair], [0], [0], [n], [pt], [1e-4])
        ke = kinetic_energy(orc, bod)
        lam, _, _ = orc.solve(P, bod, c, mu, iters=1)
        ke1 = kinetic_energy(orc, bod)
        assert ke1 <= ke * (1 + 1e-13), (trial, mu, ke, ke1)
        assert lam[0, 0] >= 0 and abs(lam[0, 1]) <= mu * lam[0, 0] + 1e-15 and abs(lam[0, 2]) <= mu * lam[0, 0] + 1e-15
    # the multi-sweep statement on one fixed case, velocities kept
    P, bod = world(orc, [block((0, 0, 1.0)), block((0.01, 0.0, 1.0 + H), mass=2 * M)], gravity=ZERO_G, warm_start=0)
    v0 = np.array([[0.3, -0.2, 0.5], [-0.1, 0.4, -0.6]]); w0 = np.array([[3.0, -2.0, 1.0], [0.5, 4.0, -1.0]])
    c = orc.Contacts.from_arrays([orc.pair_index(2, 0, 1)] * 2, [0, 1], [2, 2], [[0, 0, 1.0]] * 2,
                                 [[0.02, 0.01, 1.0 + H / 2], [-0.02, -0.01, 1.0 + H / 2]], [1e-4, 1e-4])
    kes = []
    for iters in (0, 1, 2, 3, 5, 8, 14):
        bod.v[0] = v0; bod.w[0] = w0
        orc.solve(P, bod, c, 0.5, iters=iters)
        kes.append(kinetic_energy(orc, bod))
    assert all(b <= a * (1 + 1e-13) for a, b in zip(kes, kes[1:])) and kes[-1] < 0.9 * kes[0], kes
