"""Pins of orc_collapse_test (Eq. 18, reading A17) from the mathematics, not from a restatement
of its formula: each of the three terms is driven through its threshold with a body whose displacement, rotation
or spin is constructed independently (axis-angle quaternions, Rodrigues' matrix, Eq. 3 moments), so that a wrong
frame, a dropped factor or a transposed rotation in any term fails one of these."""
import math

import numpy as np
import pytest

from paper_2606_28394_b200 import workloads as W

L_, W_, H_ = W.BLOCK_L, W.BLOCK_W, W.BLOCK_H
M = W.BLOCK_MASS
I_BODY = np.array([M / 12 * (W_ ** 2 + H_ ** 2), M / 12 * (L_ ** 2 + H_ ** 2), M / 12 * (L_ ** 2 + W_ ** 2)])   # Eq. 3


def quat_axis_angle(axis, angle):
    a = np.asarray(axis, float); a = a / np.linalg.norm(a)
    return np.concatenate([[math.cos(angle / 2)], math.sin(angle / 2) * a])


def quat_mul(p, q):
    pw, pv, qw, qv = p[0], p[1:], q[0], q[1:]
    return np.concatenate([[pw * qw - pv @ qv], pw * qv + qw * pv + np.cross(pv, qv)])


def rodrigues(axis, angle):
    a = np.asarray(axis, float); a = a / np.linalg.norm(a)
    K = np.array([[0, -a[2], a[1]], [a[2], 0, -a[0]], [-a[1], a[0], 0]])
    return np.eye(3) + math.sin(angle) * K + (1 - math.cos(angle)) * K @ K


def bodies(orc, n=3):
    """n blocks in a row, at rest; returns the oracle's Bodies view and the reference pose."""
    wl = W.make_custom([dict(pos=(0.2 * k, 0.0, 0.1), size=(L_, W_, H_), mass=M) for k in range(n)])
    bod = orc.unpack_tiles(wl.state, wl.props, n)
    return bod, bod.x[0].copy(), bod.q[0].copy()


def moved(orc, dx=0.0, angle=0.0, axis=(0.3, -0.5, 0.8), v=(0, 0, 0), w=(0, 0, 0), q_pre=None, body=1):
    bod, x0, q0 = bodies(orc)
    if q_pre is not None:                                   # start from a tilted reference orientation
        bod.q[0, body] = q_pre; q0[body] = q_pre
    d = np.array([0.6, -0.48, 0.64])                         # unit vector
    bod.x[0, body] += dx * d
    bod.q[0, body] = quat_mul(quat_axis_angle(axis, angle), bod.q[0, body])      # world-frame rotation by `angle`
    bod.v[0, body] = v; bod.w[0, body] = w
    flag, out = orc.collapse_test(bod, x0, q0, e=0, length=L_)
    return flag, out


def test_displacement_term_flips_at_half_a_block_length(orc):
    spin = (0.0, 0.0, 30.0)                                 # plenty of kinetic energy and 40 deg of rotation
    for sign, want in ((-1, False), (+1, True)):
        flag, out = moved(orc, dx=0.5 * L_ + sign * 1e-9, angle=math.radians(40), w=spin)
        assert flag is want and abs(out[0] - (0.5 * L_ + sign * 1e-9)) < 1e-12
    # the maximum over bodies, not the sum or the mean: a second body moved by less does not change it
    bod, x0, q0 = bodies(orc)
    bod.x[0, 0] += (0.01, 0, 0); bod.x[0, 2] += (0, 0.03, 0.04)
    assert abs(orc.collapse_test(bod, x0, q0, length=L_)[1][0] - 0.05) < 1e-15


@pytest.mark.parametrize("axis", [(0.3, -0.5, 0.8), (1, 0, 0), (0, 0, 1), (-0.7, 0.1, 0.2)])
def test_rotation_term_is_the_angle_of_the_relative_rotation(orc, axis):
    tilt = quat_axis_angle((0.2, 0.9, -0.4), 0.7)            # reference orientation is not the identity
    for sign, want in ((-1, False), (+1, True)):
        ang = math.radians(30) + sign * 1e-6
        flag, out = moved(orc, dx=0.6 * L_, angle=ang, axis=axis, w=(0, 20.0, 0), q_pre=tilt)
        assert flag is want and abs(out[2] - ang) < 1e-9
    # q and -q are the same rotation; angles beyond 180 deg fold back (2 acos |q . q0|)
    flag, out = moved(orc, angle=math.radians(200), axis=axis)
    assert abs(out[2] - math.radians(160)) < 1e-9


REL = 1e-6      # the mass properties reach the oracle as fp32-rounded inverses (the common input of both sides)


def close(a, b, rel=REL):
    return abs(a - b) <= rel * abs(b)


def test_kinetic_energy_is_half_m_v2_plus_half_w_I_w_in_the_body_frame(orc):
    # linear term
    _, out = moved(orc, v=(0.3, -0.4, 1.2))
    assert close(out[1], 0.5 * M * (0.09 + 0.16 + 1.44))
    # spin about each principal axis of an untilted block: 1/2 I_k w^2 with Eq. 3's moments
    for k in range(3):
        w = np.zeros(3); w[k] = 7.0
        _, out = moved(orc, w=w)
        assert close(out[1], 0.5 * I_BODY[k] * 49.0)
    # tilted block spinning about a WORLD axis: 1/2 w^T (R I R^T) w with R from Rodrigues' formula; a body-frame reading
    # of w, or R transposed, gives a different number (the three moments differ by up to 7x)
    axis, ang = (0.5, -0.3, 0.81), 1.1
    R = rodrigues(axis, ang)
    w = np.array([3.0, -5.0, 2.0])
    want = 0.5 * w @ (R @ np.diag(I_BODY) @ R.T) @ w
    wrong_frame = 0.5 * w @ np.diag(I_BODY) @ w
    wrong_transpose = 0.5 * w @ (R.T @ np.diag(I_BODY) @ R) @ w
    _, out = moved(orc, w=w, q_pre=quat_axis_angle(axis, ang))
    assert close(out[1], want) and abs(want - wrong_frame) > 0.05 * want and abs(want - wrong_transpose) > 0.05 * want
    # the sum over bodies; inactive and static bodies do not count
    bod, x0, q0 = bodies(orc)
    bod.v[0, 0] = (1, 0, 0); bod.v[0, 1] = (0, 2, 0); bod.v[0, 2] = (0, 0, 3)
    assert close(orc.collapse_test(bod, x0, q0, length=L_)[1][1], 0.5 * M * 14.0)
    bod.active[0, 2] = 0
    assert close(orc.collapse_test(bod, x0, q0, length=L_)[1][1], 0.5 * M * 5.0)


def test_energy_threshold_and_conjunction(orc):
    # E_k just below / above 5e-5 J with the other two conditions held
    for sign, want in ((-1, False), (+1, True)):
        v = math.sqrt(2 * 5e-5 * (1 + sign * 1e-5) / M)
        flag, out = moved(orc, dx=0.6 * L_, angle=math.radians(45), v=(0, v, 0))
        assert flag is want and close(out[1], 5e-5 * (1 + sign * 1e-5))
    # each condition alone, or any two, is not a collapse (Eq. 18 is a conjunction)
    assert not moved(orc, dx=L_, angle=math.radians(60))[0]
    assert not moved(orc, dx=L_, w=(0, 0, 50.0))[0]
    assert not moved(orc, angle=math.radians(60), w=(0, 0, 50.0))[0]


def test_rollout_latches_a_transient_collapse(orc):
    """The latch is an OR over the steps: a block thrown across the ground is 'collapsed' while it tumbles and stays
    latched after it has come to rest (E_k back below 5e-5 J)."""
    wl = W.make_custom([dict(pos=(0, 0, 0.04), size=(L_, W_, H_), mass=M, vel=(1.0, 0, 0), omg=(0, 25.0, 0))], mu=0.6)
    bod = orc.unpack_tiles(wl.state, wl.props, 1)
    x0, q0 = bod.x.copy(), bod.q.copy()
    P = orc.make_params(wl.params)
    flag = np.zeros(1, np.int32)
    orc.rollout(P, bod, wl.mu, 360, x0=x0, q0=q0, collapsed=flag, length=L_)
    now, out = orc.collapse_test(bod, x0[0], q0[0], e=0, length=L_)
    assert flag[0] == 1 and not now and out[1] < 5e-5 and out[0] > 0.5 * L_
