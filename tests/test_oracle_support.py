"""Pins of the NEXT-4 oracle functions: orc_support_margin (Eq. 17) against closed forms, a footprint
computed by hand, and the brute-force definition of a convex hull's supporting lines; orc_ziglar_block_analysis
(Table 1) against the table and the forces the paper prints (tests/golden/ziglar_forces.txt)."""
import math
import os

import numpy as np
import pytest

from paper_2606_28394_b200 import workloads as W

L_, W_, H_ = W.BLOCK_L, W.BLOCK_W, W.BLOCK_H
GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "ziglar_forces.txt")


def block(pos, yaw=0.0, mass=W.BLOCK_MASS, size=(L_, W_, H_), active=1.0, quat=None):
    q = (math.cos(yaw / 2), 0, 0, math.sin(yaw / 2)) if quat is None else quat
    return dict(pos=pos, quat=q, size=size, mass=mass, active=active)


def margin(orc, bodies):
    wl = W.make_custom(bodies)
    bod = orc.unpack_tiles(wl.state, wl.props, len(bodies))
    return orc.support_margin(bod, 0, eps=0.002)


def brute_margin(pts, c):
    """Definition: the hull's edges are the lines through two points with every other point on one side; the margin is the
    smallest signed distance of c to them (positive on the side of the points)."""
    best = math.inf
    n = len(pts)
    for i in range(n):
        for j in range(n):
            if i == j:
                continue
            e = pts[j] - pts[i]; ln = np.linalg.norm(e)
            if ln < 1e-12:
                continue
            nrm = np.array([-e[1], e[0]]) / ln                   # left normal
            s = (pts - pts[i]) @ nrm
            if np.all(s >= -1e-12):                              # supporting line, points to its left
                best = min(best, float((c - pts[i]) @ nrm))
    return best


def test_single_block_margin_is_its_half_width(orc):
    d, com, nh = margin(orc, [block((0.3, -0.2, H_ / 2))])
    assert nh == 4 and abs(d - W_ / 2) < 1e-9 and np.allclose(com, (0.3, -0.2), atol=1e-9)
    # yawed by 30 deg about z: same footprint rotated, same margin; COM off-centre by 5 mm along the width: margin shrinks by 5 mm
    d, _, _ = margin(orc, [block((0, 0, H_ / 2), yaw=math.radians(30))])
    assert abs(d - W_ / 2) < 1e-7
    # a block standing on its end: footprint w x h
    up = (math.cos(math.pi / 4), 0, math.sin(math.pi / 4), 0)        # 90 deg about y: length along z
    d, _, _ = margin(orc, [block((0, 0, L_ / 2), quat=up)])
    assert abs(d - H_ / 2) < 1e-7


def test_l_shaped_three_block_footprint_by_hand(orc):
    """Blocks A (along x, centre (0, 0)), B (along x, centre (0, 0.05)), C (along y, centre (0.06, 0.025)) on the ground, and
    a fourth block high above them (not on the ground) that only moves the COM.  Hull of the ground corners by hand:
    x in [-0.0375, 0.0725], y in [-0.0125, 0.0625] -- the C block's corners (0.0475..0.0725, -0.0125..0.0625) close the
    rectangle, so the hull is that rectangle.  COM = mean of the four centres (equal masses)."""
    A = block((0.0, 0.0, H_ / 2)); B = block((0.0, 0.05, H_ / 2)); Cb = block((0.06, 0.025, H_ / 2), yaw=math.pi / 2)
    top = block((0.02, 0.01, 0.2))
    d, com, nh = margin(orc, [A, B, Cb, top])
    cx, cy = (0 + 0 + 0.06 + 0.02) / 4, (0 + 0.05 + 0.025 + 0.01) / 4
    want = min(cx + 0.0375, 0.0725 - cx, cy + 0.0125, 0.0625 - cy)
    assert nh >= 4 and np.allclose(com, (cx, cy), atol=1e-8) and abs(d - want) < 1e-7      # (fp32-rounded yaw: near-collinear corners may add a vertex)
    # remove block C from the ground set by lifting it: the hull loses its right part (x <= 0.0375) and the margin follows
    d2, com2, _ = margin(orc, [A, B, block((0.06, 0.025, 0.1), yaw=math.pi / 2), top])
    want2 = min(cx + 0.0375, 0.0375 - cx, cy + 0.0125, 0.0625 - cy)
    assert abs(d2 - want2) < 1e-7 and np.allclose(com2, com)
    # an inactive body counts neither for the COM nor for the polygon; a heavier body pulls the COM
    d3, com3, _ = margin(orc, [A, B, block((0.06, 0.025, H_ / 2), yaw=math.pi / 2, active=0.0), block((0.02, 0.01, 0.2), mass=3 * W.BLOCK_MASS)])
    cx3, cy3 = (0 + 0 + 3 * 0.02) / 5, (0 + 0.05 + 3 * 0.01) / 5
    assert np.allclose(com3, (cx3, cy3), atol=1e-8) and abs(d3 - min(cx3 + 0.0375, 0.0375 - cx3, cy3 + 0.0125, 0.0625 - cy3)) < 1e-7


def test_com_outside_the_polygon_gives_a_negative_margin(orc):
    # a heavy block hanging in the air 10 cm to the side of a single supporting block
    d, com, _ = margin(orc, [block((0, 0, H_ / 2)), block((0.1, 0, 0.3), mass=9 * W.BLOCK_MASS)])
    assert abs(com[0] - 0.09) < 1e-8 and abs(d - (L_ / 2 - 0.09)) < 1e-7 and d < 0
    # nothing on the ground
    d, _, nh = margin(orc, [block((0, 0, 0.3))])
    assert nh == 0 and d < -1e29


@pytest.mark.parametrize("seed", range(6))
def test_margin_against_the_brute_force_hull_definition(orc, seed):
    """Random tumbled blocks, some on the ground: the margin equals the minimum over all supporting lines found by brute
    force over the same corner set (corners recomputed here from Rodrigues-free quaternion algebra in NumPy)."""
    rng = np.random.default_rng(seed)
    n = 7
    bodies = []
    for k in range(n):
        q = rng.standard_normal(4); q /= np.linalg.norm(q)
        z = rng.uniform(0.0, 0.08)
        bodies.append(block((rng.uniform(-0.1, 0.1), rng.uniform(-0.1, 0.1), z), quat=tuple(q)))
    wl = W.make_custom(bodies)
    bod = orc.unpack_tiles(wl.state, wl.props, n)
    d, com, nh = orc.support_margin(bod, 0, eps=0.002)
    pts = []
    for b in range(n):
        w, x, y, z = bod.q[0, b]
        R = np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                      [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                      [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])
        ez = np.abs(R[2]) @ bod.he[0, b]
        if bod.x[0, b, 2] - ez > 0.002:
            continue
        for sx in (-1, 1):
            for sy in (-1, 1):
                for sz in (-1, 1):
                    pts.append((bod.x[0, b] + R @ (np.array([sx, sy, sz]) * bod.he[0, b]))[:2])
    if not pts:
        assert nh == 0
        return
    pts = np.array(pts)
    c = bod.x[0, :, :2].mean(axis=0)
    assert np.allclose(com, c, atol=1e-12)
    assert abs(d - brute_margin(pts, c)) < 1e-9
    # invariance: translating everything leaves the margin unchanged
    bod.x[0, :, :2] += (0.37, -1.2)
    assert abs(orc.support_margin(bod, 0, eps=0.002)[0] - d) < 1e-9


def test_ziglar_block_analysis_is_table_1(orc):
    m, g = 0.0196, 9.81
    rows = {}
    for line in open(GOLD):
        if line.strip() and not line.startswith("#"):
            k, mu, f, tol = (float(t) for t in line.split())
            rows[(int(k), mu)] = (f, tol)
    for mu in (0.25, 0.40, 0.60):
        # (slot, axis) -> class, k, torque: centre block one row; side block along its length (Y) k = 3; across (X) k = 4 with torque
        for slot, axis, cls, k, tq in ((1, 0, 0, 3, False), (1, 1, 0, 3, False), (0, 0, 1, 3, False), (2, 0, 1, 3, False),
                                       (0, 1, 2, 4, True), (2, 1, 2, 4, True)):
            c, f, t = orc.ziglar_block_analysis(slot, axis, mu, m, g)
            want, tol = rows[(k, mu)]
            assert (c, t) == (cls, tq) and abs(1e3 * f - want) <= tol
