"""Pins P5-P6 of the oracle: SAT classification vs brute force, manifold vs closed forms.  CPU only."""
import itertools
import math

import numpy as np
import pytest

from paper_2606_28394_b200 import workloads as W

L, Wd, H = W.BLOCK_L, W.BLOCK_W, W.BLOCK_H


def params(orc):
    return orc.make_params(W.WorldParams(1, 2, 4))


def soup(n, seed=2839406):
    """the fp32 stage-test soup widened to fp64 with quaternions re-normalised in fp64, so that
    exact invariants (unit normal, point containment) can be asserted to 1e-12."""
    xA, qA, hA, xB, qB, hB = [a.astype(np.float64) for a in W.random_box_pairs(n, seed)]
    qA /= np.linalg.norm(qA, axis=1, keepdims=True); qB /= np.linalg.norm(qB, axis=1, keepdims=True)
    return xA, qA, hA, xB, qB, hB


# ---------------- independent brute-force overlap test (no separating axes) ----------------
_SIGNS = np.array(list(itertools.product((-1, 1), repeat=3)), dtype=float)
_EDGES = [(a, b) for a in range(8) for b in range(a + 1, 8) if np.sum(_SIGNS[a] != _SIGNS[b]) == 1]


def _verts(x, R, h):
    return x + (_SIGNS * h) @ R.T


def _seg_hits_box(p0, p1, x, R, h):
    """does the segment cross any face rectangle of the box (x,R,h)?  (local frame slab test per face)"""
    a, b = (p0 - x) @ R, (p1 - x) @ R
    for k in range(3):
        for s in (-1.0, 1.0):
            da, db = a[k] - s * h[k], b[k] - s * h[k]
            if da * db > 0 or da == db:
                continue
            t = da / (da - db)
            q = a + t * (b - a)
            o = [i for i in range(3) if i != k]
            if abs(q[o[0]]) <= h[o[0]] and abs(q[o[1]]) <= h[o[1]]:
                return True
    return False


def brute_overlap(xA, RA, hA, xB, RB, hB):
    vA, vB = _verts(xA, RA, hA), _verts(xB, RB, hB)
    if np.any(np.all(np.abs((vA - xB) @ RB) <= hB, axis=1)) or np.any(np.all(np.abs((vB - xA) @ RA) <= hA, axis=1)):
        return True
    for a, b in _EDGES:
        if _seg_hits_box(vA[a], vA[b], xB, RB, hB) or _seg_hits_box(vB[a], vB[b], xA, RA, hA):
            return True
    return False


def test_P5_sat_classification_matches_brute_force(orc):
    """north_star: SAT overlap classification agrees with brute-force vertex / edge-face queries."""
    P = params(orc)
    xA, qA, hA, xB, qB, hB = soup(3000)
    n_checked = n_hit = 0
    for k in range(len(xA)):
        mg = orc.OrcMargins(); mg.reset()
        r = orc.collide_boxes(P, xA[k], qA[k], hA[k], xB[k], qB[k], hB[k], mg)
        if mg.sat_sign < 1e-5:
            continue                       # |delta_min| >= 1e-5 m guard band
        want = brute_overlap(xA[k], orc.quat_to_R(qA[k]), hA[k], xB[k], orc.quat_to_R(qB[k]), hB[k])
        assert (r["npts"] > 0) == want, k
        n_checked += 1; n_hit += want
    assert n_checked > 2500 and 0.25 < n_hit / n_checked < 0.75


def test_P5_sat_invariants(orc):
    P = params(orc)
    xA, qA, hA, xB, qB, hB = soup(600, seed=5)
    done = 0
    for k in range(len(xA)):
        mg = orc.OrcMargins(); mg.reset()
        r = orc.collide_boxes(P, xA[k], qA[k], hA[k], xB[k], qB[k], hB[k], mg)
        if r["npts"] == 0 or min(mg.sat_sign, mg.axis_choice) < 1e-6:
            continue
        n, d = r["n"], r["sat_depth"]
        assert abs(np.linalg.norm(n) - 1) < 1e-12 and n @ (xB[k] - xA[k]) >= 0
        # moving B by (depth + tiny) along n separates the boxes; moving it by less than the
        # face-preference line (A7: every axis has delta >= 0.95 d - 1e-4 - tie) does not
        assert orc.collide_boxes(P, xA[k], qA[k], hA[k], xB[k] + (d + 1e-9) * n, qB[k], hB[k])["npts"] == 0
        s_in = 0.94 * d - 1.1e-4
        if s_in > 0:
            assert orc.collide_boxes(P, xA[k], qA[k], hA[k], xB[k] + s_in * n, qB[k], hB[k])["npts"] > 0
        # swapping A and B flips n and keeps the depth
        s = orc.collide_boxes(P, xB[k], qB[k], hB[k], xA[k], qA[k], hA[k])
        assert np.allclose(s["n"], -n, atol=1e-12) and abs(s["sat_depth"] - d) < 1e-12
        assert 1 <= r["npts"] <= 4
        assert np.all(r["depths"] >= 0) and np.all(r["depths"] <= d + 1e-12)
        # mid-surface points: within depth/2 of both boxes (face case); edge case: between the edges
        for p, dp_ in zip(r["pts"], r["depths"]):
            tol = (dp_ / 2 if r["axis"] < 6 else d) + 1e-9
            assert np.all(np.abs((p - xA[k]) @ orc.quat_to_R(qA[k])) <= hA[k] + tol)
            assert np.all(np.abs((p - xB[k]) @ orc.quat_to_R(qB[k])) <= hB[k] + tol)
        done += 1
    assert done > 150


def test_P5_axis_aligned_reduces_to_interval_overlap(orc):
    P = params(orc)
    q = np.array([1.0, 0, 0, 0])
    hA, hB = np.array([0.03, 0.02, 0.01]), np.array([0.015, 0.025, 0.02])
    for t in ([0.04, 0.0, 0.0], [0.0, -0.043, 0.001], [0.001, 0.002, 0.0295], [0.05, 0.0, 0.0]):
        t = np.array(t)
        ov = hA + hB - np.abs(t)
        r = orc.collide_boxes(P, np.zeros(3), q, hA, t, q, hB)
        if np.any(ov <= 0):
            assert r["npts"] == 0
        else:
            k = int(np.argmin(ov))
            assert r["axis"] == k and abs(r["sat_depth"] - ov[k]) < 1e-15
            assert np.allclose(r["n"], np.sign(t[k]) * np.eye(3)[k])


# ---------------- P6: manifold ----------------
def _rect_intersection(c1, psi1, h1, c2, psi2, h2):
    """independent 2-D convex intersection of two rectangles: candidate-vertex enumeration."""
    def corners(c, psi, h):
        u = np.array([math.cos(psi), math.sin(psi)]); v = np.array([-u[1], u[0]])
        return [c + sx * h[0] * u + sy * h[1] * v for sx, sy in ((-1, -1), (1, -1), (1, 1), (-1, 1))]

    def inside(p, c, psi, h):
        u = np.array([math.cos(psi), math.sin(psi)]); v = np.array([-u[1], u[0]])
        d = p - c
        return abs(d @ u) <= h[0] + 1e-12 and abs(d @ v) <= h[1] + 1e-12
    A, B = corners(c1, psi1, h1), corners(c2, psi2, h2)
    out = [p for p in A if inside(p, c2, psi2, h2)] + [p for p in B if inside(p, c1, psi1, h1)]
    for i in range(4):
        for j in range(4):
            p, r = A[i], A[(i + 1) % 4] - A[i]
            q, s = B[j], B[(j + 1) % 4] - B[j]
            den = r[0] * s[1] - r[1] * s[0]
            if abs(den) < 1e-15:
                continue
            t = ((q - p)[0] * s[1] - (q - p)[1] * s[0]) / den
            u = ((q - p)[0] * r[1] - (q - p)[1] * r[0]) / den
            if 0 <= t <= 1 and 0 <= u <= 1:
                out.append(p + t * r)
    return np.array(out)


def test_P6_tower_pair_closed_form(orc):
    """upper block across lower block, no yaw: the four corners of the 25 x 25 mm overlap square,
    at mid-depth, depth = z overlap."""
    P = params(orc)
    he = np.array([L / 2, Wd / 2, H / 2])
    ov = 1.0e-4
    xA, qA = np.zeros(3), np.array([1.0, 0, 0, 0])
    xB, qB = np.array([0.0, 0.0, H - ov]), np.array([math.cos(math.pi / 4), 0, 0, math.sin(math.pi / 4)])
    r = orc.collide_boxes(P, xA, qA, he, xB, qB, he)
    assert r["npts"] == 4 and r["axis"] == 2
    assert np.allclose(r["n"], [0, 0, 1], atol=1e-15) and abs(r["sat_depth"] - ov) < 1e-15
    assert np.allclose(r["depths"], ov, atol=1e-15)
    got = sorted(map(tuple, np.round(r["pts"], 12)))
    want = sorted((sx * Wd / 2, sy * Wd / 2, round(H / 2 - ov / 2, 12)) for sx in (-1, 1) for sy in (-1, 1))
    assert np.allclose(got, want, atol=1e-12)


def test_P6_yawed_faces_match_independent_rectangle_intersection(orc):
    P = params(orc)
    he = np.array([L / 2, Wd / 2, H / 2])
    rng = np.random.default_rng(7)
    n4 = nbig = 0
    for _ in range(200):
        psiA, psiB = rng.uniform(-math.pi, math.pi, 2)
        cB = rng.uniform(-0.03, 0.03, 2)
        ov = rng.uniform(5e-5, 5e-4)
        qA = np.array([math.cos(psiA / 2), 0, 0, math.sin(psiA / 2)])
        qB = np.array([math.cos(psiB / 2), 0, 0, math.sin(psiB / 2)])
        xB = np.array([cB[0], cB[1], H - ov])
        mg = orc.OrcMargins(); mg.reset()
        r = orc.collide_boxes(P, np.zeros(3), qA, he, xB, qB, he, mg)
        poly = _rect_intersection(np.zeros(2), psiA, he[:2], cB, psiB, he[:2])
        if len(poly) == 0:
            assert r["npts"] == 0
            continue
        if mg.clip < 1e-7:
            continue
        assert r["axis"] in (2, 5) and np.allclose(r["depths"], ov, atol=1e-12)
        assert np.allclose(r["pts"][:, 2], H / 2 - ov / 2, atol=1e-12)
        # de-duplicate the brute-force vertex list
        uniq = []
        for p in poly:
            if not any(np.linalg.norm(p - u) < 1e-9 for u in uniq):
                uniq.append(p)
        for p in r["pts"]:
            assert min(np.linalg.norm(p[:2] - u) for u in uniq) < 1e-9       # every contact is a true vertex
        if len(uniq) <= 4:
            assert r["npts"] == len(uniq); n4 += 1
        else:
            assert r["npts"] in (3, 4); nbig += 1
    assert n4 > 30 and nbig > 30


def test_P6_ground_contacts(orc):
    he = np.array([L / 2, Wd / 2, H / 2])
    r = orc.collide_ground(np.array([0.1, 0.2, H / 2 - 2e-4]), np.array([1.0, 0, 0, 0]), he)
    assert r["npts"] == 4 and np.allclose(r["depths"], 2e-4, atol=1e-15)
    assert np.allclose(r["pts"][:, 2], -1e-4, atol=1e-15)
    assert np.allclose(sorted(r["pts"][:, 0]), [0.1 - L / 2] * 2 + [0.1 + L / 2] * 2)
    # standing on an edge: two corners
    th = math.radians(20)
    q = np.array([math.cos(th / 2), math.sin(th / 2), 0, 0])
    zc = he[1] * math.sin(th) + he[2] * math.cos(th) - 1e-4
    r = orc.collide_ground(np.array([0.0, 0.0, zc]), q, he)
    assert r["npts"] == 2 and np.allclose(r["depths"], 1e-4, atol=1e-12)
    # floating: none; deeply sunk: the 4 deepest of 8
    assert orc.collide_ground(np.array([0.0, 0.0, 0.1]), q, he)["npts"] == 0
    r = orc.collide_ground(np.array([0.0, 0.0, -0.1]), q, he)
    assert r["npts"] == 4 and r["depths"].min() > 0.1


def test_edge_edge_contact_is_between_the_edges(orc):
    """two crossed boxes touching edge to edge (A8): one contact midway between the closest points."""
    P = params(orc)
    he = np.array([0.05, 0.01, 0.01])
    qa = np.array([math.cos(math.pi / 8), math.sin(math.pi / 8), 0, 0])       # A rolled 45 deg about x
    # B along y, rolled 45 deg about its own long axis: q = rot_z(90) * rot_x(45)
    cz, sz, cx, sx = math.cos(math.pi / 4), math.sin(math.pi / 4), math.cos(math.pi / 8), math.sin(math.pi / 8)
    qb = np.array([cz * cx, cz * sx, sz * sx, sz * cx])
    diag = 0.01 * math.sqrt(2)
    d = 3e-4
    xB = np.array([0.0, 0.0, 2 * diag - d])
    r = orc.collide_boxes(P, np.zeros(3), qa, he, xB, qb, he)
    assert r["axis"] == 6 and r["npts"] == 1
    assert np.allclose(r["n"], [0, 0, 1], atol=1e-12) and abs(r["sat_depth"] - d) < 1e-12
    assert np.allclose(r["pts"][0], [0, 0, diag - d / 2], atol=1e-12)
