// collide.cuh -- per-thread narrowphase of the batched Jenga step (fp32, sm_100a).
//
// S3 of DESIGN.md §2: 15-axis OBB-OBB separating-axis test (§6.2) and the
// contact manifold (§6.2.1, read as reference/incident face clipping with
// per-point depth, DESIGN.md §3 reading A8), plus box-vs-ground-plane corners (reading A9).
// One thread handles one candidate pair; all state is in registers / thread-local arrays.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace jenga {

struct Vec3 { float x, y, z; };

__device__ __forceinline__ Vec3 v3(float x, float y, float z) { Vec3 r; r.x = x; r.y = y; r.z = z; return r; }
__device__ __forceinline__ Vec3 operator+(Vec3 a, Vec3 b) { return v3(a.x + b.x, a.y + b.y, a.z + b.z); }
__device__ __forceinline__ Vec3 operator-(Vec3 a, Vec3 b) { return v3(a.x - b.x, a.y - b.y, a.z - b.z); }
__device__ __forceinline__ Vec3 operator-(Vec3 a) { return v3(-a.x, -a.y, -a.z); }
__device__ __forceinline__ Vec3 operator*(float s, Vec3 a) { return v3(s * a.x, s * a.y, s * a.z); }
__device__ __forceinline__ float dot(Vec3 a, Vec3 b) { return fmaf(a.x, b.x, fmaf(a.y, b.y, a.z * b.z)); }
__device__ __forceinline__ Vec3 cross(Vec3 a, Vec3 b) {
  return v3(fmaf(a.y, b.z, -a.z * b.y), fmaf(a.z, b.x, -a.x * b.z), fmaf(a.x, b.y, -a.y * b.x));
}
__device__ __forceinline__ Vec3 madd(Vec3 a, float s, Vec3 b) {      // a + s b
  return v3(fmaf(s, b.x, a.x), fmaf(s, b.y, a.y), fmaf(s, b.z, a.z));
}
__device__ __forceinline__ float comp(Vec3 a, int k) { return k == 0 ? a.x : (k == 1 ? a.y : a.z); }

// An oriented box: centre, the three body axes in world coordinates (columns of R, Eq. 1
// PAPER.md:147) and the half extents along them.
struct Box {
  Vec3 c;
  Vec3 ax[3];
  float he[3];
};

struct Manifold {
  int   np;        // 0 = not colliding
  int   axis;      // SAT axis id 0..14, 15 = ground
  Vec3  n;         // A -> B
  Vec3  p[4];
  float d[4];
};

struct CollideParams {
  float edge_bias_rel, edge_bias_abs, par_eps, tie_eps;
};

// ---------------------------------------------------------------- ground plane (reading A9)
// Corners below z = 0 are contacts: n = +z, depth = -z, point at mid-surface (cx, cy, z/2).
// More than four: drop the shallowest (ties: the higher corner id goes) until four remain.
__device__ inline void collide_ground(const Box& b, Manifold& m) {
  float cz[8]; float cx[8], cy[8];
  unsigned ok = 0; int nq = 0;
#pragma unroll
  for (int id = 0; id < 8; ++id) {
    float sx = (id & 1) ? b.he[0] : -b.he[0], sy = (id & 2) ? b.he[1] : -b.he[1], sz = (id & 4) ? b.he[2] : -b.he[2];
    Vec3 o = madd(madd(sx * b.ax[0], sy, b.ax[1]), sz, b.ax[2]);
    cx[id] = b.c.x + o.x; cy[id] = b.c.y + o.y; cz[id] = b.c.z + o.z;
    if (cz[id] < 0.0f) { ok |= 1u << id; ++nq; }
  }
  while (nq > 4) {
    int worst = -1; float wd = 0.0f;
#pragma unroll
    for (int id = 0; id < 8; ++id)
      if ((ok >> id) & 1u) { float dd = -cz[id]; if (worst < 0 || dd <= wd) { worst = id; wd = dd; } }
    ok &= ~(1u << worst); --nq;
  }
  m.np = 0; m.axis = 15; m.n = v3(0.0f, 0.0f, 1.0f);
#pragma unroll
  for (int id = 0; id < 8; ++id)
    if ((ok >> id) & 1u) {
      int k = m.np++;
      m.p[k] = v3(cx[id], cy[id], 0.5f * cz[id]);
      m.d[k] = -cz[id];
    }
}

// Sutherland-Hodgman against the half-space  s * ((P - c) . axis) <= e.
__device__ inline int clip_halfspace(const Vec3* in, int nin, Vec3* out, Vec3 c, Vec3 axis, float s, float e) {
  int nout = 0;
  Vec3 P = in[0];
  float dP = e - s * dot(P - c, axis);
  for (int i = 0; i < nin; ++i) {
    Vec3 Q = in[(i + 1 == nin) ? 0 : i + 1];
    float dQ = e - s * dot(Q - c, axis);
    if (dP >= 0.0f) {
      out[nout++] = P;
      if (dQ < 0.0f) { float t = dP / (dP - dQ); out[nout++] = madd(P, t, Q - P); }
    } else if (dQ >= 0.0f) {
      float t = dP / (dP - dQ); out[nout++] = madd(P, t, Q - P);
    }
    P = Q; dP = dQ;
  }
  return nout;
}

// ---------------------------------------------------------------- box vs box
struct SatResult { int axis; Vec3 n; float delta; };

__device__ __forceinline__ float absdot3(const float* he, float a, float b, float c) {
  return fmaf(he[2], fabsf(c), fmaf(he[1], fabsf(b), he[0] * fabsf(a)));
}

// 15-axis SAT: overlap delta = rA + rB - |t.L|; any delta <= 0 separates.
// Returns false if separated; otherwise the chosen axis (face preference, DESIGN §3 R-bias),
// the normal A -> B and the overlap on it.  Every multiply-add is an explicit fmaf so that the
// two places that call it (colliding-pair detection, manifold pass) take identical decisions.
__device__ __forceinline__ bool sat_boxes(const CollideParams& cp, const Box& A, const Box& B, SatResult& r) {
  const Vec3 t = B.c - A.c;
  float bestF = 0.0f, bestE = 0.0f; int iF = -1, iE = -1;
  Vec3 LF = v3(0, 0, 0), LE = v3(0, 0, 0);
  float c[3][3];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) c[i][j] = dot(A.ax[i], B.ax[j]);
  const float ta[3] = { dot(t, A.ax[0]), dot(t, A.ax[1]), dot(t, A.ax[2]) };
  const float tb[3] = { dot(t, B.ax[0]), dot(t, B.ax[1]), dot(t, B.ax[2]) };
#pragma unroll
  for (int k = 0; k < 3; ++k) {            // A's face axes, ids 0..2
    const float rB = absdot3(B.he, c[k][0], c[k][1], c[k][2]);
    const float dl = A.he[k] + rB - fabsf(ta[k]);
    if (dl <= 0.0f) return false;
    if (iF < 0 || dl < bestF - cp.tie_eps) { iF = k; bestF = dl; LF = A.ax[k]; }
  }
#pragma unroll
  for (int k = 0; k < 3; ++k) {            // B's face axes, ids 3..5
    const float rA = absdot3(A.he, c[0][k], c[1][k], c[2][k]);
    const float dl = rA + B.he[k] - fabsf(tb[k]);
    if (dl <= 0.0f) return false;
    if (dl < bestF - cp.tie_eps) { iF = 3 + k; bestF = dl; LF = B.ax[k]; }
  }
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) {          // edge axes a_i x b_j, ids 6..14
      Vec3 u = cross(A.ax[i], B.ax[j]);
      const float l2 = dot(u, u);
      if (l2 < cp.par_eps) continue;
      const float inv = 1.0f / sqrtf(l2);
      u = inv * u;
      const float rA = absdot3(A.he, dot(A.ax[0], u), dot(A.ax[1], u), dot(A.ax[2], u));
      const float rB = absdot3(B.he, dot(B.ax[0], u), dot(B.ax[1], u), dot(B.ax[2], u));
      const float dl = rA + rB - fabsf(dot(t, u));
      if (dl <= 0.0f) return false;
      if (iE < 0 || dl < bestE - cp.tie_eps) { iE = 6 + 3 * i + j; bestE = dl; LE = u; }
    }
  int ax = iF; Vec3 n = LF; float delta = bestF;
  if (iE >= 0 && bestE < fmaf(cp.edge_bias_rel, bestF, -cp.edge_bias_abs)) { ax = iE; n = LE; delta = bestE; }
  if (dot(n, t) < 0.0f) n = -n;
  r.axis = ax; r.n = n; r.delta = delta;
  return true;
}

__device__ __forceinline__ Vec3 pick3(const Vec3* a, int k) { return k == 0 ? a[0] : (k == 1 ? a[1] : a[2]); }
__device__ __forceinline__ float pickf(const float* a, int k) { return k == 0 ? a[0] : (k == 1 ? a[1] : a[2]); }

// Normal and overlap of ONE axis of a pair that sat_boxes found overlapping with this axis chosen: the same
// expressions as in sat_boxes (same fused multiply-adds), so the values are identical bit for bit.
__device__ __forceinline__ void sat_axis(const Box& A, const Box& B, int axis, SatResult& r) {
  const Vec3 t = B.c - A.c;
  Vec3 n; float delta;
  if (axis < 3) {
    n = pick3(A.ax, axis);
    const float rB = absdot3(B.he, dot(n, B.ax[0]), dot(n, B.ax[1]), dot(n, B.ax[2]));
    delta = pickf(A.he, axis) + rB - fabsf(dot(t, n));
  } else if (axis < 6) {
    n = pick3(B.ax, axis - 3);
    const float rA = absdot3(A.he, dot(A.ax[0], n), dot(A.ax[1], n), dot(A.ax[2], n));
    delta = rA + pickf(B.he, axis - 3) - fabsf(dot(t, n));
  } else {
    const int i = (axis - 6) / 3, j = (axis - 6) - 3 * i;
    Vec3 u = cross(pick3(A.ax, i), pick3(B.ax, j));
    const float inv = 1.0f / sqrtf(dot(u, u));
    u = inv * u;
    const float rA = absdot3(A.he, dot(A.ax[0], u), dot(A.ax[1], u), dot(A.ax[2], u));
    const float rB = absdot3(B.he, dot(B.ax[0], u), dot(B.ax[1], u), dot(B.ax[2], u));
    delta = rA + rB - fabsf(dot(t, u));
    n = u;
  }
  if (dot(n, t) < 0.0f) n = -n;
  r.axis = axis; r.n = n; r.delta = delta;
}

// Ground: colliding iff a corner lies below z = 0 (reading A9).
__device__ __forceinline__ bool ground_hit(const Box& b) {
  // lowest corner z = c.z - sum_k |ax_k.z| he_k  is NOT used: the per-corner sums below are the ones
  // collide_ground evaluates, so the decision is identical.
  bool hit = false;
#pragma unroll
  for (int id = 0; id < 8; ++id) {
    const float sx = (id & 1) ? b.he[0] : -b.he[0], sy = (id & 2) ? b.he[1] : -b.he[1], sz = (id & 4) ? b.he[2] : -b.he[2];
    const Vec3 o = madd(madd(sx * b.ax[0], sy, b.ax[1]), sz, b.ax[2]);
    hit = hit || (b.c.z + o.z < 0.0f);
  }
  return hit;
}

// Contact manifold for an overlapping pair (PAPER.md:273-280 read as A8).
__device__ __forceinline__ Vec3 sel3(bool c, Vec3 a, Vec3 b) { return v3(c ? a.x : b.x, c ? a.y : b.y, c ? a.z : b.z); }

// Only the clip polygons and the candidate points are indexed dynamically (thread-local arrays); the boxes, the
// reference / incident frames and the result stay in registers (axis choices go through select chains).
__device__ inline void manifold_boxes(const Box& A, const Box& B, const SatResult& sr, Manifold& m) {
  const int ax = sr.axis; const Vec3 n = sr.n; const float delta = sr.delta;
  m.axis = ax; m.n = n; m.np = 0;

  if (ax >= 6) {                            // edge-edge: closest points of the two support edges
    const int i = (ax - 6) / 3, j = (ax - 6) - 3 * i;
    Vec3 pa = A.c, pb = B.c;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const float sa = dot(A.ax[k], n) >= 0.0f ? 1.0f : -1.0f, sb = dot(B.ax[k], n) >= 0.0f ? 1.0f : -1.0f;
      const Vec3 qa = madd(pa, sa * A.he[k], A.ax[k]), qb = madd(pb, -sb * B.he[k], B.ax[k]);
      pa = sel3(k != i, qa, pa); pb = sel3(k != j, qb, pb);
    }
    const Vec3 ai = pick3(A.ax, i), bj = pick3(B.ax, j), r = pa - pb;
    const float hi = pickf(A.he, i), hj = pickf(B.he, j);
    const float bb = dot(ai, bj), cc = dot(ai, r), ff = dot(bj, r), den = 1.0f - bb * bb;
    float sA = (bb * ff - cc) / den, sB = (ff - bb * cc) / den;
    sA = fminf(fmaxf(sA, -hi), hi);
    sB = fminf(fmaxf(sB, -hj), hj);
    m.p[0] = 0.5f * (madd(pa, sA, ai) + madd(pb, sB, bj));
    m.d[0] = delta; m.np = 1;
    return;
  }

  // face case: X owns the axis (reference), Y is the other (incident)
  const bool refA = ax < 3; const int r = refA ? ax : ax - 3;
  Vec3 Xax[3], Yax[3]; float Xhe[3], Yhe[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    Xax[k] = sel3(refA, A.ax[k], B.ax[k]); Yax[k] = sel3(refA, B.ax[k], A.ax[k]);
    Xhe[k] = refA ? A.he[k] : B.he[k];     Yhe[k] = refA ? B.he[k] : A.he[k];
  }
  const Vec3 Xc = sel3(refA, A.c, B.c), Yc = sel3(refA, B.c, A.c);
  const Vec3 nref = refA ? n : -n;
  int mi = 0; float sg = -1.0f, best = 3.0e38f;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    float dk = dot(Yax[k], nref);
    if (-dk < best) { best = -dk; mi = k; sg = -1.0f; }
    if (dk < best) { best = dk; mi = k; sg = 1.0f; }
  }
  const int iu = (mi == 0) ? 1 : 0, iv = (mi == 2) ? 1 : 2;
  Vec3 poly0[8], poly1[8], inc[4];
  {
    const Vec3 fc = madd(Yc, sg * pickf(Yhe, mi), pick3(Yax, mi));
    const Vec3 eu = pickf(Yhe, iu) * pick3(Yax, iu), ev = pickf(Yhe, iv) * pick3(Yax, iv);
    inc[0] = fc - eu - ev; inc[1] = fc + eu - ev; inc[2] = fc + eu + ev; inc[3] = fc - eu + ev;
#pragma unroll
    for (int k = 0; k < 4; ++k) poly0[k] = inc[k];
  }
  const int u = (r == 0) ? 1 : 0, v = (r == 2) ? 1 : 2;
  const Vec3 xu = pick3(Xax, u), xv = pick3(Xax, v);
  const float hu = pickf(Xhe, u), hv = pickf(Xhe, v), hr = pickf(Xhe, r);
  int np = 4;
  Vec3 *pin = poly0, *pout = poly1;
#pragma unroll 1
  for (int pl = 0; pl < 4 && np; ++pl) {      // side planes +u, -u, +v, -v of the reference face (one copy of the clip code)
    np = clip_halfspace(pin, np, pout, Xc, pl < 2 ? xu : xv, (pl & 1) ? -1.0f : 1.0f, pl < 2 ? hu : hv);
    Vec3* t = pin; pin = pout; pout = t;
  }
  Vec3 cpt[8]; float cd[8]; int nc = 0;
  for (int k = 0; k < np; ++k) {
    float d = hr - dot(pin[k] - Xc, nref);
    if (d >= 0.0f) { cpt[nc] = madd(pin[k], 0.5f * d, nref); cd[nc] = d; ++nc; }
  }
  if (nc == 0) {                            // fallback: deepest incident vertex, SAT depth
    Vec3 bp = inc[0]; float bd = -3.0e38f;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      float d = hr - dot(inc[k] - Xc, nref);
      if (d > bd) { bd = d; bp = inc[k]; }
    }
    m.p[0] = madd(bp, 0.5f * delta, nref); m.d[0] = delta; m.np = 1;
    return;
  }
  unsigned keep = (1u << nc) - 1u;
  if (nc > 4) {                             // <= 4 reduction (DESIGN §2 S3)
    int i0 = 0, i1 = -1, i2 = -1, i3 = -1; float far2 = -1.0f, amax = 0.0f, amin = 0.0f;
    for (int k = 1; k < nc; ++k) if (cd[k] > cd[i0]) i0 = k;
    const Vec3 p0 = cpt[i0];
    for (int k = 0; k < nc; ++k) if (k != i0) {
      Vec3 d = cpt[k] - p0; float dd = dot(d, d);
      if (dd > far2) { far2 = dd; i1 = k; }
    }
    const Vec3 e01 = cpt[i1] - p0;
    for (int k = 0; k < nc; ++k) {
      if (k == i0 || k == i1) continue;
      float area = dot(cross(e01, cpt[k] - p0), n);
      if (area > amax) { amax = area; i2 = k; }
      if (area < amin) { amin = area; i3 = k; }
    }
    keep = (1u << i0) | (1u << i1);
    if (i2 >= 0) keep |= 1u << i2;
    if (i3 >= 0) keep |= 1u << i3;
  }
  const int no = __popc(keep);              // survivors in ascending clip-output index; static output slots
#pragma unroll
  for (int o = 0; o < 4; ++o)
    if (o < no) { const int k = __fns(keep, 0, o + 1); m.p[o] = cpt[k]; m.d[o] = cd[k]; }
  m.np = no;
}

}  // namespace jenga
