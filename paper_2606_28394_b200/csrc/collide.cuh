// collide.cuh -- per-thread narrowphase of the batched Jenga step (fp32, sm_100a).
//
// S3 of DESIGN.md §2: 15-axis OBB-OBB separating-axis test (§6.2) and the
// contact manifold (§6.2.1, read as reference/incident face clipping with
// per-point depth, DESIGN.md §3 reading A8), plus box-vs-ground-plane corners (reading A9).
// One thread handles one candidate pair.  This header holds the register-only parts (15-axis SAT, ground corners);
// the face / edge manifold reads the box records by dynamic index and clips in shared memory: kcollide.cuh.
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

}  // namespace jenga
