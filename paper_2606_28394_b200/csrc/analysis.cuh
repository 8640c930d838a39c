// analysis.cuh -- the two per-env analyses of the paper's game loop that sit beside the step:
// the support-polygon margin of Eq. 17 (§8.1) and the move classes of ziglar_block_analysis()
// (Table 1, §5.4).  Not on the timed path; one warp (one thread) per env.
#pragma once
#include "layout.cuh"

namespace jenga {

// "b comes before a on the way round": seen from hull vertex c, candidate p replaces q if p lies to the right of
// c -> q (clockwise of it), or on the line and farther away.  With every point on one side of c this is a total order
// whose maximum is the next counter-clockwise hull vertex.
__device__ __forceinline__ bool wraps_before(float cx, float cy, float qx, float qy, float px, float py) {
  const float ax = qx - cx, ay = qy - cy, bx = px - cx, by = py - cy;
  const float cr = ax * by - ay * bx;
  if (cr != 0.0f) return cr < 0.0f;
  return bx * bx + by * by > ax * ax + ay * ay;
}

// Eq. 17: support polygon = convex hull of the (x, y) of the 8 corners of every active body whose world-AABB bottom
// z - e'_z <= eps (e' = |R| e, eps = the AABB margin); COM_xy = mass-weighted mean over the active dynamic bodies;
// margin = minimum signed distance of COM_xy to the hull's edges (positive inside).  Gift wrapping: every step all 32
// lanes scan the points for the next counter-clockwise vertex (no sort).  out[env] = (margin, COM_x, COM_y, hull vertices);
// nothing on the ground: margin -1e30; one point / a segment: minus the distance to it.
__global__ void __launch_bounds__(32) k_support(const Params P, float4* out) {
  extern __shared__ float2 pts[];                               // [8 * S]
  const int env = blockIdx.x, lane = threadIdx.x, S = P.S;
  const float* st = P.state + (size_t)env * kStateRows * S;
  const float* pr = P.props + (size_t)env * kPropRows * S;
  const unsigned below = (1u << lane) - 1u;
  float msum = 0.0f, mx = 0.0f, my = 0.0f;
  int n_ground = 0;
  for (int base = 0; base < P.B; base += 32) {
    const int b = base + lane;
    bool ground = false;
    float R[9], x = 0, y = 0, hx = 0, hy = 0, hz = 0;
    if (b < P.B && pr[7 * S + b] != 0.0f) {
      x = st[b]; y = st[S + b];
      const float z = st[2 * S + b], im = pr[b];
      quat_to_R(st[3 * S + b], st[4 * S + b], st[5 * S + b], st[6 * S + b], R);
      hx = pr[4 * S + b]; hy = pr[5 * S + b]; hz = pr[6 * S + b];
      if (im > 0.0f) { const float m = 1.0f / im; msum += m; mx += m * x; my += m * y; }
      ground = z - (fabsf(R[6]) * hx + fabsf(R[7]) * hy + fabsf(R[8]) * hz) <= P.aabb_margin;
    }
    const unsigned bal = __ballot_sync(kFull, ground);
    if (ground) {
      const int slot = n_ground + __popc(bal & below);
#pragma unroll
      for (int id = 0; id < 8; ++id) {
        const float sx = (id & 1) ? hx : -hx, sy = (id & 2) ? hy : -hy, sz = (id & 4) ? hz : -hz;
        pts[8 * slot + id] = make_float2(x + R[0] * sx + R[1] * sy + R[2] * sz, y + R[3] * sx + R[4] * sy + R[5] * sz);
      }
    }
    n_ground += __popc(bal);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    msum += __shfl_xor_sync(kFull, msum, o); mx += __shfl_xor_sync(kFull, mx, o); my += __shfl_xor_sync(kFull, my, o);
  }
  const float cx = msum > 0.0f ? mx / msum : 0.0f, cy = msum > 0.0f ? my / msum : 0.0f;
  __syncwarp();
  const int n = 8 * n_ground;
  if (n == 0) { if (lane == 0) out[env] = make_float4(-1.0e30f, cx, cy, 0.0f); return; }
  // start: lowest (x, then y)
  float sx = 3.0e38f, sy = 3.0e38f;
  for (int i = lane; i < n; i += 32) { const float2 p = pts[i]; if (p.x < sx || (p.x == sx && p.y < sy)) { sx = p.x; sy = p.y; } }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const float ox = __shfl_xor_sync(kFull, sx, o), oy = __shfl_xor_sync(kFull, sy, o);
    if (ox < sx || (ox == sx && oy < sy)) { sx = ox; sy = oy; }
  }
  float ux = sx, uy = sy, d = 3.0e38f, fx = sx, fy = sy;      // current vertex, margin, the first edge's end (2-vertex case)
  int nh = 0;
  for (int it = 0; it < n + 1; ++it) {
    float qx = ux, qy = uy;                                    // candidate: the current vertex itself loses to any other point
    for (int i = lane; i < n; i += 32) { const float2 p = pts[i]; if (wraps_before(ux, uy, qx, qy, p.x, p.y)) { qx = p.x; qy = p.y; } }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const float ox = __shfl_xor_sync(kFull, qx, o), oy = __shfl_xor_sync(kFull, qy, o);
      if (wraps_before(ux, uy, qx, qy, ox, oy)) { qx = ox; qy = oy; }
    }
    qx = __shfl_sync(kFull, qx, 0); qy = __shfl_sync(kFull, qy, 0);      // one answer for the warp (ties resolve differently per lane)
    if (qx == ux && qy == uy) break;                           // a single distinct point
    ++nh;
    if (nh == 1) { fx = qx; fy = qy; }
    const float ex = qx - ux, ey = qy - uy;
    d = fminf(d, (ex * (cy - uy) - ey * (cx - ux)) / sqrtf(ex * ex + ey * ey));
    ux = qx; uy = qy;
    if (ux == sx && uy == sy) break;                           // closed
  }
  if (nh == 0) d = -sqrtf((cx - sx) * (cx - sx) + (cy - sy) * (cy - sy));
  else if (nh <= 2) {                                          // a segment: distance to it
    const float ex = fx - sx, ey = fy - sy;
    float t = ((cx - sx) * ex + (cy - sy) * ey) / (ex * ex + ey * ey);
    t = fminf(fmaxf(t, 0.0f), 1.0f);
    const float px = sx + t * ex - cx, py = sy + t * ey - cy;
    d = -sqrtf(px * px + py * py);
  }
  if (lane == 0) out[env] = make_float4(d, cx, cy, (float)(nh == 0 ? 1 : nh));
}

// Table 1: class of the move (block, axis) of every env.  The block's slot in its level follows the tower layout of the
// workloads (body id = 3 level + slot, slot 1 = centre); axis 0 = along the block's length (the paper's Y), 1 = across
// (the paper's X).  out[env] = (class 0 center_xaxis / 1 side_yaxis / 2 side_xaxis, F_min = k mu_s m g [N], torque 0/1, k).
__global__ void k_ziglar(const Params P, const int* block, const int* axis, float4* out) {
  const int env = blockIdx.x * blockDim.x + threadIdx.x;
  if (env >= P.E) return;
  const int b = block[env];
  if (b < 0 || b >= P.B) { out[env] = make_float4(-1.0f, 0.0f, 0.0f, 0.0f); return; }
  const float im = P.props[(size_t)env * kPropRows * P.S + b];
  const float m = im > 0.0f ? 1.0f / im : 0.0f;
  const float g = sqrtf(P.g[0] * P.g[0] + P.g[1] * P.g[1] + P.g[2] * P.g[2]);
  const int cls = (b % 3) == 1 ? 0 : (axis[env] == 0 ? 1 : 2);
  const float k = cls == 2 ? 4.0f : 3.0f;
  out[env] = make_float4((float)cls, k * P.mu[env] * m * g, cls == 2 ? 1.0f : 0.0f, k);
}

}  // namespace jenga
