// solve.cuh -- narrowphase dispatch, canonical colouring, contact setup, coloured PGS sweeps
// and integration for one env per CTA (see step.cuh for the mapping).
#pragma once
#include "step.cuh"

namespace jenga {

__device__ __forceinline__ Box load_box(const Smem& s, int S, int b) {
  Box X;
  X.c = v3(s.st[b], s.st[S + b], s.st[2 * S + b]);
#pragma unroll
  for (int k = 0; k < 3; ++k) X.ax[k] = v3(s.R[k * S + b], s.R[(3 + k) * S + b], s.R[(6 + k) * S + b]);
  X.he[0] = s.pr[4 * S + b]; X.he[1] = s.pr[5 * S + b]; X.he[2] = s.pr[6 * S + b];
  return X;
}

__device__ __forceinline__ void write_record(float* rec, int pair, int cand_pos, int i, int j, const Manifold& m) {
  int* ri = reinterpret_cast<int*>(rec);
  ri[RecPair] = pair; ri[RecCand] = cand_pos; ri[RecMeta] = m.axis | (m.np << 8); ri[RecA] = i; ri[RecB] = j;
  rec[RecN] = m.n.x; rec[RecN + 1] = m.n.y; rec[RecN + 2] = m.n.z;
#pragma unroll
  for (int k = 0; k < 4; ++k)
    if (k < m.np) { rec[RecPt + 4 * k] = m.p[k].x; rec[RecPt + 4 * k + 1] = m.p[k].y; rec[RecPt + 4 * k + 2] = m.p[k].z; rec[RecPt + 4 * k + 3] = m.d[k]; }
}

// S3 over the candidate list: thread k takes candidate k; colliding pairs are compacted in
// ascending pair index into s.rec.  Returns the number of colliding pairs kept (<= pc).
__device__ inline int narrowphase(const Smem& s, const Params& P, int n_cand, unsigned* status) {
  const int S = P.S;
  int n_coll = 0;
  for (int base = 0; base < n_cand; base += blockDim.x) {
    const int k = base + threadIdx.x;
    Manifold m; m.np = 0; m.axis = 0;
    int idx = 0, i = -1, j = 0;
    if (k < n_cand) {
      idx = s.cand[k];
      pair_bodies(P.B, idx, i, j);
      const Box Bj = load_box(s, S, j);
      if (i < 0) collide_ground(Bj, m);
      else { const Box Bi = load_box(s, S, i); collide_boxes(P.cp, Bi, Bj, m); }
    }
    int tot;
    const int rank = n_coll + block_rank(m.np > 0, s.scan, &tot);
    if (m.np > 0 && rank < P.pc) write_record(s.rec + (size_t)rank * kRecWords, idx, k, i, j, m);
    n_coll += tot;
  }
  if (n_coll > P.pc) { *status |= JENGA_ST_CONTACT_OVERFLOW; n_coll = P.pc; }
  __syncthreads();
  return n_coll;
}

// Canonical order (north_star (d), DESIGN §2 S4): visit the colliding pairs in ascending pair
// index; colour = lowest colour not used by an earlier pair sharing a dynamic body.  Then
// owner[] = records sorted by (colour, pair index).  Sequential by construction: thread 0 walks
// the list with one 64-bit mask per body.  Returns the number of colours.
__device__ inline int colour_pairs(const Smem& s, const Params& P, int n_coll, unsigned* status) {
  const int S = P.S;
  if (threadIdx.x == 0) {
    for (int b = 0; b < P.B; ++b) s.used[b] = 0ull;
    int ncol = 0; unsigned st = 0;
    for (int r = 0; r < n_coll; ++r) {
      const int* ri = reinterpret_cast<const int*>(s.rec + (size_t)r * kRecWords);
      const int i = ri[RecA], j = ri[RecB];
      unsigned long long m = 0ull;
      if (i >= 0 && s.pr[i] != 0.0f) m |= s.used[i];
      if (s.pr[j] != 0.0f) m |= s.used[j];
      int c = __ffsll((long long)~m) - 1;
      if (c < 0) { c = kMaxColours - 1; st |= JENGA_ST_COLOUR_OVERFLOW; }
      if (i >= 0) s.used[i] |= 1ull << c;
      s.used[j] |= 1ull << c;
      s.colour[r] = c;
      s.wrank[r] = s.ccount[c]++;
      if (c + 1 > ncol) ncol = c + 1;
    }
    int acc = 0;
    for (int c = 0; c < ncol; ++c) { const int n = s.ccount[c]; s.cstart[c] = acc; acc += n; }
    s.scan[ScNCol] = ncol;
    if (st) *status |= st;
  }
  __syncthreads();
  for (int r = threadIdx.x; r < n_coll; r += blockDim.x) s.owner[s.cstart[s.colour[r]] + s.wrank[r]] = r;
  for (int c = threadIdx.x; c < kMaxColours; c += blockDim.x) s.ccount[c] = 0;   // ready for the next step
  __syncthreads();
  (void)S;
  return s.scan[ScNCol];
}

// Per-thread solver state of one colliding pair (registers).
struct PairState {
  int a, b;            // body ids (a = -1: ground)
  int np, colour, rank;
  Vec3 n, t1, t2;      // contact frame (tangent basis: DESIGN §3 reading A10)
  Vec3 p[4];           // contact points
  float ik[4][3];      // 1 / K_dd  (Eq. 13, for d = n, t1, t2)
  float ko[4][3];      // K_01, K_02, K_12: coupling of the three rows of one contact
  float lam[4][3];     // accumulated jn, jt1, jt2
  float corr;          // Baumgarte: beta * max(0, depth_max - slop) / (imA + imB)   (Eq. 16)
};

struct BodyPair {      // the two bodies of a pair, staged from shared memory for one colour visit
  Vec3 xA, xB, vA, wA, vB, wB;
  float imA, imB, IA[6], IB[6];
};

__device__ __forceinline__ void load_bodies(const Smem& s, int S, const PairState& ps, BodyPair& bp, bool with_vel) {
  const int a = ps.a, b = ps.b;
  bp.xB = v3(s.st[b], s.st[S + b], s.st[2 * S + b]);
  bp.imB = body_dynamic(s, S, b) ? s.pr[b] : 0.0f;
#pragma unroll
  for (int k = 0; k < 6; ++k) bp.IB[k] = s.Iw[k * S + b];
  if (with_vel) {
    bp.vB = v3(s.st[7 * S + b], s.st[8 * S + b], s.st[9 * S + b]);
    bp.wB = v3(s.st[10 * S + b], s.st[11 * S + b], s.st[12 * S + b]);
  }
  if (a >= 0) {
    bp.xA = v3(s.st[a], s.st[S + a], s.st[2 * S + a]);
    bp.imA = body_dynamic(s, S, a) ? s.pr[a] : 0.0f;
#pragma unroll
    for (int k = 0; k < 6; ++k) bp.IA[k] = s.Iw[k * S + a];
    if (with_vel) {
      bp.vA = v3(s.st[7 * S + a], s.st[8 * S + a], s.st[9 * S + a]);
      bp.wA = v3(s.st[10 * S + a], s.st[11 * S + a], s.st[12 * S + a]);
    }
  } else {
    bp.xA = v3(0, 0, 0); bp.imA = 0.0f; bp.vA = v3(0, 0, 0); bp.wA = v3(0, 0, 0);
#pragma unroll
    for (int k = 0; k < 6; ++k) bp.IA[k] = 0.0f;
  }
}

__device__ __forceinline__ void store_velocities(const Smem& s, int S, const PairState& ps, const BodyPair& bp) {
  const int a = ps.a, b = ps.b;
  if (bp.imB != 0.0f) {
    s.st[7 * S + b] = bp.vB.x; s.st[8 * S + b] = bp.vB.y; s.st[9 * S + b] = bp.vB.z;
    s.st[10 * S + b] = bp.wB.x; s.st[11 * S + b] = bp.wB.y; s.st[12 * S + b] = bp.wB.z;
  }
  if (a >= 0 && bp.imA != 0.0f) {
    s.st[7 * S + a] = bp.vA.x; s.st[8 * S + a] = bp.vA.y; s.st[9 * S + a] = bp.vA.z;
    s.st[10 * S + a] = bp.wA.x; s.st[11 * S + a] = bp.wA.y; s.st[12 * S + a] = bp.wA.z;
  }
}

// a loses the impulse, b gains it (Listing 1, PAPER.md:335-336 + the angular lines, reading A11)
__device__ __forceinline__ void apply_impulse(BodyPair& bp, Vec3 rA, Vec3 rB, Vec3 Pi) {
  bp.vA = madd(bp.vA, -bp.imA, Pi);
  bp.wA = bp.wA - sym_mul(bp.IA, cross(rA, Pi));
  bp.vB = madd(bp.vB, bp.imB, Pi);
  bp.wB = bp.wB + sym_mul(bp.IB, cross(rB, Pi));
}

// S4 for the pair record r: frame, contact-space matrices, warm-start lookup.
__device__ inline void setup_pair(const Smem& s, const Params& P, int env, int r, PairState& ps) {
  const int S = P.S;
  const float* rec = s.rec + (size_t)r * kRecWords;
  const int* ri = reinterpret_cast<const int*>(rec);
  ps.rank = r; ps.a = ri[RecA]; ps.b = ri[RecB];
  const int meta = ri[RecMeta]; ps.np = (meta >> 8) & 0xff; ps.colour = s.colour[r];
  ps.n = v3(rec[RecN], rec[RecN + 1], rec[RecN + 2]);
  {   // t1 = normalise(e_k - n (n.e_k)), k = x unless |n_x| > 1/sqrt(2), then y;  t2 = n x t1
    const bool usey = fabsf(ps.n.x) > 0.70710678118654752f;
    const Vec3 e = usey ? v3(0, 1, 0) : v3(1, 0, 0);
    const float d = usey ? ps.n.y : ps.n.x;
    Vec3 u = madd(e, -d, ps.n);
    ps.t1 = rsqrtf(dot(u, u)) * u;
    ps.t2 = cross(ps.n, ps.t1);
  }
  BodyPair bp; load_bodies(s, S, ps, bp, false);
  float dmax = 0.0f;
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    ps.lam[c][0] = ps.lam[c][1] = ps.lam[c][2] = 0.0f;
    ps.ik[c][0] = ps.ik[c][1] = ps.ik[c][2] = 0.0f;
    ps.ko[c][0] = ps.ko[c][1] = ps.ko[c][2] = 0.0f;
    ps.p[c] = v3(0, 0, 0);
    if (c < ps.np) {
      ps.p[c] = v3(rec[RecPt + 4 * c], rec[RecPt + 4 * c + 1], rec[RecPt + 4 * c + 2]);
      dmax = fmaxf(dmax, rec[RecPt + 4 * c + 3]);
      const Vec3 rA = ps.a >= 0 ? ps.p[c] - bp.xA : v3(0, 0, 0), rB = ps.p[c] - bp.xB;
      const Vec3 dir[3] = { ps.n, ps.t1, ps.t2 };
      Vec3 uA[3], uB[3], wA[3], wB[3];
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        uA[d] = cross(rA, dir[d]); uB[d] = cross(rB, dir[d]);
        wA[d] = sym_mul(bp.IA, uA[d]); wB[d] = sym_mul(bp.IB, uB[d]);
      }
      const float im = bp.imA + bp.imB;
#pragma unroll
      for (int d = 0; d < 3; ++d) ps.ik[c][d] = 1.0f / (im + dot(uA[d], wA[d]) + dot(uB[d], wB[d]));
      ps.ko[c][0] = dot(uA[0], wA[1]) + dot(uB[0], wB[1]);
      ps.ko[c][1] = dot(uA[0], wA[2]) + dot(uB[0], wB[2]);
      ps.ko[c][2] = dot(uA[1], wA[2]) + dot(uB[1], wB[2]);
    }
  }
  const float ims = bp.imA + bp.imB;
  ps.corr = ims > 0.0f ? P.beta * fmaxf(0.0f, dmax - P.slop) / ims : 0.0f;

  // warm start (reading A12): a new contact inherits (jn,jt1,jt2) of the nearest not yet taken
  // previous contact point of the same pair within match_tol; slots ascending.
  if (P.warm_start) {
    const int nk = P.n_cache[env];
    const int* keys = P.cache_key + (size_t)env * P.pc * 2;
    const int pair = ri[RecPair];
    int lo = 0, hi = nk;
    while (lo < hi) { const int mid = (lo + hi) >> 1; if (keys[2 * mid] < pair) lo = mid + 1; else hi = mid; }
    if (lo < nk && keys[2 * lo] == pair) {
      const int ocnt = keys[2 * lo + 1] & 0xff;
      const float* ol = P.cache_lam + ((size_t)env * P.pc + lo) * 12;
      const float* op = P.cache_pt + ((size_t)env * P.pc + lo) * 12;
      Vec3 q[4]; float l[4][3];
#pragma unroll
      for (int o = 0; o < 4; ++o) {
        q[o] = v3(0, 0, 0); l[o][0] = l[o][1] = l[o][2] = 0.0f;
        if (o < ocnt) { q[o] = v3(op[3 * o], op[3 * o + 1], op[3 * o + 2]); l[o][0] = ol[3 * o]; l[o][1] = ol[3 * o + 1]; l[o][2] = ol[3 * o + 2]; }
      }
      unsigned taken = 0;
      const float tol2 = P.match_tol * P.match_tol;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        if (c < ps.np) {
          int bo = -1; float bd = tol2;
#pragma unroll
          for (int o = 0; o < 4; ++o)
            if (o < ocnt && !((taken >> o) & 1u)) {
              const Vec3 d = ps.p[c] - q[o]; const float dd = dot(d, d);
              if (dd < bd) { bd = dd; bo = o; }
            }
#pragma unroll
          for (int o = 0; o < 4; ++o)
            if (o == bo) { taken |= 1u << o; ps.lam[c][0] = l[o][0]; ps.lam[c][1] = l[o][1]; ps.lam[c][2] = l[o][2]; }
        }
      }
    }
  }
}

// Apply the warm-start impulses of this pair to its two bodies (one colour visit).
__device__ __forceinline__ void warm_apply(const PairState& ps, BodyPair& bp) {
#pragma unroll
  for (int c = 0; c < 4; ++c)
    if (c < ps.np) {
      const Vec3 rA = ps.p[c] - bp.xA, rB = ps.p[c] - bp.xB;
      const Vec3 Pi = madd(madd(ps.lam[c][0] * ps.n, ps.lam[c][1], ps.t1), ps.lam[c][2], ps.t2);
      apply_impulse(bp, rA, rB, Pi);
    }
}

// One Gauss-Seidel visit of a pair: slots ascending; per contact the normal row (Eq. 14,
// clamp >= 0), then t1, then t2 (Eq. 15, each clipped to +-mu_s jn)  -- Listing 1.
// The three rows of a contact act on the same two bodies, so the relative velocity of the
// contact point is read once, advanced between rows with the contact-space couplings K_ij
// (exactly the change the applied impulse causes), and the summed impulse is applied once.
__device__ __forceinline__ void solve_pair(PairState& ps, BodyPair& bp, float mu, float restitution) {
#pragma unroll
  for (int c = 0; c < 4; ++c)
    if (c < ps.np) {
      const Vec3 rA = ps.p[c] - bp.xA, rB = ps.p[c] - bp.xB;
      const Vec3 vr = (bp.vB + cross(bp.wB, rB)) - (bp.vA + cross(bp.wA, rA));
      float u0 = dot(vr, ps.n), u1 = dot(vr, ps.t1), u2 = dot(vr, ps.t2);
      // normal row
      float nw = fmaxf(ps.lam[c][0] - (1.0f + restitution) * u0 * ps.ik[c][0], 0.0f);
      const float d0 = nw - ps.lam[c][0]; ps.lam[c][0] = nw;
      u1 = fmaf(ps.ko[c][0], d0, u1); u2 = fmaf(ps.ko[c][1], d0, u2);
      // friction rows, boxed by mu * jn
      const float lim = mu * nw;
      float n1 = fminf(fmaxf(ps.lam[c][1] - u1 * ps.ik[c][1], -lim), lim);
      const float d1 = n1 - ps.lam[c][1]; ps.lam[c][1] = n1;
      u2 = fmaf(ps.ko[c][2], d1, u2);
      float n2 = fminf(fmaxf(ps.lam[c][2] - u2 * ps.ik[c][2], -lim), lim);
      const float d2 = n2 - ps.lam[c][2]; ps.lam[c][2] = n2;
      const Vec3 Pi = madd(madd(d0 * ps.n, d1, ps.t1), d2, ps.t2);
      apply_impulse(bp, rA, rB, Pi);
    }
}

// S4 (warm-start application) + S5: colour sweeps with a CTA barrier per colour.
__device__ inline void pgs_sweeps(const Smem& s, const Params& P, PairState& ps, bool have_pair,
                                  int ncol, int iters, float mu) {
  const int S = P.S;
  if (P.warm_start) {
    for (int c = 0; c < ncol; ++c) {
      if (have_pair && ps.colour == c) {
        BodyPair bp; load_bodies(s, S, ps, bp, true);
        warm_apply(ps, bp);
        store_velocities(s, S, ps, bp);
      }
      __syncthreads();
    }
  }
  for (int it = 0; it < iters; ++it)
    for (int c = 0; c < ncol; ++c) {
      if (have_pair && ps.colour == c) {
        BodyPair bp; load_bodies(s, S, ps, bp, true);
        solve_pair(ps, bp, mu, P.restitution);
        store_velocities(s, S, ps, bp);
      }
      __syncthreads();
    }
}

// S6: x += h v (Eq. 6); q <- normalise(q + h/2 [0,w] (x) q) (Eq. 2, PAPER.md:151,
// world-frame reading A3); then Eq. 16 (reading A14) once per colliding pair.
__device__ inline void integrate(const Smem& s, const Params& P, const PairState& ps, bool have_pair, int ncol,
                                 unsigned* status) {
  const int S = P.S; const float h = P.h;
  for (int b = threadIdx.x; b < P.B; b += blockDim.x) {
    if (!body_dynamic(s, S, b)) continue;
    const float vx = s.st[7 * S + b], vy = s.st[8 * S + b], vz = s.st[9 * S + b];
    const float x = s.st[b] + h * vx, y = s.st[S + b] + h * vy, z = s.st[2 * S + b] + h * vz;
    s.st[b] = x; s.st[S + b] = y; s.st[2 * S + b] = z;
    const float qw = s.st[3 * S + b], qx = s.st[4 * S + b], qy = s.st[5 * S + b], qz = s.st[6 * S + b];
    const float ox = s.st[10 * S + b], oy = s.st[11 * S + b], oz = s.st[12 * S + b];
    const float dw = -(ox * qx + oy * qy + oz * qz);
    const float dx = ox * qw + oy * qz - oz * qy;
    const float dy = oy * qw + oz * qx - ox * qz;
    const float dz = oz * qw + ox * qy - oy * qx;
    const float hh = 0.5f * h;
    const float nw = qw + hh * dw, nx = qx + hh * dx, ny = qy + hh * dy, nz = qz + hh * dz;
    const float il = 1.0f / sqrtf(nw * nw + nx * nx + ny * ny + nz * nz);
    s.st[3 * S + b] = nw * il; s.st[4 * S + b] = nx * il; s.st[5 * S + b] = ny * il; s.st[6 * S + b] = nz * il;
    if (!(isfinite(x) && isfinite(y) && isfinite(z) && isfinite(vx) && isfinite(vy) && isfinite(vz)))
      *status |= JENGA_ST_NONFINITE;
  }
  const int any = __syncthreads_or(have_pair && ps.corr > 0.0f);
  if (any) {
    for (int c = 0; c < ncol; ++c) {
      if (have_pair && ps.colour == c && ps.corr > 0.0f) {
        const int a = ps.a, b = ps.b;
        const float imB = body_dynamic(s, S, b) ? s.pr[b] : 0.0f;
        s.st[b] += imB * ps.corr * ps.n.x; s.st[S + b] += imB * ps.corr * ps.n.y; s.st[2 * S + b] += imB * ps.corr * ps.n.z;
        if (a >= 0) {
          const float imA = body_dynamic(s, S, a) ? s.pr[a] : 0.0f;
          s.st[a] -= imA * ps.corr * ps.n.x; s.st[S + a] -= imA * ps.corr * ps.n.y; s.st[2 * S + a] -= imA * ps.corr * ps.n.z;
        }
      }
      __syncthreads();
    }
  }
}

// S7: the pair's impulses and contact points become the next substep's warm-start cache.
__device__ inline void store_cache(const Params& P, int env, const Smem& s, const PairState& ps, bool have_pair, int n_coll) {
  if (have_pair) {
    const int r = ps.rank;
    const int* ri = reinterpret_cast<const int*>(s.rec + (size_t)r * kRecWords);
    int* key = P.cache_key + ((size_t)env * P.pc + r) * 2;
    key[0] = ri[RecPair]; key[1] = ((ri[RecMeta] & 0xff) << 8) | ps.np;
    float* ol = P.cache_lam + ((size_t)env * P.pc + r) * 12;
    float* op = P.cache_pt + ((size_t)env * P.pc + r) * 12;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const bool on = c < ps.np;
      ol[3 * c] = on ? ps.lam[c][0] : 0.0f; ol[3 * c + 1] = on ? ps.lam[c][1] : 0.0f; ol[3 * c + 2] = on ? ps.lam[c][2] : 0.0f;
      op[3 * c] = ps.p[c].x; op[3 * c + 1] = ps.p[c].y; op[3 * c + 2] = ps.p[c].z;
    }
  }
  if (threadIdx.x == 0) P.n_cache[env] = n_coll;
}

}  // namespace jenga
