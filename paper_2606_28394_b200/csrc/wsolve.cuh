// wsolve.cuh -- colliding-pair detection, canonical colouring, contact setup, coloured PGS sweeps,
// integration and warm-start cache for one env per warp (see wenv.cuh for the mapping).
#pragma once
#include "wenv.cuh"

namespace jenga {

__device__ __forceinline__ Box load_box(const Smem& s, int S, int b) {
  Box X;
  const float4 x = bd4(s, b, 0);
  X.c = v3(x.x, x.y, x.z);
#pragma unroll
  for (int k = 0; k < 3; ++k) X.ax[k] = v3(s.R[k * S + b], s.R[(3 + k) * S + b], s.R[(6 + k) * S + b]);
  X.he[0] = s.pr[4 * S + b]; X.he[1] = s.pr[5 * S + b]; X.he[2] = s.pr[6 * S + b];
  return X;
}

// cab word of a colliding pair: (a+1) bits 0-10 | A dynamic bit 11 | SAT axis bits 12-15 | b bits 16-26 | B dynamic bit 27
__device__ __forceinline__ unsigned pack_ab(const Smem& s, int a, int b, int axis) {
  unsigned w = (unsigned)(a + 1) | ((unsigned)axis << 12) | ((unsigned)b << 16);
  if (a >= 0 && s.bd[a * kBd + 3] != 0.0f) w |= 1u << 11;
  if (s.bd[b * kBd + 3] != 0.0f) w |= 1u << 27;
  return w;
}
__device__ __forceinline__ int ab_a(unsigned w) { return (int)(w & 0x7ffu) - 1; }
__device__ __forceinline__ int ab_b(unsigned w) { return (int)((w >> 16) & 0x7ffu); }
__device__ __forceinline__ int ab_axis(unsigned w) { return (int)((w >> 12) & 0xfu); }

// Manifold of colliding pair (a, b) whose SAT axis is known (find_colliding stored it).
__device__ __forceinline__ void pair_manifold(const Smem& s, int S, int a, int b, int axis, Manifold& m) {
  const Box Bj = load_box(s, S, b);
  if (a < 0) { collide_ground(Bj, m); return; }
  const Box Bi = load_box(s, S, a);
  SatResult sr; sat_axis(Bi, Bj, axis, sr);
  manifold_boxes(Bi, Bj, sr, m);
}

// S3, first half: which candidates collide (15-axis SAT / a ground corner below z = 0).  Lane k of a
// round takes candidate base+k; the colliding ones are compacted in ascending pair index into
// s.cpair[cur] / s.cab.  Returns the number kept (<= pc); sets CONTACT_OVERFLOW.
__device__ inline int find_colliding(const Smem& s, const Params& P, int n_cand, int cur, unsigned* status) {
  const int S = P.S, lane = lane_id();
  const unsigned below = (1u << lane) - 1u;
  int n = 0;
  for (int base = 0; base < n_cand; base += 32) {
    const int k = base + lane;
    bool hit = false; int idx = 0, i = -1, j = 0, axis = JENGA_AXIS_GROUND;
    if (k < n_cand) {
      idx = s.cand[k];
      pair_bodies(P.B, idx, i, j);
      const Box Bj = load_box(s, S, j);
      if (i < 0) hit = ground_hit(Bj);
      else { const Box Bi = load_box(s, S, i); SatResult sr; sr.axis = 0; hit = sat_boxes(P.cp, Bi, Bj, sr); axis = sr.axis; }
    }
    const unsigned bal = __ballot_sync(kFull, hit);
    const int rank = n + __popc(bal & below);
    if (hit && rank < P.pc) { s.cpair[cur][rank] = (unsigned short)idx; s.cab[rank] = pack_ab(s, i, j, axis); }
    n += __popc(bal);
  }
  if (n > P.pc) { *status |= JENGA_ST_CONTACT_OVERFLOW; n = P.pc; }
  __syncwarp();
  return n;
}

// Canonical order (north_star (d), DESIGN §2 S4): visit the colliding pairs in ascending pair index;
// colour = lowest colour not used by an earlier pair sharing a dynamic body.  Then pos[]/order[] =
// pairs sorted by (colour, pair index) and ph[] = the phase chunks (<= 32 pairs of one colour each).
// The walk is sequential by definition (lane 0, one 64-bit mask per body); when the colliding-pair
// list equals the previous substep's the previous colouring is the same function of the same input
// and is kept.
template <bool TM>
__device__ inline void colour_pairs(const Smem& s, const Params& P, int n_coll, int cur, unsigned* status) {
  const int lane = lane_id();
  bool same = n_coll == s.misc[MiNprev];
  if (same)
    for (int r = lane; r < n_coll; r += 32) same = same && (s.cpair[cur][r] == s.cpair[cur ^ 1][r]);
  same = __all_sync(kFull, same);
  if (same) return;
  for (int b = lane; b < P.B; b += 32) s.used[b] = 0ull;
  for (int c = lane; c < kMaxColours; c += 32) s.ccount[c] = 0;
  __syncwarp();
  if (lane == 0) {
    int ncol = 0; unsigned st = 0;
    for (int r = 0; r < n_coll; ++r) {
      const unsigned w = s.cab[r];
      const int a = ab_a(w), b = ab_b(w);
      unsigned long long m = 0ull;
      if (w & (1u << 11)) m |= s.used[a];
      if (w & (1u << 27)) m |= s.used[b];
      int c = __ffsll((long long)~m) - 1;
      if (c < 0) { c = kMaxColours - 1; st |= JENGA_ST_COLOUR_OVERFLOW; }
      if (a >= 0) s.used[a] |= 1ull << c;
      s.used[b] |= 1ull << c;
      s.colour[r] = (unsigned char)c;
      const int k = s.ccount[c];
      s.wrank[r] = (unsigned short)k; s.ccount[c] = k + 1;
      if (c + 1 > ncol) ncol = c + 1;
    }
    int acc = 0, nph = 0;
    for (int c = 0; c < ncol; ++c) {
      const int n = s.ccount[c];
      s.cstart[c] = acc;
      for (int st0 = acc; st0 < acc + n; ) {                     // chunks of <= 32 pairs; none straddles the TMEM boundary
        int lim = min(acc + n, st0 + 32);
        if (TM && st0 < s.pos0 && lim > s.pos0) lim = s.pos0;
        s.ph[nph++] = st0 | ((lim - st0) << 16);
        st0 = lim;
      }
      acc += n;
    }
    s.misc[MiNcol] = ncol; s.misc[MiNph] = nph;
    if (st) *status |= st;
  }
  __syncwarp();
  for (int r = lane; r < n_coll; r += 32) {
    const int k = s.cstart[s.colour[r]] + s.wrank[r];
    s.pos[r] = (unsigned short)k; s.order[k] = (unsigned short)r;
  }
  __syncwarp();
}

// ---------------------------------------------------------------- pair slots (colour-sorted solver constants)
// Header of position k (shared memory, s.hdr[f * pcA + k]):
//   0: a, b, meta = np | axis << 8 | pair index << 16 (int bits), 1/|e_k - n (n.e_k)| (tangent normalisation)
//   1: n.x n.y n.z, Baumgarte corr = beta max(0, depth_max - slop) / (imA + imB)     (Eq. 16)
// Contact constants of position k: 48 words, PairC.  ro[9c..9c+8] = p.xyz, (1+e)/K_nn, 1/K_t1t1, 1/K_t2t2,
// K_n,t1, K_n,t2, K_t1,t2 of contact c (K_dd: Eq. 13, for d = n, t1, t2); lam[3c..3c+2] = jn, jt1, jt2.
// They live in shared memory (field-major float4 [12][capS], position k - pos0) or, in the TMEM kernel for
// positions < pos0 = 32 * tmb, in tensor memory: block j = k / 32 at columns [48 j, 48 j + 48) of lane k % 32.
__device__ __forceinline__ float4& hdr4(const Smem& s, int f, int k) { return s.hdr[f * s.pcA + k]; }

struct PairC { float v[48]; };      // v[0..35] read-only constants, v[36..47] impulses
constexpr int kLam = 36;

__device__ __forceinline__ void tm_ld16(unsigned a, float* r) {
  unsigned* u = reinterpret_cast<unsigned*>(r);
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
               : "=r"(u[0]), "=r"(u[1]), "=r"(u[2]), "=r"(u[3]), "=r"(u[4]), "=r"(u[5]), "=r"(u[6]), "=r"(u[7]),
                 "=r"(u[8]), "=r"(u[9]), "=r"(u[10]), "=r"(u[11]), "=r"(u[12]), "=r"(u[13]), "=r"(u[14]), "=r"(u[15]) : "r"(a));
}
__device__ __forceinline__ void tm_st16(unsigned a, const float* r) {
  const unsigned* u = reinterpret_cast<const unsigned*>(r);
  asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
               :: "r"(a), "r"(u[0]), "r"(u[1]), "r"(u[2]), "r"(u[3]), "r"(u[4]), "r"(u[5]), "r"(u[6]), "r"(u[7]),
                  "r"(u[8]), "r"(u[9]), "r"(u[10]), "r"(u[11]), "r"(u[12]), "r"(u[13]), "r"(u[14]), "r"(u[15]) : "memory");
}
__device__ __forceinline__ void tm_st4(unsigned a, const float* r) {
  const unsigned* u = reinterpret_cast<const unsigned*>(r);
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};" :: "r"(a), "r"(u[0]), "r"(u[1]), "r"(u[2]), "r"(u[3]) : "memory");
}
__device__ __forceinline__ void tm_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// whole block j (all 32 lanes take part; lane l gets position 32 j + l)
__device__ __forceinline__ void tm_load_block(const Smem& s, int j, PairC& c) {
  const unsigned a = s.tm + 48u * (unsigned)j;
  tm_ld16(a, c.v); tm_ld16(a + 16, c.v + 16); tm_ld16(a + 32, c.v + 32);
}
__device__ __forceinline__ void tm_store_block(const Smem& s, int j, const PairC& c) {
  const unsigned a = s.tm + 48u * (unsigned)j;
  tm_st16(a, c.v); tm_st16(a + 16, c.v + 16); tm_st16(a + 32, c.v + 32);
}
__device__ __forceinline__ void tm_store_lam(const Smem& s, int j, const float* lam) {
  const unsigned a = s.tm + 48u * (unsigned)j + 36u;
  tm_st4(a, lam); tm_st4(a + 4, lam + 4); tm_st4(a + 8, lam + 8);
}
// shared-memory tier: position k >= pos0
__device__ __forceinline__ void sm_load_pair(const Smem& s, int k, PairC& c) {
  const int i = k - s.pos0;
#pragma unroll
  for (int f = 0; f < kCsF4; ++f) { const float4 t = s.cs[f * s.capS + i]; c.v[4 * f] = t.x; c.v[4 * f + 1] = t.y; c.v[4 * f + 2] = t.z; c.v[4 * f + 3] = t.w; }
}
__device__ __forceinline__ void sm_store_pair(const Smem& s, int k, const PairC& c) {
  const int i = k - s.pos0;
#pragma unroll
  for (int f = 0; f < kCsF4; ++f) s.cs[f * s.capS + i] = make_float4(c.v[4 * f], c.v[4 * f + 1], c.v[4 * f + 2], c.v[4 * f + 3]);
}
__device__ __forceinline__ void sm_store_lam(const Smem& s, int k, const float* lam) {
  const int i = k - s.pos0;
#pragma unroll
  for (int f = 0; f < 3; ++f) s.cs[(9 + f) * s.capS + i] = make_float4(lam[4 * f], lam[4 * f + 1], lam[4 * f + 2], lam[4 * f + 3]);
}
// aligned round: lane l <-> position 32 j + l (setup, cache store, lambda output).  All lanes call these.
template <bool TM>
__device__ __forceinline__ void round_load(const Smem& s, int j, int n_valid, PairC& c) {
  if (TM && 32 * j < s.pos0) { tm_load_block(s, j, c); tm_wait_ld(); }
  else if (32 * j + lane_id() < n_valid) sm_load_pair(s, 32 * j + lane_id(), c);
}
template <bool TM>
__device__ __forceinline__ void round_store(const Smem& s, int j, int n_valid, const PairC& c) {
  if (TM && 32 * j < s.pos0) { tm_store_block(s, j, c); tm_wait_st(); }
  else if (32 * j + lane_id() < n_valid) sm_store_pair(s, 32 * j + lane_id(), c);
}

struct Frame { Vec3 n, t1, t2; };

// t1 = normalise(e_k - n (n.e_k)), k = x unless |n_x| > 1/sqrt(2), then y;  t2 = n x t1   (DESIGN §3 R-basis)
__device__ __forceinline__ void tangent_raw(Vec3 n, Vec3& u) {
  const bool usey = fabsf(n.x) > 0.70710678118654752f;
  const float d = usey ? n.y : n.x;
  u = v3(fmaf(-d, n.x, usey ? 0.0f : 1.0f), fmaf(-d, n.y, usey ? 1.0f : 0.0f), -d * n.z);
}
__device__ __forceinline__ Frame make_frame(Vec3 n, float il) {
  Frame F; F.n = n;
  Vec3 u; tangent_raw(n, u);
  F.t1 = il * u;
  F.t2 = cross(n, F.t1);
  return F;
}

struct Body5 { float4 x, v, w, i0, i1; };     // x.w = inverse mass (0: static / inactive / ground)

__device__ __forceinline__ void load_body(const Smem& s, int b, Body5& o, bool with_vel) {
  if (b >= 0) {
    o.x = bd4(s, b, 0); o.i0 = bd4(s, b, 3); o.i1 = bd4(s, b, 4);
    if (with_vel) { o.v = bd4(s, b, 1); o.w = bd4(s, b, 2); }
  } else {
    o.x = o.v = o.w = o.i0 = o.i1 = make_float4(0, 0, 0, 0);
  }
}
__device__ __forceinline__ Vec3 imul(const Body5& B, Vec3 a) {      // Iw^-1 a
  return v3(fmaf(B.i0.z, a.z, fmaf(B.i0.y, a.y, B.i0.x * a.x)),
            fmaf(B.i1.x, a.z, fmaf(B.i0.w, a.y, B.i0.y * a.x)),
            fmaf(B.i1.y, a.z, fmaf(B.i1.x, a.y, B.i0.z * a.x)));
}
__device__ __forceinline__ Vec3 xyz(float4 v) { return v3(v.x, v.y, v.z); }

// S4 for one colliding pair: writes slot k from the pair's manifold.  Warm start (DESIGN §3 R-warm): a new
// contact inherits (jn,jt1,jt2) of the nearest not yet taken previous contact point of the same pair
// within match_tol; slots ascending.
__device__ inline void setup_slot(const Smem& s, const Params& P, int env, int k, int a, int b, int pair,
                                  const Manifold& m, PairC& out, int prev_buf = 0) {
  Body5 A, Bb; load_body(s, a, A, false); load_body(s, b, Bb, false);
  const Vec3 n = m.n;
  Vec3 u; tangent_raw(n, u);
  const float il = rsqrtf(dot(u, u));
  const Frame F = make_frame(n, il);
  const Vec3 dir[3] = { F.n, F.t1, F.t2 };
  const float im = A.x.w + Bb.x.w;
  float lam[4][3]; Vec3 pt[4];
  float dmax = 0.0f;
#pragma unroll
  for (int c = 0; c < 4; ++c) { lam[c][0] = lam[c][1] = lam[c][2] = 0.0f; pt[c] = v3(0, 0, 0); }
#pragma unroll
  for (int c = 0; c < 4; ++c) if (c < m.np) { pt[c] = m.p[c]; dmax = fmaxf(dmax, m.d[c]); }

  if (P.warm_start) {
    // cache entry = rank of the pair in the previous substep's colliding list: that list is still in shared memory
    // (s.cpair[prev]) inside a launch; at the first substep of a launch the keys are read from HBM.
    const int* keys = P.cache_key + (size_t)env * P.pc * 2;
    const int nprev = s.misc[MiNprev];
    int nk, lo = 0; bool found;
    if (nprev >= 0) {
      nk = nprev; int hi = nk;
      while (lo < hi) { const int mid = (lo + hi) >> 1; if ((int)s.cpair[prev_buf][mid] < pair) lo = mid + 1; else hi = mid; }
      found = lo < nk && (int)s.cpair[prev_buf][lo] == pair;
    } else {
      nk = P.n_cache[env]; int hi = nk;
      while (lo < hi) { const int mid = (lo + hi) >> 1; if (keys[2 * mid] < pair) lo = mid + 1; else hi = mid; }
      found = lo < nk && keys[2 * lo] == pair;
    }
    if (found) {
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
        if (c < m.np) {
          int bo = -1; float bdist = tol2;
#pragma unroll
          for (int o = 0; o < 4; ++o)
            if (o < ocnt && !((taken >> o) & 1u)) {
              const Vec3 d = pt[c] - q[o]; const float dd = dot(d, d);
              if (dd < bdist) { bdist = dd; bo = o; }
            }
#pragma unroll
          for (int o = 0; o < 4; ++o)
            if (o == bo) { taken |= 1u << o; lam[c][0] = l[o][0]; lam[c][1] = l[o][1]; lam[c][2] = l[o][2]; }
        }
      }
    }
  }

  const int meta = m.np | (m.axis << 8) | (pair << 16);
  hdr4(s, 0, k) = make_float4(__int_as_float(a), __int_as_float(b), __int_as_float(meta), il);
  hdr4(s, 1, k) = make_float4(n.x, n.y, n.z, im > 0.0f ? P.beta * fmaxf(0.0f, dmax - P.slop) / im : 0.0f);
  const float e1 = 1.0f + P.restitution;
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    float ik[3] = { 0, 0, 0 }, ko[3] = { 0, 0, 0 };
    if (c < m.np) {
      const Vec3 rA = a >= 0 ? pt[c] - xyz(A.x) : v3(0, 0, 0), rB = pt[c] - xyz(Bb.x);
      Vec3 uA[3], uB[3], wA[3], wB[3];
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        uA[d] = cross(rA, dir[d]); uB[d] = cross(rB, dir[d]);
        wA[d] = imul(A, uA[d]); wB[d] = imul(Bb, uB[d]);
      }
#pragma unroll
      for (int d = 0; d < 3; ++d) ik[d] = 1.0f / (im + dot(uA[d], wA[d]) + dot(uB[d], wB[d]));
      ik[0] *= e1;
      ko[0] = dot(uA[0], wA[1]) + dot(uB[0], wB[1]);
      ko[1] = dot(uA[0], wA[2]) + dot(uB[0], wB[2]);
      ko[2] = dot(uA[1], wA[2]) + dot(uB[1], wB[2]);
    }
    float* o = out.v + 9 * c;
    o[0] = pt[c].x; o[1] = pt[c].y; o[2] = pt[c].z; o[3] = ik[0]; o[4] = ik[1]; o[5] = ik[2]; o[6] = ko[0]; o[7] = ko[1]; o[8] = ko[2];
    out.v[kLam + 3 * c] = lam[c][0]; out.v[kLam + 3 * c + 1] = lam[c][1]; out.v[kLam + 3 * c + 2] = lam[c][2];
  }
}

// S3 second half + S4: lane l of round j takes colour-sorted position 32 j + l, computes the pair's manifold
// (same SAT code as find_colliding -> same decisions) and writes its header and contact constants.
template <bool TM>
__device__ inline void setup_pairs(const Smem& s, const Params& P, int env, int n_coll, int cur) {
  const int S = P.S, lane = lane_id();
  for (int j = 0; 32 * j < n_coll; ++j) {
    const int k = 32 * j + lane;
    PairC c;
#pragma unroll
    for (int t = 0; t < 48; ++t) c.v[t] = 0.0f;
    if (k < n_coll) {
      const int r = s.order[k];
      const unsigned w = s.cab[r];
      const int a = ab_a(w), b = ab_b(w);
      Manifold m; m.np = 0; m.axis = 0; m.n = v3(0, 0, 1);
      pair_manifold(s, S, a, b, ab_axis(w), m);
      setup_slot(s, P, env, k, a, b, s.cpair[cur][r], m, c, cur ^ 1);
    }
    round_store<TM>(s, j, n_coll, c);
  }
  __syncwarp();
}

// a loses the impulse, b gains it (Listing 1, PAPER.md:335-336 + the angular lines, reading A11)
__device__ __forceinline__ void apply_impulse(Body5& A, Body5& B, Vec3 rA, Vec3 rB, Vec3 Pi) {
  A.v.x = fmaf(-A.x.w, Pi.x, A.v.x); A.v.y = fmaf(-A.x.w, Pi.y, A.v.y); A.v.z = fmaf(-A.x.w, Pi.z, A.v.z);
  B.v.x = fmaf(B.x.w, Pi.x, B.v.x);  B.v.y = fmaf(B.x.w, Pi.y, B.v.y);  B.v.z = fmaf(B.x.w, Pi.z, B.v.z);
  const Vec3 cA = cross(Pi, rA), cB = cross(rB, Pi);        // -(rA x Pi), +(rB x Pi)
  A.w.x = fmaf(A.i0.z, cA.z, fmaf(A.i0.y, cA.y, fmaf(A.i0.x, cA.x, A.w.x)));
  A.w.y = fmaf(A.i1.x, cA.z, fmaf(A.i0.w, cA.y, fmaf(A.i0.y, cA.x, A.w.y)));
  A.w.z = fmaf(A.i1.y, cA.z, fmaf(A.i1.x, cA.y, fmaf(A.i0.z, cA.x, A.w.z)));
  B.w.x = fmaf(B.i0.z, cB.z, fmaf(B.i0.y, cB.y, fmaf(B.i0.x, cB.x, B.w.x)));
  B.w.y = fmaf(B.i1.x, cB.z, fmaf(B.i0.w, cB.y, fmaf(B.i0.y, cB.x, B.w.y)));
  B.w.z = fmaf(B.i1.y, cB.z, fmaf(B.i1.x, cB.y, fmaf(B.i0.z, cB.x, B.w.z)));
}

// One colour chunk of the warm-start application (S4) or of a Gauss-Seidel sweep (S5).  Lane l takes the pair at
// colour-sorted position k = start + ((l - start) mod 32), i.e. lane = k mod 32 (the lane that owns the pair's
// TMEM row): slots ascending; per contact the normal row (Eq. 14, clamp >= 0), then t1, then t2 (Eq. 15, each
// clipped to +-mu_s jn) -- Listing 1.  The three rows of a contact act on the same two bodies:
// the relative velocity of the contact point is read once, advanced between rows with the contact-space couplings
// K_ij (exactly the change the applied impulse causes), and the summed impulse is applied once (DESIGN §3
// R-couple).  Pairs of one colour share no dynamic body.
template <bool TM, bool WARM>
__device__ __forceinline__ void solve_chunk(const Smem& s, int start, int count, float mu) {
  const int lane = lane_id();
  const int k = start + ((lane - start) & 31);
  const bool active = k < start + count;
  const int jA = start >> 5;
  const bool in_tm = TM && start < s.pos0;                       // chunks never straddle pos0
  const bool span = (start & 31) + count > 32;
  PairC c;
  float keepA[12], keepB[12];                                    // impulses of the lanes that are not in this chunk
  if (in_tm) {
    tm_load_block(s, jA, c);
    PairC o;
    if (span) tm_load_block(s, jA + 1, o);
    tm_wait_ld();
    const bool mineB = (k >> 5) != jA;
#pragma unroll
    for (int t = 0; t < 12; ++t) { keepA[t] = c.v[kLam + t]; keepB[t] = span ? o.v[kLam + t] : 0.0f; }
    if (span) {
#pragma unroll
      for (int t = 0; t < 48; ++t) c.v[t] = mineB ? o.v[t] : c.v[t];
    }
  } else if (active) {
    sm_load_pair(s, k, c);
  }
  if (active) {
    const float4 h = hdr4(s, 0, k), nn = hdr4(s, 1, k);
    const int a = __float_as_int(h.x), b = __float_as_int(h.y), np = __float_as_int(h.z) & 0xff;
    Body5 A, B; load_body(s, a, A, true); load_body(s, b, B, true);
    const Frame F = make_frame(xyz(nn), h.w);
#pragma unroll
    for (int ci = 0; ci < 4; ++ci)
      if (ci < np) {
        const float* r = c.v + 9 * ci; float* l = c.v + kLam + 3 * ci;
        const Vec3 p = v3(r[0], r[1], r[2]), rA = p - xyz(A.x), rB = p - xyz(B.x);
        Vec3 Pi;
        if (WARM) {
          Pi = madd(madd(l[0] * F.n, l[1], F.t1), l[2], F.t2);
        } else {
          // vr = (vB + wB x rB) - (vA + wA x rA), each component one subtraction and four fused multiply-adds
          const Vec3 vr = v3(
            fmaf(A.w.z, rA.y, fmaf(-A.w.y, rA.z, fmaf(-B.w.z, rB.y, fmaf(B.w.y, rB.z, B.v.x - A.v.x)))),
            fmaf(A.w.x, rA.z, fmaf(-A.w.z, rA.x, fmaf(-B.w.x, rB.z, fmaf(B.w.z, rB.x, B.v.y - A.v.y)))),
            fmaf(A.w.y, rA.x, fmaf(-A.w.x, rA.y, fmaf(-B.w.y, rB.x, fmaf(B.w.x, rB.y, B.v.z - A.v.z)))));
          const float u0 = dot(vr, F.n);
          float u1 = dot(vr, F.t1), u2 = dot(vr, F.t2);
          const float nw = fmaxf(fmaf(-u0, r[3], l[0]), 0.0f);
          const float d0 = nw - l[0];
          u1 = fmaf(r[6], d0, u1); u2 = fmaf(r[7], d0, u2);
          const float lim = mu * nw;
          const float n1 = fminf(fmaxf(fmaf(-u1, r[4], l[1]), -lim), lim);
          const float d1 = n1 - l[1];
          u2 = fmaf(r[8], d1, u2);
          const float n2 = fminf(fmaxf(fmaf(-u2, r[5], l[2]), -lim), lim);
          const float d2 = n2 - l[2];
          l[0] = nw; l[1] = n1; l[2] = n2;
          Pi = madd(madd(d0 * F.n, d1, F.t1), d2, F.t2);
        }
        apply_impulse(A, B, rA, rB, Pi);
      }
    if (a >= 0) { bd4(s, a, 1) = A.v; bd4(s, a, 2) = A.w; }
    bd4(s, b, 1) = B.v; bd4(s, b, 2) = B.w;
    if (!WARM && !in_tm) sm_store_lam(s, k, c.v + kLam);
  }
  if (!WARM && in_tm) {                                          // all lanes: rows outside the chunk get their old values back
    const bool mineB = (k >> 5) != jA;
#pragma unroll
    for (int t = 0; t < 12; ++t) {
      const float mine = c.v[kLam + t];
      keepA[t] = (active && !mineB) ? mine : keepA[t];
      keepB[t] = (active && mineB) ? mine : keepB[t];
    }
    tm_store_lam(s, jA, keepA);
    if (span) tm_store_lam(s, jA + 1, keepB);
    tm_wait_st();
  }
  __syncwarp();
}

// S4 (warm-start application) + S5: the phase chunks in canonical order, `iters` sweeps.
template <bool TM>
__device__ inline void pgs_sweeps(const Smem& s, const Params& P, int iters, float mu) {
  const int nph = s.misc[MiNph];
  if (P.warm_start)
    for (int j = 0; j < nph; ++j) { const int w = s.ph[j]; solve_chunk<TM, true>(s, w & 0xffff, w >> 16, mu); }
  for (int it = 0; it < iters; ++it)
    for (int j = 0; j < nph; ++j) { const int w = s.ph[j]; solve_chunk<TM, false>(s, w & 0xffff, w >> 16, mu); }
}

// S6: x += h v (Eq. 6); q <- normalise(q + h/2 [0,w] (x) q) (Eq. 2, world-frame
// reading A3); then Eq. 16 (reading A14) once per colliding pair, colour by colour.
__device__ inline void integrate(const Smem& s, const Params& P, unsigned* status) {
  const int S = P.S, lane = lane_id(); const float h = P.h;
  for (int b = lane; b < P.B; b += 32) {
    float4 x = bd4(s, b, 0);
    if (x.w == 0.0f) continue;                                   // static or inactive
    const float4 v = bd4(s, b, 1), om = bd4(s, b, 2);
    x.x += h * v.x; x.y += h * v.y; x.z += h * v.z;
    bd4(s, b, 0) = x;
    const float qw = s.q[b], qx = s.q[S + b], qy = s.q[2 * S + b], qz = s.q[3 * S + b];
    const float dw = -(om.x * qx + om.y * qy + om.z * qz);
    const float dx = om.x * qw + om.y * qz - om.z * qy;
    const float dy = om.y * qw + om.z * qx - om.x * qz;
    const float dz = om.z * qw + om.x * qy - om.y * qx;
    const float hh = 0.5f * h;
    const float nw = qw + hh * dw, nx = qx + hh * dx, ny = qy + hh * dy, nz = qz + hh * dz;
    const float il = 1.0f / sqrtf(nw * nw + nx * nx + ny * ny + nz * nz);
    s.q[b] = nw * il; s.q[S + b] = nx * il; s.q[2 * S + b] = ny * il; s.q[3 * S + b] = nz * il;
    if (!(isfinite(x.x) && isfinite(x.y) && isfinite(x.z) && isfinite(v.x) && isfinite(v.y) && isfinite(v.z)))
      *status |= JENGA_ST_NONFINITE;
  }
  __syncwarp();
  const int nph = s.misc[MiNph];
  for (int j = 0; j < nph; ++j) {
    const int w = s.ph[j], k = (w & 0xffff) + lane;
    float4 nn = make_float4(0, 0, 0, 0);
    if (lane < (w >> 16)) nn = hdr4(s, 1, k);
    if (__any_sync(kFull, nn.w > 0.0f)) {
      if (nn.w > 0.0f) {
        const float4 hd = hdr4(s, 0, k);
        const int a = __float_as_int(hd.x), b = __float_as_int(hd.y);
        float4 xb = bd4(s, b, 0);
        if (xb.w != 0.0f) {
          const float f = xb.w * nn.w;
          xb.x += f * nn.x; xb.y += f * nn.y; xb.z += f * nn.z;
          bd4(s, b, 0) = xb;
        }
        if (a >= 0) {
          float4 xa = bd4(s, a, 0);
          if (xa.w != 0.0f) {
            const float f = xa.w * nn.w;
            xa.x -= f * nn.x; xa.y -= f * nn.y; xa.z -= f * nn.z;
            bd4(s, a, 0) = xa;
          }
        }
      }
      __syncwarp();
    }
  }
}

// Collapse latch (Eq. 18, reading A17) after a dt advance: dx_max = max_b |x_b - x_b(0)|,
// theta_max = max_b 2 acos|q_b . q_b(0)|, E_k = sum_b 1/2 m |v|^2 + 1/2 w . I_w w (body frame: R^T w against the
// principal moments); collapsed |= all three above their thresholds at this step.
__device__ inline void collapse_latch(const Smem& s, const Params& P, int env) {
  const int S = P.S, lane = lane_id();
  const float* ref = P.ref_pose + (size_t)env * 7 * S;
  float dxm = 0.0f, thm = 0.0f, ek = 0.0f;
  for (int b = lane; b < P.B; b += 32) {
    const float4 x = bd4(s, b, 0);
    if (x.w == 0.0f) continue;
    const float dx = x.x - ref[b], dy = x.y - ref[S + b], dz = x.z - ref[2 * S + b];
    dxm = fmaxf(dxm, sqrtf(dx * dx + dy * dy + dz * dz));
    const float qw = s.q[b], qx = s.q[S + b], qy = s.q[2 * S + b], qz = s.q[3 * S + b];
    const float c = fminf(fabsf(qw * ref[3 * S + b] + qx * ref[4 * S + b] + qy * ref[5 * S + b] + qz * ref[6 * S + b]), 1.0f);
    thm = fmaxf(thm, 2.0f * acosf(c));
    const float4 v = bd4(s, b, 1), w = bd4(s, b, 2);
    // R^T w with R from the new q (Eq. 1)
    const float r00 = 1.0f - 2.0f * (qy * qy + qz * qz), r01 = 2.0f * (qx * qy - qz * qw), r02 = 2.0f * (qx * qz + qy * qw);
    const float r10 = 2.0f * (qx * qy + qz * qw), r11 = 1.0f - 2.0f * (qx * qx + qz * qz), r12 = 2.0f * (qy * qz - qx * qw);
    const float r20 = 2.0f * (qx * qz - qy * qw), r21 = 2.0f * (qy * qz + qx * qw), r22 = 1.0f - 2.0f * (qx * qx + qy * qy);
    const float w0 = r00 * w.x + r10 * w.y + r20 * w.z, w1 = r01 * w.x + r11 * w.y + r21 * w.z, w2 = r02 * w.x + r12 * w.y + r22 * w.z;
    ek += 0.5f * (v.x * v.x + v.y * v.y + v.z * v.z) / x.w
        + 0.5f * (w0 * w0 / s.pr[S + b] + w1 * w1 / s.pr[2 * S + b] + w2 * w2 / s.pr[3 * S + b]);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    dxm = fmaxf(dxm, __shfl_xor_sync(kFull, dxm, o)); thm = fmaxf(thm, __shfl_xor_sync(kFull, thm, o));
    ek += __shfl_xor_sync(kFull, ek, o);
  }
  if (lane == 0) {
    if (dxm > P.collapse_dx && ek > P.collapse_ek && thm > P.collapse_theta) P.collapsed[env] = 1;
    if (P.collapse_stats) *reinterpret_cast<float4*>(P.collapse_stats + (size_t)env * 4) = make_float4(dxm, ek, thm, 0.0f);
  }
}

// Total kinetic energy of the env: sum_b 1/2 m |v|^2 + 1/2 w . I w, I in the body frame.
__device__ inline float env_kinetic_energy(const Smem& s, const Params& P) {
  const int S = P.S;
  float ek = 0.0f;
  for (int b = lane_id(); b < P.B; b += 32) {
    const float4 x = bd4(s, b, 0);
    if (x.w == 0.0f) continue;
    const float4 v = bd4(s, b, 1), w = bd4(s, b, 2);
    const float qw = s.q[b], qx = s.q[S + b], qy = s.q[2 * S + b], qz = s.q[3 * S + b];
    const float r00 = 1.0f - 2.0f * (qy * qy + qz * qz), r01 = 2.0f * (qx * qy - qz * qw), r02 = 2.0f * (qx * qz + qy * qw);
    const float r10 = 2.0f * (qx * qy + qz * qw), r11 = 1.0f - 2.0f * (qx * qx + qz * qz), r12 = 2.0f * (qy * qz - qx * qw);
    const float r20 = 2.0f * (qx * qz - qy * qw), r21 = 2.0f * (qy * qz + qx * qw), r22 = 1.0f - 2.0f * (qx * qx + qy * qy);
    const float w0 = r00 * w.x + r10 * w.y + r20 * w.z, w1 = r01 * w.x + r11 * w.y + r21 * w.z, w2 = r02 * w.x + r12 * w.y + r22 * w.z;
    ek += 0.5f * (v.x * v.x + v.y * v.y + v.z * v.z) / x.w
        + 0.5f * (w0 * w0 / s.pr[S + b] + w1 * w1 / s.pr[2 * S + b] + w2 * w2 / s.pr[3 * S + b]);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) ek += __shfl_xor_sync(kFull, ek, o);
  return ek;
}

// S7: every pair's impulses and contact points become the next substep's warm-start cache, in ascending
// pair order (cache entry r = pair rank r).  Returns the lane's (contacts, ground contacts) for the counters.
template <bool TM>
__device__ inline int2 store_cache(const Smem& s, const Params& P, int env, int n_coll) {
  const int lane = lane_id();
  int nc = 0, ng = 0;
  for (int j = 0; 32 * j < n_coll; ++j) {
    const int k = 32 * j + lane;
    PairC c; round_load<TM>(s, j, n_coll, c);
    if (k < n_coll) {
      const int r = s.order[k];
      const float4 hd = hdr4(s, 0, k);
      const int meta = __float_as_int(hd.z), np = meta & 0xff;
      nc += np; if (__float_as_int(hd.x) < 0) ng += np;
      int* key = P.cache_key + ((size_t)env * P.pc + r) * 2;
      key[0] = (int)((unsigned)meta >> 16); key[1] = meta & 0xfff;
      float* ol = P.cache_lam + ((size_t)env * P.pc + r) * 12;
      float* op = P.cache_pt + ((size_t)env * P.pc + r) * 12;
#pragma unroll
      for (int ci = 0; ci < 4; ++ci) {
        const bool on = ci < np;
#pragma unroll
        for (int t = 0; t < 3; ++t) { ol[3 * ci + t] = on ? c.v[kLam + 3 * ci + t] : 0.0f; op[3 * ci + t] = c.v[9 * ci + t]; }
      }
    }
  }
  if (lane == 0) P.n_cache[env] = n_coll;
  __syncwarp();
  return make_int2(nc, ng);
}

// ---------------------------------------------------------------- materialised outputs (stage calls / parity)
__device__ inline void write_pairs(const Smem& s, const Params& P, int env, int n_cand) {
  int* out = P.pairs + (size_t)env * P.max_pairs;
  for (int k = lane_id(); k < n_cand; k += 32) out[k] = s.cand[k];
  if (lane_id() == 0) P.n_pairs[env] = n_cand;
  __syncwarp();
}

__device__ __forceinline__ int warp_excl_scan(int v, int* total) {
  const int lane = lane_id();
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(kFull, inc, o); if (lane >= o) inc += t; }
  *total = __shfl_sync(kFull, inc, 31);
  return inc - v;
}

// Contact list in (pair, slot) order: the manifolds are recomputed from the (unchanged) poses in ascending
// pair order, so nothing has to be kept on chip for the debug output.  Leaves s.wrank[r] = contact offset.
__device__ inline int write_contacts(const Smem& s, const Params& P, int env, int n_cand, int n_coll, int cur) {
  const int S = P.S, lane = lane_id();
  int off0 = 0;
  for (int base = 0; base < n_coll; base += 32) {
    const int r = base + lane;
    Manifold m; m.np = 0; m.axis = 0; m.n = v3(0, 0, 1);
    int idx = 0;
    if (r < n_coll) {
      const unsigned w = s.cab[r];
      const int a = ab_a(w), b = ab_b(w);
      idx = s.cpair[cur][r];
      pair_manifold(s, S, a, b, ab_axis(w), m);
    }
    int tot; const int off = off0 + warp_excl_scan(m.np, &tot);
    if (r < n_coll) {
      s.wrank[r] = (unsigned short)off;
      const int* gp = P.pairs + (size_t)env * P.max_pairs;      // position of the pair in the candidate list (the
      int lo = 0, hi = n_cand;                                   // on-chip copy may already be overwritten by the slots)
      while (lo < hi) { const int mid = (lo + hi) >> 1; if (gp[mid] < idx) lo = mid + 1; else hi = mid; }
      float4* out = reinterpret_cast<float4*>(P.contacts + ((size_t)env * P.max_contacts + off) * 8);
      for (int c = 0; c < m.np; ++c) {
        const int tag = (lo & 0xffff) | (c << 16) | (m.axis << 20);
        out[2 * c] = make_float4(m.n.x, m.n.y, m.n.z, m.d[c]);
        out[2 * c + 1] = make_float4(m.p[c].x, m.p[c].y, m.p[c].z, __int_as_float(tag));
      }
    }
    off0 += tot;
  }
  if (lane == 0) P.n_contacts[env] = off0;
  __syncwarp();
  return off0;
}

// lambda in contact order; needs s.wrank[r] = contact offset of pair r.
template <bool TM>
__device__ inline void write_lambda(const Smem& s, const Params& P, int env, int n_coll) {
  for (int j = 0; 32 * j < n_coll; ++j) {
    const int k = 32 * j + lane_id();
    PairC c; round_load<TM>(s, j, n_coll, c);
    if (k < n_coll) {
      const int r = s.order[k];
      const int np = __float_as_int(hdr4(s, 0, k).z) & 0xff;
      float* out = P.lambda + ((size_t)env * P.max_contacts + s.wrank[r]) * 3;
#pragma unroll
      for (int ci = 0; ci < 4; ++ci)
        if (ci < np) { out[3 * ci] = c.v[kLam + 3 * ci]; out[3 * ci + 1] = c.v[kLam + 3 * ci + 1]; out[3 * ci + 2] = c.v[kLam + 3 * ci + 2]; }
    }
  }
}

}  // namespace jenga
