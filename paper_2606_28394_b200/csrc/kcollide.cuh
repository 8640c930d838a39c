// kcollide.cuh -- the collision kernels of a substep, one env per warp.  k_detect: S1 predict, S2 broadphase, S3 SAT
// (which candidates collide).  k_walk: S4 canonical greedy colouring (one env per thread; only envs whose pair list
// changed).  k_plan: the group's visit plan (only for groups with such an env).  k_manifold: S3 contact manifolds.  k_slot: S4 contact setup (effective masses, warm-start lookup).  Their
// products go to the scratch buffer (layout.cuh) for the next kernel.  They are separate kernels because each one's hot
// code then fits the 32 KB instruction cache (as one kernel: 70 KB, and `no_instruction` was the top stall with 16 warps
// per SM at different places in it).
#pragma once
#include "layout.cuh"

namespace jenga {

// ---------------------------------------------------------------- shared-memory arena of one env
struct CSm {
  SP<float> cb;                 // [S][cbw] collision body records: x y z im | a0 h0 | a1 h1 | a2 h2 | then q (k_detect) or Iw^-1 (k_slot)
  int cbw;                      // words per record: 20 (k_detect, k_manifold) or kCb = 28 (k_slot); a multiple of 4, odd in float4
  SP<float4> ext;               // [S]      world AABB half extents e'_x e'_y e'_z, flags (1 active | 2 dynamic)
  SP<unsigned> hitw;            // [ceil(S/32)][32] broadphase hit words of the current block of 32 rows
  SP<unsigned long long> used;  // unused (k_walk keeps the colour masks per body in its own layout)
  SP<unsigned> cab;             // [pcA]    (a+1) | A dynamic << 11 | axis << 12 | b << 16 | B dynamic << 27
  SP<unsigned short> cand;      // [mpA]    candidate pair indices, ascending
  SP<float> poly;               // [8][3][32] clip polygon of every lane (component-major: lane l <-> bank l)
  SP<unsigned short> cpair;     // [pcA]    colliding pair indices, ascending
  SP<unsigned short> cprev;     // [pcA]    pair indices of the warm-start cache (previous substep), ascending
  SP<unsigned short> pos;       // [pcA]    position of pair r
  SP<unsigned short> wrank;     // [pcA]    rank inside its colour / contact offset
  SP<unsigned char> colour;     // [pcA]
  SP<int> ph;                   // [ph_max] chunk descriptors of the GROUP in the order the solver visits them
  SP<int> chm;                  // [kMaxGroup][ph_max] per member: colour | first rank-in-colour << 6 | pairs << 20 of each chunk
  SP<int> ccount;               // [64] pairs of each colour of this env (the sibling warp reads it)
  SP<int> cfirst;               // [64] first chunk with pairs of the colour (this env's)
  SP<int> fill;                 // [nblk] lanes taken in each block (packing)
  SP<int> misc;                 // [8]
};
enum { MiNph = 0, MiNcol = 1, MiNblk = 2, MiSame = 3 };

enum { ArenaDetect = 0, ArenaManifold = 1, ArenaSlot = 2, ArenaPlan = 3 };

// k_detect: records, extents, hit words, candidate list, colliding list.  k_plan: colouring and
// plan products (no body records).  k_manifold: records, colliding list (copied from the scratch), per-lane clip
// polygons.  k_slot: records, colliding list, cache keys.
__host__ __device__ inline int cb_words(int arena) { return arena == ArenaSlot ? kCb : (arena == ArenaPlan ? 0 : 20); }

__host__ __device__ inline size_t collide_smem_words(int S, int max_pairs, int pc, int arena, int G) {
  const int pcA = round_up(pc, 8), mpA = round_up(max_pairs, 8), nblk = n_blocks(pc, G);
  if (arena == ArenaPlan) {                                // wrank, colour, ph, chm, ccount, cfirst, fill, misc
    const int phw = round_up(ph_max(nblk, G), 4);
    return round_up(pcA / 2 + pcA / 4 + (1 + kMaxGroup) * phw + 2 * kMaxColours + round_up(nblk, 4) + 8, 4);
  }
  size_t w = (size_t)cb_words(arena) * S + pcA + pcA / 2;  // cb, cab, cpair
  if (arena != ArenaManifold) w += 2 * (size_t)(pcA / 2);  // pos, wrank
  if (arena == ArenaDetect) {
    const int uh = 32 * ((S + 31) / 32);
    w += 4 * S + uh + mpA / 2 + 8;                         // ext, hitw, cand, misc
  } else if (arena == ArenaManifold) {
    w += 768;                                              // poly
  } else {
    w += pcA / 2;                                          // cprev
  }
  return round_up((int)w, 4);
}

__device__ inline CSm carve_collide(int S, int max_pairs, int pc, int base, int arena, int G) {
  const int pcA = round_up(pc, 8), mpA = round_up(max_pairs, 8), nblk = n_blocks(pc, G), phw = round_up(ph_max(nblk, G), 4);
  CSm s; int p = base;
  s.cbw = cb_words(arena);
  if (arena == ArenaPlan) {
    s.cb.off = s.cab.off = s.cpair.off = s.pos.off = s.ext.off = s.hitw.off = s.used.off = s.cand.off = s.cprev.off = s.poly.off = 0;
    s.wrank.off = p;  p += pcA / 2;
    s.colour.off = p; p += pcA / 4;
    s.ph.off = p;     p += phw;
    s.chm.off = p;    p += kMaxGroup * phw;
    s.ccount.off = p; p += kMaxColours;
    s.cfirst.off = p; p += kMaxColours;
    s.fill.off = p;   p += round_up(nblk, 4);
    s.misc.off = p;
    return s;
  }
  s.cb.off = p;     p += s.cbw * S;
  s.cab.off = p;    p += pcA;
  s.cpair.off = p;  p += pcA / 2;
  s.pos.off = s.wrank.off = 0;
  if (arena != ArenaManifold) { s.pos.off = p; p += pcA / 2; s.wrank.off = p; p += pcA / 2; }
  // the arrays of the other arena get offset 0 (never touched by this kernel)
  s.ext.off = s.hitw.off = s.used.off = s.cand.off = s.colour.off = s.ph.off = s.chm.off = 0;
  s.ccount.off = s.cfirst.off = s.fill.off = s.misc.off = s.cprev.off = s.poly.off = 0;
  if (arena == ArenaDetect) {
    s.ext.off = p;    p += 4 * S;
    s.hitw.off = p;   p += 32 * ((S + 31) / 32);
    s.cand.off = p;   p += mpA / 2;
    s.misc.off = p;
  } else if (arena == ArenaManifold) {
    s.poly.off = p;
  } else {
    s.cprev.off = p;
  }
  return s;
}

__device__ __forceinline__ Vec3 xyz(float4 v) { return v3(v.x, v.y, v.z); }
__device__ __forceinline__ Vec3 xyz4(float4 v) { return v3(v.x, v.y, v.z); }
__device__ __forceinline__ float4& cb4(const CSm& s, int b, int k) { return reinterpret_cast<float4*>(smem_f + s.cb.off + b * s.cbw)[k]; }

__device__ __forceinline__ Box load_box(const CSm& s, int b) {
  Box X;
  const float4 x = cb4(s, b, 0), a0 = cb4(s, b, 1), a1 = cb4(s, b, 2), a2 = cb4(s, b, 3);
  X.c = v3(x.x, x.y, x.z);
  X.ax[0] = v3(a0.x, a0.y, a0.z); X.ax[1] = v3(a1.x, a1.y, a1.z); X.ax[2] = v3(a2.x, a2.y, a2.z);
  X.he[0] = a0.w; X.he[1] = a1.w; X.he[2] = a2.w;
  return X;
}

// ---------------------------------------------------------------- S1: load, R, Iw^-1, AABB extents, velocity predict
// state [13][S] and props [8][S] of one env are contiguous in HBM; lane b reads column b of every row (coalesced).
// Eq. 1, I_world^-1 = R diag(I_body^-1) R^T, e'_k = sum_j |R_kj| e_j;
// v += h (g + f/m), w += h Iw^-1 (tau [- w x Iw w]) (Eq. 5; reading A2): written back to `state`.
__device__ inline void load_predict(const CSm& s, const Params& P, int env, bool predict, bool want_ext = true) {
  const int S = P.S;
  float* st = P.state + (size_t)env * kStateRows * S;
  const float* pr = P.props + (size_t)env * kPropRows * S;
  for (int b = lane_id(); b < P.B; b += 32) {
    const float px = st[b], py = st[S + b], pz = st[2 * S + b];
    const float w = st[3 * S + b], x = st[4 * S + b], y = st[5 * S + b], z = st[6 * S + b];
    const float im = pr[b], i0r = pr[S + b], i1r = pr[2 * S + b], i2r = pr[3 * S + b];
    const float hx = pr[4 * S + b], hy = pr[5 * S + b], hz = pr[6 * S + b];
    const bool act = pr[7 * S + b] != 0.0f, dyn = act && im != 0.0f;
    float R[9]; quat_to_R(w, x, y, z, R);
    float e3[3];
#pragma unroll
    for (int k = 0; k < 3; ++k)
      e3[k] = fabsf(R[3 * k]) * hx + fabsf(R[3 * k + 1]) * hy + fabsf(R[3 * k + 2]) * hz;
    if (want_ext) s.ext[b] = make_float4(e3[0], e3[1], e3[2], (act ? 1.0f : 0.0f) + (dyn ? 2.0f : 0.0f));
    float I6[6];
    world_inv_inertia(R, dyn ? i0r : 0.0f, dyn ? i1r : 0.0f, dyn ? i2r : 0.0f, I6);
    cb4(s, b, 0) = make_float4(px, py, pz, dyn ? im : 0.0f);
    cb4(s, b, 1) = make_float4(R[0], R[3], R[6], hx);        // body axis k = column k of R
    cb4(s, b, 2) = make_float4(R[1], R[4], R[7], hy);
    cb4(s, b, 3) = make_float4(R[2], R[5], R[8], hz);
    if (s.cbw == kCb) {                                      // k_slot: the effective masses need Iw^-1
      cb4(s, b, 4) = make_float4(I6[0], I6[1], I6[2], I6[3]);
      cb4(s, b, 5) = make_float4(I6[4], I6[5], 0.0f, 0.0f);
    } else if (want_ext) {
      cb4(s, b, 4) = make_float4(w, x, y, z);                // k_detect: the fp64 re-check of threshold AABB tests
    }
    if (!predict || !dyn) continue;
    float f[6] = { 0, 0, 0, 0, 0, 0 };
    if (P.f_ext) {
      const float* fe = P.f_ext + (size_t)env * kFextRows * S;
#pragma unroll
      for (int k = 0; k < 6; ++k) f[k] = fe[k * S + b];
    }
    float vx = st[7 * S + b], vy = st[8 * S + b], vz = st[9 * S + b];
    const Vec3 wv = v3(st[10 * S + b], st[11 * S + b], st[12 * S + b]);
    vx += P.h * (P.g[0] + im * f[0]); vy += P.h * (P.g[1] + im * f[1]); vz += P.h * (P.g[2] + im * f[2]);
    Vec3 tau = v3(f[3], f[4], f[5]);
    if (P.gyroscopic) {                  // I_world w = R diag(I_body) R^T w
      const float wb0 = R[0] * wv.x + R[3] * wv.y + R[6] * wv.z, wb1 = R[1] * wv.x + R[4] * wv.y + R[7] * wv.z,
                  wb2 = R[2] * wv.x + R[5] * wv.y + R[8] * wv.z;
      const float l0 = wb0 / i0r, l1 = wb1 / i1r, l2 = wb2 / i2r;
      const Vec3 Lw = v3(R[0] * l0 + R[1] * l1 + R[2] * l2, R[3] * l0 + R[4] * l1 + R[5] * l2, R[6] * l0 + R[7] * l1 + R[8] * l2);
      tau = tau - cross(wv, Lw);
    }
    const Vec3 dw = sym_mul(I6, tau);
    st[7 * S + b] = vx; st[8 * S + b] = vy; st[9 * S + b] = vz;
    st[10 * S + b] = wv.x + P.h * dw.x; st[11 * S + b] = wv.y + P.h * dw.y; st[12 * S + b] = wv.z + P.h * dw.z;
  }
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

// fp64 re-evaluation of one Eq. 10 test, every operation rounded separately (no FMA), in the order
// R from q (Eq. 1), e'_k = |R_k0| e_0 + |R_k1| e_1 + |R_k2| e_2, slack_k = (e'_i,k + e'_j,k + eps) - |x_i,k - x_j,k|.
// Used only when the fp32 slack is within 1e-5 m of zero, so that the pair list equals the fp64 definition.
#define DM(a, b) __dmul_rn((a), (b))
#define DA(a, b) __dadd_rn((a), (b))
#define DS(a, b) __dsub_rn((a), (b))
__device__ __noinline__ void ext_f64(const CSm& s, int b, double* e3) {
  const float4 q4 = cb4(s, b, 4);
  const double w = q4.x, x = q4.y, y = q4.z, z = q4.w;
  const double hx = cb4(s, b, 1).w, hy = cb4(s, b, 2).w, hz = cb4(s, b, 3).w;
  double R[9];
  R[0] = DS(1.0, DM(2.0, DA(DM(y, y), DM(z, z)))); R[1] = DM(2.0, DS(DM(x, y), DM(z, w))); R[2] = DM(2.0, DA(DM(x, z), DM(y, w)));
  R[3] = DM(2.0, DA(DM(x, y), DM(z, w))); R[4] = DS(1.0, DM(2.0, DA(DM(x, x), DM(z, z)))); R[5] = DM(2.0, DS(DM(y, z), DM(x, w)));
  R[6] = DM(2.0, DS(DM(x, z), DM(y, w))); R[7] = DM(2.0, DA(DM(y, z), DM(x, w))); R[8] = DS(1.0, DM(2.0, DA(DM(x, x), DM(y, y))));
#pragma unroll
  for (int k = 0; k < 3; ++k)
    e3[k] = DA(DA(DM(fabs(R[3 * k]), hx), DM(fabs(R[3 * k + 1]), hy)), DM(fabs(R[3 * k + 2]), hz));
}

__device__ __noinline__ bool aabb_test_f64(const CSm& s, const Params& P, int i, int j) {
  const double eps = (double)P.aabb_margin;
  double ej[3]; ext_f64(s, j, ej);
  const float4 xj = cb4(s, j, 0);
  if (i < 0) return DS(eps, DS((double)xj.z, ej[2])) >= 0.0;
  double ei[3]; ext_f64(s, i, ei);
  const float4 xi = cb4(s, i, 0);
  const double ci[3] = { xi.x, xi.y, xi.z }, cj[3] = { xj.x, xj.y, xj.z };
  double smin = 1e300;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const double slack = DS(DA(DA(ei[k], ej[k]), eps), fabs(DS(ci[k], cj[k])));
    if (slack < smin) smin = slack;
  }
  return smin >= 0.0;
}
#undef DM
#undef DA
#undef DS

// S2: ground tests, then all body pairs, in ascending canonical pair index (Eq. 10; ground test
// reading A6).  Body pairs: lane = row i of a block of 32 rows, its AABB in registers; the warp walks the columns j
// together (every lane reads body j: a shared-memory broadcast) and each lane collects its row's hits in 32-bit words;
// __popc / a warp scan of the row counts give every row its offset in the ascending list, which the lane then fills from
// its words (__ffs).  Ground candidates: __ballot_sync / __popc.  Returns the number of candidates kept (<= max_pairs);
// sets PAIR_OVERFLOW in *status.
__device__ inline int broadphase(const CSm& s, const Params& P, unsigned* status) {
  const int B = P.B, lane = lane_id();
  const float eps = P.aabb_margin;
  const unsigned below = (1u << lane) - 1u;
  int n = 0;
  for (int base = 0; base < B; base += 32) {               // ground: pair index = b
    const int j = base + lane;
    bool hit = false;
    if (j < B && cb4(s, j, 0).w != 0.0f) {
      const float sl = eps - (cb4(s, j, 0).z - s.ext[j].z);
      hit = sl >= 0.0f;
      if (fabsf(sl) < 1.0e-5f) hit = aabb_test_f64(s, P, -1, j);
    }
    const unsigned bal = __ballot_sync(kFull, hit);
    const int rank = n + __popc(bal & below);
    if (hit && rank < P.max_pairs) s.cand[rank] = (unsigned short)j;
    n += __popc(bal);
  }
  const int nW = (B + 31) >> 5;
  for (int ib = 0; ib < nW; ++ib) {
    const int i = 32 * ib + lane;
    const bool row = i < B - 1;
    float4 xi = make_float4(0, 0, 0, 0), ei = make_float4(0, 0, 0, 0);
    if (i < B) { xi = cb4(s, i, 0); ei = s.ext[i]; }
    const int fi = (int)ei.w;                               // 1 active | 2 dynamic
    for (int jb = ib; jb < nW; ++jb) {
      unsigned word = 0;
      const int j0 = 32 * jb, j1 = min(B, j0 + 32);
      for (int j = max(j0, 32 * ib + 1); j < j1; ++j) {     // uniform j: broadcast loads
        const float4 xj = cb4(s, j, 0), ej = s.ext[j];
        const int fj = (int)ej.w;
        const float s0 = (ei.x + ej.x + eps) - fabsf(xi.x - xj.x);
        const float s1 = (ei.y + ej.y + eps) - fabsf(xi.y - xj.y);
        const float s2 = (ei.z + ej.z + eps) - fabsf(xi.z - xj.z);
        const float smin = fminf(s0, fminf(s1, s2));
        bool hit = smin >= 0.0f;
        const bool consider = row && j > i && (fi & fj & 1) && ((fi | fj) & 2);
        if (consider && fabsf(smin) < 1.0e-5f) hit = aabb_test_f64(s, P, i, j);
        if (hit && consider) word |= 1u << (j - j0);
      }
      s.hitw[jb * 32 + lane] = word;
    }
    int cnt = 0;
    for (int jb = ib; jb < nW; ++jb) cnt += __popc(s.hitw[jb * 32 + lane]);
    int tot; int off = n + warp_excl_scan(cnt, &tot);
    for (int jb = ib; jb < nW; ++jb) {
      unsigned word = s.hitw[jb * 32 + lane];
      const int rowbase = B + i * (2 * B - i - 1) / 2 - i - 1 + 32 * jb;      // pair index of (i, j) = rowbase + (j - 32 jb)
      while (word) {
        const int bit = __ffs(word) - 1; word &= word - 1;
        if (off < P.max_pairs) s.cand[off] = (unsigned short)(rowbase + bit);
        ++off;
      }
    }
    n += tot;
  }
  if (n > P.max_pairs) { *status |= JENGA_ST_PAIR_OVERFLOW; n = P.max_pairs; }
  __syncwarp();
  return n;
}

// cab word of a colliding pair: (a+1) bits 0-10 | A dynamic bit 11 | SAT axis bits 12-15 | b bits 16-26 | B dynamic bit 27
__device__ __forceinline__ unsigned pack_ab(const CSm& s, int a, int b, int axis) {
  unsigned w = (unsigned)(a + 1) | ((unsigned)axis << 12) | ((unsigned)b << 16);
  if (a >= 0 && cb4(s, a, 0).w != 0.0f) w |= 1u << 11;
  if (cb4(s, b, 0).w != 0.0f) w |= 1u << 27;
  return w;
}
__device__ __forceinline__ int ab_a(unsigned w) { return (int)(w & 0x7ffu) - 1; }
__device__ __forceinline__ int ab_b(unsigned w) { return (int)((w >> 16) & 0x7ffu); }
__device__ __forceinline__ int ab_axis(unsigned w) { return (int)((w >> 12) & 0xfu); }

// ---------------------------------------------------------------- box-box manifold on the shared records
// The box records are read by dynamic index (axis k of body b = float4 1 + k of its record: axis.xyz, half extent), so
// the axis choices of the reference / incident faces are address arithmetic, not select chains; the clip polygon of
// a lane lives in the warp's shared-memory buffer s.poly (8 vertices x 3 floats per lane, component-major so that lane l
// always hits bank l): no thread-local memory anywhere in the narrowphase.
__device__ __forceinline__ float4 rec4(int off, int k) { return reinterpret_cast<const float4*>(smem_f + off)[k]; }
__device__ __forceinline__ Vec3 poly_get(int pb, int k) { return v3(smem_f[pb + (3 * k) * 32], smem_f[pb + (3 * k + 1) * 32], smem_f[pb + (3 * k + 2) * 32]); }
__device__ __forceinline__ void poly_put(int pb, int k, Vec3 p) { smem_f[pb + (3 * k) * 32] = p.x; smem_f[pb + (3 * k + 1) * 32] = p.y; smem_f[pb + (3 * k + 2) * 32] = p.z; }

// Normal and overlap of ONE axis of a pair that sat_boxes found overlapping with this axis chosen: the same
// expressions as in sat_boxes (same fused multiply-adds), so the values are identical bit for bit.
__device__ __forceinline__ void sat_axis(int oA, int oB, int axis, SatResult& r) {
  const float4 xa = rec4(oA, 0), xb = rec4(oB, 0);
  const Vec3 t = xyz4(xb) - xyz4(xa);
  const float4 a0 = rec4(oA, 1), a1 = rec4(oA, 2), a2 = rec4(oA, 3), b0 = rec4(oB, 1), b1 = rec4(oB, 2), b2 = rec4(oB, 3);
  const float heA[3] = { a0.w, a1.w, a2.w }, heB[3] = { b0.w, b1.w, b2.w };
  Vec3 n; float delta;
  if (axis < 3) {
    const float4 q = rec4(oA, 1 + axis);
    n = xyz4(q);
    const float rB = absdot3(heB, dot(n, xyz4(b0)), dot(n, xyz4(b1)), dot(n, xyz4(b2)));
    delta = q.w + rB - fabsf(dot(t, n));
  } else if (axis < 6) {
    const float4 q = rec4(oB, axis - 2);
    n = xyz4(q);
    const float rA = absdot3(heA, dot(xyz4(a0), n), dot(xyz4(a1), n), dot(xyz4(a2), n));
    delta = rA + q.w - fabsf(dot(t, n));
  } else {
    const int i = (axis - 6) / 3, j = (axis - 6) - 3 * i;
    Vec3 u = cross(xyz4(rec4(oA, 1 + i)), xyz4(rec4(oB, 1 + j)));
    const float inv = 1.0f / sqrtf(dot(u, u));
    u = inv * u;
    const float rA = absdot3(heA, dot(xyz4(a0), u), dot(xyz4(a1), u), dot(xyz4(a2), u));
    const float rB = absdot3(heB, dot(xyz4(b0), u), dot(xyz4(b1), u), dot(xyz4(b2), u));
    delta = rA + rB - fabsf(dot(t, u));
    n = u;
  }
  if (dot(n, t) < 0.0f) n = -n;
  r.axis = axis; r.n = n; r.delta = delta;
}

// Sutherland-Hodgman against the half-space  sgn * ((P - c) . axis) <= e, IN PLACE in the lane's polygon
// buffer.  Safe: iteration i has read vertices i + 1 and i + 2 before it writes, and it writes at most index i + 2
// (a convex polygon gains at most one vertex per plane).  At most 8 vertices are kept.
__device__ inline int clip_halfspace(int pb, int nin, Vec3 c, Vec3 axis, float sgn, float e) {
  int nout = 0;
  const Vec3 first = poly_get(pb, 0);
  Vec3 P = first, Q = nin > 1 ? poly_get(pb, 1) : first;
  float dP = e - sgn * dot(P - c, axis);
  for (int i = 0; i < nin; ++i) {
    const Vec3 R = i + 2 < nin ? poly_get(pb, i + 2) : first;      // the vertex after Q (wraps to vertex 0)
    const float dQ = e - sgn * dot(Q - c, axis);
    if (dP >= 0.0f) {
      if (nout < 8) poly_put(pb, nout++, P);
      if (dQ < 0.0f && nout < 8) { const float t = dP / (dP - dQ); poly_put(pb, nout++, madd(P, t, Q - P)); }
    } else if (dQ >= 0.0f && nout < 8) {
      const float t = dP / (dP - dQ); poly_put(pb, nout++, madd(P, t, Q - P));
    }
    P = Q; dP = dQ; Q = R;
  }
  return nout;
}

// Contact manifold for an overlapping pair (PAPER.md:273-280 read as A8): edge case = closest points of the two
// support edges; face case = incident face clipped against the side planes of the reference face, points below the
// reference face kept with their depth, <= 4 reduction (DESIGN §2 S3).
__device__ inline void manifold_boxes(int oA, int oB, const SatResult& sr, int pb, Manifold& m) {
  const int ax = sr.axis; const Vec3 n = sr.n; const float delta = sr.delta;
  m.axis = ax; m.n = n; m.np = 0;
  const Vec3 Ac = xyz4(rec4(oA, 0)), Bc = xyz4(rec4(oB, 0));

  if (ax >= 6) {                            // edge-edge
    const int i = (ax - 6) / 3, j = (ax - 6) - 3 * i;
    Vec3 pa = Ac, pb_ = Bc;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const float4 qa = rec4(oA, 1 + k), qb = rec4(oB, 1 + k);
      const float sa = dot(xyz4(qa), n) >= 0.0f ? 1.0f : -1.0f, sb = dot(xyz4(qb), n) >= 0.0f ? 1.0f : -1.0f;
      const Vec3 ma = madd(pa, sa * qa.w, xyz4(qa)), mb = madd(pb_, -sb * qb.w, xyz4(qb));
      if (k != i) pa = ma;
      if (k != j) pb_ = mb;
    }
    const float4 qi = rec4(oA, 1 + i), qj = rec4(oB, 1 + j);
    const Vec3 ai = xyz4(qi), bj = xyz4(qj), r = pa - pb_;
    const float hi = qi.w, hj = qj.w;
    const float bb = dot(ai, bj), cc = dot(ai, r), ff = dot(bj, r), den = 1.0f - bb * bb;
    float sA = (bb * ff - cc) / den, sB = (ff - bb * cc) / den;
    sA = fminf(fmaxf(sA, -hi), hi);
    sB = fminf(fmaxf(sB, -hj), hj);
    m.p[0] = 0.5f * (madd(pa, sA, ai) + madd(pb_, sB, bj));
    m.d[0] = delta; m.np = 1;
    return;
  }

  // face case: X owns the axis (reference), Y is the other (incident)
  const bool refA = ax < 3; const int r = refA ? ax : ax - 3;
  const int oX = refA ? oA : oB, oY = refA ? oB : oA;
  const Vec3 Xc = refA ? Ac : Bc, Yc = refA ? Bc : Ac;
  const Vec3 nref = refA ? n : -n;
  int mi = 0; float sg = -1.0f, best = 3.0e38f;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const float dk = dot(xyz4(rec4(oY, 1 + k)), nref);
    if (-dk < best) { best = -dk; mi = k; sg = -1.0f; }
    if (dk < best) { best = dk; mi = k; sg = 1.0f; }
  }
  const int iu = (mi == 0) ? 1 : 0, iv = (mi == 2) ? 1 : 2;
  Vec3 fc, eu, ev;
  {
    const float4 qm = rec4(oY, 1 + mi), qu = rec4(oY, 1 + iu), qv = rec4(oY, 1 + iv);
    fc = madd(Yc, sg * qm.w, xyz4(qm));
    eu = qu.w * xyz4(qu); ev = qv.w * xyz4(qv);
    poly_put(pb, 0, fc - eu - ev); poly_put(pb, 1, fc + eu - ev); poly_put(pb, 2, fc + eu + ev); poly_put(pb, 3, fc - eu + ev);
  }
  const int u = (r == 0) ? 1 : 0, v = (r == 2) ? 1 : 2;
  const float4 qxu = rec4(oX, 1 + u), qxv = rec4(oX, 1 + v);
  const Vec3 xu = xyz4(qxu), xv = xyz4(qxv);
  const float hu = qxu.w, hv = qxv.w, hr = rec4(oX, 1 + r).w;
  int np = 4;
#pragma unroll 1
  for (int pl = 0; pl < 4 && np; ++pl)        // side planes +u, -u, +v, -v of the reference face (one copy of the clip code)
    np = clip_halfspace(pb, np, Xc, pl < 2 ? xu : xv, (pl & 1) ? -1.0f : 1.0f, pl < 2 ? hu : hv);
  // keep the vertices below the reference face (in place: write index <= read index)
  int nc = 0;
  for (int k = 0; k < np; ++k) {
    const Vec3 q = poly_get(pb, k);
    const float d = hr - dot(q - Xc, nref);
    if (d >= 0.0f) { poly_put(pb, nc, q); ++nc; }
  }
  if (nc == 0) {                            // fallback: deepest incident vertex, SAT depth
    const Vec3 inc[4] = { fc - eu - ev, fc + eu - ev, fc + eu + ev, fc - eu + ev };
    Vec3 bp = inc[0]; float bd = -3.0e38f;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const float d = hr - dot(inc[k] - Xc, nref);
      if (d > bd) { bd = d; bp = inc[k]; }
    }
    m.p[0] = madd(bp, 0.5f * delta, nref); m.d[0] = delta; m.np = 1;
    return;
  }
  // contact point and depth of kept vertex k: the expressions of the keep test, so the depths are the same bits
#define CPT(k, P_, D_) { const Vec3 q_ = poly_get(pb, (k)); D_ = hr - dot(q_ - Xc, nref); P_ = madd(q_, 0.5f * D_, nref); }
  unsigned keep = (1u << nc) - 1u;
  if (nc > 4) {                             // <= 4 reduction (DESIGN §2 S3)
    int i0 = 0, i1 = -1, i2 = -1, i3 = -1; float far2 = -1.0f, amax = 0.0f, amin = 0.0f, d0 = 0.0f;
    Vec3 p0;
    CPT(0, p0, d0);
    for (int k = 1; k < nc; ++k) { Vec3 pk; float dk; CPT(k, pk, dk); if (dk > d0) { i0 = k; d0 = dk; p0 = pk; } }
    Vec3 p1 = p0;
    for (int k = 0; k < nc; ++k) if (k != i0) {
      Vec3 pk; float dk; CPT(k, pk, dk);
      const Vec3 d = pk - p0; const float dd = dot(d, d);
      if (dd > far2) { far2 = dd; i1 = k; p1 = pk; }
    }
    const Vec3 e01 = p1 - p0;
    for (int k = 0; k < nc; ++k) {
      if (k == i0 || k == i1) continue;
      Vec3 pk; float dk; CPT(k, pk, dk);
      const float area = dot(cross(e01, pk - p0), n);
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
    if (o < no) { const int k = __fns(keep, 0, o + 1); CPT(k, m.p[o], m.d[o]); }
#undef CPT
  m.np = no;
}

// ---------------------------------------------------------------- ground plane (reading A9)
// Corners below z = 0 are contacts: n = +z, depth = -z, point at mid-surface (cx, cy, z/2).
// More than four: drop the shallowest (ties: the higher corner id goes) until four remain; ascending corner id.
// The corners go through the lane's polygon buffer so that the survivors are fetched by index (no local memory).
__device__ inline void collide_ground(const Box& b, int pb, Manifold& m) {
  float cz[8];
  unsigned ok = 0; int nq = 0;
#pragma unroll
  for (int id = 0; id < 8; ++id) {
    const float sx = (id & 1) ? b.he[0] : -b.he[0], sy = (id & 2) ? b.he[1] : -b.he[1], sz = (id & 4) ? b.he[2] : -b.he[2];
    const Vec3 o = madd(madd(sx * b.ax[0], sy, b.ax[1]), sz, b.ax[2]);
    cz[id] = b.c.z + o.z;
    poly_put(pb, id, v3(b.c.x + o.x, b.c.y + o.y, cz[id]));
    if (cz[id] < 0.0f) { ok |= 1u << id; ++nq; }
  }
  while (nq > 4) {
    int worst = -1; float wd = 0.0f;
#pragma unroll
    for (int id = 0; id < 8; ++id)
      if ((ok >> id) & 1u) { const float dd = -cz[id]; if (worst < 0 || dd <= wd) { worst = id; wd = dd; } }
    ok &= ~(1u << worst); --nq;
  }
  m.np = nq; m.axis = 15; m.n = v3(0.0f, 0.0f, 1.0f);
#pragma unroll
  for (int o = 0; o < 4; ++o)
    if (o < nq) {
      const Vec3 c = poly_get(pb, __fns(ok, 0, o + 1));
      m.p[o] = v3(c.x, c.y, 0.5f * c.z);
      m.d[o] = -c.z;
    }
}

// Manifold of colliding pair (a, b) whose SAT axis is known (find_colliding stored it).
__device__ __forceinline__ void pair_manifold(const CSm& s, int a, int b, int axis, Manifold& m) {
  if (a < 0) { collide_ground(load_box(s, b), s.poly.off + lane_id(), m); return; }
  const int oA = s.cb.off + a * s.cbw, oB = s.cb.off + b * s.cbw;
  SatResult sr; sat_axis(oA, oB, axis, sr);
  manifold_boxes(oA, oB, sr, s.poly.off + lane_id(), m);
}

// S3, first half: which candidates collide (15-axis SAT / a ground corner below z = 0).  Lane k of a
// round takes candidate base+k; the colliding ones are compacted in ascending pair index into
// s.cpair / s.cab.  Returns the number kept (<= pc); sets CONTACT_OVERFLOW.
__device__ inline int find_colliding(const CSm& s, const Params& P, int n_cand, unsigned* status) {
  const int lane = lane_id();
  const unsigned below = (1u << lane) - 1u;
  int n = 0;
  for (int base = 0; base < n_cand; base += 32) {
    const int k = base + lane;
    bool hit = false; int idx = 0, i = -1, j = 0, axis = JENGA_AXIS_GROUND;
    if (k < n_cand) {
      idx = s.cand[k];
      pair_bodies(P.B, idx, i, j);
      const Box Bj = load_box(s, j);
      if (i < 0) hit = ground_hit(Bj);
      else { const Box Bi = load_box(s, i); SatResult sr; sr.axis = 0; hit = sat_boxes(P.cp, Bi, Bj, sr); axis = sr.axis; }
    }
    const unsigned bal = __ballot_sync(kFull, hit);
    const int rank = n + __popc(bal & below);
    if (hit && rank < P.pc) { s.cpair[rank] = (unsigned short)idx; s.cab[rank] = pack_ab(s, i, j, axis); }
    n += __popc(bal);
  }
  if (n > P.pc) { *status |= JENGA_ST_CONTACT_OVERFLOW; n = P.pc; }
  __syncwarp();
  return n;
}

// k_walk.  Canonical order (north_star (d), DESIGN §2 S4): visit the colliding pairs in ascending pair index;
// colour = lowest colour not used by an earlier pair sharing a dynamic body.  The walk of ONE env is sequential by
// definition, so a THREAD walks an env (one 64-bit colour mask per body in shared memory, [body][thread]: conflict-free)
// and the 32 lanes of a warp walk 32 envs at once -- only envs whose pair list changed (same_flag) take part.  Products, in
// the env's scratch: the colour of every pair (bytes, four per store) and meta[MetaNcol]; k_plan derives ranks and counts.
constexpr int kWalkThreads = 64;
__global__ void __launch_bounds__(kWalkThreads) k_walk(const Params P) {
  const int env = blockIdx.x * kWalkThreads + threadIdx.x, t = threadIdx.x;
  if (env >= P.E || P.same_flag[env] != 0) return;
  unsigned long long* used = reinterpret_cast<unsigned long long*>(smem_f);
  const Scratch L = scratch_layout(P.pc, P.G);
  float* scr = P.scratch + (size_t)env * P.scratch_words;
  int* meta = reinterpret_cast<int*>(scr + L.meta);
  const unsigned* gcab = reinterpret_cast<const unsigned*>(scr + L.cab);
  unsigned* gcol4 = reinterpret_cast<unsigned*>(scr + L.col);
  const int n = meta[MetaNcoll];
  for (int b = 0; b < P.B; ++b) used[b * kWalkThreads + t] = 0ull;
  int ncol = 0; unsigned st = 0, pack = 0;
  for (int r = 0; r < n; ++r) {
    const unsigned w = gcab[r];
    const int a = ab_a(w), b = ab_b(w);
    unsigned long long m = 0ull;
    if (w & (1u << 11)) m |= used[a * kWalkThreads + t];
    if (w & (1u << 27)) m |= used[b * kWalkThreads + t];
    int c = __ffsll((long long)~m) - 1;
    if (c < 0) { c = kMaxColours - 1; st |= JENGA_ST_COLOUR_OVERFLOW; }
    if (a >= 0) used[a * kWalkThreads + t] |= 1ull << c;
    used[b * kWalkThreads + t] |= 1ull << c;
    pack |= (unsigned)c << (8 * (r & 3));
    if ((r & 3) == 3 || r == n - 1) { gcol4[r >> 2] = pack; pack = 0; }
    if (c + 1 > ncol) ncol = c + 1;
  }
  meta[MetaNcol] = ncol;
  if (st) atomicOr(P.status + env, st);
}

// chunk word of a member: colour | first rank-in-colour << 6 | pairs << 20
__device__ __forceinline__ int chm_pack(int colour, int w0, int cnt) { return cnt ? (colour | (w0 << 6) | (cnt << 20)) : 0; }

// The visit plan of a group (warp-uniform: every lane runs the same steps, lane j looks after the fill of blocks j, j + 32,
// ...; both warps of the group compute the same plan from the members' colour counts).
// A visit takes pairs of the CURRENT colour of every member, at most 32 in all: first of the member with the most colours
// left (ties: the most pairs left), then of the other as far as lanes remain; a member moves to its next colour in the
// visit after its current one is used up.  So a member's colours are visited in ascending order, every pair once per
// sweep, and the pairs of one visit share no dynamic body (same colour, or different envs).  A visit becomes one chunk =
// consecutive lanes of one 32-position block, member 0's pairs first (bin packing, lowest block first: whole if a block
// has room, else cut over the emptiest blocks).  s.ph lists the chunks in visiting order; s.chm[m] says which pairs of
// member m a chunk holds; s.cfirst[c] = first chunk with pairs of colour c of member `me`.
__device__ inline void plan_group(const CSm& s, const CSm& s0, const CSm& s1, int nm, int me, int nblk, int phw, unsigned* status) {
  const int lane = lane_id();
  const SP<int> fill = s.fill;
  for (int j = lane; j < nblk; j += 32) fill[j] = 0;
  const int ncol0 = s0.misc[MiNcol], ncol1 = nm > 1 ? s1.misc[MiNcol] : 0;
  int work0 = 0, work1 = 0;
  for (int c = lane; c < ncol0; c += 32) work0 += s0.ccount[c];
  for (int c = lane; c < ncol1; c += 32) work1 += s1.ccount[c];
  work0 = __reduce_add_sync(kFull, work0); work1 = __reduce_add_sync(kFull, work1);
  int ci0 = 0, ci1 = 0, rem0 = 0, rem1 = 0, nph = 0, top = 0;
  __syncwarp();
  for (;;) {
    // the current colour of each member (empty colours are skipped)
    while (ci0 < ncol0 && rem0 == 0) { rem0 = s0.ccount[ci0]; if (rem0 == 0) ++ci0; }
    while (ci1 < ncol1 && rem1 == 0) { rem1 = s1.ccount[ci1]; if (rem1 == 0) ++ci1; }
    const int left0 = ncol0 - ci0, left1 = ncol1 - ci1;
    if (left0 <= 0 && left1 <= 0) break;
    int t0, t1;
    if (left1 > left0 || (left1 == left0 && work1 > work0)) { t1 = min(rem1, 32); t0 = min(rem0, 32 - t1); }
    else { t0 = min(rem0, 32); t1 = min(rem1, 32 - t0); }
    const int w00 = left0 > 0 ? s0.ccount[ci0] - rem0 : 0, w01 = left1 > 0 ? s1.ccount[ci1] - rem1 : 0;
    int n = t0 + t1, done = 0;
    while (n > 0) {
      int take = n, jb = -1;
      for (int base = 0; base < nblk && jb < 0; base += 32) {            // lowest block that holds it whole
        const int j = base + lane, room = j < nblk ? 32 - fill[j] : 0;
        const unsigned bal = __ballot_sync(kFull, room >= take);
        if (bal) jb = base + __ffs(bal) - 1;
      }
      if (jb < 0) {                                           // none: the emptiest block (lowest on ties) takes what fits
        int best = 0;
        for (int base = 0; base < nblk; base += 32) {
          const int j = base + lane, room = j < nblk ? 32 - fill[j] : 0;
          const int mx = __reduce_max_sync(kFull, room);
          if (mx > best) { best = mx; jb = base + __ffs(__ballot_sync(kFull, room == mx)) - 1; }
        }
        take = best;
      }
      if (jb < 0 || take <= 0 || nph >= phw) { *status |= JENGA_ST_CONTACT_OVERFLOW; break; }     // cannot happen: 32 nblk >= G pc
      const int f = fill[jb], hi = done + take;
      const int c0 = max(0, min(hi, t0) - done), lo1 = max(done, t0), c1 = max(0, hi - lo1);
      const int st0 = w00 + done, st1 = w01 + lo1 - t0;
      __syncwarp();
      if (lane == 0) {
        s.ph[nph] = ph_pack(jb, f, take);
        s.chm[nph] = chm_pack(ci0, st0, c0); s.chm[phw + nph] = chm_pack(ci1, st1, c1);
        if (me == 0 ? (c0 > 0 && st0 == 0) : (c1 > 0 && st1 == 0)) s.cfirst[me ? ci1 : ci0] = nph;
        fill[jb] = f + take;
      }
      __syncwarp();
      done += take; n -= take; ++nph;
      if (jb + 1 > top) top = jb + 1;
    }
    rem0 -= t0; work0 -= t0; if (t0 > 0 && rem0 == 0) ++ci0;
    rem1 -= t1; work1 -= t1; if (t1 > 0 && rem1 == 0) ++ci1;
  }
  if (lane == 0) { s.misc[MiNph] = nph; s.misc[MiNblk] = top; }
}

// k_detect's hand-over to k_plan: does the colliding-pair list of this env equal the one its scratch was coloured for?
// (the steady state of a standing tower: colouring and plan are functions of the lists alone and are kept).  The bodies
// + SAT axis of every pair go to the scratch for k_manifold / k_slot; a changed list replaces the stored one and
// invalidates the stamp until k_plan has re-planned the group.  same_flag[env] (a dense array: k_plan's warps read it
// coalesced and most of them leave at once) tells k_plan.
__device__ inline void publish_pairs(const CSm& s, const Params& P, int env, float* scr, const Scratch& L, int n_coll) {
  const int lane = lane_id();
  int* meta = reinterpret_cast<int*>(scr + L.meta);
  unsigned short* gpair = reinterpret_cast<unsigned short*>(scr + L.cpair);
  unsigned* gcab = reinterpret_cast<unsigned*>(scr + L.cab);
  // The colouring is a function of the pair indices AND of which bodies are dynamic (two pairs that share only a pinned
  // body may share a colour): props is the caller's and may change between calls with the pair list unchanged, so the
  // dynamic bits of the stored words are part of the comparison (the SAT axis bits are not: they do not colour anything).
  constexpr unsigned kDynBits = (1u << 11) | (1u << 27);
  bool same = meta[MetaMagic] == kMagic && meta[MetaNcoll] == n_coll;
  if (same)
    for (int r = lane; r < n_coll; r += 32) same = same && (s.cpair[r] == gpair[r]) && (((s.cab[r] ^ gcab[r]) & kDynBits) == 0u);
  same = __all_sync(kFull, same);
  for (int r = lane; r < n_coll; r += 32) gcab[r] = s.cab[r];
  if (!same) for (int r = lane; r < n_coll; r += 32) gpair[r] = s.cpair[r];
  if (lane == 0) {
    P.same_flag[env] = same ? 1 : 0;
    if (!same) { meta[MetaMagic] = 0; meta[MetaNcoll] = n_coll; }
  }
}

__device__ __forceinline__ void pair_barrier(int id) {
  if (id == 1) asm volatile("bar.sync 1, 64;" ::: "memory"); else asm volatile("bar.sync 2, 64;" ::: "memory");
}

// k_plan: S4 visit plan of the group this env belongs to, when the pair list of one of its members changed (k_walk has
// coloured the changed lists).
// One warp per env; with G = 2 the two warps of a group are neighbours in the CTA, exchange their colour counts through
// shared memory and meet at a named barrier (id 1 + warp / 2); both take the same path (the decision depends on the
// group's same_flag entries only).  A member whose own list did not change reloads ranks and counts from the scratch.
__device__ inline void plan_env(const Params& P, const int env) {
  const int warp = threadIdx.x >> 5, lane = lane_id(), G = P.G;
  const int me = G == 2 ? (env & 1) : 0;
  if (env - me >= P.E) return;                                   // no env of this warp's group exists (both warps leave)
  const bool present = env < P.E, sib_present = G == 2 && (env ^ 1) < P.E;
  const bool same_me = present ? P.same_flag[env] != 0 : true;
  const bool same_sib = sib_present ? P.same_flag[env ^ 1] != 0 : true;
  if (same_me && same_sib) return;
  const Scratch L = scratch_layout(P.pc, G);
  float* scr = P.scratch + (size_t)env * P.scratch_words;                    // touched only if present
  float* scr0 = P.scratch + (size_t)(env - me) * P.scratch_words;            // the group's first env always exists
  int* meta = reinterpret_cast<int*>(scr + L.meta);
  int* meta0 = reinterpret_cast<int*>(scr0 + L.meta);
  const int arena = (int)collide_smem_words(P.S, P.max_pairs, P.pc, ArenaPlan, G);
  const CSm s = carve_collide(P.S, P.max_pairs, P.pc, warp * arena, ArenaPlan, G);
  const CSm sib = carve_collide(P.S, P.max_pairs, P.pc, (warp ^ 1) * arena, ArenaPlan, G);
  unsigned st = 0;
  const int n_coll = present ? meta[MetaNcoll] : 0;
  unsigned char* gcol = reinterpret_cast<unsigned char*>(scr + L.col);
  unsigned short* gwrk = reinterpret_cast<unsigned short*>(scr + L.wrk);
  int* gcnt = reinterpret_cast<int*>(scr + L.ccnt);
  if (!same_me) {                                              // k_walk coloured the new list: ranks and counts, kept with it
    for (int c = lane; c < kMaxColours; c += 32) s.ccount[c] = 0;
    __syncwarp();
    const unsigned below = (1u << lane) - 1u;
    for (int base = 0; base < n_coll; base += 32) {            // rank of pair r inside its colour = pairs of that colour before it
      const int r = base + lane, c = r < n_coll ? gcol[r] : 255;
      const unsigned peers = __match_any_sync(kFull, c);
      if (r < n_coll) {
        const int k = s.ccount[c] + __popc(peers & below);
        s.colour[r] = (unsigned char)c; s.wrank[r] = (unsigned short)k; gwrk[r] = (unsigned short)k;
      }
      __syncwarp();
      if (r < n_coll && (peers & below) == 0) s.ccount[c] += __popc(peers);
      __syncwarp();
    }
    for (int c = lane; c < kMaxColours; c += 32) gcnt[c] = s.ccount[c];
    if (lane == 0) s.misc[MiNcol] = meta[MetaNcol];
    __syncwarp();
  } else {                                                     // the list is the one coloured last time
    if (present) {
      for (int r = lane; r < n_coll; r += 32) { s.colour[r] = gcol[r]; s.wrank[r] = gwrk[r]; }
      for (int c = lane; c < kMaxColours; c += 32) s.ccount[c] = gcnt[c];
    }
    if (lane == 0) s.misc[MiNcol] = present ? meta[MetaNcol] : 0;
    __syncwarp();
  }
  if (G == 2) pair_barrier(1 + (warp >> 1));
  const int nblk = P.nblk, phw = round_up(ph_max(nblk, G), 4);
  const int nm = sib_present || me == 1 ? 2 : 1;                 // members that exist
  plan_group(s, me ? sib : s, me ? s : sib, nm, me, nblk, phw, &st);
  if (G == 2) pair_barrier(1 + (warp >> 1));                    // the sibling has read this warp's colour counts (k_plan's loop reuses them)
  __syncwarp();
  const int nph = s.misc[MiNph];
  // Blocks are renumbered by the number of chunks they hold (= solver visits per sweep), most first: the first blocks
  // are the ones k_solve keeps in tensor memory, the rest are used in place in the L2-resident scratch.  Lane j = block j.
  if (const int top = s.misc[MiNblk]; top > 1 && top <= 32) {
    int cj = 0;
    for (int i = 0; i < nph; ++i) cj += (s.ph[i] >> 16) == lane ? 1 : 0;
    int id = 0;
    for (int k = 0; k < top; ++k) { const int ck = __shfl_sync(kFull, cj, k); id += (ck > cj || (ck == cj && k < lane)) ? 1 : 0; }
    for (int base = 0; base < nph; base += 32) {            // lane = chunk
      const int i = base + lane, d = i < nph ? s.ph[i] : 0;
      const int nid = __shfl_sync(kFull, id, (d >> 16) & 31);
      if (i < nph) s.ph[i] = (d & 0xffff) | (nid << 16);
    }
    __syncwarp();
  }
  if (present) {
    unsigned short* gpos = reinterpret_cast<unsigned short*>(scr + L.pos);
    for (int r = lane; r < n_coll; r += 32) {
      const int c = s.colour[r], w = s.wrank[r];
      int k = 0;
      for (int j = s.cfirst[c]; j < nph; ++j) {
        const int cm = s.chm[me * phw + j], cnt = cm >> 20, w0 = (cm >> 6) & 0x3fff;
        if (cnt && (cm & 63) == c && w >= w0 && w < w0 + cnt) {
          const int d = s.ph[j], off = me ? (s.chm[j] >> 20) : 0;
          k = 32 * (d >> 16) + (d & 0xff) + off + (w - w0);
          break;
        }
      }
      gpos[r] = (unsigned short)k;
    }
    if (lane == 0) meta[MetaMagic] = kMagic;
    flush_status(P, env, st);
  }
  if (me == 0) {                                              // group data: in the region of the group's first env
    int* gph = reinterpret_cast<int*>(scr0 + L.ph);
    for (int j = lane; j < nph; j += 32) gph[j] = s.ph[j];
    if (lane == 0) { meta0[MetaNph] = nph; meta0[MetaNblk] = s.misc[MiNblk]; }
  }
}

// One CTA per wpc envs like the other collision kernels (a persistent grid of 8 or 16 CTAs per SM measured slower: 1.13 -
// 1.16 vs 1.09 ms for detection + plan at cfg5); the loop only matters for grids the host caps.  The two warps of a group
// stay side by side (wpc is even when G = 2) and make the same decisions, so the pair barriers match.
__global__ void __launch_bounds__(128) k_plan(const Params P) {
  const int wpc = blockDim.x >> 5, warp = threadIdx.x >> 5;
  for (int base = blockIdx.x * wpc; base < P.E; base += gridDim.x * wpc) {
    plan_env(P, base + warp);
    __syncwarp();
  }
}

// ---------------------------------------------------------------- pair slots (solver constants at a position)
// The 56 words of position k (block k / 32, lane k % 32; float4 f of the pair at [block][f][lane]):
//   v[9c..9c+8], c = 0..3   p.xyz, (1+e)/K_nn, 1/K_t1t1, 1/K_t2t2, K_n,t1, K_n,t2, K_t1,t2 of contact c (K_dd: Eq. 13,
//                           PAPER.md:296, for d = n, t1, t2)
//   v[36 + 3c..], c = 0..3  the impulses jn, jt1, jt2 of contact c
//   v[48..51]               ab = record of A | record of B << 16 (solver body records of the GROUP: member m's body b is
//                           record m S + b, the ground is record G S), meta = np | axis << 8 | member << 12 | A is the
//                           ground << 13 | pair index << 16, rank r of the pair in its env's list, 1/|e_k - n (n.e_k)|
//   v[52..55]               n.x n.y n.z, Baumgarte corr = beta max(0, depth_max - slop) / (imA + imB)     (Eq. 16)
struct PairC { float v[56]; };      // v[0..35] read-only constants, v[36..47] impulses, v[48..55] header
constexpr int kLam = 36, kHdr = 48;
constexpr int kMetaMember = 1 << 12, kMetaGround = 1 << 13;

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

struct BodyK { float4 x, i0, i1; };           // x.w = inverse mass (0: static / inactive / ground)
__device__ __forceinline__ void load_bodyk(const CSm& s, int b, BodyK& o) {
  if (b >= 0) { o.x = cb4(s, b, 0); o.i0 = cb4(s, b, 4); o.i1 = cb4(s, b, 5); }
  else o.x = o.i0 = o.i1 = make_float4(0, 0, 0, 0);
}
__device__ __forceinline__ Vec3 imul(const BodyK& B, Vec3 a) {      // Iw^-1 a
  return v3(fmaf(B.i0.z, a.z, fmaf(B.i0.y, a.y, B.i0.x * a.x)),
            fmaf(B.i1.x, a.z, fmaf(B.i0.w, a.y, B.i0.y * a.x)),
            fmaf(B.i1.y, a.z, fmaf(B.i1.x, a.y, B.i0.z * a.x)));
}

// S4 for one colliding pair: header and constants of position k from the pair's manifold, written to the scratch.
// Warm start (DESIGN §3 R-warm): a new contact inherits (jn,jt1,jt2) of the nearest not yet taken previous contact
// point of the same pair within match_tol; slots ascending.  The previous pair list is s.cprev (ascending).
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" :: "l"(p)); }

// Entry of pair index `pair` in the warm-start cache (ascending list s.cprev), or -1; its impulses and points are
// prefetched into L2 (k_solve of the previous step wrote them a whole batch ago: they come from HBM) so that the loads of
// setup_slot, issued after the manifold arithmetic, do not wait for DRAM.
__device__ __forceinline__ int cache_lookup(const CSm& s, const Params& P, int env, int nprev, int pair) {
  if (!P.warm_start || nprev <= 0) return -1;
  int lo = 0, hi = nprev;
  while (lo < hi) { const int mid = (lo + hi) >> 1; if ((int)s.cprev[mid] < pair) lo = mid + 1; else hi = mid; }
  if (lo >= nprev || (int)s.cprev[lo] != pair) return -1;
  prefetch_l2(P.cache_lam + ((size_t)env * P.pc + lo) * 12);
  prefetch_l2(P.cache_pt + ((size_t)env * P.pc + lo) * 12);
  prefetch_l2(P.cache_key + ((size_t)env * P.pc + lo) * 2);
  return lo;
}

__device__ inline void setup_slot(const CSm& s, const Params& P, int env, float* scr0, const Scratch& L, int lo,
                                  int k, int r, int a, int b, int pair, const Manifold& m) {
  BodyK A, Bb; load_bodyk(s, a, A); load_bodyk(s, b, Bb);
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

  {
    if (lo >= 0) {
      const int ocnt = P.cache_key[((size_t)env * P.pc + lo) * 2 + 1] & 0xff;
      const float4* ol4 = reinterpret_cast<const float4*>(P.cache_lam + ((size_t)env * P.pc + lo) * 12);
      const float4* op4 = reinterpret_cast<const float4*>(P.cache_pt + ((size_t)env * P.pc + lo) * 12);
      float ol[12], op[12];
#pragma unroll
      for (int f = 0; f < 3; ++f) {
        const float4 a4 = ol4[f], b4 = op4[f];
        ol[4 * f] = a4.x; ol[4 * f + 1] = a4.y; ol[4 * f + 2] = a4.z; ol[4 * f + 3] = a4.w;
        op[4 * f] = b4.x; op[4 * f + 1] = b4.y; op[4 * f + 2] = b4.z; op[4 * f + 3] = b4.w;
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
              const Vec3 d = pt[c] - v3(op[3 * o], op[3 * o + 1], op[3 * o + 2]); const float dd = dot(d, d);
              if (dd < bdist) { bdist = dd; bo = o; }
            }
#pragma unroll
          for (int o = 0; o < 4; ++o)
            if (o == bo) { taken |= 1u << o; lam[c][0] = ol[3 * o]; lam[c][1] = ol[3 * o + 1]; lam[c][2] = ol[3 * o + 2]; }
        }
      }
    }
  }

  // the 14 float4 of the pair (in the blocks of the env's group) are stored as soon as their words are complete (header
  // and impulses first), so that the whole record is never live in registers at once
  float4* cs = reinterpret_cast<float4*>(scr0 + L.cs) + (size_t)(k >> 5) * (kCsF4 * 32) + (k & 31);
  const int mem = P.G == 2 ? (env & 1) : 0;
  const int meta = m.np | (m.axis << 8) | (mem ? kMetaMember : 0) | (a < 0 ? kMetaGround : 0) | (pair << 16);
  const int ab = (a >= 0 ? mem * P.S + a : P.G * P.S) | ((mem * P.S + b) << 16);
  cs[(kHdr / 4) * 32] = make_float4(__int_as_float(ab), __int_as_float(meta), __int_as_float(r), il);
  cs[(kHdr / 4 + 1) * 32] = make_float4(n.x, n.y, n.z, im > 0.0f ? P.beta * fmaxf(0.0f, dmax - P.slop) / im : 0.0f);
  const float e1 = 1.0f + P.restitution;
  PairC out;
#pragma unroll
  for (int c = 0; c < 4; ++c) { out.v[kLam + 3 * c] = lam[c][0]; out.v[kLam + 3 * c + 1] = lam[c][1]; out.v[kLam + 3 * c + 2] = lam[c][2]; }
#pragma unroll
  for (int f = kLam / 4; f < kHdr / 4; ++f) cs[f * 32] = make_float4(out.v[4 * f], out.v[4 * f + 1], out.v[4 * f + 2], out.v[4 * f + 3]);
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
#pragma unroll
    for (int f = 9 * c / 4; f < 9 * (c + 1) / 4; ++f) cs[f * 32] = make_float4(out.v[4 * f], out.v[4 * f + 1], out.v[4 * f + 2], out.v[4 * f + 3]);
  }
}

// The warm-start cache's pair list (ascending) into shared memory.
__device__ inline int load_prev_keys(const CSm& s, const Params& P, int env) {
  int nprev = P.warm_start ? P.n_cache[env] : 0;
  nprev = max(0, min(nprev, P.pc));
  const int* keys = P.cache_key + (size_t)env * P.pc * 2;
  for (int r = lane_id(); r < nprev; r += 32) s.cprev[r] = (unsigned short)keys[2 * r];
  __syncwarp();
  return nprev;
}

// S4: lane l of a round takes colliding pair r = 32 round + l (ascending pair index), fetches the manifold k_manifold
// left in the scratch and writes header and constants at the pair's position.
__device__ inline void setup_pairs(const CSm& s, const Params& P, int env, float* scr, float* scr0, const Scratch& L, int n_coll, int nprev) {
  const float4* man = reinterpret_cast<const float4*>(scr + L.man);
  for (int r = lane_id(); r < n_coll; r += 32) {
    const unsigned w = s.cab[r];
    const int a = ab_a(w), b = ab_b(w), pair = s.cpair[r];
    const int lo = cache_lookup(s, P, env, nprev, pair);
    Manifold m;
    const float4 h = man[5 * r];
    m.n = v3(h.x, h.y, h.z); m.np = __float_as_int(h.w) & 0xff; m.axis = __float_as_int(h.w) >> 8;
#pragma unroll
    for (int c = 0; c < 4; ++c) { const float4 q = man[5 * r + 1 + c]; m.p[c] = v3(q.x, q.y, q.z); m.d[c] = q.w; }
    setup_slot(s, P, env, scr0, L, lo, s.pos[r], r, a, b, pair, m);
  }
  __syncwarp();
}

// ---------------------------------------------------------------- materialised outputs (stage calls / parity)
__device__ inline void write_pairs(const CSm& s, const Params& P, int env, int n_cand) {
  int* out = P.pairs + (size_t)env * P.max_pairs;
  for (int k = lane_id(); k < n_cand; k += 32) out[k] = s.cand[k];
  if (lane_id() == 0) P.n_pairs[env] = n_cand;
  __syncwarp();
}

__device__ inline int load_candidates(const CSm& s, const Params& P, int env) {
  int n_cand = P.n_pairs[env];
  n_cand = max(0, min(n_cand, P.max_pairs));
  for (int k = lane_id(); k < n_cand; k += 32) s.cand[k] = (unsigned short)P.pairs[(size_t)env * P.max_pairs + k];
  __syncwarp();
  return n_cand;
}

// S3 second half: the manifold of every colliding pair (lane l of a round takes pair r = 32 round + l, ascending pair
// index; the SAT axis is known) into the scratch for k_slot.  With contacts_out the contact list is also written in
// (pair, slot) order (stage call / parity), and the contact offset of pair r goes to the scratch for the lambda output.
__device__ inline void manifold_pairs(const CSm& s, const Params& P, int env, float* scr, const Scratch& L, int n_coll, bool contacts_out) {
  const int lane = lane_id();
  float4* man = reinterpret_cast<float4*>(scr + L.man);
  unsigned short* gcoff = reinterpret_cast<unsigned short*>(scr + L.coff);
  const int n_cand = contacts_out ? max(0, min(P.n_pairs[env], P.max_pairs)) : 0;
  int off0 = 0;
  for (int base = 0; base < n_coll; base += 32) {
    const int r = base + lane;
    Manifold m; m.np = 0; m.axis = 0; m.n = v3(0, 0, 1);
#pragma unroll
    for (int c = 0; c < 4; ++c) { m.p[c] = v3(0, 0, 0); m.d[c] = 0.0f; }
    if (r < n_coll) {
      const unsigned w = s.cab[r];
      pair_manifold(s, ab_a(w), ab_b(w), ab_axis(w), m);
      man[5 * r] = make_float4(m.n.x, m.n.y, m.n.z, __int_as_float(m.np | (m.axis << 8)));
#pragma unroll
      for (int c = 0; c < 4; ++c) man[5 * r + 1 + c] = make_float4(m.p[c].x, m.p[c].y, m.p[c].z, m.d[c]);
    }
    if (!contacts_out) continue;
    int tot; const int off = off0 + warp_excl_scan(m.np, &tot);
    if (r < n_coll) {
      const int idx = s.cpair[r];
      gcoff[r] = (unsigned short)off;
      const int* gp = P.pairs + (size_t)env * P.max_pairs;      // position of the pair in the candidate list
      int lo = 0, hi = n_cand;
      while (lo < hi) { const int mid = (lo + hi) >> 1; if (gp[mid] < idx) lo = mid + 1; else hi = mid; }
      float4* out = reinterpret_cast<float4*>(P.contacts + ((size_t)env * P.max_contacts + off) * 8);
#pragma unroll
      for (int c = 0; c < 4; ++c)
        if (c < m.np) {
          const int tag = (lo & 0xffff) | (c << 16) | (m.axis << 20);
          out[2 * c] = make_float4(m.n.x, m.n.y, m.n.z, m.d[c]);
          out[2 * c + 1] = make_float4(m.p[c].x, m.p[c].y, m.p[c].z, __int_as_float(tag));
        }
    }
    off0 += tot;
  }
  if (contacts_out && lane == 0) { P.n_contacts[env] = off0; reinterpret_cast<int*>(scr + L.meta)[MetaNcont] = off0; }
  __syncwarp();
}

// Rebuild the colliding-pair list from a contact list in global memory (ordered (pair, slot); slot 0 carries
// the pair's normal): s.cpair, s.cab, s.wrank[r] = offset of the pair's first contact.
__device__ inline int pairs_from_contacts(const CSm& s, const Params& P, int env, int n_cont, unsigned* status) {
  const int lane = lane_id();
  const unsigned below = (1u << lane) - 1u;
  const float4* in = reinterpret_cast<const float4*>(P.contacts + (size_t)env * P.max_contacts * 8);
  const int* pairs = P.pairs + (size_t)env * P.max_pairs;
  int n = 0;
  for (int base = 0; base < n_cont; base += 32) {
    const int c = base + lane;
    bool first = false; int tag = 0;
    if (c < n_cont) { tag = __float_as_int(in[2 * c + 1].w); first = ((tag >> 16) & 3) == 0; }
    const unsigned bal = __ballot_sync(kFull, first);
    const int rank = n + __popc(bal & below);
    if (first && rank < P.pc) {
      const int idx = pairs[tag & 0xffff];
      int i, j; pair_bodies(P.B, idx, i, j);
      s.cpair[rank] = (unsigned short)idx; s.cab[rank] = pack_ab(s, i, j, (tag >> 20) & 0xf); s.wrank[rank] = (unsigned short)c;
    }
    n += __popc(bal);
  }
  if (n > P.pc) { *status |= JENGA_ST_CONTACT_OVERFLOW; n = P.pc; }
  __syncwarp();
  return n;
}

// ModeGiven (jenga_pgs_solve): slots from the contact list the caller supplied instead of the narrowphase.
__device__ inline void setup_given(const CSm& s, const Params& P, int env, float* scr, float* scr0, const Scratch& L, int n_coll, int n_cont, int nprev) {
  const float4* in = reinterpret_cast<const float4*>(P.contacts + (size_t)env * P.max_contacts * 8);
  unsigned short* gcoff = reinterpret_cast<unsigned short*>(scr + L.coff);
  for (int r = lane_id(); r < n_coll; r += 32) {
    const int c0 = gcoff[r], c1 = r + 1 < n_coll ? gcoff[r + 1] : n_cont;
    const unsigned w = s.cab[r];
    Manifold m; m.np = min(4, c1 - c0);
    const float4 f0 = in[2 * c0];
    m.n = v3(f0.x, f0.y, f0.z);
    m.axis = (__float_as_int(in[2 * c0 + 1].w) >> 20) & 0xf;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      m.p[c] = v3(0, 0, 0); m.d[c] = 0.0f;
      if (c < m.np) { const float4 a4 = in[2 * (c0 + c)], b4 = in[2 * (c0 + c) + 1]; m.p[c] = v3(b4.x, b4.y, b4.z); m.d[c] = a4.w; }
    }
    setup_slot(s, P, env, scr0, L, cache_lookup(s, P, env, nprev, s.cpair[r]), s.pos[r], r, ab_a(w), ab_b(w), s.cpair[r], m);
  }
  __syncwarp();
}

// ---------------------------------------------------------------- the kernel
// mode: ModeStep (fused substep, first half), ModeBroad (jenga_broadphase), ModeNarrow (jenga_narrowphase),
// ModeGiven (first half of jenga_pgs_solve).  honour_rest: envs whose scratch says "at rest" are skipped
// (jenga_simulate_until_rest).
// The colliding-pair list of this env from the scratch (k_detect wrote it) into the arena of k_manifold / k_slot.
__device__ inline int load_colliding(const CSm& s, const float* scr, const Scratch& L, bool want_pos) {
  const int n_coll = reinterpret_cast<const int*>(scr + L.meta)[MetaNcoll];
  const unsigned* gcab = reinterpret_cast<const unsigned*>(scr + L.cab);
  const unsigned short* gpos = reinterpret_cast<const unsigned short*>(scr + L.pos);
  const unsigned short* gpair = reinterpret_cast<const unsigned short*>(scr + L.cpair);
  for (int r = lane_id(); r < n_coll; r += 32) {
    s.cab[r] = gcab[r]; s.cpair[r] = gpair[r];
    if (want_pos) s.pos[r] = gpos[r];
  }
  __syncwarp();
  return n_coll;
}

// ---------------------------------------------------------------- the kernels
// mode: ModeStep (a substep of jenga_step), ModeBroad (jenga_broadphase: k_detect only), ModeNarrow (jenga_narrowphase),
// ModeGiven (first half of jenga_pgs_solve: the caller's contact list instead of the narrowphase).  honour_rest: envs whose
// scratch says "at rest" are skipped (jenga_simulate_until_rest).
template <int mode>
__global__ void __launch_bounds__(128, 6) k_detect(const Params P, const int honour_rest) {
  const int wpc = blockDim.x >> 5, warp = threadIdx.x >> 5, lane = lane_id();
  const int env = blockIdx.x * wpc + warp;
  if (blockIdx.x == 0 && threadIdx.x == 0) *P.work_counter = 0;      // k_solve of this substep starts its group queue at 0
  if (env >= P.E) return;
  const Scratch L = scratch_layout(P.pc, P.G);
  float* scr = P.scratch + (size_t)env * P.scratch_words;
  int* meta = reinterpret_cast<int*>(scr + L.meta);
  // an env at rest (jenga_simulate_until_rest) is skipped: it takes part in its group's plan with an empty pair list
  const bool live = !(honour_rest && meta[MetaResting]);
  if (mode == ModeBroad && !live) return;
  const CSm s = carve_collide(P.S, P.max_pairs, P.pc, warp * (int)collide_smem_words(P.S, P.max_pairs, P.pc, ArenaDetect, P.G), ArenaDetect, P.G);
  unsigned st = 0;
  int n_cand = 0, n_coll = 0;
  if (live) {
    load_predict(s, P, env, mode == ModeStep);
    if (mode == ModeStep || mode == ModeBroad) {
      n_cand = broadphase(s, P, &st);
      if (mode == ModeBroad || P.materialise) write_pairs(s, P, env, n_cand);
    } else if (mode == ModeNarrow) {
      n_cand = load_candidates(s, P, env);
    }
    if (mode == ModeStep || mode == ModeNarrow) n_coll = find_colliding(s, P, n_cand, &st);
    if (mode == ModeGiven) {
      const int n_cont = max(0, min(P.n_contacts[env], P.max_contacts));
      n_coll = pairs_from_contacts(s, P, env, n_cont, &st);
      unsigned short* gcoff = reinterpret_cast<unsigned short*>(scr + L.coff);
      for (int r = lane; r < n_coll; r += 32) gcoff[r] = s.wrank[r];       // the colouring reuses s.wrank
      if (lane == 0) meta[MetaNcont] = n_cont;
      __syncwarp();
    }
  }
  if (mode != ModeBroad) {
    publish_pairs(s, P, env, scr, L, n_coll);                  // an env at rest: an empty list
    if (!live) return;
    if (P.counters && mode == ModeStep && lane == 0) {
      atomicAdd(P.counters + JENGA_CNT_CANDIDATES, (unsigned long long)n_cand);
      atomicAdd(P.counters + JENGA_CNT_COLLIDING, (unsigned long long)n_coll);
      atomicMax(P.counters + JENGA_CNT_MAX_CANDIDATES, (unsigned long long)n_cand);
      atomicMax(P.counters + JENGA_CNT_MAX_COLLIDING, (unsigned long long)n_coll);
    }
  }
  flush_status(P, env, st);
}

template <int mode>
__global__ void __launch_bounds__(128, 5) k_manifold(const Params P, const int honour_rest) {
  const int wpc = blockDim.x >> 5, warp = threadIdx.x >> 5;
  const int env = blockIdx.x * wpc + warp;
  if (env >= P.E) return;
  const Scratch L = scratch_layout(P.pc, P.G);
  float* scr = P.scratch + (size_t)env * P.scratch_words;
  if (honour_rest && reinterpret_cast<int*>(scr + L.meta)[MetaResting]) return;
  const CSm s = carve_collide(P.S, P.max_pairs, P.pc, warp * (int)collide_smem_words(P.S, P.max_pairs, P.pc, ArenaManifold, P.G), ArenaManifold, P.G);
  load_predict(s, P, env, false, false);                                 // the records again (k_detect changed v, w only)
  const int n_coll = load_colliding(s, scr, L, false);
  manifold_pairs(s, P, env, scr, L, n_coll, mode == ModeNarrow || P.materialise);
}

template <int mode>
__global__ void __launch_bounds__(128, 2) k_slot(const Params P, const int honour_rest) {
  const int wpc = blockDim.x >> 5, warp = threadIdx.x >> 5;
  const int env = blockIdx.x * wpc + warp;
  if (env >= P.E) return;
  const Scratch L = scratch_layout(P.pc, P.G);
  float* scr = P.scratch + (size_t)env * P.scratch_words;
  int* meta = reinterpret_cast<int*>(scr + L.meta);
  if (honour_rest && meta[MetaResting]) return;
  const CSm s = carve_collide(P.S, P.max_pairs, P.pc, warp * (int)collide_smem_words(P.S, P.max_pairs, P.pc, ArenaSlot, P.G), ArenaSlot, P.G);
  load_predict(s, P, env, false, false);
  const int n_coll = load_colliding(s, scr, L, true);
  const int nprev = load_prev_keys(s, P, env);
  float* scr0 = P.scratch + (size_t)(env - (P.G == 2 ? (env & 1) : 0)) * P.scratch_words;      // the group's blocks
  if (mode == ModeGiven) setup_given(s, P, env, scr, scr0, L, n_coll, meta[MetaNcont], nprev);
  else setup_pairs(s, P, env, scr, scr0, L, n_coll, nprev);
}

}  // namespace jenga
