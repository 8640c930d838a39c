// wenv.cuh -- warp-per-env layout of the batched Jenga step (sm_100a) and stages S1, S2.
//
// Mapping: ONE WARP owns one env for the whole launch, so every synchronisation inside an env is a
// __syncwarp().  Two kernel flavours share this code (template <bool TM>):
//   TM = false  CTA = 1 warp; all solver constants in shared memory.
//   TM = true   CTA = 4 warps = 4 envs, 2 CTAs per SM; the 48 contact-constant words of the first 160
//               colour-sorted pairs of each env live in tensor memory (tcgen05.ld/st, lane = position mod 32,
//               block j = position / 32 at columns [48 j, 48 j + 48)), which frees enough shared memory for 8 envs
//               per SM.  The CTA's warps meet at a CTA barrier between the stages of a substep so that they run
//               the same code region (instruction-cache locality), nothing else is shared between them.
// Shared memory per env holds
//   * the body records (position, inverse mass, velocities, world inverse inertia: 20 floats per body,
//     read and written with 128-bit accesses by the solver),
//   * orientation, properties, rotation matrices and AABB extents as [row][S] arrays,
//   * the colliding-pair list (current and previous substep), colours, the colour-sorted order, the phase chunks,
//   * per colour-sorted position a 2-float4 header (bodies, meta, normal, Baumgarte term) and, for the positions not
//     in TMEM, the 12 float4 of contact constants, field-major (lane l of a chunk reads consecutive 16-byte words:
//     conflict-free LDS.128).  The candidate list and the colouring masks alias that region (dead before setup).
// A colour phase of the PGS is one warp instruction stream over the <= 32 pairs of a chunk; lanes are
// re-assigned to pairs every phase, so no lane idles because "its" pair has another colour.
#pragma once
#include "../../include/jenga.h"
#include "collide.cuh"

namespace jenga {

constexpr int kStateRows = 13, kPropRows = 8, kFextRows = 6;
constexpr int kMaxColours = 64;
constexpr int kBd = 20;        // floats per body record: x y z im | vx vy vz - | wx wy wz - | Ixx Ixy Ixz Iyy | Iyz Izz - -
constexpr int kHdrF4 = 2;      // float4 per pair header: (a, b, meta, 1/|t1 raw|), (n.xyz, Baumgarte corr)
constexpr int kCsF4 = 12;      // float4 of contact constants per pair: 36 read-only words + 12 impulses
// TMEM tier: the first 32 * tmb colour-sorted positions keep their contact constants in tensor memory (48 columns per
// block of 32 pairs, lane = position % 32).  tmb = 5: 256 columns per CTA of 4 warps, 2 CTAs per SM (8 envs per SM);
// tmb = 10: 512 columns, 1 CTA per SM (4 envs per SM; large configs); tmb = 0: no TMEM (1 warp per CTA).
constexpr unsigned kFull = 0xffffffffu;

struct Params {
  int E, B, S;
  float h;                  // dt / n_substeps
  int n_substeps, iters;
  float g[3];
  float restitution, aabb_margin, beta, slop;
  CollideParams cp;
  float match_tol;
  int warm_start, gyroscopic, max_pairs, max_contacts, pc, materialise, tmb;
  float* state; const float* props; const float* mu; const float* f_ext;
  int* pairs; int* n_pairs; float* contacts; int* n_contacts; float* lambda;
  int* cache_key; float* cache_lam; float* cache_pt; int* n_cache;
  unsigned* status; unsigned long long* counters;
  const float* ref_pose; int* collapsed; float* collapse_stats; int* rest_steps;
  float collapse_dx, collapse_ek, collapse_theta;           // f_d * l, eps_k, theta_th
};

// Every shared array is addressed as an offset into the one extern shared array, so that the compiler knows the
// address space (LDS/STS with 32-bit addresses; pointers carried in a struct degrade to generic LD/ST).
extern __shared__ __align__(16) float smem_f[];
template <typename T> struct SP {
  int off;                                                   // in 4-byte words
  __device__ __forceinline__ T* ptr() const { return reinterpret_cast<T*>(smem_f + off); }
  __device__ __forceinline__ T& operator[](int i) const { return reinterpret_cast<T*>(smem_f + off)[i]; }
  __device__ __forceinline__ T* operator+(int i) const { return reinterpret_cast<T*>(smem_f + off) + i; }
};

struct Smem {
  SP<float4> hdr;               // [kHdrF4][pcA] pair headers, colour-sorted position
  SP<float4> cs;                // [kCsF4][capS] contact constants of the positions kept in shared memory
  SP<float> bd;                // [S][kBd]
  SP<float> q;                  // [4][S]
  SP<float> pr;                // [8][S]  inv_m invIx invIy invIz hx hy hz active
  SP<float> R;                  // [9][S]  element (r,c) at R[(3r+c)*S + b]
  SP<float> ext;               // [3][S]
  SP<unsigned long long> used;  // [S] colour masks per body
  SP<unsigned> cab;             // [pcA] (a+1) | b << 16 of colliding pair r (ascending pair order)
  SP<unsigned short> cand;      // [mpA] candidate pair indices, ascending
  SP<unsigned short> cpair[2];  // [pcA] colliding pair indices: [cur], [prev]
  SP<unsigned short> pos;       // [pcA] colour-sorted position of pair r
  SP<unsigned short> order;     // [pcA] pair r at colour-sorted position k
  SP<unsigned short> wrank;     // [pcA] rank inside its colour / contact offset
  SP<unsigned char> colour;     // [pcA]
  SP<int> ph;                   // [kMaxColours + pcA/32 + 2] phase chunks: start | count << 16
  SP<int> ccount;               // [64]
  SP<int> cstart;               // [64]
  SP<int> misc;                 // [16]
  int pcA, capS, pos0;          // pos0 = 32 * tmb: first colour-sorted position held in cs
  unsigned tm;                  // TMEM address of this warp's lanes, column 0 (TMEM kernel)
};

enum { MiNph = 0, MiNcol = 1, MiNprev = 2 };

__host__ __device__ inline int round_up(int v, int m) { return (v + m - 1) / m * m; }

// The header + contact-constant region is dead between S7 of one substep and the setup pass of the next, which is
// when the candidate list (S2 -> first half of S3) and the colouring masks (S4) live: they alias it.
__host__ __device__ inline int cap_smem_pairs(int pc, int tmb) {
  const int pcA = round_up(pc, 8);
  return tmb ? (pcA > 32 * tmb ? pcA - 32 * tmb : 8) : pcA;
}
__host__ __device__ inline int slot_region_words(int S, int max_pairs, int pc, int tmb) {
  const int pcA = round_up(pc, 8), mpA = round_up(max_pairs, 8);
  const int a = 4 * (kHdrF4 * pcA + kCsF4 * cap_smem_pairs(pc, tmb)), b = mpA / 2 + 2 * S;
  return round_up(a > b ? a : b, 4);
}

__host__ __device__ inline size_t smem_words(int S, int max_pairs, int pc, int tmb) {
  const int pcA = round_up(pc, 8);
  size_t w = slot_region_words(S, max_pairs, pc, tmb);
  w += (size_t)(kBd + 4 + 8 + 9 + 3) * S;
  w += pcA;                        // cab
  w += 5 * (size_t)(pcA / 2);      // cpair x2, pos, order, wrank (u16)
  w += pcA / 4;                    // colour (u8)
  w += kMaxColours + pcA / 32 + 8; // ph
  w += 2 * kMaxColours + 16;       // ccount, cstart, misc
  return round_up((int)w, 4);
}

// base: word offset of this env's arena inside the CTA's dynamic shared memory
__device__ inline Smem carve(int S, int max_pairs, int pc, int tmb, int base) {
  Smem s;
  const int pcA = round_up(pc, 8), mpA = round_up(max_pairs, 8);
  s.pcA = pcA; s.capS = cap_smem_pairs(pc, tmb); s.pos0 = 32 * tmb; s.tm = 0;
  int p = base;
  s.hdr.off = p; s.cs.off = p + 4 * kHdrF4 * pcA; s.cand.off = p; s.used.off = p + mpA / 2;
  p += slot_region_words(S, max_pairs, pc, tmb);
  s.bd.off = p;  p += kBd * S;
  s.q.off = p;   p += 4 * S;
  s.pr.off = p;  p += 8 * S;
  s.R.off = p;   p += 9 * S;
  s.ext.off = p; p += 3 * S;
  s.cab.off = p; p += pcA;
  s.cpair[0].off = p; p += pcA / 2;
  s.cpair[1].off = p; p += pcA / 2;
  s.pos.off = p; p += pcA / 2;
  s.order.off = p; p += pcA / 2;
  s.wrank.off = p; p += pcA / 2;
  s.colour.off = p; p += pcA / 4;
  s.ph.off = p; p += kMaxColours + pcA / 32 + 8;
  s.ccount.off = p; p += kMaxColours;
  s.cstart.off = p; p += kMaxColours;
  s.misc.off = p;
  return s;
}

__device__ __forceinline__ int lane_id() { return threadIdx.x & 31; }

__device__ __forceinline__ float4& bd4(const Smem& s, int b, int k) { return reinterpret_cast<float4*>(smem_f + s.bd.off + b * kBd)[k]; }

__device__ __forceinline__ bool body_dynamic(const Smem& s, int S, int b) {
  return s.pr[7 * S + b] != 0.0f && s.pr[b] != 0.0f;
}

// ---------------------------------------------------------------- tile load / store
// state [13][S] and props [8][S] of one env are contiguous in HBM: 128-bit coalesced copies.
__device__ inline void load_env(const Smem& s, const Params& P, int env) {
  const int S = P.S, lane = lane_id();
  const float4* g4 = reinterpret_cast<const float4*>(P.state + (size_t)env * kStateRows * S);
  for (int i = lane; i < kStateRows * S / 4; i += 32) {
    const float4 v = g4[i];
    const int row = (4 * i) / S, b = 4 * i - row * S;
    const float e[4] = { v.x, v.y, v.z, v.w };
    if (row >= 3 && row < 7) {
      *reinterpret_cast<float4*>(s.q + (row - 3) * S + b) = v;
    } else {
      const int k = row < 3 ? row : (row < 10 ? row - 3 : row - 2);     // 0-2 -> 0-2, 7-9 -> 4-6, 10-12 -> 8-10
#pragma unroll
      for (int j = 0; j < 4; ++j) s.bd[(b + j) * kBd + k] = e[j];
    }
  }
  const float4* p4 = reinterpret_cast<const float4*>(P.props + (size_t)env * kPropRows * S);
  float4* d4 = reinterpret_cast<float4*>(s.pr.ptr());
  for (int i = lane; i < kPropRows * S / 4; i += 32) d4[i] = p4[i];
  __syncwarp();
  for (int b = lane; b < S; b += 32) {
    s.bd[b * kBd + 3] = (b < P.B && body_dynamic(s, S, b)) ? s.pr[b] : 0.0f;
    s.bd[b * kBd + 7] = 0.0f; s.bd[b * kBd + 11] = 0.0f;
  }
  __syncwarp();
}

__device__ inline void store_env(const Smem& s, const Params& P, int env) {
  const int S = P.S, lane = lane_id();
  float4* g4 = reinterpret_cast<float4*>(P.state + (size_t)env * kStateRows * S);
  for (int i = lane; i < kStateRows * S / 4; i += 32) {
    const int row = (4 * i) / S, b = 4 * i - row * S;
    float4 v;
    if (row >= 3 && row < 7) {
      v = *reinterpret_cast<const float4*>(s.q + (row - 3) * S + b);
    } else {
      const int k = row < 3 ? row : (row < 10 ? row - 3 : row - 2);
      v = make_float4(s.bd[b * kBd + k], s.bd[(b + 1) * kBd + k], s.bd[(b + 2) * kBd + k], s.bd[(b + 3) * kBd + k]);
    }
    g4[i] = v;
  }
}

__device__ __forceinline__ Vec3 sym_mul(const float* I6, Vec3 a) {   // xx xy xz yy yz zz
  return v3(fmaf(I6[2], a.z, fmaf(I6[1], a.y, I6[0] * a.x)),
            fmaf(I6[4], a.z, fmaf(I6[3], a.y, I6[1] * a.x)),
            fmaf(I6[5], a.z, fmaf(I6[4], a.y, I6[2] * a.x)));
}

// ---------------------------------------------------------------- S1: R, Iw^-1, AABB extents, velocity predict
// Eq. 1, I_world^-1 = R diag(I_body^-1) R^T, e'_k = sum_j |R_kj| e_j;
// v += h (g + f/m), w += h Iw^-1 (tau [- w x Iw w]) (Eq. 5; reading A2).
__device__ inline void pose_and_predict(const Smem& s, const Params& P, int env, bool predict) {
  const int S = P.S;
  for (int b = lane_id(); b < P.B; b += 32) {
    const float w = s.q[b], x = s.q[S + b], y = s.q[2 * S + b], z = s.q[3 * S + b];
    float R[9];
    R[0] = 1.0f - 2.0f * (y * y + z * z); R[1] = 2.0f * (x * y - z * w);        R[2] = 2.0f * (x * z + y * w);
    R[3] = 2.0f * (x * y + z * w);        R[4] = 1.0f - 2.0f * (x * x + z * z); R[5] = 2.0f * (y * z - x * w);
    R[6] = 2.0f * (x * z - y * w);        R[7] = 2.0f * (y * z + x * w);        R[8] = 1.0f - 2.0f * (x * x + y * y);
#pragma unroll
    for (int k = 0; k < 9; ++k) s.R[k * S + b] = R[k];
    const float hx = s.pr[4 * S + b], hy = s.pr[5 * S + b], hz = s.pr[6 * S + b];
#pragma unroll
    for (int k = 0; k < 3; ++k)
      s.ext[k * S + b] = fabsf(R[3 * k]) * hx + fabsf(R[3 * k + 1]) * hy + fabsf(R[3 * k + 2]) * hz;
    const bool dyn = body_dynamic(s, S, b);
    float i0 = 0.0f, i1 = 0.0f, i2 = 0.0f;
    if (dyn) { i0 = s.pr[1 * S + b]; i1 = s.pr[2 * S + b]; i2 = s.pr[3 * S + b]; }
    float I6[6]; int o = 0;
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
      for (int c = r; c < 3; ++c)
        I6[o++] = R[3 * r] * i0 * R[3 * c] + R[3 * r + 1] * i1 * R[3 * c + 1] + R[3 * r + 2] * i2 * R[3 * c + 2];
    bd4(s, b, 3) = make_float4(I6[0], I6[1], I6[2], I6[3]);
    bd4(s, b, 4) = make_float4(I6[4], I6[5], 0.0f, 0.0f);
    if (!predict || !dyn) continue;
    const float im = s.pr[b];
    float f[6] = { 0, 0, 0, 0, 0, 0 };
    if (P.f_ext) {
      const float* fe = P.f_ext + (size_t)env * kFextRows * S;
#pragma unroll
      for (int k = 0; k < 6; ++k) f[k] = fe[k * S + b];
    }
    float4 v = bd4(s, b, 1), om = bd4(s, b, 2);
    v.x += P.h * (P.g[0] + im * f[0]); v.y += P.h * (P.g[1] + im * f[1]); v.z += P.h * (P.g[2] + im * f[2]);
    Vec3 tau = v3(f[3], f[4], f[5]);
    const Vec3 wv = v3(om.x, om.y, om.z);
    if (P.gyroscopic) {                  // I_world w = R diag(I_body) R^T w
      const float wb0 = R[0] * wv.x + R[3] * wv.y + R[6] * wv.z, wb1 = R[1] * wv.x + R[4] * wv.y + R[7] * wv.z,
                  wb2 = R[2] * wv.x + R[5] * wv.y + R[8] * wv.z;
      const float l0 = wb0 / s.pr[1 * S + b], l1 = wb1 / s.pr[2 * S + b], l2 = wb2 / s.pr[3 * S + b];
      const Vec3 Lw = v3(R[0] * l0 + R[1] * l1 + R[2] * l2, R[3] * l0 + R[4] * l1 + R[5] * l2, R[6] * l0 + R[7] * l1 + R[8] * l2);
      tau = tau - cross(wv, Lw);
    }
    const Vec3 dw = sym_mul(I6, tau);
    om.x = wv.x + P.h * dw.x; om.y = wv.y + P.h * dw.y; om.z = wv.z + P.h * dw.z;
    bd4(s, b, 1) = v; bd4(s, b, 2) = om;
  }
  __syncwarp();
}

// canonical pair index -> (i, j); i = -1 for the ground
__device__ __forceinline__ void pair_bodies(int B, int idx, int& i, int& j) {
  if (idx < B) { i = -1; j = idx; return; }
  const int r = idx - B;
  const float fb = (float)(2 * B - 1);
  int a = (int)((fb - sqrtf(fb * fb - 8.0f * (float)r)) * 0.5f);
  if (a < 0) a = 0;
  while (a > 0 && a * (2 * B - a - 1) / 2 > r) --a;
  while ((a + 1) * (2 * B - a - 2) / 2 <= r) ++a;
  i = a; j = a + 1 + (r - a * (2 * B - a - 1) / 2);
}

// fp64 re-evaluation of one Eq. 10 test, every operation rounded separately (no FMA), in the order
// R from q (Eq. 1), e'_k = |R_k0| e_0 + |R_k1| e_1 + |R_k2| e_2, slack_k = (e'_i,k + e'_j,k + eps) - |x_i,k - x_j,k|.
// Used only when the fp32 slack is within 1e-5 m of zero, so that the pair list equals the fp64 definition.
#define DM(a, b) __dmul_rn((a), (b))
#define DA(a, b) __dadd_rn((a), (b))
#define DS(a, b) __dsub_rn((a), (b))
__device__ __noinline__ void ext_f64(const Smem& s, int S, int b, double* e3) {
  const double w = s.q[b], x = s.q[S + b], y = s.q[2 * S + b], z = s.q[3 * S + b];
  const double hx = s.pr[4 * S + b], hy = s.pr[5 * S + b], hz = s.pr[6 * S + b];
  double R[9];
  R[0] = DS(1.0, DM(2.0, DA(DM(y, y), DM(z, z)))); R[1] = DM(2.0, DS(DM(x, y), DM(z, w))); R[2] = DM(2.0, DA(DM(x, z), DM(y, w)));
  R[3] = DM(2.0, DA(DM(x, y), DM(z, w))); R[4] = DS(1.0, DM(2.0, DA(DM(x, x), DM(z, z)))); R[5] = DM(2.0, DS(DM(y, z), DM(x, w)));
  R[6] = DM(2.0, DS(DM(x, z), DM(y, w))); R[7] = DM(2.0, DA(DM(y, z), DM(x, w))); R[8] = DS(1.0, DM(2.0, DA(DM(x, x), DM(y, y))));
#pragma unroll
  for (int k = 0; k < 3; ++k)
    e3[k] = DA(DA(DM(fabs(R[3 * k]), hx), DM(fabs(R[3 * k + 1]), hy)), DM(fabs(R[3 * k + 2]), hz));
}

__device__ __noinline__ bool aabb_test_f64(const Smem& s, const Params& P, int i, int j) {
  const int S = P.S;
  const double eps = (double)P.aabb_margin;
  double ej[3]; ext_f64(s, S, j, ej);
  if (i < 0) return DS(eps, DS((double)s.bd[j * kBd + 2], ej[2])) >= 0.0;
  double ei[3]; ext_f64(s, S, i, ei);
  double smin = 1e300;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const double slack = DS(DA(DA(ei[k], ej[k]), eps), fabs(DS((double)s.bd[i * kBd + k], (double)s.bd[j * kBd + k])));
    if (slack < smin) smin = slack;
  }
  return smin >= 0.0;
}
#undef DM
#undef DA
#undef DS

// S2: ground tests, then all body pairs, in ascending canonical pair index; 32 tests per round, hits
// compacted with __ballot_sync/__popc into s.cand (Eq. 10; ground test reading A6).
// Returns the number of candidates kept (<= max_pairs); sets PAIR_OVERFLOW in *status.
__device__ inline int broadphase(const Smem& s, const Params& P, unsigned* status) {
  const int B = P.B, S = P.S, lane = lane_id();
  const float eps = P.aabb_margin;
  const unsigned below = (1u << lane) - 1u;
  int n = 0;
  for (int base = 0; base < B; base += 32) {               // ground: pair index = b
    const int j = base + lane;
    bool hit = false;
    if (j < B && body_dynamic(s, S, j)) {
      const float sl = eps - (s.bd[j * kBd + 2] - s.ext[2 * S + j]);
      hit = sl >= 0.0f;
      if (fabsf(sl) < 1.0e-5f) hit = aabb_test_f64(s, P, -1, j);
    }
    const unsigned bal = __ballot_sync(kFull, hit);
    const int rank = n + __popc(bal & below);
    if (hit && rank < P.max_pairs) s.cand[rank] = (unsigned short)j;
    n += __popc(bal);
  }
  const int n_bp = B * (B - 1) / 2;
  int i = 0, col = lane;                                   // lane's pair: row i, column col (j = i + 1 + col)
  for (int base = 0; base < n_bp; base += 32) {
    while (i < B - 1 && col >= B - 1 - i) { col -= B - 1 - i; ++i; }
    bool hit = false;
    const int j = i + 1 + col;
    if (i < B - 1) {
      const float4 xi = bd4(s, i, 0), xj = bd4(s, j, 0);
      const bool consider = s.pr[7 * S + i] != 0.0f && s.pr[7 * S + j] != 0.0f && (xi.w != 0.0f || xj.w != 0.0f);
      if (consider) {
        const float s0 = (s.ext[i] + s.ext[j] + eps) - fabsf(xi.x - xj.x);
        const float s1 = (s.ext[S + i] + s.ext[S + j] + eps) - fabsf(xi.y - xj.y);
        const float s2 = (s.ext[2 * S + i] + s.ext[2 * S + j] + eps) - fabsf(xi.z - xj.z);
        const float smin = fminf(s0, fminf(s1, s2));
        hit = smin >= 0.0f;
        if (fabsf(smin) < 1.0e-5f) hit = aabb_test_f64(s, P, i, j);
      }
    }
    const unsigned bal = __ballot_sync(kFull, hit);
    const int rank = n + __popc(bal & below);
    if (hit && rank < P.max_pairs) s.cand[rank] = (unsigned short)(B + i * (2 * B - i - 1) / 2 + col);
    n += __popc(bal);
    col += 32;
  }
  if (n > P.max_pairs) { *status |= JENGA_ST_PAIR_OVERFLOW; n = P.max_pairs; }
  __syncwarp();
  return n;
}

}  // namespace jenga
