// step.cuh -- CTA-level stages of the batched Jenga step (one CTA = one env, sm_100a).
//
// Mapping: the env's body tile lives in shared memory for the whole launch;
// thread t of the CTA owns candidate pair t in the narrowphase and, after the canonical
// greedy colouring, colliding pair number t of the colour-sorted order in the solver, whose
// per-contact constants (point, 3x3 contact-space matrix, accumulated impulses) stay in that
// thread's registers across all PGS iterations.  Colours are swept in order with a CTA
// barrier between them; inside a colour no two pairs share a dynamic body.
#pragma once
#include "../../include/jenga.h"
#include "collide.cuh"

namespace jenga {

constexpr int kStateRows = 13, kPropRows = 8, kFextRows = 6;
constexpr int kRecWords = 24;       // per colliding pair record in shared memory (see Rec* below)
constexpr int kMaxColours = 64;

// record layout (32-bit words): 0 pair index, 1 candidate position, 2 axis | np<<8, 3 bodyA (-1 ground),
// 4 bodyB, 5..7 normal, 8+4k..11+4k point k (xyz) and depth k
constexpr int RecPair = 0, RecCand = 1, RecMeta = 2, RecA = 3, RecB = 4, RecN = 5, RecPt = 8;

struct Params {
  int E, B, S;
  float h;                  // dt / n_substeps
  int n_substeps, iters;
  float g[3];
  float restitution, aabb_margin, beta, slop;
  CollideParams cp;
  float match_tol;
  int warm_start, gyroscopic, max_pairs, max_contacts, pc, materialise;
  float* state; const float* props; const float* mu; const float* f_ext;
  int* pairs; int* n_pairs; float* contacts; int* n_contacts; float* lambda;
  int* cache_key; float* cache_lam; float* cache_pt; int* n_cache;
  unsigned* status; unsigned long long* counters;
};

// Shared-memory carve-up of one CTA.  All arrays are [row][S] so that a warp reading one row
// for consecutive bodies hits consecutive banks.
struct Smem {
  float* st;       // [13][S] state tile
  float* pr;       // [8][S]  props tile
  float* R;        // [9][S]  rotation matrix, row-major element (r,c) at R[(3r+c)*S + b]
  float* Iw;       // [6][S]  world inverse inertia xx xy xz yy yz zz (0 for static / inactive)
  float* ext;      // [3][S]  world AABB half extents
  int*   cand;     // [max_pairs] candidate pair indices, ascending
  float* rec;      // [pc][kRecWords] colliding pair records in ascending pair order
  int*   colour;   // [pc] colour of record r
  int*   owner;    // [pc] owner[t] = record handled by thread t (colour-sorted order)
  unsigned long long* used;   // [S] colour masks per body
  int*   wrank;    // [pc] rank of record r inside its colour; later: contact offset of record r
  int*   ccount;   // [64] pairs per colour (zero between steps)
  int*   cstart;   // [64] first owner slot of each colour
  int*   scan;     // [40] warp totals + scalars
};

enum { ScN = 32, ScNColl = 33, ScNCol = 34, ScFlag = 35, ScNCont = 36, ScStatus = 37 };

__host__ __device__ inline size_t smem_words(int S, int max_pairs, int pc) {
  size_t w = (size_t)(kStateRows + kPropRows + 9 + 6 + 3) * S;
  w += max_pairs;                 // cand
  w += (size_t)pc * kRecWords;    // rec
  w += 3 * (size_t)pc;            // colour, owner, wrank
  w += 2 * kMaxColours;           // ccount, cstart
  w += 2 * (size_t)S;             // used (u64)
  w += 40;                        // scan
  return w;
}

__device__ inline Smem carve(float* base, int S, int max_pairs, int pc) {
  Smem s;
  float* p = base;
  s.st = p;  p += kStateRows * S;
  s.pr = p;  p += kPropRows * S;
  s.R = p;   p += 9 * S;
  s.Iw = p;  p += 6 * S;
  s.ext = p; p += 3 * S;
  s.used = reinterpret_cast<unsigned long long*>(p); p += 2 * S;   // S is a multiple of 4: 8-byte aligned
  s.cand = reinterpret_cast<int*>(p); p += max_pairs;
  s.rec = p; p += (size_t)pc * kRecWords;
  s.colour = reinterpret_cast<int*>(p); p += pc;
  s.owner = reinterpret_cast<int*>(p);  p += pc;
  s.wrank = reinterpret_cast<int*>(p);  p += pc;
  s.ccount = reinterpret_cast<int*>(p); p += kMaxColours;
  s.cstart = reinterpret_cast<int*>(p); p += kMaxColours;
  s.scan = reinterpret_cast<int*>(p);
  return s;
}

// ---------------------------------------------------------------- tile load / store
// state [13][S] and props [8][S] of one env are contiguous: 128-bit coalesced copies.
__device__ inline void load_tile(float* dst, const float* src, int words) {
  const float4* s4 = reinterpret_cast<const float4*>(src);
  float4* d4 = reinterpret_cast<float4*>(dst);
  for (int i = threadIdx.x; i < words / 4; i += blockDim.x) d4[i] = s4[i];
}
__device__ inline void store_tile(float* dst, const float* src, int words) {
  const float4* s4 = reinterpret_cast<const float4*>(src);
  float4* d4 = reinterpret_cast<float4*>(dst);
  for (int i = threadIdx.x; i < words / 4; i += blockDim.x) d4[i] = s4[i];
}

__device__ __forceinline__ bool body_dynamic(const Smem& s, int S, int b) {
  return s.pr[7 * S + b] != 0.0f && s.pr[0 * S + b] != 0.0f;
}

// ---------------------------------------------------------------- S1 (pose part): R, Iw^-1, AABB
// Eq. 1, I_world^-1 = R diag(I_body^-1) R^T, e'_k = sum_j |R_kj| e_j.
__device__ inline void pose_derived(const Smem& s, int B, int S) {
  for (int b = threadIdx.x; b < B; b += blockDim.x) {
    const float w = s.st[3 * S + b], x = s.st[4 * S + b], y = s.st[5 * S + b], z = s.st[6 * S + b];
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
    float i0 = 0.0f, i1 = 0.0f, i2 = 0.0f;
    if (body_dynamic(s, S, b)) { i0 = s.pr[1 * S + b]; i1 = s.pr[2 * S + b]; i2 = s.pr[3 * S + b]; }
    int o = 0;
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
      for (int c = r; c < 3; ++c)
        s.Iw[(o++) * S + b] = R[3 * r] * i0 * R[3 * c] + R[3 * r + 1] * i1 * R[3 * c + 1] + R[3 * r + 2] * i2 * R[3 * c + 2];
  }
}

__device__ __forceinline__ Vec3 sym_mul(const float* I6, Vec3 a) {   // xx xy xz yy yz zz
  return v3(I6[0] * a.x + I6[1] * a.y + I6[2] * a.z,
            I6[1] * a.x + I6[3] * a.y + I6[4] * a.z,
            I6[2] * a.x + I6[4] * a.y + I6[5] * a.z);
}

// S1 velocity part: v += h (g + f/m), w += h Iw^-1 (tau [- w x Iw w]) (Eq. 5, PAPER.md:179;
// reading A2: impulses are not multiplied by dt, only g and external loads carry h).
__device__ inline void predict_velocity(const Smem& s, const Params& P, int env) {
  const int S = P.S;
  for (int b = threadIdx.x; b < P.B; b += blockDim.x) {
    if (!body_dynamic(s, S, b)) continue;
    const float im = s.pr[b];
    float f[6] = { 0, 0, 0, 0, 0, 0 };
    if (P.f_ext) {
      const float* fe = P.f_ext + (size_t)env * kFextRows * S;
#pragma unroll
      for (int k = 0; k < 6; ++k) f[k] = fe[k * S + b];
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) s.st[(7 + k) * S + b] += P.h * (P.g[k] + im * f[k]);
    float I6[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) I6[k] = s.Iw[k * S + b];
    Vec3 tau = v3(f[3], f[4], f[5]);
    const Vec3 w = v3(s.st[10 * S + b], s.st[11 * S + b], s.st[12 * S + b]);
    if (P.gyroscopic) {
      // I_world w = R diag(I_body) R^T w
      float Rm[9];
#pragma unroll
      for (int k = 0; k < 9; ++k) Rm[k] = s.R[k * S + b];
      const float wb0 = Rm[0] * w.x + Rm[3] * w.y + Rm[6] * w.z, wb1 = Rm[1] * w.x + Rm[4] * w.y + Rm[7] * w.z,
                  wb2 = Rm[2] * w.x + Rm[5] * w.y + Rm[8] * w.z;
      const float l0 = wb0 / s.pr[1 * S + b], l1 = wb1 / s.pr[2 * S + b], l2 = wb2 / s.pr[3 * S + b];
      const Vec3 Lw = v3(Rm[0] * l0 + Rm[1] * l1 + Rm[2] * l2, Rm[3] * l0 + Rm[4] * l1 + Rm[5] * l2,
                         Rm[6] * l0 + Rm[7] * l1 + Rm[8] * l2);
      tau = tau - cross(w, Lw);
    }
    const Vec3 dw = sym_mul(I6, tau);
    s.st[10 * S + b] = w.x + P.h * dw.x; s.st[11 * S + b] = w.y + P.h * dw.y; s.st[12 * S + b] = w.z + P.h * dw.z;
  }
}

// ---------------------------------------------------------------- ordered CTA compaction
// Every thread passes a flag; returns the flag's rank among all set flags of the CTA in
// thread order, and the CTA total in *total.  Contains two barriers.
__device__ inline int block_rank(bool flag, int* warp_tot, int* total) {
  const unsigned bal = __ballot_sync(0xffffffffu, flag);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  if (lane == 0) warp_tot[wid] = __popc(bal);
  __syncthreads();
  int before = 0, tot = 0;
  for (int k = 0; k < nw; ++k) { int c = warp_tot[k]; if (k < wid) before += c; tot += c; }
  __syncthreads();
  *total = tot;
  return before + __popc(bal & ((1u << lane) - 1u));
}

// canonical pair index -> (i, j); i = -1 for the ground
__device__ __forceinline__ void pair_bodies(int B, int idx, int& i, int& j) {
  if (idx < B) { i = -1; j = idx; return; }
  const int r = idx - B;
  // row i starts at i(2B-i-1)/2
  const float fb = (float)(2 * B - 1);
  int a = (int)((fb - sqrtf(fb * fb - 8.0f * (float)r)) * 0.5f);
  if (a < 0) a = 0;
  while (a > 0 && a * (2 * B - a - 1) / 2 > r) --a;
  while ((a + 1) * (2 * B - a - 2) / 2 <= r) ++a;
  i = a; j = a + 1 + (r - a * (2 * B - a - 1) / 2);
}

// fp64 re-evaluation of one Eq. 10 test, every operation rounded separately (no FMA), in the
// order:  R from q (Eq. 1), e'_k = |R_k0| e_0 + |R_k1| e_1 + |R_k2| e_2,
// slack_k = (e'_i,k + e'_j,k + eps) - |x_i,k - x_j,k|.  Used only when the fp32 slack is within
// 1e-5 m of zero, so that the pair list equals the fp64 definition bit for bit.
__device__ inline void ext_f64(const Smem& s, int S, int b, double* e3) {
  const double w = s.st[3 * S + b], x = s.st[4 * S + b], y = s.st[5 * S + b], z = s.st[6 * S + b];
  const double hx = s.pr[4 * S + b], hy = s.pr[5 * S + b], hz = s.pr[6 * S + b];
  double R[9];
#define DM(a, b) __dmul_rn((a), (b))
#define DA(a, b) __dadd_rn((a), (b))
#define DS(a, b) __dsub_rn((a), (b))
  R[0] = DS(1.0, DM(2.0, DA(DM(y, y), DM(z, z)))); R[1] = DM(2.0, DS(DM(x, y), DM(z, w))); R[2] = DM(2.0, DA(DM(x, z), DM(y, w)));
  R[3] = DM(2.0, DA(DM(x, y), DM(z, w))); R[4] = DS(1.0, DM(2.0, DA(DM(x, x), DM(z, z)))); R[5] = DM(2.0, DS(DM(y, z), DM(x, w)));
  R[6] = DM(2.0, DS(DM(x, z), DM(y, w))); R[7] = DM(2.0, DA(DM(y, z), DM(x, w))); R[8] = DS(1.0, DM(2.0, DA(DM(x, x), DM(y, y))));
#pragma unroll
  for (int k = 0; k < 3; ++k)
    e3[k] = DA(DA(DM(fabs(R[3 * k]), hx), DM(fabs(R[3 * k + 1]), hy)), DM(fabs(R[3 * k + 2]), hz));
}

__device__ inline bool aabb_test_f64(const Smem& s, const Params& P, int i, int j) {
  const int S = P.S;
  const double eps = (double)P.aabb_margin;
  double ej[3]; ext_f64(s, S, j, ej);
  if (i < 0) {
    const double slack = DS(eps, DS((double)s.st[2 * S + j], ej[2]));
    return slack >= 0.0;
  }
  double ei[3]; ext_f64(s, S, i, ei);
  double smin = 1e300;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const double slack = DS(DA(DA(ei[k], ej[k]), eps), fabs(DS((double)s.st[k * S + i], (double)s.st[k * S + j])));
    if (slack < smin) smin = slack;
  }
  return smin >= 0.0;
}
#undef DM
#undef DA
#undef DS

// S2: all ground tests and all body pairs in ascending canonical pair index, compacted with
// __ballot_sync/__popc into s.cand (Eq. 10; ground test reading A6).
// Returns the number of candidates kept (<= max_pairs); sets PAIR_OVERFLOW in *status.
__device__ inline int broadphase(const Smem& s, const Params& P, unsigned* status) {
  const int B = P.B, S = P.S;
  const int n_tests = B + B * (B - 1) / 2;
  const float eps = P.aabb_margin;
  int n = 0;
  for (int base = 0; base < n_tests; base += blockDim.x) {
    const int idx = base + threadIdx.x;
    bool hit = false;
    if (idx < n_tests) {
      int i, j; pair_bodies(B, idx, i, j);
      bool consider; float smin;
      if (i < 0) {
        consider = body_dynamic(s, S, j);
        smin = eps - (s.st[2 * S + j] - s.ext[2 * S + j]);
      } else {
        const bool ai = s.pr[7 * S + i] != 0.0f, aj = s.pr[7 * S + j] != 0.0f;
        consider = ai && aj && (s.pr[i] != 0.0f || s.pr[j] != 0.0f);
        smin = 3.0e38f;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          const float sl = (s.ext[k * S + i] + s.ext[k * S + j] + eps) - fabsf(s.st[k * S + i] - s.st[k * S + j]);
          smin = fminf(smin, sl);
        }
      }
      if (consider) {
        hit = smin >= 0.0f;
        if (fabsf(smin) < 1.0e-5f) hit = aabb_test_f64(s, P, i, j);
      }
    }
    int tot;
    const int rank = n + block_rank(hit, s.scan, &tot);
    if (hit) { if (rank < P.max_pairs) s.cand[rank] = idx; }
    n += tot;
  }
  if (n > P.max_pairs) { *status |= JENGA_ST_PAIR_OVERFLOW; n = P.max_pairs; }
  __syncthreads();
  return n;
}

}  // namespace jenga
