// layout.cuh -- parameters, the global hand-off ("scratch") between the six kernels of a substep, and the shared
// memory arenas of the batched Jenga step (sm_100a).
//
// A substep (S1..S7 of include/jenga.h) is SIX kernels:
//   k_detect   S1 predict, S2 broadphase, S3 SAT (which candidates collide, on which axis).  One warp per env.
//   k_walk     S4 canonical greedy colouring of the envs whose pair list changed.  One THREAD per env.
//   k_plan     S4 visit plan of the env GROUP, for the groups with such an env.  One warp per env.
//   k_manifold S3 contact manifolds of the colliding pairs.  One warp per env.
//   k_slot     S4 contact setup (effective masses, warm-start lookup).  One warp per env.  Small footprints (8-11 KB of
//              shared memory per 54-body env, <= 128 registers): 16+ warps per SM hide the latencies of this branchy,
//              load-heavy half, and each kernel's hot code fits the instruction cache.  Output, in the caller-owned
//              scratch buffer: the 56 solver words (36 constants, 12 impulses, 8 header words) of every colliding pair at
//              its POSITION in the group's blocks, and the list of chunks.
//   k_solve    S4 warm-start application, S5 PGS sweeps, S6 integrate + Baumgarte, S7 cache, Eq. 18 latch.  ONE WARP PER
//              GROUP of G envs (G = 1 or 2); the blocks live in TENSOR MEMORY (tcgen05.ld/st, lane = position % 32,
//              block j = position / 32 at columns [56 j, 56 j + 56)) or are used in place in the scratch; body records
//              in shared memory.
// Groups and positions.  Envs are independent, and a warp that sweeps the colours of ONE env runs half empty (a 54-block
// tower has 7 colours of 1..27 pairs).  So G consecutive envs form a group that one solver warp owns, and the solver's
// unit of work, the VISIT, takes pairs of the current colour of EVERY member: up to 32 pairs that share no dynamic body
// (same colour within an env; different envs share nothing).  A member's colours stay in ascending order and each of
// its pairs is visited once per sweep after every pair of a lower colour: the Gauss-Seidel result of every env is the
// canonical one bit for bit (pairs of one colour commute).  A visit is a chunk of consecutive lanes of ONE 32-position
// block (bin-packed; a visit that fits no block whole is cut over the emptiest blocks): a chunk visit of the solver is
// four warp-wide TMEM loads, the contact arithmetic of the chunk's lanes, and one warp-wide store of the impulses
// (lanes outside the chunk write back what they loaded).
#pragma once
#include "../../include/jenga.h"
#include "collide.cuh"

namespace jenga {

constexpr int kStateRows = 13, kPropRows = 8, kFextRows = 6;
constexpr int kMaxColours = 64;
constexpr int kBd = 20;        // solver body record (floats): x y z im | vx vy vz Ixx | wx wy wz Ixy | Ixz Iyy Iyz Izz | qw qx qy qz   (ksolve.cuh load_bodies)
constexpr int kCb = 28;        // collision body record of k_slot: x y z im | a0.xyz h0 | a1.xyz h1 | a2.xyz h2 | Ixx Ixy Ixz Iyy | Iyz Izz - - | pad 4 (k_detect, k_manifold: 20 words, kcollide.cuh)
constexpr int kCsF4 = 14;      // float4 per pair: 36 read-only words + 12 impulses + 8 header words (kcollide.cuh PairC)
constexpr int kTmCols = 4 * kCsF4;          // tensor-memory columns of one block
constexpr int kBlkWords = kCsF4 * 4 * 32;   // words of one 32-position block in the scratch / shared tier
constexpr int kMaxGroup = 2;                // envs per solver warp
constexpr unsigned kFull = 0xffffffffu;
constexpr int kScratchHead = 64;             // global words in front of the per-env scratch: [0] = k_solve's work counter
constexpr int kMagic = 0x4a454e47;          // "JENG": scratch meta stamp of a valid colouring

enum { MetaMagic = 0, MetaNcoll, MetaNph, MetaNcol, MetaNblk, MetaResting, MetaSteps, MetaNcont, MetaWords = 16 };

// modes of the collision kernels
enum { ModeStep = 0, ModeBroad = 1, ModeNarrow = 2, ModeGiven = 3 };

struct Params {
  int E, B, S;
  float h;                  // dt / n_substeps
  int n_substeps, iters;
  float g[3];
  float restitution, aabb_margin, beta, slop;
  CollideParams cp;
  float match_tol;
  int warm_start, gyroscopic, max_pairs, max_contacts, pc, materialise, tmb, nblk;   // nblk: blocks of a GROUP
  int G;                    // envs per group (one k_solve warp): env = G * group + member
  int smb;                  // blocks per group that the tensor-memory tiers of k_solve keep in spare shared memory
  float* state; const float* props; const float* mu; const float* f_ext;
  int* pairs; int* n_pairs; float* contacts; int* n_contacts; float* lambda;
  int* cache_key; float* cache_lam; float* cache_pt; int* n_cache;
  unsigned* status; unsigned long long* counters;
  const float* ref_pose; int* collapsed; float* collapse_stats; int* rest_steps;
  float collapse_dx, collapse_ek, collapse_theta;           // f_d * l, eps_k, theta_th
  int* work_counter;                                        // next group of the running k_solve (reset by every k_detect)
  int* same_flag;                                           // [E] k_detect -> k_plan: 1 = the env's pair list is the one its colouring was made for
  float* scratch; long long scratch_words;                  // per env (the first kScratchHead words of the buffer are global)
};

__host__ __device__ inline int round_up(int v, int m) { return (v + m - 1) / m * m; }

// ---------------------------------------------------------------- scratch (global, per env), word offsets
// Every env has the same region; the blocks (cs), the chunk list (ph) and MetaNph / MetaNblk are GROUP data and live in
// the region of the group's first env (those of the other members stay untouched).
// 32-position blocks of a group: enough for G pc pairs (capacity beyond the pairs actually colliding is the packing's slack).
__host__ __device__ inline int n_blocks(int pc, int G) { return G * ((pc + 31) / 32); }
__host__ __device__ inline int ph_max(int nblk, int G) { return G * kMaxColours + 2 * nblk + 8; }

struct Scratch {
  int cs, ph, meta, pos, cpair, coff, cab, col, wrk, ccnt, man, total;
};
__host__ __device__ inline Scratch scratch_layout(int pc, int G) {
  const int pcA = round_up(pc, 8), nblk = n_blocks(pc, G);
  Scratch L; int p = 0;
  L.cs = p;    p += kBlkWords * nblk;
  L.ph = p;    p += round_up(ph_max(nblk, G), 4);
  L.meta = p;  p += MetaWords;
  L.pos = p;   p += pcA / 2;
  L.cpair = p; p += pcA / 2;
  L.coff = p;  p += pcA / 2;
  L.cab = p;   p += pcA;
  L.col = p;   p += pcA / 4;            // colour of pair r, rank inside its colour, pairs per colour: the colouring of
  L.wrk = p;   p += pcA / 2;            // the env's current pair list (k_plan re-plans a group without re-colouring a
  L.ccnt = p;  p += kMaxColours;        // member whose list did not change)
  L.man = p;   p += 20 * pcA;           // manifold of pair r: (n.xyz, np | axis << 8), 4 x (p.xyz, depth)
  L.total = round_up(p, 32);
  return L;
}

// chunk descriptor: lane0 | count << 8 | block << 16
__host__ __device__ inline int ph_pack(int block, int lane0, int count) { return lane0 | (count << 8) | (block << 16); }

// Every shared array is addressed as an offset into the one extern shared array, so that the compiler knows the
// address space (LDS/STS with 32-bit addresses; pointers carried in a struct degrade to generic LD/ST).
extern __shared__ __align__(16) float smem_f[];
template <typename T> struct SP {
  int off;                                                   // in 4-byte words
  __device__ __forceinline__ T* ptr() const { return reinterpret_cast<T*>(smem_f + off); }
  __device__ __forceinline__ T& operator[](int i) const { return reinterpret_cast<T*>(smem_f + off)[i]; }
  __device__ __forceinline__ T* operator+(int i) const { return reinterpret_cast<T*>(smem_f + off) + i; }
};

__device__ __forceinline__ int lane_id() { return threadIdx.x & 31; }

__device__ __forceinline__ void flush_status(const Params& P, int env, unsigned st) {
  st = __reduce_or_sync(kFull, st);
  if (st && lane_id() == 0) atomicOr(P.status + env, st);
}

__device__ __forceinline__ unsigned long long warp_sum(unsigned long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(kFull, v, o);
  return v;
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

// Eq. 1
__device__ __forceinline__ void quat_to_R(float w, float x, float y, float z, float* R) {
  R[0] = 1.0f - 2.0f * (y * y + z * z); R[1] = 2.0f * (x * y - z * w);        R[2] = 2.0f * (x * z + y * w);
  R[3] = 2.0f * (x * y + z * w);        R[4] = 1.0f - 2.0f * (x * x + z * z); R[5] = 2.0f * (y * z - x * w);
  R[6] = 2.0f * (x * z - y * w);        R[7] = 2.0f * (y * z + x * w);        R[8] = 1.0f - 2.0f * (x * x + y * y);
}

// I_world^-1 = R diag(I_body^-1) R^T: xx xy xz yy yz zz
__device__ __forceinline__ void world_inv_inertia(const float* R, float i0, float i1, float i2, float* I6) {
  int o = 0;
#pragma unroll
  for (int r = 0; r < 3; ++r)
#pragma unroll
    for (int c = r; c < 3; ++c)
      I6[o++] = R[3 * r] * i0 * R[3 * c] + R[3 * r + 1] * i1 * R[3 * c + 1] + R[3 * r + 2] * i2 * R[3 * c + 2];
}

__device__ __forceinline__ Vec3 sym_mul(const float* I6, Vec3 a) {   // xx xy xz yy yz zz
  return v3(fmaf(I6[2], a.z, fmaf(I6[1], a.y, I6[0] * a.x)),
            fmaf(I6[4], a.z, fmaf(I6[3], a.y, I6[1] * a.x)),
            fmaf(I6[5], a.z, fmaf(I6[4], a.y, I6[2] * a.x)));
}

}  // namespace jenga
