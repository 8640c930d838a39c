// ksolve.cuh -- sixth and last kernel of a substep, one GROUP of G envs per warp (layout.cuh): S4 warm-start application, S5
// coloured PGS sweeps, S6 integration + Baumgarte, S7 warm-start cache, Eq. 18 latch.  Inputs: the state tiles of the
// group's envs and the blocks + chunk list k_detect / k_slot left in the scratch of the group's first env.
//
// Two flavours (template <bool TM>):
//   TM = true   ONE persistent CTA per SM of 4 Q warps = 4 Q groups in flight (Q = 4, 3, 2 or 1) that owns all 512 columns
//               of tensor memory.  Warp w works in TMEM lanes 32 (w % 4) .. + 31 (its quadrant) and columns
//               [56 tmb (w / 4), + 56 tmb): the 56 words of the positions of the group's first `tmb` 32-position blocks
//               (tmb = 2, 3, 4, 9 for Q = 4, 3, 2, 1; tcgen05.ld/st.32x32b: lane = position % 32, block j at column
//               offset 56 j).  The next `smb` blocks are copied to the warp's share of the CTA's spare shared memory.
//               Blocks >= tmb + smb stay where k_slot wrote them, in the scratch (L2-resident while the group is in
//               flight): their visits load and store global memory, one visit ahead of use.
//   TM = false  CTA = 1 warp; every block in shared memory (configs too large for the TMEM tiers; small batches).
#pragma once
#include <type_traits>
#include "kcollide.cuh"

namespace jenga {

struct SSm {
  SP<float> bd;                 // [G S + 1][kBd] solver body records of the group (member m's body b: record m S + b);
                                // the last record is the ground: all zeros, never changes
  SP<float4> cs;                // [smb][kCsF4][32] blocks tmb .. tmb + smb - 1 (TM = false: tmb = 0, smb = nblk: every block)
  SP<int> ph;                   // [ph_max]
  int tmb, smb;
  unsigned tm;                  // TMEM address of this warp's lanes, first column of its group
  float4* gcs;                  // TM = true: the group's blocks in the scratch (blocks >= tmb are used in place)
};

// tmb = 0: the all-shared-memory flavour (smb is then the group's block capacity)
__host__ __device__ inline size_t solve_smem_words(int S, int pc, int tmb, int smb, int G) {
  const int nblk = n_blocks(pc, G);
  size_t w = (size_t)kBd * (G * S + 1);
  w += (size_t)kBlkWords * (tmb ? smb : nblk);
  w += round_up(ph_max(nblk, G), 4);
  return round_up((int)w, 4);
}

__device__ inline SSm carve_solve(int S, int pc, int tmb, int smb, int G, int base) {
  const int nblk = n_blocks(pc, G);
  SSm s; int p = base;
  s.tmb = tmb; s.smb = tmb ? smb : nblk; s.tm = 0; s.gcs = nullptr;
  s.cs.off = p;  p += kBlkWords * s.smb;
  s.bd.off = p;  p += kBd * (G * S + 1);
  s.ph.off = p;
  return s;
}

__device__ __forceinline__ float4& bd4(const SSm& s, int b, int k) { return reinterpret_cast<float4*>(smem_f + s.bd.off + b * kBd)[k]; }

// ---------------------------------------------------------------- TMEM access
__device__ __forceinline__ void tm_ld16(unsigned a, float* r) {
  unsigned* u = reinterpret_cast<unsigned*>(r);
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
               : "=r"(u[0]), "=r"(u[1]), "=r"(u[2]), "=r"(u[3]), "=r"(u[4]), "=r"(u[5]), "=r"(u[6]), "=r"(u[7]),
                 "=r"(u[8]), "=r"(u[9]), "=r"(u[10]), "=r"(u[11]), "=r"(u[12]), "=r"(u[13]), "=r"(u[14]), "=r"(u[15]) : "r"(a));
}
__device__ __forceinline__ void tm_ld8(unsigned a, float* r) {
  unsigned* u = reinterpret_cast<unsigned*>(r);
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(u[0]), "=r"(u[1]), "=r"(u[2]), "=r"(u[3]), "=r"(u[4]), "=r"(u[5]), "=r"(u[6]), "=r"(u[7]) : "r"(a));
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
__device__ __forceinline__ void tm_st8(unsigned a, const float* r) {
  const unsigned* u = reinterpret_cast<const unsigned*>(r);
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
               :: "r"(a), "r"(u[0]), "r"(u[1]), "r"(u[2]), "r"(u[3]), "r"(u[4]), "r"(u[5]), "r"(u[6]), "r"(u[7]) : "memory");
}
__device__ __forceinline__ void tm_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// whole block j (all 32 lanes take part; lane l gets position 32 j + l)
__device__ __forceinline__ void tm_load_block(const SSm& s, int j, PairC& c) {
  const unsigned a = s.tm + (unsigned)kTmCols * (unsigned)j;
  tm_ld16(a, c.v); tm_ld16(a + 16, c.v + 16); tm_ld16(a + 32, c.v + 32); tm_ld8(a + 48, c.v + 48);
}
__device__ __forceinline__ void tm_store_block(const SSm& s, int j, const PairC& c) {
  const unsigned a = s.tm + (unsigned)kTmCols * (unsigned)j;
  tm_st16(a, c.v); tm_st16(a + 16, c.v + 16); tm_st16(a + 32, c.v + 32); tm_st8(a + 48, c.v + 48);
}
__device__ __forceinline__ void tm_store_lam(const SSm& s, int j, const float* lam) {
  const unsigned a = s.tm + (unsigned)kTmCols * (unsigned)j + (unsigned)kLam;
  tm_st8(a, lam); tm_st4(a + 8, lam + 8);
}
// blocks outside tensor memory (j >= tmb), lane l: the warp's shared-memory copy (j < tmb + smb) or the scratch itself
__device__ __forceinline__ float4* sm_ptr(const SSm& s, int j, int l) { return s.cs.ptr() + (j - s.tmb) * (kCsF4 * 32) + l; }
__device__ __forceinline__ float4* gl_ptr(const SSm& s, int j, int l) { return s.gcs + j * (kCsF4 * 32) + l; }
// L2 eviction priorities: the rows of the in-place blocks are re-read in every sweep (keep: evict_last); what a group
// reads or writes once (tiles, blocks on their way into tensor / shared memory, the cache) should not push them out.
__device__ __forceinline__ unsigned long long l2_policy_keep() { unsigned long long p; asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p)); return p; }
__device__ __forceinline__ unsigned long long l2_policy_once() { unsigned long long p; asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p)); return p; }
// OFF: a compile-time byte offset (an immediate of the instruction: the rows of a pair are 512 bytes apart)
template <int OFF>
__device__ __forceinline__ float4 ldg_hint(const float4* a, unsigned long long pol) {
  float4 t;
  asm volatile("ld.global.L2::cache_hint.v4.f32 {%0, %1, %2, %3}, [%4 + %6], %5;" : "=f"(t.x), "=f"(t.y), "=f"(t.z), "=f"(t.w) : "l"(a), "l"(pol), "n"(OFF) : "memory");
  return t;
}
template <int OFF>
__device__ __forceinline__ void stg_hint(float4* a, float4 t, unsigned long long pol) {
  asm volatile("st.global.L2::cache_hint.v4.f32 [%0 + %6], {%1, %2, %3, %4}, %5;" :: "l"(a), "f"(t.x), "f"(t.y), "f"(t.z), "f"(t.w), "l"(pol), "n"(OFF) : "memory");
}
template <int F, int F1, class Fn> __device__ __forceinline__ void static_rows(Fn fn) { if constexpr (F < F1) { fn(std::integral_constant<int, F>()); static_rows<F + 1, F1>(fn); } }
#define JENGA_ROWS_LOAD(b) _Pragma("unroll") for (int f = 0; f < kCsF4; ++f) { const float4 t = (b)[f * 32]; c.v[4 * f] = t.x; c.v[4 * f + 1] = t.y; c.v[4 * f + 2] = t.z; c.v[4 * f + 3] = t.w; }
#define JENGA_ROWS_STORE(b, f0, f1) _Pragma("unroll") for (int f = (f0); f < (f1); ++f) (b)[f * 32] = make_float4(c.v[4 * f], c.v[4 * f + 1], c.v[4 * f + 2], c.v[4 * f + 3]);
template <bool TM>
__device__ __forceinline__ void sm_load_pair(const SSm& s, int j, int l, PairC& c) {
  if (!TM || j < s.tmb + s.smb) { const float4* b = sm_ptr(s, j, l); JENGA_ROWS_LOAD(b) }
  else {
    const float4* b = gl_ptr(s, j, l); const unsigned long long pol = l2_policy_keep();
    static_rows<0, kCsF4>([&](auto F) { constexpr int f = decltype(F)::value; const float4 t = ldg_hint<f * 512>(b, pol); c.v[4 * f] = t.x; c.v[4 * f + 1] = t.y; c.v[4 * f + 2] = t.z; c.v[4 * f + 3] = t.w; });
  }
}
template <bool TM>
__device__ __forceinline__ void sm_store_pair(const SSm& s, int j, int l, const PairC& c) {
  float4* b = sm_ptr(s, j, l); JENGA_ROWS_STORE(b, 0, kCsF4)
}
template <bool TM>
__device__ __forceinline__ void sm_store_lam(const SSm& s, int j, int l, const PairC& c) {
  if (!TM || j < s.tmb + s.smb) { float4* b = sm_ptr(s, j, l); JENGA_ROWS_STORE(b, kLam / 4, kHdr / 4) }
  else {
    float4* b = gl_ptr(s, j, l); const unsigned long long pol = l2_policy_keep();
    static_rows<kLam / 4, kHdr / 4>([&](auto F) { constexpr int f = decltype(F)::value; stg_hint<f * 512>(b, make_float4(c.v[4 * f], c.v[4 * f + 1], c.v[4 * f + 2], c.v[4 * f + 3]), pol); });
  }
}
// The lane whose pair lane `lane` loads from a block outside tensor memory: its own inside the chunk d, the chunk's first
// lane otherwise (a block in the scratch costs L2 bandwidth per sector touched; the duplicate addresses cost nothing and
// there is no divergent branch around the 14 loads).
__device__ __forceinline__ int load_lane(int d, int lane) { const int l0 = d & 0xff; return lane >= l0 && lane < l0 + ((d >> 8) & 0xff) ? lane : l0; }
// block of chunk d of this group: lane l <-> position 32 j + l.  All lanes call this.
template <bool TM>
__device__ __forceinline__ void block_load(const SSm& s, int d, PairC& c) {
  const int j = d >> 16;
  if (TM && j < s.tmb) { tm_load_block(s, j, c); tm_wait_ld(); }
  else sm_load_pair<TM>(s, j, load_lane(d, lane_id()), c);
}

// ---------------------------------------------------------------- warp / TMEM set-up
template <bool TM>
__device__ __forceinline__ SSm begin_solve(const Params& P) {
  __shared__ unsigned tm_base_s;
  const int warp = threadIdx.x >> 5;
  const int tmb = TM ? P.tmb : 0;
  SSm s = carve_solve(P.S, P.pc, tmb, P.smb, P.G, warp * (int)solve_smem_words(P.S, P.pc, tmb, P.smb, P.G));
  if (TM) {
    if (warp == 0) {
      asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                   :: "r"((unsigned)__cvta_generic_to_shared(&tm_base_s)), "r"(512) : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    s.tm = tm_base_s + ((unsigned)((warp & 3) * 32) << 16) + (unsigned)(kTmCols * tmb * (warp >> 2));
  }
  return s;
}

template <bool TM>
__device__ __forceinline__ void end_solve(const SSm& s) {
  if (TM) {
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if ((threadIdx.x >> 5) == 0)
      asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(s.tm), "r"(512) : "memory");   // warp 0: s.tm = base
  }
}

// ---------------------------------------------------------------- load
// Body records of member m from its state tile (lane b reads column b of every row: coalesced); Iw^-1 from q (Eq. 1,
// PAPER.md:168).  Record (5 float4, stride 20 words: an odd number of 16-byte words, so 8 consecutive bodies cover all
// bank groups): x y z im | v.xyz Ixx | w.xyz Ixy | Ixz Iyy Iyz Izz | q.  The solver reads the first four and writes back
// the second and third (the inertia words ride along unchanged).
__device__ inline void load_bodies(const SSm& s, const Params& P, int env, int m) {
  const int S = P.S, r0 = m * S;
  const float* st = P.state + (size_t)env * kStateRows * S;
  const float* pr = P.props + (size_t)env * kPropRows * S;
  for (int b = lane_id(); b < P.B; b += 32) {
    const float w = st[3 * S + b], x = st[4 * S + b], y = st[5 * S + b], z = st[6 * S + b];
    const float im = pr[b], i0 = pr[S + b], i1 = pr[2 * S + b], i2 = pr[3 * S + b];
    const bool dyn = pr[7 * S + b] != 0.0f && im != 0.0f;
    float R[9]; quat_to_R(w, x, y, z, R);
    float I6[6];
    world_inv_inertia(R, dyn ? i0 : 0.0f, dyn ? i1 : 0.0f, dyn ? i2 : 0.0f, I6);
    bd4(s, r0 + b, 0) = make_float4(st[b], st[S + b], st[2 * S + b], dyn ? im : 0.0f);
    bd4(s, r0 + b, 1) = make_float4(st[7 * S + b], st[8 * S + b], st[9 * S + b], I6[0]);       // v, Ixx
    bd4(s, r0 + b, 2) = make_float4(st[10 * S + b], st[11 * S + b], st[12 * S + b], I6[1]);    // w, Ixy
    bd4(s, r0 + b, 3) = make_float4(I6[2], I6[3], I6[4], I6[5]);                                // Ixz Iyy Iyz Izz
    bd4(s, r0 + b, 4) = make_float4(w, x, y, z);
  }
}

__device__ inline void store_bodies(const SSm& s, const Params& P, int env, int m) {
  const int S = P.S, r0 = m * S;
  float* st = P.state + (size_t)env * kStateRows * S;
  for (int b = lane_id(); b < P.B; b += 32) {
    const float4 x = bd4(s, r0 + b, 0), v = bd4(s, r0 + b, 1), w = bd4(s, r0 + b, 2), q = bd4(s, r0 + b, 4);
    if (x.w == 0.0f) continue;                                   // static / inactive bodies are never written
    st[b] = x.x; st[S + b] = x.y; st[2 * S + b] = x.z;
    st[3 * S + b] = q.x; st[4 * S + b] = q.y; st[5 * S + b] = q.z; st[6 * S + b] = q.w;
    st[7 * S + b] = v.x; st[8 * S + b] = v.y; st[9 * S + b] = v.z;
    st[10 * S + b] = w.x; st[11 * S + b] = w.y; st[12 * S + b] = w.z;
  }
}

// Chunk list and blocks of this group from the scratch of its first env.  Returns the number of chunks.
template <bool TM>
__device__ inline int load_slots(const SSm& s, const float* scr0, const Scratch& L) {
  const int lane = lane_id();
  const int* meta = reinterpret_cast<const int*>(scr0 + L.meta);
  const int nph = meta[MetaNph], nblk = meta[MetaNblk];
  const int* gph = reinterpret_cast<const int*>(scr0 + L.ph);
  for (int j = lane; j < nph; j += 32) s.ph[j] = gph[j];
  const float4* gcs = reinterpret_cast<const float4*>(scr0 + L.cs);
  const int ncopy = min(nblk, s.tmb + s.smb);                  // blocks beyond are used in place
  const unsigned long long once = l2_policy_once();
  for (int j = 0; j < ncopy; ++j) {
    PairC c;
#pragma unroll
    for (int f = 0; f < kCsF4; ++f) {
      const float4 t = ldg_hint<0>(gcs + (j * kCsF4 + f) * 32 + lane, once);
      c.v[4 * f] = t.x; c.v[4 * f + 1] = t.y; c.v[4 * f + 2] = t.z; c.v[4 * f + 3] = t.w;
    }
    if (TM && j < s.tmb) tm_store_block(s, j, c);
    else sm_store_pair<TM>(s, j, lane, c);
  }
  if (TM) tm_wait_st();
  __syncwarp();
  return nph;
}

struct Body5 { float4 x, v, w, i; };           // x.w = inverse mass (0: static / inactive / ground); v.w = Ixx, w.w = Ixy, i = Ixz Iyy Iyz Izz

__device__ __forceinline__ void load_body(const SSm& s, int b, Body5& o) {
  o.x = bd4(s, b, 0); o.v = bd4(s, b, 1); o.w = bd4(s, b, 2); o.i = bd4(s, b, 3);
}
// the ground's velocities stay +-0 (its inverse mass and inertia are 0), so writing them back is harmless
__device__ __forceinline__ void store_body_vel(const SSm& s, int b, const Body5& o) { bd4(s, b, 1) = o.v; bd4(s, b, 2) = o.w; }

// a loses the impulse, b gains it (Listing 1, PAPER.md:335-336 + the angular lines, reading A11)
__device__ __forceinline__ void apply_impulse(Body5& A, Body5& B, Vec3 rA, Vec3 rB, Vec3 Pi) {
  A.v.x = fmaf(-A.x.w, Pi.x, A.v.x); A.v.y = fmaf(-A.x.w, Pi.y, A.v.y); A.v.z = fmaf(-A.x.w, Pi.z, A.v.z);
  B.v.x = fmaf(B.x.w, Pi.x, B.v.x);  B.v.y = fmaf(B.x.w, Pi.y, B.v.y);  B.v.z = fmaf(B.x.w, Pi.z, B.v.z);
  const Vec3 cA = cross(Pi, rA), cB = cross(rB, Pi);        // -(rA x Pi), +(rB x Pi)
  A.w.x = fmaf(A.i.x, cA.z, fmaf(A.w.w, cA.y, fmaf(A.v.w, cA.x, A.w.x)));
  A.w.y = fmaf(A.i.z, cA.z, fmaf(A.i.y, cA.y, fmaf(A.w.w, cA.x, A.w.y)));
  A.w.z = fmaf(A.i.w, cA.z, fmaf(A.i.z, cA.y, fmaf(A.i.x, cA.x, A.w.z)));
  B.w.x = fmaf(B.i.x, cB.z, fmaf(B.w.w, cB.y, fmaf(B.v.w, cB.x, B.w.x)));
  B.w.y = fmaf(B.i.z, cB.z, fmaf(B.i.y, cB.y, fmaf(B.w.w, cB.x, B.w.y)));
  B.w.z = fmaf(B.i.w, cB.z, fmaf(B.i.z, cB.y, fmaf(B.i.x, cB.x, B.w.z)));
}

// The contact arithmetic of one pair (both passes).  Slots ascending; per contact the normal row (Eq. 14, clamp >= 0),
// then t1, then t2 (Eq. 15, each clipped to +-mu_s jn) -- Listing 1.  The three rows of a contact
// act on the same two bodies: the relative velocity of the contact point is read once, advanced between rows with the
// contact-space couplings K_ij (exactly the change the applied impulse causes), and the summed impulse is applied
// once (DESIGN §3 R-couple).  All four slots run unconditionally: an unused slot has zero constants and impulses, so its
// rows return 0 and it applies +-0 (bit-identical to skipping it, and no divergent branch per contact).
template <bool WARM>
__device__ __forceinline__ void solve_pair(PairC& c, Body5& A, Body5& B, const Frame& F, float mu) {
#pragma unroll
  for (int ci = 0; ci < 4; ++ci) {
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
}

// header words of a loaded pair
__device__ __forceinline__ int hdr_ab(const PairC& c) { return __float_as_int(c.v[kHdr]); }
__device__ __forceinline__ int hdr_meta(const PairC& c) { return __float_as_int(c.v[kHdr + 1]); }
__device__ __forceinline__ int hdr_rank(const PairC& c) { return __float_as_int(c.v[kHdr + 2]); }
__device__ __forceinline__ Frame hdr_frame(const PairC& c) { return make_frame(v3(c.v[kHdr + 4], c.v[kHdr + 5], c.v[kHdr + 6]), c.v[kHdr + 3]); }
__device__ __forceinline__ bool chunk_lane(int d, int lane) { const int l0 = d & 0xff; return lane >= l0 && lane < l0 + ((d >> 8) & 0xff); }

// S4: the cached impulses are applied once, chunk by chunk in visiting order (no impulse changes: nothing is stored).
template <bool TM>
__device__ inline void warm_start_pass(const SSm& s, int nph) {
  const int lane = lane_id();
  for (int j = 0; j < nph; ++j) {
    const int d = s.ph[j];
    PairC c; block_load<TM>(s, d, c);
    if (chunk_lane(d, lane)) {
      const int ab = hdr_ab(c), a = ab & 0xffff, b = ab >> 16;
      Body5 A, B; load_body(s, a, A); load_body(s, b, B);
      const Frame F = hdr_frame(c);
      solve_pair<true>(c, A, B, F, 0.0f);
      store_body_vel(s, a, A); store_body_vel(s, b, B);
    }
    __syncwarp();
  }
}

// S5: `iters` Gauss-Seidel sweeps over the chunks in visiting order, as ONE software-pipelined loop over the
// iters * nph chunk visits.  A visit: the chunk's pairs are lanes [lane0, lane0 + count) of block jb; they share no
// dynamic body.  As soon as the impulses of visit v are stored the block of visit v + 1 (constants, impulses, header) is
// requested from tensor memory / the scratch, so that the next visit starts with its (dependent) body loads at once.
// TMEM accesses are warp-wide: the lanes outside the chunk write back the impulses they loaded.  mu0 / mu1: the friction
// coefficients of the group's members (the pair's member is a header bit).
template <bool TM>
__device__ inline void pgs_sweeps(const SSm& s, int nph, int iters, float mu0, float mu1) {
  const int total = nph * iters, lane = lane_id();
  if (total <= 0) return;
  int d = s.ph[0], jn = 0;
  PairC c;
  if (TM && (d >> 16) < s.tmb) tm_load_block(s, d >> 16, c);
  else sm_load_pair<TM>(s, d >> 16, load_lane(d, lane), c);
#pragma unroll 1
  for (int v = 0; v < total; ++v) {
    const int jb = d >> 16;
    const bool active = chunk_lane(d, lane), in_tm = TM && jb < s.tmb;
    jn = jn + 1 == nph ? 0 : jn + 1;
    const int dn = s.ph[jn];
    if (in_tm) tm_wait_ld();
    if (active) {
      const int ab = hdr_ab(c), a = ab & 0xffff, b = ab >> 16;
      Body5 A, B; load_body(s, a, A); load_body(s, b, B);
      const Frame F = hdr_frame(c);
      solve_pair<false>(c, A, B, F, (hdr_meta(c) & kMetaMember) ? mu1 : mu0);
      store_body_vel(s, a, A); store_body_vel(s, b, B);
      if (!in_tm) sm_store_lam<TM>(s, jb, lane, c);
    }
    if (in_tm) { tm_store_lam(s, jb, c.v + kLam); tm_wait_st(); }
    __syncwarp();
    if (TM && (dn >> 16) < s.tmb) tm_load_block(s, dn >> 16, c);
    else sm_load_pair<TM>(s, dn >> 16, load_lane(dn, lane), c);
    d = dn;
  }
  if (TM) tm_wait_ld();
}

// S6, bodies of member m: x += h v (Eq. 6); q <- normalise(q + h/2 [0,w] (x) q) (Eq. 2, PAPER.md:151,
// world-frame reading A3).
__device__ inline void integrate_bodies(const SSm& s, const Params& P, int m, unsigned* status) {
  const int r0 = m * P.S; const float h = P.h;
  for (int b = lane_id(); b < P.B; b += 32) {
    float4 x = bd4(s, r0 + b, 0);
    if (x.w == 0.0f) continue;                                   // static or inactive
    const float4 v = bd4(s, r0 + b, 1), om = bd4(s, r0 + b, 2), q = bd4(s, r0 + b, 4);
    x.x += h * v.x; x.y += h * v.y; x.z += h * v.z;
    bd4(s, r0 + b, 0) = x;
    const float qw = q.x, qx = q.y, qy = q.z, qz = q.w;
    const float dw = -(om.x * qx + om.y * qy + om.z * qz);
    const float dx = om.x * qw + om.y * qz - om.z * qy;
    const float dy = om.y * qw + om.z * qx - om.x * qz;
    const float dz = om.z * qw + om.x * qy - om.y * qx;
    const float hh = 0.5f * h;
    const float nw = qw + hh * dw, nx = qx + hh * dx, ny = qy + hh * dy, nz = qz + hh * dz;
    const float il = 1.0f / sqrtf(nw * nw + nx * nx + ny * ny + nz * nz);
    bd4(s, r0 + b, 4) = make_float4(nw * il, nx * il, ny * il, nz * il);
    const float chk = (x.x + x.y + x.z) + (v.x + v.y + v.z) + (om.x + om.y + om.z) + il;      // any inf/NaN poisons the sum
    if (!isfinite(chk)) *status |= JENGA_ST_NONFINITE;
  }
}

// Per-body terms of Eq. 18 / PAPER.md:380: kinetic energy 1/2 m |v|^2 + 1/2 w . I w with I in the body frame
// (R^T w against the principal moments, R from the new q, Eq. 1).  ib: body-frame inverse moments.
__device__ __forceinline__ float body_kinetic_energy(float4 q, float4 x, float4 v, float4 w, float ib0, float ib1, float ib2) {
  float R[9]; quat_to_R(q.x, q.y, q.z, q.w, R);
  const float w0 = R[0] * w.x + R[3] * w.y + R[6] * w.z, w1 = R[1] * w.x + R[4] * w.y + R[7] * w.z, w2 = R[2] * w.x + R[5] * w.y + R[8] * w.z;
  return 0.5f * (v.x * v.x + v.y * v.y + v.z * v.z) / x.w + 0.5f * (w0 * w0 / ib0 + w1 * w1 / ib1 + w2 * w2 / ib2);
}

// Collapse latch (Eq. 18, reading A17) of member m after a dt advance: dx_max = max_b |x_b - x_b(0)|,
// theta_max = max_b 2 acos|q_b . q_b(0)|, E_k; collapsed |= all three above their thresholds at this step.
// Returns E_k (all lanes).
__device__ inline float collapse_latch(const SSm& s, const Params& P, int env, int m, bool latch) {
  const int S = P.S, lane = lane_id(), r0 = m * S;
  const float* ref = latch ? P.ref_pose + (size_t)env * 7 * S : nullptr;
  const float* pr = P.props + (size_t)env * kPropRows * S;
  float dxm = 0.0f, thm = 0.0f, ek = 0.0f;
  for (int b = lane; b < P.B; b += 32) {
    const float4 x = bd4(s, r0 + b, 0);
    if (x.w == 0.0f) continue;
    const float4 v = bd4(s, r0 + b, 1), w = bd4(s, r0 + b, 2), q = bd4(s, r0 + b, 4);
    ek += body_kinetic_energy(q, x, v, w, pr[S + b], pr[2 * S + b], pr[3 * S + b]);
    if (latch) {
      const float dx = x.x - ref[b], dy = x.y - ref[S + b], dz = x.z - ref[2 * S + b];
      dxm = fmaxf(dxm, sqrtf(dx * dx + dy * dy + dz * dz));
      const float c = fminf(fabsf(q.x * ref[3 * S + b] + q.y * ref[4 * S + b] + q.z * ref[5 * S + b] + q.w * ref[6 * S + b]), 1.0f);
      thm = fmaxf(thm, 2.0f * acosf(c));
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    dxm = fmaxf(dxm, __shfl_xor_sync(kFull, dxm, o)); thm = fmaxf(thm, __shfl_xor_sync(kFull, thm, o));
    ek += __shfl_xor_sync(kFull, ek, o);
  }
  if (latch && lane == 0) {
    if (dxm > P.collapse_dx && ek > P.collapse_ek && thm > P.collapse_theta) P.collapsed[env] = 1;
    if (P.collapse_stats) *reinterpret_cast<float4*>(P.collapse_stats + (size_t)env * 4) = make_float4(dxm, ek, thm, 0.0f);
  }
  return ek;
}

// One pass over the chunks in visiting order after the sweeps.  `baumgarte`: Eq. 16 (reading A14) once per
// colliding pair (after the bodies were integrated; pairs of a chunk share no dynamic body).  S7 (`cache_out`): every
// pair's impulses and contact points become the next substep's warm-start cache of its env (cache entry r = the pair's
// rank in the env's ascending pair list, from the header).  `lambda_out`: the impulses in contact order (stage output).
// Returns the lane's (contacts, ground contacts).
template <bool TM>
__device__ inline int2 finish_pairs(const SSm& s, const Params& P, int env0, const Scratch& L, int nph, bool baumgarte, bool cache_out, bool lambda_out) {
  const int lane = lane_id();
  const unsigned long long once = l2_policy_once();
  int nc = 0, ng = 0;
  for (int j = 0; j < nph; ++j) {
    const int d = s.ph[j];
    const bool active = chunk_lane(d, lane);
    PairC c; block_load<TM>(s, d, c);
    if (baumgarte) {
      const float corr = active ? c.v[kHdr + 7] : 0.0f;
      if (__any_sync(kFull, corr > 0.0f)) {
        if (corr > 0.0f) {
          const int ab = hdr_ab(c), a = ab & 0xffff, b = ab >> 16;
          const Vec3 n = v3(c.v[kHdr + 4], c.v[kHdr + 5], c.v[kHdr + 6]);
          float4 xb = bd4(s, b, 0);
          if (xb.w != 0.0f) {
            const float f = xb.w * corr;
            xb.x += f * n.x; xb.y += f * n.y; xb.z += f * n.z;
            bd4(s, b, 0) = xb;
          }
          float4 xa = bd4(s, a, 0);                              // the ground's record has inverse mass 0
          if (xa.w != 0.0f) {
            const float f = xa.w * corr;
            xa.x -= f * n.x; xa.y -= f * n.y; xa.z -= f * n.z;
            bd4(s, a, 0) = xa;
          }
        }
        __syncwarp();
      }
    }
    if (active) {
      const int meta = hdr_meta(c), np = meta & 0xff, r = hdr_rank(c);
      const int env = env0 + ((meta & kMetaMember) ? 1 : 0);
      nc += np; if (meta & kMetaGround) ng += np;
      if (cache_out) {
        int* key = P.cache_key + ((size_t)env * P.pc + r) * 2;
        key[0] = (int)((unsigned)meta >> 16); key[1] = meta & 0xfff;
        float4* ol = reinterpret_cast<float4*>(P.cache_lam + ((size_t)env * P.pc + r) * 12);
        float4* op = reinterpret_cast<float4*>(P.cache_pt + ((size_t)env * P.pc + r) * 12);
        float l[12], p[12];
#pragma unroll
        for (int ci = 0; ci < 4; ++ci)
#pragma unroll
          for (int t = 0; t < 3; ++t) { l[3 * ci + t] = ci < np ? c.v[kLam + 3 * ci + t] : 0.0f; p[3 * ci + t] = c.v[9 * ci + t]; }
#pragma unroll
        for (int f = 0; f < 3; ++f) {
          stg_hint<0>(ol + f, make_float4(l[4 * f], l[4 * f + 1], l[4 * f + 2], l[4 * f + 3]), once);
          stg_hint<0>(op + f, make_float4(p[4 * f], p[4 * f + 1], p[4 * f + 2], p[4 * f + 3]), once);
        }
      }
      if (lambda_out) {                                          // lambda in contact order (debug / stage output)
        const unsigned short* gcoff = reinterpret_cast<const unsigned short*>(P.scratch + (size_t)env * P.scratch_words + L.coff);
        float* out = P.lambda + ((size_t)env * P.max_contacts + gcoff[r]) * 3;
#pragma unroll
        for (int ci = 0; ci < 4; ++ci)
          if (ci < np) { out[3 * ci] = c.v[kLam + 3 * ci]; out[3 * ci + 1] = c.v[kLam + 3 * ci + 1]; out[3 * ci + 2] = c.v[kLam + 3 * ci + 2]; }
      }
    }
  }
  return make_int2(nc, ng);
}

// L2 prefetch of what the warp will read of group g (128-byte lines, lanes strided).
__device__ inline void prefetch_group(const Params& P, const Scratch& L, int g) {
  const int lane = lane_id();
  for (int m = 0; m < P.G; ++m) {
    const int e = g * P.G + m;
    if (e >= P.E) break;
    const char* st = reinterpret_cast<const char*>(P.state + (size_t)e * kStateRows * P.S);
    for (int o = 128 * lane; o < kStateRows * P.S * 4; o += 4096) prefetch_l2(st + o);
    const char* pr = reinterpret_cast<const char*>(P.props + (size_t)e * kPropRows * P.S);
    for (int o = 128 * lane; o < 4 * P.S * 4; o += 4096) prefetch_l2(pr + o);
  }
  const float* scr0 = P.scratch + (size_t)g * P.G * P.scratch_words;
  const int nblk = reinterpret_cast<const int*>(scr0 + L.meta)[MetaNblk];
  const char* cs = reinterpret_cast<const char*>(scr0 + L.cs);
  for (int o = 128 * lane; o < nblk * kBlkWords * 4; o += 4096) prefetch_l2(cs + o);
  prefetch_l2(scr0 + L.ph + 32 * (lane & 3));
}

// ---------------------------------------------------------------- the kernel
// flags: bit 0 end of a dt step (latch, counters, rest test), bit 1 PGS only (jenga_pgs_solve: no integration, no cache),
// bit 2 honour / update the per-env rest flag (jenga_simulate_until_rest).
enum { SolveEndOfStep = 1, SolvePgsOnly = 2, SolveRest = 4 };

// THREADS: the CTA size of the tier (the register budget follows it: 128 per thread with 16 warps, 168 with 12).
template <bool TM, int THREADS>
__global__ void __launch_bounds__(THREADS, 1) k_solve(const Params P, const int iters, const int flags, const float rest_ek) {
  SSm s = begin_solve<TM>(P);
  const int lane = lane_id(), G = P.G;
  const Scratch L = scratch_layout(P.pc, G);
  const int n_groups = (P.E + G - 1) / G;
  // persistent: every warp takes the next group of a global queue (an atomic counter that k_detect reset): groups differ
  // in cost by the number of colliding pairs, so a static split would leave warps idle at the end.  TMEM is allocated once
  // per CTA; the warps of a CTA never wait for one another between groups.
  // The queue is read one group ahead: while group g is solved, the state tiles and the used blocks of the warp's next
  // group are prefetched into L2 (they were written a whole batch ago, i.e. they come from HBM).
  // A batch smaller than the machine (fewer groups than warps in the grid) is spread evenly: only the first
  // ceil(groups / CTAs) warps of every CTA draw from the queue, so that no SM solves 16 groups while others idle.
  const bool draws = (int)(threadIdx.x >> 5) < (n_groups + (int)gridDim.x - 1) / (int)gridDim.x;
  int g_next = n_groups;
  if (draws && lane == 0) g_next = atomicAdd(P.work_counter, 1);
  g_next = __shfl_sync(kFull, g_next, 0);
  for (;;) {
    const int g = g_next;
    if (g >= n_groups) break;
    if (lane == 0) g_next = atomicAdd(P.work_counter, 1);
    g_next = __shfl_sync(kFull, g_next, 0);
    const int env0 = g * G, nm = min(G, P.E - env0);
    float* scr0 = P.scratch + (size_t)env0 * P.scratch_words;
    bool act[kMaxGroup]; bool any = false;
#pragma unroll
    for (int m = 0; m < kMaxGroup; ++m) {
      act[m] = m < nm;
      if (act[m] && (flags & SolveRest)) act[m] = reinterpret_cast<const int*>(scr0 + (size_t)m * P.scratch_words + L.meta)[MetaResting] == 0;
      any = any || act[m];
    }
    if (!any) continue;
    s.gcs = reinterpret_cast<float4*>(scr0 + L.cs);
#pragma unroll
    for (int m = 0; m < kMaxGroup; ++m) if (act[m]) load_bodies(s, P, env0 + m, m);
    if (lane < 5) bd4(s, G * P.S, lane) = make_float4(0, 0, 0, 0);      // the ground: inverse mass and inertia 0, at rest
    const int nph = load_slots<TM>(s, scr0, L);
    if (P.warm_start) warm_start_pass<TM>(s, nph);
    pgs_sweeps<TM>(s, nph, iters, P.mu[env0], act[kMaxGroup - 1] ? P.mu[env0 + kMaxGroup - 1] : 0.0f);
    // the next group into L2 now: requested when this group was taken (a whole group's duration ago, during which the
    // GPU streams twice the L2's size through it) the lines would be gone again by the time they are used
    if (g_next < n_groups) prefetch_group(P, L, g_next);
    if (flags & SolvePgsOnly) {
      finish_pairs<TM>(s, P, env0, L, nph, false, false, true);  // lambda in contact order only
#pragma unroll
      for (int m = 0; m < kMaxGroup; ++m) if (act[m]) store_bodies(s, P, env0 + m, m);
    } else {
      unsigned st[kMaxGroup];
#pragma unroll
      for (int m = 0; m < kMaxGroup; ++m) { st[m] = 0; if (act[m]) integrate_bodies(s, P, m, &st[m]); }
      __syncwarp();
      const int2 cc = finish_pairs<TM>(s, P, env0, L, nph, true, true, P.materialise != 0);
      __syncwarp();
      const bool eos = flags & SolveEndOfStep;
      int n_active = 0, n_steps = 0, n_colours = 0, max_colours = 0;
#pragma unroll
      for (int m = 0; m < kMaxGroup; ++m) {
        if (!act[m]) continue;
        const int env = env0 + m;
        int* meta = reinterpret_cast<int*>(scr0 + (size_t)m * P.scratch_words + L.meta);
        if (lane == 0) P.n_cache[env] = meta[MetaNcoll];
        store_bodies(s, P, env, m);
        if (eos && (P.collapsed || (flags & SolveRest))) {
          const float ek = collapse_latch(s, P, env, m, P.collapsed != nullptr);
          if ((flags & SolveRest) && lane == 0) {
            const int steps = meta[MetaSteps] + 1;
            meta[MetaSteps] = steps;
            if (P.rest_steps) P.rest_steps[env] = steps;
            if (ek < rest_ek) meta[MetaResting] = 1;
          }
        }
        if (P.counters) {
          ++n_steps;
          const int ncol = meta[MetaNcol];
          n_colours += ncol; max_colours = max(max_colours, ncol);
          for (int b = lane; b < P.B; b += 32) n_active += s.bd[(m * P.S + b) * kBd + 3] != 0.0f ? 1 : 0;
        }
        flush_status(P, env, st[m]);
      }
      if (P.counters) {
        const unsigned long long v = warp_sum((unsigned long long)cc.x), vg = warp_sum((unsigned long long)cc.y);
        n_active = __reduce_add_sync(kFull, n_active);
        if (lane == 0) {
          atomicAdd(P.counters + JENGA_CNT_CONTACTS, v);
          atomicAdd(P.counters + JENGA_CNT_CONTACT_ITERS, v * (unsigned long long)iters);
          atomicAdd(P.counters + JENGA_CNT_GROUND_CONTACTS, vg);
          atomicAdd(P.counters + JENGA_CNT_COLOURS, (unsigned long long)n_colours);
          atomicMax(P.counters + JENGA_CNT_MAX_COLOURS, (unsigned long long)max_colours);
          if (eos) {
            atomicAdd(P.counters + JENGA_CNT_ENV_STEPS, (unsigned long long)n_steps);
            atomicAdd(P.counters + JENGA_CNT_BODY_STEPS, (unsigned long long)n_active);
          }
        }
      }
    }
    __syncwarp();
  }
  end_solve<TM>(s);
}

}  // namespace jenga
