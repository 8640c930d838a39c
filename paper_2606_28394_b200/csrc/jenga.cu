// jenga.cu -- kernels and C-ABI of the batched Jenga step (include/jenga.h).  sm_100a only.
//
// One WARP per env (CTA = 32 threads).  jenga_step runs S1..S7 for n_steps*n_substeps substeps in ONE launch
// with the env's bodies and solver constants resident in shared memory; the stage entry points run a single
// stage on the same device functions so that each stage can be compared with the oracle in isolation.
#include <cuda_runtime.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "wsolve.cuh"

namespace jenga {

__device__ __forceinline__ void flush_status(const Params& P, int env, unsigned st) {
  st = __reduce_or_sync(kFull, st);
  if (st && lane_id() == 0) atomicOr(P.status + env, st);
}

__device__ __forceinline__ unsigned long long warp_sum(unsigned long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(kFull, v, o);
  return v;
}

// ---------------------------------------------------------------- warp / TMEM set-up
// TM kernels: CTA = 4 warps = 4 envs; 256 TMEM columns per CTA and 2 CTAs per SM (tmb = 5) or 512 columns and 1 CTA
// per SM (tmb = 10); warp w uses TMEM lanes 32 w .. 32 w + 31.
template <bool TM>
__device__ __forceinline__ Smem begin_warp(const Params& P, int& env) {
  __shared__ unsigned tm_base_s;
  const int warp = threadIdx.x >> 5;
  env = blockIdx.x * (TM ? 4 : 1) + warp;
  const int tmb = TM ? P.tmb : 0, cols = tmb > 5 ? 512 : 256;
  Smem s = carve(P.S, P.max_pairs, P.pc, tmb, warp * (int)smem_words(P.S, P.max_pairs, P.pc, tmb));
  if (TM) {
    if (warp == 0) {
      asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                   :: "r"((unsigned)__cvta_generic_to_shared(&tm_base_s)), "r"(cols) : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    s.tm = tm_base_s + ((unsigned)(warp * 32) << 16);
  }
  return s;
}

template <bool TM>
__device__ __forceinline__ void end_warp(const Smem& s) {
  if (TM) {
    const int cols = s.pos0 > 160 ? 512 : 256;
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if ((threadIdx.x >> 5) == 0)
      asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(s.tm), "r"(cols) : "memory");   // warp 0: s.tm = base
  }
}

// ---------------------------------------------------------------- fused step
// The 4 warps of a TMEM-kernel CTA meet at a CTA barrier before and after the PGS sweeps of every substep: they then
// run the same code region at the same time, which keeps the instruction working set of an SM (32 KB L1.5 I-cache)
// to two regions instead of eight (profiles/r1d: `no_instruction` was the top stall with 8 free-running warps).
template <bool TM>
__global__ void __launch_bounds__(TM ? 128 : 32) k_step(const Params P, const int n_steps, const float rest_ek) {
  int env;
  const Smem s = begin_warp<TM>(P, env);
  const int lane = lane_id();
  bool valid = env < P.E;            // false also once the env is at rest (jenga_simulate_until_rest)
  const bool in_range = valid;
  int steps_done = 0;
  float mu = 0.0f;
  if (valid) {
    load_env(s, P, env);
    if (lane == 0) { s.misc[MiNprev] = -1; s.misc[MiNph] = 0; s.misc[MiNcol] = 0; }
    __syncwarp();
    mu = P.mu[env];
  }
  unsigned st = 0;
  unsigned long long c_cand = 0, c_coll = 0, c_cont = 0, c_gcont = 0, c_col = 0;
  int m_cand = 0, m_coll = 0, m_col = 0, cur = 0;
  const int n_sub = n_steps * P.n_substeps;
  for (int sub = 0; sub < n_sub; ++sub) {
    int n_cand = 0, n_coll = 0;
    if (valid) {
      pose_and_predict(s, P, env, true);
      n_cand = broadphase(s, P, &st);
      if (P.materialise && sub == n_sub - 1) write_pairs(s, P, env, n_cand);   // before the slots overwrite the list
    }
    if (TM) __syncthreads();
    if (valid) {
      n_coll = find_colliding(s, P, n_cand, cur, &st);
      colour_pairs<TM>(s, P, n_coll, cur, &st);
    }
    if (TM) __syncthreads();
    if (valid) setup_pairs<TM>(s, P, env, n_coll, cur);
    if (TM) __syncthreads();
    if (valid) pgs_sweeps<TM>(s, P, P.iters, mu);
    if (TM) __syncthreads();
    if (valid) {
      if (P.materialise && sub == n_sub - 1) {
        write_contacts(s, P, env, n_cand, n_coll, cur);
        write_lambda<TM>(s, P, env, n_coll);
      }
      integrate(s, P, &st);
      if (P.collapsed && (sub + 1) % P.n_substeps == 0) collapse_latch(s, P, env);
      const int2 cc = store_cache<TM>(s, P, env, n_coll);
      c_cont += cc.x; c_gcont += cc.y;
      const int ncol = s.misc[MiNcol];
      c_cand += n_cand; c_coll += n_coll; c_col += ncol;
      m_cand = max(m_cand, n_cand); m_coll = max(m_coll, n_coll); m_col = max(m_col, ncol);
      __syncwarp();
      if (lane == 0) s.misc[MiNprev] = n_coll;
      cur ^= 1;
      __syncwarp();
      if ((sub + 1) % P.n_substeps == 0) {
        ++steps_done;
        if (rest_ek > 0.0f && env_kinetic_energy(s, P) < rest_ek) valid = false;
      }
    }
    if (rest_ek > 0.0f) {                                           // the CTA retires when all of its envs rest
      const bool all_rest = TM ? (__syncthreads_and(!valid) != 0) : !valid;
      if (all_rest) break;
    }
  }
  valid = in_range;
  if (valid) {
    if (rest_ek > 0.0f && P.rest_steps && lane == 0) P.rest_steps[env] = steps_done;
    store_env(s, P, env);
    flush_status(P, env, st);
    if (P.counters) {
      const unsigned long long v = warp_sum(c_cont), vg = warp_sum(c_gcont);
      int n_active = 0;
      for (int b = lane; b < P.B; b += 32) n_active += s.bd[b * kBd + 3] != 0.0f ? 1 : 0;
      n_active = __reduce_add_sync(kFull, n_active);
      if (lane == 0) {
        atomicAdd(P.counters + JENGA_CNT_CONTACTS, v);
        atomicAdd(P.counters + JENGA_CNT_CONTACT_ITERS, v * (unsigned long long)P.iters);
        atomicAdd(P.counters + JENGA_CNT_GROUND_CONTACTS, vg);
        atomicAdd(P.counters + JENGA_CNT_ENV_STEPS, (unsigned long long)steps_done);
        atomicAdd(P.counters + JENGA_CNT_BODY_STEPS, (unsigned long long)steps_done * n_active);
        atomicAdd(P.counters + JENGA_CNT_CANDIDATES, c_cand);
        atomicAdd(P.counters + JENGA_CNT_COLLIDING, c_coll);
        atomicAdd(P.counters + JENGA_CNT_COLOURS, c_col);
        atomicMax(P.counters + JENGA_CNT_MAX_CANDIDATES, (unsigned long long)m_cand);
        atomicMax(P.counters + JENGA_CNT_MAX_COLLIDING, (unsigned long long)m_coll);
        atomicMax(P.counters + JENGA_CNT_MAX_COLOURS, (unsigned long long)m_col);
      }
    }
  }
  end_warp<TM>(s);
}

// ---------------------------------------------------------------- stage kernels
__global__ void __launch_bounds__(32) k_broadphase(const Params P) {
  int env;
  const Smem s = begin_warp<false>(P, env);
  unsigned st = 0;
  load_env(s, P, env);
  pose_and_predict(s, P, env, false);
  const int n_cand = broadphase(s, P, &st);
  write_pairs(s, P, env, n_cand);
  flush_status(P, env, st);
}

__device__ inline int load_candidates(const Smem& s, const Params& P, int env) {
  int n_cand = P.n_pairs[env];
  n_cand = max(0, min(n_cand, P.max_pairs));
  for (int k = lane_id(); k < n_cand; k += 32) s.cand[k] = (unsigned short)P.pairs[(size_t)env * P.max_pairs + k];
  __syncwarp();
  return n_cand;
}

__global__ void __launch_bounds__(32) k_narrowphase(const Params P) {
  int env;
  const Smem s = begin_warp<false>(P, env);
  unsigned st = 0;
  load_env(s, P, env);
  pose_and_predict(s, P, env, false);
  const int n_cand = load_candidates(s, P, env);
  const int n_coll = find_colliding(s, P, n_cand, 0, &st);
  write_contacts(s, P, env, n_cand, n_coll, 0);
  flush_status(P, env, st);
}

// Rebuild the colliding-pair list from a contact list in global memory (ordered (pair, slot); slot 0 carries
// the pair's normal): s.cpair[0], s.cab, s.wrank[r] = offset of the pair's first contact.
__device__ inline int pairs_from_contacts(const Smem& s, const Params& P, int env, int n_cont, unsigned* status) {
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
      s.cpair[0][rank] = (unsigned short)idx; s.cab[rank] = pack_ab(s, i, j, (tag >> 20) & 0xf); s.wrank[rank] = (unsigned short)c;
    }
    n += __popc(bal);
  }
  if (n > P.pc) { *status |= JENGA_ST_CONTACT_OVERFLOW; n = P.pc; }
  __syncwarp();
  return n;
}

template <bool TM>
__global__ void __launch_bounds__(TM ? 128 : 32) k_pgs(const Params P, const int iters) {
  int env;
  const Smem s = begin_warp<TM>(P, env);
  const int lane = lane_id();
  if (env < P.E) {
    unsigned st = 0;
    load_env(s, P, env);
    if (lane == 0) { s.misc[MiNprev] = -1; s.misc[MiNph] = 0; s.misc[MiNcol] = 0; }
    pose_and_predict(s, P, env, false);
    const int n_cont = max(0, min(P.n_contacts[env], P.max_contacts));
    const int n_coll = pairs_from_contacts(s, P, env, n_cont, &st);
    // contact offsets survive the colouring (which reuses s.wrank) in the previous-list buffer, free in this kernel
    const SP<unsigned short> keep = s.cpair[1];
    for (int r = lane; r < n_coll; r += 32) keep[r] = s.wrank[r];
    __syncwarp();
    colour_pairs<TM>(s, P, n_coll, 0, &st);
    for (int r = lane; r < n_coll; r += 32) s.wrank[r] = keep[r];
    __syncwarp();
    const float4* in = reinterpret_cast<const float4*>(P.contacts + (size_t)env * P.max_contacts * 8);
    for (int j = 0; 32 * j < n_coll; ++j) {
      const int k = 32 * j + lane;
      PairC pc;
#pragma unroll
      for (int t = 0; t < 48; ++t) pc.v[t] = 0.0f;
      if (k < n_coll) {
        const int r = s.order[k];
        const int c0 = s.wrank[r], c1 = r + 1 < n_coll ? s.wrank[r + 1] : n_cont;
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
        setup_slot(s, P, env, k, ab_a(w), ab_b(w), s.cpair[0][r], m, pc);
      }
      round_store<TM>(s, j, n_coll, pc);
    }
    __syncwarp();
    pgs_sweeps<TM>(s, P, iters, P.mu[env]);
    write_lambda<TM>(s, P, env, n_coll);
    store_env(s, P, env);
    flush_status(P, env, st);
  }
  end_warp<TM>(s);
}

}  // namespace jenga

// =================================================================== host side / C-ABI
using jenga::Params;

struct jenga_world {
  jenga_world_desc desc;
  jenga_buffers bufs;
  Params P;
  int tmb;                 // TMEM blocks per env of the step / solve kernels: 5, 10 or 0 (no TMEM, 1 warp per CTA)
  size_t smem_step;        // dynamic shared memory per CTA of k_step / k_pgs
  size_t smem_stage;       // ... of k_broadphase / k_narrowphase (one warp per CTA, no TMEM)
};

static char g_err[512] = "no error";

static bool desc_ok(const jenga_world_desc* d) {
  if (!d || d->struct_size != sizeof(jenga_world_desc)) return false;
  if (d->n_envs <= 0 || d->n_bodies <= 0 || d->n_bodies > 360) return false;   /* pair indices are 16-bit on chip */
  if (d->body_stride < d->n_bodies || (d->body_stride & 3)) return false;
  if (d->n_substeps <= 0 || d->pgs_iters < 0 || !(d->dt > 0.0f)) return false;
  if (d->max_pairs <= 0 || d->max_pairs > 65535) return false;
  if (d->max_contacts < 4 || (d->max_contacts & 3) || d->max_contacts > 65532) return false;
  if (4 * jenga::smem_words(d->body_stride, d->max_pairs, d->max_contacts / 4, 0) > 227 * 1024) return false;
  return true;
}

static size_t env_bytes(const jenga_world_desc* d, int tmb) {
  return 4 * jenga::smem_words(d->body_stride, d->max_pairs, d->max_contacts / 4, tmb);
}

/* TMEM blocks per env.  5 (256 columns per 4-env CTA) when two such CTAs fit one SM: 8 envs per SM; else 10 (512
 * columns) when one 4-env CTA fits: 4 envs per SM; else 0: the all-shared-memory kernel, one warp per CTA.
 * JENGA_NO_TMEM=1 forces 0 (the tests use it to cover both kernels). */
static int pick_tmb(const jenga_world_desc* d) {
  const char* off = getenv("JENGA_NO_TMEM");
  if (off && off[0] == '1') return 0;
  if (2 * (4 * env_bytes(d, 5) + 1024 + 16) <= 227 * 1024) return 5;
  if (4 * env_bytes(d, 10) + 1024 + 16 <= 227 * 1024 && env_bytes(d, 0) + 1024 > 227 * 1024 / 4) return 10;
  return 0;
}

extern "C" size_t jenga_smem_bytes(const jenga_world_desc* d) {
  if (!desc_ok(d)) return 0;
  const int tmb = pick_tmb(d);
  return tmb ? 4 * env_bytes(d, tmb) : env_bytes(d, 0);
}

extern "C" int jenga_block_threads(const jenga_world_desc* d) {
  if (!desc_ok(d)) return 0;
  return pick_tmb(d) ? 128 : 32;   /* one warp per env; 4 envs per CTA in the TMEM kernel */
}

extern "C" const char* jenga_strerror(int code) {
  switch (code) {
    case JENGA_OK: return "ok";
    case JENGA_E_ARG: return "bad argument (NULL or misaligned pointer, size or capacity out of range)";
    case JENGA_E_CUDA: return g_err;
    case JENGA_E_DEVICE: return "device is not sm_100 (kernels are built for sm_100a only)";
    default: return "unknown error";
  }
}

static int cuda_fail(cudaError_t e, const char* what) {
  snprintf(g_err, sizeof(g_err), "CUDA error in %s: %s", what, cudaGetErrorString(e));
  return JENGA_E_CUDA;
}

static bool aligned16(const void* p) { return p && (((uintptr_t)p) & 15u) == 0; }

extern "C" int jenga_world_create(const jenga_world_desc* d, const jenga_buffers* b, jenga_world** out) {
  if (!out) return JENGA_E_ARG;
  *out = nullptr;
  if (!desc_ok(d) || !b) return JENGA_E_ARG;
  if (!aligned16(b->state) || !aligned16(b->props) || !b->mu || !aligned16(b->pairs) || !b->n_pairs ||
      !aligned16(b->contacts) || !b->n_contacts || !b->lambda || !b->cache_key || !b->cache_lam || !b->cache_pt ||
      !b->n_cache || !b->status)
    return JENGA_E_ARG;
  if (b->f_ext && !aligned16(b->f_ext)) return JENGA_E_ARG;
  cudaDeviceProp prop;
  cudaError_t e = cudaGetDeviceProperties(&prop, d->device);
  if (e != cudaSuccess) return cuda_fail(e, "cudaGetDeviceProperties");
  if (prop.major != 10) return JENGA_E_DEVICE;
  const size_t smem = jenga_smem_bytes(d);
  if (smem > (size_t)prop.sharedMemPerBlockOptin) return JENGA_E_ARG;
  jenga_world* w = (jenga_world*)calloc(1, sizeof(jenga_world));
  if (!w) return JENGA_E_ARG;
  w->desc = *d; w->bufs = *b; w->tmb = pick_tmb(d); w->smem_step = smem; w->smem_stage = env_bytes(d, 0);
  Params& P = w->P;
  P.E = d->n_envs; P.B = d->n_bodies; P.S = d->body_stride;
  P.h = d->dt / (float)d->n_substeps; P.n_substeps = d->n_substeps; P.iters = d->pgs_iters;
  for (int k = 0; k < 3; ++k) P.g[k] = d->gravity[k];
  P.restitution = d->restitution; P.aabb_margin = d->aabb_margin; P.beta = d->baumgarte_beta; P.slop = d->slop;
  P.cp.edge_bias_rel = d->edge_bias_rel; P.cp.edge_bias_abs = d->edge_bias_abs; P.cp.par_eps = d->par_eps; P.cp.tie_eps = d->tie_eps;
  P.match_tol = d->match_tol; P.warm_start = d->warm_start; P.gyroscopic = d->gyroscopic;
  P.max_pairs = d->max_pairs; P.max_contacts = d->max_contacts; P.pc = d->max_contacts / 4; P.materialise = d->materialise; P.tmb = w->tmb;
  P.state = b->state; P.props = b->props; P.mu = b->mu; P.f_ext = b->f_ext;
  P.pairs = b->pairs; P.n_pairs = b->n_pairs; P.contacts = b->contacts; P.n_contacts = b->n_contacts; P.lambda = b->lambda;
  P.cache_key = b->cache_key; P.cache_lam = b->cache_lam; P.cache_pt = b->cache_pt; P.n_cache = b->n_cache;
  P.status = b->status; P.counters = b->counters;
  const bool latch = d->collapse_length > 0.0f && b->ref_pose && b->collapsed;
  P.ref_pose = latch ? b->ref_pose : nullptr; P.collapsed = latch ? b->collapsed : nullptr;
  P.collapse_stats = latch ? b->collapse_stats : nullptr;
  P.rest_steps = b->rest_steps;
  P.collapse_dx = d->collapse_fd * d->collapse_length; P.collapse_ek = d->collapse_ek; P.collapse_theta = d->collapse_theta;
  struct { const void* k; size_t smem; } kernels[] = {
    { w->tmb ? (const void*)jenga::k_step<true> : (const void*)jenga::k_step<false>, w->smem_step },
    { w->tmb ? (const void*)jenga::k_pgs<true> : (const void*)jenga::k_pgs<false>, w->smem_step },
    { (const void*)jenga::k_broadphase, w->smem_stage }, { (const void*)jenga::k_narrowphase, w->smem_stage } };
  for (auto& kn : kernels) {
    e = cudaFuncSetAttribute(kn.k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kn.smem);
    if (e != cudaSuccess) { free(w); return cuda_fail(e, "cudaFuncSetAttribute"); }
    cudaFuncSetAttribute(kn.k, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  }
  *out = w;
  return JENGA_OK;
}

static int launched(const char* name) {
  const cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? JENGA_OK : cuda_fail(e, name);
}

extern "C" int jenga_world_destroy(jenga_world* w) {
  if (!w) return JENGA_E_ARG;
  free(w);
  return JENGA_OK;
}

extern "C" int jenga_set_f_ext(jenga_world* w, const float* f_ext) {
  if (!w || (f_ext && !aligned16(f_ext))) return JENGA_E_ARG;
  w->bufs.f_ext = f_ext; w->P.f_ext = f_ext;
  return JENGA_OK;
}

extern "C" int jenga_broadphase(jenga_world* w, void* stream) {
  if (!w) return JENGA_E_ARG;
  jenga::k_broadphase<<<w->P.E, 32, w->smem_stage, (cudaStream_t)stream>>>(w->P);
  return launched("k_broadphase");
}

extern "C" int jenga_narrowphase(jenga_world* w, void* stream) {
  if (!w) return JENGA_E_ARG;
  jenga::k_narrowphase<<<w->P.E, 32, w->smem_stage, (cudaStream_t)stream>>>(w->P);
  return launched("k_narrowphase");
}

extern "C" int jenga_pgs_solve(jenga_world* w, int iters, void* stream) {
  if (!w || iters < 0) return JENGA_E_ARG;
  const int it = iters > 0 ? iters : w->P.iters;
  if (w->tmb) jenga::k_pgs<true><<<(w->P.E + 3) / 4, 128, w->smem_step, (cudaStream_t)stream>>>(w->P, it);
  else jenga::k_pgs<false><<<w->P.E, 32, w->smem_step, (cudaStream_t)stream>>>(w->P, it);
  return launched("k_pgs");
}

extern "C" int jenga_step(jenga_world* w, int n_steps, void* stream) {
  if (!w || n_steps < 0) return JENGA_E_ARG;
  if (n_steps == 0) return JENGA_OK;
  if (w->tmb) jenga::k_step<true><<<(w->P.E + 3) / 4, 128, w->smem_step, (cudaStream_t)stream>>>(w->P, n_steps, 0.0f);
  else jenga::k_step<false><<<w->P.E, 32, w->smem_step, (cudaStream_t)stream>>>(w->P, n_steps, 0.0f);
  return launched("k_step");
}

extern "C" int jenga_simulate_until_rest(jenga_world* w, int max_steps, float ek_rest, void* stream) {
  if (!w || max_steps <= 0 || !(ek_rest > 0.0f)) return JENGA_E_ARG;
  if (w->tmb) jenga::k_step<true><<<(w->P.E + 3) / 4, 128, w->smem_step, (cudaStream_t)stream>>>(w->P, max_steps, ek_rest);
  else jenga::k_step<false><<<w->P.E, 32, w->smem_step, (cudaStream_t)stream>>>(w->P, max_steps, ek_rest);
  return launched("k_step (until rest)");
}

extern "C" int jenga_step_host(jenga_world* w, const float* h_in, float* h_out, int n_steps, void* stream) {
  if (!w || n_steps < 0) return JENGA_E_ARG;
  const size_t bytes = (size_t)w->P.E * jenga::kStateRows * w->P.S * sizeof(float);
  cudaStream_t st = (cudaStream_t)stream;
  if (h_in) {
    cudaError_t e = cudaMemcpyAsync(w->bufs.state, h_in, bytes, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(e, "jenga_step_host H2D");
  }
  const int rc = jenga_step(w, n_steps, stream);
  if (rc != JENGA_OK) return rc;
  if (h_out) {
    cudaError_t e = cudaMemcpyAsync(h_out, w->bufs.state, bytes, cudaMemcpyDeviceToHost, st);
    if (e != cudaSuccess) return cuda_fail(e, "jenga_step_host D2H");
  }
  return JENGA_OK;
}
