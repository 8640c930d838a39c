// jenga.cu -- C-ABI of the batched Jenga step (include/jenga.h) over the six kernels of a substep.  sm_100a only.
//
//   k_detect  (kcollide.cuh)  S1 predict, S2 broadphase, S3 SAT                                -> scratch
//   k_walk    (kcollide.cuh)  S4 greedy colouring of the envs whose pair list changed          -> scratch
//   k_plan    (kcollide.cuh)  S4 visit plan of the groups with such an env                      -> scratch
//   k_manifold (kcollide.cuh) S3 contact manifolds                                              -> scratch
//   k_slot    (kcollide.cuh)  S4 effective masses + warm-start lookup                           -> scratch
//   k_solve   (ksolve.cuh)    S4 warm start, S5 PGS sweeps, S6 integrate, S7 cache, Eq. 18 latch
// One warp per env in k_detect, k_plan, k_manifold and k_slot, one thread per env in k_walk, one warp per group of G envs
// in k_solve (layout.cuh).  jenga_step(n) enqueues n * n_substeps such sextuples of launches on the caller's stream; nothing
// returns to the host in between.  The stage entry points run the same device functions in a reduced mode.
#include <cuda_runtime.h>
#include <stdio.h>
#include <stdlib.h>
#include <new>
#include <string.h>

#include <mutex>
#include <vector>

#include "ksolve.cuh"
#include "analysis.cuh"

namespace jenga {

// jenga_simulate_until_rest: clear the per-env rest flag and step count kept in the scratch.
__global__ void k_reset_rest(const Params P) {
  const int env = blockIdx.x * blockDim.x + threadIdx.x;
  if (env >= P.E) return;
  int* meta = reinterpret_cast<int*>(P.scratch + (size_t)env * P.scratch_words + scratch_layout(P.pc, P.G).meta);
  meta[MetaResting] = 0; meta[MetaSteps] = 0;
}

}  // namespace jenga

// =================================================================== host side / C-ABI
using jenga::Params;

enum { TierAuto = 0, TierSmem = 1, TierTmem256 = 2, TierTmem512 = 3, TierTmem160 = 4, TierTmem128 = 5 };
static const size_t kSmemMax = 227 * 1024;
static const int kSmNominal = 148;     /* SMs of a B200: used by the tier heuristic only (helpers answer without a device) */

struct jenga_world {
  jenga_world_desc desc;
  jenga_buffers bufs;
  Params P;
  int tmb;                 // TMEM blocks per group of k_solve: 2, 3, 4, 9 or 0 (no TMEM, 1 warp per CTA)
  int G;                   // envs per group (= per k_solve warp)
  int wpc_collide;         // warps (= envs) per CTA of the collision kernels
  int n_sm;
  size_t smem_solve;       // dynamic shared memory per CTA of k_solve
  size_t smem_collide;     // ... of k_detect
  size_t smem_manifold, smem_slot, smem_plan;   // ... of k_manifold, k_slot, k_plan
  bool stage_bufs;         // pairs / contacts / lambda were given: the stage calls are available
  bool profiling;          // jenga_profile_enable: events around every launch of the step
  std::vector<cudaEvent_t> ev;   // e0 k_detect e1 k_manifold e2 k_slot e3 k_solve e4, per substep
  std::vector<cudaEvent_t> ev_pool;   // events of earlier reads, reused by the next marks (no create / destroy per substep)
  bool ev_broken;          // an event could not be created or recorded: the groups of five no longer line up
};

static thread_local char g_err[512] = "no error";

static size_t collide_env_bytes(const jenga_world_desc* d, int G, int arena = -1) {
  const size_t a = 4 * jenga::collide_smem_words(d->body_stride, d->max_pairs, d->max_contacts / 4, jenga::ArenaDetect, G);
  const size_t b = 4 * jenga::collide_smem_words(d->body_stride, d->max_pairs, d->max_contacts / 4, jenga::ArenaManifold, G);
  const size_t c = 4 * jenga::collide_smem_words(d->body_stride, d->max_pairs, d->max_contacts / 4, jenga::ArenaSlot, G);
  const size_t p = 4 * jenga::collide_smem_words(d->body_stride, d->max_pairs, d->max_contacts / 4, jenga::ArenaPlan, G);
  if (arena == jenga::ArenaPlan) return p;
  const size_t ab = a > b ? a : b, cp = c > p ? c : p;
  return arena == jenga::ArenaDetect ? a : (arena == jenga::ArenaManifold ? b : (arena == jenga::ArenaSlot ? c : (ab > cp ? ab : cp)));
}
/* shared memory of one k_solve warp (= one group of G envs), without / with smb blocks of spare shared memory */
static size_t solve_group_bytes(const jenga_world_desc* d, int tmb, int G, int smb = 0) {
  return 4 * jenga::solve_smem_words(d->body_stride, d->max_contacts / 4, tmb, smb, G);
}

static bool desc_ok(const jenga_world_desc* d) {
  if (!d || d->struct_size != sizeof(jenga_world_desc)) return false;
  if (d->n_envs <= 0 || d->n_bodies <= 0 || d->n_bodies > 360) return false;   /* pair indices are 16-bit on chip */
  if (d->body_stride < d->n_bodies || (d->body_stride & 3)) return false;
  if (d->n_substeps <= 0 || d->n_substeps > 64 || d->pgs_iters < 0 || !(d->dt > 0.0f)) return false;
  if (d->max_pairs <= 0 || d->max_pairs > 65535) return false;
  if (d->max_contacts < 4 || (d->max_contacts & 3) || d->max_contacts > 65532) return false;
  if (d->solver_tier < TierAuto || d->solver_tier > TierTmem128) return false;
  if (d->env_group < 0 || d->env_group > jenga::kMaxGroup) return false;
  if (collide_env_bytes(d, 1) > kSmemMax || solve_group_bytes(d, 0, 1) > kSmemMax) return false;
  return true;
}

/* Envs per k_solve warp.  Two envs share a warp when the batch still fills the machine that way (every SM gets 16 groups),
 * when two collision warps fit one CTA (the two warps of a group plan their visits together in k_detect), and when the
 * widest tensor-memory tier holds the doubled records; desc.env_group forces it (-1 if it does not fit).           */
static bool group_fits(const jenga_world_desc* d, int G) {
  if (G == 1) return true;
  return 2 * collide_env_bytes(d, G) <= kSmemMax && solve_group_bytes(d, 0, G) + 1024 <= kSmemMax;
}
static int pick_group(const jenga_world_desc* d) {
  if (d->env_group) return group_fits(d, d->env_group) ? d->env_group : -1;
  return (long long)d->n_envs >= 2ll * 16 * kSmNominal && group_fits(d, 2) ? 2 : 1;
}

/* TMEM blocks per group of k_solve: the CTA (one per SM) has 4 Q warps = 4 Q groups in flight; each group gets 512 / Q
 * columns = tmb blocks of 56: Q = 4 -> 2 blocks (16 groups per SM), Q = 3 -> 3, Q = 2 -> 4, Q = 1 -> 9; 0 = everything in
 * shared memory, one warp per CTA.  Auto takes the largest Q whose shared memory (body records of 4 Q groups) fits one
 * SM; desc.solver_tier forces a tier (-1 if it does not fit).                                                      */
static int tier_groups(int tmb) { return tmb == 2 ? 4 : (tmb == 3 ? 3 : (tmb == 4 ? 2 : (tmb == 9 ? 1 : 0))); }
static bool tier_fits(const jenga_world_desc* d, int tmb, int G) {
  return 4 * tier_groups(tmb) * solve_group_bytes(d, tmb, G) + 1024 + 16 <= kSmemMax;
}
/* The blocks of a group beyond its tensor-memory share are re-read from the scratch in every sweep: they must stay in L2
 * while the group is in flight, or every visit goes to HBM (measured at cfg5 with two envs per warp: 16 groups per SM =
 * 133 MB of blocks in flight, k_solve 6.9 ms; 12 groups per SM = 87 MB, 4.8 ms).  Capacity-based estimate, 126 MB of L2. */
static bool tier_in_l2(const jenga_world_desc* d, int tmb, int G) {
  /* blocks a group uses: about 4/5 of its capacity (cfg5: 10 of 12 with two envs per group; cfg4: 8 of 10) */
  const long long nblk = (4 * jenga::n_blocks(d->max_contacts / 4, G) + 4) / 5, out = nblk > tmb ? nblk - tmb : 0;
  return (long long)kSmNominal * 4 * tier_groups(tmb) * out * jenga::kBlkWords * 4 <= 120ll << 20;
}
static int pick_tmb(const jenga_world_desc* d, int G) {
  switch (d->solver_tier) {
    case TierSmem: return solve_group_bytes(d, 0, G) + 1024 <= kSmemMax ? 0 : -1;
    case TierTmem128: return tier_fits(d, 2, G) ? 2 : -1;
    case TierTmem160: return tier_fits(d, 3, G) ? 3 : -1;
    case TierTmem256: return tier_fits(d, 4, G) ? 4 : -1;
    case TierTmem512: return tier_fits(d, 9, G) ? 9 : -1;
    default: {
      /* auto.  A batch that does not fill the machine (148 SMs x 4 Q groups in flight) takes the tier with the fewest groups
         per SM that still holds it at once: more of every group's blocks are then in tensor memory, and below
         4 groups per SM the shared-memory tier (lowest latency per chunk visit) is the quickest.  All tiers give the same bits. */
      const long long NG = ((long long)d->n_envs + G - 1) / G;
      if (NG <= 4ll * kSmNominal && solve_group_bytes(d, 0, G) + 1024 <= kSmemMax) return 0;
      const int by_size[3] = { 9, 4, 3 };
      for (int k = 0; k < 3; ++k)
        if (NG <= 4ll * tier_groups(by_size[k]) * kSmNominal && tier_fits(d, by_size[k], G)) return by_size[k];
      const int by_width[4] = { 2, 3, 4, 9 };
      for (int k = 0; k < 4; ++k)
        if (tier_fits(d, by_width[k], G) && (tier_in_l2(d, by_width[k], G) || k == 3)) return by_width[k];
      return 0;
    }
  }
}

/* Blocks per group that a tensor-memory tier also keeps in shared memory: what the CTA's 227 KB leave per warp, at most
 * the blocks beyond the TMEM share. */
static int pick_smb(const jenga_world_desc* d, int tmb, int G) {
  if (!tmb) return 0;
  const long long warps = 4 * tier_groups(tmb), spare = (long long)kSmemMax - 1024 - 16 - warps * (long long)solve_group_bytes(d, tmb, G);
  const long long nblk = jenga::n_blocks(d->max_contacts / 4, G), smb = spare / (warps * jenga::kBlkWords * 4);
  return (int)(smb < 0 ? 0 : (smb > nblk - tmb ? (nblk > tmb ? nblk - tmb : 0) : smb));
}

/* dynamic shared memory of a k_solve CTA */
static size_t solve_cta_bytes(const jenga_world_desc* d, int tmb, int G) {
  return tmb ? 4 * tier_groups(tmb) * solve_group_bytes(d, tmb, G, pick_smb(d, tmb, G)) : solve_group_bytes(d, 0, G);
}

extern "C" size_t jenga_smem_bytes(const jenga_world_desc* d) {
  if (!desc_ok(d)) return 0;
  const int G = pick_group(d), tmb = G < 0 ? -1 : pick_tmb(d, G);
  return tmb < 0 ? 0 : solve_cta_bytes(d, tmb, G);
}

extern "C" int jenga_block_threads(const jenga_world_desc* d) {
  if (!desc_ok(d)) return 0;
  const int G = pick_group(d), tmb = G < 0 ? -1 : pick_tmb(d, G);
  return tmb < 0 ? 0 : (tmb ? 128 * tier_groups(tmb) : 32);   /* one warp per group; 4, 8, 12 or 16 groups per CTA in the TMEM tiers */
}

extern "C" int jenga_env_group(const jenga_world_desc* d) {
  if (!desc_ok(d)) return 0;
  const int G = pick_group(d);
  return G < 0 ? 0 : G;
}

extern "C" size_t jenga_scratch_bytes(const jenga_world_desc* d) {
  if (!desc_ok(d)) return 0;
  const int G = pick_group(d);
  if (G < 0) return 0;
  return ((size_t)d->n_envs * jenga::scratch_layout(d->max_contacts / 4, G).total + jenga::kScratchHead + jenga::round_up(d->n_envs, 32)) * sizeof(float);
}

extern "C" const char* jenga_strerror(int code) {
  switch (code) {
    case JENGA_OK: return "ok";
    case JENGA_E_ARG: return "bad argument (NULL or misaligned pointer, size or capacity out of range)";
    case JENGA_E_CUDA: return g_err;
    case JENGA_E_DEVICE: return "device is not sm_100 or not the current device (kernels are built for sm_100a only)";
    case JENGA_E_STATIC_CAPACITY: return "jenga_narrowphase_static: n_envs x jenga_narrowphase_static_env_bytes(desc) exceeds the built-in "
                                         "scratch (JENGA_STATIC_SCRATCH_BYTES = 8 MiB); split the batch into smaller calls";
    default: return "unknown error";
  }
}

static int cuda_fail(cudaError_t e, const char* what) {
  snprintf(g_err, sizeof(g_err), "CUDA error in %s: %s", what, cudaGetErrorString(e));
  return JENGA_E_CUDA;
}

static bool aligned16(const void* p) { return p && (((uintptr_t)p) & 15u) == 0; }

/* cudaFuncAttributeMaxDynamicSharedMemorySize is per kernel and process-wide: it is only ever raised (running maximum
 * per device), immediately before the launch that needs it, so worlds of different sizes can be used in any order.   */
enum { KnCollide = 0, KnCollideBroad, KnCollideNarrow, KnCollideGiven, KnManifold, KnManifoldNarrow, KnSlot, KnSlotGiven, KnPlan, KnWalk, KnSolveTm, KnSolveTm384, KnSolveTm256, KnSolveTm128, KnSolveSm, KnSupport, KnCount };
static std::mutex g_attr_mutex;
static size_t g_attr_max[16][KnCount];   /* bytes already granted; 0 = the 48 KB every kernel has without opting in */

static const void* kernel_ptr(int kn) {
  switch (kn) {
    case KnCollide: return (const void*)jenga::k_detect<jenga::ModeStep>;
    case KnCollideBroad: return (const void*)jenga::k_detect<jenga::ModeBroad>;
    case KnCollideNarrow: return (const void*)jenga::k_detect<jenga::ModeNarrow>;
    case KnCollideGiven: return (const void*)jenga::k_detect<jenga::ModeGiven>;
    case KnManifold: return (const void*)jenga::k_manifold<jenga::ModeStep>;
    case KnManifoldNarrow: return (const void*)jenga::k_manifold<jenga::ModeNarrow>;
    case KnSlot: return (const void*)jenga::k_slot<jenga::ModeStep>;
    case KnSlotGiven: return (const void*)jenga::k_slot<jenga::ModeGiven>;
    case KnPlan: return (const void*)jenga::k_plan;
    case KnWalk: return (const void*)jenga::k_walk;
    case KnSolveTm: return (const void*)jenga::k_solve<true, 512>;
    case KnSolveTm384: return (const void*)jenga::k_solve<true, 384>;
    case KnSolveTm256: return (const void*)jenga::k_solve<true, 256>;
    case KnSolveTm128: return (const void*)jenga::k_solve<true, 128>;
    case KnSupport: return (const void*)jenga::k_support;
    default: return (const void*)jenga::k_solve<false, 32>;
  }
}

static cudaError_t ensure_smem(int device, int kn, size_t bytes) {
  std::lock_guard<std::mutex> lock(g_attr_mutex);
  const int dv = device & 15;
  if (bytes <= g_attr_max[dv][kn]) return cudaSuccess;
  cudaError_t e = cudaFuncSetAttribute(kernel_ptr(kn), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
  if (e != cudaSuccess) return e;
  cudaFuncSetAttribute(kernel_ptr(kn), cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  g_attr_max[dv][kn] = bytes;
  return cudaSuccess;
}

extern "C" int jenga_world_create(const jenga_world_desc* d, const jenga_buffers* b, jenga_world** out) {
  if (!out) return JENGA_E_ARG;
  *out = nullptr;
  if (!desc_ok(d) || !b) return JENGA_E_ARG;
  if (!aligned16(b->state) || !aligned16(b->props) || !b->mu || !b->cache_key || !aligned16(b->cache_lam) || !aligned16(b->cache_pt) ||
      !b->n_cache || !b->status || !aligned16(b->scratch))
    return JENGA_E_ARG;
  /* the stage buffers (pairs .. lambda) are written by the stage calls and by jenga_step only with materialise = 1: a world
     that only steps may leave all five NULL (all or none) and then refuses the stage calls */
  const bool any_stage = b->pairs || b->n_pairs || b->contacts || b->n_contacts || b->lambda;
  const bool all_stage = aligned16(b->pairs) && b->n_pairs && aligned16(b->contacts) && b->n_contacts && b->lambda;
  if ((any_stage || d->materialise) && !all_stage) return JENGA_E_ARG;
  if (b->f_ext && !aligned16(b->f_ext)) return JENGA_E_ARG;
  if (d->collapse_length > 0.0f && b->ref_pose && b->collapsed &&      /* latch on: ref_pose rows and the float4 stats */
      (!aligned16(b->ref_pose) || (b->collapse_stats && !aligned16(b->collapse_stats))))
    return JENGA_E_ARG;
  if (b->scratch_bytes < jenga_scratch_bytes(d)) return JENGA_E_ARG;
  const int G = pick_group(d);
  if (G < 0) return JENGA_E_ARG;
  const int tmb = pick_tmb(d, G);
  if (tmb < 0) return JENGA_E_ARG;
  int cur = -1;
  cudaError_t e = cudaGetDevice(&cur);
  if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
  if (cur != d->device) return JENGA_E_DEVICE;       /* every call launches on the current device: it must be desc.device */
  cudaDeviceProp prop;
  e = cudaGetDeviceProperties(&prop, d->device);
  if (e != cudaSuccess) return cuda_fail(e, "cudaGetDeviceProperties");
  if (prop.major != 10) return JENGA_E_DEVICE;
  jenga_world* w = new (std::nothrow) jenga_world();
  if (!w) return JENGA_E_ARG;
  w->profiling = false; w->ev_broken = false;
  w->stage_bufs = all_stage;
  w->desc = *d; w->bufs = *b; w->tmb = tmb; w->G = G; w->n_sm = prop.multiProcessorCount;
  w->smem_solve = solve_cta_bytes(d, tmb, G);
  const size_t cb = collide_env_bytes(d, G);
  w->wpc_collide = 4 * cb <= kSmemMax ? 4 : (2 * cb <= kSmemMax ? 2 : 1);       /* G = 2: group_fits made sure of two */
  w->smem_collide = w->wpc_collide * collide_env_bytes(d, G, jenga::ArenaDetect);
  w->smem_manifold = w->wpc_collide * collide_env_bytes(d, G, jenga::ArenaManifold);
  w->smem_slot = w->wpc_collide * collide_env_bytes(d, G, jenga::ArenaSlot);
  w->smem_plan = w->wpc_collide * collide_env_bytes(d, G, jenga::ArenaPlan);
  if (w->smem_solve > (size_t)prop.sharedMemPerBlockOptin || w->smem_collide > (size_t)prop.sharedMemPerBlockOptin) { delete w; return JENGA_E_ARG; }
  Params& P = w->P;
  P.E = d->n_envs; P.B = d->n_bodies; P.S = d->body_stride;
  P.h = d->dt / (float)d->n_substeps; P.n_substeps = d->n_substeps; P.iters = d->pgs_iters;
  for (int k = 0; k < 3; ++k) P.g[k] = d->gravity[k];
  P.restitution = d->restitution; P.aabb_margin = d->aabb_margin; P.beta = d->baumgarte_beta; P.slop = d->slop;
  P.cp.edge_bias_rel = d->edge_bias_rel; P.cp.edge_bias_abs = d->edge_bias_abs; P.cp.par_eps = d->par_eps; P.cp.tie_eps = d->tie_eps;
  P.match_tol = d->match_tol; P.warm_start = d->warm_start; P.gyroscopic = d->gyroscopic;
  P.max_pairs = d->max_pairs; P.max_contacts = d->max_contacts; P.pc = d->max_contacts / 4; P.materialise = d->materialise;
  P.tmb = tmb; P.G = G; P.nblk = jenga::n_blocks(P.pc, G); P.smb = pick_smb(d, tmb, G);
  P.state = b->state; P.props = b->props; P.mu = b->mu; P.f_ext = b->f_ext;
  P.pairs = b->pairs; P.n_pairs = b->n_pairs; P.contacts = b->contacts; P.n_contacts = b->n_contacts; P.lambda = b->lambda;
  P.cache_key = b->cache_key; P.cache_lam = b->cache_lam; P.cache_pt = b->cache_pt; P.n_cache = b->n_cache;
  P.status = b->status; P.counters = b->counters;
  const bool latch = d->collapse_length > 0.0f && b->ref_pose && b->collapsed;
  P.ref_pose = latch ? b->ref_pose : nullptr; P.collapsed = latch ? b->collapsed : nullptr;
  P.collapse_stats = latch ? b->collapse_stats : nullptr;
  P.rest_steps = b->rest_steps;
  P.collapse_dx = d->collapse_fd * d->collapse_length; P.collapse_ek = d->collapse_ek; P.collapse_theta = d->collapse_theta;
  P.work_counter = (int*)b->scratch;
  P.same_flag = (int*)b->scratch + jenga::kScratchHead;
  P.scratch = (float*)b->scratch + jenga::kScratchHead + jenga::round_up(d->n_envs, 32); P.scratch_words = jenga::scratch_layout(P.pc, G).total;
  *out = w;
  return JENGA_OK;
}

static int launched(const char* name) {
  const cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? JENGA_OK : cuda_fail(e, name);
}

/* Every launch goes to the CURRENT device with pointers that belong to desc.device: on any other device the kernels would
 * fault on foreign addresses (a sticky error that ends the context), and the shared-memory opt-in below would be recorded
 * for the wrong device.  Checked at the top of every call that launches or copies. */
static int on_device(const jenga_world* w) {
  int cur = -1;
  const cudaError_t e = cudaGetDevice(&cur);
  if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
  return cur == w->desc.device ? JENGA_OK : JENGA_E_DEVICE;
}

/* recorded events go back to the pool for the next marks; `destroy` (jenga_world_destroy) frees them all */
static void drop_events(jenga_world* w, bool destroy = false) {
  for (cudaEvent_t e : w->ev) w->ev_pool.push_back(e);
  w->ev.clear();
  w->ev_broken = false;
  if (!destroy) return;
  for (cudaEvent_t e : w->ev_pool) cudaEventDestroy(e);
  w->ev_pool.clear();
}

extern "C" int jenga_world_destroy(jenga_world* w) {
  if (!w) return JENGA_E_ARG;
  drop_events(w, true);
  delete w;
  return JENGA_OK;
}

extern "C" int jenga_profile_enable(jenga_world* w, int on) {
  if (!w) return JENGA_E_ARG;
  drop_events(w);
  w->profiling = on != 0;
  return JENGA_OK;
}

extern "C" int jenga_profile_read(jenga_world* w, double* out) {
  if (!w || !out) return JENGA_E_ARG;
  /* five marks per substep, recorded by step_launches only; a mark that failed would shift every later group */
  if (w->ev_broken || w->ev.size() % 5 != 0) {
    drop_events(w);
    return cuda_fail(cudaErrorUnknown, "jenga_profile_read (an event of this interval could not be created or recorded)");
  }
  double ms[4] = { 0.0, 0.0, 0.0, 0.0 }; const size_t n = w->ev.size() / 5;
  for (size_t i = 0; i < n; ++i) {
    cudaError_t e = cudaEventSynchronize(w->ev[5 * i + 4]);
    if (e != cudaSuccess) return cuda_fail(e, "jenga_profile_read");
    for (int k = 0; k < 4; ++k) {
      float t = 0.0f;
      e = cudaEventElapsedTime(&t, w->ev[5 * i + k], w->ev[5 * i + k + 1]);
      if (e != cudaSuccess) { drop_events(w); return cuda_fail(e, "jenga_profile_read (cudaEventElapsedTime)"); }
      ms[k] += t;
    }
  }
  for (int k = 0; k < 4; ++k) out[k] = ms[k];
  out[4] = (double)n;
  drop_events(w);
  return JENGA_OK;
}


extern "C" int jenga_set_f_ext(jenga_world* w, const float* f_ext) {
  if (!w || (f_ext && !aligned16(f_ext))) return JENGA_E_ARG;
  w->bufs.f_ext = f_ext; w->P.f_ext = f_ext;
  return JENGA_OK;
}

static void mark(jenga_world* w, cudaStream_t st) {
  if (!w->profiling) return;
  cudaEvent_t e;
  if (!w->ev_pool.empty()) { e = w->ev_pool.back(); w->ev_pool.pop_back(); }
  else if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); w->ev_broken = true; return; }
  if (cudaEventRecord(e, st) != cudaSuccess) { cudaGetLastError(); w->ev_broken = true; }
  w->ev.push_back(e);
}

/* k_detect, then (except for jenga_broadphase) k_walk, k_plan, k_manifold and k_slot, for every env */
static int launch_collide(jenga_world* w, int mode, int honour_rest, cudaStream_t st) {
  int rc = on_device(w);
  if (rc != JENGA_OK) return rc;
  cudaError_t e = ensure_smem(w->desc.device, KnCollide + mode, w->smem_collide);
  if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(k_detect)");
  const int wpc = w->wpc_collide, grid = (w->P.E + wpc - 1) / wpc, thr = 32 * wpc;
  switch (mode) {
    case jenga::ModeStep: jenga::k_detect<jenga::ModeStep><<<grid, thr, w->smem_collide, st>>>(w->P, honour_rest); break;
    case jenga::ModeBroad: jenga::k_detect<jenga::ModeBroad><<<grid, thr, w->smem_collide, st>>>(w->P, honour_rest); break;
    case jenga::ModeNarrow: jenga::k_detect<jenga::ModeNarrow><<<grid, thr, w->smem_collide, st>>>(w->P, honour_rest); break;
    default: jenga::k_detect<jenga::ModeGiven><<<grid, thr, w->smem_collide, st>>>(w->P, honour_rest); break;
  }
  rc = launched("k_detect");
  if (rc != JENGA_OK || mode == jenga::ModeBroad) return rc;
  const size_t smem_walk = (size_t)jenga::kWalkThreads * w->P.B * sizeof(unsigned long long);
  e = ensure_smem(w->desc.device, KnWalk, smem_walk);
  if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(k_walk)");
  jenga::k_walk<<<(w->P.E + jenga::kWalkThreads - 1) / jenga::kWalkThreads, jenga::kWalkThreads, smem_walk, st>>>(w->P);
  rc = launched("k_walk");
  if (rc != JENGA_OK) return rc;
  e = ensure_smem(w->desc.device, KnPlan, w->smem_plan);
  if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(k_plan)");
  jenga::k_plan<<<grid, thr, w->smem_plan, st>>>(w->P);
  rc = launched("k_plan");
  if (rc != JENGA_OK) return rc;
  if (mode == jenga::ModeStep) mark(w, st);
  if (mode != jenga::ModeGiven) {                           /* manifolds (jenga_pgs_solve: the caller's contacts instead) */
    const int kn = mode == jenga::ModeStep ? KnManifold : KnManifoldNarrow;
    e = ensure_smem(w->desc.device, kn, w->smem_manifold);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(k_manifold)");
    if (mode == jenga::ModeStep) jenga::k_manifold<jenga::ModeStep><<<grid, thr, w->smem_manifold, st>>>(w->P, honour_rest);
    else jenga::k_manifold<jenga::ModeNarrow><<<grid, thr, w->smem_manifold, st>>>(w->P, honour_rest);
    rc = launched("k_manifold");
    if (rc != JENGA_OK || mode == jenga::ModeNarrow) return rc;
  }
  if (mode == jenga::ModeStep) mark(w, st);
  e = ensure_smem(w->desc.device, mode == jenga::ModeStep ? KnSlot : KnSlotGiven, w->smem_slot);
  if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(k_slot)");
  if (mode == jenga::ModeStep) jenga::k_slot<jenga::ModeStep><<<grid, thr, w->smem_slot, st>>>(w->P, honour_rest);
  else jenga::k_slot<jenga::ModeGiven><<<grid, thr, w->smem_slot, st>>>(w->P, honour_rest);
  return launched("k_slot");
}

static int launch_solve(jenga_world* w, int iters, int flags, float rest_ek, cudaStream_t st) {
  const int dev_rc = on_device(w);
  if (dev_rc != JENGA_OK) return dev_rc;
  const int q = tier_groups(w->tmb);
  const int kn = !w->tmb ? KnSolveSm : (q == 4 ? KnSolveTm : (q == 3 ? KnSolveTm384 : (q == 2 ? KnSolveTm256 : KnSolveTm128)));
  const cudaError_t e = ensure_smem(w->desc.device, kn, w->smem_solve);
  if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(k_solve)");
  /* persistent CTAs: one per SM in the TMEM tiers (it owns all 512 columns), each warp takes groups from a global queue */
  const int n_groups = (w->P.E + w->G - 1) / w->G;
  if (w->tmb) {
    /* small batches are spread over all SMs (the warps of every CTA pull groups from the same queue) */
    const int wpc = 4 * tier_groups(w->tmb), grid = n_groups < w->n_sm ? n_groups : w->n_sm;
    switch (q) {
      case 4: jenga::k_solve<true, 512><<<grid, 32 * wpc, w->smem_solve, st>>>(w->P, iters, flags, rest_ek); break;
      case 3: jenga::k_solve<true, 384><<<grid, 32 * wpc, w->smem_solve, st>>>(w->P, iters, flags, rest_ek); break;
      case 2: jenga::k_solve<true, 256><<<grid, 32 * wpc, w->smem_solve, st>>>(w->P, iters, flags, rest_ek); break;
      default: jenga::k_solve<true, 128><<<grid, 32 * wpc, w->smem_solve, st>>>(w->P, iters, flags, rest_ek); break;
    }
  } else {
    const int per_sm = (int)(kSmemMax / (w->smem_solve + 1024)), resident = w->n_sm * (per_sm < 1 ? 1 : (per_sm > 16 ? 16 : per_sm));
    jenga::k_solve<false, 32><<<n_groups < resident ? n_groups : resident, 32, w->smem_solve, st>>>(w->P, iters, flags, rest_ek);
  }
  return launched("k_solve");
}

extern "C" int jenga_broadphase(jenga_world* w, void* stream) {
  if (!w || !w->stage_bufs) return JENGA_E_ARG;
  return launch_collide(w, jenga::ModeBroad, 0, (cudaStream_t)stream);
}

extern "C" int jenga_narrowphase(jenga_world* w, void* stream) {
  if (!w || !w->stage_bufs) return JENGA_E_ARG;
  return launch_collide(w, jenga::ModeNarrow, 0, (cudaStream_t)stream);
}

extern "C" int jenga_pgs_solve(jenga_world* w, int iters, void* stream) {
  if (!w || iters < 0 || !w->stage_bufs) return JENGA_E_ARG;
  const int rc = launch_collide(w, jenga::ModeGiven, 0, (cudaStream_t)stream);
  if (rc != JENGA_OK) return rc;
  return launch_solve(w, iters > 0 ? iters : w->P.iters, jenga::SolvePgsOnly, 0.0f, (cudaStream_t)stream);
}

static int step_launches(jenga_world* w, int n_steps, int rest, float rest_ek, cudaStream_t st) {
  const int n_sub = w->P.n_substeps;
  for (int s = 0; s < n_steps; ++s)
    for (int sub = 0; sub < n_sub; ++sub) {
      mark(w, st);
      int rc = launch_collide(w, jenga::ModeStep, rest, st);
      if (rc != JENGA_OK) return rc;
      mark(w, st);
      const int flags = (sub == n_sub - 1 ? jenga::SolveEndOfStep : 0) | (rest ? jenga::SolveRest : 0);
      rc = launch_solve(w, w->P.iters, flags, rest_ek, st);
      if (rc != JENGA_OK) return rc;
      mark(w, st);
    }
  return JENGA_OK;
}

extern "C" int jenga_step(jenga_world* w, int n_steps, void* stream) {
  if (!w || n_steps < 0 || n_steps > (1 << 20)) return JENGA_E_ARG;
  return step_launches(w, n_steps, 0, 0.0f, (cudaStream_t)stream);
}

extern "C" int jenga_simulate_until_rest(jenga_world* w, int max_steps, float ek_rest, void* stream) {
  if (!w || max_steps <= 0 || max_steps > (1 << 20) || !(ek_rest > 0.0f)) return JENGA_E_ARG;
  const int dev_rc = on_device(w);
  if (dev_rc != JENGA_OK) return dev_rc;
  jenga::k_reset_rest<<<(w->P.E + 255) / 256, 256, 0, (cudaStream_t)stream>>>(w->P);
  const int rc = launched("k_reset_rest");
  if (rc != JENGA_OK) return rc;
  return step_launches(w, max_steps, 1, ek_rest, (cudaStream_t)stream);
}

extern "C" int jenga_step_host(jenga_world* w, const float* h_in, float* h_out, int n_steps, void* stream) {
  if (!w || n_steps < 0) return JENGA_E_ARG;
  const int dev_rc = on_device(w);
  if (dev_rc != JENGA_OK) return dev_rc;
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

extern "C" int jenga_support_margin(jenga_world* w, float* out, void* stream) {
  if (!w || !aligned16(out)) return JENGA_E_ARG;
  const int dev_rc = on_device(w);
  if (dev_rc != JENGA_OK) return dev_rc;
  const size_t smem = (size_t)8 * w->P.S * sizeof(float2);
  if (smem > 48 * 1024) {
    const cudaError_t e = ensure_smem(w->desc.device, KnSupport, smem);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(k_support)");
  }
  jenga::k_support<<<w->P.E, 32, smem, (cudaStream_t)stream>>>(w->P, reinterpret_cast<float4*>(out));
  return launched("k_support");
}

extern "C" int jenga_ziglar_block_analysis(jenga_world* w, const int32_t* block, const int32_t* axis, float* out, void* stream) {
  if (!w || !block || !axis || !aligned16(out)) return JENGA_E_ARG;
  const int dev_rc = on_device(w);
  if (dev_rc != JENGA_OK) return dev_rc;
  jenga::k_ziglar<<<(w->P.E + 127) / 128, 128, 0, (cudaStream_t)stream>>>(w->P, block, axis, reinterpret_cast<float4*>(out));
  return launched("k_ziglar");
}

// =================================================================== jenga_narrowphase_static: S3 with no caller scratch
// For callers that cannot hand the library device memory of their own to work in (include/jenga.h says who): the
// narrowphase as ONE kernel whose hand-off area is the array below, part of the library image on every device that
// loads it.  Nothing above this line is touched by it; it has its own per-device set-up and its own shared-memory bookkeeping.

/* The built-in hand-off area.  In HOST code this name is only a stand-in for the symbol -- its host address is not where the
 * array lives on the GPU -- so the host never passes it to a kernel: static_scratch_of() asks the runtime for the device
 * address once per device (cudaGetSymbolAddress, with that device current) and the launch passes that pointer.            */
static __device__ __align__(256) float g_static_scratch[JENGA_STATIC_SCRATCH_BYTES / sizeof(float)];

namespace jenga {

// Per-env region of the built-in area: only what the narrowphase hands from its first half to its second (the solver
// blocks, chunk list and colouring of the full layout are left out: 15.6 KB per 54-block env instead of 103 KB).
// Regions are multiples of 256 bytes; every array starts on a 16-byte boundary.
__host__ __device__ inline Scratch static_layout(int pc) {
  const int pcA = round_up(pc, 8);
  Scratch L; int p = 0;
  L.cs = L.ph = L.pos = L.col = L.wrk = L.ccnt = 0;      // not part of this layout, never addressed
  L.meta = p;  p += MetaWords;
  L.cpair = p; p += pcA / 2;
  L.coff = p;  p += pcA / 2;
  L.cab = p;   p += pcA;
  L.man = p;   p += 20 * pcA;
  L.total = round_up(p, 64);
  return L;
}

// One warp per env.  First half = k_detect<ModeNarrow> without the colouring hand-over: body records, the caller's candidate
// list, SAT -> colliding pairs (index, bodies, axis) into the env's region of the area.  Second half = k_manifold<ModeNarrow>:
// the records again in the manifold arena (it re-carves the same shared memory), the colliding list read back from the
// area, manifolds -> contacts / n_contacts in (pair, slot) order.  Same device functions, same order of arithmetic as the
// two kernels of jenga_narrowphase, so the contact list is the same bit for bit.  A warp reads back only what it wrote
// itself in this launch (ordered by __syncwarp), so the area's previous contents never matter.
// arena_words: shared-memory words per warp = the larger of the two arenas (the second must not reach into a neighbour's first).
__global__ void __launch_bounds__(128) k_narrow_static(const Params P, const int arena_words) {
  const int wpc = blockDim.x >> 5, warp = threadIdx.x >> 5, lane = lane_id();
  const int env = blockIdx.x * wpc + warp;
  if (env >= P.E) return;
  const Scratch L = static_layout(P.pc);
  float* scr = P.scratch + (size_t)env * P.scratch_words;
  int* meta = reinterpret_cast<int*>(scr + L.meta);
  unsigned st = 0;
  {
    const CSm s = carve_collide(P.S, P.max_pairs, P.pc, warp * arena_words, ArenaDetect, 1);
    load_predict(s, P, env, false);
    const int n_cand = load_candidates(s, P, env);
    const int n_coll = find_colliding(s, P, n_cand, &st);
    unsigned short* gpair = reinterpret_cast<unsigned short*>(scr + L.cpair);
    unsigned* gcab = reinterpret_cast<unsigned*>(scr + L.cab);
    for (int r = lane; r < n_coll; r += 32) { gcab[r] = s.cab[r]; gpair[r] = s.cpair[r]; }
    if (lane == 0) meta[MetaNcoll] = n_coll;
    __syncwarp();                                            // the lanes' global writes are visible to the warp from here on
  }
  {
    const CSm s = carve_collide(P.S, P.max_pairs, P.pc, warp * arena_words, ArenaManifold, 1);
    load_predict(s, P, env, false, false);
    const int n_coll = load_colliding(s, scr, L, false);
    manifold_pairs(s, P, env, scr, L, n_coll, true);
  }
  flush_status(P, env, st);
}

}  // namespace jenga

static size_t static_arena_bytes(const jenga_world_desc* d) {
  const size_t a = 4 * jenga::collide_smem_words(d->body_stride, d->max_pairs, d->max_contacts / 4, jenga::ArenaDetect, 1);
  const size_t b = 4 * jenga::collide_smem_words(d->body_stride, d->max_pairs, d->max_contacts / 4, jenga::ArenaManifold, 1);
  return a > b ? a : b;
}

/* the fields jenga_narrowphase_static reads (the rest of the descriptor is ignored) */
static bool static_desc_ok(const jenga_world_desc* d) {
  if (!d || d->struct_size != sizeof(jenga_world_desc)) return false;
  if (d->n_envs <= 0 || d->n_bodies <= 0 || d->n_bodies > 360) return false;
  if (d->body_stride < d->n_bodies || (d->body_stride & 3)) return false;
  if (d->max_pairs <= 0 || d->max_pairs > 65535) return false;
  if (d->max_contacts < 4 || (d->max_contacts & 3) || d->max_contacts > 65532) return false;
  if (d->device < 0 || d->device >= 64) return false;
  return static_arena_bytes(d) <= kSmemMax;
}

extern "C" size_t jenga_narrowphase_static_env_bytes(const jenga_world_desc* d) {
  return static_desc_ok(d) ? (size_t)jenga::static_layout(d->max_contacts / 4).total * sizeof(float) : 0;
}

/* Per-device set-up, done by the first call on that device and kept: the device address of g_static_scratch and the
 * shared-memory limit the kernel has been given there.  No allocation: two runtime queries and one attribute.          */
struct static_dev { float* ptr; size_t smem_max; bool ready; };
static static_dev g_static_dev[64];
static std::mutex g_static_mutex;

static int static_scratch_of(int device, size_t smem, float** out) {
  std::lock_guard<std::mutex> lock(g_static_mutex);
  static_dev& sd = g_static_dev[device];
  if (!sd.ready) {
    int major = 0;
    cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device);
    if (e != cudaSuccess) return cuda_fail(e, "cudaDeviceGetAttribute");
    if (major != 10) return JENGA_E_DEVICE;
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_static_scratch);          /* answers for the CURRENT device: the caller checked it is `device` */
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(g_static_scratch)");
    if (!p || (((uintptr_t)p) & 255u)) return cuda_fail(cudaErrorInvalidSymbol, "cudaGetSymbolAddress(g_static_scratch): unaligned");
    sd.ptr = (float*)p; sd.smem_max = 48 * 1024; sd.ready = true;
  }
  if (smem > sd.smem_max) {
    const cudaError_t e = cudaFuncSetAttribute((const void*)jenga::k_narrow_static, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(k_narrow_static)");
    sd.smem_max = smem;
  }
  *out = sd.ptr;
  return JENGA_OK;
}

extern "C" int jenga_narrowphase_static(const jenga_world_desc* d, const float* state, const float* props, const int32_t* pairs,
                                        const int32_t* n_pairs, float* contacts, int32_t* n_contacts, uint32_t* status, void* stream) {
  if (!static_desc_ok(d)) return JENGA_E_ARG;
  if (!aligned16(state) || !aligned16(props) || !aligned16(pairs) || !n_pairs || !aligned16(contacts) || !n_contacts || !status)
    return JENGA_E_ARG;
  const jenga::Scratch L = jenga::static_layout(d->max_contacts / 4);
  if ((unsigned long long)d->n_envs * (unsigned long long)L.total * sizeof(float) > JENGA_STATIC_SCRATCH_BYTES)
    return JENGA_E_STATIC_CAPACITY;                            /* beyond the built-in area: nothing is launched */
  int cur = -1;
  const cudaError_t e = cudaGetDevice(&cur);
  if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
  if (cur != d->device) return JENGA_E_DEVICE;                 /* the address below is the current device's copy of the array */
  const size_t arena = static_arena_bytes(d);
  const int wpc = 4 * arena <= kSmemMax ? 4 : (2 * arena <= kSmemMax ? 2 : 1);
  float* area = nullptr;
  const int rc = static_scratch_of(d->device, wpc * arena, &area);
  if (rc != JENGA_OK) return rc;
  Params P;
  memset(&P, 0, sizeof(P));                                    /* every pointer the narrowphase does not use stays NULL */
  P.E = d->n_envs; P.B = d->n_bodies; P.S = d->body_stride; P.G = 1;
  P.cp.edge_bias_rel = d->edge_bias_rel; P.cp.edge_bias_abs = d->edge_bias_abs; P.cp.par_eps = d->par_eps; P.cp.tie_eps = d->tie_eps;
  P.max_pairs = d->max_pairs; P.max_contacts = d->max_contacts; P.pc = d->max_contacts / 4;
  P.state = const_cast<float*>(state);                         /* read only here: load_predict(predict = false) */
  P.props = props; P.pairs = const_cast<int*>(pairs); P.n_pairs = const_cast<int*>(n_pairs);
  P.contacts = contacts; P.n_contacts = n_contacts; P.status = status;
  P.scratch = area; P.scratch_words = L.total;
  jenga::k_narrow_static<<<(P.E + wpc - 1) / wpc, 32 * wpc, wpc * arena, (cudaStream_t)stream>>>(P, (int)(arena / 4));
  return launched("k_narrow_static");
}
