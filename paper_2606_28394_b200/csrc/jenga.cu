// jenga.cu -- kernels and C-ABI of the batched Jenga step (include/jenga.h).  sm_100a only.
//
// One CTA per env.  jenga_step runs S1..S7 for n_steps*n_substeps substeps in ONE launch with
// the env's body tile resident in shared memory; the stage entry points run a single stage on
// the same device functions so that each stage can be compared with the oracle in isolation.
#include <cuda_runtime.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "solve.cuh"

namespace jenga {

__device__ __forceinline__ int block_excl_scan(int v, int* warp_tot, int* total) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
  if (lane == 31) warp_tot[wid] = inc;
  __syncthreads();
  int before = 0, tot = 0;
  for (int k = 0; k < nw; ++k) { const int c = warp_tot[k]; if (k < wid) before += c; tot += c; }
  __syncthreads();
  *total = tot;
  return before + inc - v;
}

struct EnvCtx { Smem s; int env; };

__device__ inline EnvCtx begin_env(const Params& P, float* smem_base) {
  EnvCtx c; c.env = blockIdx.x;
  c.s = carve(smem_base, P.S, P.max_pairs, P.pc);
  load_tile(c.s.st, P.state + (size_t)c.env * kStateRows * P.S, kStateRows * P.S);
  load_tile(c.s.pr, P.props + (size_t)c.env * kPropRows * P.S, kPropRows * P.S);
  for (int k = threadIdx.x; k < kMaxColours; k += blockDim.x) c.s.ccount[k] = 0;
  __syncthreads();
  return c;
}

__device__ inline void flush_status(const Params& P, int env, unsigned st) {
  if (st) atomicOr(P.status + env, st);
}

// contacts / lambda of the current substep in (pair, slot) order; s.wrank[r] = contact offset.
__device__ inline int contact_offsets(const Smem& s, int n_coll) {
  int np = 0;
  if ((int)threadIdx.x < n_coll)
    np = (reinterpret_cast<const int*>(s.rec + (size_t)threadIdx.x * kRecWords)[RecMeta] >> 8) & 0xff;
  int tot;
  const int off = block_excl_scan(np, s.scan, &tot);
  if ((int)threadIdx.x < n_coll) s.wrank[threadIdx.x] = off;
  __syncthreads();
  return tot;
}

__device__ inline void write_contacts(const Params& P, int env, const Smem& s, int n_coll, int n_cont) {
  if ((int)threadIdx.x < n_coll) {
    const float* rec = s.rec + (size_t)threadIdx.x * kRecWords;
    const int* ri = reinterpret_cast<const int*>(rec);
    const int np = (ri[RecMeta] >> 8) & 0xff, axis = ri[RecMeta] & 0xff, off = s.wrank[threadIdx.x];
    float4* out = reinterpret_cast<float4*>(P.contacts + ((size_t)env * P.max_contacts + off) * 8);
    for (int c = 0; c < np; ++c) {
      const int tag = (ri[RecCand] & 0xffff) | (c << 16) | (axis << 20);
      out[2 * c] = make_float4(rec[RecN], rec[RecN + 1], rec[RecN + 2], rec[RecPt + 4 * c + 3]);
      out[2 * c + 1] = make_float4(rec[RecPt + 4 * c], rec[RecPt + 4 * c + 1], rec[RecPt + 4 * c + 2], __int_as_float(tag));
    }
  }
  if (threadIdx.x == 0) P.n_contacts[env] = n_cont;
}

__device__ inline void write_lambda(const Params& P, int env, const Smem& s, const PairState& ps, bool have_pair) {
  if (have_pair) {
    float* out = P.lambda + ((size_t)env * P.max_contacts + s.wrank[ps.rank]) * 3;
#pragma unroll
    for (int c = 0; c < 4; ++c)
      if (c < ps.np) { out[3 * c] = ps.lam[c][0]; out[3 * c + 1] = ps.lam[c][1]; out[3 * c + 2] = ps.lam[c][2]; }
  }
}

__device__ inline void write_pairs(const Params& P, int env, const Smem& s, int n_cand) {
  int* out = P.pairs + (size_t)env * P.max_pairs;
  for (int k = threadIdx.x; k < n_cand; k += blockDim.x) out[k] = s.cand[k];
  if (threadIdx.x == 0) P.n_pairs[env] = n_cand;
}

// ---------------------------------------------------------------- fused step
template <int T, int MINB>
__global__ void __launch_bounds__(T, MINB) k_step(const Params P, const int n_steps) {
  extern __shared__ __align__(16) float smem_base[];
  EnvCtx cx = begin_env(P, smem_base);
  const Smem& s = cx.s; const int env = cx.env;
  const float mu = P.mu[env];
  unsigned st = 0;
  unsigned long long c_cand = 0, c_coll = 0, c_cont = 0, c_gcont = 0, c_col = 0;
  int n_active = 0;
  if (threadIdx.x == 0) for (int b = 0; b < P.B; ++b) n_active += body_dynamic(s, P.S, b) ? 1 : 0;
  const int n_sub = n_steps * P.n_substeps;
  for (int sub = 0; sub < n_sub; ++sub) {
    pose_derived(s, P.B, P.S);
    __syncthreads();
    predict_velocity(s, P, env);
    const int n_cand = broadphase(s, P, &st);
    const int n_coll = narrowphase(s, P, n_cand, &st);
    const int ncol = colour_pairs(s, P, n_coll, &st);
    const bool have = (int)threadIdx.x < n_coll;
    PairState ps; ps.np = 0; ps.colour = -1; ps.corr = 0.0f; ps.rank = 0; ps.a = -1; ps.b = 0;
    if (have) setup_pair(s, P, env, s.owner[threadIdx.x], ps);
    __syncthreads();
    pgs_sweeps(s, P, ps, have, ncol, P.iters, mu);
    int n_cont = 0;
    const bool last = sub == n_sub - 1;
    if (P.materialise && last) {
      n_cont = contact_offsets(s, n_coll);
      write_pairs(P, env, s, n_cand);
      write_contacts(P, env, s, n_coll, n_cont);
      write_lambda(P, env, s, ps, have);
    }
    integrate(s, P, ps, have, ncol, &st);
    store_cache(P, env, s, ps, have, n_coll);
    if (threadIdx.x == 0) { c_cand += n_cand; c_coll += n_coll; c_col += ncol; }
    c_cont += have ? ps.np : 0;
    c_gcont += (have && ps.a < 0) ? ps.np : 0;
    __syncthreads();
  }
  store_tile(P.state + (size_t)env * kStateRows * P.S, s.st, kStateRows * P.S);
  flush_status(P, env, st);
  if (P.counters) {
    // contacts: warp-reduce, one atomic per warp
    unsigned long long v = c_cont, vg = c_gcont;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { v += __shfl_down_sync(0xffffffffu, v, o); vg += __shfl_down_sync(0xffffffffu, vg, o); }
    if ((threadIdx.x & 31) == 0 && v) {
      atomicAdd(P.counters + JENGA_CNT_CONTACTS, v);
      atomicAdd(P.counters + JENGA_CNT_CONTACT_ITERS, v * (unsigned long long)P.iters);
      if (vg) atomicAdd(P.counters + JENGA_CNT_GROUND_CONTACTS, vg);
    }
    if (threadIdx.x == 0) {
      atomicAdd(P.counters + JENGA_CNT_ENV_STEPS, (unsigned long long)n_steps);
      atomicAdd(P.counters + JENGA_CNT_BODY_STEPS, (unsigned long long)n_steps * n_active);
      atomicAdd(P.counters + JENGA_CNT_CANDIDATES, c_cand);
      atomicAdd(P.counters + JENGA_CNT_COLLIDING, c_coll);
      atomicAdd(P.counters + JENGA_CNT_COLOURS, c_col);
    }
  }
}

// ---------------------------------------------------------------- stage kernels
template <int T, int MINB>
__global__ void __launch_bounds__(T, MINB) k_broadphase(const Params P) {
  extern __shared__ __align__(16) float smem_base[];
  EnvCtx cx = begin_env(P, smem_base);
  unsigned st = 0;
  pose_derived(cx.s, P.B, P.S);
  __syncthreads();
  const int n_cand = broadphase(cx.s, P, &st);
  write_pairs(P, cx.env, cx.s, n_cand);
  flush_status(P, cx.env, st);
}

template <int T, int MINB>
__global__ void __launch_bounds__(T, MINB) k_narrowphase(const Params P) {
  extern __shared__ __align__(16) float smem_base[];
  EnvCtx cx = begin_env(P, smem_base);
  const Smem& s = cx.s; const int env = cx.env;
  unsigned st = 0;
  pose_derived(s, P.B, P.S);
  int n_cand = P.n_pairs[env];
  if (n_cand > P.max_pairs) n_cand = P.max_pairs;
  if (n_cand < 0) n_cand = 0;
  for (int k = threadIdx.x; k < n_cand; k += blockDim.x) s.cand[k] = P.pairs[(size_t)env * P.max_pairs + k];
  __syncthreads();
  const int n_coll = narrowphase(s, P, n_cand, &st);
  const int n_cont = contact_offsets(s, n_coll);
  write_contacts(P, env, s, n_coll, n_cont);
  flush_status(P, env, st);
}

// Rebuild the per-pair records from a contact list in global memory (ordered (pair, slot); the
// contacts of one pair share the pair's normal, slot 0 carries it).
__device__ inline int records_from_contacts(const Params& P, int env, const Smem& s, unsigned* status) {
  int n_cont = P.n_contacts[env];
  if (n_cont > P.max_contacts) n_cont = P.max_contacts;
  if (n_cont < 0) n_cont = 0;
  const float4* in = reinterpret_cast<const float4*>(P.contacts + (size_t)env * P.max_contacts * 8);
  const int* pairs = P.pairs + (size_t)env * P.max_pairs;
  int n_coll = 0;
  for (int base = 0; base < n_cont; base += blockDim.x) {
    const int c = base + threadIdx.x;
    bool first = false; float4 a = make_float4(0, 0, 0, 0), b = a; int tag = 0;
    if (c < n_cont) { a = in[2 * c]; b = in[2 * c + 1]; tag = __float_as_int(b.w); first = ((tag >> 16) & 3) == 0; }
    int tot;
    const int excl = n_coll + block_rank(first, s.scan, &tot);
    if (c < n_cont) {
      const int r = first ? excl : excl - 1, slot = (tag >> 16) & 3;
      if (r >= 0 && r < P.pc) {
        float* rec = s.rec + (size_t)r * kRecWords; int* ri = reinterpret_cast<int*>(rec);
        rec[RecPt + 4 * slot] = b.x; rec[RecPt + 4 * slot + 1] = b.y; rec[RecPt + 4 * slot + 2] = b.z; rec[RecPt + 4 * slot + 3] = a.w;
        if (first) {
          const int cpos = tag & 0xffff, pidx = pairs[cpos];
          int i, j; pair_bodies(P.B, pidx, i, j);
          ri[RecPair] = pidx; ri[RecCand] = cpos; ri[RecA] = i; ri[RecB] = j;
          rec[RecN] = a.x; rec[RecN + 1] = a.y; rec[RecN + 2] = a.z;
        }
        bool lastc = c == n_cont - 1;
        if (!lastc) { const int t2 = __float_as_int(in[2 * (c + 1) + 1].w); lastc = ((t2 >> 16) & 3) == 0; }
        if (lastc) ri[RecMeta] = ((tag >> 20) & 0xf) | ((slot + 1) << 8);
      }
    }
    n_coll += tot;
  }
  if (n_coll > P.pc) { *status |= JENGA_ST_CONTACT_OVERFLOW; n_coll = P.pc; }
  __syncthreads();
  return n_coll;
}

template <int T, int MINB>
__global__ void __launch_bounds__(T, MINB) k_pgs(const Params P, const int iters) {
  extern __shared__ __align__(16) float smem_base[];
  EnvCtx cx = begin_env(P, smem_base);
  const Smem& s = cx.s; const int env = cx.env;
  unsigned st = 0;
  pose_derived(s, P.B, P.S);
  const int n_coll = records_from_contacts(P, env, s, &st);
  const int ncol = colour_pairs(s, P, n_coll, &st);
  const bool have = (int)threadIdx.x < n_coll;
  PairState ps; ps.np = 0; ps.colour = -1; ps.corr = 0.0f; ps.rank = 0; ps.a = -1; ps.b = 0;
  if (have) setup_pair(s, P, env, s.owner[threadIdx.x], ps);
  __syncthreads();
  pgs_sweeps(s, P, ps, have, ncol, iters, P.mu[env]);
  contact_offsets(s, n_coll);
  write_lambda(P, env, s, ps, have);
  store_tile(P.state + (size_t)env * kStateRows * P.S, s.st, kStateRows * P.S);
  flush_status(P, env, st);
}

}  // namespace jenga

// =================================================================== host side / C-ABI
using jenga::Params;

struct jenga_world {
  jenga_world_desc desc;
  jenga_buffers bufs;
  Params P;
  int threads;
  size_t smem;
};

static char g_err[512] = "no error";

static int pick_threads(int pc) {
  const int opts[] = { 64, 128, 192, 256, 384, 512 };
  for (int t : opts) if (pc <= t) return t;
  return 0;
}

static bool desc_ok(const jenga_world_desc* d) {
  if (!d || d->struct_size != sizeof(jenga_world_desc)) return false;
  if (d->n_envs <= 0 || d->n_bodies <= 0 || d->n_bodies > 1024) return false;
  if (d->body_stride < d->n_bodies || (d->body_stride & 3)) return false;
  if (d->n_substeps <= 0 || d->pgs_iters < 0 || !(d->dt > 0.0f)) return false;
  if (d->max_pairs <= 0 || d->max_pairs > 65535) return false;
  if (d->max_contacts < 4 || (d->max_contacts & 3)) return false;
  if (pick_threads(d->max_contacts / 4) == 0) return false;
  return true;
}

extern "C" size_t jenga_smem_bytes(const jenga_world_desc* d) {
  if (!desc_ok(d)) return 0;
  return 4 * jenga::smem_words(d->body_stride, d->max_pairs, d->max_contacts / 4);
}

extern "C" int jenga_block_threads(const jenga_world_desc* d) {
  if (!desc_ok(d)) return 0;
  return pick_threads(d->max_contacts / 4);
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

#define JENGA_DISPATCH(KERNEL, threads, smem, stream, grid, ...)                                                   \
  do {                                                                                                             \
    cudaError_t e_ = cudaSuccess;                                                                                  \
    switch (threads) {                                                                                             \
      case 64:  e_ = launch_one(jenga::KERNEL<64, 8>, 64, smem, stream, grid, __VA_ARGS__); break;                 \
      case 128: e_ = launch_one(jenga::KERNEL<128, 4>, 128, smem, stream, grid, __VA_ARGS__); break;               \
      case 192: e_ = launch_one(jenga::KERNEL<192, 3>, 192, smem, stream, grid, __VA_ARGS__); break;               \
      case 256: e_ = launch_one(jenga::KERNEL<256, 2>, 256, smem, stream, grid, __VA_ARGS__); break;               \
      case 384: e_ = launch_one(jenga::KERNEL<384, 1>, 384, smem, stream, grid, __VA_ARGS__); break;               \
      default:  e_ = launch_one(jenga::KERNEL<512, 1>, 512, smem, stream, grid, __VA_ARGS__); break;               \
    }                                                                                                              \
    if (e_ != cudaSuccess) return cuda_fail(e_, #KERNEL);                                                          \
  } while (0)

template <typename Kern, typename... Args>
static cudaError_t launch_one(Kern k, int threads, size_t smem, cudaStream_t stream, int grid, Args... args) {
  cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  k<<<grid, threads, smem, stream>>>(args...);
  return cudaGetLastError();
}

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
  w->desc = *d; w->bufs = *b; w->smem = smem; w->threads = pick_threads(d->max_contacts / 4);
  Params& P = w->P;
  P.E = d->n_envs; P.B = d->n_bodies; P.S = d->body_stride;
  P.h = d->dt / (float)d->n_substeps; P.n_substeps = d->n_substeps; P.iters = d->pgs_iters;
  for (int k = 0; k < 3; ++k) P.g[k] = d->gravity[k];
  P.restitution = d->restitution; P.aabb_margin = d->aabb_margin; P.beta = d->baumgarte_beta; P.slop = d->slop;
  P.cp.edge_bias_rel = d->edge_bias_rel; P.cp.edge_bias_abs = d->edge_bias_abs; P.cp.par_eps = d->par_eps; P.cp.tie_eps = d->tie_eps;
  P.match_tol = d->match_tol; P.warm_start = d->warm_start; P.gyroscopic = d->gyroscopic;
  P.max_pairs = d->max_pairs; P.max_contacts = d->max_contacts; P.pc = d->max_contacts / 4; P.materialise = d->materialise;
  P.state = b->state; P.props = b->props; P.mu = b->mu; P.f_ext = b->f_ext;
  P.pairs = b->pairs; P.n_pairs = b->n_pairs; P.contacts = b->contacts; P.n_contacts = b->n_contacts; P.lambda = b->lambda;
  P.cache_key = b->cache_key; P.cache_lam = b->cache_lam; P.cache_pt = b->cache_pt; P.n_cache = b->n_cache;
  P.status = b->status; P.counters = b->counters;
  *out = w;
  return JENGA_OK;
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
  JENGA_DISPATCH(k_broadphase, w->threads, w->smem, (cudaStream_t)stream, w->P.E, w->P);
  return JENGA_OK;
}

extern "C" int jenga_narrowphase(jenga_world* w, void* stream) {
  if (!w) return JENGA_E_ARG;
  JENGA_DISPATCH(k_narrowphase, w->threads, w->smem, (cudaStream_t)stream, w->P.E, w->P);
  return JENGA_OK;
}

extern "C" int jenga_pgs_solve(jenga_world* w, int iters, void* stream) {
  if (!w || iters < 0) return JENGA_E_ARG;
  const int it = iters > 0 ? iters : w->P.iters;
  JENGA_DISPATCH(k_pgs, w->threads, w->smem, (cudaStream_t)stream, w->P.E, w->P, it);
  return JENGA_OK;
}

extern "C" int jenga_step(jenga_world* w, int n_steps, void* stream) {
  if (!w || n_steps < 0) return JENGA_E_ARG;
  if (n_steps == 0) return JENGA_OK;
  JENGA_DISPATCH(k_step, w->threads, w->smem, (cudaStream_t)stream, w->P.E, w->P, n_steps);
  return JENGA_OK;
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
