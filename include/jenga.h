/* jenga.h -- C-ABI of the B200-native batched Jenga rigid-body step.
 *
 * The operation is the time step of arxiv/paper_2606_28394 (§4 "Rigid-body dynamics",
 * §6 "Collision detection", §7 "Contact solver"), batched over independent tower episodes
 * ("envs"), in the canonical order fixed by SURVEY.md §8(c) S0-S7 / DESIGN.md §2:
 *
 *   S1 predict      v += h (g + f/m), w += h Iw^-1 tau              Eq. 4-5,
 *   S2 broadphase   world-AABB overlap with margin eps              Eq. 10-11
 *   S3 narrowphase  15-axis OBB SAT + face/edge manifold (<=4 pts)  §6.2,
 *   S4 setup        r_A, r_B, tangent basis, effective masses       Eq. 12-13
 *   S5 PGS          normal rows clamped >= 0, friction rows boxed   Eq. 14-15 + Listing 1
 *   S6 integrate    x += h v, q <- normalise(q + h/2 [0,w] q),      Eq. 2, 6, 16
 *                   Baumgarte position correction per colliding pair
 *
 * Everything below is plain C: POD structs, raw pointers, sizes.  All buffer pointers are
 * DEVICE pointers owned by the caller (the Python binding allocates them as torch tensors);
 * the library never allocates or frees device memory, never synchronises and never touches
 * the default stream: every call enqueues kernels on the `cuda_stream` it is given
 * (a cudaStream_t passed as void*) and returns.  Return value: 0 = OK, negative = error
 * (JENGA_E_*); data-dependent conditions (capacity overflow, non-finite state) are
 * reported per env in `status[]`, with deterministic truncation (lowest pair indices kept).
 *
 * Indices.  Bodies 0..n_bodies-1; the ground plane z = 0 is body -1 (static).
 * Canonical pair index: ground-body b -> b; bodies i<j -> B + i(2B-i-1)/2 + (j-i-1).
 * In a pair, A is the lower id (ground first), the normal points from A to B
 * (Listing 1: a loses the impulse, b gains it).
 */
#ifndef JENGA_H_
#define JENGA_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define JENGA_OK            0
#define JENGA_E_ARG        -1   /* bad argument: NULL / misaligned pointer, capacity out of range */
#define JENGA_E_CUDA       -2   /* CUDA error on launch; text via jenga_strerror(JENGA_E_CUDA) */
#define JENGA_E_DEVICE     -3   /* device is not sm_100 (the kernels are sm_100a only), or desc.device is not the current device */

/* status[env] bit flags */
#define JENGA_ST_PAIR_OVERFLOW    1u   /* more broadphase candidates than max_pairs          */
#define JENGA_ST_CONTACT_OVERFLOW 2u   /* more colliding pairs than max_contacts/4           */
#define JENGA_ST_COLOUR_OVERFLOW  4u   /* greedy colouring needed more than 64 colours       */
#define JENGA_ST_NONFINITE        8u   /* a position or velocity became inf/NaN              */

#define JENGA_AXIS_GROUND 15           /* SAT axis id of a ground contact; 0-2 = A's face axes,
                                          3-5 = B's, 6+3i+j = a_i x b_j  */

/* counters[] slots (uint64, accumulated with atomics by jenga_step) */
enum { JENGA_CNT_ENV_STEPS = 0, JENGA_CNT_BODY_STEPS, JENGA_CNT_CANDIDATES, JENGA_CNT_COLLIDING,
       JENGA_CNT_CONTACTS, JENGA_CNT_CONTACT_ITERS, JENGA_CNT_COLOURS, JENGA_CNT_GROUND_CONTACTS,
       JENGA_CNT_MAX_CANDIDATES, JENGA_CNT_MAX_COLLIDING, JENGA_CNT_MAX_COLOURS, JENGA_CNT_RESERVED, JENGA_N_COUNTERS };
/* CONTACTS counts every contact generated (ground ones included); GROUND_CONTACTS the ground-plane subset
 * (their PGS rows touch one body, so the roofline's work model counts them separately).
 * MAX_* are running maxima per env and substep (capacity sizing: max_pairs, max_contacts/4, 64 colours).  */

typedef struct jenga_world jenga_world;   /* opaque host-side handle; owns nothing on the device */

typedef struct {
  uint32_t struct_size;                 /* = sizeof(jenga_world_desc), checked                         */
  int32_t  n_envs, n_bodies;            /* E, B                                                        */
  int32_t  body_stride;                 /* S >= B, multiple of 4 (16-byte rows)                        */
  float    dt;                          /* 1/240                                        */
  int32_t  n_substeps;                  /* each substep = S1..S7 at h = dt/n_substeps   */
  int32_t  pgs_iters;                   /* PGS sweeps per substep (paper: 14)            */
  float    gravity[3];                  /* (0,0,-9.81)                                  */
  float    restitution;                 /* e of Eq. 14                                  */
  float    aabb_margin;                 /* eps of Eq. 10, 0.002                     */
  float    baumgarte_beta, slop;        /* Eq. 16: 0.35, 4e-4                           */
  float    edge_bias_rel, edge_bias_abs;/* face preference: edge axis iff dE < rel*dF - abs*/
  float    par_eps;                     /* cross axes with |a x b|^2 < par_eps are skipped             */
  float    tie_eps;                     /* an axis replaces the incumbent only if smaller by > tie_eps */
  float    match_tol;                   /* warm-start contact-point matching radius [m]    */
  int32_t  warm_start;                  /* 1: carry (jn,jt1,jt2) between steps                         */
  int32_t  gyroscopic;                  /* 1: add -h Iw^-1 (w x Iw w) in S1 (Eq. 4); default 0         */
  int32_t  max_pairs;                   /* candidate-pair capacity per env                             */
  int32_t  max_contacts;                /* contact capacity per env, a multiple of 4 in 4..65532; colliding pairs <=
                                           max_contacts/4.  Sizes whose per-env shared-memory arenas exceed 227 KB
                                           are rejected (jenga_scratch_bytes / jenga_smem_bytes return 0)       */
  int32_t  materialise;                 /* 1: jenga_step also writes pairs/contacts/lambda of its last
                                           substep (debug / parity); 0: they stay on chip              */
  int32_t  device;                      /* CUDA device ordinal the buffers live on                     */
  float    collapse_length;             /* block length l of Eq. 18; latch off if <= 0 */
  float    collapse_fd, collapse_ek, collapse_theta;   /* f_d = 0.5, eps_k = 5e-5 J, theta_th = 30 deg in rad   */
  int32_t  solver_tier;                 /* where the PGS kernel keeps the contact constants.  0 = auto: the most groups in
                                           flight per SM that fit, or, for a batch that does not fill 148 SMs, the tier
                                           with the fewest groups per SM that still holds the batch at once (<= 592 groups:
                                           tier 1).  1 = shared memory only (one warp per CTA).  Tensor memory, one CTA per
                                           SM owning its 512 columns: 5 = 16 groups in flight with 2 blocks of 32 pairs each
                                           in TMEM, 4 = 12 groups with 3 blocks, 2 = 8 groups with 4 blocks, 3 = 4 groups with
                                           9 blocks (further blocks are served from the L2-resident scratch).  Every tier
                                           computes the same bits.  A tier that does not fit the sizes is JENGA_E_ARG. */
  int32_t  env_group;                   /* envs per warp of the PGS kernel (a "group"): 1, 2, or 0 = auto (2 when
                                           n_envs >= 4736 = 2 x 16 x 148, so that the batch still fills every SM).  With 2,
                                           a solver visit takes pairs of the current colour of BOTH envs (they share no
                                           body), so the warp's 32 lanes are filled better; each env's Gauss-Seidel order,
                                           and so its result, is the canonical one bit for bit whatever the grouping.    */
} jenga_world_desc;

/* All DEVICE pointers, caller-owned, 16-byte aligned.  PC = max_contacts/4.
 * pairs, n_pairs, contacts, n_contacts and lambda (the "stage buffers") are only written by jenga_broadphase /
 * jenga_narrowphase / jenga_pgs_solve and, when desc.materialise = 1, by jenga_step.  A world that only steps with
 * materialise = 0 may pass all five as NULL (all or none; 36 KB per 54-block env): the three stage calls then return
 * JENGA_E_ARG on that handle.                                                                            */
typedef struct {
  float       *state;      /* [E][13][S]  px py pz qw qx qy qz vx vy vz wx wy wz  */
  const float *props;      /* [E][8][S]   inv_m invIx invIy invIz hx hy hz active(0/1); I_body diagonal,
                                          Eq. 3; h* = half extents along body x,y,z       */
  const float *mu;         /* [E]         static friction mu_s per env          */
  const float *f_ext;      /* [E][6][S]   world force(3) + torque(3) applied in every substep of the
                                          call; may be NULL                                            */
  int32_t     *pairs;      /* [E][max_pairs]  ascending canonical pair indices (S2 output)             */
  int32_t     *n_pairs;    /* [E]                                                                      */
  float       *contacts;   /* [E][max_contacts][8]: nx ny nz depth px py pz tag, ordered (pair, slot);
                              tag (int bits) = position of the pair in pairs[] (bits 0-15)
                              | slot 0..3 (bits 16-17) | SAT axis id 0..15 (bits 20-23)                */
  int32_t     *n_contacts; /* [E]                                                                      */
  float       *lambda;     /* [E][max_contacts][3]  jn jt1 jt2 in contact order (S5 output)            */
  int32_t     *cache_key;  /* [E][PC][2]  warm-start cache: canonical pair index, (axis<<8 | n_points) */
  float       *cache_lam;  /* [E][PC][4][3] accumulated impulses of the previous substep               */
  float       *cache_pt;   /* [E][PC][4][3] world contact points of the previous substep               */
  int32_t     *n_cache;    /* [E]  number of valid cache pairs (0 = cold)                              */
  uint32_t    *status;     /* [E]  JENGA_ST_* flags, OR-ed in                                          */
  unsigned long long *counters; /* [JENGA_N_COUNTERS], may be NULL                                     */
  /* Collapse latch (Eq. 18, reading A17), evaluated by jenga_step after every dt
   * advance; all three may be NULL (latch off).                                                        */
  const float *ref_pose;   /* [E][7][S]  px py pz qw qx qy qz of the reference (initial) pose           */
  int32_t     *collapsed;  /* [E]  OR-latched: 1 once dx_max > f_d l, theta_max > theta_th and E_k > eps_k
                                   held at the same step                                                */
  float       *collapse_stats; /* [E][4] of the last step: dx_max [m], E_k [J], theta_max [rad], 0     */
  int32_t     *rest_steps; /* [E]  steps taken by the last jenga_simulate_until_rest; may be NULL      */
  void        *scratch;    /* jenga_scratch_bytes(desc) bytes, 16-byte aligned, ZERO-FILLED by the caller before the
                              first call: the hand-off between the six kernels of a substep (solver constants,
                              pair headers and visit chunks of every group of envs) plus per-env bookkeeping (the
                              colouring of the last pair list, the rest flag).  Contents are private to the library. */
  size_t       scratch_bytes;
} jenga_buffers;

/* Validates desc/buffers (sizes, alignment, device arch) and returns a host handle.  desc.device must be the current
 * CUDA device here and in every later call on the handle (JENGA_E_DEVICE otherwise).                    */
int jenga_world_create(const jenga_world_desc *desc, const jenga_buffers *bufs, jenga_world **out);

/* S2 on the current poses: state, props -> pairs, n_pairs.  Eq. 10.
 * Decisions are bit-exact with an fp64 evaluation of Eq. 10 on the same fp32 inputs
 * (near-threshold tests are re-evaluated in fp64 on the device).                                      */
int jenga_broadphase(jenga_world *w, void *cuda_stream);

/* S3: state, props, pairs, n_pairs -> contacts, n_contacts.  PAPER.md:261-280.                        */
int jenga_narrowphase(jenga_world *w, void *cuda_stream);

/* S4+S5 on the velocities it is given (no predict): state(v,w), contacts, pairs [, cache] ->
 * state(v,w), lambda.  `iters` overrides desc.pgs_iters when > 0.  Uses the warm-start cache
 * (read only) when desc.warm_start = 1 and n_cache[env] > 0.  Eq. 13-15, Listing 1.                   */
int jenga_pgs_solve(jenga_world *w, int iters, void *cuda_stream);

/* n_steps advances of dt (each n_substeps substeps S1..S7 = six kernel launches: detection, colouring, visit plan, manifolds, contact setup,
 * solve + integrate), all enqueued by this one call; state, cache, status and counters are updated in place.  */
int jenga_step(jenga_world *w, int n_steps, void *cuda_stream);

/* simulate_until_rest (§8.3): every env advances dt by dt until its total kinetic energy
 * E_k = sum_b 1/2 m |v|^2 + 1/2 w . I w, evaluated after every step, is below ek_rest, at most max_steps steps
 * (the paper: 400 steps, 1e-7 J); bufs.rest_steps[env] = steps taken (>= 1).  The launches of max_steps steps are
 * enqueued at once; an env at rest is flagged on the device and its warp leaves every later launch at once, so it
 * stops costing arithmetic without a host round trip.  f_ext, the warm-start cache and the collapse latch behave
 * as in jenga_step; counters add the steps actually taken.                                                */
int jenga_simulate_until_rest(jenga_world *w, int max_steps, float ek_rest, void *cuda_stream);

/* Support-polygon margin of every env (Eq. 17, §8.1): the convex hull of the (x, y) of the 8 corners of
 * every active body resting on the ground (world-AABB bottom <= aabb_margin), the mass-weighted COM_xy of the active
 * dynamic bodies, and the minimum signed distance from COM_xy to the hull's edges (positive inside).
 * out: DEVICE [E][4] fp32, 16-byte aligned: margin [m], COM_x, COM_y, number of hull vertices.  Nothing on the ground:
 * margin = -1e30, 0 vertices; a single point or a segment: minus the distance to it.                    */
int jenga_support_margin(jenga_world *w, float *out, void *cuda_stream);

/* ziglar_block_analysis() (Table 1, §5.4; Eq. 8-9): class of the move "push body
 * block[env] along axis[env]" of every env.  axis 0 = along the block's length (the paper's Y axis),
 * 1 = across it (the paper's X axis); the block's slot follows the tower layout body id = 3 level + slot,
 * slot 1 = centre block.  block, axis: DEVICE int32 [E].  out: DEVICE [E][4] fp32, 16-byte aligned: class (0 center_xaxis,
 * 1 side_yaxis, 2 side_xaxis; -1 for an invalid body id), F_min = k mu_s m g [N], torque flag, k (3 or 4).       */
int jenga_ziglar_block_analysis(jenga_world *w, const int32_t *block, const int32_t *axis, float *out, void *cuda_stream);

/* jenga_step with HOST state buffers (the end-to-end call): enqueues, on `cuda_stream`, a host->device copy
 * of h_state_in ([E][13][S] fp32, same layout as bufs.state; pinned memory recommended, pageable works but
 * serialises) into bufs.state, the fused step, and a device->host copy of bufs.state into h_state_out.
 * Either host pointer may be NULL to skip that copy.  Asynchronous like every other call: the caller
 * synchronises the stream before reading h_state_out.  The warm-start cache stays on the device.        */
int jenga_step_host(jenga_world *w, const float *h_state_in, float *h_state_out, int n_steps, void *cuda_stream);

/* Replaces bufs.f_ext for subsequent calls (NULL = no external load); takes effect for launches
 * enqueued after it returns.  Used to switch a push on and off between jenga_step calls.            */
int jenga_set_f_ext(jenga_world *w, const float *f_ext);

/* Frees the host handle (nothing on the device belongs to it). */
int jenga_world_destroy(jenga_world *w);

/* Dynamic shared memory per CTA of the PGS kernel for this descriptor (0 if invalid). */
size_t jenga_smem_bytes(const jenga_world_desc *desc);

/* Threads per CTA of the PGS kernel (one warp per group of envs: 128 Q threads in the tensor-memory tiers, 32 else). */
int jenga_block_threads(const jenga_world_desc *desc);

/* Envs per warp of the PGS kernel that this descriptor gets (desc.env_group, or what auto chooses; 0 if invalid). */
int jenga_env_group(const jenga_world_desc *desc);

/* Size of jenga_buffers.scratch for this descriptor (0 if invalid). */
size_t jenga_scratch_bytes(const jenga_world_desc *desc);

/* S3 for callers that have no device memory to lend the library as scratch.  Who that is: a plug-in inside a host program
 * whose memory pool was carved up at start-up and is closed to further requests; a control loop that must not meet the
 * device-wide stall a cudaMalloc / cudaFree implies; a thread that is inside a region of its own where the CUDA allocator
 * may not be called at all.  Such a caller can still own state / props / pairs / contacts (they are its data), but it
 * cannot size, obtain and zero a jenga_buffers.scratch, so it cannot create a jenga_world.  This ONE call does without:
 * the same narrowphase as jenga_narrowphase (§6.2: 15-axis SAT, face / edge / ground manifolds of at
 * most 4 points), bit for bit, as a single kernel launch whose hand-off area is an array built into the library image.
 *
 *   desc  the fields n_envs, n_bodies, body_stride, max_pairs, max_contacts, edge_bias_rel, edge_bias_abs, par_eps,
 *         tie_eps and device are used (struct_size is checked); everything else is ignored.
 *   IN    state [E][13][S], props [E][8][S], pairs [E][max_pairs], n_pairs [E]     (layouts as in jenga_buffers)
 *   OUT   contacts [E][max_contacts][8], n_contacts [E]; status [E] gets JENGA_ST_CONTACT_OVERFLOW OR-ed in.
 *   All seven are DEVICE pointers owned by the caller; state, props, pairs and contacts 16-byte aligned.
 *
 * Limit.  The built-in array has JENGA_STATIC_SCRATCH_BYTES (8 MiB); an env takes jenga_narrowphase_static_env_bytes(desc)
 * of it (15,616 B at max_contacts = 704: up to 537 envs per call).  A larger batch is refused with JENGA_E_STATIC_CAPACITY
 * and nothing is launched: split it into several calls on the same stream (env ranges are independent).
 * Cost.  Every GPU on which a process uses libjenga.so carries these 8 MiB from the moment the library's device code is
 * loaded there until the process exits, whether this call is ever made or not.
 * No allocation: the call makes no cudaMalloc / cudaFree / cudaMallocAsync, no host allocation of its own, and calls no
 * library routine that allocates.  The FIRST call on each device looks up the array's device address
 * (cudaGetSymbolAddress) and raises the kernel's shared-memory limit; make that first call outside any stream capture.
 * Later calls only enqueue the kernel on `cuda_stream` and return (asynchronous like the other stage calls).
 * Sharing.  There is one array per device, shared by every call from every thread and stream, and it keeps what the last
 * call left in it.  The kernel reads back only words that the same launch wrote earlier, so nothing needs to start at zero
 * and nothing is cleared -- but two calls whose kernels may run at the same time on one device (different streams, or
 * different host threads with their own streams) overwrite each other's hand-off and produce garbage without any error.
 * Keep all calls of a device on one stream, or order them with events.                                                  */
#define JENGA_STATIC_SCRATCH_BYTES (8u << 20)
#define JENGA_E_STATIC_CAPACITY -4   /* jenga_narrowphase_static: n_envs x per-env bytes exceeds JENGA_STATIC_SCRATCH_BYTES */
int jenga_narrowphase_static(const jenga_world_desc *desc, const float *state, const float *props, const int32_t *pairs,
                             const int32_t *n_pairs, float *contacts, int32_t *n_contacts, uint32_t *status, void *cuda_stream);
/* Bytes of the built-in array that one env of this descriptor takes (0 if the descriptor is out of range). */
size_t jenga_narrowphase_static_env_bytes(const jenga_world_desc *desc);

const char *jenga_strerror(int code);

/* Measurement aid (bench.py's roofline): while enabled, every launch of jenga_step / jenga_simulate_until_rest is
 * bracketed by CUDA events on the caller's stream.  jenga_profile_read synchronises on them and returns, for the launches
 * since the last enable / read, the summed device time [ms] of out[0] = the detection, colouring and plan kernels (S1, S2, SAT; S4 order),
 * out[1] = the manifold kernel, out[2] = the contact-setup kernel (effective masses, warm-start lookup), out[3] = the
 * solve + integrate kernel; out[4] = number of substeps.  `out` is a HOST array of 5 doubles.               */
int jenga_profile_enable(jenga_world *w, int on);
int jenga_profile_read(jenga_world *w, double *out);

/* Measured roofline denominators of this device: two micro-benchmarks on all SMs,
 * out[0] = FP32 thread-instructions per second (dependent-free FFMA streams, FMA = 1 instruction),
 * out[1] = shared-memory bytes per second (conflict-free LDS.128 streams), out[2] = SM count,
 * out[3], out[4] = seconds of the two timed runs, out[5] = the FFMA rate with three register operands (out[0] has
 * one uniform-register operand), out[6] = the FFMA rate when all three source registers change from one instruction to the
 * next (no operand-reuse hits: the solver's shape), out[7] = FMAs per second of the packed form fma.rn.f32x2 (two FMAs per
 * instruction) under the same no-reuse pattern.  `out` is a HOST array of 8 doubles; `scratch` a DEVICE
 * buffer of jenga_peaks_scratch_bytes() bytes.  Unlike the step calls this one synchronises the stream.  */
int jenga_measure_peaks(double *out, void *scratch, void *cuda_stream);
size_t jenga_peaks_scratch_bytes(void);

#ifdef __cplusplus
}
#endif
#endif /* JENGA_H_ */
