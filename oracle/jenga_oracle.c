/* jenga_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, sequential fp64 CPU statement of the batched Jenga rigid-body step of
 * arxiv/paper_2606_28394 (§4, §6, §7), in the canonical order of SURVEY.md §8(c)
 * S0-S7 with the readings A1-A19 (listed again in DESIGN.md §3).  It is the parity
 * reference for the CUDA path and the timed `cpu_baseline`; only tests/, bench.py's
 * cpu_baseline / --impl reference legs and __graft_entry__.smoke() may call it.  It
 * shares no code, header, table or helper with paper_2606_28394_b200/csrc.
 *
 * Build: see oracle/build.py (gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC).
 * -ffp-contract=off matters: the CUDA broadphase re-evaluates near-threshold AABB tests
 * in fp64 with separately rounded mul/add and must reproduce these decisions exactly.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"):
 *   orc_inertia_box      P3  closed form vs brute-force volume integration
 *   predict/integrate    P1  free fall closed form; P2 constant-omega rotation (world frame)
 *   orc_broadphase       P4  definition (Eq. 10); symmetric, superset of SAT, Eq. 11 form
 *   orc_collide_boxes    P5  SAT classification vs brute-force vertex/edge-face test;
 *                        P6  manifold vs independent 2-D rectangle intersection
 *   orc_solve            P7  single contact closed form, active-set LCP enumeration,
 *                            in-colour permutation invariance, KE monotone
 *   whole step           P8  incline stick/slip, P9 Ziglar rigs, P10 resting tower drift
 *   substep details      Eq. 16 above the slop (rise = beta (delta - slop); inverse-mass split, once per pair),
 *                        Eq. 14 with e > 0 ((-e)^k v_n after k iterations), external torque (n h tau / I_xx about a
 *                        principal axis; R diag(1/I) R^T tau in general), gyroscopic = 1 (first-step closed form,
 *                        angular momentum conserved), KE never rising in a row update: tests/test_oracle_pins_r3.py
 *   PARITY UNPINNED by anything in the paper (fixed by SURVEY §8(c) / DESIGN.md only):
 *   the >4-point reduction rule, the face-preference and tie constants, the tangent-basis
 *   rule, the warm-start match rule, the load split in statically indeterminate stacks.
 *
 * Layout of every per-env array (doubles, AoS): x[B][3], q[B][4] = (w,x,y,z), v[B][3],
 * w[B][3], inv_m[B], inv_I[B][3] (body-frame diagonal), he[B][3] half extents, active[B].
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* Control experiment only (oracle/oracle32.py, DESIGN.md §6 "rollout agreement"): the SAME source, same order of
 * operations, with every floating-point variable, array and struct field in fp32 (build.py adds
 * -DORC_REAL_FLOAT -fsingle-precision-constant; sqrt / fabs / acos are still libm's double routines, rounded on
 * assignment).  It answers one question -- how often does a rollout of this method flip between fp64 and fp32 arithmetic,
 * and in which direction -- and is never a parity reference.  The fp64 build does not see this line. */
#ifdef ORC_REAL_FLOAT
#define double float
#endif

#define ORC_PAIR_OVERFLOW    1u
#define ORC_CONTACT_OVERFLOW 2u
#define ORC_COLOUR_OVERFLOW  4u
#define ORC_NONFINITE        8u
#define ORC_AXIS_GROUND 15

typedef struct {
  double dt;
  double g[3];
  double restitution;
  double aabb_margin;          /* Eq. 10 epsilon */
  double beta, slop;           /* Eq. 16     */
  double edge_bias_rel, edge_bias_abs, par_eps, tie_eps;   /* A7 readings                 */
  double match_tol;            /* warm-start point matching radius (A12)                  */
  int32_t n_substeps, pgs_iters, warm_start, gyroscopic;
  int32_t max_pairs;           /* candidate capacity per env                              */
  int32_t max_contacts;        /* contact capacity per env; colliding pairs <= max_contacts/4 */
} orc_params;

/* contact list of one env, ordered by (canonical pair index, slot) */
typedef struct {
  int32_t n;
  int32_t *pair;     /* canonical pair index: ground-body b -> b; i<j -> B + i(2B-i-1)/2 + (j-i-1) */
  int32_t *slot;     /* 0..3 */
  int32_t *axis;     /* SAT axis id 0..14, 15 = ground */
  double  *nrm;      /* [n][3]  A -> B */
  double  *pt;       /* [n][3]  world */
  double  *depth;    /* [n] */
} orc_contacts;

/* warm-start cache of one env: previous step's colliding pairs and impulses */
typedef struct {
  int32_t n_pairs;
  int32_t *key_pair;  /* [cap] canonical pair index, ascending */
  int32_t *key_meta;  /* [cap] axis<<8 | n_points */
  double  *lam;       /* [cap][4][3] jn jt1 jt2 per slot */
  double  *pt;        /* [cap][4][3] world contact points of the previous step */
} orc_cache;

/* decision margins: smallest distance of any discrete decision from its threshold */
typedef struct {
  double aabb;        /* min |slack| over all Eq. 10 tests                       */
  double sat_sign;    /* min |delta| over axes deciding overlap                  */
  double axis_choice; /* min gap between chosen axis and runner-up / bias line   */
  double incident;    /* min gap of the incident-face dot product                */
  double clip;        /* min |distance| of a vertex to a clip plane / depth 0    */
  double reduce;      /* min gap in the >4 reduction arg-max decisions           */
} orc_margins;

static void margins_init(orc_margins *m) {
  m->aabb = m->sat_sign = m->axis_choice = m->incident = m->clip = m->reduce = 1e300;
}
static void mmin(double *m, double v) { if (v < *m) *m = v; }

/* ------------------------------------------------------------------ vector helpers */
static double dot3(const double *a, const double *b) { return a[0]*b[0] + a[1]*b[1] + a[2]*b[2]; }
static void cross3(const double *a, const double *b, double *c) {
  double c0 = a[1]*b[2] - a[2]*b[1], c1 = a[2]*b[0] - a[0]*b[2], c2 = a[0]*b[1] - a[1]*b[0];
  c[0] = c0; c[1] = c1; c[2] = c2;
}
static void sym_mul(const double *M /*[9] row-major*/, const double *a, double *o) {
  double o0 = M[0]*a[0] + M[1]*a[1] + M[2]*a[2];
  double o1 = M[3]*a[0] + M[4]*a[1] + M[5]*a[2];
  double o2 = M[6]*a[0] + M[7]*a[1] + M[8]*a[2];
  o[0] = o0; o[1] = o1; o[2] = o2;
}

/* Eq. 1: R[3*r+c]; column c = body axis c in world coordinates. */
void orc_quat_to_R(const double *q, double *R) {
  double w = q[0], x = q[1], y = q[2], z = q[3];
  R[0] = 1.0 - 2.0*(y*y + z*z); R[1] = 2.0*(x*y - z*w);       R[2] = 2.0*(x*z + y*w);
  R[3] = 2.0*(x*y + z*w);       R[4] = 1.0 - 2.0*(x*x + z*z); R[5] = 2.0*(y*z - x*w);
  R[6] = 2.0*(x*z - y*w);       R[7] = 2.0*(y*z + x*w);       R[8] = 1.0 - 2.0*(x*x + y*y);
}

/* Eq. 3: I_body = m/12 diag(w^2+h^2, l^2+h^2, l^2+w^2). */
void orc_inertia_box(double m, double l, double w, double h, double *I) {
  I[0] = m / 12.0 * (w*w + h*h);
  I[1] = m / 12.0 * (l*l + h*h);
  I[2] = m / 12.0 * (l*l + w*w);
}

/* I_world^-1 = R diag(I_body^-1) R^T */
static void world_inv_inertia(const double *R, const double *invI, double *Iw) {
  for (int r = 0; r < 3; ++r)
    for (int c = 0; c < 3; ++c)
      Iw[3*r+c] = R[3*r+0]*invI[0]*R[3*c+0] + R[3*r+1]*invI[1]*R[3*c+1] + R[3*r+2]*invI[2]*R[3*c+2];
}

/* Eq. 8-9, Table 1: F = k mu_s m g */
double orc_ziglar_force(double k, double mu_s, double m, double g) { return k * mu_s * m * g; }

/* canonical pair index */
int32_t orc_pair_index(int32_t B, int32_t i, int32_t j) {
  if (i < 0) return j;
  return B + i*(2*B - i - 1)/2 + (j - i - 1);
}
void orc_pair_bodies(int32_t B, int32_t idx, int32_t *i, int32_t *j) {
  if (idx < B) { *i = -1; *j = idx; return; }
  int32_t r = idx - B, a = 0;
  while (r >= B - 1 - a) { r -= B - 1 - a; ++a; }
  *i = a; *j = a + 1 + r;
}

/* ------------------------------------------------------------------ S2 broadphase */
/* Eq. 10 on world AABBs c = x, e'_k = sum_j |R_kj| e_j (A6); ground
 * candidate iff c_z - e'_z <= eps.  Output ascending canonical pair indices.           */
int32_t orc_broadphase(const orc_params *P, int32_t B, const double *x, const double *q,
                       const double *he, const double *inv_m, const int32_t *active,
                       int32_t *pairs, uint32_t *status, orc_margins *mg) {
  double *ext = (double *)malloc(sizeof(double) * 3 * (size_t)B);
  int32_t n = 0;
  const double eps = P->aabb_margin;
  for (int b = 0; b < B; ++b) {
    double R[9]; orc_quat_to_R(q + 4*b, R);
    for (int k = 0; k < 3; ++k)
      ext[3*b+k] = fabs(R[3*k+0])*he[3*b+0] + fabs(R[3*k+1])*he[3*b+1] + fabs(R[3*k+2])*he[3*b+2];
  }
  for (int b = 0; b < B; ++b) {               /* ground pairs: index b */
    if (!active[b] || inv_m[b] == 0.0) continue;
    double slack = eps - (x[3*b+2] - ext[3*b+2]);
    if (mg) mmin(&mg->aabb, fabs(slack));
    if (slack >= 0.0) {
      if (n < P->max_pairs) pairs[n++] = b; else if (status) *status |= ORC_PAIR_OVERFLOW;
    }
  }
  for (int i = 0; i < B; ++i) {
    if (!active[i]) continue;
    for (int j = i + 1; j < B; ++j) {
      if (!active[j]) continue;
      if (inv_m[i] == 0.0 && inv_m[j] == 0.0) continue;
      double smin = 1e300;
      for (int k = 0; k < 3; ++k) {
        double slack = (ext[3*i+k] + ext[3*j+k] + eps) - fabs(x[3*i+k] - x[3*j+k]);
        if (slack < smin) smin = slack;
      }
      if (mg) mmin(&mg->aabb, fabs(smin));
      if (smin >= 0.0) {
        if (n < P->max_pairs) pairs[n++] = orc_pair_index(B, i, j);
        else if (status) *status |= ORC_PAIR_OVERFLOW;
      }
    }
  }
  free(ext);
  return n;
}

/* ------------------------------------------------------------------ S3 narrowphase */
/* Ground pair (A9): corners below z=0; n=(0,0,1); depth -z; p = (cx, cy, z/2); keep the 4
 * deepest (ties -> lower corner id), emitted in ascending corner id.  Returns point count. */
int32_t orc_collide_ground(const double *x, const double *q, const double *he,
                           double *pts /*[4][3]*/, double *depths /*[4]*/, orc_margins *mg) {
  double R[9]; orc_quat_to_R(q, R);
  double c[8][3]; int ok[8]; int nq = 0;
  for (int id = 0; id < 8; ++id) {
    double s[3] = { (id & 1) ? he[0] : -he[0], (id & 2) ? he[1] : -he[1], (id & 4) ? he[2] : -he[2] };
    for (int k = 0; k < 3; ++k) c[id][k] = x[k] + (R[3*k+0]*s[0] + R[3*k+1]*s[1] + R[3*k+2]*s[2]);
    ok[id] = c[id][2] < 0.0;
    if (mg) mmin(&mg->sat_sign, fabs(c[id][2]));
    nq += ok[id];
  }
  while (nq > 4) {                      /* drop the shallowest (ties -> higher corner id) */
    int worst = -1;
    for (int id = 0; id < 8; ++id)
      if (ok[id] && (worst < 0 || -c[id][2] <= -c[worst][2])) worst = id;
    if (mg) for (int id = 0; id < 8; ++id)
      if (ok[id] && id != worst) mmin(&mg->reduce, fabs(c[id][2] - c[worst][2]));
    ok[worst] = 0; --nq;
  }
  int n = 0;
  for (int id = 0; id < 8; ++id) if (ok[id]) {
    pts[3*n+0] = c[id][0]; pts[3*n+1] = c[id][1]; pts[3*n+2] = c[id][2] / 2.0;
    depths[n] = -c[id][2]; ++n;
  }
  return n;
}

/* Sutherland-Hodgman against one half-space  s*coord <= e  ("inside" = <=) */
static int clip_plane(const double (*in)[3], int nin, double (*out)[3],
                      const double *cX, const double *axis, double s, double e, orc_margins *mg) {
  int nout = 0;
  for (int i = 0; i < nin; ++i) {
    const double *Pv = in[i], *Qv = in[(i + 1) % nin];
    double rp[3] = { Pv[0]-cX[0], Pv[1]-cX[1], Pv[2]-cX[2] };
    double rq[3] = { Qv[0]-cX[0], Qv[1]-cX[1], Qv[2]-cX[2] };
    double dP = e - s * dot3(rp, axis), dQ = e - s * dot3(rq, axis);
    if (mg) mmin(&mg->clip, fabs(dP));
    if (dP >= 0.0) {
      out[nout][0] = Pv[0]; out[nout][1] = Pv[1]; out[nout][2] = Pv[2]; ++nout;
      if (dQ < 0.0) {
        double t = dP / (dP - dQ);
        for (int k = 0; k < 3; ++k) out[nout][k] = Pv[k] + (Qv[k] - Pv[k]) * t;
        ++nout;
      }
    } else if (dQ >= 0.0) {
      double t = dP / (dP - dQ);
      for (int k = 0; k < 3; ++k) out[nout][k] = Pv[k] + (Qv[k] - Pv[k]) * t;
      ++nout;
    }
  }
  return nout;
}

/* Box pair: 15-axis SAT + manifold (PAPER.md:275-280 read as A8).
 * Returns the number of contact points (0 = not colliding).  n points A -> B.          */
int32_t orc_collide_boxes(const orc_params *P,
                          const double *xA, const double *qA, const double *heA,
                          const double *xB, const double *qB, const double *heB,
                          int32_t *axis_out, double *n_out, double *sat_depth_out,
                          double *pts /*[4][3]*/, double *depths /*[4]*/, orc_margins *mg) {
  double RA[9], RB[9], a[3][3], b[3][3], t[3];
  orc_quat_to_R(qA, RA); orc_quat_to_R(qB, RB);
  for (int k = 0; k < 3; ++k) for (int r = 0; r < 3; ++r) { a[k][r] = RA[3*r+k]; b[k][r] = RB[3*r+k]; }
  for (int k = 0; k < 3; ++k) t[k] = xB[k] - xA[k];

  double delta[15], L[15][3]; int valid[15];
  for (int id = 0; id < 15; ++id) {
    double u[3]; valid[id] = 1;
    if (id < 3) { u[0] = a[id][0]; u[1] = a[id][1]; u[2] = a[id][2]; }
    else if (id < 6) { u[0] = b[id-3][0]; u[1] = b[id-3][1]; u[2] = b[id-3][2]; }
    else {
      cross3(a[(id-6)/3], b[(id-6)%3], u);
      double l2 = dot3(u, u);
      if (l2 < P->par_eps) { valid[id] = 0; delta[id] = 1e300; continue; }
      double l = sqrt(l2); u[0] /= l; u[1] /= l; u[2] /= l;
    }
    double rA = heA[0]*fabs(dot3(a[0], u)) + heA[1]*fabs(dot3(a[1], u)) + heA[2]*fabs(dot3(a[2], u));
    double rB = heB[0]*fabs(dot3(b[0], u)) + heB[1]*fabs(dot3(b[1], u)) + heB[2]*fabs(dot3(b[2], u));
    delta[id] = rA + rB - fabs(dot3(t, u));
    L[id][0] = u[0]; L[id][1] = u[1]; L[id][2] = u[2];
  }
  {
    int sep = 0; double mn = 1e300;
    for (int id = 0; id < 15; ++id) if (valid[id]) { if (delta[id] <= 0.0) sep = 1; if (fabs(delta[id]) < mn) mn = fabs(delta[id]); }
    if (sep) {                       /* margin of a "separated" verdict: the largest gap decides */
      double gap = 0.0;
      for (int id = 0; id < 15; ++id) if (valid[id] && -delta[id] > gap) gap = -delta[id];
      if (mg) mmin(&mg->sat_sign, gap);
      return 0;
    }
    if (mg) mmin(&mg->sat_sign, mn);
  }
  /* min-penetration axis with face preference (A7): candidate replaces best only if
   * smaller by more than tie_eps; edge wins only if dE < rel*dF - abs.                 */
  int bestF = 0, bestE = -1;
  for (int id = 1; id < 6; ++id) if (delta[id] < delta[bestF] - P->tie_eps) bestF = id;
  for (int id = 6; id < 15; ++id) if (valid[id]) {
    if (bestE < 0 || delta[id] < delta[bestE] - P->tie_eps) bestE = id;
  }
  int ax = bestF;
  if (bestE >= 0 && delta[bestE] < P->edge_bias_rel * delta[bestF] - P->edge_bias_abs) ax = bestE;
  if (mg) {
    for (int id = 0; id < 6; ++id) if (id != bestF)
      mmin(&mg->axis_choice, fabs(fabs(delta[id] - delta[bestF]) - P->tie_eps));
    for (int id = 6; id < 15; ++id) if (valid[id]) {
      if (id != bestE) mmin(&mg->axis_choice, fabs(fabs(delta[id] - delta[bestE]) - P->tie_eps));
      double l2; { double u[3]; cross3(a[(id-6)/3], b[(id-6)%3], u); l2 = dot3(u, u); }
      mmin(&mg->axis_choice, fabs(l2 - P->par_eps));
    }
    if (bestE >= 0)
      mmin(&mg->axis_choice, fabs(delta[bestE] - (P->edge_bias_rel * delta[bestF] - P->edge_bias_abs)));
  }
  double n[3] = { L[ax][0], L[ax][1], L[ax][2] };
  if (dot3(n, t) < 0.0) { n[0] = -n[0]; n[1] = -n[1]; n[2] = -n[2]; }
  *axis_out = ax; *sat_depth_out = delta[ax];
  n_out[0] = n[0]; n_out[1] = n[1]; n_out[2] = n[2];

  if (ax >= 6) {                      /* edge-edge: closest points of the two support edges */
    int i = (ax - 6) / 3, j = (ax - 6) % 3;
    double pa[3] = { xA[0], xA[1], xA[2] }, pb[3] = { xB[0], xB[1], xB[2] };
    for (int k = 0; k < 3; ++k) if (k != i) {
      double s = dot3(a[k], n) >= 0.0 ? 1.0 : -1.0;
      for (int r = 0; r < 3; ++r) pa[r] += s * heA[k] * a[k][r];
    }
    for (int k = 0; k < 3; ++k) if (k != j) {
      double s = dot3(b[k], n) >= 0.0 ? 1.0 : -1.0;
      for (int r = 0; r < 3; ++r) pb[r] -= s * heB[k] * b[k][r];
    }
    double r[3] = { pa[0]-pb[0], pa[1]-pb[1], pa[2]-pb[2] };
    double bb = dot3(a[i], b[j]), c = dot3(a[i], r), f = dot3(b[j], r), den = 1.0 - bb*bb;
    double sA = (bb*f - c) / den, sB = (f - bb*c) / den;
    if (sA > heA[i]) sA = heA[i]; if (sA < -heA[i]) sA = -heA[i];
    if (sB > heB[j]) sB = heB[j]; if (sB < -heB[j]) sB = -heB[j];
    for (int k = 0; k < 3; ++k) pts[k] = 0.5 * ((pa[k] + sA*a[i][k]) + (pb[k] + sB*b[j][k]));
    depths[0] = delta[ax];
    return 1;
  }

  /* face case: reference box X owns the axis, Y is the other box */
  const int refA = ax < 3, r = ax % 3;
  const double *cX = refA ? xA : xB, *cY = refA ? xB : xA;
  const double *eX = refA ? heA : heB, *eY = refA ? heB : heA;
  double (*xX)[3] = refA ? a : b, (*yY)[3] = refA ? b : a;
  double nref[3] = { refA ? n[0] : -n[0], refA ? n[1] : -n[1], refA ? n[2] : -n[2] };
  /* incident face: outward normal sigma*y_m with the smallest dot with nref;
   * ties -> lower axis, then the - face */
  int m = 0; double sg = -1.0, best = 1e300, second = 1e300;
  for (int k = 0; k < 3; ++k) for (int sgn = -1; sgn <= 1; sgn += 2) {
    double d = sgn * dot3(yY[k], nref);
    if (d < best) { second = best; best = d; m = k; sg = (double)sgn; }
    else if (d < second) second = d;
  }
  if (mg) mmin(&mg->incident, second - best);
  int iu = (m + 1) % 3, iv = (m + 2) % 3; if (iu > iv) { int tmp = iu; iu = iv; iv = tmp; }
  double poly[2][8][3]; int np = 4;
  static const double su[4] = { -1, 1, 1, -1 }, sv[4] = { -1, -1, 1, 1 };
  for (int k = 0; k < 4; ++k) for (int c = 0; c < 3; ++c)
    poly[0][k][c] = cY[c] + sg*eY[m]*yY[m][c] + su[k]*eY[iu]*yY[iu][c] + sv[k]*eY[iv]*yY[iv][c];
  double inc[4][3]; memcpy(inc, poly[0], sizeof(inc));
  int u = (r + 1) % 3, v = (r + 2) % 3; if (u > v) { int tmp = u; u = v; v = tmp; }
  np = clip_plane(poly[0], np, poly[1], cX, xX[u], +1.0, eX[u], mg);
  if (np) np = clip_plane(poly[1], np, poly[0], cX, xX[u], -1.0, eX[u], mg);
  if (np) np = clip_plane(poly[0], np, poly[1], cX, xX[v], +1.0, eX[v], mg);
  if (np) np = clip_plane(poly[1], np, poly[0], cX, xX[v], -1.0, eX[v], mg);
  double cp[8][3], cd[8]; int nc = 0;
  for (int k = 0; k < np; ++k) {
    double rq[3] = { poly[0][k][0]-cX[0], poly[0][k][1]-cX[1], poly[0][k][2]-cX[2] };
    double d = eX[r] - dot3(rq, nref);
    if (mg) mmin(&mg->clip, fabs(d));
    if (d >= 0.0) {
      for (int c = 0; c < 3; ++c) cp[nc][c] = poly[0][k][c] + nref[c] * (d / 2.0);
      cd[nc] = d; ++nc;
    }
  }
  if (nc == 0) {                       /* A8 fallback: deepest incident vertex, SAT depth */
    int bi = 0; double bd = -1e300;
    for (int k = 0; k < 4; ++k) {
      double rq[3] = { inc[k][0]-cX[0], inc[k][1]-cX[1], inc[k][2]-cX[2] };
      double d = eX[r] - dot3(rq, nref);
      if (d > bd) { bd = d; bi = k; }
    }
    for (int c = 0; c < 3; ++c) pts[c] = inc[bi][c] + nref[c] * (delta[ax] / 2.0);
    depths[0] = delta[ax];
    return 1;
  }
  int keep[8]; for (int k = 0; k < 8; ++k) keep[k] = (k < nc);
  if (nc > 4) {                        /* <=4 reduction */
    int i0 = 0, i1 = -1, i2 = -1, i3 = -1; double far = -1.0, amax = 0.0, amin = 0.0;
    for (int k = 1; k < nc; ++k) if (cd[k] > cd[i0]) i0 = k;
    for (int k = 0; k < nc; ++k) if (k != i0) {
      double d[3] = { cp[k][0]-cp[i0][0], cp[k][1]-cp[i0][1], cp[k][2]-cp[i0][2] };
      double dd = dot3(d, d);
      if (dd > far) { far = dd; i1 = k; }
    }
    double e01[3] = { cp[i1][0]-cp[i0][0], cp[i1][1]-cp[i0][1], cp[i1][2]-cp[i0][2] };
    double area[8];
    for (int k = 0; k < nc; ++k) {
      double d[3] = { cp[k][0]-cp[i0][0], cp[k][1]-cp[i0][1], cp[k][2]-cp[i0][2] }, cr[3];
      cross3(e01, d, cr); area[k] = dot3(cr, n);
      if (k == i0 || k == i1) continue;
      if (area[k] > amax) { amax = area[k]; i2 = k; }
      if (area[k] < amin) { amin = area[k]; i3 = k; }
    }
    if (mg) {
      for (int k = 0; k < nc; ++k) {
        if (k != i0) mmin(&mg->reduce, fabs(cd[k] - cd[i0]));
        if (k != i0 && k != i1) {
          double d[3] = { cp[k][0]-cp[i0][0], cp[k][1]-cp[i0][1], cp[k][2]-cp[i0][2] };
          mmin(&mg->reduce, fabs(dot3(d, d) - far));
          if (i2 >= 0 && k != i2) mmin(&mg->reduce, fabs(area[k] - amax));
          if (i3 >= 0 && k != i3) mmin(&mg->reduce, fabs(area[k] - amin));
        }
      }
    }
    for (int k = 0; k < nc; ++k) keep[k] = (k == i0 || k == i1 || k == i2 || k == i3);
  }
  int nout = 0;
  for (int k = 0; k < nc; ++k) if (keep[k]) {
    pts[3*nout+0] = cp[k][0]; pts[3*nout+1] = cp[k][1]; pts[3*nout+2] = cp[k][2];
    depths[nout] = cd[k]; ++nout;
  }
  return nout;
}

/* S3 over a candidate list -> contact list ordered (pair, slot). */
int32_t orc_narrowphase(const orc_params *P, int32_t B, const double *x, const double *q,
                        const double *he, const int32_t *pairs, int32_t n_pairs,
                        orc_contacts *C, uint32_t *status, orc_margins *mg) {
  int32_t ncoll = 0; C->n = 0;
  const int32_t pair_cap = P->max_contacts / 4;
  for (int32_t k = 0; k < n_pairs; ++k) {
    int32_t i, j; orc_pair_bodies(B, pairs[k], &i, &j);
    double pts[12], dep[4], n[3] = { 0.0, 0.0, 1.0 }, sd = 0.0; int32_t ax = ORC_AXIS_GROUND, np;
    if (i < 0) np = orc_collide_ground(x + 3*j, q + 4*j, he + 3*j, pts, dep, mg);
    else np = orc_collide_boxes(P, x + 3*i, q + 4*i, he + 3*i, x + 3*j, q + 4*j, he + 3*j,
                                &ax, n, &sd, pts, dep, mg);
    if (np == 0) continue;
    if (ncoll >= pair_cap) { if (status) *status |= ORC_CONTACT_OVERFLOW; continue; }
    ++ncoll;
    for (int s = 0; s < np; ++s) {
      int32_t c = C->n++;
      C->pair[c] = pairs[k]; C->slot[c] = s; C->axis[c] = ax;
      for (int r = 0; r < 3; ++r) { C->nrm[3*c+r] = n[r]; C->pt[3*c+r] = pts[3*s+r]; }
      C->depth[c] = dep[s];
    }
  }
  return C->n;
}

/* ------------------------------------------------------------------ S4 + S5 */
/* greedy colouring in ascending pair index over the colliding pairs (north_star (d)):
 * colour = lowest c not used by an earlier pair sharing a dynamic body.                */
int32_t orc_colour_pairs(int32_t B, const int32_t *pair_idx, int32_t n_pairs, const double *inv_m,
                         int32_t *colour, uint32_t *status) {
  uint64_t *used = (uint64_t *)calloc((size_t)B, sizeof(uint64_t));
  int32_t ncol = 0;
  for (int32_t k = 0; k < n_pairs; ++k) {
    int32_t i, j; orc_pair_bodies(B, pair_idx[k], &i, &j);
    uint64_t m = 0;
    if (i >= 0 && inv_m[i] != 0.0) m |= used[i];
    if (inv_m[j] != 0.0) m |= used[j];
    int32_t c = 0;
    while (c < 64 && ((m >> c) & 1ull)) ++c;
    if (c >= 64) { c = 63; if (status) *status |= ORC_COLOUR_OVERFLOW; }
    colour[k] = c;
    if (i >= 0) used[i] |= 1ull << c;
    used[j] |= 1ull << c;
    if (c + 1 > ncol) ncol = c + 1;
  }
  free(used);
  return ncol;
}

/* tangent basis (A10, reading R-basis): t1 = normalise(e_k - n (n.e_k)) with
 * k = x unless |n_x| > 1/sqrt(2), then k = y;  t2 = n x t1. */
static void tangent_basis(const double *n, double *t1, double *t2) {
  int k = (fabs(n[0]) > 0.70710678118654752) ? 1 : 0;
  double e[3] = { 0, 0, 0 }; e[k] = 1.0;
  double d = n[k];
  double u[3] = { e[0] - n[0]*d, e[1] - n[1]*d, e[2] - n[2]*d };
  double l = sqrt(dot3(u, u));
  t1[0] = u[0]/l; t1[1] = u[1]/l; t1[2] = u[2]/l;
  cross3(n, t1, t2);
}

typedef struct {
  int a, b;                  /* body ids, a = -1 for the ground */
  double d[3][3];            /* n, t1, t2 */
  double k[3];               /* Eq. 13 for each direction */
  double ra[3], rb[3];
  double lam[3];             /* accumulated jn, jt1, jt2 */
} row_t;

static void apply_impulse(const row_t *r, const double *Pimp, double *v, double *w,
                          const double *inv_m, const double *Iw) {
  double c[3], dw[3];
  if (r->a >= 0 && inv_m[r->a] != 0.0) {           /* a loses */
    for (int k = 0; k < 3; ++k) v[3*r->a+k] -= inv_m[r->a] * Pimp[k];
    cross3(r->ra, Pimp, c); sym_mul(Iw + 9*r->a, c, dw);
    for (int k = 0; k < 3; ++k) w[3*r->a+k] -= dw[k];
  }
  if (inv_m[r->b] != 0.0) {                        /* b gains */
    for (int k = 0; k < 3; ++k) v[3*r->b+k] += inv_m[r->b] * Pimp[k];
    cross3(r->rb, Pimp, c); sym_mul(Iw + 9*r->b, c, dw);
    for (int k = 0; k < 3; ++k) w[3*r->b+k] += dw[k];
  }
}

static double rel_vel(const row_t *r, const double *dir, const double *v, const double *w) {
  double vb[3], va[3] = { 0, 0, 0 }, c[3];
  cross3(w + 3*r->b, r->rb, c);
  for (int k = 0; k < 3; ++k) vb[k] = v[3*r->b+k] + c[k];
  if (r->a >= 0) { cross3(w + 3*r->a, r->ra, c); for (int k = 0; k < 3; ++k) va[k] = v[3*r->a+k] + c[k]; }
  double rel[3] = { vb[0]-va[0], vb[1]-va[1], vb[2]-va[2] };
  return dot3(rel, dir);
}

/* S4 (setup, warm start, colouring) + S5 (coloured PGS sweeps, Listing 1 PAPER.md:317-347,
 * Eq. 13-15) on a given contact list.  v, w are updated in place; lam_out[n][3] gets the
 * accumulated impulses in contact order; colour_out[n] the colour of each contact's pair.
 * Iw = world inverse inertia [B][9] of the step-start pose.  cache may be NULL.
 * perm (optional, [n_colliding_pairs]) overrides the within-colour visiting order for the
 * permutation-invariance pin: pairs are visited by (colour, perm rank).                 */
void orc_solve(const orc_params *P, int32_t B, const double *x, double *v, double *w,
               const double *inv_m, const double *Iw, double mu, const orc_contacts *C,
               const orc_cache *cache, int32_t iters, double *lam_out, int32_t *colour_out,
               const int32_t *perm, uint32_t *status) {
  const int32_t n = C->n;
  if (n == 0) return;
  row_t *rows = (row_t *)malloc(sizeof(row_t) * (size_t)n);
  int32_t *pfirst = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n + 1));
  int32_t *pidx = (int32_t *)malloc(sizeof(int32_t) * (size_t)n);
  int32_t np = 0;
  for (int32_t c = 0; c < n; ++c)
    if (c == 0 || C->pair[c] != C->pair[c-1]) { pfirst[np] = c; pidx[np] = C->pair[c]; ++np; }
  pfirst[np] = n;
  /* setup */
  for (int32_t c = 0; c < n; ++c) {
    row_t *r = &rows[c]; int32_t i, j; orc_pair_bodies(B, C->pair[c], &i, &j);
    r->a = i; r->b = j;
    for (int k = 0; k < 3; ++k) {
      r->d[0][k] = C->nrm[3*c+k];
      r->ra[k] = (i >= 0) ? C->pt[3*c+k] - x[3*i+k] : 0.0;
      r->rb[k] = C->pt[3*c+k] - x[3*j+k];
    }
    tangent_basis(r->d[0], r->d[1], r->d[2]);
    for (int dd = 0; dd < 3; ++dd) {            /* Eq. 13 */
      double k_ = inv_m[j], cr[3], Ic[3], cc[3];
      cross3(r->rb, r->d[dd], cr); sym_mul(Iw + 9*j, cr, Ic); cross3(Ic, r->rb, cc);
      double ang = dot3(r->d[dd], cc);
      if (i >= 0) {
        k_ += inv_m[i];
        cross3(r->ra, r->d[dd], cr); sym_mul(Iw + 9*i, cr, Ic); cross3(Ic, r->ra, cc);
        ang += dot3(r->d[dd], cc);
      }
      r->k[dd] = k_ + ang;
    }
    r->lam[0] = r->lam[1] = r->lam[2] = 0.0;
  }
  /* warm start (A12, reading R-warm): a new contact inherits (jn,jt1,jt2) of the
   * nearest not-yet-taken previous contact point of the same pair within match_tol;
   * slots ascending, lowest old slot on ties. */
  if (P->warm_start && cache) {
    const double tol2 = P->match_tol * P->match_tol;
    for (int32_t p = 0; p < np; ++p) {
      int32_t cnt = pfirst[p+1] - pfirst[p];
      for (int32_t k = 0; k < cache->n_pairs; ++k)
        if (cache->key_pair[k] == pidx[p]) {
          int32_t ocnt = cache->key_meta[k] & 0xff; int taken[4] = { 0, 0, 0, 0 };
          for (int s = 0; s < cnt; ++s) {
            int bo = -1; double bd = tol2;
            for (int o = 0; o < ocnt; ++o) if (!taken[o]) {
              double d[3]; for (int r_ = 0; r_ < 3; ++r_) d[r_] = C->pt[3*(pfirst[p]+s)+r_] - cache->pt[(4*k + o)*3 + r_];
              double dd = dot3(d, d);
              if (dd < bd) { bd = dd; bo = o; }
            }
            if (bo >= 0) {
              taken[bo] = 1;
              for (int dd = 0; dd < 3; ++dd) rows[pfirst[p]+s].lam[dd] = cache->lam[(4*k + bo)*3 + dd];
            }
          }
          break;
        }
    }
    for (int32_t c = 0; c < n; ++c) {
      row_t *r = &rows[c]; double Pimp[3];
      for (int k = 0; k < 3; ++k) Pimp[k] = r->lam[0]*r->d[0][k] + r->lam[1]*r->d[1][k] + r->lam[2]*r->d[2][k];
      apply_impulse(r, Pimp, v, w, inv_m, Iw);
    }
  }
  /* colouring + canonical order */
  int32_t *col = (int32_t *)malloc(sizeof(int32_t) * (size_t)np);
  int32_t ncol = orc_colour_pairs(B, pidx, np, inv_m, col, status);
  int32_t *order = (int32_t *)malloc(sizeof(int32_t) * (size_t)np);
  {
    int32_t o = 0;
    for (int32_t cc = 0; cc < ncol; ++cc) {
      int32_t start = o;
      for (int32_t p = 0; p < np; ++p) if (col[p] == cc) order[o++] = p;
      if (perm)                               /* test hook: reorder inside the colour */
        for (int32_t s1 = start; s1 < o; ++s1) for (int32_t s2 = s1 + 1; s2 < o; ++s2)
          if (perm[order[s2]] < perm[order[s1]]) { int32_t tmp = order[s1]; order[s1] = order[s2]; order[s2] = tmp; }
    }
  }
  const double e = P->restitution;
  for (int32_t it = 0; it < iters; ++it)
    for (int32_t o = 0; o < np; ++o) {
      int32_t p = order[o];
      for (int32_t c = pfirst[p]; c < pfirst[p+1]; ++c) {
        row_t *r = &rows[c]; double Pimp[3];
        /* normal row, Eq. 14 */
        double vn = rel_vel(r, r->d[0], v, w);
        double dj = -(1.0 + e) * vn / r->k[0];
        double nw = r->lam[0] + dj; if (nw < 0.0) nw = 0.0;
        for (int k = 0; k < 3; ++k) Pimp[k] = (nw - r->lam[0]) * r->d[0][k];
        apply_impulse(r, Pimp, v, w, inv_m, Iw); r->lam[0] = nw;
        /* friction rows, Eq. 15 (box: each tangent clipped to +-mu*jn) */
        for (int dd = 1; dd < 3; ++dd) {
          double vt = rel_vel(r, r->d[dd], v, w);
          double lim = mu * r->lam[0];
          double nj = r->lam[dd] - vt / r->k[dd];
          if (nj > lim) nj = lim; if (nj < -lim) nj = -lim;
          for (int k = 0; k < 3; ++k) Pimp[k] = (nj - r->lam[dd]) * r->d[dd][k];
          apply_impulse(r, Pimp, v, w, inv_m, Iw); r->lam[dd] = nj;
        }
      }
    }
  for (int32_t c = 0; c < n; ++c) for (int dd = 0; dd < 3; ++dd) lam_out[3*c+dd] = rows[c].lam[dd];
  if (colour_out)
    for (int32_t p = 0; p < np; ++p) for (int32_t c = pfirst[p]; c < pfirst[p+1]; ++c) colour_out[c] = col[p];
  free(rows); free(pfirst); free(pidx); free(col); free(order);
}

/* ------------------------------------------------------------------ one substep, one env */
typedef struct {          /* optional stage outputs of the LAST substep (all may be NULL) */
  int32_t *pairs; int32_t *n_pairs;
  orc_contacts *contacts;
  double *lam;            /* [n_contacts][3] */
  int32_t *colour;        /* [n_contacts] */
  double *v_pre;          /* [B][3] velocities after S1 (input of the solve) */
  double *w_pre;
  orc_margins *margins;
} orc_trace;

static void substep(const orc_params *P, double h, int32_t B, double *x, double *q, double *v, double *w,
                    const double *inv_m, const double *inv_I, const double *he, const int32_t *active,
                    double mu, const double *f_ext, orc_cache *cache, uint32_t *status, orc_trace *tr) {
  double *Iw = (double *)calloc((size_t)B * 9, sizeof(double));
  /* S1 predict (Eq. 5; A2: only g and f_ext carry h) */
  for (int b = 0; b < B; ++b) {
    if (!active[b] || inv_m[b] == 0.0) continue;
    double R[9]; orc_quat_to_R(q + 4*b, R);
    world_inv_inertia(R, inv_I + 3*b, Iw + 9*b);
    for (int k = 0; k < 3; ++k) {
      double f = f_ext ? f_ext[6*b+k] : 0.0;
      v[3*b+k] = v[3*b+k] + h * (P->g[k] + inv_m[b] * f);
    }
    double tau[3] = { f_ext ? f_ext[6*b+3] : 0.0, f_ext ? f_ext[6*b+4] : 0.0, f_ext ? f_ext[6*b+5] : 0.0 };
    if (P->gyroscopic) {                      /* A4: off by default */
      double Ib[3] = { 1.0/inv_I[3*b], 1.0/inv_I[3*b+1], 1.0/inv_I[3*b+2] }, Iwf[9], Lw[3], gy[3];
      world_inv_inertia(R, Ib, Iwf); sym_mul(Iwf, w + 3*b, Lw); cross3(w + 3*b, Lw, gy);
      for (int k = 0; k < 3; ++k) tau[k] -= gy[k];
    }
    double dw[3]; sym_mul(Iw + 9*b, tau, dw);
    for (int k = 0; k < 3; ++k) w[3*b+k] = w[3*b+k] + h * dw[k];
  }
  if (tr && tr->v_pre) { memcpy(tr->v_pre, v, sizeof(double)*3*(size_t)B); memcpy(tr->w_pre, w, sizeof(double)*3*(size_t)B); }
  /* S2, S3 */
  int32_t *pairs = (int32_t *)malloc(sizeof(int32_t) * (size_t)(P->max_pairs > 0 ? P->max_pairs : 1));
  int32_t npairs = orc_broadphase(P, B, x, q, he, inv_m, active, pairs, status, tr ? tr->margins : NULL);
  int32_t cap = P->max_contacts > 0 ? P->max_contacts : 1;
  orc_contacts C_local, *C = &C_local;
  C->pair = (int32_t *)malloc(sizeof(int32_t)*(size_t)cap); C->slot = (int32_t *)malloc(sizeof(int32_t)*(size_t)cap);
  C->axis = (int32_t *)malloc(sizeof(int32_t)*(size_t)cap); C->nrm = (double *)malloc(sizeof(double)*3*(size_t)cap);
  C->pt = (double *)malloc(sizeof(double)*3*(size_t)cap); C->depth = (double *)malloc(sizeof(double)*(size_t)cap);
  orc_narrowphase(P, B, x, q, he, pairs, npairs, C, status, tr ? tr->margins : NULL);
  /* S4, S5 */
  double *lam = (double *)calloc((size_t)cap * 3, sizeof(double));
  int32_t *colour = (int32_t *)calloc((size_t)cap, sizeof(int32_t));
  orc_solve(P, B, x, v, w, inv_m, Iw, mu, C, cache, P->pgs_iters, lam, colour, NULL, status);
  /* S6 integrate (Eq. 6; Eq. 2 PAPER.md:151 in the world-frame reading A3) */
  for (int b = 0; b < B; ++b) {
    if (!active[b] || inv_m[b] == 0.0) continue;
    for (int k = 0; k < 3; ++k) x[3*b+k] = x[3*b+k] + h * v[3*b+k];
    double qw = q[4*b], qx = q[4*b+1], qy = q[4*b+2], qz = q[4*b+3];
    double ox = w[3*b], oy = w[3*b+1], oz = w[3*b+2];
    /* [0,omega] (x) q, Hamilton product */
    double dw_ = -(ox*qx + oy*qy + oz*qz);
    double dx_ =  ox*qw + oy*qz - oz*qy;
    double dy_ =  oy*qw + oz*qx - ox*qz;
    double dz_ =  oz*qw + ox*qy - oy*qx;
    double nw = qw + 0.5*h*dw_, nx = qx + 0.5*h*dx_, ny = qy + 0.5*h*dy_, nz = qz + 0.5*h*dz_;
    double l = sqrt(nw*nw + nx*nx + ny*ny + nz*nz);
    q[4*b] = nw/l; q[4*b+1] = nx/l; q[4*b+2] = ny/l; q[4*b+3] = nz/l;
  }
  /* Eq. 16 (A14): once per colliding pair, delta = the pair's max depth */
  for (int32_t c = 0; c < C->n; ) {
    int32_t c1 = c; double dmax = C->depth[c];
    while (c1 < C->n && C->pair[c1] == C->pair[c]) { if (C->depth[c1] > dmax) dmax = C->depth[c1]; ++c1; }
    int32_t i, j; orc_pair_bodies(B, C->pair[c], &i, &j);
    double ima = (i >= 0) ? inv_m[i] : 0.0, imb = inv_m[j];
    double pen = dmax - P->slop; if (pen < 0.0) pen = 0.0;
    if (ima + imb > 0.0) {
      double s = P->beta * pen / (ima + imb);
      for (int k = 0; k < 3; ++k) {
        if (i >= 0) x[3*i+k] -= ima * s * C->nrm[3*c+k];
        x[3*j+k] += imb * s * C->nrm[3*c+k];
      }
    }
    c = c1;
  }
  /* S7 cache */
  if (cache) {
    int32_t np = 0;
    for (int32_t c = 0; c < C->n; ++c) {
      if (c == 0 || C->pair[c] != C->pair[c-1]) {
        cache->key_pair[np] = C->pair[c]; cache->key_meta[np] = C->axis[c] << 8;
        for (int k = 0; k < 12; ++k) cache->lam[12*np+k] = 0.0;
        ++np;
      }
      cache->key_meta[np-1] += 1;
      for (int dd = 0; dd < 3; ++dd) {
        cache->lam[(4*(np-1) + C->slot[c])*3 + dd] = lam[3*c+dd];
        cache->pt[(4*(np-1) + C->slot[c])*3 + dd] = C->pt[3*c+dd];
      }
    }
    cache->n_pairs = np;
  }
  for (int b = 0; b < B; ++b) if (active[b])
    for (int k = 0; k < 3; ++k) if (!isfinite(x[3*b+k]) || !isfinite(v[3*b+k])) *status |= ORC_NONFINITE;
  if (tr) {
    if (tr->pairs) { memcpy(tr->pairs, pairs, sizeof(int32_t)*(size_t)npairs); *tr->n_pairs = npairs; }
    if (tr->contacts) {
      orc_contacts *o = tr->contacts; o->n = C->n;
      memcpy(o->pair, C->pair, sizeof(int32_t)*(size_t)C->n); memcpy(o->slot, C->slot, sizeof(int32_t)*(size_t)C->n);
      memcpy(o->axis, C->axis, sizeof(int32_t)*(size_t)C->n); memcpy(o->nrm, C->nrm, sizeof(double)*3*(size_t)C->n);
      memcpy(o->pt, C->pt, sizeof(double)*3*(size_t)C->n); memcpy(o->depth, C->depth, sizeof(double)*(size_t)C->n);
    }
    if (tr->lam) memcpy(tr->lam, lam, sizeof(double)*3*(size_t)C->n);
    if (tr->colour) memcpy(tr->colour, colour, sizeof(int32_t)*(size_t)C->n);
  }
  free(Iw); free(pairs); free(C->pair); free(C->slot); free(C->axis); free(C->nrm); free(C->pt); free(C->depth);
  free(lam); free(colour);
}

/* One dt advance (n_substeps substeps, A5) of one env.  Returns the status bits. */
uint32_t orc_step_env(const orc_params *P, int32_t B, double *x, double *q, double *v, double *w,
                      const double *inv_m, const double *inv_I, const double *he, const int32_t *active,
                      double mu, const double *f_ext, orc_cache *cache, orc_trace *tr) {
  uint32_t status = 0;
  if (tr && tr->margins) margins_init(tr->margins);
  int ns = P->n_substeps > 0 ? P->n_substeps : 1;
  for (int s = 0; s < ns; ++s)
    substep(P, P->dt / ns, B, x, q, v, w, inv_m, inv_I, he, active, mu, f_ext, cache, &status, tr);
  return status;
}

/* world inverse inertia of every body, for stage tests of orc_solve */
void orc_world_inv_inertia(int32_t B, const double *q, const double *inv_I, double *Iw) {
  for (int b = 0; b < B; ++b) { double R[9]; orc_quat_to_R(q + 4*b, R); world_inv_inertia(R, inv_I + 3*b, Iw + 9*b); }
}

/* ------------------------------------------------------------------ NEXT-1: collapse latch */
/* Eq. 18 (A17): dx_max > 0.5 l  AND  E_k > 5e-5 J  AND  theta_max > 30 deg */
int32_t orc_collapse_test(int32_t B, const double *x, const double *q, const double *v, const double *w,
                          const double *x0, const double *q0, const double *inv_m, const double *inv_I,
                          const int32_t *active, double length, double *out3) {
  double dxm = 0.0, thm = 0.0, ek = 0.0;
  for (int b = 0; b < B; ++b) {
    if (!active[b] || inv_m[b] == 0.0) continue;
    double d[3] = { x[3*b]-x0[3*b], x[3*b+1]-x0[3*b+1], x[3*b+2]-x0[3*b+2] };
    double dx = sqrt(dot3(d, d)); if (dx > dxm) dxm = dx;
    double c = fabs(q[4*b]*q0[4*b] + q[4*b+1]*q0[4*b+1] + q[4*b+2]*q0[4*b+2] + q[4*b+3]*q0[4*b+3]);
    if (c > 1.0) c = 1.0;
    double th = 2.0 * acos(c); if (th > thm) thm = th;
    double R[9]; orc_quat_to_R(q + 4*b, R);
    double wb[3];                                   /* omega in the body frame: R^T w */
    for (int k = 0; k < 3; ++k) wb[k] = R[0+k]*w[3*b] + R[3+k]*w[3*b+1] + R[6+k]*w[3*b+2];
    ek += 0.5 / inv_m[b] * dot3(v + 3*b, v + 3*b)
        + 0.5 * (wb[0]*wb[0]/inv_I[3*b] + wb[1]*wb[1]/inv_I[3*b+1] + wb[2]*wb[2]/inv_I[3*b+2]);
  }
  if (out3) { out3[0] = dxm; out3[1] = ek; out3[2] = thm; }
  return dxm > 0.5 * length && ek > 5e-5 && thm > 30.0 * 3.14159265358979323846 / 180.0;
}

/* ------------------------------------------------------------------ NEXT-4: support polygon, Ziglar move classes */
/* Eq. 17 (§8.1): support polygon = convex hull of the (x, y) of all 8 corners of every body that rests
 * on the ground, i.e. whose world-AABB bottom z_b - e'_b,z <= eps (e' = |R| e as in Eq. 10, eps = the AABB margin);
 * COM_xy = mass-weighted mean over the active dynamic bodies; margin d = minimum signed distance from COM_xy to the
 * edges of the polygon (positive inside).  Returns d; *n_hull = number of hull vertices (0: nothing on the ground,
 * d = -1e30; 1 or 2: degenerate support, d = -(distance to the point / segment)).
 * The hull is Andrew's monotone chain (textbook): sort by (x, y), lower then upper chain, strictly convex turns. */
static int cmp_xy(const void *a, const void *b) {
  const double *p = (const double *)a, *q = (const double *)b;
  if (p[0] != q[0]) return p[0] < q[0] ? -1 : 1;
  if (p[1] != q[1]) return p[1] < q[1] ? -1 : 1;
  return 0;
}
static double cross2(const double *o, const double *a, const double *b) {
  return (a[0]-o[0])*(b[1]-o[1]) - (a[1]-o[1])*(b[0]-o[0]);
}
double orc_support_margin(int32_t B, const double *x, const double *q, const double *he, const double *inv_m,
                          const int32_t *active, double eps, double *com_xy, int32_t *n_hull) {
  double *pts = (double *)malloc(sizeof(double) * 2 * 8 * (size_t)(B > 0 ? B : 1));
  int n = 0; double msum = 0.0, cx = 0.0, cy = 0.0;
  for (int b = 0; b < B; ++b) {
    if (!active[b]) continue;
    double R[9]; orc_quat_to_R(q + 4*b, R);
    if (inv_m[b] > 0.0) { double m = 1.0 / inv_m[b]; msum += m; cx += m * x[3*b]; cy += m * x[3*b+1]; }
    double ez = fabs(R[6])*he[3*b] + fabs(R[7])*he[3*b+1] + fabs(R[8])*he[3*b+2];
    if (x[3*b+2] - ez > eps) continue;
    for (int id = 0; id < 8; ++id) {
      double s[3] = { (id & 1) ? he[3*b] : -he[3*b], (id & 2) ? he[3*b+1] : -he[3*b+1], (id & 4) ? he[3*b+2] : -he[3*b+2] };
      pts[2*n]   = x[3*b]   + R[0]*s[0] + R[1]*s[1] + R[2]*s[2];
      pts[2*n+1] = x[3*b+1] + R[3]*s[0] + R[4]*s[1] + R[5]*s[2];
      ++n;
    }
  }
  if (msum > 0.0) { cx /= msum; cy /= msum; }
  if (com_xy) { com_xy[0] = cx; com_xy[1] = cy; }
  if (n == 0) { if (n_hull) *n_hull = 0; free(pts); return -1e30; }
  qsort(pts, (size_t)n, 2 * sizeof(double), cmp_xy);
  double *h = (double *)malloc(sizeof(double) * 2 * (size_t)(2 * n + 2));
  int k = 0;
  for (int i = 0; i < n; ++i) {                                  /* lower chain */
    while (k >= 2 && cross2(h + 2*(k-2), h + 2*(k-1), pts + 2*i) <= 0.0) --k;
    h[2*k] = pts[2*i]; h[2*k+1] = pts[2*i+1]; ++k;
  }
  for (int i = n - 2, t = k + 1; i >= 0; --i) {                  /* upper chain */
    while (k >= t && cross2(h + 2*(k-2), h + 2*(k-1), pts + 2*i) <= 0.0) --k;
    h[2*k] = pts[2*i]; h[2*k+1] = pts[2*i+1]; ++k;
  }
  int nh = k > 1 ? k - 1 : k;                                    /* the last point repeats the first */
  double c[2] = { cx, cy }, d = 1e300;
  if (nh >= 3) {
    for (int i = 0; i < nh; ++i) {                               /* counter-clockwise: inside is to the left of every edge */
      const double *a = h + 2*i, *b2 = h + 2*((i + 1) % nh);
      double ex = b2[0]-a[0], ey = b2[1]-a[1], len = sqrt(ex*ex + ey*ey);
      double sd = cross2(a, b2, c) / len;
      if (sd < d) d = sd;
    }
  } else if (nh == 2) {
    double ex = h[2]-h[0], ey = h[3]-h[1], l2 = ex*ex + ey*ey;
    double t = ((cx-h[0])*ex + (cy-h[1])*ey) / l2; if (t < 0) t = 0; if (t > 1) t = 1;
    double px = h[0] + t*ex - cx, py = h[1] + t*ey - cy;
    d = -sqrt(px*px + py*py);
  } else {
    d = -sqrt((cx-h[0])*(cx-h[0]) + (cy-h[1])*(cy-h[1]));
  }
  if (n_hull) *n_hull = nh;
  free(pts); free(h);
  return d;
}

/* Table 1 (§5.4): the move classes of ziglar_block_analysis().  slot: 1 = centre block of its level,
 * 0 / 2 = side blocks; axis: 0 = along the block's length (the paper's Y), 1 = across it (the paper's X,
 * PAPER.md:216).  Class 0 center_xaxis (k = 3, no torque; the centre block has one row in the table, whatever the axis),
 * 1 side_yaxis (k = 3, no torque), 2 side_xaxis (k = 4, torque on the upper layer).  F_min = k mu_s m g (Eq. 8-9). */
int32_t orc_ziglar_block_analysis(int32_t slot, int32_t axis, double mu_s, double m, double g, double *f_min, int32_t *torque) {
  int32_t cls = slot == 1 ? 0 : (axis == 0 ? 1 : 2);
  double k = cls == 2 ? 4.0 : 3.0;
  if (f_min) *f_min = orc_ziglar_force(k, mu_s, m, g);
  if (torque) *torque = cls == 2;
  return cls;
}

/* ------------------------------------------------------------------ batch rollout */
/* E envs, arrays [E][...] contiguous; OpenMP over envs only (each env is sequential).
 * f_ext may be NULL; cache arrays are caller-owned and persist between calls:
 * key_pair/key_meta [E][pc], n_keys [E], lam and cpt [E][pc][4][3], pc = max_contacts/4.
 * collapsed (optional) [E] is OR-latched every step against x0/q0; ek_out (optional) [E]. */
void orc_rollout(const orc_params *P, int32_t E, int32_t B, int32_t n_steps,
                 double *x, double *q, double *v, double *w,
                 const double *inv_m, const double *inv_I, const double *he, const int32_t *active,
                 const double *mu, const double *f_ext,
                 int32_t *key_pair, int32_t *key_meta, int32_t *n_keys, double *lam, double *cpt,
                 uint32_t *status, const double *x0, const double *q0, double length,
                 int32_t *collapsed, int64_t *contact_count) {
  const int32_t pc = P->max_contacts / 4;
#pragma omp parallel for schedule(dynamic, 1)
  for (int32_t e = 0; e < E; ++e) {
    orc_cache cache = { n_keys[e], key_pair + (size_t)e*pc, key_meta + (size_t)e*pc, lam + (size_t)e*pc*12, cpt + (size_t)e*pc*12 };
    size_t o3 = (size_t)e*B*3, o4 = (size_t)e*B*4, o1 = (size_t)e*B, o6 = (size_t)e*B*6;
    int64_t cc = 0;
    for (int32_t s = 0; s < n_steps; ++s) {
      status[e] |= orc_step_env(P, B, x+o3, q+o4, v+o3, w+o3, inv_m+o1, inv_I+o3, he+o3, active+o1,
                                mu[e], f_ext ? f_ext+o6 : NULL, &cache, NULL);
      for (int32_t k = 0; k < cache.n_pairs; ++k) cc += cache.key_meta[k] & 0xff;
      if (collapsed)
        collapsed[e] |= orc_collapse_test(B, x+o3, q+o4, v+o3, w+o3, x0+o3, q0+o4, inv_m+o1, inv_I+o3,
                                          active+o1, length, NULL);
    }
    n_keys[e] = cache.n_pairs;
    if (contact_count) contact_count[e] += cc;
  }
}

/* simulate_until_rest (§8.3): advance env by env until the total kinetic energy
 * E_k = sum_b 1/2 m |v|^2 + 1/2 w . I w, evaluated after every step, falls below ek_rest, at most max_steps
 * steps (the paper: 400, 1e-7 J).  steps_out[e] = steps taken (>= 1).  Same arrays as orc_rollout. */
void orc_rollout_until_rest(const orc_params *P, int32_t E, int32_t B, int32_t max_steps, double ek_rest,
                            double *x, double *q, double *v, double *w,
                            const double *inv_m, const double *inv_I, const double *he, const int32_t *active,
                            const double *mu,
                            int32_t *key_pair, int32_t *key_meta, int32_t *n_keys, double *lam, double *cpt,
                            uint32_t *status, int32_t *steps_out, double *ek_out) {
  const int32_t pc = P->max_contacts / 4;
#pragma omp parallel for schedule(dynamic, 1)
  for (int32_t e = 0; e < E; ++e) {
    orc_cache cache = { n_keys[e], key_pair + (size_t)e*pc, key_meta + (size_t)e*pc, lam + (size_t)e*pc*12, cpt + (size_t)e*pc*12 };
    size_t o3 = (size_t)e*B*3, o4 = (size_t)e*B*4, o1 = (size_t)e*B;
    int32_t s = 0; double out3[3] = { 0, 0, 0 };
    while (s < max_steps) {
      status[e] |= orc_step_env(P, B, x+o3, q+o4, v+o3, w+o3, inv_m+o1, inv_I+o3, he+o3, active+o1,
                                mu[e], NULL, &cache, NULL);
      ++s;
      orc_collapse_test(B, x+o3, q+o4, v+o3, w+o3, x+o3, q+o4, inv_m+o1, inv_I+o3, active+o1, 1.0, out3);
      if (out3[1] < ek_rest) break;
    }
    n_keys[e] = cache.n_pairs;
    steps_out[e] = s; if (ek_out) ek_out[e] = out3[1];
  }
}

int32_t orc_max_threads(void) {
#ifdef _OPENMP
  extern int omp_get_max_threads(void);
  return omp_get_max_threads();
#else
  return 1;
#endif
}
