/*
 * fp64 CPU ORACLE of the fixed-lag SE(2) SLAM backbone -- TEST INFRASTRUCTURE ONLY.
 * See slam_oracle.h for scope, variable order and pins.  Dense, slow, one environment at a time.
 * Nothing here is shared with (or derived from) the CUDA path.
 *
 * Citations: window of SE(2) poses + relative odometry factors PAPER.md:148; cost eq. (5)
 * PAPER.md:154-156; covariance eq. (6); sliding window / bounded memory
 * PAPER.md:144.  Where the paper is silent the readings R1-R23 apply.
 */
#include "slam_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

struct orc {
  int W, L, n, c, linear;
  int f32_storage; /* conditioning probe: round H, b, the prior and the state to fp32 (see slam_oracle.h) */
  double sig[11];
  double a[3];      /* global pose of the anchor (slot 0) */
  double* e;        /* [W][3] slot poses in the anchor frame, e[0] == 0 */
  double* m;        /* [L][2] landmarks g_l in GLOBAL coordinates (reading R17b) */
  int* active;      /* [L] */
  double *Lam, *g, *vbar; /* prior: 0.5 d'Lam d + g'd, d = v - vbar */
  double* z_odo;    /* [W][3]  z_odo[k]: slot k-1 -> k */
  int* lc_tgt;      /* [W]     target slot (< k) of the loop closure whose newer end is slot k; -1 none */
  double* z_lc;     /* [W][3] */
  int* rb_valid;    /* [W][L] */
  double* z_rb;     /* [W][L][2] range, bearing */
  int* un_valid;    /* [W]    unary absolute-pose factor on slot k (scan-match measurement) */
  double* z_un;     /* [W][3] measured global pose */
  double* om_un;    /* [W][9] its 3x3 information matrix (caller supplied, symmetric) */
};

/* ------------------------------------------------------------------ small helpers */

static double wrap_pi(double x) { return atan2(sin(x), cos(x)); }            /* R1: (-pi, pi] */
static double owrap(const orc* o, double x) { return o->linear ? x : wrap_pi(x); }

/* R3: p (+) u */
static void compose(int linear, const double* p, const double* u, double* out) {
  if (linear) { out[0] = p[0] + u[0]; out[1] = p[1] + u[1]; out[2] = p[2] + u[2]; return; }
  double c = cos(p[2]), s = sin(p[2]);
  out[0] = p[0] + c * u[0] - s * u[1];
  out[1] = p[1] + s * u[0] + c * u[1];
  out[2] = wrap_pi(p[2] + u[2]);
}

/* between(p,q): q in the frame of p */
static void between(int linear, const double* p, const double* q, double* out) {
  if (linear) { out[0] = q[0] - p[0]; out[1] = q[1] - p[1]; out[2] = q[2] - p[2]; return; }
  double c = cos(p[2]), s = sin(p[2]);
  double dx = q[0] - p[0], dy = q[1] - p[1];
  out[0] = c * dx + s * dy;
  out[1] = -s * dx + c * dy;
  out[2] = wrap_pi(q[2] - p[2]);
}

static int idx_e(int k) { return 3 * k; }                     /* k = 0 is the anchor a */
static int idx_m(const orc* o, int l) { return 3 * o->W + 2 * l; }

/* Solve A X = B (A n x n, B n x m, row-major) by Gaussian elimination with partial pivoting.
 * A and B are overwritten; X is returned in B.  Returns -1 if a pivot is 0 or non-finite. */
static int gauss_solve(double* A, double* B, int n, int m) {
  for (int k = 0; k < n; ++k) {
    int p = k;
    double best = fabs(A[k * n + k]);
    for (int i = k + 1; i < n; ++i)
      if (fabs(A[i * n + k]) > best) { best = fabs(A[i * n + k]); p = i; }
    if (!(best > 0.0) || !isfinite(best)) return -1;
    if (p != k) {
      for (int j = 0; j < n; ++j) { double t = A[k * n + j]; A[k * n + j] = A[p * n + j]; A[p * n + j] = t; }
      for (int j = 0; j < m; ++j) { double t = B[k * m + j]; B[k * m + j] = B[p * m + j]; B[p * m + j] = t; }
    }
    double inv = 1.0 / A[k * n + k];
    for (int i = k + 1; i < n; ++i) {
      double f = A[i * n + k] * inv;
      if (f == 0.0) continue;
      for (int j = k; j < n; ++j) A[i * n + j] -= f * A[k * n + j];
      for (int j = 0; j < m; ++j) B[i * m + j] -= f * B[k * m + j];
    }
  }
  for (int k = n - 1; k >= 0; --k) {
    double inv = 1.0 / A[k * n + k];
    for (int j = 0; j < m; ++j) {
      double s = B[k * m + j];
      for (int i = k + 1; i < n; ++i) s -= A[k * n + i] * B[i * m + j];
      B[k * m + j] = s * inv;
    }
  }
  return 0;
}

/* explicit inverse: Ainv = A^{-1} (A preserved) */
static int dense_inverse(const double* A, double* Ainv, int n) {
  double* T = (double*)malloc(sizeof(double) * n * n);
  memcpy(T, A, sizeof(double) * n * n);
  memset(Ainv, 0, sizeof(double) * n * n);
  for (int i = 0; i < n; ++i) Ainv[i * n + i] = 1.0;
  int rc = gauss_solve(T, Ainv, n, n);
  free(T);
  return rc;
}

/* ------------------------------------------------------------------ factors (A.2) */

/* Between factor from pose i to pose j (both in the anchor frame), measurement z = pose j in the
 * frame of pose i.  R2: r = [R_i'(t_j - t_i) - z_xy ; wrap(th_j - th_i - z_th)].
 * If i_is_frame, pose i is the anchor frame itself (identity, not a variable): no J_i block. */
static void between_factor(int linear, const double* ei, const double* ej, const double* z,
                           int i_is_frame, double* r, double* Ji, double* Jj) {
  memset(Ji, 0, 9 * sizeof(double));
  memset(Jj, 0, 9 * sizeof(double));
  if (linear) {
    for (int k = 0; k < 3; ++k) {
      r[k] = ej[k] - (i_is_frame ? 0.0 : ei[k]) - z[k];
      Jj[k * 3 + k] = 1.0;
      if (!i_is_frame) Ji[k * 3 + k] = -1.0;
    }
    return;
  }
  double zero[3] = {0, 0, 0};
  const double* p = i_is_frame ? zero : ei;
  double c = cos(p[2]), s = sin(p[2]);
  double dx = ej[0] - p[0], dy = ej[1] - p[1];
  double hx = c * dx + s * dy, hy = -s * dx + c * dy;
  r[0] = hx - z[0];
  r[1] = hy - z[1];
  r[2] = wrap_pi(ej[2] - p[2] - z[2]);
  Jj[0] = c;  Jj[1] = s;  Jj[2] = 0;
  Jj[3] = -s; Jj[4] = c;  Jj[5] = 0;
  Jj[6] = 0;  Jj[7] = 0;  Jj[8] = 1;
  if (!i_is_frame) {
    Ji[0] = -c; Ji[1] = -s; Ji[2] = hy;
    Ji[3] = s;  Ji[4] = -c; Ji[5] = -hx;
    Ji[6] = 0;  Ji[7] = 0;  Ji[8] = -1;
  }
}

/* Range-bearing factor from the pose in slot k to landmark l.  The landmark g is kept in GLOBAL
 * coordinates (reading R17b); the observing pose is x = a (+) e_k (x = a if k is the anchor slot).
 * R4: r = [ |g - t_x| - z_r ; wrap(atan2(dy,dx) - th_x - z_b) ].
 * Jacobians by the chain rule through x: Ja (2x3, wrt the anchor a), Jp (2x3, wrt e_k; zero if
 * k_is_frame), Jg (2x2, wrt the landmark). */
static void rb_factor(const double* a, const double* ek, const double* gl, const double* z, int k_is_frame,
                      double* r, double* Ja, double* Jp, double* Jg) {
  double zero[3] = {0, 0, 0};
  const double* e = k_is_frame ? zero : ek;
  double x[3];
  compose(0, a, e, x);
  double dx = gl[0] - x[0], dy = gl[1] - x[1];
  double q = dx * dx + dy * dy, rho = sqrt(q);
  r[0] = rho - z[0];
  r[1] = wrap_pi(atan2(dy, dx) - x[2] - z[1]);
  /* wrt the global observing pose x and the landmark */
  double Jx[6] = {-dx / rho, -dy / rho, 0, dy / q, -dx / q, -1};
  Jg[0] = dx / rho; Jg[1] = dy / rho;
  Jg[2] = -dy / q;  Jg[3] = dx / q;
  /* x = a (+) e:  dx/da = [[1,0,-d_y],[0,1,d_x],[0,0,1]], d = Rot(a_th) t_e;  dx/de = blockdiag(Rot(a_th),1) */
  double ca = cos(a[2]), sa = sin(a[2]);
  double ddx = ca * e[0] - sa * e[1], ddy = sa * e[0] + ca * e[1];
  double Xa[9] = {1, 0, -ddy, 0, 1, ddx, 0, 0, 1};
  double Xe[9] = {ca, -sa, 0, sa, ca, 0, 0, 0, 1};
  for (int i = 0; i < 2; ++i)
    for (int j = 0; j < 3; ++j) {
      double sa_ = 0.0, se_ = 0.0;
      for (int k = 0; k < 3; ++k) { sa_ += Jx[i * 3 + k] * Xa[k * 3 + j]; se_ += Jx[i * 3 + k] * Xe[k * 3 + j]; }
      Ja[i * 3 + j] = sa_;
      Jp[i * 3 + j] = k_is_frame ? 0.0 : se_;
    }
}

void orc_between_factor(const double* ei3, const double* ej3, const double* z3, int i_is_frame,
                        double* r3, double* Ji9, double* Jj9) {
  between_factor(0, ei3, ej3, z3, i_is_frame, r3, Ji9, Jj9);
}
void orc_rb_factor(const double* a3, const double* ek3, const double* gl2, const double* z2, int k_is_frame,
                   double* r2, double* Ja6, double* Jp6, double* Jg4) {
  rb_factor(a3, ek3, gl2, z2, k_is_frame, r2, Ja6, Jp6, Jg4);
}

/* Accumulate one factor with up to three variable blocks into the normal equations:
 *   H += J' Omega J,  grad += J' Omega r      (Omega diagonal, rdim rows)
 * block p: index idx[p] (skipped if < 0), width wid[p], Jacobian J[p] (rdim x wid[p], row-major). */
static void add_factor_n(double* H, double* grad, double* cost, int n, int rdim, const double* r,
                         const double* omega, int nblk, const int* idx, const int* wid, const double* const* J) {
  for (int p = 0; p < nblk; ++p) {
    if (idx[p] < 0) continue;
    for (int x = 0; x < wid[p]; ++x) {
      double s = 0.0;
      for (int k = 0; k < rdim; ++k) s += J[p][k * wid[p] + x] * omega[k] * r[k];
      if (grad) grad[idx[p] + x] += s;
      for (int q = 0; q < nblk; ++q) {
        if (idx[q] < 0) continue;
        for (int y = 0; y < wid[q]; ++y) {
          double h = 0.0;
          for (int k = 0; k < rdim; ++k) h += J[p][k * wid[p] + x] * omega[k] * J[q][k * wid[q] + y];
          if (H) H[(idx[p] + x) * n + idx[q] + y] += h;
        }
      }
    }
  }
  if (cost) for (int k = 0; k < rdim; ++k) *cost += 0.5 * r[k] * omega[k] * r[k];
}
static void add_factor(double* H, double* grad, double* cost, int n, int rdim, const double* r,
                       const double* omega, int ia, int wa, const double* JA, int ib, int wb,
                       const double* JB) {
  const int idx[2] = {ia, ib};
  const int wid[2] = {wa, wb};
  const double* J[2] = {JA, JB};
  add_factor_n(H, grad, cost, n, rdim, r, omega, 2, idx, wid, J);
}

/* ------------------------------------------------------------------ object */

orc* orc_create(int W, int L, const double* sig11, int linear) {
  if (W < 2 || L < 0 || (linear && L != 0)) return NULL;
  orc* o = (orc*)calloc(1, sizeof(orc));
  o->W = W; o->L = L; o->n = 3 * W + 2 * L; o->linear = linear;
  memcpy(o->sig, sig11, sizeof(double) * 11);
  int n = o->n;
  o->e = (double*)calloc(3 * W, sizeof(double));
  o->m = (double*)calloc(2 * (L + 1), sizeof(double));
  o->active = (int*)calloc(L + 1, sizeof(int));
  o->Lam = (double*)calloc((size_t)n * n, sizeof(double));
  o->g = (double*)calloc(n, sizeof(double));
  o->vbar = (double*)calloc(n, sizeof(double));
  o->z_odo = (double*)calloc(3 * W, sizeof(double));
  o->lc_tgt = (int*)calloc(W, sizeof(int));
  o->z_lc = (double*)calloc(3 * W, sizeof(double));
  o->rb_valid = (int*)calloc((size_t)W * (L + 1), sizeof(int));
  o->z_rb = (double*)calloc((size_t)W * (L + 1) * 2, sizeof(double));
  o->un_valid = (int*)calloc(W, sizeof(int));
  o->z_un = (double*)calloc(3 * W, sizeof(double));
  o->om_un = (double*)calloc(9 * W, sizeof(double));
  orc_reset(o, NULL);
  return o;
}

void orc_destroy(orc* o) {
  if (!o) return;
  free(o->e); free(o->m); free(o->active); free(o->Lam); free(o->g); free(o->vbar);
  free(o->z_odo); free(o->lc_tgt); free(o->z_lc); free(o->rb_valid); free(o->z_rb);
  free(o->un_valid); free(o->z_un); free(o->om_un);
  free(o);
}

int orc_count(const orc* o) { return o->c; }
int orc_dim(const orc* o) { return o->n; }

void orc_get_state(const orc* o, double* v) {
  memcpy(v, o->a, 3 * sizeof(double));
  memcpy(v + 3, o->e + 3, 3 * (o->W - 1) * sizeof(double));
  memcpy(v + 3 * o->W, o->m, 2 * o->L * sizeof(double));
}
void orc_set_state(orc* o, const double* v) {
  memcpy(o->a, v, 3 * sizeof(double));
  memcpy(o->e + 3, v + 3, 3 * (o->W - 1) * sizeof(double));
  memcpy(o->m, v + 3 * o->W, 2 * o->L * sizeof(double));
}
void orc_get_prior(const orc* o, double* Lam, double* g, double* vbar) {
  memcpy(Lam, o->Lam, sizeof(double) * o->n * o->n);
  memcpy(g, o->g, sizeof(double) * o->n);
  memcpy(vbar, o->vbar, sizeof(double) * o->n);
}

/* reset (R9): c = 1, anchor = init pose, prior Lambda = diag(1/sigma_p^2) on a, mean = the state */
void orc_reset(orc* o, const double* init_pose3) {
  int n = o->n;
  o->c = 1;
  for (int k = 0; k < 3; ++k) o->a[k] = init_pose3 ? init_pose3[k] : 0.0;
  memset(o->e, 0, 3 * o->W * sizeof(double));
  memset(o->m, 0, 2 * o->L * sizeof(double));
  memset(o->active, 0, o->L * sizeof(int));
  memset(o->Lam, 0, sizeof(double) * n * n);
  memset(o->g, 0, sizeof(double) * n);
  for (int k = 0; k < 3; ++k) o->Lam[k * n + k] = 1.0 / (o->sig[k] * o->sig[k]);
  for (int k = 0; k < o->W; ++k) o->lc_tgt[k] = -1;
  memset(o->rb_valid, 0, sizeof(int) * o->W * (o->L + 1));
  memset(o->un_valid, 0, sizeof(int) * o->W);
  orc_get_state(o, o->vbar);
}

static void record_rb(orc* o, int slot, const int* rb_valid, const double* rb_meas) {
  double p[3]; /* global pose of the observing slot, x = a (+) e_slot (e[0] == 0) */
  compose(0, o->a, o->e + 3 * slot, p);
  for (int l = 0; l < o->L; ++l) {
    int v = rb_valid ? (rb_valid[l] != 0) : 0;
    o->rb_valid[slot * o->L + l] = v;
    if (!v) continue;
    o->z_rb[(slot * o->L + l) * 2 + 0] = rb_meas[2 * l + 0];
    o->z_rb[(slot * o->L + l) * 2 + 1] = rb_meas[2 * l + 1];
    if (!o->active[l]) { /* R6: inverse projection from the observing pose's current estimate (global) */
      double r = rb_meas[2 * l], beta = rb_meas[2 * l + 1];
      o->m[2 * l + 0] = p[0] + r * cos(p[2] + beta);
      o->m[2 * l + 1] = p[1] + r * sin(p[2] + beta);
      o->active[l] = 1;
      o->vbar[idx_m(o, l)] = o->m[2 * l];
      o->vbar[idx_m(o, l) + 1] = o->m[2 * l + 1];
    }
  }
}

int orc_observe_first(orc* o, const int* rb_valid, const double* rb_meas) {
  if (o->c != 1) return -1;
  record_rb(o, 0, rb_valid, rb_meas);
  return 0;
}

/* Unary absolute-pose factor on the NEWEST pose (NEXT-1; the paper's scan-match measurement with a
 * caller-supplied information matrix).  x = a (+) e_k is the global pose of the slot:
 *   r = [ x - z_x ; y - z_y ; wrap(th - z_th) ],  J_a = dx/da,  J_e = dx/de_k  (as for range-bearing). */
int orc_add_unary(orc* o, const double* pose3, const double* info9) {
  int k = o->c - 1;
  o->un_valid[k] = 1;
  for (int i = 0; i < 3; ++i) o->z_un[3 * k + i] = pose3[i];
  for (int i = 0; i < 9; ++i) o->om_un[9 * k + i] = info9[i];
  return 0;
}

static void unary_factor(int linear, const double* a, const double* ek, const double* z, int k_is_frame,
                         double* r, double* Ja, double* Je) {
  double zero[3] = {0, 0, 0};
  const double* e = k_is_frame ? zero : ek;
  double x[3];
  compose(linear, a, e, x);
  r[0] = x[0] - z[0];
  r[1] = x[1] - z[1];
  r[2] = linear ? x[2] - z[2] : wrap_pi(x[2] - z[2]);
  memset(Ja, 0, 9 * sizeof(double));
  memset(Je, 0, 9 * sizeof(double));
  if (linear) {
    for (int i = 0; i < 3; ++i) { Ja[i * 3 + i] = 1.0; if (!k_is_frame) Je[i * 3 + i] = 1.0; }
    return;
  }
  double ca = cos(a[2]), sa = sin(a[2]);
  double ddx = ca * e[0] - sa * e[1], ddy = sa * e[0] + ca * e[1];
  Ja[0] = 1; Ja[2] = -ddy; Ja[4] = 1; Ja[5] = ddx; Ja[8] = 1;
  if (!k_is_frame) { Je[0] = ca; Je[1] = -sa; Je[3] = sa; Je[4] = ca; Je[8] = 1; }
}
void orc_unary_factor(const double* a3, const double* ek3, const double* z3, int k_is_frame,
                      double* r3, double* Ja9, double* Je9) {
  unary_factor(0, a3, ek3, z3, k_is_frame, r3, Ja9, Je9);
}

/* push: e_c = e_{c-1} (+) z_odo (dead-reckoned initial guess, BASELINE.json cfg 0) */
int orc_push(orc* o, const double* odom3, int lc_back, const double* lc_meas3,
             const int* rb_valid, const double* rb_meas) {
  int c = o->c;
  if (c >= o->W) return -1;
  compose(o->linear, o->e + 3 * (c - 1), odom3, o->e + 3 * c);
  for (int k = 0; k < 3; ++k) { o->z_odo[3 * c + k] = odom3[k]; o->vbar[idx_e(c) + k] = o->e[3 * c + k]; }
  o->lc_tgt[c] = -1;
  if (lc_back >= 1 && lc_back <= c) { /* R11: target = the pose lc_back steps older than the new one */
    o->lc_tgt[c] = c - lc_back;
    for (int k = 0; k < 3; ++k) o->z_lc[3 * c + k] = lc_meas3[k];
  }
  record_rb(o, c, rb_valid, rb_meas);
  o->un_valid[c] = 0;
  o->c = c + 1;
  return 0;
}

/* ------------------------------------------------------------------ normal equations (A.3) */

/* prior displacement d = v - vbar, theta components wrapped */
static void prior_d(const orc* o, double* d) {
  int n = o->n;
  double* v = (double*)malloc(sizeof(double) * n);
  orc_get_state(o, v);
  for (int i = 0; i < n; ++i) d[i] = v[i] - o->vbar[i];
  for (int k = 0; k < o->W; ++k) d[3 * k + 2] = owrap(o, d[3 * k + 2]);
  free(v);
}

/* H = Lam + sum J'Omega J, grad = (Lam d + g) + sum J'Omega r over the factors selected:
 * only_slot0 = 0: every live factor (GN system);  only_slot0 = 1: the factors touching slot 0
 * (the sub-problem that is folded into the prior by marginalization, A.5 step 1). */
static void build_system(const orc* o, int only_slot0, double* H, double* grad, double* cost) {
  int n = o->n, c = o->c, L = o->L;
  double om_odo[3], om_lc[3], om_rb[2];
  for (int k = 0; k < 3; ++k) {
    om_odo[k] = 1.0 / (o->sig[3 + k] * o->sig[3 + k]);
    om_lc[k] = 1.0 / (o->sig[6 + k] * o->sig[6 + k]);
  }
  om_rb[0] = 1.0 / (o->sig[9] * o->sig[9]);
  om_rb[1] = 1.0 / (o->sig[10] * o->sig[10]);

  double* d = (double*)malloc(sizeof(double) * n);
  prior_d(o, d);
  if (H) memcpy(H, o->Lam, sizeof(double) * n * n);
  for (int i = 0; i < n; ++i) {
    double s = o->g[i];
    for (int j = 0; j < n; ++j) s += o->Lam[i * n + j] * d[j];
    if (grad) grad[i] = s;
  }
  if (cost) {
    *cost = 0.0;
    for (int i = 0; i < n; ++i) {
      double s = 0.0;
      for (int j = 0; j < n; ++j) s += o->Lam[i * n + j] * d[j];
      *cost += 0.5 * d[i] * s + o->g[i] * d[i];
    }
  }
  free(d);

  double r[3], Ji[9], Jj[9], Ja[6], Jp[6], Jg[4];
  for (int k = 1; k < c; ++k) { /* odometry k-1 -> k */
    int i = k - 1;
    if (only_slot0 && i != 0) continue;
    between_factor(o->linear, o->e + 3 * i, o->e + 3 * k, o->z_odo + 3 * k, i == 0, r, Ji, Jj);
    add_factor(H, grad, cost, n, 3, r, om_odo, i == 0 ? -1 : idx_e(i), 3, Ji, idx_e(k), 3, Jj);
  }
  for (int k = 1; k < c; ++k) { /* loop closures lc_tgt[k] -> k */
    int i = o->lc_tgt[k];
    if (i < 0) continue;
    if (only_slot0 && i != 0) continue;
    between_factor(o->linear, o->e + 3 * i, o->e + 3 * k, o->z_lc + 3 * k, i == 0, r, Ji, Jj);
    add_factor(H, grad, cost, n, 3, r, om_lc, i == 0 ? -1 : idx_e(i), 3, Ji, idx_e(k), 3, Jj);
  }
  for (int k = 0; k < c; ++k) { /* unary absolute-pose factors: full 3x3 information */
    if (!o->un_valid[k]) continue;
    if (only_slot0 && k != 0) continue;
    double ru[3], Jua[9], Jue[9];
    unary_factor(o->linear, o->a, o->e + 3 * k, o->z_un + 3 * k, k == 0, ru, Jua, Jue);
    const double* Om = o->om_un + 9 * k;
    const int idx[2] = {0, k == 0 ? -1 : idx_e(k)};
    const double* J[2] = {Jua, Jue};
    double Or[3];
    for (int i = 0; i < 3; ++i) Or[i] = Om[i * 3] * ru[0] + Om[i * 3 + 1] * ru[1] + Om[i * 3 + 2] * ru[2];
    for (int p = 0; p < 2; ++p) {
      if (idx[p] < 0) continue;
      for (int x = 0; x < 3; ++x) {
        double sgrad = 0.0;
        for (int i = 0; i < 3; ++i) sgrad += J[p][i * 3 + x] * Or[i];
        if (grad) grad[idx[p] + x] += sgrad;
        for (int q = 0; q < 2; ++q) {
          if (idx[q] < 0) continue;
          for (int y = 0; y < 3; ++y) {
            double h = 0.0;
            for (int i = 0; i < 3; ++i)
              for (int j = 0; j < 3; ++j) h += J[p][i * 3 + x] * Om[i * 3 + j] * J[q][j * 3 + y];
            if (H) H[(idx[p] + x) * n + idx[q] + y] += h;
          }
        }
      }
    }
    if (cost) *cost += 0.5 * (ru[0] * Or[0] + ru[1] * Or[1] + ru[2] * Or[2]);
  }
  for (int k = 0; k < c; ++k) { /* range-bearing from slot k */
    if (only_slot0 && k != 0) continue;
    for (int l = 0; l < L; ++l) {
      if (!o->rb_valid[k * L + l]) continue;
      rb_factor(o->a, o->e + 3 * k, o->m + 2 * l, o->z_rb + (k * L + l) * 2, k == 0, r, Ja, Jp, Jg);
      const int idx[3] = {0, k == 0 ? -1 : idx_e(k), idx_m(o, l)};
      const int wid[3] = {3, 3, 2};
      const double* J[3] = {Ja, Jp, Jg};
      add_factor_n(H, grad, cost, n, 2, r, om_rb, 3, idx, wid, J);
    }
  }
}

/* identity rows/cols for unused pose slots (k >= c) and inactive landmarks, zero rhs (A.3) */
static void mask_unused(const orc* o, double* H, double* b) {
  int n = o->n;
  for (int i = 0; i < n; ++i) {
    int unused;
    if (i < 3 * o->W) unused = (i / 3) >= o->c;
    else unused = !o->active[(i - 3 * o->W) / 2];
    if (!unused) continue;
    for (int j = 0; j < n; ++j) { H[i * n + j] = 0.0; H[j * n + i] = 0.0; }
    H[i * n + i] = 1.0;
    if (b) b[i] = 0.0;
  }
}

void orc_set_f32_storage(orc* o, int on) { o->f32_storage = on; }

void orc_assemble(const orc* o, double* H, double* b) {
  int n = o->n;
  double* grad = (double*)malloc(sizeof(double) * n);
  build_system(o, 0, H, grad, NULL);
  for (int i = 0; i < n; ++i) grad[i] = -grad[i]; /* b = -(Lam d + g) - sum J'Omega r */
  mask_unused(o, H, grad);
  if (o->f32_storage) {
    for (int i = 0; i < n * n; ++i) H[i] = (double)(float)H[i];
    for (int i = 0; i < n; ++i) grad[i] = (double)(float)grad[i];
  }
  if (b) memcpy(b, grad, sizeof(double) * n);
  free(grad);
}

double orc_cost(const orc* o) {
  double cost = 0.0;
  build_system(o, 0, NULL, NULL, &cost);
  return cost;
}

/* solve (R12): exactly `iters` plain Gauss-Newton iterations, additive update, theta wrapped (R1) */
int orc_solve(orc* o, int iters, double* last_step_norm) {
  int n = o->n;
  double* H = (double*)malloc(sizeof(double) * n * n);
  double* b = (double*)malloc(sizeof(double) * n);
  double* v = (double*)malloc(sizeof(double) * n);
  int rc = 0;
  if (last_step_norm) *last_step_norm = 0.0;
  for (int it = 0; it < iters; ++it) {
    orc_assemble(o, H, b);
    if (gauss_solve(H, b, n, 1) != 0) { rc = -1; break; } /* b now holds delta */
    orc_get_state(o, v);
    double mx = 0.0;
    for (int i = 0; i < n; ++i) { v[i] += b[i]; if (fabs(b[i]) > mx) mx = fabs(b[i]); }
    for (int k = 0; k < o->W; ++k) v[3 * k + 2] = owrap(o, v[3 * k + 2]);
    if (o->f32_storage) for (int i = 0; i < n; ++i) v[i] = (double)(float)v[i];
    orc_set_state(o, v);
    if (last_step_norm) *last_step_norm = mx;
  }
  free(H); free(b); free(v);
  return rc;
}

/* cov (A.4, eq. (6), R13, R14): last 3x3 block of the inverse, in the newest pose's global coords */
int orc_cov(orc* o, double* cov9, double* logdet) {
  int n = o->n, c = o->c;
  double* H = (double*)malloc(sizeof(double) * n * n);
  double* P = (double*)malloc(sizeof(double) * n * n);
  orc_assemble(o, H, NULL);
  int rc = dense_inverse(H, P, n);
  double S[9];
  if (rc == 0) {
    if (c == 1) {
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) S[i * 3 + j] = P[i * n + j];
    } else {
      /* x = a (+) e, e = newest pose in the anchor frame:  J = [J_e | J_a] */
      int ie = idx_e(c - 1);
      int id[6] = {ie, ie + 1, ie + 2, 0, 1, 2};
      double S6[36], J[18];
      for (int i = 0; i < 6; ++i) for (int j = 0; j < 6; ++j) S6[i * 6 + j] = P[id[i] * n + id[j]];
      memset(J, 0, sizeof(J));
      if (o->linear) {
        for (int k = 0; k < 3; ++k) { J[k * 6 + k] = 1.0; J[k * 6 + 3 + k] = 1.0; }
      } else {
        double ca = cos(o->a[2]), sa = sin(o->a[2]);
        const double* e = o->e + 3 * (c - 1);
        double dx = ca * e[0] - sa * e[1], dy = sa * e[0] + ca * e[1];
        J[0 * 6 + 0] = ca; J[0 * 6 + 1] = -sa;
        J[1 * 6 + 0] = sa; J[1 * 6 + 1] = ca;
        J[2 * 6 + 2] = 1.0;
        J[0 * 6 + 3] = 1.0; J[0 * 6 + 5] = -dy;
        J[1 * 6 + 4] = 1.0; J[1 * 6 + 5] = dx;
        J[2 * 6 + 5] = 1.0;
      }
      for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
          double s = 0.0;
          for (int p = 0; p < 6; ++p) for (int q = 0; q < 6; ++q) s += J[i * 6 + p] * S6[p * 6 + q] * J[j * 6 + q];
          S[i * 3 + j] = s;
        }
    }
    for (int i = 0; i < 3; ++i) /* R20 */
      for (int j = i + 1; j < 3; ++j) { double t = 0.5 * (S[i * 3 + j] + S[j * 3 + i]); S[i * 3 + j] = t; S[j * 3 + i] = t; }
    double det = S[0] * (S[4] * S[8] - S[5] * S[7]) - S[1] * (S[3] * S[8] - S[5] * S[6]) +
                 S[2] * (S[3] * S[7] - S[4] * S[6]);
    if (cov9) memcpy(cov9, S, sizeof(S));
    if (logdet) *logdet = log(det); /* R15 */
  }
  free(H); free(P);
  return rc;
}

void orc_get_poses(const orc* o, double* poses) {
  memset(poses, 0, sizeof(double) * 3 * o->W);
  for (int k = 0; k < o->c; ++k) compose(o->linear, o->a, o->e + 3 * k, poses + 3 * k); /* R21 */
}

void orc_get_landmarks(const orc* o, double* lm, int* active) {
  for (int l = 0; l < o->L; ++l) {
    active[l] = o->active[l];
    lm[2 * l + 0] = o->active[l] ? o->m[2 * l] : 0.0;
    lm[2 * l + 1] = o->active[l] ? o->m[2 * l + 1] : 0.0;
  }
}

/* ------------------------------------------------------------------ marginalization (A.5) */

/* step 2: new coordinates u(v) = (a' = a (+) e_1, w = e_1, e'_k = between(e_1, e_k), g_l unchanged).
 * u is indexed like v: a' at 0, w where e_1 sits, e'_k where e_k sits, m'_l where m_l sits. */
void orc_reanchor_map(const orc* o, const double* v, double* u) {
  int W = o->W, L = o->L, c = o->c;
  memcpy(u, v, sizeof(double) * o->n);
  const double* a = v;
  const double* e1 = v + 3;
  compose(o->linear, a, e1, u);                   /* a' */
  for (int k = 2; k < c; ++k) between(o->linear, e1, v + 3 * k, u + 3 * k);
  (void)W; (void)L; /* landmarks are global: unchanged by re-anchoring */
}

/* step 3: M = du/dv at the current estimate (analytic; pinned by finite differences) */
void orc_reanchor_jac(const orc* o, double* M) {
  int n = o->n, W = o->W, L = o->L, c = o->c;
  memset(M, 0, sizeof(double) * n * n);
  for (int i = 0; i < n; ++i) M[i * n + i] = 1.0;
  const double* e1 = o->e + 3;
  if (o->linear) {
    for (int k = 0; k < 3; ++k) M[k * n + 3 + k] = 1.0;                 /* da'/de_1 = I */
    for (int j = 2; j < c; ++j)
      for (int k = 0; k < 3; ++k) M[(3 * j + k) * n + 3 + k] = -1.0;    /* de'_j/de_1 = -I */
    return;
  }
  double ca = cos(o->a[2]), sa = sin(o->a[2]);
  double dx = ca * e1[0] - sa * e1[1], dy = sa * e1[0] + ca * e1[1];   /* d = Rot(a_th) t_1 */
  /* da'/da */
  M[0 * n + 2] = -dy;
  M[1 * n + 2] = dx;
  /* da'/de_1 = blockdiag(Rot(a_th), 1) */
  M[0 * n + 3] = ca; M[0 * n + 4] = -sa;
  M[1 * n + 3] = sa; M[1 * n + 4] = ca;
  M[2 * n + 5] = 1.0;
  /* de'_k/de_1 = J_i(e_1, e_k), de'_k/de_k = J_j(e_1, e_k) */
  for (int k = 2; k < c; ++k) {
    double r[3], Ji[9], Jj[9], z[3] = {0, 0, 0};
    between_factor(0, e1, o->e + 3 * k, z, 0, r, Ji, Jj);
    for (int x = 0; x < 3; ++x)
      for (int y = 0; y < 3; ++y) {
        M[(3 * k + x) * n + 3 + y] = Ji[x * 3 + y];
        M[(3 * k + x) * n + 3 * k + y] = Jj[x * 3 + y];
      }
  }
  (void)W; (void)L; /* dg/dg = I */
}

int orc_marginalize(orc* o) {
  int n = o->n, W = o->W, L = o->L, c = o->c;
  if (c < 2) return -1;
  size_t nn = (size_t)n * n;
  double* Hs = (double*)malloc(sizeof(double) * nn);
  double* gs = (double*)malloc(sizeof(double) * n);
  double* M = (double*)malloc(sizeof(double) * nn);
  double* Nm = (double*)malloc(sizeof(double) * nn);
  double* T = (double*)malloc(sizeof(double) * nn);
  double* Hu = (double*)malloc(sizeof(double) * nn);
  double* gu = (double*)malloc(sizeof(double) * n);
  int rc = 0;

  /* 1. sub-problem: old prior + factors touching slot 0, at the current estimate (R18) */
  build_system(o, 1, Hs, gs, NULL);
  /* 3. N = M^{-1} */
  orc_reanchor_jac(o, M);
  rc = dense_inverse(M, Nm, n);
  /* 4. congruence H_u = N' H_s N, gamma_u = N' gamma_s */
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) {
      double s = 0.0;
      for (int k = 0; k < n; ++k) s += Hs[i * n + k] * Nm[k * n + j];
      T[i * n + j] = s;
    }
  for (int i = 0; i < n; ++i) {
    for (int j = 0; j < n; ++j) {
      double s = 0.0;
      for (int k = 0; k < n; ++k) s += Nm[k * n + i] * T[k * n + j];
      Hu[i * n + j] = s;
    }
    double s = 0.0;
    for (int k = 0; k < n; ++k) s += Nm[k * n + i] * gs[k];
    gu[i] = s;
  }
  /* 5. Schur complement over w (indices 3..5) */
  double Hww[9];
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) Hww[i * 3 + j] = Hu[(3 + i) * n + 3 + j];
  double Hww_inv[9];
  if (dense_inverse(Hww, Hww_inv, 3) != 0) rc = -1;
  double* Lp = (double*)calloc(nn, sizeof(double));
  double* gp = (double*)calloc(n, sizeof(double));
  for (int r = 0; r < n; ++r) {
    if (r >= 3 && r < 6) continue;
    double row[3]; /* H_rw Hww^{-1} */
    for (int j = 0; j < 3; ++j) {
      double s = 0.0;
      for (int k = 0; k < 3; ++k) s += Hu[r * n + 3 + k] * Hww_inv[k * 3 + j];
      row[j] = s;
    }
    for (int s2 = 0; s2 < n; ++s2) {
      if (s2 >= 3 && s2 < 6) continue;
      double s = Hu[r * n + s2];
      for (int k = 0; k < 3; ++k) s -= row[k] * Hu[(3 + k) * n + s2];
      Lp[r * n + s2] = s;
    }
    double s = gu[r];
    for (int k = 0; k < 3; ++k) s -= row[k] * gu[3 + k];
    gp[r] = s;
  }
  /* 7. re-index to the new slot layout: a' stays, e'_k (old 3k) -> 3(k-1) for k >= 2, landmarks stay */
  int* newidx = (int*)malloc(sizeof(int) * n);
  for (int i = 0; i < n; ++i) {
    if (i < 3) newidx[i] = i;
    else if (i < 6) newidx[i] = -1;
    else if (i < 3 * W) newidx[i] = i - 3;
    else newidx[i] = i;
  }
  memset(o->Lam, 0, sizeof(double) * nn);
  memset(o->g, 0, sizeof(double) * n);
  for (int i = 0; i < n; ++i) {
    if (newidx[i] < 0) continue;
    o->g[newidx[i]] = gp[i];
    for (int j = 0; j < n; ++j) {
      if (newidx[j] < 0) continue;
      o->Lam[newidx[i] * n + newidx[j]] = 0.5 * (Lp[i * n + j] + Lp[j * n + i]); /* R20 */
    }
  }
  /* 6. new state in the new anchor frame; shift the slot arrays */
  double v[3], e1[3];
  memcpy(e1, o->e + 3, sizeof(e1));
  compose(o->linear, o->a, e1, v);
  memcpy(o->a, v, sizeof(v));
  for (int k = 2; k < c; ++k) { between(o->linear, e1, o->e + 3 * k, v); memcpy(o->e + 3 * (k - 1), v, sizeof(v)); }
  for (int k = c - 1; k < W; ++k) memset(o->e + 3 * k, 0, 3 * sizeof(double));
  memset(o->e, 0, 3 * sizeof(double));
  for (int k = 2; k < c; ++k) {
    memcpy(o->z_odo + 3 * (k - 1), o->z_odo + 3 * k, 3 * sizeof(double));
    int t = o->lc_tgt[k] - 1;          /* targets that were slot 0 now live in the prior */
    o->lc_tgt[k - 1] = t < 0 ? -1 : t;
    memcpy(o->z_lc + 3 * (k - 1), o->z_lc + 3 * k, 3 * sizeof(double));
  }
  for (int k = 1; k < c; ++k) {
    memcpy(o->rb_valid + (k - 1) * L, o->rb_valid + k * L, sizeof(int) * L);
    memcpy(o->z_rb + (size_t)(k - 1) * L * 2, o->z_rb + (size_t)k * L * 2, sizeof(double) * 2 * L);
  }
  for (int k = 1; k < c; ++k) {
    o->un_valid[k - 1] = o->un_valid[k];
    memcpy(o->z_un + 3 * (k - 1), o->z_un + 3 * k, 3 * sizeof(double));
    memcpy(o->om_un + 9 * (k - 1), o->om_un + 9 * k, 9 * sizeof(double));
  }
  o->un_valid[c - 1] = 0;
  o->lc_tgt[c - 1] = -1;
  memset(o->rb_valid + (c - 1) * L, 0, sizeof(int) * L);
  o->c = c - 1;
  if (o->f32_storage) {
    double* sv = (double*)malloc(sizeof(double) * n);
    orc_get_state(o, sv);
    for (int i = 0; i < n; ++i) sv[i] = (double)(float)sv[i];
    orc_set_state(o, sv);
    free(sv);
    for (size_t i = 0; i < nn; ++i) o->Lam[i] = (double)(float)o->Lam[i];
    for (int i = 0; i < n; ++i) o->g[i] = (double)(float)o->g[i];
  }
  orc_get_state(o, o->vbar); /* d = 0 right after marginalization */

  free(Hs); free(gs); free(M); free(Nm); free(T); free(Hu); free(gu); free(Lp); free(gp); free(newidx);
  return rc;
}

/* ------------------------------------------------------------------ batch driver (R19) */

int orc_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

static int g_batch_f32_storage = 0;
/* optional unary factors of the batch run: un_valid[T][N] (int), un_pose[T][3][N], un_info[T][6][N] (xx,xy,yy,xt,yt,tt), float32 */
static const int* g_un_valid = 0;
static const float* g_un_pose = 0;
static const float* g_un_info = 0;
void orc_batch_set_unary(const int* valid, const float* pose, const float* info) { g_un_valid = valid; g_un_pose = pose; g_un_info = info; }
/* optional per-environment episode resets (NEXT-2): reset[T][N] (int), reset_pose[T][3][N]; applied before the push of step t */
static const int* g_reset = 0;
static const float* g_reset_pose = 0;
void orc_batch_set_resets(const int* reset, const float* pose) { g_reset = reset; g_reset_pose = pose; }
void orc_batch_set_f32_storage(int on) { g_batch_f32_storage = on; }

int orc_run_batch(int N, int W, int L, int T, int iters, const double* sig11,
                  const float* odom, const int* lc_back, const float* lc_meas,
                  const unsigned* rb_mask, const float* rb_meas,
                  const int* envs, int ne, int threads,
                  double* poses, double* cov, double* logdet, double* step) {
  int nwords = (L + 31) / 32;
  int bad = 0;
#ifdef _OPENMP
  if (threads <= 0) threads = omp_get_max_threads();
#pragma omp parallel for num_threads(threads) schedule(dynamic, 1) reduction(+ : bad)
#endif
  for (int q = 0; q < ne; ++q) {
    int env = envs[q];
    orc* o = orc_create(W, L, sig11, 0);
    o->f32_storage = g_batch_f32_storage;
    int* valid = (int*)calloc(L + 1, sizeof(int));
    double* zrb = (double*)calloc(2 * (L + 1), sizeof(double));
    int failed = 0;
    for (int t = 0; t <= T; ++t) {
      if (L > 0) {
        for (int l = 0; l < L; ++l) {
          valid[l] = (rb_mask[((size_t)t * nwords + l / 32) * N + env] >> (l % 32)) & 1u;
          zrb[2 * l + 0] = rb_meas[(((size_t)t * 2 + 0) * L + l) * N + env];
          zrb[2 * l + 1] = rb_meas[(((size_t)t * 2 + 1) * L + l) * N + env];
        }
      }
      if (t == 0) { if (L > 0) orc_observe_first(o, valid, zrb); continue; }
      double od[3], zl[3];
      for (int k = 0; k < 3; ++k) {
        od[k] = odom[((size_t)(t - 1) * 3 + k) * N + env];
        zl[k] = lc_meas ? lc_meas[((size_t)(t - 1) * 3 + k) * N + env] : 0.0;
      }
      int back = lc_back ? lc_back[(size_t)(t - 1) * N + env] : 0;
      if (g_reset && g_reset[(size_t)(t - 1) * N + env]) {
        double ip[3];
        for (int k = 0; k < 3; ++k) ip[k] = g_reset_pose[((size_t)(t - 1) * 3 + k) * N + env];
        orc_reset(o, ip);
      }
      orc_push(o, od, back, zl, valid, zrb);
      if (g_un_valid && g_un_valid[(size_t)(t - 1) * N + env]) {
        double zp[3], I6[6], I9[9];
        for (int k = 0; k < 3; ++k) zp[k] = g_un_pose[((size_t)(t - 1) * 3 + k) * N + env];
        for (int k = 0; k < 6; ++k) I6[k] = g_un_info[((size_t)(t - 1) * 6 + k) * N + env];
        I9[0] = I6[0]; I9[1] = I6[1]; I9[3] = I6[1]; I9[4] = I6[2];
        I9[2] = I6[3]; I9[6] = I6[3]; I9[5] = I6[4]; I9[7] = I6[4]; I9[8] = I6[5];
        orc_add_unary(o, zp, I9);
      }
      double sn = 0.0, S[9], ld = 0.0;
      if (orc_solve(o, iters, &sn) != 0) failed = 1;
      if (orc_cov(o, S, &ld) != 0) failed = 1;
      size_t row = (size_t)(t - 1) * ne + q;
      if (poses) orc_get_poses(o, poses + row * W * 3);
      if (cov) memcpy(cov + row * 9, S, sizeof(S));
      if (logdet) logdet[row] = ld;
      if (step) step[row] = sn;
      if (orc_count(o) == W) { if (orc_marginalize(o) != 0) failed = 1; }
    }
    bad += failed;
    free(valid); free(zrb);
    orc_destroy(o);
  }
  return bad;
}
