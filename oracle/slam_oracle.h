/*
 * fp64 CPU ORACLE of the fixed-lag SE(2) SLAM backbone.  TEST INFRASTRUCTURE ONLY.
 *
 * This is a plain, slow, dense, one-environment-at-a-time restatement of what the hot path
 * computes (§III-D eqs. (5)-(6); readings R1-R23 of DESIGN.md).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, load or
 * call it.  It shares no code with the CUDA library under paper_2603_25834_b200/csrc/.
 *
 * What it does, step by step (DESIGN.md §"Algorithm"):
 *   reset      c=1, anchor a = init pose, prior Lambda = diag(1/sigma_p^2) on a
 *   push       e_c = e_{c-1} (+) z_odo, record factors, initialise newly seen landmarks
 *   solve      `iters` plain Gauss-Newton iterations: dense H, b; delta = H^{-1} b; v <- v + delta
 *   cov        dense H at the current estimate, explicit inverse, 6x6 block of (newest pose,
 *              anchor) propagated to the newest pose's global (x,y,theta): eq. (6), last block
 *   marginalize  re-anchor + explicit Schur complement of the oldest pose (dense)
 *
 * Variable vector (natural order, NOT the GPU's elimination order):
 *   v = [ a(3) ; e_1(3) ... e_{W-1}(3) ; g_0(2) ... g_{L-1}(2) ],  n = 3W + 2L
 *   a = global pose of the oldest window pose (anchor), e_k = pose k in the anchor frame,
 *   g_l = landmark l in GLOBAL coordinates (reading R17b: anchor-frame landmarks make the information
 *   matrix couple the weakly known anchor to strongly known landmarks -- unusable in fp32).
 *   index(a)=0, index(e_k)=3k, index(m_l)=3W+2l.
 *
 * Pins (tests/test_oracle_pins.py): finite-difference Jacobians, noise-free exact recovery, the
 * pure-translation closed form, the EKF prediction recursion on odometry-only runs, equality with
 * a global-coordinate full-batch Hessian on noise-free inputs, and equality with a brute-force
 * full-batch linear least squares in `linear` mode (arbitrary noise).  Exact numbers on noisy
 * nonlinear inputs with loops/landmarks are defined by this algorithm only: "parity unpinned" by any
 * closed form for those.
 */
#ifndef SLAM_ORACLE_H
#define SLAM_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct orc orc;

/* sig: prior(3), odo(3), lc(3), rb(2) sigmas = 11 doubles.  linear != 0 selects the linear-Gaussian
 * test mode (between residual r = e_j - e_i - z, no rotations, no wrapping; L must be 0). */
orc* orc_create(int W, int L, const double* sig11, int linear);
void orc_destroy(orc*);
void orc_reset(orc*, const double* init_pose3 /* NULL -> 0 */);
int  orc_count(const orc*);
int  orc_dim(const orc*);

/* lc_back: 0 none, k>=1 loop closure to the pose k steps older (ignored if k > count-1 before the
 * push... i.e. target already left).  rb_valid[L], rb_meas[L][2] (range, bearing) may be NULL if L=0 */
int  orc_push(orc*, const double* odom3, int lc_back, const double* lc_meas3,
              const int* rb_valid, const double* rb_meas);
int  orc_observe_first(orc*, const int* rb_valid, const double* rb_meas);
/* NEXT-1: unary absolute-pose factor on the newest pose (the paper's scan-match measurement with its
 * score-scaled information matrix; the scaling itself is not given, so the 3x3
 * information is an input).  pose3 = measured GLOBAL pose, info9 = symmetric 3x3, row-major. */
int  orc_add_unary(orc*, const double* pose3, const double* info9);
void orc_unary_factor(const double* a3, const double* ek3, const double* z3, int k_is_frame,
                      double* r3, double* Ja9, double* Je9);
void orc_batch_set_unary(const int* valid, const float* pose, const float* info);
/* NEXT-2: per-environment episode resets for the batch driver: orc_reset(init pose) before the push of step t */
void orc_batch_set_resets(const int* reset, const float* pose);
/* returns 0, or -1 if H was singular.  last_step_norm (may be NULL) = max |delta| of the last iteration */
int  orc_solve(orc*, int iters, double* last_step_norm);
int  orc_cov(orc*, double* cov9, double* logdet);
int  orc_marginalize(orc*);
void orc_get_poses(const orc*, double* poses /* [W][3] global, rows >= count zero */);
void orc_get_landmarks(const orc*, double* lm /* [L][2] global */, int* active /* [L] */);

/* ---- hooks for the pin tests ---- */
void orc_get_state(const orc*, double* v /* [n] */);
void orc_set_state(orc*, const double* v /* [n] */);
void orc_get_prior(const orc*, double* Lam /* [n*n] */, double* g /* [n] */, double* vbar /* [n] */);
void orc_assemble(const orc*, double* H /* [n*n] */, double* b /* [n] */);
double orc_cost(const orc*);   /* 0.5*sum r'Omega r + 0.5 d'Lam d + g'd at the current state */
/* residual and Jacobians of one between factor in the anchor frame; i_is_frame: pose i is the anchor */
void orc_between_factor(const double* ei3, const double* ej3, const double* z3, int i_is_frame,
                        double* r3, double* Ji9, double* Jj9);
/* landmark gl in global coordinates, observing pose x = a (+) ek (x = a if k_is_frame) */
void orc_rb_factor(const double* a3, const double* ek3, const double* gl2, const double* z2, int k_is_frame,
                   double* r2, double* Ja6, double* Jp6, double* Jg4);
/* re-anchoring map u(v) of A.5 step 2 and its Jacobian M = du/dv at the current state */
void orc_reanchor_map(const orc*, const double* v, double* u);
void orc_reanchor_jac(const orc*, double* M /* [n*n] */);

/* Conditioning probe (not a second implementation): with f32 storage on, the SAME fp64 algorithm rounds
 * the assembled H and b, the marginalisation prior and the state vector to fp32 before using them.
 * The distance between this run and the plain run is a lower bound on the error of ANY implementation
 * that stores those quantities in fp32; the parity tests use it to recognise the env-steps on which
 * the stated tolerances cannot be met in fp32 at all. */
void orc_set_f32_storage(orc*, int on);
void orc_batch_set_f32_storage(int on);

/* ---- batch driver: push -> solve -> cov -> (marginalize iff count == W), T steps, a set of envs.
 * Input arrays are float32, environment-fastest, exactly as the generator wrote them and as the
 * library consumes them (include/slam.h); `envs[ne]` selects which environments to run.
 * Outputs are per selected env: poses[T][ne][W][3], cov[T][ne][9], logdet[T][ne], step[T][ne]
 * (max-norm of the last GN update).  Any output pointer may be NULL.  Returns the number of envs whose
 * H became singular (should be 0).  Uses `threads` OpenMP threads over environments (<=0: all). */
int orc_run_batch(int N, int W, int L, int T, int iters, const double* sig11,
                  const float* odom, const int* lc_back, const float* lc_meas,
                  const unsigned* rb_mask, const float* rb_meas,
                  const int* envs, int ne, int threads,
                  double* poses, double* cov, double* logdet, double* step);
int orc_max_threads(void);

#ifdef __cplusplus
}
#endif
#endif
