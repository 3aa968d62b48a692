/*
 * slam.h -- C ABI of the B200-native batched fixed-lag SE(2) SLAM backbone.
 *
 * What it computes (arxiv/paper_2603_25834, section III-D): for `batch` simulated
 * robots at once, a sliding window of the last `window` SE(2) poses connected by
 * odometry, loop-closure and range-bearing landmark factors is optimised by a few Gauss-Newton
 * iterations (eq. (5)); the newest pose's 3x3 marginal covariance is the last
 * block of the inverse Gauss-Newton Hessian (eq. (6)) and is compressed to the
 * uncertainty scalar the reward consumes (D-optimality); the window then slides
 * with bounded memory and constant cost per step by Schur-marginalising the oldest
 * pose into a Gaussian prior.  Where the paper is silent the readings R1-R25 of DESIGN.md apply.
 *
 * Conventions
 *  - Every array argument is a DEVICE pointer owned by the caller unless the name ends in `_host`.
 *  - Layout is "environment fastest": an array documented [3][N] holds element (k, env) at k*N+env.
 *  - All calls enqueue work on the stream given to slam_create and return without synchronising.
 *    Nothing is allocated after slam_create; the caller owns the workspace.
 *  - Return value: SLAM_OK or an error code; slam_last_error() gives a host string.  Numerical
 *    trouble is per environment and asynchronous: a sticky status word (slam_get_status).
 *  - All environments move in lock-step: one host-side window count (slam_count).
 *  - Not re-entrant: one context per stream, one host thread per context.
 *  - Arithmetic: fp32, except the final 6x6 -> 3x3 covariance/log-det tail (fp64, O(1) per env) and the
 *    windows the conditioning watch hands to the fp64 path (slam_set_precision).
 */
#ifndef SLAM_H
#define SLAM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct slam_ctx slam_ctx; /* opaque host object */

enum { SLAM_OK = 0, SLAM_EINVAL = 1, SLAM_ESTATE = 2, SLAM_ENOMEM = 3, SLAM_ECUDA = 4 };
/* bits of the per-environment status word */
enum { SLAM_ENV_OK = 0, SLAM_ENV_NOT_PD = 1, SLAM_ENV_NONFINITE = 2,
       SLAM_ENV_INTERNAL = 4 /* an environment did not fit the shared-memory pool: cannot happen for sizes slam_create accepts */ };

#define SLAM_MAX_WINDOW 64    /* compiled maxima: window <= 64, landmarks <= 64 */
#define SLAM_MAX_LANDMARKS 64

/* Noise model: standard deviations, all > 0.  Defaults are BASELINE.json's values. */
typedef struct {
  float prior_sigma[3]; /* 0.01, 0.01, 0.005  (x, y, theta) of the first pose            */
  float odo_sigma[3];   /* 0.05, 0.05, 0.02   odometry between-factor                     */
  float lc_sigma[3];    /* 0.10, 0.10, 0.03   loop-closure between-factor                 */
  float rb_sigma[2];    /* 0.05 (range, m), 0.01 (bearing, rad)                           */
} slam_config;

/* Fills *cfg with the defaults above. */
void slam_default_config(slam_config* cfg);

/* Bytes of device workspace slam_create needs for these sizes (0 if the sizes are invalid). */
size_t slam_workspace_bytes(int batch, int window, int landmarks);

/* Creates a context.  window in [2, SLAM_MAX_WINDOW], landmarks in [0, SLAM_MAX_LANDMARKS],
 * batch >= 1.  `workspace` is device memory, >= slam_workspace_bytes(), 256-byte aligned, owned by
 * the caller and must outlive the context.  `cuda_stream` is a cudaStream_t (NULL = default
 * stream).  The context starts reset (count = 1, prior on pose 0 at the origin).
 * Errors: SLAM_EINVAL (sizes, NULLs, alignment, sigma <= 0, workspace too small), SLAM_ECUDA. */
int slam_create(slam_ctx** out, int batch, int window, int landmarks, const slam_config* cfg /* NULL: defaults */,
                void* workspace, size_t workspace_bytes, void* cuda_stream);
void slam_destroy(slam_ctx* ctx); /* frees the host object only */

/* count = 1; anchor pose = init_pose ([3][N], NULL -> origin); prior N(init_pose, diag(prior_sigma^2))
 * on it (reading R9); clears landmarks, factors, status and a pending slam_set_unary registration. */
int slam_reset(slam_ctx* ctx, const float* init_pose);

/* NEXT-2: per-environment episode reset (episodes end after 2048 steps or on collision).
 * Environments with mask[env] != 0 restart with ONE pose at init_pose ([3][N]; NULL -> origin), the
 * first-pose prior, no landmarks, no factors and a clear status, while the others keep their windows.
 * The window stays in lock-step on the host (slam_count is the count of the never-reset environments);
 * a reset environment simply has fewer live poses until its own window is full again: it is not
 * marginalised before that, its read-outs (slam_get_poses) report only its own poses, and loop closures
 * that reach behind its reset are ignored like any loop closure that leaves the window.
 * Call it between steps (after slam_marginalize_oldest / slam_step).  A pending slam_set_unary registration
 * is kept: it belongs to the pose the next push appends, for reset environments too (mask it with `valid`). */
int slam_reset_envs(slam_ctx* ctx, const int32_t* mask, const float* init_pose);

/* S0 push (BASELINE.json "initial guess is dead-reckoned"): appends one pose with the
 * dead-reckoned guess e_c = e_{c-1} (+) odom and records this step's factors.
 *   odom    [3][N]  dx, dy, dtheta in the previous pose's frame
 *   lc_back [N]     0 = none; k >= 1 = loop closure to the pose k steps older; k > count-1 (target
 *                   already left the window) is ignored for that env.  NULL = none.
 *   lc_meas [3][N]  newest pose expressed in the target pose's frame (required iff lc_back != NULL)
 *   rb_mask [ceil(L/32)][N]  visibility bits from the NEW pose (NULL iff landmarks == 0)
 *   rb_meas [2][L][N]        range (m), bearing (rad); newly seen landmarks are initialised by
 *                            inverse projection from the new pose's guess (reading R6)
 * Errors: SLAM_ESTATE if count == window (marginalise first), SLAM_EINVAL on NULL odom etc. */
int slam_push_step(slam_ctx* ctx, const float* odom, const int32_t* lc_back, const float* lc_meas,
                   const uint32_t* rb_mask, const float* rb_meas);

/* NEXT-1: unary absolute-pose factor -- the paper's scan-match measurement, whose
 * information matrix it scales by match score and ambiguity (formula not given, so the information
 * is an input).  Registers a factor for the pose that the NEXT slam_push_step / slam_step appends:
 *   pose  [3][N]  measured GLOBAL pose (x, y, theta) of that pose
 *   info  [6][N]  symmetric 3x3 information in global coordinates, packed (xx, xy, yy, xt, yt, tt)
 *   valid [N]     non-zero where the environment has a measurement; NULL = all
 * Residual r = [x - z_x; y - z_y; wrap(theta - z_theta)].  The pointers are read by that next push
 * (stream order) and must stay valid until then; pose = info = NULL cancels.  The factor leaves the
 * window with its pose and is folded into the prior by marginalisation. */
int slam_set_unary(slam_ctx* ctx, const float* pose, const float* info, const int32_t* valid);

/* Landmark observations from pose 0; only valid right after reset (count == 1). */
int slam_observe_first(slam_ctx* ctx, const uint32_t* rb_mask, const float* rb_meas);

/* S1-S3: exactly `iters` >= 0 plain Gauss-Newton iterations (eq. (5); no damping, reading R12):
 * linearise every live factor, assemble H = Lambda + sum J'Omega J and b in shared memory, envelope
 * Cholesky, triangular solves, additive update with wrapped angles. */
int slam_solve(slam_ctx* ctx, int iters);

/* S4 (eq. (6), readings R13-R15): relinearise at the current estimate, factorise, and return the
 * newest pose's marginal covariance in GLOBAL (x, y, theta) coordinates, without forming the full
 * inverse.  cov is [9][N] (row-major 3x3 per env).  The result is cached until the next push /
 * solve / marginalise / reset, so slam_dopt after slam_marginal_cov costs one copy kernel. */
int slam_marginal_cov(slam_ctx* ctx, float* cov);
/* logdet[N] = ln det Sigma_t;  dopt[N] = det(Sigma_t)^(1/3) = exp(logdet/3) (NULL to skip). */
int slam_dopt(slam_ctx* ctx, float* logdet, float* dopt);

/* S5: Schur-complement marginalisation of the oldest pose into the Gaussian prior, re-anchoring of
 * the window to the next pose, ring-buffer advance.  Requires count >= 2 (else SLAM_ESTATE). */
int slam_marginalize_oldest(slam_ctx* ctx);

/* Fused step: push -> solve(iters) -> covariance/log-det -> marginalise iff count == window after
 * the push.  One kernel launch.  Bit-for-bit equal to the composition of the separate calls.
 * cov [9][N], logdet [N] and last_pose [3][N] (newest pose, global) may each be NULL. */
int slam_step(slam_ctx* ctx, const float* odom, const int32_t* lc_back, const float* lc_meas,
              const uint32_t* rb_mask, const float* rb_meas, int iters, float* cov, float* logdet,
              float* last_pose);

/* The same step with HOST buffers: copies the inputs to device staging inside the workspace, runs
 * slam_step, copies cov/logdet/last_pose back, all on the context's stream.  With PAGE-LOCKED host
 * buffers (cudaHostAlloc / cudaHostRegister) every copy is asynchronous and the call returns at once;
 * with pageable memory each copy blocks the host until it is done (same results).  Either way the
 * caller synchronises the stream before reading the outputs.  Errors: as slam_step; SLAM_ECUDA if a
 * copy is refused (each copy's return code is checked). */
int slam_step_host(slam_ctx* ctx, const float* odom_host, const int32_t* lc_back_host, const float* lc_meas_host,
                   const uint32_t* rb_mask_host, const float* rb_meas_host, int iters, float* cov_host,
                   float* logdet_host, float* last_pose_host);

/* Read-outs.  poses: [3][W][N] global poses of the window, slots >= count zero-filled (R21).
 * lm: [2][L][N] global landmark positions (0 where inactive); active: [ceil(L/32)][N].
 * status: [N] sticky OR of SLAM_ENV_* bits. */
int slam_get_poses(slam_ctx* ctx, float* poses);
int slam_get_landmarks(slam_ctx* ctx, float* lm, uint32_t* active);
int slam_get_status(slam_ctx* ctx, int32_t* status);

/* Device counters since the last reset, copied to stats8 ([8] uint64, device): [0] max and [1] sum of the
 * envelope words (shared-memory footprint of H) over [2] solved environment-instances, [3] rounds an
 * environment waited for space in the shared-memory pool of its CTA (it is solved one round later; the
 * result does not depend on it), [4] environment-calls that ran on the fp64 path. */
int slam_get_stats(slam_ctx* ctx, unsigned long long* stats8);

/* NEXT-4: the paper's reward, eqs. (7)-(17), elementwise over environments, meant
 * to be enqueued right after slam_dopt.  The hyper-parameters are on the paper's project page, not in
 * the paper, so they are inputs; so is the mapping from Sigma_t to the scalar U (e.g. `dopt`).
 *   R = -lambda_col                                   if collision                              (7)
 *   R = R*_explore - R_abs + R*_delta                 otherwise
 *   R_explore = lambda_explore * dcells * I,  I = c + (1-c) iota                                (8),(10)
 *   c = clip((u_hi - U_prev)/u_hi, 0, 1)^2,  iota = clip(max(U_prev - U, 0)/kappa, 0, 1)        (11),(12)
 *   R_abs = lambda_abs * exp(U_prev) * U_prev,  R_delta = lambda_delta * exp(U_prev) * (U_prev - U)  (13),(14)
 *   alpha = clip((d_min - d_crash)/(d_full - d_crash), 0, 1)                                   (15)
 *   R*_explore = R_explore * alpha;  R*_delta = R_delta * alpha if U_prev - U > 0 else R_delta (16),(17)
 * u, u_prev, dcells (eq. (9), computed by the simulator side), d_min: [N] float; collision: [N] int32
 * (non-zero = collision); reward: [N] float out.  All device pointers. */
typedef struct {
  float lambda_col, lambda_explore, lambda_abs, lambda_delta, u_hi, kappa, d_crash, d_full;
} slam_reward_params;
int slam_reward(slam_ctx* ctx, const slam_reward_params* p, const float* u, const float* u_prev, const float* dcells,
                const float* d_min, const int32_t* collision, float* reward);

/* NEXT-3: the paper's other batched stage -- correlative scan matching against a 2D log-odds occupancy
 * grid and the confidence-weighted grid update (readings R28-R34 of
 * DESIGN.md, everything below the paper's sentence is a reading).  Stateless: no context needed.
 *   grid   [N][G][G] float log-odds, row-major (y, x), square, centred on the world origin, cell = res m
 *   ranges [R][N]    R rays over 180 degrees (phi_i = -pi/2 + i pi/(R-1)); valid iff r_min <= r <= r_max
 * slam_scan_match: scores the (2hx+1)(2hy+1)(2ht+1) candidates pose_pred + (ix sxy, iy sxy, it sth)
 * (offsets in global axes) with  s = mean over valid rays of 1/(1+exp(-grid[cell(end point)]))  (0 outside
 * the grid) and returns the best candidate as pose_meas [3][N], its score [N] and the second-best
 * score [N] (the ambiguity margin; how the information matrix is scaled from them is not in the paper
 * and is left to the caller, see slam_set_unary).  Ties go to the lowest candidate index.
 * slam_grid_update: every valid ray of the scan taken at `pose` [3][N] adds -l_free*weight to the cells it
 * crosses (Amanatides-Woo traversal) and +l_occ*weight to its end cell; then the grid is clamped to
 * [-l_clamp, l_clamp].  weight [N] = the confidence (e.g. the match score).
 * The sums are accumulated with fp32 atomic adds, one per (ray, cell): the ORDER of the additions to a cell varies
 * from run to run, so a cell crossed by several rays can differ in the last bit between two runs (the cells a ray
 * crosses are integer decisions taken in fp64 and do not vary).  Everything else in this header is deterministic. */
typedef struct {
  int G; float res; int R; float r_min, r_max; int hx, hy, ht; float sxy, sth;
} slam_scan_params;
int slam_scan_match(const slam_scan_params* p, int batch, const float* grid, const float* pose_pred, const float* ranges,
                    float* pose_meas, float* score, float* second, void* cuda_stream);
int slam_grid_update(const slam_scan_params* p, int batch, float* grid, const float* pose, const float* ranges,
                     const float* weight, float l_free, float l_occ, float l_clamp, void* cuda_stream);

/* Precision of the solve (eq. (6), is the quantity at stake).  A robot
 * that dead-reckoned for a while and re-observes a landmark has information on its anchor pose spanning six
 * decades: no fp32 information-form factorisation keeps Sigma_t to 1e-3 there.  The fp32 kernel therefore watches
 * the cancellation in the anchor's pivots, r = max_i H_ii / L_ii^2 over the three anchor rows, in every
 * factorisation.  mode 1: an environment with r > ratio_hi (or a failed factorisation) is not committed by the
 * fp32 kernel; the same call is redone for it by the fp64 kernel, which keeps the environment's state and prior in
 * an fp64 shadow record until r < ratio_lo again AND the newest pose sees at least three landmarks (a robot that
 * leaves the map right after the hand-over would dead-reckon in fp32 on a prior that still carries the cancellation
 * of the ill-conditioned phase).  While the newest pose sees at least nine landmarks both thresholds count twice: with
 * that many fresh measurements per step the result hardly leans on the prior, and what fp32 loses in the anchor's
 * pivots does not accumulate (measured on 1.2e6 env-steps: the same env-steps beyond tolerance, the same number beyond
 * half of it).  mode 0: fp32 only, no watch.  mode 2: every environment on the
 * fp64 kernel (an independent second implementation: the device reference of the tests).  mode -1: the default
 * rule -- 1 for windows with landmarks or once slam_set_unary was used, else 0 (pose-only windows keep the anchor
 * out of every factor).  ratio_hi / ratio_lo: 0 keeps the current value (defaults 300 / 150).
 * Bit-for-bit equality of slam_step with the separate calls holds for environments that stay in one mode. */
int slam_set_precision(slam_ctx* ctx, int mode, float ratio_hi, float ratio_lo);

/* Allocation-free entry point, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it): ONE call runs a whole episode -- reset at the origin, (landmarks > 0:
 * the observation from pose 0 = slice 0 of rb_mask / rb_meas), then `steps` fused steps exactly like slam_step --
 * with every scratch buffer of the kernels (environment records, fp64 shadows, cost order, covariance cache) in a
 * static device array of SLAM_STATIC_MAX_BYTES inside the library instead of a caller-owned workspace.  It calls no
 * cudaMalloc / cudaFree and no allocating CUDA library routine.  Every GPU that loads the library holds the array
 * until the process exits.  Sizes whose workspace (slam_workspace_bytes) exceeds the array are rejected with
 * SLAM_ENOMEM and a message in `err` (e.g. window 20 + 24 landmarks: about 200 environments; window 6 + 5 landmarks:
 * about 2000).  ALL CALLS SHARE THE ARRAY: it keeps the last call's contents (each call clears what must start at
 * zero), and calls that overlap on the GPU -- different streams without a dependency -- race.
 *   odom [steps][3][N], lc_back [steps][N] (NULL: none), lc_meas [steps][3][N],
 *   rb_mask [steps+1][ceil(L/32)][N], rb_meas [steps+1][2][L][N]   (NULL iff landmarks == 0)
 *   cov [steps][9][N], logdet [steps][N], last_pose [steps][3][N]  (each may be NULL)     -- all DEVICE pointers
 *   err / err_len: optional host buffer for the message of a non-zero return. */
#define SLAM_STATIC_MAX_BYTES (16u << 20)
int slam_run_static(int batch, int window, int landmarks, int steps, int iters, const slam_config* cfg, const float* odom,
                    const int32_t* lc_back, const float* lc_meas, const uint32_t* rb_mask, const float* rb_meas, float* cov,
                    float* logdet, float* last_pose, void* cuda_stream, char* err, size_t err_len);

/* Measurement aid: per-kernel device time of the step launches.  slam_kernel_timing(ctx, max_steps) creates
 * 4 * max_steps CUDA events (max_steps = 0 frees them and switches the timing off; this is the one call besides
 * slam_create that creates CUDA objects); from then on every call that launches the step kernel records an event
 * before it, after it, after the fp64 kernel and after the ordering kernel, for the next max_steps such calls.
 * slam_kernel_timing_read waits for the last recorded event, stores the summed milliseconds of
 * [0] slam_step_kernel, [1] slam_ref64_kernel, [2] slam_order_kernel in ms3 (host double[3]) and the number of
 * calls they cover in *steps (host, may be NULL), and restarts the recording. */
int slam_kernel_timing(slam_ctx* ctx, int max_steps);
int slam_kernel_timing_read(slam_ctx* ctx, double* ms3, int* steps);

/* Measurement aid for the roofline's denominator ("P_fp32 ... the bench must measure it
 * with a register-resident FMA microbenchmark"): enqueues ONE launch of a kernel that fills every SM with
 * independent FP32 FMA chains held in registers (8 CTAs of 256 threads per SM, 64 FMAs per loop iteration and
 * thread, `iters` iterations, no memory traffic in the loop) and stores the number of floating-point operations
 * that launch performs (2 per FMA) in *flops (host, may be NULL).  The caller times the launch with events on
 * `cuda_stream`.  sink: device float[1], never written for the arguments used.  No context needed. */
int slam_fma_probe(long long iters, float* sink, void* cuda_stream, double* flops);

int slam_count(const slam_ctx* ctx);                /* host-side window count c in [1, window] */
long long slam_launch_count(const slam_ctx* ctx);   /* kernels launched by this context so far */
const char* slam_last_error(const slam_ctx* ctx);   /* message of the last non-zero return */

/* Introspection for the benchmark's roofline accounting: smem bytes per CTA, warps per CTA and
 * resident CTAs per SM of the step kernel for this context's sizes. */
int slam_kernel_info(const slam_ctx* ctx, int* smem_bytes_per_cta, int* warps_per_cta, int* ctas_per_sm);

#ifdef __cplusplus
}
#endif
#endif /* SLAM_H */
