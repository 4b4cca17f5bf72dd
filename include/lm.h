/*
 * lm.h -- C ABI of the B200-native batched Levenberg-Marquardt pose refinement
 *         (the trajectory optimiser's pose-error phase of CppFlow, arxiv 2309.09102, sec. III-C).
 *
 * Problem: given FK(q): R^d -> SE(3), a target path Y = [y_1..y_n], y_i in
 * SE(3), and a seed trajectory xi = [q_1..q_n], q_i in R^d, refine xi so that FK(q_i) = y_i.
 * The pose residual of waypoint i depends on q_i only, so the damped normal
 * equations (J^T J + lambda I) delta = -J^T r are block diagonal with one d x d block per
 * waypoint; this library solves B*n such blocks per LM iteration on one GPU, with the
 * accept/reject decision and the lambda update taken per waypoint on the device.
 *
 * One LM iteration of one waypoint (readings R1-R11):
 *   J = geometric Jacobian at q (world frame, flange point)
 *   delta = -(J^T J + lambda I)^-1 J^T r   (fp32 Cholesky + refinement)
 *   q+ = clamp(q + delta, q_lo, q_hi)
 *   r+ = [w_pos (p(q+) - p_t) ; w_rot Log(R(q+) R_t^T)^vee],  F+ = |r+|^2 PAPER.md:L45-47, L115-117
 *   if F+ < F: accept, lambda = max(lambda / nu_down, lambda_min)        (paper silent: DESIGN R5)
 *   else     : reject, lambda = min(lambda * nu_up,  lambda_max)
 * A waypoint is frozen once sqrt(F) < tol (DESIGN R7); tol = 0 never freezes.
 *
 * Conventions
 *   - All functions return 0 (LM_OK) or a negative lm_status; nothing throws across the ABI.
 *   - "device" pointers are CUDA device memory owned by the CALLER (e.g. torch tensors) and are
 *     borrowed until lm_free(); they must be 16-byte aligned.  "host" pointers are plain host
 *     memory read during the call only (pinned memory makes the copies asynchronous).
 *   - Device arrays are structure-of-arrays over the waypoint index w = b*n + i (b = trajectory,
 *     i = timestep):  x[k][w]  is stored at  x[k*W + w],  W = B*n.
 *   - lm_step / lm_run / lm_fk only enqueue work on the stream given to lm_init; lm_fetch
 *     synchronises that stream.  There is no CPU fallback: without a CUDA device every entry
 *     point that needs one returns LM_ECUDA.
 */
#ifndef LM_B200_H
#define LM_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LM_MAX_DOF 8
#define LM_MAX_ITERS 64 /* accept_mask is 64 bits wide */

typedef enum {
    LM_OK = 0,
    LM_EINVAL = -1, /* null pointer, dof outside 1..8, B*n == 0, misaligned pointer, lo > hi, max_iters > 64 ... */
    LM_ENOMEM = -2, /* workspace smaller than lm_workspace_bytes() */
    LM_ECUDA = -3,  /* a CUDA runtime call failed; lm_strerror() gives cudaGetErrorString */
    LM_ECAPACITY = -4 /* lm_search_static only: (dof, K, n) needs more scratch than the fixed LM_SEARCH_STATIC_BYTES */
} lm_status;

typedef struct lm_ctx lm_ctx; /* opaque, library-owned (host memory); lm_free() releases it */

/* Serial kinematic chain, HOST memory, copied by lm_init.  Modified-DH (Craig) rows (DESIGN R1):
 *   A_j = Rot_x(alpha_{j-1}) Trans_x(a_{j-1}) Rot_z(theta_j) Trans_z(d_j),
 * revolute: theta_j = theta_off_j + q_j;  prismatic: d_j = d_off_j + q_j.  Base frame = world. */
typedef struct {
    int32_t dof;               /* d, 1..8 */
    const uint8_t *joint_type; /* [d] 0 = revolute, 1 = prismatic */
    const double *dh;          /* [d][4] a_{j-1} (m), alpha_{j-1} (rad), d_j (m), theta_off_j (rad) */
    const double *q_lo, *q_hi; /* [d] joint limits (rad | m) */
    double tool[7];            /* fixed flange transform after joint d: xyz (m) + unit quaternion w,x,y,z */
} lm_chain;

#define LM_MEM_DEVICE 0
#define LM_MEM_HOST 1

typedef struct {
    int64_t B, n;             /* trajectories, waypoints per trajectory */
    const float *target_pos;  /* [3][Wt] metres; Wt = B*n, or n if shared_targets */
    const float *target_quat; /* [4][Wt] quaternion w,x,y,z (re-normalised on load, sign free: DESIGN R11) */
    int32_t shared_targets;   /* 1: all B trajectories track the same path (K candidates of one Y) */
    const float *seeds;       /* [d][B*n] seed joint values; should lie inside the joint limits */
    int32_t memory;           /* LM_MEM_DEVICE: the three arrays above are device memory, borrowed until lm_free.
                                 LM_MEM_HOST: host memory, copied into the workspace by lm_init (async on the stream
                                 if pinned); the host arrays may be reused once the stream has passed the copies. */
    void *workspace;          /* DEVICE scratch, caller-allocated, >= lm_workspace_bytes(), 256-byte aligned */
    size_t workspace_bytes;
} lm_problem;

/* LM constants.  The paper gives none (DESIGN R5); lm_default_params() fills the documented defaults. */
typedef struct {
    float lambda0;        /* initial damping, 1e-3 (BASELINE.json configs[0]) */
    float nu_up, nu_down; /* Marquardt factors, 10 and 10 */
    float lambda_min;     /* 1e-4: below ~3e-5 the fp32 pivot of the self-motion direction is noise (DESIGN R5) */
    float lambda_max;     /* 1e7 */
    float tol;            /* freeze when sqrt(F) < tol; 0 = run a fixed number of iterations (DESIGN R7/R8) */
    float w_pos, w_rot;   /* residual weights, 1 and 1 (DESIGN R2b) */
    int32_t refine_steps; /* iterative-refinement steps on the fp32 Cholesky solve, 0..2 (default 1, DESIGN R4) */
    int32_t fast_sincos;  /* 0 = accurate sincosf (default); 1 = MUFU __sincosf */
    int32_t solver;       /* LM_SOLVER_PRIMAL (default): the d x d system (J^T J + lambda I) delta = -J^T r of PAPER.md:L121;
                             LM_SOLVER_DUAL: the same step as delta = -J^T (J J^T + lambda I_6)^-1 r (6 x 6, no refinement;
                             a disclosed variant) */
    int32_t rot_residual; /* LM_ROT_LOG (default): r_rot = Log(R R_t^T)^vee (DESIGN R2);  LM_ROT_RPY: the paper's literal wording
                             (PAPER.md:L47, L115-117), the wrapped element-wise difference of roll, pitch, yaw with
                             d(rpy)/dq = E(rpy)^-1 J_w (a disclosed variant; singular at pitch = +-90 deg;
                             not combined with LM_SOLVER_DUAL or lm_traj_*) */
} lm_params;
#define LM_SOLVER_PRIMAL 0
#define LM_SOLVER_DUAL 1
#define LM_ROT_LOG 0
#define LM_ROT_RPY 1

/* lm_fetch outputs.  Every pointer is nullable; each may be DEVICE or HOST memory (detected). */
typedef struct {
    float *res_norm;           /* [W] sqrt(F) at the current q */
    float *pos_err, *rot_err;  /* [W] |p - p_t| (m) and geodesic angle (rad), unweighted */
    float *lambda;             /* [W] current lambda */
    int32_t *iters;            /* [W] iterations executed (accepted + rejected) */
    uint64_t *accept_mask;     /* [W] bit k = iteration k accepted */
    uint32_t *status;          /* [W] LM_ST_* bits */
    uint8_t *traj_converged;   /* [B] 1 iff every waypoint of the trajectory is frozen */
    int32_t *traj_iters;       /* [B] max over the trajectory's waypoints of iters */
    int64_t total_waypoint_iters; /* OUT: sum of iters over all waypoints -- numerator of the throughput metric */
    int64_t converged_trajectories; /* OUT */
} lm_stats;

#define LM_ST_FROZEN 1u    /* sqrt(F) < tol */
#define LM_ST_MAXITER 2u   /* stopped by the iteration limit, not frozen */
#define LM_ST_BREAKDOWN 4u /* a Cholesky pivot <= 0 or a non-finite step was seen (treated as a rejected step) */
#define LM_ST_NONFINITE 8u /* a non-finite trial cost was seen (rejected) */
#define LM_ST_CLAMPED 16u  /* an accepted step was clamped to a joint limit */

/* Device scratch needed for (dof, B, n); `memory` as in lm_problem (host inputs are staged in the workspace). */
size_t lm_workspace_bytes(int32_t dof, int64_t B, int64_t n, int32_t shared_targets, int32_t memory);

int lm_default_params(lm_params *out);

/* Validate, copy the chain, bind buffers; state := seeds, lambda := lambda0, iters := 0.
 * cuda_stream: a cudaStream_t (NULL = default stream).  Enqueues at most the host->device copies. */
int lm_init(lm_ctx **out, const lm_chain *chain, const lm_problem *problem, const lm_params *params,
            void *cuda_stream);

/* Exactly one LM iteration for every waypoint that is not frozen and has iters < 64.  Async.
 * lm_step is the interleaving / teacher-forcing entry point (tests, lm_plan_run's bookkeeping between phases), NOT the
 * tuned path: it is the lm_run kernel with an iteration limit of one, so per call every waypoint's state round-trips
 * through HBM (4 (2 d + 18) bytes) and FK + the Jacobian are recomputed at entry (1878 instead of 1459 FLOP at d = 7).
 * Keeping r, F and J in the state instead would move 4 (6 d + 7) more bytes each way -- at d = 7 that is 520 B per
 * waypoint-iteration, 98 us per step on 4096 x 300 at the measured HBM peak, slower than the recomputation (92 us) -- so
 * the recomputation stays; a caller that wants throughput calls lm_run (one launch for all iterations, 41 us per
 * iteration on the same batch). */
int lm_step(lm_ctx *ctx);

/* On-device loop: every waypoint iterates until frozen or until its iters == max_iters (<= 64,
 * counted from lm_init / lm_reset / lm_set_state).  ONE kernel launch, no host round trip.  Async.
 * lm_run(N) and N calls of lm_step give bit-identical results. */
int lm_run(lm_ctx *ctx, int32_t max_iters);

/* Synchronise the stream and copy out the current state.  q_out: [d][W] device or host, nullable. */
int lm_fetch(lm_ctx *ctx, float *q_out, lm_stats *stats_out);

/* HOST data (the end-to-end path): refine all B*n waypoints from host arrays (pinned memory makes the copies
 * asynchronous) and write the results to host arrays.  The batch is split into `chunks` groups of whole trajectories
 * that are pipelined over the streams of an lm_pipe (copies in, kernels, copies out), so that the host->device copy of
 * chunk k+1, the LM kernel of chunk k and the device->host copy of chunk k-1 overlap (waypoints are independent:
 * PAPER.md:L121, so the result does not depend on `chunks`).
 *
 * lm_pipe_create: the handle owns 4 streams, 2 max_chunks + 5 events and 16 max_chunks bytes of pinned memory on the
 *   device that is CURRENT at the call; nothing is process-global.  1 <= max_chunks <= LM_PIPE_MAX_CHUNKS.
 * lm_pipe_solve: problem->memory must be LM_MEM_HOST, shared_targets 0, problem->workspace DEVICE scratch of
 *   >= lm_solve_host_workspace_bytes() bytes on the handle's device, which must be the current one (else LM_EINVAL);
 *   1 <= chunks <= min(B, max_chunks).  q_out [d][B*n] and every non-null array of `stats` are HOST pointers.  The
 *   pipeline starts after everything enqueued on `cuda_stream` so far (cudaStream_t as void*, 0 = the default stream),
 *   later work on that stream is ordered after it, and the call blocks the host until every output has arrived.  One
 *   call at a time per handle; handles of different devices (or several of one device) are independent.
 * lm_pipe_destroy: releases the streams, events and pinned memory (null is a no-op).
 * lm_solve_host: lm_pipe_create + lm_pipe_solve on the default stream + lm_pipe_destroy -- the one-shot form; creating
 *   the streams costs more than a whole step, so a caller that solves repeatedly keeps a handle. */
#define LM_PIPE_MAX_CHUNKS 256
typedef struct lm_pipe lm_pipe;
size_t lm_solve_host_workspace_bytes(int32_t dof, int64_t B, int64_t n, int32_t chunks);
int lm_pipe_create(lm_pipe **pipe_out, int32_t max_chunks);
int lm_pipe_solve(lm_pipe *pipe, void *cuda_stream, const lm_chain *chain, const lm_problem *problem, const lm_params *params,
                  int32_t max_iters, int32_t chunks, float *q_out, lm_stats *stats);
void lm_pipe_destroy(lm_pipe *pipe);
int lm_solve_host(const lm_chain *chain, const lm_problem *problem, const lm_params *params, int32_t max_iters,
                  int32_t chunks, float *q_out, lm_stats *stats);

/* Restart from the seeds given to lm_init (state := seeds, lambda := lambda0, iters := 0).  Host-only, no launch. */
int lm_reset(lm_ctx *ctx);

/* Inject a state: q [d][W] and lambda [W] (device or host, lambda nullable = lambda0); iters, mask, status := 0.
 * Used for warm restarts and teacher-forced tests.  Async copies on the stream. */
int lm_set_state(lm_ctx *ctx, const float *q, const float *lambda);

/* Debug trace (device pointers, nullable, borrowed): every executed iteration overwrites
 * trial_q [d][W] = q+ and trial_F [2][W] = (F before, F+ of the trial). */
int lm_set_trace(lm_ctx *ctx, float *trial_q, float *trial_F);

/* Tuning / test knobs.  LM_OPT_BLOCK_THREADS: threads per block (multiple of 32, <= 256; 0 = default 128).
 * LM_OPT_GENERIC_KERNEL: 1 = run the generic kernel even if the chain's structure matches a
 * specialised one (the two return the same values).  Results never depend on either. */
#define LM_OPT_BLOCK_THREADS 1
#define LM_OPT_GENERIC_KERNEL 2
/* LM_OPT_LANES_PER_WAYPOINT: 1 (default: one thread owns a waypoint block), 2 or 4 = the lane-group form BASELINE.json's
 * north_star names ("thread group per waypoint block ... warp-shuffle reductions for J^T J / J^T r"): the sums over the
 * rows of J are split over 2 / 4 adjacent lanes and closed with shuffles, everything else is replicated.  Kept as a
 * MEASURED alternative (it is slower); only for chains with a specialised kernel, the default
 * residual / solver, unit weights and exact sincos (else LM_EINVAL).  Results agree with the default to rounding (the
 * summation order of the row sums differs), not bitwise. */
#define LM_OPT_LANES_PER_WAYPOINT 3
/* LM_OPT_TRAJ_FUSED (after lm_traj_attach, which resets it): where the trajectory-level step forms its normal equations.
 * 1 = in the solve kernels' producer warps, straight into shared memory (nothing of J^T J, g, rho touches HBM), 2 = in
 * per-waypoint kernels through HBM, 0 (default) = 1 when the batch has enough tiles of 32 trajectories to pay for it,
 * else 2.  With collision rows the step always takes path 2.  Both paths return the same bits. */
#define LM_OPT_TRAJ_FUSED 4
/* LM_OPT_TRAJ_COST_LANES (after lm_traj_attach; only matters with collision rows): which waypoints share a warp when the
 * trial cost and its collision rows are evaluated.  The pair loops run well when the 32 lanes of a warp see the same
 * obstacles.  2 = 32 consecutive waypoints of ONE trajectory (always alike; costs a transposition through shared memory),
 * 1 = the same waypoint of 32 trajectories of a tile (alike only if those trajectories are candidates for one path -- the
 * paper's use of the optimiser on K plans of one problem), 0 (default) = 1 with shared_targets, else 2.  Same bits. */
#define LM_OPT_TRAJ_COST_LANES 5
int lm_set_option(lm_ctx *ctx, int32_t option, int32_t value);

/* Name of the LM kernel variant this context launches: "panda7", "rand8" (compile-time chain
 * structure, csrc/lm_specs.cuh) or "generic".  Static string. */
const char *lm_kernel_name(lm_ctx *ctx);

/* Run-time specialisation (csrc/lm_jit.cu).  Only the benchmark's robots have an ahead-of-time kernel for their chain
 * STRUCTURE (which joints are prismatic, which twists are 0 / +-pi/2, which offsets vanish; csrc/lm_specs.cuh); any other
 * chain runs the generic kernel (same results, ~1.35 x the time).  lm_specialize compiles the same kernel template for
 * this context's structure with NVRTC (about one second, once per structure, device and process; cached), and lm_step /
 * lm_run of this context launch it from then on: lm_kernel_name() returns "jit".  The values are those of the generic
 * kernel bit for bit (the specialisation only drops multiplications by exact 0 / +-1).  No-op (LM_OK) for a chain that
 * already has a specialised kernel.  LM_ECUDA when libnvrtc.so.12 cannot be loaded, the compilation fails or a CUDA call
 * fails: lm_strerror(LM_ECUDA) has the reason, and the context keeps the generic kernel.  LM_OPT_GENERIC_KERNEL = 1 still
 * selects the generic kernel; the trajectory-level kernels are not specialised at run time. */
int lm_specialize(lm_ctx *ctx);

/* Forward kinematics on the device with the context's chain (S1 of the hot path):
 * q [d][count] -> pos [3][count], rot [9][count] (row-major R, SoA).  Device pointers.  Async. */
int lm_fk(lm_ctx *ctx, const float *q, int64_t count, float *pos, float *rot);

/* ------------------------------------------------------------------------------------------------
 * Trajectory-level LM step: the paper's trajectory-length term.
 *
 * Residual of ONE trajectory (Fig. 6):
 *     r = [ w_pose * r_pose ; w_diff * (q_2 - q_1, ..., q_n - q_{n-1}) ]
 * with Jacobian blocks J_i (kinematic Jacobian) on the pose rows of waypoint i and
 * -I (for q_k), +I (for q_{k+1}) on the differencing rows.  The LM update
 * (J^T J + lambda I) delta = -J^T r then has, per trajectory, the block-tridiagonal matrix
 *     diag blocks  w_pose^2 J_i^T J_i + (c_i w_diff^2 + lambda) I   (c_i = 1 at the ends, 2 inside),
 *     off-diagonal blocks  -w_diff^2 I,
 * which is solved keeping that block structure (block elimination along the waypoint index, one
 * thread per trajectory, d x d blocks in registers) plus `refine_steps` steps of iterative
 * refinement with the residual formed from J, never from J^T J (DESIGN R4 / T4).  lambda, the
 * accept/reject decision (strict decrease of |r|^2 at the clamped trial point) and
 * the iteration count are per TRAJECTORY (DESIGN T3).  w_pose = 0 gives the paper's
 * trajectory-length step on its own; w_diff = 0 reduces to B*n independent pose blocks sharing
 * one lambda per trajectory.
 *
 * The step works on the context's CURRENT joint values (after lm_run / lm_set_state) and writes
 * the result back into them, so lm_run and lm_traj_run can be alternated.
 */
typedef struct {
    float w_pose, w_diff; /* 1 and 1 (the paper gives no weights: DESIGN T1) */
    float lambda0;        /* 1e-3 */
    float nu_up, nu_down; /* 10, 10 */
    float lambda_min;     /* 1e-4 */
    float lambda_max;     /* 1e7 */
    int32_t refine_steps; /* 0..2, default 1 */
} lm_traj_params;

/* lm_traj_fetch outputs; every pointer nullable, device or host. */
typedef struct {
    float *cost;           /* [B] |r|^2 = w_pose^2 cost_pose + w_diff^2 cost_diff at the current q */
    float *cost_pose;      /* [B] sum_i |r_pose,i|^2 (pose weights w_pos / w_rot applied, w_pose not) */
    float *cost_diff;      /* [B] sum_k |q_{k+1} - q_k|^2: the trajectory-length surrogate of PAPER.md:L123 */
    float *cost_coll;      /* [B] sum of the squared collision hinge residuals (0 without capsules); cost includes it */
    float *lambda;         /* [B] */
    int32_t *iters;        /* [B] trajectory-level iterations executed since lm_traj_attach / lm_traj_reset */
    uint64_t *accept_mask; /* [B] bit k = iteration k accepted */
    uint32_t *status;      /* [B] LM_ST_MAXITER | LM_ST_BREAKDOWN | LM_ST_NONFINITE | LM_ST_CLAMPED */
    int64_t total_traj_iters; /* OUT: sum of iters */
} lm_traj_stats;

/* Device scratch for the trajectory-level step of a (dof, B, n) problem. */
size_t lm_traj_workspace_bytes(int32_t dof, int64_t B, int64_t n);

int lm_traj_default_params(lm_traj_params *out);

/* Bind a caller-owned device workspace (256-byte aligned, >= lm_traj_workspace_bytes, borrowed until
 * lm_free) and the parameters; lambda := lambda0, iters := 0 for every trajectory.  Async. */
int lm_traj_attach(lm_ctx *ctx, const lm_traj_params *params, void *workspace, size_t workspace_bytes);

/* `iters` (1..64 in total per trajectory since the last attach / reset) more trajectory-level LM
 * iterations from the context's current joint values; the result replaces them.  The per-waypoint
 * state of lm_run (lambda, iteration count, accept mask) is left as it is; |r|, the pose errors and
 * the frozen flag reported by lm_fetch are re-evaluated at the new joint values.  Kernel launches only,
 * no host round trip; async.  lm_traj_run(N) and N calls of lm_traj_run(1) give identical bits. */
int lm_traj_run(lm_ctx *ctx, int32_t iters);

/* lambda [B] := the given values (device or host; NULL = lambda0); iters, masks, status := 0.  Async. */
int lm_traj_reset(lm_ctx *ctx, const float *lambda);

/* Synchronise the stream and copy out the per-trajectory state of the trajectory-level step. */
int lm_traj_fetch(lm_ctx *ctx, lm_traj_stats *stats_out);

/* Robot-robot collision rows of the trajectory-level step:
 * the robot is a set of capsules (endpoints a, b in the frame of a link, radius c); for every listed pair and
 * every waypoint one hinge row  r = w_coll * max(0, d_safe - dist),  dist = min over t1, t2 in [0,1] of
 * |(a1 + (b1-a1) t1) - (a2 + (b2-a2) t2)| - c1 - c2  (the paper's QP), with  d r / d q = -w_coll n^T (J_p1 - J_p2)
 * at the closest points.  The rows add d x d terms to the diagonal blocks of the
 * block-tridiagonal system and their squares to the cost.  HOST pointers, copied by the call; NULL, npairs = 0
 * or w_coll = 0 removes the rows.  Requires lm_traj_attach (which also clears any capsules). */
#define LM_MAX_CAPSULES 16
#define LM_MAX_CAPSULE_PAIRS 32
typedef struct {
    int32_t ncaps;
    const int32_t *link;   /* [ncaps] -1 = base (world) frame, j = the frame joint j (0-based) moves */
    const float *a, *b;    /* [ncaps][3] endpoints in the link frame (m) */
    const float *radius;   /* [ncaps] (m) */
    int32_t npairs;
    const int32_t *pairs;  /* [npairs][2] capsule indices */
    float w_coll;          /* weight of a collision row */
    float d_safe;          /* clearance below which a pair is penalised (m) */
} lm_capsules;
int lm_traj_set_capsules(lm_ctx *ctx, const lm_capsules *model);

/* Robot-environment collision rows: obstacles are cuboids "with arbitrary spatial positioning";
 * the distance of a capsule to a cuboid is, in the cuboid's axis-aligned frame, the minimum over 0 <= t <= 1 and
 * pmin <= p <= pmax of |p - (a + (b-a) t)|, less the radius (the paper's QP); per listed (capsule, obstacle) pair
 * and waypoint one hinge row  r = w_env * max(0, d_safe - dist)  with  d r / d q = -w_env n^T J_p  at the closest
 * point of the capsule axis.  Uses the capsules of lm_traj_set_capsules (call that first; it clears the obstacles;
 * a capsule model with npairs = 0 gives environment rows only).  HOST pointers, copied by the call. */
#define LM_MAX_OBSTACLES 8
typedef struct {
    int32_t nobs;
    const float *pose;     /* [nobs][7] frame of the cuboid in the world: xyz (m) + unit quaternion w,x,y,z */
    const float *pmin, *pmax; /* [nobs][3] extents in that frame (m) */
    int32_t npairs;
    const int32_t *pairs;  /* [npairs][2] (capsule index, obstacle index) */
    float w_env;
    float d_safe;
} lm_obstacles;
int lm_traj_set_obstacles(lm_ctx *ctx, const lm_obstacles *scene);

/* Debug trace (device pointers, nullable, borrowed): every executed iteration overwrites
 * trial_q [d][W] (w-order) = the clamped trial point and trial_F [2][B] = (|r|^2 before, at the trial point). */
int lm_traj_set_trace(lm_ctx *ctx, float *trial_q, float *trial_F);

/* ------------------------------------------------------------------------------------------------
 * Non-stationary schedule with anytime bookkeeping:
 * "the optimizer optimizes for pose error exclusively until the positional and rotational error ...
 * is below the respective specified threshold at every timestep.  A trajectory length ... optimization
 * step is then taken, after which the optimizer switches back to pose only, and the cycle continues";
 * "The optimizer keeps track of the latest valid solution".
 *
 * One cycle = [pose-only phase: per-waypoint LM state reset (lambda0, 0 iterations), lm_run(pose_iters)]
 *           -> [record: a trajectory is VALID when every waypoint has pos err < pos_tol and rot err < rot_tol
 *                and no joint moves more than mjac_rev / mjac_pris across a timestep
 *               (PAPER.md:L53); valid trajectories are copied to the "latest valid" slot with their length
 *               sum_i sum_j |q_{i+1}[j] - q_i[j]|]
 *           -> [ONE trajectory-level LM iteration (lm_traj_*) for the trajectories that are pose-valid now].
 * lm_plan_run(cycles) runs `cycles` such cycles and then one more pose-only phase + record; everything is
 * enqueued on the stream, no host round trip (readings P1-P4).
 * Requires lm_traj_attach.  The freeze tolerance of the pose phase is lm_params.tol.
 */
typedef struct {
    float pos_tol;      /* 1e-4 m (0.1 mm) */
    float rot_tol;      /* 0.1 deg in rad */
    float mjac_rev;     /* 7 deg in rad */
    float mjac_pris;    /* 0.02 m */
    int32_t pose_iters; /* cap of each pose-only phase, 1..64 (default 10) */
    float min_clearance; /* with capsules / obstacles set (lm_traj_set_capsules): a valid trajectory keeps every listed pair at
                            least this far apart at every waypoint ("at no timestep ... collide"); default 0 */
} lm_plan_params;

/* lm_plan_fetch outputs; every pointer nullable, device or host. */
typedef struct {
    uint8_t *valid;             /* [B] a valid trajectory has been recorded */
    int32_t *first_valid_cycle; /* [B] cycle of the first record (0 = after the first pose phase), -1 = never */
    int32_t *records;           /* [B] number of records */
    float *length;              /* [B] trajectory length of the recorded trajectory (NaN if none) */
    float *max_pos_err, *max_rot_err; /* [B] of the CURRENT trajectory at the last record point */
    float *mjac_rev, *mjac_pris;      /* [B] likewise */
    float *cur_length;                /* [B] likewise */
    float *min_clearance;             /* [B] likewise: smallest capsule clearance (NaN without capsules) */
    int64_t valid_trajectories;       /* OUT */
} lm_plan_stats;

size_t lm_plan_workspace_bytes(int32_t dof, int64_t B, int64_t n);
int lm_plan_default_params(lm_plan_params *out);
/* Bind a caller-owned device workspace (256-byte aligned, borrowed until lm_free); clears the bookkeeping. */
int lm_plan_attach(lm_ctx *ctx, const lm_plan_params *params, void *workspace, size_t workspace_bytes);
/* Clears the bookkeeping and the trajectory-level LM state, then runs the schedule from the context's
 * current joint values.  cycles 0..64.  Async. */
int lm_plan_run(lm_ctx *ctx, int32_t cycles);
/* Synchronise; q_valid_out [d][W] (device or host, nullable) = latest valid trajectories (NaN where none). */
int lm_plan_fetch(lm_ctx *ctx, float *q_valid_out, lm_plan_stats *stats_out);

/* ---- Global discrete search over the context's B = K candidate trajectories of ONE path ------------------
 * (sec. III-B; SURVEY.md section 8f NEXT-4 iii.)  The K x n joint
 * configurations are the nodes of a layered graph, every node of timestep i-1 is joined to every node of
 * timestep i, and a dynamic program finds the path whose largest joint change across a timestep (mjac,
 * PAPER.md:L95) is smallest:
 *     c[0][k] = pen[0][k],   c[i][k] = pen[i][k] + min_k' max(c[i-1][k'], max_j |q[k][i][j] - q[k'][i-1][j]|)
 * pen = pen_limit (paper: 10) where a joint is within margin_rev (1.5 deg) / margin_pris (3 cm) of a limit,
 * plus pen_collision (paper: 100) where the smallest capsule clearance of the node is < 0 (use_clearance;
 * needs lm_traj_attach + a capsule model).  Ties go to the lowest candidate; the path ends at
 * argmin_k c[n-1][k] and is read back through the stored predecessors ("backtracking", L97).  All arithmetic
 * is fp32, rounded to nearest, in the order written above. */
#define LM_SEARCH_MAX_K 1024
typedef struct {
    float margin_rev, margin_pris; /* rad, m (1.5 deg / 3 cm) */
    float pen_limit, pen_collision; /* 10, 100 */
    int32_t use_clearance;          /* 1: add pen_collision from the capsule model set by lm_traj_set_capsules/obstacles */
} lm_search_params;

size_t lm_search_workspace_bytes(int32_t dof, int64_t K, int64_t n);
int lm_search_default_params(lm_search_params *out);
/* Runs the search on the context's CURRENT joint values (seeds if nothing has run), B = K <= LM_SEARCH_MAX_K.
 * workspace: caller-owned device memory, 256-byte aligned, >= lm_search_workspace_bytes, used during the call only.
 * Outputs (device or host, each nullable): choice_out [n] candidate index per timestep; xi_out [d][n] the
 * selected configurations (xi_search); result_out [2] = { c[n-1][choice[n-1]], mjac of xi }.
 * Synchronises the context's stream before returning.  LM_EINVAL: null / misaligned arguments, B > LM_SEARCH_MAX_K,
 * use_clearance without a capsule model; LM_ENOMEM: workspace too small. */
int lm_search(lm_ctx *ctx, const lm_search_params *params, void *workspace, size_t workspace_bytes,
              int32_t *choice_out, float *xi_out, float *result_out);

/* ---- The same search for callers that cannot allocate device memory ------------------------------------------
 * Who this is for.  lm_search, like every other call here, works in a device workspace the caller allocates.  Some
 * users of a planner cannot do that at the point where they need the search:
 *   - a re-planning loop with a deadline (the paper's planner is "anytime": it must hand back a trajectory inside a
 *     time budget).  cudaMalloc / cudaFree take driver-wide locks, can wait for all work on the device
 *     and have no bound on how long they take, so such a loop may launch kernels but must not allocate;
 *   - a process in which something else owns the GPU's memory -- a simulator or a learning framework whose caching
 *     pool has claimed nearly everything, or a deployment whose memory budget is fixed at start-up -- so a fresh
 *     cudaMalloc fails or is forbidden by policy, and the owner's pool is not reachable from C.
 * For them the scratch of the search is a fixed array inside the library image: LM_SEARCH_STATIC_BYTES (16 MiB) of
 * device memory that EVERY GPU on which this library is loaded holds from load until the process exits, used or not.
 * That is the price, and the reason the limit is modest.
 *
 * lm_search_static allocates nothing (no cudaMalloc, cudaFree, host allocation or allocating library call) and needs
 * no lm_ctx.  The caller passes only inputs and outputs:
 *   chain       HOST; only dof, joint_type, q_lo, q_hi are read (dh and tool may be anything); the fp64 limits become
 *               fp32 exactly as in lm_init (rounded into the interval).
 *   K, n        candidates and timesteps.
 *   q           DEVICE memory of the current device, [dof][K * n] fp32, element (j, k * n + i) = joint j of candidate
 *               k at timestep i -- the layout of lm_problem.seeds.  Read only.
 *   params      as for lm_search; use_clearance must be 0 (the clearance needs a capsule model, i.e. a context).
 *   cuda_stream a stream of the current device (NULL = the default stream).
 *   choice_out [n], xi_out [dof][n], result_out [2]: device or host, each nullable; same meaning as in lm_search, and
 *               bit for bit the values lm_search returns for the same q, limits and params.
 * Limit: the intermediate arrays of (dof, K, n) -- lm_search_workspace_bytes(dof, K, n), dominated by the
 * (n - 1) * K * Kpad edge costs -- must fit in LM_SEARCH_STATIC_BYTES: for 7 joints e.g. K = 175 up to n = 124,
 * K = 64 up to n = 170, K = 32 up to n = 339.  lm_search_static_fits() answers for a given size (1 / 0); a size that does not fit
 * returns LM_ECAPACITY ("exceeds the fixed scratch ...") and launches nothing.  Other errors: LM_EINVAL (null pointer,
 * dof / K / n out of range, lo > hi, q not device memory of the current device, use_clearance != 0), LM_ECUDA.
 * Set-up: the first call on each device looks up the device address of the array (cudaGetSymbolAddress, with that
 * device current) and remembers it; make that first call during start-up, before any stream capture begins.
 * Sharing: all calls on a device, from every thread and every stream, use the SAME array, and it keeps whatever the
 * previous call left in it.  Nothing in it has to start at zero -- each call overwrites every element it later reads --
 * but two calls whose kernels overlap on the GPU (different streams, or threads calling concurrently) race on it and
 * return garbage: serialise them.  The call synchronises cuda_stream before it returns, as lm_search does. */
#define LM_SEARCH_STATIC_BYTES (16u << 20)
int lm_search_static_fits(int32_t dof, int64_t K, int64_t n);
int lm_search_static(const lm_chain *chain, int64_t K, int64_t n, const float *q, const lm_search_params *params,
                     void *cuda_stream, int32_t *choice_out, float *xi_out, float *result_out);

/* Measure the FP32 FMA throughput of the current device with an FMA-only micro-kernel (16 independent
 * chains per thread, best of 5 timed launches, CUDA events on `cuda_stream`); blocks the host.
 * tflops_out: 2 * FFMA / s / 1e12.  The measured counterpart of the ALU roofline. */
int lm_fp32_peak(void *cuda_stream, double *tflops_out);

void lm_free(lm_ctx *ctx);

/* Static string for a status code; for LM_ECUDA the last CUDA error string seen by this thread. */
const char *lm_strerror(int code);

/* Diagnostics, not part of the method: kernels launched by this library in this process so far (bench.py reports it
 * as gpu_launches; the tests use it to check launch counts such as "lm_run is ONE launch"). */
int64_t lm_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* LM_B200_H */
