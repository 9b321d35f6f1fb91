/*
 * brmppi.h -- C ABI of the B200 (sm_100a) Barrier-Rate guided MPPI solver for a kinematic
 * tractor-trailer (arxiv 2508.05773).  Plain C: no C++ types, no exceptions, no torch types.
 *
 * What the calls are, and where the paper defines them:
 *   "At each control step, BR-MPPI receives the current state of the TT system and its
 *    environment, including static obstacles and predicted pedestrian motion, and generates
 *    control inputs"
 *   one MPPI solve = sample, roll out, weight, update                  (eq. 5)
 *   "u_k = u_nom,k is applied ... the last input is shifted, and the process repeats"
 *
 *   nominal control sequence initialised with zero
 *   model: eq. (6) reduced to [x, y, psi1, psi2] with controls (v, delta)
 *   barrier: eq. (16), e = 2 (discs); barrier-rate condition eq. (2)
 * The instance (4-state model, disc obstacles, per-sample alpha, hinge penalty) is the one
 * BASELINE.json's north_star names; every reading of the paper is listed in DESIGN.md.
 *
 * Pointer kinds.  Unless a parameter says DEVICE, every pointer is a HOST pointer owned by the
 * caller; the library copies in/out and keeps no reference after the call returns.
 * Ownership.  The caller owns the device workspace and the CUDA stream (with PyTorch:
 * torch.empty(bytes, dtype=torch.uint8, device="cuda").data_ptr() and
 * torch.cuda.Stream().cuda_stream); both must outlive the context.  The library never calls
 * cudaMalloc for solver data; it owns only the small host-side context object (and the CUDA
 * graph it captures for brmppi_step).
 * Errors.  Every call returns 0 (BRMPPI_OK) or a negative brmppi_status; nothing aborts, throws
 * or prints.  brmppi_strerror() maps a status to text; for BRMPPI_ERR_CUDA the text of the last
 * CUDA error seen by that call is appended.
 * Threads.  A context is not thread-safe; distinct contexts are independent.
 * Stream order.  solve / shift / set_* are enqueued on the context's stream and return without
 * waiting; get_* and brmppi_step synchronise that stream before returning.
 * No CPU fallback exists: without a CUDA device brmppi_create returns BRMPPI_ERR_CUDA.
 */
#ifndef BRMPPI_H
#define BRMPPI_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BRMPPI_MAX_DISCS 4

typedef enum {
  BRMPPI_OK = 0,
  BRMPPI_ERR_NULL = -1,                /* a required pointer was NULL                         */
  BRMPPI_ERR_INVALID_ARG = -2,         /* K<1, T<1, dt<=0, lambda<=0, sigma<0, bounds inverted,
                                          L<=0, scene out of range, unknown flag ...           */
  BRMPPI_ERR_WORKSPACE_TOO_SMALL = -3,
  BRMPPI_ERR_TOO_MANY_OBSTACLES = -4,
  BRMPPI_ERR_NONFINITE_INPUT = -5,     /* NaN/Inf in a state, goal, obstacle or control input  */
  BRMPPI_ERR_NOT_READY = -6,           /* solve/step before state and goal of every scene set;
                                          get_costs/get_final_states without FLAG_WRITE_SAMPLES */
  BRMPPI_ERR_CUDA = -7,
  BRMPPI_ERR_UNALIGNED = -8,           /* workspace not 256-byte aligned                       */
  BRMPPI_ERR_TOO_LARGE = -9            /* n exceeds the capacity of the library's static device scratch
                                          (brmppi_hitch_filter_static: BRMPPI_HITCH_STATIC_MAX_N)  */
} brmppi_status;

/* Disc obstacle with constant-velocity prediction (Assumption 2):
 * centre at rollout step t is (cx + t dt vx, cy + t dt vy).  radius > 0. */
typedef struct { float cx, cy, radius, vx, vy; } brmppi_obstacle;

/* Super-ellipse obstacle, eq. (16): centre (cx, cy), semi-axes (mx, my) along
 * the obstacle's own axes, orientation theta (rad), constant velocity (vx, vy) of the centre.
 *   h = (x'/(mx + r_v))^e + (y'/(my + r_v))^e - 1,  (x', y') = R(-theta)(c - centre(t)).
 * exponent e: 4 (parked cars in the paper) or 2 (pedestrians); other values are rejected.  The
 * barrier-rate hinge sums over discs and super-ellipses alike.  Default kernel only. */
typedef struct { float cx, cy, mx, my, theta, vx, vy; int exponent; } brmppi_superellipse;

/* Vehicle disc: body 0 = tractor axis (psi1), 1 = trailer axis (psi2); offset in metres from the
 * hitch point p_h = (x - Lh cos psi1, y - Lh sin psi1) along that axis. */
typedef struct { int body; float offset; } brmppi_disc;

/* flags */
#define BRMPPI_FLAG_WRITE_SAMPLES 1u   /* write S_k and x_T of every sample to HBM (parity /
                                          diagnostics; 20 B per sample)                        */
#define BRMPPI_FLAG_PRECISE_MATH  2u   /* sinf/cosf/tanf/logf instead of MUFU intrinsics      */
#define BRMPPI_FLAG_KERNEL_THREAD_PER_SAMPLE 4u  /* baseline kernel: one thread per sample, all
                                          steps fused (north_star item 2).  Default is the
                                          phase-split tile kernel.               */

#define BRMPPI_FLAG_PHASE_TIMING 8u     /* persistent kernel: every CTA records SM cycles per phase
                                          (clock64, bracketed by the globaltimer for the conversion
                                          to time); read with brmppi_get_phase_times            */
#define BRMPPI_FLAG_PROJECTED 32u       /* BR-MPPI proper (Sec. V-A): every sampled input is
                                          projected onto the barrier-rate equality (9) by the closed form
                                          (12) inside the rollout; per-obstacle alpha_i driven by the projected
                                          auxiliary input; no hinge penalty (w_bar is not read).  Readings:
                                          DESIGN.md reading 30.  max_obstacles <= BRMPPI_PROJECT_MAX_NO, no
                                          super-ellipses; one thread per sample.                            */
#define BRMPPI_FLAG_MPCC 64u            /* the paper's own model and tracking cost (DESIGN.md
                                          reading 31): 7-state jerk / steering-rate model, eq. (6)
                                          (PAPER.md:119-127), barrier-rate hinge on the second-order predictor (17)
                                          (PAPER.md:221-225), contouring / lag / heading / effort / progress cost
                                          (13)-(15) along a cubic reference path.  Controls are
                                          (j, omega); the state is set with brmppi_set_state7 and the path with
                                          brmppi_set_reference_path (no goal).  Default kernel: phase-split,
                                          persistent; with KERNEL_THREAD_PER_SAMPLE the simple one.
                                          Not with PROJECTED, super-ellipses or the hitch filter.               */
#define BRMPPI_FLAG_NO_CULL 16u         /* evaluate every (obstacle, disc, step) even where the
                                          hinge is provably zero (and 9.2 for BRMPPI_FLAG_MPCC);
                                          bit-identical results                                  */

typedef struct {
  int K;              /* samples per iteration, >= 1                                            */
  int T;              /* horizon steps, 1..BRMPPI_MAX_T                                         */
  int n_iter;         /* MPPI iterations per solve (no shift in between), >= 1                  */
  int n_scenes;       /* independent scenes solved per launch, >= 1; scene s uses seed + s      */
  int max_obstacles;  /* capacity per scene, 0..BRMPPI_MAX_OBSTACLES                            */
  int n_discs;        /* 1..BRMPPI_MAX_DISCS                                                    */
  brmppi_disc discs[BRMPPI_MAX_DISCS];
  float disc_radius;  /* r_v: obstacles are inflated to R + r_v                                 */
  float dt, L1, L2, Lh;
  float v_min, v_max, delta_min, delta_max;   /* hard clamp after perturbation (reading 9)      */
  float sigma_v, sigma_delta;                 /* Sigma_w = diag(sigma_v^2, sigma_delta^2)        */
  float alpha_lo, alpha_hi;                   /* alpha_k ~ U[alpha_lo, alpha_hi)                 */
  float w_pos, w_head, w_v, w_delta, w_hitch, hitch_max, w_bar, w_term, lambda;
  unsigned long long seed;
  unsigned int flags;
  int max_superellipses;  /* capacity per scene, 0..BRMPPI_MAX_SUPERELLIPSES                     */
  float hitch_kappa;      /* >= 0: the hitch-angle hinge starts at hitch_max - hitch_kappa |v|
                             (eq. (18)); 0 = fixed limit                        */
  /* Hitch-angle stabiliser, Sec. V-D (reading 28).                    */
  int hitch_filter;       /* 0 = off; 1 = brmppi_step passes U[0] through the CBF-QP below before
                             it is applied to the plant.  Never changes U itself.                 */
  float hitch_alpha;      /* alpha of condition (3), in (0, 1]         (read only if hitch_filter) */
  float hitch_qv, hitch_qdelta;   /* Q_h = diag(q_v, q_delta), both > 0 (read only if hitch_filter) */
  /* Projected rollout (read only with BRMPPI_FLAG_PROJECTED).  z = [v, omega = v tan(delta), u^alpha_1..N_o]:
   * W = Diag(Q1, Q2) with Q1 = diag(proj_qv, proj_qomega), Q2 = proj_qalpha I (all > 0), soft-bound weight
   * proj_rho >= 0 of (11a); bounds z_lo / z_hi = (v_min, -omega_max, -ualpha_max ..) / (v_max, omega_max,
   * ualpha_max ..), omega_max = max|v| tan(max|delta|); sampled u~^alpha ~ N(0, sigma_ualpha^2); stage cost
   * w_alpha * sum_i [h_i < h_buffer] max(0, alpha_i)^2.                                       */
  float proj_qv, proj_qomega, proj_qalpha, proj_rho, sigma_ualpha, ualpha_max, w_alpha, h_buffer;
  int k_offset;       /* global index of this context's first sample, >= 0: sample k of the context draws the noise
                         of sample k_offset + k and reports that index as argmin (K-sharded solves); 0 otherwise */
  /* The paper's own model and cost (read only with BRMPPI_FLAG_MPCC).  The sampled inputs are u = (j, omega):
   * box [j_min, j_max] x [omega_min, omega_max], Sigma_w = diag(sigma_j^2, sigma_omega^2); the
   * steering STATE delta is clamped to [delta_min, delta_max] after its Euler update; weights of (13): Qc
   * (contouring), Ql (lag), Qth1 / Qth2 (headings), Rj / Rw (effort), mu (progress, against nu_bar m/s); w_hitch,
   * hitch_max, hitch_kappa, w_bar, w_term, lambda, alpha_lo / alpha_hi as on the penalty path (w_term multiplies the
   * four tracking terms at the final state).  v_min .. sigma_delta's control-box meaning, w_pos, w_head, w_v and
   * w_delta are not read.  max_path_segments: capacity of the reference path, 1..BRMPPI_MAX_PATH_SEGMENTS.     */
  float j_min, j_max, omega_min, omega_max, sigma_j, sigma_omega;
  float Qc, Ql, Qth1, Qth2, Rj, Rw, mu, nu_bar;
  int max_path_segments;
} brmppi_params;

#define BRMPPI_MAX_T 512
#define BRMPPI_MAX_OBSTACLES 64
#define BRMPPI_MAX_SUPERELLIPSES 16
#define BRMPPI_PROJECT_MAX_NO 8     /* obstacles (rows of (9)) the projection handles */
#define BRMPPI_MAX_PATH_SEGMENTS 256

typedef struct brmppi_ctx brmppi_ctx;   /* opaque, library-owned host object */

typedef struct {
  float S_min;              /* smallest finite cost of the last iteration                       */
  int argmin;               /* its sample index (lowest index on ties), -1 if none finite       */
  float eta;                /* sum_k exp(-(S_k - S_min)/lambda)                                 */
  float ess;                /* effective sample size eta^2 / sum w^2                            */
  unsigned long long n;     /* global iteration counter after the last iteration                */
  int nonfinite;            /* samples whose cost was NaN/Inf (weight 0, skipped by argmin)     */
} brmppi_diag;

/* Bytes of device workspace brmppi_create needs for these parameters; 0 if they are invalid. */
size_t brmppi_workspace_bytes(const brmppi_params* p);

/* Create a context on the CURRENT CUDA device.  dev_workspace: DEVICE pointer, 256-byte aligned,
 * >= brmppi_workspace_bytes(p) bytes; cuda_stream: a cudaStream_t (NULL = legacy default
 * stream).  Nominal controls start at zero, iteration counter n = 0. */
int brmppi_create(const brmppi_params* p, void* dev_workspace, size_t workspace_bytes,
                  void* cuda_stream, brmppi_ctx** out);

/* Destroys the host object (and any captured graph).  Never frees the workspace. */
int brmppi_destroy(brmppi_ctx* ctx);

/* Vehicle state (x, y, psi1, psi2) of one scene.  psi1, psi2 are wrapped to [-pi, pi].  Not with BRMPPI_FLAG_MPCC. */
int brmppi_set_state(brmppi_ctx* ctx, int scene, const float x[4]);
/* BRMPPI_FLAG_MPCC: state x = (p_x, p_y, v, a, theta1, theta2, delta) of eq. (6) and the path parameter psi (arc
 * length of the vehicle's reference point on the path, 0 <= psi <= M dpsi, else BRMPPI_ERR_INVALID_ARG; delta must
 * lie in [delta_min, delta_max]).  theta1, theta2 are wrapped to [-pi, pi].  HOST pointer. */
int brmppi_set_state7(brmppi_ctx* ctx, int scene, const float x[7], float psi);
/* BRMPPI_FLAG_MPCC: reference path of one scene: M cubic segments on uniform knots of spacing dpsi > 0 in arc
 * length, coef[M][4][4] = coefficients c0..c3 (value = c0 + s (c1 + s (c2 + s c3)), s = psi - m dpsi) of the four
 * components (p^{x,r}, p^{y,r}, theta^{1,r}, theta^{2,r}) of segment m.  1 <= M <=
 * max_path_segments.  HOST pointer, copied.  Set it before brmppi_set_state7 (psi is checked against M dpsi). */
int brmppi_set_reference_path(brmppi_ctx* ctx, int scene, int M, float dpsi, const float* coef);
/* Goal pose (g_x, g_y, g_psi1, g_psi2).  Not with BRMPPI_FLAG_MPCC. */
int brmppi_set_goal(brmppi_ctx* ctx, int scene, const float g[4]);
/* Obstacles of one scene at rollout time 0; 0 <= n <= max_obstacles (NULL allowed when n = 0). */
int brmppi_set_obstacles(brmppi_ctx* ctx, int scene, int n, const brmppi_obstacle* obstacles);
/* State, goal and obstacles of one scene in ONE call: the same checks, meaning and error codes as brmppi_set_state +
 * brmppi_set_goal + brmppi_set_obstacles (in that order; nothing is changed if any of them would fail).  In a
 * single-scene context the three pieces leave through one host-to-device copy from a page-locked staging buffer the
 * context owns (two buffers used in turn, so the call never waits for the copy of the call before the last one);
 * with several scenes it is the three copies.  HOST pointers; asynchronous on the stream.  Not with BRMPPI_FLAG_MPCC. */
int brmppi_set_inputs(brmppi_ctx* ctx, int scene, const float x[4], const float g[4], int n,
                      const brmppi_obstacle* obstacles);
/* Super-ellipse obstacles of one scene at rollout time 0; 0 <= n <= max_superellipses (NULL allowed
 * when n = 0).  mx, my > 0; exponent 2 or 4 (else BRMPPI_ERR_INVALID_ARG). */
int brmppi_set_superellipses(brmppi_ctx* ctx, int scene, int n, const brmppi_superellipse* obstacles);
/* Nominal control sequence U[T][2] = (v, delta) per step ((j, omega) with BRMPPI_FLAG_MPCC); NULL = zeros.  Values must lie in
 * the control box (else BRMPPI_ERR_INVALID_ARG). */
int brmppi_set_nominal(brmppi_ctx* ctx, int scene, const float* U);
/* Set the global iteration counter n (the Philox counter word; reading 7).  All scenes. */
int brmppi_set_counter(brmppi_ctx* ctx, unsigned int n);
/* U = 0 and n = 0 for all scenes (state, goal and obstacles are kept). */
int brmppi_reset(brmppi_ctx* ctx);

/* One solve of every scene: n_iter x { sample, roll out, weight, update (5) }, n += n_iter.
 * Asynchronous on the stream.  A sample with non-finite cost gets weight 0; if all K are
 * non-finite U is left unchanged (diag.nonfinite == K). */
int brmppi_solve(brmppi_ctx* ctx);
/* brmppi_solve followed by brmppi_get_controls of every scene, as one call with no copy behind the solve: the
 * last iteration's update (5) writes the new nominal into page-locked host memory the context owns as well (the
 * way brmppi_step returns u0), the call waits for the stream and hands it over.  U_out: HOST, [n_scenes][T][2]
 * floats, owned by the caller.  Synchronous.  Everything else as brmppi_solve (same kernels, same results). */
int brmppi_solve_get_controls(brmppi_ctx* ctx, float* U_out);
/* One receding-horizon solve from host buffers to host buffers: brmppi_set_inputs(ctx, 0, x, g, n, obstacles)
 * followed by brmppi_solve_get_controls(ctx, U_out) -- same checks and error codes (nothing is changed or launched
 * if a check fails), same results.  In a single-scene context with a stream it is ONE graph launch: the copy of the
 * inputs from the context's page-locked staging buffer, the n_iter iterations, the last update writing U_out's
 * contents into page-locked host memory; otherwise it is the two calls.  HOST pointers; U_out [T][2] (scene 0; with
 * several scenes [n_scenes][T][2], the other scenes solved on the inputs they have).  Synchronous.  Not with
 * BRMPPI_FLAG_MPCC. */
int brmppi_solve_host(brmppi_ctx* ctx, const float x[4], const float g[4], int n, const brmppi_obstacle* obstacles,
                      float* U_out);
/* K-sharded solve.  The online-softmax state (m, eta, A[2T]) of
 * eq. (5) is associative, so G contexts (on G GPUs, or on one) can each own K/G of the samples of ONE solve:
 * same seed, state, goal, obstacles and nominal in every context, k_offset = first global sample index.
 * One MPPI iteration is then, on every shard:
 *   brmppi_shard_export(ctx, dev_record)   rollout of this shard's samples, its partials merged into ONE
 *                                          record of brmppi_shard_words(ctx) floats (per scene: m as fp64 in
 *                                          words 0-1, argmin, eta, sum w^2, nonfinite, 2 unused, A[2T]);
 *   (the caller gathers the G records in shard order: an all-gather of 4 (8 + 2T) bytes per scene and rank)
 *   brmppi_shard_import(ctx, G, dev_records)  merges them, writes U and the diagnostics, counter + 1.
 * Every shard merges the same records in the same order, so U is bit-identical on all of them.  dev_record /
 * dev_records: DEVICE pointers, 8-byte aligned, owned by the caller.  Asynchronous on the stream. */
size_t brmppi_shard_words(const brmppi_ctx* ctx);
int brmppi_shard_export(brmppi_ctx* ctx, float* dev_record);
int brmppi_shard_import(brmppi_ctx* ctx, int n_shards, const float* dev_records);

/* Warm-start shift U[t] <- U[t+1], last element kept (reading 4).  Asynchronous. */
int brmppi_shift(brmppi_ctx* ctx);
/* One closed-loop control step as a single CUDA-graph replay: solve; apply U[0] to the
 * kinematic model (one Euler step of eq. (6), psi wrapped; with BRMPPI_FLAG_MPCC the 7-state step and the
 * path-parameter update of reading 31); advance obstacles by dt * velocity;
 * shift.  Synchronises; u0_out[n_scenes][2] receives the applied control of each scene. */
int brmppi_step(brmppi_ctx* ctx, float* u0_out);

/* Results.  All synchronise the stream. */
int brmppi_get_controls(brmppi_ctx* ctx, int scene, float* U_out /* T*2 */);
int brmppi_get_state(brmppi_ctx* ctx, int scene, float x_out[4]);
int brmppi_get_state7(brmppi_ctx* ctx, int scene, float x_out[8]);   /* FLAG_MPCC: the seven states, then psi */
int brmppi_get_obstacles(brmppi_ctx* ctx, int scene, int* n_out, brmppi_obstacle* out /* max_obstacles */);
int brmppi_get_superellipses(brmppi_ctx* ctx, int scene, int* n_out, brmppi_superellipse* out /* max_superellipses */);
int brmppi_get_costs(brmppi_ctx* ctx, int scene, float* S_out /* K */);             /* FLAG_WRITE_SAMPLES */
int brmppi_get_final_states(brmppi_ctx* ctx, int scene, float* X_out /* K*4 */);    /* FLAG_WRITE_SAMPLES */
int brmppi_get_final_states7(brmppi_ctx* ctx, int scene, float* X_out /* K*8 */);   /* FLAG_WRITE_SAMPLES | FLAG_MPCC */
int brmppi_get_diag(brmppi_ctx* ctx, int scene, brmppi_diag* out);
/* What the hitch-angle stabiliser did in the last brmppi_step: u_ref = the BR-MPPI control U[0] it was
 * given, *status = 0 (rate constraint inactive, applied control = u_ref), 1 (active), 2 (no control in
 * the box satisfies the constraint; the least-violating one was applied).  With hitch_filter = 0 the
 * status is always 0.  HOST pointers; synchronises. */
int brmppi_get_hitch_filter(brmppi_ctx* ctx, int scene, float u_ref[2], int* status);

/* Device time of the two kernels of one MPPI iteration, for the roofline report.  OUTSIDE the
 * captured graph, on the context's stream, enqueues back to back and synchronises once: `reps` (+2
 * warm-up) rollout launches of every scene between two CUDA events, then `reps` (+2) update
 * launches between two events.  Returns mean milliseconds per launch (kernel + kernel-to-kernel
 * gap, as between graph nodes): out_ms[0] = rollout kernel, out_ms[1] = merge/update kernel.
 * Leaves U as ONE iteration from the current state would, and advances the iteration counter by
 * reps + 2.  1 <= reps <= 4096. */
int brmppi_time_kernels(brmppi_ctx* ctx, int reps, float out_ms[2]);

/* Per-phase device time of the LAST rollout launch, from the kernel's own clock64 stamps converted
 * with each CTA's lifetime on the globaltimer (needs BRMPPI_FLAG_PHASE_TIMING, else
 * BRMPPI_ERR_NOT_READY; default kernel only).  out_us[0..6] = mean over CTAs of the microseconds
 * spent in: scene prologue, A noise (+ obstacle tables), the Euler chain (which runs UNDER slot 3 on
 * the CTA's last four warps; not part of the sum), cost phase from the end of A to the end of the
 * last chunk, D reduction, E weighted control sums, partial write-out; out_us[7] = first CTA start to
 * last CTA end.  Synchronises. */
int brmppi_get_phase_times(brmppi_ctx* ctx, float out_us[8]);

/* Number of kernel launches this context has enqueued so far (graph replays count the kernels
 * inside the graph). */
unsigned long long brmppi_launch_count(const brmppi_ctx* ctx);

const char* brmppi_strerror(int status);

/* ---- test / measurement entry points --------------------------------------------------- */

/* Raw words of the in-kernel Philox4x32-10 generator: for k < K, t < T writes the four words
 * of the block with counter (t, n, k, tag) and key (lo32(seed), hi32(seed)) to
 * dev_out[(k*T + t)*4 + 0..3] (DEVICE pointer, K*T*4 uint32).  Uses the same device function as
 * the rollout kernels.  Synchronises. */
int brmppi_debug_philox(void* cuda_stream, unsigned long long seed, unsigned int n, int K, int T,
                        unsigned int tag, unsigned int* dev_out);

/* Arbitrary Philox4x32-10 blocks: out[i] = P(ctr[i]; key[i]) for i < n, through the generator the
 * rollout kernels use (use_curand = 0) or through the CUDA toolkit's own raw device function
 * curand_Philox4x32_10(uint4, uint2) (use_curand = 1) -- the library pin of the generator
 * (SURVEY §8(c)).  dev_ctr [n][4], dev_key [n][2], dev_out [n][4]: DEVICE pointers, 16-byte (key: 8-byte)
 * aligned.  Synchronises. */
int brmppi_debug_philox_raw(void* cuda_stream, int n, const unsigned int* dev_ctr, const unsigned int* dev_key,
                            int use_curand, unsigned int* dev_out);

/* The perturbed, clamped controls and alpha the kernels draw for (params, n, nominal U): writes
 * u[K][T][2] and alpha[K] (DEVICE pointers; either may be NULL).  dev_U_nominal: DEVICE [T][2].
 * Same device functions as the rollout kernels.  Nothing is allocated.  Synchronises. */
int brmppi_debug_sample_controls(void* cuda_stream, const brmppi_params* p, unsigned int n,
                                 const float* dev_U_nominal, float* dev_u, float* dev_alpha);

/* Hitch-angle stabiliser on its own, for n independent (state, reference control) pairs
 * (Sec. V-D).  With beta = wrap(psi1 - psi2), s = sign(beta) (+1 at 0) and
 *   h_h = hitch_max - hitch_kappa |v| - |beta|                                          eq. (18)
 *   c(u) = -s dt (psi1dot - psi2dot)(x, u) + hitch_alpha h_h        condition (3), sign of reading 1
 * the constraint is c expanded to first order in u about u_ref (reading 28: the reduced model is not
 * affine in (v, delta)), and
 *   u* = argmin q_v (v - v_ref)^2 + q_delta (delta - delta_ref)^2
 *        s.t. c(u_ref) + grad c(u_ref) . (u - u_ref) >= 0,  v_min <= v <= v_max,  delta_min <= delta <= delta_max.
 * x: HOST [n][4] states (x, y, psi1, psi2); u_ref: HOST [n][2]; u_out: HOST [n][2]; status_out: HOST
 * [n] or NULL, values as in brmppi_get_hitch_filter.  Uses p->dt, L1, L2, Lh, the control box and the
 * hitch_* fields (hitch_filter itself is ignored).  dev_scratch: DEVICE pointer to >=
 * brmppi_hitch_filter_scratch_bytes(n) bytes owned by the caller (staging for the host arrays; the
 * library allocates no device memory; BRMPPI_ERR_WORKSPACE_TOO_SMALL if it is too small).
 * Synchronises the stream.  n = 0 is a no-op. */
size_t brmppi_hitch_filter_scratch_bytes(int n);
int brmppi_hitch_filter(void* cuda_stream, const brmppi_params* p, int n, const float* x,
                        const float* u_ref, float* u_out, int* status_out, void* dev_scratch,
                        size_t scratch_bytes);

/* The same operation for callers that cannot allocate device memory at all (code under CUDA-graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): the staging that brmppi_hitch_filter takes from the caller as
 * dev_scratch lives here in a file-scope static __device__ array of BRMPPI_HITCH_STATIC_MAX_N * 36 bytes (576 KiB),
 * which every GPU that loads the library holds until the process exits.  Arguments, results and error codes as
 * brmppi_hitch_filter (all pointers HOST), plus: n > BRMPPI_HITCH_STATIC_MAX_N returns BRMPPI_ERR_TOO_LARGE and
 * touches nothing.  Calls no cudaMalloc / cudaFree and no allocating library routine; the array's device address
 * is looked up once per device (cudaGetSymbolAddress, with that device current) and kept.  Synchronises the
 * stream.  Every call on a device shares the one array: nothing in it has to start at zero (each call overwrites
 * the n entries it reads back; entries beyond n keep an earlier call's contents and are never read), but two
 * calls that overlap on the GPU -- from two host threads or two streams of the same device -- race on it:
 * serialise them. */
#define BRMPPI_HITCH_STATIC_MAX_N 16384
int brmppi_hitch_filter_static(void* cuda_stream, const brmppi_params* p, int n, const float* x,
                               const float* u_ref, float* u_out, int* status_out);

/* Closed-form projection of BR-MPPI, eq. (11)-(12), for n independent problems:
 *   min_z ||z - z_des||_W^2 + rho/2 (||z - z_lo||^2 + ||z_hi - z||^2)   s.t.  A z = b,
 *   z* = M^-1 [ p - A^T (A M^-1 A^T)^-1 (A M^-1 p - b) ],  M = W + rho I,  p = W z_des + rho/2 (z_hi + z_lo),
 * with z = [u_proj (2), u_proj^alpha (n_o)], d = 2 + n_o, 1 <= n_o <= BRMPPI_PROJECT_MAX_NO.
 * A: [n][n_o][d] row-major; b: [n][n_o]; z_des: [n][d]; z_out: [n][d] -- HOST pointers if
 * device_ptrs == 0 (copied in and out through dev_scratch, a DEVICE buffer of >=
 * brmppi_project_scratch_bytes(n, n_o) bytes owned by the caller; page-locked host arrays copy at
 * full PCIe rate, pageable ones several times slower; synchronises), DEVICE pointers, 16-byte
 * aligned for the bulk-copy path, if device_ptrs == 1 (dev_scratch unused, may be NULL; asynchronous
 * on the stream).  The library allocates no device memory either way.
 * w (the diagonal of W, all > 0), z_lo, z_hi: HOST [d], shared by all problems; rho >= 0.
 * A must have full row rank (A M^-1 A^T is factorised by Cholesky without pivoting); a rank-deficient
 * problem yields non-finite values in its own z_out row only.  How (9) builds A and b inside a rollout
 * is not part of this call.  n = 0 is a no-op. */
size_t brmppi_project_scratch_bytes(int n, int n_o);
int brmppi_project(void* cuda_stream, int n, int n_o, const float* A, const float* b, const float* z_des,
                   const float* w, float rho, const float* z_lo, const float* z_hi, float* z_out,
                   int device_ptrs, void* dev_scratch, size_t scratch_bytes);

/* Issue-rate micro-benchmarks for the roofline denominator: thread-instructions
 * per clock per SM achieved by dependent-chain-free streams of FFMA, LOP3/IADD3 (ALU pipe),
 * MUFU (XU pipe) and the FFMA+ALU mix, plus the SM count and the clock measured in-kernel.
 * out[0..7] = {ffma, alu (lop3), mufu, mix (ffma+lop3 interleaved), imad_wide, n_sms, sm_mhz of an idle SM,
 * sm_mhz seen while the FFMA kernel ran}; out[8..15] = {fmnmx, ffma2 (packed f32x2, two operands shared),
 * ffma2 with three distinct 64-bit register operands, fadd2, ffma+fmnmx interleaved, ffma2+fmnmx interleaved,
 * imad.lo, imad.hi} -- the dispatch-cost table of DESIGN.md 6.1.  Rates are whole-kernel: instructions per
 * SM / (first block start .. last block end on the globaltimer, converted with the in-kernel clock).
 * dev_scratch: DEVICE pointer to >= brmppi_measure_peaks_scratch_bytes() bytes owned by the caller
 * (the library allocates no device memory).  Synchronises. */
size_t brmppi_measure_peaks_scratch_bytes(void);
int brmppi_measure_peaks(void* cuda_stream, void* dev_scratch, size_t scratch_bytes, float out[16]);

#ifdef __cplusplus
}
#endif
#endif
