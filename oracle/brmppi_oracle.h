/*
 * brmppi_oracle.h -- CPU oracle for one BR-MPPI solve of a kinematic tractor-trailer.
 *
 * TEST INFRASTRUCTURE ONLY.  This is the plain, slow, obviously-correct restatement of the
 * method in fp64 that the CUDA path is checked against.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code, header,
 * table or constant generator with paper_2508_05773_b200/csrc/ and includes nothing from there.
 *
 * Passages followed (PAPER.md = text of arxiv 2508.05773; SURVEY.md §8(c) = the readings taken
 * where the paper is silent, all listed again in DESIGN.md):
 *   MPPI loop, weights, update (5), shift ........ PAPER.md:89-98
 *   tractor-trailer kinematics, eq. (6) ........... PAPER.md:121-127 (reduced to [x,y,psi1,psi2])
 *   discrete barrier-rate condition, eq. (2) ...... PAPER.md:64-74
 *   disc barrier = eq. (16) with e = 2 ............ PAPER.md:216-225
 *   stage + terminal cost structure, eq. (7) ...... PAPER.md:135
 *   quadratic tracking / heading / effort terms ... PAPER.md:202
 *   hitch-angle limit ............................. PAPER.md:231-235
 *   hitch-angle stabiliser: barrier (18), CBF-QP .. PAPER.md:229-239 with (3) PAPER.md:66-76
 *                                                   (reading 28)
 *
 * Pin status (tests/test_oracle_*.py, all `-m "not gpu"`):
 *   philox4x32_10 ............ pinned: published known-answer vectors + cuRAND header constants
 *   uniforms / Box-Muller .... pinned: exact representability, range, moments
 *   kinematic step ........... pinned: straight line, Euler-circle radius, hitch relaxation
 *                              closed form, steady-turn fixed point
 *   barrier / hinge .......... pinned: h=0 on the inflated circle, h=3 at 2 rho, hand-computed
 *                              step, receding sample => 0, stationary inside => T*alpha*|h|
 *   weights / update / shift . pinned: positivity, sum to 1, shift invariance, permutation
 *                              invariance, lambda->0 argmin, lambda->inf mean, sigma=0 fixed point
 *   super-ellipse barrier .... pinned: boundary points, e = 2 & m_x = m_y reduces to the disc barrier,
 *                              rotation covariance, corner value, brute force with super-ellipses
 *   hitch stabiliser ......... pinned: hand value of (18); rate condition == exact discrete condition (2)
 *                              through the pinned Euler step; gradient by finite differences; QP against
 *                              scipy SLSQP, a dense grid search and the halfspace-projection closed form;
 *                              closed-loop forward invariance of |hitch| <= limit under a jackknifing
 *                              reference.  The linearisation in u about u_ref is reading 28, not the paper's.
 *   projected rollout ........ pinned: (12) against the numpy form, KKT residuals and scipy SLSQP; A z* = b at
 *                              every (k, t); N_o = 1 scalar closed form; rho = 0 == pinv projection; rho -> inf
 *                              pulls to the centre of the bounds; rows of (9) against finite differences of h
 *                              through the pinned Euler step; far obstacle => u untouched; mpmath brute
 *                              force K<=4, T<=4.  The alpha cost's FORM is parity unpinned (reference [1] only).
 *   whole solve .............. pinned: brute force (independent mpmath transcription) K<=8, T<=5
 *   cost weights, disc placement, hinge shapes (linear barrier hinge, squared hitch hinge),
 *   scene generators ......... PARITY UNPINNED by the paper (never printed there); fixed by the
 *                              readings in DESIGN.md only.
 */
#ifndef BRMPPI_ORACLE_H
#define BRMPPI_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORC_MAX_DISCS 4

/* All lengths in metres, angles in radians, times in seconds. */
typedef struct {
  int K;                  /* samples (rollouts) per iteration                         */
  int T;                  /* horizon: controls u_0..u_{T-1}, states x_0..x_T          */
  int n_discs;            /* vehicle discs, <= ORC_MAX_DISCS                           */
  int disc_body[ORC_MAX_DISCS];     /* 0 = tractor (psi1), 1 = trailer (psi2)          */
  double disc_offset[ORC_MAX_DISCS];/* metres from the hitch point along the body axis */
  double disc_radius;     /* r_v                                                       */
  double dt, L1, L2, Lh;
  double v_min, v_max, delta_min, delta_max;
  double sigma_v, sigma_delta;
  double alpha_lo, alpha_hi;
  double w_pos, w_head, w_v, w_delta, w_hitch, hitch_max, w_bar, w_term, lambda;
  double hitch_kappa;     /* hitch limit = hitch_max - hitch_kappa |v| (eq. (18)) */
  double hitch_alpha;     /* alpha of condition (3) in the hitch stabiliser, in (0, 1] */
  double hitch_qv, hitch_qdelta;  /* Q_h = diag(q_v, q_delta) > 0 of the CBF-QP     */
  uint64_t seed;          /* Philox key = (lo32(seed), hi32(seed))                     */
} orc_params;

/* Philox4x32-10 block function (Salmon et al., SC'11). out = P(ctr; key). */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

/* f(w) = (w >> 9) * 2^-23, in [0,1), exact in fp32 and fp64.  SURVEY §8(c) reading 5. */
double orc_uniform(uint32_t w);

/* The two standard normals of (seed, n, k, t): Philox ctr = (t >> 1, n, k, 0), words (0, 1) for
 * even t and (2, 3) for odd t (readings 5, 6); Box-Muller with u1 = 1 - f(wa), u2 = f(wb).
 * z[0] -> speed channel, z[1] -> steering. */
void orc_normals(uint64_t seed, uint32_t n, uint32_t k, uint32_t t, double z[2]);

/* alpha_k of (seed, n, k): Philox ctr = (0, n, k, 1), word 0. */
double orc_alpha(const orc_params* p, uint32_t n, uint32_t k);

/* wrap(a) = a - 2 pi rint(a / 2 pi). */
double orc_wrap(double a);

/* One explicit-Euler step of the reduced eq. (6); every right-hand side at x. */
void orc_kinematic_step(const orc_params* p, const double x[4], double v, double delta,
                        double x_next[4]);

/* Centre of vehicle disc j at state x. */
void orc_disc_centre(const orc_params* p, const double x[4], int j, double c[2]);

/* h = ||c - o||^2 / (R + r_v)^2 - 1 for disc centre c and obstacle centre o, radius R. */
double orc_barrier(const orc_params* p, const double c[2], const double o[2], double R);

/* Super-ellipse barrier, eq. (16) PAPER.md:216-221 (NEXT row 2 of SURVEY §8(f)):
 *   h = |x'/(m_x + r_v)|^e + |y'/(m_y + r_v)|^e - 1,  (x', y') = R(-theta)(c - o).
 * se = (cx, cy, m_x, m_y, theta, vx, vy, e); o = the obstacle centre at the step in question. */
double orc_barrier_se(const orc_params* p, const double c[2], const double o[2], const double* se);

/* G(x) = w_pos ||p - g_p||^2 + w_head (wrap(psi1-g_psi1)^2 + wrap(psi2-g_psi2)^2). */
double orc_goal_cost(const orc_params* p, const double x[4], const double goal[4]);

/*
 * Roll out ONE sample under the given control sequence u[T][2] (already perturbed and
 * clamped) and barrier-rate alpha.  obstacles = n_obs x (cx, cy, R, vx, vy) at rollout time 0.
 * Returns S (total cost); x_T -> xT[4]; if traj != NULL it receives (T+1) x 4 states; if
 * pen_out != NULL it receives the un-weighted barrier-rate penalty sum.
 */
double orc_rollout(const orc_params* p, const double x0[4], const double goal[4], int n_obs,
                   const double* obstacles, const double* u, double alpha, double xT[4],
                   double* traj, double* pen_out);

/* Sample k of iteration n with nominal U_in[T][2]: draws alpha_k and u~_k (written to u[T][2]),
 * rolls out, returns S_k; x_T -> xT. */
double orc_sample(const orc_params* p, uint32_t n, uint32_t k, const double x0[4],
                  const double goal[4], int n_obs, const double* obstacles, const double* U_in,
                  double* u, double xT[4]);

/*
 * Weights and update from costs S[K] and sampled controls u[K][T][2]:
 *   k* = lowest k attaining the minimum finite S;  w_k = exp(-(S_k - S_k*)/lambda) (0 if S_k is
 *   not finite);  eta = sum w;  U[t] = sum_k w_k u[k][t] / eta.
 * Writes w[K] (un-normalised) if w != NULL.  Returns number of non-finite costs; if all K are
 * non-finite U_out is left untouched, *argmin = -1.
 * *gap = (second smallest S) - (smallest S)   (+inf if K == 1).
 */
int orc_weights_update(int K, int T, double lambda, const double* S, const double* u,
                       double* U_out, double* w, int* argmin, double* gap, double* eta);

/*
 * One full MPPI iteration with global iteration counter n:
 * sample, perturb + clamp, roll out, weight, update.  U_in[T][2] -> U_out[T][2] (may alias).
 * Optional outputs (NULL to skip): S[K], XT[K][4], u_all[K][T][2], w[K].
 * n_threads > 1 partitions the sample loop over pthreads; results are bit-identical to
 * n_threads == 1 because every sample is independent and the reduction is done afterwards,
 * single-threaded, in index order.
 * Returns the number of non-finite costs.
 */
int orc_iteration(const orc_params* p, uint32_t n, const double x0[4], const double goal[4],
                  int n_obs, const double* obstacles, const double* U_in, double* U_out,
                  double* S, double* XT, double* u_all, double* w, int* argmin, double* gap,
                  double* eta, int n_threads);

/* The same three calls with n_se super-ellipse obstacles (8 doubles each, layout above) next to the
 * discs; the barrier-rate hinge sums over both kinds.  The calls above are these with n_se = 0. */
double orc_rollout_se(const orc_params* p, const double x0[4], const double goal[4], int n_obs,
                      const double* obstacles, int n_se, const double* se, const double* u,
                      double alpha, double xT[4], double* traj, double* pen_out);
double orc_sample_se(const orc_params* p, uint32_t n, uint32_t k, const double x0[4],
                     const double goal[4], int n_obs, const double* obstacles, int n_se,
                     const double* se, const double* U_in, double* u, double xT[4]);
int orc_iteration_se(const orc_params* p, uint32_t n, const double x0[4], const double goal[4],
                     int n_obs, const double* obstacles, int n_se, const double* se,
                     const double* U_in, double* U_out, double* S, double* XT, double* u_all,
                     double* w, int* argmin, double* gap, double* eta, int n_threads);
void orc_advance_se(const orc_params* p, int n_se, double* se);

/* Warm-start shift: U[t] = U[t+1] for t < T-1; U[T-1] unchanged (reading 4). */
void orc_shift(int T, double* U);

/* Plant step: x0 <- Euler(x0, u0), psi wrapped to [-pi, pi); obstacles advanced by dt * vel. */
void orc_plant_step(const orc_params* p, double x0[4], const double u0[2], int n_obs,
                    double* obstacles);

/* ---- hitch-angle stabiliser, Sec. V-D (reading 28) ----------- */

/* Eq. (18): h_h = hitch_max - hitch_kappa |v| - |wrap(psi1 - psi2)|.  The reduced model has the speed
 * as an input, so "v(x)" is the speed applied over the step; |v| because the vehicle reverses. */
double orc_hitch_barrier(const orc_params* p, const double x[4], double v);

/* c(u) = [h_h(x_{k+1}) - h_h(x_k)] + alpha h_h(x_k) with |.| of the hitch angle expanded to first
 * order about x_k, i.e. the left side minus the right side of (3) in the sign of reading 1:
 *   c(u) = -s dt betadot(x_k, u) + hitch_alpha (hitch_max - hitch_kappa |v| - |beta|),
 * beta = wrap(psi1 - psi2), s = +1 if beta >= 0 else -1, betadot = psi1dot - psi2dot of eq. (6). */
double orc_hitch_rate_cond(const orc_params* p, const double x[4], const double u[2]);

/* First-order Taylor expansion of c in u about u_ref (the model is not affine in (v, delta)):
 * c(u) ~ *c0 + a . (u - u_ref).  d|v|/dv at v = 0 is taken as 0. */
void orc_hitch_constraint(const orc_params* p, const double x[4], const double u_ref[2],
                          double* c0, double a[2]);

/* u* = argmin_{u in box} q_v (v - v_ref)^2 + q_delta (delta - delta_ref)^2
 *      s.t. c0 + a . (u - u_ref) >= 0
 * solved by enumerating the active sets of the five constraints.  Returns 0 if the constraint is
 * inactive (u* = u_ref clamped into the box), 1 if it is active, 2 if box and half-plane do not
 * intersect; then u* is the point of the box with the largest a . u (coordinates with a_i = 0 keep
 * the clamped reference). */
int orc_hitch_filter(const orc_params* p, const double x[4], const double u_ref[2], double u_out[2]);

/* ---- the projected rollout: BR-MPPI proper, Sec. V-A (reading 30) ------
 *
 * At every prediction step the sampled inputs are projected onto the barrier-rate EQUALITY (9)
 *     L_f h_i(x) + L_g h_i(x) u = -(alpha_i + u^alpha_i) h_i(x),   i = 1..N_o,
 * by the closed form (12) of the soft-bounded weighted minimum-norm problem (11); the projected input
 * drives the model, the projected auxiliary input drives alpha_i.
 *
 * Readings taken for the reduced model (the paper's own model is the 7-state one):
 *  - inputs: the reduced eq. (6) is driftless and affine in w = (v, omega), omega := v tan(delta):
 *      x' = x + dt G(x) w,  G = [cos psi1, 0; sin psi1, 0; 0, 1/L1; sin(beta)/L2, -(Lh/(L1 L2)) cos(beta)],
 *    so f = 0, g = dt G and (9) is exact-affine in z = [w; u^alpha].  Sampled (v~, delta~) (perturbed and
 *    clamped as in the penalty path) give w_des = (v~, v~ tan delta~).
 *  - one constraint per obstacle, on the vehicle disc with the smallest h at x_tau
 *    (lowest index on ties): h_i = min_j h_ij.
 *  - L_g h_i = grad_x h_i . dt G(x);  L_f h_i = -(2/rho_i^2)(c - o_i) . dt vel_i: the obstacle's predicted
 *    motion (time-varying safe set), zero for a static one.
 *  - alpha_{i,0} = alpha_k for every obstacle (reading 8's per-sample draw), alpha_{i,tau+1} = alpha_{i,tau}
 *    + u^alpha_proj,i; u~^alpha_{i,tau} = sigma_ualpha zeta, zeta ~ N(0,1) from Philox counter
 *    (t, n, k, 2 + (i >> 2)), Box-Muller on words (0,1) -> zeta_0, zeta_1 and (2,3) -> zeta_2, zeta_3,
 *    obstacle i takes zeta_{i & 3}.
 *  - W = Diag(q_v, q_omega, q_alpha ... q_alpha);  z_lo / z_hi = (v_min, -omega_max, -ualpha_max ...) /
 *    (v_max, omega_max, ualpha_max ...), omega_max = max|v| tan(max|delta|).
 *  - stage cost on (x_{tau+1}, projected input): goal + heading + w_v v_p^2 + w_delta omega_p^2 + hitch
 *    hinge + w_alpha sum_i [h_i(x_{tau+1}, o_i(tau+1)) < h_buffer] max(0, alpha_{i,tau+1})^2 -- the
 *    "cost that motivates negative alpha within a buffer zone" (its exact form is in the
 *    paper's reference [1] only: PARITY UNPINNED).  No hinge penalty: the projection replaces it.
 *  - update (5) averages the SAMPLED u~ (PAPER.md:95 prints u~, not u_proj) with weights from the
 *    projected rollouts' costs.
 * Pins: tests/test_oracle_projected.py.
 */
typedef struct {
  double q_v, q_omega, q_alpha;   /* W = Diag(Q1, Q2), Q1 = diag(q_v, q_omega), Q2 = q_alpha I */
  double rho;                     /* soft-bound weight of (11a), >= 0                                          */
  double sigma_ualpha;            /* standard deviation of the sampled auxiliary inputs          */
  double ualpha_max;              /* u^alpha in [-ualpha_max, ualpha_max]: the z_lo / z_hi of (11)              */
  double w_alpha, h_buffer;       /* cost on alpha where h < h_buffer                            */
} orc_proj_params;

#define ORC_PROJ_MAX_NO 8

/* Eq. (12): z* = M^-1 [p - A^T (A M^-1 A^T)^-1 (A M^-1 p - b)], M = W + rho I,
 * p = W z_des + rho/2 (z_hi + z_lo); A is m x d row-major, W = diag(w).  The m x m system is solved by
 * Cholesky; a row whose pivot is not above 1e-14 times its own diagonal entry is dropped (multiplier 0).
 * Returns the number of dropped rows. */
int orc_project(int m, int d, const double* A, const double* b, const double* z_des, const double* w,
                double rho, const double* z_lo, const double* z_hi, double* z_out);

/* zeta[i], i < n_obs: the standard normals behind u~^alpha_{i,t} of sample k in iteration n. */
void orc_ualpha_normals(uint64_t seed, uint32_t n, uint32_t k, uint32_t t, int n_obs, double* zeta);

/* Row i of (9) at state x and step t: h = min_j h_ij(x, o(t)) (*jstar = its disc), Lg[2] = L_g h,
 * *Lf = L_f h.  obstacle = (cx, cy, R, vx, vy) at rollout time 0. */
void orc_barrier_row(const orc_params* p, const double x[4], const double* obstacle, int t, double* h,
                     int* jstar, double Lg[2], double* Lf);

/* x' = x + dt G(x) w, w = (v, omega). */
void orc_affine_step(const orc_params* p, const double x[4], const double w[2], double x_next[4]);

/* One projected rollout.  u[T][2]: sampled, clamped (v~, delta~); ualpha[T][n_obs]: sampled u~^alpha;
 * alpha0: initial alpha of every obstacle.  Optional outputs (NULL to skip): traj[(T+1)][4],
 * z_all[T][2 + n_obs] (projected z*), alpha_all[(T+1)][n_obs], Ab_all[T][n_obs][4] = (Lg0, Lg1, h, b). */
double orc_rollout_projected(const orc_params* p, const orc_proj_params* pp, const double x0[4],
                             const double goal[4], int n_obs, const double* obstacles, const double* u,
                             const double* ualpha, double alpha0, double xT[4], double* traj,
                             double* z_all, double* alpha_all, double* Ab_all);

double orc_sample_projected(const orc_params* p, const orc_proj_params* pp, uint32_t n, uint32_t k,
                            const double x0[4], const double goal[4], int n_obs, const double* obstacles,
                            const double* U_in, double* u /* T*2 */, double xT[4]);

int orc_iteration_projected(const orc_params* p, const orc_proj_params* pp, uint32_t n, const double x0[4],
                            const double goal[4], int n_obs, const double* obstacles, const double* U_in,
                            double* U_out, double* S, double* XT, double* u_all, double* w, int* argmin,
                            double* gap, double* eta, int n_threads);

/* ---- the paper's own model and tracking cost (reading 31) ------------------
 *
 * 7-state kinematic model with jerk and steering-rate inputs, eq. (6), state
 * x = [p^x, p^y, v, a, theta1, theta2, delta], u = [j, omega], explicit Euler as printed; second-order Taylor
 * predictor of the barrier, eq. (17); contouring / lag / heading / effort / progress cost,
 * eq. (13)-(15) PAPER.md:196-212, along a reference path zeta(psi) given as cubic splines in arc length.
 *
 * Readings where the paper is silent:
 *  - reference path: M cubic segments on uniform knots psi_m = m dpsi for each of (p^{x,r}, p^{y,r}, theta^{1,r},
 *    theta^{2,r}): value = c0 + c1 s + c2 s^2 + c3 s^3, s = psi - m dpsi, m = min(floor(psi / dpsi), M - 1), psi
 *    clamped to [0, M dpsi] ("third-order spline");
 *  - path parameter: psi_{k+1} = clamp(psi_k + T_s nu_k), nu_k = v_k cos(theta1_k - theta^{1,r}(psi_k)) -- "the
 *    projection velocity along the reference path";
 *  - delta is clamped to [delta_lo, delta_hi] after its Euler update (steering stops); v and a are free;
 *  - stage cost on (x_{k+1}, u_k, psi_{k+1}) (reading 3): Q_c e_c^2 + Q_l e_l^2 + Q_th1 e_th1^2 + Q_th2 e_th2^2
 *    + R_j j^2 + R_w omega^2 + mu (nu_bar - nu_{k+1})^2 + the hitch hinge of reading 15 (with |v_{k+1}|)
 *    + w_bar * sum_{i,j} max(0, (1 - alpha) h_ij(x_k, o_i(k)) - hhat_ij(x_k, u_k)): the barrier-rate condition
 *    of the penalty path with h(x_{k+1}) replaced by the predictor (17), whose hdot and hddot are the first and
 *    second Lie derivatives of h (disc j against obstacle i, reading 10) along the continuous model under the
 *    sampled input -- hddot depends on omega through d(delta)/dt, not on j (relative degree 3);
 *    terminal cost w_term * (the four tracking terms at (x_N, psi_N));
 *  - sampled inputs: clamp(U + sigma z) on (j, omega), same noise stream as the penalty path; alpha per sample
 *    (reading 8); update (5) on (j, omega).
 * Pins: tests/test_oracle_mpcc.py.  The weights are never printed in the paper (PARITY UNPINNED, like the
 * penalty path's). */
typedef struct {
  double j_min, j_max, omega_min, omega_max;     /* j in [-2, 2] m/s^3, omega in [-0.9, 0.9] rad/s */
  double sigma_j, sigma_omega;
  double delta_lo, delta_hi;
  double Qc, Ql, Qth1, Qth2, Rj, Rw, mu, nu_bar; /* weights of (13)                                             */
  int M;                                         /* cubic segments of the reference path                        */
  double dpsi;                                   /* knot spacing in arc length                                  */
  const double* coef;                            /* [M][4 components][4 coefficients c0..c3]                    */
} orc_mpcc_params;

/* eq. (6), explicit Euler, delta clamped. */
void orc7_step(const orc_params* p, const orc_mpcc_params* mp, const double x[7], const double u[2], double xn[7]);
/* (p^{x,r}, p^{y,r}, theta^{1,r}, theta^{2,r}) at arc length psi. */
void orc_path_eval(const orc_mpcc_params* mp, double psi, double out[4]);
/* nu = v cos(theta1 - theta^{1,r}(psi)). */
double orc7_progress(const orc_mpcc_params* mp, const double x[7], double psi);
/* (e^c, e^l, e^theta1, e^theta2) of (14), (15) and PAPER.md:212 (heading errors wrapped). */
void orc7_errors(const orc_mpcc_params* mp, const double x[7], double psi, double e[4]);
/* Predictor (17) for vehicle disc j against obstacle (cx, cy, R, vx, vy) at step t: returns hhat, *h = h(x). */
double orc7_hhat(const orc_params* p, const double x[7], const double u[2], const double* obstacle, int t,
                 int j, double* h);
/* One rollout under sampled, clamped inputs u[T][2]; xT[8] = final state and psi; traj (optional) [(T+1)][8]. */
double orc7_rollout(const orc_params* p, const orc_mpcc_params* mp, const double x0[7], double psi0, int n_obs,
                    const double* obstacles, const double* u, double alpha, double xT[8], double* traj);
double orc7_sample(const orc_params* p, const orc_mpcc_params* mp, uint32_t n, uint32_t k, const double x0[7],
                   double psi0, int n_obs, const double* obstacles, const double* U_in, double* u, double xT[8]);
int orc7_iteration(const orc_params* p, const orc_mpcc_params* mp, uint32_t n, const double x0[7], double psi0,
                   int n_obs, const double* obstacles, const double* U_in, double* U_out, double* S, double* XT,
                   double* u_all, double* w, int* argmin, double* gap, double* eta, int n_threads);

#ifdef __cplusplus
}
#endif
#endif
