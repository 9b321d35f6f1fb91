/*
 * brmppi_oracle.c -- CPU oracle (fp64, single pass, no blocking / fusion / reordering).
 * TEST INFRASTRUCTURE ONLY; see brmppi_oracle.h for the passages followed and the pin status.
 *
 * Build:  gcc -O2 -std=c11 -fPIC -shared -o liboracle.so brmppi_oracle.c -lm -lpthread
 *         (-ffp-contract=off so that the result does not depend on FMA availability)
 */
#include <math.h>
#include <pthread.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef ORC_FP32
/* Reading 23: the fp32 re-run mode.  The SAME source with every `double` a `float`, libm's
 * single-precision functions and (gcc -fsingle-precision-constant) single-precision literals: what a careful fp32
 * implementation of these very formulas returns, rounding after every operation.  It exists only so that the tests
 * can print the fp32 noise floor next to each tolerance (oracle/oracle32.py, tests/test_oracle_fp32_floor.py); the
 * GPU path is never compared with it, and the fp64 build below is untouched by it.
 * Build:  gcc -O2 -std=c11 -ffp-contract=off -DORC_FP32 -fsingle-precision-constant -fPIC -shared
 *             -o liboracle32.so brmppi_oracle.c -lm -lpthread */
#define double float
#define cos cosf
#define sin sinf
#define tan tanf
#define sqrt sqrtf
#define log logf
#define exp expf
#define pow powf
#define fabs fabsf
#define fmin fminf
#define fmax fmaxf
#define rint rintf
#define floor floorf
#endif

#include "brmppi_oracle.h"

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

/* ------------------------------------------------------------------------------------------
 * Philox4x32-10.  J. K. Salmon, M. A. Moraes, R. O. Dror, D. E. Shaw, "Parallel random
 * numbers: as easy as 1, 2, 3", SC'11.  One round:
 *   (hi0, lo0) = M0 * c0;  (hi1, lo1) = M1 * c2;
 *   (c0, c1, c2, c3) <- (hi1 ^ c1 ^ k0,  lo1,  hi0 ^ c3 ^ k1,  lo0)
 * and the key is bumped by (W0, W1) between rounds (not after the last).
 * ---------------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
  const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)M0 * (uint64_t)c0;
    uint64_t p1 = (uint64_t)M1 * (uint64_t)c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += W0; k1 += W1;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

double orc_uniform(uint32_t w) { return (double)(w >> 9) * (1.0 / 8388608.0); }

static void seed_key(uint64_t seed, uint32_t key[2]) {
  key[0] = (uint32_t)(seed & 0xFFFFFFFFu);
  key[1] = (uint32_t)(seed >> 32);
}

/* PAPER.md:89 "draws S independent noise rollouts w ~ N(0, Sigma_w)"; readings 5 and 6: Box-Muller on
 * two 23-bit uniforms.  One Philox block, counter (t >> 1, n, k, 0), serves the two steps 2m and
 * 2m + 1: words (0, 1) for the even step, words (2, 3) for the odd one. */
void orc_normals(uint64_t seed, uint32_t n, uint32_t k, uint32_t t, double z[2]) {
  uint32_t key[2], ctr[4] = {t >> 1, n, k, 0u}, w[4];
  seed_key(seed, key);
  orc_philox4x32_10(ctr, key, w);
  const uint32_t wa = (t & 1u) ? w[2] : w[0];
  const uint32_t wb = (t & 1u) ? w[3] : w[1];
  double u1 = 1.0 - orc_uniform(wa); /* in (0, 1] */
  double u2 = orc_uniform(wb);       /* in [0, 1) */
  double r = sqrt(-2.0 * log(u1));
  z[0] = r * cos(2.0 * M_PI * u2);
  z[1] = r * sin(2.0 * M_PI * u2);
}

/* Reading 8: one alpha per sample, U[alpha_lo, alpha_hi), Philox counter (0, n, k, 1). */
double orc_alpha(const orc_params* p, uint32_t n, uint32_t k) {
  uint32_t key[2], ctr[4] = {0u, n, k, 1u}, w[4];
  seed_key(p->seed, key);
  orc_philox4x32_10(ctr, key, w);
  return p->alpha_lo + (p->alpha_hi - p->alpha_lo) * orc_uniform(w[0]);
}

double orc_wrap(double a) { return a - 2.0 * M_PI * rint(a / (2.0 * M_PI)); }

static double clampd(double x, double lo, double hi) { return x < lo ? lo : (x > hi ? hi : x); }

/* Reduced eq. (6): explicit Euler, every right-hand side at step k. */
void orc_kinematic_step(const orc_params* p, const double x[4], double v, double delta,
                        double xn[4]) {
  double px = x[0], py = x[1], psi1 = x[2], psi2 = x[3];
  double td = tan(delta);
  double beta = psi1 - psi2;
  xn[0] = px + p->dt * v * cos(psi1);
  xn[1] = py + p->dt * v * sin(psi1);
  xn[2] = psi1 + p->dt * (v / p->L1) * td;
  xn[3] = psi2 + p->dt * (v / p->L2) * (sin(beta) - (p->Lh / p->L1) * cos(beta) * td);
}

/* Hitch point p_h = (x - Lh cos psi1, y - Lh sin psi1); disc centre = p_h + offset * body axis
 * ("cover the vehicle body with discs of radius r"; reading 11). */
void orc_disc_centre(const orc_params* p, const double x[4], int j, double c[2]) {
  double hx = x[0] - p->Lh * cos(x[2]);
  double hy = x[1] - p->Lh * sin(x[2]);
  double psi = (p->disc_body[j] == 0) ? x[2] : x[3];
  c[0] = hx + p->disc_offset[j] * cos(psi);
  c[1] = hy + p->disc_offset[j] * sin(psi);
}

/* Eq. (16) with e = 2, m_x = m_y = R, inflated by the vehicle disc radius. */
double orc_barrier(const orc_params* p, const double c[2], const double o[2], double R) {
  double rho = R + p->disc_radius;
  double dx = c[0] - o[0], dy = c[1] - o[1];
  return (dx * dx + dy * dy) / (rho * rho) - 1.0;
}

/* Eq. (16): obstacle frame p' = R(-theta_o)(c - o), semi-axes inflated by the
 * vehicle disc radius, exponent e >= 2 (even e in the paper: 4 for parked cars, 2 for pedestrians;
 * |.| makes odd or fractional e well defined too).  se = (cx, cy, m_x, m_y, theta, vx, vy, e). */
double orc_barrier_se(const orc_params* p, const double c[2], const double o[2], const double* se) {
  double ct = cos(se[4]), st = sin(se[4]);
  double dx = c[0] - o[0], dy = c[1] - o[1];
  double xp = ct * dx + st * dy;
  double yp = -st * dx + ct * dy;
  double ax = se[2] + p->disc_radius, ay = se[3] + p->disc_radius;
  return pow(fabs(xp) / ax, se[7]) + pow(fabs(yp) / ay, se[7]) - 1.0;
}

double orc_goal_cost(const orc_params* p, const double x[4], const double g[4]) {
  double ex = x[0] - g[0], ey = x[1] - g[1];
  double e1 = orc_wrap(x[2] - g[2]), e2 = orc_wrap(x[3] - g[3]);
  return p->w_pos * (ex * ex + ey * ey) + p->w_head * (e1 * e1 + e2 * e2);
}

/* Obstacle i at rollout step t: constant-velocity prediction (Assumption 2). */
static void obstacle_at(const orc_params* p, const double* obstacles, int i, int t, double o[2]) {
  const double* ob = obstacles + 5 * i;
  o[0] = ob[0] + (double)t * p->dt * ob[3];
  o[1] = ob[1] + (double)t * p->dt * ob[4];
}

double orc_rollout_se(const orc_params* p, const double x0[4], const double goal[4], int n_obs,
                      const double* obstacles, int n_se, const double* se, const double* u,
                      double alpha, double xT[4], double* traj, double* pen_out) {
  const int T = p->T, D = p->n_discs;
  double X[4] = {x0[0], x0[1], x0[2], x0[3]};
  double S = 0.0, pen_total = 0.0;
  double* hprev = (double*)malloc(sizeof(double) * (size_t)(n_obs > 0 ? n_obs : 1) * ORC_MAX_DISCS);
  double* hprev_se = (double*)malloc(sizeof(double) * (size_t)(n_se > 0 ? n_se : 1) * ORC_MAX_DISCS);

  /* h at (x_0, o(0)) */
  for (int i = 0; i < n_obs; ++i) {
    double o[2];
    obstacle_at(p, obstacles, i, 0, o);
    for (int j = 0; j < D; ++j) {
      double c[2];
      orc_disc_centre(p, X, j, c);
      hprev[i * ORC_MAX_DISCS + j] = orc_barrier(p, c, o, obstacles[5 * i + 2]);
    }
  }
  for (int i = 0; i < n_se; ++i) {   /* super-ellipse obstacles, same pairing of state and time */
    double o[2] = {se[8 * i + 0], se[8 * i + 1]};
    for (int j = 0; j < D; ++j) {
      double c[2];
      orc_disc_centre(p, X, j, c);
      hprev_se[i * ORC_MAX_DISCS + j] = orc_barrier_se(p, c, o, se + 8 * i);
    }
  }
  if (traj) memcpy(traj, X, sizeof(X));

  for (int t = 0; t < T; ++t) {
    double v = u[2 * t + 0], d = u[2 * t + 1];
    double Xn[4];
    orc_kinematic_step(p, X, v, d, Xn);

    /* barrier-rate condition h_{t+1} - h_t >= -alpha h_t (reading 1) as a
     * linear hinge penalty summed over obstacles and discs (reading 14);
     * h_{t+1} pairs x_{t+1} with o(t+1) (reading 13). */
    double pen = 0.0;
    for (int i = 0; i < n_obs; ++i) {
      double o[2];
      obstacle_at(p, obstacles, i, t + 1, o);
      for (int j = 0; j < D; ++j) {
        double c[2];
        orc_disc_centre(p, Xn, j, c);
        double hn = orc_barrier(p, c, o, obstacles[5 * i + 2]);
        double viol = (1.0 - alpha) * hprev[i * ORC_MAX_DISCS + j] - hn;
        if (viol > 0.0) pen += viol;
        hprev[i * ORC_MAX_DISCS + j] = hn;
      }
    }
    for (int i = 0; i < n_se; ++i) {
      double o[2] = {se[8 * i + 0] + (double)(t + 1) * p->dt * se[8 * i + 5],
                     se[8 * i + 1] + (double)(t + 1) * p->dt * se[8 * i + 6]};
      for (int j = 0; j < D; ++j) {
        double c[2];
        orc_disc_centre(p, Xn, j, c);
        double hn = orc_barrier_se(p, c, o, se + 8 * i);
        double viol = (1.0 - alpha) * hprev_se[i * ORC_MAX_DISCS + j] - hn;
        if (viol > 0.0) pen += viol;
        hprev_se[i * ORC_MAX_DISCS + j] = hn;
      }
    }
    pen_total += pen;

    /* stage cost on (x_{t+1}, u_t) (reading 3); hitch: squared hinge beyond the velocity-dependent
     * limit Delta_theta_max - kappa |v| of eq. (18) (reading 15, kappa = 0 in CFG0-4) */
    double hitch = fabs(orc_wrap(Xn[2] - Xn[3])) - (p->hitch_max - p->hitch_kappa * fabs(v));
    if (hitch < 0.0) hitch = 0.0;
    S += orc_goal_cost(p, Xn, goal) + p->w_v * v * v + p->w_delta * d * d +
         p->w_hitch * hitch * hitch + p->w_bar * pen;

    memcpy(X, Xn, sizeof(X));
    if (traj) memcpy(traj + 4 * (t + 1), X, sizeof(X));
  }
  S += p->w_term * orc_goal_cost(p, X, goal); /* terminal cost r_N(x_N), eq. (7) */
  memcpy(xT, X, sizeof(X));
  if (pen_out) *pen_out = pen_total;
  free(hprev);
  free(hprev_se);
  return S;
}

double orc_rollout(const orc_params* p, const double x0[4], const double goal[4], int n_obs,
                   const double* obstacles, const double* u, double alpha, double xT[4],
                   double* traj, double* pen_out) {
  return orc_rollout_se(p, x0, goal, n_obs, obstacles, 0, NULL, u, alpha, xT, traj, pen_out);
}

int orc_weights_update(int K, int T, double lambda, const double* S, const double* u,
                       double* U_out, double* w, int* argmin, double* gap, double* eta) {
  int kstar = -1, nonfinite = 0;
  double s1 = INFINITY, s2 = INFINITY;
  for (int k = 0; k < K; ++k) {
    if (!isfinite(S[k])) { ++nonfinite; continue; }
    if (S[k] < s1) { s2 = s1; s1 = S[k]; kstar = k; }   /* strict: lowest index wins ties */
    else if (S[k] < s2) { s2 = S[k]; }
  }
  if (argmin) *argmin = kstar;
  if (gap) *gap = s2 - s1;
  if (kstar < 0) { if (eta) *eta = 0.0; return nonfinite; }

  /* gamma_s = exp(-(J_s - min_j J_j)/lambda) */
  double sum_w = 0.0;
  double* wk = (double*)malloc(sizeof(double) * (size_t)K);
  for (int k = 0; k < K; ++k) {
    wk[k] = isfinite(S[k]) ? exp(-(S[k] - s1) / lambda) : 0.0;
    sum_w += wk[k];
  }
  /* u_nom <- sum_s gamma_bar_s u~_s, eq. (5) */
  for (int t = 0; t < 2 * T; ++t) {
    double acc = 0.0;
    for (int k = 0; k < K; ++k) acc += wk[k] * u[(size_t)k * 2 * T + t];
    U_out[t] = acc / sum_w;
  }
  if (w) memcpy(w, wk, sizeof(double) * (size_t)K);
  if (eta) *eta = sum_w;
  free(wk);
  return nonfinite;
}

typedef struct {
  const orc_params* p;
  uint32_t n;
  const double *x0, *goal, *obstacles, *U_in;
  int n_obs, k_begin, k_end;
  double *S, *XT, *u_all;
  int n_se;
  const double* se;
} sample_job;

/* Sample k of iteration n: draw alpha_k and the perturbed, clamped controls, roll out. */
double orc_sample_se(const orc_params* p, uint32_t n, uint32_t k, const double x0[4],
                     const double goal[4], int n_obs, const double* obstacles, int n_se,
                     const double* se, const double* U_in, double* u /* T*2 */, double xT[4]) {
  const int T = p->T;
  double alpha = orc_alpha(p, n, k);
  for (int t = 0; t < T; ++t) {
    double z[2];
    orc_normals(p->seed, n, k, (uint32_t)t, z);
    /* u~ = u_nom + w~, hard clamp to the control bounds (reading 9) */
    u[2 * t + 0] = clampd(U_in[2 * t + 0] + p->sigma_v * z[0], p->v_min, p->v_max);
    u[2 * t + 1] = clampd(U_in[2 * t + 1] + p->sigma_delta * z[1], p->delta_min, p->delta_max);
  }
  return orc_rollout_se(p, x0, goal, n_obs, obstacles, n_se, se, u, alpha, xT, NULL, NULL);
}

double orc_sample(const orc_params* p, uint32_t n, uint32_t k, const double x0[4],
                  const double goal[4], int n_obs, const double* obstacles, const double* U_in,
                  double* u /* T*2 */, double xT[4]) {
  return orc_sample_se(p, n, k, x0, goal, n_obs, obstacles, 0, NULL, U_in, u, xT);
}

static void* sample_worker(void* arg) {
  sample_job* job = (sample_job*)arg;
  const int T = job->p->T;
  for (int k = job->k_begin; k < job->k_end; ++k)
    job->S[k] = orc_sample_se(job->p, job->n, (uint32_t)k, job->x0, job->goal, job->n_obs,
                              job->obstacles, job->n_se, job->se, job->U_in,
                              job->u_all + (size_t)k * 2 * T, job->XT + 4 * (size_t)k);
  return NULL;
}

int orc_iteration_se(const orc_params* p, uint32_t n, const double x0[4], const double goal[4],
                     int n_obs, const double* obstacles, int n_se, const double* se,
                     const double* U_in, double* U_out,
                  double* S, double* XT, double* u_all, double* w, int* argmin, double* gap,
                  double* eta, int n_threads) {
  const int K = p->K, T = p->T;
  double* S_buf = S ? S : (double*)malloc(sizeof(double) * (size_t)K);
  double* XT_buf = XT ? XT : (double*)malloc(sizeof(double) * 4 * (size_t)K);
  double* u_buf = u_all ? u_all : (double*)malloc(sizeof(double) * 2 * (size_t)T * (size_t)K);
  double* U_nom = (double*)malloc(sizeof(double) * 2 * (size_t)T);
  memcpy(U_nom, U_in, sizeof(double) * 2 * (size_t)T);

  if (n_threads < 1) n_threads = 1;
  if (n_threads > K) n_threads = K;
  sample_job* jobs = (sample_job*)malloc(sizeof(sample_job) * (size_t)n_threads);
  pthread_t* tids = (pthread_t*)malloc(sizeof(pthread_t) * (size_t)n_threads);
  for (int i = 0; i < n_threads; ++i) {
    jobs[i] = (sample_job){p, n, x0, goal, obstacles, U_nom, n_obs,
                           (int)((long long)K * i / n_threads),
                           (int)((long long)K * (i + 1) / n_threads), S_buf, XT_buf, u_buf, n_se, se};
  }
  if (n_threads == 1) {
    sample_worker(&jobs[0]);
  } else {
    for (int i = 0; i < n_threads; ++i) pthread_create(&tids[i], NULL, sample_worker, &jobs[i]);
    for (int i = 0; i < n_threads; ++i) pthread_join(tids[i], NULL);
  }

  /* U_out keeps U_in if every cost is non-finite */
  if (U_out != U_in) memcpy(U_out, U_nom, sizeof(double) * 2 * (size_t)T);
  int nonfinite = orc_weights_update(K, T, p->lambda, S_buf, u_buf, U_out, w, argmin, gap, eta);

  free(jobs); free(tids); free(U_nom);
  if (!S) free(S_buf);
  if (!XT) free(XT_buf);
  if (!u_all) free(u_buf);
  return nonfinite;
}

int orc_iteration(const orc_params* p, uint32_t n, const double x0[4], const double goal[4],
                  int n_obs, const double* obstacles, const double* U_in, double* U_out,
                  double* S, double* XT, double* u_all, double* w, int* argmin, double* gap,
                  double* eta, int n_threads) {
  return orc_iteration_se(p, n, x0, goal, n_obs, obstacles, 0, NULL, U_in, U_out, S, XT, u_all, w,
                          argmin, gap, eta, n_threads);
}

/* Super-ellipse obstacles advance like discs: centre += dt * velocity (orientation fixed). */
void orc_advance_se(const orc_params* p, int n_se, double* se) {
  for (int i = 0; i < n_se; ++i) {
    se[8 * i + 0] += p->dt * se[8 * i + 5];
    se[8 * i + 1] += p->dt * se[8 * i + 6];
  }
}

void orc_shift(int T, double* U) {
  for (int t = 0; t + 1 < T; ++t) {
    U[2 * t + 0] = U[2 * (t + 1) + 0];
    U[2 * t + 1] = U[2 * (t + 1) + 1];
  }
}

void orc_plant_step(const orc_params* p, double x0[4], const double u0[2], int n_obs,
                    double* obstacles) {
  double xn[4];
  orc_kinematic_step(p, x0, u0[0], u0[1], xn);
  xn[2] = orc_wrap(xn[2]);
  xn[3] = orc_wrap(xn[3]);
  memcpy(x0, xn, sizeof(xn));
  for (int i = 0; i < n_obs; ++i) {
    obstacles[5 * i + 0] += p->dt * obstacles[5 * i + 3];
    obstacles[5 * i + 1] += p->dt * obstacles[5 * i + 4];
  }
}

/* ------------------------------------------------------------------------------------------
 * Hitch-angle stabiliser, Sec. V-D, reading 28.
 * ---------------------------------------------------------------------------------------- */

/* Eq. (18). */
double orc_hitch_barrier(const orc_params* p, const double x[4], double v) {
  double beta = orc_wrap(x[2] - x[3]);
  return p->hitch_max - p->hitch_kappa * fabs(v) - fabs(beta);
}

/* psi1dot - psi2dot of the reduced eq. (6). */
static double hitch_rate(const orc_params* p, double beta, double v, double delta) {
  double td = tan(delta);
  double psi1dot = (v / p->L1) * td;
  double psi2dot = (v / p->L2) * (sin(beta) - (p->Lh / p->L1) * cos(beta) * td);
  return psi1dot - psi2dot;
}

double orc_hitch_rate_cond(const orc_params* p, const double x[4], const double u[2]) {
  double beta = orc_wrap(x[2] - x[3]);
  double s = (beta >= 0.0) ? 1.0 : -1.0;
  return -s * p->dt * hitch_rate(p, beta, u[0], u[1]) + p->hitch_alpha * orc_hitch_barrier(p, x, u[0]);
}

void orc_hitch_constraint(const orc_params* p, const double x[4], const double u_ref[2],
                          double* c0, double a[2]) {
  double beta = orc_wrap(x[2] - x[3]);
  double s = (beta >= 0.0) ? 1.0 : -1.0;
  double v = u_ref[0], delta = u_ref[1];
  double td = tan(delta), cd = cos(delta);
  double sgn_v = (v > 0.0) ? 1.0 : ((v < 0.0) ? -1.0 : 0.0);
  /* d betadot / d v      = tan(delta)/L1 - (sin beta - (Lh/L1) cos beta tan(delta))/L2
   * d betadot / d delta  = v (1/L1 + Lh cos beta/(L1 L2)) / cos^2(delta)                   */
  double dv = td / p->L1 - (sin(beta) - (p->Lh / p->L1) * cos(beta) * td) / p->L2;
  double dd = v * (1.0 / p->L1 + p->Lh * cos(beta) / (p->L1 * p->L2)) / (cd * cd);
  *c0 = orc_hitch_rate_cond(p, x, u_ref);
  a[0] = -s * p->dt * dv - p->hitch_alpha * p->hitch_kappa * sgn_v;
  a[1] = -s * p->dt * dd;
}

int orc_hitch_filter(const orc_params* p, const double x[4], const double u_ref[2], double u_out[2]) {
  const double lo[2] = {p->v_min, p->delta_min}, hi[2] = {p->v_max, p->delta_max};
  const double q[2] = {p->hitch_qv, p->hitch_qdelta};
  double c0, a[2];
  orc_hitch_constraint(p, x, u_ref, &c0, a);

  /* Constraint lines n . u = r: the half-plane boundary and the four box edges. */
  double n[5][2] = {{a[0], a[1]}, {1, 0}, {1, 0}, {0, 1}, {0, 1}};
  double r[5] = {a[0] * u_ref[0] + a[1] * u_ref[1] - c0, lo[0], hi[0], lo[1], hi[1]};

  /* Candidates: the unconstrained minimiser, its Q-projection on each line, every pairwise
   * intersection of lines.  The minimiser of a strictly convex QP is the minimiser over the
   * affine hull of its active constraints, hence one of these. */
  double cand[16][2];
  int nc = 0;
  cand[nc][0] = u_ref[0]; cand[nc][1] = u_ref[1]; ++nc;
  for (int i = 0; i < 5; ++i) {
    double nqn = n[i][0] * n[i][0] / q[0] + n[i][1] * n[i][1] / q[1];
    if (nqn == 0.0) continue;
    double mu = (r[i] - n[i][0] * u_ref[0] - n[i][1] * u_ref[1]) / nqn;
    cand[nc][0] = u_ref[0] + mu * n[i][0] / q[0];
    cand[nc][1] = u_ref[1] + mu * n[i][1] / q[1];
    ++nc;
  }
  for (int i = 0; i < 5; ++i)
    for (int j = i + 1; j < 5; ++j) {
      double det = n[i][0] * n[j][1] - n[i][1] * n[j][0];
      if (det == 0.0) continue;
      cand[nc][0] = (r[i] * n[j][1] - n[i][1] * r[j]) / det;
      cand[nc][1] = (n[i][0] * r[j] - r[i] * n[j][0]) / det;
      ++nc;
    }

  const double eps = 1e-12;
  double scale = fabs(c0) + fabs(a[0]) * (hi[0] - lo[0]) + fabs(a[1]) * (hi[1] - lo[1]) + 1e-300;
  int best = -1;
  double best_J = 0.0;
  for (int m = 0; m < nc; ++m) {
    double v = cand[m][0], d = cand[m][1];
    if (v < lo[0] - eps * (hi[0] - lo[0]) || v > hi[0] + eps * (hi[0] - lo[0])) continue;
    if (d < lo[1] - eps * (hi[1] - lo[1]) || d > hi[1] + eps * (hi[1] - lo[1])) continue;
    double g = c0 + a[0] * (v - u_ref[0]) + a[1] * (d - u_ref[1]);
    if (g < -eps * scale) continue;
    double J = q[0] * (v - u_ref[0]) * (v - u_ref[0]) + q[1] * (d - u_ref[1]) * (d - u_ref[1]);
    if (best < 0 || J < best_J) { best = m; best_J = J; }
  }
  double uc[2];
  for (int i = 0; i < 2; ++i) uc[i] = fmin(fmax(u_ref[i], lo[i]), hi[i]);
  if (best < 0) {
    for (int i = 0; i < 2; ++i) u_out[i] = (a[i] > 0.0) ? hi[i] : ((a[i] < 0.0) ? lo[i] : uc[i]);
    return 2;
  }
  for (int i = 0; i < 2; ++i) u_out[i] = fmin(fmax(cand[best][i], lo[i]), hi[i]);
  double g_ref = c0 + a[0] * (uc[0] - u_ref[0]) + a[1] * (uc[1] - u_ref[1]);
  return (g_ref >= 0.0) ? 0 : 1;
}

/* ------------------------------------------------------------------------------------------
 * The projected rollout: BR-MPPI proper, Sec. V-A; readings in the header.
 * ---------------------------------------------------------------------------------------- */

/* Eq. (12). */
int orc_project(int m, int d, const double* A, const double* b, const double* z_des, const double* w,
                double rho, const double* z_lo, const double* z_hi, double* z_out) {
  double Minv[2 + ORC_PROJ_MAX_NO], pvec[2 + ORC_PROJ_MAX_NO], y[2 + ORC_PROJ_MAX_NO];
  double S[ORC_PROJ_MAX_NO][ORC_PROJ_MAX_NO], r[ORC_PROJ_MAX_NO], nu[ORC_PROJ_MAX_NO], diag0[ORC_PROJ_MAX_NO];
  int dropped_row[ORC_PROJ_MAX_NO], dropped = 0;
  for (int j = 0; j < d; ++j) {
    Minv[j] = 1.0 / (w[j] + rho);                                /* M = W + rho I, diagonal        */
    pvec[j] = w[j] * z_des[j] + 0.5 * rho * (z_hi[j] + z_lo[j]); /* p = W z_des + rho/2 (z_hi+z_lo) */
    y[j] = Minv[j] * pvec[j];                                    /* M^-1 p                          */
  }
  for (int i = 0; i < m; ++i) {
    double acc = -b[i];
    for (int j = 0; j < d; ++j) acc += A[i * d + j] * y[j];
    r[i] = acc;                                                  /* A M^-1 p - b                    */
    for (int k = 0; k < m; ++k) {
      double s = 0.0;
      for (int j = 0; j < d; ++j) s += A[i * d + j] * Minv[j] * A[k * d + j];
      S[i][k] = s;                                               /* A M^-1 A^T                      */
    }
    diag0[i] = S[i][i];
  }
  /* Cholesky S = L L^T in place (lower triangle), then L w = r, L^T nu = w */
  for (int k = 0; k < m; ++k) {
    double dkk = S[k][k];
    for (int q = 0; q < k; ++q) dkk -= S[k][q] * S[k][q];
    dropped_row[k] = !(dkk > 1e-14 * diag0[k]);
    if (dropped_row[k]) {
      ++dropped;
      S[k][k] = 1.0;
      for (int i = k + 1; i < m; ++i) S[i][k] = 0.0;
      for (int q = 0; q < k; ++q) S[k][q] = 0.0;
      r[k] = 0.0;
      continue;
    }
    S[k][k] = sqrt(dkk);
    for (int i = k + 1; i < m; ++i) {
      double v = S[i][k];
      for (int q = 0; q < k; ++q) v -= S[i][q] * S[k][q];
      S[i][k] = v / S[k][k];
    }
  }
  for (int i = 0; i < m; ++i) {
    double v = r[i];
    for (int q = 0; q < i; ++q) v -= S[i][q] * nu[q];
    nu[i] = v / S[i][i];
  }
  for (int i = m - 1; i >= 0; --i) {
    double v = nu[i];
    for (int q = i + 1; q < m; ++q) v -= S[q][i] * nu[q];
    nu[i] = v / S[i][i];
    if (dropped_row[i]) nu[i] = 0.0;
  }
  for (int j = 0; j < d; ++j) {
    double acc = pvec[j];
    for (int i = 0; i < m; ++i) acc -= A[i * d + j] * nu[i];
    z_out[j] = Minv[j] * acc;                                    /* M^-1 (p - A^T nu)               */
  }
  return dropped;
}

/* u~^alpha draws: counter (t, n, k, 2 + (i >> 2)); Box-Muller on (w0, w1) and (w2, w3). */
void orc_ualpha_normals(uint64_t seed, uint32_t n, uint32_t k, uint32_t t, int n_obs, double* zeta) {
  uint32_t key[2];
  seed_key(seed, key);
  for (int q = 0; 4 * q < n_obs; ++q) {
    uint32_t ctr[4] = {t, n, k, 2u + (uint32_t)q}, w[4];
    orc_philox4x32_10(ctr, key, w);
    double z4[4];
    for (int h = 0; h < 2; ++h) {
      double u1 = 1.0 - orc_uniform(w[2 * h]);
      double u2 = orc_uniform(w[2 * h + 1]);
      double rr = sqrt(-2.0 * log(u1));
      z4[2 * h + 0] = rr * cos(2.0 * M_PI * u2);
      z4[2 * h + 1] = rr * sin(2.0 * M_PI * u2);
    }
    for (int e = 0; e < 4 && 4 * q + e < n_obs; ++e) zeta[4 * q + e] = z4[e];
  }
}

/* Row i of (9): h_i on the closest disc, L_g h_i = grad_x h_i . dt G(x), L_f h_i from the
 * obstacle's predicted motion. */
void orc_barrier_row(const orc_params* p, const double x[4], const double* ob, int t, double* h_out,
                     int* jstar, double Lg[2], double* Lf) {
  double o[2] = {ob[0] + (double)t * p->dt * ob[3], ob[1] + (double)t * p->dt * ob[4]};
  double rho = ob[2] + p->disc_radius;
  int jbest = 0;
  double hbest = 0.0, cbest[2] = {0.0, 0.0};
  for (int j = 0; j < p->n_discs; ++j) {
    double c[2];
    orc_disc_centre(p, x, j, c);
    double h = orc_barrier(p, c, o, ob[2]);
    if (j == 0 || h < hbest) { hbest = h; jbest = j; cbest[0] = c[0]; cbest[1] = c[1]; }
  }
  double psi1 = x[2], psi2 = x[3], beta = psi1 - psi2;
  /* grad of h wrt the disc centre, then the chain rule through c(x) = p_h + a e(psi_body),
   * p_h = (x - Lh cos psi1, y - Lh sin psi1) */
  double gx = 2.0 * (cbest[0] - o[0]) / (rho * rho), gy = 2.0 * (cbest[1] - o[1]) / (rho * rho);
  double a = p->disc_offset[jbest];
  double dc1x = p->Lh * sin(psi1), dc1y = -p->Lh * cos(psi1);   /* d p_h / d psi1 */
  double dc2x = 0.0, dc2y = 0.0;
  if (p->disc_body[jbest] == 0) { dc1x += -a * sin(psi1); dc1y += a * cos(psi1); }
  else { dc2x = -a * sin(psi2); dc2y = a * cos(psi2); }
  double dh_dx = gx, dh_dy = gy;
  double dh_dpsi1 = gx * dc1x + gy * dc1y;
  double dh_dpsi2 = gx * dc2x + gy * dc2y;
  /* columns of G(x): d/dv = (cos psi1, sin psi1, 0, sin(beta)/L2), d/domega = (0, 0, 1/L1, -(Lh/(L1 L2)) cos beta) */
  Lg[0] = p->dt * (dh_dx * cos(psi1) + dh_dy * sin(psi1) + dh_dpsi2 * sin(beta) / p->L2);
  Lg[1] = p->dt * (dh_dpsi1 / p->L1 - dh_dpsi2 * (p->Lh / (p->L1 * p->L2)) * cos(beta));
  *Lf = -p->dt * (gx * ob[3] + gy * ob[4]);
  *h_out = hbest;
  *jstar = jbest;
}

void orc_affine_step(const orc_params* p, const double x[4], const double w[2], double xn[4]) {
  double psi1 = x[2], psi2 = x[3], beta = psi1 - psi2;
  xn[0] = x[0] + p->dt * w[0] * cos(psi1);
  xn[1] = x[1] + p->dt * w[0] * sin(psi1);
  xn[2] = psi1 + p->dt * w[1] / p->L1;
  xn[3] = psi2 + p->dt * (w[0] * sin(beta) - (p->Lh / p->L1) * w[1] * cos(beta)) / p->L2;
}

double orc_rollout_projected(const orc_params* p, const orc_proj_params* pp, const double x0[4],
                             const double goal[4], int n_obs, const double* obstacles, const double* u,
                             const double* ualpha, double alpha0, double xT[4], double* traj,
                             double* z_all, double* alpha_all, double* Ab_all) {
  const int T = p->T, d = 2 + n_obs;
  double X[4] = {x0[0], x0[1], x0[2], x0[3]};
  double alpha[ORC_PROJ_MAX_NO], S = 0.0;
  double wdiag[2 + ORC_PROJ_MAX_NO], zlo[2 + ORC_PROJ_MAX_NO], zhi[2 + ORC_PROJ_MAX_NO];
  double vabs = fmax(fabs(p->v_min), fabs(p->v_max));
  double omega_max = vabs * tan(fmax(fabs(p->delta_min), fabs(p->delta_max)));
  wdiag[0] = pp->q_v; wdiag[1] = pp->q_omega;
  zlo[0] = p->v_min; zhi[0] = p->v_max; zlo[1] = -omega_max; zhi[1] = omega_max;
  for (int i = 0; i < n_obs; ++i) {
    alpha[i] = alpha0;
    wdiag[2 + i] = pp->q_alpha; zlo[2 + i] = -pp->ualpha_max; zhi[2 + i] = pp->ualpha_max;
  }
  if (traj) memcpy(traj, X, sizeof(X));
  if (alpha_all) memcpy(alpha_all, alpha, sizeof(double) * (size_t)n_obs);

  for (int t = 0; t < T; ++t) {
    /* z_des = [w_des; u~^alpha], w_des = (v~, v~ tan delta~) */
    double zdes[2 + ORC_PROJ_MAX_NO], A[ORC_PROJ_MAX_NO * (2 + ORC_PROJ_MAX_NO)], b[ORC_PROJ_MAX_NO];
    double z[2 + ORC_PROJ_MAX_NO];
    zdes[0] = u[2 * t + 0];
    zdes[1] = u[2 * t + 0] * tan(u[2 * t + 1]);
    memset(A, 0, sizeof(A));
    for (int i = 0; i < n_obs; ++i) {
      double h, Lg[2], Lf;
      int jstar;
      zdes[2 + i] = ualpha[t * n_obs + i];
      orc_barrier_row(p, X, obstacles + 5 * i, t, &h, &jstar, Lg, &Lf);
      /* (9): L_g h u + h u^alpha = -alpha h - L_f h */
      A[i * d + 0] = Lg[0]; A[i * d + 1] = Lg[1]; A[i * d + 2 + i] = h;
      b[i] = -alpha[i] * h - Lf;
      if (Ab_all) {
        double* q = Ab_all + ((size_t)t * n_obs + i) * 4;
        q[0] = Lg[0]; q[1] = Lg[1]; q[2] = h; q[3] = b[i];
      }
    }
    if (n_obs > 0) orc_project(n_obs, d, A, b, zdes, wdiag, pp->rho, zlo, zhi, z);
    else {                                                   /* no constraint: the soft-bounded minimiser M^-1 p */
      for (int j = 0; j < 2; ++j) z[j] = (wdiag[j] * zdes[j] + 0.5 * pp->rho * (zhi[j] + zlo[j])) / (wdiag[j] + pp->rho);
    }
    if (z_all) memcpy(z_all + (size_t)t * d, z, sizeof(double) * (size_t)d);
    /* x_{tau+1} from the projected input, alpha_{tau+1} = alpha_tau + u^alpha_proj */
    double Xn[4];
    orc_affine_step(p, X, z, Xn);
    for (int i = 0; i < n_obs; ++i) alpha[i] += z[2 + i];
    /* stage cost on (x_{tau+1}, projected input) */
    double hitch = fabs(orc_wrap(Xn[2] - Xn[3])) - (p->hitch_max - p->hitch_kappa * fabs(z[0]));
    if (hitch < 0.0) hitch = 0.0;
    double ca = 0.0;
    for (int i = 0; i < n_obs; ++i) {
      double h, Lg[2], Lf;
      int jstar;
      orc_barrier_row(p, Xn, obstacles + 5 * i, t + 1, &h, &jstar, Lg, &Lf);
      if (h < pp->h_buffer && alpha[i] > 0.0) ca += alpha[i] * alpha[i];
    }
    S += orc_goal_cost(p, Xn, goal) + p->w_v * z[0] * z[0] + p->w_delta * z[1] * z[1] +
         p->w_hitch * hitch * hitch + pp->w_alpha * ca;
    memcpy(X, Xn, sizeof(X));
    if (traj) memcpy(traj + 4 * (t + 1), X, sizeof(X));
    if (alpha_all) memcpy(alpha_all + (size_t)(t + 1) * n_obs, alpha, sizeof(double) * (size_t)n_obs);
  }
  S += p->w_term * orc_goal_cost(p, X, goal);
  memcpy(xT, X, sizeof(X));
  return S;
}

double orc_sample_projected(const orc_params* p, const orc_proj_params* pp, uint32_t n, uint32_t k,
                            const double x0[4], const double goal[4], int n_obs, const double* obstacles,
                            const double* U_in, double* u, double xT[4]) {
  const int T = p->T;
  double alpha0 = orc_alpha(p, n, k);
  double* ua = (double*)malloc(sizeof(double) * (size_t)T * (size_t)(n_obs > 0 ? n_obs : 1));
  for (int t = 0; t < T; ++t) {
    double z[2], zeta[ORC_PROJ_MAX_NO];
    orc_normals(p->seed, n, k, (uint32_t)t, z);
    u[2 * t + 0] = clampd(U_in[2 * t + 0] + p->sigma_v * z[0], p->v_min, p->v_max);
    u[2 * t + 1] = clampd(U_in[2 * t + 1] + p->sigma_delta * z[1], p->delta_min, p->delta_max);
    orc_ualpha_normals(p->seed, n, k, (uint32_t)t, n_obs, zeta);
    for (int i = 0; i < n_obs; ++i) ua[t * n_obs + i] = pp->sigma_ualpha * zeta[i];
  }
  double S = orc_rollout_projected(p, pp, x0, goal, n_obs, obstacles, u, ua, alpha0, xT, NULL, NULL, NULL, NULL);
  free(ua);
  return S;
}

typedef struct {
  sample_job base;
  const orc_proj_params* pp;
} proj_job;

static void* proj_worker(void* arg) {
  proj_job* job = (proj_job*)arg;
  const sample_job* b = &job->base;
  const int T = b->p->T;
  for (int k = b->k_begin; k < b->k_end; ++k)
    b->S[k] = orc_sample_projected(b->p, job->pp, b->n, (uint32_t)k, b->x0, b->goal, b->n_obs, b->obstacles,
                                   b->U_in, b->u_all + (size_t)k * 2 * T, b->XT + 4 * (size_t)k);
  return NULL;
}

int orc_iteration_projected(const orc_params* p, const orc_proj_params* pp, uint32_t n, const double x0[4],
                            const double goal[4], int n_obs, const double* obstacles, const double* U_in,
                            double* U_out, double* S, double* XT, double* u_all, double* w, int* argmin,
                            double* gap, double* eta, int n_threads) {
  const int K = p->K, T = p->T;
  double* S_buf = S ? S : (double*)malloc(sizeof(double) * (size_t)K);
  double* XT_buf = XT ? XT : (double*)malloc(sizeof(double) * 4 * (size_t)K);
  double* u_buf = u_all ? u_all : (double*)malloc(sizeof(double) * 2 * (size_t)T * (size_t)K);
  double* U_nom = (double*)malloc(sizeof(double) * 2 * (size_t)T);
  memcpy(U_nom, U_in, sizeof(double) * 2 * (size_t)T);
  if (n_threads < 1) n_threads = 1;
  if (n_threads > K) n_threads = K;
  proj_job* jobs = (proj_job*)malloc(sizeof(proj_job) * (size_t)n_threads);
  pthread_t* tids = (pthread_t*)malloc(sizeof(pthread_t) * (size_t)n_threads);
  for (int i = 0; i < n_threads; ++i) {
    jobs[i].base = (sample_job){p, n, x0, goal, obstacles, U_nom, n_obs, (int)((long long)K * i / n_threads),
                                (int)((long long)K * (i + 1) / n_threads), S_buf, XT_buf, u_buf, 0, NULL};
    jobs[i].pp = pp;
  }
  if (n_threads == 1) proj_worker(&jobs[0]);
  else {
    for (int i = 0; i < n_threads; ++i) pthread_create(&tids[i], NULL, proj_worker, &jobs[i]);
    for (int i = 0; i < n_threads; ++i) pthread_join(tids[i], NULL);
  }
  if (U_out != U_in) memcpy(U_out, U_nom, sizeof(double) * 2 * (size_t)T);
  /* eq. (5) on the sampled u~ with the projected rollouts' costs */
  int nonfinite = orc_weights_update(K, T, p->lambda, S_buf, u_buf, U_out, w, argmin, gap, eta);
  free(jobs); free(tids); free(U_nom);
  if (!S) free(S_buf);
  if (!XT) free(XT_buf);
  if (!u_all) free(u_buf);
  return nonfinite;
}

/* ------------------------------------------------------------------------------------------
 * The paper's own model and tracking cost: eq. (6), (13)-(15), (17);
 * readings in the header (reading 31).
 * ---------------------------------------------------------------------------------------- */

/* eq. (6): x = [px, py, v, a, theta1, theta2, delta], u = [j, omega]; every RHS at step k. */
void orc7_step(const orc_params* p, const orc_mpcc_params* mp, const double x[7], const double u[2], double xn[7]) {
  double Ts = p->dt, v = x[2], a = x[3], th1 = x[4], th2 = x[5], de = x[6];
  xn[0] = x[0] + Ts * v * cos(th1);
  xn[1] = x[1] + Ts * v * sin(th1);
  xn[2] = v + Ts * a;
  xn[3] = a + Ts * u[0];
  xn[4] = th1 + Ts * (v / p->L1) * tan(de);
  xn[5] = th2 + Ts * (v / p->L2) * (sin(th1 - th2) - (p->Lh / p->L1) * cos(th1 - th2) * tan(de));
  xn[6] = clampd(de + Ts * u[1], mp->delta_lo, mp->delta_hi);
}

void orc_path_eval(const orc_mpcc_params* mp, double psi, double out[4]) {
  double L = mp->M * mp->dpsi;
  if (psi < 0.0) psi = 0.0;
  if (psi > L) psi = L;
  int m = (int)floor(psi / mp->dpsi);
  if (m > mp->M - 1) m = mp->M - 1;
  double s = psi - m * mp->dpsi;
  for (int c = 0; c < 4; ++c) {
    const double* q = mp->coef + ((size_t)m * 4 + c) * 4;
    out[c] = q[0] + s * (q[1] + s * (q[2] + s * q[3]));
  }
}

double orc7_progress(const orc_mpcc_params* mp, const double x[7], double psi) {
  double r[4];
  orc_path_eval(mp, psi, r);
  return x[2] * cos(x[4] - r[2]);
}

/* (14), (15) PAPER.md:207-210 as printed; heading errors PAPER.md:212, wrapped. */
void orc7_errors(const orc_mpcc_params* mp, const double x[7], double psi, double e[4]) {
  double r[4];
  orc_path_eval(mp, psi, r);
  double dx = x[0] - r[0], dy = x[1] - r[1];
  e[0] = sin(r[2]) * dx - cos(r[2]) * dy;
  e[1] = -cos(r[2]) * dx - sin(r[2]) * dy;
  e[2] = orc_wrap(x[4] - r[2]);
  e[3] = orc_wrap(x[5] - r[3]);
}

/* (17): hhat = h + Ts hdot + Ts^2/2 hddot along the continuous model
 *   pdot = v e(th1), vdot = a, th1dot = W1 = (v/l1) tan(delta), th2dot = W2 = (v/l2)(sin b - k cos b tan(delta)),
 *   deltadot = omega, b = th1 - th2, k = lh/l1,
 * for the disc centre c = p - lh e(th1) + a_j e(th_body) and the obstacle o(t) = o0 + t Ts vel. */
double orc7_hhat(const orc_params* p, const double x[7], const double u[2], const double* ob, int t, int j,
                 double* h_out) {
  double Ts = p->dt, v = x[2], a = x[3], th1 = x[4], th2 = x[5], de = x[6], om = u[1];
  double td = tan(de), sec2 = 1.0 / (cos(de) * cos(de));
  double b = th1 - th2, kap = p->Lh / p->L1;
  double W1 = (v / p->L1) * td;
  double W2 = (v / p->L2) * (sin(b) - kap * cos(b) * td);
  double bdot = W1 - W2;
  double W1dot = (a / p->L1) * td + (v / p->L1) * sec2 * om;
  double W2dot = (a / p->L2) * (sin(b) - kap * cos(b) * td) +
                 (v / p->L2) * (cos(b) * bdot + kap * sin(b) * bdot * td - kap * cos(b) * sec2 * om);
  double e1[2] = {cos(th1), sin(th1)}, n1[2] = {-sin(th1), cos(th1)};
  double thb = (p->disc_body[j] == 0) ? th1 : th2;
  double Wb = (p->disc_body[j] == 0) ? W1 : W2, Wbdot = (p->disc_body[j] == 0) ? W1dot : W2dot;
  double eb[2] = {cos(thb), sin(thb)}, nb[2] = {-sin(thb), cos(thb)};
  double aj = p->disc_offset[j];
  double c[2], cd[2], cdd[2];
  for (int q = 0; q < 2; ++q) {
    c[q] = x[q] - p->Lh * e1[q] + aj * eb[q];
    cd[q] = v * e1[q] - p->Lh * W1 * n1[q] + aj * Wb * nb[q];
    cdd[q] = a * e1[q] + v * W1 * n1[q] - p->Lh * (W1dot * n1[q] - W1 * W1 * e1[q]) +
             aj * (Wbdot * nb[q] - Wb * Wb * eb[q]);
  }
  double o[2] = {ob[0] + (double)t * Ts * ob[3], ob[1] + (double)t * Ts * ob[4]};
  double rho = ob[2] + p->disc_radius;
  double d[2] = {c[0] - o[0], c[1] - o[1]}, dd[2] = {cd[0] - ob[3], cd[1] - ob[4]};
  double h = (d[0] * d[0] + d[1] * d[1]) / (rho * rho) - 1.0;
  double hdot = 2.0 * (d[0] * dd[0] + d[1] * dd[1]) / (rho * rho);
  double hddot = 2.0 * (dd[0] * dd[0] + dd[1] * dd[1] + d[0] * cdd[0] + d[1] * cdd[1]) / (rho * rho);
  if (h_out) *h_out = h;
  return h + Ts * hdot + 0.5 * Ts * Ts * hddot;
}

static double mpcc_tracking(const orc_mpcc_params* mp, const double x[7], double psi) {
  double e[4];
  orc7_errors(mp, x, psi, e);
  return mp->Qc * e[0] * e[0] + mp->Ql * e[1] * e[1] + mp->Qth1 * e[2] * e[2] + mp->Qth2 * e[3] * e[3];
}

double orc7_rollout(const orc_params* p, const orc_mpcc_params* mp, const double x0[7], double psi0, int n_obs,
                    const double* obstacles, const double* u, double alpha, double xT[8], double* traj) {
  const int T = p->T, D = p->n_discs;
  double X[7], psi = psi0, S = 0.0, L = mp->M * mp->dpsi;
  memcpy(X, x0, sizeof(X));
  if (traj) { memcpy(traj, X, sizeof(X)); traj[7] = psi; }
  for (int t = 0; t < T; ++t) {
    const double* ut = u + 2 * t;
    /* barrier-rate hinge with the predictor (17) in the place of h(x_{k+1}) */
    double pen = 0.0;
    for (int i = 0; i < n_obs; ++i)
      for (int j = 0; j < D; ++j) {
        double h, hhat = orc7_hhat(p, X, ut, obstacles + 5 * i, t, j, &h);
        double viol = (1.0 - alpha) * h - hhat;
        if (viol > 0.0) pen += viol;
      }
    double Xn[7];
    orc7_step(p, mp, X, ut, Xn);
    double psin = clampd(psi + p->dt * orc7_progress(mp, X, psi), 0.0, L);
    /* stage cost (13) on (x_{k+1}, u_k, psi_{k+1}) */
    double nu = orc7_progress(mp, Xn, psin);
    double hitch = fabs(orc_wrap(Xn[4] - Xn[5])) - (p->hitch_max - p->hitch_kappa * fabs(Xn[2]));
    if (hitch < 0.0) hitch = 0.0;
    S += mpcc_tracking(mp, Xn, psin) + mp->Rj * ut[0] * ut[0] + mp->Rw * ut[1] * ut[1] +
         mp->mu * (mp->nu_bar - nu) * (mp->nu_bar - nu) + p->w_hitch * hitch * hitch + p->w_bar * pen;
    memcpy(X, Xn, sizeof(X));
    psi = psin;
    if (traj) { memcpy(traj + 8 * (t + 1), X, sizeof(X)); traj[8 * (t + 1) + 7] = psi; }
  }
  S += p->w_term * mpcc_tracking(mp, X, psi);
  memcpy(xT, X, sizeof(X));
  xT[7] = psi;
  return S;
}

double orc7_sample(const orc_params* p, const orc_mpcc_params* mp, uint32_t n, uint32_t k, const double x0[7],
                   double psi0, int n_obs, const double* obstacles, const double* U_in, double* u, double xT[8]) {
  double alpha = orc_alpha(p, n, k);
  for (int t = 0; t < p->T; ++t) {
    double z[2];
    orc_normals(p->seed, n, k, (uint32_t)t, z);
    u[2 * t + 0] = clampd(U_in[2 * t + 0] + mp->sigma_j * z[0], mp->j_min, mp->j_max);
    u[2 * t + 1] = clampd(U_in[2 * t + 1] + mp->sigma_omega * z[1], mp->omega_min, mp->omega_max);
  }
  return orc7_rollout(p, mp, x0, psi0, n_obs, obstacles, u, alpha, xT, NULL);
}

typedef struct {
  const orc_params* p;
  const orc_mpcc_params* mp;
  uint32_t n;
  const double *x0, *obstacles, *U_in;
  double psi0;
  int n_obs, k_begin, k_end;
  double *S, *XT, *u_all;
} mpcc_job;

static void* mpcc_worker(void* arg) {
  mpcc_job* b = (mpcc_job*)arg;
  const int T = b->p->T;
  for (int k = b->k_begin; k < b->k_end; ++k)
    b->S[k] = orc7_sample(b->p, b->mp, b->n, (uint32_t)k, b->x0, b->psi0, b->n_obs, b->obstacles, b->U_in,
                          b->u_all + (size_t)k * 2 * T, b->XT + 8 * (size_t)k);
  return NULL;
}

int orc7_iteration(const orc_params* p, const orc_mpcc_params* mp, uint32_t n, const double x0[7], double psi0,
                   int n_obs, const double* obstacles, const double* U_in, double* U_out, double* S, double* XT,
                   double* u_all, double* w, int* argmin, double* gap, double* eta, int n_threads) {
  const int K = p->K, T = p->T;
  double* S_buf = S ? S : (double*)malloc(sizeof(double) * (size_t)K);
  double* XT_buf = XT ? XT : (double*)malloc(sizeof(double) * 8 * (size_t)K);
  double* u_buf = u_all ? u_all : (double*)malloc(sizeof(double) * 2 * (size_t)T * (size_t)K);
  double* U_nom = (double*)malloc(sizeof(double) * 2 * (size_t)T);
  memcpy(U_nom, U_in, sizeof(double) * 2 * (size_t)T);
  if (n_threads < 1) n_threads = 1;
  if (n_threads > K) n_threads = K;
  mpcc_job* jobs = (mpcc_job*)malloc(sizeof(mpcc_job) * (size_t)n_threads);
  pthread_t* tids = (pthread_t*)malloc(sizeof(pthread_t) * (size_t)n_threads);
  for (int i = 0; i < n_threads; ++i)
    jobs[i] = (mpcc_job){p, mp, n, x0, obstacles, U_nom, psi0, n_obs, (int)((long long)K * i / n_threads),
                         (int)((long long)K * (i + 1) / n_threads), S_buf, XT_buf, u_buf};
  if (n_threads == 1) mpcc_worker(&jobs[0]);
  else {
    for (int i = 0; i < n_threads; ++i) pthread_create(&tids[i], NULL, mpcc_worker, &jobs[i]);
    for (int i = 0; i < n_threads; ++i) pthread_join(tids[i], NULL);
  }
  if (U_out != U_in) memcpy(U_out, U_nom, sizeof(double) * 2 * (size_t)T);
  int nonfinite = orc_weights_update(K, T, p->lambda, S_buf, u_buf, U_out, w, argmin, gap, eta);
  free(jobs); free(tids); free(U_nom);
  if (!S) free(S_buf);
  if (!XT) free(XT_buf);
  if (!u_all) free(u_buf);
  return nonfinite;
}
