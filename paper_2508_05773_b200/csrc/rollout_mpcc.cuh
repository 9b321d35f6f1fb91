// rollout_mpcc.cuh -- the paper's own model and tracking cost (BRMPPI_FLAG_MPCC):
// 7-state jerk / steering-rate model, eq. (6), barrier-rate hinge on the second-order Taylor
// predictor (17), contouring / lag / heading / effort / progress cost (13)-(15)
// along a cubic-spline reference path in arc length.  Readings: DESIGN.md reading 31.
//
// One thread per sample (the whole step is a serial chain: the predictor and the path parameter depend on the
// state), everything in registers; the obstacle table, the nominal and the path's coefficient table sit in
// shared memory.  In this mode DeviceParams' control box (v_min .. delta_max, sigma_v, sigma_delta) holds the
// (jerk, steering-rate) box and sigmas, so the sampler and the thread-per-sample epilogue are the penalty path's.
#pragma once

#include "rollout_thread.cuh"

namespace brmppi {

struct State7 { float x, y, v, a, t1, t2, de, psi; };

// (p^{x,r}, p^{y,r}, theta^{1,r}, theta^{2,r}) at arc length psi from the table [M][4][4] in shared memory.
__device__ __forceinline__ float4 path_eval(const float4* __restrict__ sPath, int M, float dpsi, float inv_dpsi,
                                            float psi) {
  int m = (int)floorf(psi * inv_dpsi);
  m = m > M - 1 ? M - 1 : (m < 0 ? 0 : m);
  const float s = psi - (float)m * dpsi;
  const float4* q = sPath + 4 * m;
  float r[4];
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const float4 k = q[c];
    r[c] = fmaf(s, fmaf(s, fmaf(s, k.w, k.z), k.y), k.x);
  }
  return make_float4(r[0], r[1], r[2], r[3]);
}

// One component of the same (the chain of the phase-split kernel needs theta^{1,r} only).
__device__ __forceinline__ float path_eval_component(const float4* __restrict__ sPath, int M, float dpsi,
                                                     float inv_dpsi, float psi, int comp) {
  int m = (int)floorf(psi * inv_dpsi);
  m = m > M - 1 ? M - 1 : (m < 0 ? 0 : m);
  const float s = psi - (float)m * dpsi;
  const float4 k = sPath[4 * m + comp];
  return fmaf(s, fmaf(s, fmaf(s, k.w, k.z), k.y), k.x);
}

// Q_c e_c^2 + Q_l e_l^2 + Q_th1 e_th1^2 + Q_th2 e_th2^2 at pose (x, y, t1, t2) against the path point r;
// s1 / c1 = sin / cos(t1), sr / cr = sin / cos(r.z); *nu = v cos(theta1 - theta^{1,r}).
__device__ __forceinline__ float mpcc_tracking_sc(const DeviceParams& P, float x, float y, float t1, float t2, float v,
                                                  float s1, float c1, const float4 r, float sr, float cr, float* nu) {
  const float dx = x - r.x, dy = y - r.y;
  const float ec = fmaf(sr, dx, -cr * dy);                       // (14)
  const float el = -fmaf(cr, dx, sr * dy);                       // (15)
  const float e1 = wrap_angle(t1 - r.z), e2 = wrap_angle(t2 - r.w);
  *nu = v * fmaf(c1, cr, s1 * sr);                               // v cos(theta1 - theta1r)
  return fmaf(P.Qc * ec, ec, fmaf(P.Ql * el, el, fmaf(P.Qth1 * e1, e1, P.Qth2 * e2 * e2)));
}

// The same with sin / cos of the path heading taken here; s1 / c1 = sin / cos(X.t1): the caller needs them for the
// next step anyway.
template <bool PRECISE>
__device__ __forceinline__ float mpcc_tracking(const DeviceParams& P, const State7& X, float s1, float c1,
                                               const float4 r, float* nu) {
  float sr, cr;
  sincos_t<PRECISE>(r.z, &sr, &cr);
  return mpcc_tracking_sc(P, X.x, X.y, X.t1, X.t2, X.v, s1, c1, r, sr, cr, nu);
}

// Heading rates of the continuous model, W1 = theta1', W2 = theta2', and their time derivatives under the input
// omega = delta' (sb / cb = sin / cos of the hitch angle theta1 - theta2 by the angle-difference identities).
struct MpccRates { float W1, W2, W1dot, W2dot; };

__device__ __forceinline__ MpccRates mpcc_rates(const DeviceParams& P, float v, float a, float td, float s1, float c1,
                                                float s2, float c2, float omega) {
  const float sec2 = fmaf(td, td, 1.0f);
  const float sb = s1 * c2 - c1 * s2, cb = fmaf(c1, c2, s1 * s2);
  MpccRates R;
  R.W1 = v * P.inv_L1 * td;
  const float gb = fmaf(-P.Lh_over_L1 * cb, td, sb);                       // sin b - k cos b tan(delta)
  R.W2 = v * P.inv_L2 * gb;
  const float bdot = R.W1 - R.W2;
  R.W1dot = P.inv_L1 * fmaf(a, td, v * sec2 * omega);
  const float gbdot = fmaf(bdot, fmaf(P.Lh_over_L1 * sb, td, cb), -P.Lh_over_L1 * cb * sec2 * omega);
  R.W2dot = P.inv_L2 * fmaf(a, gb, v * gbdot);
  return R;
}

// Barrier-rate hinge with the predictor (17) summed over every (obstacle, disc).  With h = |d|^2 / rho^2 - 1,
// hdot = 2 d.e / rho^2, hddot = 2 (e.e + d.acc) / rho^2 (d = disc centre - obstacle, e = their relative velocity,
// acc = the disc centre's acceleration):
//   (1 - alpha) h - hhat = -(alpha h + Ts hdot + Ts^2/2 hddot) = alpha - [alpha |d|^2 + d.(2 Ts e + Ts^2 acc) + |Ts e|^2] / rho^2,
// so everything is evaluated in step units: the caller passes vh = Ts v, ah = Ts^2 a and the rates of
// mpcc_rates(vh, ah, ..., Ts omega) (every formula is homogeneous in Ts), the obstacle table holds Ts vel.
// Lever arms a1 - l_h on e(theta1), a2 on e(theta2).  nd <= ND discs.  Obstacles [0, n_moving) are taken in the
// general form; [n_moving, n_obs) must be at rest (zero velocity: the caller's table is ordered that way), for
// which e = v_disc and g = f, so that the bracket is alpha |d|^2 + d.f + |v_disc|^2 -- the same value (every
// dropped term is an exact zero), ten instructions per (obstacle, disc) instead of sixteen.
//
// Exact culling (inv_alpha_cull > 0; the phase-split kernel unless BRMPPI_FLAG_NO_CULL): the bracket of disc j is
// Q = alpha |d|^2 + d.g + |e|^2 >= alpha |d|^2 - |d| |g| with g = f_j - 2 Ts o', so for alpha > 0 the hinge
// max(0, alpha - Q / rho^2) is zero whenever |d| >= rho + |g| / alpha (then alpha |d| (|d| - |g| / alpha) >=
// alpha rho |d| >= alpha rho^2).  With D = |p - o| the distance of the vehicle's reference point, l_max the longest
// lever (|d_j| >= D - l_max) and G = max_j (|f_jx| + |f_jy|) >= |f_j|, an obstacle contributes nothing to ANY disc
// if D >= l_max + rho + (G + 2 |Ts o'|) / alpha.  The table carries (l_max + rho) and 2 |Ts o'| with a 0.1 % + 1 mm
// margin that covers the fp32 rounding of the test and of Q; an obstacle is skipped only when every active lane of
// the warp agrees (the samples of a warp sit at the same step, close together), so the result is bit-identical.
template <int ND, bool CULL = false>
__device__ __forceinline__ float mpcc_hinge(const DeviceParams& P, const float4* __restrict__ sObs,
                                            const float4* __restrict__ sVel, int n_moving, int n_obs, int nd, float tf,
                                            float alpha, float x, float y, float vh, float ah, float s1, float c1,
                                            float s2, float c2, const MpccRates& R, float inv_alpha_cull = 0.0f) {
  // centre, velocity and f = 2 v + acc of disc j are affine in its lever arms (l1, l2): c = p + l1 e1 + l2 e2,
  // v = vh e1 + l1 W1 n1 + l2 W2 n2, acc = (ah e1 + vh W1 n1) + l1 (W1dot n1 - W1^2 e1) + l2 (W2dot n2 - W2^2 e2)
  // with e = (cos, sin), n = (-sin, cos) of the two headings; the six vectors are shared by all discs
  const float p1x = -R.W1 * s1, p1y = R.W1 * c1, p2x = -R.W2 * s2, p2y = R.W2 * c2, v0x = vh * c1, v0y = vh * s1;
  const float f0x = fmaf(2.0f, v0x, fmaf(ah, c1, vh * p1x)), f0y = fmaf(2.0f, v0y, fmaf(ah, s1, vh * p1y));
  const float f1x = fmaf(2.0f, p1x, fmaf(-R.W1dot, s1, -R.W1 * p1y)), f1y = fmaf(2.0f, p1y, fmaf(R.W1dot, c1, R.W1 * p1x));
  const float f2x = fmaf(2.0f, p2x, fmaf(-R.W2dot, s2, -R.W2 * p2y)), f2y = fmaf(2.0f, p2y, fmaf(R.W2dot, c2, R.W2 * p2x));
  float cx[ND], cy[ND], vx[ND], vy[ND], fx[ND], fy[ND];
#pragma unroll
  for (int j = 0; j < ND; ++j) {
    const float l1 = P.disc_a1[j] - P.Lh, l2 = P.disc_a2[j];
    cx[j] = fmaf(l1, c1, fmaf(l2, c2, x));
    cy[j] = fmaf(l1, s1, fmaf(l2, s2, y));
    vx[j] = fmaf(l1, p1x, fmaf(l2, p2x, v0x));
    vy[j] = fmaf(l1, p1y, fmaf(l2, p2y, v0y));
    fx[j] = fmaf(l1, f1x, fmaf(l2, f2x, f0x));
    fy[j] = fmaf(l1, f1y, fmaf(l2, f2y, f0y));
  }
  const bool cull = CULL && inv_alpha_cull > 0.0f;
  float Gv = 0.0f;
  if (CULL && cull) {
#pragma unroll
    for (int j = 0; j < ND; ++j)
      if (j < nd) Gv = fmaxf(Gv, fabsf(fx[j]) + fabsf(fy[j]));
  }
  float pen = 0.0f;
  for (int i = 0; i < n_moving; ++i) {
    const float4 o = sObs[i];
    const float4 w = sVel[i];                                  // (Ts vx, Ts vy, 2 |Ts o'|, -): the obstacle's step
    const float ox = fmaf(tf, w.x, o.x), oy = fmaf(tf, w.y, o.y);
    if (CULL && cull) {
      const float ddx = x - ox, ddy = y - oy, thr = fmaf(w.z + Gv, inv_alpha_cull, o.w);
      const bool far = fmaf(ddx, ddx, ddy * ddy) >= thr * thr;          // false on NaN
      if (__all_sync(__activemask(), far)) continue;
    }
#pragma unroll
    for (int j = 0; j < ND; ++j) {
      if (j < nd) {
        const float dx = cx[j] - ox, dy = cy[j] - oy, ex = vx[j] - w.x, ey = vy[j] - w.y;
        // d.(2 e + acc) = d.(f - 2 w): the obstacle does not accelerate
        const float gx = fmaf(-2.0f, w.x, fx[j]), gy = fmaf(-2.0f, w.y, fy[j]);
        float q = fmaf(dx, gx, fmaf(dy, gy, fmaf(ex, ex, ey * ey)));
        q = fmaf(alpha, fmaf(dx, dx, dy * dy), q);
        pen += fmaxf(fmaf(-o.z, q, alpha), 0.0f);
      }
    }
  }
  if (n_moving < n_obs) {
    float vv[ND];
#pragma unroll
    for (int j = 0; j < ND; ++j) vv[j] = fmaf(vx[j], vx[j], vy[j] * vy[j]);
    for (int i = n_moving; i < n_obs; ++i) {
      const float4 o = sObs[i];
      if (CULL && cull) {
        const float ddx = x - o.x, ddy = y - o.y, thr = fmaf(Gv, inv_alpha_cull, o.w);
        const bool far = fmaf(ddx, ddx, ddy * ddy) >= thr * thr;
        if (__all_sync(__activemask(), far)) continue;
      }
#pragma unroll
      for (int j = 0; j < ND; ++j) {
        if (j < nd) {
          const float dx = cx[j] - o.x, dy = cy[j] - o.y;
          float q = fmaf(dx, fx[j], fmaf(dy, fy[j], vv[j]));
          q = fmaf(alpha, fmaf(dx, dx, dy * dy), q);
          pen += fmaxf(fmaf(-o.z, q, alpha), 0.0f);
        }
      }
    }
  }
  return pen;
}

// Hitch hinge, effort and progress terms of (13) at (x_{k+1}, u_k): everything but tracking and barrier.
__device__ __forceinline__ float mpcc_stage_rest(const DeviceParams& P, float t1, float t2, float v, float nu, float2 u) {
  const float dn = P.nu_bar - nu;
  const float hl = fmaxf(fabsf(wrap_angle(t1 - t2)) - fmaf(-P.hitch_kappa, fabsf(v), P.hitch_max), 0.0f);
  return fmaf(P.Rj * u.x, u.x, P.Rw * u.y * u.y) + P.mu * dn * dn + P.w_hitch * hl * hl;
}

template <bool PRECISE>
__global__ void __launch_bounds__(kThreadBlock)
rollout_mpcc(const __grid_constant__ DeviceParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  // layout: obs[max_obs] float4 (ox, oy, 1/rho^2, -) | vel[max_obs] float4 (dt vx, dt vy, vx, vy) |
  //         path[M_max][4] float4 | U_nom[T] float2 | red (4 double, 4 int, 12 float) | A_w[4][2T] float
  const int T = P.T;
  float4* sObs = reinterpret_cast<float4*>(smem_raw);
  float4* sVel = sObs + P.max_obstacles;
  float4* sPath = sVel + P.max_obstacles;
  float2* sU = reinterpret_cast<float2*>(sPath + 4 * P.max_path_segments);
  double* sRedM = reinterpret_cast<double*>(sU + T + (T & 1));
  int* sRedI = reinterpret_cast<int*>(sRedM + 4);
  float* sRedF = reinterpret_cast<float*>(sRedI + 4);
  float* sA = sRedF + 12;

  const int scene = blockIdx.y;
  const int tid = threadIdx.x;
  const int k = blockIdx.x * kThreadBlock + tid;
  const bool valid = k < P.K;
  const uint32_t n = *P.counter;
  const uint32_t key0 = P.key0 + (uint32_t)scene;
  const uint32_t key1 = P.key1 + (key0 < P.key0 ? 1u : 0u);

  const float* s7 = P.state7 + 8 * scene;                         // px, py, v, a, theta1, theta2, delta, psi
  const float x0 = s7[0], y0 = s7[1];
  const int n_obs = P.n_obs[scene];
  const int M = P.path_M[scene];
  const float dpsi = P.path_dpsi[scene];
  for (int i = tid; i < T; i += kThreadBlock)
    sU[i] = reinterpret_cast<const float2*>(P.U)[scene * T + i];
  for (int i = tid; i < n_obs; i += kThreadBlock) {
    const float* ob = P.obstacles + ((size_t)scene * P.max_obstacles + i) * 5;
    const float rho = ob[2] + P.disc_radius;
    sObs[i] = make_float4(ob[0] - x0, ob[1] - y0, 1.0f / (rho * rho), 0.0f);   // vehicle-centred frame
    sVel[i] = make_float4(P.dt * ob[3], P.dt * ob[4], ob[3], ob[4]);
  }
  for (int i = tid; i < 4 * M; i += kThreadBlock) {
    float4 c = reinterpret_cast<const float4*>(P.path_coef)[(size_t)scene * 4 * P.max_path_segments + i];
    const int comp = i & 3;
    if (comp == 0) c.x -= x0;
    if (comp == 1) c.x -= y0;
    sPath[i] = c;
  }
  __syncthreads();

  double S = CUDART_INF;
  if (valid) {
    const float inv_dpsi = 1.0f / dpsi, Lpath = (float)M * dpsi;
    const float alpha = sample_alpha(P, n, (uint32_t)(k + P.k_offset), key0, key1);
    State7 X{0.0f, 0.0f, s7[2], s7[3], s7[4], s7[5], s7[6], s7[7]};
    double cost = 0.0;
    float last_track = 0.0f;
    // carried from step to step: sin / cos(theta1) and nu = v cos(theta1 - theta^{1,r}(psi)) of the current
    // state -- the stage cost of step k - 1 evaluates the same path point and the same nu as the progress of step k
    float s1, c1, nu;
    sincos_t<PRECISE>(X.t1, &s1, &c1);
    (void)mpcc_tracking<PRECISE>(P, X, s1, c1, path_eval(sPath, M, dpsi, inv_dpsi, X.psi), &nu);
#pragma unroll 1
    for (int t = 0; t < T; ++t) {
      const float2 u = sample_control<PRECISE>(P, sU[t], (uint32_t)t, n, (uint32_t)(k + P.k_offset), key0, key1);   // (j, omega)
      float s2, c2;
      sincos_t<PRECISE>(X.t2, &s2, &c2);
      const float td = tan_t<PRECISE>(X.de);
      // rates in step units (Ts W1 and Ts W2 are the Euler increments of the headings as well)
      const float vh = P.dt * X.v, ah = P.dt * P.dt * X.a;
      const MpccRates R = mpcc_rates(P, vh, ah, td, s1, c1, s2, c2, P.dt * u.y);
      const float pen = mpcc_hinge<kMaxDiscs>(P, sObs, sVel, n_obs, n_obs, P.n_discs, (float)t, alpha, X.x, X.y, vh, ah,
                                              s1, c1, s2, c2, R);          // table in the caller's order: general form
      // eq. (6), every right-hand side at step k; path parameter by the projection velocity
      State7 N;
      N.x = fmaf(vh, c1, X.x);
      N.y = fmaf(vh, s1, X.y);
      N.v = fmaf(P.dt, X.a, X.v);
      N.a = fmaf(P.dt, u.x, X.a);
      N.t1 = X.t1 + R.W1;
      N.t2 = X.t2 + R.W2;
      N.de = fminf(fmaxf(fmaf(P.dt, u.y, X.de), P.dstate_lo), P.dstate_hi);
      N.psi = fminf(fmaxf(fmaf(P.dt, nu, X.psi), 0.0f), Lpath);
      X = N;
      // stage cost (13) on (x_{k+1}, u_k, psi_{k+1})
      sincos_t<PRECISE>(X.t1, &s1, &c1);
      const float track = mpcc_tracking<PRECISE>(P, X, s1, c1, path_eval(sPath, M, dpsi, inv_dpsi, X.psi), &nu);
      last_track = track;
      const float stage = track + mpcc_stage_rest(P, X.t1, X.t2, X.v, nu, u);
      cost += (double)stage + (double)P.w_bar * (double)pen;
    }
    // terminal cost: the tracking terms at (x_N, psi_N), which the last stage cost just evaluated
    S = cost + (double)(P.w_term * last_track);
    if (P.flags & BRMPPI_FLAG_WRITE_SAMPLES) {
      P.S[(size_t)scene * P.K + k] = (float)S;
      float4* out = reinterpret_cast<float4*>(P.XT) + 2 * ((size_t)scene * P.K + k);
      out[0] = make_float4(X.x + x0, X.y + y0, X.v, X.a);
      out[1] = make_float4(X.t1, X.t2, X.de, X.psi);
    }
  }
  thread_kernel_epilogue<PRECISE>(P, sU, sRedM, sRedI, sRedF, sA, S, valid, k, scene, n, key0, key1);
}

inline size_t rollout_mpcc_smem_bytes(const DeviceParams& P) {
  return sizeof(float4) * 2 * (size_t)P.max_obstacles + sizeof(float4) * 4 * (size_t)P.max_path_segments +
         sizeof(float2) * (size_t)(P.T + (P.T & 1)) + sizeof(double) * 4 + sizeof(int) * 4 + sizeof(float) * 12 +
         sizeof(float) * 4 * 2 * (size_t)P.T;
}

}  // namespace brmppi
