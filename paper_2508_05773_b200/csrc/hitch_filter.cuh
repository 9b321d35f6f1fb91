// Hitch-angle stabiliser, Sec. V-D: barrier (18), condition (3) expanded to first
// order in u about the BR-MPPI reference (reading 28), and the 2-variable CBF-QP
//   min q_v (v - v_ref)^2 + q_delta (delta - delta_ref)^2   s.t.  c0 + a . (u - u_ref) >= 0,  u in the box.
// With a diagonal Q_h the KKT point is u_i(mu) = clamp(u_ref_i + mu a_i / q_i) for the multiplier
// mu >= 0 of the rate constraint, and g(mu) = c0 + a . (u(mu) - u_ref) is continuous, piecewise linear and
// non-decreasing with at most four breakpoints (each coordinate enters and leaves its interval once):
// the solution is the smallest mu with g(mu) >= 0, found by walking the sorted breakpoints.  One
// thread per problem; called by shift_plant (closed loop) and by hitch_filter_batch.
#pragma once
#include "brmppi_device.cuh"

namespace brmppi {

struct HitchQp { float c0, a0, a1; };

__device__ __forceinline__ HitchQp hitch_constraint(const DeviceParams& P, float psi1, float psi2, float2 r) {
  const float beta = wrap_angle(psi1 - psi2);
  const float s = beta >= 0.0f ? 1.0f : -1.0f;
  float sb, cb;
  sincosf(beta, &sb, &cb);
  const float td = tanf(r.y), cd = cosf(r.y);
  // d(psi1dot - psi2dot)/dv and /d delta of the reduced eq. (6)
  const float dv = fmaf(td, P.inv_L1, -P.inv_L2 * fmaf(-P.Lh_over_L1 * td, cb, sb));
  const float dd = r.x * P.inv_L1 * fmaf(P.Lh * P.inv_L2, cb, 1.0f) / (cd * cd);
  const float h = P.hitch_max - P.hitch_kappa * fabsf(r.x) - fabsf(beta);   // eq. (18)
  const float sgn_v = r.x > 0.0f ? 1.0f : (r.x < 0.0f ? -1.0f : 0.0f);
  HitchQp q;
  q.c0 = fmaf(-s * P.dt, r.x * dv, P.hitch_alpha * h);
  q.a0 = fmaf(-s * P.dt, dv, -P.hitch_alpha * P.hitch_kappa * sgn_v);
  q.a1 = -s * P.dt * dd;
  return q;
}

__device__ __forceinline__ float hitch_g(const HitchQp& q, float2 r, float2 w, float mu,
                                         float2 lo, float2 hi, float2* u) {
  u->x = fminf(fmaxf(fmaf(mu, w.x, r.x), lo.x), hi.x);
  u->y = fminf(fmaxf(fmaf(mu, w.y, r.y), lo.y), hi.y);
  return fmaf(q.a1, u->y - r.y, fmaf(q.a0, u->x - r.x, q.c0));
}

// Returns the filtered control; *status: 0 constraint inactive, 1 active, 2 box and half-plane disjoint.
__device__ inline float2 hitch_filter(const DeviceParams& P, float psi1, float psi2, float2 r, int* status) {
  const HitchQp q = hitch_constraint(P, psi1, psi2, r);
  const float2 lo = make_float2(P.v_min, P.delta_min), hi = make_float2(P.v_max, P.delta_max);
  const float2 w = make_float2(q.a0 / P.hitch_qv, q.a1 / P.hitch_qdelta);   // d u_i / d mu
  float2 u;
  float g_lo = hitch_g(q, r, w, 0.0f, lo, hi, &u);
  if (g_lo >= 0.0f) { *status = 0; return u; }
  // breakpoints: mu at which coordinate i reaches its lower / upper bound
  float bp[4] = {INFINITY, INFINITY, INFINITY, INFINITY};
  if (w.x != 0.0f) { bp[0] = (lo.x - r.x) / w.x; bp[1] = (hi.x - r.x) / w.x; }
  if (w.y != 0.0f) { bp[2] = (lo.y - r.y) / w.y; bp[3] = (hi.y - r.y) / w.y; }
#pragma unroll
  for (int i = 0; i < 4; ++i)
    if (!(bp[i] > 0.0f)) bp[i] = INFINITY;
#pragma unroll
  for (int i = 1; i < 4; ++i)            // insertion sort of four values
#pragma unroll
    for (int j = i; j > 0; --j)
      if (bp[j] < bp[j - 1]) { const float t = bp[j]; bp[j] = bp[j - 1]; bp[j - 1] = t; }
  float mu_lo = 0.0f;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    if (isinf(bp[i])) break;
    float2 ub;
    const float g_hi = hitch_g(q, r, w, bp[i], lo, hi, &ub);
    if (g_hi >= 0.0f) {                   // the root lies on this linear piece
      const float mu = g_hi > g_lo ? fmaf(-g_lo / (g_hi - g_lo), bp[i] - mu_lo, mu_lo) : bp[i];
      hitch_g(q, r, w, mu, lo, hi, &u);
      *status = 1;
      return u;
    }
    mu_lo = bp[i];
    g_lo = g_hi;
    u = ub;
  }
  *status = 2;                            // u = lim mu -> inf: the box point with the largest a . u
  return u;
}

// n independent problems, one thread each (brmppi_hitch_filter).
__global__ void hitch_filter_batch(const __grid_constant__ DeviceParams P, int n, const float4* x,
                                   const float2* u_ref, float2* u_out, int* status) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int st;
  const float4 xi = x[i];
  u_out[i] = hitch_filter(P, xi.z, xi.w, u_ref[i], &st);
  status[i] = st;
}

}  // namespace brmppi
