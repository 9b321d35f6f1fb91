// brmppi_device.cuh -- device-side building blocks shared by the sm_100a kernels of this
// library (and by nothing else: the CPU oracle under oracle/ has its own, independent code).
//
// Citations are to /root/reference/PAPER.md (arxiv 2508.05773) and to the numbered readings in
// DESIGN.md §3.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/brmppi.h"

namespace brmppi {

constexpr int kMaxDiscs = BRMPPI_MAX_DISCS;
constexpr int kMaxObstacles = BRMPPI_MAX_OBSTACLES;
constexpr float kTwoPi = 6.283185307179586f;
constexpr float kInvTwoPi = 0.15915494309189535f;

// Everything a kernel needs, passed by value as a __grid_constant__ parameter (constant bank,
// so scalar weights fold into FFMA operands without a load).
struct DeviceParams {
  int K, T, n_scenes, max_obstacles, n_discs, max_superellipses;
  int k_offset;               // global index of this context's first sample (Philox counter, argmin): K-sharded solves
  int disc_body[kMaxDiscs];
  float disc_offset[kMaxDiscs];
  float disc_a1[kMaxDiscs], disc_a2[kMaxDiscs];   // offset on the tractor axis / on the trailer axis (one is 0)
  float disc_radius;
  float disc_speed[kMaxDiscs];   // upper bound on the speed of each disc centre, m/s (culling)
  float dt, inv_L1, inv_L2, Lh, Lh_over_L1, Lh_over_L2;
  float v_min, v_max, delta_min, delta_max, sigma_v, sigma_delta;
  float alpha_lo, alpha_span;
  float w_pos, w_head, w_v, w_delta, w_hitch, hitch_max, hitch_kappa, w_bar, w_term;
  float inv_lambda;
  int hitch_filter;            // 1: shift_plant passes U[0] through the CBF-QP of Sec. V-D
  float hitch_alpha, hitch_qv, hitch_qdelta;
  float proj_qv, proj_qomega, proj_qalpha, proj_rho, sigma_ualpha, ualpha_max, w_alpha, h_buffer;   // BRMPPI_FLAG_PROJECTED
  // BRMPPI_FLAG_MPCC: in this mode v_min .. sigma_delta above hold the (j, omega) box and sigmas
  float dstate_lo, dstate_hi;  // clamp of the steering STATE delta
  float Qc, Ql, Qth1, Qth2, Rj, Rw, mu, nu_bar;
  int max_path_segments;
  float mpcc_lmax;             // longest lever of a disc centre about the reference point, |a1 - Lh| + |a2| (culling)
  int mpcc_noise_planes;       // rollout_mpcc_cta: the tile's sampled controls are kept in shared memory
  uint32_t key0, key1;        // Philox key of scene 0 = (lo32(seed), hi32(seed)); scene s adds s
  uint32_t flags;
  // tiling of the sample axis
  int n_partials;             // partial slots per scene (one online-softmax partial per CTA and scene)
  int S_tile;                 // persistent-CTA kernel: samples per tile
  int tiles_per_scene;        // ceil(K / S_tile)
  int total_tiles;            // tiles_per_scene * n_scenes
  int tiles_per_cta;          // CTA b owns the flat tiles [b Q, (b+1) Q); 0 = one CTA per partial slot
  int chunks, chunk_len;      // C threads per sample in the barrier phase, L steps per thread
  int t_stride;               // padded row length of the shared-memory planes
  int obs_padded;             // obstacle slots, a multiple of the group size
  int se_padded;              // super-ellipse slots, a multiple of kSeGroup (0 if none)
  int off_se;                 // shared-memory section of the super-ellipse table
  // byte offsets of the shared-memory sections (host-computed, so that the device code
  // rematerialises a pointer with one add instead of keeping it in a register)
  int off_obs, off_vel, off_thr, off_A, off_scratch, off_w, off_alpha, off_cost, off_xy,
      off_planes, off_misc;
  // workspace pointers (DEVICE)
  float* state;               // [n_scenes][4]
  float* goal;                // [n_scenes][4]
  int* n_obs;                 // [n_scenes]
  float* obstacles;           // [n_scenes][max_obstacles][5]
  int* n_se;                  // [n_scenes]
  float* se;                  // [n_scenes][max_superellipses][8]: cx, cy, mx, my, theta, vx, vy, exponent
  float* U;                   // [n_scenes][T][2]
  uint32_t* counter;          // global iteration counter n
  float* u0_applied;          // [n_scenes][2]  control applied by the last plant step
  float* u0_host;             // the same, in page-locked HOST memory the device writes directly (brmppi_step's result)
  float* U_host;              // [n_scenes][T][2]  mirror of U in page-locked host memory, written by every merge_update
  float* state7;              // [n_scenes][8]  (p_x, p_y, v, a, theta1, theta2, delta, psi)  (FLAG_MPCC)
  int* path_M;                // [n_scenes]     cubic segments of the reference path
  float* path_dpsi;           // [n_scenes]     knot spacing
  float* path_coef;           // [n_scenes][max_path_segments][4][4]
  float* hitch_ref;           // [n_scenes][4]  (v_ref, delta_ref, status as int bits, 0) of the last plant step
  double* part_m;             // [n_scenes][P]  block minimum of S (fp64)
  int* part_argmin;           // [n_scenes][P]
  float* part_eta;            // [n_scenes][P]
  float* part_w2;             // [n_scenes][P]  sum w^2 (for the ESS diagnostic)
  int* part_nonfinite;        // [n_scenes][P]
  float* part_A;              // [n_scenes][2T][P]  weighted control sums, output-major
  brmppi_diag* diag;          // [n_scenes]
  float* S;                   // [n_scenes][K]     (FLAG_WRITE_SAMPLES)
  float* XT;                  // [n_scenes][K][4]  (FLAG_WRITE_SAMPLES); [K][8] with FLAG_MPCC
  unsigned long long* phase_ns;   // [grid][8] per-CTA phase nanoseconds (FLAG_PHASE_TIMING), else null
};

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11).  Ten rounds of two 32x32->64 multiplies and two
// three-input xors; the key schedule is counter-independent, so after unrolling the compiler
// keeps key + r*W in uniform registers.  Reading 5: counter (t, n, k, tag), key from the seed.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1) {
  constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
  constexpr uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
    const uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
    const uint32_t n0 = hi1 ^ c1 ^ k0;
    const uint32_t n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += W0; k1 += W1;
  }
  return make_uint4(c0, c1, c2, c3);
}

// MUFU-backed approximations with flush-to-zero, so that no denormal fix-up code is emitted
// (every argument here is a normal number or zero).  Error: lg2 / sqrt / rcp ~1e-7 relative,
// sin / cos 2^-21.4 absolute for |x| <= pi.
__device__ __forceinline__ float fast_lg2(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float fast_sqrt(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float fast_rcp(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
// Packed fp32 pairs (sm_100 add/fma.rn.f32x2): each half rounds exactly like the scalar instruction,
// one issue slot for two results.  A pair lives in an aligned 64-bit register pair, so pack/unpack
// are register naming, not instructions.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) { f32x2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) { f32x2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ float fast_rsqrt(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float fast_sin(float x) { float y; asm("sin.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float fast_cos(float x) { float y; asm("cos.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// f(w) = (w >> 9) * 2^-23 in [0, 1): exact in fp32 (reading 5).
__device__ __forceinline__ float uniform23(uint32_t w) {
  // the 23 bits become the mantissa of a float in [1, 2); subtracting 1 is exact.  One LOP3 and
  // one FADD instead of an I2F on the 16-lane XU pipe plus an FMUL.
  return __uint_as_float(0x3f800000u | (w >> 9)) - 1.0f;
}
// 1 - f(w) in (0, 1], exact.
__device__ __forceinline__ float one_minus_uniform23(uint32_t w) {
  return 2.0f - __uint_as_float(0x3f800000u | (w >> 9));
}

// Box-Muller on two Philox words (reading 5).  z.x -> speed channel, z.y -> steering
// channel.  PRECISE selects libdevice logf/sincospif instead of MUFU lg2/sin/cos.
template <bool PRECISE>
__device__ __forceinline__ float2 box_muller(uint32_t wa, uint32_t wb) {
  const float u1 = one_minus_uniform23(wa);   // (0, 1], exact
  const float u2 = uniform23(wb);             // [0, 1)
  float r, s, c;
  if (PRECISE) {
    r = sqrtf(-2.0f * logf(u1));
    sincospif(2.0f * u2, &s, &c);
  } else {
    // -2 ln u1 = (-2 ln 2) log2(u1); MUFU.LG2 abs error ~2^-22 relative on the result.
    r = fast_sqrt(-1.3862943611198906f * fast_lg2(u1));
    // sin/cos(2 pi u2) = -sin/cos(2 pi (u2 - 1/2)): keeps the MUFU argument inside [-pi, pi),
    // where sin.approx / cos.approx have their documented 2^-21.4 absolute error; u2 - 1/2 is
    // exact in fp32.
    const float a = kTwoPi * (u2 - 0.5f);
    s = -fast_sin(a);
    c = -fast_cos(a);
  }
  return make_float2(r * c, r * s);
}

// The normals of step t of sample k in iteration n: one Philox block, counter (t >> 1, n, k, 0),
// serves steps 2m (words 0, 1) and 2m + 1 (words 2, 3) -- readings 5 and 6.
template <bool PRECISE>
__device__ __forceinline__ float2 normal_pair(uint32_t t, uint32_t n, uint32_t k, uint32_t key0,
                                              uint32_t key1) {
  const uint4 w = philox4x32_10(t >> 1, n, k, 0u, key0, key1);
  return (t & 1u) ? box_muller<PRECISE>(w.z, w.w) : box_muller<PRECISE>(w.x, w.y);
}

// alpha_k ~ U[alpha_lo, alpha_hi), Philox counter (0, n, k, 1) word 0 (reading 8).
__device__ __forceinline__ float sample_alpha(const DeviceParams& P, uint32_t n, uint32_t k,
                                              uint32_t key0, uint32_t key1) {
  const uint4 w = philox4x32_10(0u, n, k, 1u, key0, key1);
  return fmaf(P.alpha_span, uniform23(w.x), P.alpha_lo);
}

// u~ = clamp(u_nom + sigma z) (reading 9).
template <bool PRECISE>
__device__ __forceinline__ float2 sample_control(const DeviceParams& P, float2 u_nom, uint32_t t,
                                                 uint32_t n, uint32_t k, uint32_t key0,
                                                 uint32_t key1) {
  const float2 z = normal_pair<PRECISE>(t, n, k, key0, key1);
  float v = fmaf(P.sigma_v, z.x, u_nom.x);
  float d = fmaf(P.sigma_delta, z.y, u_nom.y);
  v = fminf(fmaxf(v, P.v_min), P.v_max);
  d = fminf(fmaxf(d, P.delta_min), P.delta_max);
  return make_float2(v, d);
}

// Both steps of pair m (steps 2m and 2m + 1) from ONE Philox block: what the persistent kernel uses.
template <bool PRECISE>
__device__ __forceinline__ void sample_control_pair(const DeviceParams& P, float2 u_nom0, float2 u_nom1,
                                                    uint32_t m, uint32_t n, uint32_t k, uint32_t key0,
                                                    uint32_t key1, float2* u0, float2* u1) {
  const uint4 w = philox4x32_10(m, n, k, 0u, key0, key1);
  const float2 z0 = box_muller<PRECISE>(w.x, w.y), z1 = box_muller<PRECISE>(w.z, w.w);
  u0->x = fminf(fmaxf(fmaf(P.sigma_v, z0.x, u_nom0.x), P.v_min), P.v_max);
  u0->y = fminf(fmaxf(fmaf(P.sigma_delta, z0.y, u_nom0.y), P.delta_min), P.delta_max);
  u1->x = fminf(fmaxf(fmaf(P.sigma_v, z1.x, u_nom1.x), P.v_min), P.v_max);
  u1->y = fminf(fmaxf(fmaf(P.sigma_delta, z1.y, u_nom1.y), P.delta_min), P.delta_max);
}

template <bool PRECISE>
__device__ __forceinline__ void sincos_t(float a, float* s, float* c) {
  if (PRECISE) {
    sincosf(a, s, c);
  } else {
    *s = fast_sin(a);   // MUFU.SIN after a 1/2pi multiply; abs error ~2^-21.4 for |a| <= pi,
    *c = fast_cos(a);   // growing slowly outside (|psi| stays below ~4.6 rad over a horizon)
  }
}

template <bool PRECISE>
__device__ __forceinline__ float tan_t(float a) {
  if (PRECISE) return tanf(a);
  // |delta| < 1.5 (checked at create): cos > 0, so tan = sin / sqrt(1 - sin^2); two MUFU, not three
  const float sn = fast_sin(a);
  return sn * fast_rsqrt(fmaf(-sn, sn, 1.0f));
}

// wrap(a) = a - 2 pi rint(a / 2 pi)
__device__ __forceinline__ float wrap_angle(float a) {
  return fmaf(-kTwoPi, rintf(a * kInvTwoPi), a);
}

// Same value without the XU-pipe FRND: adding and subtracting 1.5 * 2^23 rounds to the nearest
// integer (ties to even, like rintf) for |a / 2 pi| < 2^22; two FMA-pipe adds.  No fast-math
// flags are used in this build, so the compiler keeps both additions.
__device__ __forceinline__ float wrap_angle_fma(float a) {
  const float r = __fadd_rn(__fmaf_rn(a, kInvTwoPi, 12582912.0f), -12582912.0f);
  return fmaf(-kTwoPi, r, a);
}

// Vehicle state in the solve's local frame (origin at the start position).
struct State { float x, y, psi1, psi2; };

// One explicit-Euler step of the reduced eq. (6), every right-hand side at the old state
// (reading 20).  s1/c1 = sin/cos(psi1), s2/c2 = sin/cos(psi2) of the OLD state
// (sin/cos(psi1 - psi2) by the angle-difference identity, no extra MUFU).
__device__ __forceinline__ State kinematic_step(const DeviceParams& P, const State& X, float s1,
                                                float c1, float s2, float c2, float v, float tan_d) {
  const float a = P.dt * v;
  const float sb = s1 * c2 - c1 * s2;
  const float cb = fmaf(c1, c2, s1 * s2);
  State N;
  N.x = fmaf(a, c1, X.x);
  N.y = fmaf(a, s1, X.y);
  N.psi1 = fmaf(a * P.inv_L1, tan_d, X.psi1);
  N.psi2 = fmaf(a * P.inv_L2, fmaf(-P.Lh_over_L1 * tan_d, cb, sb), X.psi2);
  return N;
}

// Disc centres of the vehicle at state X given sin/cos of its two headings (reading 11).
__device__ __forceinline__ void disc_centres(const DeviceParams& P, const State& X, float s1,
                                             float c1, float s2, float c2, float cx[kMaxDiscs],
                                             float cy[kMaxDiscs]) {
  const float hx = fmaf(-P.Lh, c1, X.x), hy = fmaf(-P.Lh, s1, X.y);
#pragma unroll
  for (int j = 0; j < kMaxDiscs; ++j) {
    if (j < P.n_discs) {
      const bool trailer = P.disc_body[j] != 0;
      cx[j] = fmaf(P.disc_offset[j], trailer ? c2 : c1, hx);
      cy[j] = fmaf(P.disc_offset[j], trailer ? s2 : s1, hy);
    }
  }
}

// Same with the disc count fixed at compile time (no predicated-off fourth disc).
template <int ND>
__device__ __forceinline__ void disc_centres_n(const DeviceParams& P, float x, float y, float s1,
                                               float c1, float s2, float c2, float (&cx)[ND],
                                               float (&cy)[ND]) {
  const float hx = fmaf(-P.Lh, c1, x), hy = fmaf(-P.Lh, s1, y);
#pragma unroll
  for (int j = 0; j < ND; ++j) {
    // one of the two coefficients is zero: the same value as offset * (body axis), without a select
    cx[j] = fmaf(P.disc_a1[j], c1, fmaf(P.disc_a2[j], c2, hx));
    cy[j] = fmaf(P.disc_a1[j], s1, fmaf(P.disc_a2[j], s2, hy));
  }
}

// Goal cost G(X) =w_pos ||p - g||^2 + w_head (wrap(psi1 - g1)^2 + wrap(psi2 - g2)^2).
__device__ __forceinline__ float goal_cost(const DeviceParams& P, const State& X, const float4 g) {
  const float ex = X.x - g.x, ey = X.y - g.y;
  const float e1 = wrap_angle(X.psi1 - g.z), e2 = wrap_angle(X.psi2 - g.w);
  return fmaf(P.w_pos, fmaf(ex, ex, ey * ey), P.w_head * fmaf(e1, e1, e2 * e2));
}

// Goal + hitch stage cost with the FMA-pipe wrap (persistent-CTA kernel, fast-math mode).
__device__ __forceinline__ float tracking_cost_fma(const DeviceParams& P, const State& X, const float4 g, float v) {
  const float ex = X.x - g.x, ey = X.y - g.y;
  const float e1 = wrap_angle_fma(X.psi1 - g.z), e2 = wrap_angle_fma(X.psi2 - g.w);
  const float G = fmaf(P.w_pos, fmaf(ex, ex, ey * ey), P.w_head * fmaf(e1, e1, e2 * e2));
  const float e = fmaxf(fabsf(wrap_angle_fma(X.psi1 - X.psi2)) - fmaf(-P.hitch_kappa, fabsf(v), P.hitch_max), 0.0f);
  return fmaf(P.w_hitch * e, e, G);
}

// Hitch-angle squared hinge (reading 15).
__device__ __forceinline__ float hitch_cost(const DeviceParams& P, const State& X, float v) {
  const float e = fmaxf(fabsf(wrap_angle(X.psi1 - X.psi2)) - fmaf(-P.hitch_kappa, fabsf(v), P.hitch_max), 0.0f);
  return P.w_hitch * e * e;
}

// Lexicographic (value, index) minimum over a warp; non-finite values never win.
__device__ __forceinline__ void warp_argmin(double& m, int& idx) {
  // Three warp-wide integer minima (REDUX) instead of five shuffle rounds on a (double, int)
  // pair: the double becomes an order-preserving 64-bit key (NaN never occurs here: non-finite
  // costs were replaced by +inf), compared high word first, then low word, then the index.
  const unsigned long long b = (unsigned long long)__double_as_longlong(m);
  const unsigned long long key = (b >> 63) ? ~b : (b | 0x8000000000000000ull);
  const unsigned hi = (unsigned)(key >> 32), lo = (unsigned)key;
  const unsigned min_hi = __reduce_min_sync(0xffffffffu, hi);
  const unsigned min_lo = __reduce_min_sync(0xffffffffu, hi == min_hi ? lo : 0xffffffffu);
  const bool is_min = (hi == min_hi) && (lo == min_lo);
  const unsigned min_idx = __reduce_min_sync(0xffffffffu, is_min ? (unsigned)idx : 0xffffffffu);
  const unsigned long long mk = ((unsigned long long)min_hi << 32) | min_lo;
  const unsigned long long mb = (mk >> 63) ? (mk & 0x7fffffffffffffffull) : ~mk;
  m = __longlong_as_double((long long)mb);
  idx = (int)min_idx;
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

}  // namespace brmppi
