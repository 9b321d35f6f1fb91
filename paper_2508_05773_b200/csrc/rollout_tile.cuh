// rollout_tile.cuh -- the default rollout kernel for sm_100a: a PHASE-SPLIT TILE kernel.
//
// Why not one thread per sample (rollout_thread.cuh)?  At K = 16384 that is 512 warps for 592
// warp schedulers (148 SMs x 4): under one warp per scheduler, nothing to hide the Philox /
// MUFU / Euler dependency chains behind (SURVEY §7 hard part 1).  Only the Euler recursion is
// serial in t; noise generation is parallel over (k, t), and barrier + cost evaluation is
// parallel over (k, t, obstacle, disc) once the headings exist.  So a CTA takes a tile of
// kTileSamples = 16 samples and C = blockDim/16 threads per sample, and runs, per tile:
//
//   A  noise      thread (s, c) draws the controls of steps [cL, cL+L) of sample s: Philox ->
//                 Box-Muller -> perturb + clamp (a1, a2); stores v, delta and the heading
//                 increment dpsi1 = dt v tan(delta)/L1 to shared-memory planes; effort cost.
//   B  chain      16 threads run the serial Euler recursion of eq. (6) (a3), one sample each;
//                 psi1 overwrites dpsi1 in place, psi2 goes to a fourth plane, (x, y) is kept
//                 only at the chunk boundaries.
//   C  cost       thread (s, c) walks steps [cL, cL+L): re-integrates (x, y) from its chunk
//                 boundary (two FMAs, bit-identical to the chain), disc centres, barrier h for
//                 every (obstacle, disc) with h_t in registers, barrier-rate hinge (a4, a5),
//                 goal / heading / hitch cost (a6).  Obstacles are processed in groups of 8
//                 (padded with null obstacles whose h is identically 0), so the register count
//                 does not depend on the obstacle count.
//   D  reduce     16 threads sum the chunk partials in chunk order (fp64), take the tile's
//                 min / argmin, fold the tile into the CTA's running online-softmax state (a7).
//   E  update     threads (channel, t) rescale the running A[t] and add sum_s w_s u_s[t] from
//                 the control planes still in shared memory (a7).
//
// Trajectories and noise never leave the SM.  One partial (m, argmin, eta, A[2T]) per CTA goes
// to HBM and is merged by merge_update (update.cuh) in CTA-index order.  Tiles are assigned to
// CTAs statically (tile = blockIdx.x + i * gridDim.x): results are bit-reproducible.
#pragma once

#include <cstdlib>

#include "brmppi_device.cuh"

namespace brmppi {

constexpr int kTileSamples = 16;
constexpr int kObsGroup = 8;            // obstacles whose h_t are held in registers at a time
constexpr int kTileMaxThreads = 256;
#ifndef BRMPPI_OBS_LOAD_AHEAD
#define BRMPPI_OBS_LOAD_AHEAD 2
#endif
constexpr int kObsLoadAhead = BRMPPI_OBS_LOAD_AHEAD;

struct TilePlan {
  int tiles_per_scene, blocks_per_scene, chunks, chunk_len, t_stride, threads, obs_padded;
};

inline TilePlan make_tile_plan(int K, int T, int n_scenes, int max_obstacles) {
  TilePlan tp{};
  // C threads per sample, L = ceil(T/C) steps per thread.  A thread evaluates L+1 barrier
  // sets (h at its first state plus L new ones), so the work per sample is ~ C (L+1);
  // C in {8..16} keeps the CTA at 128-256 threads.
  int best_c = 8;
  long best_cost = -1;
  for (int c = 8; c <= 16; c += 2) {
    const int L = (T + c - 1) / c;
    const long cost = (long)c * (L + 1);
    if (best_cost < 0 || cost < best_cost) { best_cost = cost; best_c = c; }
  }
  if (const char* e = getenv("BRMPPI_TILE_CHUNKS")) {   // tuning knob for sweeps
    const int c = atoi(e);
    if (c >= 4 && c <= 16 && c % 2 == 0) best_c = c;
  }
  tp.chunks = best_c;
  tp.chunk_len = (T + best_c - 1) / best_c;
  tp.threads = kTileSamples * best_c;
  tp.t_stride = (T + 1) | 1;            // T+1 entries per row, odd length: conflict-free planes
  tp.tiles_per_scene = (K + kTileSamples - 1) / kTileSamples;
  tp.obs_padded = max_obstacles > 0 ? (max_obstacles + kObsGroup - 1) / kObsGroup * kObsGroup : kObsGroup;
  int cap = 4096 / n_scenes;
  if (cap < 128) cap = 128;
  if (const char* e = getenv("BRMPPI_TILE_MAX_BLOCKS")) {
    const int c = atoi(e);
    if (c >= 1) cap = c;
  }
  tp.blocks_per_scene = tp.tiles_per_scene < cap ? tp.tiles_per_scene : cap;
  return tp;
}

struct TileMisc {           // lives in the "misc" section
  double m;                 // running minimum of S over the CTA's tiles
  int argmin;
  float eta, w2;
  int nonfinite;
  float scale_old;          // rescale of the running sums for the tile being folded in
  int n_moving, n_groups;
  float4 x0, g;             // start state; goal in the vehicle-centred frame
  float w[kTileSamples];    // weights of the current tile
  float alpha[kTileSamples];
};

// Shared-memory carve-up, identical on host and device.
struct TileSmem {
  size_t obs, vel, xy, unom, planes, cost, A, misc, total;
};

__host__ __device__ inline TileSmem tile_smem_layout(int T, int obs_padded, int chunks, int t_stride) {
  TileSmem L{};
  size_t off = 0;
  auto take = [&](size_t b) { size_t o = off; off = (off + b + 15) / 16 * 16; return o; };
  L.obs = take(sizeof(float4) * (size_t)obs_padded);
  L.vel = take(sizeof(float2) * (size_t)obs_padded);
  L.xy = take(sizeof(float2) * (size_t)(chunks + 1) * kTileSamples);
  L.unom = take(sizeof(float2) * (size_t)T);
  L.planes = take(sizeof(float) * 4 * (size_t)kTileSamples * t_stride);
  L.cost = take(sizeof(double) * (size_t)chunks * kTileSamples);
  L.A = take(sizeof(float) * 2 * (size_t)T);
  L.misc = take(sizeof(TileMisc));
  L.total = off;
  return L;
}


// Phase C for one group of kObsGroup obstacles over the steps [t0, t1) of one sample.
// Obstacle record: (ox, oy, 1/rho^2, h0) with h = |c - o|^2 / rho^2 + h0; h0 = -1 for a real
// obstacle, and (0, 0, 0, 0) for a null one, whose h == 0 and hinge == 0 exactly.
struct GroupCost { double track, bar; };

template <bool PRECISE, int ND, bool MOVING>
__device__ __forceinline__ GroupCost cost_group(const DeviceParams& P, const float* __restrict__ pV,
                                           const float* __restrict__ pP1, const float* __restrict__ pP2,
                                           const float4* __restrict__ obs, const float2* __restrict__ vel,
                                           float x, float y, int t0, int t1, float one_minus_alpha,
                                           const float4 g, const bool first) {
  // accumulators are plain locals (never address-taken), so the "memory" clobbers below cannot
  // force them into local memory
  double track = 0.0, bar = 0.0;
  float hprev[kObsGroup][ND];
  float s1, c1, s2, c2;
  {
    sincos_t<PRECISE>(pP1[t0], &s1, &c1);
    sincos_t<PRECISE>(pP2[t0], &s2, &c2);
    float cx[ND], cy[ND];
    disc_centres_n<ND>(P, x, y, s1, c1, s2, c2, cx, cy);
    const float tf = (float)t0;
#pragma unroll
    for (int i = 0; i < kObsGroup; ++i) {
      float4 o = obs[i];
      if (MOVING) { const float2 w = vel[i]; o.x = fmaf(tf, w.x, o.x); o.y = fmaf(tf, w.y, o.y); }
#pragma unroll
      for (int j = 0; j < ND; ++j) {
        const float dx = cx[j] - o.x, dy = cy[j] - o.y;
        hprev[i][j] = fmaf(fmaf(dx, dx, dy * dy), o.z, o.w);
      }
    }
  }
  for (int t = t0; t < t1; ++t) {
    // Re-read the obstacle records from shared memory every step instead of letting the
    // compiler hoist all 8 of them (32 registers) out of the loop: occupancy matters more here
    // than 8 LDS.128 per step.
    asm volatile("" ::: "memory");
    // (x, y) of state t+1 from state t: the chain's own FMAs on the same operands
    const float a = P.dt * pV[t];
    x = fmaf(a, c1, x);
    y = fmaf(a, s1, y);
    const float psi1 = pP1[t + 1], psi2 = pP2[t + 1];
    sincos_t<PRECISE>(psi1, &s1, &c1);
    sincos_t<PRECISE>(psi2, &s2, &c2);
    float cx[ND], cy[ND];
    disc_centres_n<ND>(P, x, y, s1, c1, s2, c2, cx, cy);
    if (first) {   // block-uniform: the first group also carries the per-step tracking cost
      const State X{x, y, psi1, psi2};
      track += (double)(goal_cost(P, X, g) + hitch_cost(P, X));
    }
    const float tf = (float)(t + 1);
    float pen = 0.0f;
#pragma unroll
    for (int i = 0; i < kObsGroup; ++i) {
      // at most kObsLoadAhead obstacle records in flight: keeps the scheduler from batching all
      // eight LDS.128 (32 registers) at the top of the step
      if (i % kObsLoadAhead == 0) asm volatile("" ::: "memory");
      float4 o = obs[i];
      if (MOVING) { const float2 w = vel[i]; o.x = fmaf(tf, w.x, o.x); o.y = fmaf(tf, w.y, o.y); }
#pragma unroll
      for (int j = 0; j < ND; ++j) {
        const float dx = cx[j] - o.x, dy = cy[j] - o.y;
        const float hn = fmaf(fmaf(dx, dx, dy * dy), o.z, o.w);
        pen += fmaxf(fmaf(one_minus_alpha, hprev[i][j], -hn), 0.0f);   // barrier-rate hinge
        hprev[i][j] = hn;
      }
    }
    bar += (double)pen;
  }
  return GroupCost{track, bar};
}

}  // namespace brmppi
