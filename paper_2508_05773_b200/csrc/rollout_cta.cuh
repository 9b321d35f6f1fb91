// rollout_cta.cuh -- the default rollout kernel for sm_100a: ONE PERSISTENT CTA PER SM that walks
// a contiguous range of sample tiles through five phases (plan + shared-memory layout here, the
// kernel itself in rollout_cta_kernel.cuh).
//
// Why not one thread per sample (rollout_thread.cuh)?  At K = 16384 that is 512 warps for 592
// warp schedulers (148 SMs x 4): under one warp per scheduler, nothing to hide the Philox /
// MUFU / Euler dependency chains behind (SURVEY §7 hard part 1).  Only the Euler recursion is
// serial in t; noise generation is parallel over (k, t), and the barrier evaluation -- 8 of every
// 10 instructions -- is parallel over (k, t, obstacle, disc) once the headings exist.  So a CTA of
// 512 threads takes a tile of S samples (S = ceil(K / #SMs) when that fits in shared memory: 111
// at K = 16384, i.e. the whole problem is ONE balanced wave) and runs, per tile:
//
//   A  noise      the (sample, step-pair) items are dealt round-robin over all 512 threads: one
//                 Philox block per pair of steps -> Box-Muller -> perturb + clamp (a1, a2); stores v,
//                 delta and the heading increment dpsi1 = dt v tan(delta) / L1 to shared-memory
//                 planes.
//   B  chain      the S threads of warps 0..3 (one warp per scheduler) run the serial Euler
//                 recursion of eq. (6) (a3), one sample each, and little else (the effort cost
//                 rides along): a single in-order instruction stream per step is the critical
//                 path of the whole tile.  psi1, psi2 of every step go to shared planes, (x, y)
//                 only at the chunk boundaries.  Warp 4 sorts the obstacle tables meanwhile.
//   C  cost       thread (s, c) walks steps [cL, cL+L) of sample s: re-integrates (x, y) from its
//                 chunk boundary (two FMAs, bit-identical to the chain), disc centres, barrier h
//                 for every (obstacle, disc) with h_t in registers, barrier-rate hinge (a4, a5),
//                 goal / heading / hitch cost (a6).  Obstacles go in groups of 8 (padded with null
//                 obstacles of weight 0) held in registers; super-ellipses in groups of 4.
//   D  reduce     S threads add effort + chunk partials in a fixed order (fp64), block argmin,
//                 weights against the CTA's running minimum (online softmax, a7).
//   E  update     threads (channel, t) rescale the running A[t] and add sum_s w_s u_s[t] from the
//                 control planes still in shared memory (a7).
//
// Trajectories and noise never leave the SM.  One partial (m, argmin, eta, A[2T]) per (CTA,
// scene) goes to HBM and is merged by merge_update (update.cuh) in CTA order.  Tiles are assigned
// to CTAs statically (a contiguous range of the flat (scene, tile) list): bit-reproducible.
#pragma once

#include "brmppi_device.cuh"

namespace brmppi {

#ifndef BRMPPI_CTA_THREADS
#define BRMPPI_CTA_THREADS 512
#endif
constexpr int kCtaThreads = BRMPPI_CTA_THREADS;
constexpr int kCtaWarps = kCtaThreads / 32;
constexpr int kChainWarps = 4;                      // one per warp scheduler: the LAST four warps of the CTA
constexpr int kMaxTileSamples = kChainWarps * 32;   // 128
constexpr int kChainFirstThread = kCtaThreads - kMaxTileSamples;   // chain thread of sample s: this + s
constexpr int kWorkerThreads = kChainFirstThread;   // threads that only generate noise and evaluate costs
constexpr int kTableWarp = kCtaWarps - kChainWarps - 1;   // writes the obstacle tables of a scene
constexpr int kObsGroup = 8;                        // obstacles whose h_t are held in registers at a time
constexpr int kSeGroup = 4;                         // super-ellipses whose h_t are held in registers at a time
constexpr int kMaxChunks = 16;
constexpr int kMinChunkLen = 4;
constexpr int kPhaseSlots = 7;                      // prologue, A, chain (runs under C), B + C, D, E, partial out
constexpr int kChainSlot = 2;
constexpr size_t kSmemMax = 232448;                 // 227 KB opt-in dynamic shared memory per CTA

struct CtaMisc {            // lives in the "misc" section
  double m[2];              // running minimum of S over the CTA's tiles of this scene (by parity)
  int argmin[2];
  float eta[2], w2[2];
  int nonfinite[2];
  int n_obs, n_groups, n_se_groups;
  unsigned moving_groups;   // bit g: some obstacle of group g moves
  float4 x0, g;             // start state; goal in the vehicle-centred frame
  double redM[kChainWarps];
  int redI[kChainWarps];
  float redF[3][kChainWarps];
  unsigned long long phase_acc[kPhaseSlots], t_begin;   // BRMPPI_FLAG_PHASE_TIMING
  // chunk hand-off from the chain warps to the cost threads (one phase per tile): bar_chunk[c]
  // completes when every chain thread has stored the headings of steps <= (c + 1) L and the
  // (x, y) at the start of chunk c + 1
  unsigned long long bar_chunk[kMaxChunks];
};

struct CtaSmem {
  size_t obs, vel, thr, se, A, scratch, w, alpha, cost, xy, planes, misc, total;
};

// Shared-memory carve-up (host only: the kernel gets the byte offsets through DeviceParams, so
// that a section pointer is smem_raw + a constant-bank offset instead of a live register).
inline CtaSmem cta_smem_layout(int T, int S, int chunks, int ts, int obs_padded, int se_padded) {
  CtaSmem L{};
  size_t off = 0;
  auto take = [&](size_t b) { size_t o = off; off = (off + b + 15) / 16 * 16; return o; };
  L.obs = take(sizeof(float4) * (size_t)obs_padded);
  L.vel = take(sizeof(float2) * (size_t)obs_padded);
  L.thr = take(sizeof(float) * kMaxDiscs * (size_t)obs_padded);   // culling thresholds per (obstacle, disc)
  L.se = take(sizeof(float) * 12 * (size_t)se_padded);    // SeRecord per super-ellipse
  L.A = take(sizeof(float) * 2 * (size_t)T);
  L.scratch = take(sizeof(float) * kCtaThreads);
  L.w = take(sizeof(float) * (size_t)S);
  L.alpha = take(sizeof(float) * (size_t)S);
  L.cost = take(sizeof(double) * (size_t)chunks * S);
  L.xy = take(sizeof(float2) * (size_t)(chunks + 1) * S);
  L.planes = take(sizeof(float) * 4 * (size_t)S * ts);   // v, delta, psi1, psi2
  L.misc = take(sizeof(CtaMisc));
  L.total = off;
  return L;
}

struct CtaPlan {
  int S_tile, tiles_per_scene, total_tiles, grid, tiles_per_cta, chunks, chunk_len, ts, obs_padded,
      se_padded, n_partials;
  size_t smem;
};

// C threads per sample, L = ceil(T / C) steps per thread.  A thread evaluates L + 1 barrier
// sets (h at its first state plus L new ones); with threads to spare the smallest L wins.
inline void cta_chunking(int T, int S, int* chunks, int* chunk_len) {
  // chunks 0 .. C-2 go to the worker threads, the last chunk to the chain threads once the chain is done
  int cmax = kWorkerThreads / S + 1;
  if (cmax > kMaxChunks) cmax = kMaxChunks;
  if (cmax < 1) cmax = 1;
  int L = (T + cmax - 1) / cmax;
  const int lmin = T < kMinChunkLen ? T : kMinChunkLen;
  if (L < lmin) L = lmin;
  *chunk_len = L;
  *chunks = (T + L - 1) / L;
}

inline size_t cta_smem_bytes(int T, int S, int obs_padded, int se_padded, int* chunks, int* chunk_len, int* ts) {
  cta_chunking(T, S, chunks, chunk_len);
  *ts = (T + 1) | 1;                     // T+1 entries per row, odd length: conflict-free planes
  return cta_smem_layout(T, S, *chunks, *ts, obs_padded, se_padded).total;
}

inline CtaPlan make_cta_plan(int K, int T, int n_scenes, int max_obstacles, int max_superellipses, int n_sms) {
  CtaPlan pl{};
  pl.obs_padded = max_obstacles > 0 ? (max_obstacles + kObsGroup - 1) / kObsGroup * kObsGroup : kObsGroup;
  pl.se_padded = (max_superellipses + kSeGroup - 1) / kSeGroup * kSeGroup;
  // largest tile that fits in shared memory
  int s_max = K < kMaxTileSamples ? K : kMaxTileSamples;
  int c, l, ts;
  while (s_max > 1 && cta_smem_bytes(T, s_max, pl.obs_padded, pl.se_padded, &c, &l, &ts) > kSmemMax) --s_max;
  // fewest tiles, then cut them smaller until the last round of CTAs is full
  const long tps_min = (K + s_max - 1) / s_max;
  const long n_min = tps_min * n_scenes;
  const long rounds = (n_min + n_sms - 1) / n_sms;
  long tps = rounds * n_sms / n_scenes;
  if (tps < tps_min) tps = tps_min;
  const long tps_cap = (K + 7) / 8;      // but keep at least 8 samples per tile
  if (tps > tps_cap) tps = tps_cap > tps_min ? tps_cap : tps_min;
  pl.S_tile = (int)((K + tps - 1) / tps);
  pl.tiles_per_scene = (K + pl.S_tile - 1) / pl.S_tile;
  pl.total_tiles = pl.tiles_per_scene * n_scenes;
  int grid = pl.total_tiles < n_sms ? pl.total_tiles : n_sms;
  pl.tiles_per_cta = (pl.total_tiles + grid - 1) / grid;
  pl.grid = (pl.total_tiles + pl.tiles_per_cta - 1) / pl.tiles_per_cta;
  // CTAs whose range touches one scene: at most ceil((tps - 1) / Q) + 1
  int np = (pl.tiles_per_scene + pl.tiles_per_cta - 2) / pl.tiles_per_cta + 1;
  if (np > pl.grid) np = pl.grid;
  pl.n_partials = np;
  pl.smem = cta_smem_bytes(T, pl.S_tile, pl.obs_padded, pl.se_padded, &pl.chunks, &pl.chunk_len, &pl.ts);
  return pl;
}

}  // namespace brmppi
