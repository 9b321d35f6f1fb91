"""Parity of the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Tolerances (north_star; reading 22): Philox integers and the argmin index bit-exact;
final states, costs and controls within 1e-4 relative, i.e. |a-b| <= 1e-4 max(|b|, floor) with
floor = 1 (m, rad) for x_T and S_k, and v_max / delta_max for the two control channels.  The
argmin index is required to match only when the oracle's gap S_(2) - S_(1) exceeds
1e-3 max(1, |S_(1)|) (reading 21)."""
import numpy as np
import pytest

import scenes

pytestmark = pytest.mark.gpu

RTOL = 1e-4


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    from paper_2508_05773_b200 import brmppi
    brmppi.lib()
    return brmppi


def close(a, b, floor):
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    return np.abs(a - b) <= RTOL * np.maximum(np.abs(b), floor)


def gpu_solve(B, sc, p, flags=0, n0=0, U0=None, max_obstacles=None):
    n_obs = len(sc.obstacles)
    mo = max_obstacles if max_obstacles is not None else max(n_obs, 1)
    s = B.Solver(p, 1, mo, flags | B.FLAG_WRITE_SAMPLES)
    s.set_scene(sc)
    s.set_nominal(U0)
    s.set_counter(n0)
    s.solve()
    out = dict(U=s.get_controls(), S=s.get_costs(), XT=s.get_final_states(), diag=s.get_diag())
    s.close()
    return out


def check_against_oracle(O, got, sc, p, n0=0, U0=None, n_threads=8):
    U = np.zeros((p.T, 2)) if U0 is None else np.asarray(U0, dtype=np.float64)
    ref = O.solve(p, n0, sc.x0, sc.goal, sc.obstacles, U, n_threads=n_threads)[-1]
    okS = close(got["S"], ref["S"], 1.0)
    assert okS.all(), f"S_k: {np.count_nonzero(~okS)} of {p.K} off, worst {np.abs(got['S'] - ref['S']).max()}"
    okX = close(got["XT"], ref["XT"], 1.0)
    assert okX.all(), f"x_T worst {np.abs(got['XT'] - ref['XT']).max()}"
    floors = np.array([p.v_max, p.delta_max])
    okU = close(got["U"], ref["U"], floors[None, :])
    err = np.abs(got["U"] - ref["U"]) / (RTOL * np.maximum(np.abs(ref["U"]), floors[None, :]))
    assert okU.all(), f"U worst error = {err.max():.2f} x tolerance"
    d = got["diag"]
    if ref["gap"] > 1e-3 * max(1.0, abs(ref["S"].min())):
        assert d["argmin"] == ref["argmin"]
    assert close(d["S_min"], ref["S"].min(), 1.0)
    assert abs(d["eta"] - ref["eta"]) <= 2e-3 * ref["eta"]
    assert d["nonfinite"] == 0 and d["n"] == n0 + p.n_iter
    return dict(ref=ref, u_err=float(err.max()))


KERNELS = [pytest.param(0, id="tile"), pytest.param(4, id="thread")]


# ------------------------------------------------------------------------------------------
# Philox integers and drawn controls
# ------------------------------------------------------------------------------------------
def test_philox_bit_exact(B, O):
    rng = np.random.default_rng(0)
    for seed, n, tag in [(0, 0, 0), (0, 0, 1), (2**63 + 12345, 7, 0), (0xFFFFFFFFFFFFFFFF, 0xFFFFFFFF, 1),
                         (int(rng.integers(0, 2**62)), int(rng.integers(0, 2**31)), 0)]:
        K, T = 67, 33
        w = B.debug_philox(seed, n, K, T, tag)
        key = (seed & 0xFFFFFFFF, seed >> 32)
        for k, t in [(0, 0), (5, 3), (66, 32), (17, 0), (0, 31)] + [tuple(x) for x in rng.integers(0, 33, size=(20, 2))]:
            assert tuple(int(x) for x in w[k, t]) == O.philox((t, n, k, tag), key)


def test_philox_matches_curand_device_function(B, O):
    """Library pin (SURVEY 8(c) pin (ii)): the CUDA toolkit's own raw curand_Philox4x32_10(uint4, uint2)
    device function, this library's generator and the oracle give the same four words for random
    (counter, key) pairs -- three independent implementations of the published block function."""
    rng = np.random.default_rng(20250805)
    n = 4096
    ctr = rng.integers(0, 2**32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2**32, size=(n, 2), dtype=np.uint64).astype(np.uint32)
    ctr[0] = 0; key[0] = 0                                 # the published known-answer vectors ride along
    ctr[1] = 0xFFFFFFFF; key[1] = 0xFFFFFFFF
    ctr[2] = [0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344]; key[2] = [0xa4093822, 0x299f31d0]
    ours = B.debug_philox_raw(ctr, key, use_curand=False)
    theirs = B.debug_philox_raw(ctr, key, use_curand=True)
    assert np.array_equal(ours, theirs)
    assert [int(x) for x in theirs[0]] == [0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8]
    assert [int(x) for x in theirs[1]] == [0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd]
    assert [int(x) for x in theirs[2]] == [0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1]
    for i in list(range(3)) + [int(x) for x in rng.integers(0, n, 200)]:
        want = O.philox(tuple(int(x) for x in ctr[i]), tuple(int(x) for x in key[i]))
        assert tuple(int(x) for x in theirs[i]) == want
    assert B.debug_philox_raw(np.zeros((0, 4)), np.zeros((0, 2)), use_curand=True).shape == (0, 4)


def test_philox_layout_is_curand_state_layout(B):
    """The counter layout (t, n, k, tag) with key (lo32, hi32)(seed) is cuRAND's Philox state layout
    (curand_kernel.h: ctr.xy = offset / 4, ctr.zw = subsequence): block (0, 0, 0, 0) of seed 0."""
    w = B.debug_philox(0, 0, 1, 1, 0)
    assert [int(x) for x in w[0, 0]] == [0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8]


@pytest.mark.parametrize("flags", [0, 2], ids=["fast", "precise"])
def test_sampled_controls_match_oracle(B, O, flags):
    p = scenes.default_params(K=300, T=40, seed=99)
    U0 = np.tile([0.5, -0.1], (40, 1)).astype(np.float32)
    u, a = B.debug_sample_controls(p, 3, U0, flags)
    ref = O.iteration(p, 3, np.zeros(4), np.zeros(4), np.zeros((0, 5)), U0, want_samples=True)["u"]
    floors = np.array([p.v_max, p.delta_max])
    tol = 2e-6 if flags else 1e-5          # absolute, well inside the 1e-4 relative budget
    assert np.abs(u - ref).max() <= tol
    assert close(u, ref, floors).all()
    a_ref = np.array([O.alpha(p, 3, k) for k in range(p.K)])
    assert np.abs(a - a_ref).max() <= 1e-6
    # clamping produces exact bound values on both sides at the same places
    assert np.array_equal(u[..., 0] == p.v_max, ref[..., 0] == p.v_max)


# ------------------------------------------------------------------------------------------
# BASELINE.json configs
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("precise", [0, 2], ids=["fast", "precise"])
def test_cfg0(B, O, kernel, precise):
    sc = scenes.scene_cfg0(0)
    got = gpu_solve(B, sc, sc.params, kernel | precise)
    check_against_oracle(O, got, sc, sc.params)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_cfg1(B, O, kernel, seed):
    sc = scenes.scene_cfg1(seed)
    got = gpu_solve(B, sc, sc.params, kernel)
    check_against_oracle(O, got, sc, sc.params)


@pytest.mark.parametrize("kernel", KERNELS)
def test_cfg2_three_iterations_moving_obstacles(B, O, kernel):
    sc = scenes.scene_cfg2(0)
    got = gpu_solve(B, sc, sc.params, kernel)
    check_against_oracle(O, got, sc, sc.params)


def test_cfg2_warm_nominal_and_counter(B, O):
    sc = scenes.scene_cfg2(1)
    p = sc.params.with_(K=4096, n_iter=2)
    rng = np.random.default_rng(5)
    U0 = np.stack([rng.uniform(-1.5, 1.5, p.T), rng.uniform(-0.4, 0.4, p.T)], axis=1).astype(np.float32)
    got = gpu_solve(B, sc, p, 0, n0=1000, U0=U0)
    check_against_oracle(O, got, sc, p, n0=1000, U0=U0)


# ------------------------------------------------------------------------------------------
# edge cases: ragged tiles, tiny horizons, obstacle counts, geometry variants
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("K,T", [(1, 1), (1, 30), (17, 7), (129, 13), (1000, 50), (2049, 100), (333, 61)])
def test_ragged_sizes(B, O, kernel, K, T):
    sc = scenes.scene_static(3, 8, K=K, T=T)
    got = gpu_solve(B, sc, sc.params, kernel)
    check_against_oracle(O, got, sc, sc.params)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("n_obs", [0, 1, 7, 9, 32, 64])
def test_obstacle_counts(B, O, kernel, n_obs):
    sc = scenes.scene_static(4, n_obs, K=512, T=50)
    got = gpu_solve(B, sc, sc.params, kernel, max_obstacles=64 if n_obs else 0)
    check_against_oracle(O, got, sc, sc.params)


@pytest.mark.parametrize("kernel", KERNELS)
def test_geometry_variants(B, O, kernel):
    sc = scenes.scene_cfg2(2)
    # off-axle hitch, four discs, asymmetric bounds, other temperature
    p = sc.params.with_(K=1024, T=40, n_iter=1, Lh=1.15, L1=3.23, L2=2.9,
                        discs=((0, 1.5), (0, -0.5), (1, -1.0), (1, -2.5)), disc_radius=1.1,
                        v_min=-1.0, v_max=2.5, delta_min=-0.5, delta_max=0.7, lam=5.0, dt=0.04)
    got = gpu_solve(B, sc, p, kernel)
    check_against_oracle(O, got, sc, p)
    # one disc, vehicle starting inside an obstacle's inflated disc (h < 0 path)
    p1 = sc.params.with_(K=512, T=20, n_iter=1, discs=((0, 0.0),))
    sc1 = scenes.Scene(sc.x0, sc.goal, np.vstack([sc.obstacles, [[sc.x0[0] + 1.0, sc.x0[1], 1.0, 0.0, 0.0]]]).astype(np.float32).astype(np.float64), p1)
    got = gpu_solve(B, sc1, p1, kernel)
    check_against_oracle(O, got, sc1, p1)


@pytest.mark.parametrize("kernel", KERNELS)
def test_degenerate_noise_and_temperature(B, O, kernel):
    sc = scenes.scene_cfg1(5)
    U0 = np.tile([0.75, 0.125], (sc.params.T, 1)).astype(np.float32)
    # sigma = 0: all samples identical, U is a fixed point of the update (bit-exact)
    p = sc.params.with_(K=256, sigma_v=0.0, sigma_delta=0.0)
    got = gpu_solve(B, sc, p, kernel, U0=U0)
    assert np.array_equal(got["U"], U0)
    assert np.all(got["S"] == got["S"][0])
    assert got["diag"]["eta"] == pytest.approx(256.0)
    # lambda -> 0: U is the argmin sample's control sequence
    p = sc.params.with_(K=256, lam=1e-6)
    got = gpu_solve(B, sc, p, kernel, U0=U0)
    r = check_against_oracle(O, got, sc, p, U0=U0)
    # lambda -> infinity: plain mean
    p = sc.params.with_(K=256, lam=1e12)
    got = gpu_solve(B, sc, p, kernel, U0=U0)
    check_against_oracle(O, got, sc, p, U0=U0)
    assert got["diag"]["eta"] == pytest.approx(256.0, rel=1e-5)


def test_all_costs_nonfinite_leaves_U(B):
    sc = scenes.scene_cfg1(6)
    U0 = np.tile([0.5, 0.1], (sc.params.T, 1)).astype(np.float32)
    p = sc.params.with_(K=200, w_pos=3e38)        # every stage cost overflows fp32
    for kernel in (0, 4):
        got = gpu_solve(B, sc, p, kernel, U0=U0)
        assert np.array_equal(got["U"], U0)
        assert got["diag"]["nonfinite"] == 200 and got["diag"]["argmin"] == -1


def test_some_costs_nonfinite_get_zero_weight(B, O):
    sc = scenes.scene_cfg1(6)
    # the fp32 effort term w_v v^2 overflows to inf for samples with some |v| > ~1.06; the others
    # stay finite (huge), and the oracle's fp64 costs of the overflowing samples are larger
    # than every finite one, so both sides put all the weight on the same sample
    # (T = 1: with more steps the SUM of finite fp32 terms can exceed FLT_MAX while each term
    # and the fp64 accumulator stay finite, which is a different, benign, case)
    p = sc.params.with_(K=512, T=1, w_v=3e38)
    for kernel in (0, 4):
        got = gpu_solve(B, sc, p, kernel)
        ref = O.iteration(p, 0, sc.x0, sc.goal, sc.obstacles, np.zeros((p.T, 2)))
        n_inf = int(np.count_nonzero(~np.isfinite(got["S"])))
        assert 0 < n_inf < p.K and got["diag"]["nonfinite"] == n_inf
        floors = np.array([p.v_max, p.delta_max])
        assert close(got["U"], ref["U"], floors[None, :]).all()
        assert got["diag"]["argmin"] == ref["argmin"]


# ------------------------------------------------------------------------------------------
# batches, determinism, shift, closed loop
# ------------------------------------------------------------------------------------------
def test_batched_scenes_equal_single_scene_solves(B, O):
    scs = [scenes.scene_cfg2(s) for s in range(3)]
    p = scs[0].params.with_(K=2048, T=80, n_iter=2, seed=40)
    s = B.Solver(p, 3, 8, B.FLAG_WRITE_SAMPLES)
    for i, sc in enumerate(scs):
        s.set_scene(sc, i)
    s.solve()
    for i, sc in enumerate(scs):
        pi = p.with_(seed=40 + i)                 # scene i uses seed + i
        single = gpu_solve(B, sc, pi, 0)
        got = dict(U=s.get_controls(i), S=s.get_costs(i), XT=s.get_final_states(i), diag=s.get_diag(i))
        # same draws and arithmetic per sample; the tiling (hence the fp32/fp64 summation order
        # of the chunk partials and of the weighted sums) depends on the batch size
        assert np.allclose(got["S"], single["S"], rtol=2e-6, atol=1e-5)
        assert np.allclose(got["U"], single["U"], rtol=0, atol=2e-5)
        assert got["diag"]["argmin"] == single["diag"]["argmin"]
        check_against_oracle(O, got, sc, pi)
    s.close()


@pytest.mark.parametrize("kernel", KERNELS)
def test_replay_is_bit_reproducible(B, kernel):
    sc = scenes.scene_cfg2(3)
    p = sc.params.with_(K=8192)
    a = gpu_solve(B, sc, p, kernel)
    b = gpu_solve(B, sc, p, kernel)
    for key in ("U", "S", "XT"):
        assert np.array_equal(a[key], b[key])
    assert a["diag"] == b["diag"]


def test_shift_duplicates_tail(B):
    p = scenes.default_params(K=64, T=37)
    s = B.Solver(p, 2, 1)
    U = np.stack([np.linspace(-1, 1, 37), np.linspace(-0.5, 0.5, 37)], axis=1).astype(np.float32)
    s.set_nominal(U, 0)
    s.set_nominal(U[::-1].copy(), 1)
    s.shift()
    got0, got1 = s.get_controls(0), s.get_controls(1)
    assert np.array_equal(got0[:-1], U[1:]) and np.array_equal(got0[-1], U[-1])
    assert np.array_equal(got1[:-1], U[::-1][1:]) and np.array_equal(got1[-1], U[0])
    s.close()


def test_closed_loop_steps_match_oracle_stepwise(B, O):
    """CFG3 shape (shortened): graph-replayed control steps; after every step the oracle is
    re-seeded with the library's state so each solve / plant step / shift is compared on
    identical inputs (closed-loop trajectories of a sampled controller diverge otherwise)."""
    sc = scenes.scene_cfg2(4)                    # moving obstacles: exercises the obstacle advance
    p = sc.params.with_(K=2048, T=60, n_iter=1)
    s = B.Solver(p, 1, 8)
    s.set_scene(sc)
    x = sc.x0.copy()
    obs = sc.obstacles.copy()
    U = np.zeros((p.T, 2))
    floors = np.array([p.v_max, p.delta_max])
    for step in range(6):
        u0 = s.step()[0]
        ref = O.iteration(p, step, x, sc.goal, obs, U, n_threads=8)
        assert close(u0, ref["U"][0], floors).all()
        x_ref, obs_ref = O.plant_step(p, x, u0.astype(np.float64), obs)
        x_gpu = s.get_state().astype(np.float64)
        assert np.abs(x_gpu[:2] - x_ref[:2]).max() <= 1e-5
        dpsi = (x_gpu[2:] - x_ref[2:] + np.pi) % (2 * np.pi) - np.pi
        assert np.abs(dpsi).max() <= 1e-5
        obs_gpu = s.get_obstacles().astype(np.float64)
        assert np.abs(obs_gpu - obs_ref).max() <= 1e-5
        U_gpu = s.get_controls().astype(np.float64)
        assert close(U_gpu, O.shift(ref["U"]), floors[None, :]).all()
        assert s.get_diag()["n"] == step + 1
        x, obs, U = x_gpu, obs_gpu, U_gpu        # re-seed the oracle with the library's state
    assert s.launch_count() == 6 * 3
    s.close()


# ------------------------------------------------------------------------------------------
# full bench size: sampled outputs the oracle computes one by one + properties
# ------------------------------------------------------------------------------------------
def test_full_size_sampled_parity(B, O):
    sc = scenes.scene_cfg2(0)
    p = sc.params.with_(K=1048576, T=100, n_iter=1)
    got = gpu_solve(B, sc, p, 0)
    rng = np.random.default_rng(1)
    ks = np.concatenate([[0, 15, 16, p.K - 1, int(got["diag"]["argmin"])], rng.integers(0, p.K, 150)])
    U0 = np.zeros((p.T, 2))
    for k in ks:
        r = O.sample(p, 0, int(k), sc.x0, sc.goal, sc.obstacles, U0)
        assert close(got["S"][k], r["S"], 1.0), (k, got["S"][k], r["S"])
        assert close(got["XT"][k], r["xT"], 1.0).all()
    # properties that hold at any size
    d = got["diag"]
    assert np.isfinite(got["S"]).all() and d["nonfinite"] == 0
    assert d["argmin"] == int(np.argmin(got["S"])) or got["S"][d["argmin"]] == got["S"].min()
    assert d["S_min"] == pytest.approx(float(got["S"].min()), rel=1e-6)
    w = np.exp(-(got["S"].astype(np.float64) - float(got["S"].min())) / p.lam)
    assert d["eta"] == pytest.approx(w.sum(), rel=5e-3)
    assert got["U"][:, 0].min() >= p.v_min and got["U"][:, 0].max() <= p.v_max
    assert got["U"][:, 1].min() >= p.delta_min and got["U"][:, 1].max() <= p.delta_max


@pytest.mark.parametrize("n_obs", [32, 64])
def test_many_obstacles_at_size_sampled_parity(B, O, n_obs):
    """The multi-group, culled path in the launch configuration the sweep times (K = 16384, T = 100):
    sampled costs and final states against the oracle, every sample bit-identical to the un-culled run."""
    sc = scenes.scene_static(3, n_obs, K=16384, T=100)
    p = sc.params
    got = gpu_solve(B, sc, p, 0)
    ref = gpu_solve(B, sc, p, B.FLAG_NO_CULL)
    for key in ("S", "XT", "U"):
        assert np.array_equal(got[key], ref[key]), key
    rng = np.random.default_rng(n_obs)
    ks = np.concatenate([[0, 110, 111, p.K - 1, int(got["diag"]["argmin"])], rng.integers(0, p.K, 120)])
    U0 = np.zeros((p.T, 2))
    for k in ks:
        r = O.sample(p, 0, int(k), sc.x0, sc.goal, sc.obstacles, U0)
        assert close(got["S"][k], r["S"], 1.0), (k, got["S"][k], r["S"])
        assert close(got["XT"][k], r["xT"], 1.0).all()
    d = got["diag"]
    assert np.isfinite(got["S"]).all() and d["nonfinite"] == 0
    assert got["S"][d["argmin"]] == got["S"].min()


def test_batch64_at_size_sampled_parity(B, O):
    """BASELINE.json configs[4]'s batched launch -- 64 scenes x K = 16384, T = 80 in one launch -- on sampled
    (scene, sample) pairs against the oracle, and every scene's update inside the control box."""
    batch = scenes.scene_batch(64, 16384, 80)
    p = batch[0].params.with_(seed=0)
    s = B.Solver(p, 64, 8, B.FLAG_WRITE_SAMPLES)
    for i, sc in enumerate(batch):
        s.set_scene(sc, i)
    s.solve()
    rng = np.random.default_rng(64)
    U0 = np.zeros((p.T, 2))
    for i in [0, 1, 31, 63] + [int(x) for x in rng.integers(0, 64, 6)]:
        S, XT, U, d = s.get_costs(i), s.get_final_states(i), s.get_controls(i), s.get_diag(i)
        sc = batch[i]
        pi = p.with_(seed=i)                               # scene i draws with seed + i
        for k in [0, p.K - 1, int(d["argmin"])] + [int(x) for x in rng.integers(0, p.K, 12)]:
            r = O.sample(pi, 0, k, sc.x0, sc.goal, sc.obstacles, U0)
            assert close(S[k], r["S"], 1.0), (i, k, S[k], r["S"])
            assert close(XT[k], r["xT"], 1.0).all()
        assert S[d["argmin"]] == S.min() and d["nonfinite"] == 0
        assert U[:, 0].min() >= p.v_min and U[:, 0].max() <= p.v_max
        assert U[:, 1].min() >= p.delta_min and U[:, 1].max() <= p.delta_max
    s.close()


def test_contexts_of_different_sizes_are_independent(B, O):
    """The shared-memory limit is a per-function attribute: a small context created after a large one
    must not break the large one's next launch (and the other way round)."""
    big_sc, small_sc = scenes.scene_cfg2(2), scenes.scene_cfg0(1)
    pb, ps = big_sc.params.with_(K=16384, T=80, n_iter=1), small_sc.params
    for kernel in (0, 4):
        big = B.Solver(pb, 1, 8, kernel | B.FLAG_WRITE_SAMPLES)
        big.set_scene(big_sc)
        big.solve()
        first = big.get_costs()
        small = B.Solver(ps, 1, 1, kernel | B.FLAG_WRITE_SAMPLES)
        small.set_scene(small_sc)
        small.solve()
        small.synchronize()
        big.set_nominal(None); big.set_counter(0)
        big.solve()                                        # replays the captured graph
        assert np.array_equal(big.get_costs(), first)
        big.time_kernels(2)                                # plain launches outside the graph
        big.step()                                         # captured lazily AFTER the small context exists
        assert np.isfinite(big.get_controls()).all()
        small.solve(); small.step()
        big.close(); small.close()


# ------------------------------------------------------------------------------------------
# boundary errors
# ------------------------------------------------------------------------------------------
def test_error_codes(B):
    import ctypes as C
    import torch
    p = scenes.default_params(K=64, T=10)
    s = B.Solver(p, 1, 2)
    with pytest.raises(B.BrmppiError) as e:
        s.solve()
    assert e.value.status == B.ERR_NOT_READY
    s.set_state([0, 0, 0, 0])
    s.set_goal([1, 0, 0, 0])
    with pytest.raises(B.BrmppiError) as e:
        s.set_obstacles(np.ones((3, 5)))
    assert e.value.status == B.ERR_TOO_MANY_OBSTACLES
    with pytest.raises(B.BrmppiError) as e:
        s.set_state([np.nan, 0, 0, 0])
    assert e.value.status == B.ERR_NONFINITE_INPUT
    with pytest.raises(B.BrmppiError) as e:
        s.set_obstacles([[0, 0, -1.0, 0, 0]])
    assert e.value.status == B.ERR_INVALID_ARG
    with pytest.raises(B.BrmppiError) as e:
        s.set_state([0, 0, 0, 0], scene=1)
    assert e.value.status == B.ERR_INVALID_ARG
    with pytest.raises(B.BrmppiError) as e:
        s.set_nominal(np.tile([5.0, 0.0], (10, 1)))          # outside the control box
    assert e.value.status == B.ERR_INVALID_ARG
    with pytest.raises(B.BrmppiError) as e:
        s.get_costs()                                         # FLAG_WRITE_SAMPLES not set
    assert e.value.status == B.ERR_NOT_READY
    s.solve()
    assert np.isfinite(s.get_controls()).all()
    # psi is wrapped at set_state
    s.set_state([1.0, 2.0, 7.0, -7.0])
    x = s.get_state()
    assert abs(x[2] - (7.0 - 2 * np.pi)) < 1e-6 and abs(x[3] + (7.0 - 2 * np.pi)) < 1e-6
    s.close()
    L = B.lib()
    bad = B.make_cparams(p.with_(lam=0.0))
    assert L.brmppi_workspace_bytes(C.byref(bad)) == 0
    good = B.make_cparams(p)
    ws = torch.empty(1024, dtype=torch.uint8, device="cuda")
    ctx = C.c_void_p()
    ptr = (ws.data_ptr() + 255) // 256 * 256
    assert L.brmppi_create(C.byref(good), C.c_void_p(ptr), 512, None, C.byref(ctx)) == B.ERR_WORKSPACE_TOO_SMALL
    assert L.brmppi_create(C.byref(good), C.c_void_p(ptr + 4), 1 << 30, None, C.byref(ctx)) == B.ERR_UNALIGNED
    assert L.brmppi_create(C.byref(bad), C.c_void_p(ptr), 1 << 30, None, C.byref(ctx)) == B.ERR_INVALID_ARG
    assert L.brmppi_create(None, C.c_void_p(ptr), 1 << 30, None, C.byref(ctx)) == B.ERR_NULL
    assert B.strerror(B.ERR_TOO_MANY_OBSTACLES) == "too many obstacles"


# ------------------------------------------------------------------------------------------
# exact culling of obstacles whose hinge is provably zero
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("make", [lambda: scenes.scene_cfg2(0), lambda: scenes.scene_cfg2(5),
                                  lambda: scenes.scene_static(7, 64, K=2048, T=100),
                                  lambda: scenes.scene_cfg0(3), lambda: scenes.scene_cfg1(1),
                                  lambda: scenes.scene_cfg1(2), lambda: scenes.scene_cfg3(4),
                                  lambda: scenes.scene_static(11, 20, K=1000, T=37)],
                         ids=["cfg2a", "cfg2b", "static64", "cfg0", "cfg1a", "cfg1b", "cfg3", "static20"])
def test_culling_is_bit_exact(B, make):
    sc = make()
    p = sc.params.with_(K=min(sc.params.K, 4096), n_iter=2)
    a = gpu_solve(B, sc, p, 0)
    b = gpu_solve(B, sc, p, B.FLAG_NO_CULL)
    for key in ("S", "XT", "U"):
        assert np.array_equal(a[key], b[key]), key
    assert a["diag"] == b["diag"]


def test_culling_keeps_close_fast_obstacles(B, O):
    """Obstacles next to the vehicle, fast pedestrians, small alpha: nothing may be culled wrongly."""
    sc = scenes.scene_cfg2(6)
    obs = sc.obstacles.copy()
    obs[:4, 0:2] = sc.x0[:2] + np.array([[4.0, 3.0], [-6.0, 2.5], [9.0, -4.0], [-12.0, 5.0]])
    obs[4:, 3:5] *= 3.0                                     # 4.5 m/s pedestrians
    sc2 = scenes.Scene(sc.x0, sc.goal, obs.astype(np.float32).astype(np.float64), sc.params)
    p = sc.params.with_(K=2048, n_iter=1, alpha_lo=0.02, alpha_hi=0.3)
    a = gpu_solve(B, sc2, p, 0)
    b = gpu_solve(B, sc2, p, B.FLAG_NO_CULL)
    assert np.array_equal(a["S"], b["S"]) and np.array_equal(a["U"], b["U"])
    check_against_oracle(O, a, sc2, p)


# ------------------------------------------------------------------------------------------
# super-ellipse obstacles, eq. (16)
# ------------------------------------------------------------------------------------------
def gpu_solve_se(B, sc, p, se, flags=0, n0=0, U0=None, max_se=None):
    n_obs = len(sc.obstacles)
    s = B.Solver(p, 1, max(n_obs, 1), flags | B.FLAG_WRITE_SAMPLES, max_superellipses=max_se or max(len(se), 1))
    s.set_state(sc.x0); s.set_goal(sc.goal); s.set_obstacles(sc.obstacles); s.set_superellipses(se)
    s.set_nominal(U0)
    s.set_counter(n0)
    s.solve()
    out = dict(U=s.get_controls(), S=s.get_costs(), XT=s.get_final_states(), diag=s.get_diag())
    s.close()
    return out


def check_se(O, got, sc, p, se, n0=0, U0=None):
    U = np.zeros((p.T, 2)) if U0 is None else np.asarray(U0, dtype=np.float64)
    ref = O.solve(p, n0, sc.x0, sc.goal, sc.obstacles, U, n_threads=8, superellipses=se)[-1]
    okS = close(got["S"], ref["S"], 1.0)
    assert okS.all(), f"S_k: {np.count_nonzero(~okS)} of {p.K} off, worst {np.abs(got['S'] - ref['S']).max()}"
    assert close(got["XT"], ref["XT"], 1.0).all()
    floors = np.array([p.v_max, p.delta_max])
    err = np.abs(got["U"] - ref["U"]) / (RTOL * np.maximum(np.abs(ref["U"]), floors[None, :]))
    assert err.max() <= 1.0, f"U worst error = {err.max():.2f} x tolerance"
    if ref["gap"] > 1e-3 * max(1.0, abs(ref["S"].min())):
        assert got["diag"]["argmin"] == ref["argmin"]


@pytest.mark.parametrize("seed", [0, 1, 2])
@pytest.mark.parametrize("precise", [0, 2], ids=["fast", "precise"])
def test_superellipse_scene(B, O, seed, precise):
    sc = scenes.scene_cfg2_superellipse(seed)
    p = sc.params.with_(K=4096, n_iter=2)
    got = gpu_solve_se(B, sc, p, sc.superellipses, precise)
    check_se(O, got, sc, p, sc.superellipses)


@pytest.mark.parametrize("n_se", [1, 3, 4, 5, 16])
def test_superellipse_counts_and_discs_together(B, O, n_se):
    sc = scenes.scene_cfg2(3)                                   # 8 discs (3 moving) stay
    rng = np.random.default_rng(n_se)
    se = np.array([[sc.x0[0] + rng.uniform(-15, 15), sc.x0[1] + rng.uniform(-15, 15), rng.uniform(0.5, 2.5),
                    rng.uniform(0.4, 1.2), rng.uniform(-3, 3), rng.uniform(-1, 1), rng.uniform(-1, 1),
                    4.0 if i % 3 else 2.0] for i in range(n_se)], dtype=np.float32).astype(np.float64)
    p = sc.params.with_(K=1000, T=61, n_iter=1)
    got = gpu_solve_se(B, sc, p, se, max_se=16)
    check_se(O, got, sc, p, se)


def test_superellipse_e2_matches_disc_path(B):
    sc = scenes.scene_cfg2(2)
    p = sc.params.with_(K=2048, n_iter=1)
    a = gpu_solve(B, sc, p, 0)
    se = np.array([[o[0], o[1], o[2], o[2], 0.3 * i, o[3], o[4], 2.0] for i, o in enumerate(sc.obstacles)])
    sc2 = scenes.Scene(sc.x0, sc.goal, np.zeros((0, 5)), p)
    b = gpu_solve_se(B, sc2, p, se)
    assert np.allclose(a["S"], b["S"], rtol=1e-5, atol=1e-3)
    assert np.allclose(a["U"], b["U"], atol=1e-4) and a["diag"]["argmin"] == b["diag"]["argmin"]


def test_superellipse_closed_loop_and_errors(B, O):
    sc = scenes.scene_cfg2_superellipse(4)
    p = sc.params.with_(K=2048, T=60, n_iter=1)
    s = B.Solver(p, 1, 1, 0, max_superellipses=8)
    s.set_scene(sc)
    x, se, U = sc.x0.copy(), sc.superellipses.copy(), np.zeros((p.T, 2))
    floors = np.array([p.v_max, p.delta_max])
    for step in range(4):
        u0 = s.step()[0]
        ref = O.iteration(p, step, x, sc.goal, np.zeros((0, 5)), U, n_threads=8, superellipses=se)
        assert close(u0, ref["U"][0], floors).all()
        se_ref = O.advance_se(p, se)
        se_gpu = s.get_superellipses()
        assert np.abs(se_gpu - se_ref).max() <= 1e-5
        x, se, U = s.get_state().astype(np.float64), se_gpu.astype(np.float64), s.get_controls().astype(np.float64)
    with pytest.raises(B.BrmppiError) as e:
        s.set_superellipses(np.tile(sc.superellipses[0], (9, 1)))
    assert e.value.status == B.ERR_TOO_MANY_OBSTACLES
    bad = sc.superellipses[:1].copy(); bad[0, 7] = 3
    with pytest.raises(B.BrmppiError) as e:
        s.set_superellipses(bad)
    assert e.value.status == B.ERR_INVALID_ARG
    bad = sc.superellipses[:1].copy(); bad[0, 2] = 0.0
    with pytest.raises(B.BrmppiError) as e:
        s.set_superellipses(bad)
    assert e.value.status == B.ERR_INVALID_ARG
    s.close()
    with pytest.raises(B.BrmppiError):                          # default kernel only
        B.Solver(p, 1, 1, B.FLAG_KERNEL_THREAD_PER_SAMPLE, max_superellipses=4)


@pytest.mark.parametrize("kernel", KERNELS)
def test_velocity_dependent_hitch_limit(B, O, kernel):
    """hitch_kappa > 0 (eq. 18): start jackknifed so that the hinge is active for most samples."""
    sc = scenes.scene_cfg1(7)
    x0 = sc.x0.copy(); x0[3] = x0[2] - 1.0                     # hitch angle 1.0 rad
    sc2 = scenes.Scene(np.asarray(x0, dtype=np.float32).astype(np.float64), sc.goal, sc.obstacles, sc.params)
    p = sc.params.with_(K=1024, hitch_kappa=0.2, hitch_max=1.1)
    got = gpu_solve(B, sc2, p, kernel)
    check_against_oracle(O, got, sc2, p)
    base = gpu_solve(B, sc2, p.with_(hitch_kappa=0.0), kernel)
    assert (got["S"] >= base["S"] - 1e-3).all() and (got["S"] > base["S"] + 1e-2).any()


def test_set_inputs_equals_the_three_calls(B):
    """brmppi_set_inputs (one call, one copy in a single-scene context) leaves exactly what set_state + set_goal +
    set_obstacles leave: bit-identical solves, in a single-scene and in a two-scene context, repeated calls (the two
    staging buffers in turn), fewer obstacles than before, and the same argument errors with nothing changed."""
    sc = scenes.scene_cfg2(1)
    p = sc.params.with_(K=1500, T=40, n_iter=2)
    for n_scenes in (1, 2):
        a = B.Solver(p, n_scenes, 8, B.FLAG_WRITE_SAMPLES)
        b = B.Solver(p, n_scenes, 8, B.FLAG_WRITE_SAMPLES)
        for rep_, n_obs in enumerate((8, 8, 3, 0, 5)):
            x = sc.x0 + np.float32(0.1 * rep_)
            for i in range(n_scenes):
                a.set_state(x, i); a.set_goal(sc.goal, i); a.set_obstacles(sc.obstacles[:n_obs], i)
                b.set_inputs(x, sc.goal, sc.obstacles[:n_obs], i)
            a.set_nominal(None); b.set_nominal(None); a.set_counter(rep_); b.set_counter(rep_)
            a.solve(); b.solve()
            for i in range(n_scenes):
                assert np.array_equal(a.get_costs(i), b.get_costs(i)) and np.array_equal(a.get_controls(i), b.get_controls(i))
                assert np.array_equal(a.get_state(i), b.get_state(i)) and np.array_equal(a.get_obstacles(i), b.get_obstacles(i))
        before = b.get_state(0).copy()
        bad = sc.obstacles.copy(); bad[2, 2] = -1.0
        for args, status in (((sc.x0, sc.goal, bad), B.ERR_INVALID_ARG),
                             ((np.array([0, np.nan, 0, 0]), sc.goal, sc.obstacles), B.ERR_NONFINITE_INPUT),
                             ((sc.x0, sc.goal, np.zeros((9, 5)) + 1.0), B.ERR_TOO_MANY_OBSTACLES)):
            with pytest.raises(B.BrmppiError) as e:
                b.set_inputs(*args)
            assert e.value.status == status
        assert np.array_equal(b.get_state(0), before) and len(b.get_obstacles(0)) == 5
        a.close(); b.close()
    fresh = B.Solver(p, 1, 8, 0)
    fresh.set_inputs(sc.x0, sc.goal, sc.obstacles)      # marks state and goal as set
    fresh.solve()
    fresh.close()


def test_solve_get_controls_equals_solve_then_get_controls(B):
    """brmppi_solve_get_controls (the last update writes U into page-locked host memory too, no copy behind the
    solve) returns the bits that brmppi_solve + brmppi_get_controls return and leaves the same U on the device: one
    scene and three, repeated and mixed with plain solves, shifts and a step, and when an iteration leaves U as it
    was (every cost non-finite)."""
    sc = scenes.scene_cfg2(2)
    p = sc.params.with_(K=1200, T=37, n_iter=2)
    for n_scenes in (1, 3):
        a = B.Solver(p, n_scenes, 8, 0)
        b = B.Solver(p, n_scenes, 8, 0)
        for s in (a, b):
            for i in range(n_scenes):
                s.set_state(sc.x0 + np.float32(0.05 * i), i); s.set_goal(sc.goal, i); s.set_obstacles(sc.obstacles, i)
        for rep_ in range(4):
            a.solve()
            Ua = np.stack([a.get_controls(i) for i in range(n_scenes)])
            Ub = b.solve_get_controls()
            assert Ub.shape == (n_scenes, p.T, 2) and np.array_equal(Ua, Ub) and np.abs(Ub).max() > 0
            assert all(np.array_equal(b.get_controls(i), Ub[i]) for i in range(n_scenes))     # the device copy
            if rep_ == 1:
                a.shift(); b.shift()
            if rep_ == 2:
                assert np.array_equal(a.step(), b.step())
        a.close(); b.close()
    bad = sc.params.with_(K=256, T=20, n_iter=1, w_pos=3e38)      # every stage cost overflows fp32
    s = B.Solver(bad, 1, 8, 0)
    s.set_scene(sc)
    U0 = np.tile(np.array([[0.5, 0.1]], dtype=np.float32), (20, 1))
    s.set_nominal(U0)
    assert np.array_equal(s.solve_get_controls()[0], U0) and s.get_diag()["argmin"] == -1
    s.close()


def test_solve_host_equals_set_inputs_solve_get_controls(B):
    """brmppi_solve_host (inputs, solve and result in one call; one graph launch in a single-scene context) returns
    the bits of brmppi_set_inputs + brmppi_solve + brmppi_get_controls and leaves the same state, obstacles and U on
    the device: changing inputs and obstacle counts over repeated calls, mixed with set_inputs (the staging buffer it
    shares), in a two-scene context (the two calls underneath), and the same argument errors with nothing changed."""
    sc = scenes.scene_cfg2(3)
    p = sc.params.with_(K=1500, T=40, n_iter=2)
    for n_scenes in (1, 2):
        a = B.Solver(p, n_scenes, 8, B.FLAG_WRITE_SAMPLES)
        b = B.Solver(p, n_scenes, 8, B.FLAG_WRITE_SAMPLES)
        for s in (a, b):
            for i in range(n_scenes):
                s.set_inputs(sc.x0, sc.goal, sc.obstacles, i)
        for rep_, n_obs in enumerate((8, 8, 3, 0, 5, 8)):
            x = sc.x0 + np.float32(0.1 * rep_)
            g = sc.goal + np.float32(0.01 * rep_)
            a.set_inputs(x, g, sc.obstacles[:n_obs]); a.solve()
            Ua = np.stack([a.get_controls(i) for i in range(n_scenes)])
            Ub = b.solve_host(x, g, sc.obstacles[:n_obs])
            assert np.array_equal(Ua, Ub) and np.abs(Ub).max() > 0
            for i in range(n_scenes):
                assert np.array_equal(a.get_costs(i), b.get_costs(i)) and np.array_equal(a.get_controls(i), b.get_controls(i))
                assert np.array_equal(a.get_state(i), b.get_state(i)) and np.array_equal(a.get_obstacles(i), b.get_obstacles(i))
            if rep_ == 2:                                   # a plain set_inputs + solve in between
                a.set_inputs(sc.x0, sc.goal, sc.obstacles); b.set_inputs(sc.x0, sc.goal, sc.obstacles)
                a.solve(); b.solve()
        before, U_before = b.get_state(0).copy(), b.get_controls(0).copy()
        bad = sc.obstacles.copy(); bad[2, 2] = -1.0
        for args, status in (((sc.x0, sc.goal, bad), B.ERR_INVALID_ARG),
                             ((np.array([0, np.nan, 0, 0]), sc.goal, sc.obstacles), B.ERR_NONFINITE_INPUT),
                             ((sc.x0, sc.goal, np.zeros((9, 5)) + 1.0), B.ERR_TOO_MANY_OBSTACLES)):
            with pytest.raises(B.BrmppiError) as e:
                b.solve_host(*args)
            assert e.value.status == status
        assert np.array_equal(b.get_state(0), before) and np.array_equal(b.get_controls(0), U_before)
        a.close(); b.close()
    fresh = B.Solver(p, 1, 8, 0)
    assert np.abs(fresh.solve_host(sc.x0, sc.goal, sc.obstacles)).max() > 0      # marks state and goal as set
    fresh.close()


def test_random_configurations(B, O):
    """A seeded sweep over sizes the named cases do not visit: K from 1 to 20 000 (tiles of every width, ragged last
    tiles), T from 1 to 150 (one chunk to many, odd and even), 0 to 64 obstacles with and without motion (one to eight
    groups, table padding), one to three scenes, one to four discs, hitch offset, warm and zero nominal, a random
    iteration counter.  Per configuration: the culled launch equals the un-culled one bit for bit, and both kernels
    meet the flat tolerances on x_T and S_k against the oracle.  alpha_lo >= 0.05 and lambda >= 10 as in every recipe
    (DESIGN.md 2 says what happens below that)."""
    rng = np.random.default_rng(20250811)
    disc_sets = [((0, 2.0),), ((0, 2.0), (1, -3.0)), ((0, 2.0), (1, -2.0), (1, -6.0)), ((0, 0.0), (0, 2.5), (1, -2.0), (1, -4.5))]
    n_done = 0
    while n_done < 200:
        K = int(rng.choice([1, 7, 31, 33, 100, 333, 1000, 2049, 4097, 9000, 20000]))
        T = int(rng.choice([1, 2, 3, 5, 6, 7, 11, 12, 13, 24, 25, 40, 81, 150]))
        n_obs = int(rng.choice([0, 1, 2, 3, 5, 8, 9, 16, 17, 31, 32, 33, 64]))
        if K * T * max(n_obs, 1) > 2_000_000:
            continue
        ns = int(rng.choice([1, 1, 2, 3]))
        scs = []
        for _ in range(ns):
            sc = scenes.scene_static(int(rng.integers(0, 1000)), n_obs, K=K, T=T)
            if n_obs and rng.random() < 0.6:
                ob = sc.obstacles.copy()
                m = rng.random(n_obs) < 0.5
                ob[m, 3:] = rng.uniform(-2, 2, (int(m.sum()), 2))
                sc.obstacles = ob.astype(np.float32).astype(np.float64)
            scs.append(sc)
        p = scs[0].params.with_(discs=disc_sets[int(rng.integers(0, 4))], Lh=float(rng.choice([0.0, 0.6])),
                                alpha_lo=float(rng.choice([0.05, 0.1, 0.3])), lam=float(rng.choice([10.0, 100.0])),
                                seed=int(rng.integers(0, 2**40)))
        cap = max(n_obs, 1) if rng.random() < 0.5 else 64
        n0 = int(rng.integers(0, 100))
        U0 = None if rng.random() < 0.5 else np.tile(np.array([[0.5, 0.05]], dtype=np.float32), (T, 1))
        outs = {}
        for name, fl in (("cta", 0), ("nocull", B.FLAG_NO_CULL), ("thread", B.FLAG_KERNEL_THREAD_PER_SAMPLE)):
            s = B.Solver(p, ns, cap, fl | B.FLAG_WRITE_SAMPLES)
            for i, sc in enumerate(scs):
                s.set_scene(sc, i)
                s.set_nominal(U0, i)
            s.set_counter(n0)
            s.solve()
            outs[name] = [(s.get_costs(i), s.get_final_states(i), s.get_controls(i)) for i in range(ns)]
            s.close()
        what = f"K={K} T={T} n_obs={n_obs} scenes={ns} discs={len(p.discs)} cap={cap}"
        for i in range(ns):
            a, b, c = outs["cta"][i], outs["nocull"][i], outs["thread"][i]
            assert all(np.array_equal(x, y) for x, y in zip(a, b)), "culled != un-culled: " + what
            U = np.zeros((T, 2)) if U0 is None else U0.astype(np.float64)
            ref = O.solve(p.with_(seed=p.seed + i), n0, scs[i].x0, scs[i].goal, scs[i].obstacles, U, n_threads=8)[-1]
            for name, g in (("tile", a), ("thread", c)):
                assert close(g[0], ref["S"], 1.0).all(), f"{name} S_k: " + what
                assert close(g[1], ref["XT"], 1.0).all(), f"{name} x_T: " + what
        n_done += 1


def test_random_configurations_with_superellipses(B, O):
    """The seeded sweep with eq. (16)'s obstacles: 1 to 16 super-ellipses (e = 2 and 4, oriented, some moving) beside
    0 to 16 discs, K 1 to 9000, T 1 to 81, one to four vehicle discs, with and without unused capacity; S_k and x_T
    at the flat tolerances against the oracle."""
    rng = np.random.default_rng(20250814)
    disc_sets = [((0, 2.0),), ((0, 2.0), (1, -3.0)), ((0, 2.0), (1, -2.0), (1, -6.0)), ((0, 0.0), (0, 2.5), (1, -2.0), (1, -4.5))]
    n_done = 0
    while n_done < 80:
        K = int(rng.choice([1, 7, 31, 33, 100, 333, 1000, 2049, 9000]))
        T = int(rng.choice([1, 2, 3, 5, 6, 7, 11, 12, 13, 24, 25, 40, 81]))
        n_obs = int(rng.choice([0, 0, 1, 3, 8, 9, 16]))
        n_se = int(rng.choice([1, 2, 3, 4, 5, 8, 9, 16]))
        if K * T * (n_obs + 3 * n_se) > 4_000_000:
            continue
        sc = scenes.scene_static(int(rng.integers(0, 1000)), n_obs, K=K, T=T)
        se = np.array([[sc.x0[0] + rng.uniform(-15, 15), sc.x0[1] + rng.uniform(-15, 15), rng.uniform(0.5, 2.5),
                        rng.uniform(0.4, 1.2), rng.uniform(-3, 3), rng.uniform(-1, 1) * (i % 2), rng.uniform(-1, 1) * (i % 2),
                        4.0 if i % 3 else 2.0] for i in range(n_se)], dtype=np.float32).astype(np.float64)
        p = sc.params.with_(discs=disc_sets[int(rng.integers(0, 4))], Lh=float(rng.choice([0.0, 0.6])),
                            alpha_lo=float(rng.choice([0.05, 0.1, 0.3])), lam=float(rng.choice([10.0, 100.0])),
                            seed=int(rng.integers(0, 2**40)))
        n0 = int(rng.integers(0, 100))
        U0 = None if rng.random() < 0.5 else np.tile(np.array([[0.5, 0.05]], dtype=np.float32), (T, 1))
        got = gpu_solve_se(B, sc, p, se, n0=n0, U0=U0, max_se=n_se if rng.random() < 0.5 else 16)
        U = np.zeros((T, 2)) if U0 is None else U0.astype(np.float64)
        ref = O.solve(p, n0, sc.x0, sc.goal, sc.obstacles, U, n_threads=8, superellipses=se)[-1]
        what = f"K={K} T={T} n_obs={n_obs} n_se={n_se} discs={len(p.discs)}"
        assert close(got["S"], ref["S"], 1.0).all(), "S_k: " + what
        assert close(got["XT"], ref["XT"], 1.0).all(), "x_T: " + what
        n_done += 1
