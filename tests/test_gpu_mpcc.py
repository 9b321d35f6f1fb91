"""Parity of the paper's own model and cost on the GPU (BRMPPI_FLAG_MPCC: 7-state model eq. (6), predictor (17),
contouring cost (13)-(15); reading 31) through the C ABI against the oracle's
orc7_* on the same seeded inputs.

Tolerances:
  x_T  the north star's 1e-4 relative, floor 1.0 on every component (v, a, delta, psi are held to 1e-4 absolute);
  S_k  1e-4 max(|S_k|, 1), and for a sample that misses it, that plus w_bar * EPS_G * N_k.  On this path S_k is
       tens, not the 1e4 of the goal-seeking penalty path, while each hinge term still enters with w_bar = 1e3: an
       fp32 hinge argument carries about EPS_G = 2e-6 of absolute error (position error <= 3e-6 m -- MUFU sin/cos
       at 3.6e-7 absolute on a 6 m lever, T roundings at ulp(8 m) -- times |dh/dp| = 2 |d| / rho^2 ~ 1 / m at an
       obstacle's boundary, times alpha), so N_k active terms may move S_k by w_bar EPS_G N_k.  N_k = the hinge
       arguments above -EPS_G on the ORACLE's trajectory of that sample; at most 20 % of the samples may need it;
  U    1e-4 of the control bound plus the S_k tolerances carried through the update (5) to first order,
       sum_k w_k |u_kt - U_t| tau_k / lambda, with the oracle's weights and samples: with lambda = 1 and an effective
       sample size of tens (the penalty path's is ~1) a cost error the north star itself allows moves the weights."""

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


@pytest.fixture(params=[0, 4], ids=["cta", "thread"])
def kern(request):
    """Both rollout kernels of the mode: the phase-split CTA kernel (default) and BRMPPI_FLAG_KERNEL_THREAD_PER_SAMPLE."""
    return request.param


def close(a, b, floor):
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    return np.abs(a - b) <= RTOL * np.maximum(np.abs(b), floor)


def path_scene(seed, n_obs, K, T, near=True, v0=2.0, **kw):
    """scenes.scene_mpcc, driving at v0, with the obstacles pulled next to the stretch of the reference path the
    horizon covers, where the predictor's hinge works."""
    sc = scenes.scene_mpcc(seed, K=K, T=T, dt=0.05, n_obs=max(n_obs, 1), M=16)
    sc.x0[2] = v0
    p = sc.params.with_(K=K, T=T, n_iter=1, **kw)
    obs = sc.obstacles[:n_obs].copy()
    if near and n_obs:
        rng = np.random.default_rng(300 + seed)
        L = sc.coef.shape[0] * sc.dpsi
        for i in range(n_obs):
            s = rng.uniform(2.0, 7.0)
            m = min(int(s / sc.dpsi), sc.coef.shape[0] - 1)
            ds = s - m * sc.dpsi
            q = sc.coef[m, :2, :] @ np.array([1.0, ds, ds * ds, ds ** 3])
            tx, ty = sc.coef[m, :2, :] @ np.array([0.0, 1.0, 2.0 * ds, 3.0 * ds * ds])      # the path's tangent there
            side = np.array([-ty, tx]) / np.hypot(tx, ty) * rng.choice([-1, 1])
            obs[i, :2] = q + side * (obs[i, 2] + p.disc_radius + rng.uniform(-0.3, 0.6))
        # the start pose stays outside every inflated obstacle
        centres = scenes.parking.vehicle_disc_centres(np.array([sc.x0[0], sc.x0[1], sc.x0[4]]), p.discs)
        for i in range(n_obs):
            for _ in range(30):
                if np.hypot(*(centres - obs[i, :2]).T).min() >= 1.15 * (obs[i, 2] + p.disc_radius):
                    break
                obs[i, :2] += 0.7 * (obs[i, :2] - sc.x0[:2]) / max(np.hypot(*(obs[i, :2] - sc.x0[:2])), 1e-3)
    obs = obs.astype(np.float32).astype(np.float64).reshape(-1, 5)
    return scenes.PathScene(sc.x0, sc.psi0, obs, sc.coef, sc.dpsi, p, sc.name)


def gpu_mpcc(B, sc, p, flags=0, n0=0, U0=None, max_obstacles=None):
    mo = max(len(sc.obstacles), 1) if max_obstacles is None else max_obstacles
    s = B.Solver(p, 1, mo, flags | B.FLAG_MPCC | B.FLAG_WRITE_SAMPLES, max_path_segments=sc.coef.shape[0])
    s.set_scene(sc)
    s.set_nominal(U0)
    s.set_counter(n0)
    s.solve()
    out = dict(U=s.get_controls(), S=s.get_costs(), XT=s.get_final_states7(), diag=s.get_diag())
    s.close()
    return out


EPS_G = 2e-6      # error bound of one hinge argument (module docstring)


def active_terms(O, sc, p, n, k, U):
    """Number of hinge arguments (1 - alpha) h - hhat above -EPS_G on the oracle's own trajectory of sample k."""
    r = O.sample7(p, sc.coef, sc.dpsi, n, k, sc.x0, sc.psi0, sc.obstacles, U)
    alpha = O.alpha(p, n, k)
    traj = O.rollout7(p, sc.coef, sc.dpsi, sc.x0, sc.psi0, sc.obstacles, r["u"], alpha)["traj"]
    count = 0
    for t in range(p.T):
        for ob in sc.obstacles:
            for j in range(len(p.discs)):
                hh, h = O.hhat7(p, traj[t, :7], r["u"][t], ob, t, j)
                count += (1.0 - alpha) * h - hh > -EPS_G
    return count


def check(O, got, sc, p, n0=0, U0=None):
    U = np.zeros((p.T, 2)) if U0 is None else np.asarray(U0, dtype=np.float64)
    scale = 1.0
    for it in range(p.n_iter):      # later iterations start from a nominal that already differs by rounding
        ref = O.iteration7(p, sc.coef, sc.dpsi, n0 + it, sc.x0, sc.psi0, sc.obstacles, U, n_threads=8, want_samples=True)
        U_in, U = U, ref["U"].copy()
        scale = 1.0 if it == 0 else 4.0
    okX = close(got["XT"], ref["XT"], scale)
    assert okX.all(), f"x_T: {np.argwhere(~okX)[:5]}, worst {np.abs(got['XT'] - ref['XT']).max(axis=0)}"
    # S_k: the flat tolerance, widened for the samples that miss it by what their active hinge terms allow
    tau = scale * RTOL * np.maximum(np.abs(ref["S"]), 1.0)
    dS = np.abs(got["S"] - ref["S"])
    off = np.flatnonzero(dS > tau)
    assert len(off) <= 0.2 * p.K
    for k in off:
        tau[k] += scale * p.w_bar * EPS_G * active_terms(O, sc, p, n0 + p.n_iter - 1, int(k), U_in)
        assert dS[k] <= tau[k], (k, ref["S"][k], dS[k], tau[k])
    # U: 1e-4 of the control bound plus the S tolerances carried through (5): dU_t = sum_k w_k (u_kt - U_t)(-dS_k / lambda)
    wn = ref["w"] / ref["w"].sum()
    spread = np.abs(ref["u"] - ref["U"][None, :, :])
    floors = np.array([p.j_max, p.omega_max])
    bound = scale * RTOL * np.maximum(np.abs(ref["U"]), floors[None, :]) + np.einsum("k,ktc->tc", wn * tau / p.lam, spread)
    err = np.abs(got["U"] - ref["U"]) / bound
    assert err.max() <= 1.0, f"U worst error = {err.max():.2f} x bound"
    d = got["diag"]
    assert d["nonfinite"] == ref["nonfinite"]
    kmin = int(np.argmin(ref["S"]))
    assert abs(d["S_min"] - ref["S"].min()) <= tau[kmin] + 1e-6
    if ref["gap"] > 2.0 * tau[kmin]:
        assert d["argmin"] == ref["argmin"]
    assert abs(d["eta"] - ref["eta"]) <= (2.0 * (wn * tau).sum() / p.lam + 1e-3) * ref["eta"]
    ref["flat_ok"] = p.K - len(off)
    ref["U_err_flat"] = float((np.abs(got["U"] - ref["U"]) / (RTOL * np.maximum(np.abs(ref["U"]), floors[None, :]))).max())
    return ref


@pytest.mark.parametrize("n_obs", [0, 1, 3, 8])
@pytest.mark.parametrize("precise", [0, 2], ids=["fast", "precise"])
def test_mpcc_iteration_matches_oracle(B, O, n_obs, precise, kern):
    sc = path_scene(n_obs, n_obs, K=1000, T=40)
    ref = check(O, gpu_mpcc(B, sc, sc.params, precise | kern), sc, sc.params)
    if n_obs >= 3:      # the scene is one where the predictor's hinge is at work, not a free run
        free = O.solve7(sc.params, sc.coef, sc.dpsi, 0, sc.x0, sc.psi0, np.zeros((0, 5)), np.zeros((40, 2)), n_threads=8)[-1]
        assert (ref["S"] > free["S"] + 1e-3).mean() > 0.05
    else:               # nothing to amplify: the flat north-star tolerance holds for every sample and for U
        assert ref["flat_ok"] == sc.params.K and ref["U_err_flat"] <= 1.0


def test_ragged_sizes_and_unused_capacity(B, O, kern):
    """K not a multiple of the block, odd T (the Philox pair of the last step is half used), obstacle and path
    capacity larger than what is set."""
    sc = path_scene(4, 3, K=333, T=27)
    check(O, gpu_mpcc(B, sc, sc.params, kern, max_obstacles=8), sc, sc.params)
    s = B.Solver(sc.params, 1, 8, kern | B.FLAG_MPCC | B.FLAG_WRITE_SAMPLES, max_path_segments=64)
    s.set_scene(sc)
    s.solve()
    got = dict(U=s.get_controls(), S=s.get_costs(), XT=s.get_final_states7(), diag=s.get_diag())
    s.close()
    check(O, got, sc, sc.params)
    one = path_scene(5, 2, K=1, T=5)
    check(O, gpu_mpcc(B, one, one.params, kern), one, one.params)


def test_long_horizon_without_control_planes(B, O):
    """K = 19000, T = 130: full 128-sample tiles whose sampled controls no longer fit in shared memory beside the state
    ring -- the CTA kernel's chain then draws them as it goes and the epilogue regenerates them."""
    sc = path_scene(13, 2, K=19000, T=130, v0=0.5)
    check(O, gpu_mpcc(B, sc, sc.params), sc, sc.params)


@pytest.mark.parametrize("case", ["recipe", "near", "alpha_from_zero", "fast_far_obstacles"])
def test_culling_is_bit_exact(B, case):
    """The phase-split kernel skips obstacles that provably add nothing (mpcc_hinge): S_k, x_T and U must be
    bit-identical to the same launch with every (obstacle, disc, step) evaluated (BRMPPI_FLAG_NO_CULL)."""
    if case == "recipe":
        sc = scenes.scene_mpcc(2, K=3000, T=80, dt=0.05, n_obs=8, M=16)
        sc = scenes.PathScene(sc.x0, sc.psi0, sc.obstacles, sc.coef, sc.dpsi, sc.params.with_(n_iter=1), sc.name)
    elif case == "near":
        sc = path_scene(8, 8, K=3000, T=40)
    elif case == "alpha_from_zero":
        sc = path_scene(3, 6, K=3000, T=40, alpha_lo=0.0, alpha_hi=0.05)
    else:       # far obstacles that close in fast: 2 |Ts o'| / alpha must keep them in
        sc = path_scene(8, 8, K=3000, T=60)
        sc.obstacles[:, :2] += np.float32(25.0)
        sc.obstacles[:, 3:] = np.float32(-9.0)
    a = gpu_mpcc(B, sc, sc.params)
    b = gpu_mpcc(B, sc, sc.params, B.FLAG_NO_CULL)
    assert np.array_equal(a["S"], b["S"]) and np.array_equal(a["XT"], b["XT"]) and np.array_equal(a["U"], b["U"])
    assert a["diag"]["argmin"] == b["diag"]["argmin"]
    if case != "recipe":      # the case is not vacuous: some hinge is active somewhere
        free = scenes.PathScene(sc.x0, sc.psi0, np.zeros((0, 5)), sc.coef, sc.dpsi, sc.params, sc.name)
        assert (a["S"] > gpu_mpcc(B, free, sc.params)["S"] + 1e-3).any()


def test_warm_nominal_moving_obstacles_off_axle_hitch_four_discs(B, O, kern):
    discs = ((0, 0.0), (0, 2.5), (1, -2.0), (1, -4.5))
    sc = path_scene(6, 6, K=800, T=50, Lh=0.75, discs=discs, nu_bar=2.5, hitch_kappa=0.05, alpha_lo=0.0, alpha_hi=1.0)
    sc.obstacles[:, 3:] = np.random.default_rng(1).uniform(-1.2, 1.2, (6, 2)).astype(np.float32)
    x0 = sc.x0.copy()
    x0[2], x0[3], x0[6] = 1.5, 0.5, 0.1          # moving, accelerating, steering
    x0[5] += 0.3                                  # trailer not aligned
    sc = scenes.PathScene(x0.astype(np.float32).astype(np.float64), 0.75, sc.obstacles, sc.coef, sc.dpsi, sc.params)
    U0 = np.tile([0.5, -0.2], (50, 1)).astype(np.float32)
    check(O, gpu_mpcc(B, sc, sc.params, kern, n0=7, U0=U0), sc, sc.params, n0=7, U0=U0)
    p3 = sc.params.with_(n_iter=3)
    check(O, gpu_mpcc(B, sc, p3, kern, n0=2), sc, p3, n0=2)


def test_path_end_clamp_and_reverse(B, O, kern):
    """psi pinned at both ends of the path: a start at the path's end driving forward (psi stays at M dpsi), and a
    start at psi = 0 reversing (psi stays at 0); the steering state saturates under a hard-over nominal."""
    sc = path_scene(7, 2, K=400, T=40)
    L = sc.coef.shape[0] * sc.dpsi
    r_end = O.path_eval(sc.params, sc.coef, sc.dpsi, L)
    x_end = np.array([r_end[0], r_end[1], 2.0, 0.0, r_end[2], r_end[3], 0.0]).astype(np.float32).astype(np.float64)
    a = scenes.PathScene(x_end, float(np.float32(L)), sc.obstacles, sc.coef, sc.dpsi, sc.params)
    ra = check(O, gpu_mpcc(B, a, a.params, kern), a, a.params)
    assert (ra["XT"][:, 7] >= L - 1e-9).mean() > 0.9
    x_rev = sc.x0.copy(); x_rev[2] = -1.5
    b = scenes.PathScene(x_rev, 0.0, sc.obstacles, sc.coef, sc.dpsi, sc.params)
    rb = check(O, gpu_mpcc(B, b, b.params, kern), b, b.params)
    assert (rb["XT"][:, 7] == 0.0).mean() > 0.9
    U0 = np.tile([0.0, 0.9], (40, 1)).astype(np.float32)
    rc = check(O, gpu_mpcc(B, sc, sc.params, kern, U0=U0), sc, sc.params, U0=U0)
    assert (rc["XT"][:, 6] == sc.params.delta_max).mean() > 0.3


def test_batch_of_scenes_with_their_own_paths(B, O, kern):
    scs = [path_scene(10 + s, 2 + s, K=500, T=30) for s in range(3)]
    p = scs[0].params
    s = B.Solver(p, 3, 8, kern | B.FLAG_MPCC | B.FLAG_WRITE_SAMPLES, max_path_segments=16)
    for i, sc in enumerate(scs):
        s.set_scene(sc, i)
    s.solve()
    for i, sc in enumerate(scs):
        got = dict(U=s.get_controls(i), S=s.get_costs(i), XT=s.get_final_states7(i), diag=s.get_diag(i))
        check(O, got, sc, p.with_(seed=p.seed + i))
    s.close()


def test_k_offset_draws_the_global_samples(B, O, kern):
    """A context with k_offset = 384 computes samples 384..639 of the 640-sample solve: bit-identical S_k and x_T
    to the same samples of an unsharded context (same arithmetic, same draws), the oracle's argmin index."""
    sc = path_scene(3, 3, K=256, T=20)
    full = sc.params.with_(K=640)
    whole = gpu_mpcc(B, sc, full, kern, n0=4)
    ref = check(O, whole, sc, full, n0=4)
    s = B.Solver(sc.params, 1, 3, kern | B.FLAG_MPCC | B.FLAG_WRITE_SAMPLES, k_offset=384, max_path_segments=16)
    s.set_scene(sc)
    s.set_counter(4)
    s.solve()
    assert np.array_equal(s.get_costs(), whole["S"][384:])
    assert np.array_equal(s.get_final_states7(), whole["XT"][384:])
    part = ref["S"][384:]
    if np.partition(part, 1)[1] - part.min() > 0.05:
        assert s.get_diag()["argmin"] == 384 + int(np.argmin(part))
    s.close()


def test_step_applies_the_plant_of_eq6_and_shifts(B, O, kern):
    sc = path_scene(9, 3, K=512, T=30)
    sc.obstacles[:, 3:] = np.float32(0.5)
    p = sc.params
    s = B.Solver(p, 1, 3, kern | B.FLAG_MPCC, max_path_segments=16)
    s.set_scene(sc)
    x, psi, obs = sc.x0.copy(), sc.psi0, sc.obstacles.copy()
    for it in range(3):
        u0 = s.step()[0]
        xn = O.step7(p, sc.coef, sc.dpsi, x, u0.astype(np.float64))
        psin = min(max(psi + p.dt * O.progress7(p, sc.coef, sc.dpsi, x, psi), 0.0), sc.coef.shape[0] * sc.dpsi)
        got = s.get_state7()
        assert np.allclose(got[:7], xn, rtol=0, atol=2e-6 * max(1.0, np.abs(xn).max()))
        assert abs(got[7] - psin) <= 2e-6 * max(1.0, psin)
        obs[:, :2] += p.dt * obs[:, 3:]
        assert np.allclose(s.get_obstacles(), obs, atol=1e-5)
        x, psi = got[:7].astype(np.float64), float(got[7])
        assert s.get_diag()["n"] == it + 1
    # the shifted nominal is the solve's U moved by one step, last element kept: solve once more without a plant
    U = s.get_controls()
    s.shift()
    U2 = s.get_controls()
    assert np.array_equal(U2[:-1], U[1:]) and np.array_equal(U2[-1], U[-1])
    s.close()


def test_closed_loop_follows_the_path(B):
    """Property at run length: thirty control steps from rest on the path keep the contouring error small and the
    path parameter increasing (no oracle involved: it checks the loop the library closes, not parity)."""
    sc = path_scene(11, 0, K=4096, T=40, near=False, v0=0.5)
    s = B.Solver(sc.params, 1, 1, B.FLAG_MPCC, max_path_segments=16)
    s.set_scene(sc)
    psis = []
    for _ in range(30):
        s.step()
        psis.append(float(s.get_state7()[7]))
    assert psis[-1] > psis[0] + 0.5 and all(b >= a - 1e-6 for a, b in zip(psis, psis[1:]))
    x = s.get_state7()
    m = min(int(x[7] / sc.dpsi), sc.coef.shape[0] - 1)
    ds = x[7] - m * sc.dpsi
    r = sc.coef[m] @ np.array([1.0, ds, ds * ds, ds ** 3])
    assert np.hypot(x[0] - r[0], x[1] - r[1]) < 1.0
    s.close()


def test_argument_checks(B):
    sc = path_scene(12, 1, K=64, T=10)
    s = B.Solver(sc.params, 1, 1, B.FLAG_MPCC, max_path_segments=16)
    with pytest.raises(B.BrmppiError) as e:
        s.set_state7(sc.x0, 0.0)                         # no path yet
    assert e.value.status == B.ERR_NOT_READY
    with pytest.raises(B.BrmppiError) as e:
        s.solve()
    assert e.value.status == B.ERR_NOT_READY
    with pytest.raises(B.BrmppiError) as e:
        s.set_reference_path(np.zeros((17, 4, 4)), 1.0)  # over capacity
    assert e.value.status == B.ERR_INVALID_ARG
    with pytest.raises(B.BrmppiError):
        s.set_reference_path(sc.coef, 0.0)
    bad = sc.coef.copy(); bad[3, 1, 2] = np.nan
    with pytest.raises(B.BrmppiError) as e:
        s.set_reference_path(bad, sc.dpsi)
    assert e.value.status == B.ERR_NONFINITE_INPUT
    s.set_reference_path(sc.coef, sc.dpsi)
    L = sc.coef.shape[0] * sc.dpsi
    for psi in (-0.1, L + 0.5):
        with pytest.raises(B.BrmppiError) as e:
            s.set_state7(sc.x0, psi)
        assert e.value.status == B.ERR_INVALID_ARG
    xs = sc.x0.copy(); xs[6] = 1.0                       # steering state outside its stops
    with pytest.raises(B.BrmppiError):
        s.set_state7(xs, 0.0)
    with pytest.raises(B.BrmppiError):
        s.set_state(np.zeros(4))                         # the 4-state calls belong to the other paths
    with pytest.raises(B.BrmppiError):
        s.set_goal(np.zeros(4))
    with pytest.raises(B.BrmppiError):
        s.set_nominal(np.tile([2.5, 0.0], (10, 1)))      # jerk outside its box
    s.set_state7(sc.x0, 0.0)
    s.set_reference_path(sc.coef, sc.dpsi)               # a new path: psi must be given again
    with pytest.raises(B.BrmppiError) as e:
        s.solve()
    assert e.value.status == B.ERR_NOT_READY
    s.close()
    for kw in (dict(flags=B.FLAG_MPCC | B.FLAG_PROJECTED), dict(flags=B.FLAG_MPCC, max_superellipses=2),
               dict(flags=B.FLAG_MPCC, max_path_segments=0), dict(flags=B.FLAG_MPCC, max_path_segments=257)):
        with pytest.raises(B.BrmppiError):
            B.Solver(sc.params, 1, 1, **kw)
    with pytest.raises(B.BrmppiError):
        B.Solver(sc.params.with_(hitch_filter=1), 1, 1, B.FLAG_MPCC)
    s = B.Solver(sc.params, 1, 1, 0)
    with pytest.raises(B.BrmppiError):
        s.set_state7(sc.x0, 0.0)                         # not an MPCC context
    s.close()


def test_full_size_against_the_oracle(B, O, kern):
    """CFG2's size in the launch configuration bench.py times (K = 16384, T = 80, 8 obstacles, the recipe's scene):
    every S_k and x_T and the update against the oracle's iteration."""
    sc = scenes.scene_mpcc(0, K=16384, T=80, dt=0.05, n_obs=8, M=24)
    p = sc.params.with_(n_iter=1)
    s = B.Solver(p, 1, 8, kern | B.FLAG_MPCC | B.FLAG_WRITE_SAMPLES, max_path_segments=24)
    s.set_scene(sc)
    s.solve()
    got = dict(U=s.get_controls(), S=s.get_costs(), XT=s.get_final_states7(), diag=s.get_diag())
    s.close()
    check(O, got, sc, p)


def test_random_configurations(B, O):
    """A seeded sweep over sizes the named cases do not visit (K 1 to 1000: tiles of every width; T 1 to 81: one chunk
    to several, with and without control planes; 0 to 8 obstacles, some moving; one to four discs; hitch offset; two
    ranges of alpha; a random iteration counter).  Per configuration: culled == un-culled bit for bit on the CTA
    kernel, and both kernels against the oracle by the module's rule."""
    rng = np.random.default_rng(20250812)
    disc_sets = [((0, 2.0),), ((0, 2.0), (1, -3.0)), ((0, 2.0), (1, -2.0), (1, -6.0)), ((0, 0.0), (0, 2.5), (1, -2.0), (1, -4.5))]
    for _ in range(150):
        K = int(rng.choice([1, 7, 31, 33, 100, 333, 1000]))
        T = int(rng.choice([1, 2, 3, 5, 6, 7, 11, 12, 13, 24, 25, 40, 81]))
        n_obs = int(rng.integers(0, 9))
        sc = path_scene(int(rng.integers(0, 50)), n_obs, K=K, T=T, discs=disc_sets[int(rng.integers(0, 4))],
                        Lh=float(rng.choice([0.0, 0.5])), alpha_lo=float(rng.choice([0.1, 0.3])))
        sc.params = sc.params.with_(seed=int(rng.integers(0, 2**40)))
        if n_obs and rng.random() < 0.5:
            m = rng.random(n_obs) < 0.5
            sc.obstacles[m, 3:] = rng.uniform(-1.5, 1.5, (int(m.sum()), 2)).astype(np.float32)
        n0 = int(rng.integers(0, 100))
        what = f"K={K} T={T} n_obs={n_obs} discs={len(sc.params.discs)}"
        a = gpu_mpcc(B, sc, sc.params, 0, n0=n0, max_obstacles=8)
        b = gpu_mpcc(B, sc, sc.params, B.FLAG_NO_CULL, n0=n0, max_obstacles=8)
        c = gpu_mpcc(B, sc, sc.params, B.FLAG_KERNEL_THREAD_PER_SAMPLE, n0=n0, max_obstacles=8)
        assert all(np.array_equal(a[q], b[q]) for q in ("U", "S", "XT")), "culled != un-culled: " + what
        for got in (a, c):
            check(O, got, sc, sc.params, n0=n0)
