"""Parity of the projected rollout (BRMPPI_FLAG_PROJECTED: BR-MPPI proper, Sec. V-A) through the
C ABI against the oracle's orc_*_projected on the same seeded inputs.

Tolerance: the north star's 1e-4 relative with the floors of tests/test_gpu_parity.py for x_T, S_k and U.

One class of samples is ill-conditioned in the METHOD, not in the kernel, and is excluded by a rule the oracle
evaluates on its own trajectory: the equality (9) makes h_i evolve multiplicatively, h_{t+1} ~ (1 - alpha_i -
u^alpha_i) h_t, so a rollout that reaches an obstacle's boundary sits at h ~ 0 and leaves it again (alpha_i < 0)
by exponential growth FROM that tiny value -- where it ends depends on h at the 1e-8 level.  h = d^2/rho^2 - 1 is
a difference of O(1) numbers: fp32 resolves it to 1.2e-7.  A sample is "pinned" if |h_i(x_t)| < 1e-5 for some
(i, t) of its fp64 trajectory (fp32 then carries more than 1 % relative error in that h).  Only pinned samples
may miss the tolerance, at most 2 % of the samples may be pinned-and-off, and when any sample is off the
update U (a weighted mean over all samples) is compared at the weight those samples carry.

The second such class is a step in the COST: the alpha term of reading 30 counts alpha_i^2 only while
h_i(x_{t+1}) < h_buffer, so a state whose h lies within fp32 resolution of h_buffer (|h - h_buffer| < 1e-5 on the
oracle's trajectory) is on one side in fp64 and may be on the other in fp32, and S_k moves by w_alpha alpha_i^2 with
x_T unchanged (found by a randomised sweep: K = 2500, T = 3, h = 0.5000001 against h_buffer = 0.5).  Such a sample
is treated like a pinned one."""
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


def near_scene(seed, n_obs, K, T, **kw):
    """CFG2-shaped scene whose obstacles sit where the projection has work to do."""
    sc = scenes.scene_cfg2(seed)
    rng = np.random.default_rng(100 + seed)
    obs = sc.obstacles[:n_obs].copy()
    obs[:, :2] = sc.x0[:2] + rng.uniform(-10, 10, (n_obs, 2))
    p = sc.params.with_(K=K, T=T, n_iter=1, **kw)
    # the start pose stays outside every inflated obstacle (h >= 0.2 for every disc): push offenders away
    centres = scenes.parking.vehicle_disc_centres(sc.x0[:3], p.discs)
    for i in range(n_obs):
        for _ in range(20):
            d = np.hypot(*(centres - obs[i, :2]).T).min()
            if d >= 1.1 * (obs[i, 2] + p.disc_radius):
                break
            obs[i, :2] += 1.5 * (obs[i, :2] - sc.x0[:2]) / max(np.hypot(*(obs[i, :2] - sc.x0[:2])), 1e-3)
    obs = obs.astype(np.float32).astype(np.float64)
    return scenes.Scene(sc.x0, sc.goal, obs, p)


def gpu_projected(B, sc, p, flags=0, n0=0, U0=None):
    s = B.Solver(p, 1, max(len(sc.obstacles), 1), flags | B.FLAG_PROJECTED | B.FLAG_WRITE_SAMPLES)
    s.set_scene(sc)
    s.set_nominal(U0)
    s.set_counter(n0)
    s.solve()
    out = dict(U=s.get_controls(), S=s.get_costs(), XT=s.get_final_states(), diag=s.get_diag())
    s.close()
    return out


def pinned(O, sc, p, n, k, U):
    """min over (obstacle, step) of |h| along the oracle's own projected trajectory of sample k."""
    no = len(sc.obstacles)
    if no == 0:
        return False
    u = O.sample_projected(p, n, k, sc.x0, sc.goal, sc.obstacles, U)["u"]
    ua = np.array([p.sigma_ualpha * O.ualpha_normals(p.seed, n, k, t, no) for t in range(p.T)])
    r = O.rollout_projected(p, sc.x0, sc.goal, sc.obstacles, u, ua, O.alpha(p, n, k))
    if float(np.abs(r["Ab"][:, :, 2]).min()) < 1e-5:
        return True
    # at the edge of the alpha cost's indicator: h_i(x_{t+1}) next to h_buffer (module docstring)
    for t in range(1, p.T + 1):
        for ob in sc.obstacles:
            if abs(O.barrier_row(p, r["traj"][t], ob, t)[0] - p.h_buffer) < 1e-5:
                return True
    return False


def check(O, got, sc, p, n0=0, U0=None):
    U = np.zeros((p.T, 2)) if U0 is None else np.asarray(U0, dtype=np.float64)
    refs = O.solve_projected(p, n0, sc.x0, sc.goal, sc.obstacles, U, n_threads=8)
    ref = refs[-1]
    U_last = U if p.n_iter == 1 else refs[-2]["U"]
    okS = close(got["S"], ref["S"], 1.0)
    okX = close(got["XT"], ref["XT"], 1.0).all(axis=1)
    bad = np.flatnonzero(~(okS & okX))
    assert len(bad) <= 0.02 * p.K, f"{len(bad)} of {p.K} samples off; worst dS {np.abs(got['S'] - ref['S']).max()}"
    if p.n_iter == 1:
        for k in bad:       # each sample that is off must be pinned to a boundary by the oracle's own measure
            assert pinned(O, sc, p, n0, int(k), U_last), (k, got["S"][k], ref["S"][k], got["XT"][k], ref["XT"][k])
    floors = np.array([p.v_max, p.delta_max])
    err = np.abs(got["U"] - ref["U"]) / (RTOL * np.maximum(np.abs(ref["U"]), floors[None, :]))
    if len(bad) == 0 and p.n_iter == 1:
        assert err.max() <= 1.0, f"U worst error = {err.max():.2f} x tolerance"
    else:   # the samples that are off can move U by at most their share of the weight (controls are bounded)
        share = ref["w"][bad].sum() / ref["eta"] if len(bad) else 0.0
        bound = 1.0 + 2.0 * (share + (1e-3 if p.n_iter > 1 else 0.0)) / RTOL
        assert err.max() <= bound, f"U worst error = {err.max():.2f} x tolerance, bound {bound:.2f}"
    d = got["diag"]
    if ref["gap"] > 1e-3 * max(1.0, abs(ref["S"].min())) and len(bad) == 0:
        assert d["argmin"] == ref["argmin"]
    return len(bad)


@pytest.mark.parametrize("n_obs", [1, 2, 3, 4, 5, 8])
@pytest.mark.parametrize("precise", [0, 2], ids=["fast", "precise"])
def test_projected_iteration_matches_oracle(B, O, n_obs, precise):
    sc = near_scene(n_obs, n_obs, K=1000, T=40)
    got = gpu_projected(B, sc, sc.params, precise)
    check(O, got, sc, sc.params)


def test_no_obstacles_and_unused_capacity(B, O):
    sc = near_scene(3, 3, K=600, T=30)
    empty = scenes.Scene(sc.x0, sc.goal, np.zeros((0, 5)), sc.params)
    check(O, gpu_projected(B, empty, sc.params), empty, sc.params)
    # 3 obstacles in a context with room for 8: the unused rows must change nothing
    s = B.Solver(sc.params, 1, 8, B.FLAG_PROJECTED | B.FLAG_WRITE_SAMPLES)
    s.set_scene(sc)
    s.solve()
    a = dict(U=s.get_controls(), S=s.get_costs(), XT=s.get_final_states(), diag=s.get_diag())
    s.close()
    check(O, a, sc, sc.params)


def test_warm_nominal_moving_obstacles_off_axle_hitch(B, O):
    sc = near_scene(5, 8, K=800, T=50, Lh=0.75, proj_rho=1.0, h_buffer=2.0, w_alpha=3.0)
    U0 = np.tile([1.2, 0.15], (50, 1)).astype(np.float32)
    got = gpu_projected(B, sc, sc.params, 0, n0=7, U0=U0)
    check(O, got, sc, sc.params, n0=7, U0=U0)
    p3 = sc.params.with_(n_iter=3)
    got = gpu_projected(B, sc, p3, 0, n0=2)
    check(O, got, sc, p3, n0=2)


def test_pinned_samples_are_the_only_ones_off(B, O):
    """A start INSIDE an inflated obstacle drives many rollouts onto its boundary (h -> 0): those are the
    samples the rule in the module docstring excludes, every other one still meets 1e-4."""
    sc = near_scene(8, 8, K=1000, T=40)
    obs = sc.obstacles.copy()
    c = scenes.parking.vehicle_disc_centres(sc.x0[:3], sc.params.discs)[1]
    obs[3, :2] = c + np.array([0.0, 0.96 * (obs[3, 2] + sc.params.disc_radius)])
    sc2 = scenes.Scene(sc.x0, sc.goal, obs.astype(np.float32).astype(np.float64), sc.params)
    got = gpu_projected(B, sc2, sc2.params)
    check(O, got, sc2, sc2.params)


def test_cfg2_shape_and_paper_shape_sampled(B, O):
    """CFG2's K = 16384, T = 80, eight obstacles, and the paper's 5000 rollouts x H = 120 x 8 obstacles
    (PAPER.md:243): sampled (k) against the oracle, plus size-independent properties."""
    for K, T, dt in ((16384, 80, 0.05), (5000, 120, 0.04)):
        sc = near_scene(0, 8, K=K, T=T, dt=dt)
        p = sc.params
        got = gpu_projected(B, sc, p)
        rng = np.random.default_rng(K)
        ks = np.concatenate([[0, 127, 128, K - 1, int(got["diag"]["argmin"])], rng.integers(0, K, 120)])
        U0 = np.zeros((T, 2))
        n_bad = 0
        for k in ks:
            r = O.sample_projected(p, 0, int(k), sc.x0, sc.goal, sc.obstacles, U0)
            ok = close(got["S"][k], r["S"], 1.0) and close(got["XT"][k], r["xT"], 1.0).all()
            if not ok:
                assert pinned(O, sc, p, 0, int(k), U0), (k, got["S"][k], r["S"])
                n_bad += 1
        assert n_bad <= 3, n_bad
        d = got["diag"]
        assert np.isfinite(got["S"]).all() and d["nonfinite"] == 0
        assert got["S"][d["argmin"]] == got["S"].min()
        assert got["U"][:, 0].min() >= p.v_min and got["U"][:, 0].max() <= p.v_max
        assert got["U"][:, 1].min() >= p.delta_min and got["U"][:, 1].max() <= p.delta_max


def test_projection_keeps_rollouts_out_of_the_obstacle(B, O):
    """The point of the method: with the projection the sampled rollouts end outside the inflated obstacle they
    are driven at; the penalty-free unprojected ones (w_bar = 0) end inside it."""
    p = scenes.default_params(K=2048, T=60, dt=0.1, discs=((0, 2.0),), sigma_v=0.3, sigma_delta=0.05,
                              proj_qalpha=50.0, sigma_ualpha=0.05, w_bar=0.0, alpha_lo=0.1, alpha_hi=0.3)
    obs = np.array([[10.0, 0.0, 1.0, 0.0, 0.0]])
    sc = scenes.Scene(np.zeros(4), np.array([20.0, 0, 0, 0]), obs, p)
    U0 = np.tile([2.0, 0.0], (p.T, 1)).astype(np.float32)
    got = gpu_projected(B, sc, p, U0=U0)
    cx = got["XT"][:, 0] + 2.0 * np.cos(got["XT"][:, 2]) - 10.0
    cy = got["XT"][:, 1] + 2.0 * np.sin(got["XT"][:, 2])
    h_end = (cx**2 + cy**2) / (1.0 + p.disc_radius) ** 2 - 1.0
    assert (h_end > -1e-3).mean() > 0.99
    s = B.Solver(p, 1, 1, B.FLAG_WRITE_SAMPLES)
    s.set_scene(sc); s.set_nominal(U0); s.solve()
    XT = s.get_final_states(); s.close()
    # unprojected: they drive on towards the goal at 2 m/s x 6 s and pass through the obstacle region
    assert (XT[:, 0] > 9.0).mean() > 0.9


def test_closed_loop_and_errors(B, O):
    sc = near_scene(2, 8, K=512, T=30)
    s = B.Solver(sc.params, 1, 8, B.FLAG_PROJECTED)
    s.set_scene(sc)
    for _ in range(5):
        u0 = s.step()
        assert np.isfinite(u0).all()
    assert s.launch_count() == 5 * 3
    s.close()
    with pytest.raises(B.BrmppiError):
        B.Solver(sc.params, 1, 9, B.FLAG_PROJECTED)                      # more rows than the projection handles
    with pytest.raises(B.BrmppiError):
        B.Solver(sc.params, 1, 8, B.FLAG_PROJECTED, max_superellipses=2)
    with pytest.raises(B.BrmppiError):
        B.Solver(sc.params.with_(proj_qalpha=0.0), 1, 8, B.FLAG_PROJECTED)
    with pytest.raises(B.BrmppiError):
        B.Solver(sc.params.with_(proj_rho=-1.0), 1, 8, B.FLAG_PROJECTED)
    B.Solver(sc.params.with_(proj_qalpha=0.0), 1, 8, 0).close()          # not read without the flag


def test_random_configurations(B, O):
    """A seeded sweep over sizes the named cases do not visit (K 1 to 1000, T 1 to 60, 0 to 8 obstacles -- every
    obstacle-capacity instantiation, with unused capacity --, some moving, one to four discs, hitch offset, two
    projection weights rho, warm and zero nominal, a random iteration counter), each against the oracle by the
    module's rule."""
    rng = np.random.default_rng(20250813)
    disc_sets = [((0, 2.0),), ((0, 2.0), (1, -3.0)), ((0, 2.0), (1, -2.0), (1, -6.0)), ((0, 0.0), (0, 2.5), (1, -2.0), (1, -4.5))]
    n_off = 0
    for _ in range(200):
        K = int(rng.choice([1, 7, 31, 33, 100, 129, 333, 1000]))
        T = int(rng.choice([1, 2, 3, 5, 6, 7, 11, 12, 13, 24, 25, 40, 60]))
        n_obs = int(rng.integers(0, 9))
        sc = near_scene(int(rng.integers(0, 40)), n_obs, K=K, T=T, discs=disc_sets[int(rng.integers(0, 4))],
                        Lh=float(rng.choice([0.0, 0.75])), proj_rho=float(rng.choice([0.1, 1.0])))
        sc.params = sc.params.with_(seed=int(rng.integers(0, 2**40)))
        if n_obs and rng.random() < 0.5:
            m = rng.random(n_obs) < 0.5
            sc.obstacles[m, 3:] = rng.uniform(-1.5, 1.5, (int(m.sum()), 2)).astype(np.float32)
        n0 = int(rng.integers(0, 100))
        U0 = None if rng.random() < 0.5 else np.tile(np.array([[0.8, 0.1]], dtype=np.float32), (T, 1))
        cap = max(n_obs, 1) if rng.random() < 0.5 else 8
        s = B.Solver(sc.params, 1, cap, B.FLAG_PROJECTED | B.FLAG_WRITE_SAMPLES)
        s.set_scene(sc)
        s.set_nominal(U0)
        s.set_counter(n0)
        s.solve()
        got = dict(U=s.get_controls(), S=s.get_costs(), XT=s.get_final_states(), diag=s.get_diag())
        s.close()
        n_off += check(O, got, sc, sc.params, n0=n0, U0=U0)
    assert n_off <= 200         # pinned-and-off samples stay the exception over the whole sweep
