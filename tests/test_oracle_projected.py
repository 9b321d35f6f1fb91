"""Pins of the projected rollout in the C oracle (BR-MPPI proper, Sec. V-A; readings in
oracle/brmppi_oracle.h and DESIGN.md reading 30).  None of them retypes the oracle's formulas: the
closed form (12) is checked against the numpy form (another solver), against the optimality conditions of
(11) themselves and against scipy's constrained minimiser; the rows of (9) against finite differences of the
barrier through the (separately pinned) Euler step; the rollout against the constraint it has to satisfy at
every step; the whole sample against an mpmath transcription that solves the KKT system of (11) instead of
evaluating (12)."""
import math

import mpmath as mp
import numpy as np
import pytest

import scenes
from scenes.projection import projection_batch
from oracle import projection as OP
from test_oracle_bruteforce import philox_py, wrap, M32


def P(**kw):
    return scenes.default_params(**kw)


# ---- (12) ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n_o", [1, 2, 3, 5, 8])
@pytest.mark.parametrize("dense", [False, True])
def test_closed_form_against_numpy_solver_and_kkt(O, n_o, dense):
    B = projection_batch(40 + n_o, 50, n_o, dense=dense)
    for i in range(50):
        A, b, zd = B["A"][i], B["b"][i], B["z_des"][i]
        z, dropped = O.project(A, b, zd, B["w"], B["rho"], B["z_lo"], B["z_hi"])
        assert dropped == 0
        ref = OP.project(A, b, zd, B["w"], B["rho"], B["z_lo"], B["z_hi"])       # LAPACK solve, not Cholesky
        assert np.abs(z - ref).max() <= 1e-9 * max(1.0, np.abs(ref).max())
        assert np.abs(A @ z - b).max() <= 1e-10 * (1.0 + np.abs(A) @ np.abs(z)).max()   # feasibility (11b)
        # stationarity of (11a) on null(A): its gradient 2 W (z - z_des) + rho (2 z - z_lo - z_hi) is a
        # combination of the rows of A
        g = 2 * B["w"] * (z - zd) + B["rho"] * (2 * z - B["z_lo"] - B["z_hi"])
        coef = np.linalg.lstsq(A.T, g, rcond=None)[0]
        assert np.abs(A.T @ coef - g).max() <= 1e-8 * max(1.0, np.abs(g).max())


def test_closed_form_against_scipy_slsqp(O):
    from scipy.optimize import minimize
    B = projection_batch(3, 12, 4)
    for i in range(12):
        A, b, zd = B["A"][i], B["b"][i], B["z_des"][i]
        z, _ = O.project(A, b, zd, B["w"], B["rho"], B["z_lo"], B["z_hi"])
        f = lambda x: OP.objective(x, zd, B["w"], B["rho"], B["z_lo"], B["z_hi"])
        r = minimize(f, np.zeros(6), constraints=[dict(type="eq", fun=lambda x: A @ x - b)], method="SLSQP",
                     options=dict(ftol=1e-14, maxiter=500))
        assert r.success and np.abs(r.x - z).max() <= 2e-6
        assert f(z) <= r.fun + 1e-9


def test_single_constraint_scalar_form_and_limits(O):
    """N_o = 1: z* = y - M^-1 a (a.y - b) / (a.M^-1 a), y = M^-1 p (the projection onto one hyperplane in the
    M-metric).  rho = 0: the weighted minimum-norm projection (10), z_des + W^-1/2 pinv(A W^-1/2)(b - A z_des).
    rho -> inf: the Euclidean projection of the centre of the bounds onto {A z = b}."""
    rng = np.random.default_rng(1)
    for _ in range(20):
        a = rng.normal(size=3); b = rng.normal(); zd = rng.normal(size=3)
        w = rng.uniform(0.2, 3, 3); rho = rng.uniform(0, 2); lo = -rng.uniform(0.5, 2, 3); hi = rng.uniform(0.5, 2, 3)
        z, _ = O.project(a[None, :], [b], zd, w, rho, lo, hi)
        Minv = 1 / (w + rho)
        y = Minv * (w * zd + 0.5 * rho * (lo + hi))
        want = y - Minv * a * (a @ y - b) / (a @ (Minv * a))
        assert np.abs(z - want).max() <= 1e-12
    B = projection_batch(9, 10, 5)
    for i in range(10):
        A, b, zd, w = B["A"][i], B["b"][i], B["z_des"][i], B["w"]
        z0, _ = O.project(A, b, zd, w, 0.0, B["z_lo"], B["z_hi"])
        want = zd + (1 / np.sqrt(w)) * (np.linalg.pinv(A / np.sqrt(w)[None, :]) @ (b - A @ zd))
        assert np.abs(z0 - want).max() <= 1e-10
        zi, _ = O.project(A, b, zd, w, 1e9, B["z_lo"], B["z_hi"])
        c = 0.5 * (B["z_lo"] + B["z_hi"])
        want = c + np.linalg.pinv(A) @ (b - A @ c)
        assert np.abs(zi - want).max() <= 1e-6


def test_rank_deficient_row_is_dropped(O):
    B = projection_batch(5, 1, 4)
    A, b, zd = B["A"][0].copy(), B["b"][0].copy(), B["z_des"][0]
    A[3] = A[1]; b[3] = b[1]                               # the same constraint twice
    z, dropped = O.project(A, b, zd, B["w"], B["rho"], B["z_lo"], B["z_hi"])
    assert dropped == 1
    want, _ = O.project(A[:3], b[:3], zd, B["w"], B["rho"], B["z_lo"], B["z_hi"])
    assert np.abs(z - want).max() <= 1e-12 and np.abs(A @ z - b).max() <= 1e-10


# ---- rows of (9) -----------------------------------------------------------------------------------
def test_barrier_row_hand_value(O):
    """One tractor disc 2 m ahead of the axle, obstacle 3 m ahead of the disc, rho = 2: h = 9/4 - 1,
    grad_c h = 2 (c - o) / rho^2 = (-1.5, 0); driving forward lowers h by 1.5 dt per m/s, steering does nothing
    to first order (the disc moves sideways, perpendicular to c - o)."""
    p = P(dt=0.125, discs=((0, 2.0),), disc_radius=1.25, L1=4.0, Lh=0.0)     # all exactly representable
    h, j, Lg, Lf = O.barrier_row(p, [0, 0, 0, 0], [5.0, 0.0, 0.75, -0.5, 2.0], 0)
    assert j == 0 and h == pytest.approx(1.25, rel=1e-15)
    assert Lg[0] == pytest.approx(-0.1875, rel=1e-14) and abs(Lg[1]) <= 1e-16
    # L_f h = -grad_c h . dt vel = -(-1.5)(0.125)(-0.5) = -0.09375: an obstacle coming closer lowers h
    assert Lf == pytest.approx(-0.09375, rel=1e-14)
    # the disc with the smallest h is the active one; ties -> lowest index
    p3 = P(dt=0.1)
    hs = [O.barrier(p3, O.disc_centre(p3, [0, 0, 0.3, -0.2], jj), [-4.0, -1.0], 1.0) for jj in range(3)]
    h, j, _, _ = O.barrier_row(p3, [0, 0, 0.3, -0.2], [-4.0, -1.0, 1.0, 0, 0], 0)
    assert h == min(hs) and j == int(np.argmin(hs))


@pytest.mark.parametrize("Lh", [0.0, 0.75])
def test_lie_derivatives_against_finite_differences(O, Lh):
    """L_g h . w is the first-order change of h (of the active disc) under x' = x + dt G(x) w: central
    differences through orc_affine_step; L_f h is the exact change of h under the obstacle's step minus the
    second-order term |dt vel|^2 / rho^2."""
    rng = np.random.default_rng(7)
    p = P(dt=0.05, Lh=Lh)
    for _ in range(40):
        x = np.array([rng.uniform(-5, 5), rng.uniform(-5, 5), rng.uniform(-3, 3), rng.uniform(-3, 3)])
        ob = np.array([rng.uniform(-12, 12), rng.uniform(-12, 12), rng.uniform(0.4, 1.5), rng.uniform(-1.5, 1.5), rng.uniform(-1.5, 1.5)])
        t = int(rng.integers(0, 30))
        h, j, Lg, Lf = O.barrier_row(p, x, ob, t)
        o_t = ob[:2] + t * p.dt * ob[3:5]
        hj = lambda xx, oo: O.barrier(p, O.disc_centre(p, xx, j), oo, ob[2])
        assert hj(x, o_t) == pytest.approx(h, rel=1e-14)
        eps = 1e-4
        for e in range(2):
            w = np.zeros(2); w[e] = eps
            fd = (hj(O.affine_step(p, x, w), o_t) - hj(O.affine_step(p, x, -w), o_t)) / (2 * eps)
            assert fd == pytest.approx(Lg[e], rel=2e-6, abs=1e-9)
        rho = ob[2] + p.disc_radius
        dv = p.dt * ob[3:5]
        assert hj(x, o_t + dv) - h == pytest.approx(Lf + dv @ dv / rho**2, rel=1e-10, abs=1e-13)


def test_affine_step_is_the_euler_step_in_other_inputs(O):
    rng = np.random.default_rng(3)
    p = P(dt=0.05, Lh=0.4)
    for _ in range(20):
        x = rng.uniform(-3, 3, 4); v = rng.uniform(-2, 2); d = rng.uniform(-0.6, 0.6)
        a = O.affine_step(p, x, [v, v * math.tan(d)])
        b = O.kinematic_step(p, x, v, d)
        assert np.abs(a - b).max() <= 1e-14


def test_ualpha_normals_moments_and_layout(O):
    """Unit normals, independent across obstacles and of the control noise; obstacle i of block q = i >> 2."""
    z = np.array([O.ualpha_normals(5, 1, k, t, 8) for k in range(400) for t in range(25)])
    assert np.abs(z.mean(axis=0)).max() <= 4 / math.sqrt(len(z))
    assert np.abs(z.var(axis=0) - 1).max() <= 0.05
    c = np.corrcoef(z.T)
    assert np.abs(c - np.eye(8)).max() <= 0.04
    assert np.array_equal(O.ualpha_normals(5, 1, 7, 3, 3), O.ualpha_normals(5, 1, 7, 3, 8)[:3])
    zc = np.array([O.normals(5, 1, k, t) for k in range(400) for t in range(25)])
    assert np.abs(np.corrcoef(np.hstack([z[:, :2], zc]).T) - np.eye(4)).max() <= 0.04


# ---- the rollout -----------------------------------------------------------------------------------
def _random_rollout(O, seed, n_obs, **kw):
    sc = scenes.scene_cfg2(seed)
    p = sc.params.with_(K=4, T=25, **kw)
    rng = np.random.default_rng(seed)
    obs = sc.obstacles[:n_obs].copy()
    obs[:, :2] = sc.x0[:2] + rng.uniform(-9, 9, (n_obs, 2))          # close enough to matter
    obs = obs.astype(np.float32).astype(np.float64)
    u = np.stack([np.clip(rng.normal(0.5, 1.0, p.T), p.v_min, p.v_max), np.clip(rng.normal(0, 0.3, p.T), p.delta_min, p.delta_max)], axis=1)
    ua = p.sigma_ualpha * rng.normal(size=(p.T, n_obs))
    return sc, p, obs, u, ua


@pytest.mark.parametrize("n_obs", [1, 3, 8])
def test_rollout_satisfies_the_equality_at_every_step(O, n_obs):
    """(9) holds at every prediction step with the PROJECTED inputs, alpha follows alpha + u^alpha_proj
    (PAPER.md:183), the trajectory is the affine step of the projected input."""
    for seed in range(3):
        sc, p, obs, u, ua = _random_rollout(O, seed, n_obs)
        r = O.rollout_projected(p, sc.x0, sc.goal, obs, u, ua, 0.4)
        for t in range(p.T):
            for i in range(n_obs):
                Lg0, Lg1, h, b = r["Ab"][t, i]
                lhs = Lg0 * r["z"][t, 0] + Lg1 * r["z"][t, 1] + h * r["z"][t, 2 + i]
                assert abs(lhs - b) <= 1e-9 * (1 + abs(b) + abs(h))
                # b = -alpha h - L_f h and the row is the one barrier_row gives at the rollout's own state
                hh, _, Lg, Lf = O.barrier_row(p, r["traj"][t], obs[i], t)
                assert (hh, Lg[0], Lg[1]) == (h, Lg0, Lg1)
                assert b == pytest.approx(-r["alpha"][t, i] * hh - Lf, rel=1e-14, abs=1e-15)
            assert np.abs(r["alpha"][t + 1] - (r["alpha"][t] + r["z"][t, 2:])).max() <= 1e-15
            assert np.abs(r["traj"][t + 1] - O.affine_step(p, r["traj"][t], r["z"][t, :2])).max() == 0.0
        assert np.all(r["alpha"][0] == 0.4)


def test_far_obstacles_leave_the_input_alone_and_no_obstacle_is_plain_mppi(O):
    sc, p, obs, u, ua = _random_rollout(O, 1, 2, proj_rho=0.0, w_delta=0.0)
    far = obs.copy(); far[:, :2] += 1e5
    r = O.rollout_projected(p, sc.x0, sc.goal, far, u, ua, 0.4)
    w_des = np.stack([u[:, 0], u[:, 0] * np.tan(u[:, 1])], axis=1)
    assert np.abs(r["z"][:, :2] - w_des).max() <= 1e-6          # the alpha channel absorbs the constraint
    r0 = O.rollout_projected(p, sc.x0, sc.goal, np.zeros((0, 5)), u, np.zeros((p.T, 0)), 0.4)
    plain = O.rollout(p, sc.x0, sc.goal, np.zeros((0, 5)), u, 0.4, want_traj=True)
    assert np.abs(r0["traj"] - plain["traj"]).max() <= 1e-12
    assert r0["S"] == pytest.approx(plain["S"], rel=1e-12)      # w_delta = 0: omega^2 vs delta^2 is the only difference


def test_projection_turns_the_vehicle_away(O):
    """Driving straight at an obstacle with alpha fixed near 0 (q_alpha huge, no sampled u^alpha): the
    equality h' = -(alpha) h lets h decay no faster than alpha h per step, so the vehicle must slow down;
    without the projection it drives through."""
    p = P(T=40, dt=0.1, discs=((0, 2.0),), proj_qalpha=1e6, proj_rho=0.0, sigma_ualpha=0.0)
    obs = np.array([[9.0, 0.0, 0.7, 0.0, 0.0]])
    u = np.tile([2.0, 0.0], (p.T, 1))
    r = O.rollout_projected(p, [0, 0, 0, 0], [20, 0, 0, 0], obs, u, np.zeros((p.T, 1)), 0.2)
    hs = [O.barrier_row(p, x, obs[0], 0)[0] for x in r["traj"]]
    assert min(hs) > 0 and hs[-1] < 0.1 * hs[0]                 # approaches, never enters
    assert all(h1 >= 0.79 * h0 for h0, h1 in zip(hs, hs[1:]))   # h_{t+1} ~ (1 - alpha) h_t up to 2nd order
    plain = O.rollout(p, [0, 0, 0, 0], [20, 0, 0, 0], obs, u, 0.2, want_traj=True)
    assert min(O.barrier(p, O.disc_centre(p, x, 0), obs[0, :2], 0.7) for x in plain["traj"]) < 0


def test_alpha_cost_counts_positive_alpha_inside_the_buffer(O):
    sc, p, obs, u, ua = _random_rollout(O, 2, 3, w_alpha=0.0)
    obs[:, :2] = sc.x0[:2] + np.array([[3.0, 2.0], [-7.0, -2.5], [40.0, 0.0]], dtype=np.float32)
    r0 = O.rollout_projected(p, sc.x0, sc.goal, obs, u, ua, 0.6)
    pw = p.with_(w_alpha=3.0, h_buffer=2.0)
    r1 = O.rollout_projected(pw, sc.x0, sc.goal, obs, u, ua, 0.6)
    want = 0.0
    for t in range(p.T):
        for i in range(3):
            h = O.barrier_row(p, r0["traj"][t + 1], obs[i], t + 1)[0]
            a = r0["alpha"][t + 1, i]
            if h < 2.0 and a > 0:
                want += 3.0 * a * a
    assert want > 0 and r1["S"] - r0["S"] == pytest.approx(want, rel=1e-10)
    assert np.array_equal(r0["traj"], r1["traj"])               # a cost, not a constraint


# ---- brute force -----------------------------------------------------------------------------------
def brute_force_projected(p, n, x0, goal, obstacles, U):
    """Independent mpmath transcription of one projected iteration.  The projection is NOT evaluated by (12):
    the KKT system of (11), [2M  A^T; A  0][z; mu] = [2p; b], is solved by LU instead."""
    mpf = mp.mpf
    K, T, No, D = p.K, p.T, len(obstacles), len(p.discs)
    key = (p.seed & M32, p.seed >> 32)
    f = lambda w: mpf(w >> 9) / 2**23
    bm = lambda wa, wb: (mp.sqrt(-2 * mp.log(1 - f(wa))) * mp.cos(2 * mp.pi * f(wb)), mp.sqrt(-2 * mp.log(1 - f(wa))) * mp.sin(2 * mp.pi * f(wb)))
    dt, L1, L2, Lh = mpf(p.dt), mpf(p.L1), mpf(p.L2), mpf(p.Lh)
    vabs = max(abs(mpf(p.v_min)), abs(mpf(p.v_max)))
    om = vabs * mp.tan(max(abs(mpf(p.delta_min)), abs(mpf(p.delta_max))))
    wd = [mpf(p.proj_qv), mpf(p.proj_qomega)] + [mpf(p.proj_qalpha)] * No
    lo = [mpf(p.v_min), -om] + [-mpf(p.ualpha_max)] * No
    hi = [mpf(p.v_max), om] + [mpf(p.ualpha_max)] * No
    rho = mpf(p.proj_rho)

    def centre(X, j):
        body, off = p.discs[j]
        ang = X[2] if body == 0 else X[3]
        return (X[0] - Lh * mp.cos(X[2]) + mpf(off) * mp.cos(ang), X[1] - Lh * mp.sin(X[2]) + mpf(off) * mp.sin(ang))

    def hval(X, i, j, t):
        c = centre(X, j)
        ox = mpf(float(obstacles[i][0])) + t * dt * mpf(float(obstacles[i][3]))
        oy = mpf(float(obstacles[i][1])) + t * dt * mpf(float(obstacles[i][4]))
        r = mpf(float(obstacles[i][2])) + mpf(p.disc_radius)
        return ((c[0] - ox) ** 2 + (c[1] - oy) ** 2) / r**2 - 1

    def step(X, w):
        b = X[2] - X[3]
        return (X[0] + dt * w[0] * mp.cos(X[2]), X[1] + dt * w[0] * mp.sin(X[2]), X[2] + dt * w[1] / L1,
                X[3] + dt * (w[0] * mp.sin(b) - Lh / L1 * w[1] * mp.cos(b)) / L2)

    def G(s):
        return mpf(p.w_pos) * ((s[0] - mpf(float(goal[0]))) ** 2 + (s[1] - mpf(float(goal[1]))) ** 2) + \
            mpf(p.w_head) * (wrap(s[2] - mpf(float(goal[2]))) ** 2 + wrap(s[3] - mpf(float(goal[3]))) ** 2)

    S, XT, us = [], [], []
    for k in range(K):
        alpha = [mpf(p.alpha_lo) + (mpf(p.alpha_hi) - mpf(p.alpha_lo)) * f(philox_py((0, n, k, 1), key)[0])] * No
        X = tuple(mpf(float(a)) for a in x0)
        cost, uk = mpf(0), []
        for t in range(T):
            w4 = philox_py((t >> 1, n, k, 0), key)
            zv, zd = bm(w4[2], w4[3]) if t & 1 else bm(w4[0], w4[1])
            v = min(max(mpf(float(U[t][0])) + mpf(p.sigma_v) * zv, mpf(p.v_min)), mpf(p.v_max))
            d = min(max(mpf(float(U[t][1])) + mpf(p.sigma_delta) * zd, mpf(p.delta_min)), mpf(p.delta_max))
            uk.append((v, d))
            zeta = []
            for q in range((No + 3) // 4):
                b4 = philox_py((t, n, k, 2 + q), key)
                zeta += list(bm(b4[0], b4[1])) + list(bm(b4[2], b4[3]))
            zdes = [v, v * mp.tan(d)] + [mpf(p.sigma_ualpha) * zeta[i] for i in range(No)]
            # rows of (9) by differentiating h numerically-free: mpmath's own derivative of t -> h(step(X, t e))
            rows, rhs = [], []
            for i in range(No):
                hs = [hval(X, i, j, t) for j in range(D)]
                js = hs.index(min(hs))
                h = hs[js]
                Lg = [mp.diff(lambda s, e=e: hval(step(X, [s if e == 0 else 0, s if e == 1 else 0]), i, js, t), 0) for e in range(2)]
                # L_f h: derivative of h along the obstacle's motion over one step
                Lf = mp.diff(lambda s: hval(X, i, js, t + s), 0)
                rows.append(Lg + [h if c == i else mpf(0) for c in range(No)])
                rhs.append(-alpha[i] * h - Lf)
            d_ = 2 + No
            if No:
                KKT = mp.zeros(d_ + No)
                r_ = mp.zeros(d_ + No, 1)
                for j in range(d_):
                    KKT[j, j] = 2 * (wd[j] + rho)
                    r_[j] = 2 * (wd[j] * zdes[j] + rho / 2 * (lo[j] + hi[j]))
                    for i in range(No):
                        KKT[j, d_ + i] = rows[i][j]
                        KKT[d_ + i, j] = rows[i][j]
                for i in range(No):
                    r_[d_ + i] = rhs[i]
                sol = mp.lu_solve(KKT, r_)
                z = [sol[j] for j in range(d_)]
            else:
                z = [(wd[j] * zdes[j] + rho / 2 * (lo[j] + hi[j])) / (wd[j] + rho) for j in range(2)]
            Xn = step(X, z[:2])
            alpha = [alpha[i] + z[2 + i] for i in range(No)]
            hitch = max(mpf(0), abs(wrap(Xn[2] - Xn[3])) - (mpf(p.hitch_max) - mpf(p.hitch_kappa) * abs(z[0])))
            ca = sum(alpha[i] ** 2 for i in range(No)
                     if min(hval(Xn, i, j, t + 1) for j in range(D)) < mpf(p.h_buffer) and alpha[i] > 0)
            cost += G(Xn) + mpf(p.w_v) * z[0] ** 2 + mpf(p.w_delta) * z[1] ** 2 + mpf(p.w_hitch) * hitch**2 + mpf(p.w_alpha) * ca
            X = Xn
        S.append(cost + mpf(p.w_term) * G(X))
        XT.append(X)
        us.append(uk)
    smin = min(S)
    g = [mp.exp(-(s - smin) / mpf(p.lam)) for s in S]
    Unew = [[sum(g[k] * us[k][t][c] for k in range(K)) / sum(g) for c in range(2)] for t in range(T)]
    return dict(S=S, XT=XT, U=Unew, argmin=S.index(smin))


@pytest.mark.parametrize("case", [0, 1, 2])
def test_projected_iteration_matches_bruteforce(O, case):
    sc = scenes.scene_cfg0(case)
    if case == 0:      # one static obstacle
        p = sc.params.with_(K=4, T=4, seed=11, h_buffer=30.0)
        obs, x0, U = sc.obstacles, sc.x0, np.zeros((4, 2))
    elif case == 1:    # off-axle hitch, a moving obstacle and one overlapping the vehicle, warm nominal, 5 obstacles (two Philox blocks)
        p = sc.params.with_(K=3, T=3, seed=2**40 + 3, Lh=0.75, dt=0.25, lam=3.0, h_buffer=5.0, proj_rho=1.5)
        obs = np.array([[3.0, 0.5, 1.0, -1.0, 0.25], [-5.0, 1.0, 1.5, 0.0, 0.0], [6.0, -4.0, 0.5, 0.3, 0.3],
                        [0.0, 9.0, 1.0, 0.0, -1.0], [-9.0, -9.0, 1.2, 0.0, 0.0]], dtype=np.float32).astype(float)
        x0 = np.array([0.5, -0.25, 0.4, -0.9], dtype=np.float32).astype(float)
        U = np.array([[1.0, 0.2], [-0.5, -0.3], [1.9, 0.55]], dtype=np.float32).astype(float)
    else:              # no obstacle at all: soft-bounded plain MPPI
        p = sc.params.with_(K=4, T=3, seed=5, dt=0.2, proj_rho=0.7)
        obs, x0, U = np.zeros((0, 5)), sc.x0, np.array([[-1.5, 0.1]] * 3, dtype=np.float32).astype(float)
    n = 4
    ref = brute_force_projected(p, n, x0, sc.goal, obs, U)
    got = O.iteration_projected(p, n, x0, sc.goal, obs, U)
    assert got["argmin"] == ref["argmin"]
    for k in range(p.K):
        assert abs(got["S"][k] - ref["S"][k]) <= 1e-10 * max(1, abs(ref["S"][k]))
        for c in range(4):
            assert abs(got["XT"][k][c] - ref["XT"][k][c]) <= 1e-11
    for t in range(p.T):
        for c in range(2):
            assert abs(got["U"][t][c] - ref["U"][t][c]) <= 1e-11
