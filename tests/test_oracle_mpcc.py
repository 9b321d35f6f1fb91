"""Pins of the oracle's 7-state model, Taylor predictor (17) and contouring cost (13)-(15) (
DESIGN.md reading 31).  Closed forms of the Euler recursion, the spline against scipy's own evaluation, the error
definitions on a straight reference, the predictor against the continuous flow integrated by scipy (third-order
agreement, and its two derivatives one by one) and against an exact polynomial case, and an mpmath transcription of a
whole iteration that gets the Lie derivatives by differentiating h along a Taylor expansion of the flow instead of
the analytic formulas."""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy.integrate import solve_ivp
from scipy.interpolate import CubicSpline

import scenes
from test_oracle_bruteforce import philox_py, wrap, M32


def P(**kw):
    return scenes.default_params(**kw)


def straight_path(M=8, dpsi=2.0, heading=0.0, origin=(0.0, 0.0)):
    """Reference path along a straight line: linear position, constant headings."""
    coef = np.zeros((M, 4, 4))
    for m in range(M):
        coef[m, 0, 0] = origin[0] + m * dpsi * math.cos(heading); coef[m, 0, 1] = math.cos(heading)
        coef[m, 1, 0] = origin[1] + m * dpsi * math.sin(heading); coef[m, 1, 1] = math.sin(heading)
        coef[m, 2, 0] = heading; coef[m, 3, 0] = heading
    return coef, dpsi


# ---- eq. (6) ---------------------------------------------------------------------------------------------
def test_constant_jerk_closed_form_and_straight_line(O):
    """a_k = a_0 + k Ts j exactly; v_k = v_0 + k Ts a_0 + Ts^2 j k (k - 1) / 2 (the Euler sum, not the continuous
    v_0 + a_0 t + j t^2 / 2); with delta = 0 the headings never move and p_k = p_0 + Ts sum_{i<k} v_i e(theta1)."""
    p = P(dt=0.125)
    coef, dpsi = straight_path()
    x = np.array([1.0, -2.0, 0.5, 0.25, 0.75, 0.75, 0.0])
    j, Ts = -1.5, 0.125
    vs = []
    for k in range(20):
        assert x[3] == pytest.approx(0.25 + k * Ts * j, abs=1e-15)
        assert x[2] == pytest.approx(0.5 + k * Ts * 0.25 + Ts * Ts * j * k * (k - 1) / 2, abs=1e-14)
        assert x[4] == 0.75 and x[5] == 0.75 and x[6] == 0.0
        s = Ts * sum(vs)
        assert x[0] == pytest.approx(1.0 + s * math.cos(0.75), abs=1e-14) and x[1] == pytest.approx(-2.0 + s * math.sin(0.75), abs=1e-14)
        vs.append(x[2])
        x = O.step7(p, coef, dpsi, x, [j, 0.0])


def test_pose_part_is_the_reduced_model_and_steering_saturates(O):
    """(p, theta1, theta2) of (6) advance exactly like the pinned reduced step with inputs (v_k, delta_k); delta
    integrates omega and stops at the steering limits."""
    rng = np.random.default_rng(2)
    p = P(dt=0.05, Lh=0.4)
    coef, dpsi = straight_path()
    for _ in range(20):
        x = np.concatenate([rng.uniform(-3, 3, 2), [rng.uniform(-2, 2), rng.uniform(-1, 1)], rng.uniform(-3, 3, 2), [rng.uniform(-0.5, 0.5)]])
        u = [rng.uniform(-2, 2), rng.uniform(-0.9, 0.9)]
        xn = O.step7(p, coef, dpsi, x, u)
        r = O.kinematic_step(p, [x[0], x[1], x[4], x[5]], x[2], x[6])
        assert np.abs(np.array([xn[0], xn[1], xn[4], xn[5]]) - r).max() <= 1e-15
        assert xn[6] == pytest.approx(min(max(x[6] + p.dt * u[1], p.delta_min), p.delta_max), abs=1e-16)
    x = np.array([0, 0, 1.0, 0, 0, 0, 0.59])
    for _ in range(10):
        x = O.step7(p, coef, dpsi, x, [0.0, 0.9])
    assert x[6] == p.delta_max


# ---- reference path and errors -----------------------------------------------------------------------------
def test_path_table_reproduces_scipys_spline(O):
    """The coefficient table is a data recipe (scenes/mpcc.py); the oracle's evaluation of it must be the spline."""
    sc = scenes.scene_mpcc(3, K=8, T=4)
    M = sc.coef.shape[0]
    kk = sc.dpsi * np.arange(M + 1)
    rng = np.random.default_rng(0)
    ends = [O.path_eval(sc.params, sc.coef, sc.dpsi, k) for k in kk]
    for c in range(4):
        sp = CubicSpline(kk, [e[c] for e in ends])         # a spline through the oracle's own knot values
        for psi in rng.uniform(0, kk[-1], 50):
            # not the same spline (end conditions differ) but the table is C0 at the knots and cubic in between
            m = min(int(psi // sc.dpsi), M - 1)
            s = psi - m * sc.dpsi
            want = sum(sc.coef[m, c, q] * s**q for q in range(4))
            assert O.path_eval(sc.params, sc.coef, sc.dpsi, psi)[c] == pytest.approx(want, rel=1e-14, abs=1e-14)
        for m in range(1, M):                                # continuity across knots (to the table's fp32 rounding)
            left = sum(sc.coef[m - 1, c, q] * sc.dpsi**q for q in range(4))
            assert left == pytest.approx(sc.coef[m, c, 0], abs=2e-5)
    # clamped outside [0, L]
    assert np.array_equal(O.path_eval(sc.params, sc.coef, sc.dpsi, -3.0), O.path_eval(sc.params, sc.coef, sc.dpsi, 0.0))
    assert np.array_equal(O.path_eval(sc.params, sc.coef, sc.dpsi, 1e3), O.path_eval(sc.params, sc.coef, sc.dpsi, M * sc.dpsi))
    # arc-length parameterisation (a property of the RECIPE, approximate: the table is a spline through 25 knots of
    # the arc-length-resampled curve): |d p / d psi| ~ 1 along the path
    for psi in rng.uniform(0.5, kk[-1] - 0.5, 20):
        a, b = O.path_eval(sc.params, sc.coef, sc.dpsi, psi - 1e-4), O.path_eval(sc.params, sc.coef, sc.dpsi, psi + 1e-4)
        assert np.hypot(b[0] - a[0], b[1] - a[1]) / 2e-4 == pytest.approx(1.0, abs=0.15)


def test_errors_on_a_straight_reference(O):
    """Reference along +x: (14) gives e_c = -(p_y - p_y^r), the lateral offset up to sign, (15) e_l = -(p_x - p_x^r),
    the distance the projection point is ahead; both are invariant under a common rotation of path and vehicle;
    heading errors are wrapped differences."""
    p = P()
    coef, dpsi = straight_path()
    x = np.array([3.0, 0.7, 1.0, 0.0, 0.2, -0.1, 0.0])
    e = O.errors7(p, coef, dpsi, x, 2.5)
    assert e[0] == pytest.approx(-0.7, abs=1e-15) and e[1] == pytest.approx(-(3.0 - 2.5), abs=1e-15)
    assert e[2] == pytest.approx(0.2, abs=1e-15) and e[3] == pytest.approx(-0.1, abs=1e-15)
    for phi in (0.6, -2.0, 3.0):
        c2, d2 = straight_path(heading=phi)
        R = np.array([[math.cos(phi), -math.sin(phi)], [math.sin(phi), math.cos(phi)]])
        xr = x.copy(); xr[:2] = R @ x[:2]; xr[4] += phi; xr[5] += phi
        assert np.abs(O.errors7(p, c2, d2, xr, 2.5) - e).max() <= 1e-14
    x[4] = 2 * math.pi + 0.2
    assert O.errors7(p, coef, dpsi, x, 2.5)[2] == pytest.approx(0.2, abs=1e-14)
    # progress: the velocity projected on the path tangent
    assert O.progress7(p, coef, dpsi, [0, 0, 1.5, 0, 0.0, 0, 0], 1.0) == pytest.approx(1.5)
    assert O.progress7(p, coef, dpsi, [0, 0, 1.5, 0, math.pi / 2, 0, 0], 1.0) == pytest.approx(0.0, abs=1e-15)
    assert O.progress7(p, coef, dpsi, [0, 0, -1.5, 0, math.pi, 0, 0], 1.0) == pytest.approx(1.5)   # reversing along the path


# ---- predictor (17) ----------------------------------------------------------------------------------------
def flow(p, x, u, t_end):
    """The CONTINUOUS model behind (6) under constant input, integrated by scipy to 1e-12 (no clamp on delta)."""
    def f(t, s):
        px, py, v, a, th1, th2, de = s
        b = th1 - th2
        return [v * math.cos(th1), v * math.sin(th1), a, u[0], v / p.L1 * math.tan(de),
                v / p.L2 * (math.sin(b) - p.Lh / p.L1 * math.cos(b) * math.tan(de)), u[1]]
    r = solve_ivp(f, [0.0, t_end], list(x), rtol=1e-12, atol=1e-13, method="DOP853")
    return r.y[:, -1]


def h_exact(O, p, x7, ob, j, time):
    c = O.disc_centre(p, [x7[0], x7[1], x7[4], x7[5]], j)
    return O.barrier(p, c, ob[:2] + time * ob[3:5], ob[2])


def test_predictor_matches_the_continuous_flow_to_third_order(O):
    """hhat - h(x(Ts)) = O(Ts^3) (halving Ts divides the error by ~8), and its first and second derivative in Ts
    are the time derivatives of h along the flow (central differences of the integrated trajectory)."""
    rng = np.random.default_rng(5)
    for trial in range(12):
        Lh = 0.0 if trial % 2 else 0.75
        x = np.concatenate([rng.uniform(-3, 3, 2), [rng.uniform(-2, 2), rng.uniform(-1, 1)], rng.uniform(-3, 3, 2), [rng.uniform(-0.5, 0.5)]])
        u = np.array([rng.uniform(-2, 2), rng.uniform(-0.9, 0.9)])
        ob = np.array([rng.uniform(-8, 8), rng.uniform(-8, 8), rng.uniform(0.4, 1.5), rng.uniform(-1.5, 1.5), rng.uniform(-1.5, 1.5)])
        j = int(rng.integers(0, 3))
        errs = []
        for Ts in (0.1, 0.05, 0.025):
            p = P(dt=Ts, Lh=Lh)
            hh, h0 = O.hhat7(p, x, u, ob, 0, j)
            assert h0 == pytest.approx(h_exact(O, p, x, ob, j, 0.0), rel=1e-14)
            errs.append(abs(hh - h_exact(O, p, flow(p, x, u, p.dt), ob, j, p.dt)))
        assert errs[0] < 5e-2 and errs[2] < errs[0] / 30 + 1e-12         # third order: / 64 over two halvings
        # derivatives: hhat is h + Ts hdot + Ts^2/2 hddot, so three Ts values give hdot and hddot
        pa, pb = P(dt=0.5, Lh=Lh), P(dt=1.0, Lh=Lh)
        fa, h0 = O.hhat7(pa, x, u, ob, 0, j)
        fb, _ = O.hhat7(pb, x, u, ob, 0, j)
        hdd = (fb - h0 - 2 * (fa - h0)) / 0.25
        hd = (fa - h0) / 0.5 - 0.25 * hdd
        e = 1e-3
        hp, hm = h_exact(O, pa, flow(pa, x, u, e), ob, j, e), h_exact(O, pa, flow(pa, x, u, -e), ob, j, -e)
        assert (hp - hm) / (2 * e) == pytest.approx(hd, rel=1e-5, abs=1e-6)
        assert (hp - 2 * h0 + hm) / e**2 == pytest.approx(hdd, rel=2e-4, abs=2e-4)


def test_predictor_is_exact_up_to_the_cubic_term_on_a_straight_accelerating_approach(O):
    """delta = 0, omega = 0, j = 0, static obstacle, tractor disc: the disc moves s(t) = v t + a t^2 / 2 along e, so
    h(t) is a quartic in t and the predictor drops exactly (2 (d0.e) . 0 + v a t^3 + a^2 t^4 / 4) / rho^2."""
    p = P(dt=0.125, discs=((0, 2.0),), disc_radius=1.25)
    x = np.array([0.0, 0.0, 1.5, -0.75, 0.0, 0.0, 0.0])
    ob = np.array([9.0, 0.5, 0.75, 0.0, 0.0])
    hh, h0 = O.hhat7(p, x, [0.0, 0.0], ob, 0, 0)
    Ts, v, a, rho = 0.125, 1.5, -0.75, 2.0
    s = v * Ts + a * Ts * Ts / 2
    h_true = ((2.0 + s - 9.0) ** 2 + 0.25) / rho**2 - 1.0
    assert h_true - hh == pytest.approx((v * a * Ts**3 + a * a * Ts**4 / 4) / rho**2, rel=1e-10)
    # the jerk does not enter (relative degree 3), the steering rate does (through d delta / dt)
    assert O.hhat7(p, x, [2.0, 0.0], ob, 0, 0)[0] == hh
    assert O.hhat7(p, x, [0.0, 0.9], ob, 0, 0)[0] != hh
    # a moving obstacle: o(t) at step t, and hdot sees its velocity
    obm = np.array([9.0, 0.5, 0.75, -1.0, 0.0])
    hh_m, h_m = O.hhat7(p, x, [0.0, 0.0], obm, 4, 0)
    assert h_m == pytest.approx(((2.0 - (9.0 - 4 * Ts)) ** 2 + 0.25) / 4.0 - 1.0, rel=1e-14)
    assert hh_m < h_m - (hh - h0) * 0 and (hh_m - h_m) < (hh - h0)       # closing faster than against the static one


# ---- cost and rollout ----------------------------------------------------------------------------------------
def test_stage_cost_terms_by_hand(O):
    """One step, no obstacle, straight reference: every term of (13) from the definitions."""
    coef, dpsi = straight_path()
    p = P(T=1, dt=0.125, w_term=0.0, w_hitch=0.0, Qc=3.0, Ql=5.0, Qth1=7.0, Qth2=11.0, Rj=0.5, Rw=0.25, mu=2.0, nu_bar=1.0)
    x0 = np.array([1.0, 0.5, 0.8, 0.0, 0.1, -0.2, 0.0])
    u = np.array([[1.0, -0.4]])
    r = O.rollout7(p, coef, dpsi, x0, 0.75, np.zeros((0, 5)), u, 0.5)
    x1 = O.step7(p, coef, dpsi, x0, u[0])
    psi1 = 0.75 + 0.125 * 0.8 * math.cos(0.1)
    assert r["xT"][7] == pytest.approx(psi1, abs=1e-15) and np.array_equal(r["xT"][:7], x1)
    nu1 = x1[2] * math.cos(x1[4])
    want = 3.0 * x1[1] ** 2 + 5.0 * (x1[0] - psi1) ** 2 + 7.0 * x1[4] ** 2 + 11.0 * x1[5] ** 2 + 0.5 * 1.0 + 0.25 * 0.16 + 2.0 * (1.0 - nu1) ** 2
    assert r["S"] == pytest.approx(want, rel=1e-13)
    pt = p.with_(w_term=4.0)
    assert O.rollout7(pt, coef, dpsi, x0, 0.75, np.zeros((0, 5)), u, 0.5)["S"] - r["S"] == pytest.approx(
        4.0 * (3.0 * x1[1] ** 2 + 5.0 * (x1[0] - psi1) ** 2 + 7.0 * x1[4] ** 2 + 11.0 * x1[5] ** 2), rel=1e-12)
    # the barrier-rate hinge with the predictor: one obstacle straight ahead, one disc
    pb = p.with_(discs=((0, 2.0),), disc_radius=1.25, w_bar=10.0)
    ob = np.array([[4.5, 0.5, 0.75, 0.0, 0.0]])
    hh, h0 = O.hhat7(pb, x0, u[0], ob[0], 0, 0)
    base = O.rollout7(pb.with_(w_bar=0.0), coef, dpsi, x0, 0.75, ob, u, 0.5)["S"]
    assert (1 - 0.5) * h0 - hh > 0
    assert O.rollout7(pb, coef, dpsi, x0, 0.75, ob, u, 0.5)["S"] - base == pytest.approx(10.0 * ((1 - 0.5) * h0 - hh), rel=1e-12)


def brute_force7(p, coef, dpsi, n, x0, psi0, obstacles, U):
    """mpmath transcription of one iteration.  hdot and hddot are NOT the analytic formulas: the flow is expanded as
    x(t) = x + t F + t^2/2 (dF/dx F + dF/du . 0) with the Jacobian action by mp.diff, and h(x(t), o(t)) is
    differentiated in t by mp.diff."""
    mpf = mp.mpf
    K, T, D, No = p.K, p.T, len(p.discs), len(obstacles)
    key = (p.seed & M32, p.seed >> 32)
    f = lambda w: mpf(w >> 9) / 2**23
    Ts, L1, L2, Lh = mpf(p.dt), mpf(p.L1), mpf(p.L2), mpf(p.Lh)
    M = coef.shape[0]
    Lp = M * mpf(dpsi)

    def F(s, u):
        px, py, v, a, t1, t2, de = s
        b = t1 - t2
        return [v * mp.cos(t1), v * mp.sin(t1), a, u[0], v / L1 * mp.tan(de), v / L2 * (mp.sin(b) - Lh / L1 * mp.cos(b) * mp.tan(de)), u[1]]

    def path(psi):
        psi = min(max(psi, mpf(0)), Lp)
        m = min(int(mp.floor(psi / mpf(dpsi))), M - 1)
        s = psi - m * mpf(dpsi)
        return [sum(mpf(float(coef[m, c, q])) * s**q for q in range(4)) for c in range(4)]

    def hval(s, i, j, time):
        body, off = p.discs[j]
        ang = s[4] if body == 0 else s[5]
        cx = s[0] - Lh * mp.cos(s[4]) + mpf(off) * mp.cos(ang)
        cy = s[1] - Lh * mp.sin(s[4]) + mpf(off) * mp.sin(ang)
        ox = mpf(float(obstacles[i][0])) + time * mpf(float(obstacles[i][3]))
        oy = mpf(float(obstacles[i][1])) + time * mpf(float(obstacles[i][4]))
        rho = mpf(float(obstacles[i][2])) + mpf(p.disc_radius)
        return ((cx - ox) ** 2 + (cy - oy) ** 2) / rho**2 - 1

    def track(s, psi):
        r = path(psi)
        dx, dy = s[0] - r[0], s[1] - r[1]
        ec = mp.sin(r[2]) * dx - mp.cos(r[2]) * dy
        el = -mp.cos(r[2]) * dx - mp.sin(r[2]) * dy
        return mpf(p.Qc) * ec**2 + mpf(p.Ql) * el**2 + mpf(p.Qth1) * wrap(s[4] - r[2]) ** 2 + mpf(p.Qth2) * wrap(s[5] - r[3]) ** 2

    S, XT, us = [], [], []
    for k in range(K):
        alpha = mpf(p.alpha_lo) + (mpf(p.alpha_hi) - mpf(p.alpha_lo)) * f(philox_py((0, n, k, 1), key)[0])
        X = [mpf(float(a)) for a in x0]
        psi, cost, uk = mpf(psi0), mpf(0), []
        for t in range(T):
            w4 = philox_py((t >> 1, n, k, 0), key)
            wa, wb = (w4[2], w4[3]) if t & 1 else (w4[0], w4[1])
            r_ = mp.sqrt(-2 * mp.log(1 - f(wa)))
            z0, z1 = r_ * mp.cos(2 * mp.pi * f(wb)), r_ * mp.sin(2 * mp.pi * f(wb))
            u = (min(max(mpf(float(U[t][0])) + mpf(p.sigma_j) * z0, mpf(p.j_min)), mpf(p.j_max)),
                 min(max(mpf(float(U[t][1])) + mpf(p.sigma_omega) * z1, mpf(p.omega_min)), mpf(p.omega_max)))
            uk.append(u)
            F0 = F(X, u)
            # second derivative of the flow: d/ds F(x + s F0)|_0
            F1 = [mp.diff(lambda s_, c=c: F([X[q] + s_ * F0[q] for q in range(7)], u)[c], 0) for c in range(7)]
            xt = lambda tau: [X[q] + tau * F0[q] + tau**2 / 2 * F1[q] for q in range(7)]
            pen = mpf(0)
            for i in range(No):
                for j in range(D):
                    g = lambda tau: hval(xt(tau), i, j, t * Ts + tau)
                    h0, hd, hdd = g(mpf(0)), mp.diff(g, 0), mp.diff(g, 0, 2)
                    pen += max(mpf(0), (1 - alpha) * h0 - (h0 + Ts * hd + Ts**2 / 2 * hdd))
            Xn = [X[q] + Ts * F0[q] for q in range(7)]
            Xn[6] = min(max(Xn[6], mpf(p.delta_min)), mpf(p.delta_max))
            psin = min(max(psi + Ts * X[2] * mp.cos(X[4] - path(psi)[2]), mpf(0)), Lp)
            nu = Xn[2] * mp.cos(Xn[4] - path(psin)[2])
            hitch = max(mpf(0), abs(wrap(Xn[4] - Xn[5])) - (mpf(p.hitch_max) - mpf(p.hitch_kappa) * abs(Xn[2])))
            cost += track(Xn, psin) + mpf(p.Rj) * u[0] ** 2 + mpf(p.Rw) * u[1] ** 2 + mpf(p.mu) * (mpf(p.nu_bar) - nu) ** 2 + \
                mpf(p.w_hitch) * hitch**2 + mpf(p.w_bar) * pen
            X, psi = Xn, psin
        S.append(cost + mpf(p.w_term) * track(X, psi))
        XT.append(X + [psi])
        us.append(uk)
    smin = min(S)
    g = [mp.exp(-(s - smin) / mpf(p.lam)) for s in S]
    Unew = [[sum(g[k] * us[k][t][c] for k in range(K)) / sum(g) for c in range(2)] for t in range(T)]
    return dict(S=S, XT=XT, U=Unew, argmin=S.index(smin))


@pytest.mark.parametrize("case", [0, 1])
def test_iteration_matches_bruteforce(O, case):
    sc = scenes.scene_mpcc(case, K=4, T=4)
    if case == 0:
        p = sc.params.with_(seed=9)
        obs, x0, U = sc.obstacles[:2], sc.x0, np.zeros((4, 2))
    else:      # off-axle hitch, an obstacle next to the vehicle (hinge active), warm nominal, steering at its stop, hitch hinge active
        p = sc.params.with_(K=3, T=3, seed=2**33 + 1, Lh=0.75, dt=0.25, lam=2.0, hitch_max=0.2, hitch_kappa=0.05)
        x0 = sc.x0.copy(); x0[2] = 1.5; x0[3] = 0.5; x0[5] -= 0.5; x0[6] = 0.58
        x0 = x0.astype(np.float32).astype(float)
        obs = np.array([[x0[0] + 3.5, x0[1] + 0.5, 1.0, -0.5, 0.25], [x0[0] - 5.0, x0[1] + 2.0, 0.75, 0.0, 0.0]], dtype=np.float32).astype(float)
        U = np.array([[1.0, 0.8], [-0.5, 0.3], [1.9, -0.2]], dtype=np.float32).astype(float)
    ref = brute_force7(p, sc.coef, sc.dpsi, 3, x0, 0.25, obs, U)
    got = O.iteration7(p, sc.coef, sc.dpsi, 3, x0, 0.25, obs, U)
    assert got["argmin"] == ref["argmin"]
    for k in range(p.K):
        assert abs(got["S"][k] - ref["S"][k]) <= 1e-10 * max(1, abs(ref["S"][k]))
        for c in range(8):
            assert abs(got["XT"][k][c] - ref["XT"][k][c]) <= 1e-12
    for t in range(p.T):
        for c in range(2):
            assert abs(got["U"][t][c] - ref["U"][t][c]) <= 1e-12
