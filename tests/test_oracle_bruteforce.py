"""Brute force pin (NS: "results match brute force at K<=8, T<=5"): an independent transcription
of one BR-MPPI iteration in pure Python with mpmath at 50 digits, structured differently from the
oracle on purpose -- everything is materialised (all controls, all trajectories, the full table of
barrier values h[k][t][i][j]) and the cost is assembled from those tables afterwards, the softmax
is written as normalised weights.  The C oracle must agree to 1e-12."""
import mpmath as mp
import numpy as np
import pytest

import scenes

mp.mp.dps = 50
M32 = 0xFFFFFFFF


def philox_py(ctr, key):
    c = list(ctr)
    k = list(key)
    for _ in range(10):
        p0 = 0xD2511F53 * c[0]
        p1 = 0xCD9E8D57 * c[2]
        c = [((p1 >> 32) ^ c[1] ^ k[0]) & M32, p1 & M32, ((p0 >> 32) ^ c[3] ^ k[1]) & M32, p0 & M32]
        k = [(k[0] + 0x9E3779B9) & M32, (k[1] + 0xBB67AE85) & M32]
    return c


def wrap(a):
    return a - 2 * mp.pi * mp.nint(a / (2 * mp.pi))


def brute_force(p, n, x0, goal, obstacles, U, superellipses=()):
    K, T, D = p.K, p.T, len(p.discs)
    key = (p.seed & M32, p.seed >> 32)
    f = lambda w: mp.mpf(w >> 9) / 2**23
    mpf = mp.mpf
    # 1. all controls and alphas
    u = [[None] * T for _ in range(K)]
    alpha = []
    for k in range(K):
        alpha.append(mpf(p.alpha_lo) + (mpf(p.alpha_hi) - mpf(p.alpha_lo)) * f(philox_py((0, n, k, 1), key)[0]))
        for t in range(T):
            w = philox_py((t >> 1, n, k, 0), key)       # one block per pair of steps (reading 6)
            wa, wb = (w[2], w[3]) if t & 1 else (w[0], w[1])
            r = mp.sqrt(-2 * mp.log(1 - f(wa)))
            zv, zd = r * mp.cos(2 * mp.pi * f(wb)), r * mp.sin(2 * mp.pi * f(wb))
            v = min(max(mpf(U[t][0]) + mpf(p.sigma_v) * zv, mpf(p.v_min)), mpf(p.v_max))
            d = min(max(mpf(U[t][1]) + mpf(p.sigma_delta) * zd, mpf(p.delta_min)), mpf(p.delta_max))
            u[k][t] = (v, d)
    # 2. all trajectories
    X = [[None] * (T + 1) for _ in range(K)]
    for k in range(K):
        X[k][0] = tuple(mpf(float(a)) for a in x0)
        for t in range(T):
            x, y, p1, p2 = X[k][t]
            v, d = u[k][t]
            X[k][t + 1] = (x + p.dt * v * mp.cos(p1), y + p.dt * v * mp.sin(p1),
                           p1 + p.dt * v / mpf(p.L1) * mp.tan(d),
                           p2 + p.dt * v / mpf(p.L2) * (mp.sin(p1 - p2) - mpf(p.Lh) / mpf(p.L1) * mp.cos(p1 - p2) * mp.tan(d)))
    # 3. barrier table
    def h(k, t, i, j):
        x, y, p1, p2 = X[k][t]
        body, off = p.discs[j]
        ang = p1 if body == 0 else p2
        cx = x - mpf(p.Lh) * mp.cos(p1) + mpf(off) * mp.cos(ang)
        cy = y - mpf(p.Lh) * mp.sin(p1) + mpf(off) * mp.sin(ang)
        ox = mpf(float(obstacles[i][0])) + t * mpf(p.dt) * mpf(float(obstacles[i][3]))
        oy = mpf(float(obstacles[i][1])) + t * mpf(p.dt) * mpf(float(obstacles[i][4]))
        rho = mpf(float(obstacles[i][2])) + mpf(p.disc_radius)
        return ((cx - ox) ** 2 + (cy - oy) ** 2) / rho**2 - 1
    def h_se(k, t, i, j):      # eq. (16)
        x, y, p1, p2 = X[k][t]
        body, off = p.discs[j]
        ang = p1 if body == 0 else p2
        cx = x - mpf(p.Lh) * mp.cos(p1) + mpf(off) * mp.cos(ang)
        cy = y - mpf(p.Lh) * mp.sin(p1) + mpf(off) * mp.sin(ang)
        ocx, ocy, mx, my, th, vx, vy, e = (mpf(float(a)) for a in superellipses[i])
        dx, dy = cx - (ocx + t * mpf(p.dt) * vx), cy - (ocy + t * mpf(p.dt) * vy)
        xp = mp.cos(th) * dx + mp.sin(th) * dy
        yp = -mp.sin(th) * dx + mp.cos(th) * dy
        return abs(xp / (mx + mpf(p.disc_radius))) ** e + abs(yp / (my + mpf(p.disc_radius))) ** e - 1
    H = [[[[h(k, t, i, j) for j in range(D)] for i in range(len(obstacles))] +
          [[h_se(k, t, i, j) for j in range(D)] for i in range(len(superellipses))]
          for t in range(T + 1)] for k in range(K)]
    # 4. costs from the tables
    def G(s):
        return mpf(p.w_pos) * ((s[0] - mpf(float(goal[0]))) ** 2 + (s[1] - mpf(float(goal[1]))) ** 2) + \
            mpf(p.w_head) * (wrap(s[2] - mpf(float(goal[2]))) ** 2 + wrap(s[3] - mpf(float(goal[3]))) ** 2)
    S = []
    for k in range(K):
        bar = sum(max(mpf(0), (1 - alpha[k]) * H[k][t][i][j] - H[k][t + 1][i][j])
                  for t in range(T) for i in range(len(obstacles) + len(superellipses)) for j in range(D))
        track = sum(G(X[k][t + 1]) for t in range(T))
        effort = sum(mpf(p.w_v) * u[k][t][0] ** 2 + mpf(p.w_delta) * u[k][t][1] ** 2 for t in range(T))
        hitch = sum(mpf(p.w_hitch) * max(mpf(0), abs(wrap(X[k][t + 1][2] - X[k][t + 1][3])) - (mpf(p.hitch_max) - mpf(p.hitch_kappa) * abs(u[k][t][0]))) ** 2
                    for t in range(T))
        S.append(track + effort + hitch + mpf(p.w_bar) * bar + mpf(p.w_term) * G(X[k][T]))
    # 5. normalised softmax weights and update
    smin = min(S)
    g = [mp.exp(-(s - smin) / mpf(p.lam)) for s in S]
    gbar = [x / sum(g) for x in g]
    Unew = [[sum(gbar[k] * u[k][t][c] for k in range(K)) for c in range(2)] for t in range(T)]
    return dict(S=S, U=Unew, XT=[X[k][T] for k in range(K)], argmin=S.index(smin))


@pytest.mark.parametrize("case", [0, 1, 2, 3])
def test_oracle_matches_bruteforce(O, case):
    sc = scenes.scene_cfg0(case)
    if case == 0:
        p = sc.params.with_(K=8, T=5, seed=11)
        obs = sc.obstacles
        x0, U = sc.x0, np.zeros((5, 2))
    elif case == 1:   # off-axle hitch, two obstacles (one moving, one overlapping the vehicle), warm nominal
        p = sc.params.with_(K=6, T=4, seed=2**40 + 3, Lh=0.75, dt=0.25, lam=3.0)
        obs = np.array([[3.0, 0.5, 1.0, -1.0, 0.25], [-5.0, 1.0, 1.5, 0.0, 0.0]], dtype=np.float32).astype(float)
        x0 = np.array([0.5, -0.25, 0.4, -0.9], dtype=np.float32).astype(float)
        U = np.array([[1.0, 0.2], [-0.5, -0.3], [1.9, 0.55], [0.0, 0.0]], dtype=np.float32).astype(float)
    elif case == 3:   # super-ellipse obstacles: a rotated parked car (e = 4) under the trailer's path, a walking pedestrian (e = 2)
        p = sc.params.with_(K=6, T=5, seed=5, dt=0.2)
        obs = sc.obstacles
        x0, U = sc.x0, np.array([[-1.5, 0.1]] * 5, dtype=np.float32).astype(float)
        se = np.array([[-9.0, 2.5, 2.25, 0.9, 0.6, 0.0, 0.0, 4.0], [-3.0, -2.0, 0.4, 0.4, 0.0, 0.3, 1.2, 2.0]], dtype=np.float32).astype(float)
    else:             # large hitch angle and headings near +-pi (wrap paths active)
        p = sc.params.with_(K=5, T=3, seed=77, sigma_v=1.0, sigma_delta=0.5, dt=0.5, hitch_kappa=0.15)   # eq. (18) limit active
        obs = sc.obstacles
        x0 = np.array([1.0, 2.0, 3.0, -2.9], dtype=np.float32).astype(float)
        U = np.array([[-1.0, 0.5]] * 3, dtype=np.float32).astype(float)
    if case != 3:
        se = np.zeros((0, 8))
    n = 4
    ref = brute_force(p, n, x0, sc.goal, obs, U, [tuple(r) for r in se])
    got = O.iteration(p, n, x0, sc.goal, obs, U, superellipses=se)
    assert got["argmin"] == ref["argmin"]
    for k in range(p.K):
        assert abs(got["S"][k] - ref["S"][k]) <= 1e-12 * max(1, abs(ref["S"][k]))
        for c in range(4):
            assert abs(got["XT"][k][c] - ref["XT"][k][c]) <= 1e-12
    for t in range(p.T):
        for c in range(2):
            assert abs(got["U"][t][c] - ref["U"][t][c]) <= 1e-12
