"""Pins of the CPU oracle against what the paper and the mathematics fix (SURVEY.md §8(c) "Pins").

None of these re-types the oracle's own formula: they are published known-answer vectors, closed
forms of the continuous/discrete kinematics, hand-worked numbers, invariants of the softmax
update, and an independent 50-digit brute force (tests/test_oracle_bruteforce.py).  A dropped
term, a wrong sign, a transposed index or a shifted time index fails at least one of them."""
import math
import os
import re

import numpy as np
import pytest

import scenes

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def P(**kw):
    return scenes.default_params(**kw)


# ------------------------------------------------------------------------------------------
# Philox integers
# ------------------------------------------------------------------------------------------
def test_philox_known_answers(O):
    n = 0
    for line in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(x, 16) for x in line.split()]
        assert O.philox(w[0:4], w[4:6]) == tuple(w[6:10])
        n += 1
    assert n == 3


def test_philox_constants_match_curand_header(O):
    """The toolkit's own Philox header must carry the multipliers / Weyl constants that reproduce
    the KATs: a generator with those constants swapped (M0<->M1) fails the KAT above; this test
    documents where the constants come from on this box."""
    hdr = "/usr/local/cuda/include/curand_philox4x32_x.h"
    if not os.path.exists(hdr):
        pytest.skip("CUDA toolkit header not present")
    txt = open(hdr).read()
    consts = {m.group(1): int(m.group(2), 16)
              for m in re.finditer(r"#define\s+(PHILOX_\w+)\s+\(?0x([0-9A-Fa-f]+)", txt)}
    assert consts["PHILOX_M4x32_0"] == 0xD2511F53
    assert consts["PHILOX_M4x32_1"] == 0xCD9E8D57
    assert consts["PHILOX_W32_0"] == 0x9E3779B9
    assert consts["PHILOX_W32_1"] == 0xBB67AE85


def test_philox_counter_and_key_sensitivity(O):
    """Every counter word and key word matters (a mixed-up word order would alias streams)."""
    base = O.philox((1, 2, 3, 4), (5, 6))
    seen = {base}
    for i in range(4):
        c = [1, 2, 3, 4]
        c[i] += 1
        seen.add(O.philox(c, (5, 6)))
    seen.add(O.philox((1, 2, 3, 4), (6, 6)))
    seen.add(O.philox((1, 2, 3, 4), (5, 7)))
    assert len(seen) == 7
    # swapping two counter words is not a symmetry
    assert O.philox((2, 1, 3, 4), (5, 6)) != base


def test_noise_stream_layout(O):
    """Counter layout (t, n, k, tag) and key (lo32(seed), hi32(seed)) -- DESIGN.md reading 5/7.
    orc_normals / orc_alpha must consume exactly those blocks."""
    seed, n, k = 0x1234567890ABCDEF, 7, 4242
    for t in (16, 17, 0, 1):                       # one block per pair of steps (reading 6)
        w = O.philox((t >> 1, n, k, 0), (seed & 0xFFFFFFFF, seed >> 32))
        wa, wb = (w[2], w[3]) if t & 1 else (w[0], w[1])
        u1 = 1.0 - (wa >> 9) / 2.0**23
        u2 = (wb >> 9) / 2.0**23
        r = math.sqrt(-2.0 * math.log(u1))
        z = O.normals(seed, n, k, t)
        assert z[0] == pytest.approx(r * math.cos(2 * math.pi * u2), rel=1e-14, abs=1e-15)
        assert z[1] == pytest.approx(r * math.sin(2 * math.pi * u2), rel=1e-14, abs=1e-15)
    assert not np.allclose(O.normals(seed, n, k, 16), O.normals(seed, n, k, 17))
    p = P(seed=seed, alpha_lo=0.25, alpha_hi=0.75)
    wa = O.philox((0, n, k, 1), (seed & 0xFFFFFFFF, seed >> 32))
    assert O.alpha(p, n, k) == pytest.approx(0.25 + 0.5 * ((wa[0] >> 9) / 2.0**23), rel=1e-15)


# ------------------------------------------------------------------------------------------
# uniforms / normals
# ------------------------------------------------------------------------------------------
def test_uniform_exact_and_range(O):
    assert O.uniform(0) == 0.0
    assert O.uniform(0x1FF) == 0.0                      # low 9 bits dropped
    assert O.uniform(0x200) == 2.0**-23
    assert O.uniform(0xFFFFFFFF) == 1.0 - 2.0**-23       # < 1
    rng = np.random.default_rng(0)
    for w in rng.integers(0, 2**32, size=200):
        u = O.uniform(int(w))
        assert 0.0 <= u < 1.0
        assert float(np.float32(u)) == u                 # exactly representable in fp32
        assert float(np.float32(1.0 - u)) == 1.0 - u     # and so is u1 = 1 - f


def test_normal_moments(O):
    """Box-Muller on the Philox stream: standard normal, the two channels uncorrelated."""
    n_s, n_t = 2500, 100
    z = np.array([O.normals(12345, 3, k, t) for k in range(n_s) for t in range(n_t)])
    n = z.shape[0]
    assert abs(z[:, 0].mean()) < 4 / math.sqrt(n)
    assert abs(z[:, 1].mean()) < 4 / math.sqrt(n)
    assert abs(z[:, 0].var() - 1) < 0.01
    assert abs(z[:, 1].var() - 1) < 0.01
    assert abs(np.mean(z[:, 0] * z[:, 1])) < 4 / math.sqrt(n)
    # 4th moment of a standard normal is 3 (a uniform or a mis-scaled radius fails this)
    assert abs(np.mean(z[:, 0] ** 4) - 3) < 0.1
    assert np.abs(z).max() < 5.65                        # sqrt(-2 ln 2^-23) = 5.6467


def test_alpha_range_and_mean(O):
    p = P(seed=9)
    a = np.array([O.alpha(p, 0, k) for k in range(20000)])
    assert a.min() >= p.alpha_lo and a.max() < p.alpha_hi
    assert abs(a.mean() - 0.5 * (p.alpha_lo + p.alpha_hi)) < 4 * (p.alpha_hi - p.alpha_lo) / math.sqrt(12 * a.size)
    # alpha is a different stream from the control noise of the same (n, k)
    assert O.alpha(p, 0, 5) != O.alpha(p, 1, 5)


# ------------------------------------------------------------------------------------------
# kinematics: closed forms (eq. 6 reduced)
# ------------------------------------------------------------------------------------------
def roll(O, p, x, v, d, n):
    xs = [np.array(x, dtype=float)]
    for _ in range(n):
        xs.append(O.kinematic_step(p, xs[-1], v, d))
    return np.array(xs)


def test_straight_line(O):
    p = P(dt=0.125)
    psi = 0.7
    xs = roll(O, p, [1.0, -2.0, psi, psi], 1.5, 0.0, 40)
    T = 40
    assert xs[-1, 0] == pytest.approx(1.0 + T * 0.125 * 1.5 * math.cos(psi), rel=1e-13)
    assert xs[-1, 1] == pytest.approx(-2.0 + T * 0.125 * 1.5 * math.sin(psi), rel=1e-13)
    assert np.all(xs[:, 2] == psi) and np.all(xs[:, 3] == psi)   # headings exactly constant
    # reversing moves the other way
    xr = roll(O, p, [0, 0, 0, 0], -1.0, 0.0, 8)
    assert xr[-1, 0] == pytest.approx(-1.0) and xr[-1, 1] == 0.0


def test_euler_circle_radius(O):
    """Constant (v, delta): the Euler vertices lie exactly on a circle of radius
    R_E = |v| dt / (2 sin(|dtheta|/2)), dtheta = dt v tan(delta)/L1, which -> L1/tan(delta)."""
    p = P(dt=0.1, L1=4.0)
    v, d = 1.5, 0.3
    xs = roll(O, p, [0, 0, 0.2, 0.2], v, d, 300)
    dth = p.dt * v * math.tan(d) / p.L1
    R_E = abs(v) * p.dt / (2 * math.sin(abs(dth) / 2))
    # circumcentre from three vertices, then all vertices equidistant
    (ax, ay), (bx, by), (cx, cy) = xs[0, :2], xs[100, :2], xs[200, :2]
    dd = 2 * (ax * (by - cy) + bx * (cy - ay) + cx * (ay - by))
    ux = ((ax**2 + ay**2) * (by - cy) + (bx**2 + by**2) * (cy - ay) + (cx**2 + cy**2) * (ay - by)) / dd
    uy = ((ax**2 + ay**2) * (cx - bx) + (bx**2 + by**2) * (ax - cx) + (cx**2 + cy**2) * (bx - ax)) / dd
    r = np.hypot(xs[:, 0] - ux, xs[:, 1] - uy)
    assert np.max(np.abs(r - R_E)) < 1e-10
    assert R_E == pytest.approx(p.L1 / math.tan(d), rel=1e-4)       # NS: radius L1 / tan(delta)
    assert xs[-1, 2] == pytest.approx(0.2 + 300 * dth, rel=1e-12)   # heading rate v tan(delta)/L1
    # left turn for positive steer when driving forward: centre is to the left of the heading
    left = np.array([-math.sin(0.2), math.cos(0.2)])
    assert np.dot([ux - xs[0, 0], uy - xs[0, 1]], left) > 0


def test_hitch_relaxation_closed_form(O):
    """delta = 0, v > 0: beta = psi1 - psi2 obeys beta' = -(v/L2) sin(beta), solution
    tan(beta/2) = tan(beta0/2) exp(-v t / L2).  Euler converges at O(dt); v < 0 diverges."""
    beta0, v, t_end = 0.8, 2.0, 4.0
    errs = []
    for dt in (0.1, 0.05, 0.025):
        p = P(dt=dt, L2=8.0)
        n = round(t_end / p.dt)
        xs = roll(O, p, [0, 0, beta0, 0.0], v, 0.0, n)
        beta = xs[-1, 2] - xs[-1, 3]
        exact = 2 * math.atan(math.tan(beta0 / 2) * math.exp(-v * n * p.dt / p.L2))
        errs.append(beta - exact)
    assert abs(errs[0]) < 5e-3
    assert errs[0] / errs[1] == pytest.approx(2.0, rel=0.1)
    assert errs[1] / errs[2] == pytest.approx(2.0, rel=0.1)
    # reversing: the hitch angle grows (jackknife instability)
    p = P(dt=0.05)
    xs = roll(O, p, [0, 0, 0.1, 0.0], -2.0, 0.0, 80)
    assert abs(xs[-1, 2] - xs[-1, 3]) > 0.1 * 2


def test_steady_turn_fixed_point(O):
    """Lh = 0: beta* = asin(L2 tan(delta) / L1) is an exact fixed point of the Euler map."""
    p = P(dt=0.05, L1=4.0, L2=8.0, Lh=0.0)
    d, v = 0.3, 1.0
    beta = math.asin(p.L2 * math.tan(d) / p.L1)
    xs = roll(O, p, [0, 0, beta, 0.0], v, d, 400)
    assert np.max(np.abs((xs[:, 2] - xs[:, 3]) - beta)) < 1e-12


def test_steady_turn_with_hitch_offset(O):
    """Lh != 0: steady state solves sin(b) - (Lh/L1) tan(d) cos(b) = L2 tan(d)/L1, i.e.
    b = asin(c / sqrt(1+a^2)) + atan(a), a = (Lh/L1) tan d, c = L2 tan d / L1.  Pins the sign
    and the Lh/L1 factor of the off-axle hitch term of eq. (6)."""
    p = P(dt=0.05, L1=3.25, L2=3.0, Lh=1.125)
    d, v = 0.25, 1.0
    a = (p.Lh / p.L1) * math.tan(d)
    c = p.L2 * math.tan(d) / p.L1
    beta = math.asin(c / math.sqrt(1 + a * a)) + math.atan(a)
    xs = roll(O, p, [0, 0, beta, 0.0], v, d, 400)
    assert np.max(np.abs((xs[:, 2] - xs[:, 3]) - beta)) < 1e-12
    # and one hand-worked step: x=(0,0,pi/2,0), v=2, delta=atan(0.5), dt=0.05
    # beta = pi/2: sin=1, cos=0  => psi2' = 0 + 0.05*(2/3)*(1 - 0) = 1/30; psi1' = pi/2 + 0.05*(2/3.25)*0.5
    xn = O.kinematic_step(p, [0, 0, math.pi / 2, 0.0], 2.0, math.atan(0.5))
    assert xn[3] == pytest.approx(p.dt * 2.0 / 3.0, rel=1e-12)
    assert xn[2] == pytest.approx(math.pi / 2 + p.dt * (2 / 3.25) * 0.5, rel=1e-12)
    assert xn[0] == pytest.approx(0.0, abs=1e-15) and xn[1] == pytest.approx(p.dt * 2.0, rel=1e-12)


def test_euler_uses_old_state_everywhere(O):
    """Every right-hand side at step k: psi2's update must see psi1_k, and
    x, y must see psi1_k (a semi-implicit variant fails)."""
    p = P(dt=0.5, L1=4.0, L2=8.0)
    x = [0.0, 0.0, math.pi / 2, 0.0]
    xn = O.kinematic_step(p, x, 1.0, math.atan(1.0))      # tan(delta) = 1
    assert xn[0] == pytest.approx(0.0, abs=1e-16)          # cos(pi/2) = 0, not cos(psi1')
    assert xn[1] == pytest.approx(0.5)
    assert xn[2] == pytest.approx(math.pi / 2 + 0.5 * 0.25)
    assert xn[3] == pytest.approx(0.5 * (1 / 8.0) * math.sin(math.pi / 2))


# ------------------------------------------------------------------------------------------
# barrier, hinge penalty
# ------------------------------------------------------------------------------------------
def test_barrier_values(O):
    p = P(disc_radius=1.25)
    R = 0.75                                    # rho = 2
    assert O.barrier(p, [2.0, 0.0], [0.0, 0.0], R) == 0.0           # on the inflated circle
    assert O.barrier(p, [0.0, 4.0], [0.0, 0.0], R) == 3.0           # at distance 2 rho
    assert O.barrier(p, [1.0, 1.0], [1.0, 1.0], R) == -1.0          # at the centre
    assert O.barrier(p, [3.0, 5.0], [0.0, 1.0], R) == 25.0 / 4 - 1  # offsets in both axes


def test_disc_centres(O):
    p = P(Lh=0.5, discs=((0, 2.0), (1, -2.0), (1, -6.0)))
    x = [1.0, 2.0, math.pi / 2, math.pi]        # tractor points +y, trailer points -x
    # hitch point = (1, 2 - 0.5) = (1, 1.5)
    np.testing.assert_allclose(O.disc_centre(p, x, 0), [1.0, 3.5], atol=1e-15)   # +2 along +y
    np.testing.assert_allclose(O.disc_centre(p, x, 1), [3.0, 1.5], atol=1e-15)   # -2 along -x => +x
    np.testing.assert_allclose(O.disc_centre(p, x, 2), [7.0, 1.5], atol=1e-15)


def test_hand_worked_barrier_rate_step(O):
    """x0 = origin, heading 0, one disc at the tractor (+2 m), v = 1, dt = 0.125, obstacle at
    (5, 0) with R = 0.75, r_v = 1.25 (rho = 2):
        h_0 = (5-2)^2/4 - 1 = 1.25;   after the step the disc is at 2.125: h_1 = 2.875^2/4 - 1
        = 1.06640625.   alpha = 0.125: (1-alpha) h_0 - h_1 = 1.09375 - 1.06640625 = 0.02734375 > 0.
        alpha = 0.5   : 0.625 - 1.0664 < 0  => no penalty."""
    p = P(T=1, dt=0.125, disc_radius=1.25, discs=((0, 2.0),), w_pos=0.0, w_head=0.0, w_v=0.0,
          w_delta=0.0, w_hitch=0.0, w_term=0.0, w_bar=1000.0)
    obs = [[5.0, 0.0, 0.75, 0.0, 0.0]]
    r = O.rollout(p, [0, 0, 0, 0], [0, 0, 0, 0], obs, [[1.0, 0.0]], 0.125)
    assert r["pen"] == 0.02734375
    assert r["S"] == 27.34375
    r = O.rollout(p, [0, 0, 0, 0], [0, 0, 0, 0], obs, [[1.0, 0.0]], 0.5)
    assert r["pen"] == 0.0 and r["S"] == 0.0


def test_receding_sample_has_zero_penalty(O):
    """NS invariant: outside every disc with h increasing => exactly zero barrier penalty."""
    p = P(T=30, dt=0.1)
    obs = [[6.0, 0.5, 1.0, 0.0, 0.0], [8.0, -3.0, 0.5, 0.0, 0.0]]
    u = np.tile([-1.5, 0.0], (30, 1))           # reversing straight away from both obstacles
    for a in (0.1, 0.5, 1.0):
        r = O.rollout(p, [0, 0, 0, 0], [-10, 0, 0, 0], obs, u, a, want_traj=True)
        assert r["pen"] == 0.0
    # approaching fast with small alpha is penalised
    r = O.rollout(p, [0, 0, 0, 0], [-10, 0, 0, 0], obs, -u, 0.1)
    assert r["pen"] > 0.0


def test_stationary_inside_disc(O):
    """v = 0 inside a disc: h constant < 0, each step costs alpha |h| per (obstacle, disc)."""
    p = P(T=7, dt=0.1, disc_radius=1.25, discs=((0, 2.0),))
    obs = [[3.0, 0.0, 0.75, 0.0, 0.0]]          # disc centre (2,0) is 1 m from it: h = 1/4 - 1
    u = np.zeros((7, 2))
    r = O.rollout(p, [0, 0, 0, 0], [0, 0, 0, 0], obs, u, 0.4)
    assert r["pen"] == pytest.approx(7 * 0.4 * 0.75, rel=1e-14)


def test_moving_obstacle_pairs_with_time(O):
    """h_{t+1} uses (x_{t+1}, o(t+1)): an obstacle moving with the vehicle keeps h constant
    (=> no penalty outside); a static reading of the same obstacle would change h."""
    p = P(T=10, dt=0.125, disc_radius=1.25, discs=((0, 2.0),))
    u = np.tile([1.0, 0.0], (10, 1))
    obs_moving = [[6.0, 0.0, 0.75, 1.0, 0.0]]   # same velocity as the vehicle, 4 m ahead of disc
    r = O.rollout(p, [0, 0, 0, 0], [0, 0, 0, 0], obs_moving, u, 0.1)
    assert r["pen"] == 0.0                       # h == 3 throughout, (1-a)*3 - 3 < 0
    obs_static = [[6.0, 0.0, 0.75, 0.0, 0.0]]
    r2 = O.rollout(p, [0, 0, 0, 0], [0, 0, 0, 0], obs_static, u, 0.1)
    assert r2["pen"] > 0.0
    # obstacle running into a parked vehicle from behind the disc
    obs_hit = [[-2.0, 0.0, 0.75, 2.0, 0.0]]
    r3 = O.rollout(p, [0, 0, 0, 0], [0, 0, 0, 0], obs_hit, np.zeros((10, 2)), 0.1)
    # by hand: o(t) = -2 + 0.25 t, c = 2: h_t = (4 - 0.25 t)^2/4 - 1
    h = [(4 - 0.25 * t) ** 2 / 4 - 1 for t in range(11)]
    pen = sum(max(0.0, 0.9 * h[t] - h[t + 1]) for t in range(10))
    assert r3["pen"] == pytest.approx(pen, rel=1e-13)


# ------------------------------------------------------------------------------------------
# cost terms one at a time (PAPER.md:135 structure; terms of CFG0)
# ------------------------------------------------------------------------------------------
ZERO_W = dict(w_pos=0.0, w_head=0.0, w_v=0.0, w_delta=0.0, w_hitch=0.0, w_term=0.0, w_bar=0.0)


def test_cost_terms_closed_form(O):
    T, dt, v = 8, 0.25, 1.0
    u = np.tile([v, 0.0], (T, 1))
    x0, goal = [0, 0, 0, 0], [3.0, 1.0, 0.0, 0.0]
    # position term only: stage cost on x_{t+1}, t = 0..T-1  (reading 3)
    p = P(T=T, dt=dt, **{**ZERO_W, "w_pos": 0.5})
    S = O.rollout(p, x0, goal, [], u, 0.5)["S"]
    assert S == pytest.approx(sum(0.5 * ((dt * v * (t + 1) - 3.0) ** 2 + 1.0) for t in range(T)))
    # terminal only: w_term * G(x_T) with G's own weights
    p = P(T=T, dt=dt, **{**ZERO_W, "w_pos": 0.5, "w_term": 4.0})
    S2 = O.rollout(p, x0, goal, [], u, 0.5)["S"]
    assert S2 - S == pytest.approx(4.0 * 0.5 * ((dt * v * T - 3.0) ** 2 + 1.0))
    # effort on the applied control
    p = P(T=T, dt=dt, **{**ZERO_W, "w_v": 0.25, "w_delta": 2.0})
    uu = np.tile([1.5, -0.5], (T, 1))
    assert O.rollout(p, x0, goal, [], uu, 0.5)["S"] == pytest.approx(T * (0.25 * 2.25 + 2.0 * 0.25))
    # heading with wrap: psi = -pi + 0.1 vs goal pi - 0.1 is an error of 0.2, not 2 pi - 0.2
    p = P(T=1, dt=dt, **{**ZERO_W, "w_head": 1.0})
    S = O.rollout(p, [0, 0, -math.pi + 0.1, -math.pi + 0.1], [0, 0, math.pi - 0.1, math.pi - 0.1],
                  [], np.zeros((1, 2)), 0.5)["S"]
    assert S == pytest.approx(2 * 0.2**2, rel=1e-12)
    # hitch: squared hinge beyond hitch_max, v = 0 keeps the angle
    p = P(T=5, dt=dt, **{**ZERO_W, "w_hitch": 10.0, "hitch_max": 1.25})
    S = O.rollout(p, [0, 0, 1.5, 0.0], goal, [], np.zeros((5, 2)), 0.5)["S"]
    assert S == pytest.approx(5 * 10.0 * 0.25**2)
    S = O.rollout(p, [0, 0, 0.0, 1.5], goal, [], np.zeros((5, 2)), 0.5)["S"]      # |.|
    assert S == pytest.approx(5 * 10.0 * 0.25**2)
    S = O.rollout(p, [0, 0, 1.0, 0.0], goal, [], np.zeros((5, 2)), 0.5)["S"]      # below the limit
    assert S == 0.0
    # hitch angle is wrapped: psi1 - psi2 = 2 pi - 0.1 is a hitch angle of 0.1
    S = O.rollout(p, [0, 0, math.pi - 0.05, -math.pi + 0.05], goal, [], np.zeros((5, 2)), 0.5)["S"]
    assert S == 0.0


def test_wrap(O):
    assert O.wrap(0.3) == 0.3
    assert O.wrap(2 * math.pi + 0.3) == pytest.approx(0.3, abs=1e-15)
    assert O.wrap(-math.pi - 0.1) == pytest.approx(math.pi - 0.1, abs=1e-15)
    assert abs(O.wrap(7 * math.pi)) == pytest.approx(math.pi)


# ------------------------------------------------------------------------------------------
# weights / update / shift
# ------------------------------------------------------------------------------------------
def test_weights_positive_sum_to_one_shift_and_permutation_invariant(O):
    rng = np.random.default_rng(3)
    K, T = 64, 6
    S = rng.uniform(100, 130, K)
    u = rng.normal(size=(K, T, 2))
    r = O.weights_update(S, u, 1.0)
    w = r["w"] / r["eta"]
    assert np.all(w > 0) and w.sum() == pytest.approx(1.0, rel=1e-14)
    assert r["w"][r["argmin"]] == 1.0 and r["argmin"] == int(np.argmin(S))
    # textbook definition of the update (softmax average), written with library routines
    ref = np.einsum("k,ktc->tc", np.exp(-(S - S.min())) / np.exp(-(S - S.min())).sum(), u)
    np.testing.assert_allclose(r["U"], ref, rtol=1e-13, atol=1e-15)
    # adding a constant to every cost changes nothing (the min-shift).  The
    # constant is a power of two small enough that S + c stays exact to ~1e-13
    r2 = O.weights_update(S + 64.0, u, 1.0)
    np.testing.assert_allclose(r2["U"], r["U"], rtol=1e-11)
    # permuting the samples changes nothing
    perm = rng.permutation(K)
    r3 = O.weights_update(S[perm], u[perm], 1.0)
    np.testing.assert_allclose(r3["U"], r["U"], rtol=1e-12)
    assert perm[r3["argmin"]] == r["argmin"]
    # gap = second smallest - smallest
    ss = np.sort(S)
    assert r["gap"] == pytest.approx(ss[1] - ss[0], rel=1e-12)


def test_lambda_limits(O):
    rng = np.random.default_rng(4)
    K, T = 32, 5
    S = rng.uniform(0, 50, K)
    u = rng.normal(size=(K, T, 2))
    r = O.weights_update(S, u, 1e-6)                     # lambda -> 0 selects the argmin sample
    assert np.array_equal(r["U"], u[np.argmin(S)])
    assert np.all(np.isfinite(r["U"]))
    r = O.weights_update(S, u, 1e12)                     # lambda -> inf: plain mean
    np.testing.assert_allclose(r["U"], u.mean(axis=0), rtol=1e-9, atol=1e-12)


def test_ties_and_nonfinite(O):
    u = np.arange(4 * 2 * 2, dtype=float).reshape(4, 2, 2)
    r = O.weights_update([5.0, 3.0, 3.0, 9.0], u, 1e-6)
    assert r["argmin"] == 1                              # lowest index among ties
    np.testing.assert_allclose(r["U"], 0.5 * (u[1] + u[2]))   # ties share the mass equally
    r = O.weights_update([np.inf, 3.0, np.nan, 9.0], u, 1e-6)
    assert r["argmin"] == 1 and r["nonfinite"] == 2
    np.testing.assert_allclose(r["U"], u[1])
    r = O.weights_update([np.inf, np.nan], u[:2], 1.0)
    assert r["argmin"] == -1 and r["nonfinite"] == 2


def test_iteration_fixed_point_and_mean(O):
    sc = scenes.scene_cfg0(0)
    # sigma = 0: every sample equals the nominal, U is a fixed point of the update
    p = sc.params.with_(K=16, T=10, sigma_v=0.0, sigma_delta=0.0)
    U0 = np.tile([0.75, 0.125], (10, 1))
    r = O.iteration(p, 0, sc.x0, sc.goal, sc.obstacles, U0, want_samples=True)
    assert np.array_equal(r["U"], U0)
    assert np.all(r["S"] == r["S"][0])
    # all cost weights zero: S = 0 for all k, update = plain sample mean of the clamped controls
    p = sc.params.with_(K=64, T=10, **ZERO_W)
    r = O.iteration(p, 5, sc.x0, sc.goal, sc.obstacles, U0, want_samples=True)
    assert np.all(r["S"] == 0.0)
    np.testing.assert_allclose(r["U"], r["u"].mean(axis=0), rtol=1e-13)
    # the update is a convex combination of clamped controls: stays inside the box
    p = sc.params.with_(K=64, T=10, sigma_v=5.0, sigma_delta=5.0)
    r = O.iteration(p, 0, sc.x0, sc.goal, sc.obstacles, U0, want_samples=True)
    assert r["u"][..., 0].min() >= p.v_min and r["u"][..., 0].max() <= p.v_max
    assert r["u"][..., 1].min() >= p.delta_min and r["u"][..., 1].max() <= p.delta_max
    assert (r["u"][..., 0] == p.v_max).any() and (r["u"][..., 1] == p.delta_min).any()
    assert r["U"][:, 0].min() >= p.v_min and r["U"][:, 0].max() <= p.v_max
    # the sampled controls are u_nom + sigma z with the documented stream
    p = sc.params.with_(K=8, T=10)
    r = O.iteration(p, 2, sc.x0, sc.goal, sc.obstacles, U0, want_samples=True)
    z = O.normals(p.seed, 2, 3, 7)
    assert r["u"][3, 7, 0] == pytest.approx(np.clip(0.75 + p.sigma_v * z[0], p.v_min, p.v_max), rel=1e-15)
    assert r["u"][3, 7, 1] == pytest.approx(np.clip(0.125 + p.sigma_delta * z[1], p.delta_min, p.delta_max), rel=1e-15)


def test_iteration_counter_gives_fresh_noise_and_threads_are_bit_identical(O):
    sc = scenes.scene_cfg0(1)
    p = sc.params.with_(K=200, T=12)
    U0 = np.zeros((12, 2))
    a = O.iteration(p, 0, sc.x0, sc.goal, sc.obstacles, U0)
    b = O.iteration(p, 1, sc.x0, sc.goal, sc.obstacles, U0)
    assert not np.array_equal(a["S"], b["S"])
    c = O.iteration(p, 0, sc.x0, sc.goal, sc.obstacles, U0, n_threads=3)
    for key in ("U", "S", "XT"):
        assert np.array_equal(a[key], c[key])
    assert a["argmin"] == c["argmin"]


def test_shift_and_plant(O):
    U = np.arange(10, dtype=float).reshape(5, 2)
    Us = O.shift(U)
    np.testing.assert_array_equal(Us[:4], U[1:])
    np.testing.assert_array_equal(Us[4], U[4])            # tail duplicated, not zero-filled
    p = P(dt=0.5)
    obs = [[1.0, 2.0, 0.5, 0.25, -0.5]]
    x, ob = O.plant_step(p, [0, 0, math.pi - 0.01, 0.0], [2.0, math.atan(1.0)], obs)
    # psi1' = pi - 0.01 + 0.5*(2/4)*1 = pi + 0.24 -> wrapped to -pi + 0.24
    assert x[2] == pytest.approx(-math.pi + 0.24, abs=1e-12)
    assert x[0] == pytest.approx(0.5 * 2.0 * math.cos(math.pi - 0.01))
    np.testing.assert_allclose(ob[0], [1.125, 1.75, 0.5, 0.25, -0.5])


def test_velocity_dependent_hitch_limit(O):
    """Eq. (18): the hitch hinge starts at hitch_max - kappa |v|.  One step with
    delta = 0 from a hitch angle of 1.0 rad: psi1 stays, psi2 moves by dt (v / L2) sin(beta)."""
    p = P(T=1, dt=0.1, w_pos=0.0, w_head=0.0, w_v=0.0, w_delta=0.0, w_term=0.0, w_hitch=10.0, hitch_max=1.2)
    x0 = [0.0, 0.0, 1.0, 0.0]
    for v in (2.0, -2.0, 0.5):
        beta1 = 1.0 - p.dt * (v / p.L2) * math.sin(1.0)              # hitch angle after the step (fp32-rounded dt)
        for kappa in (0.0, 0.05, 0.2):
            pk = p.with_(hitch_kappa=kappa)
            r = O.rollout(pk, x0, [0, 0, 0, 0], np.zeros((0, 5)), [[v, 0.0]], 0.5)
            lim = pk.hitch_max - pk.hitch_kappa * abs(v)              # parameters are fp32-rounded doubles
            want = pk.w_hitch * max(0.0, abs(beta1) - lim) ** 2
            assert r["S"] == pytest.approx(want, rel=1e-9, abs=1e-12), (v, kappa)
    # kappa = 0.2, |v| = 2: limit 0.8 < 0.9...: active; kappa = 0: inactive
    assert O.rollout(p.with_(hitch_kappa=0.2), x0, [0, 0, 0, 0], np.zeros((0, 5)), [[2.0, 0.0]], 0.5)["S"] > 0
    assert O.rollout(p, x0, [0, 0, 0, 0], np.zeros((0, 5)), [[2.0, 0.0]], 0.5)["S"] == 0.0
