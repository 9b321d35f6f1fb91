"""Pins of the oracle's super-ellipse barrier, eq. (16) of the paper (SURVEY §8(f)
NEXT row 2): values the formula fixes independently of the implementation."""
import math

import numpy as np
import pytest

import scenes

P = scenes.default_params


def test_boundary_inside_outside(O):
    p = P(disc_radius=0.0)
    se = [1.0, -2.0, 2.0, 1.0, 0.0, 0.0, 0.0, 4.0]          # axis-aligned, semi-axes 2 x 1
    o = se[:2]
    for pt, want in [((3.0, -2.0), 0.0), ((-1.0, -2.0), 0.0), ((1.0, -1.0), 0.0), ((1.0, -3.0), 0.0),
                     ((1.0, -2.0), -1.0), ((3.0, -1.0), 1.0), ((5.0, -2.0), 15.0), ((1.0, 0.0), 15.0)]:
        assert O.barrier_se(p, pt, o, se) == pytest.approx(want, abs=1e-12)


def test_hand_worked_rotated(O):
    # theta = 90 deg: x' = dy, y' = -dx.  Point (1, 2), semi-axes (2, 1), no inflation:
    # x' = 2, y' = -1  ->  (2/2)^4 + (1/1)^4 - 1 = 1
    p = P(disc_radius=0.0)
    se = [0.0, 0.0, 2.0, 1.0, math.pi / 2, 0.0, 0.0, 4.0]
    assert O.barrier_se(p, (1.0, 2.0), (0.0, 0.0), se) == pytest.approx(1.0, abs=1e-12)
    # the same point seen by the unrotated obstacle: (1/2)^4 + 2^4 - 1
    se[4] = 0.0
    assert O.barrier_se(p, (1.0, 2.0), (0.0, 0.0), se) == pytest.approx(1 / 16 + 16 - 1, abs=1e-12)


def test_inflation_by_disc_radius(O):
    p = P(disc_radius=1.3)
    r = p.disc_radius
    se = [0.0, 0.0, 2.25, 0.9, 0.3, 0.0, 0.0, 4.0]
    c, s = math.cos(0.3), math.sin(0.3)
    ax, ay = 2.25 + r, 0.9 + r
    assert O.barrier_se(p, (ax * c, ax * s), (0, 0), se) == pytest.approx(0.0, abs=1e-12)      # along the long axis
    assert O.barrier_se(p, (-ay * s, ay * c), (0, 0), se) == pytest.approx(0.0, abs=1e-12)     # along the short axis
    q = 2 ** -0.25                                                                              # the "corner" of e = 4
    assert O.barrier_se(p, (q * ax * c - q * ay * s, q * ax * s + q * ay * c), (0, 0), se) == pytest.approx(0.0, abs=1e-12)


def test_e2_equal_axes_is_the_disc_barrier(O):
    p = P()
    rng = np.random.default_rng(3)
    for _ in range(50):
        c, o = rng.uniform(-20, 20, 2), rng.uniform(-20, 20, 2)
        R, th = rng.uniform(0.3, 2.0), rng.uniform(-math.pi, math.pi)
        se = [o[0], o[1], R, R, th, 0.0, 0.0, 2.0]
        assert O.barrier_se(p, c, o, se) == pytest.approx(O.barrier(p, c, o, R), rel=1e-12, abs=1e-12)


def test_rotation_covariance(O):
    p = P()
    rng = np.random.default_rng(4)
    for _ in range(20):
        o = rng.uniform(-5, 5, 2)
        d = rng.uniform(-6, 6, 2)
        th, phi = rng.uniform(-3, 3, 2)
        se = [o[0], o[1], 2.25, 0.9, th, 0, 0, 4.0]
        h0 = O.barrier_se(p, o + d, o, se)
        rot = np.array([[math.cos(phi), -math.sin(phi)], [math.sin(phi), math.cos(phi)]])
        se2 = list(se)
        se2[4] = th + phi
        assert O.barrier_se(p, o + rot @ d, o, se2) == pytest.approx(h0, rel=1e-11, abs=1e-11)


def test_rollout_with_e2_superellipses_equals_discs(O):
    """A whole iteration with moving circular super-ellipses is bit-identical to the disc path."""
    sc = scenes.scene_cfg2(1)
    p = sc.params.with_(K=64, T=30, n_iter=1)
    U = np.zeros((p.T, 2))
    a = O.iteration(p, 3, sc.x0, sc.goal, sc.obstacles, U)
    se = np.array([[o[0], o[1], o[2], o[2], 0.4 * i, o[3], o[4], 2.0] for i, o in enumerate(sc.obstacles)])
    b = O.iteration(p, 3, sc.x0, sc.goal, np.zeros((0, 5)), U, superellipses=se)
    assert np.abs(a["S"] - b["S"]).max() <= 1e-9 * np.abs(a["S"]).max()
    assert a["argmin"] == b["argmin"] and np.abs(a["U"] - b["U"]).max() <= 1e-10


def test_receding_and_stationary(O):
    p = P(T=10, dt=0.1)
    se = np.array([[0.0, 5.0, 2.25, 0.9, 0.0, 0.0, 0.0, 4.0]])
    # driving away along +x from a car that sits beside the path: h grows, penalty exactly 0
    u = np.tile([1.5, 0.0], (p.T, 1))
    r = O.rollout(p, [8.0, 0.0, 0.0, 0.0], [20, 0, 0, 0], np.zeros((0, 5)), u, 0.5, superellipses=se)
    assert r["pen"] == 0.0
    # standing still inside the inflated car: every step costs alpha |h| per disc inside
    u0 = np.zeros((p.T, 2))
    x_in = [0.0, 5.0, 0.0, 0.0]
    r = O.rollout(p, x_in, [0, 0, 0, 0], np.zeros((0, 5)), u0, 0.25, superellipses=se)
    hs = [O.barrier_se(p, O.disc_centre(p, x_in, j), se[0, :2], se[0]) for j in range(3)]
    want = p.T * 0.25 * sum(-h for h in hs if h < 0)
    assert any(h < 0 for h in hs) and r["pen"] == pytest.approx(want, rel=1e-12)


def test_advance_moves_the_centre_only_and_like_a_disc(O):
    """orc_advance_se: centre += dt * velocity, everything else untouched (hand value), and the same
    displacement the plant step gives a disc obstacle with that velocity (Assumption 2)."""
    p = P(dt=0.25)
    se = np.array([[1.0, -2.0, 2.25, 0.9, 0.7, 0.8, -0.4, 4.0],
                   [5.0, 5.0, 0.4, 0.4, 0.0, 0.0, 0.0, 2.0]])
    out = O.advance_se(p, se)
    want = se.copy()
    want[0, 0] = 1.0 + 0.25 * 0.8      # 1.2
    want[0, 1] = -2.0 + 0.25 * -0.4    # -2.1
    assert np.array_equal(out, want)
    assert np.array_equal(se[0, :2], [1.0, -2.0])          # the input is not modified
    discs = np.array([[1.0, -2.0, 0.5, 0.8, -0.4], [5.0, 5.0, 0.4, 0.0, 0.0]])
    _, discs_next = O.plant_step(p, np.zeros(4), np.zeros(2), discs)
    assert np.array_equal(out[:, :2], discs_next[:, :2])
    # n steps of advance == the position the rollout pairs with step n: o(n) = o(0) + n dt vel
    cur = se
    for _ in range(7):
        cur = O.advance_se(p, cur)
    assert cur[0, 0] == pytest.approx(1.0 + 7 * 0.25 * 0.8, rel=1e-15)
    assert cur[0, 1] == pytest.approx(-2.0 + 7 * 0.25 * -0.4, rel=1e-15)
