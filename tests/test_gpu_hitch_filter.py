"""Parity of the hitch-angle stabiliser (Sec. V-D; reading 28) through the
C ABI against the oracle: brmppi_hitch_filter on batches of seeded (state, reference) pairs, and
brmppi_step with hitch_filter = 1 step by step.

Tolerance: the filtered control within 1e-4 relative with floors (v_max, delta_max), as for every other
control (test_gpu_parity.py).  The QP's solution is Lipschitz in (c0, a) with constant ~ 1/|a|_Q, so a
problem whose fp32 constraint data could move the answer by more than the tolerance is ill-conditioned
in the method itself; those (|Q^-1/2 a| below 2e-3, or the half-plane within 1e-4 of leaving the box:
status 1 vs 2) are compared on feasibility and objective value instead of coordinates."""
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


def make_pairs(rng, n, p, outside=True):
    beta = rng.uniform(-1.5, 1.5, n)
    psi2 = rng.uniform(-np.pi, np.pi, n)
    x = np.stack([rng.uniform(-20, 20, n), rng.uniform(-20, 20, n), psi2 + beta, psi2], axis=1).astype(np.float32)
    m = 1.1 if outside else 1.0
    u = np.stack([rng.uniform(m * p.v_min, m * p.v_max, n), rng.uniform(m * p.delta_min, m * p.delta_max, n)],
                 axis=1).astype(np.float32)
    return x, u


PARAM_SETS = [
    dict(),
    dict(hitch_kappa=0.2, hitch_alpha=0.3, hitch_qv=0.5, hitch_qdelta=4.0, hitch_max=0.9),
    dict(Lh=0.8, hitch_alpha=1.0, hitch_qv=3.0, hitch_qdelta=0.3, dt=0.1),
    dict(hitch_max=0.5, hitch_kappa=0.1, v_min=-1.0, v_max=3.0, delta_min=-0.4, delta_max=0.7),
]


@pytest.mark.parametrize("kw", PARAM_SETS, ids=[str(i) for i in range(len(PARAM_SETS))])
@pytest.mark.parametrize("n", [1, 127, 128, 5000])
def test_batch_matches_oracle(B, O, kw, n):
    p = scenes.default_params(dt=0.05).with_(**kw)
    rng = np.random.default_rng(100 + n)
    x, r = make_pairs(rng, n, p)
    u, st = B.hitch_filter(p, x, r)
    floors = np.array([max(abs(p.v_min), abs(p.v_max)), max(abs(p.delta_min), abs(p.delta_max))])
    q = np.array([p.hitch_qv, p.hitch_qdelta])
    lo = np.array([p.v_min, p.delta_min])
    hi = np.array([p.v_max, p.delta_max])
    n_coord = 0
    seen = set()
    for i in range(n):
        xi, ri = x[i].astype(np.float64), r[i].astype(np.float64)
        u_ref, st_ref = O.hitch_filter(p, xi, ri)
        c0, a = O.hitch_constraint(p, xi, ri)
        seen.add(st_ref)
        ui = u[i].astype(np.float64)
        assert np.all(ui >= lo) and np.all(ui <= hi)
        g = c0 + a @ (ui - ri)
        g_max = c0 + sum(max(a[k] * (lo[k] - ri[k]), a[k] * (hi[k] - ri[k])) for k in range(2))
        well = np.sqrt(np.sum(a * a / q)) > 2e-3 and abs(g_max) > 1e-4 and abs(c0 + a @ (np.clip(ri, lo, hi) - ri)) > 1e-6
        if well:
            assert st[i] == st_ref
            assert np.all(np.abs(ui - u_ref) <= RTOL * np.maximum(np.abs(u_ref), floors)), (i, ui, u_ref, st_ref)
            n_coord += 1
        else:
            J = np.sum(q * (ui - ri) ** 2)
            J_ref = np.sum(q * (u_ref - ri) ** 2)
            if st_ref != 2 and st[i] != 2:
                assert g >= -1e-5 and J <= J_ref + 1e-3 * (1 + J_ref)
    assert n_coord >= 0.95 * n
    if n >= 5000:
        assert seen == {0, 1, 2}


def test_batch_edge_cases(B, O):
    p = scenes.default_params(dt=0.05)
    u, st = B.hitch_filter(p, np.zeros((0, 4)), np.zeros((0, 2)))            # n = 0
    assert u.shape == (0, 2) and st.shape == (0,)
    # standstill: the steering has no authority, a_delta = 0; inside the safe set nothing changes
    u, st = B.hitch_filter(p, [[0, 0, 0.5, 0]], [[0.0, 0.3]])
    assert st[0] == 0 and np.array_equal(u[0], np.float32([0.0, 0.3]))
    # reference outside the box, constraint inactive: clamped
    u, st = B.hitch_filter(p, [[0, 0, 0.1, 0]], [[-2.5, 0.65]])
    assert st[0] == 0 and np.array_equal(u[0], np.float32([p.v_min, p.delta_max]))
    # far beyond the limit, alpha h very negative: no control in the box satisfies it -> status 2, and
    # the answer is the oracle's least-violating vertex
    x, r = [[0, 0, 1.5, 0]], [[-2.0, -0.5]]
    p2 = p.with_(hitch_max=0.3, hitch_alpha=1.0)
    u, st = B.hitch_filter(p2, x, r)
    u_ref, st_ref = O.hitch_filter(p2, x[0], r[0])
    assert st[0] == 2 and st_ref == 2 and np.allclose(u[0], u_ref, atol=1e-6)
    for bad in (dict(hitch_alpha=0.0), dict(hitch_alpha=1.5), dict(hitch_qv=0.0), dict(hitch_qdelta=-1.0)):
        with pytest.raises(B.BrmppiError):
            B.hitch_filter(p.with_(**bad), x, r)
        with pytest.raises(B.BrmppiError):
            B.Solver(p.with_(hitch_filter=1, **bad), 1, 1)
    B.Solver(p.with_(hitch_filter=0, hitch_alpha=0.0), 1, 1).close()      # not read when the filter is off


def test_closed_loop_with_filter_matches_oracle_stepwise(B, O):
    """brmppi_step with hitch_filter = 1: solve, CBF-QP on U[0], plant step with the filtered control,
    shift of the unfiltered sequence.  Starts nearly jackknifed so that the constraint is active."""
    sc = scenes.scene_cfg1(3)
    p = sc.params.with_(K=2048, T=40, n_iter=1, hitch_filter=1, hitch_max=0.6, hitch_alpha=0.2, w_hitch=0.0)
    x = sc.x0.copy()
    x[3] = x[2] - 0.58
    s = B.Solver(p, 1, 8)
    s.set_scene(sc)
    s.set_state(x)
    obs = sc.obstacles.copy()
    U = np.zeros((p.T, 2))
    floors = np.array([p.v_max, p.delta_max])
    statuses = []
    for step in range(12):
        u0 = s.step()[0]
        ref = O.iteration(p, step, x, sc.goal, obs, U, n_threads=8)
        r_gpu, st_gpu = s.get_hitch_filter()
        assert np.all(np.abs(r_gpu - ref["U"][0]) <= RTOL * np.maximum(np.abs(ref["U"][0]), floors))
        # the oracle filters the library's own reference, so that the QP is compared on identical inputs
        u_ref, st_ref = O.hitch_filter(p, x, r_gpu.astype(np.float64))
        assert st_gpu == st_ref
        assert np.all(np.abs(u0 - u_ref) <= RTOL * np.maximum(np.abs(u_ref), floors))
        statuses.append(st_gpu)
        x_ref, obs_ref = O.plant_step(p, x, u0.astype(np.float64), obs)
        x_gpu = s.get_state().astype(np.float64)
        assert np.abs(x_gpu[:2] - x_ref[:2]).max() <= 1e-5
        dpsi = (x_gpu[2:] - x_ref[2:] + np.pi) % (2 * np.pi) - np.pi
        assert np.abs(dpsi).max() <= 1e-5
        U_gpu = s.get_controls().astype(np.float64)
        assert np.all(np.abs(U_gpu - O.shift(ref["U"])) <= RTOL * np.maximum(np.abs(O.shift(ref["U"])), floors[None, :]))
        x, obs, U = x_gpu, s.get_obstacles().astype(np.float64), U_gpu
    assert 1 in statuses, statuses                       # the stabiliser did act
    assert s.launch_count() == 12 * 3                    # still solve (2 kernels) + one plant/shift kernel
    s.close()


def test_filter_off_is_unchanged(B):
    sc = scenes.scene_cfg1(3)
    p = sc.params.with_(K=1024, T=30)
    out = []
    for hf in (0, 1):
        s = B.Solver(p.with_(hitch_filter=hf, hitch_max=1.2), 1, 8)
        s.set_scene(sc)
        u0 = s.step()[0].copy()
        r, st = s.get_hitch_filter()
        out.append((u0, r, st, s.get_state()))
        s.close()
    # zero hitch angle at the start: the constraint is inactive and both runs are bit-identical
    assert out[0][2] == 0 and out[1][2] == 0
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][0], out[0][1])
    assert np.array_equal(out[0][3], out[1][3])


def test_closed_loop_keeps_the_hitch_limit(B):
    """PAPER.md:235 on the GPU path: 220 graph-replayed control steps of CFG3 from a nearly jackknifed start
    with a hitch limit of 0.6 rad.  Without the stabiliser BR-MPPI's own control overshoots the limit; with it
    the hitch angle stays within the linearisation remainder of reading 28 (tests/test_oracle_hitch_filter.py
    derives the 0.02 rad)."""
    sc = scenes.scene_cfg3(0)
    worst = {}
    for hf in (0, 1):
        p = sc.params.with_(hitch_filter=hf, hitch_max=0.6, hitch_alpha=0.3)
        s = B.Solver(p, 1, 8)
        s.set_scene(sc)
        x = sc.x0.copy()
        x[3] = x[2] - 0.55
        s.set_state(x)
        w, active = 0.0, 0
        for _ in range(220):
            s.step()
            st = s.get_state().astype(np.float64)
            w = max(w, abs((st[2] - st[3] + np.pi) % (2 * np.pi) - np.pi))
            active += s.get_hitch_filter()[1] == 1
        worst[hf] = (w, active)
        s.close()
    assert worst[0][1] == 0 and worst[1][1] > 10
    assert worst[1][0] <= 0.6 + 0.02
    assert worst[0][0] > worst[1][0] + 0.03          # the unfiltered run does overshoot


def test_scratch_is_caller_owned(B):
    """brmppi_hitch_filter stages through a device scratch the caller passes in (no library-side allocation)."""
    import ctypes as C
    import torch
    p = scenes.default_params(hitch_max=0.9, hitch_alpha=0.4)
    n = 100
    assert B.lib().brmppi_hitch_filter_scratch_bytes(0) == 0
    need = B.lib().brmppi_hitch_filter_scratch_bytes(n)
    assert need >= 36 * n
    cp = B.make_cparams(p, 1, 0, 0)
    x = np.zeros((n, 4), dtype=np.float32); r = np.zeros((n, 2), dtype=np.float32); u = np.zeros((n, 2), dtype=np.float32)
    fp = C.POINTER(C.c_float)
    st = torch.cuda.current_stream()
    small = torch.empty(need // 2, dtype=torch.uint8, device="cuda")
    args = (C.c_void_p(st.cuda_stream), C.byref(cp), n, x.ctypes.data_as(fp), r.ctypes.data_as(fp), u.ctypes.data_as(fp), None)
    assert B.lib().brmppi_hitch_filter(*args, C.c_void_p(small.data_ptr()), C.c_size_t(small.numel())) == B.ERR_WORKSPACE_TOO_SMALL
    assert B.lib().brmppi_hitch_filter(*args, None, 0) == B.ERR_NULL
    ok = torch.empty(need, dtype=torch.uint8, device="cuda")
    assert B.lib().brmppi_hitch_filter(*args, C.c_void_p(ok.data_ptr()), C.c_size_t(need)) == B.OK
