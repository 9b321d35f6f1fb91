"""Parity of brmppi_project (eq. (11)-(12)) through the C ABI against oracle/projection.py
on the same seeded (9)-shaped problems.

Tolerance: the flat |z - z_ref| <= 1e-4 max(|z_ref|, 1) of the north star for every (9)-shaped problem of the
recipe (A = [L_g h | diag(h)]; measured on 3000 problems per N_o: worst error 2.0e-5 at N_o = 7 although
cond(S) of S = A M^-1 A^T reaches 7e4 -- Cholesky's error follows the diagonally scaled condition number,
which the diag(h) block keeps small; table in DESIGN.md 6.9).  A DENSE random A is not what (9) produces; the
call accepts it, and there fp32 Cholesky loses cond(S) eps_32 (2.6e-4 seen at cond 2e4), so those cases are
compared at 1e-4 max(1, cond(S) / 1e3).  The equality constraint itself is checked in fp64 on the fp32
result: |A z - b| <= 2e-5 (1 + |A| |z|)."""
import numpy as np
import pytest

from scenes.projection import projection_batch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    from paper_2508_05773_b200 import brmppi
    brmppi.lib()
    return brmppi


@pytest.fixture(scope="module")
def OP():
    from oracle import projection
    return projection


def check(OP, z, P, idx, dense=False):
    Minv = 1.0 / (P["w"] + P["rho"])
    worst = 0.0
    for i in idx:
        ref = OP.project(P["A"][i], P["b"][i], P["z_des"][i], P["w"], P["rho"], P["z_lo"], P["z_hi"])
        tol = 1e-4
        if dense:
            tol *= max(1.0, np.linalg.cond((P["A"][i] * Minv[None, :]) @ P["A"][i].T) / 1e3)
        zi = z[i].astype(np.float64)
        err = np.abs(zi - ref) / np.maximum(np.abs(ref), 1.0)
        assert err.max() <= tol, (i, err.max())
        worst = max(worst, err.max() / tol)
        res = np.abs(P["A"][i] @ zi - P["b"][i])
        assert np.all(res <= 2e-5 * (1.0 + np.abs(P["A"][i]) @ np.abs(zi))), (i, res)
    return worst


@pytest.mark.parametrize("n_o", [1, 2, 3, 4, 5, 6, 7, 8])
@pytest.mark.parametrize("n", [1, 127, 129, 1000])
def test_host_pointers_match_oracle(B, OP, n_o, n):
    dense = (n % 2 == 0)
    P = projection_batch(1000 * n_o + n, n, n_o, dense=dense)
    z = B.project(P["A"], P["b"], P["z_des"], P["w"], P["rho"], P["z_lo"], P["z_hi"])
    assert z.shape == (n, n_o + 2) and np.isfinite(z).all()
    check(OP, z, P, range(n), dense=dense)


def test_device_pointers_full_size_sampled(B, OP):
    """The paper's per-solve count: 5000 rollouts x 120 steps = 600 000 projections with eight obstacles
    (PAPER.md:243), device-resident, sampled rows against the oracle; host- and device-pointer calls agree
    bit for bit."""
    import torch
    n, n_o = 600_000, 8
    P = projection_batch(7, n, n_o)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()
    z = B.project(dev(P["A"]), dev(P["b"]), dev(P["z_des"]), P["w"], P["rho"], P["z_lo"], P["z_hi"])
    torch.cuda.synchronize()
    z = z.cpu().numpy()
    assert np.isfinite(z).all()
    idx = np.concatenate([[0, 1, 127, 128, n - 129, n - 128, n - 1], np.random.default_rng(0).integers(0, n, 300)])
    check(OP, z, P, idx)
    # A CTA of the big launch walks ~10 blocks through one shared-memory stage that is refilled while it
    # computes; a launch of <= 443 blocks gives every CTA a single block.  Same arithmetic per problem, so
    # windows of the big result must equal their own small launches bit for bit (this caught a missing
    # proxy fence before the refill: rows of the next block overwrote loads still in flight).
    for start_blk in (0, 1500, 4687 - 440):
        sl = slice(start_blk * 128, (start_blk + 440) * 128)
        z_win = B.project(P["A"][sl], P["b"][sl], P["z_des"][sl], P["w"], P["rho"], P["z_lo"], P["z_hi"])
        assert np.array_equal(z_win, z[sl]), start_blk
    sl = slice(n - 960, n)                       # 7 full blocks + the 64-problem tail in both launches
    z_host = B.project(P["A"][sl], P["b"][sl], P["z_des"][sl], P["w"], P["rho"], P["z_lo"], P["z_hi"])
    assert np.array_equal(z_host, z[sl])


@pytest.mark.parametrize("n_o", [3, 6, 7])
def test_many_blocks_per_cta_other_sizes(B, OP, n_o):
    """Odd N_o (scalar shared loads) and another even one through the persistent multi-block path."""
    import torch
    n = 128 * 3000 + 77
    P = projection_batch(40 + n_o, n, n_o)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()
    z = B.project(dev(P["A"]), dev(P["b"]), dev(P["z_des"]), P["w"], P["rho"], P["z_lo"], P["z_hi"]).cpu().numpy()
    check(OP, z, P, np.concatenate([[0, 127, 128, n - 78, n - 77, n - 1], np.random.default_rng(1).integers(0, n, 150)]))
    sl = slice(128 * 1000, 128 * 1400)
    z_win = B.project(P["A"][sl], P["b"][sl], P["z_des"][sl], P["w"], P["rho"], P["z_lo"], P["z_hi"])
    assert np.array_equal(z_win, z[sl])


def test_rho_zero_and_large(B, OP):
    P = projection_batch(5, 256, 4)
    for rho in (0.0, 50.0):
        P["rho"] = rho
        z = B.project(P["A"], P["b"], P["z_des"], P["w"], rho, P["z_lo"], P["z_hi"])
        check(OP, z, P, range(256))


def test_edge_cases_and_errors(B):
    P = projection_batch(1, 4, 3)
    z = B.project(P["A"][:0], P["b"][:0], P["z_des"][:0], P["w"], P["rho"], P["z_lo"], P["z_hi"])   # n = 0
    assert z.shape == (0, 5)
    # a rank-deficient problem (two equal rows) spoils its own row only
    A = P["A"].copy()
    A[2, 1] = A[2, 0]
    z = B.project(A, P["b"], P["z_des"], P["w"], P["rho"], P["z_lo"], P["z_hi"])
    z_ok = B.project(P["A"], P["b"], P["z_des"], P["w"], P["rho"], P["z_lo"], P["z_hi"])
    assert np.array_equal(z[[0, 1, 3]], z_ok[[0, 1, 3]])
    with pytest.raises(B.BrmppiError):
        B.project(np.zeros((2, 9, 11)), np.zeros((2, 9)), np.zeros((2, 11)), np.ones(11), 0.1, -np.ones(11), np.ones(11))
    w_bad = P["w"].copy()
    w_bad[1] = 0.0
    with pytest.raises(B.BrmppiError):
        B.project(P["A"], P["b"], P["z_des"], w_bad, P["rho"], P["z_lo"], P["z_hi"])
    with pytest.raises(B.BrmppiError):
        B.project(P["A"], P["b"], P["z_des"], P["w"], -1.0, P["z_lo"], P["z_hi"])


def test_unaligned_device_pointers_take_the_generic_path(B, OP):
    """Views that start one problem into an odd-N_o batch are not 16-byte aligned (63, 7 and 9 words per
    problem): no bulk copy is legal, the call falls back to the LDG kernel and must still be right."""
    import torch
    n, n_o = 700, 7
    P = projection_batch(9, n, n_o)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()
    A, b, zd = dev(P["A"]), dev(P["b"]), dev(P["z_des"])
    assert A[1:].data_ptr() % 16 != 0 and A[1:].is_contiguous()
    z_all = B.project(A, b, zd, P["w"], P["rho"], P["z_lo"], P["z_hi"]).cpu().numpy()
    z_view = B.project(A[1:], b[1:], zd[1:], P["w"], P["rho"], P["z_lo"], P["z_hi"]).cpu().numpy()
    assert np.array_equal(z_view, z_all[1:])          # same arithmetic on both paths
    check(OP, z_all, P, range(0, n, 5))


def test_caller_owned_scratch_and_pinned_staging(B, OP):
    """The host-pointer form stages through a device scratch the CALLER owns (the library allocates no device
    memory): too small -> BRMPPI_ERR_WORKSPACE_TOO_SMALL, NULL -> BRMPPI_ERR_NULL; page-locked host tensors go
    through the same call and give the same bits as numpy arrays."""
    import ctypes as C
    import torch
    n, n_o = 300, 5
    P = projection_batch(21, n, n_o)
    need = B.lib().brmppi_project_scratch_bytes(n, n_o)
    assert need >= 4 * (n * n_o * (n_o + 2) + n * n_o + 2 * n * (n_o + 2))
    assert B.lib().brmppi_project_scratch_bytes(0, n_o) == 0 and B.lib().brmppi_project_scratch_bytes(n, 9) == 0
    z_np = B.project(P["A"], P["b"], P["z_des"], P["w"], P["rho"], P["z_lo"], P["z_hi"])
    small = torch.empty(need // 2, dtype=torch.uint8, device="cuda")
    with pytest.raises(B.BrmppiError) as e:
        B.project(P["A"], P["b"], P["z_des"], P["w"], P["rho"], P["z_lo"], P["z_hi"], scratch=small)
    assert e.value.status == B.ERR_WORKSPACE_TOO_SMALL
    A = np.ascontiguousarray(P["A"], dtype=np.float32)
    st = torch.cuda.current_stream()
    f = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    w, lo, hi = f(P["w"]), f(P["z_lo"]), f(P["z_hi"])
    fp = C.POINTER(C.c_float)
    out = np.zeros((n, n_o + 2), dtype=np.float32)
    b_, z_ = f(P["b"]), f(P["z_des"])
    r = B.lib().brmppi_project(C.c_void_p(st.cuda_stream), n, n_o, C.c_void_p(A.ctypes.data), C.c_void_p(b_.ctypes.data),
                               C.c_void_p(z_.ctypes.data), w.ctypes.data_as(fp), float(P["rho"]), lo.ctypes.data_as(fp),
                               hi.ctypes.data_as(fp), C.c_void_p(out.ctypes.data), 0, None, 0)
    assert r == B.ERR_NULL
    pin = lambda a: torch.from_numpy(f(a)).pin_memory()
    big = torch.empty(need, dtype=torch.uint8, device="cuda")
    z_pin = B.project(pin(P["A"]), pin(P["b"]), pin(P["z_des"]), P["w"], P["rho"], P["z_lo"], P["z_hi"], scratch=big)
    assert np.array_equal(z_pin, z_np)
    check(OP, z_np, P, range(0, n, 3))
