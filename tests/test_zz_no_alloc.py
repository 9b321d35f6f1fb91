"""brmppi_hitch_filter_static: the hitch-angle stabiliser (Sec. V-D) through the library's static
device scratch, for callers that cannot allocate device memory (include/brmppi.h).  Its output is compared with the
existing path's (brmppi_hitch_filter with a caller-owned scratch, itself checked against the oracle in
test_gpu_hitch_filter.py) on two calls in a row that share the static array -- the second one smaller, so that
stale entries of the first would show -- within the tolerance of the other control tests: 1e-4 relative with floors
(v_max, delta_max); the statuses must be equal.  The file is named so that pytest collects it last."""
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


def pairs(rng, n, p):
    beta = rng.uniform(-1.5, 1.5, n)
    psi2 = rng.uniform(-np.pi, np.pi, n)
    x = np.stack([rng.uniform(-20, 20, n), rng.uniform(-20, 20, n), psi2 + beta, psi2], axis=1).astype(np.float32)
    u = np.stack([rng.uniform(1.1 * p.v_min, 1.1 * p.v_max, n), rng.uniform(1.1 * p.delta_min, 1.1 * p.delta_max, n)],
                 axis=1).astype(np.float32)
    return x, u


def test_static_scratch_matches_the_caller_scratch_path_twice(B):
    p = scenes.default_params(dt=0.05).with_(hitch_kappa=0.2, hitch_alpha=0.3, hitch_qv=0.5, hitch_qdelta=4.0, hitch_max=0.9)
    floors = np.array([max(abs(p.v_min), abs(p.v_max)), max(abs(p.delta_min), abs(p.delta_max))])
    rng = np.random.default_rng(7)
    seen = set()
    for n in (B.HITCH_STATIC_MAX_N, 1000):          # the full capacity, then a smaller batch over the same array
        x, r = pairs(rng, n, p)
        u_ref, st_ref = B.hitch_filter(p, x, r)
        u, st = B.hitch_filter_static(p, x, r)
        assert np.array_equal(st, st_ref)
        assert (np.abs(u - u_ref) <= RTOL * np.maximum(np.abs(u_ref), floors[None, :])).all()
        seen |= set(st.tolist())
    assert seen == {0, 1, 2}                         # all three outcomes of the QP were exercised


def test_capacity_and_argument_errors(B):
    p = scenes.default_params(dt=0.05)
    x, r = pairs(np.random.default_rng(1), B.HITCH_STATIC_MAX_N + 1, p)
    with pytest.raises(B.BrmppiError) as e:
        B.hitch_filter_static(p, x, r)
    assert e.value.status == B.ERR_TOO_LARGE and "static" in str(e.value)
    u, st = B.hitch_filter_static(p, x[:0], r[:0])   # n = 0 is a no-op
    assert u.shape == (0, 2) and st.shape == (0,)
    with pytest.raises(B.BrmppiError) as e:
        B.hitch_filter_static(p.with_(hitch_alpha=0.0), x[:4], r[:4])
    assert e.value.status == B.ERR_INVALID_ARG
