"""The oracle's fp32 re-run mode (SURVEY 8(c) reading 23; oracle/oracle32.py, oracle/fp32_floor.py): the fp32 noise
floor of every parity quantity is printed next to its tolerance (run with -s to see the table), and where the floor
exceeds the tolerance the report must say so and name the rule the parity test uses instead.  CPU only; the GPU path
is never compared with the fp32 build."""
import numpy as np

import scenes
from oracle import fp32_floor


def test_fp32_build_draws_the_same_noise_and_is_a_different_build(O):
    from oracle import oracle32 as O32
    assert O32._FP32 and not O._FP32 and O32._LIB != O._LIB
    p = scenes.default_params()
    for (n, k, t) in ((0, 0, 0), (3, 17, 5), (9, 4095, 79)):
        z64, z32 = O.normals(p.seed, n, k, t), O32.normals(p.seed, n, k, t)
        assert z32.dtype == np.float32 and np.allclose(z32, z64, rtol=0, atol=4e-6)   # Box-Muller in float: ~1e-6
        assert abs(O32.alpha(p, n, k) - O.alpha(p, n, k)) <= 1e-7                       # exact uniform, one rounding
    # one Euler step: fp32 rounding, not a different formula
    x = np.array([1.0, -2.0, 0.3, -0.2])
    assert np.allclose(O32.kinematic_step(p, x, 1.5, 0.2), O.kinematic_step(p, x, 1.5, 0.2), rtol=0, atol=1e-6)


def test_fp32_floor_is_reported_beside_every_tolerance(capsys):
    rows = fp32_floor.report(K=512, n_threads=8)
    with capsys.disabled():
        print("\n" + fp32_floor.markdown(rows))
    by = {(r["path"], r["quantity"]): r for r in rows}
    assert len(by) == len(rows) >= 15
    for r in rows:
        assert np.isfinite(r["floor_max"]) and r["tolerance"] == 1e-4
        if not r["attainable"]:                       # said, not hidden: and the parity rule used instead is named
            assert r["note"], r
    # the flat tolerance on x_T and S_k is attainable in fp32 on every path of the penalty family, with margin
    for (path, q), r in by.items():
        if q in ("x_T", "S_k") and ("penalty" in path or "super-ellipses" in path):
            assert r["floor_max"] <= 0.25 * r["tolerance"], r
    # final states of the other two paths too, away from the amplifying samples
    assert by[("7-state model + (13), (17), cfg2mpcc shape", "x_T")]["floor_max"] <= 0.25e-4
    assert by[("projected rollout (Sec. V-A), cfg2 shape", "x_T")]["floor_p99"] <= 0.25e-4
