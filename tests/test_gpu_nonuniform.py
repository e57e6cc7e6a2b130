"""GPU parity on NON-UNIFORM 2-theta grids (hyper.general_grid = 1, R31) against the fp64 oracle, whose
non-uniform path is pinned in tests/test_nonuniform_grid_pins.py.  Tolerances as in tests/test_gpu_parity.py."""
import math

import numpy as np
import pytest

from oracle import xrdvi_oracle as orc
from paper_2501_09308_b200 import Xrdvi, XrdviError, synth

from test_gpu_parity import check_eval

pytestmark = pytest.mark.gpu


def jitter(x, seed, amp=0.35):
    rng = np.random.default_rng(seed)
    step = (x[-1] - x[0]) / (x.shape[0] - 1)
    xj = x.copy()
    xj[1:-1] += rng.uniform(-amp, amp, x.shape[0] - 2) * step
    assert np.all(np.diff(xj) > 0)
    return xj


def both(wl, x, **hyper):
    hp = dict(wl.hyper)
    hp.update(hyper)
    o = orc.Oracle(x, wl.y, wl.background, wl.peak_ofs, wl.peak_pos, wl.peak_int, **hp)
    gpu = Xrdvi(x, wl.y, wl.background, wl.peak_ofs, wl.peak_pos, wl.peak_int, S_max=wl.S, general_grid=1, **hp)
    return o, gpu


def test_jittered_config1_three_states():
    wl = synth.make_workload(1, S=64)
    x = jitter(wl.two_theta, seed=5)
    o, gpu = both(wl, x)
    assert gpu.pair_count == o.pair_count() and gpu.n_c == o.n_c
    st0, _ = gpu.get_state()
    np.testing.assert_allclose(st0, o.init_state(), rtol=1e-6)
    check_eval(gpu, o, st0, 64, seed=1, iteration=1)
    gpu.fit(60, seed=1)
    st, _ = gpu.get_state()
    check_eval(gpu, o, st, 64, seed=1, iteration=61)
    rnd = synth.random_state(wl.K, 1, 1, seed=4)
    rnd[:, :, 0, :, 0] += math.log(1.0 / o.lambda_h()) - 2.0
    check_eval(gpu, o, rnd, 64, seed=2, iteration=7)


def test_jittered_config0_fit_and_ragged_grid():
    wl = synth.make_workload(0)
    x = jitter(wl.two_theta, seed=9, amp=0.4)                       # N = 1001: a ragged last tile; steps from 0.2 to 1.8 of the mean
    o, gpu = both(wl, x)
    st0, _ = gpu.get_state()
    check_eval(gpu, o, st0, wl.S, seed=3, iteration=1, n_prof=16)
    st_g, inc_g, tr_g = gpu.fit(200, seed=3, want_trace=True)
    st_r, _, tr_r = o.fit(o.init_state(), 200, wl.S, seed=3, want_trace=True)
    np.testing.assert_allclose(tr_g[:3], tr_r[:3], rtol=1e-4)
    check_eval(gpu, o, st_g, wl.S, seed=3, iteration=201, n_prof=16)
    for k in wl.true_phases[0]:
        np.testing.assert_allclose(st_g[0, 0, 0, k, :3], st_r[0, 0, 0, k, :3], atol=0.03)


def test_general_path_with_asymmetry_poisson_and_dense_window():
    wl = synth.make_workload(0, asym=(0.8, 1.3), peak_counts=2.0e4)
    x = jitter(wl.two_theta, seed=2)
    o, gpu = both(wl, x)
    assert gpu.C == 5
    st = synth.random_state(wl.K, 1, 1, seed=3, classes=5)
    st[0, 0, 0, :, 0] += math.log(1.0 / o.lambda_h()) - 1.0
    check_eval(gpu, o, st, wl.S, seed=4, iteration=2, n_prof=8)
    wl2 = synth.make_workload(1, S=32, K=8)
    o2, gpu2 = both(wl2, jitter(wl2.two_theta, seed=3), window_W=0.0)      # dense: every point in every window
    st2, _ = gpu2.get_state()
    check_eval(gpu2, o2, st2, 32, seed=1, iteration=1, n_prof=2)


def test_uniform_grid_through_the_general_path_and_rejections():
    wl = synth.make_workload(1, S=32, K=10)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl, general_grid=1)                          # a uniform grid is accepted with the flag
    st0, _ = gpu.get_state()
    check_eval(gpu, o, st0, 32, seed=1, iteration=1)
    ref = Xrdvi.from_workload(wl)
    e_a, g_a = gpu.elbo_grad(S=32, seed=1, iteration=1)
    e_b, g_b = ref.elbo_grad(S=32, seed=1, iteration=1)
    np.testing.assert_allclose(e_a, e_b, rtol=1e-6)                        # same model, other arithmetic order
    x = jitter(wl.two_theta, seed=1)
    with pytest.raises(XrdviError) as ei:                                  # non-uniform without the flag
        Xrdvi(x, wl.y, wl.background, wl.peak_ofs, wl.peak_pos, wl.peak_int, S_max=32, **wl.hyper)
    assert ei.value.code == -3
    xr = wl.two_theta.copy()
    xr[10] = xr[9] + 0.1 * (xr[11] - xr[9]) / 2                            # steps 0.1 and 1.9 of the mean: ratio 19
    with pytest.raises(XrdviError) as ei:
        Xrdvi(xr, wl.y, wl.background, wl.peak_ofs, wl.peak_pos, wl.peak_int, S_max=32, general_grid=1, **wl.hyper)
    assert ei.value.code == -3
