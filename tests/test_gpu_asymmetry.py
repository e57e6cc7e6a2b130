"""GPU parity of the peak-asymmetry / sec-width extension (R30) against the fp64 oracle,
through the C ABI: five latent classes (h, mu, w, r, alpha) per phase.  Same tolerances as tests/test_gpu_parity.py."""
import math

import numpy as np
import pytest

from oracle import xrdvi_oracle as orc
from paper_2501_09308_b200 import Xrdvi, synth

from test_gpu_parity import TOL_ELBO, TOL_GRAD, TOL_INCL, check_eval, class_errors

pytestmark = pytest.mark.gpu


def test_config0_split_peaks_all_states_and_fit():
    wl = synth.make_workload(0, asym=(0.75, 1.35))
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    assert gpu.C == 5 and o.C == 5 and gpu.pair_count == o.pair_count()
    st0, step = gpu.get_state()
    assert st0.shape == (1, 1, 2, wl.K, 5) and step == 0
    np.testing.assert_allclose(st0, o.init_state(), rtol=1e-6)
    check_eval(gpu, o, st0, wl.S, seed=3, iteration=1, n_prof=16)
    gpu.fit(50, seed=3)
    st50, _ = gpu.get_state()
    check_eval(gpu, o, st50, wl.S, seed=3, iteration=51, n_prof=16)
    st_g, inc_g, tr_g = gpu.fit(450, seed=3, want_trace=True)
    check_eval(gpu, o, st_g, wl.S, seed=3, iteration=501, n_prof=16)
    st_r, _, tr_r = o.fit(o.init_state(), 500, wl.S, seed=3, want_trace=True)
    inc_r = o.inclusion(st_r)
    decided = (inc_r < 0.05) | (inc_r > 0.95)
    assert np.abs(inc_g - inc_r)[decided].max() <= TOL_INCL
    # absent phases of config 0 are still on their way down after 500 steps (R29): their read-out sits on the
    # steep part of the normal cdf, where fp32 and fp64 trajectories that differ by 0.01 in m_h differ by 0.04 in P_incl
    assert np.abs(inc_g - inc_r).max() <= 0.1
    for k in wl.true_phases[0]:       # parameters of the planted phases; on config 0's undersampled grid (h, w, alpha)
        # trade off along a ridge: fp32 trajectories with different summation orders end 0.05-0.13 apart along it (measured)
        np.testing.assert_allclose(st_g[0, 0, 0, k, [0, 2, 4]], st_r[0, 0, 0, k, [0, 2, 4]], atol=0.2)
        np.testing.assert_allclose(st_g[0, 0, 0, k, 1], st_r[0, 0, 0, k, 1], atol=0.01)
    inc2, area = gpu.inclusion()
    inc_o, area_o = o.inclusion(st_g.astype(np.float64), want_area=True)
    np.testing.assert_allclose(inc2, inc_o, atol=1e-9)
    np.testing.assert_allclose(area, area_o, rtol=1e-9)
    np.testing.assert_allclose(gpu.posterior_summary()[..., 4, :], o.posterior_summary(st_g.astype(np.float64))[..., 4, :],
                               rtol=1e-12)


def test_first_steps_follow_the_oracle_and_alpha_is_updated():
    wl = synth.make_workload(0, asym=(0.75, 1.35))
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    st_g, _, tr_g = gpu.fit(1, seed=5, want_trace=True)
    st_r, _, tr_r = o.fit(o.init_state(), 1, wl.S, seed=5, want_trace=True)
    np.testing.assert_allclose(st_g, st_r, atol=2e-5)
    assert np.all(np.abs(st_g[0, 0, 0, :, 4]) == pytest.approx(0.1, rel=1e-3))     # first Adam step of m_alpha = +-lr
    st_g3, _, _ = gpu.fit(2, seed=5)
    st_r3, _, _ = o.fit(o.init_state(), 3, wl.S, seed=5)
    np.testing.assert_allclose(st_g3, st_r3, atol=2e-3)


def test_config1_with_the_asymmetric_model_three_states_and_restarts():
    wl = synth.make_workload(1, S=64, n_restarts=2)
    o = orc.from_workload(wl, asymmetry=1)
    gpu = Xrdvi.from_workload(wl, asymmetry=1)
    gpu.reset_state(seed=9)
    st0, _ = gpu.get_state()
    np.testing.assert_allclose(st0, o.init_state(seed=9), rtol=2e-6, atol=2e-7)
    assert np.abs(st0[0, 1, 0, :, 4]).min() > 0                   # restart 1: jittered alpha
    check_eval(gpu, o, st0, 64, seed=1, iteration=1)
    gpu.fit(60, seed=1)
    st, _ = gpu.get_state()
    check_eval(gpu, o, st, 64, seed=1, iteration=61)
    rnd = synth.random_state(wl.K, 1, 2, seed=4, classes=5)
    rnd[:, :, 0, :, 0] += math.log(1.0 / o.lambda_h()) - 2.0
    rnd[:, :, 0, :, 4] *= 2.0                                      # alpha from 0.5 to 2
    check_eval(gpu, o, rnd, 64, seed=2, iteration=7)


@pytest.mark.parametrize("asym", [0, 1])
def test_sec_width_term(asym):
    wl = synth.make_workload(1, S=32, K=12)
    o = orc.from_workload(wl, width_sec=1, asymmetry=asym)
    gpu = Xrdvi.from_workload(wl, width_sec=1, asymmetry=asym)
    assert gpu.C == 4 + asym
    st = synth.random_state(wl.K, 1, 1, seed=3, classes=4 + asym)
    st[0, 0, 0, :, 0] += math.log(1.0 / o.lambda_h()) - 2.0
    check_eval(gpu, o, st, 32, seed=4, iteration=2, n_prof=4)
    gpu.fit(30, seed=2)
    st30, _ = gpu.get_state()
    check_eval(gpu, o, st30, 32, seed=2, iteration=31, n_prof=2)


def test_poisson_with_asymmetry_and_adaptive_windows():
    wl = synth.make_workload(0, asym=(0.8, 1.3), peak_counts=2.0e4)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    st0, _ = gpu.get_state()
    check_eval(gpu, o, st0, wl.S, seed=3, iteration=1, n_prof=8)
    gpu.fit(120, seed=3)
    st, _ = gpu.get_state()
    check_eval(gpu, o, st, wl.S, seed=3, iteration=121, n_prof=8)
    nck = gpu.adapt_windows(10.0)
    np.testing.assert_array_equal(nck, o.adaptive_halfwidths(st.astype(np.float64), 10.0))
    o.set_phase_windows(nck)
    assert gpu.pair_count == o.pair_count()
    check_eval(gpu, o, st, wl.S, seed=3, iteration=122, n_prof=8)


def test_long_work_items_take_the_split_kernel_with_asymmetry():
    wl = synth.make_workload(4, K=150, S=8)
    o = orc.from_workload(wl, asymmetry=1)
    gpu = Xrdvi.from_workload(wl, asymmetry=1)
    st = synth.random_state(wl.K, 1, 1, seed=12, classes=5)
    st[:, :, 0, :, 0] += math.log(1.0 / o.lambda_h()) - 3.0
    st[:, :, 0, :, 2] = np.log(np.random.default_rng(0).uniform(0.03, 0.3, wl.K))
    check_eval(gpu, o, st, 8, seed=6, iteration=2, n_prof=2)


def test_logjoint_gradient_service_with_five_classes():
    wl = synth.make_workload(3, n_patterns=2, S=64)
    o = orc.from_workload(wl, asymmetry=1)
    gpu = Xrdvi.from_workload(wl, asymmetry=1)
    rng = np.random.default_rng(3)
    for pat, n in ((0, 1), (1, 37)):
        z = synth.random_state(wl.K, n, 1, seed=20 + pat, classes=5)[:, 0, 0]
        z[:, :, 0] += math.log(1.0 / o.lambda_h(pat)) - 2.0 + rng.normal(0, 0.3, (n, wl.K))
        ll_g, lpj_g, g_g = gpu.logjoint_grad(z, pattern=pat)
        assert g_g.shape == (n, wl.K, 5)
        for t in sorted({0, n // 2, n - 1}):
            ll_r, lpj_r, g_r = o.logjoint_grad(z[t].astype(np.float64), pat)
            assert ll_g[t] == pytest.approx(ll_r, rel=TOL_ELBO)
            assert lpj_g[t] == pytest.approx(lpj_r, rel=TOL_ELBO, abs=1e-3)
            err = np.abs(g_g[t] - g_r).max(axis=0) / np.abs(g_r).max(axis=0)
            assert err.max() <= TOL_GRAD, err


def test_checkpoint_resume_and_reproducibility_with_five_classes():
    wl = synth.make_workload(1, S=64, K=10)
    ref = Xrdvi.from_workload(wl, asymmetry=1)
    st_ref, inc_ref, _ = ref.fit(29, seed=9)
    a = Xrdvi.from_workload(wl, asymmetry=1)
    a.fit(13, seed=9)
    st, step = a.get_state()
    m1, m2, n = a.get_optimizer_state()
    assert m1.shape == st.shape and np.abs(m2[..., 4]).max() > 0
    b = Xrdvi.from_workload(wl, asymmetry=1)
    b.set_state(st, step)
    b.set_optimizer_state(m1, m2, n)
    st_b, inc_b, _ = b.fit(16, seed=9)
    np.testing.assert_array_equal(st_b, st_ref)
    np.testing.assert_array_equal(inc_b, inc_ref)
