"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (full P, R, S, so the
same kernel shape, grid and workspace), on outputs the oracle can compute in seconds:

  cfg 1  K=50, S=256: everything (profile, ll per draw, ELBO, gradient) at three states;
  cfg 2  R=32 x S=4096 (131 072 sample-instances in one launch): ll of every draw and ELBO + gradient of two
         sampled restarts (first and last), ll of sampled draws of others one by one;
  cfg 3  P=1024 x S=128: ELBO + gradient + ll of sampled patterns (first, middle, last);
  cfg 4  K=1000, M~175k, N=8001, +-400-point window, S=256: ll of sampled draws one by one, ELBO and gradient
         of the whole evaluation;
plus properties that hold at any size (restarts with identical state and identical counters would coincide;
every ll finite; gradient of l is 1 + O(.)).  Tolerances as in test_gpu_parity.py (north_star).
"""
import numpy as np
import pytest

from oracle import xrdvi_oracle as orc
from paper_2501_09308_b200 import Xrdvi, synth

pytestmark = pytest.mark.gpu

TOL_ELBO = 1e-4
TOL_GRAD = 1e-3
TOL_PROFILE = 1e-4


def class_err(g_gpu, g_ref):
    """g [..., 2, K, 4] -> max over classes of max_k |diff| / max_k |ref|."""
    err = np.abs(g_gpu.astype(np.float64) - g_ref).max(axis=-2)
    ref = np.abs(g_ref).max(axis=-2)
    return float((err / ref).max())


def profile_one_draw(o, state64, seed, iteration, inst, s):
    """profile of ONE draw computed piece by piece with the oracle (eps -> zeta -> profile)."""
    pat = inst // o.R
    st = state64.reshape(o.P * o.R, 2, o.K, 4)[inst]
    zeta = np.empty((o.K, 4))
    for k in range(o.K):
        zeta[k] = st[0, k] + np.exp(st[1, k]) * orc.eps(seed, iteration, inst, s, k)
    return o.profile(zeta, pat), pat


def ll_one_draw(o, state64, seed, iteration, inst, s):
    """log-likelihood of ONE draw computed piece by piece with the oracle (eps -> zeta -> profile -> ll)."""
    f, pat = profile_one_draw(o, state64, seed, iteration, inst, s)
    return o.loglik(f, pat)


def check_profiles(gpu, o, st, S, seed, iteration, picks):
    """element-wise profile of sampled draws (instance, s) at full size: first / last group of the launch, so that both
    ends of the grid of CTAs (and, at config 4, of the ticket queue) are hit"""
    st64 = st.astype(np.float64)
    for inst, s in picks:
        f_g, _ = gpu.debug_profile(1, state=st, S=S, seed=seed, iteration=iteration, first=inst * S + s)
        f_r, _ = profile_one_draw(o, st64, seed, iteration, inst, s)
        assert np.abs(f_g[0] - f_r).max() / np.abs(f_r).max() <= TOL_PROFILE, (inst, s)


def test_config1_full_size_three_states():
    wl = synth.make_workload(1)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    assert gpu.pair_count == o.pair_count()
    for n_fit, it in ((0, 1), (50, 51), (450, 501)):
        if n_fit:
            gpu.fit(n_fit, seed=1)
        st, _ = gpu.get_state()
        elbo_r, grad_r, ll_r, f_r = o.elbo_grad(st.astype(np.float64), wl.S, 1, it, want_ll=True, n_profiles=3)
        f_g, ll_g = gpu.debug_profile(wl.S, state=st, S=wl.S, seed=1, iteration=it, want_f=False)
        np.testing.assert_allclose(ll_g, ll_r.reshape(-1), rtol=TOL_ELBO)
        f_g, _ = gpu.debug_profile(3, state=st, S=wl.S, seed=1, iteration=it)
        for t in range(3):
            assert np.abs(f_g[t] - f_r[t]).max() / np.abs(f_r[t]).max() <= TOL_PROFILE
        elbo_g, grad_g = gpu.elbo_grad(state=st, S=wl.S, seed=1, iteration=it)
        np.testing.assert_allclose(elbo_g, elbo_r, rtol=TOL_ELBO)
        assert class_err(grad_g, grad_r) <= TOL_GRAD
    inc, area = gpu.inclusion()
    truth = wl.true_phases[0]
    assert np.all(inc[0, 0, truth] > 0.99)                       # the planted phases are found
    assert area[0, 0, truth].sum() > 0.9


def test_config2_full_size_sampled_restarts():
    wl = synth.make_workload(2)
    assert (wl.R, wl.S) == (32, 4096)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    gpu.reset_state(seed=5)
    gpu.fit(3, seed=2)                                           # a few full-size steps away from the start
    st, step = gpu.get_state()
    assert step == 3
    st64 = st.astype(np.float64)
    elbo_g, grad_g = gpu.elbo_grad(state=st, S=wl.S, seed=2, iteration=9)
    _, ll_g = gpu.debug_profile(wl.R * wl.S, state=st, S=wl.S, seed=2, iteration=9, want_f=False)
    ll_g = ll_g.reshape(wl.R, wl.S)
    assert np.isfinite(ll_g).all() and np.isfinite(grad_g).all()
    for rst in (0, wl.R - 1):
        e_r, g_r, ll_r = o.elbo_grad_range(st64, wl.S, 2, 9, rst, 1, want_ll=True)
        np.testing.assert_allclose(ll_g[rst], ll_r[0], rtol=TOL_ELBO)
        np.testing.assert_allclose(elbo_g[0, rst], e_r[0], rtol=TOL_ELBO)
        assert class_err(grad_g[0, rst], g_r[0]) <= TOL_GRAD
    check_profiles(gpu, o, st, wl.S, 2, 9, [(0, 0), (0, 31), (wl.R - 1, wl.S - 32), (wl.R - 1, wl.S - 1)])
    rng = np.random.default_rng(0)
    for _ in range(12):                                          # other restarts: sampled draws one by one
        rst, s = int(rng.integers(1, wl.R - 1)), int(rng.integers(0, wl.S))
        assert ll_g[rst, s] == pytest.approx(ll_one_draw(o, st64, 2, 9, rst, s), rel=TOL_ELBO)


def test_config3_full_size_sampled_patterns():
    wl = synth.make_workload(3)
    assert (wl.P, wl.S) == (1024, 128)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    gpu.fit(2, seed=4)
    st, _ = gpu.get_state()
    st64 = st.astype(np.float64)
    elbo_g, grad_g = gpu.elbo_grad(state=st, S=wl.S, seed=4, iteration=7)
    _, ll_g = gpu.debug_profile(wl.P * wl.S, state=st, S=wl.S, seed=4, iteration=7, want_f=False)
    ll_g = ll_g.reshape(wl.P, wl.S)
    assert np.isfinite(ll_g).all() and np.isfinite(grad_g).all()
    for pat in (0, 511, 1023):
        e_r, g_r, ll_r = o.elbo_grad_range(st64, wl.S, 4, 7, pat, 1, want_ll=True)
        np.testing.assert_allclose(ll_g[pat], ll_r[0], rtol=TOL_ELBO)
        np.testing.assert_allclose(elbo_g[pat, 0], e_r[0], rtol=TOL_ELBO)
        assert class_err(grad_g[pat, 0], g_r[0]) <= TOL_GRAD
    check_profiles(gpu, o, st, wl.S, 4, 7, [(0, 0), (0, 31), (wl.P - 1, wl.S - 32), (wl.P - 1, wl.S - 1)])
    rng = np.random.default_rng(1)
    for _ in range(12):
        pat, s = int(rng.integers(0, wl.P)), int(rng.integers(0, wl.S))
        assert ll_g[pat, s] == pytest.approx(ll_one_draw(o, st64, 4, 7, pat, s), rel=TOL_ELBO)


def test_config4_full_size():
    wl = synth.make_workload(4)
    assert (wl.K, wl.N, wl.S) == (1000, 8001, 256)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    assert gpu.n_c == 400 and gpu.pair_count == o.pair_count()
    gpu.fit(2, seed=6)
    st, _ = gpu.get_state()
    st64 = st.astype(np.float64)
    _, ll_g = gpu.debug_profile(wl.S, state=st, S=wl.S, seed=6, iteration=5, want_f=False)
    assert np.isfinite(ll_g).all()
    for s in (0, 31, 32, 100, 255):
        assert ll_g[s] == pytest.approx(ll_one_draw(o, st64, 6, 5, 0, s), rel=TOL_ELBO)
    check_profiles(gpu, o, st, wl.S, 6, 5, [(0, 0), (0, 31), (0, wl.S - 32), (0, wl.S - 1)])
    # whole evaluation: 3.6e10 pair evaluations in the fp64 oracle (about a minute on 16 host cores)
    elbo_g, grad_g = gpu.elbo_grad(state=st, S=wl.S, seed=6, iteration=5)
    e_r, g_r, ll_r = o.elbo_grad_range(st64, wl.S, 6, 5, 0, 1, want_ll=True)
    np.testing.assert_allclose(ll_g, ll_r[0], rtol=TOL_ELBO)
    np.testing.assert_allclose(elbo_g[0, 0], e_r[0], rtol=TOL_ELBO)
    assert class_err(grad_g[0, 0], g_r[0]) <= TOL_GRAD


def _fit_parity(iterations, S=None):
    """Fit config 1 at full size (K=50, S=256 unless given) on both sides with the same draws; compare what is unique
    (R22): inclusion probabilities (north_star: 0.02 absolute), area ratios and the identified parameters of the planted
    phases."""
    wl = synth.make_workload(1) if S is None else synth.make_workload(1, S=S)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    st_g, inc_g, tr_g = gpu.fit(iterations, seed=1, want_trace=True)
    st_r, _, tr_r = o.fit(o.init_state(), iterations, wl.S, seed=1, want_trace=True)
    inc_r, area_r = o.inclusion(st_r, want_area=True)
    _, area_g = gpu.inclusion()
    d_inc = float(np.abs(inc_g - inc_r).max())
    assert d_inc <= 0.02, d_inc
    assert np.abs(area_g - area_r).max() <= 0.01
    np.testing.assert_allclose(tr_g[:3, 0, 0], tr_r[:3, 0, 0], rtol=TOL_ELBO)
    # later the fp32 and fp64 trajectories decorrelate (R22) and the S-draw ELBO estimate fluctuates from step to
    # step: the tails agree as distributions, not entry by entry
    n_tail = min(200, iterations // 2)
    spread = float(tr_r[-n_tail:].std())
    assert abs(float(np.median(tr_g[-n_tail:])) - float(np.median(tr_r[-n_tail:]))) <= max(spread, 1e-3 * abs(float(tr_r[-1, 0, 0])))
    for k in wl.true_phases[0]:
        np.testing.assert_allclose(st_g[0, 0, 0, k, :3], st_r[0, 0, 0, k, :3], atol=0.02)
    print(f"fit parity, {iterations} iterations: max |dP_incl| = {d_inc:.2e}, max |d area ratio| = "
          f"{float(np.abs(area_g - area_r).max()):.2e}, ELBO tail median GPU {float(np.median(tr_g[-n_tail:])):.2f} "
          f"oracle {float(np.median(tr_r[-n_tail:])):.2f} (spread {spread:.1f})")
    return d_inc, inc_g, inc_r, wl


def test_config1_full_size_fit_inclusion_parity_200_iterations():
    _fit_parity(200)


def test_config1_whole_2000_iteration_fit_inclusion_parity_at_32_draws():
    """The metric's own workload end to end -- the 2000-iteration K=50 (2^50 combination) fit -- against the oracle in
    the default GPU suite: both sides with S = 32 draws per step (a minute of fp64 oracle instead of eight at S = 256,
    which stays opt-in below)."""
    d_inc, inc_g, inc_r, wl = _fit_parity(2000, S=32)
    truth = wl.true_phases[0]
    assert np.all(inc_g[0, 0, truth] > 0.99) and np.all(inc_r[0, 0, truth] > 0.99)
    assert np.delete(inc_g[0, 0], truth).max() < 0.5              # no absent phase is read as present (R29: converged)


@pytest.mark.skipif(not __import__("os").environ.get("XRDVI_LONG"), reason="8 min of fp64 oracle: set XRDVI_LONG=1")
def test_config1_full_fit_2000_iterations_inclusion_parity():
    d_inc, inc_g, inc_r, wl = _fit_parity(2000)
    truth = wl.true_phases[0]
    print("max |dP_incl| =", d_inc, "planted", truth, "P_incl(GPU) planted", inc_g[0, 0, truth],
          "largest absent", np.delete(inc_g[0, 0], truth).max())
    assert np.all(inc_g[0, 0, truth] > 0.99)
