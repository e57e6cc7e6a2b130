"""Pins of the oracle's Poisson likelihood (hyper.likelihood = 1; the paper's A12-A16, PAPER.md:247-261;
DESIGN.md reading R24) against things other than itself: scipy's Poisson log-pmf, central finite
differences, the stationarity of ll at f = y, and the paper's qualitative result on count data."""
import math

import numpy as np
import pytest
import scipy.stats

from oracle import xrdvi_oracle as orc
from paper_2501_09308_b200 import synth


def count_problem(seed=5, K=3, M=4, N=241, **hyper):
    rng = np.random.default_rng(seed)
    x = 20.0 + 0.02 * np.arange(N)
    ofs = np.arange(K + 1, dtype=np.int64) * M
    pos = np.concatenate([np.sort(rng.uniform(20.3, 24.5, M)) for _ in range(K)])
    inten = rng.uniform(5.0, 100.0, K * M)
    bg = 30.0 + 2.0 * (x - 20.0)
    y = rng.poisson(bg + 200.0 * np.exp(-0.5 * ((x - 22.0) / 0.05) ** 2)).astype(np.float64)
    hp = dict(window_W=10.0, fwhm_ref=0.15, w_rate=30.0, lambda_h=0.02, likelihood=1)
    hp.update(hyper)
    return orc.Oracle(x, y, bg, ofs, pos, inten, **hp), rng


def rand_zeta(rng, K):
    z = np.empty((K, 4))
    z[:, 0] = rng.normal(1.0, 0.5, K)
    z[:, 1] = rng.normal(0.0, 0.03, K)
    z[:, 2] = np.log(rng.uniform(0.05, 0.2, K))
    z[:, 3] = rng.normal(0.0, 1.0, K)
    return z


def test_poisson_loglik_is_scipy_logpmf_sum():
    o, rng = count_problem()
    z = rand_zeta(rng, o.K)
    f = o.profile(z)
    assert f.min() > 0
    ref = scipy.stats.poisson.logpmf(o.y[0].astype(np.int64), f).sum()
    assert o.loglik(f) == pytest.approx(ref, rel=1e-12)
    # the likelihood switch changes nothing else: same profile, same prior term as the Gaussian problem
    og, _ = count_problem(likelihood=0, noise_sigma=3.0)
    np.testing.assert_array_equal(og.profile(z), f)
    assert og.logprior_jac(z) == o.logprior_jac(z)
    assert og.loglik(f) != o.loglik(f)


def test_poisson_loglik_is_stationary_at_f_equal_y():
    """d ll / d f_i = y_i / f_i - 1 vanishes at f = y and ll is maximal there (term by term)."""
    o, rng = count_problem()
    y = np.maximum(o.y[0], 0.5)
    ll0 = o.loglik(y)
    for s in (-0.02, 0.02):
        assert o.loglik(y * (1.0 + s)) < ll0
    d = 1e-4
    assert abs(o.loglik(y * (1 + d)) - o.loglik(y * (1 - d))) < 1e-6 * abs(ll0)


@pytest.mark.parametrize("W", [0.0, 10.0])
def test_poisson_logjoint_gradient_by_central_differences(W):
    o, rng = count_problem(window_W=W)
    z = rand_zeta(rng, o.K)
    ll, lpj, g = o.logjoint_grad(z)
    assert ll == pytest.approx(o.loglik(o.profile(z)), rel=1e-14)
    for k in range(o.K):
        for c in range(4):
            d = 1e-6
            zp, zm = z.copy(), z.copy()
            zp[k, c] += d
            zm[k, c] -= d
            fp = o.loglik(o.profile(zp)) + o.logprior_jac(zp)
            fm = o.loglik(o.profile(zm)) + o.logprior_jac(zm)
            fd = (fp - fm) / (2 * d)
            assert g[k, c] == pytest.approx(fd, rel=2e-6, abs=1e-6 * np.abs(g).max())


def test_poisson_elbo_gradient_by_central_differences_of_fixed_draw_estimator():
    o, rng = count_problem()
    st = np.zeros((1, 1, 2, o.K, 4))
    st[0, 0, 0] = rand_zeta(rng, o.K)
    st[0, 0, 1] = math.log(0.05)
    e0, g = o.elbo_grad(st, 4, 9, 3)
    for idx in [(0, 0, 0, 1, 0), (0, 0, 0, 2, 2), (0, 0, 1, 0, 1), (0, 0, 1, 1, 3)]:
        d = 1e-6
        sp, sm = st.copy(), st.copy()
        sp[idx] += d
        sm[idx] -= d
        fd = (o.elbo_grad(sp, 4, 9, 3)[0][0, 0] - o.elbo_grad(sm, 4, 9, 3)[0][0, 0]) / (2 * d)
        assert g[idx] == pytest.approx(fd, rel=5e-6, abs=1e-6 * np.abs(g).max())


def test_count_data_fit_recovers_planted_phases():
    """PAPER.md:140 on synthetic COUNT data (config 0 recipe, peak 2e4 counts, Poisson noise)."""
    wl = synth.make_workload(0, peak_counts=2.0e4)
    assert wl.hyper["likelihood"] == 1 and np.all(wl.y >= 0) and np.all(wl.y == np.round(wl.y))
    o = orc.from_workload(wl)
    st, _, tr = o.fit(o.init_state(), 500, wl.S, seed=11, want_trace=True)
    inc, area = o.inclusion(st, want_area=True)
    truth = sorted(wl.true_phases[0])
    absent = [k for k in range(o.K) if k not in truth]
    assert np.all(inc[0, 0, truth] > 0.99)
    assert area[0, 0, truth].sum() > 0.93 and area[0, 0, absent].max() < 0.03
    for k in truth:
        assert math.exp(st[0, 0, 0, k, 0]) == pytest.approx(wl.true_params[0][k][0], rel=0.2)
    assert tr[-50:].mean() > tr[:50].mean()
