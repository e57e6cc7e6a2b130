"""Pins of the oracle on NON-UNIFORM 2-theta grids (reading R31; xrdvi_create takes any strictly
increasing grid, "uniform fast path") -- CPU only.  The profile of A3-A8 is a function of x_i alone, so
nothing but the window bookkeeping depends on the spacing: R31 keeps the integer window |i - j_m| <= n_c of R16 with j_m the
NEAREST grid point and n_c from the mean step."""
import math

import numpy as np
import pytest
import scipy.stats

from oracle import xrdvi_oracle as orc
from paper_2501_09308_b200 import synth

from test_oracle_pins import FWHM_TO_SIGMA, rand_zeta


def jittered_grid(N=401, lo=20.0, hi=28.0, seed=2, amp=0.35):
    rng = np.random.default_rng(seed)
    step = (hi - lo) / (N - 1)
    x = lo + step * np.arange(N)
    x[1:-1] += rng.uniform(-amp, amp, N - 2) * step           # strictly increasing for amp < 0.5
    assert np.all(np.diff(x) > 0)
    return x


def problem_on(x, seed=7, K=3, M=6, **hyper):
    rng = np.random.default_rng(seed)
    ofs = np.arange(K + 1, dtype=np.int64) * M
    pos = np.concatenate([np.sort(rng.uniform(x[0] - 0.1, x[-1] + 0.1, M)) for _ in range(K)])   # some outside
    inten = rng.uniform(5.0, 100.0, K * M)
    y = rng.uniform(0.0, 50.0, x.shape[0])
    bg = 1.0 + 0.1 * (x - x[0])
    hp = dict(window_W=10.0, fwhm_ref=0.15, w_shape=3.0, w_rate=30.0, noise_sigma=2.0, lambda_h=0.7)
    hp.update(hyper)
    return orc.Oracle(x, y, bg, ofs, pos, inten, **hp), rng


def test_nearest_index_is_the_uniform_formula_on_a_uniform_grid():
    wl = synth.make_workload(1)
    x = wl.two_theta
    step = (x[-1] - x[0]) / (x.shape[0] - 1)
    pos = np.concatenate([wl.peak_pos[::7], [x[0] - 0.3, x[0] - 0.011, x[-1] + 0.011, x[-1] + 0.7]])
    for p in pos:
        j = math.floor((p - x[0]) / step + 0.5)
        d_lo, d_hi = abs(p - (x[0] + step * j)), step / 2
        if abs(d_lo - d_hi) < 1e-9:                            # an exact tie may go either way
            continue
        assert orc.nearest_index(x, p) == j


def test_windowed_profile_on_a_jittered_grid_is_the_masked_library_sum():
    x = jittered_grid()
    o, rng = problem_on(x)
    z = rand_zeta(rng, o.K)
    h, mu, w, r = np.exp(z[:, 0]), z[:, 1], np.exp(z[:, 2]), 1 / (1 + np.exp(-z[:, 3]))
    step = (x[-1] - x[0]) / (x.shape[0] - 1)
    n_c = math.ceil(10.0 * 0.15 / step - 1e-9)
    assert o.n_c == n_c
    idx = np.arange(x.shape[0])
    f = o.B[0].copy()
    pairs = 0
    for k in range(o.K):
        for m in range(o.ofs[k], o.ofs[k + 1]):
            p = o.pos[m]
            if x[0] < p < x[-1]:
                j = int(np.argmin(np.abs(x - p)))                  # nearest grid point
            else:
                j = orc.nearest_index(x, p)                        # beyond the grid: continued with the mean step
                assert j <= 0 or j >= x.shape[0] - 1
            mask = np.abs(idx - j) <= n_c
            pairs += int(mask.sum())
            rho = p + mu[k]
            v = (1 - r[k]) * scipy.stats.norm.pdf(x, rho, w[k] * FWHM_TO_SIGMA) + r[k] * scipy.stats.cauchy.pdf(x, rho, w[k] / 2)
            f += h[k] * o.inten[m] * np.where(mask, v, 0.0)
    np.testing.assert_allclose(o.profile(z), f, rtol=1e-12)
    assert o.pair_count() == pairs


def test_dense_profile_does_not_depend_on_the_other_grid_points():
    """Dense mode: f(x_i) is a function of x_i alone, so a non-uniform grid made of points of a fine uniform grid carries
    the fine grid's values bit for bit."""
    fine = 20.0 + 0.01 * np.arange(801)
    rng = np.random.default_rng(4)
    pick = np.sort(rng.choice(801, size=300, replace=False))
    pick[0], pick[-1] = 0, 800
    pick = np.unique(pick)
    x = fine[pick]
    assert np.ptp(np.diff(x)) > 0.005                            # really non-uniform
    of, _ = problem_on(fine, window_W=0.0)
    on = orc.Oracle(x, of.y[0][pick], of.B[0][pick], of.ofs, of.pos, of.inten, **{**of.hyper})
    z = rand_zeta(np.random.default_rng(1), of.K)
    np.testing.assert_array_equal(on.profile(z), of.profile(z)[pick])


def test_a_grid_uniform_to_1e_6_of_the_step_is_treated_as_uniform():
    x = 20.0 + 0.02 * np.arange(401)
    xp = x.copy()
    xp[1:-1] += np.random.default_rng(0).uniform(-4e-9, 4e-9, 399)   # 2e-7 of the step
    o1, _ = problem_on(x)
    o2, _ = problem_on(xp)
    assert o1.pair_count() == o2.pair_count()
    z = rand_zeta(np.random.default_rng(1), o1.K)
    np.testing.assert_allclose(o2.profile(z), o1.profile(z), rtol=1e-6)


@pytest.mark.parametrize("W", [0.0, 10.0])
def test_logjoint_gradient_on_a_jittered_grid_by_central_differences(W):
    x = jittered_grid(N=301, hi=26.0)
    o, rng = problem_on(x, window_W=W)
    z = rand_zeta(rng, o.K)
    ll, lpj, g = o.logjoint_grad(z)
    for k in range(o.K):
        for c in range(4):
            hstep = 1e-6
            zp, zm = z.copy(), z.copy()
            zp[k, c] += hstep
            zm[k, c] -= hstep
            fd = ((o.loglik(o.profile(zp)) + o.logprior_jac(zp)) - (o.loglik(o.profile(zm)) + o.logprior_jac(zm))) / (2 * hstep)
            assert g[k, c] == pytest.approx(fd, rel=5e-6, abs=2e-6 * np.abs(g).max())
