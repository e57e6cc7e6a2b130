"""Pins of the oracle's per-phase (adaptive) windows, reading R27 (second
half; `north_star`: "pseudo-Voigt truncated at a problem-defined +-W FWHM cutoff").  CPU only.

Checked against things other than the oracle itself: scipy pdfs summed peak by peak under a mask written out
here, the closed-form pair count, central finite differences, locality invariants, hand-computed half-widths.
"""
import math

import numpy as np
import pytest
import scipy.stats

from oracle import xrdvi_oracle as orc
from paper_2501_09308_b200 import synth

FWHM_TO_SIGMA = 1.0 / (2.0 * math.sqrt(2.0 * math.log(2.0)))


def tiny_problem(K=4, M=6, N=401, lo=20.0, hi=28.0, seed=11, **hyper):
    rng = np.random.default_rng(seed)
    x = lo + (hi - lo) * np.arange(N) / (N - 1)
    ofs = np.arange(K + 1, dtype=np.int64) * M
    pos = np.concatenate([np.sort(rng.uniform(lo - 0.2, hi + 0.2, M)) for _ in range(K)])   # some outside the grid
    inten = rng.uniform(5.0, 100.0, K * M)
    y = rng.uniform(0.0, 50.0, N)
    bg = 1.0 + 0.1 * (x - lo)
    hp = dict(window_W=10.0, fwhm_ref=0.15, w_shape=3.0, w_rate=30.0, noise_sigma=2.0, lambda_h=0.7)
    hp.update(hyper)
    return orc.Oracle(x, y, bg, ofs, pos, inten, **hp), rng


def rand_zeta(rng, K):
    z = np.empty((K, 4))
    z[:, 0] = rng.normal(-1.0, 0.5, K)
    z[:, 1] = rng.normal(0.0, 0.03, K)
    z[:, 2] = np.log(rng.uniform(0.05, 0.2, K))
    z[:, 3] = rng.normal(0.0, 1.0, K)
    return z


def masked_library_profile(o, z, n_ck):
    """sum over phases and peaks of scipy's normal / Cauchy pdfs, each masked to |i - j_m| <= n_ck[k]"""
    h, mu, w, r = np.exp(z[:, 0]), z[:, 1], np.exp(z[:, 2]), 1.0 / (1.0 + np.exp(-z[:, 3]))
    f = o.B[0].copy()
    delta = (o.x[-1] - o.x[0]) / (o.N - 1)
    idx = np.arange(o.N)
    for k in range(o.K):
        for m in range(o.ofs[k], o.ofs[k + 1]):
            rho = o.pos[m] + mu[k]
            v = ((1 - r[k]) * scipy.stats.norm.pdf(o.x, rho, w[k] * FWHM_TO_SIGMA)
                 + r[k] * scipy.stats.cauchy.pdf(o.x, rho, w[k] / 2.0))
            j = math.floor((o.pos[m] - o.x[0]) / delta + 0.5)
            f += h[k] * o.inten[m] * np.where(np.abs(idx - j) <= n_ck[k], v, 0.0)
    return f


def test_per_phase_profile_equals_masked_library_sum_and_pair_count():
    o, rng = tiny_problem()
    assert o.n_c == 75
    n_ck = np.array([75, 12, 0, 40])
    o.set_phase_windows(n_ck)
    z = rand_zeta(rng, o.K)
    f = o.profile(z)
    ref = masked_library_profile(o, z, n_ck)
    assert np.abs(f - ref).max() <= 1e-12 * np.abs(ref).max()
    # closed-form count: every peak contributes the clipped length of [j - n, j + n]
    delta = (o.x[-1] - o.x[0]) / (o.N - 1)
    count = 0
    for k in range(o.K):
        for m in range(o.ofs[k], o.ofs[k + 1]):
            j = math.floor((o.pos[m] - o.x[0]) / delta + 0.5)
            count += max(0, min(o.N - 1, j + n_ck[k]) - max(0, j - n_ck[k]) + 1)
    assert o.pair_count() == count
    # the static window is the special case n_ck = n_c, and None restores it
    static = tiny_problem()[0]
    o.set_phase_windows(np.full(o.K, 75))
    assert np.array_equal(o.profile(z), static.profile(z)) and o.pair_count() == static.pair_count()
    o.set_phase_windows(n_ck)
    o.set_phase_windows(None)
    assert np.array_equal(o.profile(z), static.profile(z))


def test_window_of_a_phase_touches_only_that_phase():
    o, rng = tiny_problem()
    z = rand_zeta(rng, o.K)
    base = o.profile(z)
    for k in range(o.K):
        n_ck = np.full(o.K, 75)
        n_ck[k] = 3
        o.set_phase_windows(n_ck)
        f = o.profile(z)
        zk = z.copy()
        zk[k, 0] = -80.0                                   # phase k switched off: the other phases' part
        others = o.profile(zk)
        o.set_phase_windows(None)
        assert not np.array_equal(f, base)                 # the narrow window does cut something ...
        assert np.allclose(others, o.profile(zk), rtol=0, atol=1e-30)   # ... but only of phase k
        # inside the narrow window nothing changes: points within 3 of every peak of phase k keep their value
        delta = (o.x[-1] - o.x[0]) / (o.N - 1)
        js = [math.floor((o.pos[m] - o.x[0]) / delta + 0.5) for m in range(o.ofs[k], o.ofs[k + 1])]
        # (a point can still lose the tail of ANOTHER peak of phase k, so compare only the cut amount's sign)
        assert np.all(f <= base + 1e-12 * np.abs(base).max())          # truncation only removes positive terms
        assert len(js) == o.ofs[k + 1] - o.ofs[k]


def test_rejected_half_widths():
    o, _ = tiny_problem()
    with pytest.raises(ValueError):
        o.set_phase_windows(np.array([76, 1, 1, 1]))       # wider than the create-time window
    with pytest.raises(ValueError):
        o.set_phase_windows(np.array([-1, 1, 1, 1]))
    dense, _ = tiny_problem(window_W=0.0)
    with pytest.raises(ValueError):
        dense.set_phase_windows(np.array([1, 1, 1, 1]))


def test_gradients_by_central_differences_with_per_phase_windows():
    wl = synth.make_workload(0)
    o = orc.from_workload(wl)
    n_ck = np.array([22, 9, 15, 4, 22, 11])
    o.set_phase_windows(n_ck)
    rng = np.random.default_rng(5)
    z = rand_zeta(rng, o.K)
    z[:, 0] = math.log(o.lambda_h() ** -1 / o.K) + rng.normal(0, 0.3, o.K)
    ll, lpj, g = o.logjoint_grad(z)
    for k in range(o.K):
        for c in range(4):
            hs = 1e-6
            zp, zm = z.copy(), z.copy()
            zp[k, c] += hs
            zm[k, c] -= hs
            fd = ((o.loglik(o.profile(zp)) + o.logprior_jac(zp))
                  - (o.loglik(o.profile(zm)) + o.logprior_jac(zm))) / (2 * hs)
            assert g[k, c] == pytest.approx(fd, rel=2e-6, abs=1e-6 * np.abs(g).max())
    # fixed-draw ELBO estimator
    S, seed, it = 4, 17, 3
    st = synth.random_state(o.K, 1, 1, seed=2).astype(np.float64)
    st[0, 0, 0, :, 0] += math.log(1.0 / o.lambda_h()) + 1.0
    elbo, grad = o.elbo_grad(st, S, seed, it)
    scale = np.abs(grad).max()
    for _ in range(12):
        j = tuple(int(v) for v in (0, 0, rng.integers(2), rng.integers(o.K), rng.integers(4)))
        sp, sm = st.copy(), st.copy()
        sp[j] += 1e-6
        sm[j] -= 1e-6
        fd = (o.elbo_grad(sp, S, seed, it)[0][0, 0] - o.elbo_grad(sm, S, seed, it)[0][0, 0]) / 2e-6
        assert grad[j] == pytest.approx(fd, rel=5e-6, abs=2e-7 * scale)


def test_refresh_rule_hand_computed():
    # config 1 grid: step 0.02 deg, static window 75 points; n_min = ceil(2 W) = 20 points
    wl = synth.make_workload(1)
    o = orc.from_workload(wl)
    assert o.n_c == 75
    K = o.K
    st = np.zeros((1, 1, 2, K, 4))
    st[0, 0, 1] = -12.0                                    # variational sd e^-12: E[w] = exp(m_w) to 1e-11
    st[0, 0, 0, :, 2] = math.log(0.1)
    # phase 0: FWHM 0.05, shift +0.03 -> (10*0.05 + 0.03)/0.02 = 26.5 -> 27
    st[0, 0, 0, 0, 2], st[0, 0, 0, 0, 1] = math.log(0.05), 0.03
    # phase 1: same with a negative shift (|mu| counts) -> 27
    st[0, 0, 0, 1, 2], st[0, 0, 0, 1, 1] = math.log(0.05), -0.03
    # phase 2: FWHM 0.2 -> 100 points -> clamped to the static 75
    st[0, 0, 0, 2, 2] = math.log(0.2)
    # phase 3: FWHM 0.01 -> 5 points -> floor n_min = 20
    st[0, 0, 0, 3, 2] = math.log(0.01)
    # phase 4: FWHM 0.1 exactly -> 50 (the 1e-9 guard keeps an exact ratio from rounding up)
    # phase 5: lognormal mean: m_w = ln 0.1, sd 0.5 -> E[w] = 0.1 e^{0.125} = 0.11331 -> 56.66 -> 57
    st[0, 0, 1, 5, 2] = math.log(0.5)
    n = o.adaptive_halfwidths(st, 10.0)
    assert list(n[:6]) == [27, 27, 75, 20, 50, 57]
    assert np.all(n[6:] == 50)
    # W scales the cutoff: W = 5 halves it (n_min = 10)
    n5 = o.adaptive_halfwidths(st, 5.0)
    assert list(n5[:6]) == [14, 14, 50, 10, 25, 29]


def test_refresh_rule_takes_the_widest_instance():
    wl = synth.make_workload(0)
    o = orc.from_workload(wl, n_restarts=3, window_W=10.0, fwhm_ref=0.3)    # step 0.07, n_c = 43, n_min = 20
    assert o.n_c == 43
    st = np.zeros((1, 3, 2, o.K, 4))
    st[:, :, 1] = -12.0
    st[:, :, 0, :, 2] = math.log(0.15)                     # 1.5 / 0.07 = 21.4 -> 22
    st[0, 1, 0, 2, 2] = math.log(0.2)                      # restart 1 widens phase 2: 2.0 / 0.07 = 28.6 -> 29
    st[0, 2, 0, 4, 1] = 0.1                                # restart 2 shifts phase 4: 1.6 / 0.07 = 22.9 -> 23
    n = o.adaptive_halfwidths(st, 10.0)
    assert list(n) == [22, 22, 29, 22, 23, 22]


def test_adaptive_fit_recovers_planted_phases_and_shrinks_the_work():
    """Config 0 (absent phases shrink to ~0 area): a fit whose windows are refreshed every 100
    steps to +-5 FWHM does 45 % less work and lands on the same phases as the static +-22-point fit.
    (Config 0's 0.07 deg grid undersamples the peaks, so absent phases sit near the 1 % threshold: the check
    is on area ratios, as in test_fit_recovers_planted_phases_config0.)"""
    wl = synth.make_workload(0)
    o = orc.from_workload(wl)
    full_pairs = o.pair_count()
    st_static, _, _ = o.fit(o.init_state(0), 500, wl.S, seed=1)
    st, hist = o.fit_adaptive(o.init_state(0), 500, wl.S, seed=1, refresh_every=100, W=5.0)
    assert len(hist) == 4 and all(h.min() >= 10 and h.max() <= 22 for h in hist)
    assert o.pair_count() < 0.6 * full_pairs
    inc, area = o.inclusion(st, want_area=True)
    inc, area = inc[0, 0], area[0, 0]
    truth = sorted(wl.true_phases[0])
    absent = [k for k in range(o.K) if k not in truth]
    assert np.all(inc[truth] > 0.99)
    assert area[truth].sum() > 0.93 and area[absent].max() < 0.03
    o.set_phase_windows(None)
    assert np.abs(inc - o.inclusion(st_static)[0, 0]).max() < 0.02
