"""Pins of the oracle's peak-asymmetry extension (reading R30) -- CPU only.

The paper's profile function has a fifth parameter per phase, the asymmetry alpha_k (A9/A10, PAPER.md:234-239:
A(x; alpha) = alpha for x >= rho, 1 below), with prior alpha_k ~ Norm(1.00, 0.20) (B.2), and names a
sec(.) width term; the equations that USE A and sec are missing from PAPER.md.  Reading R30: A multiplies
the WIDTH on the high-angle side at unchanged height (continuous at x = rho, area (1 + alpha) / 2); the sec term is the
angle-dependent width w_k sec(p_m / 2).  Everything here checks oracle/xrdvi_oracle.c against something other than
itself: the symmetric oracle (already pinned), scipy pdfs, quadrature, closed forms, finite differences, Philox words.
"""
import math

import numpy as np
import pytest
import scipy.integrate
import scipy.stats

from oracle import xrdvi_oracle as orc
from paper_2501_09308_b200 import synth

from test_oracle_pins import FWHM_TO_SIGMA, rand_zeta, tiny_problem


def rand_zeta5(rng, K):
    z = np.empty((K, 5))
    z[:, :4] = rand_zeta(rng, K)
    z[:, 4] = rng.normal(0.0, 0.2, K)
    return z


# --------------------------------------------------------------------------- the split shape
@pytest.mark.parametrize("w,r,alpha", [(0.05, 0.0, 1.4), (0.1, 0.4, 0.7), (0.3, 1.0, 1.25)])
def test_split_shape_sides_area_continuity_and_half_height(w, r, alpha):
    rho = 31.7
    xs = np.concatenate([rho - np.geomspace(1e-4, 5.0, 40), rho + np.geomspace(1e-4, 5.0, 40)])
    for x in xs:
        v = orc.pseudo_voigt_asym(x, rho, w, r, alpha)
        wa = w * (alpha if x >= rho else 1.0)                 # A9: the high-angle side is alpha times wider ...
        scale = alpha if x >= rho else 1.0                    # ... at the height of width w
        ref = scale * ((1 - r) * scipy.stats.norm.pdf(x, rho, wa * FWHM_TO_SIGMA)
                       + r * scipy.stats.cauchy.pdf(x, rho, wa / 2))
        assert v == pytest.approx(ref, rel=1e-12)
    # continuity at the peak position, where both sides take the symmetric peak height
    top = orc.pseudo_voigt(rho, rho, w, r)
    assert orc.pseudo_voigt_asym(rho, rho, w, r, alpha) == top
    assert orc.pseudo_voigt_asym(rho - 1e-13, rho, w, r, alpha) == pytest.approx(top, rel=1e-9)
    # half height at rho - w/2 and at rho + alpha w/2
    assert orc.pseudo_voigt_asym(rho - w / 2, rho, w, r, alpha) == pytest.approx(top / 2, rel=1e-12)
    assert orc.pseudo_voigt_asym(rho + alpha * w / 2, rho, w, r, alpha) == pytest.approx(top / 2, rel=1e-12)
    # area: each half scales with its width -> (1 + alpha) / 2 minus the Lorentzian tails beyond +-X
    X = 400.0
    lo, _ = scipy.integrate.quad(lambda x: orc.pseudo_voigt_asym(x, rho, w, r, alpha), rho - X, rho, limit=400,
                                 points=[rho - 5 * w], epsabs=0, epsrel=1e-11)
    hi, _ = scipy.integrate.quad(lambda x: orc.pseudo_voigt_asym(x, rho, w, r, alpha), rho, rho + X, limit=400,
                                 points=[rho + 5 * w * alpha], epsabs=0, epsrel=1e-11)
    tail = lambda width: r * (0.5 - math.atan(2 * X / width) / math.pi)   # Cauchy mass beyond X on one side
    assert lo == pytest.approx(0.5 - tail(w), rel=1e-9)
    assert hi == pytest.approx(alpha * (0.5 - tail(alpha * w)), rel=1e-9)
    assert lo + hi == pytest.approx((1 + alpha) / 2, abs=2 * r * alpha * w / (math.pi * X) * 1.01 + 1e-9)


def test_alpha_one_is_the_symmetric_model_bit_for_bit():
    """zeta_alpha = 0 (alpha = 1): profile, ll and the four old gradient classes equal the symmetric oracle exactly;
    log prior + Jacobian differs by the alpha term alone."""
    for W in (0.0, 10.0):
        o4, rng = tiny_problem(window_W=W)
        o5, _ = tiny_problem(window_W=W, asymmetry=1)
        assert (o4.C, o5.C) == (4, 5)
        z4 = rand_zeta(rng, o4.K)
        z5 = np.concatenate([z4, np.zeros((o4.K, 1))], axis=1)
        np.testing.assert_array_equal(o5.profile(z5), o4.profile(z4))
        ll4, lpj4, g4 = o4.logjoint_grad(z4)
        ll5, lpj5, g5 = o5.logjoint_grad(z5)
        assert ll5 == ll4
        np.testing.assert_array_equal(g5[:, :4], g4)
        assert lpj5 - lpj4 == pytest.approx(o4.K * scipy.stats.norm.logpdf(1.0, 1.0, 0.2), rel=1e-12)


def test_profile_is_a_sum_of_split_library_pdfs_and_only_the_high_side_moves():
    o, rng = tiny_problem(asymmetry=1, window_W=0.0)
    z = rand_zeta5(rng, o.K)
    h, mu, w, r, al = np.exp(z[:, 0]), z[:, 1], np.exp(z[:, 2]), 1 / (1 + np.exp(-z[:, 3])), np.exp(z[:, 4])
    f = o.B[0].copy()
    for k in range(o.K):
        for m in range(o.ofs[k], o.ofs[k + 1]):
            rho = o.pos[m] + mu[k]
            hi = o.x >= rho
            wa = np.where(hi, al[k] * w[k], w[k])
            v = np.where(hi, al[k], 1.0) * ((1 - r[k]) * scipy.stats.norm.pdf(o.x, rho, wa * FWHM_TO_SIGMA)
                                            + r[k] * scipy.stats.cauchy.pdf(o.x, rho, wa / 2))
            f += h[k] * o.inten[m] * v
    np.testing.assert_allclose(o.profile(z), f, rtol=1e-12)
    # one peak, one phase: changing alpha leaves every point below the peak position untouched
    x = 20.0 + 0.02 * np.arange(301)
    one = orc.Oracle(x, np.ones(301), None, [0, 1], [23.004], [50.0], window_W=0.0, asymmetry=1, noise_sigma=1.0,
                     lambda_h=1.0)
    za = np.array([[0.0, 0.003, math.log(0.1), 0.3, math.log(0.8)]])
    zb = za.copy()
    zb[0, 4] = math.log(1.3)
    fa, fb = one.profile(za), one.profile(zb)
    below = x < 23.004 + 0.003
    np.testing.assert_array_equal(fa[below], fb[below])
    assert np.all(fb[~below] > fa[~below])


def test_sec_width_term_is_the_peak_by_peak_width_factor():
    """hyper.width_sec: w_mk = w_k sec(p_m / 2), p_m in degrees of 2 theta (the sec of, size-broadening
    form), at the table position: a profile of single-peak phases equals the plain profile with each width scaled."""
    x = 60.0 + 0.02 * np.arange(1501)                           # 60 .. 90 deg: sec(theta) = 1.155 .. 1.414
    pos = np.array([63.0, 71.5, 84.25])
    ofs = np.arange(4, dtype=np.int64)
    inten = np.array([40.0, 100.0, 70.0])
    hp = dict(window_W=0.0, noise_sigma=1.0, lambda_h=1.0)
    o_sec = orc.Oracle(x, np.ones(1501), None, ofs, pos, inten, width_sec=1, **hp)
    o_pl = orc.Oracle(x, np.ones(1501), None, ofs, pos, inten, **hp)
    z = np.array([[0.2, 0.01, math.log(0.08), -0.5], [-0.3, -0.02, math.log(0.12), 0.9], [0.0, 0.0, math.log(0.1), 0.0]])
    zs = z.copy()
    zs[:, 2] += np.log(1.0 / np.cos(np.radians(pos / 2)))        # the same widths, put in by hand
    np.testing.assert_allclose(o_sec.profile(z), o_pl.profile(zs), rtol=1e-13)
    # with several peaks per phase the factor differs peak by peak: finite differences pin the gradient
    wl = synth.make_workload(0)
    o = orc.from_workload(wl, width_sec=1, asymmetry=1)
    check_logjoint_fd(o, seed=5)


# --------------------------------------------------------------------------- gradients
def check_logjoint_fd(o, seed):
    rng = np.random.default_rng(seed)
    z = rand_zeta5(rng, o.K) if o.C == 5 else rand_zeta(rng, o.K)
    z[:, 0] = math.log(o.lambda_h() ** -1 / o.K) + rng.normal(0, 0.3, o.K)
    ll, lpj, g = o.logjoint_grad(z)
    assert ll == pytest.approx(o.loglik(o.profile(z)), rel=1e-14)
    assert lpj == pytest.approx(o.logprior_jac(z), rel=1e-14)
    for k in range(o.K):
        for c in range(o.C):
            hstep = 1e-6
            zp, zm = z.copy(), z.copy()
            zp[k, c] += hstep
            zm[k, c] -= hstep
            fd = ((o.loglik(o.profile(zp)) + o.logprior_jac(zp))
                  - (o.loglik(o.profile(zm)) + o.logprior_jac(zm))) / (2 * hstep)
            assert g[k, c] == pytest.approx(fd, rel=5e-6, abs=2e-6 * np.abs(g).max()), (k, c)


@pytest.mark.parametrize("W,likelihood", [(0.0, 0), (10.0, 0), (10.0, 1)])
def test_logjoint_gradient_in_all_five_classes_by_central_differences(W, likelihood):
    """The split shape has a kink at x = rho (A9), but the sums over grid points are differentiable wherever no grid
    point sits exactly on a peak centre: central differences of the log-joint pin all five classes."""
    wl = synth.make_workload(0, peak_counts=2.0e4) if likelihood else synth.make_workload(0)
    o = orc.from_workload(wl, window_W=W, asymmetry=1)
    check_logjoint_fd(o, seed=3)


def test_elbo_gradient_by_central_differences_of_fixed_draw_estimator():
    wl = synth.make_workload(0)
    o = orc.from_workload(wl, asymmetry=1)
    S, seed, it = 4, 99, 5
    st = synth.random_state(o.K, 1, 1, seed=1, classes=5).astype(np.float64)
    st[0, 0, 0, :, 0] += math.log(1.0 / o.lambda_h()) + 1.0
    elbo, grad = o.elbo_grad(st, S, seed, it)
    assert grad.shape == (1, 1, 2, o.K, 5)
    rng = np.random.default_rng(0)
    scale = np.abs(grad).max()
    picks = [(0, 0, ml, k, 4) for ml in (0, 1) for k in range(o.K)]          # every alpha entry ...
    picks += [tuple(int(v) for v in (0, 0, rng.integers(2), rng.integers(o.K), rng.integers(4))) for _ in range(8)]
    for j in picks:
        hstep = 1e-6
        sp, sm = st.copy(), st.copy()
        sp[j] += hstep
        sm[j] -= hstep
        fd = (o.elbo_grad(sp, S, seed, it)[0][0, 0] - o.elbo_grad(sm, S, seed, it)[0][0, 0]) / (2 * hstep)
        assert grad[j] == pytest.approx(fd, rel=5e-6, abs=2e-7 * scale), j


# --------------------------------------------------------------------------- prior, draws, initial state
def test_alpha_prior_jacobian_and_its_closed_form_expectation():
    o, rng = tiny_problem(K=1, M=2, asymmetry=1)
    o4, _ = tiny_problem(K=1, M=2)
    z = rand_zeta5(rng, 1)
    al = math.exp(z[0, 4])
    extra = scipy.stats.norm.logpdf(al, 1.0, 0.2) + z[0, 4]                  # B.2 + log |d alpha / d zeta|
    assert o.logprior_jac(z) - o4.logprior_jac(z[:, :4]) == pytest.approx(extra, rel=1e-12)
    # E_q of the alpha term in closed form: E[(e^zeta - 1)^2] = e^{2m + 2s^2} - 2 e^{m + s^2/2} + 1
    m, s = 0.15, 0.2
    closed = -(math.exp(2 * m + 2 * s * s) - 2 * math.exp(m + s * s / 2) + 1) / (2 * 0.2 ** 2) \
        - math.log(0.2 * math.sqrt(2 * math.pi)) + m
    n = 40000
    vals = np.empty(n)
    z0 = np.array([[0.0, 0.0, math.log(0.1), 0.0, 0.0]])
    base = o.logprior_jac(z0) - (scipy.stats.norm.logpdf(1.0, 1.0, 0.2))
    for i in range(n):
        zi = z0.copy()
        zi[0, 4] = m + s * orc.eps_alpha(2024, 3, 0, i, 0)
        vals[i] = o.logprior_jac(zi) - base
    se = vals.std(ddof=1) / math.sqrt(n)
    assert abs(vals.mean() - closed) < 4.0 * se


def test_fifth_normal_is_box_muller_of_a_second_philox_call():
    seed, it, inst, s, k = (5 << 32) | 77, 12, 3, 41, 7
    w = orc.philox4x32_10([it, s, k | 0x80000000, inst], [seed & 0xFFFFFFFF, seed >> 32])
    u0, u1 = ((w[0] >> 9) + 0.5) / 2 ** 23, ((w[1] >> 9) + 0.5) / 2 ** 23
    assert orc.eps_alpha(seed, it, inst, s, k) == pytest.approx(math.sqrt(-2 * math.log(u0)) * math.cos(2 * math.pi * u1),
                                                                rel=1e-14)
    assert abs(orc.eps_alpha(seed, it, inst, s, k) - orc.eps(seed, it, inst, s, k)[0]) > 1e-6   # not the first call's
    e = np.array([orc.eps_alpha(9, 1, 0, i, 0) for i in range(200000)])
    assert abs(e.mean()) < 0.01 and abs(e.var() - 1.0) < 0.01 and abs(scipy.stats.kurtosis(e)) < 0.05


def test_elbo_is_mean_of_logjoint_plus_entropy_with_five_classes():
    wl = synth.make_workload(0)
    o = orc.from_workload(wl, asymmetry=1)
    S, seed, it = 3, 5, 2
    st = o.init_state()
    assert st.shape == (1, 1, 2, o.K, 5) and np.all(st[0, 0, 0, :, 4] == 0.0)      # alpha starts at 1
    np.testing.assert_array_equal(st[..., :4], orc.from_workload(wl).init_state())
    st[0, 0, 0, :, 4] = 0.1
    elbo, grad, ll = o.elbo_grad(st, S, seed, it, want_ll=True)
    acc = 0.0
    for s in range(S):
        z = np.empty((o.K, 5))
        for k in range(o.K):
            e5 = np.concatenate([orc.eps(seed, it, 0, s, k), [orc.eps_alpha(seed, it, 0, s, k)]])
            z[k] = st[0, 0, 0, k] + np.exp(st[0, 0, 1, k]) * e5
        l1, l2, _ = o.logjoint_grad(z)
        assert ll[0, 0, s] == pytest.approx(l1, rel=1e-14)
        acc += l1 + l2
    ent = (st[0, 0, 1] + 0.5 * math.log(2 * math.pi * math.e)).sum()
    assert elbo[0, 0] == pytest.approx(acc / S + ent, rel=1e-13)


def test_restart_jitter_of_alpha():
    wl = synth.make_workload(0, n_restarts=3)
    o = orc.from_workload(wl, asymmetry=1)
    st = o.init_state(seed=4)
    w = orc.philox4x32_10([0xFFFFFFFF, 2, 1 | 0x80000000, 0], [4, 0])
    u0, u1 = ((w[0] >> 9) + 0.5) / 2 ** 23, ((w[1] >> 9) + 0.5) / 2 ** 23
    assert st[0, 2, 0, 1, 4] == pytest.approx(0.05 * math.sqrt(-2 * math.log(u0)) * math.cos(2 * math.pi * u1), rel=1e-12)
    assert np.all(st[0, 0, 0, :, 4] == 0.0)


# --------------------------------------------------------------------------- read-outs, windows, fit
def test_readouts_with_the_area_factor_and_the_alpha_marginal():
    o, rng = tiny_problem(asymmetry=1)
    st = synth.random_state(o.K, 1, 1, seed=3, classes=5).astype(np.float64)
    inc, area = o.inclusion(st, want_area=True)
    A = np.array([o.inten[o.ofs[k]:o.ofs[k + 1]].sum() for k in range(o.K)])
    m, s = st[0, 0, 0], np.exp(st[0, 0, 1])
    Ea = scipy.stats.lognorm.mean(s[:, 4], scale=np.exp(m[:, 4]))
    Aeff = A * (1 + Ea) / 2                                                   # area of a split peak: (1 + alpha) / 2
    Eh = scipy.stats.lognorm.mean(s[:, 0], scale=np.exp(m[:, 0]))
    Tbar = (Aeff * Eh).sum()
    np.testing.assert_allclose(inc[0, 0], scipy.stats.lognorm.sf(0.01 * Tbar / Aeff, s[:, 0], scale=np.exp(m[:, 0])),
                               rtol=1e-10, atol=1e-14)
    np.testing.assert_allclose(area[0, 0], Aeff * Eh / Tbar, rtol=1e-12)
    summ = o.posterior_summary(st)
    assert summ.shape == (1, 1, o.K, 5, 5)
    for k in range(o.K):
        d = scipy.stats.lognorm(s[k, 4], scale=math.exp(m[k, 4]))
        np.testing.assert_allclose(summ[0, 0, k, 4], [d.mean(), d.std(), d.ppf(0.025), d.ppf(0.5), d.ppf(0.975)], rtol=1e-9)
    np.testing.assert_allclose(summ[0, 0, :, :4], orc.Oracle(o.x, o.y, o.B, o.ofs, o.pos, o.inten, **{
        **o.hyper, "asymmetry": 0}).posterior_summary(st[..., :4])[0, 0], rtol=1e-12)


def test_adaptive_window_rule_covers_the_wider_side():
    wl = synth.make_workload(1, K=4)
    o = orc.from_workload(wl, asymmetry=1)
    st = o.init_state()
    st[0, 0, 0, :, 2] = math.log(0.05)
    st[0, 0, 1, :, 2] = -12.0
    st[0, 0, 0, :, 4] = np.log([1.0, 1.5, 0.6, 1.9])
    st[0, 0, 1, :, 4] = -12.0
    n = o.adaptive_halfwidths(st, 10.0)
    # W E[w] max(1, E[alpha]) / Delta = 10 * 0.05 * (1, 1.5, 1, 1.9) / 0.02 = 25, 37.5, 25, 47.5 -> ceil
    np.testing.assert_array_equal(n, [25, 38, 25, 48])


def test_fit_recovers_planted_asymmetry():
    """Config-0 recipe with split peaks (alpha ~ U(0.75, 1.35) per planted phase) on a grid that resolves them: the
    asymmetric model recovers alpha of every planted phase; the symmetric model fits the same data worse."""
    wl = synth.make_workload(0, grid=(10.0, 45.0, 1751), asym=(0.75, 1.35))
    o5 = orc.from_workload(wl)
    assert o5.C == 5
    st5, _, tr5 = o5.fit(o5.init_state(), 600, wl.S, seed=11, want_trace=True)
    for k, prm in wl.true_params[0].items():
        a_fit = math.exp(st5[0, 0, 0, k, 4])
        assert a_fit == pytest.approx(prm[4], abs=0.1), (k, prm[4])   # narrow peaks (3 points per FWHM) lean to the prior
        assert (a_fit - 1.0) * (prm[4] - 1.0) > 0.0                   # ... but on the right side of 1
        assert math.exp(st5[0, 0, 0, k, 0]) == pytest.approx(prm[0], rel=0.1)
        assert math.exp(st5[0, 0, 0, k, 2]) == pytest.approx(prm[2], rel=0.2)
    o4 = orc.from_workload(wl, asymmetry=0)
    st4, _, tr4 = o4.fit(o4.init_state(), 600, wl.S, seed=11, want_trace=True)
    assert tr5[-50:].mean() > tr4[-50:].mean() + 20.0          # measured: 36 nats
