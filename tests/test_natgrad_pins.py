"""Pins of the oracle's natural-gradient update (hyper.optimizer = 1, reading R25; north_star:
"an Adam/natural-gradient update kernel") against things other than its own formula:
the Fisher metric of a Gaussian in (m, ln sigma) from a numerical KL Hessian, the covariance of the step under
a rescaling of the latent coordinate, and the one-step solution of a Gaussian target."""
import math

import numpy as np
import pytest

from oracle import xrdvi_oracle as orc
from paper_2501_09308_b200 import synth


def oracle(lr):
    wl = synth.make_workload(0)
    return orc.from_workload(wl, optimizer=1, lr=lr), wl


def kl_gauss(m1, s1, m0, s0):
    """KL( N(m1, s1^2) || N(m0, s0^2) ), textbook closed form."""
    return math.log(s0 / s1) + (s1 * s1 + (m1 - m0) ** 2) / (2 * s0 * s0) - 0.5


def test_step_uses_the_fisher_metric_of_the_gaussian_family():
    """F = Hessian of KL(q_theta+d || q_theta) at d = 0 in theta = (m, l); the step must be lr F^-1 grad."""
    o, wl = oracle(lr=0.37)
    rng = np.random.default_rng(0)
    st = synth.random_state(o.K, 1, 1, seed=2).astype(np.float64)
    g = rng.normal(0, 1.0, st.shape) * 1e-3
    new = o.natgrad_step(st, g)
    d = 1e-4
    for k, c in ((0, 0), (3, 2), (5, 3)):
        m, l = st[0, 0, 0, k, c], st[0, 0, 1, k, c]
        s = math.exp(l)
        f_mm = (kl_gauss(m + d, s, m, s) + kl_gauss(m - d, s, m, s)) / d ** 2          # = 1/s^2
        f_ll = (kl_gauss(m, s * math.exp(d), m, s) + kl_gauss(m, s * math.exp(-d), m, s)) / d ** 2   # = 2
        assert new[0, 0, 0, k, c] - m == pytest.approx(0.37 * g[0, 0, 0, k, c] / f_mm, rel=1e-5)
        assert new[0, 0, 1, k, c] - l == pytest.approx(0.37 * g[0, 0, 1, k, c] / f_ll, rel=1e-5)


def test_step_is_covariant_under_rescaling_of_the_latent():
    """zeta' = c zeta  =>  m' = c m, l' = l + ln c, dE/dm' = (dE/dm)/c, dE/dl' = dE/dl; a natural-gradient
    step commutes with the rescaling (a plain gradient step does not)."""
    o, wl = oracle(lr=0.2)
    rng = np.random.default_rng(1)
    st = synth.random_state(o.K, 1, 1, seed=3).astype(np.float64)
    g = rng.normal(0, 0.05, st.shape)
    c = 3.7
    st2, g2 = st.copy(), g.copy()
    st2[:, :, 0] *= c
    st2[:, :, 1] += math.log(c)
    g2[:, :, 0] /= c
    a, b = o.natgrad_step(st, g), o.natgrad_step(st2, g2)
    np.testing.assert_allclose(b[:, :, 0], c * a[:, :, 0], rtol=1e-12)
    np.testing.assert_allclose(b[:, :, 1], a[:, :, 1] + math.log(c), rtol=1e-12)


def test_gaussian_target_is_solved_in_one_unit_step_and_is_a_fixed_point():
    """Target N(0, s^2): ELBO(m, l) = -(m^2 + e^{2l})/(2 s^2) + l + const.  At sigma = s a step with lr = 1
    lands on m = 0; (0, ln s) does not move; l is clamped to [-12, 2]."""
    o, wl = oracle(lr=1.0)
    s = 0.3
    st = np.zeros((1, 1, 2, o.K, 4))
    st[0, 0, 0] = np.random.default_rng(2).normal(0, 1, (o.K, 4))
    st[0, 0, 1] = math.log(s)
    grad = np.empty_like(st)
    grad[0, 0, 0] = -st[0, 0, 0] / s ** 2
    grad[0, 0, 1] = -np.exp(2 * st[0, 0, 1]) / s ** 2 + 1.0
    new = o.natgrad_step(st, grad)
    np.testing.assert_allclose(new[0, 0, 0], 0.0, atol=1e-15)
    np.testing.assert_allclose(new[0, 0, 1], math.log(s), rtol=1e-15)
    again = o.natgrad_step(new, np.zeros_like(new))
    np.testing.assert_array_equal(again, new)
    big = o.natgrad_step(st, np.full_like(st, 1e3))
    assert np.all(big[0, 0, 1] == 2.0)
    small = o.natgrad_step(st, np.full_like(st, -1e3))
    assert np.all(small[0, 0, 1] == -12.0)


def test_natural_gradient_fit_increases_the_elbo():
    o, wl = oracle(lr=0.01)
    st, _, tr = o.fit(o.init_state(), 200, wl.S, seed=11, want_trace=True)
    assert np.isfinite(st).all()
    assert tr[-20:].mean() > tr[:20].mean() + 100.0
