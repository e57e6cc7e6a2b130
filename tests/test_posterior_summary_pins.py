"""Pins of the oracle's marginal summaries (orc_posterior_summary, reading R28; SURVEY.md 8(f) NEXT-4
second half: "posterior summaries (Fig. 6-style marginals)") against things other than its own formulas:
scipy's log-normal / normal distributions, adaptive quadrature and Monte-Carlo sampling of the logit-normal,
symmetry and small-sigma limits."""
import numpy as np
import pytest
from scipy import integrate, special, stats

from oracle import xrdvi_oracle as orc
from paper_2501_09308_b200 import synth


@pytest.fixture(scope="module")
def case():
    wl = synth.make_workload(0)
    o = orc.from_workload(wl)
    st = synth.random_state(o.K, 1, 1, seed=11).astype(np.float64)
    # spread of widths of q: narrow, prior-like and wide components in every class
    st[0, 0, 1] = np.log(np.array([0.02, 0.3, 1.0, 2.5, 0.1, 0.7])[: o.K, None] * np.ones((1, 4)))
    st[0, 0, 0, :, 3] = np.array([-3.0, -0.5, 0.0, 0.4, 2.0, 5.0])[: o.K]
    return o, st, o.posterior_summary(st)[0, 0]


def test_lognormal_classes_match_scipy(case):
    o, st, out = case
    for c in (0, 2):
        for k in range(o.K):
            m, s = st[0, 0, 0, k, c], np.exp(st[0, 0, 1, k, c])
            d = stats.lognorm(s=s, scale=np.exp(m))
            assert out[k, c, 0] == pytest.approx(d.mean(), rel=1e-12)
            assert out[k, c, 1] == pytest.approx(d.std(), rel=1e-10)
            assert out[k, c, 2:] == pytest.approx(d.ppf([0.025, 0.5, 0.975]), rel=1e-10)


def test_shift_class_is_the_normal_itself(case):
    o, st, out = case
    for k in range(o.K):
        m, s = st[0, 0, 0, k, 1], np.exp(st[0, 0, 1, k, 1])
        assert out[k, 1, 0] == m and out[k, 1, 1] == s
        assert out[k, 1, 2:] == pytest.approx(stats.norm(m, s).ppf([0.025, 0.5, 0.975]), rel=1e-10, abs=1e-13)


def test_mixing_class_against_adaptive_quadrature_and_sampling(case):
    o, st, out = case
    rng = np.random.default_rng(5)
    for k in range(o.K):
        m, s = st[0, 0, 0, k, 3], np.exp(st[0, 0, 1, k, 3])
        e1 = integrate.quad(lambda z: special.expit(m + s * z) * stats.norm.pdf(z), -np.inf, np.inf, epsabs=1e-13)[0]
        e2 = integrate.quad(lambda z: special.expit(m + s * z) ** 2 * stats.norm.pdf(z), -np.inf, np.inf, epsabs=1e-13)[0]
        assert out[k, 3, 0] == pytest.approx(e1, abs=1e-10)
        assert out[k, 3, 1] == pytest.approx(np.sqrt(e2 - e1 * e1), abs=1e-8)
        r = special.expit(rng.normal(m, s, 400_000))
        assert out[k, 3, 0] == pytest.approx(r.mean(), abs=4 * r.std() / np.sqrt(r.size) + 1e-6)
        assert out[k, 3, 1] == pytest.approx(r.std(), rel=2e-2, abs=1e-5)
        assert out[k, 3, 2:] == pytest.approx(np.quantile(r, [0.025, 0.5, 0.975]), abs=5e-3)
        assert out[k, 3, 2:] == pytest.approx(special.expit(stats.norm(m, s).ppf([0.025, 0.5, 0.975])), rel=1e-10)


def test_symmetry_small_sigma_limit_and_ordering(case):
    o, st, out = case
    assert out[2, 3, 0] == pytest.approx(0.5, abs=1e-13)            # m_r = 0: logit-normal symmetric about 1/2
    assert out[2, 3, 3] == pytest.approx(0.5, abs=1e-15)
    m = st[0, 0, 0, 0, 3]                                            # sigma = 0.02: delta method
    g = special.expit(m)
    assert out[0, 3, 0] == pytest.approx(g + 0.5 * 0.02 ** 2 * g * (1 - g) * (1 - 2 * g), abs=1e-8)
    assert out[0, 3, 1] == pytest.approx(0.02 * g * (1 - g), rel=2e-3)
    tiny = st.copy()                                                 # sigma = e^-12 (the clamp of R10): no cancellation
    tiny[0, 0, 1, :, 3] = -12.0
    t = o.posterior_summary(tiny)[0, 0]
    gk = special.expit(tiny[0, 0, 0, :, 3])
    assert t[:, 3, 1] == pytest.approx(np.exp(-12.0) * gk * (1 - gk), rel=1e-6)
    assert t[:, 3, 0] == pytest.approx(gk, abs=1e-11)
    assert np.all(out[..., 2] < out[..., 3]) and np.all(out[..., 3] < out[..., 4])
    assert np.all(out[..., 1] > 0)
    assert np.all(out[:, 3, 2:] > 0) and np.all(out[:, 3, 2:] < 1) and np.all(out[:, 3, 0] < 1)
