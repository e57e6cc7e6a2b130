"""Brute force over all 2^K phase combinations at tiny K, against the variational inclusion
probabilities of the fp64 oracle (BASELINE.json north_star; SURVEY.md 8(c) "Pins": inclusion).

The discrete problem the paper replaces (2^K indicator combinations) is enumerated
exactly for K = 6: for every subset gamma the nuisances (mu, w, r) are fixed at the fitted variational
means and the evidence is integrated EXACTLY over the scales h_gamma >= 0:

    Z_gamma = int_{h >= 0} prod_k lambda e^{-lambda h_k} N(y; B + C_gamma^T h, sigma_n^2) dh
            = c_0 lambda^{|g|} (2 pi)^{|g|/2} |Lam|^{-1/2} exp(b^T Lam^{-1} b / 2) Pr[N(Lam^{-1} b, Lam^{-1}) >= 0]

with Lam = C C^T / sigma_n^2, b = C (y - B) / sigma_n^2 - lambda 1 (completing the square; c_0 is common to
all subsets), the orthant probability from scipy's multivariate-normal cdf (Genz).  Uniform prior over
subsets.  This is independent of the variational machinery (no q, no ELBO, no Adam): it only uses the
oracle's per-phase unit profile, which test_oracle_pins.py pins against scipy pdfs.

Criterion: the maximum-evidence subset equals {k : P_incl(k) > 1/2} and equals the planted
set; every phase falls on the same side of 1/2 under both; max |difference| is bounded.  The Occam factor
makes exact inclusion of absent phases small but not zero (measured here: 0.002-0.18).  The criterion is asserted on
P_incl itself (the R15 read-out at incl_tau = 1 %) for a converged fit on a grid that resolves the peaks; what happens
on config 0's own undersampled grid and after its own 500 iterations is DESIGN.md reading R29 and is asserted too.
"""
import functools
import itertools
import math

import numpy as np
import pytest
import scipy.stats

from oracle import xrdvi_oracle as orc
from paper_2501_09308_b200 import synth


def unit_profiles(o, zeta):
    """C_k(x_i): windowed profile of phase k alone at h_k = 1 and the nuisances of `zeta` (via the oracle's
    profile function and its linearity in h, which is pinned separately)."""
    C = np.empty((o.K, o.N))
    for k in range(o.K):
        z = zeta.copy()
        z[:, 0] = -745.0            # exp(-745) = 5e-324: the other phases contribute nothing
        z[k, 0] = 0.0
        C[k] = o.profile(z) - o.B[0]
    return C


def log_evidence(C, resid, sigma_n, lam):
    g = C.shape[0]
    if g == 0:
        return 0.0
    Lam = C @ C.T / sigma_n ** 2
    b = C @ resid / sigma_n ** 2 - lam
    cov = np.linalg.inv(Lam)
    cov = 0.5 * (cov + cov.T)
    hhat = cov @ b
    sign, logdet = np.linalg.slogdet(Lam)
    assert sign > 0
    if g == 1:
        orth = scipy.stats.norm.sf(0.0, loc=hhat[0], scale=math.sqrt(cov[0, 0]))
    else:
        # Pr[X >= 0] = Pr[-X <= 0]
        orth = scipy.stats.multivariate_normal.cdf(np.zeros(g), mean=-hhat, cov=cov, maxpts=200000 * g,
                                                   abseps=1e-10, releps=1e-10)
    return g * math.log(lam) + 0.5 * g * math.log(2 * math.pi) - 0.5 * logdet + 0.5 * b @ hhat + math.log(max(orth, 1e-300))


RESOLVED_GRID = (10.0, 80.0, 3501)      # config-0 recipe on a 0.02 deg grid that resolves the 0.05-0.15 deg peaks
ITS_CONVERGED = 2000                     # absent-phase scales decay slowly under Adam (R29)


@functools.lru_cache(maxsize=None)
def fitted(seed, resolved, its):
    wl = synth.make_workload(0, seed=seed, grid=RESOLVED_GRID if resolved else None)
    o = orc.from_workload(wl)
    assert o.K == 6
    st, _, _ = o.fit(o.init_state(), its, wl.S, seed=11)
    return wl, o, st


def exact_posterior(o, st):
    """All 64 subsets with the nuisances at the variational means: exact inclusion probability of every phase,
    the maximum-evidence subset, and the noise-limited ("detection-limit") area ratio of every phase, i.e. the
    exact posterior sd of h_k in the full linear model times A_k over the fitted total area."""
    zeta = st[0, 0, 0].copy()
    C = unit_profiles(o, zeta)
    resid = o.y[0] - o.B[0]
    sig, lam = o.sigma_n(), o.lambda_h()
    subsets, logZ = [], []
    for n in range(o.K + 1):
        for g in itertools.combinations(range(o.K), n):
            subsets.append(g)
            logZ.append(log_evidence(C[list(g)], resid, sig, lam))
    logZ = np.array(logZ)
    post = np.exp(logZ - logZ.max())
    post /= post.sum()
    inc_bf = np.array([sum(p for g, p in zip(subsets, post) if k in g) for k in range(o.K)])
    cov = np.linalg.inv(C @ C.T / sig ** 2)
    hhat = cov @ (C @ resid / sig ** 2 - lam)
    A = np.array([o.inten[o.ofs[k]:o.ofs[k + 1]].sum() for k in range(o.K)])
    detlim = np.sqrt(np.diag(cov)) * A / (A * np.maximum(hhat, 0.0)).sum()
    return inc_bf, subsets[int(np.argmax(post))], detlim


@pytest.mark.parametrize("seed", [1000, 2024])
def test_variational_inclusion_probability_against_all_64_subsets(seed):
    """The pin north_star asks for, on P_incl ITSELF (R15 read-out at the model's own incl_tau = 1 %):
    {k : P_incl(k) > 1/2} = maximum-evidence subset = planted set, every phase on the same side of 1/2 under the
    exact posterior and under q, and the absent phases' probabilities close.  Instance: config-0 recipe on a grid that
    resolves the peaks, fitted to convergence (R29)."""
    wl, o, st = fitted(seed, True, ITS_CONVERGED)
    inc_vi = o.inclusion(st)[0, 0]
    inc_bf, best, detlim = exact_posterior(o, st)
    truth = tuple(sorted(wl.true_phases[0]))
    absent = [k for k in range(o.K) if k not in truth]
    tau = o.hyper["incl_tau"]
    assert best == truth                                              # exact posterior mode = planted set
    assert tuple(k for k in range(o.K) if inc_vi[k] > 0.5) == truth   # variational read-out: the same set
    for k in range(o.K):
        assert (inc_bf[k] > 0.5) == (inc_vi[k] > 0.5) == (k in truth)
    assert np.abs(inc_bf - inc_vi)[list(truth)].max() < 1e-3          # true phases: both say "certainly in"
    assert inc_vi[absent].max() < 0.15 and inc_bf[absent].max() < 0.25
    assert np.abs(inc_bf - inc_vi)[absent].max() < 0.2                # Occam factor vs area threshold: close, not equal
    assert detlim.max() < 0.75 * tau                                  # the instance is decidable at tau (R29)
    print("absent phases: exact", inc_bf[absent], "variational", inc_vi[absent], "noise-limited area", detlim[absent])


@pytest.mark.parametrize("seed", [1000, 2024])
def test_inclusion_on_config0_grid_and_its_documented_exception(seed):
    """Config 0 proper (0.07 deg grid, peaks of 0.05-0.15 deg FWHM undersampled): the noise-limited area of an absent
    phase is 0.4-0.8 % of the total, i.e. comparable with tau = 1 %, so the area-ratio read-out R15 cannot decide every
    absent phase (R29).  Rule asserted here: true phases are in under both; an absent phase is out under
    both UNLESS its noise-limited area is >= 0.75 tau (seed 1000 has one such phase: P_incl = 0.52, exact 0.03)."""
    wl, o, st = fitted(seed, False, ITS_CONVERGED)
    inc_vi = o.inclusion(st)[0, 0]
    inc_bf, best, detlim = exact_posterior(o, st)
    truth = tuple(sorted(wl.true_phases[0]))
    tau = o.hyper["incl_tau"]
    assert best == truth
    undecided = []
    for k in range(o.K):
        if k in truth:
            assert inc_vi[k] > 0.99 and inc_bf[k] > 0.99
            continue
        assert inc_bf[k] < 0.35
        if inc_vi[k] >= 0.5:
            assert detlim[k] >= 0.75 * tau, (k, inc_vi[k], detlim[k])
            undecided.append(k)
        assert inc_vi[k] < 0.6                                         # never "certainly in"
    assert len(undecided) == (1 if seed == 1000 else 0)
    print("undecided absent phases", undecided, "variational", inc_vi, "exact", inc_bf, "noise-limited area", detlim)


def test_absent_phases_have_not_converged_after_500_iterations():
    """R29, first half: config 0's own 500 iterations leave the absent phases' scales above their noise limit -- their
    area ratios are still falling (2.2 % -> 0.7 %, 1.9 % -> 1.2 % between 500 and 2000 steps at seed 1000), so at 500
    steps P_incl of an absent phase can read 0.99.  The GPU-vs-oracle 0.02 gate at 500 steps compares such values."""
    wl, o, st500 = fitted(1000, False, 500)
    _, _, st2000 = fitted(1000, False, ITS_CONVERGED)
    truth = sorted(wl.true_phases[0])
    absent = [k for k in range(o.K) if k not in truth]
    inc500, area500 = (a[0, 0] for a in o.inclusion(st500, want_area=True))
    inc2000, area2000 = (a[0, 0] for a in o.inclusion(st2000, want_area=True))
    assert inc500[truth].min() > 0.99 and inc2000[truth].min() > 0.99
    assert area500[absent].max() > 1.5 * area2000[absent].max()       # still shrinking
    assert inc500[absent].max() > 0.9 and inc2000[absent].max() < 0.6
    assert np.all(area2000[absent] < area500[absent] + 1e-3)


def test_subset_evidence_one_dimensional_closed_form():
    """The building block against direct quadrature in one dimension (a plausible sign / factor slip in the
    completed square fails here)."""
    rng = np.random.default_rng(3)
    N = 60
    c = np.abs(rng.normal(0, 1, N))
    sigma_n, lam = 0.7, 1.3
    y = 0.8 * c + rng.normal(0, sigma_n, N)
    import scipy.integrate
    f = lambda h: lam * math.exp(-lam * h) * math.exp(-0.5 * ((y - c * h) ** 2).sum() / sigma_n ** 2
                                                       + 0.5 * (y ** 2).sum() / sigma_n ** 2)
    ref, _ = scipy.integrate.quad(f, 0, 10, epsabs=0, epsrel=1e-11, limit=400)
    got = math.exp(log_evidence(c[None, :], y, sigma_n, lam))
    assert got == pytest.approx(ref, rel=1e-8)


def test_elbo_is_a_lower_bound_on_the_exact_log_evidence():
    """Pins the ABSOLUTE value of the ELBO (all normalising constants, Jacobians, entropy): with the nuisances
    (mu, w, r) frozen (variational sd e^-12) the model has only the scales h, whose evidence is exact (the full-set
    term of the 2^K enumeration above).  ELBO_h = ELBO - [log prior + log Jacobian + entropy of the frozen
    coordinates] must not exceed ln Z_h, and after a fit the gap (= KL(q_h || posterior)) is a few nats."""
    wl = synth.make_workload(0)
    o = orc.from_workload(wl)
    st, _, _ = o.fit(o.init_state(), 500, wl.S, seed=11)
    st = st.copy()
    st[0, 0, 1, :, 1:] = -12.0                                   # freeze mu, w, r at their variational means
    zeta = st[0, 0, 0]
    hy = o.hyper
    frozen = 0.0
    for k in range(o.K):
        mu, zw, zr = zeta[k, 1], zeta[k, 2], zeta[k, 3]
        w, r = math.exp(zw), 1.0 / (1.0 + math.exp(-zr))
        frozen += scipy.stats.norm.logpdf(mu, 0.0, hy["mu_sigma"])                                   # B.2
        frozen += scipy.stats.gamma.logpdf(w, hy["w_shape"], scale=1.0 / hy["w_rate"]) + zw          # + log |dw/dzeta|
        frozen += scipy.stats.uniform.logpdf(r) + math.log(r) + math.log(1.0 - r)                    # + log |dr/dzeta|
        frozen += 3 * (-12.0 + 0.5 * math.log(2 * math.pi * math.e))                                 # entropy of the 3
    # exact log evidence over h >= 0 with the nuisances fixed: all K phases included
    C = unit_profiles(o, zeta)
    resid = o.y[0] - o.B[0]
    sig, lam = o.sigma_n(), o.lambda_h()
    ln_c0 = -0.5 * float(resid @ resid) / sig ** 2 - o.N * math.log(sig) - 0.5 * o.N * math.log(2 * math.pi)
    ln_z = ln_c0 + log_evidence(C, resid, sig, lam)

    S = 4096
    vals = []
    for it in range(4):                                          # four independent draws sets: mean and its error
        elbo, _ = o.elbo_grad(st, S, 77, 100 + it)
        vals.append(elbo[0, 0] - frozen)
    elbo_h, se = float(np.mean(vals)), float(np.std(vals, ddof=1) / math.sqrt(len(vals)))
    gap = ln_z - elbo_h
    print(f"ln Z_h = {ln_z:.3f}, ELBO_h = {elbo_h:.3f} +- {se:.3f}, gap = {gap:.3f}")
    assert gap > -4.0 * se - 1e-6                                # a lower bound ...
    assert gap < 8.0                                             # ... and a tight one after the fit (KL of q_h)
    # a deliberately bad q_h (shifted by one nat in every ln h) is a much worse bound, but still a bound
    bad = st.copy()
    bad[0, 0, 0, :, 0] += 1.0
    elbo_bad = o.elbo_grad(bad, S, 77, 200)[0][0, 0] - frozen
    assert elbo_bad < elbo_h - 10.0 and elbo_bad < ln_z
