"""Randomised small problems through the C ABI against the oracle: odd sizes (N not a multiple of 16, K = 1, phases with one
peak, tiles without any record, windows from 0 points to dense, peaks outside the grid, S not a multiple of 32, several
patterns x restarts), every likelihood / model switch.  These hit the table builder's corners (record-granular share cuts,
empty shares, staged and unstaged lists, ticket-queue selection) that the five configs do not."""
import math

import numpy as np
import pytest

from oracle import xrdvi_oracle as orc
from paper_2501_09308_b200 import Xrdvi

from test_gpu_parity import TOL_ELBO, TOL_GRAD, class_errors

pytestmark = pytest.mark.gpu


def random_problem(seed):
    rng = np.random.default_rng(seed)
    N = int(rng.choice([17, 33, 100, 257, 640, 1001, 2049]))
    step = float(rng.choice([0.01, 0.02, 0.05]))
    lo = float(rng.uniform(5.0, 60.0))
    x = lo + step * np.arange(N)
    K = int(rng.choice([1, 2, 3, 7, 19, 60]))
    counts = rng.integers(1, int(rng.choice([2, 6, 40])) + 1, size=K)
    ofs = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    M = int(ofs[-1])
    span = x[-1] - x[0]
    pos = rng.uniform(x[0] - 0.2 * span, x[-1] + 0.2 * span, M)
    if rng.random() < 0.5:                                   # clustered peaks: some tiles crowded, others empty
        pos = x[0] + span * np.clip(rng.normal(0.3, 0.08, M), -0.1, 1.1)
    for k in range(K):
        pos[ofs[k]:ofs[k + 1]].sort()
    inten = rng.uniform(0.5, 100.0, M)
    inten[rng.random(M) < 0.05] = 0.0                        # dummy peaks
    for k in range(K):
        if inten[ofs[k]:ofs[k + 1]].sum() == 0.0:
            inten[ofs[k]] = 1.0
    P, R = int(rng.choice([1, 1, 2, 3])), int(rng.choice([1, 1, 2]))
    S = int(rng.choice([1, 5, 32, 33, 70]))
    poisson = rng.random() < 0.3
    y = rng.uniform(0.0, 40.0, (P, N))
    bg = 1.0 + rng.uniform(0.0, 2.0, (P, N))
    if poisson:
        y = rng.poisson(y + bg).astype(np.float64)
    W = float(rng.choice([0.0, 0.02, 1.0, 4.0, 10.0, 30.0]))
    hp = dict(window_W=W, fwhm_ref=float(rng.choice([0.05, 0.15, 0.4])), w_shape=3.0, w_rate=30.0,
              noise_sigma=float(rng.uniform(0.5, 3.0)), lambda_h=float(rng.uniform(0.2, 2.0)), n_patterns=P, n_restarts=R,
              likelihood=int(poisson), asymmetry=int(rng.random() < 0.3), width_sec=int(rng.random() < 0.2),
              general_grid=int(rng.random() < 0.25))
    if hp["general_grid"]:
        x = x.copy()
        x[1:-1] += rng.uniform(-0.3, 0.3, N - 2) * step
    return x, y, bg, ofs, pos, inten, hp, S


@pytest.mark.parametrize("seed", list(range(24)))
def test_random_problem(seed):
    x, y, bg, ofs, pos, inten, hp, S = random_problem(1000 + seed)
    o = orc.Oracle(x, y, bg, ofs, pos, inten, **{k: v for k, v in hp.items() if k != "general_grid"})   # the oracle takes any grid
    gpu = Xrdvi(x, y, bg, ofs, pos, inten, S_max=S, **hp)
    assert gpu.pair_count == o.pair_count()
    gpu.reset_state(seed=seed)
    st, _ = gpu.get_state()
    np.testing.assert_allclose(st, o.init_state(seed=seed), rtol=2e-6, atol=2e-7)
    rng = np.random.default_rng(seed)
    st = st + rng.normal(0.0, 0.2, st.shape).astype(np.float32)
    st[..., 0, :, 1] *= 0.1                                  # shifts of a few hundredths of a degree
    if hp["asymmetry"]:
        st[..., 0, :, 4] *= 0.5
    elbo_r, grad_r, ll_r = o.elbo_grad(st.astype(np.float64), S, 7, 3, want_ll=True)
    elbo_g, grad_g = gpu.elbo_grad(state=st, S=S, seed=7, iteration=3)
    f_g, ll_g = gpu.debug_profile(min(S, 4), state=st, S=S, seed=7, iteration=3, want_f=False)
    tol_ll = TOL_ELBO if not hp["likelihood"] else 3e-4       # Poisson ll is a sum of terms of both signs
    np.testing.assert_allclose(ll_g, ll_r.reshape(-1)[:min(S, 4)], rtol=tol_ll, atol=1e-3)
    np.testing.assert_allclose(elbo_g, elbo_r, rtol=tol_ll, atol=1e-3)
    # class-normalised over phases AND instances: with K = 1 a single entry would be its own scale, and the entries of
    # d ELBO / d l are means of terms that cancel (SURVEY.md 8(c) "Parity metrics")
    err = np.abs(grad_g.astype(np.float64) - grad_r).max(axis=(0, 1, 3))
    ref = np.maximum(np.abs(grad_r).max(axis=(0, 1, 3)), 1e-3)
    assert (err / ref).max() <= TOL_GRAD, (hp, err / ref)
    st2, inc, _ = gpu.fit(3, S=S, seed=5)
    assert np.isfinite(st2).all() and np.isfinite(inc).all()
    gpu.close()
    # the same three steps on a second handle: bit for bit (fixed summation orders, no race between the kernels of a step)
    gpu_b = Xrdvi(x, y, bg, ofs, pos, inten, S_max=S, **hp)
    gpu_b.reset_state(seed=seed)
    st2_b, inc_b, _ = gpu_b.fit(3, S=S, seed=5)
    assert np.array_equal(st2, st2_b) and np.array_equal(inc, inc_b)
    gpu_b.close()


@pytest.mark.parametrize("seed", list(range(16)))
def test_random_problem_many_instances_fit_is_repeatable(seed):
    """The same generator with up to 72 instances and up to 300 draws: a 30-step fit on two handles, the second in two
    pieces, bit for bit (summation orders are fixed; the kernels of consecutive steps overlap only where it is safe)."""
    x, y, bg, ofs, pos, inten, hp, S = random_problem(5000 + seed)
    rng = np.random.default_rng(seed)
    P, R = int(rng.choice([1, 2, 5, 9])), int(rng.choice([1, 3, 8]))
    y = np.tile(y[:1], (P, 1)) * rng.uniform(0.5, 1.5, (P, 1))
    bg = np.tile(bg[:1], (P, 1))
    if hp["likelihood"]:
        y = np.round(y)
    hp["n_patterns"], hp["n_restarts"] = P, R
    S = int(rng.choice([1, 5, 32, 33, 70, 256, 300]))
    a = Xrdvi(x, y, bg, ofs, pos, inten, S_max=S, **hp)
    st_a, inc_a, _ = a.fit(30, S=S, seed=9)
    b = Xrdvi(x, y, bg, ofs, pos, inten, S_max=S, **hp)
    b.fit(17, S=S, seed=9)
    st_b, inc_b, _ = b.fit(13, S=S, seed=9)
    assert np.isfinite(st_a).all() and np.isfinite(inc_a).all()
    assert np.array_equal(st_a, st_b) and np.array_equal(inc_a, inc_b)
    # and the ELBO / gradient at the fitted state against the oracle
    o = orc.Oracle(x, y, bg, ofs, pos, inten, **{k: v for k, v in hp.items() if k != "general_grid"})
    Se = min(S, 33)
    elbo_r, grad_r = o.elbo_grad(st_a.astype(np.float64), Se, 7, 3)[:2]
    elbo_g, grad_g = a.elbo_grad(state=st_a, S=Se, seed=7, iteration=3)
    tol = TOL_ELBO if not hp["likelihood"] else 3e-4
    np.testing.assert_allclose(elbo_g, elbo_r, rtol=tol, atol=1e-3)
    err = np.abs(grad_g.astype(np.float64) - grad_r).max(axis=(0, 1, 3))
    ref = np.maximum(np.abs(grad_r).max(axis=(0, 1, 3)), 1e-3)
    assert (err / ref).max() <= TOL_GRAD, (hp, err / ref)
    a.close(); b.close()
