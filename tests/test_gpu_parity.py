"""Parity of the CUDA path (through the C ABI) against the fp64 oracle on the same seeded inputs
and the same Philox draws.  Tolerances are north_star's: profile / ll / ELBO relative 1e-4,
gradients relative 1e-3 (class-normalised, SURVEY.md 8(c) "Parity metrics"), inclusion 0.02 absolute."""
import math

import numpy as np
import pytest

from oracle import xrdvi_oracle as orc
from paper_2501_09308_b200 import Xrdvi, synth

pytestmark = pytest.mark.gpu

TOL_PROFILE = 1e-4
TOL_ELBO = 1e-4
TOL_GRAD = 1e-3
TOL_INCL = 0.02


def class_errors(g_gpu, g_ref):
    """max_k |g_gpu - g_ref| / max_k |g_ref| per (pattern, restart, m|l, class)."""
    err = np.abs(g_gpu.astype(np.float64) - g_ref).max(axis=3)
    ref = np.abs(g_ref).max(axis=3)
    return err / ref


def check_eval(gpu, o, state, S, seed, iteration, n_prof=4):
    elbo_r, grad_r, ll_r, f_r = o.elbo_grad(state.astype(np.float64), S, seed, iteration, want_ll=True,
                                            n_profiles=n_prof)
    f_g, ll_g = gpu.debug_profile(n_prof, state=state, S=S, seed=seed, iteration=iteration)
    for t in range(n_prof):
        assert np.abs(f_g[t] - f_r[t]).max() / np.abs(f_r[t]).max() <= TOL_PROFILE
    ll_flat = ll_r.reshape(-1)
    np.testing.assert_allclose(ll_g, ll_flat[:n_prof], rtol=TOL_ELBO)
    elbo_g, grad_g = gpu.elbo_grad(state=state, S=S, seed=seed, iteration=iteration)
    np.testing.assert_allclose(elbo_g, elbo_r, rtol=TOL_ELBO)
    ce = class_errors(grad_g, grad_r)
    assert ce.max() <= TOL_GRAD, ce
    return ce.max()


# --------------------------------------------------------------------------- a-1 draws
def test_philox_words_bit_exact_and_normals():
    wl = synth.make_workload(0, n_restarts=2)
    gpu = Xrdvi.from_workload(wl, S_max=40)
    seed, it, S = (7 << 32) | 12345, 77, 40
    eps, raw = gpu.debug_draws(2 * S, S=S, seed=seed, iteration=it)
    for t in (0, 1, 17, 39, 40, 79):
        inst, s = divmod(t, S)
        for k in range(wl.K):
            ref = orc.philox4x32_10([it, s, k, inst], [seed & 0xFFFFFFFF, seed >> 32])
            assert [int(v) for v in raw[t, k]] == ref                      # bit-exact integer work
            np.testing.assert_allclose(eps[t, k], orc.eps(seed, it, inst, s, k), rtol=0, atol=4e-6)
    # published known-answer vector through the device generator: counter (it=0,s=0,k=0,inst=0), key 0
    eps0, raw0 = gpu.debug_draws(1, S=S, seed=0, iteration=0)
    assert [int(v) for v in raw0[0, 0]] == [0x6627E8D5, 0xE169C58D, 0xBC57AC4C, 0x9B00DBD8]


# --------------------------------------------------------------------------- configs
def test_config0_all_states():
    wl = synth.make_workload(0)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    assert gpu.pair_count == o.pair_count() and gpu.n_c == o.n_c
    st0, step = gpu.get_state()
    assert step == 0
    np.testing.assert_allclose(st0, o.init_state(), rtol=1e-6)
    check_eval(gpu, o, st0, wl.S, seed=3, iteration=1, n_prof=16)
    gpu.fit(50, seed=3)
    st50, step = gpu.get_state()
    assert step == 50
    check_eval(gpu, o, st50, wl.S, seed=3, iteration=51, n_prof=16)
    gpu.fit(450, seed=3)
    st500, _ = gpu.get_state()
    check_eval(gpu, o, st500, wl.S, seed=3, iteration=501, n_prof=16)


def test_config0_fit_inclusion_parity():
    wl = synth.make_workload(0)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    st_g, inc_g, tr_g = gpu.fit(500, seed=11, want_trace=True)
    st_r, _, tr_r = o.fit(o.init_state(), 500, wl.S, seed=11, want_trace=True)
    inc_r = o.inclusion(st_r)
    assert np.abs(inc_g - inc_r).max() <= TOL_INCL
    # the first steps follow the oracle closely (before fp32/fp64 trajectories drift apart)
    np.testing.assert_allclose(tr_g[:3], tr_r[:3], rtol=TOL_ELBO)
    # identified parameters of the planted phases agree
    for k in wl.true_phases[0]:
        np.testing.assert_allclose(st_g[0, 0, 0, k, :3], st_r[0, 0, 0, k, :3], atol=0.02)
    inc2, area = gpu.inclusion()
    np.testing.assert_array_equal(inc2, inc_g)
    assert area.sum() == pytest.approx(1.0, rel=1e-9)


def test_single_adam_step_matches_oracle():
    wl = synth.make_workload(0)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    st_g, _, _ = gpu.fit(1, seed=5)
    st_r, _, _ = o.fit(o.init_state(), 1, wl.S, seed=5)
    np.testing.assert_allclose(st_g, st_r, atol=2e-5)
    st_g2, _, _ = gpu.fit(2, seed=5)                              # steps 2 and 3 continue the counter
    st_r3, _, _ = o.fit(o.init_state(), 3, wl.S, seed=5)
    np.testing.assert_allclose(st_g2, st_r3, atol=2e-3)


def test_config1_reduced_draws():
    wl = synth.make_workload(1, S=64)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    assert gpu.pair_count == o.pair_count()
    st0, _ = gpu.get_state()
    check_eval(gpu, o, st0, 64, seed=1, iteration=1)
    gpu.fit(50, seed=1)
    st50, _ = gpu.get_state()
    check_eval(gpu, o, st50, 64, seed=1, iteration=51)
    gpu.fit(250, seed=1)
    st300, _ = gpu.get_state()
    check_eval(gpu, o, st300, 64, seed=1, iteration=301)


def test_config2_restarts_batched():
    wl = synth.make_workload(2, n_restarts=3, S=32)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    gpu.reset_state(seed=9)
    st0, _ = gpu.get_state()
    np.testing.assert_allclose(st0, o.init_state(seed=9), rtol=2e-6, atol=2e-7)
    assert np.abs(st0[0, 1, 0] - st0[0, 0, 0]).min() > 0          # restarts are jittered
    check_eval(gpu, o, st0, 32, seed=2, iteration=4, n_prof=2)


def test_config3_patterns_batched():
    wl = synth.make_workload(3, n_patterns=3, S=32)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    st = synth.random_state(wl.K, 3, 1, seed=4)
    st[:, :, 0, :, 0] += np.log(1.0 / np.array([o.lambda_h(p) for p in range(3)]))[:, None, None] - 2.0
    elbo_r, grad_r, ll_r = o.elbo_grad(st.astype(np.float64), 32, 8, 3, want_ll=True)
    elbo_g, grad_g = gpu.elbo_grad(state=st, S=32, seed=8, iteration=3)
    np.testing.assert_allclose(elbo_g, elbo_r, rtol=TOL_ELBO)
    assert class_errors(grad_g, grad_r).max() <= TOL_GRAD
    f_g, ll_g = gpu.debug_profile(96, state=st, S=32, seed=8, iteration=3, want_f=False)
    np.testing.assert_allclose(ll_g, ll_r.reshape(-1), rtol=TOL_ELBO)


def test_config4_reduced_library():
    wl = synth.make_workload(4, K=60, S=8)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    assert gpu.n_c == 400 and gpu.pair_count == o.pair_count()
    st0, _ = gpu.get_state()
    check_eval(gpu, o, st0, 8, seed=6, iteration=2, n_prof=2)
    st = synth.random_state(wl.K, 1, 1, seed=12)
    st[:, :, 0, :, 0] += math.log(1.0 / o.lambda_h()) - 3.0
    st[:, :, 0, :, 2] = np.log(np.random.default_rng(0).uniform(0.03, 0.3, wl.K))
    check_eval(gpu, o, st, 8, seed=6, iteration=2, n_prof=2)


# --------------------------------------------------------------------------- edge cases
def test_dense_mode_ragged_sizes_and_out_of_range_peaks():
    rng = np.random.default_rng(5)
    N = 203                                                        # not a multiple of 4 or 8
    x = 20.0 + 0.02 * np.arange(N)
    ofs = np.array([0, 3, 4, 9], dtype=np.int64)
    pos = np.array([19.0, 21.0, 23.9, 22.5, 10.0, 20.01, 24.05, 24.06, 30.0])   # some outside the grid
    inten = rng.uniform(1, 100, 9)
    y = rng.uniform(0, 30, N)
    for W in (0.0, 3.0):
        hp = dict(window_W=W, fwhm_ref=0.1, noise_sigma=1.5, lambda_h=0.5, w_rate=30.0)
        o = orc.Oracle(x, y, None, ofs, pos, inten, **hp)
        gpu = Xrdvi(x, y, None, ofs, pos, inten, S_max=5, **hp)
        assert gpu.pair_count == o.pair_count()
        st = synth.random_state(3, 1, 1, seed=1)
        st[:, :, 0, :, 0] += 2.0
        check_eval(gpu, o, st, 5, seed=1, iteration=0, n_prof=5)
        gpu.close()


def test_results_are_bitwise_reproducible():
    wl = synth.make_workload(1, S=64)
    outs = []
    for _ in range(2):
        gpu = Xrdvi.from_workload(wl)
        st, inc, tr = gpu.fit(20, seed=3, want_trace=True)
        e, g = gpu.elbo_grad(S=64, seed=3, iteration=99)
        outs.append((st, inc, tr, e, g))
        gpu.close()
    for a, b in zip(outs[0], outs[1]):
        np.testing.assert_array_equal(a, b)


def test_error_paths_on_device():
    wl = synth.make_workload(0)
    gpu = Xrdvi.from_workload(wl)
    from paper_2501_09308_b200 import XrdviError
    with pytest.raises(XrdviError):
        gpu.elbo_grad(S=wl.S + 64)
    with pytest.raises(XrdviError):
        gpu.fit(-1)


# --------------------------------------------------------------------------- Poisson likelihood (A12-A16)
def test_poisson_config0_all_states_and_fit():
    wl = synth.make_workload(0, peak_counts=2.0e4)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    st0, _ = gpu.get_state()
    np.testing.assert_allclose(st0, o.init_state(), rtol=1e-6)
    check_eval(gpu, o, st0, wl.S, seed=3, iteration=1, n_prof=16)
    st_g, inc_g, tr_g = gpu.fit(500, seed=3, want_trace=True)
    check_eval(gpu, o, st_g, wl.S, seed=3, iteration=501, n_prof=16)
    st_r, _, tr_r = o.fit(o.init_state(), 500, wl.S, seed=3, want_trace=True)
    np.testing.assert_allclose(tr_g[:3], tr_r[:3], rtol=TOL_ELBO)
    assert np.abs(inc_g - o.inclusion(st_r)).max() <= TOL_INCL
    for k in wl.true_phases[0]:
        np.testing.assert_allclose(st_g[0, 0, 0, k, :3], st_r[0, 0, 0, k, :3], atol=0.02)


def test_poisson_config1_reduced_draws_and_zero_counts():
    wl = synth.make_workload(1, S=64, peak_counts=300.0)          # low counts: many y = 0 points
    assert (wl.y == 0).sum() > 10
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    st0, _ = gpu.get_state()
    check_eval(gpu, o, st0, 64, seed=1, iteration=1)
    gpu.fit(100, seed=1)
    st, _ = gpu.get_state()
    check_eval(gpu, o, st, 64, seed=1, iteration=101)


def test_poisson_rejects_non_positive_background():
    from paper_2501_09308_b200 import XrdviError
    wl = synth.make_workload(0, peak_counts=1.0e3)
    bg = wl.background.copy()
    bg[0, 17] = 0.0
    with pytest.raises(XrdviError):
        Xrdvi(wl.two_theta, wl.y, bg, wl.peak_ofs, wl.peak_pos, wl.peak_int, S_max=4, **wl.hyper)
    y = wl.y.copy()
    y[0, 5] = -1.0
    with pytest.raises(XrdviError):
        Xrdvi(wl.two_theta, y, wl.background, wl.peak_ofs, wl.peak_pos, wl.peak_int, S_max=4, **wl.hyper)


# --------------------------------------------------------------------------- natural-gradient update (R25)
def test_natural_gradient_steps_match_oracle():
    wl = synth.make_workload(0)
    o = orc.from_workload(wl, optimizer=1, lr=0.01)
    gpu = Xrdvi.from_workload(wl, optimizer=1, lr=0.01)
    st_g, _, tr_g = gpu.fit(1, seed=5, want_trace=True)
    st_r, _, tr_r = o.fit(o.init_state(), 1, wl.S, seed=5, want_trace=True)
    np.testing.assert_allclose(st_g, st_r, rtol=1e-4, atol=2e-5)
    st_g, inc_g, tr_g = gpu.fit(199, seed=5, want_trace=True)            # steps 2..200 continue the counter
    st_r, _, tr_r = o.fit(o.init_state(), 200, wl.S, seed=5, want_trace=True)
    np.testing.assert_allclose(tr_g[:3, 0, 0], tr_r[1:4, 0, 0], rtol=TOL_ELBO)
    assert tr_g[-20:].mean() > tr_r[:20].mean() + 100.0                   # the ELBO rises
    assert np.abs(inc_g - o.inclusion(st_r)).max() <= TOL_INCL
    check_eval(gpu, o, st_g, wl.S, seed=5, iteration=201)
    from paper_2501_09308_b200 import XrdviError
    with pytest.raises(XrdviError):
        Xrdvi.from_workload(wl, optimizer=2)


# --------------------------------------------------------------------------- log-joint gradient service (NEXT-4)
def check_logjoint(gpu, o, zeta, pat):
    ll_g, lpj_g, g_g = gpu.logjoint_grad(zeta, pattern=pat)
    for t in range(zeta.shape[0]):
        ll_r, lpj_r, g_r = o.logjoint_grad(zeta[t].astype(np.float64), pat)
        assert ll_g[t] == pytest.approx(ll_r, rel=TOL_ELBO)
        assert lpj_g[t] == pytest.approx(lpj_r, rel=TOL_ELBO, abs=1e-3)
        err = np.abs(g_g[t] - g_r).max(axis=0) / np.abs(g_r).max(axis=0)       # per latent class, over phases
        assert err.max() <= TOL_GRAD, err


def test_logjoint_gradient_service_matches_oracle():
    wl = synth.make_workload(3, n_patterns=3, S=64)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    rng = np.random.default_rng(3)
    for pat, n in ((0, 1), (2, 37), (1, 64)):
        st = synth.random_state(wl.K, n, 1, seed=20 + pat)[:, 0, 0]            # [n][K][4] points near a fit
        st[:, :, 0] += math.log(1.0 / o.lambda_h(pat)) - 2.0 + rng.normal(0, 0.3, (n, wl.K))
        ll_g, lpj_g, g_g = gpu.logjoint_grad(st, pattern=pat)
        for t in sorted({0, n // 2, n - 1}):
            ll_r, lpj_r, g_r = o.logjoint_grad(st[t].astype(np.float64), pat)
            assert ll_g[t] == pytest.approx(ll_r, rel=TOL_ELBO)
            assert lpj_g[t] == pytest.approx(lpj_r, rel=TOL_ELBO, abs=1e-3)
            err = np.abs(g_g[t] - g_r).max(axis=0) / np.abs(g_r).max(axis=0)
            assert err.max() <= TOL_GRAD, err
    # the state of a fit is untouched by the service, and a fit still runs after it
    st0, step = gpu.get_state()
    gpu.logjoint_grad(synth.random_state(wl.K, 3, 1, seed=1)[:, 0, 0], pattern=0)
    st1, _ = gpu.get_state()
    np.testing.assert_array_equal(st0, st1)
    gpu.fit(3, seed=2)
    from paper_2501_09308_b200 import XrdviError
    with pytest.raises(XrdviError):
        gpu.logjoint_grad(np.zeros((65, wl.K, 4), np.float32))                 # n > S_max rounded up to 32
    with pytest.raises(XrdviError):
        gpu.logjoint_grad(np.zeros((1, wl.K, 4), np.float32), pattern=3)


def test_logjoint_gradient_service_chunks_and_poisson():
    wl = synth.make_workload(4, K=60, S=256)                                   # 4 groups per launch, 7 groups: 2 launches
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    n = 200
    st = synth.random_state(wl.K, n, 1, seed=5)[:, 0, 0]
    st[:, :, 0] += math.log(1.0 / o.lambda_h()) - 3.0
    st[:, :, 2] = np.log(np.random.default_rng(1).uniform(0.03, 0.3, (n, wl.K)))
    ll_g, lpj_g, g_g = gpu.logjoint_grad(st)
    for t in (0, 31, 32, 127, 128, 199):
        ll_r, lpj_r, g_r = o.logjoint_grad(st[t].astype(np.float64))
        assert ll_g[t] == pytest.approx(ll_r, rel=TOL_ELBO)
        assert lpj_g[t] == pytest.approx(lpj_r, rel=TOL_ELBO, abs=1e-3)
        err = np.abs(g_g[t] - g_r).max(axis=0) / np.abs(g_r).max(axis=0)
        assert err.max() <= TOL_GRAD, err
    wlp = synth.make_workload(0, peak_counts=5.0e3)
    op = orc.from_workload(wlp)
    gp = Xrdvi.from_workload(wlp)
    stp = synth.random_state(wlp.K, 9, 1, seed=8)[:, 0, 0]
    stp[:, :, 0] += math.log(1.0 / op.lambda_h()) - 1.0
    check_logjoint(gp, op, stp, 0)


# --------------------------------------------------------------------------- extreme latents
def test_extreme_widths_shifts_and_mixing():
    """Very narrow and very wide peaks, shifts of many grid points, mixing at both ends, tiny and huge scales:
    the Gaussian-core / Lorentz-tail split, the shared reciprocals and the grid-index coordinates must hold."""
    wl = synth.make_workload(1, S=32, K=12)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    K = wl.K
    st = synth.random_state(K, 1, 1, seed=3)
    st[0, 0, 0, :, 0] += math.log(1.0 / o.lambda_h()) - 2.0
    # FWHM (deg) from half a grid step to twice the window; narrower peaks amplify the fp32 rounding of the
    # sampled shift (3e-8 deg at |mu| = 0.5) by 2/w beyond 1e-4 of the peak height
    st[0, 0, 0, :, 2] = np.log([0.01, 0.015, 0.02, 0.05, 0.1, 0.2, 0.5, 1.0, 3.0, 0.03, 0.3, 0.08])
    st[0, 0, 0, :, 1] = [0.5, -0.5, 0.3, -0.2, 0.0, 0.01, -0.01, 0.1, -0.1, 0.02, 0.0, 0.25]             # shift (deg)
    st[0, 0, 0, :, 3] = [-20, 20, -8, 8, 0, 1, -1, 3, -3, 0.5, 15, -15]                                  # logit r
    st[0, 0, 0, 3, 0] -= 12.0                                                                              # h tiny
    st[0, 0, 0, 5, 0] += 3.0                                                                               # h large
    st[0, 0, 1] = math.log(0.02)
    st[0, 0, 1, :, 2] = math.log(0.3)                                                                      # wide spread of w inside a group
    check_eval(gpu, o, st, 32, seed=4, iteration=2, n_prof=4)
    ll_g, lpj_g, g_g = gpu.logjoint_grad(st[0, 0, 0][None])
    ll_r, lpj_r, g_r = o.logjoint_grad(st[0, 0, 0].astype(np.float64))
    assert ll_g[0] == pytest.approx(ll_r, rel=TOL_ELBO)
    assert (np.abs(g_g[0] - g_r).max(axis=0) / np.abs(g_r).max(axis=0)).max() <= TOL_GRAD


# --------------------------------------------------------------------------- split (ticket-queue) tile kernel
def test_split_kernel_on_long_work_items():
    """elbo_split_kernel (one-warp work items, partial profiles through L2) is what the library selects when a share
    of a tile's list holds >= 512 records (config 4 at full size).  Config 4 with K = 150 reaches that on a problem the
    oracle finishes in seconds (668 records per share, window +-400 points); K = 60 (test_config4_reduced_library) and
    config 1 take the fused kernel.  Parity at two states, determinism across two handles, Poisson."""
    wl = synth.make_workload(4, K=150, S=8)
    o = orc.from_workload(wl)
    outs = []
    for rep in range(2):
        gpu = Xrdvi.from_workload(wl)
        assert gpu.pair_count == o.pair_count() and gpu.pair_count // (((wl.N + 15) // 16) * 4 * 16) >= 512
        st0, _ = gpu.get_state()
        if rep == 0:
            check_eval(gpu, o, st0, 8, seed=6, iteration=2, n_prof=2)
        st, inc, tr = gpu.fit(12, seed=3, want_trace=True)
        e, g = gpu.elbo_grad(S=8, seed=3, iteration=99)
        e5, g5 = gpu.elbo_grad(S=5, seed=3, iteration=5)                  # ragged group
        outs.append((st, inc, tr, e, g, e5, g5))
        if rep == 0:
            check_eval(gpu, o, st, 8, seed=3, iteration=13, n_prof=2)
        gpu.close()
    for a, b in zip(outs[0], outs[1]):
        np.testing.assert_array_equal(a, b)


# --------------------------------------------------------------------------- checkpoint / resume, restarts, streams
def test_checkpoint_resume_is_bitwise_the_uninterrupted_fit():
    """fit(n) + get_state + get_optimizer_state, then set_state + set_optimizer_state + fit(m) on ANOTHER handle of
    the same problem equals fit(n + m) bit for bit (set_state alone restarts Adam)."""
    wl = synth.make_workload(1, S=64, K=10)
    ref = Xrdvi.from_workload(wl)
    st_ref, inc_ref, _ = ref.fit(37, seed=9)
    a = Xrdvi.from_workload(wl)
    a.fit(21, seed=9)
    st, step = a.get_state()
    m1, m2, adam_steps = a.get_optimizer_state()
    assert step == 21 and adam_steps == 21 and np.abs(m2).max() > 0
    b = Xrdvi.from_workload(wl)
    b.set_state(st, step)
    b.set_optimizer_state(m1, m2, adam_steps)
    st_b, inc_b, _ = b.fit(16, seed=9)
    np.testing.assert_array_equal(st_b, st_ref)
    np.testing.assert_array_equal(inc_b, inc_ref)
    from paper_2501_09308_b200 import XrdviError
    with pytest.raises(XrdviError):
        b.set_optimizer_state(m1, m2, 99)                         # more Adam steps than completed steps


def test_set_state_alone_starts_a_fresh_adam():
    """set_state zeroes the moments AND restarts the bias correction: the steps after it are the oracle's Adam steps
    1, 2, ... from zero moments on the draws of iterations step + 1, step + 2, ..."""
    wl = synth.make_workload(0)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    gpu.fit(30, seed=5)
    st, step = gpu.get_state()
    gpu.set_state(st, step)
    assert gpu.get_optimizer_state()[2] == 0
    st_g, _, _ = gpu.fit(3, seed=5)
    ref = st.astype(np.float64)
    m1, m2 = np.zeros_like(ref), np.zeros_like(ref)
    for it in range(3):
        _, grad = o.elbo_grad(ref, wl.S, 5, step + 1 + it)
        ref = o.adam_step(ref, grad, m1, m2, it + 1)
    np.testing.assert_allclose(st_g, ref, atol=2e-3)
    first = Xrdvi.from_workload(wl)
    first.set_state(st, step)
    st1, _, _ = first.fit(1, seed=5)
    np.testing.assert_allclose(np.abs(st1 - st)[0, 0, 0], 0.1, rtol=2e-3)   # fresh Adam: first step = lr * sign(g)


def test_restart_offset_draws_the_jitter_of_a_later_restart():
    wl1, wl3 = synth.make_workload(0), synth.make_workload(0, n_restarts=3)
    o3 = orc.from_workload(wl3)
    gpu = Xrdvi.from_workload(wl1)
    ref = o3.init_state(seed=9)
    for off in (0, 1, 2):
        gpu.reset_state(seed=9, restart_offset=off)
        st, _ = gpu.get_state()
        np.testing.assert_allclose(st[0, 0], ref[0, off], rtol=2e-6, atol=2e-7)
    assert np.abs(ref[0, 2, 0] - ref[0, 0, 0]).min() > 0


def test_library_owned_stream_when_null_is_passed():
    """A C caller may pass stream 0: the legacy default stream cannot be captured into a CUDA Graph, so xrdvi_create
    makes a private stream; results equal those on a caller-provided stream."""
    wl = synth.make_workload(0)
    a, b = Xrdvi.from_workload(wl), Xrdvi.from_workload(wl, library_stream=True)
    ra, rb = a.fit(25, seed=4, want_trace=True), b.fit(25, seed=4, want_trace=True)
    for x, y in zip(ra, rb):
        np.testing.assert_array_equal(x, y)
    b.close()


def test_two_handles_interleaved_and_resumed_fit():
    """Handles are independent (own workspace, control block, graphs); a fit split into pieces (odd lengths, so
    both the 8-step and the 1-step graph run) equals the fit in one piece, bit for bit."""
    wl_a, wl_b = synth.make_workload(0), synth.make_workload(1, S=64, K=10)
    ref = {}
    for name, wl in (("a", wl_a), ("b", wl_b)):
        g = Xrdvi.from_workload(wl)
        ref[name] = g.fit(37, seed=9, want_trace=True)
        g.close()
    ga, gb = Xrdvi.from_workload(wl_a), Xrdvi.from_workload(wl_b)
    tr_a, tr_b = [], []
    for n in (5, 9, 16, 7):                                         # 37 steps in four pieces, alternating handles
        sa, ia, ta = ga.fit(n, seed=9, want_trace=True)
        gb.elbo_grad(S=64, seed=1, iteration=3)                     # an evaluation in between must not disturb b's fit
        sb, ib, tb = gb.fit(n, seed=9, want_trace=True)
        ga.logjoint_grad(synth.random_state(wl_a.K, 2, 1, seed=1)[:, 0, 0])
        tr_a.append(ta)
        tr_b.append(tb)
    np.testing.assert_array_equal(sa, ref["a"][0])
    np.testing.assert_array_equal(ia, ref["a"][1])
    np.testing.assert_array_equal(np.concatenate(tr_a), ref["a"][2])
    np.testing.assert_array_equal(sb, ref["b"][0])
    np.testing.assert_array_equal(ib, ref["b"][1])
    np.testing.assert_array_equal(np.concatenate(tr_b), ref["b"][2])
    assert ga.get_state()[1] == 37 and gb.get_state()[1] == 37


def test_debug_timeline_rows_are_consistent():
    """xrdvi_debug_timeline: one row per warp of the launch, ordered stamps, SM ids of a B200, every record counted."""
    from paper_2501_09308_b200 import XrdviError
    wl = synth.make_workload(1, S=64)
    g = Xrdvi.from_workload(wl)
    before, _ = g.get_state()
    rows = g.debug_timeline(seed=3)
    after, _ = g.get_state()
    assert np.array_equal(before, after)                       # the state is not touched
    assert len(rows) > 0 and (rows[:, 0] > 0).all()
    t0, t1, t2 = (rows[:, i].astype(np.int64) for i in range(3))
    assert (t1 >= t0).all() and (t2 >= t1).all()
    assert (t2.max() - t0.min()) < 50_000_000                  # one launch: far below 50 ms
    sm = (rows[:, 3] & np.uint64(0xFFFFFFFF)).astype(np.int64)
    assert sm.max() < 160 and len(np.unique(sm)) > 100
    rec = (rows[:, 3] >> np.uint64(32)).astype(np.int64)
    # every (peak, tile) record is owned by exactly one share per group: 2 groups here, and the records of a draw
    # hold pair_count in-window pairs of at most 16 points each
    groups = 2
    assert rec.sum() % groups == 0
    assert rec.sum() // groups * 16 >= g.pair_count
    with pytest.raises(XrdviError):
        g.debug_timeline(capacity=8)
    g.close()


def test_debug_update_timeline_rows_are_consistent():
    """xrdvi_debug_update_timeline: one row per CTA of update_draw_kernel plus the next tile kernel's start; the stamps of
    a CTA are ordered, every CTA is resident before its wait returns, the next step begins after the last CTA is done, and
    the stamped run is the same fit as an unstamped one."""
    wl = synth.make_workload(1, S=64)
    g = Xrdvi.from_workload(wl)
    rows = g.debug_update_timeline(steps=12, seed=3).astype(np.int64)
    n_cta = wl.K + 2
    assert rows.shape == (n_cta + 1, 8)
    u = rows[:n_cta]
    phase, ll = u[:wl.K], u[wl.K:]
    assert (np.diff(phase, axis=1) >= 0).all()
    assert (np.diff(ll[:, [0, 1, 2, 3, 7]], axis=1) >= 0).all() and (ll[:, 4:7] == 0).all()
    assert rows[n_cta, 0] >= u[:, 7].max()                   # the next tile kernel waits for the whole launch
    assert 0 < rows[n_cta, 1] <= u[:, 2].min()               # and this launch for the whole tile kernel of its step
    assert (u[:, 7].max() - u[:, 2].min()) < 50_000          # ns: the serial section is a few microseconds
    h = Xrdvi.from_workload(wl)
    st_h, _, _ = h.fit(12, seed=3)
    st_g, _ = g.get_state()
    assert np.array_equal(st_g, st_h)
    summ = h.update_timeline_summary(steps=6, seed=3)
    assert summ["ctas"] == n_cta and 0 < summ["last_phase_cta_done_ns"] <= summ["next_tile_kernel_past_its_wait_ns"] < 50_000
    from paper_2501_09308_b200 import XrdviError
    with pytest.raises(XrdviError):
        g.debug_update_timeline(steps=1)                     # needs a stamped step and a step after it
