"""Parity of the CUDA path with per-phase (adaptive) windows, reading R27, against the fp64 oracle:
same seeded inputs, same Philox draws, the same half-widths set on both sides.  Tolerances as
tests/test_gpu_parity.py (north_star): profile / ll / ELBO relative 1e-4, class-normalised gradient 1e-3,
inclusion 0.02 absolute; half-widths and pair counts are integers and must agree exactly."""
import numpy as np
import pytest

from oracle import xrdvi_oracle as orc
from paper_2501_09308_b200 import Xrdvi, XrdviError, synth
from test_gpu_parity import TOL_INCL, check_eval

pytestmark = pytest.mark.gpu


def test_per_phase_windows_config1_three_states():
    wl = synth.make_workload(1, S=64)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    rng = np.random.default_rng(3)
    n_ck = rng.integers(0, 76, wl.K)
    n_ck[:6] = (0, 1, 7, 8, 75, 16)            # no neighbour, one, just below / at half a tile, the cap, a tile
    assert np.array_equal(gpu.get_phase_windows(), np.full(wl.K, 75))
    full = gpu.pair_count
    gpu.set_phase_windows(n_ck)
    o.set_phase_windows(n_ck)
    assert np.array_equal(gpu.get_phase_windows(), n_ck)
    assert gpu.pair_count == o.pair_count() < full
    st0, step0 = gpu.get_state()
    check_eval(gpu, o, st0, 64, seed=1, iteration=1)
    gpu.fit(60, seed=1)
    st60, step = gpu.get_state()
    assert step == step0 + 60
    check_eval(gpu, o, st60, 64, seed=1, iteration=61)
    # a change of windows keeps state, moments and step; the graph is re-captured for the new tables
    n2 = np.minimum(n_ck + 9, 75)
    gpu.set_phase_windows(n2)
    o.set_phase_windows(n2)
    st_same, step_same = gpu.get_state()
    assert step_same == step and np.array_equal(st_same, st60)
    assert gpu.pair_count == o.pair_count()
    gpu.fit(40, seed=1)
    st100, _ = gpu.get_state()
    check_eval(gpu, o, st100, 64, seed=1, iteration=101)
    # NULL restores the static window bit for bit
    gpu.set_phase_windows(None)
    o.set_phase_windows(None)
    assert gpu.pair_count == full == o.pair_count()
    ref = Xrdvi.from_workload(wl)
    e1, g1 = gpu.elbo_grad(state=st100, S=64, seed=5, iteration=9)
    e2, g2 = ref.elbo_grad(state=st100, S=64, seed=5, iteration=9)
    assert np.array_equal(e1, e2) and np.array_equal(g1, g2)


def test_per_phase_windows_batched_poisson_and_wide_library():
    # restarts + patterns share one table set
    wl = synth.make_workload(3, n_patterns=2, n_restarts=2, S=32)
    o, gpu = orc.from_workload(wl), Xrdvi.from_workload(wl)
    n_ck = np.random.default_rng(8).integers(5, 76, wl.K)
    gpu.set_phase_windows(n_ck)
    o.set_phase_windows(n_ck)
    st0, _ = gpu.get_state()
    check_eval(gpu, o, st0, 32, seed=2, iteration=3, n_prof=2)
    # the paper's Poisson likelihood (R24), ragged last tile
    wl0 = synth.make_workload(0, peak_counts=1.0e4)
    o0, g0 = orc.from_workload(wl0), Xrdvi.from_workload(wl0)
    n0 = np.array([22, 3, 10, 0, 17, 8])
    g0.set_phase_windows(n0)
    o0.set_phase_windows(n0)
    s0, _ = g0.get_state()
    check_eval(g0, o0, s0, wl0.S, seed=2, iteration=1, n_prof=4)
    # config 4's +-400-point window (a peak spans 51 tiles), reduced library
    wl4 = synth.make_workload(4, K=60, S=8)
    o4, g4 = orc.from_workload(wl4), Xrdvi.from_workload(wl4)
    n4 = np.random.default_rng(1).integers(20, 401, wl4.K)
    g4.set_phase_windows(n4)
    o4.set_phase_windows(n4)
    assert g4.pair_count == o4.pair_count()
    s4, _ = g4.get_state()
    check_eval(g4, o4, s4, 8, seed=6, iteration=2, n_prof=2)


def test_refresh_rule_matches_oracle_exactly():
    wl = synth.make_workload(1, n_restarts=3, S=32)
    o, gpu = orc.from_workload(wl), Xrdvi.from_workload(wl)
    gpu.reset_state(seed=4)
    gpu.fit(40, seed=4)
    st, _ = gpu.get_state()
    for W in (10.0, 6.0, 3.5):
        n_gpu = gpu.adapt_windows(W)
        n_ref = o.adaptive_halfwidths(st.astype(np.float64), W)
        assert np.array_equal(n_gpu, n_ref)
        assert np.array_equal(gpu.get_phase_windows(), n_ref)
    # hand-set state: widths 0.05 .. 0.25 deg, shifts, a wide variational sd
    st2 = st.copy()
    st2[:, :, 0, :, 2] = np.log(np.linspace(0.01, 0.25, wl.K))[None, None, :]
    st2[0, 1, 0, :, 1] = np.linspace(-0.2, 0.2, wl.K)
    st2[0, 2, 1, ::7, 2] = np.log(0.6)
    gpu.set_state(st2, step=40)
    assert np.array_equal(gpu.adapt_windows(10.0), o.adaptive_halfwidths(st2.astype(np.float64), 10.0))


def test_adaptive_fit_config0_inclusion_parity():
    wl = synth.make_workload(0)
    o, gpu = orc.from_workload(wl), Xrdvi.from_workload(wl)
    full = gpu.pair_count
    st_g, inc_g, tr_g = gpu.fit_adaptive(500, refresh_every=100, W=5.0, seed=1, want_trace=True)
    st_r, hist = o.fit_adaptive(o.init_state(0), 500, wl.S, seed=1, refresh_every=100, W=5.0)
    assert np.abs(inc_g - o.inclusion(st_r)).max() <= TOL_INCL
    assert np.abs(gpu.get_phase_windows().astype(np.int64) - hist[-1]).max() <= 1     # fp32 / fp64 trajectories
    assert gpu.pair_count < 0.6 * full
    assert np.isfinite(tr_g).all() and tr_g[-50:].mean() > tr_g[:50].mean()
    for k in wl.true_phases[0]:
        np.testing.assert_allclose(st_g[0, 0, 0, k, :3], st_r[0, 0, 0, k, :3], atol=0.02)
    # the same fit driven piece by piece through the C ABI is bitwise the same
    g2 = Xrdvi.from_workload(wl)
    for piece in range(5):
        g2.fit(100, seed=1, want_state=False, want_incl=False)
        if piece < 4:
            g2.adapt_windows(5.0)
    st2, _ = g2.get_state()
    assert np.array_equal(st2, st_g)


def test_adaptive_fit_config1_inclusion_parity_reduced_draws():
    wl = synth.make_workload(1, S=32)
    o, gpu = orc.from_workload(wl), Xrdvi.from_workload(wl)
    full = gpu.pair_count
    st_g, inc_g, _ = gpu.fit_adaptive(150, refresh_every=50, W=10.0, seed=2)
    st_r, hist = o.fit_adaptive(o.init_state(0), 150, 32, seed=2, refresh_every=50, W=10.0)
    assert np.abs(inc_g - o.inclusion(st_r)).max() <= TOL_INCL
    assert np.abs(gpu.get_phase_windows().astype(np.int64) - hist[-1]).max() <= 1
    assert gpu.pair_count < 0.9 * full
    # the final state evaluates to the oracle's numbers under the windows now in force
    o.set_phase_windows(gpu.get_phase_windows())
    check_eval(gpu, o, st_g, 32, seed=2, iteration=151)


def test_window_error_paths():
    wl = synth.make_workload(0)
    gpu = Xrdvi.from_workload(wl)
    with pytest.raises(XrdviError):
        gpu.set_phase_windows(np.array([23, 1, 1, 1, 1, 1]))
    with pytest.raises(XrdviError):
        gpu.set_phase_windows(np.array([-1, 1, 1, 1, 1, 1]))
    with pytest.raises(XrdviError):
        gpu.adapt_windows(0.0)
    with pytest.raises(XrdviError):
        gpu.fit_adaptive(10, refresh_every=0, W=5.0)
    assert np.array_equal(gpu.get_phase_windows(), np.full(6, 22))       # nothing changed
    dense = Xrdvi.from_workload(wl, window_W=0.0)
    with pytest.raises(XrdviError):
        dense.set_phase_windows(np.ones(6, dtype=np.int32))
    with pytest.raises(XrdviError):
        dense.adapt_windows(5.0)


# --------------------------------------------------------------------------- full sizes, bench launch configuration
def test_config1_full_size_adaptive_fit_and_evaluation():
    """K=50, S=256 (the headline launch shape): 300 steps with a refresh every 100, then everything (ll of every
    draw, profiles, ELBO, gradient) under the windows left in force, and the inclusion probabilities of the
    oracle's own adaptive fit with the same draws."""
    wl = synth.make_workload(1)
    o, gpu = orc.from_workload(wl), Xrdvi.from_workload(wl)
    st_g, inc_g, _ = gpu.fit_adaptive(300, refresh_every=100, W=10.0, seed=1)
    n_g = gpu.get_phase_windows()
    assert n_g.min() >= 20 and n_g.max() <= 75 and gpu.pair_count < 0.9 * 629906
    st_r, hist = o.fit_adaptive(o.init_state(0), 300, wl.S, seed=1, refresh_every=100, W=10.0)
    assert np.abs(n_g.astype(np.int64) - hist[-1]).max() <= 1
    assert np.abs(inc_g - o.inclusion(st_r)).max() <= TOL_INCL
    o.set_phase_windows(n_g)
    assert gpu.pair_count == o.pair_count()
    elbo_r, grad_r, ll_r = o.elbo_grad(st_g.astype(np.float64), wl.S, 1, 301, want_ll=True)
    _, ll_g = gpu.debug_profile(wl.S, state=st_g, S=wl.S, seed=1, iteration=301, want_f=False)
    np.testing.assert_allclose(ll_g, ll_r.reshape(-1), rtol=1e-4)
    check_eval(gpu, o, st_g, wl.S, seed=1, iteration=301, n_prof=3)


def test_config4_full_size_adapted_windows_sampled_draws():
    """K=1000, N=8001, S=256, +-400-point cap: windows adapted after 3 steps (W = 20: 111..400 points); ll of sampled
    draws one by one with the oracle under the same half-widths, pair counts equal."""
    from test_gpu_fullsize import ll_one_draw
    wl = synth.make_workload(4)
    o, gpu = orc.from_workload(wl), Xrdvi.from_workload(wl)
    gpu.fit(3, seed=6)
    n_g = gpu.adapt_windows(20.0)
    st, _ = gpu.get_state()
    st64 = st.astype(np.float64)
    assert np.array_equal(n_g, o.adaptive_halfwidths(st64, 20.0))
    o.set_phase_windows(n_g)
    assert gpu.pair_count == o.pair_count() < 137387988
    _, ll_g = gpu.debug_profile(wl.S, state=st, S=wl.S, seed=6, iteration=7, want_f=False)
    assert np.isfinite(ll_g).all()
    for s in (0, 31, 32, 131, 255):
        assert ll_g[s] == pytest.approx(ll_one_draw(o, st64, 6, 7, 0, s), rel=1e-4)
    e, g = gpu.elbo_grad(state=st, S=wl.S, seed=6, iteration=7)
    assert np.isfinite(e).all() and np.isfinite(g).all()
