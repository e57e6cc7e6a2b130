"""Fits with many instances: `update_draw_kernel` then runs in several waves of CTAs (K + gpi CTAs of 256 threads per
instance; a B200 holds about 300 of them at a time).  What a CTA of that kernel reads BEFORE its grid-dependency wait --
its own step counter `ctl->u_step`, which fixes the Philox iteration of the next draws and the Adam bias correction -- must
not move while CTAs of the same launch have yet to start.  A launch that moved it early would give the
late instances the draws of the wrong iteration: the fit would leave the oracle's by the size of an Adam step (0.1) and two
handles would not agree bit for bit."""
import numpy as np
import pytest

from oracle import xrdvi_oracle as orc
from paper_2501_09308_b200 import Xrdvi, synth

pytestmark = pytest.mark.gpu


def test_fit_of_200_patterns_follows_the_oracle_and_is_repeatable():
    P, S, steps = 200, 32, 10
    wl = synth.make_workload(3, n_patterns=P, K=6, S=S)          # config 3's recipe: P patterns share one library
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    st_g, inc_g, tr_g = gpu.fit(steps, S=S, seed=3, want_trace=True)
    st_r, _, tr_r = o.fit(o.init_state(0), steps, S, seed=3, want_trace=True)
    # ten Adam steps of 0.1 each: fp32 against fp64 stays within 1e-3, a wrong draw iteration does not
    assert np.abs(st_g.astype(np.float64) - st_r).max() <= 2e-3
    np.testing.assert_allclose(tr_g, np.asarray(tr_r).reshape(tr_g.shape), rtol=1e-4)
    assert np.abs(inc_g - o.inclusion(st_r)).max() <= 0.02
    # every pattern, first to last, took the same number of steps with the same draws on a second handle
    gpu2 = Xrdvi.from_workload(wl)
    st_2, inc_2, tr_2 = gpu2.fit(steps, S=S, seed=3, want_trace=True)
    assert np.array_equal(st_g, st_2) and np.array_equal(tr_g, tr_2) and np.array_equal(inc_g, inc_2)
    # and in two pieces (the step counter is handed from launch to launch, and from run to run by the host)
    gpu3 = Xrdvi.from_workload(wl)
    gpu3.fit(4, S=S, seed=3)
    st_3, _, _ = gpu3.fit(steps - 4, S=S, seed=3)
    assert np.array_equal(st_g, st_3)


def test_fit_of_12_restarts_of_4096_draws_is_repeatable():
    """Config 2's shape (many draws per instance: the update kernel's long path, K + 128 CTAs per instance)."""
    wl = synth.make_workload(2, n_restarts=12, K=5)
    a, b = Xrdvi.from_workload(wl), Xrdvi.from_workload(wl)
    st_a, inc_a, _ = a.fit(6, seed=9)
    st_b, inc_b, _ = b.fit(6, seed=9)
    assert np.array_equal(st_a, st_b) and np.array_equal(inc_a, inc_b)
    o = orc.from_workload(synth.make_workload(2, n_restarts=12, K=5, S=64))
    # the same six steps with 64 of the draws per step on both sides (the oracle's cost is per draw)
    c = Xrdvi.from_workload(wl)
    st_c, _, _ = c.fit(6, S=64, seed=9)
    st_r, _, _ = o.fit(o.init_state(0), 6, 64, seed=9)
    assert np.abs(st_c.astype(np.float64) - st_r).max() <= 2e-3
