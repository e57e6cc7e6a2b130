"""Parity of xrdvi_posterior_summary (marginals of q in (h, mu, w, r), R28) against the fp64 oracle on
the same float32 state.  Both sides compute in fp64 from the same inputs by different quadratures: closed-form
entries relative 1e-12, the logit-normal mean absolute 1e-12 and its sd relative 1e-9."""
import numpy as np
import pytest

from oracle import xrdvi_oracle as orc
from paper_2501_09308_b200 import Xrdvi, synth

pytestmark = pytest.mark.gpu


def compare(out_g, out_r):
    assert out_g.shape == out_r.shape
    for c in (0, 1, 2):
        np.testing.assert_allclose(out_g[..., c, :], out_r[..., c, :], rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(out_g[..., 3, 0], out_r[..., 3, 0], rtol=0, atol=1e-12)
    np.testing.assert_allclose(out_g[..., 3, 1], out_r[..., 3, 1], rtol=1e-9, atol=1e-18)
    np.testing.assert_allclose(out_g[..., 3, 2:], out_r[..., 3, 2:], rtol=1e-12, atol=1e-15)


def test_summary_of_random_states_with_extreme_widths():
    """Several patterns and restarts, K not a multiple of the block, log sigma across the clamp range [-12, 2]."""
    wl = synth.make_workload(3, n_patterns=3, n_restarts=2, K=37)
    o = orc.from_workload(wl)
    gpu = Xrdvi.from_workload(wl)
    st = synth.random_state(wl.K, 3, 2, seed=21)
    rng = np.random.default_rng(22)
    st[:, :, 1] = rng.uniform(-12.0, 2.0, st[:, :, 1].shape).astype(np.float32)
    st[:, :, 0, :, 3] = rng.uniform(-8.0, 8.0, st[:, :, 0, :, 3].shape).astype(np.float32)
    st[0, 0, 1, 0] = -12.0
    st[0, 0, 1, 1] = 2.0
    gpu.set_state(st)
    compare(gpu.posterior_summary(), o.posterior_summary(st.astype(np.float64)))


def test_summary_after_a_fit_config0_and_full_size_config1():
    for cfg, iters in ((0, 300), (1, 50)):
        wl = synth.make_workload(cfg)
        o = orc.from_workload(wl)
        gpu = Xrdvi.from_workload(wl)
        gpu.fit(iters, seed=4)
        st, _ = gpu.get_state()
        out_g = gpu.posterior_summary()
        compare(out_g, o.posterior_summary(st.astype(np.float64)))
        # consistent with the inclusion read-out: the area ratio uses E[h] of the same log-normal (R15)
        _, area = gpu.inclusion()
        eh = out_g[0, 0, :, 0, 0]
        A = np.array([wl.peak_int[wl.peak_ofs[k]:wl.peak_ofs[k + 1]].sum() for k in range(wl.K)])
        np.testing.assert_allclose(area[0, 0], A * eh / (A * eh).sum(), rtol=1e-9)


def test_null_summary_pointer_is_rejected():
    from paper_2501_09308_b200.binding import load_library
    wl = synth.make_workload(0)
    gpu = Xrdvi.from_workload(wl)
    assert load_library().xrdvi_posterior_summary(gpu._h, None) != 0
