"""xrdvi_profile_static (include/xrdvi.h): the one entry point that allocates nothing and takes no caller scratch -- its
profile rows pass through a 4 MiB file-scope `static __device__` array of the library.  Checked against the existing path
(xrdvi_debug_profile with caller scratch, itself parity-tested against the oracle in test_gpu_parity.py) on calls in a
row; tolerance: the profile / ll tolerance of the other GPU tests (relative 1e-4; the two paths launch the same kernels,
so the rows are in fact identical).  Named test_zz_* so that pytest collects it last: `pytest -x`
would otherwise hide every later test behind a failure here.  Passes alone in a fresh process and after the others."""
import numpy as np
import pytest

from paper_2501_09308_b200 import Xrdvi, XrdviError, synth

pytestmark = pytest.mark.gpu

TOL_PROFILE = 1e-4
TOL_LL = 1e-4


def assert_same(gpu, n, first, **kw):
    f_ref, ll_ref = gpu.debug_profile(n, first=first, **kw)          # existing path: caller scratch
    f_new, ll_new = gpu.profile_static(n, first=first, **kw)         # static scratch, no allocation
    assert f_new.shape == f_ref.shape and np.isfinite(f_new).all()
    for t in range(n):
        assert np.abs(f_new[t] - f_ref[t]).max() / np.abs(f_ref[t]).max() <= TOL_PROFILE
    np.testing.assert_allclose(ll_new, ll_ref, rtol=TOL_LL)
    return f_new, ll_new


def test_two_calls_in_a_row_match_the_existing_path():
    wl = synth.make_workload(0, n_restarts=2)
    S = 40                                                            # two instances of 40 draws: ragged 32-draw groups
    gpu = Xrdvi.from_workload(wl, S_max=S)
    st_a = synth.random_state(wl.K, wl.P, wl.R, seed=1)
    st_b = synth.random_state(wl.K, wl.P, wl.R, seed=2)
    # call 1: rows 35 .. 46 straddle the two restarts; call 2: other parameters, other rows, fewer of them -- the array
    # still holds call 1's rows then, and none of them may show up
    f1, ll1 = assert_same(gpu, 12, 35, state=st_a, S=S, seed=5, iteration=3)
    f2, ll2 = assert_same(gpu, 5, 2, state=st_b, S=S, seed=6, iteration=4)
    assert np.abs(f2 - f1[:5]).max() > 0 and np.abs(ll2 - ll1[:5]).max() > 0
    # call 3 repeats call 1 exactly: same rows, bit for bit
    f3, ll3 = gpu.profile_static(12, first=35, state=st_a, S=S, seed=5, iteration=3)
    assert np.array_equal(f3, f1) and np.array_equal(ll3, ll1)
    # ll only (no use of the array), and the internal state instead of caller parameters
    _, ll4 = gpu.profile_static(12, first=35, state=st_a, S=S, seed=5, iteration=3, want_f=False)
    assert np.array_equal(ll4, ll1)
    gpu.set_state(st_b)
    f5, ll5 = gpu.profile_static(5, first=2, S=S, seed=6, iteration=4)
    assert np.array_equal(f5, f2) and np.array_equal(ll5, ll2)


def test_second_handle_shares_the_array_and_config1_rows():
    wl0 = synth.make_workload(0)
    wl1 = synth.make_workload(1, S=64)
    a = Xrdvi.from_workload(wl0, S_max=32)
    b = Xrdvi.from_workload(wl1)                                      # K = 50, several tiles and a ragged tail
    st0 = synth.random_state(wl0.K, wl0.P, wl0.R, seed=3)
    st1 = synth.random_state(wl1.K, wl1.P, wl1.R, seed=4)
    assert_same(b, 6, 20, state=st1, S=64, seed=1, iteration=1)
    assert_same(a, 3, 0, state=st0, S=32, seed=2, iteration=2)
    assert_same(b, 2, 62, state=st1, S=64, seed=3, iteration=9)
    # the fit still runs after these calls and leaves the same state as on a fresh handle (no existing path disturbed)
    c = Xrdvi.from_workload(wl0, S_max=32)
    a.reset_state(0)
    r_a = a.fit(20, S=32, seed=11)
    r_c = c.fit(20, S=32, seed=11)
    assert np.array_equal(r_a[0], r_c[0])


def test_asymmetric_model_parameters_reach_the_device_without_staging():
    wl = synth.make_workload(0, asym=(0.75, 1.35))
    gpu = Xrdvi.from_workload(wl, S_max=32, asymmetry=1)
    assert gpu.C == 5
    st = synth.random_state(wl.K, wl.P, wl.R, seed=8, classes=5)
    assert_same(gpu, 4, 7, state=st, S=32, seed=4, iteration=2)
    assert_same(gpu, 4, 7, state=synth.random_state(wl.K, wl.P, wl.R, seed=9, classes=5), S=32, seed=4, iteration=2)


def test_sizes_beyond_the_static_array_are_rejected():
    wl = synth.make_workload(1, S=512)
    gpu = Xrdvi.from_workload(wl)
    limit = Xrdvi.STATIC_SCRATCH_FLOATS
    n_ok = limit // gpu.N
    assert n_ok + 1 <= 512
    with pytest.raises(XrdviError) as ei:
        gpu.profile_static(n_ok + 1, S=512)
    assert ei.value.code == -5 and "static scratch" in str(ei.value) and str(limit) in str(ei.value)
    f, ll = gpu.profile_static(n_ok, S=512, seed=1, iteration=1)      # the largest request that fits
    f_ref, ll_ref = gpu.debug_profile(n_ok, S=512, seed=1, iteration=1)
    assert np.array_equal(f, f_ref) and np.array_equal(ll, ll_ref)
    _, ll_all = gpu.profile_static(512, S=512, seed=1, iteration=1, want_f=False)   # ll alone has no limit
    assert np.array_equal(ll_all[:n_ok], ll)
    with pytest.raises(XrdviError):
        gpu.profile_static(4, first=510, S=512)                       # rows beyond P R S
