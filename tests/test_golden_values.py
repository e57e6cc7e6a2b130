"""Stored fp64 oracle values (tests/golden/cfg0_oracle_values.txt, written by tests/golden/make_golden.py from
oracle/ only).  CPU: the oracle still reproduces them (guards against silent drift of its arithmetic).
GPU: the CUDA path matches them without running the oracle in the same process."""
import importlib.util
import pathlib

import numpy as np
import pytest

GOLDEN = pathlib.Path(__file__).resolve().parent / "golden"


def load_golden():
    vals = {}
    for ln in (GOLDEN / "cfg0_oracle_values.txt").read_text().splitlines():
        if ln.startswith("#") or not ln.strip():
            continue
        case, q, idx, v = ln.split()
        vals.setdefault(case, {}).setdefault(q, []).append(float(v))
    return {c: {q: np.array(v) for q, v in d.items()} for c, d in vals.items()}


def make_golden_module():
    spec = importlib.util.spec_from_file_location("make_golden", GOLDEN / "make_golden.py")
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def test_oracle_reproduces_its_stored_values():
    gold = load_golden()
    for name, o, st, S, seed, it in make_golden_module().cases():
        elbo, grad, ll = o.elbo_grad(st, S, seed, it, want_ll=True)
        np.testing.assert_allclose(elbo[0, 0], gold[name]["elbo"][0], rtol=1e-12)
        np.testing.assert_allclose(ll[0, 0], gold[name]["ll"], rtol=1e-12)
        np.testing.assert_allclose(grad.reshape(-1), gold[name]["grad"], rtol=1e-9, atol=1e-9)


@pytest.mark.gpu
def test_cuda_path_matches_the_stored_oracle_values():
    from paper_2501_09308_b200 import Xrdvi, synth
    gold = load_golden()
    mod = make_golden_module()
    for name, o, st, S, seed, it in mod.cases():                        # the oracle objects are not evaluated here
        wl = synth.make_workload(0, peak_counts=2.0e4) if name.startswith("poisson") else synth.make_workload(0)
        gpu = Xrdvi.from_workload(wl)
        if name == "gauss_windows":
            gpu.set_phase_windows(mod.PHASE_WINDOWS)
        st32 = st.astype(np.float32)
        assert np.array_equal(st32.astype(np.float64), st)              # golden states are fp32-exact
        elbo, grad = gpu.elbo_grad(state=st32, S=S, seed=seed, iteration=it)
        _, ll = gpu.debug_profile(S, state=st32, S=S, seed=seed, iteration=it, want_f=False)
        assert elbo[0, 0] == pytest.approx(gold[name]["elbo"][0], rel=1e-4)
        np.testing.assert_allclose(ll, gold[name]["ll"], rtol=1e-4)
        g_ref = gold[name]["grad"].reshape(2, wl.K, 4)
        err = np.abs(grad[0, 0] - g_ref).max(axis=1) / np.abs(g_ref).max(axis=1)
        assert err.max() <= 1e-3, (name, err)
