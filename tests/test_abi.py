"""CPU-side checks of the boundary: the library loads, exports every symbol include/xrdvi.h
declares, the hyper struct mirrors the header, and argument validation fails loudly (no GPU needed)."""
import ctypes as C
import pathlib
import re

import numpy as np
import pytest

from paper_2501_09308_b200 import binding, build

ROOT = pathlib.Path(__file__).resolve().parents[1]


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load_library()


def _declared(header_name):
    header = (ROOT / "include" / header_name).read_text()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    return set(re.findall(r"\b(xrdvi_[a-z_]+)\s*\(", header))


def test_every_declared_symbol_is_exported(lib):
    """include/xrdvi.h (product boundary) and include/xrdvi_debug.h (read-backs / timing) are both exported by
    libxrdvi.so; include/xrdvi_measure.h (pipe-rate microbenchmark) is NOT: it lives in its own library."""
    assert _declared("xrdvi.h") == set(binding.EXPORTS)
    assert _declared("xrdvi_debug.h") == set(binding.DEBUG_EXPORTS)
    for name in binding.EXPORTS + binding.DEBUG_EXPORTS:
        assert hasattr(lib, name), name
    assert _declared("xrdvi_measure.h") == {"xrdvi_pipe_rates"}
    assert not hasattr(lib, "xrdvi_pipe_rates")


def test_measure_library_builds_and_exports_its_symbol():
    path = build.build_measure()
    M = C.CDLL(str(path))
    assert hasattr(M, "xrdvi_pipe_rates")


def test_product_library_reads_no_environment_knob():
    """The tuning knobs (kernel shape, fused / split, PDL, staging) exist only under -DXRDVI_TUNING."""
    blob = (ROOT / "paper_2501_09308_b200" / "libxrdvi.so").read_bytes()
    for knob in (b"XRDVI_TILE_SHAPE", b"XRDVI_FUSED", b"XRDVI_SPLIT", b"XRDVI_NO_PDL", b"XRDVI_NO_UNROLL", b"XRDVI_NO_STAGE", b"XRDVI_G_BLOCK"):
        assert knob not in blob, knob


def test_hyper_struct_mirrors_header(lib):
    hy = binding.default_hyper()
    assert hy.size == C.sizeof(binding.Hyper)
    assert (hy.mu_sigma, hy.w_shape, hy.w_rate) == (0.03, 3.0, 100.0)          # PAPER.md:274 (B.2)
    assert hy.incl_tau == 0.01
    assert (hy.lr, hy.beta1, hy.beta2, hy.adam_eps) == (0.1, 0.9, 0.999, 1e-8)
    assert hy.init_log_sigma == pytest.approx(np.log(0.1))
    assert (hy.n_patterns, hy.n_restarts, hy.likelihood, hy.optimizer) == (1, 1, 0, 0)


def test_workspace_bytes(lib):
    hy = binding.default_hyper()
    small = lib.xrdvi_workspace_bytes(1001, 6, 120, 16, 0.07, C.byref(hy))
    big = lib.xrdvi_workspace_bytes(4001, 50, 4500, 256, 0.02, C.byref(hy))
    assert 0 < small < big < 1 << 30
    # the high-throughput configs stay far below the 180 GB of one B200
    hy3 = binding.default_hyper(n_patterns=1024)
    assert lib.xrdvi_workspace_bytes(4001, 50, 4500, 128, 0.02, C.byref(hy3)) < 8 << 30
    hy4 = binding.default_hyper(window_W=20.0, fwhm_ref=0.3)
    assert lib.xrdvi_workspace_bytes(8001, 1000, 175000, 256, 0.015, C.byref(hy4)) < 8 << 30
    dense = binding.default_hyper(window_W=0.0)
    assert lib.xrdvi_workspace_bytes(1001, 6, 120, 16, 0.07, C.byref(dense)) > small
    assert lib.xrdvi_workspace_bytes(1, 6, 120, 16, 0.07, C.byref(hy)) == 0
    assert lib.xrdvi_workspace_bytes(1001, 6, 120, 16, 0.0, C.byref(hy)) == 0
    hy.size = 3
    assert lib.xrdvi_workspace_bytes(1001, 6, 120, 16, 0.07, C.byref(hy)) == 0


def test_create_rejects_bad_arguments_before_touching_cuda(lib):
    hy = binding.default_hyper()
    x = np.linspace(10, 80, 101)
    y = np.ones(101)
    ofs = np.array([0, 2, 4], dtype=np.int64)
    pos = np.array([20.0, 30.0, 40.0, 50.0])
    inten = np.array([1.0, 2.0, 3.0, 4.0])
    out = C.c_void_p()
    dp = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))  # noqa: E731
    ip = lambda a: a.ctypes.data_as(C.POINTER(C.c_int64))   # noqa: E731

    def create(x=x, ofs=ofs, inten=inten, hy=hy):
        return lib.xrdvi_create(dp(x), len(x), dp(y), None, 2, ip(ofs), dp(pos), dp(inten), C.byref(hy), 16, 0,
                                None, C.c_void_p(256), 1 << 20, C.byref(out))

    xs = x.copy(); xs[5] = xs[4]
    assert create(x=xs) == -2 and b"increasing" in lib.xrdvi_last_error()
    xn = x.copy(); xn[7] += 0.01
    assert create(x=xn) == -3
    assert create(ofs=np.array([0, 0, 4], dtype=np.int64)) == -4
    assert create(inten=np.array([1.0, -2.0, 3.0, 4.0])) == -1
    hb = binding.default_hyper(likelihood=2)          # 0 Gaussian and 1 Poisson are the only likelihoods
    assert create(hy=hb) == -1
    assert out.value is None


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(binding.XrdviError):
        binding.Xrdvi(np.linspace(0, 1, 11), np.ones(11), None, [0, 1], [0.5], [1.0], S_max=4)
