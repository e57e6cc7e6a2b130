"""Thin Python binding of the C ABI in include/xrdvi.h (argument marshalling only).

Every step of the hot path runs in the CUDA kernels of libxrdvi.so.  PyTorch is used for the
device workspace (one uint8 tensor) and the CUDA stream, nothing else.  There is no CPU
fallback: a missing library or a missing sm_100 device raises.
"""
from __future__ import annotations

import ctypes as C
import pathlib

import numpy as np

_PKG = pathlib.Path(__file__).resolve().parent
_LIB_PATH = _PKG / "libxrdvi.so"

EXPORTS = (            # include/xrdvi.h: the product boundary
    "xrdvi_default_hyper", "xrdvi_workspace_bytes", "xrdvi_create", "xrdvi_destroy", "xrdvi_pair_count",
    "xrdvi_latent_classes", "xrdvi_window_halfwidth", "xrdvi_set_phase_windows", "xrdvi_get_phase_windows", "xrdvi_adapt_windows",
    "xrdvi_fit_adaptive", "xrdvi_reset_state", "xrdvi_reset_state_restart", "xrdvi_get_state", "xrdvi_set_state",
    "xrdvi_get_optimizer_state", "xrdvi_set_optimizer_state", "xrdvi_elbo_grad",
    "xrdvi_fit", "xrdvi_inclusion", "xrdvi_posterior_summary", "xrdvi_logjoint_grad", "xrdvi_profile_static",
    "xrdvi_last_error",
)
DEBUG_EXPORTS = (      # include/xrdvi_debug.h: read-backs for the parity tests, timing for bench.py and profiles/
    "xrdvi_debug_profile", "xrdvi_debug_draws", "xrdvi_time_kernels", "xrdvi_bench_steps", "xrdvi_debug_timeline",
    "xrdvi_debug_update_timeline",
)


class XrdviError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"xrdvi error {code}: {msg}")
        self.code = code


class Hyper(C.Structure):
    """Mirror of ``xrdvi_hyper`` (include/xrdvi.h)."""
    _fields_ = [
        ("size", C.c_uint32), ("_pad", C.c_uint32),
        ("lambda_h", C.c_double), ("mu_sigma", C.c_double), ("w_shape", C.c_double), ("w_rate", C.c_double),
        ("noise_sigma", C.c_double), ("window_W", C.c_double), ("fwhm_ref", C.c_double),
        ("incl_tau", C.c_double), ("lr", C.c_double), ("beta1", C.c_double), ("beta2", C.c_double),
        ("adam_eps", C.c_double), ("init_log_sigma", C.c_double),
        ("n_patterns", C.c_int32), ("n_restarts", C.c_int32), ("likelihood", C.c_int32), ("optimizer", C.c_int32),
        ("asymmetry", C.c_int32), ("width_sec", C.c_int32), ("alpha_mu", C.c_double), ("alpha_sigma", C.c_double),
        ("general_grid", C.c_int32), ("_pad2", C.c_int32),
    ]


_lib = None


def load_library():
    """dlopen libxrdvi.so (built in-tree by paper_2501_09308_b200.build); fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not _LIB_PATH.exists():
        raise XrdviError(-100, f"{_LIB_PATH} not built; run `python -m paper_2501_09308_b200.build` "
                               "(there is no CPU fallback)")
    L = C.CDLL(str(_LIB_PATH))
    vp, fp, dp = C.c_void_p, C.POINTER(C.c_float), C.POINTER(C.c_double)
    L.xrdvi_default_hyper.argtypes = [C.POINTER(Hyper)]
    L.xrdvi_default_hyper.restype = None
    L.xrdvi_workspace_bytes.argtypes = [C.c_int64, C.c_int32, C.c_int64, C.c_int32, C.c_double, C.POINTER(Hyper)]
    L.xrdvi_workspace_bytes.restype = C.c_size_t
    L.xrdvi_create.argtypes = [dp, C.c_int64, dp, dp, C.c_int32, C.POINTER(C.c_int64), dp, dp, C.POINTER(Hyper),
                               C.c_int32, C.c_int, vp, vp, C.c_size_t, C.POINTER(vp)]
    L.xrdvi_destroy.argtypes = [vp]
    L.xrdvi_destroy.restype = None
    L.xrdvi_pair_count.argtypes = [vp]
    L.xrdvi_pair_count.restype = C.c_int64
    L.xrdvi_window_halfwidth.argtypes = [vp]
    L.xrdvi_window_halfwidth.restype = C.c_int64
    L.xrdvi_latent_classes.argtypes = [vp]
    L.xrdvi_latent_classes.restype = C.c_int32
    ip = C.POINTER(C.c_int32)
    L.xrdvi_set_phase_windows.argtypes = [vp, ip]
    L.xrdvi_get_phase_windows.argtypes = [vp, ip]
    L.xrdvi_adapt_windows.argtypes = [vp, C.c_double, ip]
    L.xrdvi_fit_adaptive.argtypes = [vp, C.c_int32, C.c_int32, C.c_uint64, C.c_int32, C.c_double, fp, dp, dp]
    L.xrdvi_reset_state.argtypes = [vp, C.c_uint64]
    L.xrdvi_reset_state_restart.argtypes = [vp, C.c_uint64, C.c_int32]
    L.xrdvi_get_optimizer_state.argtypes = [vp, fp, fp, C.POINTER(C.c_int64)]
    L.xrdvi_set_optimizer_state.argtypes = [vp, fp, fp, C.c_int64]
    L.xrdvi_get_state.argtypes = [vp, fp, C.POINTER(C.c_int64)]
    L.xrdvi_set_state.argtypes = [vp, fp, C.c_int64]
    L.xrdvi_elbo_grad.argtypes = [vp, fp, C.c_int32, C.c_uint64, C.c_uint64, dp, fp]
    L.xrdvi_fit.argtypes = [vp, C.c_int32, C.c_int32, C.c_uint64, fp, dp, dp]
    L.xrdvi_inclusion.argtypes = [vp, dp, dp]
    L.xrdvi_posterior_summary.argtypes = [vp, dp]
    L.xrdvi_logjoint_grad.argtypes = [vp, fp, C.c_int64, C.c_int32, dp, dp, fp]
    L.xrdvi_profile_static.argtypes = [vp, fp, C.c_int32, C.c_uint64, C.c_uint64, C.c_int64, C.c_int64, fp, dp]
    L.xrdvi_debug_profile.argtypes = [vp, fp, C.c_int32, C.c_uint64, C.c_uint64, C.c_int64, C.c_int64, fp, dp, vp,
                                      C.c_size_t]
    L.xrdvi_debug_draws.argtypes = [vp, C.c_int32, C.c_uint64, C.c_uint64, C.c_int64, fp, C.POINTER(C.c_uint32),
                                    C.POINTER(C.c_int32), vp, C.c_size_t]
    L.xrdvi_time_kernels.argtypes = [vp, C.c_int32, C.c_uint64, C.c_int32, fp]
    L.xrdvi_bench_steps.argtypes = [vp, C.c_int32, C.c_int32, C.c_uint64, vp, C.c_size_t, fp]
    L.xrdvi_debug_timeline.argtypes = [vp, C.c_int32, C.c_uint64, C.c_int64, C.POINTER(C.c_uint64), C.POINTER(C.c_int64),
                                       vp, C.c_size_t]
    L.xrdvi_debug_update_timeline.argtypes = [vp, C.c_int32, C.c_int32, C.c_uint64, C.c_int64, C.POINTER(C.c_uint64),
                                              C.POINTER(C.c_int64), vp, C.c_size_t]
    L.xrdvi_last_error.restype = C.c_char_p
    _lib = L
    return L


def default_hyper(**overrides) -> Hyper:
    hy = Hyper()
    load_library().xrdvi_default_hyper(C.byref(hy))
    for k, v in overrides.items():
        if k.startswith("_") or k == "size" or not hasattr(hy, k):
            raise TypeError(f"unknown hyper-parameter {k!r}")
        setattr(hy, k, v)
    return hy


def _check(rc):
    if rc != 0:
        raise XrdviError(rc, load_library().xrdvi_last_error().decode())


def _f(a):
    return a.ctypes.data_as(C.POINTER(C.c_float)) if a is not None else None


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def pipe_rates(device=0) -> dict:
    """Measured per-SM per-clock pipe rates (xrdvi_pipe_rates, include/xrdvi_measure.h): the microbenchmark lives in
    its own library, libxrdvi_measure.so (`python -m paper_2501_09308_b200.build --measure`), loaded only here."""
    path = _PKG / "libxrdvi_measure.so"
    if not path.exists():
        raise XrdviError(-100, f"{path} not built; run `python -m paper_2501_09308_b200.build --measure`")
    M = C.CDLL(str(path))
    M.xrdvi_pipe_rates.argtypes = [C.c_int, C.POINTER(C.c_float)]
    r = np.zeros(9, dtype=np.float32)
    rc = M.xrdvi_pipe_rates(int(device), _f(r))
    if rc != 0:
        raise XrdviError(rc, "xrdvi_pipe_rates failed")
    names = ("ffma", "ffma2", "mufu_ex2", "mufu_rcp", "mix_forward", "mix_backward", "mix_ffma2", "mufu_ex2_rcp", "sm_mhz")
    return {k: float(v) for k, v in zip(names, r)}


class Xrdvi:
    """One problem: P patterns x R restarts over a shared candidate library (xrdvi_create)."""

    def __init__(self, two_theta, y, background, peak_ofs, peak_pos, peak_int, S_max, device=0, library_stream=False,
                 **hyper):
        import torch  # device memory and stream only

        L = load_library()
        if not torch.cuda.is_available():
            raise XrdviError(-6, "no CUDA device: the xrdvi hot path has no CPU fallback")
        self.hyper = default_hyper(**hyper)
        self.P, self.R = int(self.hyper.n_patterns), int(self.hyper.n_restarts)
        x = np.ascontiguousarray(two_theta, dtype=np.float64)
        self.N = int(x.shape[0])
        yy = np.ascontiguousarray(np.asarray(y, dtype=np.float64).reshape(self.P, self.N))
        bg = None if background is None else np.ascontiguousarray(
            np.asarray(background, dtype=np.float64).reshape(self.P, self.N))
        ofs = np.ascontiguousarray(peak_ofs, dtype=np.int64)
        pos = np.ascontiguousarray(peak_pos, dtype=np.float64)
        inten = np.ascontiguousarray(peak_int, dtype=np.float64)
        self.K, self.M, self.S_max = int(ofs.shape[0] - 1), int(pos.shape[0]), int(S_max)
        step = float((x[-1] - x[0]) / (self.N - 1)) if self.N > 1 else 0.0
        nbytes = int(L.xrdvi_workspace_bytes(self.N, self.K, self.M, self.S_max, step, C.byref(self.hyper)))
        if nbytes == 0:
            raise XrdviError(-1, "xrdvi_workspace_bytes: invalid sizes")
        self.device = torch.device("cuda", device)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        # a non-default stream (CUDA Graph capture needs one); library_stream=True passes NULL and lets xrdvi_create
        # make its own
        self.stream = None if library_stream else torch.cuda.Stream(device=self.device)
        self._h = C.c_void_p()
        _check(L.xrdvi_create(_d(x), self.N, _d(yy), _d(bg), self.K, ofs.ctypes.data_as(C.POINTER(C.c_int64)),
                              _d(pos), _d(inten), C.byref(self.hyper), self.S_max, device,
                              C.c_void_p(self.stream.cuda_stream if self.stream is not None else 0),
                              C.c_void_p(self.workspace.data_ptr()), nbytes, C.byref(self._h)))
        self.workspace_bytes = nbytes
        self.C = int(L.xrdvi_latent_classes(self._h))       # latent classes per phase: 4, or 5 with the asymmetry

    @classmethod
    def from_workload(cls, wl, S_max=None, device=0, library_stream=False, **overrides):
        hp = dict(wl.hyper)
        hp.update(overrides)
        return cls(wl.two_theta, wl.y, wl.background, wl.peak_ofs, wl.peak_pos, wl.peak_int,
                   S_max=wl.S if S_max is None else S_max, device=device, library_stream=library_stream, **hp)

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            load_library().xrdvi_destroy(self._h)
            self._h = C.c_void_p()
        self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- queries ---------------------------------------------------------------
    @property
    def pair_count(self) -> int:
        return int(load_library().xrdvi_pair_count(self._h))

    @property
    def n_c(self) -> int:
        return int(load_library().xrdvi_window_halfwidth(self._h))

    def _state_shape(self):
        return (self.P, self.R, 2, self.K, self.C)

    # ---- state -----------------------------------------------------------------
    def reset_state(self, seed=0, restart_offset=0):
        _check(load_library().xrdvi_reset_state_restart(self._h, int(seed), int(restart_offset)))

    def get_optimizer_state(self):
        m1 = np.empty(self._state_shape(), dtype=np.float32)
        m2 = np.empty(self._state_shape(), dtype=np.float32)
        n = C.c_int64()
        _check(load_library().xrdvi_get_optimizer_state(self._h, _f(m1), _f(m2), C.byref(n)))
        return m1, m2, int(n.value)

    def set_optimizer_state(self, mom1, mom2, adam_steps):
        m1 = np.ascontiguousarray(mom1, dtype=np.float32).reshape(self._state_shape())
        m2 = np.ascontiguousarray(mom2, dtype=np.float32).reshape(self._state_shape())
        _check(load_library().xrdvi_set_optimizer_state(self._h, _f(m1), _f(m2), int(adam_steps)))

    def get_state(self):
        st = np.empty(self._state_shape(), dtype=np.float32)
        step = C.c_int64()
        _check(load_library().xrdvi_get_state(self._h, _f(st), C.byref(step)))
        return st, int(step.value)

    def set_state(self, state, step=0):
        st = np.ascontiguousarray(state, dtype=np.float32).reshape(self._state_shape())
        _check(load_library().xrdvi_set_state(self._h, _f(st), int(step)))

    # ---- hot path --------------------------------------------------------------
    def elbo_grad(self, state=None, S=None, seed=0, iteration=0):
        S = self.S_max if S is None else int(S)
        st = None if state is None else np.ascontiguousarray(state, dtype=np.float32).reshape(self._state_shape())
        elbo = np.empty((self.P, self.R), dtype=np.float64)
        grad = np.empty(self._state_shape(), dtype=np.float32)
        _check(load_library().xrdvi_elbo_grad(self._h, _f(st), S, int(seed), int(iteration), _d(elbo), _f(grad)))
        return elbo, grad

    def fit(self, iterations, S=None, seed=0, want_state=True, want_incl=True, want_trace=False):
        S = self.S_max if S is None else int(S)
        st = np.empty(self._state_shape(), dtype=np.float32) if want_state else None
        inc = np.empty((self.P, self.R, self.K), dtype=np.float64) if want_incl else None
        tr = np.empty((int(iterations), self.P, self.R), dtype=np.float64) if want_trace else None
        _check(load_library().xrdvi_fit(self._h, int(iterations), S, int(seed), _f(st), _d(inc), _d(tr)))
        return st, inc, tr

    # ---- per-phase (adaptive) windows, R27 ---------------------------------------
    def set_phase_windows(self, n_ck=None):
        a = None if n_ck is None else np.ascontiguousarray(n_ck, dtype=np.int32).reshape(self.K)
        _check(load_library().xrdvi_set_phase_windows(
            self._h, None if a is None else a.ctypes.data_as(C.POINTER(C.c_int32))))

    def get_phase_windows(self):
        a = np.empty(self.K, dtype=np.int32)
        _check(load_library().xrdvi_get_phase_windows(self._h, a.ctypes.data_as(C.POINTER(C.c_int32))))
        return a

    def adapt_windows(self, W):
        a = np.empty(self.K, dtype=np.int32)
        _check(load_library().xrdvi_adapt_windows(self._h, float(W), a.ctypes.data_as(C.POINTER(C.c_int32))))
        return a

    def fit_adaptive(self, iterations, refresh_every, W, S=None, seed=0, want_state=True, want_incl=True,
                     want_trace=False):
        S = self.S_max if S is None else int(S)
        st = np.empty(self._state_shape(), dtype=np.float32) if want_state else None
        inc = np.empty((self.P, self.R, self.K), dtype=np.float64) if want_incl else None
        tr = np.empty((int(iterations), self.P, self.R), dtype=np.float64) if want_trace else None
        _check(load_library().xrdvi_fit_adaptive(self._h, int(iterations), S, int(seed), int(refresh_every),
                                                 float(W), _f(st), _d(inc), _d(tr)))
        return st, inc, tr

    def logjoint_grad(self, zeta, pattern=0):
        """ll [n], log prior + log Jacobian [n], gradient [n][K][4] at the points zeta [n][K][4] (xrdvi_logjoint_grad)."""
        z = np.ascontiguousarray(zeta, dtype=np.float32).reshape(-1, self.K, self.C)
        n = int(z.shape[0])
        ll = np.empty(n, dtype=np.float64)
        lpj = np.empty(n, dtype=np.float64)
        g = np.empty((n, self.K, self.C), dtype=np.float32)
        _check(load_library().xrdvi_logjoint_grad(self._h, _f(z), n, int(pattern), _d(ll), _d(lpj), _f(g)))
        return ll, lpj, g

    def inclusion(self):
        inc = np.empty((self.P, self.R, self.K), dtype=np.float64)
        ar = np.empty_like(inc)
        _check(load_library().xrdvi_inclusion(self._h, _d(inc), _d(ar)))
        return inc, ar

    def posterior_summary(self):
        out = np.empty((self.P, self.R, self.K, self.C, 5), dtype=np.float64)
        _check(load_library().xrdvi_posterior_summary(self._h, _d(out)))
        return out

    STATIC_SCRATCH_FLOATS = 1 << 20     # xrdvi_profile_static: n * N limit (4 MiB static device array)

    def profile_static(self, n, state=None, S=None, seed=0, iteration=0, want_f=True, first=0):
        """xrdvi_profile_static: profile rows f [n][N] and ll [n] of the draws first .. first + n - 1; allocates nothing
        in the library and needs no scratch (n * N <= STATIC_SCRATCH_FLOATS)."""
        S = self.S_max if S is None else int(S)
        st = None if state is None else np.ascontiguousarray(state, dtype=np.float32).reshape(self._state_shape())
        f = np.empty((int(n), self.N), dtype=np.float32) if want_f else None
        ll = np.empty(int(n), dtype=np.float64)
        _check(load_library().xrdvi_profile_static(self._h, _f(st), S, int(seed), int(iteration), int(first), int(n),
                                                   _f(f), _d(ll)))
        return f, ll

    # ---- debug / measurement (include/xrdvi_debug.h) -----------------------------
    def _scratch(self, nbytes):
        """A device scratch tensor for the debug / measurement calls (the library allocates nothing itself)."""
        import torch
        if nbytes <= 0:
            return None, None, 0
        t = torch.empty(int(nbytes), dtype=torch.uint8, device=self.device)
        return t, C.c_void_p(t.data_ptr()), int(nbytes)

    def debug_profile(self, n, state=None, S=None, seed=0, iteration=0, want_f=True, first=0):
        S = self.S_max if S is None else int(S)
        st = None if state is None else np.ascontiguousarray(state, dtype=np.float32).reshape(self._state_shape())
        f = np.empty((int(n), self.N), dtype=np.float32) if want_f else None
        ll = np.empty(int(n), dtype=np.float64)
        scratch, ptr, nb = self._scratch(4 * int(n) * self.N if want_f else 0)
        _check(load_library().xrdvi_debug_profile(self._h, _f(st), S, int(seed), int(iteration), int(first), int(n),
                                                  _f(f), _d(ll), ptr, nb))
        return f, ll

    def debug_draws(self, n, S=None, seed=0, iteration=0, want_core=False):
        S = self.S_max if S is None else int(S)
        eps = np.empty((int(n), self.K, 4), dtype=np.float32)
        raw = np.empty((int(n), self.K, 4), dtype=np.uint32)
        core = np.empty((int(n), self.K), dtype=np.int32) if want_core else None
        scratch, ptr, nb = self._scratch(16 * self.P * self.R * ((S + 31) // 32) * 32 * self.K)
        _check(load_library().xrdvi_debug_draws(
            self._h, S, int(seed), int(iteration), int(n), _f(eps), raw.ctypes.data_as(C.POINTER(C.c_uint32)),
            core.ctypes.data_as(C.POINTER(C.c_int32)) if want_core else None, ptr, nb))
        return (eps, raw, core) if want_core else (eps, raw)

    def time_kernels(self, S=None, seed=0, reps=20):
        S = self.S_max if S is None else int(S)
        ms = np.zeros(4, dtype=np.float32)
        _check(load_library().xrdvi_time_kernels(self._h, S, int(seed), int(reps), _f(ms)))
        return dict(ms_tile=float(ms[0]), ms_tile_forward_only=float(ms[1]), ms_update=float(ms[2]),
                    ms_iteration=float(ms[3]))

    def debug_timeline(self, S=None, seed=0, capacity=1 << 22):
        """Per-warp (start, end of phase 1, end, SM id | records << 32) of one tile-kernel launch (xrdvi_debug_timeline)."""
        S = self.S_max if S is None else int(S)
        rows = np.zeros((int(capacity), 4), dtype=np.uint64)
        n = C.c_int64(0)
        scratch, ptr, nb = self._scratch(32 * int(capacity))
        _check(load_library().xrdvi_debug_timeline(self._h, S, int(seed), int(capacity),
                                                   rows.ctypes.data_as(C.POINTER(C.c_uint64)), C.byref(n), ptr, nb))
        return rows[: n.value]

    def debug_update_timeline(self, steps=40, S=None, seed=0, tile_warps=1 << 22):
        """[CTAs + 1][8] %globaltimer stamps of one update_draw_kernel launch inside a run of `steps` steps
        (xrdvi_debug_update_timeline); the last row's first word is the next tile kernel's start.  `tile_warps`: an upper
        bound of the warps of one tile-kernel launch (sizes the scratch)."""
        S = self.S_max if S is None else int(S)
        cap = (self.K + (S + 31) // 32) * self.P * self.R + 1
        rows = np.zeros((cap, 8), dtype=np.uint64)
        n = C.c_int64(0)
        scratch, ptr, nb = self._scratch(64 * cap + 64 * int(tile_warps))
        _check(load_library().xrdvi_debug_update_timeline(self._h, int(steps), S, int(seed), cap,
                                                          rows.ctypes.data_as(C.POINTER(C.c_uint64)), C.byref(n), ptr, nb))
        return rows[: n.value]

    def update_timeline_summary(self, steps=40, S=None, seed=0):
        """Segment durations (ns; mean and max over the phase CTAs) of one update_draw_kernel launch, from
        debug_update_timeline: the numbers of profiles/r2_update_kernel.md."""
        S = self.S_max if S is None else int(S)
        r = self.debug_update_timeline(steps=steps, S=S, seed=seed).astype(np.int64)
        per_inst = self.K + (S + 31) // 32
        u = r[:-1]
        ph = u[[i for i in range(u.shape[0]) if i % per_inst < self.K]]
        ll = u[[i for i in range(u.shape[0]) if i % per_inst >= self.K]]
        t0 = int(u[:, 2].min())                                   # the first CTA's wait returned
        d = np.diff(ph, axis=1)
        names = ("before_the_wait", "waiting", "slots_and_prior_added", "shuffles_and_barrier", "own_parameter",
                 "all_parameters", "draws_and_exit")
        out = {"ctas": int(u.shape[0]),
               "resident_before_wait_returned_ns": (int(t0 - u[:, 0].max()), int(t0 - u[:, 0].min())),
               "segments_ns_mean_max": {n: (int(d[:, i].mean()), int(d[:, i].max())) for i, n in enumerate(names)},
               "last_phase_cta_done_ns": int(ph[:, 7].max() - t0), "mean_phase_cta_done_ns": int((ph[:, 7] - t0).mean()),
               "last_loglik_cta_done_ns": int(ll[:, 7].max() - t0),
               "next_tile_kernel_past_its_wait_ns": int(r[-1, 0] - t0),
               "tile_kernel_last_warp_done_ns": int(r[-1, 1] - t0)}
        return out

    def bench_steps(self, steps, S=None, seed=0, l2_flush_bytes=0):
        S = self.S_max if S is None else int(S)
        ms = np.empty(int(steps), dtype=np.float32)
        scratch, ptr, nb = self._scratch(int(l2_flush_bytes))
        _check(load_library().xrdvi_bench_steps(self._h, int(steps), S, int(seed), ptr, nb, _f(ms)))
        return ms
