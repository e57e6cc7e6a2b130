"""ctypes wrapper around oracle/xrdvi_oracle.c (fp64 CPU oracle).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and the
cpu_baseline / --impl reference legs of bench.py.  The product package
(paper_2501_09308_b200) never imports this module, and this module never imports
the product's CUDA binding.
"""
from __future__ import annotations

import ctypes as C
import pathlib
import sys

import numpy as np

_HERE = pathlib.Path(__file__).resolve().parent
sys.path.insert(0, str(_HERE))
import build as _build  # noqa: E402  (oracle/build.py)

sys.path.pop(0)


class OrcHyper(C.Structure):
    _fields_ = [
        ("lambda_h", C.c_double), ("mu_sigma", C.c_double),
        ("w_shape", C.c_double), ("w_rate", C.c_double),
        ("noise_sigma", C.c_double),
        ("window_W", C.c_double), ("fwhm_ref", C.c_double),
        ("incl_tau", C.c_double),
        ("lr", C.c_double), ("beta1", C.c_double), ("beta2", C.c_double), ("adam_eps", C.c_double),
        ("init_log_sigma", C.c_double),
        ("n_patterns", C.c_int32), ("n_restarts", C.c_int32),
        ("likelihood", C.c_int32), ("optimizer", C.c_int32),
        ("asymmetry", C.c_int32), ("width_sec", C.c_int32),
        ("alpha_mu", C.c_double), ("alpha_sigma", C.c_double),
    ]


DEFAULTS = dict(lambda_h=0.0, mu_sigma=0.03, w_shape=3.0, w_rate=100.0, noise_sigma=0.0,
                window_W=10.0, fwhm_ref=0.15, incl_tau=0.01, lr=0.1, beta1=0.9, beta2=0.999,
                adam_eps=1e-8, init_log_sigma=float(np.log(0.1)), n_patterns=1, n_restarts=1, likelihood=0, optimizer=0,
                asymmetry=0, width_sec=0, alpha_mu=1.0, alpha_sigma=0.2)

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(str(path))
        dp = C.POINTER(C.c_double)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [dp, C.c_int64, dp, dp, C.c_int32, C.POINTER(C.c_int64), dp, dp,
                                 C.POINTER(OrcHyper)]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32)] * 3
        L.orc_eps.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, dp]
        L.orc_window_halfwidth.restype = C.c_int64
        L.orc_window_halfwidth.argtypes = [C.c_void_p]
        L.orc_pair_count.restype = C.c_int64
        L.orc_pair_count.argtypes = [C.c_void_p]
        for name in ("orc_sigma_n", "orc_lambda_h"):
            getattr(L, name).restype = C.c_double
            getattr(L, name).argtypes = [C.c_void_p, C.c_int32]
        for name in ("orc_gauss", "orc_lorentz"):
            getattr(L, name).restype = C.c_double
            getattr(L, name).argtypes = [C.c_double] * 3
        L.orc_pseudo_voigt.restype = C.c_double
        L.orc_pseudo_voigt.argtypes = [C.c_double] * 4
        L.orc_pseudo_voigt_asym.restype = C.c_double
        L.orc_pseudo_voigt_asym.argtypes = [C.c_double] * 5
        L.orc_eps_alpha.restype = C.c_double
        L.orc_eps_alpha.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32]
        L.orc_nearest_index.restype = C.c_int64
        L.orc_nearest_index.argtypes = [dp, C.c_int64, C.c_double]
        L.orc_classes.restype = C.c_int32
        L.orc_classes.argtypes = [C.c_void_p]
        L.orc_profile.argtypes = [C.c_void_p, C.c_int32, dp, dp]
        L.orc_loglik.restype = C.c_double
        L.orc_loglik.argtypes = [C.c_void_p, C.c_int32, dp]
        L.orc_logprior_jac.restype = C.c_double
        L.orc_logprior_jac.argtypes = [C.c_void_p, C.c_int32, dp]
        L.orc_logjoint_grad.argtypes = [C.c_void_p, C.c_int32, dp, dp, dp, dp, dp]
        L.orc_elbo_grad.argtypes = [C.c_void_p, dp, C.c_int32, C.c_uint64, C.c_uint64, dp, dp, dp, dp,
                                    C.c_int64]
        L.orc_elbo_grad_range.argtypes = [C.c_void_p, dp, C.c_int32, C.c_uint64, C.c_uint64, C.c_int32, C.c_int32,
                                          dp, dp, dp, dp, C.c_int64]
        L.orc_adam_step.argtypes = [C.c_void_p, dp, dp, dp, dp, C.c_int64]
        L.orc_natgrad_step.argtypes = [C.c_void_p, dp, dp]
        L.orc_init_state.argtypes = [C.c_void_p, C.c_uint64, dp]
        L.orc_fit.argtypes = [C.c_void_p, dp, dp, dp, C.c_int32, C.c_int32, C.c_uint64, C.c_int64, dp]
        L.orc_inclusion.argtypes = [C.c_void_p, dp, dp, dp]
        L.orc_posterior_summary.argtypes = [C.c_void_p, dp, dp]
        L.orc_set_phase_windows.restype = C.c_int
        L.orc_set_phase_windows.argtypes = [C.c_void_p, C.POINTER(C.c_int64)]
        L.orc_adaptive_halfwidths.argtypes = [C.c_void_p, dp, C.c_double, C.POINTER(C.c_int64)]
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def eps(seed, iteration, inst, s, k):
    out = np.empty(4, dtype=np.float64)
    lib().orc_eps(int(seed), int(iteration), int(inst), int(s), int(k), _dp(out))
    return out


def gauss(x, rho, w):
    return lib().orc_gauss(float(x), float(rho), float(w))


def lorentz(x, rho, w):
    return lib().orc_lorentz(float(x), float(rho), float(w))


def pseudo_voigt(x, rho, w, r):
    return lib().orc_pseudo_voigt(float(x), float(rho), float(w), float(r))


def pseudo_voigt_asym(x, rho, w, r, alpha):
    return lib().orc_pseudo_voigt_asym(float(x), float(rho), float(w), float(r), float(alpha))


def eps_alpha(seed, iteration, inst, s, k):
    return float(lib().orc_eps_alpha(int(seed), int(iteration), int(inst), int(s), int(k)))


def nearest_index(x, p):
    x = np.ascontiguousarray(x, dtype=np.float64)
    return int(lib().orc_nearest_index(_dp(x), int(x.shape[0]), float(p)))


def num_threads():
    return int(lib().orc_num_threads())


class Oracle:
    """One problem (P patterns x R restarts) held by the C oracle."""

    def __init__(self, two_theta, y, background, peak_ofs, peak_pos, peak_int, **hyper):
        L = lib()
        hp = dict(DEFAULTS)
        unknown = set(hyper) - set(hp)
        if unknown:
            raise TypeError(f"unknown hyper-parameters: {sorted(unknown)}")
        hp.update(hyper)
        self.hyper = hp
        self.x = np.ascontiguousarray(two_theta, dtype=np.float64)
        self.N = int(self.x.shape[0])
        self.P, self.R = int(hp["n_patterns"]), int(hp["n_restarts"])
        self.y = np.ascontiguousarray(np.asarray(y, dtype=np.float64).reshape(self.P, self.N))
        self.B = None if background is None else np.ascontiguousarray(
            np.asarray(background, dtype=np.float64).reshape(self.P, self.N))
        self.ofs = np.ascontiguousarray(peak_ofs, dtype=np.int64)
        self.K = int(self.ofs.shape[0] - 1)
        self.pos = np.ascontiguousarray(peak_pos, dtype=np.float64)
        self.inten = np.ascontiguousarray(peak_int, dtype=np.float64)
        self.M = int(self.pos.shape[0])
        self._hs = OrcHyper(**hp)
        self._h = L.orc_create(_dp(self.x), self.N, _dp(self.y), _dp(self.B), self.K,
                               self.ofs.ctypes.data_as(C.POINTER(C.c_int64)), _dp(self.pos),
                               _dp(self.inten), C.byref(self._hs))
        self.C = int(L.orc_classes(self._h))        # latent classes per phase: 4, or 5 with the asymmetry (R30)
        self._mom = None
        self.step = 0

    def __del__(self):
        try:
            if getattr(self, "_h", None):
                lib().orc_destroy(self._h)
                self._h = None
        except Exception:
            pass

    # ---- scalars -----------------------------------------------------------
    @property
    def n_c(self):
        return int(lib().orc_window_halfwidth(self._h))

    def pair_count(self):
        return int(lib().orc_pair_count(self._h))

    def sigma_n(self, pat=0):
        return float(lib().orc_sigma_n(self._h, pat))

    def lambda_h(self, pat=0):
        return float(lib().orc_lambda_h(self._h, pat))

    # ---- model pieces ------------------------------------------------------
    def _zeta(self, zeta):
        z = np.ascontiguousarray(zeta, dtype=np.float64).reshape(self.K, self.C)
        return z

    def profile(self, zeta, pat=0):
        z = self._zeta(zeta)
        f = np.empty(self.N, dtype=np.float64)
        lib().orc_profile(self._h, pat, _dp(z), _dp(f))
        return f

    def loglik(self, f, pat=0):
        f = np.ascontiguousarray(f, dtype=np.float64)
        return float(lib().orc_loglik(self._h, pat, _dp(f)))

    def logprior_jac(self, zeta, pat=0):
        z = self._zeta(zeta)
        return float(lib().orc_logprior_jac(self._h, pat, _dp(z)))

    def logjoint_grad(self, zeta, pat=0):
        z = self._zeta(zeta)
        ll, lpj = C.c_double(), C.c_double()
        g = np.empty((self.K, self.C), dtype=np.float64)
        lib().orc_logjoint_grad(self._h, pat, _dp(z), C.byref(ll), C.byref(lpj), _dp(g), None)
        return ll.value, lpj.value, g

    # ---- ELBO --------------------------------------------------------------
    def _state(self, state):
        st = np.ascontiguousarray(state, dtype=np.float64).reshape(self.P, self.R, 2, self.K, self.C)
        return st

    def elbo_grad(self, state, S, seed, iteration, want_ll=False, n_profiles=0):
        st = self._state(state)
        elbo = np.empty((self.P, self.R), dtype=np.float64)
        grad = np.empty_like(st)
        ll = np.empty((self.P, self.R, S), dtype=np.float64) if want_ll else None
        f = np.empty((n_profiles, self.N), dtype=np.float64) if n_profiles else None
        lib().orc_elbo_grad(self._h, _dp(st), int(S), int(seed), int(iteration), _dp(elbo), _dp(grad),
                            _dp(ll), _dp(f), int(n_profiles))
        out = [elbo, grad]
        if want_ll:
            out.append(ll)
        if n_profiles:
            out.append(f)
        return tuple(out)

    def elbo_grad_range(self, state, S, seed, iteration, inst0, n_inst, want_ll=False):
        """ELBO / gradient (/ ll per draw) of instances inst0 .. inst0+n_inst-1 only (inst = pat*R + rst)."""
        st = self._state(state)
        elbo = np.empty(n_inst, dtype=np.float64)
        grad = np.empty((n_inst, 2, self.K, self.C), dtype=np.float64)
        ll = np.empty((n_inst, S), dtype=np.float64) if want_ll else None
        lib().orc_elbo_grad_range(self._h, _dp(st), int(S), int(seed), int(iteration), int(inst0), int(n_inst),
                                  _dp(elbo), _dp(grad), _dp(ll), None, 0)
        return (elbo, grad, ll) if want_ll else (elbo, grad)

    def init_state(self, seed=0):
        st = np.empty((self.P, self.R, 2, self.K, self.C), dtype=np.float64)
        lib().orc_init_state(self._h, int(seed), _dp(st))
        return st

    def adam_step(self, state, grad, mom1, mom2, step):
        st = self._state(state).copy()
        g = np.ascontiguousarray(grad, dtype=np.float64)
        lib().orc_adam_step(self._h, _dp(st), _dp(g), _dp(mom1), _dp(mom2), int(step))
        return st

    def natgrad_step(self, state, grad):
        st = self._state(state).copy()
        g = np.ascontiguousarray(grad, dtype=np.float64)
        lib().orc_natgrad_step(self._h, _dp(st), _dp(g))
        return st

    def fit(self, state, iterations, S, seed, first_step=1, mom=None, want_trace=False):
        """Returns (state, (mom1, mom2), trace).  Steps first_step .. first_step+iterations-1."""
        st = self._state(state).copy()
        if mom is None:
            mom = (np.zeros_like(st), np.zeros_like(st))
        m1, m2 = (np.ascontiguousarray(mom[0], dtype=np.float64).copy(),
                  np.ascontiguousarray(mom[1], dtype=np.float64).copy())
        tr = np.empty((iterations, self.P, self.R), dtype=np.float64) if want_trace else None
        lib().orc_fit(self._h, _dp(st), _dp(m1), _dp(m2), int(iterations), int(S), int(seed),
                      int(first_step), _dp(tr))
        return st, (m1, m2), tr

    # ---- adaptive windows (R27) ---------------------------------------------
    def set_phase_windows(self, n_ck=None):
        """Per-phase window half-widths (points), 0 <= n_ck[k] <= n_c; None restores the static window."""
        if n_ck is None:
            lib().orc_set_phase_windows(self._h, None)
            return
        a = np.ascontiguousarray(n_ck, dtype=np.int64).reshape(self.K)
        if lib().orc_set_phase_windows(self._h, a.ctypes.data_as(C.POINTER(C.c_int64))) != 0:
            raise ValueError("per-phase half-widths need a windowed problem and 0 <= n_ck <= n_c")

    def adaptive_halfwidths(self, state, W):
        st = self._state(state)
        out = np.empty(self.K, dtype=np.int64)
        lib().orc_adaptive_halfwidths(self._h, _dp(st), float(W), out.ctypes.data_as(C.POINTER(C.c_int64)))
        return out

    def fit_adaptive(self, state, iterations, S, seed, refresh_every, W):
        """R27: `iterations` steps in pieces of `refresh_every`; after every piece but the last the per-phase
        windows are refreshed from the current state.  Starts from the windows currently set.  Returns
        (state, list of the half-width vectors set after each refresh)."""
        st, mom, done, hist = self._state(state).copy(), None, 0, []
        while done < iterations:
            n = min(int(refresh_every), iterations - done)
            st, mom, _ = self.fit(st, n, S, seed, first_step=done + 1, mom=mom)
            done += n
            if done < iterations:
                nck = self.adaptive_halfwidths(st, W)
                self.set_phase_windows(nck)
                hist.append(nck)
        return st, hist

    def inclusion(self, state, want_area=False):
        st = self._state(state)
        inc = np.empty((self.P, self.R, self.K), dtype=np.float64)
        ar = np.empty_like(inc) if want_area else None
        lib().orc_inclusion(self._h, _dp(st), _dp(inc), _dp(ar))
        return (inc, ar) if want_area else inc

    def posterior_summary(self, state):
        """Marginals of q in (h, mu, w, r): [P][R][K][4][5] = (mean, sd, q2.5, q50, q97.5) (reading R28)."""
        st = self._state(state)
        out = np.empty((self.P, self.R, self.K, self.C, 5), dtype=np.float64)
        lib().orc_posterior_summary(self._h, _dp(st), _dp(out))
        return out


def from_workload(wl, **overrides):
    """Oracle for a paper_2501_09308_b200.synth.Workload (inputs only; no product code runs)."""
    hp = dict(wl.hyper)
    hp.update(overrides)
    return Oracle(wl.two_theta, wl.y, wl.background, wl.peak_ofs, wl.peak_pos, wl.peak_int, **hp)
