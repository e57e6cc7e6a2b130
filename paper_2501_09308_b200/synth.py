"""Seeded synthetic XRD workloads (the five BASELINE.json configs).

This module is the *instrument simulator*: it draws candidate peak tables and
observed patterns.  It serves both the CUDA path and the fp64 oracle with the
same inputs and holds none of the method's inference arithmetic (no ELBO, no
gradient, no window, no Philox).  The patterns are generated DENSE
(untruncated pseudo-Voigt, plain numpy) exactly as SURVEY.md §8(d) states; they
stand in for the paper's TiO2 measurement and AtomWork-Adv candidate tables
(PAPER.md:84-86), which are not available offline.

Recipe (BASELINE.json `configs`), host numpy
``default_rng(1000 + cfg)``:
  peaks / phase : 20 (cfg 0), U{30..150} (cfg 1-3), U{50..300} (cfg 4)
  positions     : U(lo, hi), sorted
  intensities   : I = 100 * (1 + Pareto(1.5)) / max
  true phases   : 3 / U{2..4} / as cfg 1 / U{1..5} per pattern / 5
  true params   : h ~ U(0.5, 2), shift ~ N(0, 0.02), FWHM ~ U(0.05, 0.15)
                  (cfg 4: U(0.03, 0.3)), mixing ~ U(0.2, 0.8)
  background    : b0 + b1 (x - lo), b0 ~ 2 % of max signal (passed as B)
  noise         : N(0, sigma_n), sigma_n = 1 % of max signal
  cfg 1-3       : two absent "confuser" phases whose peaks are a true phase's
                  peaks + U(-0.1, 0.1) deg with re-drawn intensities.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

_A_G = 2.0 * math.sqrt(math.log(2.0) / math.pi)
_A_L = 2.0 / math.pi


@dataclasses.dataclass
class Workload:
    """One synthetic problem: inputs of ``xrdvi_create`` plus run settings."""

    cfg: int
    two_theta: np.ndarray          # [N] float64, uniform grid
    y: np.ndarray                  # [P, N] float64 observed intensities
    background: np.ndarray         # [P, N] float64
    peak_ofs: np.ndarray           # [K+1] int64 CSR offsets
    peak_pos: np.ndarray           # [M] float64 (deg), sorted inside each phase
    peak_int: np.ndarray           # [M] float64, max 100 per phase
    hyper: dict                    # keyword overrides for the hyper struct
    S: int                         # Monte-Carlo draws per (pattern, restart)
    iterations: int
    true_phases: list              # per pattern: sorted list of planted phase ids
    true_params: list              # per pattern: dict k -> (h, shift, fwhm, mix)

    @property
    def N(self) -> int:
        return int(self.two_theta.shape[0])

    @property
    def K(self) -> int:
        return int(self.peak_ofs.shape[0] - 1)

    @property
    def M(self) -> int:
        return int(self.peak_pos.shape[0])

    @property
    def P(self) -> int:
        return int(self.y.shape[0])

    @property
    def R(self) -> int:
        return int(self.hyper.get("n_restarts", 1))


def _pseudo_voigt_pattern(x, pos, inten, h, shift, fwhm, mix, alpha=1.0):
    """Dense instrument response of one phase (plain numpy, fp64).  alpha != 1: split peaks, the high-angle side
    alpha times wider at the same height (A9/A10)."""
    out = np.zeros_like(x)
    # chunk the (peak x point) plane to bound memory
    for a in range(0, pos.shape[0], 64):
        p = pos[a:a + 64, None] + shift
        t = (x[None, :] - p) / fwhm
        if alpha != 1.0:
            t = np.where(t >= 0.0, t / alpha, t)
        g = (_A_G / fwhm) * np.exp(-4.0 * math.log(2.0) * t * t)
        l = (_A_L / fwhm) / (1.0 + 4.0 * t * t)
        out += (inten[a:a + 64, None] * ((1.0 - mix) * g + mix * l)).sum(axis=0)
    return h * out


_SPEC = {
    # cfg: (K, (Mlo, Mhi), N, lo, hi, P, R, S, its, W, fwhm_ref, (fw_lo, fw_hi), (w_shape, w_rate))
    0: (6, (20, 20), 1001, 10.0, 80.0, 1, 1, 16, 500, 10.0, 0.15, (0.05, 0.15), (3.0, 30.0)),
    1: (50, (30, 150), 4001, 10.0, 90.0, 1, 1, 256, 2000, 10.0, 0.15, (0.05, 0.15), (3.0, 30.0)),
    2: (50, (30, 150), 4001, 10.0, 90.0, 1, 32, 4096, 2000, 10.0, 0.15, (0.05, 0.15), (3.0, 30.0)),
    3: (50, (30, 150), 4001, 10.0, 90.0, 1024, 1, 128, 1000, 10.0, 0.15, (0.05, 0.15), (3.0, 30.0)),
    4: (1000, (50, 300), 8001, 5.0, 125.0, 1, 1, 256, 2000, 20.0, 0.3, (0.03, 0.3), (2.0, 12.0)),
}


def make_workload(cfg: int, n_patterns: int | None = None, n_restarts: int | None = None,
                  S: int | None = None, K: int | None = None, seed: int | None = None,
                  peak_counts: float | None = None, grid: tuple | None = None,
                  noise_frac: float = 0.01, asym: tuple | None = None) -> Workload:
    """Build config ``cfg`` (0..4).  Optional overrides shrink a config for tests
    (e.g. ``n_patterns=4`` for cfg 3) without changing its per-pattern recipe.

    ``peak_counts``: COUNT data for the paper's Poisson likelihood: signal + background
    are scaled so that their maximum is ``peak_counts`` and y ~ Poisson(signal + background) replaces the
    Gaussian noise; the planted scales h are multiplied by the same factor and ``hyper['likelihood'] = 1``.

    ``grid = (lo, hi, N)`` replaces the config's 2theta range and point count (same recipe otherwise), e.g. config 0
    on a 0.02 deg grid that resolves its peaks: ``grid=(10.0, 80.0, 3501)``.  ``noise_frac``: Gaussian noise sigma as a
    fraction of the maximum signal (the configs' 1 %).  ``asym = (lo, hi)``: every planted phase gets a peak asymmetry
    alpha ~ U(lo, hi) (split peaks); ``true_params`` entries then carry alpha as a fifth value and
    ``hyper['asymmetry'] = 1``."""
    if cfg not in _SPEC:
        raise ValueError(f"unknown config {cfg}")
    (K0, (mlo, mhi), N, lo, hi, P0, R0, S0, its, W, fwhm_ref, (fw_lo, fw_hi), (w_shape, w_rate)) = _SPEC[cfg]
    K = K0 if K is None else int(K)
    P = P0 if n_patterns is None else int(n_patterns)
    R = R0 if n_restarts is None else int(n_restarts)
    S = S0 if S is None else int(S)
    if grid is not None:
        lo, hi, N = float(grid[0]), float(grid[1]), int(grid[2])
    rng = np.random.default_rng((1000 + cfg) if seed is None else seed)

    x = lo + (hi - lo) * np.arange(N, dtype=np.float64) / (N - 1)

    # ---- candidate library ------------------------------------------------
    counts = rng.integers(mlo, mhi + 1, size=K)
    pos_list, int_list = [], []
    for k in range(K):
        p = np.sort(rng.uniform(lo, hi, size=counts[k]))
        i = 1.0 + rng.pareto(1.5, size=counts[k])
        pos_list.append(p)
        int_list.append(100.0 * i / i.max())

    # ---- which phases are planted ------------------------------------------
    n_conf = 2 if cfg in (1, 2, 3) else 0
    K_plain = K - n_conf                     # the last n_conf phases are confusers
    true_phases, true_params = [], []
    for pat in range(P):
        if cfg == 0:
            nt = 3
        elif cfg in (1, 2):
            nt = int(rng.integers(2, 5))
        elif cfg == 3:
            nt = int(rng.integers(1, 6))
        else:
            nt = 5
        nt = min(nt, K_plain)
        ids = np.sort(rng.choice(K_plain, size=nt, replace=False))
        true_phases.append([int(v) for v in ids])
        prm = {}
        for k in ids:
            prm[int(k)] = (float(rng.uniform(0.5, 2.0)), float(rng.normal(0.0, 0.02)),
                           float(rng.uniform(fw_lo, fw_hi)), float(rng.uniform(0.2, 0.8)))
            if asym is not None:
                prm[int(k)] = prm[int(k)] + (float(rng.uniform(asym[0], asym[1])),)
        true_params.append(prm)

    # ---- confusers: absent phases shadowing true phases of pattern 0 --------
    for c in range(n_conf):
        src = true_phases[0][c % len(true_phases[0])]
        p = np.sort(np.clip(pos_list[src] + rng.uniform(-0.1, 0.1, size=pos_list[src].shape[0]),
                            lo, hi))
        i = 1.0 + rng.pareto(1.5, size=p.shape[0])
        pos_list[K_plain + c] = p
        int_list[K_plain + c] = 100.0 * i / i.max()
        counts[K_plain + c] = p.shape[0]

    peak_ofs = np.zeros(K + 1, dtype=np.int64)
    peak_ofs[1:] = np.cumsum(counts)
    peak_pos = np.concatenate(pos_list).astype(np.float64)
    peak_int = np.concatenate(int_list).astype(np.float64)

    # ---- observed patterns --------------------------------------------------
    y = np.empty((P, N), dtype=np.float64)
    bg = np.empty((P, N), dtype=np.float64)
    for pat in range(P):
        sig = np.zeros(N, dtype=np.float64)
        for k, prm in true_params[pat].items():
            sig += _pseudo_voigt_pattern(x, pos_list[k], int_list[k], *prm)
        smax = float(sig.max())
        b0 = 0.02 * smax
        b1 = rng.uniform(-0.5, 0.5) * b0 / (hi - lo)
        bg[pat] = b0 + b1 * (x - lo)
        sigma_n = float(noise_frac) * smax
        if peak_counts is None:
            y[pat] = sig + bg[pat] + rng.normal(0.0, sigma_n, size=N)
        else:
            c = float(peak_counts) / float((sig + bg[pat]).max())
            bg[pat] *= c
            y[pat] = rng.poisson(c * sig + bg[pat]).astype(np.float64)
            true_params[pat] = {k: (prm[0] * c,) + tuple(prm[1:]) for k, prm in true_params[pat].items()}

    hyper = dict(window_W=W, fwhm_ref=fwhm_ref, w_shape=w_shape, w_rate=w_rate,
                 n_patterns=P, n_restarts=R)
    if peak_counts is not None:
        hyper["likelihood"] = 1
    if asym is not None:
        hyper["asymmetry"] = 1
    return Workload(cfg=cfg, two_theta=x, y=y, background=bg, peak_ofs=peak_ofs,
                    peak_pos=peak_pos, peak_int=peak_int, hyper=hyper, S=S, iterations=its,
                    true_phases=true_phases, true_params=true_params)


def random_state(K: int, P: int, R: int, seed: int, spread: float = 0.3, classes: int = 4) -> np.ndarray:
    """A seeded float32 variational state [P][R][2][K][classes] near a plausible fit
    (used by parity tests to probe ELBO/gradient away from the initial state); classes = 5 adds the
    asymmetry latent ln alpha ~ N(0, 0.15)."""
    rng = np.random.default_rng(seed)
    st = np.zeros((P, R, 2, K, classes), dtype=np.float32)
    st[:, :, 0, :, 0] = rng.normal(-3.0, 1.5 * spread + 0.5, size=(P, R, K))
    st[:, :, 0, :, 1] = rng.normal(0.0, 0.02, size=(P, R, K))
    st[:, :, 0, :, 2] = np.log(0.1) + rng.normal(0.0, spread, size=(P, R, K))
    st[:, :, 0, :, 3] = rng.normal(0.0, 1.0, size=(P, R, K))
    st[:, :, 1, :, :4] = np.log(0.1) + rng.normal(0.0, spread, size=(P, R, K, 4))
    if classes == 5:
        st[:, :, 0, :, 4] = rng.normal(0.0, 0.15, size=(P, R, K))
        st[:, :, 1, :, 4] = np.log(0.05) + rng.normal(0.0, spread, size=(P, R, K))
    return st
