/*
 * xrdvi.h -- C ABI of the B200-native ELBO-and-gradient hot path of
 * "Rapid, Comprehensive Search of Crystalline Phases from X-ray Diffraction in Seconds via
 * GPU-Accelerated Bayesian Variational Inference" (arXiv 2501.09308).
 *
 * Citations are PAPER.md:<line> (the paper's text) and DESIGN.md "Readings" R<n> (how a silent,
 * ambiguous or garbled passage is read; the same table binds the fp64 oracle).
 *
 * Problem statement (A1-A2): measured pattern D = {(x_i, y_i)}, i < N, and a
 * candidate set F = {F_k}, k < K, F_k = {(p_m, I_m)}, m < M_k (ragged).  Profile model
 * (A3-A8):
 *     f(x_i) = B(x_i) + sum_k h_k sum_m I_m [ (1-r_k) G(x_i; p_m+mu_k, w_k) + r_k L(x_i; p_m+mu_k, w_k) ]
 * with unit-area, FWHM-parameterised G and L (R1), a static +-n_c-point window per peak (R16), Gaussian
 * noise of known sigma_n (R3) or the paper's Poisson counts (A12-A16, hyper.likelihood = 1, R24), priors h~Exp(lambda_h) (eq.3), mu~N(0,mu_sigma),
 * w~Gam(w_shape, rate w_rate), r~U(0,1) (B.2), and a mean-field Gaussian q (eq.10,
 * PAPER.md:131) over the unconstrained latents zeta = (ln h, mu, ln w, logit r) (R6).
 *
 * General rules
 *  - Every function returns 0 (XRDVI_OK) or a negative XRDVI_E_* code; on failure outputs are
 *    untouched and xrdvi_last_error() (thread-local) describes the failure.  No exception or abort
 *    crosses this boundary.  There is NO CPU fallback: without a CUDA device of compute capability
 *    10.x every call fails with XRDVI_E_NOT_SM100 / XRDVI_E_CUDA.
 *  - Pointers are HOST pointers unless the parameter says "device".  The caller owns every array;
 *    inputs are copied during the call and never retained; outputs are written to caller memory.
 *  - All device work is enqueued on the stream given at create; calls that return host outputs
 *    synchronise that stream before returning.  Calls on one handle are not thread-safe.
 *  - Results are bitwise reproducible for equal inputs (all reductions have a fixed order).
 *
 * Layout of variational parameters ("state"): float [P][R][2][K][4]; [..][0] = m (mean), [..][1] =
 * l = log sigma; the last axis is the latent class (h, mu, w, r) -- (h, mu, w, r, alpha), i.e. [K][5], when
 * hyper.asymmetry = 1 (R30).  An "instance" is inst = pat*R + rst.
 */
#ifndef XRDVI_H
#define XRDVI_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct xrdvi xrdvi; /* opaque; one per problem (P patterns x R restarts) */

enum {
    XRDVI_OK = 0,
    XRDVI_E_INVALID_ARG = -1,
    XRDVI_E_UNSORTED_GRID = -2,      /* 2theta not strictly increasing                      */
    XRDVI_E_NONUNIFORM_GRID = -3,    /* 2theta not uniform to 1e-6 of the step and hyper.general_grid = 0, or its steps
                                        differ by more than a factor 16 (R16, R31: see xrdvi_create)         */
    XRDVI_E_EMPTY_PHASE = -4,        /* a phase with M_k = 0                                 */
    XRDVI_E_WORKSPACE_TOO_SMALL = -5,
    XRDVI_E_CUDA = -6,
    XRDVI_E_NOT_SM100 = -7
};

/* Hyper-parameters (POD, versioned by .size = sizeof(xrdvi_hyper)).  xrdvi_default_hyper fills the
 * paper's values (B.2; threshold PAPER.md:140) and the DESIGN.md readings.          */
typedef struct {
    uint32_t size;
    uint32_t _pad;
    double lambda_h;       /* rate of the Exp prior on h (eq.3).  <=0: auto 1/eta_h per pattern,
                              eta_h = max(y-B) * fwhm_ref / max(I) (R13)                          */
    double mu_sigma;       /* 0.03 deg (B.2)                                                      */
    double w_shape;        /* 3   (B.2)                                                           */
    double w_rate;         /* 100 (B.2; lambda is a RATE, R12)                                     */
    double noise_sigma;    /* Gaussian sigma_n.  <=0: auto 0.01 * max(y-B) per pattern (R4)       */
    double window_W;       /* static cutoff c = window_W * fwhm_ref (deg).  <=0: dense (R16)      */
    double fwhm_ref;       /* 0.15 deg                                                            */
    double incl_tau;       /* 0.01: area-ratio threshold (R15)                      */
    double lr, beta1, beta2, adam_eps; /* Adam ascent: 0.1, 0.9, 0.999, 1e-8 (R10)                */
    double init_log_sigma; /* ln 0.1 (R11)                                                        */
    int32_t n_patterns;    /* P >= 1                                                              */
    int32_t n_restarts;    /* R >= 1                                                              */
    int32_t likelihood;    /* 0 Gaussian with known sigma_n (R3, the graded path); 1 Poisson, the paper's
                              A12-A16: ll = sum y ln f - f - ln y!; needs y >= 0 and
                              background > 0 everywhere (R24), noise_sigma is ignored                */
    int32_t optimizer;     /* 0 Adam ascent (R10); 1 natural-gradient ascent of the mean-field Gaussian:
                              m += lr sigma^2 dELBO/dm, l += lr (dELBO/dl)/2, l clamped to [-12, 2] (R25);
                              plain steps, no trust region: needs a small lr (0.01 at config 0)             */
    int32_t asymmetry;     /* 1: the paper's peak asymmetry (A9/A10; R30): a FIFTH latent per phase,
                              alpha_k = exp(zeta_alpha) ~ Norm(alpha_mu, alpha_sigma); the high-angle side of every peak
                              (x >= p_m + mu_k) is alpha_k times wider at unchanged height (area (1 + alpha_k)/2).
                              Every [..][K][4] array of this header becomes [..][K][5] (class order h, mu, w, r, alpha);
                              xrdvi_latent_classes() returns the count.  0 (default): the four-latent model          */
    int32_t width_sec;     /* 1: angle-dependent width w_k sec(p_m / 2) per peak (the sec of; R30)      */
    double alpha_mu;       /* 1.00 (B.2)                                                          */
    double alpha_sigma;    /* 0.20 (B.2)                                                                        */
    int32_t general_grid;  /* 0 (default): two_theta must be uniform (the fast path).  1: any strictly increasing grid whose
                              steps differ by at most a factor 16 (R31): j_m = the grid point nearest to p_m, the window stays
                              |i - j_m| <= n_c with n_c from the MEAN step; the kernels read per-tile point offsets and
                              per-record bases (x_{i0} - p_m, fp64-computed) instead of (i - j_m) Delta, every record takes
                              the per-point bodies (about half the speed).  The flag sizes the workspace, so it is part
                              of xrdvi_workspace_bytes' input; a uniform grid is accepted with it as well               */
    int32_t _pad2;
} xrdvi_hyper;

void xrdvi_default_hyper(xrdvi_hyper* hyp);

/* Bytes of device workspace xrdvi_create needs for draws up to S_max per (pattern, restart).
 * two_theta_step = (two_theta[N-1] - two_theta[0]) / (N-1), the grid step in degrees (it fixes the window
 * half-width n_c, R16).  Depends only on the sizes (an upper bound over peak positions).  0 on invalid
 * arguments.                                                                                       */
size_t xrdvi_workspace_bytes(int64_t N, int32_t K, int64_t M, int32_t S_max, double two_theta_step,
                             const xrdvi_hyper* hyp);

/* Build a problem.
 *  two_theta [N]     strictly increasing (deg).  Uniform (the paper's grid) is the fast path: the peak
 *                    encoding (nearest grid index + fp64 offset, R16) and the packed bodies use the constant step.  A
 *                    grid that departs from uniform by more than 1e-6 of the step needs hyper.general_grid = 1 (R31),
 *                    else XRDVI_E_NONUNIFORM_GRID
 *  y [P][N]          observed intensities;  background [P][N] or NULL (-> 0) (R5: B is an input)
 *  peak_ofs [K+1]    CSR offsets into peak_pos / peak_int ([M], M = peak_ofs[K]); any order inside
 *                    a phase; peaks with no in-window grid point are dropped (R16)
 *  device, cuda_stream   CUDA device ordinal and a cudaStream_t the library enqueues all its work on.  It must be
 *                    capturable into a CUDA Graph; NULL (the legacy default stream cannot be captured) makes
 *                    xrdvi_create create a private non-blocking stream, destroyed by xrdvi_destroy
 *  workspace         DEVICE pointer, >= xrdvi_workspace_bytes(...) bytes, 256-byte aligned, owned by
 *                    the caller and kept alive until xrdvi_destroy
 * Preprocessing (sorting, grid-index encoding j_m/delta_m, window tables) is done on the host in
 * fp64; the state is initialised as xrdvi_reset_state(h, 0).                                       */
int xrdvi_create(const double* two_theta, int64_t N, const double* y, const double* background,
                 int32_t K, const int64_t* peak_ofs, const double* peak_pos, const double* peak_int,
                 const xrdvi_hyper* hyp, int32_t S_max, int device, void* cuda_stream,
                 void* workspace, size_t workspace_bytes, xrdvi** out);

void xrdvi_destroy(xrdvi* h);

/* In-window (m,i) pairs per sample-instance: the unit of the throughput metric.                    */
int64_t xrdvi_pair_count(const xrdvi* h);
/* Latent classes per phase C: 4 (h, mu, w, r), or 5 with hyper.asymmetry (+ alpha).  Wherever this header writes
 * [K][4] (states, gradients, moments, zeta, summaries) the last axis has C entries.                   */
int32_t xrdvi_latent_classes(const xrdvi* h);
/* Window half-width n_c in grid points (N for dense).                                              */
int64_t xrdvi_window_halfwidth(const xrdvi* h);

/* ---- Per-phase (adaptive) windows: DESIGN.md reading R27 of north_star's "pseudo-Voigt truncated at a
 * problem-defined +-W FWHM cutoff" (second half).  The paper evaluates every peak on
 * the whole grid; the window is this build's model reading R16.
 *
 * xrdvi_set_phase_windows: replace the static half-width n_c by per-phase ones, n_ck int32 [K] HOST,
 *   0 <= n_ck[k] <= n_c (the create-time window sizes the workspace); NULL restores the static window.  A pair
 *   (m, i), m a peak of phase k, is in the model iff |i - j_m| <= n_ck[k] and 0 <= i < N.  Rebuilds the per-tile
 *   tables on the host (integers only) and uploads them; variational state, Adam moments and step counter are
 *   untouched; xrdvi_pair_count follows.  Synchronises the stream.  XRDVI_E_INVALID_ARG on a dense problem
 *   (window_W <= 0) or an out-of-range value (nothing changed then).
 * xrdvi_get_phase_windows: the half-widths in force, n_ck int32 [K] HOST (all n_c after create).
 * xrdvi_adapt_windows: the refresh rule.  Reads the variational state and sets
 *     n_ck[k] = min(n_c, max(ceil(2 W - 1e-9), ceil(max_inst(W E_q[w_k] + |E_q[mu_k]|) / Delta - 1e-9))),
 *     E_q[w_k] = exp(m_w + sigma_w^2 / 2), E_q[mu_k] = m_mu, the maximum over the (pattern, restart) instances,
 *   i.e. +-W FWHM around the shifted peak centre at the variational means, never narrower than the window of
 *   a peak of FWHM 2 Delta.  fp64 on the host from the fp32 state.  n_ck_out int32 [K] HOST or NULL.
 * xrdvi_fit_adaptive: `iterations` steps as xrdvi_fit, in pieces of `refresh_every` steps with
 *   xrdvi_adapt_windows(h, W) between the pieces (not after the last).  Starts from the windows in force and
 *   leaves the last refreshed ones in force.  Outputs as xrdvi_fit (host buffers, NULL to skip; elbo_trace
 *   rows older than 4096 steps within a piece are NaN).                                                     */
int xrdvi_set_phase_windows(xrdvi* h, const int32_t* n_ck);
int xrdvi_get_phase_windows(const xrdvi* h, int32_t* n_ck);
int xrdvi_adapt_windows(xrdvi* h, double W, int32_t* n_ck_out);
int xrdvi_fit_adaptive(xrdvi* h, int32_t iterations, int32_t S, uint64_t seed, int32_t refresh_every, double W,
                       float* var_params_out, double* incl_prob, double* elbo_trace);

/* (Re)initialise the variational state (R11), zero the Adam moments and the step counter.
 * Restart r > 0 is jittered with Philox counter (0xFFFFFFFF, r, k, pat) under `seed`.
 * xrdvi_reset_state_restart: the same with the restart index shifted, r = rst + restart_offset >= 0 -- instance
 * (pat, rst) starts where restart rst + restart_offset of a larger problem would (independent replicas of one
 * problem on several GPUs: rank as the offset gives every replica its own jittered start).            */
int xrdvi_reset_state(xrdvi* h, uint64_t seed);
int xrdvi_reset_state_restart(xrdvi* h, uint64_t seed, int32_t restart_offset);
/* Copy the state out / in: var_params float [P][R][2][K][4].  set_state sets the step counter to `step` (number of
 * completed optimisation steps; the next step draws with Philox iteration step + 1) and starts a FRESH Adam: the
 * moments are zeroed and the bias correction restarts with them (first step after set_state = lr * sign(g)).
 * To continue a fit exactly (checkpoint / resume), also carry the optimiser state:
 * xrdvi_get_optimizer_state: mom1, mom2 float [P][R][2][K][4] (Adam's first / second moments; either may be NULL),
 *   *adam_steps = steps the moments have accumulated (the exponent of the bias correction).
 * xrdvi_set_optimizer_state: after xrdvi_set_state; 0 <= adam_steps <= step.  fit(n) + get_state +
 *   get_optimizer_state, then set_state + set_optimizer_state + fit(m) on any handle of the same problem is bitwise
 *   fit(n + m) (tested).                                                                              */
int xrdvi_get_state(xrdvi* h, float* var_params, int64_t* step);
int xrdvi_set_state(xrdvi* h, const float* var_params, int64_t step);
int xrdvi_get_optimizer_state(xrdvi* h, float* mom1, float* mom2, int64_t* adam_steps);
int xrdvi_set_optimizer_state(xrdvi* h, const float* mom1, const float* mom2, int64_t adam_steps);

/* One ELBO-and-gradient evaluation (eq.7 PAPER.md:111 as a Monte-Carlo mean over S reparameterised
 * draws + analytic entropy, R7/R8):
 *  var_params   float [P][R][2][K][4] or NULL (use the internal state; it is not modified)
 *  S            draws per (pattern, restart), 1 <= S <= S_max
 *  seed, iteration   Philox4x32-10 key and counter word 0; draw (s, k, inst) uses counter
 *               (iteration, s, k, inst) (R18)
 *  elbo         double [P][R];   grad  float [P][R][2][K][4] = d ELBO / d (m, l); either may be NULL */
int xrdvi_elbo_grad(xrdvi* h, const float* var_params, int32_t S, uint64_t seed, uint64_t iteration,
                    double* elbo, float* grad);

/* `iterations` ascent steps (Adam, or natural gradient if hyper.optimizer = 1) from the internal state, each one a replay of a CUDA
 * Graph; step t uses Philox iteration t, t
 * continuing from the state's step counter + 1 (the graph holds two kernels: the fused profile/residual/
 * backward kernel and the reduce + Adam + next-draw kernel).  Outputs (each may be NULL, nothing is copied then):
 *  var_params_out float [P][R][2][K][4]; incl_prob double [P][R][K] (R15);
 *  elbo_trace double [iterations][P][R] (only the last 4096 iterations are kept; older rows = NaN)  */
int xrdvi_fit(xrdvi* h, int32_t iterations, int32_t S, uint64_t seed, float* var_params_out,
              double* incl_prob, double* elbo_trace);

/* Posterior inclusion probability and area ratio per phase from the internal state (R15):
 * incl_prob, area_ratio double [P][R][K], either may be NULL.                                      */
int xrdvi_inclusion(xrdvi* h, double* incl_prob, double* area_ratio);

/* Marginal summaries of the fitted q in the constrained parameters (R28; the posterior marginals of the
 * paper's Fig. 6, SURVEY.md 8(f) NEXT-4 second half), from the internal state, computed on the device in fp64:
 * zeta ~ N(m, sigma^2) (eq.(10)) pushed through the bijections of R6 -- h, w log-normal, mu normal,
 * r logit-normal (mean / sd by quadrature).
 *  summary  host double [P][R][K][4][5], classes (h, mu, w, r) x (mean, sd, 2.5 %, 50 %, 97.5 % quantile); owned by
 *           the caller, must not be NULL (XRDVI_E_INVALID_ARG).  Synchronous on the handle's stream.          */
int xrdvi_posterior_summary(xrdvi* h, double* summary);

/* Log-joint gradient service: log p(Y, Phi) + log |dPhi/dzeta| and its gradient at n
 * caller-supplied points of the unconstrained latent space, for one pattern -- what a gradient-based sampler of the
 * paper's model (the MCMC rows of Table 1) evaluates per leapfrog step.  The same
 * profile / residual / backward kernels run on the points as on Monte-Carlo draws; no variational state is read
 * or modified (the per-step draw buffers are overwritten).
 *  zeta     float [n][K][4] = (ln h, mu, ln w, logit r) per phase (R6);  1 <= n <= S_max rounded up to 32
 *  pattern  index of the observed pattern, 0 <= pattern < P
 *  ll       double [n]: log-likelihood (Gaussian or Poisson, hyper.likelihood)
 *  lpj      double [n]: log prior + log Jacobian;   grad float [n][K][4] = d (ll + lpj) / d zeta
 *  ll, lpj, grad may each be NULL.                                                                           */
int xrdvi_logjoint_grad(xrdvi* h, const float* zeta, int64_t n, int32_t pattern, double* ll, double* lpj,
                        float* grad);

/* Model profile and log-likelihood of chosen draws WITHOUT any allocation and without caller scratch, for callers that
 * cannot call cudaMalloc (tight serving loops, harnesses that forbid it, code around a CUDA graph capture): draw +
 * forward pass (a-1 .. a-4: eq.(3)-(8) PAPER.md:206-232 profile, residual, ll) at (var_params or the internal state
 * when NULL, S, seed, iteration), exactly as the fit evaluates them.  The profile rows pass through a file-scope
 * `static __device__` array of the library: 1 048 576 floats = 4 MiB on every GPU that loads the library, held until the
 * process exits; its device address is resolved once per device in xrdvi_create (cudaGetSymbolAddress).
 *  var_params  host float [P][R][2][K][C] (C = xrdvi_latent_classes) or NULL;  1 <= S <= S_max
 *  first, n    the sample-instances first .. first + n - 1 in (pattern, restart, s) order, 0 <= first, first + n <= P R S
 *  f           host float [n][N]: S_F + B of each row (owned by the caller), or NULL
 *  ll          host double [n]: log-likelihood of each row, or NULL
 * Limit: n * N <= 1 048 576 when f is wanted, else XRDVI_E_WORKSPACE_TOO_SMALL (message states both numbers; ask for fewer
 * rows per call).  XRDVI_E_INVALID_ARG for S / first / n out of range; XRDVI_E_CUDA if the array's address could not be
 * resolved at create.  Calls no cudaMalloc / cudaFree / allocating routine, host or device.  Synchronous on the handle's
 * stream; the variational state is not modified (the per-step draw buffers are overwritten, as by xrdvi_elbo_grad).
 * EVERY call on a GPU, from any handle, shares the one array, which keeps the last call's rows (each call zeroes the
 * part it uses first): calls whose GPU work overlaps (handles on different streams, several host threads) RACE on it --
 * serialise them.                                                                                               */
int xrdvi_profile_static(xrdvi* h, const float* var_params, int32_t S, uint64_t seed, uint64_t iteration,
                         int64_t first, int64_t n, float* f, double* ll);

const char* xrdvi_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* XRDVI_H */
