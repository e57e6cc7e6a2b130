// xrdvi_kernels.cuh -- sm_100a kernels of the ELBO-and-gradient hot path.
//
// Data-parallel axes: a *sample-instance* t = (pattern, restart, draw s) lives in one LANE; 32
// consecutive draws of one (pattern, restart) form a *group* g, so every warp works on one run of grid
// points for 32 draws at once: peak records and observed data are warp-uniform (broadcast loads),
// latents are lane-private, all global traffic is 128-byte coalesced.
//
// One optimisation step is two kernels:
//   elbo_tile_kernel   (a-3, a-4, a-5, a-6 likelihood part) one CTA per (TW consecutive 16-point tiles, group).
//                      Every tile has a static, PHASE-MAJOR list of the peaks whose window reaches it, split at
//                      phase boundaries into PS shares; warp (tile, share) walks its share twice:
//                      phase 1 synthesises the profile of the tile in 16 registers per lane (the PS partial
//                      profiles are summed through shared memory), the residual e = (y - f)/sigma_n^2 goes
//                      back to all shares through shared memory and then lives in REGISTERS;
//                      phase 2 accumulates the six backward sums of each peak over the 16 points, folds them
//                      per phase, applies the chain rule and reduces over the 32 draws with warp shuffles
//                      (fixed tree) to 8 floats per (tile, phase, group).
//   elbo_split_kernel  the same two phases as one-warp work items on a ticket queue, partial profiles through
//                      L2 instead of a CTA barrier; chosen for launches with few tile-warps and long items.
//   update_draw_kernel (a-6 prior part, a-7, a-8, a-1, a-2) one CTA per (phase, instance): fixed-order
//                      reduction of the partials and of the per-draw prior terms, ELBO, Adam ascent
//                      on the 8 variational parameters of the phase, then the Philox draws and the
//                      transform for the NEXT step.
//
// Coordinates: t' = 2 (x_i - p_m - mu) / w, so that  G = exp(-4 ln2 t^2) = 2^(-t'^2)  and
// L = 1/(1+4t^2) = 1/(1+t'^2)  (PAPER.md:221-232 with the unit-area FWHM shapes, reading R1).  A peak is
// stored as (j_m, delta_m) with p_m = x_{j_m} + delta_m computed in fp64 at create, so
// t' = (i - j_m) * (Delta*2/w) + (-delta_m - mu) * 2/w  has no fp32 cancellation at high angles.
//
// Instruction diet: the path is bound by SM issue slots (4 warp-instructions per
// clock), then by the MUFU pipe (16 lanes/SM/clk, shared by ex2 and rcp).  Measures:
//   * Gaussian core / Lorentz tail: 2^(-t'^2) < 2^-24 for |t'| > 4.9, so outside a per-(group, phase)
//     core half-width n_g (from the largest sampled w and |mu| of the 32 draws) only L is evaluated;
//   * shared reciprocal: 1/ua and 1/ub of two neighbouring points come from ONE rcp(ua*ub);
//   * (peak, tile) pairs whose 16 points are all in-window and all tail take a branch-free unrolled body;
//     the others are processed quad by quad (out-of-window quads skipped, partial quads masked);
//   * backward first moments use t' = t0 + p*step: sum e L^2 t' = t0 sum e L^2 + step sum (p e) L^2 with
//     p*e held in registers, so the inner loop needs no multiplication by t'.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace xrdvi_dev {

constexpr int kPT = 16;         // grid points per thread in phase 1 (one warp = one 16-point tile)
constexpr int kTraceCap = 4096; // iterations of ELBO trace kept on the device
constexpr int kUpdThreads = 256;
constexpr float kGaussCut = 4.9f;   // |t'| beyond which 2^(-t'^2) < 2^-24 is dropped

constexpr float kAG = 0.93943727869965132f;  // 2 sqrt(ln2/pi)
constexpr float kAL = 0.63661977236758134f;  // 2/pi
constexpr float kLn2 = 0.69314718055994531f;

struct __align__(16) PeakRec {   // 16 bytes (one LDG.128); one record per (peak, 16-point tile its window reaches)
    int dj;        // nearest grid index j_m of the peak minus the first grid index of the tile
    float delta;   // p_m - x_{j_m}  (|delta| <= Delta/2), fp64-computed
    float inten;   // I_m
    int full;      // bit 0: all 16 points of the tile exist and lie inside the peak's window; bits 1..30: the window
                   // half-width n_c,k of the peak's phase in points (per-phase windows, R27; read by the edge bodies)
};

struct PatConst {  // per observed pattern
    float inv_sn;      // 1/sigma_n
    float inv_sn2;     // 1/sigma_n^2
    float lambda_h;    // rate of the Exp prior
    float log_lambda_h;
    double ll_const;   // Gaussian: -N ln sigma_n - N/2 ln 2pi;  Poisson: sum_i (y ln y - y - ln y!)
    float ll_scale;    // ll = ll_scale * (sum of llpart) + ll_const: -1/2 (Gaussian), 1 (Poisson)
    float pad;
};

struct Ctl {       // device-resident control block (so that graph replays need no new arguments)
    unsigned long long seed;
    long long step;        // completed optimisation steps
    long long trace_base;  // step index of trace row 0
    long long iteration_override;  // >= 0: Philox iteration for elbo_grad/debug; < 0: use step + 1
    long long adam_t0;             // step count at which the Adam moments were last zeroed: bias correction uses step + 1 - adam_t0
    unsigned int pending;          // update_draw_kernel has run and finish_step has not: 1 evaluation, 2 step
    unsigned int ticket;           // next work item of elbo_split_kernel (re-armed by the launch's last CTA)
    unsigned int finished;         // CTAs of the current elbo_split_kernel launch that are done
    unsigned int pad;
    // The step as update_draw_kernel sees it, kept by that kernel itself so that it may be read BEFORE griddep_wait
    // (finish_step of the tile kernel moves `step`): step = u_step + u_acc / (CTAs of a launch).  The host sets u_step =
    // step and u_acc = 0 at the start of a run; every CTA of an optimisation step adds 1 to u_acc when it is done
    // (fire and forget).  A CTA of a later wave of the same launch reads u_acc with some of that launch's additions
    // in it, but never all of them (its own is missing), so the quotient is the same for every CTA of a launch.
    long long u_step;
    unsigned long long u_acc;
};

struct Dev {
    // sizes
    int N, K, P, R, PR, n_c, n_seg, n_tile, n_slots, TW, PS;   // n_seg = ceil(n_tile / TW) segments of TW tiles
    int S, gpi, G;       // draws, groups per instance, groups (run-time)
    int likelihood;      // 0 Gaussian with known sigma_n (R3), 1 Poisson (A12-A16; R24)
    int optimizer;       // 0 Adam (R10), 1 natural gradient (R25)
    int split;           // 1: backward launches with PS > 1 use elbo_split_kernel (long work items)
    float delta;         // grid step (deg)
    float gcut;          // kGaussCut / (2 Delta): core half-width in points per unit of w
    float inv_delta;
    // priors / optimiser
    float mu_inv_var, mu_logc, w_shape, w_rate, w_logc;
    float lr, beta1, beta2, adam_eps;
    // static tables
    const float* yb;          // [P][N]  y - B
    const float* bg;          // [P][N]
    const PeakRec* pk_tile;   // per-tile phase-major peak lists, concatenated (+1 padding record)
    const int4* run_tab;      // [n_slots + 1] phase runs of the tile lists: (m0, m1) range in pk_tile, .z = phase,
                              //               .w = output slot in part8 (slots are numbered phase-major)
    const int2* share_rng;    // [n_tile][PS]: range of runs of the share
    const int* seg_order;     // [n_seg] segments (TW tiles) by decreasing work (LPT dispatch order)
    const int* slot_ofs;      // [K+1] output slots of phase k: [slot_ofs[k], slot_ofs[k+1]), tiles in increasing order
    const PatConst* pat;      // [P]
    const double* area;       // [K] A_k = sum_m I_m
    // state
    float* var;               // [PR][2][K][4]
    float* mom1;
    float* mom2;
    float* grad;              // [PR][2][K][4]
    double* elbo;             // [PR]
    double* elbo_k;           // [PR][K+1]  per-phase ELBO terms ([K] unused)
    double* ll_t;             // [PR][S_pad]
    double* ll_g;             // [G] sum of ll_t over the 32 draws of a group
    double* trace;            // [kTraceCap][PR]
    Ctl* ctl;
    // per-iteration buffers
    float4* lat;              // [G][K][32]  (2/w, -mu*2/w, h(1-r)aG/w, h r aL/w)
    float4* eps;              // [G][K][32]
    float* rr;                // [G][K][32]  r
    int* ng;                  // [G][K]      Gaussian core half-width in grid points
    float* llpart;            // [G][n_seg][32] the segment's part of ll (tile_residual), per draw
    float* part8;             // [G][n_slots][8] (g_h, g_mu, g_w, g_r, g_h eps_h, ...) summed over 32 draws
    // log-joint gradient service (xrdvi_logjoint_grad): per-draw output instead of the sum over the draws
    float* partial;           // [G][n_tile][PS][16][32] partial profiles of elbo_split_kernel (PS > 1 only)
    unsigned int* tile_cnt;   // [G][n_tile] partial profiles that have arrived
    unsigned int* tile_cnt2;  // [G][n_tile] phase-2 items that are done
    float* pd;                // nullptr, or [groups of the launch][n_slots][4][32] d ll / d zeta per (run, class, draw)
    int g_base;               // group of blockIdx.x = 0 in elbo_tile_kernel (0 except in the service)
    long long dbg_first;      // first sample-instance of the debug profile read-back (xrdvi_debug_profile)
    const int2* tile_rng;     // [n_tile + 1] (first run, first record) of every tile's lists
    int stage;                // 1: elbo_tile_kernel copies the tile's lists into shared memory (they fit: host check)
    int g_block;              // draw groups per dispatch chunk of elbo_tile_kernel (their latent records stay in L2)
    int upd_smem;             // dynamic shared memory of update_draw_kernel launches (bytes; its short path stages slot rows there)
    // peak asymmetry and the sec width term (reading R30; hyper.asymmetry / hyper.width_sec).  asym = 1: a fifth latent
    // alpha_k per phase; every state array has a companion for it ([PR][2][K]: m_alpha, l_alpha)
    int asym, sec;
    int general;              // 1: non-uniform 2theta grid (R31): per-tile point offsets and per-record bases instead of (i - j) Delta
    float reach_pad;          // slack of the Gaussian-core half-width in points: 1.5 on a uniform grid (|delta_m| <= Delta/2, rounding)
    const float* tile_off;    // [n_tile][16] x_{i0 + p} - x_{i0} (general = 1)
    const float* pk_base;     // [records] x_{i0} - p_m of the record's tile and peak, fp64-computed (general = 1)
    int model;                // 1: asym, sec or general is on: the tile kernels run tile_phase*_asym (per-draw rows of 160 floats)
    float alpha_mu, alpha_inv_var, alpha_logc;   // prior Norm(alpha_mu, alpha_sigma): mean, 1/sigma^2, -ln(sigma sqrt(2 pi))
    const float* pk_sec;      // [records] cos(p_m / 2) = 1 / sec factor of the record's peak (sec = 1 only)
    const float* sec_max;     // [K] largest sec factor of the phase's peaks (1 without the sec term)
    float* var_a;             // [PR][2][K]
    float* mom1_a;
    float* mom2_a;
    float* grad_a;
    float* ia;                // [G][K][32] 1 / alpha of the draw
    float* eps_a;             // [G][K][32]
    float* parta;             // [G][n_slots][2] (g_alpha, g_alpha eps_alpha) summed over the 32 draws
    // measurement (xrdvi_debug_timeline): nullptr, or [warps of the launch][4] = (start, end of phase 1, end, SM id | records << 32)
    unsigned long long* tl;
    // measurement (xrdvi_debug_update_timeline): nullptr, or [CTAs of update_draw_kernel][8] %globaltimer stamps of
    // thread 0 of every CTA of update_draw_kernel<true>
    unsigned long long* tlu;
};

// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// Programmatic dependent launch (sm_90+): a kernel launched with the programmatic-serialization attribute may start
// before its predecessor in the stream has finished; griddep_wait() blocks until the predecessor has completed and
// its writes are visible (a no-op for a normal launch), griddep_launch_dependents() lets the successor start
// launching.  Everything that reads or overwrites data of the predecessor comes after griddep_wait().  The tile kernels
// call griddep_launch_dependents() AFTER their griddep_wait(): their successor, update_draw_kernel, may then read
// before its own wait whatever the kernels before the tile kernel wrote (they have completed).
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
// Per-warp timeline stamps of the tile kernels (xrdvi_debug_timeline; d.tl == nullptr in every other launch, a
// warp-uniform test on a kernel parameter).  Each stamp is stored at once, nothing stays live across the phases.
__device__ __forceinline__ void tl_stamp(unsigned long long* tl, unsigned row, int col) {
    if (tl && (threadIdx.x & 31) == 0) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        tl[static_cast<size_t>(row) * 4 + col] = t;
    }
}
__device__ __forceinline__ void tlu_stamp(unsigned long long* tlu, unsigned row, int col) {   // thread 0 of a CTA
    if (tlu && threadIdx.x == 0) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        tlu[static_cast<size_t>(row) * 8 + col] = t;
    }
}
__device__ __forceinline__ void tl_tag(unsigned long long* tl, unsigned row, int records) {
    if (tl && (threadIdx.x & 31) == 0) {
        unsigned sm;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(sm));
        tl[static_cast<size_t>(row) * 4 + 3] = sm | (static_cast<unsigned long long>(records) << 32);
    }
}
__device__ __forceinline__ void griddep_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

__device__ __forceinline__ float rcp_approx(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Philox4x32-10 (Salmon et al., SC'11), counter (c0..c3), key (k0,k1).
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        const unsigned hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
        k.x += 0x9E3779B9u;
        k.y += 0xBB67AE85u;
    }
    return c;
}

__device__ __forceinline__ float uniform23(unsigned w) {
    return (static_cast<float>(w >> 9) + 0.5f) * (1.0f / 8388608.0f);  // exact in fp32
}

__device__ __forceinline__ float4 normals_from_words(uint4 w) {
    const float u0 = uniform23(w.x), u1 = uniform23(w.y), u2 = uniform23(w.z), u3 = uniform23(w.w);
    const float r0 = sqrtf(-2.0f * logf(u0)), r1 = sqrtf(-2.0f * logf(u2));
    float s0, c0, s1, c1;
    sincospif(2.0f * u1, &s0, &c0);
    sincospif(2.0f * u3, &s1, &c1);
    return make_float4(r0 * c0, r0 * s0, r1 * c1, r1 * s1);
}

struct Phys { float zh, zw, zr, h, mu, w, r; };

// zeta = m + exp(l) * eps; h = exp(zeta_h), mu = zeta_mu, w = exp(zeta_w), r = sigmoid(zeta_r)  (R6)
__device__ __forceinline__ Phys transform(const float4 m, const float4 sg, const float4 ep) {
    Phys q;
    q.zh = fmaf(sg.x, ep.x, m.x);
    q.mu = fmaf(sg.y, ep.y, m.y);
    q.zw = fmaf(sg.z, ep.z, m.z);
    q.zr = fmaf(sg.w, ep.w, m.w);
    q.h = expf(q.zh);
    q.w = expf(q.zw);
    q.r = 1.0f / (1.0f + expf(-q.zr));
    return q;
}

__device__ __forceinline__ long long philox_iteration(const Ctl* ctl) {
    const long long o = ctl->iteration_override;
    return o >= 0 ? o : ctl->step + 1;
}

// a-2, second half: latent record, eps, r and the group's Gaussian-core half-width of phase k for the lane's
// draw.  Must be called by all 32 lanes of a warp whose lanes hold consecutive draws of group g (the core
// half-width n_g is a warp maximum); `valid` = false for padding lanes, which contribute nothing.
__device__ __forceinline__ void emit_latent(const Dev& d, int g, int k, bool valid, const Phys& q, const float4 ep,
                                            float alpha = 1.0f, float ep_a = 0.0f) {
    const int lane = threadIdx.x & 31;
    // 1/w is capped at 5e7 (w >= 2e-8 deg: far outside the model's regime) so that the shared reciprocal
    // rcp(ua ub) of two points can never see an overflowed product
    const float iw = fminf(1.0f / q.w, 5.0e7f);
    const float iw2 = 2.0f * iw;
    float4 lt = make_float4(iw2, -q.mu * iw2, q.h * (1.0f - q.r) * kAG * iw, q.h * q.r * kAL * iw);
    // Gaussian core half-width in grid points for this draw: |t'| <= kGaussCut  <=>
    // |i - j| <= kGaussCut w / (2 Delta) + |delta_m + mu| / Delta; |delta_m| <= Delta/2, +1 for rounding
    // (R30: the high-angle side is alpha times wider, the widest peak of the phase sec_max times)
    float wide = q.w;
    if (d.asym) wide *= fmaxf(alpha, 1.0f);
    if (d.sec) wide *= d.sec_max[k];
    float reach = fmaf(d.gcut, wide, fabsf(q.mu) * d.inv_delta) + d.reach_pad;
    if (!valid) {
        lt = make_float4(1.0f, 0.0f, 0.0f, 0.0f);
        reach = 0.0f;
    }
    if (!(reach < 1.0e9f)) reach = 1.0e9f;  // also catches NaN
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) reach = fmaxf(reach, __shfl_xor_sync(0xffffffffu, reach, o));
    const size_t o = (static_cast<size_t>(g) * d.K + k) * 32 + lane;
    d.lat[o] = lt;
    d.eps[o] = ep;
    d.rr[o] = q.r;
    if (d.asym) {
        d.ia[o] = valid ? fminf(1.0f / alpha, 1.0e6f) : 1.0f;
        d.eps_a[o] = ep_a;
    }
    if (lane == 0) d.ng[static_cast<size_t>(g) * d.K + k] = static_cast<int>(reach) + 1;
}

// R30: the normal of the fifth latent: first Box-Muller output of a second Philox call, bit 31 of the phase word set.
__device__ __forceinline__ float normal_alpha(unsigned it, unsigned s, unsigned k, unsigned inst, unsigned long long seed) {
    const uint4 w = philox4x32_10(make_uint4(it, s, k | 0x80000000u, inst),
                                  make_uint2(static_cast<unsigned>(seed), static_cast<unsigned>(seed >> 32)));
    const float u0 = uniform23(w.x), u1 = uniform23(w.y);
    float sn, cs;
    sincospif(2.0f * u1, &sn, &cs);
    return sqrtf(-2.0f * logf(u0)) * cs;
}

// a-1 + a-2 for one (instance, phase k, draw s): Philox draw, transform, latent record (all 32 lanes of a warp).
__device__ __forceinline__ void draw_one(const Dev& d, int inst, int k, int s, unsigned it, unsigned long long seed,
                                         const float4 m, const float4 l, uint4* __restrict__ raw_out,
                                         float m_a = 0.0f, float l_a = 0.0f) {
    const int g = inst * d.gpi + (s >> 5);
    const uint4 words = philox4x32_10(make_uint4(it, static_cast<unsigned>(s), static_cast<unsigned>(k),
                                                 static_cast<unsigned>(inst)),
                                      make_uint2(static_cast<unsigned>(seed), static_cast<unsigned>(seed >> 32)));
    const float4 ep = normals_from_words(words);
    const float4 sg = make_float4(expf(l.x), expf(l.y), expf(l.z), expf(l.w));
    float alpha = 1.0f, ep_a = 0.0f;
    if (d.asym) {
        ep_a = normal_alpha(it, static_cast<unsigned>(s), static_cast<unsigned>(k), static_cast<unsigned>(inst), seed);
        alpha = expf(fmaf(expf(l_a), ep_a, m_a));
    }
    emit_latent(d, g, k, s < d.S, transform(m, sg, ep), ep, alpha, ep_a);
    if (raw_out) raw_out[(static_cast<size_t>(g) * d.K + k) * 32 + (threadIdx.x & 31)] = words;
}

// Stand-alone draw kernel (first step of a fit, xrdvi_elbo_grad, debug).  grid (ceil(K/4), G), block 128.
__global__ void __launch_bounds__(128) draw_transform_kernel(const Dev d, const float* __restrict__ var,
                                                              uint4* __restrict__ raw_out) {
    const int lane = threadIdx.x & 31;
    const int k = blockIdx.x * 4 + (threadIdx.x >> 5);
    const int g = blockIdx.y;
    if (k >= d.K) return;
    const int inst = g / d.gpi;
    const int s = (g - inst * d.gpi) * 32 + lane;
    const float4 m = *reinterpret_cast<const float4*>(var + (static_cast<size_t>(inst) * 2 * d.K + k) * 4);
    const float4 l = *reinterpret_cast<const float4*>(var + (static_cast<size_t>(inst) * 2 * d.K + d.K + k) * 4);
    float m_a = 0.0f, l_a = 0.0f;
    if (d.asym) {   // the companion of `var` for alpha sits right behind it: var_a = var + PR * 8 * K (host layout)
        const float* va = var + static_cast<size_t>(d.PR) * 8 * d.K;
        m_a = va[static_cast<size_t>(inst) * 2 * d.K + k];
        l_a = va[static_cast<size_t>(inst) * 2 * d.K + d.K + k];
    }
    draw_one(d, inst, k, s, static_cast<unsigned>(philox_iteration(d.ctl)), d.ctl->seed, m, l, raw_out, m_a, l_a);
}

// ------------------------------------------------------------------------------------------------
// Packed FP32x2 arithmetic (Blackwell: fma/mul/add.rn.f32x2 on 64-bit register pairs).  One instruction does two
// IEEE single-precision operations: the same FP32 rate as FFMA, HALF the issue slots -- and the path is bound by
// issue slots (profiles/).  A quad of grid points 4Q .. 4Q+3 is held as X = (4Q, 4Q+2), Y = (4Q+1, 4Q+3), so that
// the two shared reciprocals of a quad, r = (1/(u_a u_b), 1/(u_c u_d)), give L_X = r * u_Y and L_Y = r * u_X without
// any swap of register halves.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 rcp2(f32x2 v) {      // two MUFU.RCP on the halves
    float lo, hi;
    unpack2(v, lo, hi);
    return pack2(rcp_approx(lo), rcp_approx(hi));
}
__device__ __forceinline__ f32x2 ex2neg2(f32x2 v) {   // (2^-lo, 2^-hi): two MUFU.EX2
    float lo, hi;
    unpack2(v, lo, hi);
    return pack2(ex2_approx(-lo), ex2_approx(-hi));
}

// Per-(peak, tile) constants of the packed bodies: t' of the quad's X and Y points advance by 4 step per quad.
struct Quad2 {
    f32x2 tX, tY;     // t' at (0, 2) and (1, 3) of the current quad
    f32x2 step4;      // (4 step, 4 step)
};
__device__ __forceinline__ Quad2 quad2_begin(float t0, float step) {
    Quad2 q;
    q.tX = pack2(t0, fmaf(2.0f, step, t0));
    q.tY = pack2(t0 + step, fmaf(3.0f, step, t0));
    const float s4 = 4.0f * step;
    q.step4 = pack2(s4, s4);
    return q;
}

// Phase 1, full tile: acc2[2Q] (X points) and acc2[2Q+1] (Y points) += I [c_L L (+ c_G G)].
template <bool CORE>
__device__ __forceinline__ void fwd_tile2(float t0, float step, float cg2, float cl, f32x2 (&acc2)[kPT / 2]) {
    Quad2 q = quad2_begin(t0, step);
    const f32x2 one2 = pack2(1.0f, 1.0f), cl2 = pack2(cl, cl), cg22 = pack2(cg2, cg2);
#pragma unroll
    for (int Q = 0; Q < kPT / 4; ++Q) {
        const f32x2 uX = fma2(q.tX, q.tX, one2), uY = fma2(q.tY, q.tY, one2);
        const f32x2 rc = mul2(rcp2(mul2(uX, uY)), cl2);
        acc2[2 * Q] = fma2(rc, uY, acc2[2 * Q]);
        acc2[2 * Q + 1] = fma2(rc, uX, acc2[2 * Q + 1]);
        if (CORE) {
            acc2[2 * Q] = fma2(cg22, ex2neg2(uX), acc2[2 * Q]);
            acc2[2 * Q + 1] = fma2(cg22, ex2neg2(uY), acc2[2 * Q + 1]);
        }
        if (Q + 1 < kPT / 4) {
            q.tX = add2(q.tX, q.step4);
            q.tY = add2(q.tY, q.step4);
        }
    }
}

// Phase 2, full tile: the six sums of Acc6, each as a pair of partial sums (X points, Y points).  e t' is formed per
// quad: two more packed multiplications per quad than weights p e_p held in registers would need (sum e L^2 t' =
// t0 a5 + step sum p e L^2), but sixteen registers fewer, which measures faster (profiles/r2_dead_ends.md, "kept").
struct Acc6x2 { f32x2 a1, a2, a3t, a4t, a5, a6t; };
template <bool CORE>
__device__ __forceinline__ void bwd_tile2(float t0, float step, const f32x2 (&e2)[kPT / 2], Acc6x2& a) {
    Quad2 q = quad2_begin(t0, step);
    const f32x2 one2 = pack2(1.0f, 1.0f);
#pragma unroll
    for (int Q = 0; Q < kPT / 4; ++Q) {
        const f32x2 uX = fma2(q.tX, q.tX, one2), uY = fma2(q.tY, q.tY, one2);
        const f32x2 r = rcp2(mul2(uX, uY));
        const f32x2 LX = mul2(r, uY), LY = mul2(r, uX);
        const f32x2 L2X = mul2(LX, LX), L2Y = mul2(LY, LY);
        const f32x2 etX = mul2(e2[2 * Q], q.tX), etY = mul2(e2[2 * Q + 1], q.tY);
        a.a1 = fma2(e2[2 * Q], LX, fma2(e2[2 * Q + 1], LY, a.a1));
        a.a5 = fma2(e2[2 * Q], L2X, fma2(e2[2 * Q + 1], L2Y, a.a5));
        a.a3t = fma2(etX, L2X, fma2(etY, L2Y, a.a3t));
        if (CORE) {
            const f32x2 gX = ex2neg2(uX), gY = ex2neg2(uY);
            a.a2 = fma2(e2[2 * Q], gX, fma2(e2[2 * Q + 1], gY, a.a2));
            a.a4t = fma2(etX, gX, fma2(etY, gY, a.a4t));
            a.a6t = fma2(mul2(etX, q.tX), gX, fma2(mul2(etY, q.tY), gY, a.a6t));
        }
        if (Q + 1 < kPT / 4) {
            q.tX = add2(q.tX, q.step4);
            q.tY = add2(q.tY, q.step4);
        }
    }
}
__device__ __forceinline__ float hsum2(f32x2 v) {
    float lo, hi;
    unpack2(v, lo, hi);
    return lo + hi;
}

// ------------------------------------------------------------------------------------------------
// Phase-1 building blocks (profile).  acc[p] += I_m [ c_G 2^(-t'^2) + c_L / (1 + t'^2) ].
// Two neighbouring points share one reciprocal: 1/ua = ub * rcp(ua ub).
// The Gaussian uses u = 1 + t'^2 as well: 2^(-t'^2) = 2 * 2^(-u), the factor 2 is folded into cg2 = 2 c_G.
template <bool CORE>
__device__ __forceinline__ void fwd_pair(float ta, float tb, float cg2, float cl, float& acca, float& accb) {
    const float ua = fmaf(ta, ta, 1.0f), ub = fmaf(tb, tb, 1.0f);
    const float rc = rcp_approx(ua * ub) * cl;
    acca = fmaf(rc, ub, acca);
    accb = fmaf(rc, ua, accb);
    if (CORE) {
        acca = fmaf(cg2, ex2_approx(-ua), acca);
        accb = fmaf(cg2, ex2_approx(-ub), accb);
    }
}

// Per-(peak, tile) geometry in tile coordinates (warp-uniform): in-window points p_lo <= p <= p_hi, Gaussian
// core c_lo <= p <= c_hi.
struct PeakGeo { int p_lo, p_hi, c_lo, c_hi; };

// One quad (points 4Q .. 4Q+3) of a window-edge (peak, tile) pair in phase 1: quads outside the window are
// skipped, out-of-window points of a partial quad get a zero coefficient, the Gaussian is added if the core
// touches the quad.  One compact body per quad (these pairs are 2 of ~10 per peak; code size matters more).
template <int Q>
__device__ __forceinline__ void fwd_quad_generic(const PeakGeo& g, float t0, float step, float cg2, float cl,
                                                 f32x2& accX, f32x2& accY) {
    const int lo = max(g.p_lo, 4 * Q), hi = min(g.p_hi, 4 * Q + 3);
    if (lo > hi) return;                                   // quad outside the window
    const unsigned span = static_cast<unsigned>(hi - lo);
    float u[4], m[4], a[4];
    unpack2(accX, a[0], a[2]);
    unpack2(accY, a[1], a[3]);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float t = fmaf(static_cast<float>(4 * Q + i), step, t0);
        u[i] = fmaf(t, t, 1.0f);
        m[i] = static_cast<unsigned>(4 * Q + i - lo) <= span ? 1.0f : 0.0f;
    }
    const float r01 = rcp_approx(u[0] * u[1]) * cl, r23 = rcp_approx(u[2] * u[3]) * cl;
    a[0] = fmaf(r01 * u[1], m[0], a[0]);
    a[1] = fmaf(r01 * u[0], m[1], a[1]);
    a[2] = fmaf(r23 * u[3], m[2], a[2]);
    a[3] = fmaf(r23 * u[2], m[3], a[3]);
    if (g.c_hi >= 4 * Q && g.c_lo <= 4 * Q + 3) {
#pragma unroll
        for (int i = 0; i < 4; ++i) a[i] = fmaf(cg2 * m[i], ex2_approx(-u[i]), a[i]);
    }
    accX = pack2(a[0], a[2]);
    accY = pack2(a[1], a[3]);
}

// ------------------------------------------------------------------------------------------------
// Phase-2 building blocks.  Per (peak, tile) with t'_p = t0 + p step and e_p the residual:
//   a1 = sum e L, a5 = sum e L^2, a3t = sum e L^2 t'       (Lorentz part, every in-window point)
//   a2 = sum e g, a4t = sum e g t', a6t = sum e g t'^2     (Gaussian part, core points only; g = 2^(-u) = G/2,
//                                                           u = 1 + t'^2)
struct Acc6 { float a1, a2, a3t, a4t, a5, a6t; };

template <int Q>
__device__ __forceinline__ void bwd_quad_generic(const PeakGeo& g, float t0, float step, f32x2 eX, f32x2 eY,
                                                 Acc6& a) {
    const int lo = max(g.p_lo, 4 * Q), hi = min(g.p_hi, 4 * Q + 3);
    if (lo > hi) return;
    const unsigned span = static_cast<unsigned>(hi - lo);
    float u[4], ev[4], qv[4], tv[4];
    unpack2(eX, ev[0], ev[2]);
    unpack2(eY, ev[1], ev[3]);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float t = fmaf(static_cast<float>(4 * Q + i), step, t0);
        tv[i] = t;
        u[i] = fmaf(t, t, 1.0f);
        const bool in = static_cast<unsigned>(4 * Q + i - lo) <= span;   // out-of-window points: zero residual
        ev[i] = in ? ev[i] : 0.0f;
        qv[i] = ev[i] * t;
    }
    const float r01 = rcp_approx(u[0] * u[1]), r23 = rcp_approx(u[2] * u[3]);
    const float L[4] = {r01 * u[1], r01 * u[0], r23 * u[3], r23 * u[2]};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float L2 = L[i] * L[i];
        a.a1 = fmaf(ev[i], L[i], a.a1);
        a.a5 = fmaf(ev[i], L2, a.a5);
        a.a3t = fmaf(qv[i], L2, a.a3t);
    }
    if (g.c_hi >= 4 * Q && g.c_lo <= 4 * Q + 3) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float gg = ex2_approx(-u[i]);
            a.a2 = fmaf(ev[i], gg, a.a2);
            a.a4t = fmaf(qv[i], gg, a.a4t);
            a.a6t = fmaf(qv[i] * tv[i], gg, a.a6t);
        }
    }
}

// Fixed-tree reduction of 8 per-lane values over the 32 lanes; lane c < 8 returns the total of v[c].
// Rounds 1-3 halve the number of values each lane carries (transpose-reduce), rounds 4-5 are plain
// butterflies: 9 shuffles instead of 40.
__device__ __forceinline__ float warp_reduce8(float (&v)[8]) {
    const int lane = threadIdx.x & 31;
    float w4[4], w2[2];
    {
        const bool up = lane & 16;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float send = up ? v[i] : v[i + 4];
            const float keep = up ? v[i + 4] : v[i];
            w4[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
        }
    }
    {
        const bool up = lane & 8;
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const float send = up ? w4[i] : w4[i + 2];
            const float keep = up ? w4[i + 2] : w4[i];
            w2[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
        }
    }
    float w1;
    {
        const bool up = lane & 4;
        const float send = up ? w2[0] : w2[1];
        const float keep = up ? w2[1] : w2[0];
        w1 = keep + __shfl_xor_sync(0xffffffffu, send, 4);
    }
    w1 += __shfl_xor_sync(0xffffffffu, w1, 2);
    w1 += __shfl_xor_sync(0xffffffffu, w1, 1);
    // a lane now holds the total of value c = 4*bit4 + 2*bit3 + bit2 of its lane index; move it to lane c
    const int src = ((lane & 4) ? 16 : 0) | ((lane & 2) ? 8 : 0) | ((lane & 1) ? 4 : 0);
    return __shfl_sync(0xffffffffu, w1, src);
}


// Poisson likelihood of one grid point (A12-A16; R24): y = (y - B) + B, f = S_F + B (A3);
// returns (d ll / d f, the point's term of ll minus its f-independent part):
//   e = y/f - 1,   term = y ln(f/y) + (y - f)   (-f if y = 0).
// Kept out of line: it runs once per point and tile and would otherwise put ~1000 instructions (IEEE divisions,
// log1pf) between the two hot phases of the kernel.
__device__ __noinline__ float2 poisson_point(float ymb, float b, float s_f) {
    const float yv = ymb + b, f = s_f + b;
    const float diff = ymb - s_f;                           // y - f
    float term;
    if (yv > 0.0f) {
        const float x = -diff / yv;                         // f/y - 1
        term = yv * (log1pf(x) - x);
    } else {
        term = -f;
    }
    return make_float2(diff / f, term);
}

// Warp-uniform geometry of a window-edge (peak, tile) pair in tile coordinates.
__device__ __forceinline__ PeakGeo edge_geo(int dj, int ngc, int n_c, int plim) {
    PeakGeo g;
    g.p_lo = dj - n_c;
    g.p_hi = min(dj + n_c, plim);
    g.c_lo = dj - ngc;
    g.c_hi = dj + ngc;
    return g;
}

// a-7 (last part), as a device function: ELBO of every instance = mean log-likelihood + sum over the phases of (mean
// log prior + log Jacobian + entropy), summed in phase order; trace row and step counter of an optimisation step.
// Called by ALL threads of ONE CTA; does nothing unless an update_draw_kernel has run since the last call
// (ctl->pending).  The tile kernel of the next step calls it (its last CTA in launch order): neither the tile
// kernel nor this function needs the other's results, and the next update_draw_kernel starts after both.
__device__ __forceinline__ void finish_step(const Dev& d) {
    const unsigned int pending = d.ctl->pending;           // 0 nothing, 1 evaluation only, 2 optimisation step
    if (pending == 0u) return;                             // uniform over the CTA
    const long long step = d.ctl->step;
    for (int inst = threadIdx.x; inst < d.PR; inst += blockDim.x) {
        const double* __restrict__ ek = d.elbo_k + static_cast<size_t>(inst) * (d.K + 1);
        double llsum = 0.0;                                    // groups in order
        for (int gi = 0; gi < d.gpi; ++gi) llsum += d.ll_g[static_cast<size_t>(inst) * d.gpi + gi];
        double el = llsum * (1.0 / static_cast<double>(d.S));
        for (int kk = 0; kk < d.K; ++kk) el += ek[kk];
        d.elbo[inst] = el;
        if (pending == 2u) {
            const long long row = step - d.ctl->trace_base;
            if (row >= 0) d.trace[static_cast<size_t>(row % kTraceCap) * d.PR + inst] = el;
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        if (pending == 2u) d.ctl->step = step + 1;
        d.ctl->pending = 0u;
    }
}

// ------------------------------------------------------------------------------------------------
// Where a warp reads the static per-tile tables from: global memory (warp-uniform LDG.128 broadcasts through L1/L2),
// or the copy of the tile's lists that elbo_tile_kernel staged in shared memory with bulk asynchronous copies
// (north_star: "per-tile peak windows ... staged through shared memory/TMA"; LDS.128 broadcasts).
struct SrcGlobal {
    const PeakRec* __restrict__ pkt;
    const int4* __restrict__ runs;
    __device__ __forceinline__ PeakRec rec(int m) const { return pkt[m]; }
    __device__ __forceinline__ int4 run(int r) const { return runs[r]; }
};
struct SrcShared {   // shared-window byte addresses of record 0 / run 0 (i.e. already offset by the tile's first index)
    unsigned rec0, run0;
    __device__ __forceinline__ PeakRec rec(int m) const {
        PeakRec v;
        asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];"
                     : "=r"(v.dj), "=f"(v.delta), "=f"(v.inten), "=r"(v.full) : "r"(rec0 + 16u * static_cast<unsigned>(m)));
        return v;
    }
    __device__ __forceinline__ int4 run(int r) const {
        int4 v;
        asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];"
                     : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(run0 + 16u * static_cast<unsigned>(r)));
        return v;
    }
};

// Bulk asynchronous copy global -> shared memory completed on an mbarrier (cp.async.bulk; SASS UBLKCP).
constexpr int kStageRec = 224;   // records / run headers (incl. the one after the last run) a staged tile list may hold
constexpr int kStageRun = 64;
__device__ __forceinline__ unsigned smem_u32(const void* p) { return static_cast<unsigned>(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ void mbar_init(unsigned mbar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned mbar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned mbar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(mbar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned mbar, unsigned parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tWAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}"
        ::"r"(mbar), "r"(parity) : "memory");
}
template <bool STAGE> struct TileSrc;
template <> struct TileSrc<false> { typedef SrcGlobal type; };
template <> struct TileSrc<true> { typedef SrcShared type; };

// ------------------------------------------------------------------------------------------------
// a-3 .. a-6 (likelihood part): profile + residual + backward of one 16-point tile for one group of 32 draws.
// A warp owns one tile and one share of the tile's phase runs, in BOTH phases.  A run = the peaks of one phase
// that reach the tile; its header carries the phase, so the per-phase latents are loaded once per run (prefetched
// one run ahead) and the run index is the output slot of phase 2.
struct TileCtx {
    int g;              // group (32 draws) of this warp
    int i0, plim;       // first grid index of the tile, last valid point of the tile (< 0: no point)
    int pat;            // observed pattern of the group
    const float4* lat;  // latent records of the group, already offset by the lane
    const int* ngk;     // Gaussian-core half-widths of the group
};

__device__ __forceinline__ TileCtx tile_ctx(const Dev& d, int g, int tile) {
    TileCtx c;
    c.g = g;
    c.i0 = tile * kPT;
    c.plim = min(kPT - 1, d.N - 1 - c.i0);
    c.pat = (g / d.gpi) / d.R;
    c.lat = d.lat + static_cast<size_t>(g) * d.K * 32 + (threadIdx.x & 31);
    c.ngk = d.ng + static_cast<size_t>(g) * d.K;
    return c;
}

// Phase 1: acc[p] = profile of the runs [rng.x, rng.y) on the 16 points of the tile (acc is overwritten).  The
// accumulators live as packed pairs (quad Q: acc2[2Q] = points (4Q, 4Q+2), acc2[2Q+1] = points (4Q+1, 4Q+3)).
template <class Src>
__device__ __forceinline__ void tile_phase1(const Dev& d, const Src& src, const TileCtx& c, int2 rng, float (&acc)[kPT]) {
    f32x2 acc2[kPT / 2];
#pragma unroll
    for (int i = 0; i < kPT / 2; ++i) acc2[i] = 0ull;
    if (rng.x < rng.y) {
        int4 run_n = src.run(rng.x);
        float4 lt_n = c.lat[static_cast<size_t>(run_n.z) * 32];
        int ng_n = c.ngk[run_n.z];
        for (int r = rng.x; r < rng.y; ++r) {
            const int4 run = run_n;
            const float4 lt = lt_n;
            const int ngc = ng_n;
            run_n = src.run(r + 1);                         // run_tab carries one padding entry
            lt_n = c.lat[static_cast<size_t>(run_n.z) * 32];
            ng_n = c.ngk[run_n.z];
            const float step = d.delta * lt.x;
            const unsigned core_span = static_cast<unsigned>(kPT - 1 + 2 * ngc);
#pragma unroll 1
            for (int m = run.x; m < run.y; ++m) {
                const PeakRec pk = src.rec(m);
                const float t0 = fmaf(static_cast<float>(-pk.dj), step, fmaf(-pk.delta, lt.x, lt.y));
                const float cl = pk.inten * lt.w;
                const bool core = static_cast<unsigned>(pk.dj + ngc) <= core_span;   // Gaussian core touches the tile
                if (pk.full & 1) {   // branch-free bodies: Lorentz tail only, or tail + Gaussian on all 16 points
                    if (!core) {
                        fwd_tile2<false>(t0, step, 0.0f, cl, acc2);
                    } else {
                        fwd_tile2<true>(t0, step, 2.0f * pk.inten * lt.z, cl, acc2);
                    }
                } else {         // window edge: quad by quad
                    const PeakGeo geo = edge_geo(pk.dj, ngc, pk.full >> 1, c.plim);
                    const float cg2 = 2.0f * pk.inten * lt.z;
                    fwd_quad_generic<0>(geo, t0, step, cg2, cl, acc2[0], acc2[1]);
                    fwd_quad_generic<1>(geo, t0, step, cg2, cl, acc2[2], acc2[3]);
                    fwd_quad_generic<2>(geo, t0, step, cg2, cl, acc2[4], acc2[5]);
                    fwd_quad_generic<3>(geo, t0, step, cg2, cl, acc2[6], acc2[7]);
                }
            }
        }
    }
#pragma unroll
    for (int Q = 0; Q < kPT / 4; ++Q) {
        unpack2(acc2[2 * Q], acc[4 * Q], acc[4 * Q + 2]);
        unpack2(acc2[2 * Q + 1], acc[4 * Q + 1], acc[4 * Q + 3]);
    }
}

// a-4: residual e = d ll / d f (0 beyond the grid) from the complete profile acc (without B); returns the
// tile's part of ll:
//   Gaussian (R3):  e = (y - f)/sigma_n^2,  part = sum ((y - f)/sigma_n)^2            (ll = -1/2 sum + const)
//   Poisson (A16):  e = y/f - 1,            part = sum y ln(f/y) + (y - f)  (-f if y = 0)   (ll = sum + const)
__device__ __forceinline__ float tile_residual(const Dev& d, const TileCtx& c, const float (&acc)[kPT], float (&ev)[kPT]) {
    const PatConst pc = d.pat[c.pat];
    const float* __restrict__ yb = d.yb + static_cast<size_t>(c.pat) * d.N;
    float ss = 0.0f;
    if (d.likelihood == 0) {
#pragma unroll
        for (int p = 0; p < kPT; ++p) {
            float r = 0.0f;
            if (p <= c.plim) r = yb[c.i0 + p] - acc[p];
            const float z = r * pc.inv_sn;
            ss = fmaf(z, z, ss);
            ev[p] = r * pc.inv_sn2;
        }
    } else {
        const float* __restrict__ bgp = d.bg + static_cast<size_t>(c.pat) * d.N;
#pragma unroll
        for (int p = 0; p < kPT; ++p) {
            ev[p] = 0.0f;
            if (p <= c.plim) {
                const float2 ed = poisson_point(yb[c.i0 + p], bgp[c.i0 + p], acc[p]);
                ev[p] = ed.x;
                ss += ed.y;
            }
        }
    }
    return ss;
}

// a-4 on one quad (points 4 Q .. 4 Q + 3) of the tile: the PS = 4 warps of a CTA take one quad each.
__device__ __forceinline__ float quad_residual(const Dev& d, const TileCtx& c, int Q, const float4 acc, float4& ev) {
    const PatConst pc = d.pat[c.pat];
    const float* __restrict__ yb = d.yb + static_cast<size_t>(c.pat) * d.N + c.i0 + 4 * Q;
    const float a[4] = {acc.x, acc.y, acc.z, acc.w};
    float e[4];
    float ss = 0.0f;
    if (d.likelihood == 0) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            float r = 0.0f;
            if (4 * Q + i <= c.plim) r = yb[i] - a[i];
            const float z = r * pc.inv_sn;
            ss = fmaf(z, z, ss);
            e[i] = r * pc.inv_sn2;
        }
    } else {
        const float* __restrict__ bgp = d.bg + static_cast<size_t>(c.pat) * d.N + c.i0 + 4 * Q;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            e[i] = 0.0f;
            if (4 * Q + i <= c.plim) {
                const float2 ed = poisson_point(yb[i], bgp[i], a[i]);
                e[i] = ed.x;
                ss += ed.y;
            }
        }
    }
    ev = make_float4(e[0], e[1], e[2], e[3]);
    return ss;
}

// debug read-back of the profile f = S_F + B of the first n_dbg sample-instances (parity tests)
__device__ __forceinline__ void tile_debug_profile(const Dev& d, const TileCtx& c, const float (&acc)[kPT],
                                                   float* __restrict__ f_dbg, long long n_dbg) {
    const int inst = c.g / d.gpi;
    const int s = (c.g - inst * d.gpi) * 32 + (threadIdx.x & 31);
    const long long t = static_cast<long long>(inst) * d.S + s - d.dbg_first;   // row of the read-back buffer
    if (s < d.S && t >= 0 && t < n_dbg) {
        const float* __restrict__ bg = d.bg + static_cast<size_t>(c.pat) * d.N;
#pragma unroll
        for (int p = 0; p < kPT; ++p)
            if (p <= c.plim) f_dbg[t * d.N + c.i0 + p] = acc[p] + bg[c.i0 + p];
    }
}

// Phase 2: six sums per phase run [rng.x, rng.y) over the tile from the residual e, chain rule, reduction over the
// 32 draws (or, in the gradient service, per-draw output to row pd_row of d.pd).
template <class Src>
__device__ __forceinline__ void tile_phase2(const Dev& d, const Src& src, const TileCtx& c, int2 rng, const float (&e)[kPT],
                                            int pd_row) {
    if (rng.x >= rng.y) return;
    const int lane = threadIdx.x & 31;
    f32x2 e2[kPT / 2];                   // packed like the accumulators of phase 1
#pragma unroll
    for (int Q = 0; Q < kPT / 4; ++Q) {
        e2[2 * Q] = pack2(e[4 * Q], e[4 * Q + 2]);
        e2[2 * Q + 1] = pack2(e[4 * Q + 1], e[4 * Q + 3]);
    }
    const float4* __restrict__ epsg = d.eps + static_cast<size_t>(c.g) * d.K * 32 + lane;
    const float* __restrict__ rrg = d.rr + static_cast<size_t>(c.g) * d.K * 32 + lane;
    float* __restrict__ part = d.part8 + static_cast<size_t>(c.g) * d.n_slots * 8;

    int4 run_n = src.run(rng.x);
    float4 lt_n = c.lat[static_cast<size_t>(run_n.z) * 32];
    int ng_n = c.ngk[run_n.z];
    for (int r = rng.x; r < rng.y; ++r) {
        const int4 run = run_n;
        const float4 lt = lt_n;
        const int ngc = ng_n;
        run_n = src.run(r + 1);
        lt_n = c.lat[static_cast<size_t>(run_n.z) * 32];
        ng_n = c.ngk[run_n.z];
        // loads of the flush, issued early
        const float4 ep = epsg[static_cast<size_t>(run.z) * 32];
        const float rmix = rrg[static_cast<size_t>(run.z) * 32];
        const float step = d.delta * lt.x;
        const unsigned core_span = static_cast<unsigned>(kPT - 1 + 2 * ngc);
        // sums over the peaks of the run, I_m folded in:
        //   B1 = sum I e L, B3 = sum I e L^2 t', B5 = sum I e L^2; B2 = sum I e G, B4 = sum I e G t', B6 = sum I e G t'^2
        float B1 = 0.f, B2 = 0.f, B3 = 0.f, B4 = 0.f, B5 = 0.f, B6 = 0.f;
#pragma unroll 1
        for (int m = run.x; m < run.y; ++m) {
            const PeakRec pk = src.rec(m);
            const float t0 = fmaf(static_cast<float>(-pk.dj), step, fmaf(-pk.delta, lt.x, lt.y));
            const bool core = static_cast<unsigned>(pk.dj + ngc) <= core_span;
            if ((pk.full & 1) && !core) {
                Acc6x2 a2 = {0ull, 0ull, 0ull, 0ull, 0ull, 0ull};
                bwd_tile2<false>(t0, step, e2, a2);
                const float a1 = hsum2(a2.a1), a5 = hsum2(a2.a5);
                B3 = fmaf(pk.inten, hsum2(a2.a3t), B3);
                B1 = fmaf(pk.inten, a1, B1);
                B5 = fmaf(pk.inten, a5, B5);
            } else {
                Acc6 a = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
                if (pk.full & 1) {
                    Acc6x2 a2 = {0ull, 0ull, 0ull, 0ull, 0ull, 0ull};
                    bwd_tile2<true>(t0, step, e2, a2);
                    a.a1 = hsum2(a2.a1); a.a2 = hsum2(a2.a2); a.a3t = hsum2(a2.a3t);
                    a.a4t = hsum2(a2.a4t); a.a5 = hsum2(a2.a5); a.a6t = hsum2(a2.a6t);
                } else {
                    const PeakGeo geo = edge_geo(pk.dj, ngc, pk.full >> 1, c.plim);
                    bwd_quad_generic<0>(geo, t0, step, e2[0], e2[1], a);
                    bwd_quad_generic<1>(geo, t0, step, e2[2], e2[3], a);
                    bwd_quad_generic<2>(geo, t0, step, e2[4], e2[5], a);
                    bwd_quad_generic<3>(geo, t0, step, e2[6], e2[7], a);
                }
                const float i2 = 2.0f * pk.inten;           // g = G/2 in the Gaussian sums
                B1 = fmaf(pk.inten, a.a1, B1);
                B2 = fmaf(i2, a.a2, B2);
                B5 = fmaf(pk.inten, a.a5, B5);
                B3 = fmaf(pk.inten, a.a3t, B3);
                B4 = fmaf(i2, a.a4t, B4);
                B6 = fmaf(i2, a.a6t, B6);
            }
        }
        // chain rule for the likelihood part (per draw), then sum over the 32 draws of the group
        const float cG = lt.z, cL = lt.w;
        float v[8];
        v[0] = fmaf(cL, B1, cG * B2);
        v[1] = lt.x * (2.0f * cL * B3 + (2.0f * kLn2) * cG * B4);
        v[2] = -(cL * (2.0f * B5 - B1) + cG * (B2 - (2.0f * kLn2) * B6));
        v[3] = (1.0f - rmix) * cL * B1 - rmix * cG * B2;
        if (d.pd) {   // gradient service: keep the draws apart
            float* __restrict__ o = d.pd + (static_cast<size_t>(pd_row) * d.n_slots + run.w) * 128 + lane;
            o[0] = v[0]; o[32] = v[1]; o[64] = v[2]; o[96] = v[3];
            continue;
        }
        v[4] = v[0] * ep.x; v[5] = v[1] * ep.y; v[6] = v[2] * ep.z; v[7] = v[3] * ep.w;
        const float tot = warp_reduce8(v);
        if (lane < 8) part[static_cast<size_t>(run.w) * 8 + lane] = tot;
    }
}

// ------------------------------------------------------------------------------------------------
// Peak asymmetry and sec width term (reading R30; A9/A10 PAPER.md:234-239, prior PAPER.md:274,
// the sec of).  t'' = t' / A, A = alpha for t' >= 0 (x >= rho), 1 below; heights unchanged.  With
// ia = 1 / alpha and mx = max(t', 0):   t'' = t' + mx (ia - 1),   d t''/d mu = -(2/w) (1 on the low, ia on the high side)
// so that  sum e L^2 t'' (d t''/d mu factor) = sum e L^2 [t' + mx (ia^2 - 1)],  and  d t''/d alpha = -t''/alpha on the high
// side only:  alpha d f/d alpha = I [2 c_L t''^2 L^2 + 2 ln2 c_G t''^2 G]_high,  t''_high = mx ia.
// The sec term multiplies the width of the record's peak by sec(p_m / 2): t', the step and both heights get the factor
// inv_s = cos(p_m / 2), the mu chain one more.
// Records whose 16 points are in-window and outside the Gaussian core lie wholly on ONE side of the peak for all 32
// draws (the core half-width covers the largest sampled shift), so they keep the packed bodies with (t0, step) scaled
// by ia on the high side; core and window-edge records take the scalar per-point bodies below.
template <int Q>
__device__ __forceinline__ void fwd_quad_asym(const PeakGeo& g, const float (&o)[kPT], float t0, float sx, float iam1,
                                              float cg2, float cl, f32x2& accX, f32x2& accY) {
    const int lo = max(g.p_lo, 4 * Q), hi = min(g.p_hi, 4 * Q + 3);
    if (lo > hi) return;                                   // quad outside the window
    const unsigned span = static_cast<unsigned>(hi - lo);
    float u[4], m[4], a[4];
    unpack2(accX, a[0], a[2]);
    unpack2(accY, a[1], a[3]);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        float t = fmaf(o[4 * Q + i], sx, t0);              // o_p = x_{i0+p} - x_{i0} (p Delta on a uniform grid), sx = 2 / w_m
        t = fmaf(fmaxf(t, 0.0f), iam1, t);                 // high-angle side: t' / alpha
        u[i] = fmaf(t, t, 1.0f);
        m[i] = static_cast<unsigned>(4 * Q + i - lo) <= span ? 1.0f : 0.0f;
    }
    const float r01 = rcp_approx(u[0] * u[1]) * cl, r23 = rcp_approx(u[2] * u[3]) * cl;
    a[0] = fmaf(r01 * u[1], m[0], a[0]);
    a[1] = fmaf(r01 * u[0], m[1], a[1]);
    a[2] = fmaf(r23 * u[3], m[2], a[2]);
    a[3] = fmaf(r23 * u[2], m[3], a[3]);
    if (g.c_hi >= 4 * Q && g.c_lo <= 4 * Q + 3) {
#pragma unroll
        for (int i = 0; i < 4; ++i) a[i] = fmaf(cg2 * m[i], ex2_approx(-u[i]), a[i]);
    }
    accX = pack2(a[0], a[2]);
    accY = pack2(a[1], a[3]);
}

// a1 = sum e L, a5 = sum e L^2, a2 = sum e g as in Acc6, a6u = sum e u g (g = 2^-u = G/2, u = 1 + t''^2);
// a3m = sum e L^2 tm, a4m = sum e g tm with tm = t' + mx (ia^2 - 1) (the mu chain); h1 = sum e mx^2 L^2, h2 = sum e mx^2 g.
struct Acc8 { float a1, a2, a5, a6u, a3m, a4m, h1, h2; };

template <int Q>
__device__ __forceinline__ void bwd_quad_asym(const PeakGeo& g, const float (&o)[kPT], float t0, float sx, float iam1,
                                              float ia2m1, f32x2 eX, f32x2 eY, Acc8& a) {
    const int lo = max(g.p_lo, 4 * Q), hi = min(g.p_hi, 4 * Q + 3);
    if (lo > hi) return;
    const unsigned span = static_cast<unsigned>(hi - lo);
    float u[4], ev[4], tm[4], em[4];
    unpack2(eX, ev[0], ev[2]);
    unpack2(eY, ev[1], ev[3]);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float tp = fmaf(o[4 * Q + i], sx, t0);
        const float mx = fmaxf(tp, 0.0f);
        const float t = fmaf(mx, iam1, tp);
        tm[i] = fmaf(mx, ia2m1, tp);
        u[i] = fmaf(t, t, 1.0f);
        const bool in = static_cast<unsigned>(4 * Q + i - lo) <= span;   // out-of-window points: zero residual
        ev[i] = in ? ev[i] : 0.0f;
        em[i] = ev[i] * mx * mx;
    }
    const float r01 = rcp_approx(u[0] * u[1]), r23 = rcp_approx(u[2] * u[3]);
    const float L[4] = {r01 * u[1], r01 * u[0], r23 * u[3], r23 * u[2]};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float L2 = L[i] * L[i];
        a.a1 = fmaf(ev[i], L[i], a.a1);
        a.a5 = fmaf(ev[i], L2, a.a5);
        a.a3m = fmaf(ev[i] * tm[i], L2, a.a3m);
        a.h1 = fmaf(em[i], L2, a.h1);
    }
    if (g.c_hi >= 4 * Q && g.c_lo <= 4 * Q + 3) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float gg = ex2_approx(-u[i]);
            a.a2 = fmaf(ev[i], gg, a.a2);
            a.a6u = fmaf(ev[i] * u[i], gg, a.a6u);
            a.a4m = fmaf(ev[i] * tm[i], gg, a.a4m);
            a.h2 = fmaf(em[i], gg, a.h2);
        }
    }
}

// Offsets of the tile's 16 points from its first one: p Delta on a uniform grid, the table of R31 otherwise.
__device__ __forceinline__ void tile_offsets(const Dev& d, const TileCtx& c, float (&o)[kPT]) {
    if (d.general) {
        const float4* __restrict__ t = reinterpret_cast<const float4*>(d.tile_off + static_cast<size_t>(c.i0));   // i0 = 16 tile
#pragma unroll
        for (int v = 0; v < kPT / 4; ++v) {
            const float4 q = t[v];
            o[4 * v] = q.x; o[4 * v + 1] = q.y; o[4 * v + 2] = q.z; o[4 * v + 3] = q.w;
        }
    } else {
#pragma unroll
        for (int p = 0; p < kPT; ++p) o[p] = static_cast<float>(p) * d.delta;
    }
}

// Phase 1 with the asymmetry / sec term (R30).  ia_g: 1 / alpha of the group's draws, already offset by the lane.
template <class Src>
__device__ __forceinline__ void tile_phase1_asym(const Dev& d, const Src& src, const TileCtx& c, int2 rng, float (&acc)[kPT]) {
    f32x2 acc2[kPT / 2];
#pragma unroll
    for (int i = 0; i < kPT / 2; ++i) acc2[i] = 0ull;
    const float* __restrict__ iag = d.ia + static_cast<size_t>(c.g) * d.K * 32 + (threadIdx.x & 31);
    float o[kPT];                                           // point offsets of the tile from its first point
    tile_offsets(d, c, o);
    for (int r = rng.x; r < rng.y; ++r) {
        const int4 run = src.run(r);
        const float4 lt = c.lat[static_cast<size_t>(run.z) * 32];
        const int ngc = c.ngk[run.z];
        const float ia = d.asym ? iag[static_cast<size_t>(run.z) * 32] : 1.0f;
        const float iam1 = ia - 1.0f;
        const float step_k = d.delta * lt.x;
        const unsigned core_span = static_cast<unsigned>(kPT - 1 + 2 * ngc);
#pragma unroll 1
        for (int m = run.x; m < run.y; ++m) {
            const PeakRec pk = src.rec(m);
            const float inv_s = d.sec ? d.pk_sec[m] : 1.0f;
            float step = step_k * inv_s;
            // t' at the first point of the tile: grid-index form on a uniform grid, x_{i0} - p_m from the table otherwise
            float t0 = (d.general ? fmaf(d.pk_base[m], lt.x, lt.y)
                                  : fmaf(static_cast<float>(-pk.dj), step_k, fmaf(-pk.delta, lt.x, lt.y))) * inv_s;
            const float cl = pk.inten * lt.w * inv_s;
            const bool core = static_cast<unsigned>(pk.dj + ngc) <= core_span;
            if ((pk.full & 1) && !core && !d.general) {     // one side of the peak for every draw: packed body
                if (pk.dj < 0) { t0 *= ia; step *= ia; }    // the tile lies above the peak: high-angle side
                fwd_tile2<false>(t0, step, 0.0f, cl, acc2);
            } else {
                const PeakGeo geo = edge_geo(pk.dj, ngc, pk.full >> 1, c.plim);
                const float cg2 = 2.0f * pk.inten * lt.z * inv_s;
                const float sx = lt.x * inv_s;
                fwd_quad_asym<0>(geo, o, t0, sx, iam1, cg2, cl, acc2[0], acc2[1]);
                fwd_quad_asym<1>(geo, o, t0, sx, iam1, cg2, cl, acc2[2], acc2[3]);
                fwd_quad_asym<2>(geo, o, t0, sx, iam1, cg2, cl, acc2[4], acc2[5]);
                fwd_quad_asym<3>(geo, o, t0, sx, iam1, cg2, cl, acc2[6], acc2[7]);
            }
        }
    }
#pragma unroll
    for (int Q = 0; Q < kPT / 4; ++Q) {
        unpack2(acc2[2 * Q], acc[4 * Q], acc[4 * Q + 2]);
        unpack2(acc2[2 * Q + 1], acc[4 * Q + 1], acc[4 * Q + 3]);
    }
}

// Phase 2 with the asymmetry / sec term: ten values per run, (g_h, g_mu, g_w, g_r, g (x) eps) into part8 and
// (g_alpha, g_alpha eps_alpha) into parta; per-draw mode: five classes per run.
template <class Src>
__device__ __forceinline__ void tile_phase2_asym(const Dev& d, const Src& src, const TileCtx& c, int2 rng, const float (&e)[kPT],
                                                 int pd_row) {
    if (rng.x >= rng.y) return;
    const int lane = threadIdx.x & 31;
    f32x2 e2[kPT / 2];
#pragma unroll
    for (int Q = 0; Q < kPT / 4; ++Q) {
        e2[2 * Q] = pack2(e[4 * Q], e[4 * Q + 2]);
        e2[2 * Q + 1] = pack2(e[4 * Q + 1], e[4 * Q + 3]);
    }
    const size_t gk = static_cast<size_t>(c.g) * d.K * 32 + lane;
    float off[kPT];
    tile_offsets(d, c, off);
    for (int r = rng.x; r < rng.y; ++r) {
        const int4 run = src.run(r);
        const size_t o = gk + static_cast<size_t>(run.z) * 32;
        const float4 lt = c.lat[static_cast<size_t>(run.z) * 32];
        const int ngc = c.ngk[run.z];
        const float4 ep = d.eps[o];
        const float rmix = d.rr[o];
        const float ia = d.asym ? d.ia[o] : 1.0f;
        const float ep_a = d.asym ? d.eps_a[o] : 0.0f;
        const float iam1 = ia - 1.0f, ia2 = ia * ia, ia2m1 = ia2 - 1.0f;
        const float step_k = d.delta * lt.x;
        const unsigned core_span = static_cast<unsigned>(kPT - 1 + 2 * ngc);
        // per run, I_m / s_m folded in: B1 = sum e L, B5 = sum e L^2, B2 = sum e G, B6 = sum e G t''^2,
        // B3 = sum e L^2 t'' (mu-chain factor), B4 = sum e G t'' (same), H1 = sum_high e L^2 t''^2, H2 = sum_high e G t''^2
        float B1 = 0.f, B2 = 0.f, B3 = 0.f, B4 = 0.f, B5 = 0.f, B6 = 0.f, H1 = 0.f, H2 = 0.f;
#pragma unroll 1
        for (int m = run.x; m < run.y; ++m) {
            const PeakRec pk = src.rec(m);
            const float inv_s = d.sec ? d.pk_sec[m] : 1.0f;
            float step = step_k * inv_s;
            float t0 = (d.general ? fmaf(d.pk_base[m], lt.x, lt.y)
                                  : fmaf(static_cast<float>(-pk.dj), step_k, fmaf(-pk.delta, lt.x, lt.y))) * inv_s;
            const float wI = pk.inten * inv_s;              // height factor of the record
            const bool core = static_cast<unsigned>(pk.dj + ngc) <= core_span;
            if ((pk.full & 1) && !core && !d.general) {
                const bool high = pk.dj < 0;
                if (high) { t0 *= ia; step *= ia; }
                Acc6x2 a2 = {0ull, 0ull, 0ull, 0ull, 0ull, 0ull};
                bwd_tile2<false>(t0, step, e2, a2);
                const float a1 = hsum2(a2.a1), a5 = hsum2(a2.a5), m3 = hsum2(a2.a3t);   // m3 = sum e L^2 t''
                B1 = fmaf(wI, a1, B1);
                B5 = fmaf(wI, a5, B5);
                B3 = fmaf(wI * inv_s * (high ? ia : 1.0f), m3, B3);
                if (high) H1 = fmaf(wI, a1 - a5, H1);       // t''^2 L^2 = L - L^2
            } else {
                const PeakGeo geo = edge_geo(pk.dj, ngc, pk.full >> 1, c.plim);
                Acc8 a = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
                const float sx = lt.x * inv_s;
                bwd_quad_asym<0>(geo, off, t0, sx, iam1, ia2m1, e2[0], e2[1], a);
                bwd_quad_asym<1>(geo, off, t0, sx, iam1, ia2m1, e2[2], e2[3], a);
                bwd_quad_asym<2>(geo, off, t0, sx, iam1, ia2m1, e2[4], e2[5], a);
                bwd_quad_asym<3>(geo, off, t0, sx, iam1, ia2m1, e2[6], e2[7], a);
                const float i2 = 2.0f * wI;                 // g = G/2 in the Gaussian sums
                B1 = fmaf(wI, a.a1, B1);
                B2 = fmaf(i2, a.a2, B2);
                B5 = fmaf(wI, a.a5, B5);
                B6 = fmaf(i2, a.a6u - a.a2, B6);
                B3 = fmaf(wI * inv_s, a.a3m, B3);
                B4 = fmaf(i2 * inv_s, a.a4m, B4);
                H1 = fmaf(wI * ia2, a.h1, H1);
                H2 = fmaf(i2 * ia2, a.h2, H2);
            }
        }
        const float cG = lt.z, cL = lt.w;
        float v[8];
        v[0] = fmaf(cL, B1, cG * B2);
        v[1] = lt.x * (2.0f * cL * B3 + (2.0f * kLn2) * cG * B4);
        v[2] = -(cL * (2.0f * B5 - B1) + cG * (B2 - (2.0f * kLn2) * B6));
        v[3] = (1.0f - rmix) * cL * B1 - rmix * cG * B2;
        const float va = d.asym ? 2.0f * cL * H1 + (2.0f * kLn2) * cG * H2 : 0.0f;   // alpha d ll / d alpha
        if (d.pd) {   // gradient service: keep the draws apart, five classes per run
            float* __restrict__ o5 = d.pd + (static_cast<size_t>(pd_row) * d.n_slots + run.w) * 160 + lane;
            o5[0] = v[0]; o5[32] = v[1]; o5[64] = v[2]; o5[96] = v[3]; o5[128] = va;
            continue;
        }
        v[4] = v[0] * ep.x; v[5] = v[1] * ep.y; v[6] = v[2] * ep.z; v[7] = v[3] * ep.w;
        const float tot = warp_reduce8(v);
        float* __restrict__ part = d.part8 + static_cast<size_t>(c.g) * d.n_slots * 8;
        if (lane < 8) part[static_cast<size_t>(run.w) * 8 + lane] = tot;
        float s0 = va, s1 = va * ep_a;
#pragma unroll
        for (int of = 16; of > 0; of >>= 1) {               // fixed butterfly: every lane ends with the totals
            s0 += __shfl_xor_sync(0xffffffffu, s0, of);
            s1 += __shfl_xor_sync(0xffffffffu, s1, of);
        }
        if (lane == 0)
            *reinterpret_cast<float2*>(d.parta + (static_cast<size_t>(c.g) * d.n_slots + run.w) * 2) = make_float2(s0, s1);
    }
}

// Fused variant: grid (G, n_seg), block 32*TW*PS; segment = TW consecutive tiles.  Warp w owns tile (w % TW) of the
// segment and share (w / TW) of that tile's runs; the PS partial profiles meet in shared memory.  Used when the
// launch has enough tile-warps without splitting (PS = 1: no barrier is ever waited on) and for forward-only runs.
#ifndef XRDVI_TILE_WARPS_PER_SM
#define XRDVI_TILE_WARPS_PER_SM 24          // register budget: 65536 / (32 * 24) = 85 -> 80 registers per thread
#endif
#ifndef XRDVI_TILE_WARPS_PER_SM_SHARED
#define XRDVI_TILE_WARPS_PER_SM_SHARED 20   // CTAs with several warps (few-group launches): 96 registers, no spills
#endif
// Resident CTAs per SM the register budget is set for.  Launches with millions of one-warp CTAs (PS = 1) are
// throughput-bound and want 24 warps per SM; the few-group launches (config 1: 2008 CTAs of 4 warps) are bound by the
// latency of each warp's own instruction stream, where 96 registers without spills beat 80 with (measured 0.169 vs
// 0.180 ms, profiles/).
constexpr int tile_ctas_per_sm(int TW, int PS) {
    const int warps = TW * PS;
    const int budget = warps > 1 ? XRDVI_TILE_WARPS_PER_SM_SHARED : XRDVI_TILE_WARPS_PER_SM;
    return budget / warps > 0 ? budget / warps : 1;
}
// STAGE (TW = 1): thread 0 copies the tile's record list and run headers into shared memory with two bulk asynchronous
// copies completed on an mbarrier (north_star: "per-tile peak windows ... staged through shared memory/TMA"); the
// tables are static, so the copies are issued BEFORE griddepcontrol.wait and overlap the predecessor kernel's drain.
// All PS shares of the CTA then read records and run headers with LDS.128 broadcasts in both phases.
// MODEL 0: the base profile (A3-A8); MODEL 1: with the peak asymmetry / sec width term of R30 (tile_phase*_asym).
template <int TW, int PS, bool BWD, bool STAGE, int MODEL>
__global__ void __launch_bounds__(32 * TW * PS, tile_ctas_per_sm(TW, PS))
elbo_tile_kernel(const Dev d, float* __restrict__ f_dbg, long long n_dbg) {
    static_assert(!STAGE || TW == 1, "staging holds one tile list per CTA");
    __shared__ float4 e_s[TW][kPT / 4][32];
    constexpr bool kQuadShare = (PS == 4 && TW == 1);       // residual formed by four warps, one quad each
    __shared__ float ss_s[kQuadShare ? 4 : TW][32];
    __shared__ __align__(16) float acc_s[PS > 1 ? (kQuadShare ? PS : PS - 1) * TW * kPT : 1][32];
    __shared__ __align__(128) PeakRec rec_s[STAGE ? kStageRec : 1];
    __shared__ __align__(16) int4 run_s[STAGE ? kStageRun : 1];
    __shared__ __align__(8) unsigned long long mbar_s;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int tw = w % TW, ps = w / TW;
    // grid (G, n_seg), dispatched blockIdx.x fastest.  The dispatch order is cut into chunks of g_block draw groups; inside a
    // chunk the CTAs run TILE-major (all groups of the chunk on the heaviest tile first, the lightest tiles last), so the
    // latent records of a chunk (g_block x K x 1.2 KB, sized to stay in L2) are read from DRAM once, not once per tile:
    // with every group in one chunk, config 2 streamed all 241 MB of latents through DRAM for each of its 251 tiles
    // (79 GB per launch, ncu; profiles/r2_*).  Config 1 (8 groups) is one chunk.
    const unsigned lin = blockIdx.y * gridDim.x + blockIdx.x;
    const unsigned per_chunk = static_cast<unsigned>(d.g_block) * gridDim.y;
    const unsigned chunk = lin / per_chunk, rem = lin - chunk * per_chunk;
    const unsigned gb = (chunk + 1) * d.g_block <= gridDim.x ? d.g_block : gridDim.x - chunk * d.g_block;
    const unsigned seg_pos = rem / gb;
    const int group = static_cast<int>(chunk * d.g_block + (rem - seg_pos * gb));
    const int seg = d.seg_order[seg_pos];                   // static tables: may be read before the predecessor is done
    const int tile = seg * TW + tw;
    const bool live = tile < d.n_tile;                      // the last segment may have fewer than TW tiles
    typename TileSrc<STAGE>::type src;
    if constexpr (STAGE) {
        const int2 t0 = d.tile_rng[tile], t1 = d.tile_rng[tile + 1];
        const unsigned mb = smem_u32(&mbar_s);
        if (threadIdx.x == 0) {
            mbar_init(mb, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            const unsigned rb = 16u * static_cast<unsigned>(t1.y - t0.y), hb = 16u * static_cast<unsigned>(t1.x - t0.x + 1);
            mbar_expect_tx(mb, rb + hb);
            if (rb) bulk_g2s(smem_u32(&rec_s[0]), d.pk_tile + t0.y, rb, mb);
            bulk_g2s(smem_u32(&run_s[0]), d.run_tab + t0.x, hb, mb);      // + the header after the last run
        }
        src.rec0 = smem_u32(&rec_s[0]) - 16u * static_cast<unsigned>(t0.y);
        src.run0 = smem_u32(&run_s[0]) - 16u * static_cast<unsigned>(t0.x);
    } else {
        src = SrcGlobal{d.pk_tile, d.run_tab};
    }
    const TileCtx c = tile_ctx(d, d.g_base + group, tile);
    int2 rng = make_int2(0, 0);
    if (live) rng = d.share_rng[tile * PS + ps];
    if constexpr (STAGE) {
        if (PS > 1) __syncthreads();                        // the mbarrier is initialised before anybody polls it
        mbar_wait(smem_u32(&mbar_s), 0u);
    }
    griddep_wait();                                         // latents, control block: written by the predecessor
    // Only now may the successor (update_draw_kernel) begin: whatever it reads BEFORE its own griddep_wait was written
    // by the update_draw_kernel before this launch, which has completed once any CTA here is past the wait.
    griddep_launch_dependents();
    if (blockIdx.x == gridDim.x - 1 && blockIdx.y == gridDim.y - 1) finish_step(d);   // previous step's ELBO / count
    const unsigned tl_row = lin * (TW * PS) + w;
    tl_stamp(d.tl, tl_row, 0);
    if (d.tl) tl_tag(d.tl, tl_row, rng.x < rng.y ? d.run_tab[rng.y - 1].y - d.run_tab[rng.x].x : 0);

    float acc[kPT];
#pragma unroll
    for (int p = 0; p < kPT; ++p) acc[p] = 0.0f;
    if constexpr (MODEL == 1) tile_phase1_asym(d, src, c, rng, acc);
    else tile_phase1(d, src, c, rng, acc);

    if constexpr (kQuadShare) {
        // every share leaves its partial profile in shared memory as one float4 per quad; warp q then sums quad q over the
        // shares in share order, forms its residual and its part of ll: a quarter of the serial section per warp
        float4* __restrict__ aq = reinterpret_cast<float4*>(&acc_s[0][0]);     // [share][quad][lane]
#pragma unroll
        for (int v = 0; v < kPT / 4; ++v)
            aq[(ps * 4 + v) * 32 + lane] = make_float4(acc[4 * v], acc[4 * v + 1], acc[4 * v + 2], acc[4 * v + 3]);
        __syncthreads();
        float4 a = aq[ps * 32 + lane];
#pragma unroll
        for (int q = 1; q < PS; ++q) {
            const float4 b = aq[(q * 4 + ps) * 32 + lane];
            a.x += b.x; a.y += b.y; a.z += b.z; a.w += b.w;
        }
        float4 ev;
        const float ss = quad_residual(d, c, ps, a, ev);
        if (BWD) e_s[0][ps][lane] = ev;
        ss_s[ps][lane] = ss;
        if (f_dbg) {
            const int inst = c.g / d.gpi;
            const int sd = (c.g - inst * d.gpi) * 32 + lane;
            const long long t = static_cast<long long>(inst) * d.S + sd - d.dbg_first;
            if (sd < d.S && t >= 0 && t < n_dbg) {
                const float* __restrict__ bg = d.bg + static_cast<size_t>(c.pat) * d.N + c.i0 + 4 * ps;
                const float av[4] = {a.x, a.y, a.z, a.w};
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    if (4 * ps + i <= c.plim) f_dbg[t * d.N + c.i0 + 4 * ps + i] = av[i] + bg[i];
            }
        }
        __syncthreads();
        if (w == 0)
            d.llpart[(static_cast<size_t>(c.g) * d.n_seg + seg) * 32 + lane] =
                ((ss_s[0][lane] + ss_s[1][lane]) + ss_s[2][lane]) + ss_s[3][lane];
    } else {
    if (PS > 1) {   // sum the PS partial profiles of the tile: shares 1.. in order onto share 0
        if (ps > 0) {
#pragma unroll
            for (int p = 0; p < kPT; ++p) acc_s[((ps - 1) * TW + tw) * kPT + p][lane] = acc[p];
        }
        __syncthreads();
        if (ps == 0) {
#pragma unroll
            for (int q = 1; q < PS; ++q)
#pragma unroll
                for (int p = 0; p < kPT; ++p) acc[p] += acc_s[((q - 1) * TW + tw) * kPT + p][lane];
        }
    }
    if (ps == 0) {
        float ev[kPT];
        const float ss = tile_residual(d, c, acc, ev);
        if (BWD) {
#pragma unroll
            for (int v = 0; v < kPT / 4; ++v)
                e_s[tw][v][lane] = make_float4(ev[4 * v], ev[4 * v + 1], ev[4 * v + 2], ev[4 * v + 3]);
        }
        ss_s[tw][lane] = ss;
        if (f_dbg && live) tile_debug_profile(d, c, acc, f_dbg, n_dbg);
    }
    __syncthreads();
    if (w == 0) {  // fixed-order sum over the tiles of the segment
        float ss = ss_s[0][lane];
#pragma unroll
        for (int v = 1; v < TW; ++v) ss += ss_s[v][lane];
        d.llpart[(static_cast<size_t>(c.g) * d.n_seg + seg) * 32 + lane] = ss;
    }
    }
    tl_stamp(d.tl, tl_row, 1);
    if (!BWD) return;
    if (rng.x >= rng.y) { tl_stamp(d.tl, tl_row, 2); return; }
    float e[kPT];
#pragma unroll
    for (int v = 0; v < kPT / 4; ++v) {
        const float4 t = e_s[tw][v][lane];
        e[4 * v] = t.x; e[4 * v + 1] = t.y; e[4 * v + 2] = t.z; e[4 * v + 3] = t.w;
    }
    if constexpr (MODEL == 1) tile_phase2_asym(d, src, c, rng, e, group);
    else tile_phase2(d, src, c, rng, e, group);
    tl_stamp(d.tl, tl_row, 2);
}

// Split variant for launches with few tile-warps (PS > 1; configs 1 and 4): one warp per CTA, work items taken from a
// ticket counter in the order  [phase-1 items of all tiles by decreasing work] [phase-2 items in the same order]:
//   phase-1 item (tile, share, group): partial profile of the share's runs -> global memory (L2), then a release
//                                      increment of the (tile, group) counter;
//   phase-2 item (tile, share, group): waits until the PS partial profiles of its (tile, group) have arrived (their
//                                      items have lower tickets, i.e. they are running or done: no deadlock), sums
//                                      them in share order, forms the residual and runs its share of phase 2.
// No barrier inside a CTA, items half as long as a fused CTA, phase-2 work fills the tail of phase 1.  All sums keep
// a fixed order, so results do not depend on the schedule.  grid: n_items * 2 (BWD) or n_items + n_tile * G CTAs
// (a persistent variant, 3552 CTAs looping over tickets, measured 3 % slower).
template <int PS, bool BWD, int MODEL>
__global__ void __launch_bounds__(32, XRDVI_TILE_WARPS_PER_SM) elbo_split_kernel(const Dev d, float* __restrict__ f_dbg, long long n_dbg) {
    const int lane = threadIdx.x;
    griddep_wait();
    griddep_launch_dependents();                           // after the wait: see elbo_tile_kernel
    if (blockIdx.x == gridDim.x - 1) finish_step(d);       // previous step's ELBO / count
    const unsigned n_items = static_cast<unsigned>(d.n_tile) * PS * d.G;
    unsigned ticket = 0;
    if (lane == 0) ticket = atomicAdd(&d.ctl->ticket, 1u);
    ticket = __shfl_sync(0xffffffffu, ticket, 0);
    const bool second = ticket >= n_items;
    tl_stamp(d.tl, ticket, 0);
    if (second) tl_stamp(d.tl, ticket, 1);                 // a phase-2 item: no phase-1 part
    unsigned item = second ? ticket - n_items : ticket;
    int ps, gi, pos;
    if (second && !BWD) {            // forward only: one phase-2 item per (tile, group), played by share 0
        ps = 0;
        gi = item % d.G;
        pos = item / d.G;
    } else {
        gi = item % d.G;
        item /= d.G;
        ps = item % PS;
        pos = item / PS;
    }
    const int tile = d.seg_order[pos];                     // TW = 1: segments are tiles
    const TileCtx c = tile_ctx(d, d.g_base + gi, tile);
    const int2 rng = d.share_rng[tile * PS + ps];
    if (d.tl) tl_tag(d.tl, ticket, rng.x < rng.y ? d.run_tab[rng.y - 1].y - d.run_tab[rng.x].x : 0);
    const size_t tg = static_cast<size_t>(gi) * d.n_tile + tile;
    float* __restrict__ partial = d.partial + tg * (PS * kPT * 32) + lane;

    if (!second) {
        float acc[kPT];
#pragma unroll
        for (int p = 0; p < kPT; ++p) acc[p] = 0.0f;
        if constexpr (MODEL == 1) tile_phase1_asym(d, SrcGlobal{d.pk_tile, d.run_tab}, c, rng, acc);
        else tile_phase1(d, SrcGlobal{d.pk_tile, d.run_tab}, c, rng, acc);
#pragma unroll
        for (int p = 0; p < kPT; ++p) __stcg(partial + (ps * kPT + p) * 32, acc[p]);
        __threadfence();
        __syncwarp();
        if (lane == 0) atomicAdd(&d.tile_cnt[tg], 1u);
        tl_stamp(d.tl, ticket, 1);
    } else {
        if (lane == 0) {
            while (atomicAdd(&d.tile_cnt[tg], 0u) < static_cast<unsigned>(PS)) __nanosleep(64);
        }
        __syncwarp();
        __threadfence();
        float acc[kPT];
#pragma unroll
        for (int p = 0; p < kPT; ++p) acc[p] = __ldcg(partial + p * 32);
#pragma unroll
        for (int q = 1; q < PS; ++q)
#pragma unroll
            for (int p = 0; p < kPT; ++p) acc[p] += __ldcg(partial + (q * kPT + p) * 32);
        float ev[kPT];
        const float ss = tile_residual(d, c, acc, ev);
        if (ps == 0) {
            d.llpart[(static_cast<size_t>(c.g) * d.n_seg + tile) * 32 + lane] = ss;
            if (f_dbg) tile_debug_profile(d, c, acc, f_dbg, n_dbg);
        }
        if (BWD) {
            if constexpr (MODEL == 1) tile_phase2_asym(d, SrcGlobal{d.pk_tile, d.run_tab}, c, rng, ev, gi);
            else tile_phase2(d, SrcGlobal{d.pk_tile, d.run_tab}, c, rng, ev, gi);
        }
        __syncwarp();
        if (lane == 0) {   // the last phase-2 item of the (tile, group) re-arms its counters for the next launch
            const unsigned n_second = BWD ? PS : 1;
            if (atomicAdd(&d.tile_cnt2[tg], 1u) == n_second - 1) {
                d.tile_cnt[tg] = 0u;
                d.tile_cnt2[tg] = 0u;
            }
        }
    }
    tl_stamp(d.tl, ticket, 2);
    if (lane == 0) {       // the last CTA of the launch re-arms the ticket counter
        __threadfence();
        if (atomicAdd(&d.ctl->finished, 1u) == gridDim.x - 1) {
            d.ctl->ticket = 0u;
            d.ctl->finished = 0u;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// deterministic block reduction of NV doubles per thread (fixed shuffle tree, then warps in order)
template <int NV, int NWARPS>
__device__ __forceinline__ void block_reduce(double (&v)[NV], double* smem /* [NWARPS][NV] */) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[i] += __shfl_xor_sync(0xffffffffu, v[i], o);
    }
    if (lane == 0) {
#pragma unroll
        for (int i = 0; i < NV; ++i) smem[warp * NV + i] = v[i];
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        double a = 0.0;
        for (int w = 0; w < NWARPS; ++w) a += smem[w * NV + i];
        v[i] = a;
    }
    __syncthreads();
}

// a-6 (prior part) + a-7 + a-8 + next a-1/a-2.  grid (K + gpi, PR), block 256.  This kernel is the serial section
// between two tile kernels, so it is written for latency: every load a thread needs is issued before the first
// dependent instruction, and the work that does not depend on the reduced gradient (the prior and Jacobian terms of
// the own draw, the bias corrections, the Philox normals of the next step) runs while the output slots arrive.
//  blockIdx.x = k < K       : reduce the part8 slots of phase k and the per-draw prior/Jacobian terms over the S
//                             draws of instance blockIdx.y -> grad; Adam ascent on the 8 (10) parameters of (inst, k);
//                             draws + transform of the next step for (inst, k, all s)          (do_update)
//  blockIdx.x = K + gi      : log-likelihood of the 32 draws of group gi of the instance (sum of llpart over the
//                             segments: warp w sums the segments t = w mod 8 in increasing order, the eight sums are
//                             combined in a fixed tree) and their sum ll_g
//  Short path (at most one draw per thread, and the phase's slot rows of all groups of the instance fit the dynamic
//  shared memory of the launch, d.upd_smem: configs 0, 1, 3): thread 0 requests the rows with one bulk asynchronous
//  copy per group right after the wait (cp.async.bulk on an mbarrier: no registers in flight, no address arithmetic),
//  and every thread reads its rows from shared memory.  Long path: the loops over global memory.  Both add in the same
//  order (slots in index order, then the draws, fixed shuffle tree, warps in order): results do not depend on the path.
//  The ELBO is assembled, and the step counted, by finish_step (next tile kernel, or finish_step_kernel).
constexpr int kLlBatch = 32;    // llpart loads a thread of a log-likelihood CTA keeps in flight

__device__ __forceinline__ void prior_terms(const Dev& d, const PatConst& pc, const float4 m, const float4 sg, const float4 ep,
                                            float (&gz)[4], float& lp) {
    const Phys q = transform(m, sg, ep);
    gz[0] = 1.0f - pc.lambda_h * q.h;
    gz[1] = -q.mu * d.mu_inv_var;
    gz[2] = d.w_shape - d.w_rate * q.w;
    gz[3] = 1.0f - 2.0f * q.r;
    const float az = fabsf(q.zr);
    lp = (pc.log_lambda_h - pc.lambda_h * q.h + q.zh)
       + (-0.5f * q.mu * q.mu * d.mu_inv_var + d.mu_logc)
       + (d.w_logc + d.w_shape * q.zw - d.w_rate * q.w)
       - (az + 2.0f * log1pf(expf(-az)));
}
// alpha = exp(zeta) ~ Norm(alpha_mu, alpha_sigma) (B.2 PAPER.md:274) + log Jacobian (R30): (log term, g_alpha)
__device__ __forceinline__ float2 prior_alpha(const Dev& d, float m_a, float sg_a, float ea) {
    const float za = fmaf(sg_a, ea, m_a), al = expf(za), da = al - d.alpha_mu;
    return make_float2(-0.5f * da * da * d.alpha_inv_var + d.alpha_logc + za, 1.0f - da * d.alpha_inv_var * al);
}

// STAMP: the instantiation xrdvi_debug_update_timeline launches (thread 0 of every CTA leaves %globaltimer stamps in d.tlu);
// every other launch takes STAMP = false, which has none of that code.
template <bool STAMP>
__global__ void __launch_bounds__(kUpdThreads, 2) update_draw_kernel(const Dev d, const float* __restrict__ var_in,
                                                                  int do_update) {
    constexpr int kW = kUpdThreads / 32;
    __shared__ double red[kW * 11];
    __shared__ double ll_s[kW][32];
    __shared__ float new_ml[10];
    const int inst = blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int pat = inst / d.R;
    const PatConst pc = d.pat[pat];
    // static tables: the slot range of the phase, before the wait
    extern __shared__ __align__(128) float rows_s[];           // short path: [gpi][n_sl][8] slot rows of the phase
    __shared__ __align__(8) unsigned long long mbar_s;
    const int k = blockIdx.x;
    int s0 = 0, n_sl = 0;
    if (k < d.K) { s0 = d.slot_ofs[k]; n_sl = d.slot_ofs[k + 1] - s0; }
    const int n_part = n_sl * d.gpi;
    const int s_pad = d.gpi * 32;
    const bool fast = k < d.K && s_pad <= kUpdThreads && static_cast<long long>(n_part) * 32 <= d.upd_smem;
    if (fast && n_part > 0) {
        if (threadIdx.x == 0) {
            mbar_init(smem_u32(&mbar_s), 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncthreads();                                        // the mbarrier is initialised before anybody polls it
    }
    // Also before the wait: everything the previous update_draw_kernel (or the host) wrote -- the variational parameters,
    // the moments, the normals of this step's draws, the step counter u_step.  That kernel has completed: the tile kernel
    // between the two lets this one start only after its own griddep_wait.  What the tile kernel writes (the output
    // slots, llpart, ctl->step / pending through finish_step) is read after the wait.
    // These loads bypass L1 (ld.global.cg): the SM may still hold lines the previous launches of this kernel read.
    const unsigned tlu_row = blockIdx.y * gridDim.x + blockIdx.x;
    if constexpr (STAMP) tlu_stamp(d.tlu, tlu_row, 0);                          // [0] the CTA is resident
    const long long step = __ldcg(&d.ctl->u_step) +        // completed steps; this is step + 1
        static_cast<long long>(__ldcg(&d.ctl->u_acc) / (static_cast<unsigned long long>(gridDim.x) * gridDim.y));
    const unsigned long long seed = __ldcg(&d.ctl->seed);
    const double inv_s = 1.0 / static_cast<double>(d.S);
    const unsigned it_n = static_cast<unsigned>(step + 2);
    float4 m = make_float4(0.f, 0.f, 0.f, 0.f), l = m;
    float m_a = 0.0f, l_a = 0.0f;
    // the parameter this thread updates (threads 0..7: (m, l) x 4 classes; 8, 9: alpha), its moments, the bias corrections
    const bool upd_thread = k < d.K && (threadIdx.x < 8 || (threadIdx.x < 10 && d.asym));
    const bool is_l = threadIdx.x < 8 ? threadIdx.x >= 4 : threadIdx.x == 9;
    const size_t o_par = threadIdx.x < 8
        ? (static_cast<size_t>(inst) * 2 * d.K + (is_l ? d.K : 0) + k) * 4 + (threadIdx.x & 3)
        : static_cast<size_t>(inst) * 2 * d.K + (is_l ? d.K : 0) + k;
    float x_par = 0.0f, m1_par = 0.0f, m2_par = 0.0f;
    float bc1 = 1.0f, bc2 = 1.0f;                    // Adam bias corrections of this step
    if (k < d.K) {
        m = __ldcg(reinterpret_cast<const float4*>(var_in + (static_cast<size_t>(inst) * 2 * d.K + k) * 4));
        l = __ldcg(reinterpret_cast<const float4*>(var_in + (static_cast<size_t>(inst) * 2 * d.K + d.K + k) * 4));
        // R30: the fifth latent's parameters sit behind the [PR][2][K][4] block of every state array
        const float* __restrict__ va_in = var_in + static_cast<size_t>(d.PR) * 8 * d.K + static_cast<size_t>(inst) * 2 * d.K;
        if (d.asym) { m_a = __ldcg(va_in + k); l_a = __ldcg(va_in + d.K + k); }
        if (upd_thread) {
            x_par = threadIdx.x < 8 ? __ldcg(var_in + o_par) : (is_l ? l_a : m_a);
            if (do_update && d.optimizer != 1) {
                m1_par = __ldcg((threadIdx.x < 8 ? d.mom1 : d.mom1_a) + o_par);
                m2_par = __ldcg((threadIdx.x < 8 ? d.mom2 : d.mom2_a) + o_par);
                const float stepf = static_cast<float>(step + 1 - __ldcg(&d.ctl->adam_t0));
                bc1 = 1.0f - powf(d.beta1, stepf);
                bc2 = 1.0f - powf(d.beta2, stepf);
            }
        }
    }
    // short path: prior + Jacobian terms of the thread's draw and the Philox normals of its next draw
    const bool has_draw = fast && static_cast<int>(threadIdx.x) < d.S;
    float4 ep = make_float4(0.f, 0.f, 0.f, 0.f), ep_n = ep;
    float ea = 0.0f, epa_n = 0.0f;
    float gz[4] = {0.f, 0.f, 0.f, 0.f}, lp = 0.0f;
    float2 pr_a = make_float2(0.f, 0.f);
    if (fast) {
        const int s = threadIdx.x;
        if (has_draw) {
            const size_t o_draw = (static_cast<size_t>(inst * d.gpi + (s >> 5)) * d.K + k) * 32 + lane;
            ep = __ldcg(d.eps + o_draw);
            if (d.asym) ea = __ldcg(d.eps_a + o_draw);
            const float4 sg = make_float4(expf(l.x), expf(l.y), expf(l.z), expf(l.w));
            prior_terms(d, pc, m, sg, ep, gz, lp);
            if (d.asym) pr_a = prior_alpha(d, m_a, expf(l_a), ea);
        }
        if (do_update && s < s_pad) {
            const uint2 key = make_uint2(static_cast<unsigned>(seed), static_cast<unsigned>(seed >> 32));
            ep_n = normals_from_words(philox4x32_10(
                make_uint4(it_n, static_cast<unsigned>(s), static_cast<unsigned>(k), static_cast<unsigned>(inst)), key));
            if (d.asym) epa_n = normal_alpha(it_n, static_cast<unsigned>(s), static_cast<unsigned>(k), static_cast<unsigned>(inst), seed);
        }
    }
    if constexpr (STAMP) tlu_stamp(d.tlu, tlu_row, 1);                          // [1] done with what needs no output of the tile kernel
    griddep_launch_dependents();
    griddep_wait();                               // output slots, llpart: written by the tile kernel
    if constexpr (STAMP) tlu_stamp(d.tlu, tlu_row, 2);                          // [2] the wait returned
    if (fast && n_part > 0 && threadIdx.x == 0) {               // the slot rows of the phase, one contiguous piece per group
        const unsigned mb = smem_u32(&mbar_s), piece = 32u * static_cast<unsigned>(n_sl);
        mbar_expect_tx(mb, piece * static_cast<unsigned>(d.gpi));
        const float* __restrict__ src = d.part8 + (static_cast<size_t>(inst) * d.gpi * d.n_slots + s0) * 8;
        for (int gi = 0; gi < d.gpi; ++gi)
            bulk_g2s(smem_u32(rows_s) + piece * gi, src + static_cast<size_t>(gi) * d.n_slots * 8, piece, mb);
    }

    if (k >= d.K) {
        const int gi = k - d.K;
        const int g = inst * d.gpi + gi;
        const float* __restrict__ lp_g = d.llpart + static_cast<size_t>(g) * d.n_seg * 32 + lane;
        const int n_i = warp < d.n_seg ? (d.n_seg - warp + kW - 1) / kW : 0;   // segments warp, warp + 8, ...
        double a = 0.0;
        for (int i = 0; i < n_i; i += kLlBatch) {      // kLlBatch loads in flight, added in segment order
            float x[kLlBatch];
#pragma unroll
            for (int j = 0; j < kLlBatch; ++j) x[j] = i + j < n_i ? lp_g[static_cast<size_t>(warp + kW * (i + j)) * 32] : 0.0f;
#pragma unroll
            for (int j = 0; j < kLlBatch; ++j)
                if (i + j < n_i) a += static_cast<double>(x[j]);
        }
        if constexpr (STAMP) tlu_stamp(d.tlu, tlu_row, 3);                      // [3] log-likelihood CTA: the tiles are added
        ll_s[warp][lane] = a;
        __syncthreads();
        if (warp == 0) {
            const double a8 = ((ll_s[0][lane] + ll_s[1][lane]) + (ll_s[2][lane] + ll_s[3][lane])) +
                              ((ll_s[4][lane] + ll_s[5][lane]) + (ll_s[6][lane] + ll_s[7][lane]));
            const int s = gi * 32 + lane;
            double ll = 0.0;
            if (s < d.S) {
                ll = static_cast<double>(pc.ll_scale) * a8 + pc.ll_const;
                d.ll_t[static_cast<size_t>(inst) * s_pad + s] = ll;
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) ll += __shfl_xor_sync(0xffffffffu, ll, o);
            if (lane == 0) d.ll_g[g] = ll;
        }
        if (k == d.K && inst == 0 && threadIdx.x == 0) d.ctl->pending = do_update ? 2u : 1u;
        if (do_update && threadIdx.x == 0) atomicAdd(&d.ctl->u_acc, 1ull);    // this CTA is done (result unused: a reduction)
        if constexpr (STAMP) tlu_stamp(d.tlu, tlu_row, 7);
        return;
    }

    double v[11];   // [0..3] sum g, [4..7] sum g eps, [8] sum log prior + log Jacobian, [9] sum g_alpha, [10] sum g_alpha eps_alpha
#pragma unroll
    for (int i = 0; i < 11; ++i) v[i] = 0.0;

    if (fast) {
        if (d.asym) {     // the alpha pair of every slot (R30 only): from global memory, under the bulk copies
            for (int idx = threadIdx.x; idx < n_part; idx += kUpdThreads) {
                const int gi = idx / n_sl, sl = s0 + (idx - gi * n_sl);
                const float2 pa = *reinterpret_cast<const float2*>(
                    d.parta + (static_cast<size_t>(inst * d.gpi + gi) * d.n_slots + sl) * 2);
                v[9] += pa.x;
                v[10] += pa.y;
            }
        }
        // likelihood part, slots in index order (row idx of the staged block = group gi, slot s0 + idx - gi n_sl)
        if (n_part > 0) {
            mbar_wait(smem_u32(&mbar_s), 0u);
            for (int idx = threadIdx.x; idx < n_part; idx += kUpdThreads) {
                const float4 a = *reinterpret_cast<const float4*>(rows_s + static_cast<size_t>(idx) * 8);
                const float4 b = *reinterpret_cast<const float4*>(rows_s + static_cast<size_t>(idx) * 8 + 4);
                v[0] += a.x; v[1] += a.y; v[2] += a.z; v[3] += a.w;
                v[4] += b.x; v[5] += b.y; v[6] += b.z; v[7] += b.w;
            }
        }
        if (has_draw) {
            const float e4[4] = {ep.x, ep.y, ep.z, ep.w};
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                v[c] += static_cast<double>(gz[c]);
                v[4 + c] += static_cast<double>(gz[c] * e4[c]);
            }
            v[8] += static_cast<double>(lp);
            if (d.asym) {
                v[8] += static_cast<double>(pr_a.x);
                v[9] += static_cast<double>(pr_a.y);
                v[10] += static_cast<double>(pr_a.y * ea);
            }
        }
    } else {
        // likelihood part: partials of phase k, all groups of the instance
        for (int idx = threadIdx.x; idx < n_part; idx += kUpdThreads) {
            const int gi = idx / n_sl, sl = s0 + (idx - gi * n_sl);
            const float4* __restrict__ pp = reinterpret_cast<const float4*>(
                d.part8 + (static_cast<size_t>(inst * d.gpi + gi) * d.n_slots + sl) * 8);
            const float4 a = pp[0], b = pp[1];
            v[0] += a.x; v[1] += a.y; v[2] += a.z; v[3] += a.w;
            v[4] += b.x; v[5] += b.y; v[6] += b.z; v[7] += b.w;
        }
        if (d.asym) {
            for (int idx = threadIdx.x; idx < n_part; idx += kUpdThreads) {
                const int gi = idx / n_sl, sl = s0 + (idx - gi * n_sl);
                const float2 pa = *reinterpret_cast<const float2*>(
                    d.parta + (static_cast<size_t>(inst * d.gpi + gi) * d.n_slots + sl) * 2);
                v[9] += pa.x;
                v[10] += pa.y;
            }
        }
        // prior + Jacobian part, per draw
        const float4 sg = make_float4(expf(l.x), expf(l.y), expf(l.z), expf(l.w));
        const float sg_a = expf(l_a);
        for (int s = threadIdx.x; s < d.S; s += kUpdThreads) {
            const int g = inst * d.gpi + (s >> 5);
            const float4 ep = d.eps[(static_cast<size_t>(g) * d.K + k) * 32 + lane];
            float gz[4], lp;
            prior_terms(d, pc, m, sg, ep, gz, lp);
            const float e4[4] = {ep.x, ep.y, ep.z, ep.w};
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                v[c] += static_cast<double>(gz[c]);
                v[4 + c] += static_cast<double>(gz[c] * e4[c]);
            }
            v[8] += static_cast<double>(lp);
            if (d.asym) {
                const float ea = d.eps_a[(static_cast<size_t>(g) * d.K + k) * 32 + lane];
                const float2 pr_a = prior_alpha(d, m_a, sg_a, ea);
                v[8] += static_cast<double>(pr_a.x);
                v[9] += static_cast<double>(pr_a.y);
                v[10] += static_cast<double>(pr_a.y * ea);
            }
        }
    }

    if constexpr (STAMP) tlu_stamp(d.tlu, tlu_row, 3);                          // [3] phase CTA: slots and prior terms are added
    // deterministic block reduction: fixed shuffle tree inside a warp, then thread i < 11 adds the warps' sums of
    // value i in warp order.  Thread i < 8 owns parameter i, threads 8 / 9 the alpha pair (sums 9 / 10), thread 10 sum 8.
    const int n_red = d.asym ? 11 : 9;
#pragma unroll
    for (int i = 0; i < 11; ++i) {
        if (i < n_red) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v[i] += __shfl_xor_sync(0xffffffffu, v[i], o);
        }
    }
    if (lane == 0) {
#pragma unroll
        for (int i = 0; i < 11; ++i) red[warp * 11 + i] = v[i];
    }
    __syncthreads();
    if constexpr (STAMP) tlu_stamp(d.tlu, tlu_row, 4);                          // [4] shuffle trees and the barrier
    if (threadIdx.x < 11) {
        const int col = threadIdx.x < 8 ? threadIdx.x : threadIdx.x == 10 ? 8 : threadIdx.x + 1;
        double tot = 0.0;
#pragma unroll
        for (int w = 0; w < kW; ++w) tot += red[w * 11 + col];
        if (threadIdx.x == 10) {
            // mean log prior + Jacobian of the phase, plus its entropy sum_c (l_c + 1/2 ln 2 pi e)
            d.elbo_k[static_cast<size_t>(inst) * (d.K + 1) + k] =
                tot * inv_s + (static_cast<double>(l.x) + static_cast<double>(l.y) + static_cast<double>(l.z) +
                               static_cast<double>(l.w)) + 4.0 * 1.4189385332046727 +
                (d.asym ? static_cast<double>(l_a) + 1.4189385332046727 : 0.0);
        } else if (upd_thread) {
            const int c = threadIdx.x & 3;
            const float lc = threadIdx.x >= 8 ? l_a : c == 0 ? l.x : c == 1 ? l.y : c == 2 ? l.z : l.w;
            const float sgc = expf(lc);
            const double gd = is_l ? tot * inv_s * static_cast<double>(sgc) + 1.0 : tot * inv_s;
            const float gj = static_cast<float>(gd);
            (threadIdx.x < 8 ? d.grad : d.grad_a)[o_par] = gj;
            float x = x_par;
            if (do_update) {   // l clamped to [-12, 2]
                if (d.optimizer == 1) {   // natural-gradient ascent: Fisher metric diag(1/sigma^2, 2) (R25)
                    x += d.lr * (is_l ? 0.5f * gj : sgc * sgc * gj);
                } else {                  // Adam ascent, bias-corrected (R10)
                    // the roundings are written out (one product rounded, the other fused), so that the moments do
                    // not depend on how a compiler version contracts the two-term sums
                    const float m1 = __fmaf_rn(gj, 1.0f - d.beta1, __fmul_rn(d.beta1, m1_par));
                    const float m2 = __fmaf_rn(m2_par, d.beta2, __fmul_rn(__fmul_rn(1.0f - d.beta2, gj), gj));
                    (threadIdx.x < 8 ? d.mom1 : d.mom1_a)[o_par] = m1;
                    (threadIdx.x < 8 ? d.mom2 : d.mom2_a)[o_par] = m2;
                    x += d.lr * (m1 / bc1) / (sqrtf(m2 / bc2) + d.adam_eps);
                }
                if (is_l) x = fminf(fmaxf(x, -12.0f), 2.0f);
                (threadIdx.x < 8 ? d.var : d.var_a)[o_par] = x;
            }
            new_ml[threadIdx.x] = x;
        }
    }
    if constexpr (STAMP) tlu_stamp(d.tlu, tlu_row, 5);                          // [5] the parameter of thread 0 is updated
    if (do_update) {       // draws of the next step from the updated parameters
        __syncthreads();
        if constexpr (STAMP) tlu_stamp(d.tlu, tlu_row, 6);                      // [6] all parameters of the phase are updated
        const float4 mn = make_float4(new_ml[0], new_ml[1], new_ml[2], new_ml[3]);
        const float4 ln = make_float4(new_ml[4], new_ml[5], new_ml[6], new_ml[7]);
        const float mna = d.asym ? new_ml[8] : 0.0f, lna = d.asym ? new_ml[9] : 0.0f;
        if (fast) {
            const int s = threadIdx.x;
            if (s < s_pad) {   // whole warps
                const float4 sgn = make_float4(expf(ln.x), expf(ln.y), expf(ln.z), expf(ln.w));
                float alpha = 1.0f;
                if (d.asym) alpha = expf(fmaf(expf(lna), epa_n, mna));
                emit_latent(d, inst * d.gpi + (s >> 5), k, s < d.S, transform(mn, sgn, ep_n), ep_n, alpha, epa_n);
            }
        } else {
            for (int s = threadIdx.x; s < s_pad; s += kUpdThreads) draw_one(d, inst, k, s, it_n, seed, mn, ln, nullptr, mna, lna);
        }
    }
    if (do_update && threadIdx.x == 0) atomicAdd(&d.ctl->u_acc, 1ull);        // this CTA is done (result unused: a reduction)
    if constexpr (STAMP) tlu_stamp(d.tlu, tlu_row, 7);                          // [7] done
}

// a-7 (last part): ELBO of every instance = mean log-likelihood + sum over the phases of (mean log prior + log
// Jacobian + entropy), summed in phase order; trace row and step counter of an optimisation step.
// grid 1, block 256: finish_step after the last step of a run and after single evaluations.
__global__ void __launch_bounds__(256) finish_step_kernel(const Dev d) { finish_step(d); }

// a-10: inclusion probability and area ratio (R15), fp64.  grid PR, block 128.
__global__ void __launch_bounds__(128) inclusion_kernel(const Dev d, double tau, double* __restrict__ incl,
                                                        double* __restrict__ ratio) {
    __shared__ double red[4];
    const int inst = blockIdx.x;
    const float* m = d.var + static_cast<size_t>(inst) * 8 * d.K;
    const float* l = m + 4 * d.K;
    // R30: a split peak has area (1 + alpha) / 2, alpha at its mean under q
    const float* ma = d.var_a + static_cast<size_t>(inst) * 2 * d.K;
    auto area_of = [&](int k) {
        double a = d.area[k];
        if (d.asym) {
            const double sa = exp(static_cast<double>(ma[d.K + k]));
            a *= 0.5 * (1.0 + exp(static_cast<double>(ma[k]) + 0.5 * sa * sa));
        }
        return a;
    };
    double v[1] = {0.0};
    for (int k = threadIdx.x; k < d.K; k += 128) {
        const double s = exp(static_cast<double>(l[4 * k]));
        v[0] += area_of(k) * exp(static_cast<double>(m[4 * k]) + 0.5 * s * s);
    }
    block_reduce<1, 4>(v, red);
    const double tbar = v[0];
    for (int k = threadIdx.x; k < d.K; k += 128) {
        const double s = exp(static_cast<double>(l[4 * k]));
        const double ak = area_of(k);
        const double z = (static_cast<double>(m[4 * k]) - log(tau * tbar / ak)) / s;
        incl[static_cast<size_t>(inst) * d.K + k] = 0.5 * erfc(-z * 0.70710678118654752440);
        ratio[static_cast<size_t>(inst) * d.K + k] = ak * exp(static_cast<double>(m[4 * k]) + 0.5 * s * s) / tbar;
    }
}

// Marginal summaries of q in the constrained parameters (R28; the paper's Fig. 6 marginals), fp64.
// grid (ceil(K / 4), PR), block 128: one warp per phase.  out [PR][K][4][5] = mean, sd, 2.5 %, 50 %, 97.5 % quantile.
// h, w log-normal, mu normal (closed forms, lanes 0..2); r logit-normal: trapezoid rule on z in [-10, 10], step 1/32,
// of (r - r0) and (r - r0)^2 against the normal density, r0 = sigmoid(m) (centred, so a narrow q does not cancel),
// the 641 points strided over the lanes and folded by a fixed-order shuffle tree.  The integrand is analytic in
// |Im z| < pi / sigma >= 0.42 (sigma <= e^2, R10): trapezoid error ~ e^-85.
__global__ void __launch_bounds__(128) posterior_summary_kernel(const Dev d, double* __restrict__ out) {
    const int lane = threadIdx.x & 31;
    const int k = blockIdx.x * 4 + (threadIdx.x >> 5);
    if (k >= d.K) return;
    const int inst = blockIdx.y;
    const float* mp = d.var + static_cast<size_t>(inst) * 8 * d.K + 4 * k;
    const double z975 = 1.95996398454005423552;
    const int C5 = d.asym ? 25 : 20;                       // classes x 5 values per phase
    double* ok = out + (static_cast<size_t>(inst) * d.K + k) * C5;
    if (lane == 4 && d.asym) {                             // alpha = exp(zeta): log-normal (R30)
        const float* ma = d.var_a + static_cast<size_t>(inst) * 2 * d.K;
        const double m = static_cast<double>(ma[k]), s = exp(static_cast<double>(ma[d.K + k]));
        const double mean = exp(m + 0.5 * s * s);
        double* o = ok + 20;
        o[0] = mean; o[1] = sqrt(expm1(s * s)) * mean;
        o[2] = exp(m - s * z975); o[3] = exp(m); o[4] = exp(m + s * z975);
    }
    if (lane < 3) {
        const double m = static_cast<double>(mp[lane]);
        const double s = exp(static_cast<double>(mp[4 * d.K + lane]));
        double* o = ok + 5 * lane;
        if (lane == 1) {
            o[0] = m; o[1] = s; o[2] = m - s * z975; o[3] = m; o[4] = m + s * z975;
        } else {
            const double mean = exp(m + 0.5 * s * s);
            o[0] = mean; o[1] = sqrt(expm1(s * s)) * mean;
            o[2] = exp(m - s * z975); o[3] = exp(m); o[4] = exp(m + s * z975);
        }
    }
    const double m = static_cast<double>(mp[3]);
    const double s = exp(static_cast<double>(mp[4 * d.K + 3]));
    const double r0 = 1.0 / (1.0 + exp(-m));
    double a0 = 0.0, a1 = 0.0, a2 = 0.0;
    for (int i = -320 + lane; i <= 320; i += 32) {
        const double z = i * 0.03125;
        const double ph = ((i == -320 || i == 320) ? 0.5 : 1.0) * exp(-0.5 * z * z);
        const double dr = 1.0 / (1.0 + exp(-(m + s * z))) - r0;
        a0 += ph; a1 += ph * dr; a2 += ph * dr * dr;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a0 += __shfl_xor_sync(0xffffffffu, a0, o);
        a1 += __shfl_xor_sync(0xffffffffu, a1, o);
        a2 += __shfl_xor_sync(0xffffffffu, a2, o);
    }
    if (lane == 3) {
        const double e1 = a1 / a0, e2 = a2 / a0;
        double* o = ok + 15;
        o[0] = r0 + e1; o[1] = sqrt(fmax(e2 - e1 * e1, 0.0));
        o[2] = 1.0 / (1.0 + exp(-(m - s * z975))); o[3] = r0; o[4] = 1.0 / (1.0 + exp(-(m + s * z975)));
    }
}

// R11 initial state.  grid PR, block 128 over phases.
__global__ void __launch_bounds__(128) init_state_kernel(const Dev d, const float* __restrict__ m_h0 /*[P]*/,
                                                         float m_w0, float init_log_sigma, unsigned long long seed,
                                                         int restart_offset) {
    const int inst = blockIdx.x;
    const int pat = inst / d.R, rst = inst - pat * d.R + restart_offset;   // the restart index the jitter is drawn for
    for (int k = threadIdx.x; k < d.K; k += 128) {
        float4 m = make_float4(m_h0[pat], 0.0f, m_w0, 0.0f);
        if (rst > 0) {
            const uint4 w = philox4x32_10(make_uint4(0xFFFFFFFFu, static_cast<unsigned>(rst), static_cast<unsigned>(k),
                                                     static_cast<unsigned>(pat)),
                                          make_uint2(static_cast<unsigned>(seed), static_cast<unsigned>(seed >> 32)));
            const float4 ep = normals_from_words(w);
            m.x += 0.5f * ep.x; m.y += 0.01f * ep.y; m.z += 0.2f * ep.z; m.w += 0.5f * ep.w;
        }
        float* o = d.var + (static_cast<size_t>(inst) * 2 * d.K + k) * 4;
        o[0] = m.x; o[1] = m.y; o[2] = m.z; o[3] = m.w;
        float* ol = o + 4 * d.K;
        ol[0] = ol[1] = ol[2] = ol[3] = init_log_sigma;
        if (d.asym) {   // R30: alpha starts at 1; restart jitter 0.05 eps from a second Philox call (bit 31 of the phase word)
            float m_a = 0.0f;
            if (rst > 0)
                m_a = 0.05f * normal_alpha(0xFFFFFFFFu, static_cast<unsigned>(rst), static_cast<unsigned>(k),
                                           static_cast<unsigned>(pat), seed);
            d.var_a[static_cast<size_t>(inst) * 2 * d.K + k] = m_a;
            d.var_a[static_cast<size_t>(inst) * 2 * d.K + d.K + k] = init_log_sigma;
        }
    }
    const int per = 8 * d.K;
    for (int j = threadIdx.x; j < per; j += 128) {
        d.mom1[static_cast<size_t>(inst) * per + j] = 0.0f;
        d.mom2[static_cast<size_t>(inst) * per + j] = 0.0f;
    }
    if (d.asym)
        for (int j = threadIdx.x; j < 2 * d.K; j += 128) {
            d.mom1_a[static_cast<size_t>(inst) * 2 * d.K + j] = 0.0f;
            d.mom2_a[static_cast<size_t>(inst) * 2 * d.K + j] = 0.0f;
        }
}

// ------------------------------------------------------------------------------------------------
// Log-joint gradient service (the gradient an HMC / MCMC sampler of the paper's Table 1 needs):
// the caller supplies the unconstrained latents zeta [n][K][4] of n points; the tile kernel runs on them exactly
// as on draws and leaves d ll / d zeta per draw in d.pd.

// a-2 for supplied points.  grid (ceil(K/4), groups of this launch), block 128.  Point of lane:
// s = (s_group0 + blockIdx.y) * 32 + lane.
__global__ void __launch_bounds__(128) zeta_latent_kernel(const Dev d, const float4* __restrict__ zeta,
                                                          const float* __restrict__ zeta_a, int n, int s_group0) {
    const int lane = threadIdx.x & 31;
    const int k = blockIdx.x * 4 + (threadIdx.x >> 5);
    if (k >= d.K) return;
    const int s = (s_group0 + blockIdx.y) * 32 + lane;
    const bool valid = s < n;
    const float4 z = valid ? zeta[static_cast<size_t>(s) * d.K + k] : make_float4(0.f, 0.f, 0.f, 0.f);
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
    const float alpha = (d.asym && valid) ? expf(zeta_a[static_cast<size_t>(s) * d.K + k]) : 1.0f;
    emit_latent(d, d.g_base + blockIdx.y, k, valid, transform(z, zero, zero), zero, alpha, 0.0f);
}

// Sum of the per-run gradients of phase k over the tiles (fixed order) + prior and Jacobian part (a-6).
// grid (K, groups of this launch), block 32 (lane = point).  Also the phase's log prior + log Jacobian -> lpk.
__global__ void __launch_bounds__(32) logjoint_grad_kernel(const Dev d, const float4* __restrict__ zeta,
                                                           const float* __restrict__ zeta_a, int n, int s_group0, int pat,
                                                           float4* __restrict__ grad, float* __restrict__ grad_a,
                                                           float* __restrict__ lpk) {
    const int lane = threadIdx.x, k = blockIdx.x, gi = blockIdx.y;
    const int s = (s_group0 + gi) * 32 + lane;
    if (s >= n) return;
    const PatConst pc = d.pat[pat];
    const int row = d.model ? 160 : 128;                   // floats per (run, 32 points): 4 or 5 classes
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0, a4 = 0.0;
    for (int j = d.slot_ofs[k]; j < d.slot_ofs[k + 1]; ++j) {
        const float* __restrict__ o = d.pd + (static_cast<size_t>(gi) * d.n_slots + j) * row + lane;
        a0 += static_cast<double>(o[0]); a1 += static_cast<double>(o[32]);
        a2 += static_cast<double>(o[64]); a3 += static_cast<double>(o[96]);
        if (d.asym) a4 += static_cast<double>(o[128]);
    }
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
    const Phys q = transform(zeta[static_cast<size_t>(s) * d.K + k], zero, zero);
    grad[static_cast<size_t>(s) * d.K + k] =
        make_float4(static_cast<float>(a0 + static_cast<double>(1.0f - pc.lambda_h * q.h)),
                    static_cast<float>(a1 + static_cast<double>(-q.mu * d.mu_inv_var)),
                    static_cast<float>(a2 + static_cast<double>(d.w_shape - d.w_rate * q.w)),
                    static_cast<float>(a3 + static_cast<double>(1.0f - 2.0f * q.r)));
    const float az = fabsf(q.zr);
    float lp = (pc.log_lambda_h - pc.lambda_h * q.h + q.zh) + (-0.5f * q.mu * q.mu * d.mu_inv_var + d.mu_logc) +
               (d.w_logc + d.w_shape * q.zw - d.w_rate * q.w) - (az + 2.0f * log1pf(expf(-az)));
    if (d.asym) {
        const float za = zeta_a[static_cast<size_t>(s) * d.K + k], al = expf(za), da = al - d.alpha_mu;
        grad_a[static_cast<size_t>(s) * d.K + k] =
            static_cast<float>(a4 + static_cast<double>(1.0f - da * d.alpha_inv_var * al));
        lp += -0.5f * da * da * d.alpha_inv_var + d.alpha_logc + za;
    }
    lpk[(static_cast<size_t>(gi) * d.K + k) * 32 + lane] = lp;
}

// ll and log prior + log Jacobian per point.  grid (groups of this launch), block 32.
__global__ void __launch_bounds__(32) logjoint_scalar_kernel(const Dev d, int n, int s_group0, int pat,
                                                             const float* __restrict__ lpk, double* __restrict__ ll,
                                                             double* __restrict__ lpj) {
    const int lane = threadIdx.x, gi = blockIdx.x;
    const int s = (s_group0 + gi) * 32 + lane;
    if (s >= n) return;
    const PatConst pc = d.pat[pat];
    const float* __restrict__ lp = d.llpart + static_cast<size_t>(d.g_base + gi) * d.n_seg * 32 + lane;
    double a = 0.0;
    for (int t = 0; t < d.n_seg; ++t) a += static_cast<double>(lp[static_cast<size_t>(t) * 32]);
    ll[s] = static_cast<double>(pc.ll_scale) * a + pc.ll_const;
    double b = 0.0;
    for (int k = 0; k < d.K; ++k) b += static_cast<double>(lpk[(static_cast<size_t>(gi) * d.K + k) * 32 + lane]);
    lpj[s] = b;
}

}  // namespace xrdvi_dev
