// xrdvi_kernels.cuh -- sm_100a kernels of the ELBO-and-gradient hot path.
//
// Data-parallel axes: a *sample-instance* t = (pattern, restart, draw s) lives in one LANE; 32
// consecutive draws of one (pattern, restart) form a *group* g, so every warp works on one 2theta tile
// (forward) or one peak chunk (backward) for 32 draws at once: peak records and observed data are
// warp-uniform (broadcast loads), latents are lane-private, all global traffic is 128-byte coalesced.
//
// Coordinates: t' = 2 (x_i - p_m - mu) / w, so that  G = exp(-4 ln2 t^2) = 2^(-t'^2)  and
// L = 1/(1+4t^2) = 1/(1+t'^2)  (PAPER.md:221-232 with the unit-area FWHM shapes, reading R1).  A peak is
// stored as (j_m, delta_m) with p_m = x_{j_m} + delta_m computed in fp64 at create, so
// t' = (i - j_m) * (Delta*2/w) + (-delta_m - mu) * 2/w  has no fp32 cancellation at high angles.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace xrdvi_dev {

constexpr int kFwdP = 8;        // grid points per thread in the forward kernel
constexpr int kFwdWarps = 4;    // warps (= tiles) per forward block
constexpr int kBwdWarps = 4;    // warps (= peak units) per backward block
constexpr int kTraceCap = 4096; // iterations of ELBO trace kept on the device

constexpr float kAG = 0.93943727869965132f;  // 2 sqrt(ln2/pi)
constexpr float kAL = 0.63661977236758134f;  // 2/pi
constexpr float kLn2 = 0.69314718055994531f;

struct PeakRec {   // 16 bytes
    int j;         // nearest grid index of the peak (may lie outside [0,N))
    float delta;   // p_m - x_j  (|delta| <= Delta/2), fp64-computed
    float inten;   // I_m
    int k;         // phase
};

struct PatConst {  // per observed pattern
    float inv_sn;      // 1/sigma_n
    float inv_sn2;     // 1/sigma_n^2
    float lambda_h;    // rate of the Exp prior
    float log_lambda_h;
    double ll_const;   // -N ln sigma_n - N/2 ln 2pi
};

struct Ctl {       // device-resident control block (so that graph replays need no new arguments)
    unsigned long long seed;
    long long step;        // completed optimisation steps
    long long trace_base;  // step index of trace row 0
    long long iteration_override;  // >= 0: Philox iteration for elbo_grad/debug; < 0: use step + 1
};

struct Dev {
    // sizes
    int N, NQ, K, P, R, PR, n_c, ntile, n_units, Mv;
    int S, gpi, G;       // draws, groups per instance, groups (run-time)
    float delta;         // grid step (deg)
    // priors / optimiser
    float mu_inv_var, mu_logc, w_shape, w_rate, w_logc;
    float lr, beta1, beta2, adam_eps;
    // static tables
    const float* yb;          // [P][N]  y - B
    const float* bg;          // [P][N]
    const PeakRec* pk_fwd;    // [Mv] sorted by j
    const int2* tile_rng;     // [ntile] peak range [x,y) of each forward tile
    const PeakRec* pk_bwd;    // [Mv] phase-major
    const int4* units;        // [n_units] (k, m0, m1, -)
    const int* unit_ofs;      // [K+1] units of phase k
    const PatConst* pat;      // [P]
    const double* area;       // [K] A_k = sum_m I_m
    // state
    float* var;               // [PR][2][K][4]
    float* mom1;
    float* mom2;
    float* grad;              // [PR][2][K][4]
    double* elbo;             // [PR]
    double* elbo_k;           // [PR][K]
    double* ll_t;             // [PR][S_pad]
    double* trace;            // [kTraceCap][PR]
    Ctl* ctl;
    // per-iteration buffers
    float4* lat;              // [G][K][32]  (2/w, -mu*2/w, h(1-r)aG/w, h r aL/w)
    float4* eps;              // [G][K][32]
    float4* e;                // [G][NQ][32] residual e_i = (y_i - f_i)/sigma_n^2, 4 points per float4
    float* llpart;            // [G][ntile][32] sum over the tile of ((y-f)/sigma_n)^2
    float* sums;              // [G][n_units][6][32]
};

// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
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
__device__ __forceinline__ Phys transform(const float4 m, const float4 l, const float4 ep) {
    Phys q;
    q.zh = fmaf(expf(l.x), ep.x, m.x);
    q.mu = fmaf(expf(l.y), ep.y, m.y);
    q.zw = fmaf(expf(l.z), ep.z, m.z);
    q.zr = fmaf(expf(l.w), ep.w, m.w);
    q.h = expf(q.zh);
    q.w = expf(q.zw);
    q.r = 1.0f / (1.0f + expf(-q.zr));
    return q;
}

__device__ __forceinline__ long long philox_iteration(const Ctl* ctl) {
    const long long o = ctl->iteration_override;
    return o >= 0 ? o : ctl->step + 1;
}

// ------------------------------------------------------------------------------------------------
// a-1 + a-2: draws and transform.  grid (ceil(K/4), G), block 128: thread = (phase k, lane).
__global__ void __launch_bounds__(128) draw_transform_kernel(const Dev d, const float* __restrict__ var,
                                                              uint4* __restrict__ raw_out) {
    const int lane = threadIdx.x & 31;
    const int k = blockIdx.x * 4 + (threadIdx.x >> 5);
    const int g = blockIdx.y;
    if (k >= d.K) return;
    const int inst = g / d.gpi;
    const int s = (g - inst * d.gpi) * 32 + lane;
    const unsigned long long seed = d.ctl->seed;
    const unsigned it = static_cast<unsigned>(philox_iteration(d.ctl));
    const uint4 words = philox4x32_10(make_uint4(it, static_cast<unsigned>(s), static_cast<unsigned>(k),
                                                 static_cast<unsigned>(inst)),
                                      make_uint2(static_cast<unsigned>(seed), static_cast<unsigned>(seed >> 32)));
    const float4 ep = normals_from_words(words);
    const float4 m = *reinterpret_cast<const float4*>(var + (static_cast<size_t>(inst) * 2 * d.K + k) * 4);
    const float4 l = *reinterpret_cast<const float4*>(var + (static_cast<size_t>(inst) * 2 * d.K + d.K + k) * 4);
    const Phys q = transform(m, l, ep);
    const float iw = 1.0f / q.w;
    const float iw2 = 2.0f * iw;
    float4 lt = make_float4(iw2, -q.mu * iw2, q.h * (1.0f - q.r) * kAG * iw, q.h * q.r * kAL * iw);
    if (s >= d.S) lt = make_float4(1.0f, 0.0f, 0.0f, 0.0f);  // padding lanes contribute nothing
    const size_t o = (static_cast<size_t>(g) * d.K + k) * 32 + lane;
    d.lat[o] = lt;
    d.eps[o] = ep;
    if (raw_out) raw_out[o] = words;
}

// ------------------------------------------------------------------------------------------------
// a-3 + a-4: fused profile + residual.  grid (ceil(ntile/kFwdWarps), G), block 32*kFwdWarps.
// Warp = one tile of kFwdP consecutive grid points for the 32 draws of group g.
__global__ void __launch_bounds__(32 * kFwdWarps) forward_kernel(const Dev d, float* __restrict__ f_dbg,
                                                                  long long n_dbg) {
    const int lane = threadIdx.x & 31;
    const int tile = blockIdx.x * kFwdWarps + (threadIdx.x >> 5);
    const int g = blockIdx.y;
    if (tile >= d.ntile) return;
    const int i0 = tile * kFwdP;
    const int2 rng = d.tile_rng[tile];
    const float4* __restrict__ lat = d.lat + static_cast<size_t>(g) * d.K * 32 + lane;
    const int full_lo = i0 + kFwdP - 1 - d.n_c, full_hi = i0 + d.n_c;

    float acc[kFwdP];
#pragma unroll
    for (int p = 0; p < kFwdP; ++p) acc[p] = 0.0f;

    for (int m = rng.x; m < rng.y; ++m) {
        const PeakRec pk = d.pk_fwd[m];
        const float4 lt = lat[static_cast<size_t>(pk.k) * 32];
        const float step = d.delta * lt.x;
        const float tc = fmaf(-pk.delta, lt.x, lt.y);
        const float t0 = fmaf(static_cast<float>(i0 - pk.j), step, tc);
        const float cg = pk.inten * lt.z, cl = pk.inten * lt.w;
        if (pk.j >= full_lo && pk.j <= full_hi) {  // window covers the whole tile (warp-uniform)
#pragma unroll
            for (int p = 0; p < kFwdP; ++p) {
                const float t = fmaf(static_cast<float>(p), step, t0);
                const float q = t * t;
                acc[p] = fmaf(cg, ex2_approx(-q), acc[p]);
                acc[p] = fmaf(cl, rcp_approx(1.0f + q), acc[p]);
            }
        } else {
#pragma unroll
            for (int p = 0; p < kFwdP; ++p) {
                const int dn = i0 + p - pk.j;
                const bool in = (dn >= -d.n_c) && (dn <= d.n_c);
                const float t = fmaf(static_cast<float>(p), step, t0);
                const float q = t * t;
                const float v = fmaf(cg, ex2_approx(-q), cl * rcp_approx(1.0f + q));
                acc[p] += in ? v : 0.0f;
            }
        }
    }

    // epilogue: residual, e = (y - f)/sigma_n^2, partial sum of ((y - f)/sigma_n)^2
    const int inst = g / d.gpi;
    const int pat = inst / d.R;
    const PatConst pc = d.pat[pat];
    const float* __restrict__ yb = d.yb + static_cast<size_t>(pat) * d.N;
    float ev[kFwdP];
    float ss = 0.0f;
#pragma unroll
    for (int p = 0; p < kFwdP; ++p) {
        const int i = i0 + p;
        float r = 0.0f;
        if (i < d.N) r = yb[i] - acc[p];
        const float z = r * pc.inv_sn;
        ss = fmaf(z, z, ss);
        ev[p] = r * pc.inv_sn2;
    }
    float4* __restrict__ eo = d.e + (static_cast<size_t>(g) * d.NQ + (i0 >> 2)) * 32 + lane;
#pragma unroll
    for (int v = 0; v < kFwdP / 4; ++v)
        if ((i0 >> 2) + v < d.NQ) eo[static_cast<size_t>(v) * 32] = make_float4(ev[4 * v], ev[4 * v + 1], ev[4 * v + 2], ev[4 * v + 3]);
    d.llpart[(static_cast<size_t>(g) * d.ntile + tile) * 32 + lane] = ss;

    if (f_dbg) {  // debug read-back of the profile (parity tests); warp-uniform branch
        const int s = (g - inst * d.gpi) * 32 + lane;
        const long long t = static_cast<long long>(inst) * d.S + s;
        if (s < d.S && t < n_dbg) {
            const float* __restrict__ bg = d.bg + static_cast<size_t>(pat) * d.N;
#pragma unroll
            for (int p = 0; p < kFwdP; ++p)
                if (i0 + p < d.N) f_dbg[t * d.N + i0 + p] = acc[p] + bg[i0 + p];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// a-5: backward six sums.  grid (ceil(n_units/kBwdWarps), G), block 32*kBwdWarps.
// Warp = one unit (a chunk of peaks of one phase) for the 32 draws of group g.  Sums in t' units:
//   B1 = sum e I L, B2 = sum e I G, B3 = sum e I L^2 t', B4 = sum e I G t', B5 = sum e I L^2, B6 = sum e I G t'^2
__global__ void __launch_bounds__(32 * kBwdWarps) backward_kernel(const Dev d) {
    const int lane = threadIdx.x & 31;
    const int unit = blockIdx.x * kBwdWarps + (threadIdx.x >> 5);
    const int g = blockIdx.y;
    if (unit >= d.n_units) return;
    const int4 un = d.units[unit];
    const float4 lt = d.lat[(static_cast<size_t>(g) * d.K + un.x) * 32 + lane];
    const float step = d.delta * lt.x;
    const float4* __restrict__ eg = d.e + static_cast<size_t>(g) * d.NQ * 32 + lane;

    float B1 = 0.f, B2 = 0.f, B3 = 0.f, B4 = 0.f, B5 = 0.f, B6 = 0.f;
    for (int m = un.y; m < un.z; ++m) {
        const PeakRec pk = d.pk_bwd[m];
        const int lo = max(0, pk.j - d.n_c), hi = min(d.N - 1, pk.j + d.n_c);
        const int q0 = lo >> 2, q1 = hi >> 2;
        const float tc = fmaf(-pk.delta, lt.x, lt.y);
        float a1 = 0.f, a2 = 0.f, a3 = 0.f, a4 = 0.f, a5 = 0.f, a6 = 0.f;
        for (int q = q0; q <= q1; ++q) {
            float4 e4 = eg[static_cast<size_t>(q) * 32];
            if (q == q0 || q == q1) {  // ragged ends of the window (warp-uniform)
                const int ib = q * 4;
                if (ib + 0 < lo || ib + 0 > hi) e4.x = 0.f;
                if (ib + 1 < lo || ib + 1 > hi) e4.y = 0.f;
                if (ib + 2 < lo || ib + 2 > hi) e4.z = 0.f;
                if (ib + 3 < lo || ib + 3 > hi) e4.w = 0.f;
            }
            const float tq = fmaf(static_cast<float>(q * 4 - pk.j), step, tc);
            const float ee[4] = {e4.x, e4.y, e4.z, e4.w};
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const float t = fmaf(static_cast<float>(c), step, tq);
                const float qq = t * t;
                const float G = ex2_approx(-qq);
                const float L = rcp_approx(1.0f + qq);
                const float x = ee[c] * L;
                a1 += x;
                const float y = x * L;
                a5 += y;
                a3 = fmaf(y, t, a3);
                const float z = ee[c] * G;
                a2 += z;
                const float zt = z * t;
                a4 += zt;
                a6 = fmaf(zt, t, a6);
            }
        }
        B1 = fmaf(pk.inten, a1, B1);
        B2 = fmaf(pk.inten, a2, B2);
        B3 = fmaf(pk.inten, a3, B3);
        B4 = fmaf(pk.inten, a4, B4);
        B5 = fmaf(pk.inten, a5, B5);
        B6 = fmaf(pk.inten, a6, B6);
    }
    float* __restrict__ so = d.sums + (static_cast<size_t>(g) * d.n_units + unit) * 6 * 32 + lane;
    so[0] = B1; so[32] = B2; so[64] = B3; so[96] = B4; so[128] = B5; so[160] = B6;
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

// a-6 + a-7: chain rule, prior/Jacobian gradient, mean over the S draws.
// grid (K, PR), block 128: threads stride over the draws of instance inst for phase k.
constexpr int kChainThreads = 128;
__global__ void __launch_bounds__(kChainThreads) chain_reduce_kernel(const Dev d, const float* __restrict__ var) {
    __shared__ double red[(kChainThreads / 32) * 9];
    const int k = blockIdx.x, inst = blockIdx.y;
    const int pat = inst / d.R;
    const PatConst pc = d.pat[pat];
    const float4 m = *reinterpret_cast<const float4*>(var + (static_cast<size_t>(inst) * 2 * d.K + k) * 4);
    const float4 l = *reinterpret_cast<const float4*>(var + (static_cast<size_t>(inst) * 2 * d.K + d.K + k) * 4);
    const float sg[4] = {expf(l.x), expf(l.y), expf(l.z), expf(l.w)};
    const int u0 = d.unit_ofs[k], u1 = d.unit_ofs[k + 1];
    double v[9];
#pragma unroll
    for (int i = 0; i < 9; ++i) v[i] = 0.0;

    for (int s = threadIdx.x; s < d.S; s += kChainThreads) {
        const int g = inst * d.gpi + (s >> 5), lane = s & 31;
        float B[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        for (int u = u0; u < u1; ++u) {
            const float* __restrict__ sp = d.sums + (static_cast<size_t>(g) * d.n_units + u) * 6 * 32 + lane;
#pragma unroll
            for (int c = 0; c < 6; ++c) B[c] += sp[c * 32];
        }
        const float4 ep = d.eps[(static_cast<size_t>(g) * d.K + k) * 32 + lane];
        const Phys q = transform(m, l, ep);
        const float iw = 1.0f / q.w;
        const float cLp = q.r * kAL * iw, cGp = (1.0f - q.r) * kAG * iw;
        const float dh = cLp * B[0] + cGp * B[1];
        const float dr = q.h * iw * (kAL * B[0] - kAG * B[1]);
        const float dmu = q.h * iw * (4.0f * cLp * B[2] + 4.0f * kLn2 * cGp * B[3]);
        const float dw = -q.h * iw * (cLp * (2.0f * B[4] - B[0]) + cGp * (B[1] - 2.0f * kLn2 * B[5]));
        const float gz[4] = {fmaf(dh, q.h, 1.0f - pc.lambda_h * q.h),
                             dmu - q.mu * d.mu_inv_var,
                             fmaf(dw, q.w, d.w_shape - d.w_rate * q.w),
                             fmaf(dr, q.r * (1.0f - q.r), 1.0f - 2.0f * q.r)};
        const float az = fabsf(q.zr);
        const float lp = (pc.log_lambda_h - pc.lambda_h * q.h + q.zh)
                       + (-0.5f * q.mu * q.mu * d.mu_inv_var + d.mu_logc)
                       + (d.w_logc + d.w_shape * q.zw - d.w_rate * q.w)
                       - (az + 2.0f * log1pf(expf(-az)));
        const float e4[4] = {ep.x, ep.y, ep.z, ep.w};
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            v[c] += static_cast<double>(gz[c]);
            v[4 + c] += static_cast<double>(gz[c] * e4[c] * sg[c]);
        }
        v[8] += static_cast<double>(lp);
    }
    block_reduce<9, kChainThreads / 32>(v, red);
    if (threadIdx.x < 4) {
        const double inv_s = 1.0 / static_cast<double>(d.S);
        const int c = threadIdx.x;
        d.grad[(static_cast<size_t>(inst) * 2 * d.K + k) * 4 + c] = static_cast<float>(v[c] * inv_s);
        d.grad[(static_cast<size_t>(inst) * 2 * d.K + d.K + k) * 4 + c] = static_cast<float>(v[4 + c] * inv_s + 1.0);
        if (c == 0) d.elbo_k[static_cast<size_t>(inst) * d.K + k] = v[8] * inv_s;
    }
}

// a-7 (ELBO) + a-8 (Adam ascent).  grid PR, block 256.
constexpr int kFinThreads = 256;
__global__ void __launch_bounds__(kFinThreads) finalize_update_kernel(const Dev d, const float* __restrict__ var_in,
                                                                      int do_update) {
    __shared__ double red[(kFinThreads / 32) * 1];
    const int inst = blockIdx.x;
    const int pat = inst / d.R;
    const PatConst pc = d.pat[pat];
    double v[1] = {0.0};
    for (int s = threadIdx.x; s < d.S; s += kFinThreads) {
        const int g = inst * d.gpi + (s >> 5), lane = s & 31;
        const float* __restrict__ lp = d.llpart + static_cast<size_t>(g) * d.ntile * 32 + lane;
        double a = 0.0;
        for (int t = 0; t < d.ntile; ++t) a += static_cast<double>(lp[static_cast<size_t>(t) * 32]);
        const double ll = -0.5 * a + pc.ll_const;
        d.ll_t[static_cast<size_t>(inst) * d.gpi * 32 + s] = ll;
        v[0] += ll;
    }
    block_reduce<1, kFinThreads / 32>(v, red);
    const long long step = d.ctl->step + 1;
    if (threadIdx.x == 0) {
        double el = v[0] / static_cast<double>(d.S);
        for (int k = 0; k < d.K; ++k) el += d.elbo_k[static_cast<size_t>(inst) * d.K + k];
        const float* l = var_in + (static_cast<size_t>(inst) * 2 * d.K + d.K) * 4;
        double ent = 0.0;
        for (int j = 0; j < 4 * d.K; ++j) ent += static_cast<double>(l[j]) + 1.4189385332046727;  // 1/2 ln(2 pi e)
        el += ent;
        d.elbo[inst] = el;
        if (do_update) {
            const long long row = step - 1 - d.ctl->trace_base;
            if (row >= 0) d.trace[static_cast<size_t>(row % kTraceCap) * d.PR + inst] = el;
        }
    }
    if (!do_update) return;
    __syncthreads();  // thread 0 has read l for the entropy before anyone overwrites it
    const float bc1 = 1.0f - powf(d.beta1, static_cast<float>(step));
    const float bc2 = 1.0f - powf(d.beta2, static_cast<float>(step));
    const int per = 8 * d.K;
    for (int j = threadIdx.x; j < per; j += kFinThreads) {
        const size_t o = static_cast<size_t>(inst) * per + j;
        const float gj = d.grad[o];
        const float m1 = d.beta1 * d.mom1[o] + (1.0f - d.beta1) * gj;
        const float m2 = d.beta2 * d.mom2[o] + (1.0f - d.beta2) * gj * gj;
        d.mom1[o] = m1;
        d.mom2[o] = m2;
        float x = d.var[o] + d.lr * (m1 / bc1) / (sqrtf(m2 / bc2) + d.adam_eps);
        if (j >= per / 2) x = fminf(fmaxf(x, -12.0f), 2.0f);
        d.var[o] = x;
    }
}

__global__ void bump_step_kernel(Ctl* ctl) { ctl->step += 1; }

// a-10: inclusion probability and area ratio (R15), fp64.  grid PR, block 128.
__global__ void __launch_bounds__(128) inclusion_kernel(const Dev d, double tau, double* __restrict__ incl,
                                                        double* __restrict__ ratio) {
    __shared__ double red[4];
    const int inst = blockIdx.x;
    const float* m = d.var + static_cast<size_t>(inst) * 8 * d.K;
    const float* l = m + 4 * d.K;
    double v[1] = {0.0};
    for (int k = threadIdx.x; k < d.K; k += 128) {
        const double s = exp(static_cast<double>(l[4 * k]));
        v[0] += d.area[k] * exp(static_cast<double>(m[4 * k]) + 0.5 * s * s);
    }
    block_reduce<1, 4>(v, red);
    const double tbar = v[0];
    for (int k = threadIdx.x; k < d.K; k += 128) {
        const double s = exp(static_cast<double>(l[4 * k]));
        const double z = (static_cast<double>(m[4 * k]) - log(tau * tbar / d.area[k])) / s;
        incl[static_cast<size_t>(inst) * d.K + k] = 0.5 * erfc(-z * 0.70710678118654752440);
        ratio[static_cast<size_t>(inst) * d.K + k] = d.area[k] * exp(static_cast<double>(m[4 * k]) + 0.5 * s * s) / tbar;
    }
}

// R11 initial state.  grid PR, block 128 over phases.
__global__ void __launch_bounds__(128) init_state_kernel(const Dev d, const float* __restrict__ m_h0 /*[P]*/,
                                                         float m_w0, float init_log_sigma, unsigned long long seed) {
    const int inst = blockIdx.x;
    const int pat = inst / d.R, rst = inst - pat * d.R;
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
    }
    const int per = 8 * d.K;
    for (int j = threadIdx.x; j < per; j += 128) {
        d.mom1[static_cast<size_t>(inst) * per + j] = 0.0f;
        d.mom2[static_cast<size_t>(inst) * per + j] = 0.0f;
    }
}

}  // namespace xrdvi_dev
