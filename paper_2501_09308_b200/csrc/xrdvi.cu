// xrdvi.cu -- C ABI (include/xrdvi.h), host preprocessing in fp64, launch logic and CUDA Graph.
// There is no CPU fallback anywhere in this file: every compute step is a kernel in
// xrdvi_kernels.cuh; the host only validates, sorts and encodes the static tables at create.
#include "../../include/xrdvi.h"
#include "xrdvi_kernels.cuh"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <limits>
#include <string>
#include <vector>

using namespace xrdvi_dev;

namespace {

thread_local std::string g_err;

int fail(int code, const std::string& msg) {
    g_err = msg;
    return code;
}

#define CU(call)                                                                                     \
    do {                                                                                             \
        cudaError_t e_ = (call);                                                                     \
        if (e_ != cudaSuccess)                                                                       \
            return fail(XRDVI_E_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_));          \
    } while (0)

size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

struct Plan {   // workspace carve; identical arithmetic in workspace_bytes and create
    int P, R, PR, S_pad, gpi_max, G_max, NQ, ntile, K;
    int unit_peaks;    // target peaks per backward unit
    int units_cap;     // upper bound on the number of units
    long long M;
    size_t total;
    size_t o_yb, o_bg, o_pkf, o_tile, o_pkb, o_units, o_uofs, o_pat, o_area, o_mh0;
    size_t o_var, o_vartmp, o_mom1, o_mom2, o_grad, o_elbo, o_elbok, o_llt, o_trace, o_ctl;
    size_t o_lat, o_eps, o_e, o_llpart, o_sums, o_dbg;
};

bool make_plan(int64_t N, int32_t K, int64_t M, int32_t S_max, const xrdvi_hyper* hyp, Plan* pl) {
    if (N < 2 || K < 1 || M < 1 || S_max < 1 || !hyp) return false;
    if (N > (1 << 28) || M > (1ll << 30) || K > (1 << 24)) return false;
    Plan p{};
    p.P = std::max(1, hyp->n_patterns);
    p.R = std::max(1, hyp->n_restarts);
    p.PR = p.P * p.R;
    p.K = K;
    p.M = M;
    p.S_pad = (S_max + 31) / 32 * 32;
    p.gpi_max = p.S_pad / 32;
    p.G_max = p.PR * p.gpi_max;
    if (p.G_max > 65535 || p.PR > 65535) return false;  // grid.y limit
    p.NQ = static_cast<int>((N + 3) / 4);
    p.ntile = static_cast<int>((N + kFwdP - 1) / kFwdP);
    // backward units: enough warps to fill 148 SMs x 16 warps, at least one unit per phase
    const long long want = std::max<long long>(K, (148ll * 16 + p.G_max - 1) / p.G_max);
    p.unit_peaks = static_cast<int>(std::max<long long>(4, (M + want - 1) / want));
    p.units_cap = static_cast<int>(M / p.unit_peaks + K + 1);
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t r = o; o = align_up(o + bytes); return r; };
    const size_t var_b = sizeof(float) * p.PR * 8 * static_cast<size_t>(K);
    p.o_yb = take(sizeof(float) * p.P * N);
    p.o_bg = take(sizeof(float) * p.P * N);
    p.o_pkf = take(sizeof(PeakRec) * M);
    p.o_tile = take(sizeof(int2) * p.ntile);
    p.o_pkb = take(sizeof(PeakRec) * M);
    p.o_units = take(sizeof(int4) * p.units_cap);
    p.o_uofs = take(sizeof(int) * (K + 1));
    p.o_pat = take(sizeof(PatConst) * p.P);
    p.o_area = take(sizeof(double) * K);
    p.o_mh0 = take(sizeof(float) * p.P);
    p.o_var = take(var_b);
    p.o_vartmp = take(var_b);
    p.o_mom1 = take(var_b);
    p.o_mom2 = take(var_b);
    p.o_grad = take(var_b);
    p.o_elbo = take(sizeof(double) * p.PR);
    p.o_elbok = take(sizeof(double) * p.PR * K);
    p.o_llt = take(sizeof(double) * p.PR * p.S_pad);
    p.o_trace = take(sizeof(double) * kTraceCap * p.PR);
    p.o_ctl = take(sizeof(Ctl));
    p.o_lat = take(sizeof(float4) * static_cast<size_t>(p.G_max) * K * 32);
    p.o_eps = take(sizeof(float4) * static_cast<size_t>(p.G_max) * K * 32);
    p.o_e = take(sizeof(float4) * static_cast<size_t>(p.G_max) * p.NQ * 32);
    p.o_llpart = take(sizeof(float) * static_cast<size_t>(p.G_max) * p.ntile * 32);
    p.o_sums = take(sizeof(float) * static_cast<size_t>(p.G_max) * p.units_cap * 6 * 32);
    p.o_dbg = take(sizeof(double) * (2 * static_cast<size_t>(p.PR) * K + 64));
    p.total = o;
    *pl = p;
    return true;
}

}  // namespace

struct xrdvi {
    Plan plan{};
    Dev dev{};
    xrdvi_hyper hyp{};
    int device = 0;
    cudaStream_t stream = nullptr;
    char* ws = nullptr;
    int64_t N = 0, M = 0, pairs = 0;
    int K = 0;
    int n_c = 0;
    std::vector<float> m_h0;   // per pattern initial m_h
    float m_w0 = 0.f;
    long long step_host = 0;   // mirror of ctl.step
    // CUDA Graph of one optimisation step, keyed by S
    cudaGraphExec_t graph_exec = nullptr;
    int graph_S = -1;
    cudaEvent_t ev[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
};

namespace {

void set_S(xrdvi* h, int S) {
    h->dev.S = S;
    h->dev.gpi = (S + 31) / 32;
    h->dev.G = h->plan.PR * h->dev.gpi;
}

// enqueue the kernels of one evaluation (and optionally the Adam update) on the stream
int enqueue_iteration(xrdvi* h, const float* var, int do_update, float* f_dbg, long long n_dbg,
                      uint4* raw_out, bool forward_only) {
    const Dev& d = h->dev;
    cudaStream_t st = h->stream;
    draw_transform_kernel<<<dim3((d.K + 3) / 4, d.G), 128, 0, st>>>(d, var, raw_out);
    forward_kernel<<<dim3((d.ntile + kFwdWarps - 1) / kFwdWarps, d.G), 32 * kFwdWarps, 0, st>>>(d, f_dbg, n_dbg);
    if (!forward_only) {
        backward_kernel<<<dim3((d.n_units + kBwdWarps - 1) / kBwdWarps, d.G), 32 * kBwdWarps, 0, st>>>(d);
        chain_reduce_kernel<<<dim3(d.K, d.PR), kChainThreads, 0, st>>>(d, var);
    }
    finalize_update_kernel<<<d.PR, kFinThreads, 0, st>>>(d, var, do_update);
    if (do_update) bump_step_kernel<<<1, 1, 0, st>>>(d.ctl);
    CU(cudaGetLastError());
    return XRDVI_OK;
}

int write_ctl(xrdvi* h, uint64_t seed, long long step, long long trace_base, long long it_override) {
    Ctl c;
    c.seed = seed;
    c.step = step;
    c.trace_base = trace_base;
    c.iteration_override = it_override;
    CU(cudaMemcpyAsync(h->dev.ctl, &c, sizeof(Ctl), cudaMemcpyHostToDevice, h->stream));
    CU(cudaStreamSynchronize(h->stream));  // c lives on this stack frame
    return XRDVI_OK;
}

int check_S(xrdvi* h, int32_t S) {
    if (!h) return fail(XRDVI_E_INVALID_ARG, "null handle");
    if (S < 1 || S > h->plan.S_pad) return fail(XRDVI_E_INVALID_ARG, "S out of range [1, S_max]");
    return XRDVI_OK;
}

int ensure_graph(xrdvi* h, int S) {
    if (h->graph_exec && h->graph_S == S) return XRDVI_OK;
    if (h->graph_exec) { cudaGraphExecDestroy(h->graph_exec); h->graph_exec = nullptr; }
    set_S(h, S);
    cudaGraph_t graph = nullptr;
    CU(cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal));
    int rc = enqueue_iteration(h, h->dev.var, 1, nullptr, 0, nullptr, false);
    cudaError_t e = cudaStreamEndCapture(h->stream, &graph);
    if (rc != XRDVI_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
    if (e != cudaSuccess) return fail(XRDVI_E_CUDA, std::string("cudaStreamEndCapture: ") + cudaGetErrorString(e));
    e = cudaGraphInstantiate(&h->graph_exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) return fail(XRDVI_E_CUDA, std::string("cudaGraphInstantiate: ") + cudaGetErrorString(e));
    h->graph_S = S;
    return XRDVI_OK;
}

}  // namespace

extern "C" {

const char* xrdvi_last_error(void) { return g_err.c_str(); }

void xrdvi_default_hyper(xrdvi_hyper* hy) {
    if (!hy) return;
    std::memset(hy, 0, sizeof(*hy));
    hy->size = sizeof(xrdvi_hyper);
    hy->lambda_h = 0.0;
    hy->mu_sigma = 0.03;
    hy->w_shape = 3.0;
    hy->w_rate = 100.0;
    hy->noise_sigma = 0.0;
    hy->window_W = 10.0;
    hy->fwhm_ref = 0.15;
    hy->incl_tau = 0.01;
    hy->lr = 0.1;
    hy->beta1 = 0.9;
    hy->beta2 = 0.999;
    hy->adam_eps = 1e-8;
    hy->init_log_sigma = std::log(0.1);
    hy->n_patterns = 1;
    hy->n_restarts = 1;
    hy->likelihood = 0;
}

size_t xrdvi_workspace_bytes(int64_t N, int32_t K, int64_t M, int32_t S_max, const xrdvi_hyper* hyp) {
    Plan pl;
    if (!hyp || hyp->size != sizeof(xrdvi_hyper)) return 0;
    if (!make_plan(N, K, M, S_max, hyp, &pl)) return 0;
    return pl.total;
}

int xrdvi_create(const double* x, int64_t N, const double* y, const double* bgin, int32_t K,
                 const int64_t* ofs, const double* pos, const double* inten, const xrdvi_hyper* hyp,
                 int32_t S_max, int device, void* cuda_stream, void* workspace, size_t workspace_bytes,
                 xrdvi** out) {
    if (!x || !y || !ofs || !pos || !inten || !hyp || !out || !workspace)
        return fail(XRDVI_E_INVALID_ARG, "null argument");
    if (hyp->size != sizeof(xrdvi_hyper)) return fail(XRDVI_E_INVALID_ARG, "xrdvi_hyper.size mismatch");
    if (hyp->likelihood != 0) return fail(XRDVI_E_INVALID_ARG, "only the Gaussian likelihood (0) is built");
    if (N < 2 || K < 1 || S_max < 1) return fail(XRDVI_E_INVALID_ARG, "N >= 2, K >= 1, S_max >= 1 required");
    if (hyp->n_patterns < 1 || hyp->n_restarts < 1) return fail(XRDVI_E_INVALID_ARG, "P, R >= 1 required");
    if (!(hyp->mu_sigma > 0) || !(hyp->w_shape > 0) || !(hyp->w_rate > 0) || !(hyp->fwhm_ref > 0) ||
        !(hyp->incl_tau > 0) || !(hyp->lr > 0))
        return fail(XRDVI_E_INVALID_ARG, "non-positive hyper-parameter");
    if (ofs[0] != 0) return fail(XRDVI_E_INVALID_ARG, "peak_ofs[0] != 0");
    for (int k = 0; k < K; ++k) {
        if (ofs[k + 1] < ofs[k]) return fail(XRDVI_E_INVALID_ARG, "peak_ofs not non-decreasing");
        if (ofs[k + 1] == ofs[k]) return fail(XRDVI_E_EMPTY_PHASE, "phase " + std::to_string(k) + " has no peaks");
    }
    const int64_t M = ofs[K];
    for (int64_t i = 1; i < N; ++i)
        if (!(x[i] > x[i - 1])) return fail(XRDVI_E_UNSORTED_GRID, "two_theta not strictly increasing");
    const double delta = (x[N - 1] - x[0]) / static_cast<double>(N - 1);
    for (int64_t i = 0; i < N; ++i)
        if (std::fabs(x[i] - (x[0] + delta * static_cast<double>(i))) > 1e-6 * delta)
            return fail(XRDVI_E_NONUNIFORM_GRID, "two_theta is not a uniform grid (this build needs one)");
    for (int64_t m = 0; m < M; ++m)
        if (!std::isfinite(pos[m]) || !std::isfinite(inten[m]) || inten[m] < 0.0)
            return fail(XRDVI_E_INVALID_ARG, "peak position/intensity not finite or negative intensity");

    int dev_count = 0;
    CU(cudaGetDeviceCount(&dev_count));
    if (device < 0 || device >= dev_count) return fail(XRDVI_E_CUDA, "no such CUDA device");
    cudaDeviceProp prop;
    CU(cudaGetDeviceProperties(&prop, device));
    if (prop.major != 10) return fail(XRDVI_E_NOT_SM100, "device is not compute capability 10.x (sm_100a build)");
    CU(cudaSetDevice(device));

    Plan pl;
    if (!make_plan(N, K, M, S_max, hyp, &pl)) return fail(XRDVI_E_INVALID_ARG, "sizes out of range");
    if (workspace_bytes < pl.total) return fail(XRDVI_E_WORKSPACE_TOO_SMALL, "workspace too small: need " + std::to_string(pl.total));
    if (reinterpret_cast<uintptr_t>(workspace) % 256) return fail(XRDVI_E_INVALID_ARG, "workspace not 256-byte aligned");

    // ---- fp64 preprocessing (R16) ----------------------------------------------------------------
    const int P = pl.P;
    long long n_c;
    if (hyp->window_W > 0.0) n_c = static_cast<long long>(std::ceil(hyp->window_W * hyp->fwhm_ref / delta - 1e-9));
    else {         // dense: every point is inside every window, wherever the peak lies
        n_c = N;
        for (int64_t m = 0; m < M; ++m) {
            const long long j = static_cast<long long>(std::floor((pos[m] - x[0]) / delta + 0.5));
            n_c = std::max<long long>(n_c, std::max<long long>(std::llabs(j), std::llabs(N - 1 - j)) + 1);
        }
    }
    if (n_c > (1ll << 30)) return fail(XRDVI_E_INVALID_ARG, "peak positions too far from the grid");
    struct HP { long long j; double d; double I; int k; };
    std::vector<HP> kept;
    kept.reserve(M);
    std::vector<double> area(K, 0.0);
    double imax = 0.0;
    long long pairs = 0;
    for (int k = 0; k < K; ++k)
        for (int64_t m = ofs[k]; m < ofs[k + 1]; ++m) {
            area[k] += inten[m];
            imax = std::max(imax, inten[m]);
            const long long j = static_cast<long long>(std::floor((pos[m] - x[0]) / delta + 0.5));
            const long long lo = std::max<long long>(0, j - n_c), hi = std::min<long long>(N - 1, j + n_c);
            if (lo > hi) continue;  // no in-range grid point
            pairs += hi - lo + 1;
            const double xj = (j >= 0 && j < N) ? x[j] : x[0] + delta * static_cast<double>(j);
            kept.push_back({j, pos[m] - xj, inten[m], k});
        }
    const int Mv = static_cast<int>(kept.size());
    for (int k = 0; k < K; ++k)
        if (!(area[k] > 0.0)) return fail(XRDVI_E_EMPTY_PHASE, "phase " + std::to_string(k) + " has zero total intensity");

    // forward table: sorted by j (stable in (j, k, original order)); tile ranges by binary search
    std::vector<HP> fw = kept;
    std::stable_sort(fw.begin(), fw.end(), [](const HP& a, const HP& b) { return a.j < b.j; });
    std::vector<PeakRec> pk_fwd(std::max(Mv, 1)), pk_bwd(std::max(Mv, 1));
    for (int m = 0; m < Mv; ++m)
        pk_fwd[m] = {static_cast<int>(fw[m].j), static_cast<float>(fw[m].d), static_cast<float>(fw[m].I), fw[m].k};
    std::vector<int2> tile_rng(pl.ntile);
    for (int t = 0; t < pl.ntile; ++t) {
        const long long i0 = static_cast<long long>(t) * kFwdP;
        const long long jlo = i0 - n_c, jhi = i0 + kFwdP - 1 + n_c;
        auto a = std::lower_bound(fw.begin(), fw.end(), jlo, [](const HP& p, long long v) { return p.j < v; });
        auto b = std::upper_bound(fw.begin(), fw.end(), jhi, [](long long v, const HP& p) { return v < p.j; });
        tile_rng[t] = make_int2(static_cast<int>(a - fw.begin()), static_cast<int>(b - fw.begin()));
    }
    // backward table: phase-major (kept is already phase-major), split into units of ~unit_peaks peaks
    std::vector<int4> units;
    std::vector<int> unit_ofs(K + 1, 0);
    {
        int m = 0;
        for (int k = 0; k < K; ++k) {
            int m_end = m;
            while (m_end < Mv && kept[m_end].k == k) ++m_end;
            const int cnt = m_end - m;
            unit_ofs[k] = static_cast<int>(units.size());
            if (cnt > 0) {
                const int nu = (cnt + pl.unit_peaks - 1) / pl.unit_peaks;
                for (int u = 0; u < nu; ++u) {
                    const int a = m + static_cast<int>(static_cast<long long>(cnt) * u / nu);
                    const int b = m + static_cast<int>(static_cast<long long>(cnt) * (u + 1) / nu);
                    units.push_back(make_int4(k, a, b, 0));
                }
            }
            m = m_end;
        }
        unit_ofs[K] = static_cast<int>(units.size());
        for (int q = 0; q < Mv; ++q)
            pk_bwd[q] = {static_cast<int>(kept[q].j), static_cast<float>(kept[q].d), static_cast<float>(kept[q].I), kept[q].k};
    }
    if (static_cast<int>(units.size()) > pl.units_cap) return fail(XRDVI_E_INVALID_ARG, "internal: unit bound exceeded");
    if (units.empty()) units.push_back(make_int4(0, 0, 0, 0));

    // observed data and per-pattern constants
    std::vector<float> yb(static_cast<size_t>(P) * N), bgf(static_cast<size_t>(P) * N);
    std::vector<PatConst> pat(P);
    std::vector<float> m_h0(P);
    for (int p = 0; p < P; ++p) {
        double smax = -std::numeric_limits<double>::infinity();
        for (int64_t i = 0; i < N; ++i) {
            const double b = bgin ? bgin[p * N + i] : 0.0;
            const double v = y[p * N + i] - b;
            if (!std::isfinite(v)) return fail(XRDVI_E_INVALID_ARG, "non-finite observation");
            smax = std::max(smax, v);
            yb[p * N + i] = static_cast<float>(v);
            bgf[p * N + i] = static_cast<float>(b);
        }
        const double sn = hyp->noise_sigma > 0.0 ? hyp->noise_sigma : 0.01 * smax;           // R4
        const double eta_h = smax * hyp->fwhm_ref / (imax > 0.0 ? imax : 1.0);               // R13
        const double lam = hyp->lambda_h > 0.0 ? hyp->lambda_h : 1.0 / eta_h;
        if (!(sn > 0.0) || !(lam > 0.0) || !(eta_h > 0.0))
            return fail(XRDVI_E_INVALID_ARG, "auto noise_sigma / lambda_h needs max(y - B) > 0");
        pat[p].inv_sn = static_cast<float>(1.0 / sn);
        pat[p].inv_sn2 = static_cast<float>(1.0 / (sn * sn));
        pat[p].lambda_h = static_cast<float>(lam);
        pat[p].log_lambda_h = static_cast<float>(std::log(lam));
        pat[p].ll_const = -static_cast<double>(N) * std::log(sn) - 0.5 * static_cast<double>(N) * std::log(2.0 * M_PI);
        m_h0[p] = static_cast<float>(std::log(eta_h / static_cast<double>(K)));               // R11
    }

    // ---- handle + upload -------------------------------------------------------------------------
    xrdvi* h = new xrdvi();
    h->plan = pl;
    h->hyp = *hyp;
    h->device = device;
    h->stream = static_cast<cudaStream_t>(cuda_stream);
    h->ws = static_cast<char*>(workspace);
    h->N = N; h->M = M; h->K = K; h->pairs = pairs; h->n_c = static_cast<int>(n_c);
    h->m_h0 = m_h0;
    h->m_w0 = static_cast<float>(std::log(hyp->w_shape / hyp->w_rate));
    Dev& d = h->dev;
    char* w = h->ws;
    d.N = static_cast<int>(N); d.NQ = pl.NQ; d.K = K; d.P = pl.P; d.R = pl.R; d.PR = pl.PR;
    d.n_c = static_cast<int>(n_c); d.ntile = pl.ntile; d.n_units = static_cast<int>(units.size()); d.Mv = Mv;
    d.delta = static_cast<float>(delta);
    d.mu_inv_var = static_cast<float>(1.0 / (hyp->mu_sigma * hyp->mu_sigma));
    d.mu_logc = static_cast<float>(-std::log(hyp->mu_sigma * std::sqrt(2.0 * M_PI)));
    d.w_shape = static_cast<float>(hyp->w_shape);
    d.w_rate = static_cast<float>(hyp->w_rate);
    d.w_logc = static_cast<float>(hyp->w_shape * std::log(hyp->w_rate) - std::lgamma(hyp->w_shape));
    d.lr = static_cast<float>(hyp->lr); d.beta1 = static_cast<float>(hyp->beta1);
    d.beta2 = static_cast<float>(hyp->beta2); d.adam_eps = static_cast<float>(hyp->adam_eps);
    d.yb = reinterpret_cast<float*>(w + pl.o_yb);
    d.bg = reinterpret_cast<float*>(w + pl.o_bg);
    d.pk_fwd = reinterpret_cast<PeakRec*>(w + pl.o_pkf);
    d.tile_rng = reinterpret_cast<int2*>(w + pl.o_tile);
    d.pk_bwd = reinterpret_cast<PeakRec*>(w + pl.o_pkb);
    d.units = reinterpret_cast<int4*>(w + pl.o_units);
    d.unit_ofs = reinterpret_cast<int*>(w + pl.o_uofs);
    d.pat = reinterpret_cast<PatConst*>(w + pl.o_pat);
    d.area = reinterpret_cast<double*>(w + pl.o_area);
    d.var = reinterpret_cast<float*>(w + pl.o_var);
    d.mom1 = reinterpret_cast<float*>(w + pl.o_mom1);
    d.mom2 = reinterpret_cast<float*>(w + pl.o_mom2);
    d.grad = reinterpret_cast<float*>(w + pl.o_grad);
    d.elbo = reinterpret_cast<double*>(w + pl.o_elbo);
    d.elbo_k = reinterpret_cast<double*>(w + pl.o_elbok);
    d.ll_t = reinterpret_cast<double*>(w + pl.o_llt);
    d.trace = reinterpret_cast<double*>(w + pl.o_trace);
    d.ctl = reinterpret_cast<Ctl*>(w + pl.o_ctl);
    d.lat = reinterpret_cast<float4*>(w + pl.o_lat);
    d.eps = reinterpret_cast<float4*>(w + pl.o_eps);
    d.e = reinterpret_cast<float4*>(w + pl.o_e);
    d.llpart = reinterpret_cast<float*>(w + pl.o_llpart);
    d.sums = reinterpret_cast<float*>(w + pl.o_sums);
    set_S(h, S_max);

    cudaStream_t st = h->stream;
    auto up = [&](size_t off, const void* src, size_t bytes) {
        return cudaMemcpyAsync(w + off, src, bytes, cudaMemcpyHostToDevice, st);
    };
    cudaError_t ce = cudaSuccess;
    auto chk = [&](cudaError_t e) { if (ce == cudaSuccess) ce = e; };
    chk(up(pl.o_yb, yb.data(), sizeof(float) * yb.size()));
    chk(up(pl.o_bg, bgf.data(), sizeof(float) * bgf.size()));
    chk(up(pl.o_pkf, pk_fwd.data(), sizeof(PeakRec) * std::max(Mv, 1)));
    chk(up(pl.o_tile, tile_rng.data(), sizeof(int2) * tile_rng.size()));
    chk(up(pl.o_pkb, pk_bwd.data(), sizeof(PeakRec) * std::max(Mv, 1)));
    chk(up(pl.o_units, units.data(), sizeof(int4) * units.size()));
    chk(up(pl.o_uofs, unit_ofs.data(), sizeof(int) * unit_ofs.size()));
    chk(up(pl.o_pat, pat.data(), sizeof(PatConst) * pat.size()));
    chk(up(pl.o_area, area.data(), sizeof(double) * area.size()));
    chk(up(pl.o_mh0, m_h0.data(), sizeof(float) * m_h0.size()));
    chk(cudaMemsetAsync(w + pl.o_trace, 0xFF, sizeof(double) * kTraceCap * pl.PR, st));
    chk(cudaStreamSynchronize(st));  // host staging vectors go out of scope below
    for (auto& e : h->ev) chk(cudaEventCreate(&e));
    if (ce != cudaSuccess) {
        delete h;
        return fail(XRDVI_E_CUDA, std::string("upload: ") + cudaGetErrorString(ce));
    }
    int rc = xrdvi_reset_state(h, 0);
    if (rc != XRDVI_OK) { xrdvi_destroy(h); return rc; }
    *out = h;
    return XRDVI_OK;
}

void xrdvi_destroy(xrdvi* h) {
    if (!h) return;
    if (h->graph_exec) cudaGraphExecDestroy(h->graph_exec);
    for (auto& e : h->ev) if (e) cudaEventDestroy(e);
    delete h;
}

int64_t xrdvi_pair_count(const xrdvi* h) { return h ? h->pairs : -1; }
int64_t xrdvi_window_halfwidth(const xrdvi* h) { return h ? h->n_c : -1; }

int xrdvi_reset_state(xrdvi* h, uint64_t seed) {
    if (!h) return fail(XRDVI_E_INVALID_ARG, "null handle");
    CU(cudaSetDevice(h->device));
    init_state_kernel<<<h->plan.PR, 128, 0, h->stream>>>(h->dev, reinterpret_cast<const float*>(h->ws + h->plan.o_mh0),
                                                          h->m_w0, static_cast<float>(h->hyp.init_log_sigma), seed);
    CU(cudaGetLastError());
    h->step_host = 0;
    return write_ctl(h, 0, 0, 0, -1);
}

int xrdvi_get_state(xrdvi* h, float* var_params, int64_t* step) {
    if (!h) return fail(XRDVI_E_INVALID_ARG, "null handle");
    CU(cudaSetDevice(h->device));
    if (var_params) {
        CU(cudaMemcpyAsync(var_params, h->dev.var, sizeof(float) * h->plan.PR * 8 * h->K, cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
    }
    if (step) *step = h->step_host;
    return XRDVI_OK;
}

int xrdvi_set_state(xrdvi* h, const float* var_params, int64_t step) {
    if (!h || !var_params || step < 0) return fail(XRDVI_E_INVALID_ARG, "null handle/state or negative step");
    CU(cudaSetDevice(h->device));
    const size_t b = sizeof(float) * h->plan.PR * 8 * h->K;
    CU(cudaMemcpyAsync(h->dev.var, var_params, b, cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemsetAsync(h->dev.mom1, 0, b, h->stream));
    CU(cudaMemsetAsync(h->dev.mom2, 0, b, h->stream));
    h->step_host = step;
    return write_ctl(h, 0, step, step, -1);
}

int xrdvi_elbo_grad(xrdvi* h, const float* var_params, int32_t S, uint64_t seed, uint64_t iteration,
                    double* elbo, float* grad) {
    int rc = check_S(h, S);
    if (rc) return rc;
    CU(cudaSetDevice(h->device));
    const size_t b = sizeof(float) * h->plan.PR * 8 * h->K;
    const float* var = h->dev.var;
    if (var_params) {
        float* tmp = reinterpret_cast<float*>(h->ws + h->plan.o_vartmp);
        CU(cudaMemcpyAsync(tmp, var_params, b, cudaMemcpyHostToDevice, h->stream));
        var = tmp;
    }
    set_S(h, S);
    rc = write_ctl(h, seed, h->step_host, h->step_host, static_cast<long long>(iteration & 0xFFFFFFFFull));
    if (rc) return rc;
    rc = enqueue_iteration(h, var, 0, nullptr, 0, nullptr, false);
    if (rc) return rc;
    std::vector<double> el(elbo ? h->plan.PR : 0);
    std::vector<float> gr(grad ? h->plan.PR * 8 * static_cast<size_t>(h->K) : 0);
    if (elbo) CU(cudaMemcpyAsync(el.data(), h->dev.elbo, sizeof(double) * h->plan.PR, cudaMemcpyDeviceToHost, h->stream));
    if (grad) CU(cudaMemcpyAsync(gr.data(), h->dev.grad, b, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    if (elbo) std::memcpy(elbo, el.data(), sizeof(double) * el.size());
    if (grad) std::memcpy(grad, gr.data(), b);
    return XRDVI_OK;
}

int xrdvi_fit(xrdvi* h, int32_t iterations, int32_t S, uint64_t seed, float* var_out, double* incl, double* trace) {
    int rc = check_S(h, S);
    if (rc) return rc;
    if (iterations < 0) return fail(XRDVI_E_INVALID_ARG, "iterations < 0");
    CU(cudaSetDevice(h->device));
    rc = ensure_graph(h, S);
    if (rc) return rc;
    set_S(h, S);
    const long long step0 = h->step_host;
    rc = write_ctl(h, seed, step0, step0, -1);
    if (rc) return rc;
    for (int it = 0; it < iterations; ++it) CU(cudaGraphLaunch(h->graph_exec, h->stream));
    h->step_host = step0 + iterations;
    const int PR = h->plan.PR;
    std::vector<float> vo(var_out ? PR * 8 * static_cast<size_t>(h->K) : 0);
    std::vector<double> inc(incl ? PR * static_cast<size_t>(h->K) : 0);
    std::vector<double> tr;
    if (var_out) CU(cudaMemcpyAsync(vo.data(), h->dev.var, sizeof(float) * vo.size(), cudaMemcpyDeviceToHost, h->stream));
    if (incl) {
        double* dbg = reinterpret_cast<double*>(h->ws + h->plan.o_dbg);
        inclusion_kernel<<<PR, 128, 0, h->stream>>>(h->dev, h->hyp.incl_tau, dbg, dbg + static_cast<size_t>(PR) * h->K);
        CU(cudaGetLastError());
        CU(cudaMemcpyAsync(inc.data(), dbg, sizeof(double) * inc.size(), cudaMemcpyDeviceToHost, h->stream));
    }
    const int kept = std::min(iterations, kTraceCap);
    if (trace && kept > 0) {
        tr.resize(static_cast<size_t>(kTraceCap) * PR);
        CU(cudaMemcpyAsync(tr.data(), h->dev.trace, sizeof(double) * tr.size(), cudaMemcpyDeviceToHost, h->stream));
    }
    CU(cudaStreamSynchronize(h->stream));
    if (var_out) std::memcpy(var_out, vo.data(), sizeof(float) * vo.size());
    if (incl) std::memcpy(incl, inc.data(), sizeof(double) * inc.size());
    if (trace) {
        for (int it = 0; it < iterations; ++it)
            for (int i = 0; i < PR; ++i)
                trace[static_cast<size_t>(it) * PR + i] =
                    (it >= iterations - kept) ? tr[static_cast<size_t>(it % kTraceCap) * PR + i]
                                              : std::numeric_limits<double>::quiet_NaN();
    }
    return XRDVI_OK;
}

int xrdvi_inclusion(xrdvi* h, double* incl, double* ratio) {
    if (!h) return fail(XRDVI_E_INVALID_ARG, "null handle");
    CU(cudaSetDevice(h->device));
    const int PR = h->plan.PR;
    const size_t n = static_cast<size_t>(PR) * h->K;
    double* dbg = reinterpret_cast<double*>(h->ws + h->plan.o_dbg);
    inclusion_kernel<<<PR, 128, 0, h->stream>>>(h->dev, h->hyp.incl_tau, dbg, dbg + n);
    CU(cudaGetLastError());
    std::vector<double> buf(2 * n);
    CU(cudaMemcpyAsync(buf.data(), dbg, sizeof(double) * 2 * n, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    if (incl) std::memcpy(incl, buf.data(), sizeof(double) * n);
    if (ratio) std::memcpy(ratio, buf.data() + n, sizeof(double) * n);
    return XRDVI_OK;
}

int xrdvi_debug_profile(xrdvi* h, const float* var_params, int32_t S, uint64_t seed, uint64_t iteration,
                        int64_t n, float* f, double* ll) {
    int rc = check_S(h, S);
    if (rc) return rc;
    CU(cudaSetDevice(h->device));
    const long long T = static_cast<long long>(h->plan.PR) * S;
    if (n < 0 || n > T) return fail(XRDVI_E_INVALID_ARG, "n out of range");
    const size_t b = sizeof(float) * h->plan.PR * 8 * h->K;
    const float* var = h->dev.var;
    if (var_params) {
        float* tmp = reinterpret_cast<float*>(h->ws + h->plan.o_vartmp);
        CU(cudaMemcpyAsync(tmp, var_params, b, cudaMemcpyHostToDevice, h->stream));
        var = tmp;
    }
    set_S(h, S);
    rc = write_ctl(h, seed, h->step_host, h->step_host, static_cast<long long>(iteration & 0xFFFFFFFFull));
    if (rc) return rc;
    float* f_dev = nullptr;
    if (f && n > 0) CU(cudaMalloc(&f_dev, sizeof(float) * n * h->N));  // debug path only
    rc = enqueue_iteration(h, var, 0, f_dev, n, nullptr, true);
    if (rc) { cudaFree(f_dev); return rc; }
    std::vector<double> llh(static_cast<size_t>(h->plan.PR) * h->plan.S_pad);
    cudaError_t e = cudaMemcpyAsync(llh.data(), h->dev.ll_t, sizeof(double) * llh.size(), cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess && f_dev) e = cudaMemcpyAsync(f, f_dev, sizeof(float) * n * h->N, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    cudaFree(f_dev);
    if (e != cudaSuccess) return fail(XRDVI_E_CUDA, std::string("debug_profile: ") + cudaGetErrorString(e));
    if (ll) {
        const int gpi32 = h->dev.gpi * 32;
        for (long long t = 0; t < n; ++t) ll[t] = llh[static_cast<size_t>(t / S) * gpi32 + (t % S)];
    }
    return XRDVI_OK;
}

int xrdvi_debug_draws(xrdvi* h, int32_t S, uint64_t seed, uint64_t iteration, int64_t n, float* eps, uint32_t* raw) {
    int rc = check_S(h, S);
    if (rc) return rc;
    CU(cudaSetDevice(h->device));
    const long long T = static_cast<long long>(h->plan.PR) * S;
    if (n < 0 || n > T || !eps) return fail(XRDVI_E_INVALID_ARG, "n out of range or eps NULL");
    set_S(h, S);
    rc = write_ctl(h, seed, h->step_host, h->step_host, static_cast<long long>(iteration & 0xFFFFFFFFull));
    if (rc) return rc;
    const Dev& d = h->dev;
    const size_t cnt = static_cast<size_t>(d.G) * d.K * 32;
    uint4* raw_dev = nullptr;
    CU(cudaMalloc(&raw_dev, sizeof(uint4) * cnt));  // debug path only
    draw_transform_kernel<<<dim3((d.K + 3) / 4, d.G), 128, 0, h->stream>>>(d, d.var, raw_dev);
    std::vector<float4> eh(cnt);
    std::vector<uint4> rh(cnt);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(eh.data(), d.eps, sizeof(float4) * cnt, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(rh.data(), raw_dev, sizeof(uint4) * cnt, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    cudaFree(raw_dev);
    if (e != cudaSuccess) return fail(XRDVI_E_CUDA, std::string("debug_draws: ") + cudaGetErrorString(e));
    for (long long t = 0; t < n; ++t) {
        const int inst = static_cast<int>(t / S), s = static_cast<int>(t % S);
        const int g = inst * d.gpi + s / 32, lane = s % 32;
        for (int k = 0; k < d.K; ++k) {
            const size_t o = (static_cast<size_t>(g) * d.K + k) * 32 + lane;
            std::memcpy(eps + (static_cast<size_t>(t) * d.K + k) * 4, &eh[o], sizeof(float4));
            if (raw) std::memcpy(raw + (static_cast<size_t>(t) * d.K + k) * 4, &rh[o], sizeof(uint4));
        }
    }
    return XRDVI_OK;
}

int xrdvi_time_kernels(xrdvi* h, int32_t S, uint64_t seed, int32_t reps, float* ms_fwd, float* ms_bwd, float* ms_iter) {
    int rc = check_S(h, S);
    if (rc) return rc;
    if (reps < 1) return fail(XRDVI_E_INVALID_ARG, "reps < 1");
    CU(cudaSetDevice(h->device));
    set_S(h, S);
    rc = write_ctl(h, seed, h->step_host, h->step_host, -1);
    if (rc) return rc;
    const Dev& d = h->dev;
    cudaStream_t st = h->stream;
    double tf = 0.0, tb = 0.0, ti = 0.0;
    for (int r = 0; r < reps + 1; ++r) {   // first pass is a warm-up
        CU(cudaEventRecord(h->ev[0], st));
        draw_transform_kernel<<<dim3((d.K + 3) / 4, d.G), 128, 0, st>>>(d, d.var, nullptr);
        CU(cudaEventRecord(h->ev[1], st));
        forward_kernel<<<dim3((d.ntile + kFwdWarps - 1) / kFwdWarps, d.G), 32 * kFwdWarps, 0, st>>>(d, nullptr, 0);
        CU(cudaEventRecord(h->ev[2], st));
        backward_kernel<<<dim3((d.n_units + kBwdWarps - 1) / kBwdWarps, d.G), 32 * kBwdWarps, 0, st>>>(d);
        CU(cudaEventRecord(h->ev[3], st));
        chain_reduce_kernel<<<dim3(d.K, d.PR), kChainThreads, 0, st>>>(d, d.var);
        finalize_update_kernel<<<d.PR, kFinThreads, 0, st>>>(d, d.var, 0);
        CU(cudaEventRecord(h->ev[4], st));
        CU(cudaGetLastError());
        CU(cudaStreamSynchronize(st));
        if (r == 0) continue;
        float a = 0, b = 0, c = 0;
        CU(cudaEventElapsedTime(&a, h->ev[1], h->ev[2]));
        CU(cudaEventElapsedTime(&b, h->ev[2], h->ev[3]));
        CU(cudaEventElapsedTime(&c, h->ev[0], h->ev[4]));
        tf += a; tb += b; ti += c;
    }
    if (ms_fwd) *ms_fwd = static_cast<float>(tf / reps);
    if (ms_bwd) *ms_bwd = static_cast<float>(tb / reps);
    if (ms_iter) *ms_iter = static_cast<float>(ti / reps);
    return XRDVI_OK;
}

int xrdvi_bench_steps(xrdvi* h, int32_t steps, int32_t S, uint64_t seed, size_t flush_bytes, float* ms_steps) {
    int rc = check_S(h, S);
    if (rc) return rc;
    if (steps < 1 || !ms_steps) return fail(XRDVI_E_INVALID_ARG, "steps < 1 or ms_steps NULL");
    CU(cudaSetDevice(h->device));
    rc = ensure_graph(h, S);
    if (rc) return rc;
    set_S(h, S);
    rc = write_ctl(h, seed, h->step_host, h->step_host, -1);
    if (rc) return rc;
    void* flush = nullptr;
    if (flush_bytes) CU(cudaMalloc(&flush, flush_bytes));  // measurement path only
    std::vector<cudaEvent_t> ev(2 * static_cast<size_t>(steps), nullptr);
    cudaError_t e = cudaSuccess;
    for (auto& x : ev) if (e == cudaSuccess) e = cudaEventCreate(&x);
    if (e == cudaSuccess && flush) e = cudaMemsetAsync(flush, 0, flush_bytes, h->stream);
    for (int i = 0; i < steps && e == cudaSuccess; ++i) {
        e = cudaEventRecord(ev[2 * i], h->stream);
        if (e == cudaSuccess) e = cudaGraphLaunch(h->graph_exec, h->stream);
        if (e == cudaSuccess) e = cudaEventRecord(ev[2 * i + 1], h->stream);
        if (e == cudaSuccess && flush) e = cudaMemsetAsync(flush, i & 0xFF, flush_bytes, h->stream);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    h->step_host += steps;
    for (int i = 0; i < steps && e == cudaSuccess; ++i) e = cudaEventElapsedTime(&ms_steps[i], ev[2 * i], ev[2 * i + 1]);
    for (auto& x : ev) if (x) cudaEventDestroy(x);
    if (flush) cudaFree(flush);
    if (e != cudaSuccess) return fail(XRDVI_E_CUDA, std::string("bench_steps: ") + cudaGetErrorString(e));
    return XRDVI_OK;
}

}  // extern "C"
