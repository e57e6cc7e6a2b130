// xrdvi.cu -- C ABI (include/xrdvi.h), host preprocessing in fp64, launch logic and CUDA Graph.
// There is no CPU fallback anywhere in this file: every compute step is a kernel in
// xrdvi_kernels.cuh; the host only validates, sorts and encodes the static tables at create.
#include "../../include/xrdvi.h"
#include "../../include/xrdvi_debug.h"
#include "xrdvi_kernels.cuh"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <mutex>
#include <numeric>
#include <string>
#include <vector>

using namespace xrdvi_dev;

// Scratch of xrdvi_profile_static (include/xrdvi.h), the one entry point that needs no caller scratch: profile rows
// float [n][N] between the forward kernel and the copy to the caller.  kStaticScratchFloats floats = 4 MiB, held by every
// GPU that loads this library until the process exits.  In host code this NAME is a host-side stand-in, not a device
// address: static_scratch_address() below resolves it once per device, and only that pointer is given to a kernel.
constexpr size_t kStaticScratchFloats = size_t(1) << 20;
static __device__ __align__(256) float g_static_scratch[kStaticScratchFloats];

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

// Device address of g_static_scratch on `device`, which must be the CURRENT device (every device that loads the module has
// its own copy of the array).  Resolved once per device, at set-up (xrdvi_create), cached with its return code.
constexpr int kMaxDevices = 64;
struct StaticScratch { float* ptr = nullptr; cudaError_t err = cudaSuccess; bool done = false; };
StaticScratch g_static[kMaxDevices];
std::mutex g_static_mu;

cudaError_t static_scratch_address(int device, float** ptr) {
    *ptr = nullptr;
    if (device < 0 || device >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_static_mu);
    StaticScratch& e = g_static[device];
    if (!e.done) {
        void* p = nullptr;
        e.err = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e.err != cudaSuccess) { p = nullptr; (void)cudaGetLastError(); }   // reported by xrdvi_profile_static, not here
        e.ptr = static_cast<float*>(p);
        e.done = true;
    }
    *ptr = e.ptr;
    return e.err;
}


struct Plan {   // workspace carve; identical arithmetic in workspace_bytes and create
    int P, R, PR, S_pad, gpi_max, G_max, K;
    int TW, PS, split, NW, SP, n_seg, n_tile;
    long long M, n_c, tile_cap, slots_cap;
    size_t total;
    size_t o_yb, o_bg, o_pkt, o_runs, o_srng, o_sord, o_sofs, o_pat, o_area, o_mh0;
    size_t o_var, o_vartmp, o_mom1, o_mom2, o_grad, o_elbo, o_elbok, o_llt, o_llg, o_trace, o_ctl;
    size_t o_lat, o_eps, o_rr, o_ng, o_llpart, o_part8, o_dbg;
    size_t o_pd, o_lpk, o_zeta, o_gradz, o_lls, o_partial, o_tcnt, o_summ;
    size_t o_trng, o_ia, o_epsa, o_parta, o_pksec, o_secmax, o_tileoff, o_pkbase;
    int pd_groups;     // groups one launch of the log-joint gradient service handles
};

// window half-width in grid points (R16); dense (W <= 0) is represented by n_c = -1 here
long long window_points(const xrdvi_hyper* hyp, double step) {
    if (!(hyp->window_W > 0.0)) return -1;
    return static_cast<long long>(std::ceil(hyp->window_W * hyp->fwhm_ref / step - 1e-9));
}

// CTA shape of elbo_tile_kernel: TW tiles of 16 points per segment, PS shares of each tile's peak list
// (TW * PS warps).  Many groups: no split.  Few groups (config 1: 8): split peak lists, so that the SMs still see
// several warps per scheduler.  n_sm <= 0 (xrdvi_workspace_bytes, which knows no device): the decision for 256 SMs, whose
// workspace bounds that of every smaller device (PS = 4 needs more than PS = 1).
void choose_shape(int64_t N, int G_max, int n_sm, int* TW, int* PS) {
#ifdef XRDVI_TUNING
    if (const char* e = std::getenv("XRDVI_TILE_SHAPE")) {   // sweep knob of the measurement build: "TWxPS"
        int a = 0, b = 0;
        if (std::sscanf(e, "%dx%d", &a, &b) == 2 && (a == 1 || a == 2 || a == 4) && (b == 1 || b == 2 || b == 3 || b == 4 || b == 5 || b == 6 || b == 8) && a * b <= 16) {
            *TW = a; *PS = b;
            return;
        }
    }
#endif
    // measured on B200 (profiles/r1_v5_shape_sweep.md, repeated with staged lists in profiles/r2_*): one tile per CTA
    // is best everywhere; launches with fewer than 8 tile-warps per resident warp slot (configs 1 and 4: 2008 / 4008)
    // want the peak lists split four ways, the others (configs 2, 3: 1e6) no split
    const long long tiles = (N + 15) / 16 * static_cast<long long>(G_max);   // warps at PS = 1
    const int sms = (n_sm <= 0 || n_sm > 256) ? 256 : n_sm;                   // no device: the largest count the bound covers
    const long long resident = static_cast<long long>(sms) * 24;              // warps the GPU holds at 80 registers
    *TW = 1;
    *PS = tiles >= 8 * resident ? 1 : 4;
}

bool make_plan(int64_t N, int32_t K, int64_t M, int32_t S_max, double step, const xrdvi_hyper* hyp, int n_sm, Plan* pl) {
    if (N < 2 || K < 1 || M < 1 || S_max < 1 || !hyp || !(step > 0.0)) return false;
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
    choose_shape(N, p.G_max, n_sm, &p.TW, &p.PS);
    p.NW = p.TW * p.PS;
    p.SP = kPT * p.TW;
    p.n_seg = static_cast<int>((N + p.SP - 1) / p.SP);
    p.n_tile = static_cast<int>((N + kPT - 1) / kPT);
    if (p.n_seg > 65535) return false;                  // grid.y limit of elbo_tile_kernel
    p.n_c = window_points(hyp, step);
    // entries of the per-tile phase-major lists: a peak appears once per 16-point tile its window touches
    const long long per_peak = p.n_c < 0 ? p.n_tile : std::min<long long>(p.n_tile, (2 * p.n_c + kPT) / kPT + 1);
    p.tile_cap = M * per_peak;
    // long work items (an upper bound of the records of one of PS shares of a tile >= 512; config 4): one-warp items on a
    // ticket queue (elbo_split_kernel) instead of PS-warp CTAs
    p.split = (p.PS > 1 && p.TW == 1 && p.tile_cap / (static_cast<long long>(p.n_tile) * p.PS) >= 512) ? 1 : 0;
    // one output slot per (tile, phase present in the tile), plus one per run a share boundary cuts
    p.slots_cap = std::min<long long>(static_cast<long long>(p.n_tile) * K, p.tile_cap) + static_cast<long long>(p.n_tile) * (p.PS - 1);
    if (p.tile_cap > (1ll << 31) - 1 || p.slots_cap > (1ll << 31) - 1) return false;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t r = o; o = align_up(o + bytes); return r; };
    const size_t var_b = sizeof(float) * p.PR * 10 * static_cast<size_t>(K);   // [PR][2][K][4], then [PR][2][K] for alpha (R30)
    const size_t gk32 = static_cast<size_t>(p.G_max) * K * 32;
    p.o_yb = take(sizeof(float) * p.P * N);
    p.o_bg = take(sizeof(float) * p.P * N);
    p.o_pkt = take(sizeof(PeakRec) * (p.tile_cap + 1));
    p.o_runs = take(sizeof(int4) * (p.slots_cap + 1));
    p.o_srng = take(sizeof(int2) * static_cast<size_t>(p.n_tile) * p.PS);
    p.o_sord = take(sizeof(int) * p.n_seg);
    p.o_sofs = take(sizeof(int) * (K + 1));
    p.o_pat = take(sizeof(PatConst) * p.P);
    p.o_area = take(sizeof(double) * K);
    p.o_mh0 = take(sizeof(float) * p.P);
    p.o_var = take(var_b);
    p.o_vartmp = take(var_b);
    p.o_mom1 = take(var_b);
    p.o_mom2 = take(var_b);
    p.o_grad = take(var_b);
    p.o_elbo = take(sizeof(double) * p.PR);
    p.o_elbok = take(sizeof(double) * p.PR * (K + 1));
    p.o_llt = take(sizeof(double) * p.PR * p.S_pad);
    p.o_llg = take(sizeof(double) * p.G_max);
    p.o_trace = take(sizeof(double) * kTraceCap * p.PR);
    p.o_ctl = take(sizeof(Ctl));
    p.o_lat = take(sizeof(float4) * gk32);
    p.o_eps = take(sizeof(float4) * gk32);
    p.o_rr = take(sizeof(float) * gk32);
    p.o_ng = take(sizeof(int) * static_cast<size_t>(p.G_max) * K);
    p.o_llpart = take(sizeof(float) * static_cast<size_t>(p.G_max) * p.n_seg * 32);
    p.o_part8 = take(sizeof(float) * static_cast<size_t>(p.G_max) * std::max<long long>(p.slots_cap, 1) * 8);
    p.o_dbg = take(sizeof(double) * (2 * static_cast<size_t>(p.PR) * K + 64));
    p.o_summ = take(sizeof(double) * 25 * static_cast<size_t>(p.PR) * K);   // marginal summaries (R28; 5 classes with R30)
    // log-joint gradient service: per-draw partials of at most 64 MiB worth of groups (at least one)
    const size_t pd_group_bytes = sizeof(float) * 160 * static_cast<size_t>(std::max<long long>(p.slots_cap, 1));
    p.pd_groups = static_cast<int>(std::min<size_t>(p.gpi_max, std::max<size_t>(1, (size_t(64) << 20) / pd_group_bytes)));
    p.o_pd = take(pd_group_bytes * p.pd_groups);
    p.o_lpk = take(sizeof(float) * 32 * static_cast<size_t>(K) * p.pd_groups);
    p.o_zeta = take(sizeof(float) * 5 * static_cast<size_t>(p.S_pad) * K);    // float4 [S_pad][K], then float [S_pad][K] (alpha)
    p.o_gradz = take(sizeof(float) * 5 * static_cast<size_t>(p.S_pad) * K);
    p.o_lls = take(sizeof(double) * 2 * p.S_pad);
    // split kernel (PS > 1): partial profiles of every (group, tile, share) and two counters per (group, tile)
    p.o_partial = take(p.split ? sizeof(float) * kPT * 32 * static_cast<size_t>(p.G_max) * p.n_tile * p.PS : 0);
    p.o_tcnt = take(sizeof(unsigned int) * 2 * static_cast<size_t>(p.G_max) * p.n_tile);
    p.o_trng = take(sizeof(int2) * (static_cast<size_t>(p.n_tile) + 1));
    const bool model = hyp->asymmetry || hyp->width_sec || hyp->general_grid;    // R30 / R31 buffers only when in use
    p.o_ia = take(model ? sizeof(float) * gk32 : 0);
    p.o_epsa = take(model ? sizeof(float) * gk32 : 0);
    p.o_parta = take(model ? sizeof(float) * 2 * static_cast<size_t>(p.G_max) * std::max<long long>(p.slots_cap, 1) : 0);
    p.o_pksec = take(hyp->width_sec ? sizeof(float) * (p.tile_cap + 1) : 0);
    p.o_secmax = take(sizeof(float) * K);
    p.o_tileoff = take(hyp->general_grid ? sizeof(float) * kPT * static_cast<size_t>(p.n_tile) : 0);
    p.o_pkbase = take(hyp->general_grid ? sizeof(float) * (p.tile_cap + 1) : 0);
    p.total = o;
    *pl = p;
    return true;
}

// ---- static tables (R16, R27) -----------------------------------------------------------------------
struct HostPeak { long long j; double d; double I; int k; double inv_s; double pos; };   // nearest grid index, p_m - x_j, intensity, phase, cos(p_m / 2) (R30)

struct Tables {
    std::vector<PeakRec> pk_tile;     // per-tile phase-major peak lists (+1 padding record)
    std::vector<float> pk_sec;        // cos(p_m / 2) of every record's peak (sec width term, R30)
    std::vector<float> pk_base;       // x_{i0} - p_m of every record (general grid, R31)
    std::vector<int4> run_tab;        // (m0, m1, phase, slot) per phase run (+1 padding header)
    std::vector<int2> share_rng;      // [n_tile][PS] run ranges of the shares
    std::vector<int> seg_order, slot_ofs;
    std::vector<int2> tile_rng;       // [n_tile + 1] (first run, first record) of every tile's lists
    int max_tile_rec = 0, max_tile_runs = 0;
    int n_slots = 0;
    long long pairs = 0;              // in-window (peak, point) pairs per draw
};

// Per-tile phase-major lists: the peaks whose window reaches the tile, stable-sorted by phase; PS contiguous shares
// split at phase boundaries and balanced by clipped pair count; one output slot per (tile, phase present in the
// tile).  `nck[k]` is the window half-width of phase k in points (the static n_c for every phase at create; per
// phase after xrdvi_set_phase_windows, R27); peaks with no in-range grid point are dropped.  All in integers.
const char* build_tables(const Plan& pl, int64_t N, int K, const std::vector<HostPeak>& all,
                         const std::vector<long long>& nck, const std::vector<double>& xgrid, Tables* T) {
    std::vector<HostPeak> fw;
    fw.reserve(all.size());
    long long pairs = 0;
    for (const HostPeak& p : all) {
        const long long lo = std::max<long long>(0, p.j - nck[p.k]), hi = std::min<long long>(N - 1, p.j + nck[p.k]);
        if (lo > hi) continue;  // no in-range grid point
        pairs += hi - lo + 1;
        fw.push_back(p);
    }
    // (phase, grid index, input order) order: the order of the entries inside every tile list.  The callers hand the peaks
    // over phase by phase, so one stable sort by grid index inside every phase's range does it (two stable sorts of the
    // whole list otherwise: 0.34 of the 0.86 ms of a config-1 table build).
    if (std::is_sorted(fw.begin(), fw.end(), [](const HostPeak& a, const HostPeak& b) { return a.k < b.k; })) {
        for (size_t b = 0; b < fw.size();) {
            size_t e = b + 1;
            while (e < fw.size() && fw[e].k == fw[b].k) ++e;
            std::stable_sort(fw.begin() + b, fw.begin() + e, [](const HostPeak& a, const HostPeak& b2) { return a.j < b2.j; });
            b = e;
        }
    } else {
        std::stable_sort(fw.begin(), fw.end(), [](const HostPeak& a, const HostPeak& b) { return a.j < b.j; });
        std::stable_sort(fw.begin(), fw.end(), [](const HostPeak& a, const HostPeak& b) { return a.k < b.k; });
    }
    const int PSn = pl.PS, TWn = pl.TW, n_tile = pl.n_tile;
    auto tiles_of = [&](const HostPeak& p, int* t0, int* t1) {
        const long long lo = std::max<long long>(0, p.j - nck[p.k]), hi = std::min<long long>(N - 1, p.j + nck[p.k]);
        *t0 = static_cast<int>(lo / kPT);
        *t1 = static_cast<int>(hi / kPT);
    };
    // pass 1: entries and phase runs per tile
    std::vector<long long> ent_base(n_tile + 1, 0);
    std::vector<int> run_base(n_tile + 1, 0), last_k(n_tile, -1);
    for (const HostPeak& p : fw) {
        int t0, t1;
        tiles_of(p, &t0, &t1);
        for (int t = t0; t <= t1; ++t) {
            ++ent_base[t + 1];
            if (last_k[t] != p.k) { last_k[t] = p.k; ++run_base[t + 1]; }
        }
    }
    for (int t = 0; t < n_tile; ++t) { ent_base[t + 1] += ent_base[t]; run_base[t + 1] += run_base[t]; }
    const long long n_ent = ent_base[n_tile];
    const int n_runs = run_base[n_tile];
    if (n_ent > pl.tile_cap || n_runs > pl.slots_cap) return "internal: table bound exceeded";
    // pass 2: fill the lists, the run headers (m0, m1, phase, 0) and the clipped pair count of every run
    T->pk_sec.assign(static_cast<size_t>(n_ent) + 1, 1.0f);
    T->pk_base.assign(xgrid.empty() ? 0 : static_cast<size_t>(n_ent) + 1, 0.0f);
    T->pk_tile.assign(static_cast<size_t>(n_ent) + 1, PeakRec{0, 0.f, 0.f, 0});   // +1: the kernel prefetches one
    T->run_tab.assign(static_cast<size_t>(n_runs) + 1, make_int4(0, 0, 0, 0));    // record / header past the end
    T->share_rng.assign(static_cast<size_t>(n_tile) * PSn, make_int2(0, 0));
    std::vector<long long> seg_work(pl.n_seg, 0);
    std::vector<int> rec_w(static_cast<size_t>(n_ent), 0);   // in-window points of every record (share balance)
    std::vector<long long> ent_cur(ent_base.begin(), ent_base.end() - 1);
    std::vector<int> run_cur(run_base.begin(), run_base.end() - 1);
    std::fill(last_k.begin(), last_k.end(), -1);
    long long pairs_check = 0;
    for (const HostPeak& p : fw) {
        int t0, t1;
        tiles_of(p, &t0, &t1);
        const long long n = nck[p.k];
        for (int t = t0; t <= t1; ++t) {
            const long long i0 = static_cast<long long>(t) * kPT, i1 = std::min<long long>(i0 + kPT - 1, N - 1);
            const long long wq = std::min(i1, p.j + n) - std::max(i0, p.j - n) + 1;   // >= 1 by construction
            const long long dj = p.j - i0;
            const bool full = (i1 - i0 == kPT - 1) && dj - n <= 0 && dj + n >= kPT - 1;
            const long long e = ent_cur[t]++;
            T->pk_tile[e] = PeakRec{static_cast<int>(dj), static_cast<float>(p.d), static_cast<float>(p.I),
                                    static_cast<int>(n << 1) | (full ? 1 : 0)};
            T->pk_sec[e] = static_cast<float>(p.inv_s);
            if (!xgrid.empty()) T->pk_base[e] = static_cast<float>(xgrid[i0] - p.pos);   // fp64 difference (R31)
            if (last_k[t] != p.k) {
                last_k[t] = p.k;
                T->run_tab[run_cur[t]++] = make_int4(static_cast<int>(e), static_cast<int>(e), p.k, 0);
            }
            const int r = run_cur[t] - 1;
            T->run_tab[r].y = static_cast<int>(e) + 1;
            rec_w[e] = static_cast<int>(wq);
            seg_work[t / TWn] += wq;
            pairs_check += wq;
        }
    }
    // pass 3: PS contiguous shares per tile, balanced by in-window pair count at RECORD granularity: a share boundary
    // that falls inside a phase run cuts the run in two (two headers, two output slots of the same phase: the reduction
    // over the slots of a phase does not care), so that the shares of a tile -- which meet at a barrier -- carry equal
    // work whatever the sizes of the phases.  Rebuilds run_tab / run_base with the cut runs.
    {
        std::vector<int4> runs2;
        runs2.reserve(static_cast<size_t>(n_runs) + static_cast<size_t>(n_tile) * PSn);
        std::vector<int> run_base2(n_tile + 1, 0);
        for (int t = 0; t < n_tile; ++t) {
            run_base2[t] = static_cast<int>(runs2.size());
            const long long e0 = ent_base[t], e1 = ent_base[t + 1];
            long long tot = 0;
            for (long long e = e0; e < e1; ++e) tot += rec_w[e];
            std::vector<long long> cuts(PSn + 1, e1);        // share w = records [cuts[w], cuts[w + 1])
            cuts[0] = e0;
            {
                long long cum = 0, e = e0;
                for (int w = 1; w < PSn; ++w) {
                    const long long goal = tot * w / PSn;
                    while (e < e1 && cum + rec_w[e] <= goal) { cum += rec_w[e]; ++e; }
                    cuts[w] = e;
                }
            }
            int w = 0;
            std::vector<int> share_first(PSn + 1, 0);
            for (int r = run_base[t]; r < run_base[t + 1]; ++r) {
                long long m0 = T->run_tab[r].x;
                const long long m1 = T->run_tab[r].y;
                while (m0 < m1) {
                    while (w < PSn && cuts[w + 1] <= m0) { ++w; share_first[w] = static_cast<int>(runs2.size()); }
                    const long long stop = std::min(m1, w < PSn ? cuts[w + 1] : m1);
                    runs2.push_back(make_int4(static_cast<int>(m0), static_cast<int>(stop), T->run_tab[r].z, 0));
                    m0 = stop;
                }
            }
            while (w < PSn) { ++w; share_first[w] = static_cast<int>(runs2.size()); }
            for (int q = 0; q < PSn; ++q)
                T->share_rng[static_cast<size_t>(t) * PSn + q] = make_int2(std::max(share_first[q], run_base2[t]), share_first[q + 1]);
            T->share_rng[static_cast<size_t>(t) * PSn].x = run_base2[t];
        }
        run_base2[n_tile] = static_cast<int>(runs2.size());
        if (static_cast<long long>(runs2.size()) > pl.slots_cap) return "internal: table bound exceeded (cut runs)";
        runs2.push_back(make_int4(0, 0, 0, 0));              // the header past the end
        T->run_tab.swap(runs2);
        run_base.swap(run_base2);
    }
    const int n_runs2 = static_cast<int>(T->run_tab.size()) - 1;
    std::vector<int> slot_phase(n_runs2);
    for (int r = 0; r < n_runs2; ++r) slot_phase[r] = T->run_tab[r].z;
    if (pairs_check != pairs) return "internal: tile tables do not cover every pair once";
    const int n_slots = n_runs2;
    // output slots numbered phase-major (the reduction over the tiles of a phase reads one contiguous range);
    // within a phase in increasing tile order
    T->slot_ofs.assign(K + 1, 0);
    for (int s = 0; s < n_slots; ++s) ++T->slot_ofs[slot_phase[s] + 1];
    for (int k = 0; k < K; ++k) T->slot_ofs[k + 1] += T->slot_ofs[k];
    {
        std::vector<int> fill(T->slot_ofs.begin(), T->slot_ofs.end() - 1);
        for (int s = 0; s < n_slots; ++s) T->run_tab[s].w = fill[slot_phase[s]]++;
    }
    T->seg_order.resize(pl.n_seg);
    std::iota(T->seg_order.begin(), T->seg_order.end(), 0);
    std::stable_sort(T->seg_order.begin(), T->seg_order.end(), [&](int a, int b) { return seg_work[a] > seg_work[b]; });
    T->tile_rng.resize(static_cast<size_t>(n_tile) + 1);
    T->max_tile_rec = T->max_tile_runs = 0;
    for (int t = 0; t <= n_tile; ++t) {
        T->tile_rng[t] = make_int2(run_base[t], static_cast<int>(ent_base[t]));
        if (t < n_tile) {
            T->max_tile_rec = std::max(T->max_tile_rec, static_cast<int>(ent_base[t + 1] - ent_base[t]));
            T->max_tile_runs = std::max(T->max_tile_runs, run_base[t + 1] - run_base[t]);
        }
    }
    T->n_slots = n_slots;
    T->pairs = pairs;
    return nullptr;
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
    int n_c = 0;               // create-time (static) half-width; the cap of the per-phase ones
    bool windowed = false;     // hyper.window_W > 0
    double delta = 0.0;        // grid step
    std::vector<HostPeak> peaks;   // every input peak, CSR order (xrdvi_set_phase_windows rebuilds the tables from it)
    std::vector<double> xgrid;     // the grid, kept only for hyper.general_grid (R31: per-record bases x_{i0} - p_m)
    std::vector<long long> n_ck;   // [K] half-width per phase in force (R27); all n_c after create
    std::vector<float> m_h0;   // per pattern initial m_h
    float m_w0 = 0.f;
    long long step_host = 0;   // mirror of ctl.step
    long long adam_t0 = 0;     // mirror of ctl.adam_t0 (step count at which the Adam moments were last zeroed)
    bool own_stream = false;   // the stream was created by xrdvi_create (caller passed 0)
    float* static_scratch = nullptr;               // device address of g_static_scratch on h->device (set at create)
    cudaError_t static_scratch_err = cudaSuccess;  // what cudaGetSymbolAddress returned there
    // CUDA Graph of one optimisation step, keyed by S
    cudaGraphExec_t graph_exec = nullptr;    // one step
    cudaGraphExec_t graph_execU = nullptr;   // kUnroll steps: programmatic launches also across step boundaries
    int graph_S = -1;
    int max_phase_slots = 0;   // output slots of the widest phase at create
    cudaEvent_t ev[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
};

namespace {

// Dynamic shared memory of update_draw_kernel: room for the slot rows (32 bytes each) of the widest phase over all
// groups of an instance, if every draw of an instance has a thread of its own and the rows fit; else 0 (its long path).
constexpr int kUpdSmemCap = 96 * 1024;

int set_S(xrdvi* h, int S) {
    h->dev.S = S;
    h->dev.gpi = (S + 31) / 32;
    h->dev.G = h->plan.PR * h->dev.gpi;
    const long long rows = static_cast<long long>(h->max_phase_slots) * h->dev.gpi * 32;
    h->dev.upd_smem = (h->dev.gpi * 32 <= kUpdThreads && rows <= kUpdSmemCap) ? static_cast<int>(rows) : 0;
    return XRDVI_OK;
}

// Upload a set of static tables and make them the ones in force.  The Dev block (kernel argument, held by value in
// the captured graphs) does not change after create: `n_slots` is only the row stride of the backward's output
// slots and stays at the create-time count (per-phase windows are never wider than the static one, so a later
// table set has at most as many (tile, phase) runs), and the fused / ticket-queue choice is made once.  A refresh
// therefore needs no graph re-capture.
int install_tables(xrdvi* h, const Tables& T, const std::vector<long long>& nck, bool at_create) {
    const Plan& pl = h->plan;
    Dev& d = h->dev;
    cudaStream_t st = h->stream;
    char* w = h->ws;
    if (!at_create && T.n_slots > d.n_slots) return fail(XRDVI_E_INVALID_ARG, "internal: more output slots than at create");
    CU(cudaStreamSynchronize(st));   // nothing in flight may still read the old tables
    CU(cudaMemcpyAsync(w + pl.o_pkt, T.pk_tile.data(), sizeof(PeakRec) * T.pk_tile.size(), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(w + pl.o_runs, T.run_tab.data(), sizeof(int4) * T.run_tab.size(), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(w + pl.o_srng, T.share_rng.data(), sizeof(int2) * T.share_rng.size(), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(w + pl.o_sord, T.seg_order.data(), sizeof(int) * T.seg_order.size(), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(w + pl.o_sofs, T.slot_ofs.data(), sizeof(int) * T.slot_ofs.size(), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(w + pl.o_trng, T.tile_rng.data(), sizeof(int2) * T.tile_rng.size(), cudaMemcpyHostToDevice, st));
    if (h->hyp.general_grid)
        CU(cudaMemcpyAsync(w + pl.o_pkbase, T.pk_base.data(), sizeof(float) * T.pk_base.size(), cudaMemcpyHostToDevice, st));
    if (h->hyp.width_sec)
        CU(cudaMemcpyAsync(w + pl.o_pksec, T.pk_sec.data(), sizeof(float) * T.pk_sec.size(), cudaMemcpyHostToDevice, st));
    if (at_create) {
        // widest phase in output slots (per-phase windows only ever shrink it): sizes update_draw_kernel's staging buffer
        h->max_phase_slots = 0;
        for (size_t k = 0; k + 1 < T.slot_ofs.size(); ++k)
            h->max_phase_slots = std::max(h->max_phase_slots, T.slot_ofs[k + 1] - T.slot_ofs[k]);
        d.n_slots = std::max(T.n_slots, 1);
        d.split = pl.split;
        // bulk-copy staging (TW = 1) needs every tile list to fit the shared-memory buffers; decided once (the per-phase
        // windows of R27 only ever shrink the lists), because the Dev block is held by value in the captured graphs
        d.stage = (pl.TW == 1 && T.max_tile_rec <= kStageRec && T.max_tile_runs <= kStageRun - 1) ? 1 : 0;
#ifdef XRDVI_TUNING
        if (std::getenv("XRDVI_NO_STAGE")) d.stage = 0;     // A/B knob of the measurement build
#endif
        CU(cudaMemsetAsync(w + pl.o_part8, 0, sizeof(float) * static_cast<size_t>(pl.G_max) * d.n_slots * 8, st));
    }
    CU(cudaStreamSynchronize(st));   // T belongs to the caller
    h->pairs = T.pairs;
    h->n_ck = nck;
    return XRDVI_OK;
}

// Few tile-warps (PS > 1) and long work items: one-warp CTAs on a ticket queue (elbo_split_kernel) instead of PS-warp
// CTAs with a barrier.  Measured on B200: config 4 (4300 peaks per item) 22.4 vs 23.5 ms per step, config 1 (39 peaks
// per item) 0.1967 vs 0.1933 ms: the partial profiles through L2 only pay off for long items.
// Launch with the programmatic-stream-serialization attribute (the kernel may begin while its predecessor drains; it
// calls griddep_wait() before touching the predecessor's data).  pdl = false: a plain launch.
template <typename... KArgs, typename... Args>
void launch_k(void (*kernel)(KArgs...), dim3 grid, dim3 block, cudaStream_t st, bool pdl, size_t smem, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

bool use_split(const Dev& d) {
#ifdef XRDVI_TUNING
    if (std::getenv("XRDVI_FUSED")) return false;            // A/B knobs of the measurement build
    if (std::getenv("XRDVI_SPLIT")) return d.TW == 1 && d.PS > 1;
#endif
    return d.TW == 1 && d.PS > 1 && d.split;
}

// one CTA shape: the staged variant when the tile lists fit (TW = 1), the R30 model variant when the asymmetry or the
// sec term is on (instantiated for TW = 1 only; make_plan never selects another TW for them)
template <int TW, int PS, bool BWD>
void launch_tile_shape(const Dev& d, dim3 grid, cudaStream_t st, bool pdl, float* f_dbg, long long n_dbg) {
    const dim3 block(32 * TW * PS);
    if constexpr (TW == 1) {
        if (d.model) {
            if (d.stage) launch_k(elbo_tile_kernel<1, PS, BWD, true, 1>, grid, block, st, pdl, size_t(0), d, f_dbg, n_dbg);
            else launch_k(elbo_tile_kernel<1, PS, BWD, false, 1>, grid, block, st, pdl, size_t(0), d, f_dbg, n_dbg);
            return;
        }
        if (d.stage) { launch_k(elbo_tile_kernel<1, PS, BWD, true, 0>, grid, block, st, pdl, size_t(0), d, f_dbg, n_dbg); return; }
    }
    launch_k(elbo_tile_kernel<TW, PS, BWD, false, 0>, grid, block, st, pdl, size_t(0), d, f_dbg, n_dbg);
}

template <int PS, bool BWD>
void launch_split_shape(const Dev& d, dim3 grid, cudaStream_t st, bool pdl, float* f_dbg, long long n_dbg) {
    if (d.model) launch_k(elbo_split_kernel<PS, BWD, 1>, grid, dim3(32), st, pdl, size_t(0), d, f_dbg, n_dbg);
    else launch_k(elbo_split_kernel<PS, BWD, 0>, grid, dim3(32), st, pdl, size_t(0), d, f_dbg, n_dbg);
}

template <bool BWD>
void launch_tile(const Dev& d, cudaStream_t st, float* f_dbg, long long n_dbg, bool pdl = false) {
    if (BWD && use_split(d)) {   // forward-only launches (debug, timing) always take the fused kernel
        const unsigned items = static_cast<unsigned>(d.n_tile) * d.PS * d.G;
        const dim3 grid(BWD ? 2 * items : items + static_cast<unsigned>(d.n_tile) * d.G);
        switch (d.PS) {
            case 4: launch_split_shape<4, BWD>(d, grid, st, pdl, f_dbg, n_dbg); break;
#ifdef XRDVI_TUNING
            case 3: launch_split_shape<3, BWD>(d, grid, st, pdl, f_dbg, n_dbg); break;
            case 2: launch_split_shape<2, BWD>(d, grid, st, pdl, f_dbg, n_dbg); break;
            case 5: launch_split_shape<5, BWD>(d, grid, st, pdl, f_dbg, n_dbg); break;
            case 6: launch_split_shape<6, BWD>(d, grid, st, pdl, f_dbg, n_dbg); break;
            case 8: launch_split_shape<8, BWD>(d, grid, st, pdl, f_dbg, n_dbg); break;
#endif
            default: break;
        }
        return;
    }
    const dim3 grid(d.G, d.n_seg);   // x = draw group (dispatched fastest), y = position in seg_order
#define XRDVI_TILE_CASE(TW_, PS_) \
    case TW_ * 16 + PS_: launch_tile_shape<TW_, PS_, BWD>(d, grid, st, pdl, f_dbg, n_dbg); break;
    switch (d.TW * 16 + d.PS) {
        XRDVI_TILE_CASE(1, 1) XRDVI_TILE_CASE(1, 4)      // the shapes choose_shape selects
#ifdef XRDVI_TUNING
        XRDVI_TILE_CASE(1, 2) XRDVI_TILE_CASE(1, 3) XRDVI_TILE_CASE(1, 5) XRDVI_TILE_CASE(1, 6) XRDVI_TILE_CASE(1, 8)
        XRDVI_TILE_CASE(2, 1) XRDVI_TILE_CASE(2, 2) XRDVI_TILE_CASE(2, 4) XRDVI_TILE_CASE(2, 8)
        XRDVI_TILE_CASE(4, 1) XRDVI_TILE_CASE(4, 2) XRDVI_TILE_CASE(4, 4)
#endif
        default: break;
    }
#undef XRDVI_TILE_CASE
}

void launch_draw(const Dev& d, cudaStream_t st, const float* var, uint4* raw_out) {
    draw_transform_kernel<<<dim3((d.K + 3) / 4, d.G), 128, 0, st>>>(d, var, raw_out);
}

// one optimisation step as the graph replays it: fused profile/residual/backward, then reduce + Adam +
// the draws of the next step.  The draws of the FIRST step come from launch_draw.
int enqueue_step(xrdvi* h) {
    const Dev& d = h->dev;
#ifdef XRDVI_TUNING
    static const bool pdl = std::getenv("XRDVI_NO_PDL") == nullptr;    // A/B knob of the measurement build
#else
    const bool pdl = true;
#endif
    // both kernels may start while their predecessor drains (programmatic dependent launch); each waits with
    // griddep_wait() before it touches the predecessor's data
    launch_tile<true>(d, h->stream, nullptr, 0, pdl);                  // also finishes the previous step (ELBO, count)
    if (d.tlu)   // xrdvi_debug_update_timeline: the stamped instantiation
        launch_k(update_draw_kernel<true>, dim3(d.K + d.gpi, d.PR), dim3(kUpdThreads), h->stream, pdl, static_cast<size_t>(d.upd_smem), d,
                 static_cast<const float*>(d.var), 1);
    else
        launch_k(update_draw_kernel<false>, dim3(d.K + d.gpi, d.PR), dim3(kUpdThreads), h->stream, pdl, static_cast<size_t>(d.upd_smem), d,
                 static_cast<const float*>(d.var), 1);
    CU(cudaGetLastError());
    return XRDVI_OK;
}

// after the last step of a run (and after an evaluation): the pending ELBO assembly / step count
int enqueue_finish(xrdvi* h) {
    finish_step_kernel<<<1, 256, 0, h->stream>>>(h->dev);
    CU(cudaGetLastError());
    return XRDVI_OK;
}

// one evaluation at `var` without touching the state: draw -> tile -> reduce
int enqueue_eval(xrdvi* h, const float* var, float* f_dbg, long long n_dbg, bool forward_only) {
    const Dev& d = h->dev;
    launch_draw(d, h->stream, var, nullptr);
    if (forward_only) launch_tile<false>(d, h->stream, f_dbg, n_dbg);
    else launch_tile<true>(d, h->stream, f_dbg, n_dbg);
    // forward_only leaves stale partials in part8: the gradient output of this launch is not used then
    update_draw_kernel<false><<<dim3(d.K + d.gpi, d.PR), kUpdThreads, d.upd_smem, h->stream>>>(d, var, 0);
    CU(cudaGetLastError());
    return enqueue_finish(h);
}

int write_ctl(xrdvi* h, uint64_t seed, long long step, long long trace_base, long long it_override) {
    Ctl c{};
    c.seed = seed;
    c.step = step;
    c.u_step = step;
    c.trace_base = trace_base;
    c.iteration_override = it_override;
    c.adam_t0 = h->adam_t0;
    CU(cudaMemcpyAsync(h->dev.ctl, &c, sizeof(Ctl), cudaMemcpyHostToDevice, h->stream));
    CU(cudaStreamSynchronize(h->stream));  // c lives on this stack frame
    return XRDVI_OK;
}

int check_S(xrdvi* h, int32_t S) {
    if (!h) return fail(XRDVI_E_INVALID_ARG, "null handle");
    if (S < 1 || S > h->plan.S_pad) return fail(XRDVI_E_INVALID_ARG, "S out of range [1, S_max]");
    return XRDVI_OK;
}

constexpr int kUnroll = 8;   // steps per graph of the long graph

int capture_steps(xrdvi* h, int n, cudaGraphExec_t* out) {
    cudaGraph_t graph = nullptr;
    CU(cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal));
    int rc = XRDVI_OK;
    for (int i = 0; i < n && rc == XRDVI_OK; ++i) rc = enqueue_step(h);
    cudaError_t e = cudaStreamEndCapture(h->stream, &graph);
    if (rc != XRDVI_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
    if (e != cudaSuccess) return fail(XRDVI_E_CUDA, std::string("cudaStreamEndCapture: ") + cudaGetErrorString(e));
    e = cudaGraphInstantiate(out, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) return fail(XRDVI_E_CUDA, std::string("cudaGraphInstantiate: ") + cudaGetErrorString(e));
    return XRDVI_OK;
}

int ensure_graph(xrdvi* h, int S) {
    if (h->graph_exec && h->graph_execU && h->graph_S == S) return XRDVI_OK;
    if (h->graph_exec) { cudaGraphExecDestroy(h->graph_exec); h->graph_exec = nullptr; }
    if (h->graph_execU) { cudaGraphExecDestroy(h->graph_execU); h->graph_execU = nullptr; }
    int rc = set_S(h, S);
    if (rc == XRDVI_OK) rc = capture_steps(h, 1, &h->graph_exec);
    if (rc == XRDVI_OK) rc = capture_steps(h, kUnroll, &h->graph_execU);
    if (rc != XRDVI_OK) return rc;
    h->graph_S = S;
    return XRDVI_OK;
}

// `n` optimisation steps: as many kUnroll-step graphs as fit, single-step graphs for the rest
int launch_steps(xrdvi* h, int n) {
#ifdef XRDVI_TUNING
    static const bool no_unroll = std::getenv("XRDVI_NO_UNROLL") != nullptr;   // A/B knob of the measurement build
#else
    const bool no_unroll = false;
#endif
    int i = 0;
    if (!no_unroll)
        for (; i + kUnroll <= n; i += kUnroll) CU(cudaGraphLaunch(h->graph_execU, h->stream));
    for (; i < n; ++i) CU(cudaGraphLaunch(h->graph_exec, h->stream));
    return XRDVI_OK;
}

// start of a run of optimisation steps: control block, then the draws of step step0 + 1
int begin_steps(xrdvi* h, int S, uint64_t seed) {
    int rc = ensure_graph(h, S);
    if (rc) return rc;
    set_S(h, S);
    rc = write_ctl(h, seed, h->step_host, h->step_host, -1);
    if (rc) return rc;
    launch_draw(h->dev, h->stream, h->dev.var, nullptr);
    CU(cudaGetLastError());
    return XRDVI_OK;
}

// External <-> device layout of a state-shaped array.  External (include/xrdvi.h): float [PR][2][K][C], C = 4 or 5
// (hyper.asymmetry, R30).  Device: the [PR][2][K][4] block of the four base classes, followed by [PR][2][K] for alpha.
size_t block_floats(const xrdvi* h) { return static_cast<size_t>(h->plan.PR) * (h->hyp.asymmetry ? 10 : 8) * h->K; }

int download_block(xrdvi* h, const float* dev, float* out) {   // synchronises the stream
    const size_t n = block_floats(h);
    if (!h->hyp.asymmetry) {
        CU(cudaMemcpyAsync(out, dev, sizeof(float) * n, cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
        return XRDVI_OK;
    }
    std::vector<float> tmp(n);
    CU(cudaMemcpyAsync(tmp.data(), dev, sizeof(float) * n, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    const size_t rows = static_cast<size_t>(h->plan.PR) * 2 * h->K;   // (inst, m | l, k)
    const float* a = tmp.data() + rows * 4;
    for (size_t r = 0; r < rows; ++r) {
        for (int c = 0; c < 4; ++c) out[r * 5 + c] = tmp[r * 4 + c];
        out[r * 5 + 4] = a[r];
    }
    return XRDVI_OK;
}

int upload_block(xrdvi* h, const float* in, float* dev) {      // synchronises the stream
    const size_t n = block_floats(h);
    if (!h->hyp.asymmetry) {
        CU(cudaMemcpyAsync(dev, in, sizeof(float) * n, cudaMemcpyHostToDevice, h->stream));
        CU(cudaStreamSynchronize(h->stream));
        return XRDVI_OK;
    }
    std::vector<float> tmp(n);
    const size_t rows = static_cast<size_t>(h->plan.PR) * 2 * h->K;
    float* a = tmp.data() + rows * 4;
    for (size_t r = 0; r < rows; ++r) {
        for (int c = 0; c < 4; ++c) tmp[r * 4 + c] = in[r * 5 + c];
        a[r] = in[r * 5 + 4];
    }
    CU(cudaMemcpyAsync(dev, tmp.data(), sizeof(float) * n, cudaMemcpyHostToDevice, h->stream));
    CU(cudaStreamSynchronize(h->stream));
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
    hy->optimizer = 0;
    hy->asymmetry = 0;
    hy->width_sec = 0;
    hy->alpha_mu = 1.0;        // B.2
    hy->alpha_sigma = 0.2;
    hy->general_grid = 0;
}

size_t xrdvi_workspace_bytes(int64_t N, int32_t K, int64_t M, int32_t S_max, double two_theta_step,
                             const xrdvi_hyper* hyp) {
    Plan pl;
    if (!hyp || hyp->size != sizeof(xrdvi_hyper)) return 0;
    if (!make_plan(N, K, M, S_max, two_theta_step, hyp, 0, &pl)) return 0;
    return pl.total;
}

int xrdvi_create(const double* x, int64_t N, const double* y, const double* bgin, int32_t K,
                 const int64_t* ofs, const double* pos, const double* inten, const xrdvi_hyper* hyp,
                 int32_t S_max, int device, void* cuda_stream, void* workspace, size_t workspace_bytes,
                 xrdvi** out) {
    if (!x || !y || !ofs || !pos || !inten || !hyp || !out || !workspace)
        return fail(XRDVI_E_INVALID_ARG, "null argument");
    if (hyp->size != sizeof(xrdvi_hyper)) return fail(XRDVI_E_INVALID_ARG, "xrdvi_hyper.size mismatch");
    if (hyp->likelihood != 0 && hyp->likelihood != 1)
        return fail(XRDVI_E_INVALID_ARG, "likelihood must be 0 (Gaussian) or 1 (Poisson)");
    if (hyp->optimizer != 0 && hyp->optimizer != 1)
        return fail(XRDVI_E_INVALID_ARG, "optimizer must be 0 (Adam) or 1 (natural gradient)");
    if ((hyp->asymmetry != 0 && hyp->asymmetry != 1) || (hyp->width_sec != 0 && hyp->width_sec != 1))
        return fail(XRDVI_E_INVALID_ARG, "asymmetry and width_sec must be 0 or 1");
    if (hyp->asymmetry && !(hyp->alpha_sigma > 0)) return fail(XRDVI_E_INVALID_ARG, "non-positive alpha_sigma");
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
    const double delta = (x[N - 1] - x[0]) / static_cast<double>(N - 1);   // the (mean) step
    bool uniform = true;
    double step_min = x[1] - x[0], step_max = step_min;
    for (int64_t i = 0; i < N; ++i) {
        if (std::fabs(x[i] - (x[0] + delta * static_cast<double>(i))) > 1e-6 * delta) uniform = false;
        if (i > 0) { step_min = std::min(step_min, x[i] - x[i - 1]); step_max = std::max(step_max, x[i] - x[i - 1]); }
    }
    if (!uniform && !hyp->general_grid)
        return fail(XRDVI_E_NONUNIFORM_GRID, "two_theta is not a uniform grid (set hyper.general_grid = 1 for the general path)");
    if (!uniform && step_max > 16.0 * step_min)
        return fail(XRDVI_E_NONUNIFORM_GRID, "two_theta steps differ by more than a factor 16");
    const bool general = hyp->general_grid != 0;          // the general path also takes a uniform grid
    // R31: nearest grid point of p (the lower one on a tie); beyond the grid continued with the mean step
    auto nearest = [&](double p) -> long long {
        if (uniform) return static_cast<long long>(std::floor((p - x[0]) / delta + 0.5));
        if (p <= x[0]) return -static_cast<long long>(std::floor((x[0] - p) / delta + 0.5));
        if (p >= x[N - 1]) return N - 1 + static_cast<long long>(std::floor((p - x[N - 1]) / delta + 0.5));
        const double* hi = std::lower_bound(x, x + N, p);  // first x_i >= p; 0 < hi - x < N here
        const long long i1 = hi - x, i0 = i1 - 1;
        return (x[i1] - p) < (p - x[i0]) ? i1 : i0;
    };
    for (int64_t m = 0; m < M; ++m)
        if (!std::isfinite(pos[m]) || !std::isfinite(inten[m]) || inten[m] < 0.0)
            return fail(XRDVI_E_INVALID_ARG, "peak position/intensity not finite or negative intensity");

    int dev_count = 0;
    CU(cudaGetDeviceCount(&dev_count));
    if (device < 0 || device >= dev_count) return fail(XRDVI_E_CUDA, "no such CUDA device");
    int cc_major = 0, n_sm = 0;   // two attribute queries: cudaGetDeviceProperties costs ~1 ms per call
    CU(cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, device));
    CU(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, device));
    if (cc_major != 10) return fail(XRDVI_E_NOT_SM100, "device is not compute capability 10.x (sm_100a build)");
    CU(cudaSetDevice(device));

    Plan pl;
    if (!make_plan(N, K, M, S_max, delta, hyp, n_sm, &pl)) return fail(XRDVI_E_INVALID_ARG, "sizes out of range");
    if (workspace_bytes < pl.total) return fail(XRDVI_E_WORKSPACE_TOO_SMALL, "workspace too small: need " + std::to_string(pl.total));
    if (reinterpret_cast<uintptr_t>(workspace) % 256) return fail(XRDVI_E_INVALID_ARG, "workspace not 256-byte aligned");

    // ---- fp64 preprocessing (R16) ----------------------------------------------------------------
    const int P = pl.P;
    long long n_c = pl.n_c;
    if (n_c < 0) {     // dense: every point is inside every window, wherever the peak lies
        n_c = N;
        for (int64_t m = 0; m < M; ++m) {
            const long long j = nearest(pos[m]);
            n_c = std::max<long long>(n_c, std::max<long long>(std::llabs(j), std::llabs(N - 1 - j)) + 1);
        }
    }
    if (n_c > (1ll << 29)) return fail(XRDVI_E_INVALID_ARG, "peak positions too far from the grid");
    std::vector<HostPeak> all_peaks;
    all_peaks.reserve(M);
    std::vector<double> area(K, 0.0);
    std::vector<float> sec_max(K, 1.0f);
    double imax = 0.0;
    for (int k = 0; k < K; ++k)
        for (int64_t m = ofs[k]; m < ofs[k + 1]; ++m) {
            area[k] += inten[m];
            imax = std::max(imax, inten[m]);
            const long long j = nearest(pos[m]);
            const double xj = (j >= 0 && j < N) ? x[j] : x[0] + delta * static_cast<double>(j);
            const double inv_s = hyp->width_sec ? std::cos(0.5 * pos[m] * M_PI / 180.0) : 1.0;   // R30: 1 / sec(p_m / 2)
            if (!(inv_s > 1e-3)) return fail(XRDVI_E_INVALID_ARG, "width_sec needs peak positions below 180 deg");
            sec_max[k] = std::max(sec_max[k], static_cast<float>(1.0 / inv_s));
            all_peaks.push_back({j, pos[m] - xj, inten[m], k, inv_s, pos[m]});
        }
    for (int k = 0; k < K; ++k)
        if (!(area[k] > 0.0)) return fail(XRDVI_E_EMPTY_PHASE, "phase " + std::to_string(k) + " has zero total intensity");
    const std::vector<long long> nck0(K, n_c);
    Tables tabs;
    const std::vector<double> xgrid = general ? std::vector<double>(x, x + N) : std::vector<double>();
    if (const char* terr = build_tables(pl, N, K, all_peaks, nck0, xgrid, &tabs)) return fail(XRDVI_E_INVALID_ARG, terr);

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
            if (hyp->likelihood == 1 && (!(y[p * N + i] >= 0.0) || !(b > 0.0)))   // R24
                return fail(XRDVI_E_INVALID_ARG, "Poisson likelihood needs y >= 0 and background > 0 everywhere");
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
        pat[p].ll_scale = -0.5f;
        if (hyp->likelihood == 1) {   // A16: sum_i { y ln f - f - ln y! } = sum_i { y ln(f/y) + (y - f) } + sum_i { y ln y - y - ln y! }
            double c = 0.0;
            for (int64_t i = 0; i < N; ++i) {
                const double yv = y[p * N + i];
                c += (yv > 0.0 ? yv * std::log(yv) - yv : 0.0) - std::lgamma(yv + 1.0);
            }
            pat[p].ll_const = c;
            pat[p].ll_scale = 1.0f;
        }
        m_h0[p] = static_cast<float>(std::log(eta_h / static_cast<double>(K)));               // R11
    }

    // ---- handle + upload -------------------------------------------------------------------------
    xrdvi* h = new xrdvi();
    h->plan = pl;
    h->hyp = *hyp;
    h->device = device;
    h->stream = static_cast<cudaStream_t>(cuda_stream);
    if (!h->stream) {   // the legacy default stream cannot be captured into a CUDA Graph: use a private non-blocking stream
        cudaError_t se = cudaStreamCreateWithFlags(&h->stream, cudaStreamNonBlocking);
        if (se != cudaSuccess) { delete h; return fail(XRDVI_E_CUDA, std::string("cudaStreamCreateWithFlags: ") + cudaGetErrorString(se)); }
        h->own_stream = true;
    }
    h->ws = static_cast<char*>(workspace);
    h->N = N; h->M = M; h->K = K; h->n_c = static_cast<int>(n_c);
    h->windowed = pl.n_c >= 0;
    h->delta = delta;
    h->peaks = std::move(all_peaks);
    h->xgrid = xgrid;
    h->m_h0 = m_h0;
    h->m_w0 = static_cast<float>(std::log(hyp->w_shape / hyp->w_rate));
    Dev& d = h->dev;
    char* w = h->ws;
    d.N = static_cast<int>(N); d.K = K; d.P = pl.P; d.R = pl.R; d.PR = pl.PR;
    d.n_c = static_cast<int>(n_c); d.TW = pl.TW; d.PS = pl.PS; d.n_seg = pl.n_seg; d.n_tile = pl.n_tile;
    d.likelihood = hyp->likelihood;
    d.optimizer = hyp->optimizer;
    d.delta = static_cast<float>(delta);
    // Gaussian-core half-width in POINTS: with the smallest step on a general grid (R31), and a slack that covers
    // |p_m - x_{j_m}| <= step_max / 2 in units of that step
    const double core_step = general ? step_min : delta;
    d.gcut = static_cast<float>(static_cast<double>(kGaussCut) / (2.0 * core_step));
    d.inv_delta = static_cast<float>(1.0 / core_step);
    d.general = general ? 1 : 0;
    d.reach_pad = general ? static_cast<float>(1.0 + 0.5 * step_max / step_min + 1e-3) : 1.5f;
    d.tile_off = reinterpret_cast<float*>(w + pl.o_tileoff);
    d.pk_base = reinterpret_cast<float*>(w + pl.o_pkbase);
    d.mu_inv_var = static_cast<float>(1.0 / (hyp->mu_sigma * hyp->mu_sigma));
    d.mu_logc = static_cast<float>(-std::log(hyp->mu_sigma * std::sqrt(2.0 * M_PI)));
    d.w_shape = static_cast<float>(hyp->w_shape);
    d.w_rate = static_cast<float>(hyp->w_rate);
    d.w_logc = static_cast<float>(hyp->w_shape * std::log(hyp->w_rate) - std::lgamma(hyp->w_shape));
    d.lr = static_cast<float>(hyp->lr); d.beta1 = static_cast<float>(hyp->beta1);
    d.beta2 = static_cast<float>(hyp->beta2); d.adam_eps = static_cast<float>(hyp->adam_eps);
    d.yb = reinterpret_cast<float*>(w + pl.o_yb);
    d.bg = reinterpret_cast<float*>(w + pl.o_bg);
    d.pk_tile = reinterpret_cast<PeakRec*>(w + pl.o_pkt);
    d.run_tab = reinterpret_cast<int4*>(w + pl.o_runs);
    d.share_rng = reinterpret_cast<int2*>(w + pl.o_srng);
    d.seg_order = reinterpret_cast<int*>(w + pl.o_sord);
    d.slot_ofs = reinterpret_cast<int*>(w + pl.o_sofs);
    d.pat = reinterpret_cast<PatConst*>(w + pl.o_pat);
    d.area = reinterpret_cast<double*>(w + pl.o_area);
    d.var = reinterpret_cast<float*>(w + pl.o_var);
    d.mom1 = reinterpret_cast<float*>(w + pl.o_mom1);
    d.mom2 = reinterpret_cast<float*>(w + pl.o_mom2);
    d.grad = reinterpret_cast<float*>(w + pl.o_grad);
    d.elbo = reinterpret_cast<double*>(w + pl.o_elbo);
    d.elbo_k = reinterpret_cast<double*>(w + pl.o_elbok);
    d.ll_t = reinterpret_cast<double*>(w + pl.o_llt);
    d.ll_g = reinterpret_cast<double*>(w + pl.o_llg);
    d.trace = reinterpret_cast<double*>(w + pl.o_trace);
    d.ctl = reinterpret_cast<Ctl*>(w + pl.o_ctl);
    d.lat = reinterpret_cast<float4*>(w + pl.o_lat);
    d.eps = reinterpret_cast<float4*>(w + pl.o_eps);
    d.rr = reinterpret_cast<float*>(w + pl.o_rr);
    d.ng = reinterpret_cast<int*>(w + pl.o_ng);
    d.llpart = reinterpret_cast<float*>(w + pl.o_llpart);
    d.part8 = reinterpret_cast<float*>(w + pl.o_part8);
    d.pd = nullptr;
    d.g_base = 0;
    d.dbg_first = 0;
    d.partial = reinterpret_cast<float*>(w + pl.o_partial);
    d.tile_cnt = reinterpret_cast<unsigned int*>(w + pl.o_tcnt);
    d.tile_cnt2 = d.tile_cnt + static_cast<size_t>(pl.G_max) * pl.n_tile;
    d.tile_rng = reinterpret_cast<int2*>(w + pl.o_trng);
    d.stage = 0;
    {   // dispatch chunk: as many draw groups as keep their latent records (K x 32 x 36 B each, + alpha) within 16 MB of L2
        const long long per_group = static_cast<long long>(K) * 32 * 44;
        d.g_block = static_cast<int>(std::min<long long>(std::max<long long>((16ll << 20) / per_group, 8), 65535));
#ifdef XRDVI_TUNING
        if (const char* e = std::getenv("XRDVI_G_BLOCK")) d.g_block = std::max(1, std::atoi(e));   // A/B knob
#endif
    }
    d.asym = hyp->asymmetry;
    d.sec = hyp->width_sec;
    d.model = (hyp->asymmetry || hyp->width_sec || hyp->general_grid) ? 1 : 0;
    d.alpha_mu = static_cast<float>(hyp->alpha_mu);
    d.alpha_inv_var = static_cast<float>(1.0 / (hyp->alpha_sigma * hyp->alpha_sigma));
    d.alpha_logc = static_cast<float>(-std::log(hyp->alpha_sigma * std::sqrt(2.0 * M_PI)));
    d.pk_sec = reinterpret_cast<float*>(w + pl.o_pksec);
    d.sec_max = reinterpret_cast<float*>(w + pl.o_secmax);
    const size_t a_ofs = static_cast<size_t>(pl.PR) * 8 * K;      // the alpha companion sits behind every [PR][2][K][4] block
    d.var_a = d.var + a_ofs;
    d.mom1_a = d.mom1 + a_ofs;
    d.mom2_a = d.mom2 + a_ofs;
    d.grad_a = d.grad + a_ofs;
    d.ia = reinterpret_cast<float*>(w + pl.o_ia);
    d.eps_a = reinterpret_cast<float*>(w + pl.o_epsa);
    d.parta = reinterpret_cast<float*>(w + pl.o_parta);
    set_S(h, S_max);

    cudaStream_t st = h->stream;
    auto up = [&](size_t off, const void* src, size_t bytes) {
        return cudaMemcpyAsync(w + off, src, bytes, cudaMemcpyHostToDevice, st);
    };
    cudaError_t ce = cudaSuccess;
    auto chk = [&](cudaError_t e) { if (ce == cudaSuccess) ce = e; };
    chk(up(pl.o_yb, yb.data(), sizeof(float) * yb.size()));
    chk(up(pl.o_bg, bgf.data(), sizeof(float) * bgf.size()));
    chk(up(pl.o_pat, pat.data(), sizeof(PatConst) * pat.size()));
    chk(up(pl.o_area, area.data(), sizeof(double) * area.size()));
    chk(up(pl.o_secmax, sec_max.data(), sizeof(float) * sec_max.size()));
    std::vector<float> tile_off;
    if (general) {   // R31: offsets of every tile's points from its first one, fp64 differences
        tile_off.assign(static_cast<size_t>(pl.n_tile) * kPT, 0.0f);
        for (int64_t i = 0; i < N; ++i) tile_off[i] = static_cast<float>(x[i] - x[i / kPT * kPT]);
        for (size_t i = N; i < tile_off.size(); ++i) tile_off[i] = tile_off[N - 1] + static_cast<float>(delta * (i - (N - 1)));
        chk(up(pl.o_tileoff, tile_off.data(), sizeof(float) * tile_off.size()));
    }
    chk(up(pl.o_mh0, m_h0.data(), sizeof(float) * m_h0.size()));
    chk(cudaMemsetAsync(w + pl.o_tcnt, 0, sizeof(unsigned int) * 2 * static_cast<size_t>(pl.G_max) * pl.n_tile, st));
    chk(cudaMemsetAsync(w + pl.o_trace, 0xFF, sizeof(double) * kTraceCap * pl.PR, st));
    chk(cudaStreamSynchronize(st));  // host staging vectors go out of scope below
    for (auto& e : h->ev) chk(cudaEventCreate(&e));

    if (ce != cudaSuccess) {
        delete h;
        return fail(XRDVI_E_CUDA, std::string("upload: ") + cudaGetErrorString(ce));
    }
    int rc = install_tables(h, tabs, nck0, true);
    if (rc == XRDVI_OK) {      // the update kernel's staging buffer: up to kUpdSmemCap of dynamic shared memory, sized by set_S
        set_S(h, S_max);
        cudaError_t e = cudaFuncSetAttribute(update_draw_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kUpdSmemCap);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(update_draw_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kUpdSmemCap);
        if (e != cudaSuccess) rc = fail(XRDVI_E_CUDA, std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e));
    }
    if (rc == XRDVI_OK) rc = xrdvi_reset_state(h, 0);
    if (rc != XRDVI_OK) { xrdvi_destroy(h); return rc; }
    // set-up of xrdvi_profile_static: `device` is current here; a failure only disables that entry point
    h->static_scratch_err = static_scratch_address(device, &h->static_scratch);
    *out = h;
    return XRDVI_OK;
}

void xrdvi_destroy(xrdvi* h) {
    if (!h) return;
    if (h->graph_exec) cudaGraphExecDestroy(h->graph_exec);
    if (h->graph_execU) cudaGraphExecDestroy(h->graph_execU);
    for (auto& e : h->ev) if (e) cudaEventDestroy(e);
    if (h->own_stream) { cudaStreamSynchronize(h->stream); cudaStreamDestroy(h->stream); }
    delete h;
}

int64_t xrdvi_pair_count(const xrdvi* h) { return h ? h->pairs : -1; }
int64_t xrdvi_window_halfwidth(const xrdvi* h) { return h ? h->n_c : -1; }
int32_t xrdvi_latent_classes(const xrdvi* h) { return h ? (h->hyp.asymmetry ? 5 : 4) : -1; }

// ---- per-phase (adaptive) windows, R27 ---------------------------------------------------------------
int xrdvi_set_phase_windows(xrdvi* h, const int32_t* n_ck) {
    if (!h) return fail(XRDVI_E_INVALID_ARG, "null handle");
    if (!h->windowed) return fail(XRDVI_E_INVALID_ARG, "per-phase windows need a windowed problem (window_W > 0)");
    std::vector<long long> nck(h->K, h->n_c);
    if (n_ck)
        for (int k = 0; k < h->K; ++k) {
            if (n_ck[k] < 0 || n_ck[k] > h->n_c)
                return fail(XRDVI_E_INVALID_ARG, "half-width of phase " + std::to_string(k) + " outside [0, n_c]");
            nck[k] = n_ck[k];
        }
    if (nck == h->n_ck) return XRDVI_OK;
    CU(cudaSetDevice(h->device));
    Tables tabs;
    if (const char* terr = build_tables(h->plan, h->N, h->K, h->peaks, nck, h->xgrid, &tabs)) return fail(XRDVI_E_INVALID_ARG, terr);
    return install_tables(h, tabs, nck, false);
}

int xrdvi_get_phase_windows(const xrdvi* h, int32_t* n_ck) {
    if (!h || !n_ck) return fail(XRDVI_E_INVALID_ARG, "null handle/output");
    for (int k = 0; k < h->K; ++k) n_ck[k] = static_cast<int32_t>(h->n_ck[k]);
    return XRDVI_OK;
}

int xrdvi_adapt_windows(xrdvi* h, double W, int32_t* n_ck_out) {
    if (!h) return fail(XRDVI_E_INVALID_ARG, "null handle");
    if (!h->windowed) return fail(XRDVI_E_INVALID_ARG, "per-phase windows need a windowed problem (window_W > 0)");
    if (!(W > 0.0) || !std::isfinite(W)) return fail(XRDVI_E_INVALID_ARG, "W must be positive");
    CU(cudaSetDevice(h->device));
    const int K = h->K, PR = h->plan.PR;
    std::vector<float> var(static_cast<size_t>(PR) * 10 * K);
    CU(cudaMemcpyAsync(var.data(), h->dev.var, sizeof(float) * block_floats(h), cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    const float* var_a = var.data() + static_cast<size_t>(PR) * 8 * K;   // alpha companion (R30)
    // the rule, in fp64 on the host from the fp32 state (this is table preprocessing, like create):
    // cutoff_k = max over instances of W E_q[w_k] + |E_q[mu_k]|, E_q[w] = exp(m_w + sigma_w^2 / 2)
    const long long n_min = static_cast<long long>(std::ceil(2.0 * W - 1e-9));
    std::vector<int32_t> nck(K);
    for (int k = 0; k < K; ++k) {
        double cut = 0.0;
        double smax = 1.0;      // R30: the widest peak of the phase under the sec term
        if (h->hyp.width_sec)
            for (const HostPeak& p : h->peaks) if (p.k == k) smax = std::max(smax, 1.0 / p.inv_s);
        for (int i = 0; i < PR; ++i) {
            const float* m = var.data() + static_cast<size_t>(i) * 8 * K;
            const float* l = m + 4 * static_cast<size_t>(K);
            const double sw = std::exp(static_cast<double>(l[4 * k + 2]));
            double wbar = std::exp(static_cast<double>(m[4 * k + 2]) + 0.5 * sw * sw) * smax;
            if (h->hyp.asymmetry) {   // R30: the high-angle side is alpha times wider
                const double sa = std::exp(static_cast<double>(var_a[static_cast<size_t>(i) * 2 * K + K + k]));
                const double abar = std::exp(static_cast<double>(var_a[static_cast<size_t>(i) * 2 * K + k]) + 0.5 * sa * sa);
                if (abar > 1.0) wbar *= abar;
            }
            const double ci = W * wbar + std::fabs(static_cast<double>(m[4 * k + 1]));
            if (!std::isfinite(ci)) return fail(XRDVI_E_INVALID_ARG, "non-finite variational state");
            cut = std::max(cut, ci);
        }
        long long n = static_cast<long long>(std::ceil(std::min(cut / h->delta, 4e9) - 1e-9));
        n = std::min<long long>(std::max(n, n_min), h->n_c);
        nck[k] = static_cast<int32_t>(n);
    }
    int rc = xrdvi_set_phase_windows(h, nck.data());
    if (rc) return rc;
    if (n_ck_out) std::memcpy(n_ck_out, nck.data(), sizeof(int32_t) * K);
    return XRDVI_OK;
}

int xrdvi_fit_adaptive(xrdvi* h, int32_t iterations, int32_t S, uint64_t seed, int32_t refresh_every, double W,
                       float* var_out, double* incl, double* trace) {
    int rc = check_S(h, S);
    if (rc) return rc;
    if (iterations < 0 || refresh_every < 1) return fail(XRDVI_E_INVALID_ARG, "iterations >= 0 and refresh_every >= 1 required");
    if (!h->windowed) return fail(XRDVI_E_INVALID_ARG, "per-phase windows need a windowed problem (window_W > 0)");
    if (!(W > 0.0) || !std::isfinite(W)) return fail(XRDVI_E_INVALID_ARG, "W must be positive");
    int done = 0;
    while (iterations - done > refresh_every) {
        rc = xrdvi_fit(h, refresh_every, S, seed, nullptr, nullptr,
                       trace ? trace + static_cast<size_t>(done) * h->plan.PR : nullptr);
        if (rc) return rc;
        done += refresh_every;
        rc = xrdvi_adapt_windows(h, W, nullptr);
        if (rc) return rc;
    }
    return xrdvi_fit(h, iterations - done, S, seed, var_out, incl,
                     trace ? trace + static_cast<size_t>(done) * h->plan.PR : nullptr);
}

int xrdvi_reset_state(xrdvi* h, uint64_t seed) { return xrdvi_reset_state_restart(h, seed, 0); }

int xrdvi_reset_state_restart(xrdvi* h, uint64_t seed, int32_t restart_offset) {
    if (!h) return fail(XRDVI_E_INVALID_ARG, "null handle");
    if (restart_offset < 0 || restart_offset > (1 << 30)) return fail(XRDVI_E_INVALID_ARG, "restart_offset out of range");
    CU(cudaSetDevice(h->device));
    init_state_kernel<<<h->plan.PR, 128, 0, h->stream>>>(h->dev, reinterpret_cast<const float*>(h->ws + h->plan.o_mh0),
                                                          h->m_w0, static_cast<float>(h->hyp.init_log_sigma), seed,
                                                          restart_offset);
    CU(cudaGetLastError());
    h->step_host = 0;
    h->adam_t0 = 0;
    return write_ctl(h, 0, 0, 0, -1);
}

int xrdvi_get_state(xrdvi* h, float* var_params, int64_t* step) {
    if (!h) return fail(XRDVI_E_INVALID_ARG, "null handle");
    CU(cudaSetDevice(h->device));
    if (var_params)
        if (int rc = download_block(h, h->dev.var, var_params)) return rc;
    if (step) *step = h->step_host;
    return XRDVI_OK;
}

int xrdvi_set_state(xrdvi* h, const float* var_params, int64_t step) {
    if (!h || !var_params || step < 0) return fail(XRDVI_E_INVALID_ARG, "null handle/state or negative step");
    CU(cudaSetDevice(h->device));
    const size_t b = sizeof(float) * block_floats(h);
    if (int rc = upload_block(h, var_params, h->dev.var)) return rc;
    CU(cudaMemsetAsync(h->dev.mom1, 0, b, h->stream));
    CU(cudaMemsetAsync(h->dev.mom2, 0, b, h->stream));
    h->step_host = step;
    h->adam_t0 = step;               // fresh moments: the bias correction restarts with them
    return write_ctl(h, 0, step, step, -1);
}

int xrdvi_get_optimizer_state(xrdvi* h, float* mom1, float* mom2, int64_t* adam_steps) {
    if (!h) return fail(XRDVI_E_INVALID_ARG, "null handle");
    CU(cudaSetDevice(h->device));
    if (mom1) if (int rc = download_block(h, h->dev.mom1, mom1)) return rc;
    if (mom2) if (int rc = download_block(h, h->dev.mom2, mom2)) return rc;
    if (adam_steps) *adam_steps = h->step_host - h->adam_t0;
    return XRDVI_OK;
}

int xrdvi_set_optimizer_state(xrdvi* h, const float* mom1, const float* mom2, int64_t adam_steps) {
    if (!h || !mom1 || !mom2) return fail(XRDVI_E_INVALID_ARG, "null handle/moments");
    if (adam_steps < 0 || adam_steps > h->step_host) return fail(XRDVI_E_INVALID_ARG, "adam_steps outside [0, step]");
    CU(cudaSetDevice(h->device));
    if (int rc = upload_block(h, mom1, h->dev.mom1)) return rc;
    if (int rc = upload_block(h, mom2, h->dev.mom2)) return rc;
    h->adam_t0 = h->step_host - adam_steps;
    return write_ctl(h, 0, h->step_host, h->step_host, -1);   // synchronises: the host buffers may go
}

// shared prologue of the evaluation entry points: stage var_params (or use the state), set S and the
// Philox iteration
static int begin_eval(xrdvi* h, const float* var_params, int32_t S, uint64_t seed, uint64_t iteration, const float** var) {
    int rc = check_S(h, S);
    if (rc) return rc;
    CU(cudaSetDevice(h->device));
    *var = h->dev.var;
    if (var_params) {
        float* tmp = reinterpret_cast<float*>(h->ws + h->plan.o_vartmp);
        if (int urc = upload_block(h, var_params, tmp)) return urc;
        *var = tmp;
    }
    rc = set_S(h, S);
    if (rc) return rc;
    return write_ctl(h, seed, h->step_host, h->step_host, static_cast<long long>(iteration & 0xFFFFFFFFull));
}

int xrdvi_elbo_grad(xrdvi* h, const float* var_params, int32_t S, uint64_t seed, uint64_t iteration,
                    double* elbo, float* grad) {
    const float* var = nullptr;
    int rc = begin_eval(h, var_params, S, seed, iteration, &var);
    if (rc) return rc;
    rc = enqueue_eval(h, var, nullptr, 0, false);
    if (rc) return rc;
    std::vector<double> el(elbo ? h->plan.PR : 0);
    std::vector<float> gr(grad ? block_floats(h) : 0);
    if (elbo) CU(cudaMemcpyAsync(el.data(), h->dev.elbo, sizeof(double) * h->plan.PR, cudaMemcpyDeviceToHost, h->stream));
    if (grad) { if (int drc = download_block(h, h->dev.grad, gr.data())) return drc; }
    CU(cudaStreamSynchronize(h->stream));
    if (elbo) std::memcpy(elbo, el.data(), sizeof(double) * el.size());
    if (grad) std::memcpy(grad, gr.data(), sizeof(float) * gr.size());
    return XRDVI_OK;
}

int xrdvi_fit(xrdvi* h, int32_t iterations, int32_t S, uint64_t seed, float* var_out, double* incl, double* trace) {
    int rc = check_S(h, S);
    if (rc) return rc;
    if (iterations < 0) return fail(XRDVI_E_INVALID_ARG, "iterations < 0");
    CU(cudaSetDevice(h->device));
    if (iterations > 0) {
        rc = begin_steps(h, S, seed);
        if (rc) return rc;
        rc = launch_steps(h, iterations);
        if (rc) return rc;
        rc = enqueue_finish(h);
        if (rc) return rc;
        h->step_host += iterations;
    }
    const int PR = h->plan.PR;
    std::vector<float> vo(var_out ? block_floats(h) : 0);
    std::vector<double> inc(incl ? PR * static_cast<size_t>(h->K) : 0);
    std::vector<double> tr;
    if (var_out) { if (int drc = download_block(h, h->dev.var, vo.data())) return drc; }
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

int xrdvi_posterior_summary(xrdvi* h, double* summary) {
    if (!h) return fail(XRDVI_E_INVALID_ARG, "null handle");
    if (!summary) return fail(XRDVI_E_INVALID_ARG, "summary is NULL");
    CU(cudaSetDevice(h->device));
    const size_t n = (h->hyp.asymmetry ? 25 : 20) * static_cast<size_t>(h->plan.PR) * h->K;
    double* dev = reinterpret_cast<double*>(h->ws + h->plan.o_summ);
    posterior_summary_kernel<<<dim3((h->K + 3) / 4, h->plan.PR), 128, 0, h->stream>>>(h->dev, dev);
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(summary, dev, sizeof(double) * n, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return XRDVI_OK;
}

int xrdvi_debug_profile(xrdvi* h, const float* var_params, int32_t S, uint64_t seed, uint64_t iteration,
                        int64_t first, int64_t n, float* f, double* ll, void* scratch, size_t scratch_bytes) {
    const float* var = nullptr;
    int rc = begin_eval(h, var_params, S, seed, iteration, &var);
    if (rc) return rc;
    const long long T = static_cast<long long>(h->plan.PR) * S;
    if (first < 0 || n < 0 || first + n > T) return fail(XRDVI_E_INVALID_ARG, "first / n out of range");
    float* f_dev = nullptr;
    if (f && n > 0) {
        if (!scratch || scratch_bytes < sizeof(float) * static_cast<size_t>(n) * h->N)
            return fail(XRDVI_E_WORKSPACE_TOO_SMALL, "debug_profile: scratch smaller than n * N floats");
        f_dev = static_cast<float*>(scratch);
    }
    h->dev.dbg_first = first;
    rc = enqueue_eval(h, var, f_dev, n, true);
    h->dev.dbg_first = 0;
    if (rc) return rc;
    std::vector<double> llh(static_cast<size_t>(h->plan.PR) * h->plan.S_pad);
    cudaError_t e = cudaMemcpyAsync(llh.data(), h->dev.ll_t, sizeof(double) * llh.size(), cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess && f_dev) e = cudaMemcpyAsync(f, f_dev, sizeof(float) * n * h->N, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return fail(XRDVI_E_CUDA, std::string("debug_profile: ") + cudaGetErrorString(e));
    if (ll) {
        const int gpi32 = h->dev.gpi * 32;
        for (long long t = 0; t < n; ++t) ll[t] = llh[static_cast<size_t>((first + t) / S) * gpi32 + ((first + t) % S)];
    }
    return XRDVI_OK;
}

// The same evaluation as xrdvi_debug_profile with the caller's scratch replaced by g_static_scratch: no device or host
// allocation on this path (no std::vector either), so it may be called where cudaMalloc is forbidden.
int xrdvi_profile_static(xrdvi* h, const float* var_params, int32_t S, uint64_t seed, uint64_t iteration,
                         int64_t first, int64_t n, float* f, double* ll) {
    int rc = check_S(h, S);
    if (rc) return rc;
    const long long T = static_cast<long long>(h->plan.PR) * S;
    if (first < 0 || n < 0 || first + n > T) return fail(XRDVI_E_INVALID_ARG, "profile_static: first / n out of range");
    const size_t want = f ? static_cast<size_t>(n) * static_cast<size_t>(h->N) : 0;
    if (want > kStaticScratchFloats)
        return fail(XRDVI_E_WORKSPACE_TOO_SMALL,
                    "profile_static: n * N = " + std::to_string(want) + " floats exceed the static scratch of " +
                        std::to_string(kStaticScratchFloats) + " floats (4 MiB); ask for fewer rows per call");
    if (want && !h->static_scratch)
        return fail(XRDVI_E_CUDA, std::string("profile_static: cudaGetSymbolAddress failed at create: ") +
                                      cudaGetErrorString(h->static_scratch_err));
    CU(cudaSetDevice(h->device));
    const float* var = h->dev.var;
    if (var_params) {   // external [PR][2][K][C] -> device [PR][2][K][4] (+ [PR][2][K] for alpha, R30), strided copies
        float* tmp = reinterpret_cast<float*>(h->ws + h->plan.o_vartmp);
        const size_t rows = static_cast<size_t>(h->plan.PR) * 2 * h->K;
        if (!h->hyp.asymmetry) {
            CU(cudaMemcpyAsync(tmp, var_params, sizeof(float) * rows * 4, cudaMemcpyHostToDevice, h->stream));
        } else {
            CU(cudaMemcpy2DAsync(tmp, 4 * sizeof(float), var_params, 5 * sizeof(float), 4 * sizeof(float), rows,
                                 cudaMemcpyHostToDevice, h->stream));
            CU(cudaMemcpy2DAsync(tmp + rows * 4, sizeof(float), var_params + 4, 5 * sizeof(float), sizeof(float), rows,
                                 cudaMemcpyHostToDevice, h->stream));
        }
        var = tmp;
    }
    rc = set_S(h, S);
    if (rc) return rc;
    rc = write_ctl(h, seed, h->step_host, h->step_host, static_cast<long long>(iteration & 0xFFFFFFFFull));   // synchronises
    if (rc) return rc;
    float* f_dev = want ? h->static_scratch : nullptr;
    // every call shares the array and finds the previous call's rows in it: start from zero, so that a point the kernel
    // did not write can never be read as this call's result
    if (f_dev) CU(cudaMemsetAsync(f_dev, 0, sizeof(float) * want, h->stream));
    h->dev.dbg_first = first;
    rc = enqueue_eval(h, var, f_dev, f_dev ? n : 0, true);
    h->dev.dbg_first = 0;
    if (rc) return rc;
    cudaError_t e = cudaSuccess;
    if (f_dev) e = cudaMemcpyAsync(f, f_dev, sizeof(float) * want, cudaMemcpyDeviceToHost, h->stream);
    if (ll && n > 0) {   // ll_t is [PR][gpi * 32]: one contiguous piece per instance the rows touch
        const int gpi32 = h->dev.gpi * 32;
        for (long long inst = first / S; inst <= (first + n - 1) / S && e == cudaSuccess; ++inst) {
            const long long lo = std::max<long long>(first, inst * S), hi = std::min<long long>(first + n, (inst + 1) * S);
            e = cudaMemcpyAsync(ll + (lo - first), h->dev.ll_t + static_cast<size_t>(inst) * gpi32 + (lo - inst * S),
                                sizeof(double) * static_cast<size_t>(hi - lo), cudaMemcpyDeviceToHost, h->stream);
        }
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return fail(XRDVI_E_CUDA, std::string("profile_static: ") + cudaGetErrorString(e));
    return XRDVI_OK;
}

int xrdvi_debug_draws(xrdvi* h, int32_t S, uint64_t seed, uint64_t iteration, int64_t n, float* eps, uint32_t* raw,
                      int32_t* core_halfwidth, void* scratch, size_t scratch_bytes) {
    const float* var = nullptr;
    int rc = begin_eval(h, nullptr, S, seed, iteration, &var);
    if (rc) return rc;
    const long long T = static_cast<long long>(h->plan.PR) * S;
    if (n < 0 || n > T || !eps) return fail(XRDVI_E_INVALID_ARG, "n out of range or eps NULL");
    const Dev& d = h->dev;
    const size_t cnt = static_cast<size_t>(d.G) * d.K * 32;
    if (!scratch || scratch_bytes < sizeof(uint4) * cnt)
        return fail(XRDVI_E_WORKSPACE_TOO_SMALL, "debug_draws: scratch smaller than 16 bytes per (draw slot, phase)");
    uint4* raw_dev = static_cast<uint4*>(scratch);
    launch_draw(d, h->stream, var, raw_dev);
    std::vector<float4> eh(cnt);
    std::vector<uint4> rh(cnt);
    std::vector<int> ngh(static_cast<size_t>(d.G) * d.K);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(eh.data(), d.eps, sizeof(float4) * cnt, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(rh.data(), raw_dev, sizeof(uint4) * cnt, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(ngh.data(), d.ng, sizeof(int) * ngh.size(), cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return fail(XRDVI_E_CUDA, std::string("debug_draws: ") + cudaGetErrorString(e));
    for (long long t = 0; t < n; ++t) {
        const int inst = static_cast<int>(t / S), s = static_cast<int>(t % S);
        const int g = inst * d.gpi + s / 32, lane = s % 32;
        for (int k = 0; k < d.K; ++k) {
            const size_t o = (static_cast<size_t>(g) * d.K + k) * 32 + lane;
            std::memcpy(eps + (static_cast<size_t>(t) * d.K + k) * 4, &eh[o], sizeof(float4));
            if (raw) std::memcpy(raw + (static_cast<size_t>(t) * d.K + k) * 4, &rh[o], sizeof(uint4));
            if (core_halfwidth) core_halfwidth[static_cast<size_t>(t) * d.K + k] = ngh[static_cast<size_t>(g) * d.K + k];
        }
    }
    return XRDVI_OK;
}

int xrdvi_logjoint_grad(xrdvi* h, const float* zeta, int64_t n, int32_t pattern, double* ll, double* lpj, float* grad) {
    if (!h || !zeta) return fail(XRDVI_E_INVALID_ARG, "null handle or zeta");
    if (n < 1 || n > h->plan.S_pad) return fail(XRDVI_E_INVALID_ARG, "n out of range [1, S_max rounded up to 32]");
    if (pattern < 0 || pattern >= h->plan.P) return fail(XRDVI_E_INVALID_ARG, "pattern out of range");
    CU(cudaSetDevice(h->device));
    const int K = h->K;
    const bool asym = h->hyp.asymmetry != 0;
    const size_t nk = static_cast<size_t>(n) * K;
    // device layout: float4 [n][K] for the four base classes, then float [n][K] for alpha (R30); the caller's arrays are
    // [n][K][C]
    float* zeta_dev = reinterpret_cast<float*>(h->ws + h->plan.o_zeta);
    float* grad_dev = reinterpret_cast<float*>(h->ws + h->plan.o_gradz);
    float* zeta_a = zeta_dev + 4 * static_cast<size_t>(h->plan.S_pad) * K;
    float* grad_a = grad_dev + 4 * static_cast<size_t>(h->plan.S_pad) * K;
    double* ll_dev = reinterpret_cast<double*>(h->ws + h->plan.o_lls);
    double* lpj_dev = ll_dev + h->plan.S_pad;
    float* lpk = reinterpret_cast<float*>(h->ws + h->plan.o_lpk);
    cudaStream_t st = h->stream;
    std::vector<float> z4, za;
    if (asym) {
        z4.resize(nk * 4);
        za.resize(nk);
        for (size_t r = 0; r < nk; ++r) {
            for (int c = 0; c < 4; ++c) z4[r * 4 + c] = zeta[r * 5 + c];
            za[r] = zeta[r * 5 + 4];
        }
        CU(cudaMemcpyAsync(zeta_dev, z4.data(), sizeof(float) * 4 * nk, cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(zeta_a, za.data(), sizeof(float) * nk, cudaMemcpyHostToDevice, st));
    } else {
        CU(cudaMemcpyAsync(zeta_dev, zeta, sizeof(float) * 4 * nk, cudaMemcpyHostToDevice, st));
    }
    set_S(h, static_cast<int>(n));                    // the n points take the place of the draws of one instance
    const int gpi = h->dev.gpi;
    const int inst = pattern * h->plan.R;             // restart 0 of the pattern: only its buffers are used
    for (int c0 = 0; c0 < gpi; c0 += h->plan.pd_groups) {
        const int ng = std::min(h->plan.pd_groups, gpi - c0);
        Dev dd = h->dev;
        dd.g_base = inst * gpi + c0;
        dd.G = ng;
        dd.pd = reinterpret_cast<float*>(h->ws + h->plan.o_pd);
        zeta_latent_kernel<<<dim3((K + 3) / 4, ng), 128, 0, st>>>(dd, reinterpret_cast<const float4*>(zeta_dev), zeta_a,
                                                                 static_cast<int>(n), c0);
        launch_tile<true>(dd, st, nullptr, 0);
        logjoint_grad_kernel<<<dim3(K, ng), 32, 0, st>>>(dd, reinterpret_cast<const float4*>(zeta_dev), zeta_a,
                                                        static_cast<int>(n), c0, pattern,
                                                        reinterpret_cast<float4*>(grad_dev), grad_a, lpk);
        logjoint_scalar_kernel<<<ng, 32, 0, st>>>(dd, static_cast<int>(n), c0, pattern, lpk, ll_dev, lpj_dev);
        CU(cudaGetLastError());
    }
    std::vector<double> llh(ll ? n : 0), lph(lpj ? n : 0);
    std::vector<float> gh(grad ? nk * 4 : 0), ga(grad && asym ? nk : 0);
    if (ll) CU(cudaMemcpyAsync(llh.data(), ll_dev, sizeof(double) * n, cudaMemcpyDeviceToHost, st));
    if (lpj) CU(cudaMemcpyAsync(lph.data(), lpj_dev, sizeof(double) * n, cudaMemcpyDeviceToHost, st));
    if (grad) CU(cudaMemcpyAsync(gh.data(), grad_dev, sizeof(float) * 4 * nk, cudaMemcpyDeviceToHost, st));
    if (grad && asym) CU(cudaMemcpyAsync(ga.data(), grad_a, sizeof(float) * nk, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    if (ll) std::memcpy(ll, llh.data(), sizeof(double) * n);
    if (lpj) std::memcpy(lpj, lph.data(), sizeof(double) * n);
    if (grad) {
        if (!asym) std::memcpy(grad, gh.data(), sizeof(float) * 4 * nk);
        else
            for (size_t r = 0; r < nk; ++r) {
                for (int c = 0; c < 4; ++c) grad[r * 5 + c] = gh[r * 4 + c];
                grad[r * 5 + 4] = ga[r];
            }
    }
    return XRDVI_OK;
}

int xrdvi_time_kernels(xrdvi* h, int32_t S, uint64_t seed, int32_t reps, float* ms /* [4] */) {
    int rc = check_S(h, S);
    if (rc) return rc;
    if (reps < 1 || !ms) return fail(XRDVI_E_INVALID_ARG, "reps < 1 or ms NULL");
    CU(cudaSetDevice(h->device));
    rc = set_S(h, S);
    if (rc) return rc;
    rc = write_ctl(h, seed, h->step_host, h->step_host, -1);
    if (rc) return rc;
    const Dev& d = h->dev;
    cudaStream_t st = h->stream;
    double tt = 0.0, tf = 0.0, tu = 0.0, ti = 0.0;
    for (int r = 0; r < reps + 1; ++r) {   // first pass is a warm-up
        CU(cudaEventRecord(h->ev[0], st));
        launch_draw(d, st, d.var, nullptr);
        CU(cudaEventRecord(h->ev[1], st));
        launch_tile<true>(d, st, nullptr, 0);
        CU(cudaEventRecord(h->ev[2], st));
        update_draw_kernel<false><<<dim3(d.K + d.gpi, d.PR), kUpdThreads, d.upd_smem, st>>>(d, d.var, 0);
        CU(cudaEventRecord(h->ev[3], st));
        launch_tile<false>(d, st, nullptr, 0);
        CU(cudaEventRecord(h->ev[4], st));
        CU(cudaGetLastError());
        CU(cudaStreamSynchronize(st));
        if (r == 0) continue;
        float a = 0, b = 0, c = 0, e = 0;
        CU(cudaEventElapsedTime(&a, h->ev[1], h->ev[2]));
        CU(cudaEventElapsedTime(&b, h->ev[2], h->ev[3]));
        CU(cudaEventElapsedTime(&c, h->ev[3], h->ev[4]));
        CU(cudaEventElapsedTime(&e, h->ev[0], h->ev[3]));
        tt += a; tu += b; tf += c; ti += e;
    }
    ms[0] = static_cast<float>(tt / reps);
    ms[1] = static_cast<float>(tf / reps);
    ms[2] = static_cast<float>(tu / reps);
    ms[3] = static_cast<float>(ti / reps);
    return XRDVI_OK;
}

int xrdvi_debug_timeline(xrdvi* h, int32_t S, uint64_t seed, int64_t capacity, uint64_t* rows, int64_t* n_rows,
                         void* scratch, size_t scratch_bytes) {
    int rc = check_S(h, S);
    if (rc) return rc;
    if (!rows || !n_rows || capacity < 1) return fail(XRDVI_E_INVALID_ARG, "rows / n_rows NULL or capacity < 1");
    CU(cudaSetDevice(h->device));
    rc = set_S(h, S);
    if (rc) return rc;
    rc = write_ctl(h, seed, h->step_host, h->step_host, -1);
    if (rc) return rc;
    Dev d = h->dev;                                       // a copy with the stamp buffer attached
    const long long warps = use_split(d) ? 2ll * d.n_tile * d.PS * d.G : static_cast<long long>(d.n_seg) * d.G * d.TW * d.PS;
    if (warps > capacity) return fail(XRDVI_E_INVALID_ARG, "capacity < warps of the launch");
    if (!scratch || scratch_bytes < sizeof(unsigned long long) * 4 * static_cast<size_t>(warps))
        return fail(XRDVI_E_WORKSPACE_TOO_SMALL, "debug_timeline: scratch smaller than 32 bytes per warp of the launch");
    unsigned long long* buf = static_cast<unsigned long long*>(scratch);
    cudaStream_t st = h->stream;
    cudaError_t e = cudaSuccess;
    for (int pass = 0; pass < 3 && e == cudaSuccess; ++pass) {       // two warm-up passes, the third is stamped
        launch_draw(h->dev, st, h->dev.var, nullptr);
        d.tl = pass == 2 ? buf : nullptr;
        if (pass == 2) e = cudaMemsetAsync(buf, 0, sizeof(unsigned long long) * 4 * warps, st);
        launch_tile<true>(d, st, nullptr, 0);
        update_draw_kernel<false><<<dim3(d.K + d.gpi, d.PR), kUpdThreads, h->dev.upd_smem, st>>>(h->dev, h->dev.var, 0);
        if (e == cudaSuccess) e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(rows, buf, sizeof(unsigned long long) * 4 * warps, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return fail(XRDVI_E_CUDA, std::string("debug_timeline: ") + cudaGetErrorString(e));
    *n_rows = warps;
    return enqueue_finish(h) ? XRDVI_E_CUDA : XRDVI_OK;
}

int xrdvi_debug_update_timeline(xrdvi* h, int32_t steps, int32_t S, uint64_t seed, int64_t capacity, uint64_t* rows,
                                int64_t* n_rows, void* scratch, size_t scratch_bytes) {
    int rc = check_S(h, S);
    if (rc) return rc;
    if (steps < 2 || !rows || !n_rows) return fail(XRDVI_E_INVALID_ARG, "steps < 2 or NULL output");
    CU(cudaSetDevice(h->device));
    rc = begin_steps(h, S, seed);
    if (rc) return rc;
    const Dev& d = h->dev;
    const long long n_cta = static_cast<long long>(d.K + d.gpi) * d.PR;
    if (n_cta + 1 > capacity) return fail(XRDVI_E_INVALID_ARG, "capacity < CTAs of update_draw_kernel + 1");
    // the tile kernel of the step after the stamped one leaves its per-warp stamps (as in xrdvi_debug_timeline) behind the
    // update kernel's rows: the earliest of them is the time at which the next step could begin
    const long long warps = use_split(d) ? 2ll * d.n_tile * d.PS * d.G : static_cast<long long>(d.n_seg) * d.G * d.TW * d.PS;
    const size_t u_bytes = sizeof(unsigned long long) * 8 * static_cast<size_t>(n_cta);
    const size_t t_bytes = sizeof(unsigned long long) * 4 * static_cast<size_t>(warps);
    if (!scratch || scratch_bytes < u_bytes + 2 * t_bytes)
        return fail(XRDVI_E_WORKSPACE_TOO_SMALL,
                    "debug_update_timeline: scratch smaller than 64 bytes per CTA of the update kernel + 64 per warp of the tile kernel");
    unsigned long long* buf = static_cast<unsigned long long*>(scratch);
    unsigned long long* buf_t = buf + 8 * n_cta;            // tile kernel of the step after the stamped update kernel
    unsigned long long* buf_t0 = buf_t + 4 * warps;         // tile kernel of the same step
    cudaStream_t st = h->stream;
    cudaError_t e = cudaMemsetAsync(buf, 0, u_bytes + 2 * t_bytes, st);
    // the steps as xrdvi_fit enqueues them (programmatic launches), outside a graph
    for (int i = 0; i < steps && e == cudaSuccess && rc == XRDVI_OK; ++i) {
        h->dev.tlu = i == steps - 2 ? buf : nullptr;
        h->dev.tl = i == steps - 1 ? buf_t : i == steps - 2 ? buf_t0 : nullptr;
        rc = enqueue_step(h);
    }
    h->dev.tlu = nullptr;
    h->dev.tl = nullptr;
    if (rc == XRDVI_OK) rc = enqueue_finish(h);
    if (rc == XRDVI_OK) h->step_host += steps;
    std::vector<unsigned long long> tl(static_cast<size_t>(warps) * 8);
    if (e == cudaSuccess) e = cudaMemcpyAsync(rows, buf, u_bytes, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(tl.data(), buf_t, 2 * t_bytes, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return fail(XRDVI_E_CUDA, std::string("debug_update_timeline: ") + cudaGetErrorString(e));
    if (rc != XRDVI_OK) return rc;
    unsigned long long first = 0, last_end = 0;              // next tile kernel's first start; this step's tile kernel's last end
    for (long long w = 0; w < warps; ++w) {
        if (tl[4 * w] && (!first || tl[4 * w] < first)) first = tl[4 * w];
        last_end = std::max(last_end, tl[4 * (warps + w) + 2]);
    }
    for (int c = 0; c < 8; ++c) rows[8 * n_cta + c] = c == 0 ? first : c == 1 ? last_end : 0;
    *n_rows = n_cta + 1;
    return XRDVI_OK;
}

int xrdvi_bench_steps(xrdvi* h, int32_t steps, int32_t S, uint64_t seed, void* flush, size_t flush_bytes, float* ms_steps) {
    int rc = check_S(h, S);
    if (rc) return rc;
    if (steps < 1 || !ms_steps) return fail(XRDVI_E_INVALID_ARG, "steps < 1 or ms_steps NULL");
    CU(cudaSetDevice(h->device));
    rc = begin_steps(h, S, seed);
    if (rc) return rc;
    if (!flush) flush_bytes = 0;
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
    if (e == cudaSuccess) { finish_step_kernel<<<1, 256, 0, h->stream>>>(h->dev); e = cudaGetLastError(); }
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    h->step_host += steps;
    for (int i = 0; i < steps && e == cudaSuccess; ++i) e = cudaEventElapsedTime(&ms_steps[i], ev[2 * i], ev[2 * i + 1]);
    for (auto& x : ev) if (x) cudaEventDestroy(x);
    if (e != cudaSuccess) return fail(XRDVI_E_CUDA, std::string("bench_steps: ") + cudaGetErrorString(e));
    return XRDVI_OK;
}

}  // extern "C"
