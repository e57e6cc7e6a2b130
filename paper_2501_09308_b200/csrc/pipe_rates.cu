// pipe_rates.cu -- microbenchmark of the SM issue / FP32 / MUFU rates that bound the hot path.
// Measured, not assumed: the ALU roofline bench.py reports divides by these per-SM, per-clock rates
// (DESIGN.md "Roofline").  One CTA of 1024 threads per SM; every thread runs `iters` rounds of 8
// independent dependency chains of one instruction kind; cycles come from clock64() inside the kernel,
// so the figures are per SM clock, independent of the clock frequency.
#include "../../include/xrdvi_measure.h"

enum { XRDVI_OK = 0, XRDVI_E_INVALID_ARG = -1, XRDVI_E_CUDA = -6, XRDVI_E_NOT_SM100 = -7 };   // as include/xrdvi.h

#include <cuda_runtime.h>
#include <string>
#include <vector>

namespace {

enum Kind { kFfma = 0, kFfma2 = 1, kEx2 = 2, kRcp = 3, kMixFwd = 4, kMixBwd = 5, kFmul2Mix = 6, kEx2Rcp = 7, kNumKinds = 8 };

template <int KIND>
__global__ void __launch_bounds__(1024) rate_kernel(int iters, float seed, float* sink, long long* cycles) {
    float x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = seed + 0.001f * static_cast<float>(threadIdx.x + i);
    const float a = 0.999f, b = 0.0001f;
    unsigned long long xa = 0, xb = 0, xx[8];
    if (KIND == kFfma2 || KIND == kFmul2Mix) {
        asm volatile("mov.b64 %0, {%1, %1};" : "=l"(xa) : "f"(a));
        asm volatile("mov.b64 %0, {%1, %1};" : "=l"(xb) : "f"(b));
#pragma unroll
        for (int i = 0; i < 8; ++i) asm volatile("mov.b64 %0, {%1, %1};" : "=l"(xx[i]) : "f"(x[i]));
    }
    __syncthreads();
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
        if (KIND == kFfma) {
#pragma unroll
            for (int i = 0; i < 8; ++i) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(x[i]) : "f"(a), "f"(b));
        } else if (KIND == kFfma2) {
#pragma unroll
            for (int i = 0; i < 8; ++i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(xx[i]) : "l"(xa), "l"(xb));
        } else if (KIND == kEx2) {
#pragma unroll
            for (int i = 0; i < 8; ++i) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(x[i]));
        } else if (KIND == kRcp) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {   // rcp followed by an add: ptxas folds rcp(rcp(x)) otherwise
                asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(x[i]));
                asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(x[i]) : "f"(a));
            }
        } else if (KIND == kEx2Rcp) {       // 4 ex2 chains + 4 (rcp, add) chains: is the MUFU rate shared?
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(x[i]));
                asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(x[i + 4]));
                asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(x[i + 4]) : "f"(a));
            }
        } else if (KIND == kMixFwd) {   // 5 FP32 + 2 MUFU per "pair" (plain forward), 4 pairs per round
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(x[i]) : "f"(a), "f"(b));
                asm volatile("mul.rn.f32 %0, %1, %1;" : "=f"(x[i + 4]) : "f"(x[i]));
                asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(x[i + 4]));
                asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(x[i]) : "f"(a), "f"(x[i + 4]));
                asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(x[i + 4]) : "f"(a));
                asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(x[i + 4]));
                asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(x[i]) : "f"(b), "f"(x[i + 4]));
            }
        } else if (KIND == kMixBwd) {   // 14 FP32 + 2 MUFU per pair (plain backward), 2 pairs per round
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(x[i + 2]) : "f"(x[i]));
                asm volatile("rcp.approx.ftz.f32 %0, %1;" : "=f"(x[i + 4]) : "f"(x[i]));
#pragma unroll
                for (int j = 0; j < 7; ++j) {
                    asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(x[i + 6]) : "f"(x[i + 2]), "f"(a));
                    asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(x[i]) : "f"(x[i + 4]), "f"(b));
                }
            }
        } else {                        // kFmul2Mix: 7 packed FP32x2 + 2 MUFU per pair-of-pairs
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(x[i + 2]) : "f"(x[i]));
                asm volatile("rcp.approx.ftz.f32 %0, %1;" : "=f"(x[i + 4]) : "f"(x[i]));
#pragma unroll
                for (int j = 0; j < 7; ++j)
                    asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(xx[i * 4 + (j & 3)]) : "l"(xa), "l"(xb));
            }
        }
    }
    const long long t1 = clock64();
    float acc = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        acc += x[i];
        float lo, hi;
        asm volatile("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(xx[i]));
        acc += lo + hi;
    }
    if (acc == 123.456f) sink[0] = acc;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

thread_local std::string g_err2;

}  // namespace

extern "C" {

// rates float [9]: lane-operations per SM clock of
//  [0] FFMA (3-register), [1] FFMA2 counted as 2 FMAs per lane, [2] MUFU.EX2, [3] MUFU.RCP,
//  [4] warp-instruction issue rate x32 of the plain forward mix (5 FP32 : 2 MUFU),
//  [5] same for the plain backward mix (14 FP32 : 2 MUFU), [6] same for 7 FFMA2 : 2 MUFU,
//  [7] MUFU operations of 4 EX2 + 4 RCP chains run together (is the 16/clk rate shared?),
//  [8] SM clock in MHz during the run (cycles / CUDA-event time of the FFMA kernel).
int xrdvi_pipe_rates(int device, float* rates) {
    if (!rates) return XRDVI_E_INVALID_ARG;
    if (cudaSetDevice(device) != cudaSuccess) return XRDVI_E_CUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return XRDVI_E_CUDA;
    if (prop.major != 10) return XRDVI_E_NOT_SM100;
    const int n_sm = prop.multiProcessorCount, iters = 16384;
    float* sink = nullptr;
    long long* cyc = nullptr;
    if (cudaMalloc(&sink, 64) != cudaSuccess || cudaMalloc(&cyc, sizeof(long long) * n_sm) != cudaSuccess) return XRDVI_E_CUDA;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    std::vector<long long> h(n_sm);
    // lane-operations per thread per round for each kind
    const double ops_per_round[kNumKinds] = {8, 16, 8, 8, 28, 32, 18, 8};
    for (int kind = 0; kind < kNumKinds; ++kind) {
        float ms = 0.f;
        for (int rep = 0; rep < 2; ++rep) {   // rep 0 warms up
            cudaEventRecord(e0);
            switch (kind) {
                case kFfma: rate_kernel<kFfma><<<n_sm, 1024>>>(iters, 1.0f, sink, cyc); break;
                case kFfma2: rate_kernel<kFfma2><<<n_sm, 1024>>>(iters, 1.0f, sink, cyc); break;
                case kEx2: rate_kernel<kEx2><<<n_sm, 1024>>>(iters, 1.0f, sink, cyc); break;
                case kRcp: rate_kernel<kRcp><<<n_sm, 1024>>>(iters, 1.0f, sink, cyc); break;
                case kMixFwd: rate_kernel<kMixFwd><<<n_sm, 1024>>>(iters, 1.0f, sink, cyc); break;
                case kMixBwd: rate_kernel<kMixBwd><<<n_sm, 1024>>>(iters, 1.0f, sink, cyc); break;
                case kEx2Rcp: rate_kernel<kEx2Rcp><<<n_sm, 1024>>>(iters, 1.0f, sink, cyc); break;
                default: rate_kernel<kFmul2Mix><<<n_sm, 1024>>>(iters, 1.0f, sink, cyc); break;
            }
            cudaEventRecord(e1);
            if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(sink); cudaFree(cyc); return XRDVI_E_CUDA; }
            cudaEventElapsedTime(&ms, e0, e1);
        }
        cudaMemcpy(h.data(), cyc, sizeof(long long) * n_sm, cudaMemcpyDeviceToHost);
        double mean = 0.0;
        for (long long c : h) mean += static_cast<double>(c);
        mean /= n_sm;
        rates[kind] = static_cast<float>(1024.0 * iters * ops_per_round[kind] / mean);
        if (kind == kFfma) rates[8] = static_cast<float>(mean / (ms * 1e-3) / 1e6);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    cudaFree(cyc);
    return XRDVI_OK;
}

}  // extern "C"
