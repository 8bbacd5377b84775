// qlga_peak.cu -- issue-rate microbenchmarks of the plain floating-point pipes (sm_100a): the measured
// denominator of the "alu" roofline ("measure with an FMA microbenchmark").
//
// Every thread runs NCHAIN independent dependent chains of one instruction kind (DFMA, FFMA, or the packed
// two-wide FFMA2), 1024 resident threads per SM, so that neither latency nor occupancy limits the issue
// rate; the result is counted in thread-instructions (one per lane: an FFMA2 counts as two).  Two clocks:
// CUDA events around the launch (instructions per second at the clock the GPU held) and clock64() inside
// the kernel (instructions per SM cycle, independent of the clock).
#include <stdint.h>
#include "qlga_internal.h"

namespace qlga {

constexpr int NCHAIN = 8;

template <int KIND>
__global__ void __launch_bounds__(256, 4) peak_kernel(double a, double b, int iters, double* sink,
                                                      unsigned long long* cycles) {
    const long long t0 = clock64();
    const double seed = 1.0 + 1e-9 * (double)(blockIdx.x * blockDim.x + threadIdx.x);
    double acc = 0.0;
    if (KIND == 0) {
        double x[NCHAIN];
#pragma unroll
        for (int k = 0; k < NCHAIN; ++k) x[k] = seed + k;
#pragma unroll 1
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int k = 0; k < NCHAIN; ++k) x[k] = fma(x[k], a, b);
        }
#pragma unroll
        for (int k = 0; k < NCHAIN; ++k) acc += x[k];
    } else if (KIND == 1) {
        float x[NCHAIN];
        const float fa = (float)a, fb = (float)b;
#pragma unroll
        for (int k = 0; k < NCHAIN; ++k) x[k] = (float)seed + k;
#pragma unroll 1
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int k = 0; k < NCHAIN; ++k) x[k] = fmaf(x[k], fa, fb);
        }
#pragma unroll
        for (int k = 0; k < NCHAIN; ++k) acc += x[k];
    } else {
        float2 x[NCHAIN];
        const float2 fa = make_float2((float)a, (float)a), fb = make_float2((float)b, (float)b);
#pragma unroll
        for (int k = 0; k < NCHAIN; ++k) x[k] = make_float2((float)seed + k, (float)seed - k);
#pragma unroll 1
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int k = 0; k < NCHAIN; ++k) x[k] = __ffma2_rn(x[k], fa, fb);
        }
#pragma unroll
        for (int k = 0; k < NCHAIN; ++k) acc += x[k].x + x[k].y;
    }
    const long long t1 = clock64();
    if (acc == 12345.6789) *sink = acc;                 // keeps the chains alive
    if (threadIdx.x == 0) atomicMax(cycles, (unsigned long long)(t1 - t0));
}

}  // namespace qlga

using namespace qlga;

// include/qlga.h: qlga_issue_peak
extern "C" qlga_status qlga_issue_peak(int kind, void* cuda_stream, double* instr_per_s,
                                       double* instr_per_clk_per_sm, double* ms_out) {
    if (kind < 0 || kind > 2 || !instr_per_s || !instr_per_clk_per_sm) return QLGA_EINVAL;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return QLGA_ECUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return QLGA_ECUDA;
    double* sink = nullptr;
    unsigned long long* cyc = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    qlga_status st = QLGA_ECUDA;
    const int iters = 16384, blocks = sms * 4, threads = 256;
    const double per_thread = (double)iters * 4 * NCHAIN * (kind == 2 ? 2 : 1);
    float ms = 0.f, best = 1e30f;
    unsigned long long hc = 0, best_cyc = ~0ull;
    if (cudaMalloc(&sink, sizeof(double)) != cudaSuccess) goto done;
    if (cudaMalloc(&cyc, sizeof(unsigned long long)) != cudaSuccess) goto done;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) goto done;
    for (int rep = 0; rep < 4; ++rep) {                  // the first launch warms up; best of the next three
        if (cudaMemsetAsync(cyc, 0, sizeof(unsigned long long), stream) != cudaSuccess) goto done;
        cudaEventRecord(e0, stream);
        if (kind == 0) peak_kernel<0><<<blocks, threads, 0, stream>>>(0.999999, 1e-6, iters, sink, cyc);
        else if (kind == 1) peak_kernel<1><<<blocks, threads, 0, stream>>>(0.999999, 1e-6, iters, sink, cyc);
        else peak_kernel<2><<<blocks, threads, 0, stream>>>(0.999999, 1e-6, iters, sink, cyc);
        cudaEventRecord(e1, stream);
        if (cudaGetLastError() != cudaSuccess) goto done;
        if (cudaEventSynchronize(e1) != cudaSuccess) goto done;
        cudaEventElapsedTime(&ms, e0, e1);
        if (cudaMemcpy(&hc, cyc, sizeof(hc), cudaMemcpyDeviceToHost) != cudaSuccess) goto done;
        if (rep > 0 && ms < best) best = ms;
        if (rep > 0 && hc < best_cyc) best_cyc = hc;
    }
    *instr_per_s = per_thread * blocks * threads / (best * 1e-3);
    // four 256-thread CTAs are resident per SM and run side by side for the whole kernel
    *instr_per_clk_per_sm = per_thread * 4 * threads / (double)best_cyc;
    if (ms_out) *ms_out = best;
    st = QLGA_OK;
done:
    if (st != QLGA_OK) cudaGetLastError();
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(sink); cudaFree(cyc);
    return st;
}
