// probe.cu -- measurement helper, not part of the stage: the FP64 fused-multiply-add issue rate of the device.
//
// The stage kernel is bound by FP64 arithmetic as much as by HBM, and the driver-written
// MEASURED_PEAKS.json holds no FP64 figure, so bench.py measures the denominator of its "alu" roofline live:
// every thread runs kChains independent dependent-DFMA chains (enough to cover the pipe latency at full
// occupancy); the rate is DFMA lane-operations per second over all SMs, timed with CUDA events.
#include "rad_internal.h"

namespace rad {
namespace {

constexpr int kChains = 8;

__global__ void __launch_bounds__(256) k_probe_dfma(double *out, int iters, double a, double b) {
    double x[kChains];
#pragma unroll
    for (int q = 0; q < kChains; q++) x[q] = threadIdx.x + q;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int q = 0; q < kChains; q++) x[q] = fma(x[q], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < kChains; q++) s += x[q];
    if (s == 123.456) out[0] = s;  // never true for the arguments used; keeps the chains alive
}

}  // namespace

// returns 0 on success; *dfma_per_sec = lane-level DFMA operations per second (x2 = FP64 flop/s)
int probe_dfma_rate(double *dfma_per_sec, long long *launches) {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1;
    double *d = nullptr;
    if (cudaMalloc((void **)&d, sizeof(double)) != cudaSuccess) return -1;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int iters = 1 << 14, blocks = sms * 8, threads = 256;
    double best = 0.0;
    for (int rep = 0; rep < 5; rep++) {
        cudaEventRecord(e0, 0);
        k_probe_dfma<<<blocks, threads>>>(d, iters, 0.999999, 1e-9);
        cudaEventRecord(e1, 0);
        if (cudaEventSynchronize(e1) != cudaSuccess) { best = -1.0; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double rate = (double)blocks * threads * kChains * (double)iters / (ms * 1e-3);
        if (rep > 0 && rate > best) best = rate;  // first repetition is warm-up
        if (launches) (*launches)++;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(d);
    if (best <= 0.0) return -1;
    *dfma_per_sec = best;
    return 0;
}

}  // namespace rad
