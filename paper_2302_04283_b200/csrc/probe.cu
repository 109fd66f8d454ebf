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

// NM independent DMMA m8n8k4 accumulator chains and NF independent DFMA chains per thread, interleaved: do the FP64 matrix
// instruction and the scalar FP64 instruction draw on the same pipe?
template <int NM, int NF>
__global__ void __launch_bounds__(512) k_probe_pipes(double *out, int iters, double a, double b) {
    double c0[NM > 0 ? NM : 1], c1[NM > 0 ? NM : 1], x[NF > 0 ? NF : 1];
#pragma unroll
    for (int q = 0; q < NM; q++) { c0[q] = threadIdx.x; c1[q] = q; }
#pragma unroll
    for (int q = 0; q < NF; q++) x[q] = threadIdx.x + q;
    const double A = a + threadIdx.x, B = b;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int q = 0; q < NM; q++)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};" : "+d"(c0[q]), "+d"(c1[q]) : "d"(A), "d"(B));
#pragma unroll
        for (int q = 0; q < NF; q++) x[q] = fma(x[q], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < NM; q++) s += c0[q] + c1[q];
#pragma unroll
    for (int q = 0; q < NF; q++) s += x[q];
    if (s == 123.456) out[0] = s;
}

template <int NM, int NF>
double time_pipes(double *d, int blocks, int iters, long long *launches) {
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 3; rep++) {
        cudaEventRecord(e0, 0);
        k_probe_pipes<NM, NF><<<blocks, 512>>>(d, iters, 0.999999, 1e-9);
        cudaEventRecord(e1, 0);
        if (cudaEventSynchronize(e1) != cudaSuccess) { best = -1.f; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
        if (launches) (*launches)++;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return best;
}

}  // namespace

// out[0..5]: multiply-add lane operations per second of (DMMA alone, DFMA alone, DMMA in the mix, DFMA in the mix, DMMA in a mix with
// fewer matrix chains, DFMA in that mix); one DMMA m8n8k4 = 256 multiply-adds.  16 warps per SM.  Returns 0 on success.
int probe_fp64_pipes(double *out6, long long *launches) {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1;
    double *d = nullptr;
    if (cudaMalloc((void **)&d, sizeof(double)) != cudaSuccess) return -1;
    const int iters = 1 << 13, blocks = sms;
    const double warps = (double)blocks * 16, thr = warps * 32;
    const double t_m = time_pipes<4, 0>(d, blocks, iters, launches), t_f = time_pipes<0, 8>(d, blocks, iters, launches);
    const double t_mix = time_pipes<4, 8>(d, blocks, iters, launches), t_mix1 = time_pipes<1, 8>(d, blocks, iters, launches);
    cudaFree(d);
    if (t_m <= 0 || t_f <= 0 || t_mix <= 0 || t_mix1 <= 0) return -1;
    out6[0] = warps * 4 * 256.0 * iters / (t_m * 1e-3);
    out6[1] = thr * 8 * (double)iters / (t_f * 1e-3);
    out6[2] = warps * 4 * 256.0 * iters / (t_mix * 1e-3);
    out6[3] = thr * 8 * (double)iters / (t_mix * 1e-3);
    out6[4] = warps * 1 * 256.0 * iters / (t_mix1 * 1e-3);
    out6[5] = thr * 8 * (double)iters / (t_mix1 * 1e-3);
    return 0;
}

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
