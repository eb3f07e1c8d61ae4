// mf_probe.cu — FP64-pipe micro-benchmarks behind mf_probe_fp64(): the measured denominators of the
// "alu" roofline in bench.py (MEASURED_PEAKS.json has no FP64 entry).  Register-only loops, 8 independent
// chains per thread so that latency is covered, grid = 8 CTAs of 256 threads per SM.
#include "mf_kernels.h"

namespace mf {

constexpr int CH = 8;

template <int OP>
__global__ void __launch_bounds__(256) k_probe(double* out, int iters, double seed, long long* cycles)
{
    double x[CH], y[CH], z[CH];
#pragma unroll
    for (int c = 0; c < CH; ++c) { x[c] = seed + 1e-3 * (threadIdx.x + c); y[c] = 1.0 + 1e-9 * (threadIdx.x + c) * seed; z[c] = 1e-9 * (threadIdx.x - c) * seed; }
    const double a = 1.0 + 1e-9, b = 1e-9;
    long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int c = 0; c < CH; ++c) {
            if (OP == 0) x[c] = fma(x[c], a, b);
            if (OP == 1) x[c] = x[c] + b;
            if (OP == 2) x[c] = x[c] * a;
            if (OP == 3) x[c] = 1.0 / (x[c] + 0.5);
            if (OP == 4) x[c] = sqrt(x[c] + 2.0);
            if (OP == 5) x[c] = fma(y[c], z[c], x[c]);   // three distinct register operands: the register file needs 3 cycles for them
        }
    }
    long long t1 = clock64();
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < CH; ++c) s += x[c] + (OP == 5 ? y[c] + z[c] : 0.0);
    if (s == 123.456) out[0] = s;             // keeps the loop alive
    if (blockIdx.x == 0 && threadIdx.x == 0 && cycles) *cycles = t1 - t0;
}

template <int OP>
static double run_probe(int sms, int iters, double* d_out, long long* d_cyc, double* clock_hz)
{
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int grid = sms * 8;
    k_probe<OP><<<grid, 256>>>(d_out, iters / 8, 1.0, nullptr);      // warm-up
    cudaEventRecord(e0);
    k_probe<OP><<<grid, 256>>>(d_out, iters, 1.0, d_cyc);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (clock_hz) {
        long long cyc = 0;
        cudaMemcpy(&cyc, d_cyc, sizeof(cyc), cudaMemcpyDeviceToHost);
        *clock_hz = (double)cyc / (ms * 1e-3);                        // block 0 ran for ~ the whole kernel
    }
    return (double)grid * 256.0 * CH * (double)iters / (ms * 1e-3);
}

int probe_fp64(double out[8])
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return -1;
    double* d_out = nullptr;
    long long* d_cyc = nullptr;
    if (cudaMalloc(&d_out, 64) != cudaSuccess || cudaMalloc(&d_cyc, 8) != cudaSuccess) return -1;
    const int sms = prop.multiProcessorCount;
    double hz = 0.0;
    out[0] = run_probe<0>(sms, 1 << 14, d_out, d_cyc, &hz);
    out[1] = run_probe<1>(sms, 1 << 14, d_out, d_cyc, nullptr);
    out[2] = run_probe<2>(sms, 1 << 14, d_out, d_cyc, nullptr);
    out[3] = run_probe<3>(sms, 1 << 11, d_out, d_cyc, nullptr);
    out[4] = run_probe<4>(sms, 1 << 11, d_out, d_cyc, nullptr);
    out[5] = hz;
    out[6] = (double)sms;
    out[7] = run_probe<5>(sms, 1 << 14, d_out, d_cyc, nullptr);
    cudaFree(d_out); cudaFree(d_cyc);
    return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

} // namespace mf
