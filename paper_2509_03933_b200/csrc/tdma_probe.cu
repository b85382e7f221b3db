// fp64 ALU probe ("fp64 peak is not in MEASURED_PEAKS.json; measure it").  The path is
// bound by HBM in its general form, but its serial chains are chains of dependent fp64 multiply-adds
// and reciprocals, and the shared-coefficient form (16 B per real cell) moves so few bytes per
// flop that the fp64 pipe becomes the second roofline.  tdma_probe_fp64 measures, on the current
// device: the DFMA issue rate with many independent chains (throughput) and the cycles per
// dependent DFMA, per dependent Newton reciprocal (rcp_nr of tdma_fused_tma.cuh) and per IEEE division.
#include "../../include/tdma.h"

#include <cuda_runtime.h>

namespace {

__device__ __forceinline__ double rcp_nr_probe(double x)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    double e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    e = fma(-x, r, 1.0);
    return fma(r, e, r);
}

// 8 independent chains per thread, `iters` rounds: 8 * iters DFMA per thread
__global__ void __launch_bounds__(256) dfma_throughput_kernel(double *out, double a, double b, int iters)
{
    double v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = (double)(threadIdx.x + i);
    for (int n = 0; n < iters; ++n) {
#pragma unroll
        for (int i = 0; i < 8; ++i) v[i] = fma(v[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += v[i];
    if (s == 123.456) out[0] = s;          // never true: keeps the chains alive
}

// one warp, one dependent chain: cycles per operation
template <int OP>
__global__ void latency_kernel(double *out, long long *cycles, double a, double b, int iters)
{
    double v = a;
    const long long t0 = clock64();
    for (int n = 0; n < iters; ++n) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            if (OP == 0) v = fma(v, a, b);
            else if (OP == 1) v = rcp_nr_probe(v) + b;     // + b keeps v away from a fixed point
            else v = b / v + a;
        }
    }
    const long long t1 = clock64();
    if (threadIdx.x == 0) { cycles[0] = t1 - t0; out[0] = v; }
}

}  // namespace

extern "C" int tdma_probe_fp64(double *result, int n)
{
    if (!result || n < 6) return TDMA_ERR_INVALID_ARG;
    int dev = 0, sms = 0, khz = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return TDMA_ERR_CUDA;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev);
    double *out = nullptr;
    long long *cyc = nullptr;
    if (cudaMalloc(&out, 64) != cudaSuccess || cudaMalloc(&cyc, 64) != cudaSuccess) { cudaFree(out); return TDMA_ERR_ALLOC; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int iters = 1 << 14, blocks = sms * 8;
    dfma_throughput_kernel<<<blocks, 256>>>(out, 0.999999, 1e-9, iters);        // warm-up
    cudaEventRecord(e0);
    dfma_throughput_kernel<<<blocks, 256>>>(out, 0.999999, 1e-9, iters);
    cudaEventRecord(e1);
    cudaError_t e = cudaEventSynchronize(e1);
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    const double dfma = (double)blocks * 256.0 * 8.0 * iters;
    result[0] = 2.0 * dfma / (ms * 1e-3) / 1e12;                     // TFLOP/s (DFMA = 2 flop)
    // per SM and cycle, from the SM cycles the same kernel takes (clock64 of one resident warp)
    long long h = 0;
    const int lit = 1 << 12;
    double lat[3] = {0, 0, 0};
    for (int op = 0; op < 3 && e == cudaSuccess; ++op) {
        for (int pass = 0; pass < 2; ++pass) {
            if (op == 0) latency_kernel<0><<<1, 32>>>(out, cyc, 0.999999, 1e-9, lit);
            else if (op == 1) latency_kernel<1><<<1, 32>>>(out, cyc, 1.25, 0.3, lit);
            else latency_kernel<2><<<1, 32>>>(out, cyc, 1.25, 0.3, lit);
        }
        e = cudaMemcpy(&h, cyc, sizeof(h), cudaMemcpyDeviceToHost);
        lat[op] = (double)h / (8.0 * lit);
    }
    result[1] = dfma / (ms * 1e-3) / ((double)sms * khz * 1e3);      // DFMA per SM per cycle at the nominal clock
    result[2] = lat[0];                                               // cycles per dependent DFMA
    result[3] = lat[1] - lat[0] * 0.0;                                // cycles per dependent rcp_nr (+ one DADD)
    result[4] = lat[2];                                               // cycles per dependent IEEE division (+ one DADD)
    result[5] = khz * 1e-3;                                           // nominal SM clock, MHz
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out); cudaFree(cyc);
    return e == cudaSuccess ? TDMA_OK : TDMA_ERR_CUDA;
}
