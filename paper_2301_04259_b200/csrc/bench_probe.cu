// libsoap_b200_bench.so: measurement aids for bench.py.  NOT part of the product library (libsoap_b200.so) nor of its C ABI
// (include/soap_b200.h): nothing on the hot path calls into this file, and the product never loads it.
//
// soap_bench_fp32_rate: the device's FP32 FMA rate with the instruction forms the shift-interpolate-accumulate kernels use
// (probe.cuh) - the denominator of bench.py's `"bound": "alu"` roofline, checked on the box instead of taken on trust.
#include <algorithm>
#include <cuda_runtime.h>

#include "probe.cuh"

extern "C" {

// Runs a register-only kernel of independent FMA chains (8 CTAs of 256 threads per SM, 16 accumulators per thread) on
// `device`, default stream, and stores the best of four timed repetitions in FMAs per second in *fma_per_s (HOST).
// packed != 0: fma.rn.f32x2 with a scalar-broadcast operand (SASS FFMA2); 0: plain FFMA.  Synchronous.
// Returns 0, or the cudaError_t of the call that failed.
int soap_bench_fp32_rate(int device, int packed, double *fma_per_s) {
    using namespace soap;
    if (!fma_per_s) return (int)cudaErrorInvalidValue;
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return (int)e;
    int n_sm = 0;
    if ((e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, device)) != cudaSuccess) return (int)e;
    float *sink = nullptr;  // never written (see the kernel); any valid address will do
    if ((e = cudaMalloc(reinterpret_cast<void **>(&sink), sizeof(float))) != cudaSuccess) return (int)e;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int iters = 4096, grid = n_sm * 8;  // 8 CTAs of 256 threads per SM: 64 warps, every sub-partition full
    double best = 0.0;
    for (int rep = 0; rep < 5; ++rep) {  // the first repetition warms up; best of the rest
        cudaEventRecord(e0, nullptr);
        if (packed) fp32_probe_kernel<true><<<grid, kProbeThreads>>>(iters, 1.0000001f, sink);
        else fp32_probe_kernel<false><<<grid, kProbeThreads>>>(iters, 1.0000001f, sink);
        cudaEventRecord(e1, nullptr);
        if ((e = cudaEventSynchronize(e1)) != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double fma = (double)grid * kProbeThreads * (double)iters * 8.0 * kProbeChains;
        if (rep > 0 && ms > 0.f) best = std::max(best, fma / (ms * 1e-3));
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    *fma_per_s = best;
    return (int)e;
}

}  // extern "C"
