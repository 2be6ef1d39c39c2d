// Measures the FP32 FMA rate of the device with the instruction forms the shift-interpolate-accumulate kernels use: the
// denominator of bench.py's `"bound": "alu"` roofline checked on the box instead of taken on trust.
// 16 independent accumulators per thread, no memory traffic; `packed` = fma.rn.f32x2 with a scalar-broadcast operand (SASS
// FFMA2, the inner loops' form), else plain FFMA.  Not part of the hot path.
#pragma once
#include <cuda_runtime.h>

#include "ptx_helpers.cuh"

namespace soap {

constexpr int kProbeThreads = 256;
constexpr int kProbeChains = 16;  // fp32 accumulators per thread (8 packed pairs)

template <bool PACKED>
__global__ void __launch_bounds__(kProbeThreads) fp32_probe_kernel(int iters, float w, float *__restrict__ sink) {
    float2 acc[kProbeChains / 2], u[kProbeChains / 2];
#pragma unroll
    for (int k = 0; k < kProbeChains / 2; ++k) {
        acc[k] = make_float2(0.f, 0.f);
        u[k] = make_float2(1.f + (float)(threadIdx.x + k), 2.f + (float)k);
    }
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int rep = 0; rep < 8; ++rep) {
#pragma unroll
            for (int k = 0; k < kProbeChains / 2; ++k) {
                if (PACKED) {
                    acc[k] = fma2(bcast2(w), u[k], acc[k]);
                } else {
                    acc[k].x = fmaf(w, u[k].x, acc[k].x);
                    acc[k].y = fmaf(w, u[k].y, acc[k].y);
                }
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < kProbeChains / 2; ++k) s += acc[k].x + acc[k].y;
    if (s == 123.456f) sink[0] = s;  // keeps the loop alive; never true for the values used
}

}  // namespace soap
