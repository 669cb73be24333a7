// gt_measure.cuh -- measurement utility, not on the path: the FP32 FMA peak of the device, the denominator of the
// FP32 kernel's roofline (bench.py "alu" bound; SURVEY 8d asks for a MEASURED register-only FMA loop next to the
// nominal 148 SM x 128 lanes x 2 x clock).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gt {

// 8 independent FMA chains per thread, registers only; 1024 threads per CTA, one wave of CTAs over the SMs.
__global__ void __launch_bounds__(1024) fma_peak_kernel(float* __restrict__ out, int iters, float a, float b) {
    float x0 = threadIdx.x * 1e-6f, x1 = x0 + 1.f, x2 = x0 + 2.f, x3 = x0 + 3.f, x4 = x0 + 4.f, x5 = x0 + 5.f, x6 = x0 + 6.f, x7 = x0 + 7.f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            x0 = fmaf(x0, a, b); x1 = fmaf(x1, a, b); x2 = fmaf(x2, a, b); x3 = fmaf(x3, a, b);
            x4 = fmaf(x4, a, b); x5 = fmaf(x5, a, b); x6 = fmaf(x6, a, b); x7 = fmaf(x7, a, b);
        }
    }
    const float s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == 123.456f) out[blockIdx.x * blockDim.x + threadIdx.x] = s;      // never true: keeps the chains alive
}

}  // namespace gt
