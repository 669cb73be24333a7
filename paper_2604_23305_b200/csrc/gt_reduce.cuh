// gt_reduce.cuh -- plan-time statistics of the caller's large DEVICE arrays (source cube, PWV screen).
//
// The tensor kernel feeds fp16 operand pairs to tcgen05.mma, so gt_plan_create must know the largest
// spectrum element the generator can produce before it fixes the operand scale:
//   max_nu max( |Xn(nu)|, |G(nu)| max_pixels |cube[pixel][nu]| )
// and it must refuse arrays that hold NaN or Inf (they would reach table indices).
// One pass over the array, column-wise: a[row][col] -> absmax[col] (and sum[col] in double).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gt {

// grid = (ceil(n_cols / 256), row blocks); thread = one column, strided over its block's rows (coalesced across the
// warp).  |x| of a finite float orders like its bit pattern, and NaN / Inf patterns (>= 0x7F800000) order above every
// finite value, so one atomicMax on the bits gives the maximum AND the non-finite flag.
__global__ void __launch_bounds__(256)
colstat_kernel(const float* __restrict__ a, int64_t n_rows, int32_t n_cols, uint32_t* __restrict__ absmax_bits,
               double* __restrict__ sum) {
    const int32_t c = blockIdx.x * 256 + threadIdx.x;
    if (c >= n_cols) return;
    const int64_t per = (n_rows + gridDim.y - 1) / gridDim.y;
    const int64_t r0 = (int64_t)blockIdx.y * per, r1 = min(n_rows, r0 + per);
    uint32_t m = 0u;
    double s = 0.0;
    for (int64_t r = r0; r < r1; ++r) {
        const float v = __ldg(a + r * n_cols + c);
        m = max(m, __float_as_uint(v) & 0x7FFFFFFFu);
        s += (double)v;
    }
    if (r1 > r0) {
        atomicMax(absmax_bits + c, m);
        if (sum) atomicAdd(sum + c, s);
    }
}

}  // namespace gt
