// gt_reduce.cuh -- plan-time statistics of the caller's large DEVICE arrays (source cube, PWV screen).
//
// The tensor kernel feeds fp16 operand pairs to tcgen05.mma, so gt_plan_create must know the largest
// spectrum element the generator can produce before it fixes the operand scale:
//   max_nu max( |Xn(nu)|, |G(nu)| max_pixels |cube[pixel][nu]| )
// and it must refuse arrays that hold NaN or Inf (they would reach table indices).
// One pass over the array, column-wise: a[row][col] -> absmax[col], sum[col] in double, and the signed minimum and
// maximum per column (banded corrections: the range of the PWV screen and the sign of the cube bound
// the spectrum elements from below as well).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

namespace gt {

// order-preserving map float -> uint32 (finite values and infinities): atomicMin / atomicMax on the keys give min / max
__host__ __device__ __forceinline__ uint32_t float_key(float v) {
#ifdef __CUDA_ARCH__
    const uint32_t b = __float_as_uint(v);
#else
    uint32_t b; memcpy(&b, &v, 4);
#endif
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__host__ __device__ __forceinline__ float key_float(uint32_t k) {
    const uint32_t b = (k & 0x80000000u) ? (k & 0x7FFFFFFFu) : ~k;
#ifdef __CUDA_ARCH__
    return __uint_as_float(b);
#else
    float v; memcpy(&v, &b, 4); return v;
#endif
}

// grid = (ceil(n_cols / 256), row blocks); thread = one column, strided over its block's rows (coalesced across the
// warp).  |x| of a finite float orders like its bit pattern, and NaN / Inf patterns (>= 0x7F800000) order above every
// finite value, so one atomicMax on the bits gives the maximum AND the non-finite flag.
// min_key must be initialised to 0xFFFFFFFF and max_key to 0 (both may be nullptr).
__global__ void __launch_bounds__(256)
colstat_kernel(const float* __restrict__ a, int64_t n_rows, int32_t n_cols, uint32_t* __restrict__ absmax_bits,
               double* __restrict__ sum, uint32_t* __restrict__ min_key = nullptr, uint32_t* __restrict__ max_key = nullptr) {
    const int32_t c = blockIdx.x * 256 + threadIdx.x;
    if (c >= n_cols) return;
    const int64_t per = (n_rows + gridDim.y - 1) / gridDim.y;
    const int64_t r0 = (int64_t)blockIdx.y * per, r1 = min(n_rows, r0 + per);
    uint32_t m = 0u, lo = 0xFFFFFFFFu, hi = 0u;
    double s = 0.0;
    for (int64_t r = r0; r < r1; ++r) {
        const float v = __ldg(a + r * n_cols + c);
        m = max(m, __float_as_uint(v) & 0x7FFFFFFFu);
        const uint32_t k = float_key(v);
        lo = min(lo, k); hi = max(hi, k);
        s += (double)v;
    }
    if (r1 > r0) {
        atomicMax(absmax_bits + c, m);
        if (sum) atomicAdd(sum + c, s);
        if (min_key) atomicMin(min_key + c, lo);
        if (max_key) atomicMax(max_key + c, hi);
    }
}

}  // namespace gt
