// gt_screen.cuh -- pre-processing of the atmosphere screen (R24), SURVEY row f4.
//   PWV[y][x] = PWV_0 + (1 / 6.587) sum_{i,j} K[j][i] EPL[(y + j) mod ny][(x + i) mod nx]          (Eq. 4 + footprint)
// K = the aperture footprint on the screen grid (Gaussian illumination of Eq. 2 truncated at R_tel, unit sum),
// built in double by the caller of the kernel (gt_prepare_screen).  Not separable (the disc), so it is a direct
// 2-D convolution: a block makes a 32 x 32 output tile from a shared-memory halo tile; 8 B of HBM per pixel.
#pragma once
#include "gt_common.cuh"

namespace gt {

struct ScreenParams {
    const float* epl;      // [ny][nx]
    float* pwv;            // [ny][nx]
    const float* K;        // [2 ry + 1][2 rx + 1]
    int32_t nx, ny, rx, ry;
    float scale, pwv0;     // 1 / 6.587, PWV_0
};

constexpr int kScreenTile = 32;

__device__ __forceinline__ int wrap_index(int a, int n) { a %= n; return a < 0 ? a + n : a; }

// grid (ceil(nx / 32), ceil(ny / 32)), block 256 = 32 x 8; dynamic shared memory = halo tile + weights
__global__ void __launch_bounds__(256) screen_los_kernel(ScreenParams p) {
    extern __shared__ float sm_screen[];
    const int tw = kScreenTile + 2 * p.rx, th = kScreenTile + 2 * p.ry, kw = 2 * p.rx + 1, kh = 2 * p.ry + 1;
    float* tile = sm_screen;
    float* wk = sm_screen + (size_t)tw * th;
    const int x0 = blockIdx.x * kScreenTile, y0 = blockIdx.y * kScreenTile;
    for (int idx = threadIdx.x; idx < tw * th; idx += 256) {
        const int r = idx / tw, c = idx - r * tw;
        tile[idx] = __ldg(p.epl + (size_t)wrap_index(y0 - p.ry + r, p.ny) * p.nx + wrap_index(x0 - p.rx + c, p.nx));
    }
    for (int idx = threadIdx.x; idx < kw * kh; idx += 256) wk[idx] = p.K[idx];
    __syncthreads();
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    for (int j = 0; j < kh; ++j)
        for (int i = 0; i < kw; ++i) {
            const float w = wk[j * kw + i];
            if (w == 0.f) continue;                                    // outside the aperture (block-uniform)
#pragma unroll
            for (int k = 0; k < 4; ++k) acc[k] = fmaf(w, tile[(ty + 8 * k + j) * tw + tx + i], acc[k]);
        }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int x = x0 + tx, y = y0 + ty + 8 * k;
        if (x < p.nx && y < p.ny) p.pwv[(size_t)y * p.nx + x] = fmaf(acc[k], p.scale, p.pwv0);
    }
}

}  // namespace gt
