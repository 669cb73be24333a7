// gt_pink_tk.cuh -- step 6b, the paper's own method: Timmer & Koenig (1995) pink noise (PAPER.md:223,
// DESIGN.md R21).  For detector d = (spaxel s, channel c) with one-sided PSD P(f) = A_d f^-alpha_d and
// N = n_samples, f_k = k f_s / N:
//     X_0 = 0,   X_k = sqrt(P(f_k) f_s N / 4) (z0 + i z1)   (0 < k < N/2),   X_{N/2} = sqrt(P f_s N) z0  (N even)
//     (z0, z1) = normals 0, 1 of Philox(seed; c0 = k, c1 = s, c2 = c, c3 = 3)
//     x_n = (1/N) sum_k X_k e^{2 pi i k n / N}  over the Hermitian extension  = irfft(X)
// Plan creation: tk_spectrum_kernel fills the half spectra (already divided by N) of all detectors,
// cuFFT (a library FFT is a legitimate step) transforms them in place, batched, to the real series
// [n_det][N + 2]; gt_simulate adds the slice of a launch to the TOD with a tiled transpose
// (series are detector-major, the TOD is time-major).
#pragma once
#include "gt_common.cuh"

namespace gt {

constexpr uint32_t kStreamPinkTk = 3u;

struct TkParams {
    int64_t n_det, n_samples;
    int32_t n_chan;
    double f_sample;
    const float* amp;        // [n_det] sqrt(A f_s / (4 N))      (= sqrt(P f_s N / 4) / N without the f^-alpha/2 factor)
    const float* half_alpha; // [n_det] alpha / 2
    float* series;           // [n_det][ld] fp32, ld = 2 (N/2 + 1): half spectrum (complex) before, real series after the FFT
    int64_t ld;
    uint32_t seed_lo, seed_hi;
    uint32_t spaxel_base;    // global index of the plan's spaxel 0 (Philox counter word 1)
    const float2* kelvin_ab; // [n_chan] (a, b) of T = a + b P, applied to the total in tk_add_kernel's write (nullptr: none)
};

// thread = (detector, frequency index k), k fastest
__global__ void __launch_bounds__(256) tk_spectrum_kernel(TkParams p) {
    const int64_t K = p.n_samples / 2;
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= p.n_det * (K + 1)) return;
    const int64_t d = idx / (K + 1), k = idx - d * (K + 1);
    float re = 0.f, im = 0.f;
    if (k > 0) {
        const uint4 w = philox4x32_10((uint32_t)k, p.spaxel_base + (uint32_t)(d / p.n_chan), (uint32_t)(d % p.n_chan), kStreamPinkTk,
                                      p.seed_lo, p.seed_hi);
        float z0, z1;
        normal_pair(w.x, w.y, z0, z1);
        const float fk = (float)((double)k * p.f_sample / (double)p.n_samples);
        const float sig = p.amp[d] * exp2f(-p.half_alpha[d] * __log2f(fk));      // sqrt(P(f_k) f_s N / 4) / N
        if (2 * k == p.n_samples) { re = 2.0f * sig * z0; im = 0.f; }            // Nyquist term: sqrt(P f_s N) / N
        else { re = sig * z0; im = sig * z1; }
    }
    float2* row = reinterpret_cast<float2*>(p.series + d * p.ld);
    row[k] = make_float2(re, im);
}

// tod[(t_local) * n_det + d] += series[d * ld + t0 + t_local]; 32 x 32 tiles through shared memory
__global__ void __launch_bounds__(256) tk_add_kernel(TkParams p, int64_t t0, int64_t T, float* __restrict__ tod) {
    __shared__ float tile[32][33];
    const int64_t tb = (int64_t)blockIdx.x * 32, db = (int64_t)blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;              // 32 x 8
#pragma unroll
    for (int i = 0; i < 32; i += 8) {
        const int64_t d = db + ty + i, t = tb + tx;
        tile[ty + i][tx] = (d < p.n_det && t < T) ? p.series[d * p.ld + t0 + t] : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 32; i += 8) {
        const int64_t t = tb + ty + i, d = db + tx;
        if (d < p.n_det && t < T) {
            const float total = tod[t * p.n_det + d] + tile[tx][ty + i];
            if (p.kelvin_ab) { const float2 ab = __ldg(p.kelvin_ab + d % p.n_chan); tod[t * p.n_det + d] = fmaf(ab.y, total, ab.x); }
            else tod[t * p.n_det + d] = total;
        }
    }
}

}  // namespace gt
