// gt_beam.cuh -- pre-processing of the source cube (R25), SURVEY row f4.
//   F_nu(rho) = |int_0^R A(r) J0(2 pi r rho / lambda) r dr|^2 / F_nu(0),  A(r) = exp(-k r^2),  k = |t_edge|/20 ln10 / R^2   (Eq. 2-3)
//   P[j][i][nu] = A_p daz del sum_{dj,di} F_nu(di daz, dj del) I[j - dj][i - di][nu] cos(el_first + (j - dj) del)      (Eq. 1)
// beam_weights_kernel evaluates the Hankel integral in double (composite Simpson, kBeamQuad intervals) on one
// quadrant of the (2 r + 1)^2 pixel offsets and mirrors it; beam_conv_kernel is the direct convolution, one
// thread per (pixel, frequency) with the frequency fastest so that cube and weight loads are coalesced.
#pragma once
#include "gt_common.cuh"

namespace gt {

constexpr int kBeamQuad = 1024;       // Simpson intervals over [0, R_tel]: the integrand has < 10 oscillations

struct BeamParams {
    int32_t n_az, n_el, n_freq, r_pix;
    double nu0, dnu, daz, del, el_first, R_tel, k_taper, scale;   // scale = A_p daz del
    const float* I;      // [n_el][n_az][n_freq]
    float* P;            // [n_el][n_az][n_freq]
    float* W;            // [2 r + 1][2 r + 1][n_freq]
};

// grid (ceil(n_freq / 128), r + 1, r + 1), block 128: thread = (nu, dj >= 0, di >= 0)
__global__ void __launch_bounds__(128) beam_weights_kernel(BeamParams p) {
    const int f = blockIdx.x * blockDim.x + threadIdx.x, di = blockIdx.y, dj = blockIdx.z;
    if (f >= p.n_freq) return;
    const double lam = 299792458.0 / (p.nu0 + (double)f * p.dnu);
    const double rho = sqrt((di * p.daz) * (di * p.daz) + (dj * p.del) * (dj * p.del));
    const double b = 2.0 * 3.14159265358979323846 * rho / lam, h = p.R_tel / (double)kBeamQuad;
    double s = 0.0;                                    // Simpson: the r = 0 node contributes 0 (factor r)
    for (int q = 1; q <= kBeamQuad; ++q) {
        const double r = (double)q * h;
        const double w = (q == kBeamQuad) ? 1.0 : ((q & 1) ? 4.0 : 2.0);
        s += w * exp(-p.k_taper * r * r) * j0(b * r) * r;
    }
    s *= h / 3.0;
    const double g0 = p.k_taper > 0.0 ? -expm1(-p.k_taper * p.R_tel * p.R_tel) / (2.0 * p.k_taper) : 0.5 * p.R_tel * p.R_tel;
    const float F = (float)((s / g0) * (s / g0));
    const int kw = 2 * p.r_pix + 1;
    const int js[2] = {p.r_pix + dj, p.r_pix - dj}, is[2] = {p.r_pix + di, p.r_pix - di};
    for (int a = 0; a < 2; ++a)
        for (int c = 0; c < 2; ++c) p.W[((size_t)js[a] * kw + is[c]) * p.n_freq + f] = F;
}

// grid (ceil(n_freq / 128), n_az, n_el), block 128
__global__ void __launch_bounds__(128) beam_conv_kernel(BeamParams p) {
    const int f = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y, j = blockIdx.z;
    if (f >= p.n_freq) return;
    const int r = p.r_pix, kw = 2 * r + 1;
    double acc = 0.0;
    for (int dj = -r; dj <= r; ++dj) {
        const int js = j - dj;
        if (js < 0 || js >= p.n_el) continue;
        const double cw = cos(p.el_first + (double)js * p.del);
        double row = 0.0;
        for (int di = -r; di <= r; ++di) {
            const int is = i - di;
            if (is < 0 || is >= p.n_az) continue;
            row += (double)__ldg(p.W + ((size_t)(dj + r) * kw + (di + r)) * p.n_freq + f) *
                   (double)__ldg(p.I + ((size_t)js * p.n_az + is) * p.n_freq + f);
        }
        acc += cw * row;
    }
    p.P[((size_t)j * p.n_az + i) * p.n_freq + f] = (float)(p.scale * acc);
}

}  // namespace gt
