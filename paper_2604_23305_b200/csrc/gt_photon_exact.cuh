// gt_photon_exact.cuh -- photon noise from the paper's full Eq. 17 (R23).
//   NEP^2 / 2 = dnu sum_nu Fm P (h nu + g) + dnu sum_nu Fm^2 P^2,   g = 2 Delta_Al / eta_pb
// Both contractions run through the fused tensor kernel: the part linear in the generated element goes through
// the filter L = (Fm (h nu + g) + 2 Fm^2 Y) / E0, the quadratic part through Fm^2 on squared elements; both come
// back divided by the energy E0 = h nu_max + g so that they are O(P_KID).  This kernel forms
//   sigma = sqrt((lin + sq) f_s) sqrt(E0)       (Eq. 18: NEP sqrt(f_s / 2))
// and adds sigma z to the power with the same Philox normal as the narrow-band mode (Eq. 19).
#pragma once
#include "gt_common.cuh"

namespace gt {

struct PhotonExactParams {
    float* tod;                    // [n_rows][n_chan] noiseless P_KID in, P_KID + P_wn out
    const float *lin, *sq;         // [n_rows][n_chan] the two contractions / E0
    int64_t n_rows, t0;
    int32_t n_chan, n_spaxel;
    float f_sample, sqrt_e0;
    uint32_t seed_lo, seed_hi, spaxel_base;
};

// block = 256 threads walking spans of 32 whole rows, as kelvin_kernel
__global__ void __launch_bounds__(256) photon_exact_kernel(PhotonExactParams p) {
    constexpr int kRows = 32;
    const int64_t n_span = (p.n_rows + kRows - 1) / kRows;
    for (int64_t sp = blockIdx.x; sp < n_span; sp += gridDim.x) {
        const int64_t r0 = sp * kRows;
        const uint32_t len = (uint32_t)(min((int64_t)kRows, p.n_rows - r0) * p.n_chan);
        const size_t base = (size_t)r0 * p.n_chan;
        for (uint32_t j = threadIdx.x; j < len; j += 256) {
            const uint32_t rl = j / (uint32_t)p.n_chan, c = j - rl * (uint32_t)p.n_chan;
            const int64_t r = r0 + rl;
            const uint32_t n = (uint32_t)(p.t0 + r / p.n_spaxel), s = p.spaxel_base + (uint32_t)(r % p.n_spaxel);
            const uint4 w = philox4x32_10(n, s, c, kStreamPhoton, p.seed_lo, p.seed_hi);
            const float half_nep2 = fmaxf(__ldcs(p.lin + base + j) + __ldcs(p.sq + base + j), 0.f);
            const float sigma = sqrt_fast(half_nep2 * p.f_sample) * p.sqrt_e0;
            p.tod[base + j] = fmaf(sigma, normal_cos(w.x, w.y), p.tod[base + j]);
        }
    }
}

}  // namespace gt
