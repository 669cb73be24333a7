// gt_common_mode.cuh -- the one cross-spaxel step of the paper: common-mode subtraction, Eq. 25-26.
//
//   T*_a,i(t,f) = T_b,i / eta_i  -  (1 - eta_i) / (eta_i N_out)  sum_j S_j T_b,j / (1 - eta_j),
//   eta_j(t,f) = eta_atm,z(f)^csc(el_j(t))   (Eq. 10 on the zenith transmission at the observation's mean PWV),
//   S_j = 1 where the spaxel offset sqrt(dphi_j^2 + dtheta_j^2) > r_out, N_out = sum_j S_j.
//
// Spaxel-sharded runs: every rank holds a sub-range of the spaxels, forms its PARTIAL sum over its
// own spaxels with cm_partial_kernel, the [t x chan] partial sums are added across ranks (one all-reduce), and
// cm_apply_kernel finishes Eq. 25 on the rank's own slab.  Both kernels are HBM-bound passes over the TOD (4 B read per
// detector-sample for the partial sums, 8 B read-modify-write for the result); the transmission is formed in double as
// exp(csc ln eta_z), and 1 - eta as -expm1(csc ln eta_z): no cancellation where the atmosphere is nearly transparent.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gt {

struct CmParams {
    const double *sinE, *cosE;        // per sample: sin / cos(el0 + el[n])   (the plan's geometry tables)
    const double *sin_del, *cos_del;  // per spaxel
    const double* ln_eta_z;           // [n_chan] ln of the zenith transmission at the mean PWV, at the channel centres
    const float* weight;              // [n_spaxel] S_j (0 or 1)
    int64_t t0, T;
    int32_t n_spaxel, n_chan;
    double inv_n_out;                 // 1 / N_out over ALL spaxels of the instrument (apply only)
};

// csc of the absolute elevation of (sample t0 + t, spaxel s) by the addition formula, as the geometry kernel
__device__ __forceinline__ double cm_csc(const CmParams& p, int64_t t, int s) {
    const int64_t n = p.t0 + t;
    return 1.0 / (p.sinE[n] * p.cos_del[s] + p.cosE[n] * p.sin_del[s]);
}

// grid.x = samples, threads stride over channels: partial[t][c] = sum over this plan's spaxels of S_s T_b / (1 - eta)
__global__ void __launch_bounds__(128)
cm_partial_kernel(CmParams p, const float* __restrict__ tod, float* __restrict__ partial) {
    const int64_t t = blockIdx.x;
    for (int c = threadIdx.x; c < p.n_chan; c += blockDim.x) {
        const double le = p.ln_eta_z[c];
        double acc = 0.0;
        for (int s = 0; s < p.n_spaxel; ++s) {
            if (p.weight[s] == 0.f) continue;
            const double one_minus_eta = -expm1(cm_csc(p, t, s) * le);
            acc += (double)__ldcs(tod + ((size_t)t * p.n_spaxel + s) * p.n_chan + c) / one_minus_eta;
        }
        partial[(size_t)t * p.n_chan + c] = (float)acc;
    }
}

// grid.x = samples x spaxels, threads stride over channels: tod <- T*_a in place
__global__ void __launch_bounds__(128)
cm_apply_kernel(CmParams p, float* __restrict__ tod, const float* __restrict__ sum) {
    const int64_t r = blockIdx.x;
    const int64_t t = r / p.n_spaxel;
    const int s = (int)(r - t * p.n_spaxel);
    const double csc = cm_csc(p, t, s);
    for (int c = threadIdx.x; c < p.n_chan; c += blockDim.x) {
        const double x = csc * p.ln_eta_z[c], eta = exp(x), one_minus_eta = -expm1(x);
        const size_t i = (size_t)r * p.n_chan + c;
        const double cm = (double)__ldg(sum + (size_t)t * p.n_chan + c) * p.inv_n_out;
        tod[i] = (float)(((double)tod[i] - one_minus_eta * cm) / eta);
    }
}

}  // namespace gt
