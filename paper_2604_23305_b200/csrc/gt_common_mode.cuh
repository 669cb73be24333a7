// gt_common_mode.cuh -- the one cross-spaxel step of the paper: common-mode subtraction, Eq. 25-26.
//
//   T*_a,i(t,f) = T_b,i / eta_i  -  (1 - eta_i) / (eta_i N_out)  sum_j S_j T_b,j / (1 - eta_j),
//   eta_j(t,f) = eta_atm,z(f)^csc(el_j(t))   (Eq. 10 on the zenith transmission at the observation's mean PWV),
//   S_j = 1 where the spaxel offset sqrt(dphi_j^2 + dtheta_j^2) > r_out, N_out = sum_j S_j.
//
// Spaxel-sharded runs: every rank holds a sub-range of the spaxels, forms its PARTIAL sum over its
// own spaxels with cm_partial_kernel, the [t x chan] partial sums are added across ranks (one all-reduce), and
// cm_apply_kernel finishes Eq. 25 on the rank's own slab.  Both kernels are passes over the TOD (4 B read per
// detector-sample for the partial sums, 8 B read-modify-write for the result); the transmission is formed in double as
// exp(csc ln eta_z), and 1 - eta as -expm1(csc ln eta_z): no cancellation where the atmosphere is nearly transparent
// (cm_eta: from the values at a reference airmass and a short polynomial in the airmass difference).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gt {

constexpr int kCmBatch = 8;           // TOD values fetched ahead per thread (apply kernel)

struct CmParams {
    const double *sinE, *cosE;        // per sample: sin / cos(el0 + el[n])   (the plan's geometry tables)
    const double *sin_del, *cos_del;  // per spaxel
    const double* ln_eta_z;           // [4][n_chan]: ln of the zenith transmission at the mean PWV at the channel centres (le),
                                      //   then eta0 = exp(csc0 le), om0 = 1 - eta0 = -expm1(csc0 le) and 1 / eta0 at the reference airmass csc0
    const float* weight;              // [n_spaxel] S_j (0 or 1)
    int64_t t0, T;
    int32_t n_spaxel, n_chan;
    double inv_n_out;                 // 1 / N_out over ALL spaxels of the instrument (apply only)
    double csc0;                      // reference airmass (boresight): eta = eta0 exp((csc - csc0) le)
};

// csc of the absolute elevation of (sample t0 + t, spaxel s) by the addition formula, as the geometry kernel
__device__ __forceinline__ double cm_csc(const CmParams& p, int64_t t, int s) {
    const int64_t n = p.t0 + t;
    return 1.0 / (p.sinE[n] * p.cos_del[s] + p.cosE[n] * p.sin_del[s]);
}

// eta = exp(csc le) and 1 - eta = -expm1(csc le) to double accuracy, from the per-channel values at the reference airmass:
//   eta = eta0 (1 + u),  1 - eta = om0 - eta0 u,  1 / eta = (1 + w) / eta0,   u = expm1(x),  w = expm1(-x),  x = (csc - csc0) le.
// Over a scan the airmass moves by 1e-3 or so of csc0, so |x| << 1 and u, w are SMALL CORRECTIONS: they are evaluated in
// fp32 (Taylor polynomial of degree 4: x^5 / 120 < 2.6e-9 for |x| <= 0.05 and 3e-16 for the |x| ~ 1e-3 of a scan; the fp32
// rounding of u, 6e-8 |x|, is below 3e-9 of eta) and only folded into the double values eta0, om0 = -expm1(csc0 le) (no
// cancellation) and 1 / eta0 with one DFMA each.
// Beyond |x| = 0.05 the library functions in double.  The double-precision exp, expm1 and divisions per element were what
// bound these kernels (15 ms each per C4 step: FP64 is a narrow pipe on this GPU).
__device__ __forceinline__ float cm_expm1_small(float x) {
    return x * fmaf(x, fmaf(x, fmaf(x, 1.0f / 24, 1.0f / 6), 0.5f), 1.0f);
}
// 1 / d for d in the normal fp32 range: fp32 reciprocal (2^-23) and one Newton step in double (2^-46)
__device__ __forceinline__ double cm_rcp(double d) {
    const double r = (double)__frcp_rn((float)d);
    return fma(r, fma(-d, r, 1.0), r);
}

// le4 = [4][n_chan]: fills eta0 = exp(csc0 le), om0 = -expm1(csc0 le) and 1 / eta0 = exp(-csc0 le) behind the le the host uploaded
__global__ void __launch_bounds__(128) cm_ref_kernel(double* __restrict__ le4, int32_t n_chan, double csc0) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_chan) return;
    const double x = csc0 * le4[c];
    le4[n_chan + c] = exp(x);
    le4[2 * n_chan + c] = -expm1(x);
    le4[3 * n_chan + c] = exp(-x);
}

// shared memory of both kernels: [n_spaxel] double csc - csc0 of this sample's lines of sight, [n_spaxel] the same in float,
// [n_spaxel] float S_j
__device__ __forceinline__ void cm_stage_sample(const CmParams& p, int64_t t, double* s_dcsc, float*& s_dcf, float*& s_w) {
    s_dcf = reinterpret_cast<float*>(s_dcsc + p.n_spaxel);
    s_w = s_dcf + p.n_spaxel;
    for (int s = threadIdx.x; s < p.n_spaxel; s += blockDim.x) {
        const double d = cm_csc(p, t, s) - p.csc0;
        s_dcsc[s] = d; s_dcf[s] = (float)d; s_w[s] = p.weight[s];
    }
    __syncthreads();
}
inline size_t cm_smem_bytes(int n_spaxel) { return (size_t)n_spaxel * (sizeof(double) + 2 * sizeof(float)); }

// grid.x = samples, threads stride over channels: partial[t][c] = sum over this plan's spaxels of S_s T_b / (1 - eta)
__global__ void __launch_bounds__(128, 16)          // read-only and fp32-heavy: 32 registers hold it (5.3 ms per C4 step; 8 blocks: 6.6)
cm_partial_kernel(CmParams p, const float* __restrict__ tod, float* __restrict__ partial) {
    extern __shared__ double s_dcsc[];
    float *s_dcf, *s_w;
    const int64_t t = blockIdx.x;
    cm_stage_sample(p, t, s_dcsc, s_dcf, s_w);
    for (int c = threadIdx.x; c < p.n_chan; c += blockDim.x) {
        const double le = p.ln_eta_z[c], eta0 = p.ln_eta_z[p.n_chan + c], om0 = p.ln_eta_z[2 * p.n_chan + c];
        const float lef = (float)le;
        double acc = 0.0;
        const float* col = tod + (size_t)t * p.n_spaxel * p.n_chan + c;
        for (int s = 0; s < p.n_spaxel; ++s) {
            if (s_w[s] == 0.f) continue;
            const float x = s_dcf[s] * lef;
            // 1 - eta lies in (0, 1): far inside the fp32 range unless the channel is transparent to 1e-30
            double one_minus_eta = fma(-eta0, (double)cm_expm1_small(x), om0);
            if (!(fabsf(x) <= 0.05f)) one_minus_eta = -expm1((s_dcsc[s] + p.csc0) * le);
            acc = fma((double)__ldcs(col + (size_t)s * p.n_chan), one_minus_eta > 1e-30 ? cm_rcp(one_minus_eta) : 1.0 / one_minus_eta, acc);
        }
        partial[(size_t)t * p.n_chan + c] = (float)acc;
    }
}

// grid.x = samples, threads stride over channels and walk the sample's spaxels: tod <- T*_a in place.  (One block per
// (sample, spaxel) row re-read the four per-channel constants, 32 B, for every 4-byte element.)
__global__ void __launch_bounds__(128, 8)           // 8 values in flight per thread need the 64 registers (8.1 ms per C4 step; 12 blocks: 10.1, 16: 12.1)
cm_apply_kernel(CmParams p, float* __restrict__ tod, const float* __restrict__ sum) {
    extern __shared__ double s_dcsc[];
    float *s_dcf, *s_w;
    const int64_t t = blockIdx.x;
    cm_stage_sample(p, t, s_dcsc, s_dcf, s_w);
    for (int c = threadIdx.x; c < p.n_chan; c += blockDim.x) {
        const double le = p.ln_eta_z[c], eta0 = p.ln_eta_z[p.n_chan + c], om0 = p.ln_eta_z[2 * p.n_chan + c], inv0 = p.ln_eta_z[3 * p.n_chan + c];
        const float lef = (float)le;
        const double cm = (double)__ldg(sum + (size_t)t * p.n_chan + c) * p.inv_n_out;
        float* col = tod + (size_t)t * p.n_spaxel * p.n_chan + c;
        for (int sb = 0; sb < p.n_spaxel; sb += kCmBatch) {
            float cur[kCmBatch];                       // loads of a batch first: a load after a store to the same array would wait for it
#pragma unroll
            for (int b = 0; b < kCmBatch; ++b) cur[b] = sb + b < p.n_spaxel ? __ldcs(col + (size_t)(sb + b) * p.n_chan) : 0.f;
#pragma unroll
            for (int b = 0; b < kCmBatch; ++b) {
                const int s = sb + b;
                if (s < p.n_spaxel) {
                    const float x = s_dcf[s] * lef;
                    double one_minus_eta = fma(-eta0, (double)cm_expm1_small(x), om0);
                    double inv_eta = fma(inv0, (double)cm_expm1_small(-x), inv0);
                    if (!(fabsf(x) <= 0.05f)) {
                        const double y = (s_dcsc[s] + p.csc0) * le;
                        one_minus_eta = -expm1(y); inv_eta = exp(-y);
                    }
                    __stcs(col + (size_t)s * p.n_chan, (float)(fma(-one_minus_eta, cm, (double)cur[b]) * inv_eta));
                }
            }
        }
    }
}

}  // namespace gt
