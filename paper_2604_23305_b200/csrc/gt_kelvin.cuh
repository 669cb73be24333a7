// gt_kelvin.cuh -- brightness-temperature output (R22).
// Plan creation simulates the skydip in double precision: for the K zenith PWV values pwv_k = lo + k step,
// blank sky, boresight elevation el0,
//     eta_atm(nu) = eta_z(nu, pwv_k)^(1 / sin el0)                              (Eq. 10, LUT bilinear)
//     P_KID[k][c] = dnu sum_nu Fm[c][nu] ((1 - eta_atm) Xd(nu) + Yd(nu))        (Eq. 11, 12, 16 collapsed, S = 0)
//     T_b[k][c]   = sum_nu Fm[c][nu] ((1 - eta_atm) T_atm + eta_atm T_cmb) / sum_nu Fm[c][nu]
// then the least-squares line T_b = a_c + b_c P_KID per channel.  gt_simulate applies it to the finished TOD.
#pragma once
#include "gt_common.cuh"

namespace gt {

struct SkydipParams {
    int32_t n_chan, n_freq, n_freq_pad, n_pwv, K;
    double dnu, lut_pwv0, lut_dpwv, pwv_lo, pwv_step, csc0, T_atm, T_cmb;
    const float* lut_r;      // [n_pwv][n_freq_pad] LUT resampled on the frequency grid
    const float* filt;       // [n_chan][n_freq] (the caller's device array)
    const double *Xd, *Yd;   // [n_freq] collapsed cascade in W/Hz: P_nu = (1 - eta_atm) Xd + eta_atm G S + Yd
    double *P, *T;           // [K][n_chan]
    double* ab;              // [2][n_chan]: a, b
    float2* abf;             // [n_chan] (a, b) in fp32 for the epilogue
    int32_t* bad;            // set to 1 + channel when a channel cannot be calibrated
};

__device__ __forceinline__ double block_sum_256(double v, double* sh) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += sh[i];
    return s;
}

// grid (n_chan, K), block 256
__global__ void __launch_bounds__(256) skydip_kernel(SkydipParams p) {
    __shared__ double sh[8];
    const int c = blockIdx.x, k = blockIdx.y;
    const double pwv = p.pwv_lo + (double)k * p.pwv_step;
    double q = (pwv - p.lut_pwv0) / p.lut_dpwv;
    q = fmin(fmax(q, 0.0), (double)(p.n_pwv - 1));
    int ip = (int)floor(q);
    if (ip > p.n_pwv - 2) ip = p.n_pwv - 2;
    if (ip < 0) ip = 0;
    const double fq = q - (double)ip;
    const float* L0 = p.lut_r + (size_t)ip * p.n_freq_pad;
    const float* L1 = p.lut_r + (size_t)min(ip + 1, p.n_pwv - 1) * p.n_freq_pad;
    const float* F = p.filt + (size_t)c * p.n_freq;
    double sP = 0.0, sT = 0.0, sF = 0.0;
    for (int i = threadIdx.x; i < p.n_freq; i += 256) {
        const double l0 = (double)L0[i], l1 = (double)L1[i];
        const double eta = pow(l0 + fq * (l1 - l0), p.csc0);
        const double f = (double)F[i];
        sP += f * ((1.0 - eta) * p.Xd[i] + p.Yd[i]);
        sT += f * ((1.0 - eta) * p.T_atm + eta * p.T_cmb);
        sF += f;
    }
    sP = block_sum_256(sP, sh); sT = block_sum_256(sT, sh); sF = block_sum_256(sF, sh);
    if (threadIdx.x == 0) {
        p.P[(size_t)k * p.n_chan + c] = p.dnu * sP;
        p.T[(size_t)k * p.n_chan + c] = sF != 0.0 ? sT / sF : 0.0;
        if (sF == 0.0) atomicMax(p.bad, 1 + c);
    }
}

// thread = channel: least squares over the K skydip points
__global__ void __launch_bounds__(128) skydip_fit_kernel(SkydipParams p) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= p.n_chan) return;
    double Pm = 0.0, Tm = 0.0;
    for (int k = 0; k < p.K; ++k) { Pm += p.P[(size_t)k * p.n_chan + c]; Tm += p.T[(size_t)k * p.n_chan + c]; }
    Pm /= (double)p.K; Tm /= (double)p.K;
    double spp = 0.0, spt = 0.0;
    for (int k = 0; k < p.K; ++k) {
        const double dP = p.P[(size_t)k * p.n_chan + c] - Pm, dT = p.T[(size_t)k * p.n_chan + c] - Tm;
        spp += dP * dP; spt += dP * dT;
    }
    double a = 0.0, b = 0.0;
    if (spp > 0.0) { b = spt / spp; a = Tm - b * Pm; }
    else atomicMax(p.bad, 1 + c);
    p.ab[c] = a; p.ab[p.n_chan + c] = b;
    p.abf[c] = make_float2((float)a, (float)b);
}

// tod[r][c] = a_c + b_c tod[r][c].  A block walks spans of 32 whole rows (contiguous, so the channel of an
// element is a 32-bit remainder of its offset in the span); 8 B per detector-sample.
constexpr int kKelvinRows = 32;
__global__ void __launch_bounds__(256) kelvin_kernel(float* __restrict__ tod, int64_t n_rows, int32_t n_chan,
                                                      const float2* __restrict__ abf) {
    const int64_t n_span = (n_rows + kKelvinRows - 1) / kKelvinRows;
    for (int64_t sp = blockIdx.x; sp < n_span; sp += gridDim.x) {
        const int64_t r0 = sp * kKelvinRows;
        const uint32_t len = (uint32_t)(min((int64_t)kKelvinRows, n_rows - r0) * n_chan);
        float* base = tod + r0 * n_chan;
        for (uint32_t j = threadIdx.x; j < len; j += 256) {
            const float2 ab = __ldg(abf + j % (uint32_t)n_chan);
            base[j] = fmaf(ab.y, base[j], ab.x);
        }
    }
}

}  // namespace gt
