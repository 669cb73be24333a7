// gt_fused_fp32.cuh -- steps 2-6a as ONE kernel on the FP32 CUDA cores (GT_VARIANT_FP32).
//
// north_star allows "FP32 CUDA cores if that is measured to be faster" than the split-TF32
// tensor path; this kernel is that measured alternative and the first correct CUDA path.
// Roofline: FP32 FMA pipe (2 * n_chan * n_freq flop per row), see DESIGN.md.
//
// Per CTA: a tile of BM = 64 rows x (32*TN) channels.  For each slab of BK = 32 frequencies
//   generate  A[k][row] = eps*Xn + eta*(G*S)      (steps 2-4 collapsed)
//   load      B[k][c]   = Fm^T slab               (coalesced from the transposed filter)
//   contract  acc[row][c] += A[k][row] * B[k][c]  (8 x TN register tile per thread)
// Every kF32_FlushSlabs slabs the register accumulators are added into the output tile (which
// the same thread owns) and cleared: an FFMA chain over 4000 positive terms drifts past the 1e-5
// gate (measured 1.8e-5 at n_freq = 4000), a chain of 512 does not.
// Epilogue: P_KID = (flushed + acc)*scale + bias[c]; photon noise (Philox keyed (seed, n, s, c)); store.
// The [n_freq x rows] spectrum lives only in shared memory.
#pragma once
#include "gt_common.cuh"

namespace gt {

struct FusedParams {
    const RowParam* rows;     // [n_rows] of this launch
    int64_t n_rows;
    int64_t t0;               // first sample of this launch (row r -> n = t0 + r / n_spaxel)
    int32_t n_spaxel, n_chan, n_freq, n_freq_pad;
    // collapsed-cascade coefficients per frequency (scaled by 1/P_ref), [n_freq_pad]
    const float *Xn, *Gs;
    // zenith transmission LUT resampled on the frequency grid, [n_pwv][n_freq_pad]
    const float* lut_r;
    // source cube [n_el][n_az][n_freq] (NULL = blank sky), n_az for the row stride
    const float* cube; int32_t n_az;
    // transposed zero-padded filter [n_freq_pad][n_chan_pad]
    const float* filt_t; int32_t n_chan_pad;
    // epilogue
    float scale;              // P_ref * dnu
    const float *bias;        // [n_chan_pad] dnu * sum_nu Fm * Y   (W)
    const float *noise_c1, *noise_c2;   // [n_chan_pad] h f_c f_s, f_s / dnu_c
    const float4* chan4;                // [n_chan_pad] {bias, noise_c1, noise_c2, 0}: one 16-byte load per output
    int32_t photon_noise; uint32_t seed_lo, seed_hi;
    uint32_t spaxel_base;     // global index of the plan's spaxel 0: Philox counter word 1 = spaxel_base + s
    float nep_f_sample, nep_sqrt_e0;   // Eq. 17 pass of the tensor kernel: sigma = sqrt(P f_s) sqrt(E0)
    float* out;               // [n_rows][n_chan]
};

// steps 2-4 for one (row, nu) element, collapsed form:
//   P_nu = eps * Xn + eta * (G * S) + Y,  eta = eta_z^csc,  eps = 1 - eta;  Y goes into bias[c].
__device__ __forceinline__ float element_value(float eta_z, float csc, float Xn, float GS) {
    const float eta = exp2f(csc * __log2f(eta_z));
    return fmaf(1.0f - eta, Xn, eta * GS);
}

constexpr int kF32_BM = 64, kF32_BK = 32, kF32_Threads = 256, kF32_AStride = 68;
constexpr int kF32_FlushSlabs = 16;     // 512 frequencies per accumulation segment

template <int TN>
__global__ void __launch_bounds__(kF32_Threads)
fused_fp32_kernel(const FusedParams p) {
    constexpr int NCB = 32 * TN;                    // channels per CTA
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* As = reinterpret_cast<float*>(smem_raw);                   // [BK][AStride]
    float* Bs = As + kF32_BK * kF32_AStride;                          // [BK][NCB]
    RowParam* rp_s = reinterpret_cast<RowParam*>(Bs + kF32_BK * NCB); // [BM]

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t row0 = (int64_t)blockIdx.x * kF32_BM;
    const int c0 = blockIdx.y * NCB;

    if (tid < kF32_BM) {
        RowParam rp;
        if (row0 + tid < p.n_rows) rp = p.rows[row0 + tid];
        else { rp.fp = 0.f; rp.csc = 1.f; rp.ip = 0; rp.pix = -1; rp.w00 = rp.w01 = rp.w10 = rp.w11 = 0.f; }
        rp_s[tid] = rp;
    }
    __syncthreads();

    float acc[8][TN];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < TN; ++j) acc[i][j] = 0.f;

    const size_t nf = (size_t)p.n_freq;
    int n_flushed = 0;
    for (int k0 = 0; k0 < p.n_freq_pad; k0 += kF32_BK) {
        // ---- segment boundary: move the partial sums into the output tile (thread-private elements) ----
        if (k0 > 0 && (k0 / kF32_BK) % kF32_FlushSlabs == 0) {
#pragma unroll
            for (int j = 0; j < TN; ++j) {
                const int c = c0 + lane + 32 * j;
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const int64_t r = row0 + warp * 8 + i;
                    if (c < p.n_chan && r < p.n_rows) {
                        float* o = p.out + (size_t)r * p.n_chan + c;
                        *o = n_flushed ? *o + acc[i][j] : acc[i][j];
                    }
                    acc[i][j] = 0.f;
                }
            }
            ++n_flushed;
        }
        // ---- generate the A slab: lane = frequency, 8 rows per thread ----
        {
            const int nu = k0 + lane;
            const float Xn = __ldg(p.Xn + nu), G = __ldg(p.Gs + nu);
            const bool in_grid = nu < p.n_freq;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int row = warp + 8 * i;
                const RowParam rp = rp_s[row];
                const float L0 = __ldg(p.lut_r + (size_t)rp.ip * p.n_freq_pad + nu);
                const float L1 = __ldg(p.lut_r + (size_t)(rp.ip + 1) * p.n_freq_pad + nu);
                const float eta_z = fmaf(rp.fp, L1 - L0, L0);
                float S = 0.f;
                if (rp.pix >= 0 && in_grid) {
                    const float* c00 = p.cube + (size_t)rp.pix * nf + nu;
                    S = rp.w00 * __ldg(c00) + rp.w01 * __ldg(c00 + nf)
                      + rp.w10 * __ldg(c00 + (size_t)p.n_az * nf) + rp.w11 * __ldg(c00 + (size_t)(p.n_az + 1) * nf);
                }
                As[lane * kF32_AStride + row] = element_value(eta_z, rp.csc, Xn, G * S);
            }
        }
        // ---- load the B slab ----
        {
            const float4* src = reinterpret_cast<const float4*>(p.filt_t + (size_t)k0 * p.n_chan_pad + c0);
            constexpr int V = NCB / 4;                              // float4 per k-row
            for (int idx = tid; idx < kF32_BK * V; idx += kF32_Threads) {
                const int k = idx / V, v = idx % V;
                reinterpret_cast<float4*>(Bs + k * NCB)[v] = __ldg(src + (size_t)k * (p.n_chan_pad / 4) + v);
            }
        }
        __syncthreads();
        // ---- contract ----
#pragma unroll 4
        for (int k = 0; k < kF32_BK; ++k) {
            const float4 a0 = *reinterpret_cast<const float4*>(As + k * kF32_AStride + warp * 8);
            const float4 a1 = *reinterpret_cast<const float4*>(As + k * kF32_AStride + warp * 8 + 4);
            const float a[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
            float b[TN];
#pragma unroll
            for (int j = 0; j < TN; ++j) b[j] = Bs[k * NCB + lane + 32 * j];
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < TN; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
        }
        __syncthreads();
    }

    // ---- epilogue: bias, photon noise (Eq. 18-19), store ----
#pragma unroll
    for (int j = 0; j < TN; ++j) {
        const int c = c0 + lane + 32 * j;
        if (c >= p.n_chan) continue;
        const float bias = __ldg(p.bias + c), n1 = __ldg(p.noise_c1 + c), n2 = __ldg(p.noise_c2 + c);
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int64_t r = row0 + warp * 8 + i;
            if (r >= p.n_rows) continue;
            float a = acc[i][j];
            if (n_flushed) a += p.out[(size_t)r * p.n_chan + c];
            float P = fmaf(a, p.scale, bias);
            if (p.photon_noise) {
                const uint32_t n = (uint32_t)(p.t0 + r / p.n_spaxel), s = (uint32_t)(r % p.n_spaxel);
                P = fmaf(photon_sigma(P, n1, n2), photon_normal(n, p.spaxel_base + s, (uint32_t)c, p.seed_lo, p.seed_hi), P);
            }
            p.out[(size_t)r * p.n_chan + c] = P;
        }
    }
}

}  // namespace gt
