// gt_pink.cuh -- step 6b: per-detector AR(1)-cascade pink noise (R18) added to the TOD.
//
//   x_j[n] = phi_j x_j[n-1] + sqrt(1 - phi_j^2) eps_j[n],   P_pn[n] = sum_j g_j x_j[n],
//   eps_j[n] = normal j of Philox(seed; n, spaxel, chan, stream 1 (j<4) / 2 (j>=4)),
//   x_j[-1]  = normal j of Philox(seed; 0xFFFFFFFF, spaxel, chan, stream 1/2).
//
// The recurrence is sequential in n but LINEAR, so a chunk of T samples is cut into segments
// of kPinkSeg samples that run in parallel (detectors x segments threads):
//   pink_local : x from a ZERO state inside each segment, adds sum_j g_j x_j to the TOD,
//                stores the segment's end state e_j                       (HBM: TOD read+write)
//   pink_carry : per detector, sequential over segments: true state at each segment start
//                c[seg+1] = phi^len c[seg] + e[seg]; final state -> plan   (tiny)
//   pink_fixup : adds sum_j g_j phi_j^(m+1) c_j[seg] at offset m of each segment (TOD read+write)
// HBM-bound: 16 B per detector-sample of traffic on top of the fused kernel's 4 B.
#pragma once
#include "gt_common.cuh"

namespace gt {

constexpr int kPinkSeg = 64;
constexpr int kPinkBatch = 8;      // TOD values fetched ahead per thread
constexpr int kPinkMaxJ = 8;

struct PinkParams {
    int32_t J, n_chan;
    int64_t n_det;                 // n_spaxel * n_chan
    float phi[kPinkMaxJ], sq[kPinkMaxJ];     // phi_j, sqrt(1 - phi_j^2)
    const float* gain;             // [n_det][J]
    float* state;                  // [n_det][J] x_j at the sample before the chunk
    float* seg;                    // [n_seg][n_det][J] scratch: e (after local), c (after carry)
    uint32_t seed_lo, seed_hi;
};

__device__ __forceinline__ void pink_normals(const PinkParams& p, uint32_t c0, uint32_t s, uint32_t c,
                                             float z[kPinkMaxJ]) {
    const uint4 w = philox4x32_10(c0, s, c, kStreamPinkLo, p.seed_lo, p.seed_hi);
    normal_pair(w.x, w.y, z[0], z[1]);
    normal_pair(w.z, w.w, z[2], z[3]);
    if (p.J > 4) {
        const uint4 v = philox4x32_10(c0, s, c, kStreamPinkHi, p.seed_lo, p.seed_hi);
        normal_pair(v.x, v.y, z[4], z[5]);
        normal_pair(v.z, v.w, z[6], z[7]);
    } else {
        z[4] = z[5] = z[6] = z[7] = 0.f;
    }
}

// state <- x_j[-1] (called when a run starts at sample 0)
__global__ void __launch_bounds__(256) pink_init_kernel(PinkParams p) {
    const int64_t d = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (d >= p.n_det) return;
    float z[kPinkMaxJ];
    pink_normals(p, kCounterInit, (uint32_t)(d / p.n_chan), (uint32_t)(d % p.n_chan), z);
#pragma unroll
    for (int j = 0; j < kPinkMaxJ; ++j)
        if (j < p.J) p.state[d * p.J + j] = z[j];
}

// thread = (segment, detector); detectors fastest so that TOD accesses coalesce.
template <int JM>      // JM = 4 or 8: number of AR(1) stages the unrolled loops cover (J <= JM)
__global__ void __launch_bounds__(256)
pink_local_kernel(PinkParams p, int64_t t0, int64_t T, float* __restrict__ tod) {
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t n_seg = (T + kPinkSeg - 1) / kPinkSeg;
    if (idx >= n_seg * p.n_det) return;
    const int64_t sg = idx / p.n_det, d = idx % p.n_det;
    const uint32_t s = (uint32_t)(d / p.n_chan), c = (uint32_t)(d % p.n_chan);
    float g[kPinkMaxJ], x[kPinkMaxJ];
#pragma unroll
    for (int j = 0; j < JM; ++j) { g[j] = j < p.J ? p.gain[d * p.J + j] : 0.f; x[j] = 0.f; }
    const int64_t m0 = sg * kPinkSeg, m1 = min(m0 + (int64_t)kPinkSeg, T);
    // batches of kPinkBatch samples: the TOD values are fetched first (independent loads in flight while the
    // Philox / Box-Muller arithmetic runs), the recurrence itself stays strictly sequential in m
    for (int64_t mb = m0; mb < m1; mb += kPinkBatch) {
        float cur[kPinkBatch];
#pragma unroll
        for (int b = 0; b < kPinkBatch; ++b) cur[b] = mb + b < m1 ? __ldcs(tod + (mb + b) * p.n_det + d) : 0.f;
#pragma unroll
        for (int b = 0; b < kPinkBatch; ++b) {
            const int64_t m = mb + b;
            if (m < m1) {
                float z[kPinkMaxJ];
                pink_normals(p, (uint32_t)(t0 + m), s, c, z);
                float pn = 0.f;
#pragma unroll
                for (int j = 0; j < JM; ++j) {
                    x[j] = fmaf(p.phi[j], x[j], p.sq[j] * z[j]);
                    pn = fmaf(g[j], x[j], pn);
                }
                tod[m * p.n_det + d] = cur[b] + pn;
            }
        }
    }
#pragma unroll
    for (int j = 0; j < JM; ++j)
        if (j < p.J) p.seg[(sg * p.n_det + d) * p.J + j] = x[j];
}

// thread = (detector, stage): walks the segments, replaces e[seg] by the state at the segment start.
// The chain c <- phi^len c + e is a dependent FMA per segment, but its inputs are not: they are
// fetched 16 segments at a time so that the walk costs one memory round trip per batch instead of one
// per segment.
__global__ void __launch_bounds__(256) pink_carry_kernel(PinkParams p, int64_t T) {
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= p.n_det * p.J) return;
    const int j = (int)(idx % p.J);
    const int64_t n_seg = (T + kPinkSeg - 1) / kPinkSeg;
    const int64_t stride = p.n_det * p.J;                  // seg[sg][d][j]: idx is the offset inside one segment slice
    float cst = p.state[idx];
    const float phi = p.phi[j];
    const float phiL = powf(phi, (float)kPinkSeg);
    constexpr int kBatch = 16;
    for (int64_t s0 = 0; s0 < n_seg; s0 += kBatch) {
        float e[kBatch];
#pragma unroll
        for (int b = 0; b < kBatch; ++b) e[b] = s0 + b < n_seg ? p.seg[(s0 + b) * stride + idx] : 0.f;
#pragma unroll
        for (int b = 0; b < kBatch; ++b) {
            const int64_t sg = s0 + b;
            if (sg < n_seg) {
                p.seg[sg * stride + idx] = cst;
                const int64_t len = min((int64_t)kPinkSeg, T - sg * kPinkSeg);
                cst = fmaf(len == kPinkSeg ? phiL : powf(phi, (float)len), cst, e[b]);
            }
        }
    }
    p.state[idx] = cst;
}

template <int JM>
__global__ void __launch_bounds__(256)
pink_fixup_kernel(PinkParams p, int64_t T, float* __restrict__ tod) {
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t n_seg = (T + kPinkSeg - 1) / kPinkSeg;
    if (idx >= n_seg * p.n_det) return;
    const int64_t sg = idx / p.n_det, d = idx % p.n_det;
    float a[kPinkMaxJ];       // g_j * phi_j^(m+1) * c_j
#pragma unroll
    for (int j = 0; j < JM; ++j)
        a[j] = j < p.J ? p.gain[d * p.J + j] * p.seg[(sg * p.n_det + d) * p.J + j] : 0.f;
    const int64_t m0 = sg * kPinkSeg, m1 = min(m0 + (int64_t)kPinkSeg, T);
    for (int64_t mb = m0; mb < m1; mb += kPinkBatch) {
        float cur[kPinkBatch];
#pragma unroll
        for (int b = 0; b < kPinkBatch; ++b) cur[b] = mb + b < m1 ? __ldcs(tod + (mb + b) * p.n_det + d) : 0.f;
#pragma unroll
        for (int b = 0; b < kPinkBatch; ++b) {
            const int64_t m = mb + b;
            if (m < m1) {
                float add = 0.f;
#pragma unroll
                for (int j = 0; j < JM; ++j) { a[j] *= p.phi[j]; add += a[j]; }
                tod[m * p.n_det + d] = cur[b] + add;
            }
        }
    }
}

}  // namespace gt
