// gt_pink.cuh -- step 6b: per-detector AR(1)-cascade pink noise (R18) added to the TOD.
//
//   x_j[n] = phi_j x_j[n-1] + sqrt(1 - phi_j^2) eps_j[n],   P_pn[n] = sum_j g_j x_j[n],
//   eps_j[n] = normal j of Philox(seed; n, spaxel, chan, stream 1 (j<4) / 2 (j>=4)),
//   x_j[-1]  = normal j of Philox(seed; 0xFFFFFFFF, spaxel, chan, stream 1/2).
//
// The recurrence is sequential in n but LINEAR, so a chunk of T samples is cut into segments of
// kPinkSeg samples that run in parallel (segments x detectors threads) and are chained through their end
// states in a single kernel (pink_chain_kernel): 8 B per detector-sample of HBM traffic on top of the
// fused kernel's 4 B, one Philox call per detector-sample.
#pragma once
#include "gt_common.cuh"
#include "gt_tc_ptx.cuh"     // packed fp32 pairs (FFMA2 / FMUL2 / FADD2)

namespace gt {

#ifndef GT_PINK_SEG
#define GT_PINK_SEG 64
#endif
constexpr int kPinkSeg = GT_PINK_SEG;
constexpr int kPinkBatch = 8;      // TOD values fetched ahead per thread
constexpr int kPinkMaxJ = 8;

struct PinkParams {
    int32_t J, n_chan;
    int64_t n_det;                 // n_spaxel * n_chan
    float phi[kPinkMaxJ], sq[kPinkMaxJ];     // phi_j, sqrt(1 - phi_j^2)
    const float* gain;             // [n_det][J]
    float* state;                  // [n_det][J] x_j at the sample before the chunk
    float* seg;                    // [n_seg][n_det][J] scratch: inclusive end state of every segment
    uint32_t* flags;               // [n_seg][n_det / 256] end state published; zeroed before every launch
    uint32_t* ticket;              // block ticket counter; zeroed before every launch
    uint32_t seed_lo, seed_hi;
    uint32_t spaxel_base;          // global index of the plan's spaxel 0 (Philox counter word 1)
    const float2* kelvin_ab;       // [n_chan] (a, b) of the brightness-temperature map T = a + b P, applied to the total of
                                   // Eq. 21 in the same write (nullptr: output in W, or applied elsewhere)
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
    pink_normals(p, kCounterInit, p.spaxel_base + (uint32_t)(d / p.n_chan), (uint32_t)(d % p.n_chan), z);
#pragma unroll
    for (int j = 0; j < kPinkMaxJ; ++j)
        if (j < p.J) p.state[d * p.J + j] = z[j];
}

// ONE pass over the TOD.  Block = 256 detectors x one segment of kPinkSeg samples; blocks take their
// (segment, detector block) from a ticket counter, so a block's predecessor (same detectors, previous
// segment) always started earlier.  Per thread:
//   1. the segment's series from a ZERO state (Philox + Box-Muller + J FMAs per sample), kept in shared
//      memory, and its end state e_j;
//   2. the true state at the segment start c_j: the plan state for segment 0, else the predecessor's
//      inclusive end state, published through global memory and a flag (acquire / release);
//   3. own inclusive end state phi_j^len c_j + e_j published at once (the chain advances before the TOD
//      is touched), the last segment's goes back into the plan state;
//   4. TOD += series + sum_j g_j phi_j^(m+1) c_j, one read-modify-write.
// The recurrence is linear, so 1 + 4 equals running it from the true state.
template <int JM>      // JM = 4 or 8: number of AR(1) stages the unrolled loops cover (J <= JM)
__global__ void __launch_bounds__(256)
pink_chain_kernel(PinkParams p, int64_t t0, int64_t T, float* __restrict__ tod) {
    extern __shared__ float s_pn[];                     // [kPinkSeg][256]
    __shared__ uint32_t s_ticket;
    const int tid = threadIdx.x;
    const uint32_t n_dblk = (uint32_t)((p.n_det + 255) / 256);
    if (tid == 0) s_ticket = atomicAdd(p.ticket, 1u);
    __syncthreads();
    const int64_t sg = s_ticket / n_dblk;
    const uint32_t db = s_ticket % n_dblk;
    const int64_t d = (int64_t)db * 256 + tid;
    const bool valid = d < p.n_det;
    const int64_t m0 = sg * kPinkSeg;
    const int len = (int)min((int64_t)kPinkSeg, T - m0);
    // The stages are worked in PAIRS (2i, 2i + 1) on packed fp32 (FFMA2 / FMUL2: two IEEE operations per issue slot; the
    // kernel is bound by instruction issue, profiles/r02a_pink.md): a pair shares one Box-Muller radius, its normals are
    // the cosine and the sine branch, so  x2 <- phi2 x2 + r (sq2 * (cos, sin)).
    using ptx::f32x2; using ptx::pk2; using ptx::upk2; using ptx::fma2; using ptx::mul2; using ptx::add2;
    float g[JM];
    f32x2 x2[JM / 2], g2[JM / 2], phi2[JM / 2], sq2[JM / 2];
#pragma unroll
    for (int j = 0; j < JM; ++j) g[j] = (valid && j < p.J) ? p.gain[d * p.J + j] : 0.f;
#pragma unroll
    for (int i = 0; i < JM / 2; ++i) {
        x2[i] = pk2(0.f, 0.f); g2[i] = pk2(g[2 * i], g[2 * i + 1]);
        phi2[i] = pk2(p.phi[2 * i], p.phi[2 * i + 1]); sq2[i] = pk2(p.sq[2 * i], p.sq[2 * i + 1]);
    }
    if (valid) {
        const uint32_t s = p.spaxel_base + (uint32_t)(d / p.n_chan), c = (uint32_t)(d % p.n_chan);
        const PhiloxKeys keys = philox_keys(p.seed_lo, p.seed_hi);      // the ten round keys, once per thread (21.6 -> 21.2 ms per C4 step)
        for (int m = 0; m < len; ++m) {        // two or four samples in flight (unrolled) gain nothing: 19.6 vs 19.8-20.1 ms per C4 step
            uint32_t w[JM];
            {
                const uint4 a = philox4x32_10((uint32_t)(t0 + m0 + m), s, c, kStreamPinkLo, keys);
                w[0] = a.x; w[1] = a.y; w[2] = a.z; w[3] = a.w;
            }
            if constexpr (JM > 4) {
                if (p.J > 4) {
                    const uint4 b = philox4x32_10((uint32_t)(t0 + m0 + m), s, c, kStreamPinkHi, keys);
                    w[4] = b.x; w[5] = b.y; w[6] = b.z; w[7] = b.w;
                } else {
                    w[4] = w[5] = w[6] = w[7] = 0u;       // stages 4-7 carry zero gains and zero states
                }
            }
            f32x2 pn2 = pk2(0.f, 0.f);
#pragma unroll
            for (int i = 0; i < JM / 2; ++i) {
                const float r = bm_radius(w[2 * i]);
                float sn, cs;
                __sincosf(bm_angle(w[2 * i + 1]), &sn, &cs);
                x2[i] = fma2(pk2(r, r), mul2(sq2[i], pk2(cs, sn)), mul2(phi2[i], x2[i]));
                pn2 = fma2(g2[i], x2[i], pn2);
            }
            const float2 pn = upk2(pn2);
            s_pn[m * 256 + tid] = pn.x + pn.y;
        }
    }
    float x[JM];
#pragma unroll
    for (int i = 0; i < JM / 2; ++i) { const float2 v = upk2(x2[i]); x[2 * i] = v.x; x[2 * i + 1] = v.y; }
    // state at the segment start
    if (sg > 0) {
        if (tid == 0) {
            const uint32_t* flag = p.flags + (size_t)(sg - 1) * n_dblk + db;
            uint32_t v;
            do {
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(flag) : "memory");
                if (v == 0u) __nanosleep(100);
            } while (v == 0u);
        }
        __syncthreads();
    }
    float cin[JM];
#pragma unroll
    for (int j = 0; j < JM; ++j) {
        cin[j] = 0.f;
        if (valid && j < p.J)
            cin[j] = sg > 0 ? __ldcg(p.seg + ((sg - 1) * p.n_det + d) * p.J + j) : p.state[d * p.J + j];
    }
    // publish the inclusive end state, then release the successor
    if (valid) {
#pragma unroll
        for (int j = 0; j < JM; ++j)
            if (j < p.J) {
                const float cout = fmaf(powf(p.phi[j], (float)len), cin[j], x[j]);
                __stcg(p.seg + (sg * p.n_det + d) * p.J + j, cout);
                if (m0 + len >= T) p.state[d * p.J + j] = cout;
            }
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        uint32_t* flag = p.flags + (size_t)sg * n_dblk + db;
        asm volatile("st.release.gpu.global.u32 [%0], %1;" :: "l"(flag), "r"(1u) : "memory");
    }
    // one read-modify-write of the TOD
    if (valid) {
        f32x2 a2[JM / 2];
#pragma unroll
        for (int i = 0; i < JM / 2; ++i) a2[i] = mul2(g2[i], pk2(cin[2 * i], cin[2 * i + 1]));
        float* col = tod + m0 * p.n_det + d;
        const float2 kab = p.kelvin_ab ? __ldg(p.kelvin_ab + d % p.n_chan) : make_float2(0.f, 1.f);
        for (int mb = 0; mb < len; mb += kPinkBatch) {
            float cur[kPinkBatch];
#pragma unroll
            for (int b = 0; b < kPinkBatch; ++b) cur[b] = mb + b < len ? __ldcs(col + (int64_t)(mb + b) * p.n_det) : 0.f;
#pragma unroll
            for (int b = 0; b < kPinkBatch; ++b) {
                const int m = mb + b;
                if (m < len) {
                    f32x2 add2v = pk2(0.f, 0.f);
#pragma unroll
                    for (int i = 0; i < JM / 2; ++i) { a2[i] = mul2(a2[i], phi2[i]); add2v = add2(add2v, a2[i]); }
                    const float2 add = upk2(add2v);
                    const float total = cur[b] + (s_pn[m * 256 + tid] + (add.x + add.y));
                    col[(int64_t)m * p.n_det] = p.kelvin_ab ? fmaf(kab.y, total, kab.x) : total;
                }
            }
        }
    }
}

}  // namespace gt
