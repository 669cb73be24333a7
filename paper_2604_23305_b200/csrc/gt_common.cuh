// gt_common.cuh -- shared device-side definitions of the CUDA path (libgateau_b200.so).
// Shares nothing with oracle/: the constants and the Philox rounds below are restated from
// PAPER.md / DESIGN.md for the device.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gt {

// ---- per-row record handed from the geometry kernel to the fused kernel (32 B) --------
struct __align__(16) RowParam {
    float fp;          // LUT fraction in PWV
    float csc;         // airmass 1/sin(E), Eq. 10
    int32_t ip;        // lower LUT row
    int32_t pix;       // source pixel index jv*n_az + ju of the lower-left tap, -1 = outside (S = 0)
    float w00, w01, w10, w11;   // bilinear source weights (jv,ju) (jv,ju+1) (jv+1,ju) (jv+1,ju+1)
};
static_assert(sizeof(RowParam) == 32, "RowParam must be 32 bytes");

// ---- Philox4x32-10 (Salmon et al. SC'11; R19) --------------------------------
// counter = (c0 = sample n, c1 = spaxel, c2 = channel, c3 = stream), key = 64-bit seed.
constexpr uint32_t kPhiloxM0 = 0xD2511F53u, kPhiloxM1 = 0xCD9E8D57u;
constexpr uint32_t kPhiloxW0 = 0x9E3779B9u, kPhiloxW1 = 0xBB67AE85u;
constexpr uint32_t kStreamPhoton = 0u, kStreamPinkLo = 1u, kStreamPinkHi = 2u;
constexpr uint32_t kCounterInit = 0xFFFFFFFFu;

__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(kPhiloxM0, c0), lo0 = kPhiloxM0 * c0;
        const uint32_t hi1 = __umulhi(kPhiloxM1, c2), lo1 = kPhiloxM1 * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += kPhiloxW0; k1 += kPhiloxW1;
    }
    return make_uint4(c0, c1, c2, c3);
}

// The same with the ten round keys made by the caller (a loop that draws one block per iteration keeps them in registers
// instead of re-deriving them every time).
struct PhiloxKeys { uint32_t k0[10], k1[10]; };
__device__ __forceinline__ PhiloxKeys philox_keys(uint32_t k0, uint32_t k1) {
    PhiloxKeys K;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        K.k0[r] = k0 + (uint32_t)r * kPhiloxW0; K.k1[r] = k1 + (uint32_t)r * kPhiloxW1;
        asm volatile("" : "+r"(K.k0[r]), "+r"(K.k1[r]));          // opaque: not re-materialised inside the loop
    }
    return K;
}
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const PhiloxKeys& K) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(kPhiloxM0, c0), lo0 = kPhiloxM0 * c0;
        const uint32_t hi1 = __umulhi(kPhiloxM1, c2), lo1 = kPhiloxM1 * c2;
        const uint32_t n0 = hi1 ^ c1 ^ K.k0[r];
        const uint32_t n2 = hi0 ^ c3 ^ K.k1[r];
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    }
    return make_uint4(c0, c1, c2, c3);
}

// W independent Philox4x32-10 blocks at once: the ten rounds of one block are a strictly serial
// chain (~10 cycles per round), so a lone warp only fills its issue slots if it interleaves
// several blocks.  Same arithmetic as philox4x32_10; counters differ in word 2 (the channel).
template <int W>
__device__ __forceinline__ void philox4x32_10_multi(uint32_t c0, uint32_t c1, const uint32_t (&c2)[W], uint32_t c3,
                                                    uint32_t k0, uint32_t k1, uint32_t (&o0)[W], uint32_t (&o1)[W]) {
    uint32_t a[W], b[W], c[W], d[W];
#pragma unroll
    for (int i = 0; i < W; ++i) { a[i] = c0; b[i] = c1; c[i] = c2[i]; d[i] = c3; }
#pragma unroll
    for (int r = 0; r < 10; ++r) {
#pragma unroll
        for (int i = 0; i < W; ++i) {
            const uint32_t hi0 = __umulhi(kPhiloxM0, a[i]), lo0 = kPhiloxM0 * a[i];
            const uint32_t hi1 = __umulhi(kPhiloxM1, c[i]), lo1 = kPhiloxM1 * c[i];
            a[i] = hi1 ^ b[i] ^ k0; b[i] = lo1; c[i] = hi0 ^ d[i] ^ k1; d[i] = lo0;
        }
        k0 += kPhiloxW0; k1 += kPhiloxW1;
    }
#pragma unroll
    for (int i = 0; i < W; ++i) { o0[i] = a[i]; o1[i] = b[i]; }      // words 0 and 1
}
template <int W>
__device__ __forceinline__ void philox4x32_10_multi4(uint32_t c0, uint32_t c1, const uint32_t (&c2)[W], uint32_t c3,
                                                     uint32_t k0, uint32_t k1, uint4 (&o)[W]) {
    uint32_t a[W], b[W], c[W], d[W];
#pragma unroll
    for (int i = 0; i < W; ++i) { a[i] = c0; b[i] = c1; c[i] = c2[i]; d[i] = c3; }
#pragma unroll
    for (int r = 0; r < 10; ++r) {
#pragma unroll
        for (int i = 0; i < W; ++i) {
            const uint32_t hi0 = __umulhi(kPhiloxM0, a[i]), lo0 = kPhiloxM0 * a[i];
            const uint32_t hi1 = __umulhi(kPhiloxM1, c[i]), lo1 = kPhiloxM1 * c[i];
            a[i] = hi1 ^ b[i] ^ k0; b[i] = lo1; c[i] = hi0 ^ d[i] ^ k1; d[i] = lo0;
        }
        k0 += kPhiloxW0; k1 += kPhiloxW1;
    }
#pragma unroll
    for (int i = 0; i < W; ++i) o[i] = make_uint4(a[i], b[i], c[i], d[i]);
}

// U(w) = ((w >> 9) + 1/2) 2^-23 in (0,1): exact in fp32 (R19), as ONE fused multiply-add (the product and the
// sum are both exact, so this equals the two-step form bit for bit).
__device__ __forceinline__ float uniform01(uint32_t w) {
    return fmaf((float)(w >> 9), 1.0f / 8388608.0f, 0.5f / 8388608.0f);
}

// Box-Muller: z0 = sqrt(-2 ln U(w0)) cos(2 pi U(w1)), z1 = ... sin(...).  MUFU log/sin/cos: the
// normals only need ~1e-3 absolute accuracy for the 2e-5 TOD gate (sigma/P ~ 1e-3).
// MUFU.SQRT (2^-22 relative): sqrtf's IEEE path costs a dozen instructions and a slow-path call
__device__ __forceinline__ float sqrt_fast(float x) {
    float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r;
}
// radius sqrt(-2 ln U(w)) = sqrt(-2 ln2 log2 U): U >= 2^-24 is a normal number, so the bare MUFU.LG2 serves (__logf adds a
// denormal branch of three instructions) and the two constants fold into one multiply
__device__ __forceinline__ float bm_radius(uint32_t w) {
    float l; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(l) : "f"(uniform01(w)));
    return sqrt_fast(-1.38629436111989061883f * l);
}
// angle 2 pi U(w) in one fused multiply-add (one rounding instead of two: 2^-24 relative, far inside MUFU.SIN's own error)
__device__ __forceinline__ float bm_angle(uint32_t w) {
    return fmaf((float)(w >> 9), 6.28318530717958647692f / 8388608.0f, 3.14159265358979323846f / 8388608.0f);
}
__device__ __forceinline__ float normal_cos(uint32_t w0, uint32_t w1) {
    return bm_radius(w0) * __cosf(bm_angle(w1));
}
__device__ __forceinline__ void normal_pair(uint32_t w0, uint32_t w1, float& z0, float& z1) {
    const float r = bm_radius(w0);
    float s, c;
    __sincosf(bm_angle(w1), &s, &c);
    z0 = r * c; z1 = r * s;
}

// Photon noise (stream 0, R19): one block yields four normals and serves the channels b + 128 q + {0, 32, 64, 96}:
// channel c uses normal photon_slot(c) of the block with counter word 2 = photon_block(c).
__device__ __forceinline__ uint32_t photon_block(uint32_t c) { return ((c >> 7) << 5) | (c & 31u); }
__device__ __forceinline__ uint32_t photon_slot(uint32_t c) { return (c >> 5) & 3u; }
__device__ __forceinline__ void normals_of_block(const uint4& w, float (&z)[4]) {
    normal_pair(w.x, w.y, z[0], z[1]);
    normal_pair(w.z, w.w, z[2], z[3]);
}
// one channel on its own (FP32 kernel: the whole block for one normal; the tensor kernel's finisher uses all four)
__device__ __forceinline__ float photon_normal(uint32_t n, uint32_t spaxel, uint32_t c, uint32_t seed_lo, uint32_t seed_hi) {
    const uint4 w = philox4x32_10(n, spaxel, photon_block(c), kStreamPhoton, seed_lo, seed_hi);
    const uint32_t k = photon_slot(c);
    const float r = bm_radius(k < 2u ? w.x : w.z), a = bm_angle(k < 2u ? w.y : w.w);
    return r * ((k & 1u) ? __sinf(a) : __cosf(a));
}

// sigma of Eq. 18 in north_star's narrow-band form (R17):
// sigma^2 = (2 h f_c P + 2 P^2 / dnu_c) f_s / 2 = P (c1 + P c2), c1 = h f_c f_s, c2 = f_s / dnu_c.
__device__ __forceinline__ float photon_sigma(float P, float c1, float c2) {
    const float v = P * (c1 + P * c2);
    return v > 0.0f ? sqrt_fast(v) : 0.0f;
}

}  // namespace gt
