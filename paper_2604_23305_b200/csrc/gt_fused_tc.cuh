// gt_fused_tc.cuh -- steps 2-6a as ONE tcgen05 tensor-core kernel (GT_VARIANT_TENSOR).
//
//   P_KID[row][c] = dnu * sum_nu Fm[c][nu] * P[row][nu]                       (Eq. 16)
// is a dense [rows x n_freq] . [n_freq x n_chan] contraction whose left operand is GENERATED
// (steps 2-4, collapsed cascade of DESIGN.md) and never exists in HBM.  Per persistent CTA
// (one per SM) and per tile of 128 rows:
//
//   generator warps (8)   : 32-frequency slab of the spectrum for 128 rows -> split into
//                           tf32 hi + lo -> shared memory in the UMMA K-major SWIZZLE_128B layout
//   loader warp (1 lane)  : filter slab images (hi, lo; pre-split, pre-swizzled at plan time)
//                           global -> shared by cp.async.bulk, mbarrier complete_tx
//   MMA warp (1 lane)     : tcgen05.mma.kind::tf32, M = 128, N <= 128 per column group, K = 8:
//                           acc += A_hi.B_hi + A_lo.B_hi + A_hi.B_lo     ("3xTF32", fp32 accumulate
//                           in tensor memory; the dropped A_lo.B_lo term is ~2^-22 relative)
//   epilogue warps (4)    : SEGMENTED ACCUMULATION.  The tensor core's fp32 accumulate truncates
//                           (measured: -2.7e-5 relative after 500 chained MMAs of positive terms,
//                           DESIGN.md "Accumulation in tensor memory"), so no accumulator lives
//                           longer than `seg` slabs: the <= 384 padded channels of a tile are cut
//                           into <= 3 column groups of <= 128 columns that rotate through FOUR
//                           128-column tensor-memory buffers; at a (staggered) segment boundary a
//                           group moves to the spare buffer and the epilogue warps add the
//                           finished partial sums (tcgen05.ld) into a per-CTA, L2-resident fp32
//                           scratch tile [column][row] with round-to-nearest FADDs.  After the
//                           last segment they transpose the scratch tile into the TOD:
//                           P = sum*scale + bias[c], photon noise (Eq. 18-19), coalesced stores.
//
// Pipelines: A ring (2 stages, generator -> MMA), B ring (loader -> MMA), accumulator buffers
// flush_full / buf_free (MMA <-> epilogue); all mbarrier based.
#pragma once
#include <vector>
#include <cstring>
#include <algorithm>
#include "gt_common.cuh"
#include "gt_fused_fp32.cuh"
#include "gt_tc_ptx.cuh"
#include "../../include/gateau_b200.h"

namespace gt {

constexpr int kTcBM = 128;                 // rows per tile (UMMA M)
constexpr int kTcBK = 32;                  // frequencies per A stage / B unit: one 128-byte swizzle row
constexpr int kTcUK = 8;                   // K of one tcgen05.mma.kind::tf32
constexpr int kTcAStages = 2;
constexpr int kTcAPartBytes = kTcBM * kTcBK * 4;            // 16 KB (hi or lo)
constexpr int kTcAStageBytes = 2 * kTcAPartBytes;           // 32 KB
constexpr int kTcEpiWarps = 4, kTcGenWarps = 8;
// warp roles, aligned to warpgroups of 4 warps so that setmaxnreg can move registers between them:
//   WG0 = warps 0-3 flush (tensor-memory lane quarter = warp), WG1 = loader, MMA, 2 idle,
//   WG2-3 = generators, WG4 = finishers.  The kernel starts with 96 registers per thread (640 threads);
//   setmaxnreg can only redistribute that pool: 128 x (112 + 40 + 2*128 + 72) = 128 x 5*96.
constexpr int kTcWarpLoader = 4, kTcWarpMma = 5, kTcWarpGen0 = 8;
constexpr int kTcFinWarps = 4, kTcWarpFin0 = kTcWarpGen0 + kTcGenWarps;            // 16
constexpr int kTcThreads = 32 * (kTcWarpFin0 + kTcFinWarps);                        // 640
constexpr int kTcRegsFlush = 112, kTcRegsCtl = 40, kTcRegsGen = 128, kTcRegsFin = 72;
static_assert(kTcRegsFlush + kTcRegsCtl + 2 * kTcRegsGen + kTcRegsFin <= 5 * 96, "setmaxnreg pool");
constexpr int kTcMaxGroupChan = 384;       // channels per tile: 3 column groups of 128 (+ 1 spare buffer = 512 columns)
constexpr int kTcBufCols = 128, kTcNumBuf = 4, kTcMaxCg = 3;
constexpr int kTcSegDefault = 8;           // slabs (of 32 frequencies) per accumulation segment
constexpr int kTcMaxBStages = 4;
constexpr int kTcSmemLimit = 227 * 1024;

struct TcTables {
    unsigned char* filt_img = nullptr;   // [group][kb][part hi/lo][NBtot rows][128 B swizzled]
    float* scratch = nullptr;            // [num CTAs][2][nb_tot][128] fp32 partial sums (L2 resident)
    int32_t n_groups = 0;                // channel groups (tiles along the channel axis) of <= 384 channels
    int32_t nb_tot = 0;                  // padded channels per group (multiple of 32)
    int32_t n_cg = 0;                    // column groups per tile, widths 128,..,remainder
    int32_t seg = kTcSegDefault;         // slabs per accumulation segment
    int32_t n_kb = 0;                    // n_freq_pad / 32
    int32_t unit_bytes = 0;              // nb_tot * 128
    int32_t b_stages = 0;
    int32_t smem_bytes = 0;
};

inline const char*& tc_error_ref() { static const char* e = ""; return e; }
inline const char* tc_error() { return tc_error_ref(); }

// round-to-nearest (ties away) fp32 -> tf32 on the host, finite inputs
inline float host_tf32(float x) {
    uint32_t b; std::memcpy(&b, &x, 4);
    b = (b + 0x1000u) & 0xFFFFE000u;
    float r; std::memcpy(&r, &b, 4);
    return r;
}

// Splits the filter into tf32 hi/lo parts and lays every (group, 32-frequency slab, part) out as
// the exact shared-memory image tcgen05.mma reads (K-major, SWIZZLE_128B): the loader is a flat copy.
inline gt_status build_tc_tables(const std::vector<float>& filt, int n_chan, int n_freq, int n_freq_pad,
                                 TcTables& t, cudaStream_t st) {
    const int G = (n_chan + kTcMaxGroupChan - 1) / kTcMaxGroupChan;
    int per = (n_chan + G - 1) / G;
    const int nbt = (per + 31) / 32 * 32;
    t.n_groups = G; t.nb_tot = nbt;
    t.n_cg = (nbt + kTcBufCols - 1) / kTcBufCols;
    t.n_kb = n_freq_pad / kTcBK;
    t.unit_bytes = nbt * 128;
    const int fixed = kTcAStages * kTcAStageBytes + 1024 /*alignment slack*/ + 256 /*barriers*/;   // barriers use 164 B
    t.b_stages = std::min(kTcMaxBStages, (kTcSmemLimit - fixed) / t.unit_bytes);
    if (t.b_stages < 2) { tc_error_ref() = "filter slab does not fit in shared memory"; return GT_ERR_UNSUPPORTED; }
    t.smem_bytes = fixed + t.b_stages * t.unit_bytes;

    const size_t total = (size_t)G * t.n_kb * 2 * t.unit_bytes;
    std::vector<float> img(total / 4, 0.f);
    for (int g = 0; g < G; ++g)
        for (int n = 0; n < nbt; ++n) {
            const int ch = g * nbt + n;
            if (ch >= n_chan) continue;
            for (int i = 0; i < n_freq; ++i) {
                const float f = filt[(size_t)ch * n_freq + i];
                const float hi = host_tf32(f), lo = host_tf32(f - hi);
                const int kb = i / kTcBK, kk = i % kTcBK;
                const size_t unit0 = ((size_t)(g * t.n_kb + kb) * 2) * (t.unit_bytes / 4);
                const size_t off = (size_t)n * 32 + (size_t)(((kk >> 2) ^ (n & 7)) << 2) + (kk & 3);
                img[unit0 + off] = hi;
                img[unit0 + t.unit_bytes / 4 + off] = lo;
            }
        }
    if (cudaMalloc(reinterpret_cast<void**>(&t.filt_img), total) != cudaSuccess) {
        cudaGetLastError(); tc_error_ref() = "cudaMalloc of the filter image failed"; return GT_ERR_OOM;
    }
    if (cudaMemcpyAsync(t.filt_img, img.data(), total, cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess) {
        cudaGetLastError(); tc_error_ref() = "upload of the filter image failed"; return GT_ERR_CUDA;
    }
    return GT_OK;
}
// per-CTA scratch tile of partial sums; grid = one CTA per SM
inline gt_status alloc_tc_scratch(TcTables& t, int num_sms) {
    if (t.scratch) return GT_OK;
    const size_t bytes = (size_t)num_sms * 2 * t.nb_tot * kTcBM * sizeof(float);     // two tiles per CTA
    if (cudaMalloc(reinterpret_cast<void**>(&t.scratch), bytes) != cudaSuccess) {
        cudaGetLastError(); tc_error_ref() = "cudaMalloc of the partial-sum scratch failed"; return GT_ERR_OOM;
    }
    return GT_OK;
}
inline void free_tc_tables(TcTables& t) {
    if (t.filt_img) cudaFree(t.filt_img);
    if (t.scratch) cudaFree(t.scratch);
    t.filt_img = nullptr; t.scratch = nullptr;
}

struct TcParams {
    FusedParams f;
    const unsigned char* filt_img;
    float* scratch;
    int32_t n_groups, nb_tot, n_cg, seg, n_kb, unit_bytes, b_stages;
    int32_t n_row_tiles;
    int32_t cube_vec;           // 1: cube spectra can be read as aligned float4
};

// shared-memory map relative to the 1024-byte aligned base:
//   [0, 64 KB)                      A ring: stage s at s*32 KB = {hi 16 KB, lo 16 KB}
//   [64 KB, 64 KB + NBS*unit)       B ring
//   then barriers: a_full[2] a_empty[2] b_full[4] b_empty[4] flush_full[4] buf_free[4] tile_done[2]
//   scratch_free[2], tensor-memory slot
struct TcSmem {
    uint32_t a, b, a_full, a_empty, b_full, b_empty, flush_full, buf_free, tile_done, scratch_free, slot;
    __device__ TcSmem(uint32_t base, int b_stages, int unit_bytes) {
        a = base; b = base + kTcAStages * kTcAStageBytes;
        const uint32_t bar = b + (uint32_t)b_stages * (uint32_t)unit_bytes;
        a_full = bar; a_empty = bar + 16; b_full = bar + 32; b_empty = bar + 64;
        flush_full = bar + 96; buf_free = bar + 128; tile_done = bar + 160; scratch_free = bar + 176; slot = bar + 192;
    }
};

// Column groups of a tile and the rotation of their accumulators through the tensor-memory
// buffers.  The MMA thread and the epilogue warps each run one instance over the same
// (tile, slab, group) sequence, so they agree on which buffer a group occupies without talking.
struct TcRotation {
    int n_cg, seg, n_kb;
    int buf[kTcMaxCg];             // buffer each group accumulates into
    int fifo[kTcNumBuf]; int head, count;   // free buffers, oldest first
    __device__ TcRotation(int n_cg_, int seg_, int n_kb_) : n_cg(n_cg_), seg(seg_), n_kb(n_kb_), head(0), count(0) {
        for (int g = 0; g < kTcMaxCg; ++g) buf[g] = g;
        for (int b = n_cg_; b < kTcNumBuf; ++b) fifo[count++] = b;
    }
    // group g closes a segment after slab kb (staggered so that flushes do not coincide)
    __device__ bool boundary(int kb, int g) const {
        return kb == n_kb - 1 || ((kb + 1 + (g * seg) / n_cg) % seg) == 0;
    }
    // moves group g to the oldest free buffer; returns the buffer it leaves
    __device__ int rotate(int g) {
        const int old = buf[g];
        const int nb = fifo[head];
        fifo[head] = old;                   // count stays the same: pop head, push tail (ring of size count)
        head = (head + 1) % count;
        buf[g] = nb;
        return old;
    }
    __device__ static int col0(int g) { return g * kTcBufCols; }
    __device__ int width(int g, int nb_tot) const { return min(kTcBufCols, nb_tot - g * kTcBufCols); }
};

__device__ __forceinline__ float4 ldg4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }

template <bool VEC>
__global__ void __launch_bounds__(kTcThreads, 1)
fused_tc_kernel(const TcParams p) {
    extern __shared__ unsigned char smem_raw[];
    const uint32_t raw = ptx::smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;
    const TcSmem sm(base, p.b_stages, p.unit_bytes);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const FusedParams& f = p.f;

    if (tid == 0) {
        for (int s = 0; s < kTcAStages; ++s) {
            ptx::mbar_init(sm.a_full + 8 * s, 32 * kTcGenWarps);
            ptx::mbar_init(sm.a_empty + 8 * s, 1);
        }
        for (int s = 0; s < kTcMaxBStages; ++s) {
            ptx::mbar_init(sm.b_full + 8 * s, 1);
            ptx::mbar_init(sm.b_empty + 8 * s, 1);
        }
        for (int b = 0; b < kTcNumBuf; ++b) {
            ptx::mbar_init(sm.flush_full + 8 * b, 1);
            ptx::mbar_init(sm.buf_free + 8 * b, 32 * kTcEpiWarps);
        }
        for (int b = 0; b < 2; ++b) {
            ptx::mbar_init(sm.tile_done + 8 * b, 32 * kTcEpiWarps);
            ptx::mbar_init(sm.scratch_free + 8 * b, 32 * kTcFinWarps);
        }
        ptx::fence_mbar_init();
    }
    if (warp == kTcWarpMma) {
        ptx::tmem_alloc(sm.slot, 512);
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = *reinterpret_cast<const volatile uint32_t*>(smem_raw + (sm.slot - raw));

    const int64_t n_tiles = (int64_t)p.n_row_tiles * p.n_groups;

    if (warp >= kTcWarpGen0 && warp < kTcWarpFin0) {
        // =========================== generator: steps 2-4 -> A ring ===========================
        ptx::setmaxnreg_inc<kTcRegsGen>();
        const int gw = warp - kTcWarpGen0;
        const int rsub = gw * 4 + (lane >> 3), chunk = lane & 7;
        const uint32_t swz = (uint32_t)((chunk ^ (rsub & 7)) << 4);
        const size_t nf = (size_t)f.n_freq, nfp = (size_t)f.n_freq_pad;
        uint32_t it = 0;
        for (int64_t tl = blockIdx.x; tl < n_tiles; tl += gridDim.x) {
            const int64_t row0 = (tl / p.n_groups) * kTcBM;
            float fp[4], csc[4], w00[4], w01[4], w10[4], w11[4];
            const float* lutp[4];
            const float* cubep[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int64_t R = row0 + rsub + 32 * j;
                RowParam rp;
                if (R < f.n_rows) {
                    const int4* src = reinterpret_cast<const int4*>(f.rows + R);
                    const int4 a = __ldg(src), b = __ldg(src + 1);
                    rp.fp = __int_as_float(a.x); rp.csc = __int_as_float(a.y); rp.ip = a.z; rp.pix = a.w;
                    rp.w00 = __int_as_float(b.x); rp.w01 = __int_as_float(b.y);
                    rp.w10 = __int_as_float(b.z); rp.w11 = __int_as_float(b.w);
                } else {
                    rp.fp = 0.f; rp.csc = 1.f; rp.ip = 0; rp.pix = -1; rp.w00 = rp.w01 = rp.w10 = rp.w11 = 0.f;
                }
                fp[j] = rp.fp; csc[j] = rp.csc; w00[j] = rp.w00; w01[j] = rp.w01; w10[j] = rp.w10; w11[j] = rp.w11;
                lutp[j] = f.lut_r + (size_t)rp.ip * nfp + chunk * 4;
                cubep[j] = (rp.pix >= 0 && f.cube) ? f.cube + (size_t)rp.pix * nf + chunk * 4 : nullptr;
            }
            for (int kb = 0; kb < p.n_kb; ++kb, ++it) {
                const uint32_t stage = it & 1u, ph = (it >> 1) & 1u;
                const int nu0 = kb * kTcBK + chunk * 4;
                const float4 X = ldg4(f.Xn + nu0), G = ldg4(f.Gs + nu0);
                float4 L0[4], L1[4], S[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    L0[j] = ldg4(lutp[j] + kb * kTcBK);
                    L1[j] = ldg4(lutp[j] + nfp + kb * kTcBK);
                    S[j] = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (cubep[j] != nullptr && nu0 < f.n_freq) {
                        const float* c00 = cubep[j] + kb * kTcBK;
                        const float* c01 = c00 + nf;
                        const float* c10 = c00 + (size_t)f.n_az * nf;
                        const float* c11 = c10 + nf;
                        if (VEC) {
                            const float4 a = ldg4(c00), b = ldg4(c01), c = ldg4(c10), d = ldg4(c11);
                            S[j].x = w00[j] * a.x + w01[j] * b.x + w10[j] * c.x + w11[j] * d.x;
                            S[j].y = w00[j] * a.y + w01[j] * b.y + w10[j] * c.y + w11[j] * d.y;
                            S[j].z = w00[j] * a.z + w01[j] * b.z + w10[j] * c.z + w11[j] * d.z;
                            S[j].w = w00[j] * a.w + w01[j] * b.w + w10[j] * c.w + w11[j] * d.w;
                        } else {
                            float s4[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                            for (int e = 0; e < 4; ++e)
                                if (nu0 + e < f.n_freq)
                                    s4[e] = w00[j] * __ldg(c00 + e) + w01[j] * __ldg(c01 + e)
                                          + w10[j] * __ldg(c10 + e) + w11[j] * __ldg(c11 + e);
                            S[j] = make_float4(s4[0], s4[1], s4[2], s4[3]);
                        }
                    }
                }
                ptx::mbar_wait(sm.a_empty + 8 * stage, ph ^ 1u);
                unsigned char* a_hi = smem_raw + (sm.a - raw) + stage * kTcAStageBytes;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    float4 v, hi, lo;
                    v.x = element_value(fmaf(fp[j], L1[j].x - L0[j].x, L0[j].x), csc[j], X.x, G.x * S[j].x);
                    v.y = element_value(fmaf(fp[j], L1[j].y - L0[j].y, L0[j].y), csc[j], X.y, G.y * S[j].y);
                    v.z = element_value(fmaf(fp[j], L1[j].z - L0[j].z, L0[j].z), csc[j], X.z, G.z * S[j].z);
                    v.w = element_value(fmaf(fp[j], L1[j].w - L0[j].w, L0[j].w), csc[j], X.w, G.w * S[j].w);
                    hi.x = ptx::to_tf32(v.x); hi.y = ptx::to_tf32(v.y); hi.z = ptx::to_tf32(v.z); hi.w = ptx::to_tf32(v.w);
                    lo.x = ptx::to_tf32(v.x - hi.x); lo.y = ptx::to_tf32(v.y - hi.y);
                    lo.z = ptx::to_tf32(v.z - hi.z); lo.w = ptx::to_tf32(v.w - hi.w);
                    const uint32_t off = (uint32_t)(rsub + 32 * j) * 128u + swz;
                    *reinterpret_cast<float4*>(a_hi + off) = hi;
                    *reinterpret_cast<float4*>(a_hi + kTcAPartBytes + off) = lo;
                }
                ptx::fence_proxy_async_smem();
                ptx::mbar_arrive(sm.a_full + 8 * stage);
            }
        }
    } else if (warp >= kTcWarpLoader && warp < kTcWarpGen0) {
      ptx::setmaxnreg_dec<kTcRegsCtl>();
      if (warp == kTcWarpLoader) {
        // =========================== loader: filter slab images -> B ring =====================
        if (lane == 0) {
            uint32_t ub = 0;
            for (int64_t tl = blockIdx.x; tl < n_tiles; tl += gridDim.x) {
                const int g = (int)(tl % p.n_groups);
                const unsigned char* src = p.filt_img + (size_t)g * p.n_kb * 2 * (size_t)p.unit_bytes;
                for (int u = 0; u < 2 * p.n_kb; ++u, ++ub) {
                    const uint32_t bs = ub % (uint32_t)p.b_stages, bph = (ub / (uint32_t)p.b_stages) & 1u;
                    ptx::mbar_wait(sm.b_empty + 8 * bs, bph ^ 1u);
                    ptx::mbar_arrive_expect_tx(sm.b_full + 8 * bs, (uint32_t)p.unit_bytes);
                    ptx::bulk_g2s(sm.b + bs * (uint32_t)p.unit_bytes, src + (size_t)u * p.unit_bytes,
                                  (uint32_t)p.unit_bytes, sm.b_full + 8 * bs);
                }
            }
        }
        __syncwarp();
      } else if (warp == kTcWarpMma) {
        // =========================== MMA issuer =================================================
        if (lane == 0) {
            TcRotation rot(p.n_cg, p.seg, p.n_kb);
            uint32_t idesc[kTcMaxCg], uses[kTcNumBuf] = {0u, 0u, 0u, 0u};
            bool fresh[kTcMaxCg];              // next MMA into buf[g] overwrites (first of a segment)
#pragma unroll
            for (int g = 0; g < kTcMaxCg; ++g) {
                idesc[g] = ptx::idesc_tf32(kTcBM, g < p.n_cg ? rot.width(g, p.nb_tot) : 16);
                fresh[g] = true;
            }
            uint32_t it = 0, ub = 0;
            for (int64_t tl = blockIdx.x; tl < n_tiles; tl += gridDim.x) {
                for (int kb = 0; kb < p.n_kb; ++kb, ++it) {
                    const uint32_t stage = it & 1u, ph = (it >> 1) & 1u;
                    // a group that has just moved to another buffer waits until the epilogue has drained it
#pragma unroll
                    for (int g = 0; g < kTcMaxCg; ++g)
                        if (g < p.n_cg && fresh[g]) {
                            const int b = rot.buf[g];
                            if (uses[b] > 0) ptx::mbar_wait(sm.buf_free + 8 * b, (uses[b] - 1u) & 1u);
                        }
                    ptx::mbar_wait(sm.a_full + 8 * stage, ph);
                    const uint32_t a_hi = sm.a + stage * kTcAStageBytes, a_lo = a_hi + kTcAPartBytes;
                    {   // filter hi part: acc += A_hi.B_hi + A_lo.B_hi
                        const uint32_t bs = ub % (uint32_t)p.b_stages, bph = (ub / (uint32_t)p.b_stages) & 1u;
                        ptx::mbar_wait(sm.b_full + 8 * bs, bph);
                        ptx::tc_fence_after();
                        const uint32_t b0 = sm.b + bs * (uint32_t)p.unit_bytes;
#pragma unroll
                        for (int k = 0; k < kTcBK / kTcUK; ++k)
#pragma unroll
                            for (int g = 0; g < kTcMaxCg; ++g)
                                if (g < p.n_cg) {
                                    const uint64_t bd = ptx::smem_desc_sw128(b0 + (uint32_t)(g * kTcBufCols) * 128u + k * 32u);
                                    const uint32_t d = tmem_base + (uint32_t)(rot.buf[g] * kTcBufCols);
                                    ptx::mma_tf32_ss(d, ptx::smem_desc_sw128(a_hi + k * 32u), bd, idesc[g], (k != 0 || !fresh[g]) ? 1u : 0u);
                                    ptx::mma_tf32_ss(d, ptx::smem_desc_sw128(a_lo + k * 32u), bd, idesc[g], 1u);
                                }
                        ptx::tc_commit(sm.b_empty + 8 * bs);
                        ++ub;
                    }
                    {   // filter lo part: acc += A_hi.B_lo
                        const uint32_t bs = ub % (uint32_t)p.b_stages, bph = (ub / (uint32_t)p.b_stages) & 1u;
                        ptx::mbar_wait(sm.b_full + 8 * bs, bph);
                        ptx::tc_fence_after();
                        const uint32_t b0 = sm.b + bs * (uint32_t)p.unit_bytes;
#pragma unroll
                        for (int k = 0; k < kTcBK / kTcUK; ++k)
#pragma unroll
                            for (int g = 0; g < kTcMaxCg; ++g)
                                if (g < p.n_cg) {
                                    const uint64_t bd = ptx::smem_desc_sw128(b0 + (uint32_t)(g * kTcBufCols) * 128u + k * 32u);
                                    ptx::mma_tf32_ss(tmem_base + (uint32_t)(rot.buf[g] * kTcBufCols),
                                                     ptx::smem_desc_sw128(a_hi + k * 32u), bd, idesc[g], 1u);
                                }
                        ptx::tc_commit(sm.b_empty + 8 * bs);
                        ++ub;
                    }
                    ptx::tc_commit(sm.a_empty + 8 * stage);
                    // segment boundaries: hand the finished partial sums to the epilogue, move on to a free buffer
#pragma unroll
                    for (int g = 0; g < kTcMaxCg; ++g) {
                        if (g >= p.n_cg) continue;
                        fresh[g] = false;
                        if (rot.boundary(kb, g)) {
                            const int old = rot.rotate(g);
                            ptx::tc_commit(sm.flush_full + 8 * old);
                            ++uses[old];
                            fresh[g] = true;
                        }
                    }
                }
            }
        }
        __syncwarp();
      }
    } else if (warp >= kTcWarpFin0) {
        // ============ finisher: scratch tile -> P = sum*scale + bias, photon noise -> TOD ========
        ptx::setmaxnreg_dec<kTcRegsFin>();
        const int q = warp - kTcWarpFin0;
        uint32_t ti = 0;
        for (int64_t tl = blockIdx.x; tl < n_tiles; tl += gridDim.x, ++ti) {
            const int64_t row0 = (tl / p.n_groups) * kTcBM;
            const int cg0 = (int)(tl % p.n_groups) * p.nb_tot;
            const int n_valid = min(p.nb_tot, f.n_chan - cg0);            // real channels of this group
            const uint32_t sb = ti & 1u;
            const float* sc = p.scratch + ((size_t)blockIdx.x * 2 + sb) * p.nb_tot * kTcBM;
            ptx::mbar_wait(sm.tile_done + 8 * sb, (ti >> 1) & 1u);
            constexpr int kMaxPerLane = kTcMaxGroupChan / 32;             // 12
            for (int r = q; r < kTcBM; r += kTcFinWarps) {
                const int64_t Rr = row0 + r;
                if (Rr >= f.n_rows) break;
                const uint32_t n = (uint32_t)(f.t0 + Rr / f.n_spaxel), s = (uint32_t)(Rr % f.n_spaxel);
                float* o = f.out + (size_t)Rr * f.n_chan + cg0;
                float x[kMaxPerLane];
#pragma unroll
                for (int j = 0; j < kMaxPerLane; ++j) {
                    const int c = lane + 32 * j;
                    x[j] = c < n_valid ? __ldcg(sc + (size_t)c * kTcBM + r) : 0.f;
                }
#pragma unroll
                for (int j = 0; j < kMaxPerLane; ++j) {
                    const int c = lane + 32 * j;
                    if (c < n_valid) {
                        float P = fmaf(x[j], f.scale, __ldg(f.bias + cg0 + c));
                        if (f.photon_noise) {
                            const uint4 w = philox4x32_10(n, s, (uint32_t)(cg0 + c), kStreamPhoton, f.seed_lo, f.seed_hi);
                            P = fmaf(photon_sigma(P, __ldg(f.noise_c1 + cg0 + c), __ldg(f.noise_c2 + cg0 + c)),
                                     normal_cos(w.x, w.y), P);
                        }
                        o[c] = P;
                    }
                }
            }
            ptx::mbar_arrive(sm.scratch_free + 8 * sb);
        }
    } else {
        // ============ epilogue: segment flushes of the accumulators into the scratch tile =======
        ptx::setmaxnreg_inc<kTcRegsFlush>();
        const int q = warp;                                    // tensor-memory lane quarter
        const int trow = 32 * q + lane;                        // tile row = tensor-memory lane
        TcRotation rot(p.n_cg, p.seg, p.n_kb);
        uint32_t fulls[kTcNumBuf] = {0u, 0u, 0u, 0u};
        uint32_t ti = 0;
        for (int64_t tl = blockIdx.x; tl < n_tiles; tl += gridDim.x, ++ti) {
            const uint32_t sb = ti & 1u;
            float* const sc = p.scratch + ((size_t)blockIdx.x * 2 + sb) * p.nb_tot * kTcBM;
            if (ti >= 2) ptx::mbar_wait(sm.scratch_free + 8 * sb, ((ti >> 1) - 1u) & 1u);   // finisher done with tile ti-2
            bool first[kTcMaxCg] = {true, true, true};
            for (int kb = 0; kb < p.n_kb; ++kb)
#pragma unroll
                for (int g = 0; g < kTcMaxCg; ++g) {
                    if (g >= p.n_cg || !rot.boundary(kb, g)) continue;
                    const int b = rot.rotate(g);
                    const int wg = rot.width(g, p.nb_tot);
                    float* scg = sc + (size_t)(g * kTcBufCols) * kTcBM + trow;
                    const uint32_t taddr = tmem_base + ((uint32_t)(32 * q) << 16) + (uint32_t)(b * kTcBufCols);
                    const bool add = !first[g];
                    uint32_t v[32];
                    float pa[32], pb[32];
                    // the running sums of the first 32 columns are fetched while the MMAs still run
                    if (add) {
#pragma unroll
                        for (int i = 0; i < 32; ++i) pa[i] = __ldcg(scg + (size_t)i * kTcBM);
                    }
                    ptx::mbar_wait(sm.flush_full + 8 * b, fulls[b] & 1u);
                    ++fulls[b];
                    ptx::tc_fence_after();
                    for (int c0 = 0; c0 < wg; c0 += 64) {
                        const bool two = c0 + 32 < wg;
                        ptx::tmem_ld_32x32(taddr + (uint32_t)c0, v);
                        if (add && two) {
#pragma unroll
                            for (int i = 0; i < 32; ++i) pb[i] = __ldcg(scg + (size_t)(c0 + 32 + i) * kTcBM);
                        }
                        ptx::tmem_ld_wait();
#pragma unroll
                        for (int i = 0; i < 32; ++i)
                            __stcg(scg + (size_t)(c0 + i) * kTcBM, add ? pa[i] + __uint_as_float(v[i]) : __uint_as_float(v[i]));
                        if (two) {
                            ptx::tmem_ld_32x32(taddr + (uint32_t)(c0 + 32), v);
                            if (add && c0 + 64 < wg) {
#pragma unroll
                                for (int i = 0; i < 32; ++i) pa[i] = __ldcg(scg + (size_t)(c0 + 64 + i) * kTcBM);
                            }
                            ptx::tmem_ld_wait();
#pragma unroll
                            for (int i = 0; i < 32; ++i)
                                __stcg(scg + (size_t)(c0 + 32 + i) * kTcBM, add ? pb[i] + __uint_as_float(v[i]) : __uint_as_float(v[i]));
                        }
                    }
                    ptx::tc_fence_before();
                    ptx::mbar_arrive(sm.buf_free + 8 * b);
                    first[g] = false;
                }
            // every partial sum of the tile is in the scratch tile: hand it to the finisher warps
            ptx::mbar_arrive(sm.tile_done + 8 * sb);
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == kTcWarpMma) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc(tmem_base, 512);
    }
}

inline cudaError_t launch_fused_tc(const FusedParams& fp, const TcTables& t, int num_sms, cudaStream_t st) {
    TcParams p{};
    p.f = fp; p.filt_img = t.filt_img;
    p.scratch = t.scratch;
    p.n_groups = t.n_groups; p.nb_tot = t.nb_tot; p.n_cg = t.n_cg; p.seg = t.seg > 0 ? t.seg : kTcSegDefault; p.n_kb = t.n_kb;
    p.unit_bytes = t.unit_bytes; p.b_stages = t.b_stages;
    p.n_row_tiles = (int32_t)((fp.n_rows + kTcBM - 1) / kTcBM);
    p.cube_vec = (fp.cube == nullptr) || ((fp.n_freq % 4 == 0) && ((reinterpret_cast<uintptr_t>(fp.cube) & 15u) == 0));
    const int64_t n_tiles = (int64_t)p.n_row_tiles * p.n_groups;
    const unsigned grid = (unsigned)std::min<int64_t>(n_tiles, num_sms);
    static int smem_set[2] = {0, 0};
    cudaError_t e;
    if (p.cube_vec) {
        if (smem_set[1] < t.smem_bytes) {
            e = cudaFuncSetAttribute(fused_tc_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, t.smem_bytes);
            if (e != cudaSuccess) return e;
            smem_set[1] = t.smem_bytes;
        }
        fused_tc_kernel<true><<<grid, kTcThreads, t.smem_bytes, st>>>(p);
    } else {
        if (smem_set[0] < t.smem_bytes) {
            e = cudaFuncSetAttribute(fused_tc_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, t.smem_bytes);
            if (e != cudaSuccess) return e;
            smem_set[0] = t.smem_bytes;
        }
        fused_tc_kernel<false><<<grid, kTcThreads, t.smem_bytes, st>>>(p);
    }
    return cudaGetLastError();
}

}  // namespace gt
