// gt_fused_tc.cuh -- steps 2-6a as ONE tcgen05 tensor-core kernel (GT_VARIANT_TENSOR, GT_VARIANT_TENSOR_FULL).
//
//   P_KID[row][c] = dnu * sum_nu Fm[c][nu] * P[row][nu]                       (Eq. 16)
// is a dense [rows x n_freq] . [n_freq x n_chan] contraction whose left operand is GENERATED
// (steps 2-4, collapsed cascade of DESIGN.md) and never exists in HBM.  Per persistent CTA
// (one per SM) and per tile of 128 rows:
//
//   generator warps (16)  : 64-frequency slab of the spectrum for 128 rows -> fp16 pair (hi, lo) of the
//                           scaled value (22 mantissa bits) -> shared memory, UMMA K-major SWIZZLE_128B.
//                           A warp works on two rows x the whole slab (a thread walks four rows), on packed
//                           fp32 pairs (FFMA2 / FMUL2 / FADD2); the L1's LSU data pipe (the 16-byte cube taps)
//                           sets the cycles of the kernel (profiles/r02e_fused_tc.md)
//   loader warp (1 lane)  : filter slab images (hi, lo; pre-split, pre-swizzled at plan time; CTA pair:
//                           this CTA's half) global -> shared by cp.async.bulk, mbarrier complete_tx
//   MMA warp (1 lane)     : tcgen05.mma.cta_group::2.kind::f16, M = 256 per CTA pair, N <= 128 per column
//                           group, K = 16:  acc += A_hi.B_hi + A_lo.B_hi + A_hi.B_lo  (the three-term split
//                           of north_star with fp16 pieces: every product of two 11-bit pieces is exact in
//                           the fp32 accumulate, the dropped A_lo.B_lo term is 2^-22 relative).  BANDED
//                           CORRECTIONS: the two correction products of a (column group, slab) block are
//                           issued only where the plan could not bound them below 1e-6 of the channel's
//                           power in the worst case (corr_on): 54 % fewer on C4
//   flush warps (4)       : SEGMENTED ACCUMULATION.  The tensor core's fp32 accumulate truncates
//                           (measured: -2.7e-5 relative after 500 chained MMAs of positive terms,
//                           DESIGN.md "Accumulation in tensor memory"), so no accumulator lives
//                           longer than `seg` slabs: the <= 384 padded channels of a tile are cut
//                           into <= 3 column groups of <= 128 columns that rotate through FOUR
//                           128-column tensor-memory buffers; at a (staggered) segment boundary a
//                           group moves to the spare buffer and the epilogue warps add the
//                           finished partial sums (tcgen05.ld) into a per-CTA, L2-resident fp32
//                           scratch tile [column][row] with round-to-nearest FADDs.  After the
//                           last segment the finisher warps (8) transpose the scratch tile into the TOD:
//                           P = sum*scale + bias[c], photon noise (Eq. 18-19; one Philox block per four
//                           channels, R19), coalesced stores.
//
// Pipelines: A ring (2 stages, generators of both CTAs -> leader's MMA thread), B ring (loader -> MMA, the
// peer's halves relayed by a forwarder), accumulator buffers flush_full / buf_free (MMA <-> flush), scratch
// tiles tile_done / scratch_free (flush <-> finisher); all mbarrier based, CTA-scope waits.
#pragma once
#include <vector>
#include <cstring>
#include <algorithm>
#include <cstdlib>
#include <cstdio>
#include <cmath>
#include <atomic>
#include <thread>
#include <cuda_fp16.h>
#include "gt_common.cuh"
#include "gt_fused_fp32.cuh"
#include "gt_tc_ptx.cuh"
#include "../../include/gateau_b200.h"

namespace gt {

constexpr int kTcBM = 128;                 // rows per tile (UMMA M)
constexpr int kTcBK = 64;                  // frequencies per A stage / B unit: one 128-byte swizzle row of 64 fp16
constexpr float kTcSqScale = 1.0f / 256.0f;   // squared elements (v = O(256)) are scaled back into fp16 range
constexpr int kTcHB = 32;                  // frequencies per generator step group (8 lanes x 4): half a slab
constexpr int kTcKSteps = 4;               // K = 16 MMAs per 128-byte operand row
// Operand scaling into the fp16 range: exact powers of two chosen at plan time and
// undone in the epilogue.  A (spectrum): ONE scale per plan, from the largest element the generator can produce
// (max |Xn|, max |G| max |cube|), so that it lands in [2^kTcAMaxLog2 - 1, 2^kTcAMaxLog2).  B (filter): one scale PER
// CHANNEL, so that the row maximum lands in [2^14, 2^15): a delta filter 1/dnu ~ 1e-8, a row-normalised filter ~ 1e-10
// and a filter of peak 1 all keep their 22 bits.
constexpr int kTcAMaxLog2 = 11;            // |A| < 2048: the squared elements of Eq. 17 (A^2 / 256) still fit fp16
constexpr int kTcBMaxLog2 = 15;            // row maximum of |B| < 32768
#ifndef GT_TC_A_STAGES
#define GT_TC_A_STAGES 2
#endif
constexpr int kTcAStages = GT_TC_A_STAGES;   // <= 4
#ifndef GT_TC_PAIR
#define GT_TC_PAIR 1
#endif
// CTA pair (cta_group::2): two CTAs on one TPC compute two row tiles with M = 256 MMAs; each holds half of every
// filter unit in shared memory, so the filter is fetched from L2, written to and read from shared memory once per pair.
constexpr bool kTcPair = GT_TC_PAIR != 0;
// Timing diagnostics (parts of the kernel switched off through GATEAU_TC_DEBUG) exist only in tuning builds
// (-DGT_TC_DIAG): the product kernel carries no such branches.
#ifdef GT_TC_DIAG
#define GT_DIAG(p, bit) (((p).debug & (bit)) != 0)
#else
#define GT_DIAG(p, bit) false
#endif
constexpr int kTcAPartBytes = kTcBM * 128;                  // 16 KB (hi or lo part: 128 rows of 64 fp16)
constexpr int kTcAStageBytes = 2 * kTcAPartBytes;           // 32 KB
constexpr int kTcEpiWarps = 4, kTcGenWarps = 16;
constexpr int kTcStageBytes = 16 * 32 * 4;                  // one flush batch: 16 columns x 32 rows of fp32
// warp roles, aligned to warpgroups of 4 warps so that setmaxnreg can move registers between them:
//   WG0 = warps 0-3 flush (tensor-memory lane quarter = warp), WG1-4 = generators (4 warps per scheduler: the
//   per-element dependency chain lg2 -> ex2 -> split only fills the issue slots with thread-level parallelism),
//   WG5-6 = finishers (two warps per scheduler: the ten dependent Philox rounds of one warp leave its scheduler
//   idle, measured 9.87 -> 9.45 ms on a 16 000-sample C4 launch against one finisher warpgroup with 88 registers),
//   WG7 = 2 idle, loader, MMA.  The kernel starts with 64 registers per thread (1024 threads); setmaxnreg can only
//   redistribute that pool: 128 x (56 + 4*80 + 2*48 + 40) = 128 x 8*64.  GT_TC_FIN_WARPS = 4 is the earlier
//   896-thread layout (72 registers at start, one finisher warpgroup with 88).
// The warp scheduler favours the highest warp id among eligible warps: the two single-thread control
// roles sit in the LAST warpgroup so that the MMA issue stream is never starved by generator warps.
constexpr int kTcWarpGen0 = 4;
constexpr int kTcRowsPerThread = kTcBM / (4 * kTcGenWarps), kTcRowStride = 4 * kTcGenWarps;   // 2 rows, 64 apart
#ifndef GT_TC_FIN_WARPS
#define GT_TC_FIN_WARPS 8
#endif
constexpr int kTcFinWarps = GT_TC_FIN_WARPS, kTcWarpFin0 = kTcWarpGen0 + kTcGenWarps;   // 4 or 8 finisher warps from warp 20
static_assert(kTcFinWarps == 4 || kTcFinWarps == 8, "finishers fill whole warpgroups");
constexpr int kTcWarpCtl0 = kTcWarpFin0 + kTcFinWarps;                              // 24 (28)
constexpr int kTcWarpLoader = kTcWarpCtl0 + 2, kTcWarpMma = kTcWarpCtl0 + 3;        // 26, 27 (30, 31)
constexpr int kTcThreads = 32 * (kTcWarpCtl0 + 4);                                  // 896 (1024)
constexpr int kTcRegsBase = (65536 / kTcThreads) / 8 * 8;                           // 72 (64): registers per thread at kernel start
#ifndef GT_TC_REGS_FLUSH
#define GT_TC_REGS_FLUSH 56
#endif
#ifndef GT_TC_REGS_FIN
#define GT_TC_REGS_FIN (GT_TC_FIN_WARPS == 8 ? 48 : 88)
#endif
// finisher: channels in flight per lane, and whether the next row's partial sums are fetched a row ahead
#ifndef GT_TC_FIN_QW
#define GT_TC_FIN_QW 3      // Philox blocks (quads of channels) in flight per finisher lane: 1 or 3
#endif
#ifndef GT_TC_FIN_PREFETCH
#define GT_TC_FIN_PREFETCH (GT_TC_FIN_WARPS == 8 ? 0 : 1)
#endif
constexpr int kTcRegsFlush = GT_TC_REGS_FLUSH, kTcRegsCtl = 40, kTcRegsGen = 80, kTcRegsFin = GT_TC_REGS_FIN;
static_assert(kTcRegsFlush + kTcRegsCtl + 4 * kTcRegsGen + (kTcFinWarps / 4) * kTcRegsFin <= (kTcThreads / 128) * kTcRegsBase, "setmaxnreg pool");
constexpr int kTcMaxGroupChan = 384;       // channels per tile: 3 column groups of 128 (+ 1 spare buffer = 512 columns)
constexpr int kTcBufCols = 128, kTcNumBuf = 4, kTcMaxCg = 3;
constexpr int kTcSegDefault = 12;          // slabs (of 64 frequencies) per accumulation segment (measured max error on the C4 window 6.5e-6 of the 1e-5 gate, narrow channels on segment edges 0.8e-6; 8: 4.9e-6, 16: 9.4e-6)
// The tensor core's fp32 accumulate TRUNCATES (measured): the 16 products of an MMA are aligned
// to the running sum and cut at kTcTruncGrain of its unit in the last place (two guard bits), the new sum is cut to
// the unit itself.  Positive products far above the grain therefore lose 16 x grain / 2 + 1/2 = 2.5 ulp per MMA;
// products below the grain are dropped whole; the split's correction products (random signs) lose 1/2 ulp per MMA
// once they reach the grain and nothing below it.  The plan tabulates, per (channel, segment), how many ulps of its
// final sum a segment loses (from the channel's own filter and a reference spectrum: a narrow channel whose mass
// arrives in the first slab of a segment loses 2.5 ulp per later 16-frequency step, one whose mass arrives last
// loses nothing) and the flush warps add them back in units of the ulp of the partial sum they hold.
constexpr double kTcTruncGrain = 0.25;
#ifndef GT_TC_TRUNC_ULP
#define GT_TC_TRUNC_ULP 0.9f
#endif
constexpr float kTcTruncUlp = GT_TC_TRUNC_ULP;      // overall factor on the table (0.9: the model with factor 1 left a mean error of +0.9e-6 on the config windows); tuning builds calibrate with 0 (off)
#ifndef GT_TC_MAX_B_STAGES
#define GT_TC_MAX_B_STAGES 3
#endif
constexpr int kTcMaxBStages = GT_TC_MAX_B_STAGES;   // <= 4 (barrier slots)
// Banded corrections (DESIGN.md section 6 "Banded corrections"): the two correction products of the split, A_lo.Fm_hi and
// A_hi.Fm_lo, are each at most 2^-12 of the main product element by element.  For a (column group, slab) block in which every
// channel of the group has so little of its filter that BOTH corrections of ALL skipped blocks together stay, in the worst
// case over the spectra the plan can produce, below kTcSkipBudget of the channel's power, the MMA thread issues only
// A_hi.Fm_hi (a third of the tensor work of that block).  0 switches the skipping off.
#ifndef GT_TC_SKIP_BUDGET
#define GT_TC_SKIP_BUDGET 1e-6
#endif
constexpr double kTcSkipBudget = GT_TC_SKIP_BUDGET;
constexpr int kTcSmemLimit = 227 * 1024;

struct TcTables {
    unsigned char* filt_img = nullptr;   // [group][kb][part hi/lo][NBtot rows][128 B swizzled]
    float* scratch = nullptr;            // [num CTAs][2][nb_tot / 4][128][4] fp32 partial sums (L2 resident)
    int32_t n_groups = 0;                // channel groups (tiles along the channel axis) of <= 384 channels
    int32_t nb_tot = 0;                  // padded channels per group (multiple of 32)
    int32_t n_cg = 0;                    // column groups per tile, widths 128,..,remainder
    int32_t seg = kTcSegDefault;         // slabs per accumulation segment
    int32_t n_kb = 0;                    // n_freq_pad / 64
    int32_t unit_bytes = 0;              // nb_tot * 128
    int32_t b_stages = 0;
    int32_t smem_bytes = 0;
    float* comp = nullptr;               // [group][n_seg][nb_tot] truncation compensation in ulp of the segment sum, times 2^-23
    int32_t n_seg = 0;                   // segments per tile (max over the column groups)
    unsigned char* corr_on = nullptr;    // [group][n_kb] bit cg: A_lo.Fm_hi of column group cg is issued for this slab; bit 4 + cg: A_hi.Fm_lo
    int64_t n_corr_blocks = 0, n_corr_skipped = 0;     // correction products per (group, column group, slab): 2 each; how many are skipped
};

// plan-time host loops over channels / samples are independent: a plain thread pool per call (plan creation is part of
// the end-to-end time bench.py reports)
template <class F>
inline void host_parallel_for(int64_t n, F&& f) {
    const int64_t nt = std::max<int64_t>(1, std::min<int64_t>({(int64_t)std::thread::hardware_concurrency(), (int64_t)16, n}));
    if (nt == 1) { for (int64_t i = 0; i < n; ++i) f(i); return; }
    std::vector<std::thread> th;
    for (int64_t k = 0; k < nt; ++k)
        th.emplace_back([=, &f]() { for (int64_t i = k * n / nt; i < (k + 1) * n / nt; ++i) f(i); });
    for (auto& t : th) t.join();
}

// device memory of the tables: the plan layer installs its pool allocator here (gateau_b200.cu); plain cudaMalloc otherwise
using TcAllocFn = cudaError_t (*)(void**, size_t);
using TcFreeFn = void (*)(void*);
inline cudaError_t tc_default_alloc(void** p, size_t n) { return cudaMalloc(p, n); }
inline void tc_default_free(void* p) { cudaFree(p); }
inline TcAllocFn& tc_alloc_fn() { static TcAllocFn f = tc_default_alloc; return f; }
inline TcFreeFn& tc_free_fn() { static TcFreeFn f = tc_default_free; return f; }

inline const char*& tc_error_ref() { static thread_local const char* e = ""; return e; }
inline const char* tc_error() { return tc_error_ref(); }

// Expected number of ulps (of the FINAL segment sum S) that one chained MMA loses when the accumulator stands at
// p S: the loss is ~1 ulp of the accumulator, ulp(p S) / ulp(S) = 2^floor(log2(p m)) for S = m 2^e; the flush warps
// know e (they hold S) but the plan only knows the profile p, so the table carries the mean over a log-uniform
// mantissa m in [1,2): 2^k (1 + f) with log2 p = k + f.  Signed like p (the truncation is toward zero).
inline double tc_ulp_ratio(double p) {
    if (p == 0.0 || !std::isfinite(p)) return 0.0;
    const double a = std::fabs(p), l = std::log2(a), k = std::floor(l);
    const double r = std::ldexp(1.0 + (l - k), (int)std::max(-60.0, std::min(60.0, k)));
    return p < 0.0 ? -r : r;
}

// Splits the filter into fp16 hi/lo parts and lays every (group, 64-frequency slab, part) out as
// the exact shared-memory image tcgen05.mma reads (K-major, SWIZZLE_128B): the loader is a flat copy.
// Channel c is scaled by its own power of two 2^kb[c] so that its largest |value| lands in [2^14, 2^15);
// inv_scale[c] = 2^-kb[c] goes into the epilogue constant of the channel.
// a_ref [n_freq]: a reference spectrum in the generator's scaled units (any positive multiple will do), used only for
// the truncation-compensation table: W[c][segment] = kTcTruncUlp 2^-23 sum over the MMAs of the segment of
// tc_ulp_ratio(accumulator after that MMA / final segment sum), in the order the MMA thread issues them.
// filt1 != nullptr (the Eq. 17 pass): no split -- unit 0 = fp16(2^kb filt), unit 1 = fp16(2^kb filt1), one scale per
// channel from the larger of the two maxima; one accumulation segment per tile and no compensation table (sigma needs 1e-3).
// What the plan knows about the elements the generator can produce, for the banded corrections: per frequency the range
// of the elements in the generator's scaled units, per channel the part of the channel's power that does not pass through
// the contraction (the bias), in units of the contraction sum.  nullptr: no skipping.
// Two masks per (column group, slab), each with half of kTcSkipBudget of the channel's smallest possible power:
//   A_lo.Fm_hi: |A_lo| <= 2^-12 |element|, sign unknown: worst case 2^-12 sum |Fm| max|v| over the skipped slabs;
//   A_hi.Fm_lo: Fm_lo is known, so the sum over the skipped slabs is bounded by |sum Fm_lo v_mid| + sum |Fm_lo| (v_rad +
//               2^-12 max|v|) with v_mid, v_rad the centre and half width of the element's range (the signs of Fm_lo
//               cancel as they do in the product itself).
struct TcSkipBounds {
    const std::vector<double>* v_min;    // [n_freq] smallest element (may be negative)
    const std::vector<double>* v_max;    // [n_freq] largest element
    const std::vector<double>* floor_c;  // [n_chan], >= 0
};

inline gt_status build_tc_tables(const std::vector<float>& filt, int n_chan, int n_freq, int n_freq_pad,
                                 const std::vector<double>& a_ref, TcTables& t, std::vector<float>& inv_scale,
                                 cudaStream_t st, const std::vector<float>* filt1 = nullptr, const TcSkipBounds* sb = nullptr) {
    const int G = (n_chan + kTcMaxGroupChan - 1) / kTcMaxGroupChan;
    int per = (n_chan + G - 1) / G;
    // several groups: every group starts on a multiple of 128 channels, so that a finisher lane's quads of channels
    // (lane + 128 m + {0, 32, 64, 96}: one Philox block each, R19) never straddle two groups
    const int nbt = G > 1 ? (per + 127) / 128 * 128 : (per + 31) / 32 * 32;
    t.n_groups = G; t.nb_tot = nbt;
    t.n_cg = (nbt + kTcBufCols - 1) / kTcBufCols;
    t.n_kb = n_freq_pad / kTcBK;
    if (t.seg <= 0) t.seg = kTcSegDefault;
    if (filt1) t.seg = t.n_kb;
    // one unit = the rows one CTA holds of one (slab, part): all nb_tot rows, or (CTA pair) the half of every
    // column group this CTA supplies to the M = 256 MMAs (rank r: columns [r w/2, (r+1) w/2) of a group of width w)
    constexpr int kRanks = kTcPair ? 2 : 1;
    t.unit_bytes = nbt * 128 / kRanks;
    const int fixed = kTcAStages * kTcAStageBytes + 1024 /*alignment slack*/ + 320 /*barriers*/ + kTcBM * 32 /*row constants*/ + kTcEpiWarps * kTcBufCols * 4 /*compensation weights of the next flush, per flush warp*/
                    + kTcEpiWarps * 2 * kTcStageBytes /*flush staging: two 2 KB batches per flush warp*/;
    t.b_stages = std::min(kTcMaxBStages, (kTcSmemLimit - fixed) / t.unit_bytes);
    if (t.b_stages < 2) { tc_error_ref() = "filter slab does not fit in shared memory"; return GT_ERR_UNSUPPORTED; }
    t.smem_bytes = fixed + t.b_stages * t.unit_bytes;

    // segment of every slab, per column group: the host-side twin of TcRotation::boundary
    std::vector<int> seg_of((size_t)t.n_cg * t.n_kb);
    t.n_seg = 1;
    for (int cg = 0; cg < t.n_cg; ++cg) {
        int cnt = (cg * t.seg) / t.n_cg, si = 0;
        for (int kb = 0; kb < t.n_kb; ++kb) {
            seg_of[(size_t)cg * t.n_kb + kb] = si;
            if (kb != t.n_kb - 1 && ++cnt == t.seg) { cnt = 0; ++si; }
        }
        t.n_seg = std::max(t.n_seg, si + 1);
    }

    inv_scale.assign((size_t)G * nbt, 1.0f);
    const size_t total = (size_t)G * t.n_kb * 2 * kRanks * t.unit_bytes;
    std::vector<float> img(total / 4, 0.f);
    std::vector<float> comp((size_t)G * t.n_seg * nbt, 0.f);
    uint16_t* img16 = reinterpret_cast<uint16_t*>(img.data());
    std::atomic<int> bad{0};
    // per (channel, 16-frequency K step): the step's share of the contraction for the reference spectrum (compensation
    // table); per (channel, slab): the worst-case |correction| of the slab in units of its budget (banded corrections)
    const size_t n_steps = (size_t)t.n_kb * kTcKSteps;
    std::vector<double> part_all((size_t)G * nbt * n_steps, 0.0);
    const bool skipping = sb != nullptr && !filt1 && kTcSkipBudget > 0.0;
    const size_t n_cost = skipping ? (size_t)G * nbt * t.n_kb : 0;
    std::vector<float> cost(n_cost, 0.f), flo_a(n_cost, 0.f), flo_r(n_cost, 0.f);   // in units of the channel's budget; INFINITY: no skipping
    // per frequency, for the correction bounds: 2^12 x the largest |A_lo| = |v - fp16(v)| (2^-12 |v| in fp16's normal range,
    // half a subnormal step 2^-25 below it), centre of the bracket, half width + the largest |A_hi - v|, max(0, v_min)
    std::vector<double> b_abs(skipping ? n_freq : 0), b_mid(b_abs.size()), b_rad(b_abs.size()), b_pos(b_abs.size());
    for (size_t i = 0; i < b_abs.size(); ++i) {
        const double vmin = (*sb->v_min)[i], vmax = (*sb->v_max)[i];
        b_abs[i] = std::max(std::fabs(vmin), std::fabs(vmax)) + std::ldexp(1.0, -13);
        b_mid[i] = 0.5 * (vmax + vmin);
        b_rad[i] = 0.5 * (vmax - vmin) + std::ldexp(b_abs[i], -12);
        b_pos[i] = std::max(0.0, vmin);
    }
    // ---- phase A, per channel: scale, shared-memory image, reference profile, correction bounds ----
    host_parallel_for((int64_t)G * nbt, [&](int64_t gn) {
        const int g = (int)(gn / nbt), n = (int)(gn % nbt);
        const int ch = g * nbt + n;
        if (ch >= n_chan) return;
        double* part = part_all.data() + (size_t)gn * n_steps;
        const float* frow = filt.data() + (size_t)ch * n_freq;
        const float* frow1 = filt1 ? filt1->data() + (size_t)ch * n_freq : nullptr;
        float amax = 0.f;
        bool negative = false;
        for (int i = 0; i < n_freq; ++i) {
            if (!std::isfinite(frow[i]) || (frow1 && !std::isfinite(frow1[i]))) { bad = 1; return; }
            amax = std::max(amax, std::fabs(frow[i]));
            negative |= frow[i] < 0.f;
            if (frow1) amax = std::max(amax, std::fabs(frow1[i]));
        }
        int kb_c = 0;
        if (amax > 0.f) { int e; std::frexp(amax, &e); kb_c = std::max(-100, std::min(100, kTcBMaxLog2 - e)); }
        inv_scale[(size_t)g * nbt + n] = std::ldexp(1.0f, -kb_c);
        // which CTA holds row n, and where inside its unit
        const int cg = n / kTcBufCols, col0 = cg * kTcBufCols, w = std::min(kTcBufCols, nbt - col0);
        const int rk = kTcPair ? (n - col0) / (w / 2) : 0;
        const int nl = kTcPair ? col0 / 2 + (n - col0) - rk * (w / 2) : n;        // local row
        double lo_sum = 0.0;                                                     // smallest contraction sum, scaled filter
        const float two_kb = std::ldexp(1.0f, kb_c);                             // a power of two: the products below are exact
        for (int kb = 0; kb < t.n_kb; ++kb) {
            // (group tile, slab, unit, rank): units are laid out [g][kb][unit][rank]; inside, K-major SWIZZLE_128B rows of
            // 64 fp16: 16-byte chunk (kk / 8) XOR (row % 8)
            uint16_t* const u0 = img16 + ((size_t)((g * t.n_kb + kb) * 2 + 0) * kRanks + rk) * (t.unit_bytes / 2) + (size_t)nl * 64;
            uint16_t* const u1 = img16 + ((size_t)((g * t.n_kb + kb) * 2 + 1) * kRanks + rk) * (t.unit_bytes / 2) + (size_t)nl * 64;
            const int i_lo = kb * kTcBK, i_hi = std::min(n_freq, i_lo + kTcBK);
            double pk[kTcKSteps] = {}, c_s = 0.0, a_s = 0.0, r_s = 0.0;          // sums of this slab, in registers
            for (int i = i_lo; i < i_hi; ++i) {
                const int kk = i - i_lo;
                const float f = frow[i] * two_kb;
                const __half fh = __float2half_rn(f);
                const __half fl = __float2half_rn(frow1 ? frow1[i] * two_kb : f - __half2float(fh));
                const int off = (((kk >> 3) ^ (nl & 7)) << 3) + (kk & 7);
                u0[off] = __half_as_ushort(fh);                // unit 0: Fm_hi
                u1[off] = __half_as_ushort(fl);                // unit 1: Fm_lo
                pk[kk >> 4] += (double)f * a_ref[i];
                if (skipping) {
                    const double flo = (double)__half2float(fl);
                    c_s += std::fabs((double)f) * b_abs[i];
                    a_s += flo * b_mid[i];
                    r_s += std::fabs(flo) * b_rad[i];
                    lo_sum += (double)f * b_pos[i];
                }
            }
            for (int k = 0; k < kTcKSteps; ++k) part[(size_t)kb * kTcKSteps + k] = pk[k];
            if (skipping) {
                cost[(size_t)gn * t.n_kb + kb] = (float)c_s; flo_a[(size_t)gn * t.n_kb + kb] = (float)a_s; flo_r[(size_t)gn * t.n_kb + kb] = (float)r_s;
            }
        }
        if (skipping) {
            // the channel's power is at least floor + sum Fm max(0, v_min) (all in units of the scaled contraction sum);
            // each of the two corrections gets half of the budget
            const double denom = 0.5 * kTcSkipBudget * ((*sb->floor_c)[ch] * std::ldexp(1.0, kb_c) + lo_sum);
            const bool never = negative || !(denom > 0.0) || !std::isfinite(denom);
            for (int kb = 0; kb < t.n_kb; ++kb) {
                const size_t k = (size_t)gn * t.n_kb + kb;
                cost[k] = never ? INFINITY : (float)(std::ldexp((double)cost[k], -12) / denom);
                flo_a[k] = never ? INFINITY : (float)((double)flo_a[k] / denom);
                flo_r[k] = never ? INFINITY : (float)((double)flo_r[k] / denom);
            }
        }
    });
    if (bad) { tc_error_ref() = "the filter holds a NaN or Inf"; return GT_ERR_VALUE; }
    // ---- phase B, per (group, column group): the slabs whose corrections are skipped.  Slabs are tried in the order of
    //      their largest cost over the group's channels; one is taken while every channel's total stays within its budget
    //      (1 in these units).  Bit cg of corr_on: A_lo.Fm_hi issued; bit 4 + cg: A_hi.Fm_lo issued. ----
    std::vector<unsigned char> corr_on((size_t)G * t.n_kb, 0xFF);
    t.n_corr_blocks = 2 * (int64_t)G * t.n_cg * t.n_kb; t.n_corr_skipped = 0;
    if (skipping) {
        for (int g = 0; g < G; ++g)
            for (int cg = 0; cg < t.n_cg; ++cg) {
                const int n0 = cg * kTcBufCols, n1 = std::min({nbt, n0 + kTcBufCols, n_chan - g * nbt});
                if (n1 <= n0) continue;
                auto at = [&](const std::vector<float>& a, int n, int kb) { return a[((size_t)g * nbt + n) * t.n_kb + kb]; };
                std::vector<std::pair<float, int>> order(t.n_kb);
                // A_lo.Fm_hi: additive worst case
                for (int kb = 0; kb < t.n_kb; ++kb) {
                    float m = 0.f;
                    for (int n = n0; n < n1; ++n) m = std::max(m, at(cost, n, kb));
                    order[kb] = {m, kb};
                }
                std::sort(order.begin(), order.end());
                std::vector<double> used(n1 - n0, 0.0), sum_a(n1 - n0, 0.0);
                for (const auto& o : order) {
                    if (!(o.first <= 1.f)) break;
                    bool fits = true;
                    for (int n = n0; n < n1 && fits; ++n) fits = used[n - n0] + at(cost, n, o.second) <= 1.0;
                    if (!fits) break;
                    for (int n = n0; n < n1; ++n) used[n - n0] += at(cost, n, o.second);
                    corr_on[(size_t)g * t.n_kb + o.second] &= (unsigned char)~(1u << cg);
                    ++t.n_corr_skipped;
                }
                // A_hi.Fm_lo: |signed sum| + radius
                for (int kb = 0; kb < t.n_kb; ++kb) {
                    float m = 0.f;
                    for (int n = n0; n < n1; ++n) m = std::max(m, std::fabs(at(flo_a, n, kb)) + at(flo_r, n, kb));
                    order[kb] = {m, kb};
                }
                std::sort(order.begin(), order.end());
                std::fill(used.begin(), used.end(), 0.0);
                for (const auto& o : order) {
                    if (!(o.first <= 1.f)) break;
                    bool fits = true;
                    for (int n = n0; n < n1 && fits; ++n)
                        fits = std::fabs(sum_a[n - n0] + at(flo_a, n, o.second)) + used[n - n0] + at(flo_r, n, o.second) <= 1.0;
                    if (!fits) continue;                             // a later slab may still fit (the signed sums cancel)
                    for (int n = n0; n < n1; ++n) { sum_a[n - n0] += at(flo_a, n, o.second); used[n - n0] += at(flo_r, n, o.second); }
                    corr_on[(size_t)g * t.n_kb + o.second] &= (unsigned char)~(16u << cg);
                    ++t.n_corr_skipped;
                }
            }
    }
#ifdef GT_TC_DIAG
    if (skipping && std::getenv("GATEAU_TC_PRINT_MASK")) {           // tuning builds only
        for (int g = 0; g < G; ++g) {
            std::fprintf(stderr, "corr_on group %d:", g);
            for (int kb = 0; kb < t.n_kb; ++kb) std::fprintf(stderr, " %02x", corr_on[(size_t)g * t.n_kb + kb]);
            std::fprintf(stderr, "\n");
        }
    }
#endif
    // ---- phase C, per channel: truncation compensation ----
    host_parallel_for((int64_t)G * nbt, [&](int64_t gn) {
        {
            const int g = (int)(gn / nbt), n = (int)(gn % nbt);
            const int ch = g * nbt + n;
            if (ch >= n_chan) return;
            const double* part = part_all.data() + (size_t)gn * n_steps;
            const int cg = n / kTcBufCols;
            // walk the MMAs of every segment in issue order.  Per slab the MMA thread issues,
            // for k = 0..3, A_hi.Fm_hi (moves the accumulator by part[kb][k]) and A_lo.Fm_hi, then for k = 0..3 A_hi.Fm_lo
            // (the two corrections only where corr_on says so).
            for (int s0 = 0, kb0 = 0; kb0 < t.n_kb; ++s0) {
                int kb1 = kb0;
                while (kb1 < t.n_kb && seg_of[(size_t)cg * t.n_kb + kb1] == s0) ++kb1;
                double S = 0.0;
                for (int kb = kb0; kb < kb1; ++kb) for (int k = 0; k < kTcKSteps; ++k) S += part[(size_t)kb * kTcKSteps + k];
                double W = 0.0;
                if (S != 0.0) {
                    // losses in ulp of the accumulator at that moment; x = mean product of the step in those ulps
                    // (E[1/m] = 0.72 over the mantissa m of the final sum, whose exponent the flush warps know)
                    auto step_x = [&](double part_k, double r) { return r > 0.0 ? std::fabs(part_k / S) / 16.0 / (std::ldexp(0.72, -23) * r) : 0.0; };
                    auto loss_main = [&](double x) { return x < kTcTruncGrain ? 16.0 * x : 16.0 * kTcTruncGrain / 2.0 + 0.5; };
                    auto loss_corr = [&](double x) { return 0.5 * std::min(1.0, x * std::ldexp(1.0, -12) / 1.4142 / kTcTruncGrain); };
                    double acc = 0.0;
                    for (int kb = kb0; kb < kb1; ++kb) {
                        const bool corr_lo = (corr_on[(size_t)g * t.n_kb + kb] >> cg) & 1u, corr_flo = (corr_on[(size_t)g * t.n_kb + kb] >> (4 + cg)) & 1u;
                        for (int k = 0; k < kTcKSteps; ++k) {
                            const double pk = part[(size_t)kb * kTcKSteps + k];
                            acc += pk;
                            const double r = tc_ulp_ratio(acc / S), x = step_x(pk, std::fabs(r));
                            W += r * (loss_main(x) + (corr_lo ? loss_corr(x) : 0.0));
                        }
                        const double r = tc_ulp_ratio(acc / S);
                        if (corr_flo) for (int k = 0; k < kTcKSteps; ++k) W += r * loss_corr(step_x(part[(size_t)kb * kTcKSteps + k], std::fabs(r)));
                    }
                    // a profile that overshoots or changes sign (filters with negative lobes) is not a profile the
                    // row's own sums need follow: keep the compensation inside what a one-signed sum can lose
                    const double w_max = (16.0 * kTcTruncGrain / 2.0 + 1.5) * kTcKSteps * (kb1 - kb0);
                    W = std::max(0.0, std::min(W, w_max));
                }
                if (filt1) W = 0.0;
                comp[((size_t)g * t.n_seg + s0) * nbt + n] = (float)(W * (double)kTcTruncUlp * std::ldexp(1.0, -23));
                kb0 = kb1;
            }
        }
    });
    if (bad) { tc_error_ref() = "the filter holds a NaN or Inf"; return GT_ERR_VALUE; }
    if (tc_alloc_fn()(reinterpret_cast<void**>(&t.filt_img), total) != cudaSuccess ||
        tc_alloc_fn()(reinterpret_cast<void**>(&t.corr_on), corr_on.size()) != cudaSuccess ||
        tc_alloc_fn()(reinterpret_cast<void**>(&t.comp), comp.size() * sizeof(float)) != cudaSuccess) {
        cudaGetLastError(); tc_error_ref() = "cudaMalloc of the filter image failed"; return GT_ERR_OOM;
    }
    if (cudaMemcpyAsync(t.filt_img, img.data(), total, cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(t.comp, comp.data(), comp.size() * sizeof(float), cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(t.corr_on, corr_on.data(), corr_on.size(), cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess) {
        cudaGetLastError(); tc_error_ref() = "upload of the filter image failed"; return GT_ERR_CUDA;
    }
    return GT_OK;
}
// per-CTA scratch tile of partial sums; grid = one CTA per SM
inline gt_status alloc_tc_scratch(TcTables& t, int num_sms) {
    if (t.scratch) return GT_OK;
    const size_t bytes = (size_t)num_sms * 2 * t.nb_tot * kTcBM * sizeof(float);     // two tiles per CTA
    if (tc_alloc_fn()(reinterpret_cast<void**>(&t.scratch), bytes) != cudaSuccess) {
        cudaGetLastError(); tc_error_ref() = "cudaMalloc of the partial-sum scratch failed"; return GT_ERR_OOM;
    }
    return GT_OK;
}
inline void free_tc_tables(TcTables& t) {
    if (t.filt_img) tc_free_fn()(t.filt_img);
    if (t.scratch) tc_free_fn()(t.scratch);
    if (t.comp) tc_free_fn()(t.comp);
    if (t.corr_on) tc_free_fn()(t.corr_on);
    t.filt_img = nullptr; t.scratch = nullptr; t.comp = nullptr; t.corr_on = nullptr;
}

struct TcParams {
    FusedParams f;
    const unsigned char* filt_img;
    float* scratch;
    const float* comp;          // [group][n_seg][nb_tot] truncation compensation (build_tc_tables)
    const unsigned char* corr_on;   // [group][n_kb] bit cg: column group cg gets A_lo.Fm_hi in this slab, bit 4 + cg: A_hi.Fm_lo (banded corrections)
    int32_t n_seg;
    int32_t n_groups, nb_tot, n_cg, seg, n_kb, unit_bytes, b_stages;
    int32_t n_row_tiles;
    int32_t cube_vec;           // 1: cube spectra can be read as aligned float4
    int32_t debug;              // timing diagnostics only (GATEAU_TC_DEBUG): 1 = generator skips its arithmetic, 2 = no MMAs issued, 4 = no filter copies, 8 = no finisher work
};

// shared-memory map relative to the 1024-byte aligned base:
//   [0, NAS*32 KB)                  A ring: stage s at s*32 KB = {hi 16 KB, lo 16 KB}
//   [NAS*32 KB, .. + NBS*unit)      B ring
//   then barriers: a_full[2] a_empty[2] b_full[4] b_empty[4] flush_full[4] buf_free[4] tile_done[2]
//   scratch_free[2], tensor-memory slot
struct TcSmem {
    uint32_t a, b, a_full, a_empty, b_full, b_empty, flush_full, buf_free, tile_done, scratch_free, b_peer, slot, rowp, wcomp, stage;
    __device__ TcSmem(uint32_t base, int b_stages, int unit_bytes) {
        a = base; b = base + kTcAStages * kTcAStageBytes;
        const uint32_t bar = b + (uint32_t)b_stages * (uint32_t)unit_bytes;
        a_full = bar; a_empty = bar + 32; b_full = bar + 64; b_empty = bar + 96;
        flush_full = bar + 128; buf_free = bar + 160; tile_done = bar + 192; scratch_free = bar + 208; b_peer = bar + 224; slot = bar + 256;
        rowp = bar + 320;
        wcomp = rowp + kTcBM * 32;
        stage = wcomp + kTcEpiWarps * kTcBufCols * 4;
    }
};

// Column groups of a tile and the rotation of their accumulators through the tensor-memory
// buffers.  The MMA thread and the epilogue warps each run one instance over the same
// (tile, slab, group) sequence, so they agree on which buffer a group occupies without talking.
// All state is packed into registers (2 bits per buffer id): the MMA thread's issue loop must
// stay far below the 2112 cycles the tensor pipe needs per slab.
struct TcRotation {
    int n_cg, seg, n_kb;
    uint32_t bufs;                 // buffer of group g in bits [2g, 2g+2)
    uint32_t fifo;                 // free buffers, oldest in bits [0, 2)
    int shift;                     // 2 * (number of free buffers - 1)
    int cnt[kTcMaxCg];             // position of the group in its (staggered) segment grid
    __device__ TcRotation(int n_cg_, int seg_, int n_kb_) : n_cg(n_cg_), seg(seg_), n_kb(n_kb_) {
        bufs = 0u | (1u << 2) | (2u << 4);
        fifo = 0u; int c = 0;
        for (int b = n_cg_; b < kTcNumBuf; ++b, ++c) fifo |= (uint32_t)b << (2 * c);
        shift = 2 * (c - 1);
#pragma unroll
        for (int g = 0; g < kTcMaxCg; ++g) cnt[g] = (g * seg_) / n_cg_;
    }
    __device__ __forceinline__ int buf(int g) const { return (int)((bufs >> (2 * g)) & 3u); }
    // called once per (slab, group) in slab order: does group g close a segment after slab kb?
    // Returns the number of slabs of the segment that closes (0: no boundary).
    // called once per (slab, group) in slab order: does group g close a segment after slab kb?
    __device__ __forceinline__ bool boundary(int kb, int g) {
        if (kb == n_kb - 1) { cnt[g] = (g * seg) / n_cg; return true; }
        if (++cnt[g] == seg) { cnt[g] = 0; return true; }
        return false;
    }
    // moves group g to the oldest free buffer; returns the buffer it leaves
    __device__ __forceinline__ int rotate(int g) {
        const uint32_t old = (bufs >> (2 * g)) & 3u, nb = fifo & 3u;
        fifo = (fifo >> 2) | (old << shift);
        bufs = (bufs & ~(3u << (2 * g))) | (nb << (2 * g));
        return (int)old;
    }
    __device__ __forceinline__ int width(int g, int nb_tot) const { return min(kTcBufCols, nb_tot - g * kTcBufCols); }
};

// steps 2-4 for one (row, nu) element as in element_value (gt_fused_fp32.cuh), with the two MUFU
// operations issued as single instructions: eta_z is in (0,1] and csc >= 1, so log2 is <= 0 and finite
// and 2^(csc log2 eta_z) underflows to 0 exactly where eta_atm is below 1e-38.
__device__ __forceinline__ float element_value_fast(float eta_z, float csc, float Xn, float G, float S) {
    const float eta = ptx::ex2_ftz(csc * ptx::lg2_ftz(eta_z));
    return fmaf(eta, fmaf(G, S, -Xn), Xn);           // (1 - eta) Xn + eta G S in two FMAs
}

// Writes 4 consecutive frequencies (lane-chunk `chunk` of half `h` of a 64-frequency slab) of tile row `row`
// into an A stage as the fp16 pair (hi, lo) of the scaled value: hi = fp16(s v), lo = fp16(s v - hi), 22
// mantissa bits together.  Part 0 holds hi, part 1 lo, each as K-major SWIZZLE_128B rows of 64 fp16.  The filter
// is split the same way at plan time and the contraction is issued as hi.Fm_hi + lo.Fm_hi + hi.Fm_lo with
// kind::f16 MMAs (K = 16, fp32 accumulate): north_star's three-term split with the accuracy of 3xTF32 (each
// product of two 11-bit pieces is exact in fp32, the dropped lo.Fm_lo is 2^-22) at 3/8 of its tensor time and
// half of its operand bytes.
__device__ __forceinline__ void store_split(unsigned char* a_stage, int row, int chunk, int h, const float4& v) {
    const float2 s01 = make_float2(v.x, v.y), s23 = make_float2(v.z, v.w);      // v is already scaled: the plan folds kTcScaleA into Xn and Gs
    const __half2 h01 = __float22half2_rn(s01), h23 = __float22half2_rn(s23);
    const float2 b01 = __half22float2(h01), b23 = __half22float2(h23);
    const __half2 l01 = __float22half2_rn(ptx::upk2(ptx::sub2(ptx::pk2(s01.x, s01.y), ptx::pk2(b01.x, b01.y))));    // FADD2
    const __half2 l23 = __float22half2_rn(ptx::upk2(ptx::sub2(ptx::pk2(s23.x, s23.y), ptx::pk2(b23.x, b23.y))));
    uint2 hi2, lo2;
    hi2.x = *reinterpret_cast<const uint32_t*>(&h01); hi2.y = *reinterpret_cast<const uint32_t*>(&h23);
    lo2.x = *reinterpret_cast<const uint32_t*>(&l01); lo2.y = *reinterpret_cast<const uint32_t*>(&l23);
    const uint32_t c16 = (uint32_t)(h * 4 + (chunk >> 1)), sub = (uint32_t)(chunk & 1) * 8u;
    unsigned char* dst = a_stage + (uint32_t)row * 128u + ((c16 ^ (uint32_t)(row & 7)) << 4) + sub;
    *reinterpret_cast<uint2*>(dst) = hi2;
    *reinterpret_cast<uint2*>(dst + kTcAPartBytes) = lo2;
}

// Eq. 17 pass (NEP = true): the same shared-memory slots hold fp16(v) in part 0 and fp16(v^2 / 256) in part 1 (single
// terms: sigma only needs 1e-3); the filter units hold L and Fm^2 kPref 256 / E0 on one per-channel scale, so that
// part 0 . unit 0 + part 1 . unit 1 accumulates the linear and the quadratic term of NEP^2 into ONE accumulator.
__device__ __forceinline__ void store_nep(unsigned char* a_stage, int row, int chunk, int h, const float4& v) {
    const __half2 h01 = __float22half2_rn(make_float2(v.x, v.y)), h23 = __float22half2_rn(make_float2(v.z, v.w));
    const __half2 q01 = __float22half2_rn(make_float2(v.x * v.x * kTcSqScale, v.y * v.y * kTcSqScale));
    const __half2 q23 = __float22half2_rn(make_float2(v.z * v.z * kTcSqScale, v.w * v.w * kTcSqScale));
    uint2 a2, b2;
    a2.x = *reinterpret_cast<const uint32_t*>(&h01); a2.y = *reinterpret_cast<const uint32_t*>(&h23);
    b2.x = *reinterpret_cast<const uint32_t*>(&q01); b2.y = *reinterpret_cast<const uint32_t*>(&q23);
    const uint32_t c16 = (uint32_t)(h * 4 + (chunk >> 1)), sub = (uint32_t)(chunk & 1) * 8u;
    unsigned char* dst = a_stage + (uint32_t)row * 128u + ((c16 ^ (uint32_t)(row & 7)) << 4) + sub;
    *reinterpret_cast<uint2*>(dst) = a2;
    *reinterpret_cast<uint2*>(dst + kTcAPartBytes) = b2;
}

// element (column, row) of a scratch tile laid out [row / 32][column / 16][row % 32][16 columns]: the 16 columns x 32 rows one
// flush batch moves are 2 KB contiguous (one bulk copy), and inside them a row's 16 columns are 64 contiguous bytes, so a
// finisher warp (lane = channel, one row) touches two 64-byte pieces per load instead of eight 16-byte ones.  The four
// 16-byte chunks of a row are XOR-swizzled with bits 1-2 of the row: the flush warps' 16-byte shared stores (lane = row) are
// then conflict-free, and the bulk copy carries the permutation into the scratch tile unchanged.
__device__ __forceinline__ size_t tc_scratch_index(int col, int row, int nb_tot) {
    return ((size_t)(row >> 5) * (size_t)(nb_tot >> 4) + (size_t)(col >> 4)) * 512 + (size_t)(row & 31) * 16
         + (size_t)((((col >> 2) & 3) ^ ((row >> 1) & 3)) << 2) + (size_t)(col & 3);
}

__device__ __forceinline__ float4 ldg4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }

template <bool VEC, bool NEP>
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
            ptx::mbar_init(sm.a_full + 8 * s, (kTcPair ? 2 : 1) * kTcGenWarps);      // pair: the leader also counts the peer's generators
            ptx::mbar_init(sm.a_empty + 8 * s, 1);
        }
        for (int s = 0; s < kTcMaxBStages; ++s) {
            ptx::mbar_init(sm.b_full + 8 * s, 1);
            ptx::mbar_init(sm.b_empty + 8 * s, 1);
            ptx::mbar_init(sm.b_peer + 8 * s, 1);
        }
        for (int b = 0; b < kTcNumBuf; ++b) {
            ptx::mbar_init(sm.flush_full + 8 * b, 1);
            ptx::mbar_init(sm.buf_free + 8 * b, (kTcPair ? 2 : 1) * kTcEpiWarps);
        }
        for (int b = 0; b < 2; ++b) {
            ptx::mbar_init(sm.tile_done + 8 * b, kTcEpiWarps);
            ptx::mbar_init(sm.scratch_free + 8 * b, kTcFinWarps);
        }
        ptx::fence_mbar_init();
    }
    if (warp == kTcWarpMma) {
        if constexpr (kTcPair) { ptx::tmem_alloc2(sm.slot, 512); ptx::tmem_relinquish2(); }
        else { ptx::tmem_alloc(sm.slot, 512); ptx::tmem_relinquish(); }
    }
    ptx::tc_fence_before();
    if constexpr (kTcPair) ptx::cluster_sync_all(); else __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = *reinterpret_cast<const volatile uint32_t*>(smem_raw + (sm.slot - raw));

    // Work distribution.  Single CTA: tile = (row tile, channel group), strided over the grid.  CTA pair: the
    // pair takes two consecutive row tiles of one channel group (rank r the r-th of them); both CTAs run the
    // same number of iterations, a row tile past the end is computed on default rows and never stored.
    const uint32_t rank = kTcPair ? ptx::cluster_ctarank() : 0u;
    const int64_t worker = kTcPair ? (int64_t)ptx::cluster_id_x() : (int64_t)blockIdx.x;
    const int64_t n_workers = kTcPair ? (int64_t)ptx::cluster_nctaid_x() : (int64_t)gridDim.x;
    const int64_t n_tiles = kTcPair ? (int64_t)((p.n_row_tiles + 1) / 2) * p.n_groups : (int64_t)p.n_row_tiles * p.n_groups;
    // arrive on a barrier the leader CTA waits on / wait for a signal that may come from the peer CTA
    auto arrive_leader = [&](uint32_t bar) {
        if (kTcPair && rank != 0) ptx::mbar_arrive_cluster(ptx::mapa(bar, 0)); else ptx::mbar_arrive(bar);
    };
    auto wait_pair = [&](uint32_t bar, uint32_t parity) {
        ptx::mbar_wait_relaxed(bar, parity);      // CTA-scope acquire: a cluster-scope one would invalidate L1 on every wait
    };
    auto wait_lead = [&](uint32_t bar, uint32_t parity) {          // leader's waits on barriers the peer also arrives on
        ptx::mbar_wait(bar, parity);
    };
    auto commit_pair = [&](uint32_t bar) {                          // completion of the MMAs issued so far, signalled to both CTAs
        if constexpr (kTcPair) ptx::tc_commit2(bar, (uint16_t)3); else ptx::tc_commit(bar);
    };
    auto mma_f16 = [&](uint32_t d, uint64_t a, uint64_t b, uint32_t id, uint32_t acc) {       // kind::f16, K = 16
        if constexpr (kTcPair) ptx::mma2_f16_ss(d, a, b, id, acc); else ptx::mma_f16_ss(d, a, b, id, acc);
    };
    // Row tiles are TIME-MAJOR: row tile rt = (block of 128 consecutive samples tb, spaxel s), tile row r = sample
    // tb*128 + r of the launch.  Consecutive samples of one spaxel point ~1 source pixel apart, so their 2 x 2 tap
    // footprints share cube lines (L1 hits) and, almost always, the two LUT rows.
    const int64_t n_t = f.n_rows / f.n_spaxel;                      // samples in this launch
    auto tile_rt = [&](int64_t tl) -> int64_t {
        const int64_t rt = tl / p.n_groups;
        return kTcPair ? 2 * rt + rank : rt;
    };
    // global row (t * n_spaxel + s) of tile row r, or -1 past the end of the launch
    auto tile_row = [&](int64_t rt, int r) -> int64_t {
        const int64_t tb = rt / f.n_spaxel, s = rt - tb * f.n_spaxel, t = tb * kTcBM + r;
        return t < n_t ? t * f.n_spaxel + s : -1;
    };
    if (warp >= kTcWarpGen0 && warp < kTcWarpFin0) {
        // =========================== generator: steps 2-4 -> A ring ===========================
        ptx::setmaxnreg_inc<kTcRegsGen>();
        const int gw = warp - kTcWarpGen0;
        // general path (any n_freq, no 16-byte loads): rows of this thread rsub and rsub + 64; a warp's four rows are
        // {0,4,1,5} or {2,6,3,7} of an 8-row swizzle group, in lane order (conflict-free 8-byte shared stores per half warp)
        const int q4 = lane >> 3;
        const int rsub = (gw >> 1) * 8 + (gw & 1) * 2 + (q4 >> 1) + (q4 & 1) * 4, chunk = lane & 7;
        const size_t nf = (size_t)f.n_freq, nfp = (size_t)f.n_freq_pad;
        uint32_t a_st = 0, a_ph = 0;           // A-ring stage and its phase parity
        if constexpr (VEC) {
            // Warp = TWO rows x the whole 64-frequency slab (half warp = one row, lane = 4 frequencies); a thread walks FOUR
            // rows (32 apart) per slab.  Against the earlier map (warp = four rows x half a slab, two rows per thread) the
            // per-frequency vectors Xn, G and the LUT rows, which every row of the tile shares, are fetched once per slab
            // and four rows instead of once per half slab and two rows: half the 16-byte loads whose 512 bytes per warp hold
            // only 128-256 distinct ones (the L1's wavefront pipe is this kernel's busiest unit, profiles/r02b), and a half
            // warp's 8-byte shared stores cover one whole 128-byte row: conflict-free by construction.
            // The loads of the next row are issued before the current one is computed; the per-row constants live in
            // shared memory (each warp only reads rows it wrote itself).
            struct Tap { float4 c00, c01, c10, c11; };
            struct Lut { float4 L0, L1; };
            constexpr int kRows = 4, kStride = 2 * kTcGenWarps;          // rows of a thread: r0 + 32 j
            static_assert(kRows * kStride == kTcBM, "generator rows");
            const int q2 = lane >> 4, c16 = lane & 15, r0 = 2 * gw + q2;
            RowParam* rowp = reinterpret_cast<RowParam*>(smem_raw + (sm.rowp - raw));
            for (int64_t tl = worker; tl < n_tiles; tl += n_workers) {
                const int64_t rt = tile_rt(tl);
                __syncwarp();
                if (c16 < kRows) {
                    const int64_t R = tile_row(rt, r0 + kStride * c16);
                    RowParam rp;
                    if (R >= 0) {
                        const int4* src = reinterpret_cast<const int4*>(f.rows + R);
                        const int4 a = __ldg(src), b = __ldg(src + 1);
                        rp.fp = __int_as_float(a.x); rp.csc = __int_as_float(a.y); rp.ip = a.z; rp.pix = a.w;
                        rp.w00 = __int_as_float(b.x); rp.w01 = __int_as_float(b.y);
                        rp.w10 = __int_as_float(b.z); rp.w11 = __int_as_float(b.w);
                    } else {
                        rp.fp = 0.f; rp.csc = 1.f; rp.ip = 0; rp.pix = -1; rp.w00 = rp.w01 = rp.w10 = rp.w11 = 0.f;
                    }
                    if (f.cube == nullptr || rp.pix < 0) { rp.pix = 0; rp.w00 = rp.w01 = rp.w10 = rp.w11 = 0.f; }
                    rowp[gw * 8 + c16 * 2 + q2] = rp;      // slot of row (j = c16, q2): the warp's two rows of one j are adjacent
                }
                __syncwarp();
                // 32-bit element offsets of this thread's rows (plan creation rejects tables of 2^32 elements or more).
                // Rows outside the cube carry zero weights and read pixel 0; padded frequencies read the last real
                // chunk (their filter entries are zero), so every load is unconditional and in bounds.
                uint32_t lut_off[kRows], cube_off[kRows];
#pragma unroll
                for (int j = 0; j < kRows; ++j) {
                    const int4 a = *reinterpret_cast<const int4*>(rowp + gw * 8 + j * 2 + q2);   // fp, csc, ip, pix
                    lut_off[j] = (uint32_t)a.z * (uint32_t)nfp + (uint32_t)c16 * 4u;
                    cube_off[j] = (uint32_t)a.w * (uint32_t)nf;
                }
                // The base pointer lives in a per-thread register pair (it gets an opaque zero added): "base + 4 * offset" then
                // compiles to LEA + LEA.HI.X on the integer pipe.  With the base in a uniform register it is IMAD.MOV (the
                // constant 4) + IMAD.WIDE on the FMA pipe, which the packed FFMA2 stream already keeps busy: 78.0-79.2 ->
                // 76.5 ms per C4 step.
                const float* cube_base = f.cube != nullptr ? f.cube : f.lut_r;
                {
                    uint32_t zero;                                    // lane >> 5: always 0, opaque to the compiler
                    asm volatile("mov.u32 %0, %%laneid;" : "=r"(zero));
                    cube_base += zero >> 5;
                }
                const uint32_t tap01 = f.cube != nullptr ? (uint32_t)nf : 0u;
                const uint32_t tap10 = f.cube != nullptr ? (uint32_t)f.n_az * (uint32_t)nf : 0u;
                const uint32_t nu_last = (uint32_t)(max(f.n_freq, 4) - 4) & ~3u;     // 16-byte aligned (n_freq % 4 == 0 with a cube)
                // The two LUT rows are looked up per SAMPLE, but the PWV moves by ~1e-4 of a LUT step per sample: the
                // rows of a thread nearly always share them.  They are fetched for row 0 of every slab and re-fetched for
                // a later row only where its LUT row differs from the one before.
                bool new_lut[kRows];
#pragma unroll
                for (int j = 1; j < kRows; ++j) new_lut[j] = lut_off[j] != lut_off[j - 1];
                auto issue_lut = [&](int kb, int j, Lut& l) {
                    const uint32_t lo = lut_off[j] + (uint32_t)kb * kTcBK;
                    l.L0 = ldg4(f.lut_r + lo); l.L1 = ldg4(f.lut_r + (lo + (uint32_t)nfp));
                };
                auto issue = [&](int kb, int j, Tap& t) {
                    if (GT_DIAG(p, 16)) return;
                    const uint32_t co = cube_off[j] + min((uint32_t)kb * kTcBK + (uint32_t)c16 * 4u, nu_last);
                    t.c00 = ldg4(cube_base + co);           t.c01 = ldg4(cube_base + (co + tap01));
                    t.c10 = ldg4(cube_base + (co + tap10)); t.c11 = ldg4(cube_base + (co + tap10 + tap01));
                };
                auto compute = [&](int j, const Tap& cur, const Lut& lut, const float4& X, const float4& G, uint32_t stage) {
                    const RowParam* rp = rowp + gw * 8 + j * 2 + q2;
                    const float2 fc = *reinterpret_cast<const float2*>(rp);                    // fp, csc (registers for them cost spills: measured 91 -> 108 ms)
                    const float4 w = *reinterpret_cast<const float4*>(&rp->w00);
                    float4 v;
                    // steps 2-4 on pairs of frequencies: every fp32 operation below is one FFMA2 / FMUL2 / FADD2 for two
                    // elements (the same IEEE operations in the same order as the scalar form, half the issue slots)
                    {
                        using namespace ptx;
                        const f32x2 w00 = pk2(w.x, w.x), w01 = pk2(w.y, w.y), w10 = pk2(w.z, w.z), w11 = pk2(w.w, w.w);
                        const f32x2 fp2 = pk2(fc.x, fc.x), csc2 = pk2(fc.y, fc.y);
                        auto pair = [&](float c00x, float c00y, float c01x, float c01y, float c10x, float c10y, float c11x, float c11y,
                                        float l0x, float l0y, float l1x, float l1y, float Xx, float Xy, float Gx, float Gy,
                                        float& vx, float& vy) {
                            f32x2 S2 = mul2(w00, pk2(c00x, c00y));
                            S2 = fma2(w01, pk2(c01x, c01y), S2);
                            S2 = fma2(w10, pk2(c10x, c10y), S2);
                            S2 = fma2(w11, pk2(c11x, c11y), S2);
                            const f32x2 L0 = pk2(l0x, l0y);
                            const float2 ez = upk2(fma2(fp2, sub2(pk2(l1x, l1y), L0), L0));
                            const float2 lg = upk2(mul2(csc2, pk2(lg2_ftz(ez.x), lg2_ftz(ez.y))));
                            const f32x2 eta = pk2(ex2_ftz(lg.x), ex2_ftz(lg.y));
                            const float2 r = upk2(fma2(eta, fma2(pk2(Gx, Gy), S2, pk2(-Xx, -Xy)), pk2(Xx, Xy)));
                            vx = r.x; vy = r.y;
                        };
                        pair(cur.c00.x, cur.c00.y, cur.c01.x, cur.c01.y, cur.c10.x, cur.c10.y, cur.c11.x, cur.c11.y,
                             lut.L0.x, lut.L0.y, lut.L1.x, lut.L1.y, X.x, X.y, G.x, G.y, v.x, v.y);
                        pair(cur.c00.z, cur.c00.w, cur.c01.z, cur.c01.w, cur.c10.z, cur.c10.w, cur.c11.z, cur.c11.w,
                             lut.L0.z, lut.L0.w, lut.L1.z, lut.L1.w, X.z, X.w, G.z, G.w, v.z, v.w);
                    }
                    const int row = r0 + kStride * j;
                    if constexpr (NEP) store_nep(smem_raw + (sm.a - raw) + stage * kTcAStageBytes, row, c16 & 7, c16 >> 3, v);
                    else store_split(smem_raw + (sm.a - raw) + stage * kTcAStageBytes, row, c16 & 7, c16 >> 3, v);
                };
                Tap t0, t1;
                Lut lut;
                issue(0, 0, t0);
                for (int kb = 0; kb < p.n_kb; ++kb, a_ph ^= (++a_st == kTcAStages), a_st = a_st == kTcAStages ? 0u : a_st) {
                    const uint32_t stage = a_st, ph = a_ph;
                    if (GT_DIAG(p, 1)) {
                        wait_pair(sm.a_empty + 8 * stage, ph ^ 1u);
                        __syncwarp();
                        if (lane == 0) arrive_leader(sm.a_full + 8 * stage);
                        continue;
                    }
                    issue_lut(kb, 0, lut);
                    const float4 X = ldg4(f.Xn + kb * kTcBK + c16 * 4), G = ldg4(f.Gs + kb * kTcBK + c16 * 4);
                    issue(kb, 1, t1);
                    wait_pair(sm.a_empty + 8 * stage, ph ^ 1u);
                    compute(0, t0, lut, X, G, stage);
                    issue(kb, 2, t0);
                    if (new_lut[1]) issue_lut(kb, 1, lut);
                    compute(1, t1, lut, X, G, stage);
                    issue(kb, 3, t1);
                    if (new_lut[2]) issue_lut(kb, 2, lut);
                    compute(2, t0, lut, X, G, stage);
                    if (kb + 1 < p.n_kb) issue(kb + 1, 0, t0);
                    if (new_lut[3]) issue_lut(kb, 3, lut);
                    compute(3, t1, lut, X, G, stage);
                    // one arrival per warp: 512 per-thread arrivals on one mbarrier serialise (~5 cycles each)
                    ptx::fence_proxy_async_smem();
                    __syncwarp();
                    if (lane == 0) arrive_leader(sm.a_full + 8 * stage);
                }
            }
        } else
        for (int64_t tl = worker; tl < n_tiles; tl += n_workers) {
            const int64_t rt = tile_rt(tl);
            float fp[kTcRowsPerThread], csc[kTcRowsPerThread], w00[kTcRowsPerThread], w01[kTcRowsPerThread], w10[kTcRowsPerThread], w11[kTcRowsPerThread];
            const float* lutp[kTcRowsPerThread];
            const float* cubep[kTcRowsPerThread];
#pragma unroll
            for (int j = 0; j < kTcRowsPerThread; ++j) {
                const int64_t R = tile_row(rt, rsub + kTcRowStride * j);
                RowParam rp;
                if (R >= 0) {
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
            for (int kb = 0; kb < p.n_kb; ++kb, a_ph ^= (++a_st == kTcAStages), a_st = a_st == kTcAStages ? 0u : a_st) {
                const uint32_t stage = a_st, ph = a_ph;
                if (GT_DIAG(p, 1)) {
                    wait_pair(sm.a_empty + 8 * stage, ph ^ 1u);
                    __syncwarp();
                    if (lane == 0) arrive_leader(sm.a_full + 8 * stage);
                    continue;
                }
                for (int h = 0; h < 2; ++h) {
                const int hb = 2 * kb + h;
                const int nu0 = hb * kTcHB + chunk * 4;
                const float4 X = ldg4(f.Xn + nu0), G = ldg4(f.Gs + nu0);
                float4 L0[kTcRowsPerThread], L1[kTcRowsPerThread], S[kTcRowsPerThread];
#pragma unroll
                for (int j = 0; j < kTcRowsPerThread; ++j) {
                    L0[j] = ldg4(lutp[j] + hb * kTcHB);
                    L1[j] = ldg4(lutp[j] + nfp + hb * kTcHB);
                    S[j] = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (cubep[j] != nullptr && nu0 < f.n_freq) {
                        const float* c00 = cubep[j] + hb * kTcHB;
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
                if (h == 0) wait_pair(sm.a_empty + 8 * stage, ph ^ 1u);
                unsigned char* a_hi = smem_raw + (sm.a - raw) + stage * kTcAStageBytes;
#pragma unroll
                for (int j = 0; j < kTcRowsPerThread; ++j) {
                    float4 v;
                    v.x = element_value_fast(fmaf(fp[j], L1[j].x - L0[j].x, L0[j].x), csc[j], X.x, G.x, S[j].x);
                    v.y = element_value_fast(fmaf(fp[j], L1[j].y - L0[j].y, L0[j].y), csc[j], X.y, G.y, S[j].y);
                    v.z = element_value_fast(fmaf(fp[j], L1[j].z - L0[j].z, L0[j].z), csc[j], X.z, G.z, S[j].z);
                    v.w = element_value_fast(fmaf(fp[j], L1[j].w - L0[j].w, L0[j].w), csc[j], X.w, G.w, S[j].w);
                    if constexpr (NEP) store_nep(a_hi, rsub + kTcRowStride * j, chunk, h, v);
                    else store_split(a_hi, rsub + kTcRowStride * j, chunk, h, v);
                }
                }
                ptx::fence_proxy_async_smem();
                __syncwarp();
                if (lane == 0) arrive_leader(sm.a_full + 8 * stage);
            }
        }
    } else if (warp >= kTcWarpCtl0) {
      ptx::setmaxnreg_dec<kTcRegsCtl>();
      if (warp == kTcWarpLoader) {
        // =========================== loader: filter slab images -> B ring =====================
        // (pair: each CTA copies its half of every unit, the rows of the N/2 columns it supplies to the MMA)
        if (lane == 0) {
            uint32_t bs = 0, bph = 0;
            for (int64_t tl = worker; tl < n_tiles; tl += n_workers) {
                const int g = (int)(tl % p.n_groups);
                const size_t stride = (size_t)p.unit_bytes * (kTcPair ? 2 : 1);
                const unsigned char* src = p.filt_img + (size_t)g * p.n_kb * 2 * stride + (size_t)rank * p.unit_bytes;
                for (int u = 0; u < 2 * p.n_kb; ++u) {
                    wait_pair(sm.b_empty + 8 * bs, bph ^ 1u);
                    if (GT_DIAG(p, 4)) ptx::mbar_arrive(sm.b_full + 8 * bs);
                    else {
                        ptx::mbar_arrive_expect_tx(sm.b_full + 8 * bs, (uint32_t)p.unit_bytes);
                        ptx::bulk_g2s(sm.b + bs * (uint32_t)p.unit_bytes, src + (size_t)u * stride,
                                      (uint32_t)p.unit_bytes, sm.b_full + 8 * bs);
                    }
                    if (++bs == (uint32_t)p.b_stages) { bs = 0; bph ^= 1u; }
                }
            }
        }
        __syncwarp();
      } else if (kTcPair && warp == kTcWarpCtl0 && rank != 0) {
        // =========================== forwarder (peer CTA): tells the leader that our half unit has landed ====
        if (lane == 0) {
            uint32_t bs = 0, bph = 0;
            for (int64_t tl = worker; tl < n_tiles; tl += n_workers)
                for (int u = 0; u < 2 * p.n_kb; ++u) {
                    ptx::mbar_wait(sm.b_full + 8 * bs, bph);
                    ptx::mbar_arrive_cluster(ptx::mapa(sm.b_peer + 8 * bs, 0));
                    if (++bs == (uint32_t)p.b_stages) { bs = 0; bph ^= 1u; }
                }
        }
        __syncwarp();
      } else if (warp == kTcWarpMma && rank == 0) {
        // =========================== MMA issuer (pair: the leader CTA issues for both) ===============
        {   // the whole warp runs the loop (uniform control flow); one elected lane issues
            TcRotation rot(p.n_cg, p.seg, p.n_kb);
            uint32_t idesc[kTcMaxCg];
            uint32_t fresh = 7u;               // bit g: next MMA into buf(g) overwrites (first of a segment)
            uint32_t used = 0u, par = 0u;      // bit b: buffer b was flushed before / parity of its flush count
#pragma unroll
            for (int g = 0; g < kTcMaxCg; ++g) idesc[g] = ptx::idesc_f16(kTcPair ? 2 * kTcBM : kTcBM, g < p.n_cg ? rot.width(g, p.nb_tot) : 16);
            const bool issue = !GT_DIAG(p, 2);
            constexpr int kGroupDesc = (kTcBufCols * 128 >> 4) / (kTcPair ? 2 : 1);   // descriptor step between column groups (pair: half the rows)
            uint32_t a_st = 0, a_ph = 0, bs = 0, bph = 0;
            for (int64_t tl = worker; tl < n_tiles; tl += n_workers) {
                const unsigned char* const corr_t = p.corr_on + (size_t)(tl % p.n_groups) * p.n_kb;
                for (int kb = 0; kb < p.n_kb; ++kb, a_ph ^= (++a_st == kTcAStages), a_st = a_st == kTcAStages ? 0u : a_st) {
                    const uint32_t stage = a_st, ph = a_ph;
                    // banded corrections: bit g = column group g gets A_lo.Fm_hi in this slab, bit 4 + g = A_hi.Fm_lo (fetched
                    // before the waits below: an L1/L2 hit whose latency they cover)
                    const uint32_t corr = NEP ? 0xFFu : (uint32_t)__ldg(corr_t + kb);
                    uint32_t d[kTcMaxCg];
                    // a group that has just moved to another buffer waits until the epilogue has drained it
#pragma unroll
                    for (int g = 0; g < kTcMaxCg; ++g) {
                        const uint32_t b = (uint32_t)rot.buf(g);
                        d[g] = tmem_base + b * (uint32_t)kTcBufCols;
                        if (g < p.n_cg && (fresh >> g & 1u) && (used >> b & 1u))
                            wait_lead(sm.buf_free + 8 * b, par >> b & 1u);
                    }
                    wait_lead(sm.a_full + 8 * stage, ph);
                    const uint64_t ad_hi = ptx::smem_desc_sw128(sm.a + stage * kTcAStageBytes);
                    const uint64_t ad_lo = ad_hi + (uint64_t)(kTcAPartBytes >> 4);
                    {   // unit 0: acc += A_hi.Fm_hi + A_lo.Fm_hi
                        ptx::mbar_wait(sm.b_full + 8 * bs, bph);
                        if constexpr (kTcPair) ptx::mbar_wait(sm.b_peer + 8 * bs, bph);
                        ptx::tc_fence_after();
                        const uint64_t bd0 = ptx::smem_desc_sw128(sm.b + bs * (uint32_t)p.unit_bytes);
                        if (issue && ptx::elect_one()) {
#pragma unroll
                            for (int k = 0; k < kTcKSteps; ++k)
#pragma unroll
                                for (int g = 0; g < kTcMaxCg; ++g)
                                    if (g < p.n_cg) {
                                        const uint64_t bd = bd0 + (uint64_t)(g * kGroupDesc + k * 2);
                                        mma_f16(d[g], ad_hi + (uint64_t)(k * 2), bd, idesc[g], (k != 0 || !(fresh >> g & 1u)) ? 1u : 0u);
                                        if constexpr (!NEP) if (corr >> g & 1u) mma_f16(d[g], ad_lo + (uint64_t)(k * 2), bd, idesc[g], 1u);
                                    }
                        }
                        __syncwarp();
                        if (ptx::elect_one()) commit_pair(sm.b_empty + 8 * bs);
                        if (++bs == (uint32_t)p.b_stages) { bs = 0; bph ^= 1u; }
                    }
                    {   // unit 1: acc += A_hi.Fm_lo
                        ptx::mbar_wait(sm.b_full + 8 * bs, bph);
                        if constexpr (kTcPair) ptx::mbar_wait(sm.b_peer + 8 * bs, bph);
                        ptx::tc_fence_after();
                        const uint64_t bd0 = ptx::smem_desc_sw128(sm.b + bs * (uint32_t)p.unit_bytes);
                        if (issue && ptx::elect_one()) {
#pragma unroll
                            for (int k = 0; k < kTcKSteps; ++k)
#pragma unroll
                                for (int g = 0; g < kTcMaxCg; ++g)
                                    if (g < p.n_cg && (corr >> (4 + g) & 1u))
                                        mma_f16(d[g], (NEP ? ad_lo : ad_hi) + (uint64_t)(k * 2),
                                                        bd0 + (uint64_t)(g * kGroupDesc + k * 2), idesc[g], 1u);
                        }
                        __syncwarp();
                        if (ptx::elect_one()) commit_pair(sm.b_empty + 8 * bs);
                        if (++bs == (uint32_t)p.b_stages) { bs = 0; bph ^= 1u; }
                    }
                    if (ptx::elect_one()) commit_pair(sm.a_empty + 8 * stage);
                    // segment boundaries: hand the finished partial sums to the epilogue, move on to a free buffer
                    fresh = 0u;
#pragma unroll
                    for (int g = 0; g < kTcMaxCg; ++g) {
                        if (g < p.n_cg && rot.boundary(kb, g)) {
                            const uint32_t old = (uint32_t)rot.rotate(g);
                            if (ptx::elect_one()) commit_pair(sm.flush_full + 8 * old);
                            par ^= (used >> old & 1u) << old;      // parity of (flush count - 1) once used
                            used |= 1u << old;
                            fresh |= 1u << g;
                        }
                    }
                }
            }
        }
        __syncwarp();
      }
    } else if (warp >= kTcWarpFin0 && warp < kTcWarpCtl0) {
        // ============ finisher: scratch tile -> P = sum*scale + bias, photon noise -> TOD ========
        if constexpr (kTcRegsFin > kTcRegsBase) ptx::setmaxnreg_inc<kTcRegsFin>(); else if constexpr (kTcRegsFin < kTcRegsBase) ptx::setmaxnreg_dec<kTcRegsFin>();
        const int q = warp - kTcWarpFin0;
        uint32_t ti = 0;
        for (int64_t tl = worker; tl < n_tiles; tl += n_workers, ++ti) {
            const int64_t rt = tile_rt(tl);
            const int64_t tb = rt / f.n_spaxel;
            const uint32_t s = (uint32_t)(rt - tb * f.n_spaxel);
            const int cg0 = (int)(tl % p.n_groups) * p.nb_tot;
            const int n_valid = min(p.nb_tot, f.n_chan - cg0);            // real channels of this group
            const uint32_t sb = ti & 1u;
            const float* sc = p.scratch + ((size_t)blockIdx.x * 2 + sb) * p.nb_tot * kTcBM;
            ptx::mbar_wait_relaxed(sm.tile_done + 8 * sb, (ti >> 1) & 1u);
            constexpr int kMaxPerLane = kTcMaxGroupChan / 32;             // 12
            constexpr bool kPrefetch = GT_TC_FIN_PREFETCH != 0;
            float x[kMaxPerLane], xn[kPrefetch ? kMaxPerLane : 1];
            if constexpr (kPrefetch) {
#pragma unroll
                for (int j = 0; j < kMaxPerLane; ++j) {
                    const int c = lane + 32 * j;
                    xn[j] = c < n_valid ? __ldcg(sc + tc_scratch_index(c, q, p.nb_tot)) : 0.f;
                }
            }
            for (int r = q; r < kTcBM; r += kTcFinWarps) {
                const int64_t t = tb * kTcBM + r;                         // sample of this row within the launch
                if (t >= n_t || GT_DIAG(p, 8)) break;
                const uint32_t n = (uint32_t)(f.t0 + t);
                float* o = f.out + (size_t)(t * f.n_spaxel + s) * f.n_chan + cg0;
                if constexpr (kPrefetch) {
                    // this row's partial sums were fetched during the previous row; fetch the next row's now
#pragma unroll
                    for (int j = 0; j < kMaxPerLane; ++j) {
                        x[j] = xn[j];
                        const int c = lane + 32 * j;
                        xn[j] = (c < n_valid && r + kTcFinWarps < kTcBM) ? __ldcg(sc + tc_scratch_index(c, r + kTcFinWarps, p.nb_tot)) : 0.f;
                    }
                } else {
                    // all of this row's partial sums are requested at once; the other finisher warp of the scheduler covers the latency
#pragma unroll
                    for (int j = 0; j < kMaxPerLane; ++j) {
                        const int c = lane + 32 * j;
                        x[j] = c < n_valid ? __ldcg(sc + tc_scratch_index(c, r, p.nb_tot)) : 0.f;
                    }
                }
                // One Philox block per FOUR channels (R19): the lane owns channels lane + 32 j, and the four channels
                // lane + 128 m + {0, 32, 64, 96} of quad m share the block 32 (cg0 / 128 + m) + lane (group starts are
                // multiples of 128, build_tc_tables), whose four normals are the cosine and sine branches of two
                // Box-Muller pairs.  QW blocks are interleaved: the ten rounds of one block are a serial chain.
                constexpr int kQuads = kMaxPerLane / 4, QW = GT_TC_FIN_QW;
                const uint32_t blk0 = (((uint32_t)cg0 >> 7) << 5) + (uint32_t)lane;
#pragma unroll
                for (int m0 = 0; m0 < kQuads; m0 += QW) {
                    if (lane + 128 * m0 >= n_valid) break;
                    float z[QW][4];
                    if (NEP || f.photon_noise) {
                        uint32_t cc[QW];
                        uint4 w[QW];
#pragma unroll
                        for (int i = 0; i < QW; ++i) cc[i] = blk0 + 32u * (uint32_t)(m0 + i);
                        philox4x32_10_multi4<QW>(n, f.spaxel_base + s, cc, kStreamPhoton, f.seed_lo, f.seed_hi, w);
#pragma unroll
                        for (int i = 0; i < QW; ++i) normals_of_block(w[i], z[i]);
                    } else {
#pragma unroll
                        for (int i = 0; i < QW; ++i) z[i][0] = z[i][1] = z[i][2] = z[i][3] = 0.f;
                    }
#pragma unroll
                    for (int i = 0; i < QW; ++i) {
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            const int j = 4 * (m0 + i) + k, c = lane + 32 * j;
                            if (j < kMaxPerLane && c < n_valid) {
                                const float4 k4 = __ldg(f.chan4 + cg0 + c);   // bias, h f_c f_s, f_s / dnu_c, 2^-kb (the channel's filter scale)
                                float P = fmaf(x[j] * k4.w, f.scale, k4.x);
                                if constexpr (NEP) {
                                    // Eq. 17 pass: P = NEP^2 / (2 E0) of this detector-sample; the TOD already holds the noiseless power of
                                    // the first pass: tod += sqrt(P f_s) sqrt(E0) z, z = the normal of the narrow-band mode (Eq. 18-19)
                                    const float sigma = sqrt_fast(fmaxf(P, 0.f) * f.nep_f_sample) * f.nep_sqrt_e0;
                                    P = fmaf(sigma, z[i][k], __ldcs(o + c));
                                } else if (f.photon_noise) {
                                    P = fmaf(photon_sigma(P, k4.y, k4.z), z[i][k], P);
                                }
                                __stcs(o + c, P);                          // streaming store: the TOD must not evict the scratch tiles from L2
                            }
                        }
                    }
                }
            }
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(sm.scratch_free + 8 * sb);
        }
    } else {
        // ============ epilogue: segment flushes of the accumulators into the scratch tile =======
        ptx::setmaxnreg_dec<kTcRegsFlush>();
        const int q = warp;                                    // tensor-memory lane quarter (tile row = tensor-memory lane 32 q + lane)
        TcRotation rot(p.n_cg, p.seg, p.n_kb);
        uint32_t fulls = 0u;                                   // bit b: parity of buffer b's flush count
        uint32_t ti = 0;
        for (int64_t tl = worker; tl < n_tiles; tl += n_workers, ++ti) {
            const uint32_t sb = ti & 1u;
            float* const sc = p.scratch + ((size_t)blockIdx.x * 2 + sb) * p.nb_tot * kTcBM;
            if (ti >= 2) ptx::mbar_wait_relaxed(sm.scratch_free + 8 * sb, ((ti >> 1) - 1u) & 1u);   // finisher done with tile ti-2
            bool first[kTcMaxCg] = {true, true, true};
            int segi[kTcMaxCg] = {0, 0, 0};                      // segment of the tile each group is in
            const float* const comp_t = p.comp + (size_t)(tl % p.n_groups) * p.n_seg * p.nb_tot;
            for (int kb = 0; kb < p.n_kb; ++kb)
#pragma unroll
                for (int g = 0; g < kTcMaxCg; ++g) {
                    if (g >= p.n_cg || !rot.boundary(kb, g)) continue;
                    const int b = rot.rotate(g);
                    const int wg = rot.width(g, p.nb_tot);
                    // truncation-compensation weights of this (group, segment): fetched into this warp's own shared-memory
                    // strip BEFORE the wait, so that the flush itself never waits on global memory for them
                    float4* const wsm = reinterpret_cast<float4*>(smem_raw + (sm.wcomp - raw)) + q * (kTcBufCols / 4);
                    {
                        const float4* const comp4 = reinterpret_cast<const float4*>(comp_t + (size_t)segi[g] * p.nb_tot + g * kTcBufCols);
                        __syncwarp();
                        wsm[lane] = 4 * lane < wg ? __ldg(comp4 + lane) : make_float4(0.f, 0.f, 0.f, 0.f);
                        __syncwarp();
                    }
                    ++segi[g];
                    // The partial sums go to the scratch tile through the bulk-copy engine: 16 columns x this warp's 32 rows
                    // (2 KB, contiguous in the scratch layout) are staged in shared memory and sent with ONE
                    // cp.async.bulk (first segment: store) or cp.reduce.async.bulk.add.f32 (later segments: the L2 adds,
                    // round to nearest) -- the flush never waits for a load of the running sums, so its duration no longer
                    // depends on the L2 round trip and the accumulator buffer is handed back after ~8 short batches.
                    float* const scw = sc + tc_scratch_index(g * kTcBufCols, 32 * q, p.nb_tot);            // this warp's strip of the group
                    const uint32_t taddr = tmem_base + ((uint32_t)(32 * q) << 16) + (uint32_t)(b * kTcBufCols);
                    const bool add = !first[g];
                    uint32_t v[16];
                    wait_pair(sm.flush_full + 8 * b, fulls >> b & 1u);
                    fulls ^= 1u << b;
                    ptx::tc_fence_after();
                    // 32 columns (two tcgen05.ld of 16) per round: both halves go into this warp's 4 KB staging strip, ONE
                    // proxy fence and ONE 4 KB bulk copy per round.  wg is a multiple of 32.
                    float4* const stg = reinterpret_cast<float4*>(smem_raw + (sm.stage - raw)) + q * (2 * kTcStageBytes / 16) + lane * 4;
                    const uint32_t stg_s = sm.stage + (uint32_t)(q * 2 * kTcStageBytes);
                    for (int c0 = 0; c0 < wg; c0 += 32) {
                        ptx::tmem_ld_32x16(taddr + (uint32_t)c0, v);
                        // the strip was last read by the bulk copy of the previous round
                        if (lane == 0) ptx::bulk_wait_read<0>();
                        ptx::tmem_ld_wait();
                        __syncwarp();
#pragma unroll
                        for (int hh = 0; hh < 2; ++hh) {
                            if (hh == 1) {
                                ptx::tmem_ld_32x16(taddr + (uint32_t)(c0 + 16), v);
                                ptx::tmem_ld_wait();
                                if (c0 + 32 >= wg) {
                                    // all of the group's columns are in registers: the accumulator buffer can go back to the MMA thread
                                    ptx::tc_fence_before();
                                    __syncwarp();
                                    if (lane == 0) arrive_leader(sm.buf_free + 8 * b);
                                }
                            }
#pragma unroll
                            for (int i = 0; i < 4; ++i) {
                                // truncation compensation: the segment lost w ulp of its own sum (table of the plan, per
                                // channel and segment); +-2^e of the sum = its sign and exponent bits
#ifndef GT_TC_NO_COMP
                                const float4 w4 = wsm[(c0 + 16 * hh) / 4 + i];
#else
                                const float4 w4 = make_float4(0.f, 0.f, 0.f, 0.f);      // tuning builds: cost of the table look-up
#endif
                                float4 sum;
                                sum.x = fmaf(__uint_as_float(v[4 * i] & 0xFF800000u), w4.x, __uint_as_float(v[4 * i]));
                                sum.y = fmaf(__uint_as_float(v[4 * i + 1] & 0xFF800000u), w4.y, __uint_as_float(v[4 * i + 1]));
                                sum.z = fmaf(__uint_as_float(v[4 * i + 2] & 0xFF800000u), w4.z, __uint_as_float(v[4 * i + 2]));
                                sum.w = fmaf(__uint_as_float(v[4 * i + 3] & 0xFF800000u), w4.w, __uint_as_float(v[4 * i + 3]));
                                stg[hh * (kTcStageBytes / 16) + (i ^ ((lane >> 1) & 3))] = sum;      // [16-column batch][row][16 columns, chunks swizzled], as the scratch tile
                            }
                        }
                        ptx::fence_proxy_async_smem();
                        __syncwarp();
                        if (lane == 0) {
                            float* const dst = scw + (size_t)(c0 / 16) * (32 * 16);
                            if (add) ptx::bulk_reduce_add_f32_s2g(dst, stg_s, 2 * kTcStageBytes); else ptx::bulk_s2g(dst, stg_s, 2 * kTcStageBytes);
                            ptx::bulk_commit();
                        }
                    }
                    first[g] = false;
                }
            // every partial sum of the tile is on its way: once this warp's bulk copies have completed, hand the
            // tile to the finisher warps
            if (lane == 0) { ptx::bulk_wait_all(); __threadfence(); ptx::mbar_arrive(sm.tile_done + 8 * sb); }
            __syncwarp();
        }
    }

    ptx::tc_fence_before();
    if constexpr (kTcPair) ptx::cluster_sync_all(); else __syncthreads();     // pair: the peer's shared and tensor memory stay alive until both are done
    if (warp == kTcWarpMma) {
        ptx::tc_fence_after();
        if constexpr (kTcPair) ptx::tmem_dealloc2(tmem_base, 512); else ptx::tmem_dealloc(tmem_base, 512);
    }
}

// nep = true: the second pass of the exact photon noise (Eq. 17, R23): the generator writes fp16(v) and
// fp16(v^2 / 256), the tables hold L and the scaled Fm^2, the finisher turns the contraction into sigma and adds sigma z
// to the TOD the first pass wrote.
inline cudaError_t launch_fused_tc(const FusedParams& fp, const TcTables& t, int num_sms, cudaStream_t st, bool nep = false) {
    TcParams p{};
    p.f = fp; p.filt_img = t.filt_img;
    // FusedParams::scale carries the spectrum scale of the plan; the per-channel filter scale is chan4.w
    p.scratch = t.scratch; p.comp = t.comp; p.corr_on = t.corr_on; p.n_seg = t.n_seg;
    p.n_groups = t.n_groups; p.nb_tot = t.nb_tot; p.n_cg = t.n_cg; p.seg = t.seg > 0 ? t.seg : kTcSegDefault; p.n_kb = t.n_kb;
    p.unit_bytes = t.unit_bytes; p.b_stages = t.b_stages;
    p.n_row_tiles = (int32_t)(((fp.n_rows / fp.n_spaxel + kTcBM - 1) / kTcBM) * fp.n_spaxel);      // time-major: blocks of 128 samples x spaxels
#ifdef GT_TC_DIAG
    if (const char* e = std::getenv("GATEAU_TC_DEBUG")) p.debug = std::atoi(e);      // tuning builds only
#endif
    p.cube_vec = (fp.cube == nullptr) || ((fp.n_freq % 4 == 0) && ((reinterpret_cast<uintptr_t>(fp.cube) & 15u) == 0));
    const int64_t n_tiles = kTcPair ? (int64_t)((p.n_row_tiles + 1) / 2) * p.n_groups : (int64_t)p.n_row_tiles * p.n_groups;
    const int64_t workers = kTcPair ? num_sms / 2 : num_sms;
    const unsigned grid = (unsigned)(std::min<int64_t>(n_tiles, workers) * (kTcPair ? 2 : 1));
    auto kern = nep ? (p.cube_vec ? fused_tc_kernel<true, true> : fused_tc_kernel<false, true>)
                       : (p.cube_vec ? fused_tc_kernel<true, false> : fused_tc_kernel<false, false>);
    // set on every launch: the attribute is per device
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, t.smem_bytes);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(kTcThreads); cfg.dynamicSmemBytes = (size_t)t.smem_bytes; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = kTcPair ? 2 : 1; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    e = cudaLaunchKernelEx(&cfg, kern, p);
    if (e != cudaSuccess) return e;
    return cudaGetLastError();
}

}  // namespace gt
