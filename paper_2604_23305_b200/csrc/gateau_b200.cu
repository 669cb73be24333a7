// gateau_b200.cu -- C ABI (include/gateau_b200.h), plan (host double-precision precompute,
// device tables, streams) and kernel launches of libgateau_b200.so.
//
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo -O3 -shared -Xcompiler -fPIC
// No code is shared with oracle/ and nothing here runs the path on the CPU: the host code
// only validates, derives per-frequency/per-channel constants once per plan, and launches.
#include "../../include/gateau_b200.h"

#include <cmath>
#include <cstdio>
#include <cstdarg>
#include <cstring>
#include <cstdlib>
#include <string>
#include <vector>
#include <new>
#include <atomic>

#include "gt_common.cuh"
#include "gt_geometry.cuh"
#include "gt_fused_fp32.cuh"
#include "gt_fused_tc.cuh"
#include "gt_pink.cuh"
#include "gt_pink_tk.cuh"
#include "gt_kelvin.cuh"
#include "gt_screen.cuh"
#include "gt_beam.cuh"
#include "gt_reduce.cuh"
#include "gt_measure.cuh"
#include "gt_common_mode.cuh"
#include <cufft.h>

// ---- gt_common_mode_static: the [t x chan] partial sums of Eq. 25 in library-owned static device memory ----
// Part of the module image: every GPU that loads this library holds these 8 MB until the process exits.  In HOST code the
// name below is a host-side stand-in, not a device address (a kernel given it faults, or silently uses the wrong memory
// where the GPU can reach host memory): host code uses the address cudaGetSymbolAddress returns, resolved once per
// device at plan creation (cm_static_resolve) with that device current.
static __device__ __align__(256) float g_cm_static_scratch[GT_COMMON_MODE_STATIC_MAX];

namespace {
float* g_cm_static_ptr[64] = {};          // per device: device address of g_cm_static_scratch (nullptr = not resolved yet)
std::atomic<bool> g_cm_static_ok[64] = {};

// set-up, once per device, with that device current (called by gt_plan_create)
cudaError_t cm_static_resolve(int dev) {
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    if (g_cm_static_ok[dev].load(std::memory_order_acquire)) return cudaSuccess;
    float* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_cm_static_scratch);
    if (e != cudaSuccess) return e;
    if (ptr == nullptr) return cudaErrorInvalidSymbol;
    g_cm_static_ptr[dev] = ptr;            // racing plan creations on one device store the same value
    g_cm_static_ok[dev].store(true, std::memory_order_release);
    return cudaSuccess;
}
}  // namespace

namespace {

// CODATA exact values (PAPER.md names h, k_B implicitly through P^JN; R4)
constexpr double kH = 6.62607015e-34, kKB = 1.380649e-23, kPi = 3.14159265358979323846;
// Spectrum scale: the kernels work on P_nu / p_ref with p_ref = k_B 300 K 2^-e, e chosen per plan so that the largest
// element the generator can produce lands just below 2^kTcAMaxLog2, the range the tensor kernel's fp16 operand split
// wants.
constexpr double kPref0 = kKB * 300.0;

thread_local std::string g_create_error = "";

// single-moded Johnson-Nyquist / Planck spectral power h nu / (exp(h nu / kT) - 1), 0 at T = 0
double jn_power(double nu, double T) {
    if (!(T > 0.0)) return 0.0;
    return kH * nu / std::expm1(kH * nu / (kKB * T));
}

// Device memory of the plans comes from ONE library-owned stream-ordered pool per device that keeps what plans return
// (release threshold = everything): creating and destroying plans back to back -- an observation per plan, as bench.py's
// end-to-end leg does -- does not pay cudaMalloc / cudaFree of the 0.5 GB chunk buffers each time.
// gt_release_cached_memory() gives the cached blocks back to the driver.
cudaStream_t g_pool_stream[64] = {};      // the pool's own (non-blocking) stream: allocations and releases are ordered on it
cudaMemPool_t plan_pool(int dev) {
    static cudaMemPool_t pools[64] = {};
    if (dev < 0 || dev >= 64) return nullptr;
    if (!pools[dev]) {
        if (cudaStreamCreateWithFlags(&g_pool_stream[dev], cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); return nullptr; }
        cudaMemPoolProps props{};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool = nullptr;
        if (cudaMemPoolCreate(&pool, &props) != cudaSuccess) { cudaGetLastError(); return nullptr; }
        uint64_t keep = UINT64_MAX;
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        pools[dev] = pool;
    }
    return pools[dev];
}

// the same pool for the tensor kernel's tables (gt_fused_tc.cuh): plain pointers, so the device of the pool is looked up
cudaError_t pool_alloc_raw(void** p, size_t bytes) {
    int dev = 0;
    cudaMemPool_t pool = cudaGetDevice(&dev) == cudaSuccess ? plan_pool(dev) : nullptr;
    if (!pool) return cudaMalloc(p, bytes);
    cudaError_t e = cudaMallocFromPoolAsync(p, std::max<size_t>(bytes, 1), pool, g_pool_stream[dev]);
    if (e == cudaSuccess) e = cudaStreamSynchronize(g_pool_stream[dev]);
    return e;
}
void pool_free_raw(void* p) {
    int dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess && plan_pool(dev)) cudaFreeAsync(p, g_pool_stream[dev]); else cudaFree(p);
}

template <class T>
struct DevBuf {
    T* p = nullptr; size_t n = 0; int pool_dev = -1;
    // allocation and release are ordered on the pool's own stream; an allocation is synchronised before it is handed out,
    // a release happens only after the plan's streams have been synchronised (gt_plan_destroy) or before first use
    cudaError_t alloc(size_t count) {
        release(); n = count;
        const size_t bytes = std::max<size_t>(count, 1) * sizeof(T);
        int dev = 0;
        cudaMemPool_t pool = cudaGetDevice(&dev) == cudaSuccess ? plan_pool(dev) : nullptr;
        if (pool) {
            cudaError_t e = cudaMallocFromPoolAsync(reinterpret_cast<void**>(&p), bytes, pool, g_pool_stream[dev]);
            if (e == cudaSuccess) e = cudaStreamSynchronize(g_pool_stream[dev]);
            if (e == cudaSuccess) { pool_dev = dev; return e; }
            cudaGetLastError(); p = nullptr;
        }
        pool_dev = -1;
        return cudaMalloc(reinterpret_cast<void**>(&p), bytes);
    }
    cudaError_t upload(const std::vector<T>& h, cudaStream_t st) {
        cudaError_t e = alloc(h.size());
        if (e != cudaSuccess || h.empty()) return e;
        return cudaMemcpyAsync(p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice, st);
    }
    void release() {
        if (p) { if (pool_dev >= 0) cudaFreeAsync(p, g_pool_stream[pool_dev]); else cudaFree(p); }
        p = nullptr; n = 0; pool_dev = -1;
    }
    ~DevBuf() { release(); }
};

}  // namespace

struct gt_plan {
    // sizes
    int32_t n_freq = 0, n_freq_pad = 0, n_chan = 0, n_chan_pad = 0, n_spaxel = 0, n_pwv = 0, J = 0;
    int64_t n_samples = 0, chunk_samples = 0, chunk_dev = 0;      // samples per launch: host-output chunks / device output
    int32_t photon_noise = 0, pink_noise = 0, variant = GT_VARIANT_FP32;
    bool tc_full = false;             // GT_VARIANT_TENSOR_FULL: every correction product of the split is issued
    int32_t spaxel_base = 0;         // global index of spaxel 0 of this plan (Philox counter word 1)
    int device = 0;
    uint64_t seed = 0;
    float scale = 0.f;
    double p_ref = kPref0;           // W/Hz per unit of the generated spectrum
    // borrowed
    const float* cube = nullptr; int32_t n_az = 0, n_el = 0;
    // geometry
    gt::GeoParams geo{};
    DevBuf<double> d_tan_az, d_tan_el, d_sinE, d_cosE, d_az, d_el;
    DevBuf<double> d_sp;             // 6 per-spaxel tables back to back
    // fused-kernel tables
    DevBuf<float> d_Xn, d_Gs, d_lut_r, d_filt_t, d_bias, d_c1, d_c2;
    DevBuf<float4> d_chan4;
    // exact Eq. 17 photon noise (R23): two more filter sets for the tensor kernel and their outputs
    int32_t photon_mode = 0;
    gt::TcTables tc_nep;                        // filter units L and Fm^2 kPref 256 / E0 of the second pass
    DevBuf<float4> d_chan4_nep;
    float sqrt_e0 = 0.f, f_sample = 0.f;
    int32_t output_unit = 0;                    // 1: brightness temperature through the skydip map (R22)
    DevBuf<double> d_kelvin_ab;                 // [2][n_chan] a, b
    DevBuf<float2> d_kelvin_abf;                // [n_chan] (a, b)
    gt::TcTables tc;                 // tensor-kernel operand images
    // pink
    gt::PinkParams pink{};
    DevBuf<float> d_gain, d_state, d_seg;
    DevBuf<uint32_t> d_pink_sync;
    int32_t pink_method = 0;         // 0 AR(1) cascade, 1 Timmer & Koenig
    gt::TkParams tk{};
    DevBuf<float> d_tk_amp, d_tk_halpha, d_tk_series;   // ticket counter + per-(segment, detector block) flags of the chained pink kernel
    int64_t pink_next_t = 0;
    // scratch
    DevBuf<gt::RowParam> d_rows;     // [chunk rows]
    DevBuf<float> d_chunk[2];        // device TOD chunks (host output only), allocated lazily
    DevBuf<float> d_pwv[2];
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_ready[2] = {nullptr, nullptr}, ev_copied[2] = {nullptr, nullptr};
    std::vector<cudaEvent_t> ev_fused;       // start/stop pairs of the last call
    std::vector<cudaEvent_t> ev_tl;          // host-output calls: per chunk {compute begin, compute end, copy begin, copy end} (timing enabled)
    int32_t n_tl_last = 0;
    int32_t n_fused_last = 0;
    int64_t launches = 0;
    int num_sms = 148;
    // common-mode subtraction (Eq. 25-26): what the plan keeps of its inputs for it
    std::vector<float> h_lut;  int32_t n_nu_lut = 0;
    double lut_nu0 = 0, lut_dnu = 0, lut_pwv0 = 0, lut_dpwv = 0;
    std::vector<double> h_daz, h_del, h_fc;
    DevBuf<double> d_ln_eta_z;  DevBuf<float> d_cm_weight;      // common mode: [4][n_chan] le, eta0, 1 - eta0, 1 / eta0; [n_spaxel] S_j
    double cm_csc0 = 1.0;                                      // reference airmass of the common-mode kernels (boresight)
    // diagnostics (SURVEY section 5 "Metrics"): rows seen by the geometry kernel, rows outside the cube, PWV clamps
    DevBuf<unsigned long long> d_counters;   // [3] outside cube, PWV below / above the LUT
    int64_t rows_done = 0;
    cudaStream_t last_stream = nullptr;
    std::string error;
};

namespace {

gt_status fail(gt_plan* p, gt_status st, const char* fmt, ...) {
    char buf[512];
    va_list ap; va_start(ap, fmt); vsnprintf(buf, sizeof buf, fmt, ap); va_end(ap);
    if (p) p->error = buf; else g_create_error = buf;
    return st;
}

#define GT_CUDA(plan, expr)                                                                   \
    do { cudaError_t e_ = (expr);                                                             \
         if (e_ != cudaSuccess) return fail(plan, e_ == cudaErrorMemoryAllocation ? GT_ERR_OOM : GT_ERR_CUDA, \
                                            "%s: %s", #expr, cudaGetErrorString(e_)); } while (0)

// copy a small DEVICE array to the host (plan creation only)
gt_status fetch(const float* dev, size_t n, std::vector<float>& out, const char* what) {
    out.resize(n);
    cudaError_t e = cudaMemcpy(out.data(), dev, n * sizeof(float), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return fail(nullptr, GT_ERR_CUDA, "reading %s from device: %s", what, cudaGetErrorString(e));
    return GT_OK;
}

gt_status validate(const gt_config* c) {
    if (!c) return fail(nullptr, GT_ERR_NULL, "cfg is NULL");
    if (!c->az_rad || !c->el_rad || !c->daz_rad || !c->del_rad || !c->screen || !c->atm_lut || !c->filt ||
        !c->f_center_hz) return fail(nullptr, GT_ERR_NULL, "a required array pointer is NULL");
    if (c->n_freq <= 0 || c->n_samples <= 0 || c->n_spaxel <= 0 || c->n_chan <= 0 || c->nx <= 0 || c->ny <= 0 ||
        c->n_pwv < 2 || c->n_nu_lut < 2 || c->n_stage < 0 || c->chunk_samples < 0)
        return fail(nullptr, GT_ERR_SHAPE, "a size is non-positive (n_freq/n_samples/n_spaxel/n_chan/nx/ny/n_pwv/n_nu_lut/n_stage)");
    if (c->n_samples > 0xFFFFFFFELL) return fail(nullptr, GT_ERR_SHAPE, "n_samples exceeds the 32-bit Philox counter word");
    if (c->spaxel_index_base < 0) return fail(nullptr, GT_ERR_VALUE, "spaxel_index_base is negative");
    {
        // Eq. 10 needs every line of sight above the horizon: sin(el0 + el[n] + del[s]) > 0 for all n, s
        double e_lo = c->el_rad[0], e_hi = c->el_rad[0], d_lo = c->del_rad[0], d_hi = c->del_rad[0];
        bool finite = std::isfinite(c->el0_rad);
        for (int64_t n = 0; n < c->n_samples; ++n) {
            finite = finite && std::isfinite(c->az_rad[n]) && std::isfinite(c->el_rad[n]);
            e_lo = std::min(e_lo, c->el_rad[n]); e_hi = std::max(e_hi, c->el_rad[n]);
        }
        for (int s = 0; s < c->n_spaxel; ++s) {
            finite = finite && std::isfinite(c->daz_rad[s]) && std::isfinite(c->del_rad[s]);
            d_lo = std::min(d_lo, c->del_rad[s]); d_hi = std::max(d_hi, c->del_rad[s]);
        }
        if (!finite) return fail(nullptr, GT_ERR_VALUE, "the scan pattern or the spaxel offsets hold a NaN or Inf");
        if (!(c->el0_rad + e_lo + d_lo > 0.0) || !(c->el0_rad + e_hi + d_hi < 3.14159265358979323846))
            return fail(nullptr, GT_ERR_VALUE, "a line of sight is at or below the horizon: el0 + el + del spans [%g, %g] rad",
                        c->el0_rad + e_lo + d_lo, c->el0_rad + e_hi + d_hi);
    }
    if (c->n_stage > 0 && !c->stages) return fail(nullptr, GT_ERR_NULL, "stages is NULL with n_stage > 0");
    if (c->cube && (c->n_az < 2 || c->n_el < 2)) return fail(nullptr, GT_ERR_SHAPE, "source cube needs n_az, n_el >= 2");
    if (c->cube && (double)c->n_az * (double)c->n_el * (double)c->n_freq >= 4294967296.0)
        return fail(nullptr, GT_ERR_SHAPE, "source cube of 2^32 elements or more is not supported (32-bit tap offsets)");
    if (c->cube && (!(c->daz_grid_rad > 0) || !(c->del_grid_rad > 0)))
        return fail(nullptr, GT_ERR_VALUE, "source grid steps must be positive");
    if (!(c->f_sample_hz > 0) || !(c->dnu_hz > 0) || !(c->nu0_hz > 0) || !(c->dx_m > 0) || !(c->dy_m > 0) ||
        !(c->lut_dnu_hz > 0) || !(c->lut_dpwv_mm > 0))
        return fail(nullptr, GT_ERR_VALUE, "f_sample, dnu, nu0, dx, dy, lut_dnu, lut_dpwv must be positive");
    if (c->T_cmb_K < 0 || c->T_atm_K < 0) return fail(nullptr, GT_ERR_VALUE, "negative temperature");
    for (int k = 0; k < c->n_stage; ++k) {
        const gt_stage& s = c->stages[k];
        if (s.T_K < 0) return fail(nullptr, GT_ERR_VALUE, "stage %d: negative temperature", k + 1);
        if (!s.eta_nu && !(s.eta_scalar >= 0.0 && s.eta_scalar <= 1.0))
            return fail(nullptr, GT_ERR_VALUE, "stage %d: eta_scalar outside [0,1]", k + 1);
    }
    if (c->pink_method != 0 && c->pink_method != 1) return fail(nullptr, GT_ERR_VALUE, "unknown pink_method %d", c->pink_method);
    if (c->photon_mode != 0 && c->photon_mode != 1) return fail(nullptr, GT_ERR_VALUE, "unknown photon_mode %d", c->photon_mode);
    if (c->photon_noise && c->photon_mode == 1) {
        if (c->variant == GT_VARIANT_FP32) return fail(nullptr, GT_ERR_UNSUPPORTED, "photon_mode = 1 (Eq. 17) runs on the tensor variant only");
        if (!(c->kid_gap_J >= 0.0) || !(c->eta_pb > 0.0) || !std::isfinite(c->kid_gap_J) || !std::isfinite(c->eta_pb))
            return fail(nullptr, GT_ERR_VALUE, "kid_gap_J = %g, eta_pb = %g are not a valid pair-breaking energy and efficiency", c->kid_gap_J, c->eta_pb);
    }
    if (c->output_unit != 0 && c->output_unit != 1) return fail(nullptr, GT_ERR_VALUE, "unknown output_unit %d", c->output_unit);
    if (c->output_unit == 1) {
        if (c->skydip_n < 2 || c->skydip_n > 64) return fail(nullptr, GT_ERR_SHAPE, "skydip_n = %d is outside 2..64", c->skydip_n);
        if (!(c->skydip_pwv_hi_mm > c->skydip_pwv_lo_mm) || !std::isfinite(c->skydip_pwv_lo_mm) || !std::isfinite(c->skydip_pwv_hi_mm))
            return fail(nullptr, GT_ERR_VALUE, "skydip PWV range [%g, %g] mm is empty", c->skydip_pwv_lo_mm, c->skydip_pwv_hi_mm);
        if (!(std::sin(c->el0_rad) > 0.0)) return fail(nullptr, GT_ERR_VALUE, "skydip: boresight elevation is not above the horizon");
    }
    if (c->pink_noise && c->pink_method == 0) {
        if (c->pink_n_stage < 1 || c->pink_n_stage > gt::kPinkMaxJ)
            return fail(nullptr, GT_ERR_SHAPE, "pink_n_stage must be in 1..8");
        if (!c->pink_A || !c->pink_alpha || !c->pink_f_corner_hz)
            return fail(nullptr, GT_ERR_NULL, "pink noise arrays are NULL");
    }
    if (c->pink_noise && c->pink_method == 1 && (!c->pink_A || !c->pink_alpha))
        return fail(nullptr, GT_ERR_NULL, "pink noise arrays are NULL");
    if (c->variant != GT_VARIANT_DEFAULT && c->variant != GT_VARIANT_FP32 && c->variant != GT_VARIANT_TENSOR && c->variant != GT_VARIANT_TENSOR_FULL)
        return fail(nullptr, GT_ERR_VALUE, "unknown variant %d", c->variant);
    // LUT must cover the frequency grid (R13)
    const double r_lo = (c->nu0_hz - c->lut_nu0_hz) / c->lut_dnu_hz;
    const double r_hi = (c->nu0_hz + (c->n_freq - 1) * c->dnu_hz - c->lut_nu0_hz) / c->lut_dnu_hz;
    if (r_lo < -1e-9 || r_hi > (c->n_nu_lut - 1) + 1e-9)
        return fail(nullptr, GT_ERR_RANGE, "atm_lut frequency range does not cover the frequency grid");
    return GT_OK;
}

template <int TN>
cudaError_t launch_fp32(const gt::FusedParams& fp, int grid_y, cudaStream_t st) {
    const size_t smem = (size_t)(gt::kF32_BK * gt::kF32_AStride + gt::kF32_BK * 32 * TN) * sizeof(float)
                      + gt::kF32_BM * sizeof(gt::RowParam);
    // set on every launch: the attribute is per device and a microsecond is nothing next to the kernel
    cudaError_t e = cudaFuncSetAttribute(gt::fused_fp32_kernel<TN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)((fp.n_rows + gt::kF32_BM - 1) / gt::kF32_BM), grid_y);
    gt::fused_fp32_kernel<TN><<<grid, gt::kF32_Threads, smem, st>>>(fp);
    return cudaGetLastError();
}

// channels per CTA of the FP32 kernel = 32 * TN; pick the smallest instantiated TN that covers
// n_chan in one block column, else 11 with several block columns.
int fp32_tn(int n_chan) {
    const int need = (n_chan + 31) / 32;
    for (int tn : {1, 2, 4, 6, 8, 11}) if (tn >= need) return tn;
    return 11;
}

cudaError_t launch_fused_fp32(const gt_plan* p, const gt::FusedParams& fp, cudaStream_t st) {
    const int tn = fp32_tn(p->n_chan);
    const int gy = (p->n_chan + 32 * tn - 1) / (32 * tn);
    switch (tn) {
        case 1: return launch_fp32<1>(fp, gy, st);
        case 2: return launch_fp32<2>(fp, gy, st);
        case 4: return launch_fp32<4>(fp, gy, st);
        case 6: return launch_fp32<6>(fp, gy, st);
        case 8: return launch_fp32<8>(fp, gy, st);
        default: return launch_fp32<11>(fp, gy, st);
    }
}

// One chunk: geometry -> fused -> (pink).  dst/pwv_dst are DEVICE pointers.
gt_status run_chunk(gt_plan* p, int64_t t0, int64_t T, float* dst, float* pwv_dst, bool noise,
                    cudaStream_t st, int fused_slot) {
    const int64_t n_rows = T * p->n_spaxel;
    if (n_rows == 0) return GT_OK;
    gt::geometry_kernel<<<(unsigned)((n_rows + 255) / 256), 256, 0, st>>>(p->geo, t0, n_rows, p->d_rows.p, pwv_dst, nullptr, p->d_counters.p);
    GT_CUDA(p, cudaGetLastError());
    p->launches++;
    p->rows_done += n_rows;

    gt::FusedParams fp{};
    fp.rows = p->d_rows.p; fp.n_rows = n_rows; fp.t0 = t0;
    fp.n_spaxel = p->n_spaxel; fp.n_chan = p->n_chan; fp.n_freq = p->n_freq; fp.n_freq_pad = p->n_freq_pad;
    fp.Xn = p->d_Xn.p; fp.Gs = p->d_Gs.p; fp.lut_r = p->d_lut_r.p;
    fp.cube = p->cube; fp.n_az = p->n_az;
    fp.filt_t = p->d_filt_t.p; fp.n_chan_pad = p->n_chan_pad;
    fp.scale = p->scale; fp.bias = p->d_bias.p; fp.noise_c1 = p->d_c1.p; fp.noise_c2 = p->d_c2.p; fp.chan4 = p->d_chan4.p;
    const bool exact = noise && p->photon_noise && p->photon_mode == 1;
    fp.photon_noise = (noise && !exact) ? p->photon_noise : 0;
    fp.seed_lo = (uint32_t)(p->seed & 0xffffffffu); fp.seed_hi = (uint32_t)(p->seed >> 32);
    fp.spaxel_base = (uint32_t)p->spaxel_base;
    fp.out = dst;

    while ((int)p->ev_fused.size() < 2 * (fused_slot + 1)) {
        cudaEvent_t e; GT_CUDA(p, cudaEventCreate(&e)); p->ev_fused.push_back(e);
    }
    GT_CUDA(p, cudaEventRecord(p->ev_fused[2 * fused_slot], st));
    if (p->variant == GT_VARIANT_FP32) {
        GT_CUDA(p, launch_fused_fp32(p, fp, st));
    } else {
        GT_CUDA(p, gt::launch_fused_tc(fp, p->tc, p->num_sms, st));
    }
    if (exact) {
        // Eq. 17: a second pass of the fused kernel contracts the spectrum with L and its square with Fm^2 into ONE
        // accumulator (single fp16 terms, one segment), and its finisher adds sigma z to the TOD of the first pass
        gt::FusedParams fn = fp;
        fn.chan4 = p->d_chan4_nep.p; fn.nep_f_sample = p->f_sample; fn.nep_sqrt_e0 = p->sqrt_e0;
        p->tc_nep.scratch = p->tc.scratch;                                       // the passes run one after another
        GT_CUDA(p, gt::launch_fused_tc(fn, p->tc_nep, p->num_sms, st, true));
        p->launches += 1;
    }
    GT_CUDA(p, cudaEventRecord(p->ev_fused[2 * fused_slot + 1], st));
    p->launches++;
    p->n_fused_last = fused_slot + 1;

    // brightness-temperature output (the gt_simulate path; gt_debug_pkid stays in W): the map T = a_c + b_c (total of Eq. 21)
    // rides on the last kernel that writes the TOD -- the pink-noise kernels -- and is a pass of its own only without them
    const bool kelvin = noise && p->output_unit == 1;
    bool kelvin_done = false;
    if (noise && p->pink_noise && p->pink_method == 1) {
        dim3 grid((unsigned)((T + 31) / 32), (unsigned)((p->tk.n_det + 31) / 32));
        p->tk.kelvin_ab = kelvin ? p->d_kelvin_abf.p : nullptr; kelvin_done = kelvin;
        gt::tk_add_kernel<<<grid, 256, 0, st>>>(p->tk, t0, T, dst);
        GT_CUDA(p, cudaGetLastError());
        p->launches += 1;
    } else if (noise && p->pink_noise) {
        const int64_t n_seg = (T + gt::kPinkSeg - 1) / gt::kPinkSeg;
        const int64_t n_thr = n_seg * p->pink.n_det;
        if ((size_t)(n_thr * p->J) > p->d_seg.n) GT_CUDA(p, p->d_seg.alloc((size_t)(n_thr * p->J)));
        p->pink.seg = p->d_seg.p;
        const int64_t n_dblk = (p->pink.n_det + 255) / 256;
        const size_t n_flags = (size_t)(n_seg * n_dblk) + 1;                 // + the ticket counter
        if (n_flags > p->d_pink_sync.n) GT_CUDA(p, p->d_pink_sync.alloc(n_flags));
        GT_CUDA(p, cudaMemsetAsync(p->d_pink_sync.p, 0, n_flags * sizeof(uint32_t), st));
        p->pink.flags = p->d_pink_sync.p + 1; p->pink.ticket = p->d_pink_sync.p;
        p->pink.kelvin_ab = kelvin ? p->d_kelvin_abf.p : nullptr; kelvin_done = kelvin;
        const size_t smem = (size_t)gt::kPinkSeg * 256 * sizeof(float);
        GT_CUDA(p, cudaFuncSetAttribute(gt::pink_chain_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        GT_CUDA(p, cudaFuncSetAttribute(gt::pink_chain_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        if (p->J <= 4) gt::pink_chain_kernel<4><<<(unsigned)(n_seg * n_dblk), 256, smem, st>>>(p->pink, t0, T, dst);
        else           gt::pink_chain_kernel<8><<<(unsigned)(n_seg * n_dblk), 256, smem, st>>>(p->pink, t0, T, dst);
        GT_CUDA(p, cudaGetLastError());
        p->launches += 1;
    }
    if (kelvin && !kelvin_done) {
        const int64_t n_span = (n_rows + gt::kKelvinRows - 1) / gt::kKelvinRows;
        gt::kelvin_kernel<<<(unsigned)std::min<int64_t>(n_span, 16 * p->num_sms), 256, 0, st>>>(dst, n_rows, p->n_chan, p->d_kelvin_abf.p);
        GT_CUDA(p, cudaGetLastError());
        p->launches += 1;
    }
    return GT_OK;
}

bool is_device_ptr(const void* ptr) {
    cudaPointerAttributes a{};
    if (cudaPointerGetAttributes(&a, ptr) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

gt_status simulate_impl(gt_plan* p, int64_t t_begin, int64_t t_count, float* out, float* pwv_out,
                        bool noise, cudaStream_t st) {
    if (!p) return fail(nullptr, GT_ERR_NULL, "plan is NULL");
    if (t_begin < 0 || t_count < 0 || t_begin + t_count > p->n_samples)
        return fail(p, GT_ERR_RANGE, "sample range [%lld, %lld) outside [0, %lld)", (long long)t_begin,
                    (long long)(t_begin + t_count), (long long)p->n_samples);
    if (t_count == 0) return GT_OK;
    if (!out) return fail(p, GT_ERR_NULL, "output pointer is NULL");
    {
        int dev = -1;
        GT_CUDA(p, cudaGetDevice(&dev));
        if (dev != p->device) return fail(p, GT_ERR_VALUE, "the plan lives on device %d, the current device is %d", p->device, dev);
    }
    p->last_stream = st;
    const bool pink = noise && p->pink_noise && p->pink_method == 0;      // the AR(1) cascade carries state between calls
    if (pink) {
        if (t_begin == 0) {
            gt::pink_init_kernel<<<(unsigned)((p->pink.n_det + 255) / 256), 256, 0, st>>>(p->pink);
            GT_CUDA(p, cudaGetLastError());
            p->launches++;
            p->pink_next_t = 0;
        } else if (t_begin != p->pink_next_t) {
            return fail(p, GT_ERR_VALUE, "pink noise is a recurrence: expected t_begin = %lld (or 0), got %lld",
                        (long long)p->pink_next_t, (long long)t_begin);
        }
    }
    p->n_fused_last = 0; p->n_tl_last = 0;
    const bool dev_out = is_device_ptr(out);
    const bool dev_pwv = pwv_out ? is_device_ptr(pwv_out) : true;
    if (pwv_out && dev_pwv != dev_out)
        return fail(p, GT_ERR_VALUE, "tod_out and pwv_out must be the same kind of memory");
    const int64_t chunk = dev_out ? p->chunk_dev : p->chunk_samples;
    const size_t row_floats = (size_t)p->n_spaxel * p->n_chan;
    int slot = 0, k = 0;
    for (int64_t t = t_begin; t < t_begin + t_count; t += chunk, ++k) {
        const int64_t T = std::min(chunk, t_begin + t_count - t);
        const size_t off = (size_t)(t - t_begin);
        if (dev_out) {
            gt_status s = run_chunk(p, t, T, out + off * row_floats, pwv_out ? pwv_out + off * p->n_spaxel : nullptr,
                                    noise, st, k);
            if (s != GT_OK) return s;
        } else {
            // double-buffered device chunk -> side-stream D2H, overlapped with the next chunk
            if (!p->d_chunk[slot].p) GT_CUDA(p, p->d_chunk[slot].alloc((size_t)chunk * row_floats));
            if (pwv_out && !p->d_pwv[slot].p) GT_CUDA(p, p->d_pwv[slot].alloc((size_t)chunk * p->n_spaxel));
            GT_CUDA(p, cudaStreamWaitEvent(st, p->ev_copied[slot], 0));      // buffer free again?
            while ((int)p->ev_tl.size() < 4 * (k + 1)) { cudaEvent_t e; GT_CUDA(p, cudaEventCreate(&e)); p->ev_tl.push_back(e); }
            GT_CUDA(p, cudaEventRecord(p->ev_tl[4 * k + 0], st));
            gt_status s = run_chunk(p, t, T, p->d_chunk[slot].p, pwv_out ? p->d_pwv[slot].p : nullptr, noise, st, k);
            if (s != GT_OK) return s;
            GT_CUDA(p, cudaEventRecord(p->ev_tl[4 * k + 1], st));
            GT_CUDA(p, cudaEventRecord(p->ev_ready[slot], st));
            GT_CUDA(p, cudaStreamWaitEvent(p->copy_stream, p->ev_ready[slot], 0));
            GT_CUDA(p, cudaEventRecord(p->ev_tl[4 * k + 2], p->copy_stream));
            GT_CUDA(p, cudaMemcpyAsync(out + off * row_floats, p->d_chunk[slot].p, (size_t)T * row_floats * sizeof(float),
                                       cudaMemcpyDeviceToHost, p->copy_stream));
            if (pwv_out)
                GT_CUDA(p, cudaMemcpyAsync(pwv_out + off * p->n_spaxel, p->d_pwv[slot].p,
                                           (size_t)T * p->n_spaxel * sizeof(float), cudaMemcpyDeviceToHost, p->copy_stream));
            GT_CUDA(p, cudaEventRecord(p->ev_tl[4 * k + 3], p->copy_stream));
            GT_CUDA(p, cudaEventRecord(p->ev_copied[slot], p->copy_stream));
            p->n_tl_last = k + 1;
            slot ^= 1;
        }
    }
    if (pink) p->pink_next_t = t_begin + t_count;
    if (!dev_out) GT_CUDA(p, cudaStreamSynchronize(p->copy_stream));
    return GT_OK;
}

}  // namespace

// =========================================================================================
extern "C" {

gt_status gt_plan_create(const gt_config* cfg, void* cuda_stream, gt_plan** out_plan) {
    if (!out_plan) return fail(nullptr, GT_ERR_NULL, "out_plan is NULL");
    *out_plan = nullptr;
    if (gt_status s = validate(cfg)) return s;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(nullptr, GT_ERR_CUDA, "no CUDA device: libgateau_b200 has no CPU fallback");
    }
    const gt_config& c = *cfg;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    gt_plan* p = new (std::nothrow) gt_plan();
    if (!p) return fail(nullptr, GT_ERR_OOM, "host allocation failed");
    struct Guard { gt_plan* p; ~Guard() { if (p) gt_plan_destroy(p); } } guard{p};
#define GT_CUDA0(expr)                                                                              \
    do { cudaError_t e_ = (expr);                                                                   \
         if (e_ != cudaSuccess) return fail(nullptr, e_ == cudaErrorMemoryAllocation ? GT_ERR_OOM : GT_ERR_CUDA, \
                                            "%s: %s", #expr, cudaGetErrorString(e_)); } while (0)
    {
        // single attributes, not cudaGetDeviceProperties: that call fills every field through the driver and was measured
        // at ~2 ms per plan normally and, intermittently, at 14 ms and more (outliers of 50-100 ms in the end-to-end leg)
        int dev = 0, sms = 0, major = 0, minor = 0;
        GT_CUDA0(cudaGetDevice(&dev));
        GT_CUDA0(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        GT_CUDA0(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        GT_CUDA0(cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev));
        p->device = dev;
        p->num_sms = sms;
        if (major != 10) return fail(nullptr, GT_ERR_UNSUPPORTED, "built for sm_100a, device is sm_%d%d", major, minor);
    }
    GT_CUDA0(cudaStreamSynchronize(st));
    gt::tc_alloc_fn() = pool_alloc_raw; gt::tc_free_fn() = pool_free_raw;

    const int nf = c.n_freq, nc = c.n_chan, ns = c.n_spaxel;
    const int nfp = (nf + 63) / 64 * 64;      // the tensor kernel works in slabs of 64 frequencies
    p->n_freq = nf; p->n_freq_pad = nfp; p->n_chan = nc; p->n_spaxel = ns; p->n_pwv = c.n_pwv;
    p->n_samples = c.n_samples; p->photon_noise = c.photon_noise != 0; p->pink_noise = c.pink_noise != 0;
    p->seed = c.seed; p->cube = c.cube; p->n_az = c.n_az; p->n_el = c.n_el; p->spaxel_base = c.spaxel_index_base;
    p->tc_full = c.variant == GT_VARIANT_TENSOR_FULL;
    p->variant = (c.variant == GT_VARIANT_FP32) ? GT_VARIANT_FP32 : GT_VARIANT_TENSOR;   // DEFAULT -> tensor: measured 8x faster than the FP32 kernel on C4

    // ---- statistics of the large device arrays: non-finite values are refused, the cube's per-frequency maximum
    //      bounds the spectrum elements (operand range of the tensor kernel), the means feed the reference spectrum ----
    std::vector<float> cube_max(nf, 0.f), cube_lo(nf, 0.f), cube_hi(nf, 0.f);     // |.| maximum; signed range including 0 (outside the cube)
    std::vector<double> cube_mean(nf, 0.0);
    double screen_mean = 0.0, screen_lo = 0.0, screen_hi = 0.0;
    {
        const int64_t n_pix = c.cube ? (int64_t)c.n_az * c.n_el : 0;
        DevBuf<uint32_t> d_max; DevBuf<double> d_sum;
        const size_t n_stat = (size_t)nf + (size_t)c.nx;
        GT_CUDA0(d_max.alloc(3 * n_stat)); GT_CUDA0(d_sum.alloc(n_stat));           // |.| max bits, min keys, max keys
        GT_CUDA0(cudaMemsetAsync(d_max.p, 0, n_stat * sizeof(uint32_t), st));
        GT_CUDA0(cudaMemsetAsync(d_max.p + n_stat, 0xFF, n_stat * sizeof(uint32_t), st));
        GT_CUDA0(cudaMemsetAsync(d_max.p + 2 * n_stat, 0, n_stat * sizeof(uint32_t), st));
        GT_CUDA0(cudaMemsetAsync(d_sum.p, 0, n_stat * sizeof(double), st));
        if (c.cube) {
            const unsigned gy = (unsigned)std::min<int64_t>(n_pix, std::max<int64_t>(1, (8 * p->num_sms) / ((nf + 255) / 256)));
            gt::colstat_kernel<<<dim3((unsigned)((nf + 255) / 256), gy), 256, 0, st>>>(c.cube, n_pix, nf, d_max.p, d_sum.p,
                                                                                      d_max.p + n_stat, d_max.p + 2 * n_stat);
            GT_CUDA0(cudaGetLastError());
        }
        {
            const unsigned gy = (unsigned)std::min<int64_t>(c.ny, std::max<int64_t>(1, (8 * p->num_sms) / ((c.nx + 255) / 256)));
            gt::colstat_kernel<<<dim3((unsigned)((c.nx + 255) / 256), gy), 256, 0, st>>>(c.screen, c.ny, c.nx, d_max.p + nf, d_sum.p + nf,
                                                                                        d_max.p + n_stat + nf, d_max.p + 2 * n_stat + nf);
            GT_CUDA0(cudaGetLastError());
        }
        p->launches += c.cube ? 2 : 1;
        std::vector<uint32_t> h_max(3 * n_stat); std::vector<double> h_sum(n_stat);
        GT_CUDA0(cudaMemcpyAsync(h_max.data(), d_max.p, 3 * n_stat * sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
        GT_CUDA0(cudaMemcpyAsync(h_sum.data(), d_sum.p, n_stat * sizeof(double), cudaMemcpyDeviceToHost, st));
        GT_CUDA0(cudaStreamSynchronize(st));
        for (int i = 0; i < nf; ++i) {
            if (h_max[i] >= 0x7F800000u) return fail(nullptr, GT_ERR_VALUE, "the source cube holds a NaN or Inf (frequency index %d)", i);
            std::memcpy(&cube_max[i], &h_max[i], sizeof(float));
            cube_mean[i] = n_pix ? h_sum[i] / (double)n_pix : 0.0;
            if (n_pix) {
                cube_lo[i] = std::min(0.f, gt::key_float(h_max[n_stat + i]));
                cube_hi[i] = std::max(0.f, gt::key_float(h_max[2 * n_stat + i]));
            }
        }
        for (int i = 0; i < c.nx; ++i) {
            if (h_max[nf + i] >= 0x7F800000u) return fail(nullptr, GT_ERR_VALUE, "the PWV screen holds a NaN or Inf (column %d)", i);
            screen_mean += h_sum[nf + i];
            const double lo = gt::key_float(h_max[n_stat + nf + i]), hi = gt::key_float(h_max[2 * n_stat + nf + i]);
            screen_lo = i ? std::min(screen_lo, lo) : lo; screen_hi = i ? std::max(screen_hi, hi) : hi;
        }
        screen_mean /= (double)c.nx * (double)c.ny;
    }

    // ---- small device arrays needed on the host ----
    std::vector<float> h_lut, h_filt, h_front;
    if (gt_status s = fetch(c.atm_lut, (size_t)c.n_pwv * c.n_nu_lut, h_lut, "atm_lut")) return s;
    if (gt_status s = fetch(c.filt, (size_t)nc * nf, h_filt, "filt")) return s;
    if (c.eta_front_nu) if (gt_status s = fetch(c.eta_front_nu, nf, h_front, "eta_front_nu")) return s;
    std::vector<std::vector<float>> h_stage(c.n_stage);
    for (int k = 0; k < c.n_stage; ++k)
        if (c.stages[k].eta_nu) if (gt_status s = fetch(c.stages[k].eta_nu, nf, h_stage[k], "stage eta_nu")) return s;
    for (float v : h_front) if (!(v >= 0.f && v <= 1.f)) return fail(nullptr, GT_ERR_VALUE, "eta_front_nu outside [0,1]");
    for (auto& hs : h_stage) for (float v : hs) if (!(v >= 0.f && v <= 1.f)) return fail(nullptr, GT_ERR_VALUE, "stage eta_nu outside [0,1]");
    for (float v : h_lut) if (!(v > 0.f && v <= 1.f)) return fail(nullptr, GT_ERR_VALUE, "atm_lut outside (0,1]");
    for (float v : h_filt) if (!std::isfinite(v)) return fail(nullptr, GT_ERR_VALUE, "filt holds a NaN or Inf");

    // ---- collapsed cascade, double precision ----
    // P_final(nu) = eta_atm * (b1 + a*S) + b0 after Eq. 11 and Eq. 12 for k = 0..n_stage:
    //   after the atmosphere:  a = eta_front, b1 = B_cmb - B_atm, b0 = B_atm
    //   plain stage k:         a *= eta_k; b1 *= eta_k; b0 = eta_k b0 + (1-eta_k) B(T_k)
    //   coupled stage k:       a *= eta_k; b1 = eta_k b1 + (1-eta_k)(B_cmb - B_atm); b0 = eta_k b0 + (1-eta_k) B_atm
    // With eps = 1 - eta_atm:  P_final = eps*(-b1) + eta_atm*(a*S) + (b0 + b1);  all three terms >= 0.
    std::vector<double> Y(nf), Xd(nf), Gd(nf);
    double v_max = 0.0;                        // largest |element| the generator can produce, in W/Hz
    for (int i = 0; i < nf; ++i) {
        const double nu = c.nu0_hz + (double)i * c.dnu_hz;
        const double Bc = jn_power(nu, c.T_cmb_K), Ba = jn_power(nu, c.T_atm_K);
        double a = c.eta_front_nu ? (double)h_front[i] : 1.0, b1 = Bc - Ba, b0 = Ba;
        for (int k = 0; k < c.n_stage; ++k) {
            const gt_stage& s = c.stages[k];
            const double e = s.eta_nu ? (double)h_stage[k][i] : s.eta_scalar;
            a *= e;
            if (s.couple_atmosphere) { b1 = e * b1 + (1.0 - e) * (Bc - Ba); b0 = e * b0 + (1.0 - e) * Ba; }
            else                     { b1 = e * b1;                         b0 = e * b0 + (1.0 - e) * jn_power(nu, s.T_K); }
        }
        Xd[i] = -b1; Gd[i] = a; Y[i] = b0 + b1;
        // an element is the convex combination (1 - eta) Xn + eta G S of its two end points, eta in [0,1]
        v_max = std::max(v_max, std::max(std::fabs(b1), a * (double)cube_max[i]));
    }
    if (!std::isfinite(v_max)) return fail(nullptr, GT_ERR_RANGE, "the spectrum is not finite (stage temperatures, source cube)");
    {
        // p_ref = k_B 300 K 2^-e with v_max / p_ref in [2^(kTcAMaxLog2 - 1), 2^kTcAMaxLog2): exact power of two on top of
        // k_B 300 K, so the fp16 (hi, lo) pairs of the elements keep 22 bits down to ~1e-4 of the largest one
        int e = 8;
        if (v_max > 0.0) { int x; std::frexp(v_max / kPref0, &x); e = gt::kTcAMaxLog2 - x; }
        e = std::max(-900, std::min(900, e));
        p->p_ref = std::ldexp(kPref0, -e);
        const double s = p->p_ref * c.dnu_hz;
        if (!(s > 1e-37) || !(s < 1e37) || !(1.0 / p->p_ref < 1e37))
            return fail(nullptr, GT_ERR_RANGE, "spectrum of at most %g W/Hz cannot be scaled into the fp32 range of the kernels", v_max);
        p->scale = (float)s;
    }
    const double kPref = p->p_ref;
    std::vector<float> Xn(nfp, 0.f), Gs(nfp, 0.f);
    for (int i = 0; i < nf; ++i) { Xn[i] = (float)(Xd[i] / kPref); Gs[i] = (float)(Gd[i] / kPref); }

    // ---- LUT resampled on the frequency grid (bilinear is separable, R14) ----
    std::vector<float> lut_r((size_t)c.n_pwv * nfp, 1.0f);
    for (int i = 0; i < nf; ++i) {
        const double nu = c.nu0_hz + (double)i * c.dnu_hz;
        const double r = (nu - c.lut_nu0_hz) / c.lut_dnu_hz;
        long ir = (long)std::floor(r);
        if (ir > c.n_nu_lut - 2) ir = c.n_nu_lut - 2;
        if (ir < 0) ir = 0;
        const double fr = r - (double)ir;
        for (int q = 0; q < c.n_pwv; ++q) {
            const double L0 = h_lut[(size_t)q * c.n_nu_lut + ir], L1 = h_lut[(size_t)q * c.n_nu_lut + ir + 1];
            lut_r[(size_t)q * nfp + i] = (float)((1.0 - fr) * L0 + fr * L1);
        }
    }

    // ---- reference spectrum (any positive multiple): the mean line of sight -- screen mean + drift at mid-run, boresight
    //      airmass, mean cube spectrum.  Used only to shape the truncation-compensation table of the tensor kernel. ----
    std::vector<double> a_ref(nf, 1.0);
    {
        const double pwv = screen_mean + c.pwv0_a_mm + c.pwv0_b_mm_per_s * 0.5 * (double)c.n_samples / c.f_sample_hz;
        double q = (pwv - c.lut_pwv0_mm) / c.lut_dpwv_mm;
        if (!(q >= 0.0)) q = 0.0;
        if (q > (double)(c.n_pwv - 1)) q = (double)(c.n_pwv - 1);
        const int ip = (int)std::min<double>(std::floor(q), c.n_pwv - 2);
        const double fpq = q - ip, csc0 = 1.0 / std::max(std::sin(c.el0_rad), 1e-3);
        double top = 0.0;
        for (int i = 0; i < nf; ++i) {
            const double ez = (1.0 - fpq) * lut_r[(size_t)ip * nfp + i] + fpq * lut_r[(size_t)(ip + 1) * nfp + i];
            const double eta = std::pow(ez, csc0);
            a_ref[i] = (1.0 - eta) * Xd[i] + eta * Gd[i] * cube_mean[i];
            top = std::max(top, std::fabs(a_ref[i]));
        }
        bool ok = top > 0.0;
        for (int i = 0; i < nf && ok; ++i) ok = a_ref[i] >= 0.0 && std::isfinite(a_ref[i]);
        if (!ok) std::fill(a_ref.begin(), a_ref.end(), 1.0);              // no usable reference: flat
        else for (double& v : a_ref) v = v / top + 1e-6;                  // keeps channels in fully transparent bands alive
    }

    // ---- filter: transposed/padded copy (FP32 variant), per-channel constants ----
    const int tn = fp32_tn(nc);
    const int ncp = ((nc + 32 * tn - 1) / (32 * tn)) * 32 * tn;
    p->n_chan_pad = ncp;
    std::vector<float> bias(ncp, 0.f), c1(ncp, 0.f), c2(ncp, 0.f), cw(ncp, 1.f);
    {
        std::atomic<int> bad_ch{-1};
        gt::host_parallel_for(nc, [&](int64_t ch) {
            double sb = 0.0, s1 = 0.0, s2 = 0.0;
            for (int i = 0; i < nf; ++i) {
                const double f = h_filt[(size_t)ch * nf + i];
                sb += f * Y[i]; s1 += f * c.dnu_hz; s2 += f * f * c.dnu_hz;
            }
            bias[ch] = (float)(c.dnu_hz * sb);
            const double dnu_c = c.dnu_eff_hz ? c.dnu_eff_hz[ch] : (s2 > 0 ? s1 * s1 / s2 : 1.0);
            if (!(dnu_c > 0)) { bad_ch = (int)ch; return; }
            c1[ch] = (float)(kH * c.f_center_hz[ch] * c.f_sample_hz);
            c2[ch] = (float)(c.f_sample_hz / dnu_c);
        });
        if (bad_ch >= 0) return fail(nullptr, GT_ERR_VALUE, "dnu_eff[%d] is not positive", (int)bad_ch);
    }
    if (p->variant == GT_VARIANT_FP32) {
        std::vector<float> ft((size_t)nfp * ncp, 0.f);
        for (int ch = 0; ch < nc; ++ch)
            for (int i = 0; i < nf; ++i) ft[(size_t)i * ncp + ch] = h_filt[(size_t)ch * nf + i];
        GT_CUDA0(p->d_filt_t.upload(ft, st));
        GT_CUDA0(cudaStreamSynchronize(st));
    } else {
#ifdef GT_TC_DIAG
        if (const char* e = std::getenv("GATEAU_TC_SEG")) {          // tuning builds only: slabs per accumulation segment
            const int v = std::atoi(e);
            if (v > 0) p->tc.seg = v;
        }
#endif
        std::vector<float> inv;
        // banded corrections: the range of the elements the generator can produce, per frequency (scaled units), and what
        // every channel's power holds at least.  An element is (1 - eta) Xn + eta G S:
        //   eta = eta_z(nu, PWV)^csc; PWV lies between pwv0(t) + the screen's minimum and maximum, so eta_z (bilinear in PWV:
        //   a convex combination of two adjacent table rows) lies between the smallest and the largest entry of the table
        //   rows that range touches; csc lies between its values at the lowest and highest elevation of the scan;
        //   S (bilinear in the cube, zero outside) lies between the cube's minimum and maximum at that frequency, and 0.
        // The expression is bilinear in (eta, S): its extremes are at the corners of that box.  1e-3 of margin covers the
        // kernel's fp32 arithmetic (MUFU ex2 / lg2: ~1e-6).
        std::vector<double> v_hi(nf), v_lo(nf), floor_c(nc);
        {
            const double t_end = (double)(c.n_samples - 1) / c.f_sample_hz;
            const double p0 = c.pwv0_a_mm, p1 = c.pwv0_a_mm + c.pwv0_b_mm_per_s * t_end;
            auto row_of = [&](double pwv) {
                double q = (pwv - c.lut_pwv0_mm) / c.lut_dpwv_mm;
                if (!(q >= 0.0)) q = 0.0;
                if (q > (double)(c.n_pwv - 1)) q = (double)(c.n_pwv - 1);
                return q;
            };
            const int r0 = (int)std::floor(row_of(std::min(p0, p1) + screen_lo));
            const int r1 = std::min(c.n_pwv - 1, (int)std::floor(row_of(std::max(p0, p1) + screen_hi)) + 1);
            double e_lo = 1e300, e_hi = -1e300, d_lo = 1e300, d_hi = -1e300;
            for (int64_t n = 0; n < c.n_samples; ++n) { e_lo = std::min(e_lo, c.el_rad[n]); e_hi = std::max(e_hi, c.el_rad[n]); }
            for (int sidx = 0; sidx < ns; ++sidx) { d_lo = std::min(d_lo, c.del_rad[sidx]); d_hi = std::max(d_hi, c.del_rad[sidx]); }
            const double E_lo = c.el0_rad + e_lo + d_lo, E_hi = c.el0_rad + e_hi + d_hi;
            const bool el_ok = E_lo > 1e-3 && E_hi < kPi - 1e-3;
            // csc is unimodal on (0, pi) with its minimum 1 at pi/2
            const double csc_hi = el_ok ? std::max(1.0 / std::sin(E_lo), 1.0 / std::sin(E_hi)) * (1.0 + 1e-6) : 0.0;
            const double csc_lo = el_ok ? ((E_lo <= 0.5 * kPi && E_hi >= 0.5 * kPi) ? 1.0 : std::min(1.0 / std::sin(E_lo), 1.0 / std::sin(E_hi)) * (1.0 - 1e-6)) : 1.0;
            for (int i = 0; i < nf; ++i) {
                float z_lo = 1.f, z_hi = 0.f;
                for (int q = r0; q <= r1; ++q) { z_lo = std::min(z_lo, lut_r[(size_t)q * nfp + i]); z_hi = std::max(z_hi, lut_r[(size_t)q * nfp + i]); }
                const double eta_hi = std::pow((double)z_hi, csc_lo), eta_lo = el_ok ? std::pow((double)z_lo, csc_hi) : 0.0;
                const double x = Xd[i], gs_lo = Gd[i] * (double)(Gd[i] >= 0 ? cube_lo[i] : cube_hi[i]), gs_hi = Gd[i] * (double)(Gd[i] >= 0 ? cube_hi[i] : cube_lo[i]);
                double hi = -1e300, lo = 1e300;
                for (double eta : {eta_lo, eta_hi})
                    for (double gs : {gs_lo, gs_hi}) { const double v = (1.0 - eta) * x + eta * gs; hi = std::max(hi, v); lo = std::min(lo, v); }
                const double pad = 1e-3 * std::max(std::fabs(hi), std::fabs(lo));
                v_hi[i] = (hi + pad) / kPref;
                v_lo[i] = (lo - pad) / kPref;
            }
        }
        for (int ch = 0; ch < nc; ++ch) floor_c[ch] = std::max(0.0, (double)bias[ch] / (double)p->scale);
        const gt::TcSkipBounds sb{&v_lo, &v_hi, &floor_c};            // {v_min, v_max, floor}
        if (gt_status s = gt::build_tc_tables(h_filt, nc, nf, nfp, a_ref, p->tc, inv, st, nullptr, c.variant == GT_VARIANT_TENSOR_FULL ? nullptr : &sb)) {
            return fail(nullptr, s, "tensor variant: %s", gt::tc_error());
        }
        for (int ch = 0; ch < nc; ++ch) cw[ch] = inv[ch];            // channel ch = column ch % nb_tot of channel group ch / nb_tot
        if (gt_status s = gt::alloc_tc_scratch(p->tc, p->num_sms)) return fail(nullptr, s, "tensor variant: %s", gt::tc_error());
        if (c.photon_noise && c.photon_mode == 1) {
            // Eq. 17 with P_nu = kPref v + Y (v = the generated element):
            //   NEP^2 / (2 dnu) = sum Fm (h nu + g) P + sum Fm^2 P^2
            //                   = kPref sum [Fm (h nu + g) + 2 Fm^2 Y] v + kPref^2 sum Fm^2 v^2 + sum [Fm (h nu + g) Y + Fm^2 Y^2]
            // divided by E0 = h nu_max + g (so that it is O(P_KID)):  kPref dnu [sum L v + sum Q' (v^2 / 256)] + const,
            //   L = (Fm (h nu + g) + 2 Fm^2 Y) / E0,   Q' = Fm^2 256 kPref / E0
            const double g = 2.0 * c.kid_gap_J / c.eta_pb;
            const double E0 = kH * (c.nu0_hz + (double)(nf - 1) * c.dnu_hz) + g;
            std::vector<float> L((size_t)nc * nf), Q((size_t)nc * nf);
            std::vector<float4> c4n(ncp, make_float4(0.f, 0.f, 0.f, 1.f));
            for (int ch = 0; ch < nc; ++ch) {
                double sb = 0.0;
                for (int i = 0; i < nf; ++i) {
                    const double f = h_filt[(size_t)ch * nf + i], e = kH * (c.nu0_hz + (double)i * c.dnu_hz) + g;
                    L[(size_t)ch * nf + i] = (float)((f * e + 2.0 * f * f * Y[i]) / E0);
                    Q[(size_t)ch * nf + i] = (float)(f * f * kPref / ((double)gt::kTcSqScale * E0));
                    sb += f * e * Y[i] + f * f * Y[i] * Y[i];
                }
                c4n[ch].x = (float)(c.dnu_hz * sb / E0);
            }
            std::vector<float> inv_n;
            if (gt_status s = gt::build_tc_tables(L, nc, nf, nfp, a_ref, p->tc_nep, inv_n, st, &Q)) return fail(nullptr, s, "tensor variant (Eq. 17 filters): %s", gt::tc_error());
            for (int ch = 0; ch < nc; ++ch) c4n[ch].w = inv_n[ch];
            GT_CUDA0(p->d_chan4_nep.upload(c4n, st));
            GT_CUDA0(cudaStreamSynchronize(st));
            p->sqrt_e0 = (float)std::sqrt(E0);
            p->f_sample = (float)c.f_sample_hz;
        }
    }
    GT_CUDA0(p->d_Xn.upload(Xn, st)); GT_CUDA0(p->d_Gs.upload(Gs, st)); GT_CUDA0(p->d_lut_r.upload(lut_r, st));
    GT_CUDA0(p->d_bias.upload(bias, st)); GT_CUDA0(p->d_c1.upload(c1, st)); GT_CUDA0(p->d_c2.upload(c2, st));
    {
        std::vector<float4> c4(ncp);
        for (int ch = 0; ch < ncp; ++ch) c4[ch] = make_float4(bias[ch], c1[ch], c2[ch], cw[ch]);
        GT_CUDA0(p->d_chan4.upload(c4, st));
        GT_CUDA0(cudaStreamSynchronize(st));
    }
    p->h_lut = h_lut; p->n_nu_lut = c.n_nu_lut; p->lut_nu0 = c.lut_nu0_hz; p->lut_dnu = c.lut_dnu_hz;
    p->lut_pwv0 = c.lut_pwv0_mm; p->lut_dpwv = c.lut_dpwv_mm;
    p->h_daz.assign(c.daz_rad, c.daz_rad + ns); p->h_del.assign(c.del_rad, c.del_rad + ns);
    p->h_fc.assign(c.f_center_hz, c.f_center_hz + nc);
    GT_CUDA0(p->d_ln_eta_z.alloc((size_t)4 * nc)); GT_CUDA0(p->d_cm_weight.alloc((size_t)ns));
    { const double s0 = std::sin(c.el0_rad); p->cm_csc0 = s0 > 1e-3 ? 1.0 / s0 : 1.0; }
    GT_CUDA0(cm_static_resolve(p->device));     // device address of the static scratch of gt_common_mode_static
    GT_CUDA0(p->d_counters.alloc(3));
    GT_CUDA0(cudaMemsetAsync(p->d_counters.p, 0, 3 * sizeof(unsigned long long), st));

    // ---- geometry tables: per-sample and per-spaxel transcendental inputs from the host libm ----
    {
        const int64_t nt = c.n_samples;
        std::vector<double> ta(nt), te(nt), sE(nt), cE(nt), az(c.az_rad, c.az_rad + nt), el(c.el_rad, c.el_rad + nt);
        gt::host_parallel_for(nt, [&](int64_t n) {
            ta[n] = std::tan(c.az_rad[n]); te[n] = std::tan(c.el_rad[n]);
            const double E = c.el0_rad + c.el_rad[n];
            sE[n] = std::sin(E); cE[n] = std::cos(E);
        });
        GT_CUDA0(p->d_tan_az.upload(ta, st)); GT_CUDA0(p->d_tan_el.upload(te, st));
        GT_CUDA0(p->d_sinE.upload(sE, st)); GT_CUDA0(p->d_cosE.upload(cE, st));
        GT_CUDA0(p->d_az.upload(az, st)); GT_CUDA0(p->d_el.upload(el, st));
        std::vector<double> sp((size_t)6 * ns);
        for (int s = 0; s < ns; ++s) {
            sp[0 * ns + s] = std::tan(c.daz_rad[s]); sp[1 * ns + s] = std::tan(c.del_rad[s]);
            sp[2 * ns + s] = std::sin(c.del_rad[s]); sp[3 * ns + s] = std::cos(c.del_rad[s]);
            sp[4 * ns + s] = c.daz_rad[s];           sp[5 * ns + s] = c.del_rad[s];
        }
        GT_CUDA0(p->d_sp.upload(sp, st));
        GT_CUDA0(cudaStreamSynchronize(st));       // host vectors go out of scope
        gt::GeoParams& g = p->geo;
        g.tan_az = p->d_tan_az.p; g.tan_el = p->d_tan_el.p; g.sinE = p->d_sinE.p; g.cosE = p->d_cosE.p;
        g.az = p->d_az.p; g.el = p->d_el.p;
        g.tan_daz = p->d_sp.p; g.tan_del = p->d_sp.p + ns; g.sin_del = p->d_sp.p + 2 * ns;
        g.cos_del = p->d_sp.p + 3 * ns; g.daz = p->d_sp.p + 4 * ns; g.del = p->d_sp.p + 5 * ns;
        g.n_spaxel = ns; g.f_sample = c.f_sample_hz;
        g.screen = c.screen; g.nx = c.nx; g.ny = c.ny; g.dx = c.dx_m; g.dy = c.dy_m;
        g.h_col = c.h_column_m; g.wind = c.wind_mps; g.pwv0_a = c.pwv0_a_mm; g.pwv0_b = c.pwv0_b_mm_per_s;
        g.n_pwv = c.n_pwv; g.lut_pwv0 = c.lut_pwv0_mm; g.lut_dpwv = c.lut_dpwv_mm;
        g.has_cube = c.cube != nullptr; g.n_az = c.n_az; g.n_el = c.n_el;
        g.az_min = c.az_min_rad; g.daz_grid = c.daz_grid_rad; g.el_min = c.el_min_rad; g.del_grid = c.del_grid_rad;
    }

    // ---- brightness-temperature output: the skydip and its linear map (R22) ----
    p->output_unit = c.output_unit;
    p->photon_mode = c.photon_mode;
    if (c.output_unit == 1) {
        const int K = c.skydip_n;
        DevBuf<double> d_Xd, d_Yd, d_P, d_T; DevBuf<int32_t> d_bad;
        GT_CUDA0(d_Xd.upload(Xd, st)); GT_CUDA0(d_Yd.upload(Y, st));
        GT_CUDA0(d_P.alloc((size_t)K * nc)); GT_CUDA0(d_T.alloc((size_t)K * nc)); GT_CUDA0(d_bad.alloc(1));
        GT_CUDA0(p->d_kelvin_ab.alloc((size_t)2 * nc)); GT_CUDA0(p->d_kelvin_abf.alloc((size_t)nc));
        GT_CUDA0(cudaMemsetAsync(d_bad.p, 0, sizeof(int32_t), st));
        gt::SkydipParams k{};
        k.n_chan = nc; k.n_freq = nf; k.n_freq_pad = nfp; k.n_pwv = c.n_pwv; k.K = K;
        k.dnu = c.dnu_hz; k.lut_pwv0 = c.lut_pwv0_mm; k.lut_dpwv = c.lut_dpwv_mm;
        k.pwv_lo = c.skydip_pwv_lo_mm; k.pwv_step = (c.skydip_pwv_hi_mm - c.skydip_pwv_lo_mm) / (double)(K - 1);
        k.csc0 = 1.0 / std::sin(c.el0_rad); k.T_atm = c.T_atm_K; k.T_cmb = c.T_cmb_K;
        k.lut_r = p->d_lut_r.p; k.filt = c.filt; k.Xd = d_Xd.p; k.Yd = d_Yd.p; k.P = d_P.p; k.T = d_T.p;
        k.ab = p->d_kelvin_ab.p; k.abf = p->d_kelvin_abf.p; k.bad = d_bad.p;
        gt::skydip_kernel<<<dim3((unsigned)nc, (unsigned)K), 256, 0, st>>>(k);
        GT_CUDA0(cudaGetLastError());
        gt::skydip_fit_kernel<<<(unsigned)((nc + 127) / 128), 128, 0, st>>>(k);
        GT_CUDA0(cudaGetLastError());
        int32_t bad = 0;
        GT_CUDA0(cudaMemcpyAsync(&bad, d_bad.p, sizeof(bad), cudaMemcpyDeviceToHost, st));
        GT_CUDA0(cudaStreamSynchronize(st));
        p->launches += 2;
        if (bad) return fail(nullptr, GT_ERR_VALUE, "skydip: channel %d cannot be calibrated (its filter sums to zero or its power does not vary with PWV)", bad - 1);
    }

    p->pink_method = c.pink_method;
    // ---- Timmer & Koenig pink noise (R21): the series of every detector, once ----
    if (p->pink_noise && p->pink_method == 1) {
        const int64_t N = c.n_samples, K = N / 2, n_det = (int64_t)ns * nc, ld = 2 * (K + 1);
        std::vector<float> amp((size_t)n_det), halpha((size_t)n_det);
        for (int64_t d = 0; d < n_det; ++d) {
            if (!(c.pink_A[d] >= 0) || !(c.pink_alpha[d] >= 0))
                return fail(nullptr, GT_ERR_VALUE, "pink noise level of detector %lld is invalid", (long long)d);
            amp[d] = (float)std::sqrt(c.pink_A[d] * c.f_sample_hz / (4.0 * (double)N));
            halpha[d] = (float)(0.5 * c.pink_alpha[d]);
        }
        GT_CUDA0(p->d_tk_amp.upload(amp, st)); GT_CUDA0(p->d_tk_halpha.upload(halpha, st));
        GT_CUDA0(p->d_tk_series.alloc((size_t)(n_det * ld)));
        gt::TkParams& k = p->tk;
        k.n_det = n_det; k.n_samples = N; k.n_chan = nc; k.f_sample = c.f_sample_hz;
        k.amp = p->d_tk_amp.p; k.half_alpha = p->d_tk_halpha.p; k.series = p->d_tk_series.p; k.ld = ld;
        k.seed_lo = (uint32_t)(c.seed & 0xffffffffu); k.seed_hi = (uint32_t)(c.seed >> 32);
        k.spaxel_base = (uint32_t)c.spaxel_index_base;
        const int64_t n_thr = n_det * (K + 1);
        gt::tk_spectrum_kernel<<<(unsigned)((n_thr + 255) / 256), 256, 0, st>>>(k);
        GT_CUDA0(cudaGetLastError());
        p->launches++;
        if (N >= 2) {
            cufftHandle h;
            int n[1] = {(int)N}, inembed[1] = {(int)(K + 1)}, onembed[1] = {(int)ld};
            if (N > 0x7fffffffLL) return fail(nullptr, GT_ERR_SHAPE, "n_samples too large for the FFT");
            if (cufftPlanMany(&h, 1, n, inembed, 1, (int)(K + 1), onembed, 1, (int)ld, CUFFT_C2R, (int)n_det) != CUFFT_SUCCESS)
                return fail(nullptr, GT_ERR_OOM, "cufftPlanMany failed (length %lld, batch %lld)", (long long)N, (long long)n_det);
            cufftResult r = cufftSetStream(h, st);
            if (r == CUFFT_SUCCESS)
                r = cufftExecC2R(h, reinterpret_cast<cufftComplex*>(p->d_tk_series.p), p->d_tk_series.p);   // in place
            cudaError_t e = cudaStreamSynchronize(st);
            cufftDestroy(h);
            if (r != CUFFT_SUCCESS || e != cudaSuccess) return fail(nullptr, GT_ERR_CUDA, "inverse FFT of the pink-noise spectra failed");
        }
        GT_CUDA0(cudaStreamSynchronize(st));       // amp / halpha host vectors go out of scope
    }

    // ---- pink-noise coefficients of the AR(1) cascade (R18) ----
    if (p->pink_noise && p->pink_method == 0) {
        const int J = c.pink_n_stage;
        p->J = J;
        gt::PinkParams& k = p->pink;
        k.J = J; k.n_chan = nc; k.n_det = (int64_t)ns * nc;
        k.seed_lo = (uint32_t)(c.seed & 0xffffffffu); k.seed_hi = (uint32_t)(c.seed >> 32);
        k.spaxel_base = (uint32_t)c.spaxel_index_base;
        double lnrho = 1.0;
        if (J >= 2) lnrho = std::log(c.pink_f_corner_hz[0] / c.pink_f_corner_hz[J - 1]) / (double)(J - 1);
        for (int j = 0; j < gt::kPinkMaxJ; ++j) { k.phi[j] = 0.f; k.sq[j] = 0.f; }
        for (int j = 0; j < J; ++j) {
            if (!(c.pink_f_corner_hz[j] > 0)) return fail(nullptr, GT_ERR_VALUE, "pink corner frequency must be positive");
            const double phi = std::exp(-2.0 * kPi * c.pink_f_corner_hz[j] / c.f_sample_hz);
            k.phi[j] = (float)phi; k.sq[j] = (float)std::sqrt(1.0 - phi * phi);
        }
        std::vector<float> gain((size_t)k.n_det * J);
        for (int64_t d = 0; d < k.n_det; ++d)
            for (int j = 0; j < J; ++j) {
                const double A = c.pink_A[d], al = c.pink_alpha[d], fj = c.pink_f_corner_hz[j];
                const double g2 = A * lnrho * std::sin(kPi * al / 2.0) * std::pow(fj, 1.0 - al);
                if (!(g2 >= 0)) return fail(nullptr, GT_ERR_VALUE, "pink noise level of detector %lld is invalid", (long long)d);
                gain[(size_t)d * J + j] = (float)std::sqrt(g2);
            }
        GT_CUDA0(p->d_gain.upload(gain, st));
        GT_CUDA0(p->d_state.alloc((size_t)k.n_det * J));
        GT_CUDA0(cudaStreamSynchronize(st));
        k.gain = p->d_gain.p; k.state = p->d_state.p; k.seg = nullptr;
    }

    // ---- chunking and streams ----
    {
        const double bytes_per_sample = (double)ns * nc * sizeof(float);
        int64_t chunk = c.chunk_samples > 0 ? c.chunk_samples
                                            : (int64_t)std::max(1.0, std::floor(512.0 * 1048576.0 / bytes_per_sample));
        chunk = std::min(chunk, c.n_samples);
        if (c.chunk_samples == 0 && chunk > gt::kPinkSeg) chunk = chunk / gt::kPinkSeg * gt::kPinkSeg;
        p->chunk_samples = chunk;
        // device output needs no staging buffers: larger launches (about 2^22 rows, 134 MB of RowParam) keep the persistent
        // kernel's tail (the last partial wave of tiles, and the cluster barrier the pairs end on) below half a per cent
        int64_t chunk_dev = chunk;
        if (c.chunk_samples == 0) {
            chunk_dev = std::max<int64_t>(chunk, std::min<int64_t>(c.n_samples, (1 << 22) / std::max(ns, 1)));
            if (chunk_dev > gt::kPinkSeg) chunk_dev = chunk_dev / gt::kPinkSeg * gt::kPinkSeg;
        }
        p->chunk_dev = chunk_dev;
        GT_CUDA0(p->d_rows.alloc((size_t)std::max(chunk, chunk_dev) * ns));
        GT_CUDA0(cudaStreamCreateWithFlags(&p->copy_stream, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            GT_CUDA0(cudaEventCreateWithFlags(&p->ev_ready[i], cudaEventDisableTiming));
            GT_CUDA0(cudaEventCreateWithFlags(&p->ev_copied[i], cudaEventDisableTiming));
        }
    }
    GT_CUDA0(cudaStreamSynchronize(st));
    guard.p = nullptr;
    *out_plan = p;
    return GT_OK;
}

gt_status gt_simulate(gt_plan* plan, int64_t t_begin, int64_t t_count, float* tod_out, float* pwv_out,
                      void* cuda_stream) {
    return simulate_impl(plan, t_begin, t_count, tod_out, pwv_out, true, reinterpret_cast<cudaStream_t>(cuda_stream));
}

gt_status gt_debug_pkid(gt_plan* plan, int64_t t_begin, int64_t t_count, float* pkid_out, void* cuda_stream) {
    return simulate_impl(plan, t_begin, t_count, pkid_out, nullptr, false, reinterpret_cast<cudaStream_t>(cuda_stream));
}

gt_status gt_plan_destroy(gt_plan* plan) {
    if (!plan) return GT_OK;
    // wait for the work this plan enqueued (its last stream and its copy stream), not for the whole device
    if (plan->last_stream != nullptr || plan->launches > 0) cudaStreamSynchronize(plan->last_stream);
    if (plan->copy_stream) { cudaStreamSynchronize(plan->copy_stream); cudaStreamDestroy(plan->copy_stream); }
    for (int i = 0; i < 2; ++i) {
        if (plan->ev_ready[i]) cudaEventDestroy(plan->ev_ready[i]);
        if (plan->ev_copied[i]) cudaEventDestroy(plan->ev_copied[i]);
    }
    for (cudaEvent_t e : plan->ev_fused) cudaEventDestroy(e);
    for (cudaEvent_t e : plan->ev_tl) cudaEventDestroy(e);
    plan->tc_nep.scratch = nullptr;                                     // alias of tc.scratch
    gt::free_tc_tables(plan->tc_nep);
    gt::free_tc_tables(plan->tc);
    delete plan;
    return GT_OK;
}

const char* gt_last_error(const gt_plan* plan) {
    return plan ? plan->error.c_str() : g_create_error.c_str();
}

gt_status gt_debug_geometry(gt_plan* plan, int64_t t_begin, int64_t t_count, gt_georec* host_records_out) {
    gt_plan* p = plan;
    if (!p) return fail(nullptr, GT_ERR_NULL, "plan is NULL");
    if (!host_records_out) return fail(p, GT_ERR_NULL, "host_records_out is NULL");
    if (t_begin < 0 || t_count < 0 || t_begin + t_count > p->n_samples) return fail(p, GT_ERR_RANGE, "sample range outside the plan");
    const int64_t n_rows = t_count * p->n_spaxel;
    if (n_rows == 0) return GT_OK;
    DevBuf<gt_georec> rec;
    GT_CUDA(p, rec.alloc((size_t)n_rows));
    gt::geometry_kernel<<<(unsigned)((n_rows + 255) / 256), 256>>>(p->geo, t_begin, n_rows, nullptr, nullptr, rec.p, nullptr);
    GT_CUDA(p, cudaGetLastError());
    p->launches++;
    GT_CUDA(p, cudaMemcpy(host_records_out, rec.p, (size_t)n_rows * sizeof(gt_georec), cudaMemcpyDeviceToHost));
    return GT_OK;
}

__global__ void debug_philox_kernel(uint32_t k0, uint32_t k1, uint32_t c0_begin, int64_t count,
                                    uint32_t c1, uint32_t c2, uint32_t c3, uint4* out) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < count) out[i] = gt::philox4x32_10(c0_begin + (uint32_t)i, c1, c2, c3, k0, k1);
}

gt_status gt_debug_philox(uint64_t seed, uint32_t c0_begin, int64_t count, uint32_t c1, uint32_t c2, uint32_t c3,
                          uint32_t* host_out_words) {
    if (!host_out_words) return fail(nullptr, GT_ERR_NULL, "host_out_words is NULL");
    if (count < 0) return fail(nullptr, GT_ERR_SHAPE, "count is negative");
    if (count == 0) return GT_OK;
    DevBuf<uint4> out;
    GT_CUDA(nullptr, out.alloc((size_t)count));
    debug_philox_kernel<<<(unsigned)((count + 255) / 256), 256>>>((uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32),
                                                                  c0_begin, count, c1, c2, c3, out.p);
    GT_CUDA(nullptr, cudaGetLastError());
    GT_CUDA(nullptr, cudaMemcpy(host_out_words, out.p, (size_t)count * sizeof(uint4), cudaMemcpyDeviceToHost));
    return GT_OK;
}

gt_status gt_prepare_source(const float* I_dev, int32_t n_az, int32_t n_el, int32_t n_freq, double nu0_hz, double dnu_hz,
                            double daz_rad, double del_rad, double el_first_rad, double R_tel_m, double t_edge_db,
                            int32_t r_pix, float* P_dev, void* cuda_stream) {
    if (!I_dev || !P_dev) return fail(nullptr, GT_ERR_NULL, "gt_prepare_source: NULL cube pointer");
    if (I_dev == P_dev) return fail(nullptr, GT_ERR_VALUE, "gt_prepare_source: input and output must be distinct buffers");
    if (n_az <= 0 || n_el <= 0 || n_freq <= 0 || n_az > 65535 || n_el > 65535)
        return fail(nullptr, GT_ERR_SHAPE, "gt_prepare_source: cube size %d x %d x %d", n_el, n_az, n_freq);
    if (r_pix < 0 || r_pix > 64) return fail(nullptr, GT_ERR_SHAPE, "gt_prepare_source: r_pix = %d is outside 0..64", r_pix);
    if (!(nu0_hz > 0) || !(nu0_hz + (n_freq - 1) * dnu_hz > 0) || !(daz_rad > 0) || !(del_rad > 0) || !(R_tel_m > 0) ||
        !std::isfinite(t_edge_db) || !std::isfinite(el_first_rad))
        return fail(nullptr, GT_ERR_VALUE, "gt_prepare_source: frequencies, pixel pitch and R_tel must be positive");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int kw = 2 * r_pix + 1;
    DevBuf<float> d_W;
    GT_CUDA(nullptr, d_W.alloc((size_t)kw * kw * n_freq));
    gt::BeamParams b{};
    b.n_az = n_az; b.n_el = n_el; b.n_freq = n_freq; b.r_pix = r_pix;
    b.nu0 = nu0_hz; b.dnu = dnu_hz; b.daz = daz_rad; b.del = del_rad; b.el_first = el_first_rad; b.R_tel = R_tel_m;
    b.k_taper = std::fabs(t_edge_db) / 20.0 * std::log(10.0) / (R_tel_m * R_tel_m);
    b.scale = 3.14159265358979323846 * R_tel_m * R_tel_m * daz_rad * del_rad;
    b.I = I_dev; b.P = P_dev; b.W = d_W.p;
    const unsigned gf = (unsigned)((n_freq + 127) / 128);
    gt::beam_weights_kernel<<<dim3(gf, (unsigned)(r_pix + 1), (unsigned)(r_pix + 1)), 128, 0, st>>>(b);
    GT_CUDA(nullptr, cudaGetLastError());
    gt::beam_conv_kernel<<<dim3(gf, (unsigned)n_az, (unsigned)n_el), 128, 0, st>>>(b);
    GT_CUDA(nullptr, cudaGetLastError());
    GT_CUDA(nullptr, cudaStreamSynchronize(st));          // the beam table goes out of scope
    return GT_OK;
}

gt_status gt_prepare_screen(const float* epl_dev, int32_t nx, int32_t ny, double dx_m, double dy_m,
                            double R_tel_m, double t_edge_db, double pwv0_mm, float* pwv_dev, void* cuda_stream) {
    if (!epl_dev || !pwv_dev) return fail(nullptr, GT_ERR_NULL, "gt_prepare_screen: NULL screen pointer");
    if (epl_dev == pwv_dev) return fail(nullptr, GT_ERR_VALUE, "gt_prepare_screen: input and output must be distinct buffers");
    if (nx <= 0 || ny <= 0) return fail(nullptr, GT_ERR_SHAPE, "gt_prepare_screen: screen size %d x %d", nx, ny);
    if (!(dx_m > 0) || !(dy_m > 0) || !(R_tel_m > 0) || !std::isfinite(t_edge_db) || !std::isfinite(pwv0_mm))
        return fail(nullptr, GT_ERR_VALUE, "gt_prepare_screen: dx, dy and R_tel must be positive, t_edge and pwv0 finite");
    const double qx = std::floor(R_tel_m / dx_m), qy = std::floor(R_tel_m / dy_m);
    if (qx > 64.0 || qy > 64.0) return fail(nullptr, GT_ERR_UNSUPPORTED, "gt_prepare_screen: the aperture spans more than 64 pixels");
    const int rx = (int)qx, ry = (int)qy, kw = 2 * rx + 1, kh = 2 * ry + 1;
    std::vector<double> Kd((size_t)kw * kh, 0.0);
    double sum = 0.0;
    for (int j = -ry; j <= ry; ++j)
        for (int i = -rx; i <= rx; ++i) {
            const double r2 = (i * dx_m) * (i * dx_m) + (j * dy_m) * (j * dy_m);
            if (r2 < R_tel_m * R_tel_m) sum += Kd[(size_t)(j + ry) * kw + (i + rx)] = std::pow(10.0, -std::fabs(t_edge_db) / 20.0 * r2 / (R_tel_m * R_tel_m));
        }
    std::vector<float> Kf(Kd.size());
    for (size_t i = 0; i < Kd.size(); ++i) Kf[i] = (float)(Kd[i] / sum);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    DevBuf<float> d_K;
    GT_CUDA(nullptr, d_K.upload(Kf, st));
    gt::ScreenParams sp{};
    sp.epl = epl_dev; sp.pwv = pwv_dev; sp.K = d_K.p; sp.nx = nx; sp.ny = ny; sp.rx = rx; sp.ry = ry;
    sp.scale = (float)(1.0 / 6.587); sp.pwv0 = (float)pwv0_mm;
    const size_t smem = ((size_t)(gt::kScreenTile + 2 * rx) * (gt::kScreenTile + 2 * ry) + (size_t)kw * kh) * sizeof(float);
    GT_CUDA(nullptr, cudaFuncSetAttribute(gt::screen_los_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    dim3 grid((unsigned)((nx + gt::kScreenTile - 1) / gt::kScreenTile), (unsigned)((ny + gt::kScreenTile - 1) / gt::kScreenTile));
    gt::screen_los_kernel<<<grid, 256, smem, st>>>(sp);
    GT_CUDA(nullptr, cudaGetLastError());
    GT_CUDA(nullptr, cudaStreamSynchronize(st));          // d_K and Kf go out of scope
    return GT_OK;
}

int64_t gt_launch_count(const gt_plan* plan) { return plan ? plan->launches : 0; }

gt_status gt_release_cached_memory(void) {
    int dev = 0;
    GT_CUDA(nullptr, cudaGetDevice(&dev));
    if (cudaMemPool_t pool = plan_pool(dev)) {
        GT_CUDA(nullptr, cudaDeviceSynchronize());
        GT_CUDA(nullptr, cudaMemPoolTrimTo(pool, 0));
    }
    return GT_OK;
}

gt_status gt_plan_counters(gt_plan* plan, int64_t* rows, int64_t* rows_outside_cube, int64_t* pwv_below_lut, int64_t* pwv_above_lut) {
    if (!plan) return fail(nullptr, GT_ERR_NULL, "plan is NULL");
    unsigned long long h[3] = {0, 0, 0};
    GT_CUDA(plan, cudaStreamSynchronize(plan->last_stream));
    GT_CUDA(plan, cudaMemcpy(h, plan->d_counters.p, sizeof h, cudaMemcpyDeviceToHost));
    if (rows) *rows = plan->rows_done;
    if (rows_outside_cube) *rows_outside_cube = (int64_t)h[0];
    if (pwv_below_lut) *pwv_below_lut = (int64_t)h[1];
    if (pwv_above_lut) *pwv_above_lut = (int64_t)h[2];
    return GT_OK;
}

gt_status gt_pink_state_export(gt_plan* plan, float* host_state, int64_t* next_t) {
    if (!plan || !host_state || !next_t) return fail(plan, GT_ERR_NULL, "gt_pink_state_export: NULL argument");
    if (!plan->pink_noise || plan->pink_method != 0) return fail(plan, GT_ERR_UNSUPPORTED, "the plan carries no AR(1) pink-noise state");
    GT_CUDA(plan, cudaStreamSynchronize(plan->last_stream));
    GT_CUDA(plan, cudaMemcpy(host_state, plan->d_state.p, (size_t)plan->pink.n_det * plan->J * sizeof(float), cudaMemcpyDeviceToHost));
    *next_t = plan->pink_next_t;
    return GT_OK;
}

gt_status gt_pink_state_import(gt_plan* plan, const float* host_state, int64_t next_t) {
    if (!plan || !host_state) return fail(plan, GT_ERR_NULL, "gt_pink_state_import: NULL argument");
    if (!plan->pink_noise || plan->pink_method != 0) return fail(plan, GT_ERR_UNSUPPORTED, "the plan carries no AR(1) pink-noise state");
    if (next_t < 1 || next_t > plan->n_samples) return fail(plan, GT_ERR_RANGE, "next_t = %lld is outside 1..n_samples", (long long)next_t);
    GT_CUDA(plan, cudaStreamSynchronize(plan->last_stream));
    GT_CUDA(plan, cudaMemcpy(plan->d_state.p, host_state, (size_t)plan->pink.n_det * plan->J * sizeof(float), cudaMemcpyHostToDevice));
    plan->pink_next_t = next_t;
    return GT_OK;
}

gt_status gt_debug_chunking(const gt_plan* plan, int64_t* host_chunk, int64_t* device_chunk) {
    if (!plan) return fail(nullptr, GT_ERR_NULL, "plan is NULL");
    if (host_chunk) *host_chunk = plan->chunk_samples;
    if (device_chunk) *device_chunk = plan->chunk_dev;
    return GT_OK;
}

const char* gt_variant_name(const gt_plan* plan) {
    if (!plan) return "";
    return plan->variant == GT_VARIANT_FP32 ? "fp32-ffma" : plan->tc_full ? "tcgen05-3xf16-split-full" : "tcgen05-3xf16-split";
}

gt_status gt_debug_kelvin_map(gt_plan* plan, double* a_out, double* b_out) {
    if (!plan || !a_out || !b_out) return fail(plan, GT_ERR_NULL, "gt_debug_kelvin_map: NULL argument");
    if (plan->output_unit != 1) return fail(plan, GT_ERR_UNSUPPORTED, "the plan's output unit is W: no skydip map");
    const size_t nb = (size_t)plan->n_chan * sizeof(double);
    if (cudaMemcpy(a_out, plan->d_kelvin_ab.p, nb, cudaMemcpyDeviceToHost) != cudaSuccess ||
        cudaMemcpy(b_out, plan->d_kelvin_ab.p + plan->n_chan, nb, cudaMemcpyDeviceToHost) != cudaSuccess)
        return fail(plan, GT_ERR_CUDA, "gt_debug_kelvin_map: copy failed");
    return GT_OK;
}

namespace {
// ln eta_atm,z at the channel centres: bilinear on the lookup table's own grid at (f_c, mean PWV), PWV clamped to the
// table (R13); uploads it and the Eq. 26 weights S_j.  Returns N_out of this plan's spaxels.
gt_status cm_setup(gt_plan* p, double pwv_mean_mm, double r_out_rad, gt::CmParams& k, int32_t* n_out, cudaStream_t st) {
    if (!(pwv_mean_mm == pwv_mean_mm) || !(r_out_rad >= 0.0)) return fail(p, GT_ERR_VALUE, "common mode: pwv_mean and r_out must be a number and non-negative");
    const int n_pwv = p->n_pwv, nn = p->n_nu_lut;
    double q = (pwv_mean_mm - p->lut_pwv0) / p->lut_dpwv;
    if (!(q >= 0.0)) q = 0.0;
    if (q > (double)(n_pwv - 1)) q = (double)(n_pwv - 1);
    const int ip = (int)std::min<double>(std::floor(q), n_pwv - 2);
    const double fpq = q - ip;
    std::vector<double> le((size_t)p->n_chan);
    for (int c = 0; c < p->n_chan; ++c) {
        const double r = (p->h_fc[c] - p->lut_nu0) / p->lut_dnu;
        if (r < -1e-9 || r > (nn - 1) + 1e-9) return fail(p, GT_ERR_RANGE, "common mode: channel centre %d lies outside the lookup table", c);
        int ir = (int)std::floor(r);
        ir = std::max(0, std::min(ir, nn - 2));
        const double fr = r - ir;
        const float* L0 = p->h_lut.data() + (size_t)ip * nn + ir;
        const float* L1 = L0 + nn;
        const double ez = (1.0 - fpq) * ((1.0 - fr) * L0[0] + fr * L0[1]) + fpq * ((1.0 - fr) * L1[0] + fr * L1[1]);
        le[c] = std::log(ez);
        if (!(le[c] < 0.0)) return fail(p, GT_ERR_VALUE, "common mode: the atmosphere is fully transparent in channel %d (1 - eta_atm = 0 in Eq. 25)", c);
    }
    std::vector<float> w((size_t)p->n_spaxel);
    int32_t n = 0;
    for (int s = 0; s < p->n_spaxel; ++s) { w[s] = std::hypot(p->h_daz[s], p->h_del[s]) > r_out_rad ? 1.f : 0.f; n += w[s] != 0.f; }
    GT_CUDA(p, cudaMemcpyAsync(p->d_ln_eta_z.p, le.data(), le.size() * sizeof(double), cudaMemcpyHostToDevice, st));
    GT_CUDA(p, cudaMemcpyAsync(p->d_cm_weight.p, w.data(), w.size() * sizeof(float), cudaMemcpyHostToDevice, st));
    gt::cm_ref_kernel<<<(unsigned)((p->n_chan + 127) / 128), 128, 0, st>>>(p->d_ln_eta_z.p, p->n_chan, p->cm_csc0);   // eta0, 1 - eta0 at the reference airmass
    GT_CUDA(p, cudaGetLastError());
    GT_CUDA(p, cudaStreamSynchronize(st));                 // the host vectors go out of scope
    k.sinE = p->d_sinE.p; k.cosE = p->d_cosE.p; k.sin_del = p->d_sp.p + 2 * p->n_spaxel; k.cos_del = p->d_sp.p + 3 * p->n_spaxel;
    k.ln_eta_z = p->d_ln_eta_z.p; k.weight = p->d_cm_weight.p; k.n_spaxel = p->n_spaxel; k.n_chan = p->n_chan;
    k.csc0 = p->cm_csc0;
    if (n_out) *n_out = n;
    return GT_OK;
}
}  // namespace

gt_status gt_common_mode_partial(gt_plan* plan, int64_t t_begin, int64_t t_count, const float* tod_K_dev, double pwv_mean_mm,
                                 double r_out_rad, float* partial_dev, int32_t* n_out, void* cuda_stream) {
    if (!plan || !tod_K_dev || !partial_dev || !n_out) return fail(plan, GT_ERR_NULL, "gt_common_mode_partial: NULL argument");
    if (t_begin < 0 || t_count < 0 || t_begin + t_count > plan->n_samples) return fail(plan, GT_ERR_RANGE, "sample range outside the plan");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    gt::CmParams k{};
    if (gt_status s = cm_setup(plan, pwv_mean_mm, r_out_rad, k, n_out, st)) return s;
    if (t_count == 0) return GT_OK;
    k.t0 = t_begin; k.T = t_count;
    gt::cm_partial_kernel<<<(unsigned)t_count, 128, gt::cm_smem_bytes(plan->n_spaxel), st>>>(k, tod_K_dev, partial_dev);
    GT_CUDA(plan, cudaGetLastError());
    plan->launches += 2; plan->last_stream = st;          // cm_ref_kernel (cm_setup) + this pass
    return GT_OK;
}

gt_status gt_common_mode_apply(gt_plan* plan, int64_t t_begin, int64_t t_count, float* tod_K_dev, double pwv_mean_mm,
                               const float* sum_dev, int32_t n_out_total, void* cuda_stream) {
    if (!plan || !tod_K_dev || !sum_dev) return fail(plan, GT_ERR_NULL, "gt_common_mode_apply: NULL argument");
    if (t_begin < 0 || t_count < 0 || t_begin + t_count > plan->n_samples) return fail(plan, GT_ERR_RANGE, "sample range outside the plan");
    if (n_out_total < 1) return fail(plan, GT_ERR_VALUE, "common mode: no spaxel lies outside r_out (N_out = 0 in Eq. 25)");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    gt::CmParams k{};
    if (gt_status s = cm_setup(plan, pwv_mean_mm, 0.0, k, nullptr, st)) return s;
    if (t_count == 0) return GT_OK;
    k.t0 = t_begin; k.T = t_count; k.inv_n_out = 1.0 / (double)n_out_total;
    if (t_count > 0x7fffffffLL) return fail(plan, GT_ERR_SHAPE, "common mode: more than 2^31 samples in one call");
    gt::cm_apply_kernel<<<(unsigned)t_count, 128, gt::cm_smem_bytes(plan->n_spaxel), st>>>(k, tod_K_dev, sum_dev);
    GT_CUDA(plan, cudaGetLastError());
    plan->launches += 2; plan->last_stream = st;          // cm_ref_kernel (cm_setup) + this pass
    return GT_OK;
}

gt_status gt_common_mode_static(gt_plan* plan, int64_t t_begin, int64_t t_count, float* tod_K_dev, double pwv_mean_mm,
                                double r_out_rad, int32_t* n_out, void* cuda_stream) {
    if (!plan || !tod_K_dev || !n_out) return fail(plan, GT_ERR_NULL, "gt_common_mode_static: NULL argument");
    if (t_begin < 0 || t_count < 0 || t_begin + t_count > plan->n_samples) return fail(plan, GT_ERR_RANGE, "sample range outside the plan");
    constexpr int kMaxChan = 4096, kMaxSpaxel = 4096;      // the per-channel / per-spaxel constants are built on the stack
    if (plan->n_chan > kMaxChan || plan->n_spaxel > kMaxSpaxel)
        return fail(plan, GT_ERR_SHAPE, "gt_common_mode_static: at most %d channels and %d spaxels (the plan has %d and %d)",
                    kMaxChan, kMaxSpaxel, plan->n_chan, plan->n_spaxel);
    if (t_count * (int64_t)plan->n_chan > (int64_t)GT_COMMON_MODE_STATIC_MAX)
        return fail(plan, GT_ERR_SHAPE, "gt_common_mode_static: t_count * n_chan = %lld exceeds the static scratch of %lld "
                    "elements (GT_COMMON_MODE_STATIC_MAX): call it on windows of at most %lld samples, or use "
                    "gt_common_mode_partial / gt_common_mode_apply with a buffer of your own",
                    (long long)(t_count * plan->n_chan), (long long)GT_COMMON_MODE_STATIC_MAX,
                    (long long)(GT_COMMON_MODE_STATIC_MAX / plan->n_chan));
    if (t_count * plan->n_spaxel > 0x7fffffffLL) return fail(plan, GT_ERR_SHAPE, "common mode: more than 2^31 rows in one call");
    {
        int dev = -1;
        GT_CUDA(plan, cudaGetDevice(&dev));
        if (dev != plan->device) return fail(plan, GT_ERR_VALUE, "the plan lives on device %d, the current device is %d", plan->device, dev);
    }
    float* const scratch = g_cm_static_ok[plan->device].load(std::memory_order_acquire) ? g_cm_static_ptr[plan->device] : nullptr;
    if (!scratch) return fail(plan, GT_ERR_CUDA, "gt_common_mode_static: the static scratch of device %d was never resolved", plan->device);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    gt_plan* const p = plan;
    if (!(pwv_mean_mm == pwv_mean_mm) || !(r_out_rad >= 0.0)) return fail(p, GT_ERR_VALUE, "common mode: pwv_mean and r_out must be a number and non-negative");
    // the constants of cm_setup (same arithmetic), in stack arrays instead of vectors: nothing is allocated, on either side
    double le[kMaxChan];
    float w[kMaxSpaxel];
    {
        const int n_pwv = p->n_pwv, nn = p->n_nu_lut;
        double q = (pwv_mean_mm - p->lut_pwv0) / p->lut_dpwv;
        if (!(q >= 0.0)) q = 0.0;
        if (q > (double)(n_pwv - 1)) q = (double)(n_pwv - 1);
        const int ip = (int)std::min<double>(std::floor(q), n_pwv - 2);
        const double fpq = q - ip;
        for (int c = 0; c < p->n_chan; ++c) {
            const double r = (p->h_fc[c] - p->lut_nu0) / p->lut_dnu;
            if (r < -1e-9 || r > (nn - 1) + 1e-9) return fail(p, GT_ERR_RANGE, "common mode: channel centre %d lies outside the lookup table", c);
            int ir = (int)std::floor(r);
            ir = std::max(0, std::min(ir, nn - 2));
            const double fr = r - ir;
            const float* L0 = p->h_lut.data() + (size_t)ip * nn + ir;
            const float* L1 = L0 + nn;
            const double ez = (1.0 - fpq) * ((1.0 - fr) * L0[0] + fr * L0[1]) + fpq * ((1.0 - fr) * L1[0] + fr * L1[1]);
            le[c] = std::log(ez);
            if (!(le[c] < 0.0)) return fail(p, GT_ERR_VALUE, "common mode: the atmosphere is fully transparent in channel %d (1 - eta_atm = 0 in Eq. 25)", c);
        }
    }
    int32_t n = 0;
    for (int s = 0; s < p->n_spaxel; ++s) { w[s] = std::hypot(p->h_daz[s], p->h_del[s]) > r_out_rad ? 1.f : 0.f; n += w[s] != 0.f; }
    *n_out = n;
    if (n < 1) return fail(p, GT_ERR_VALUE, "common mode: no spaxel lies outside r_out (N_out = 0 in Eq. 25)");
    if (t_count == 0) return GT_OK;
    GT_CUDA(p, cudaMemcpyAsync(p->d_ln_eta_z.p, le, (size_t)p->n_chan * sizeof(double), cudaMemcpyHostToDevice, st));
    GT_CUDA(p, cudaMemcpyAsync(p->d_cm_weight.p, w, (size_t)p->n_spaxel * sizeof(float), cudaMemcpyHostToDevice, st));
    gt::cm_ref_kernel<<<(unsigned)((p->n_chan + 127) / 128), 128, 0, st>>>(p->d_ln_eta_z.p, p->n_chan, p->cm_csc0);   // eta0, 1 - eta0 at the reference airmass
    GT_CUDA(p, cudaGetLastError());
    GT_CUDA(p, cudaStreamSynchronize(st));                 // the stack arrays go out of scope
    gt::CmParams k{};
    k.sinE = p->d_sinE.p; k.cosE = p->d_cosE.p; k.sin_del = p->d_sp.p + 2 * p->n_spaxel; k.cos_del = p->d_sp.p + 3 * p->n_spaxel;
    k.ln_eta_z = p->d_ln_eta_z.p; k.weight = p->d_cm_weight.p; k.n_spaxel = p->n_spaxel; k.n_chan = p->n_chan;
    k.t0 = t_begin; k.T = t_count; k.inv_n_out = 1.0 / (double)n; k.csc0 = p->cm_csc0;
    // cm_partial_kernel overwrites every element [0, t_count * n_chan) it later reads: nothing in the shared array has to
    // start at zero, and what the previous call left behind is never read
    gt::cm_partial_kernel<<<(unsigned)t_count, 128, gt::cm_smem_bytes(p->n_spaxel), st>>>(k, tod_K_dev, scratch);
    GT_CUDA(p, cudaGetLastError());
    gt::cm_apply_kernel<<<(unsigned)t_count, 128, gt::cm_smem_bytes(p->n_spaxel), st>>>(k, tod_K_dev, scratch);
    GT_CUDA(p, cudaGetLastError());
    p->launches += 3; p->last_stream = st;
    return GT_OK;
}

gt_status gt_debug_corrections(const gt_plan* plan, int64_t* blocks, int64_t* skipped) {
    if (!plan || !blocks || !skipped) return GT_ERR_NULL;
    *blocks = plan->variant == GT_VARIANT_TENSOR ? plan->tc.n_corr_blocks : 0;
    *skipped = plan->variant == GT_VARIANT_TENSOR ? plan->tc.n_corr_skipped : 0;
    return GT_OK;
}

gt_status gt_debug_timeline(gt_plan* plan, int32_t capacity, int32_t* n_chunks, double* ms_out) {
    if (!plan || !n_chunks || !ms_out) return fail(plan, GT_ERR_NULL, "gt_debug_timeline: NULL argument");
    *n_chunks = std::min(plan->n_tl_last, capacity);
    for (int k = 0; k < *n_chunks; ++k)
        for (int j = 0; j < 4; ++j) {
            GT_CUDA(plan, cudaEventSynchronize(plan->ev_tl[4 * k + j]));
            float ms = 0.f;
            GT_CUDA(plan, cudaEventElapsedTime(&ms, plan->ev_tl[0], plan->ev_tl[4 * k + j]));
            ms_out[4 * k + j] = ms;
        }
    return GT_OK;
}

gt_status gt_measure_fp32_fma(void* cuda_stream, double* tflops_out) {
    if (!tflops_out) return fail(nullptr, GT_ERR_NULL, "gt_measure_fp32_fma: NULL argument");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int dev = 0, sm_count = 0;
    GT_CUDA(nullptr, cudaGetDevice(&dev));
    GT_CUDA(nullptr, cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev));
    const int blocks = 2 * sm_count, iters = 1 << 14;     // 2 CTAs of 1024 threads per SM = every resident thread slot
    DevBuf<float> out;
    GT_CUDA(nullptr, out.alloc((size_t)blocks * 1024));
    cudaEvent_t e0, e1;
    GT_CUDA(nullptr, cudaEventCreate(&e0)); GT_CUDA(nullptr, cudaEventCreate(&e1));
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {                                    // first pass warms up; best of the rest
        cudaEventRecord(e0, st);
        gt::fma_peak_kernel<<<blocks, 1024, 0, st>>>(out.p, iters, 0.999f, 1e-3f);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) break;
        float ms = 0.f; cudaEventElapsedTime(&ms, e0, e1);
        const double flop = 2.0 * 8.0 * 16.0 * (double)iters * 1024.0 * (double)blocks;
        if (rep > 0 && ms > 0.f) best = std::max(best, flop / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    GT_CUDA(nullptr, cudaGetLastError());
    *tflops_out = best;
    return GT_OK;
}

double gt_last_fused_ms(gt_plan* plan, int32_t* n_launches) {
    if (n_launches) *n_launches = 0;
    if (!plan || plan->n_fused_last == 0) return 0.0;
    double total = 0.0;
    for (int i = 0; i < plan->n_fused_last; ++i) {
        if (cudaEventSynchronize(plan->ev_fused[2 * i + 1]) != cudaSuccess) return -1.0;
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, plan->ev_fused[2 * i], plan->ev_fused[2 * i + 1]) != cudaSuccess) return -1.0;
        total += ms;
    }
    if (n_launches) *n_launches = plan->n_fused_last;
    return total;
}

}  // extern "C"
