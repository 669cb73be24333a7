/*
 * gateau_b200.h -- C ABI of libgateau_b200.so, the B200 (sm_100a) hot path of the gateau
 * observation simulator of arXiv 2604.23305.
 *
 * The library computes, for every (time sample n, spaxel s), the signal chain of
 * PAPER.md Sect. 2.4-2.7 (lines 125-229) and writes time-ordered data (TOD):
 *
 *   step 0  pointing            phi(t_n)+dphi_s, theta(t_n)+dtheta_s
 *   step 1  screen sampling     Eq. 9 frozen-flow coordinates, bilinear PWV
 *   step 2  transmission        bilinear eta_atm,z(nu,PWV), Eq. 10 airmass
 *   step 3  source sampling     bilinear P_nu,src, zero outside; Eq. 11
 *   step 4  cascade             Eq. 12 for the atmosphere and every stage
 *   step 5  contraction         Eq. 16 P_KID = sum_nu eta_filt P_nu dnu
 *   step 6a photon noise        Eq. 18-19 with the narrow-band NEP
 *   step 6b pink noise          per-detector AR(1) cascade (R18)
 *   step 7  output              Eq. 21, TOD [t][spaxel][chan] fp32
 *
 * Every step runs in hand-written CUDA kernels; there is no CPU fallback: without a
 * CUDA device every entry point that computes returns GT_ERR_CUDA.
 *
 * Pointer kinds are stated per field: HOST pointers are read (copied) during
 * gt_plan_create and may be freed afterwards; DEVICE pointers are BORROWED: the caller
 * allocates them (e.g. torch.empty(..., device="cuda").data_ptr()), they must stay
 * valid and unchanged until gt_plan_destroy.  The library owns what it allocates.
 *
 * Errors: every call returns a gt_status, never throws, never aborts.  On error
 * *out_plan is NULL / outputs are unspecified; gt_last_error gives a message.
 */
#ifndef GATEAU_B200_H
#define GATEAU_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gt_plan gt_plan;                 /* opaque, owned by the library */

typedef enum {
    GT_OK = 0,
    GT_ERR_NULL = 1,          /* a required pointer is NULL                                   */
    GT_ERR_SHAPE = 2,         /* a size is non-positive or inconsistent                       */
    GT_ERR_VALUE = 3,         /* a value is outside its domain (eta not in [0,1], T < 0, ...) */
    GT_ERR_RANGE = 4,         /* a range is not covered (LUT nu range, sample range)          */
    GT_ERR_OOM = 5,
    GT_ERR_CUDA = 6,          /* CUDA runtime error, or no CUDA device                        */
    GT_ERR_UNSUPPORTED = 7
} gt_status;

/* One optical stage k >= 1 of the cascade, Eq. 12.  The atmosphere is
 * always the extra stage k = 0 and is not listed here (R5). */
typedef struct {
    const float* eta_nu;      /* DEVICE [n_freq] efficiency per frequency, or NULL => eta_scalar */
    double       eta_scalar;
    double       T_K;         /* physical temperature of the stage                              */
    int32_t      couple_atmosphere; /* 1: the parasitic term is the sky seen through the
                                 atmosphere, (1-eta_atm) B(T_atm) + eta_atm B(T_cmb) */
} gt_stage;

/* Kernel variant for step 2-6a (the fused generator + contraction + photon-noise kernel). */
enum {
    GT_VARIANT_DEFAULT = 0,   /* tcgen05 tensor-core kernel, three-term split of the fp32 operands */
    GT_VARIANT_FP32    = 1,   /* FP32 CUDA-core kernel (the measured alternative of north_star)  */
    GT_VARIANT_TENSOR  = 2,   /* tcgen05 kernel, explicitly                                      */
    GT_VARIANT_TENSOR_FULL = 3 /* tcgen05 kernel issuing EVERY correction product of the split: no banded corrections
                                  (DESIGN.md section 6.1).  The reference the banded kernel is tested against; ~10 % slower. */
};

typedef struct {
    /* uniform frequency grid nu_i = nu0 + i dnu, i < n_freq */
    int32_t n_freq;  double nu0_hz, dnu_hz;
    /* sampling: t_n = n / f_sample */
    int64_t n_samples;  double f_sample_hz;
    /* scan pattern: HOST [n_samples], radians relative to the scan centre;
       el0_rad = absolute elevation of the scan centre, used only for the airmass (Eq. 10) */
    const double *az_rad, *el_rad;  double el0_rad;
    /* spaxel pointing offsets: HOST [n_spaxel], radians */
    int32_t n_spaxel;  const double *daz_rad, *del_rad;
    /* source cube P_nu,src in W/Hz: DEVICE [n_el][n_az][n_freq], frequency
       fastest, or NULL = blank sky.  Grid node (j,i) sits at (el_min + j del_grid, az_min + i daz_grid). */
    const float* cube;  int32_t n_az, n_el;
    double az_min_rad, daz_grid_rad, el_min_rad, del_grid_rad;
    /* Eq. 11 front end: DEVICE [n_freq] eta_t*eta_surf*eta_pol, NULL => 1; T_cmb 0 => no CMB term */
    const float* eta_front_nu;  double T_cmb_K;
    /* frozen-flow PWV screen (Eq. 9): DEVICE [ny][nx] in mm, periodic; pixel size, column
       height h, wind speed along +x, and the mean PWV drift PWV_0(t) = a + b t added on top */
    const float* screen;  int32_t nx, ny;
    double dx_m, dy_m, h_column_m, wind_mps, pwv0_a_mm, pwv0_b_mm_per_s;
    /* zenith transmission lookup table: DEVICE [n_pwv][n_nu_lut] */
    const float* atm_lut;  int32_t n_pwv, n_nu_lut;
    double lut_nu0_hz, lut_dnu_hz, lut_pwv0_mm, lut_dpwv_mm, T_atm_K;
    /* optical stages k = 1..n_stage: HOST array of gt_stage */
    int32_t n_stage;  const gt_stage* stages;
    /* dispersive element (Eq. 16): DEVICE [n_chan][n_freq] transmission */
    int32_t n_chan;  const float* filt;
    const double* f_center_hz;    /* HOST [n_chan] channel centre (photon noise h nu)            */
    const double* dnu_eff_hz;     /* HOST [n_chan] effective bandwidth, NULL => derived from filt */
    /* noise: Philox4x32-10 keyed by seed, counter (n, spaxel, chan, stream) (R19).  Photon noise (stream 0)
       uses all four normals of a block: channel c takes normal (c / 32) % 4 of the block with counter word 2 =
       32 (c / 128) + c % 32; pink noise (streams 1, 2) takes the four normals of block (n, spaxel, c) for its four stages */
    uint64_t seed;  int32_t photon_noise, pink_noise;
    const double *pink_A, *pink_alpha;     /* HOST [n_spaxel*n_chan] PSD level A and slope alpha */
    int32_t pink_n_stage;  const double* pink_f_corner_hz;   /* HOST [J] corner frequencies, J <= 8 */
    /* streaming: samples per device chunk when the output is host memory; 0 => library picks */
    int64_t chunk_samples;
    /* one of GT_VARIANT_* */
    int32_t variant;
    /* pink-noise method: 0 = per-detector AR(1) cascade (north_star; pink_n_stage, pink_f_corner_hz used),
       1 = Timmer & Koenig: the whole series of every detector is drawn in the Fourier domain
       with PSD A f^-alpha and transformed back at plan creation (R21; needs
       n_spaxel*n_chan*n_samples*4 B of device memory; any sample range may then be simulated in any order) */
    int32_t pink_method;
    /* output unit (R22): 0 = detected power [W]; 1 = brightness temperature [K].
       For 1 the plan simulates a skydip at plan creation -- blank sky on the boresight at elevation el0, the
       zenith PWV taking skydip_n (2..64) evenly spaced values in [skydip_pwv_lo_mm, skydip_pwv_hi_mm] -- records
       the noiseless P_KID[c] and the filter-weighted line-of-sight temperature
       T_b[c] = sum_nu Fm[c][nu] ((1 - eta_atm) T_atm + eta_atm T_cmb) / sum_nu Fm[c][nu], fits the least-squares
       line T_b = a_c + b_c P_KID per channel, and gt_simulate returns a_c + b_c * (Eq. 21 total).
       GT_ERR_VALUE if a channel's filter sums to zero or its P_KID does not vary over the skydip. */
    int32_t output_unit;
    int32_t skydip_n;
    double skydip_pwv_lo_mm, skydip_pwv_hi_mm;
    /* photon-noise model when photon_noise != 0: 0 = north_star's narrow-band form (R17);
       1 = the paper's Eq. 17: NEP^2 = 2 sum_nu Fm P_nu (h nu + Fm P_nu + 2 kid_gap_J / eta_pb) dnu on the
       row's own spectrum (shot + bunching + generation-recombination), sigma = NEP sqrt(f_sample / 2), same Philox
       normal as mode 0 (R23).  Mode 1 runs the fused kernel a second time per launch (tensor variant only:
       GT_ERR_UNSUPPORTED with GT_VARIANT_FP32): the spectrum is generated again and contracted, as single fp16 terms, with
       Fm (h nu + g) + 2 Fm^2 Y and (its square) with Fm^2 into one accumulator; sigma is accurate to ~1e-3.
       kid_gap_J = Delta_Al (188 micro-eV in the paper, :103), eta_pb = pair-breaking efficiency (0.4). */
    int32_t photon_mode;
    double kid_gap_J, eta_pb;
    /* Global index of this plan's spaxel 0 (default 0).  A plan may hold a sub-range of an instrument's spaxels
       (spaxel-sharded runs): the Philox counter word 1 is spaxel_index_base + s, so that the shard
       reproduces the TOD of the same spaxels in a plan that holds them all, bit for bit.  >= 0. */
    int32_t spaxel_index_base;
} gt_config;

/* Value ranges (tensor variant).  The fused kernel contracts fp16 (hi, lo) operand pairs:
 *   - filt: any finite values (negative lobes of an Eq. 7 filterbank included).  Every channel is scaled by its own
 *     power of two, so a delta filter 1/dnu, a row-normalised filter and a transmission of peak 1 are equally accurate;
 *     inside one channel, values below 2^-39 of the channel's largest are rounded to multiples of 2^-39 of it.
 *   - spectrum: the plan takes the largest element it can meet (max over nu of |(B_atm - B_cmb) prod eta_k| and
 *     |eta_front prod eta_k| max |cube|, one device reduction over the cube) and scales by a power of two; elements
 *     below 2^-36 of that maximum are rounded to multiples of it.  NaN / Inf in cube, screen, filt, LUT or the
 *     per-frequency efficiencies: GT_ERR_VALUE.  A spectrum whose scale leaves the fp32 range: GT_ERR_RANGE.
 * Threads and streams: a plan owns one set of work buffers.  It may be used by one thread and one stream at a time;
 * calls on the same plan must be ordered by the caller (same stream, or events).  A plan belongs to the device that was
 * current at gt_plan_create; calling it with another device current returns GT_ERR_VALUE. */

/* Per-row geometry record returned by gt_debug_geometry: the integers are the quantities
 * "index, scan and RNG counters" that must match the oracle bit for bit. */
typedef struct {
    int64_t n;                   /* global sample index (= Philox counter word 0)          */
    int32_t iu0, iv0;            /* wrapped lower-left screen cell                          */
    int32_t ju, jv;              /* lower-left source cell, -1/-1 outside the cube          */
    int32_t ip;                  /* lower LUT row in PWV                                    */
    int32_t pad_;
    double  fu, fv, gu, gv, fp;  /* bilinear fractions                                      */
    double  pwv_mm;              /* zenith PWV on the line of sight incl. drift             */
    double  csc;                 /* 1 / sin(absolute elevation)                             */
} gt_georec;

/* Validates cfg, copies every HOST array, reads the small DEVICE arrays it needs for
 * plan-time constants (LUT, filter, per-frequency efficiencies) and uploads the derived
 * tables.  cuda_stream: a cudaStream_t (NULL = default stream) used for the uploads.
 * Returns GT_OK and *out_plan, or an error and *out_plan = NULL. */
gt_status gt_plan_create(const gt_config* cfg, void* cuda_stream, gt_plan** out_plan);

/* Simulates samples n = t_begin .. t_begin+t_count-1 for all spaxels and channels.
 *   tod_out  [t_count][n_spaxel][n_chan] fp32, DEVICE memory or (pinned or pageable) HOST
 *            memory; detected with cudaPointerGetAttributes.
 *   pwv_out  optional (NULL ok) [t_count][n_spaxel] fp32 zenith PWV, same memory kind rule.
 * DEVICE output: the kernels write in place and the call returns after enqueueing on
 * cuda_stream (asynchronous).  HOST output: the TOD is produced in chunks of
 * chunk_samples into two device buffers and copied out on an internal side stream while
 * the next chunk computes; the call returns after the last copy has completed (blocking).
 * With pink noise on, the AR(1) state advances with the call: calls must cover
 * contiguous increasing ranges, or restart from t_begin = 0 (else GT_ERR_VALUE).  With
 * pink noise off any range is legal.  t_count = 0 is legal and does nothing. */
gt_status gt_simulate(gt_plan* plan, int64_t t_begin, int64_t t_count,
                      float* tod_out, float* pwv_out, void* cuda_stream);

/* Device memory of the plans comes from a library-owned stream-ordered pool that keeps what destroyed plans return, so
 * that creating plans back to back (one observation per plan) does not pay cudaMalloc / cudaFree every time.  This call
 * returns the cached blocks of the current device to the driver (it synchronises the device). */
gt_status gt_release_cached_memory(void);

/* Frees everything the plan owns, after waiting for the work the plan itself enqueued (the stream of its last call
 * and its internal copy stream).  NULL-safe. */
gt_status gt_plan_destroy(gt_plan* plan);

/* Pre-processing utility (R25; not part of a plan): turns a specific-intensity cube
 * I_nu [W m^-2 Hz^-1 sr^-1] into the spectral power cube P_nu,src [W/Hz] that gt_config.cube expects.
 *   F_nu(rho) = |int_0^R A(r) J0(2 pi r rho / lambda) r dr|^2 / F_nu(0)        the far field of the circular aperture
 *               with A(r) = 10^(-|t_edge_db| / 20 * r^2 / R_tel^2), r < R_tel (Eq. 2-3: the 2-D Fourier transform of
 *               a circularly symmetric illumination is this Hankel transform), peak 1
 *   P[j][i][nu] = pi R_tel^2 daz del sum_{|dj|,|di| <= r_pix} F_nu(di daz, dj del) I[j - dj][i - di][nu]
 *                 cos(el_first + (j - dj) del)                                  (Eq. 1, rectangle rule; I = 0 outside)
 * I_dev, P_dev: DEVICE [n_el][n_az][n_freq] fp32 (the cube layout of gt_config), distinct, caller-owned.
 * nu = nu0_hz + k dnu_hz; daz_rad, del_rad = the cube's pixel pitch; el_first_rad = absolute elevation of row 0.
 * Needs (2 r_pix + 1)^2 n_freq * 4 B of device scratch for the beam table.  Synchronises cuda_stream.
 * GT_ERR_SHAPE for non-positive sizes or r_pix outside 0..64, GT_ERR_VALUE for non-positive nu0, pitch or R_tel. */
gt_status gt_prepare_source(const float* I_dev, int32_t n_az, int32_t n_el, int32_t n_freq, double nu0_hz, double dnu_hz,
                            double daz_rad, double del_rad, double el_first_rad, double R_tel_m, double t_edge_db,
                            int32_t r_pix, float* P_dev, void* cuda_stream);
/* Pre-processing utility (R24; not part of a plan): turns an extra-path-length screen
 * into the line-of-sight PWV screen that gt_config.screen expects.
 *   pwv[y][x] = pwv0_mm + (1 / 6.587) sum_{i,j} K[j][i] epl[(y + j) mod ny][(x + i) mod nx]      (Eq. 4, then :92)
 * K = the aperture footprint on the screen grid: 10^(-|t_edge_db| / 20 * r^2 / R_tel^2) for r < R_tel (the Gaussian
 * illumination of Eq. 2 with the given edge taper), 0 outside, r^2 = (i dx)^2 + (j dy)^2, normalised to unit sum.
 * epl_dev, pwv_dev: DEVICE [ny][nx] fp32, distinct buffers, caller-owned.  Synchronises cuda_stream before returning
 * (the footprint weights are a temporary of the call).
 * GT_ERR_SHAPE for non-positive sizes, GT_ERR_VALUE for non-positive dx, dy, R_tel,
 * GT_ERR_UNSUPPORTED if R_tel spans more than 64 pixels in x or y. */
gt_status gt_prepare_screen(const float* epl_dev, int32_t nx, int32_t ny, double dx_m, double dy_m,
                            double R_tel_m, double t_edge_db, double pwv0_mm, float* pwv_dev, void* cuda_stream);

/* Common-mode subtraction, Eq. 25-26, on a TOD in brightness temperature (output_unit = 1):
 *   T*_a,i(t,f) = T_b,i / eta_i - (1 - eta_i) / (eta_i N_out) sum_j S_j T_b,j / (1 - eta_j),
 *   eta_j(t,f) = eta_atm,z(f)^csc(el0 + el[t] + del[j]) (Eq. 10), eta_atm,z(f) = the plan's lookup table, bilinear at
 *   (f_center[f], pwv_mean_mm) (the zenith PWV averaged over the observation; clamped to the table),
 *   S_j = 1 where sqrt(daz_j^2 + del_j^2) > r_out_rad, N_out = sum_j S_j.
 * The sum over spaxels is the only cross-spaxel term of the paper, so it is split for spaxel-sharded runs (one plan per
 * spaxel sub-range, spaxel_index_base):
 *   gt_common_mode_partial: partial_dev[t][chan] (DEVICE, fp32, overwritten) = sum over THIS plan's spaxels of
 *       S_j T_b,j / (1 - eta_j), and *n_out = this plan's number of spaxels with S_j = 1.  tod_K_dev DEVICE
 *       [t_count][n_spaxel][n_chan], read only.
 *   -- the caller adds partial sums and n_out over the plans (one all-reduce over [t x chan]) --
 *   gt_common_mode_apply: tod_K_dev <- T*_a in place, given sum_dev[t][chan] over ALL spaxels and n_out_total >= 1.
 * A single plan holding every spaxel calls both with its own partial sum.  Asynchronous on cuda_stream (after a short
 * synchronous upload of per-channel constants).  GT_ERR_RANGE if a channel centre lies outside the table,
 * GT_ERR_VALUE if a channel is fully transparent (1 - eta = 0) or n_out_total < 1. */
gt_status gt_common_mode_partial(gt_plan* plan, int64_t t_begin, int64_t t_count, const float* tod_K_dev, double pwv_mean_mm,
                                 double r_out_rad, float* partial_dev, int32_t* n_out, void* cuda_stream);
gt_status gt_common_mode_apply(gt_plan* plan, int64_t t_begin, int64_t t_count, float* tod_K_dev, double pwv_mean_mm,
                               const float* sum_dev, int32_t n_out_total, void* cuda_stream);

/* The same subtraction (Eq. 25-26, single plan holding every spaxel: partial sum, then apply) for callers that cannot
 * allocate device memory -- code under CUDA-graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The
 * [t_count][n_chan] partial sums, which gt_common_mode_partial / _apply take as a caller-owned buffer, live in ONE
 * file-scope static device array of GT_COMMON_MODE_STATIC_MAX floats (8 MB) inside the library: every GPU that loads the
 * library holds it until the process exits.  The call allocates nothing, on the device or on the host (no cudaMalloc,
 * cudaFree, pool or allocating library routine: the per-channel and per-spaxel constants are built on the stack and
 * copied into tables the plan already owns); its device address is resolved once per device at gt_plan_create.
 *   tod_K_dev: DEVICE [t_count][n_spaxel][n_chan] fp32, brightness temperature, overwritten in place with T*_a.
 *   *n_out = N_out of the plan's spaxels.  Results are bit-identical to gt_common_mode_partial + gt_common_mode_apply.
 * Limits: t_count * n_chan <= GT_COMMON_MODE_STATIC_MAX (call it on windows of samples), n_chan <= 4096,
 * n_spaxel <= 4096: GT_ERR_SHAPE beyond them, with the limit in the message.  GT_ERR_VALUE if N_out = 0; otherwise the
 * errors of gt_common_mode_partial.
 * EVERY call on a device shares the array, which keeps the last call's contents (never read: the partial sums overwrite
 * all t_count * n_chan elements before they are used, so nothing needs clearing).  Calls that overlap on the GPU -- two
 * streams, two plans, two host threads on one device -- RACE on it: serialise them (one stream, or events).  Asynchronous
 * on cuda_stream after a short synchronous upload of the constants, like gt_common_mode_partial. */
#define GT_COMMON_MODE_STATIC_MAX 2097152
gt_status gt_common_mode_static(gt_plan* plan, int64_t t_begin, int64_t t_count, float* tod_K_dev, double pwv_mean_mm,
                                double r_out_rad, int32_t* n_out, void* cuda_stream);

/* Message of the last error on this plan; plan == NULL => the calling thread's last
 * gt_plan_create error.  Never NULL. */
const char* gt_last_error(const gt_plan* plan);

/* ---- test hooks (not part of the user path) ---- */
/* Geometry records of rows (t_begin .. t_begin+t_count-1) x (all spaxels) into HOST memory
 * host_records_out[t_count*n_spaxel], computed by the same device code as gt_simulate. */
gt_status gt_debug_geometry(gt_plan* plan, int64_t t_begin, int64_t t_count,
                            gt_georec* host_records_out);
/* Raw Philox4x32-10 output words of the device generator for `count` consecutive values
 * of counter word 0 starting at c0_begin, fixed (c1, c2, c3), key = seed: HOST
 * out_words[count][4].  Needs no plan. */
gt_status gt_debug_philox(uint64_t seed, uint32_t c0_begin, int64_t count,
                          uint32_t c1, uint32_t c2, uint32_t c3, uint32_t* host_out_words);
/* Noiseless channel power (Eq. 16 only, noise switched off regardless of the plan) for the
 * same range as gt_simulate; pkid_out follows the tod_out rules.  Does not touch the
 * pink-noise state. */
gt_status gt_debug_pkid(gt_plan* plan, int64_t t_begin, int64_t t_count,
                        float* pkid_out, void* cuda_stream);
/* Samples per kernel launch: *host_chunk when the output is host memory (= chunk_samples, or the library's pick),
 * *device_chunk when it is device memory.  The parity tests place sampled rows on both sides of these seams. */
gt_status gt_debug_chunking(const gt_plan* plan, int64_t* host_chunk, int64_t* device_chunk);
/* Number of kernels this library launched since the plan was created. */
int64_t gt_launch_count(const gt_plan* plan);
/* Diagnostic counters since plan creation (any pointer may be NULL): rows = (sample, spaxel) pairs the
 * geometry kernel processed for gt_simulate / gt_debug_pkid; rows_outside_cube = rows whose pointing fell outside the
 * source cube (they see blank sky); pwv_below_lut / pwv_above_lut = rows whose line-of-sight PWV was
 * clamped to the first / last row of the lookup table (R13).  Synchronises the plan's last stream. */
gt_status gt_plan_counters(gt_plan* plan, int64_t* rows, int64_t* rows_outside_cube,
                           int64_t* pwv_below_lut, int64_t* pwv_above_lut);
/* Checkpoint / restart at call granularity: everything but the AR(1) pink-noise state is a pure function
 * of the sample index (counter-based RNG), so a run can be resumed by another plan of the same configuration.
 *   export: host_state [n_spaxel * n_chan * pink_n_stage] fp32 = x_j of every detector at the last simulated sample
 *           (detector-major, stage fastest), *next_t = the sample the next gt_simulate must start at.
 *   import: sets both; the next gt_simulate must start at next_t (1 <= next_t <= n_samples; 0 needs no import).
 * GT_ERR_UNSUPPORTED unless the plan has pink_noise != 0 with pink_method = 0.  Both synchronise the plan's last stream. */
gt_status gt_pink_state_export(gt_plan* plan, float* host_state, int64_t* next_t);
gt_status gt_pink_state_import(gt_plan* plan, const float* host_state, int64_t next_t);
/* Name of the fused-kernel variant the plan resolved to ("tcgen05-3xf16-split", "fp32-ffma"). */
const char* gt_variant_name(const gt_plan* plan);
/* Device time [ms] the fused kernel took in the last gt_simulate / gt_debug_pkid call, summed
 * over its launches (CUDA events on the launching stream); synchronises the stream.  Also
 * returns the number of launches in *n_launches (NULL ok). */
double gt_last_fused_ms(gt_plan* plan, int32_t* n_launches);
/* Banded corrections of the tensor variant: *blocks = correction products of the three-term split,
 * two (A_lo.Fm_hi and A_hi.Fm_lo) per (channel group, column group, 64-frequency slab) block of the contraction;
 * *skipped = how many of them are not issued because the plan proved them negligible there (worst case over the spectra
 * the plan can produce, all skipped products of a channel together, below 1e-6 of the channel's smallest power).
 * Both 0 for GT_VARIANT_FP32.  Test and reporting hook. */
gt_status gt_debug_corrections(const gt_plan* plan, int64_t* blocks, int64_t* skipped);
/* Measurement hooks (bench.py).  gt_debug_timeline: device timeline of the last HOST-output gt_simulate call, per chunk
 * k < *n_chunks <= capacity: ms_out[4 k + {0,1,2,3}] = {compute begin, compute end, copy begin, copy end} in ms after the
 * first chunk's compute begin (CUDA events on the compute stream and on the internal copy stream): shows the D2H copy
 * of chunk k running under the kernels of chunk k+1.  gt_measure_fp32_fma: FP32 FMA peak of the current device in
 * TFLOP/s from a register-only FMA loop (8 chains per thread, every thread slot resident), best of 5. */
gt_status gt_debug_timeline(gt_plan* plan, int32_t capacity, int32_t* n_chunks, double* ms_out);
gt_status gt_measure_fp32_fma(void* cuda_stream, double* tflops_out);
/* Test hook: the per-channel skydip map T_b = a + b P_KID of a plan with output_unit = 1, copied to the HOST
 * arrays a_out, b_out [n_chan] (double).  GT_ERR_UNSUPPORTED if the plan's output unit is W. */
gt_status gt_debug_kelvin_map(gt_plan* plan, double* a_out, double* b_out);

#ifdef __cplusplus
}
#endif
#endif
