/*
 * gateau_oracle.h -- C interface of the CPU ORACLE.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load this library.  It shares
 * no code, header, table or constant generator with the CUDA path under
 * paper_2604_23305_b200/csrc/ and neither includes the other.
 *
 * It is a plain double-precision transcription of the per-(time sample, spaxel,
 * frequency) signal chain of arXiv 2604.23305 ("gateau"), Sect. 2.4-2.7
 * (lines 125-229), in the paper's order and notation.  Where the paper is silent,
 * ambiguous or garbled the reading taken is listed in DESIGN.md ("Readings").
 *
 * All pointers are HOST pointers.  Large arrays are the same fp32 bytes handed to the
 * CUDA path (cube, screen, LUT, filter, per-frequency efficiencies); they are widened
 * to double on use.  Everything else is double.
 */
#ifndef GATEAU_ORACLE_H
#define GATEAU_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* One optical stage k >= 1 of the radiative transfer cascade, Eq. 12. */
typedef struct {
    const float* eta_nu;        /* [n_freq] or NULL => eta_scalar at every frequency          */
    double       eta_scalar;
    double       T_K;           /* physical temperature T_k                                   */
    int32_t      couple_atmosphere; /* 1: parasitic term is the sky          */
} go_stage;

typedef struct {
    /* uniform frequency grid nu_i = nu0 + i*dnu */
    int32_t n_freq;  double nu0_hz, dnu_hz;
    /* sampling: t_n = n / f_sample */
    int64_t n_samples;  double f_sample_hz;
    /* scan pattern phi(t_n), theta(t_n) relative to the scan centre and
       the absolute centre elevation theta_0 used for the airmass (Eq. 10)             */
    const double *az_rad, *el_rad;  double el0_rad;
    /* spaxel pointing offsets (Delta phi_i, Delta theta_i) */
    int32_t n_spaxel;  const double *daz_rad, *del_rad;
    /* source cube P_nu,src [n_el][n_az][n_freq] in W/Hz, or NULL = blank sky */
    const float* cube;  int32_t n_az, n_el;
    double az_min_rad, daz_grid_rad, el_min_rad, del_grid_rad;
    /* Eq. 11 front end: eta_t*eta_surf*eta_pol per frequency (NULL => 1) and T_CMB (0 => none) */
    const float* eta_front_nu;  double T_cmb_K;
    /* frozen-flow PWV screen [ny][nx] in mm (Eq. 9) */
    const float* screen;  int32_t nx, ny;
    double dx_m, dy_m, h_column_m, wind_mps, pwv0_a_mm, pwv0_b_mm_per_s;
    /* zenith transmission lookup table eta_atm,z [n_pwv][n_nu_lut] */
    const float* atm_lut;  int32_t n_pwv, n_nu_lut;
    double lut_nu0_hz, lut_dnu_hz, lut_pwv0_mm, lut_dpwv_mm, T_atm_K;
    /* optical stages k = 1..n_stage (the atmosphere is always the extra stage 0) */
    int32_t n_stage;  const go_stage* stages;
    /* dispersive element: transmission eta_filt [n_chan][n_freq] (Eq. 16) */
    int32_t n_chan;  const float* filt;
    const double *f_center_hz;      /* [n_chan]                                          */
    const double *dnu_eff_hz;       /* [n_chan] or NULL => derived from the filter rows  */
    /* noise */
    uint64_t seed;  int32_t photon_noise, pink_noise;
    const double *pink_A, *pink_alpha;          /* [n_spaxel*n_chan]                     */
    int32_t pink_n_stage;  const double* pink_f_corner_hz;   /* [J], J <= 8             */
} go_config;

/* Per-row (t, spaxel) geometry record: the integers are compared bit-exactly with the
   CUDA path, the fractions to 1e-6 absolute. */
typedef struct {
    int64_t n;                  /* global sample index                                   */
    int32_t iu0, iv0;           /* wrapped lower-left screen cell                        */
    int32_t ju, jv;             /* lower-left source cell, -1/-1 when outside the cube   */
    int32_t ip;                 /* lower LUT row in PWV                                  */
    int32_t pad_;
    double  fu, fv, gu, gv, fp; /* bilinear fractions                                    */
    double  pwv_mm;             /* line-of-sight zenith PWV incl. drift                  */
    double  csc;                /* 1/sin(absolute elevation)                             */
} go_georec;

/* ---- elementary pieces (pinned individually by tests) ---- */
double go_planck(double nu_hz, double T_K);                       /* P^JN_nu(T) */
void   go_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
double go_uniform(uint32_t w);                                    /* (0,1), 23 bits + half    */
void   go_normals4(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                   double z[4]);                                  /* Box-Muller x2            */
double go_photon_normal(uint64_t seed, uint32_t n, uint32_t s, uint32_t ch);   /* R19: block 32 (ch div 128) + ch mod 32, normal (ch div 32) mod 4 */
void   go_normals_bulk(uint64_t seed, uint32_t c0_begin, int64_t count, uint32_t c1, uint32_t c2,
                       uint32_t c3, double* z /*[count][4]*/);
double go_photon_sigma(double P_W, double f_center_hz, double dnu_eff_hz, double f_sample_hz);
void   go_dnu_eff(const go_config* cfg, double* out /*[n_chan]*/);
void   go_pink_coeffs(const go_config* cfg, int32_t spaxel, int32_t chan,
                      double* phi /*[J]*/, double* gain /*[J]*/);

/* ---- the path ---- */
/* Geometry for rows (n = t_begin..t_begin+t_count-1) x (all spaxels); out[t_count*n_spaxel]. */
int go_geometry(const go_config* cfg, int64_t t_begin, int64_t t_count, go_georec* out);
/* Spectrum entering the dispersive element for one row; optional intermediates.          */
int go_row_spectrum(const go_config* cfg, int64_t n, int32_t spaxel,
                    double* P_final /*[n_freq]*/, double* eta_atm /*[n_freq] or NULL*/,
                    double* S_src /*[n_freq] or NULL*/);
/* Full chain for a contiguous block of samples, all spaxels.  Any output may be NULL.
   tod        [t_count][n_spaxel][n_chan]  Eq. 21 with the noise terms switched on in cfg
   pkid       [t_count][n_spaxel][n_chan]  noiseless Eq. 16
   pwv        [t_count][n_spaxel]          zenith PWV
   Pink noise is a recurrence from n = 0: the call regenerates it from 0 up to t_begin. */
int go_simulate(const go_config* cfg, int64_t t_begin, int64_t t_count,
                double* tod, double* pkid, double* pwv);
/* Noiseless power + photon-noise term for an arbitrary list of rows (sampled parity).    */
int go_simulate_rows(const go_config* cfg, int64_t n_rows, const int64_t* t_idx,
                     const int32_t* s_idx, double* pkid /*[n_rows][n_chan]*/,
                     double* wn /*[n_rows][n_chan] or NULL*/);
/* Pink-noise series P_pn for selected detectors, samples t_begin..t_begin+t_count-1.     */
int go_pink_series(const go_config* cfg, int64_t n_det, const int32_t* s_idx,
                   const int32_t* c_idx, int64_t t_begin, int64_t t_count,
                   double* out /*[n_det][t_count]*/);

int go_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
