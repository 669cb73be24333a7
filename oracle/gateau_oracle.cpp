/*
 * gateau_oracle.cpp -- plain double-precision CPU ORACLE for the gateau hot path.
 *
 * TEST INFRASTRUCTURE ONLY (see gateau_oracle.h).  Slow and literal on purpose: every
 * function follows one passage of arXiv 2604.23305 in the paper's order; no
 * blocking, fusion or re-association.  The only hoisting is that P^JN_nu(T) of a fixed
 * temperature is tabulated once per frequency (a pure function of nu and T, same
 * expression, same value) instead of being re-evaluated for every row.
 *
 * Build: g++ -O2 -std=c++17 -fopenmp -ffp-contract=off -fno-fast-math -shared -fPIC
 *   -ffp-contract=off matters: the geometry index arithmetic must round every + - * /
 *   separately so that the integer cell indices are the IEEE-754 ones (DESIGN.md,
 *   "canonical geometry arithmetic").
 *
 * Parity pins: tests/test_oracle_*.py (closed forms, invariants, library routines, brute
 * force).  Unpinned: absolute physical realism of the synthetic inputs (out of scope).
 */
#include "gateau_oracle.h"

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

/* CODATA 2018 exact values */
constexpr double kPlanck_h    = 6.62607015e-34;   /* J s  */
constexpr double kBoltzmann_k = 1.380649e-23;     /* J/K  */
constexpr double kPi          = 3.14159265358979323846;

/* ------------------------------------------------------------------------------------
 * P^JN_nu(T): single-moded Johnson-Nyquist spectral power (Nyquist 1928
 * quantum form, one mode, one polarisation): h nu / (exp(h nu / k T) - 1) [W/Hz].
 * Reading R4: the paper names it without a formula; B(nu, 0) = 0.
 * ---------------------------------------------------------------------------------- */
double planck(double nu, double T) {
    if (!(T > 0.0)) return 0.0;
    const double x = kPlanck_h * nu / (kBoltzmann_k * T);
    return kPlanck_h * nu / std::expm1(x);
}

/* ------------------------------------------------------------------------------------
 * Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  Counter (c0..c3), key (k0,k1).
 * Round: two 32x32->64 products; output (hi1^c1^k0, lo1, hi0^c3^k1, lo0); the key is
 * bumped by the Weyl constants between rounds.  Written from the published description.
 * ---------------------------------------------------------------------------------- */
constexpr uint32_t PHILOX_M0 = 0xD2511F53u, PHILOX_M1 = 0xCD9E8D57u;
constexpr uint32_t PHILOX_W0 = 0x9E3779B9u, PHILOX_W1 = 0xBB67AE85u;

void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = (uint64_t)PHILOX_M0 * c0;
        const uint64_t p1 = (uint64_t)PHILOX_M1 * c2;
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n1 = lo1;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        const uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += PHILOX_W0; k1 += PHILOX_W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* U(w) = ((w >> 9) + 1/2) * 2^-23 in (0,1): 23 random bits plus a half, so every value is
 * exactly representable in binary32 as well as binary64 (reading R19). */
double uniform01(uint32_t w) { return ((double)(w >> 9) + 0.5) * (1.0 / 8388608.0); }

/* Four standard normals from one Philox block: Box-Muller on (w0,w1) and on (w2,w3).
 * Counter layout (reading R19): c0 = sample index n, c1 = spaxel, c2 = channel (pink noise) or
 * channel block (photon noise, see photon_normal),
 * c3 = stream; key = (seed low 32, seed high 32). */
void normals4(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, double z[4]) {
    const uint32_t ctr[4] = {c0, c1, c2, c3};
    const uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32)};
    uint32_t w[4];
    philox4x32_10(ctr, key, w);
    const double r0 = std::sqrt(-2.0 * std::log(uniform01(w[0])));
    const double a0 = 2.0 * kPi * uniform01(w[1]);
    const double r1 = std::sqrt(-2.0 * std::log(uniform01(w[2])));
    const double a1 = 2.0 * kPi * uniform01(w[3]);
    z[0] = r0 * std::cos(a0);
    z[1] = r0 * std::sin(a0);
    z[2] = r1 * std::cos(a1);
    z[3] = r1 * std::sin(a1);
}

constexpr uint32_t STREAM_PHOTON = 0, STREAM_PINK_LO = 1, STREAM_PINK_HI = 2;
constexpr uint32_t COUNTER_INIT  = 0xFFFFFFFFu;    /* c0 used for the AR(1) initial states */

/* The photon-noise normal of detector-sample (n, spaxel s, channel ch) (reading R19): one Philox block of
 * stream 0 yields four independent normals (Box-Muller's cosine and sine branches of both word pairs) and serves
 * the four channels b + 128 q + {0, 32, 64, 96}, b = ch mod 32, q = ch div 128:
 *   counter = (n, s, 32 q + b, 0),  normal index k = (ch div 32) mod 4. */
double photon_normal(uint64_t seed, uint32_t n, uint32_t s, uint32_t ch) {
    double z[4];
    normals4(seed, n, s, 32u * (ch / 128u) + ch % 32u, STREAM_PHOTON, z);
    return z[(ch / 32u) % 4u];
}

/* Eq. 17-18 in north_star's narrow-band form (reading R17):
 * sigma^2 = (2 h f_c P + 2 P^2 / dnu_c) * f_sample / 2. */
double photon_sigma(double P, double f_c, double dnu_c, double f_s) {
    const double nep2 = 2.0 * kPlanck_h * f_c * P + 2.0 * P * P / dnu_c;
    return std::sqrt((nep2 > 0.0 ? nep2 : 0.0) * f_s / 2.0);
}

/* Default effective bandwidth of channel c (reading R17): the flat-spectrum reduction of
 * Eq. 17's bunching term, (sum F dnu)^2 / (sum F^2 dnu). */
double dnu_eff_default(const go_config& c, int ch) {
    double s1 = 0.0, s2 = 0.0;
    for (int i = 0; i < c.n_freq; ++i) {
        const double f = (double)c.filt[(size_t)ch * c.n_freq + i];
        s1 += f * c.dnu_hz;
        s2 += f * f * c.dnu_hz;
    }
    return s1 * s1 / s2;
}

double dnu_eff_of(const go_config& c, int ch) {
    return c.dnu_eff_hz ? c.dnu_eff_hz[ch] : dnu_eff_default(c, ch);
}

/* AR(1)-cascade coefficients for detector (spaxel, chan) (reading R18):
 * phi_j = exp(-2 pi f_j / f_s);  g_j^2 = A ln(rho) sin(pi alpha / 2) f_j^(1-alpha),
 * ln(rho) = ln(f_0 / f_{J-1}) / (J-1)  (1 when J == 1). */
void pink_coeffs(const go_config& c, int s, int ch, double* phi, double* gain) {
    const int J = c.pink_n_stage;
    const size_t d = (size_t)s * c.n_chan + ch;
    const double A = c.pink_A[d], alpha = c.pink_alpha[d];
    double lnrho = 1.0;
    if (J >= 2) lnrho = std::log(c.pink_f_corner_hz[0] / c.pink_f_corner_hz[J - 1]) / (double)(J - 1);
    for (int j = 0; j < J; ++j) {
        const double fj = c.pink_f_corner_hz[j];
        phi[j]  = std::exp(-2.0 * kPi * fj / c.f_sample_hz);
        gain[j] = std::sqrt(A * lnrho * std::sin(kPi * alpha / 2.0) * std::pow(fj, 1.0 - alpha));
    }
}

/* One detector's pink-noise series for samples [t_begin, t_begin+t_count): the recurrence
 * always starts at n = 0 from the drawn initial state x_j[-1]. */
void pink_series(const go_config& c, int s, int ch, int64_t t_begin, int64_t t_count, double* out) {
    const int J = c.pink_n_stage;
    double phi[8], gain[8], x[8], z[8];
    pink_coeffs(c, s, ch, phi, gain);
    normals4(c.seed, COUNTER_INIT, (uint32_t)s, (uint32_t)ch, STREAM_PINK_LO, z);
    if (J > 4) normals4(c.seed, COUNTER_INIT, (uint32_t)s, (uint32_t)ch, STREAM_PINK_HI, z + 4);
    for (int j = 0; j < J; ++j) x[j] = z[j];
    for (int64_t n = 0; n < t_begin + t_count; ++n) {
        normals4(c.seed, (uint32_t)n, (uint32_t)s, (uint32_t)ch, STREAM_PINK_LO, z);
        if (J > 4) normals4(c.seed, (uint32_t)n, (uint32_t)s, (uint32_t)ch, STREAM_PINK_HI, z + 4);
        double pn = 0.0;
        for (int j = 0; j < J; ++j) {
            x[j] = phi[j] * x[j] + std::sqrt(1.0 - phi[j] * phi[j]) * z[j];
            pn += gain[j] * x[j];
        }
        if (n >= t_begin) out[n - t_begin] = pn;
    }
}

/* Positive modulo for cell indices (periodic screen, reading R7). */
int64_t pmod(int64_t a, int64_t m) { const int64_t r = a % m; return r < 0 ? r + m : r; }

/* ------------------------------------------------------------------------------------
 * Steps 0-1 and the index part of steps 2-3 for one row (sample n, spaxel s).
 * PAPER.md:137 (pointing), Eq. 9 :141-145 (screen coordinates), :147 (bilinear PWV),
 * Eq. 10 :149 (airmass).  Canonical arithmetic: only + - * / floor on
 * doubles, tangent/sine of a sum formed with the addition formulas from per-sample and
 * per-spaxel libm values, so the CUDA path can reproduce the integers bit for bit.
 * ---------------------------------------------------------------------------------- */
void row_geometry(const go_config& c, int64_t n, int s, go_georec& g) {
    g.n = n; g.pad_ = 0;
    const double t = (double)n / c.f_sample_hz;

    /* tan(phi(t) + dphi_i), tan(theta(t) + dtheta_i) */
    const double ta_n = std::tan(c.az_rad[n]), ta_s = std::tan(c.daz_rad[s]);
    const double te_n = std::tan(c.el_rad[n]), te_s = std::tan(c.del_rad[s]);
    const double tan_a = (ta_n + ta_s) / (1.0 - ta_n * ta_s);
    const double tan_e = (te_n + te_s) / (1.0 - te_n * te_s);

    /* Eq. 9; wind along +x (R10); boresight at t=0 on the screen centre (R8) */
    const double x = c.h_column_m * tan_a + c.wind_mps * t;
    const double y = c.h_column_m * tan_e;
    const double u = x / c.dx_m + 0.5 * (double)c.nx;
    const double v = y / c.dy_m + 0.5 * (double)c.ny;
    const double fl_u = std::floor(u), fl_v = std::floor(v);
    g.fu = u - fl_u;  g.fv = v - fl_v;
    const int64_t iu = (int64_t)fl_u, iv = (int64_t)fl_v;
    const int64_t iu0 = pmod(iu, c.nx), iu1 = pmod(iu + 1, c.nx);
    const int64_t iv0 = pmod(iv, c.ny), iv1 = pmod(iv + 1, c.ny);
    g.iu0 = (int32_t)iu0;  g.iv0 = (int32_t)iv0;

    /* bilinear PWV + mean drift PWV_0(t) */
    const double s00 = (double)c.screen[(size_t)iv0 * c.nx + iu0];
    const double s01 = (double)c.screen[(size_t)iv0 * c.nx + iu1];
    const double s10 = (double)c.screen[(size_t)iv1 * c.nx + iu0];
    const double s11 = (double)c.screen[(size_t)iv1 * c.nx + iu1];
    const double row0 = (1.0 - g.fu) * s00 + g.fu * s01;
    const double row1 = (1.0 - g.fu) * s10 + g.fu * s11;
    g.pwv_mm = ((1.0 - g.fv) * row0 + g.fv * row1) + (c.pwv0_a_mm + c.pwv0_b_mm_per_s * t);

    /* LUT cell in PWV: clamp (R13) */
    double q = (g.pwv_mm - c.lut_pwv0_mm) / c.lut_dpwv_mm;
    if (q < 0.0) q = 0.0;
    if (q > (double)(c.n_pwv - 1)) q = (double)(c.n_pwv - 1);
    int64_t ip = (int64_t)std::floor(q);
    if (ip > c.n_pwv - 2) ip = c.n_pwv - 2;
    g.ip = (int32_t)ip;  g.fp = q - (double)ip;

    /* airmass: sin of the absolute elevation theta(t) + theta_0 + dtheta_i (Eq. 10) */
    const double E_n = c.el0_rad + c.el_rad[n];
    const double sinE = std::sin(E_n) * std::cos(c.del_rad[s]) + std::cos(E_n) * std::sin(c.del_rad[s]);
    g.csc = 1.0 / sinE;

    /* source cell, flat az/el grid (R11), inclusive edges (R12) */
    g.ju = -1; g.jv = -1; g.gu = 0.0; g.gv = 0.0;
    if (c.cube) {
        const double a = c.az_rad[n] + c.daz_rad[s];
        const double e = c.el_rad[n] + c.del_rad[s];
        const double us = (a - c.az_min_rad) / c.daz_grid_rad;
        const double vs = (e - c.el_min_rad) / c.del_grid_rad;
        if (!(us < 0.0 || us > (double)(c.n_az - 1) || vs < 0.0 || vs > (double)(c.n_el - 1))) {
            int64_t ju = (int64_t)std::floor(us), jv = (int64_t)std::floor(vs);
            if (ju > c.n_az - 2) ju = c.n_az - 2;
            if (jv > c.n_el - 2) jv = c.n_el - 2;
            g.ju = (int32_t)ju;  g.jv = (int32_t)jv;
            g.gu = us - (double)ju;  g.gv = vs - (double)jv;
        }
    }
}

/* Row-invariant tables: P^JN of every fixed temperature on the frequency grid. */
struct Tables {
    std::vector<double> nu, B_cmb, B_atm;
    std::vector<std::vector<double>> B_stage;
    std::vector<int64_t> ir;  std::vector<double> fr;      /* LUT cell / fraction in nu */
};

void build_tables(const go_config& c, Tables& tb) {
    const int nf = c.n_freq;
    tb.nu.resize(nf); tb.B_cmb.resize(nf); tb.B_atm.resize(nf); tb.ir.resize(nf); tb.fr.resize(nf);
    tb.B_stage.assign(c.n_stage, std::vector<double>(nf));
    for (int i = 0; i < nf; ++i) {
        const double nu = c.nu0_hz + (double)i * c.dnu_hz;
        tb.nu[i] = nu;
        tb.B_cmb[i] = planck(nu, c.T_cmb_K);
        tb.B_atm[i] = planck(nu, c.T_atm_K);
        for (int k = 0; k < c.n_stage; ++k) tb.B_stage[k][i] = planck(nu, c.stages[k].T_K);
        const double r = (nu - c.lut_nu0_hz) / c.lut_dnu_hz;
        int64_t ir = (int64_t)std::floor(r);
        if (ir > c.n_nu_lut - 2) ir = c.n_nu_lut - 2;
        if (ir < 0) ir = 0;
        tb.ir[i] = ir;  tb.fr[i] = r - (double)ir;
    }
}

/* ------------------------------------------------------------------------------------
 * Steps 2-4 for one row: the spectrum P_nu entering the dispersive element.
 * ---------------------------------------------------------------------------------- */
void row_spectrum(const go_config& c, const Tables& tb, const go_georec& g,
                  double* P_out, double* eta_out, double* S_out) {
    const int nf = c.n_freq;
    const size_t nl = (size_t)c.n_nu_lut;
    for (int i = 0; i < nf; ++i) {
        /* step 2: bilinear eta_atm,z(nu, PWV) then Eq. 10 (R14, R15) */
        const size_t ir = (size_t)tb.ir[i];
        const double fr = tb.fr[i];
        const double L00 = (double)c.atm_lut[(size_t)g.ip * nl + ir];
        const double L01 = (double)c.atm_lut[(size_t)g.ip * nl + ir + 1];
        const double L10 = (double)c.atm_lut[(size_t)(g.ip + 1) * nl + ir];
        const double L11 = (double)c.atm_lut[(size_t)(g.ip + 1) * nl + ir + 1];
        const double eta_z = (1.0 - g.fp) * ((1.0 - fr) * L00 + fr * L01)
                           +        g.fp  * ((1.0 - fr) * L10 + fr * L11);
        const double eta_atm = std::pow(eta_z, g.csc);

        /* step 3: bilinear source, zero outside the grid */
        double S = 0.0;
        if (g.ju >= 0) {
            const size_t na = (size_t)c.n_az, f = (size_t)nf;
            const double c00 = (double)c.cube[((size_t)g.jv * na + g.ju) * f + i];
            const double c01 = (double)c.cube[((size_t)g.jv * na + g.ju + 1) * f + i];
            const double c10 = (double)c.cube[((size_t)(g.jv + 1) * na + g.ju) * f + i];
            const double c11 = (double)c.cube[((size_t)(g.jv + 1) * na + g.ju + 1) * f + i];
            S = (1.0 - g.gv) * ((1.0 - g.gu) * c00 + g.gu * c01)
              +        g.gv  * ((1.0 - g.gu) * c10 + g.gu * c11);
        }

        /* Eq. 11: front-end coupling and CMB */
        const double eta_front = c.eta_front_nu ? (double)c.eta_front_nu[i] : 1.0;
        double P = eta_front * S + tb.B_cmb[i];

        /* Eq. 12, stage 0: the atmosphere */
        P = eta_atm * P + (1.0 - eta_atm) * tb.B_atm[i];

        /* Eq. 12, optical stages k = 1..n_stage */
        for (int k = 0; k < c.n_stage; ++k) {
            const go_stage& st = c.stages[k];
            const double eta_k = st.eta_nu ? (double)st.eta_nu[i] : st.eta_scalar;
            const double J_k = st.couple_atmosphere
                ? (1.0 - eta_atm) * tb.B_atm[i] + eta_atm * tb.B_cmb[i]
                : tb.B_stage[k][i];
            P = eta_k * P + (1.0 - eta_k) * J_k;
        }
        P_out[i] = P;
        if (eta_out) eta_out[i] = eta_atm;
        if (S_out)   S_out[i] = S;
    }
}

/* Step 5, Eq. 16 with the rectangle rule on the uniform grid (R16). */
double contract_channel(const go_config& c, int ch, const double* P) {
    double acc = 0.0;
    const float* F = c.filt + (size_t)ch * c.n_freq;
    for (int i = 0; i < c.n_freq; ++i) acc += (double)F[i] * P[i];
    return c.dnu_hz * acc;
}

int check(const go_config* c) {
    if (!c || !c->az_rad || !c->el_rad || !c->daz_rad || !c->del_rad || !c->screen ||
        !c->atm_lut || !c->filt || !c->f_center_hz) return 1;
    if (c->n_freq <= 0 || c->n_samples <= 0 || c->n_spaxel <= 0 || c->n_chan <= 0 ||
        c->nx <= 0 || c->ny <= 0 || c->n_pwv < 2 || c->n_nu_lut < 2 || c->n_stage < 0) return 2;
    if (c->n_stage > 0 && !c->stages) return 1;
    if (c->cube && (c->n_az < 2 || c->n_el < 2)) return 2;
    if (c->pink_noise && (c->pink_n_stage < 1 || c->pink_n_stage > 8 || !c->pink_A ||
                          !c->pink_alpha || !c->pink_f_corner_hz)) return 3;
    return 0;
}

}  // namespace

extern "C" {

double go_planck(double nu_hz, double T_K) { return planck(nu_hz, T_K); }

void go_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    philox4x32_10(ctr, key, out);
}

double go_uniform(uint32_t w) { return uniform01(w); }

void go_normals4(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, double z[4]) {
    normals4(seed, c0, c1, c2, c3, z);
}

double go_photon_normal(uint64_t seed, uint32_t n, uint32_t s, uint32_t ch) { return photon_normal(seed, n, s, ch); }

void go_normals_bulk(uint64_t seed, uint32_t c0_begin, int64_t count, uint32_t c1, uint32_t c2,
                     uint32_t c3, double* z) {
    for (int64_t k = 0; k < count; ++k) normals4(seed, c0_begin + (uint32_t)k, c1, c2, c3, z + 4 * k);
}

double go_photon_sigma(double P_W, double f_center_hz, double dnu_eff_hz, double f_sample_hz) {
    return photon_sigma(P_W, f_center_hz, dnu_eff_hz, f_sample_hz);
}

void go_dnu_eff(const go_config* cfg, double* out) {
    for (int ch = 0; ch < cfg->n_chan; ++ch) out[ch] = dnu_eff_of(*cfg, ch);
}

void go_pink_coeffs(const go_config* cfg, int32_t spaxel, int32_t chan, double* phi, double* gain) {
    pink_coeffs(*cfg, spaxel, chan, phi, gain);
}

int go_geometry(const go_config* cfg, int64_t t_begin, int64_t t_count, go_georec* out) {
    if (int e = check(cfg)) return e;
    if (t_begin < 0 || t_count < 0 || t_begin + t_count > cfg->n_samples) return 4;
    const int ns = cfg->n_spaxel;
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < t_count * ns; ++r)
        row_geometry(*cfg, t_begin + r / ns, (int)(r % ns), out[r]);
    return 0;
}

int go_row_spectrum(const go_config* cfg, int64_t n, int32_t spaxel,
                    double* P_final, double* eta_atm, double* S_src) {
    if (int e = check(cfg)) return e;
    if (n < 0 || n >= cfg->n_samples || spaxel < 0 || spaxel >= cfg->n_spaxel) return 4;
    Tables tb; build_tables(*cfg, tb);
    go_georec g; row_geometry(*cfg, n, spaxel, g);
    row_spectrum(*cfg, tb, g, P_final, eta_atm, S_src);
    return 0;
}

int go_simulate_rows(const go_config* cfg, int64_t n_rows, const int64_t* t_idx,
                     const int32_t* s_idx, double* pkid, double* wn) {
    if (int e = check(cfg)) return e;
    const go_config& c = *cfg;
    Tables tb; build_tables(c, tb);
    std::vector<double> dnu_c(c.n_chan);
    for (int ch = 0; ch < c.n_chan; ++ch) dnu_c[ch] = dnu_eff_of(c, ch);
    int bad = 0;
#pragma omp parallel
    {
        std::vector<double> P(c.n_freq);
#pragma omp for schedule(dynamic, 4)
        for (int64_t r = 0; r < n_rows; ++r) {
            const int64_t n = t_idx[r]; const int s = s_idx[r];
            if (n < 0 || n >= c.n_samples || s < 0 || s >= c.n_spaxel) {
#pragma omp atomic write
                bad = 1;
                continue;
            }
            go_georec g; row_geometry(c, n, s, g);
            row_spectrum(c, tb, g, P.data(), nullptr, nullptr);
            for (int ch = 0; ch < c.n_chan; ++ch) {
                const double pk = contract_channel(c, ch, P.data());
                pkid[(size_t)r * c.n_chan + ch] = pk;
                if (wn) {
                    wn[(size_t)r * c.n_chan + ch] = photon_sigma(pk, c.f_center_hz[ch], dnu_c[ch], c.f_sample_hz)
                                                  * photon_normal(c.seed, (uint32_t)n, (uint32_t)s, (uint32_t)ch);
                }
            }
        }
    }
    return bad ? 4 : 0;
}

int go_pink_series(const go_config* cfg, int64_t n_det, const int32_t* s_idx, const int32_t* c_idx,
                   int64_t t_begin, int64_t t_count, double* out) {
    if (int e = check(cfg)) return e;
    if (!cfg->pink_noise) return 3;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t d = 0; d < n_det; ++d)
        pink_series(*cfg, s_idx[d], c_idx[d], t_begin, t_count, out + (size_t)d * t_count);
    return 0;
}

int go_simulate(const go_config* cfg, int64_t t_begin, int64_t t_count,
                double* tod, double* pkid, double* pwv) {
    if (int e = check(cfg)) return e;
    const go_config& c = *cfg;
    if (t_begin < 0 || t_count < 0 || t_begin + t_count > c.n_samples) return 4;
    Tables tb; build_tables(c, tb);
    const int ns = c.n_spaxel, nc = c.n_chan;
    std::vector<double> dnu_c(nc);
    for (int ch = 0; ch < nc; ++ch) dnu_c[ch] = dnu_eff_of(c, ch);

    /* steps 0-6a, rows independent */
#pragma omp parallel
    {
        std::vector<double> P(c.n_freq);
#pragma omp for schedule(dynamic, 4)
        for (int64_t r = 0; r < t_count * ns; ++r) {
            const int64_t n = t_begin + r / ns; const int s = (int)(r % ns);
            go_georec g; row_geometry(c, n, s, g);
            if (pwv) pwv[r] = g.pwv_mm;
            if (!tod && !pkid) continue;
            row_spectrum(c, tb, g, P.data(), nullptr, nullptr);
            for (int ch = 0; ch < nc; ++ch) {
                const double pk = contract_channel(c, ch, P.data());          /* Eq. 16 */
                if (pkid) pkid[(size_t)r * nc + ch] = pk;
                if (tod) {
                    double wn = 0.0;
                    if (c.photon_noise) {                                      /* Eq. 18-19 */
                        wn = photon_sigma(pk, c.f_center_hz[ch], dnu_c[ch], c.f_sample_hz)
                           * photon_normal(c.seed, (uint32_t)n, (uint32_t)s, (uint32_t)ch);
                    }
                    tod[(size_t)r * nc + ch] = pk + wn;
                }
            }
        }
    }
    /* step 6b + Eq. 21: tod = (P_KID + P_wn) + P_pn */
    if (tod && c.pink_noise) {
#pragma omp parallel
        {
            std::vector<double> pn((size_t)t_count);
#pragma omp for schedule(dynamic, 1)
            for (int64_t d = 0; d < (int64_t)ns * nc; ++d) {
                const int s = (int)(d / nc), ch = (int)(d % nc);
                pink_series(c, s, ch, t_begin, t_count, pn.data());
                for (int64_t k = 0; k < t_count; ++k)
                    tod[((size_t)k * ns + s) * nc + ch] += pn[k];
            }
        }
    }
    return 0;
}

int go_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
