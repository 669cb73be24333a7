// gt_geometry.cuh -- steps 0-1 and the index part of steps 2-3 (Eq. 9-10).
//
// One thread per row (sample n, spaxel s).  HBM-bound and tiny (< 1 % of the path): 4 screen
// taps + ~100 B of per-sample/per-spaxel constants in, one 32-byte RowParam out.
//
// "Canonical geometry arithmetic": every + - * / below is a separately rounded
// IEEE-754 binary64 operation (__dadd_rn/__dmul_rn/__ddiv_rn are never contracted into FMAs),
// in the order DESIGN.md fixes, and the transcendental inputs (tan/sin/cos per sample and per
// spaxel) come from the host's libm at plan time.  The integer cell indices are therefore the
// IEEE ones on any machine, which is what makes "index, scan and RNG counters bit-exact" a
// meaningful gate.
#pragma once
#include "gt_common.cuh"
#include "../../include/gateau_b200.h"

namespace gt {

struct GeoParams {
    // per-sample tables (device, double): tan(az), tan(el), sin(el0+el), cos(el0+el), az, el
    const double *tan_az, *tan_el, *sinE, *cosE, *az, *el;
    // per-spaxel tables (device, double)
    const double *tan_daz, *tan_del, *sin_del, *cos_del, *daz, *del;
    int32_t n_spaxel;
    double f_sample;
    // screen
    const float* screen; int32_t nx, ny;
    double dx, dy, h_col, wind, pwv0_a, pwv0_b;
    // LUT in PWV
    int32_t n_pwv; double lut_pwv0, lut_dpwv;
    // source grid
    int32_t has_cube, n_az, n_el;
    double az_min, daz_grid, el_min, del_grid;
};

__device__ __forceinline__ int64_t pmod64(int64_t a, int64_t m) {
    const int64_t r = a % m;
    return r < 0 ? r + m : r;
}

// rows r = 0 .. n_rows-1 of the chunk starting at sample t0: n = t0 + r / n_spaxel, s = r % n_spaxel.
__global__ void __launch_bounds__(256)
geometry_kernel(GeoParams g, int64_t t0, int64_t n_rows, RowParam* __restrict__ rows,
                float* __restrict__ pwv_out, gt_georec* __restrict__ rec_out,
                unsigned long long* __restrict__ counters) {       // [3] rows outside the cube, PWV below / above the LUT (NULL ok)
    const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_rows) return;
    const unsigned active = __activemask();
    const int64_t n = t0 + r / g.n_spaxel;
    const int s = (int)(r % g.n_spaxel);

    const double t = __ddiv_rn((double)n, g.f_sample);

    // tan(phi(t) + dphi_s), tan(theta(t) + dtheta_s) by the addition formula
    const double ta_n = g.tan_az[n], ta_s = g.tan_daz[s];
    const double te_n = g.tan_el[n], te_s = g.tan_del[s];
    const double tan_a = __ddiv_rn(__dadd_rn(ta_n, ta_s), __dsub_rn(1.0, __dmul_rn(ta_n, ta_s)));
    const double tan_e = __ddiv_rn(__dadd_rn(te_n, te_s), __dsub_rn(1.0, __dmul_rn(te_n, te_s)));

    // Eq. 9: frozen-flow screen coordinates, wind along +x, boresight(t=0) on the screen centre
    const double x = __dadd_rn(__dmul_rn(g.h_col, tan_a), __dmul_rn(g.wind, t));
    const double y = __dmul_rn(g.h_col, tan_e);
    const double u = __dadd_rn(__ddiv_rn(x, g.dx), __dmul_rn(0.5, (double)g.nx));
    const double v = __dadd_rn(__ddiv_rn(y, g.dy), __dmul_rn(0.5, (double)g.ny));
    const double fl_u = floor(u), fl_v = floor(v);
    const double fu = __dsub_rn(u, fl_u), fv = __dsub_rn(v, fl_v);
    const int64_t iu = (int64_t)fl_u, iv = (int64_t)fl_v;
    const int64_t iu0 = pmod64(iu, g.nx), iu1 = pmod64(iu + 1, g.nx);
    const int64_t iv0 = pmod64(iv, g.ny), iv1 = pmod64(iv + 1, g.ny);

    // bilinear PWV + drift PWV_0(t)
    const double s00 = (double)__ldg(g.screen + (size_t)iv0 * g.nx + iu0);
    const double s01 = (double)__ldg(g.screen + (size_t)iv0 * g.nx + iu1);
    const double s10 = (double)__ldg(g.screen + (size_t)iv1 * g.nx + iu0);
    const double s11 = (double)__ldg(g.screen + (size_t)iv1 * g.nx + iu1);
    const double omfu = __dsub_rn(1.0, fu), omfv = __dsub_rn(1.0, fv);
    const double row0 = __dadd_rn(__dmul_rn(omfu, s00), __dmul_rn(fu, s01));
    const double row1 = __dadd_rn(__dmul_rn(omfu, s10), __dmul_rn(fu, s11));
    const double pwv = __dadd_rn(__dadd_rn(__dmul_rn(omfv, row0), __dmul_rn(fv, row1)),
                                 __dadd_rn(g.pwv0_a, __dmul_rn(g.pwv0_b, t)));

    // LUT cell in PWV, clamped (R13)
    double q = __ddiv_rn(__dsub_rn(pwv, g.lut_pwv0), g.lut_dpwv);
    const bool clamp_lo = !(q >= 0.0), clamp_hi = q > (double)(g.n_pwv - 1);     // a NaN is clamped to row 0 as well: every index stays in bounds
    if (clamp_lo) q = 0.0;
    if (clamp_hi) q = (double)(g.n_pwv - 1);
    int64_t ip = (int64_t)floor(q);
    if (ip > g.n_pwv - 2) ip = g.n_pwv - 2;
    if (ip < 0) ip = 0;
    const double fp = __dsub_rn(q, (double)ip);

    // Eq. 10 airmass: sin(E + dtheta_s) by the addition formula
    const double sinE = __dadd_rn(__dmul_rn(g.sinE[n], g.cos_del[s]), __dmul_rn(g.cosE[n], g.sin_del[s]));
    const double csc = __ddiv_rn(1.0, sinE);

    // source cell: flat grid, inclusive edges, zero outside
    int32_t ju = -1, jv = -1;
    double gu = 0.0, gv = 0.0;
    if (g.has_cube) {
        const double a = __dadd_rn(g.az[n], g.daz[s]);
        const double e = __dadd_rn(g.el[n], g.del[s]);
        const double us = __ddiv_rn(__dsub_rn(a, g.az_min), g.daz_grid);
        const double vs = __ddiv_rn(__dsub_rn(e, g.el_min), g.del_grid);
        if (!(us < 0.0 || us > (double)(g.n_az - 1) || vs < 0.0 || vs > (double)(g.n_el - 1))) {
            int64_t j0 = (int64_t)floor(us), j1 = (int64_t)floor(vs);
            if (j0 > g.n_az - 2) j0 = g.n_az - 2;
            if (j1 > g.n_el - 2) j1 = g.n_el - 2;
            ju = (int32_t)j0; jv = (int32_t)j1;
            gu = __dsub_rn(us, (double)j0); gv = __dsub_rn(vs, (double)j1);
        }
    }

    if (rows) {
        RowParam rp;
        rp.fp = (float)fp;
        rp.csc = (float)csc;
        rp.ip = (int32_t)ip;
        rp.pix = ju < 0 ? -1 : jv * g.n_az + ju;
        rp.w00 = (float)((1.0 - gv) * (1.0 - gu));
        rp.w01 = (float)((1.0 - gv) * gu);
        rp.w10 = (float)(gv * (1.0 - gu));
        rp.w11 = (float)(gv * gu);
        rows[r] = rp;
    }
    if (pwv_out) pwv_out[r] = (float)pwv;
    if (counters) {
        // diagnostics: one atomic per warp and event kind, only where the event occurs (both are rare)
        const unsigned b0 = __ballot_sync(active, g.has_cube && ju < 0), b1 = __ballot_sync(active, clamp_lo), b2 = __ballot_sync(active, clamp_hi);
        if ((threadIdx.x & 31) == __ffs(active) - 1) {
            if (b0) atomicAdd(counters + 0, (unsigned long long)__popc(b0));
            if (b1) atomicAdd(counters + 1, (unsigned long long)__popc(b1));
            if (b2) atomicAdd(counters + 2, (unsigned long long)__popc(b2));
        }
    }
    if (rec_out) {
        gt_georec o;
        o.n = n; o.iu0 = (int32_t)iu0; o.iv0 = (int32_t)iv0; o.ju = ju; o.jv = jv;
        o.ip = (int32_t)ip; o.pad_ = 0;
        o.fu = fu; o.fv = fv; o.gu = gu; o.gv = gv; o.fp = fp; o.pwv_mm = pwv; o.csc = csc;
        rec_out[r] = o;
    }
}

}  // namespace gt
