// upd_prep.cuh -- the per-cell constants of the velocity update (Sec. 2.3, Eqs. 7-10; R5).
//
// One thread turns a cell's moment record, its nine coefficients and tau into UPD_NC fp32 constants that
// update_warp_kernel reads.  The function is shared by upd_prep_kernel (stand-alone fp_velocity_update) and by the
// closure kernels, which call it right after they produced the coefficients when they run inside fp_step: the
// thread already holds the record, tau and the coefficients, so the separate one-thread-per-cell kernel and its
// 11 us latency chain disappear from the step.
//
// layout of the constants: [0..2] U_hi, [3..5] U_lo, [6..11] B = C + I/tau (11,12,13,22,23,33), [12..14] gamma,
// [15..17] eps2*h, [18] eps2, [19] 3 theta, [20] E1, [21] (1-E1) tau, [22] sqrt(theta (1-E2)), [23] active,
// [24] tau^2 (1-E1)^2 / (3 theta), [25] 2 tau (E1-E2) / (3 theta),
// [26] |c|^2 beyond which a particle's drift is re-evaluated in fp64 (upd_far_cell in update.cu), [27] the same for the paths
// that give a cell all 32 lanes and subtract U as hi + lo (no bulk-velocity rounding shift)
#pragma once
#include "common.cuh"

#define UPD_NC 28                  // floats of per-cell constants
#ifndef UPD_FAR_S
#define UPD_FAR_S 1.5                 // drift terms the fast path accepts, in thermal speeds (see [26] below)
#endif
#ifndef UPD_FAR_FLOOR
#define UPD_FAR_FLOOR 1.0            // ... but never a range below sigma^2 (4.0 left particles at 1.6-2 sigma of bimodal
                                     // Mach-9 cells, cubic term ~5 thermal speeds, on the fast path: up to 1.85x the tolerance;
                                     // the step time does not depend on it: those cells hold a particle beyond 2 sigma anyway)
#endif

// rec: the cell's record (13 or 29 doubles, any address space), cf: its nine coefficients as stored in fp32.
// Returns FP_FLAG_SKIPPED when the cell holds particles that the update leaves untouched, else 0.
__device__ __forceinline__ uint32_t upd_prep_cell(const double* rec, int stride, const float* cf, double tau, float dt,
                                                  float eps2_scale, float* __restrict__ o)
{
    const double n = rec[0];
    const double theta = (rec[4] + rec[7] + rec[9]) / 3.0;
    const bool active = n >= 2.0 && (theta > 0.0) && isfinite(theta);
    if (!active) {
        o[23] = 0.0f;
        return n > 0.0 ? (uint32_t)FP_FLAG_SKIPPED : 0u;
    }
    const double U0 = rec[1], U1 = rec[2], U2 = rec[3];
    const float Uh0 = (float)U0, Uh1 = (float)U1, Uh2 = (float)U2;
    double h0, h1, h2;
    if (stride == 13) { h0 = rec[10]; h1 = rec[11]; h2 = rec[12]; }
    else { h0 = rec[10] + rec[13] + rec[15]; h1 = rec[11] + rec[16] + rec[18]; h2 = rec[12] + rec[17] + rec[19]; }
    // one thread walks this chain alone, so keep it short: two reciprocals, one exp, one sqrt
    const double itau = 1.0 / tau, ith = 1.0 / theta;
    const double E1 = exp(-(double)dt * itau), E2 = E1 * E1;
    const double p0 = rec[4] * ith - 1.0, p1 = rec[5] * ith, p2 = rec[6] * ith, p3 = rec[7] * ith - 1.0,
                 p4 = rec[8] * ith, p5 = rec[9] * ith - 1.0;
    const double eps2 = (double)eps2_scale * fabs(p0 * (p3 * p5 - p4 * p4) - p1 * (p1 * p5 - p4 * p2) + p2 * (p1 * p4 - p3 * p2)) * itau * ith;
    const double i3t = ith * (1.0 / 3.0);
    float4* o4 = reinterpret_cast<float4*>(o);      // cellc rows are 112 B apart and 16 B aligned
    o4[0] = make_float4(Uh0, Uh1, Uh2, (float)(U0 - (double)Uh0));
    o4[1] = make_float4((float)(U1 - (double)Uh1), (float)(U2 - (double)Uh2), (float)((double)cf[0] + itau), cf[1]);
    o4[2] = make_float4(cf[2], (float)((double)cf[3] + itau), cf[4], (float)((double)cf[5] + itau));
    o4[3] = make_float4(cf[6], cf[7], cf[8], (float)(eps2 * h0));
    o4[4] = make_float4((float)(eps2 * h1), (float)(eps2 * h2), (float)eps2, (float)(3.0 * theta));
    o4[5] = make_float4((float)E1, (float)((1.0 - E1) * tau), (float)sqrt(theta * (1.0 - E2)), 1.0f);
    // [26]: in fp32 a drift term T costs ~6e-8 |T| of absolute error per rounding, and the terms of N cancel against each
    // other.  A particle stays on the fast path while its linear, quadratic and cubic terms, (1-E1) tau |B| |c|,
    // (1-E1) tau |gamma| c^2 and (1-E1) tau eps2 |c|^3, each stay below UPD_FAR_S thermal speeds, i.e. while
    // |c|^2 < min((s / (kap |B|))^2, s / (kap |gamma|), (s / (kap eps2))^(2/3)) with s = UPD_FAR_S sqrt(theta); the range is
    // never taken below UPD_FAR_FLOOR theta.  Equilibrium cells (B, gamma, eps2 ~ 0): infinity.  (Randomised comparison
    // with the oracle: at 3 thermal speeds and a floor of 25 theta, cells of a few particles -- whose eps2 is
    // O(1 / (tau theta)) -- missed the 1e-6 tolerance by up to 2x.)
    const double kap = (1.0 - E1) * tau, s3 = UPD_FAR_S * sqrt(theta);
    const double gmax = fmax(fabs((double)cf[6]), fmax(fabs((double)cf[7]), fabs((double)cf[8])));
    double far2_hl;
    double far2 = fmin(gmax > 0.0 ? s3 / (kap * gmax) : INFINITY, eps2 > 0.0 ? cbrt((s3 / (kap * eps2)) * (s3 / (kap * eps2))) : INFINITY);
    {   // the linear term (1-E1) tau |B c| <= kap |B|_inf |c| as well (B = C + I/tau vanishes in equilibrium)
        const double b0 = fabs((double)cf[0] + itau) + fabs((double)cf[1]) + fabs((double)cf[2]);
        const double b1 = fabs((double)cf[1]) + fabs((double)cf[3] + itau) + fabs((double)cf[4]);
        const double b2 = fabs((double)cf[2]) + fabs((double)cf[4]) + fabs((double)cf[5] + itau);
        const double bmax = fmax(b0, fmax(b1, b2));
        if (bmax > 0.0) far2 = fmin(far2, (s3 / (kap * bmax)) * (s3 / (kap * bmax)));
        far2 = fmin(fmax(far2, UPD_FAR_FLOOR * theta), 3.0e38);
        // The fast path subtracts U as ONE fp32 number: every c of the cell is off by up to d = 2^-24 |U|.  The drift's
        // Jacobian |dN/dc| <= |B| + 2 |gamma| |c| + 3 eps2 c^2 multiplies that shift: a particle stays on the fast path while
        // (1-E1) tau |dN/dc| d < 2e-7 thermal speeds.  Binding in hypersonic cells with a strongly non-linear drift (two- and
        // three-particle cells, whose eps2 is O(1 / (tau theta))): there the bound is below every |c| and the cell always
        // takes the fp64 path.
        const double du = 5.97e-8 * fmax(fabs(U0), fmax(fabs(U1), fabs(U2)));
        const double T = 2.0e-7 * sqrt(theta), A0 = kap * bmax * du, A1 = 2.0 * kap * gmax * du, A2 = 3.0 * kap * eps2 * du;
        double xu = INFINITY;                                // the |c| at which A2 x^2 + A1 x + A0 reaches T
        if (A0 >= T) xu = 0.0;
        else if (A2 > 0.0) xu = (-A1 + sqrt(A1 * A1 + 4.0 * A2 * (T - A0))) / (2.0 * A2);
        else if (A1 > 0.0) xu = (T - A0) / A1;
        far2_hl = far2;                                      // [27]: the range of the paths that subtract U as hi + lo (32 lanes per cell)
        far2 = fmin(far2, xu * xu);
    }
    o4[6] = make_float4((float)(tau * tau * (1.0 - E1) * (1.0 - E1) * i3t), (float)(2.0 * tau * (E1 - E2) * i3t), (float)far2, (float)far2_hl);
    return 0u;
}
