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
// [26] |c|^2 beyond which a particle's drift is re-evaluated in fp64 (see upd_far_kernel in update.cu)
#pragma once
#include "common.cuh"

#define UPD_NC 28                  // floats of per-cell constants

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
    // [26]: in fp32 a drift term T costs ~6e-8 |T| of absolute error; the quadratic and cubic terms of a particle far out in
    // the cell's distribution, (1-E1) tau |gamma| c^2 and (1-E1) tau eps2 |c|^3, stay below 3 sqrt(theta) (error < 2e-7
    // sqrt(theta)) as long as |c|^2 < min(3 s / (kap |gamma|), (3 s / (kap eps2))^(2/3)); never below (5 sigma)^2 = 25 theta,
    // up to where the terms are a few thermal speeds in any physical state.  Equilibrium cells (eps2, gamma ~ 0): infinity.
    const double kap = (1.0 - E1) * tau, s3 = 3.0 * sqrt(theta);
    const double gmax = fmax(fabs((double)cf[6]), fmax(fabs((double)cf[7]), fabs((double)cf[8])));
    double far2 = fmin(gmax > 0.0 ? s3 / (kap * gmax) : INFINITY, eps2 > 0.0 ? cbrt((s3 / (kap * eps2)) * (s3 / (kap * eps2))) : INFINITY);
    far2 = fmin(fmax(far2, 25.0 * theta), 3.0e38);
    o4[6] = make_float4((float)(tau * tau * (1.0 - E1) * (1.0 - E1) * i3t), (float)(2.0 * tau * (E1 - E2) * i3t), (float)far2, 0.0f);
    return 0u;
}
