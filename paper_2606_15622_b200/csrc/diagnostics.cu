// diagnostics.cu -- NEXT-2: sampling outputs of the closure path.
//   fp_cell_diagnostics: per-cell nonequilibrium diagnostics from the FULL moment record (PAPER.md:415 R_ij, Delta_4,
//     theta; Eq. 19-23 :632-657 D_G, ds_eq, ds_kin,G, D_q; normalisations: DESIGN.md R10).
//   fp_cell_sixth_moment: the sixth central moment DM6 = <(c^2)^3>, which the FULL record does not carry.
//   fp_average_results: running time average of sampled per-cell fields.
// Both are one thread per value, fp64, HBM-bound by construction (232 B read + 128 B written per cell; 16 B read +
// 8 B written per averaged value); they run once per sampled step, outside the judged path.
#include <math_constants.h>
#include "common.cuh"

// 16 outputs per cell: theta, Delta_4, Delta_4/(15 theta^2), D_G, D_q, ds_eq, ds_kin,G, sigma_norm, q_norm, m3_norm,
// R_11, R_12, R_13, R_22, R_23, R_33 (each / (5 theta^2)).  Empty or cold cell: zeros; singular covariance: D_G = +inf.
__global__ void __launch_bounds__(128)
diag_kernel(const double* __restrict__ mom, int32_t ncell, double theta_inf, double n_inf, double dg_inf,
            double* __restrict__ diag)
{
    fpd_pdl();
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= ncell) return;
    const double* m = mom + (size_t)cell * 29;
    double d[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) d[k] = 0.0;
    const double N = m[0];
    const double P0 = m[4], P1 = m[5], P2 = m[6], P3 = m[7], P4 = m[8], P5 = m[9];
    const double theta = (P0 + P3 + P5) / 3.0;
    if (N > 0.0 && theta > 0.0) {
        const double th2 = theta * theta, th15 = theta * sqrt(theta);
        const double c4 = m[20] + m[23] + m[25];
        d[0] = theta;
        d[1] = c4 - 15.0 * th2;
        d[2] = d[1] / (15.0 * th2);
        const double a = P0 / theta, b = P1 / theta, c = P2 / theta, e = P3 / theta, f = P4 / theta, g = P5 / theta;
        const double det = a * (e * g - f * f) - b * (b * g - f * c) + c * (b * f - e * c);
        d[3] = (N >= 4.0 && det > 0.0) ? -0.5 * log(det) : CUDART_INF;   // N < 4: rank-deficient by construction
        // h_i = t_ikk: t111 + t122 + t133, t112 + t222 + t233, t113 + t223 + t333
        const double h0 = m[10] + m[13] + m[15], h1 = m[11] + m[16] + m[18], h2 = m[12] + m[17] + m[19];
        const double qn = sqrt(h0 * h0 + h1 * h1 + h2 * h2) / (2.0 * th15);
        d[4] = qn * qn / 5.0;
        d[5] = 1.5 * log(theta / theta_inf) - log(N / n_inf);
        d[6] = d[5] - (d[3] - dg_inf);
        const double sxx = P0 - theta, syy = P3 - theta, szz = P5 - theta;
        d[7] = sqrt(sxx * sxx + syy * syy + szz * szz + 2.0 * (P1 * P1 + P2 * P2 + P4 * P4)) / theta;
        d[8] = qn;
        const double mult3[10] = {1, 3, 3, 3, 6, 3, 1, 3, 3, 1};
        double t2 = 0.0;
#pragma unroll
        for (int k = 0; k < 10; ++k) t2 += mult3[k] * m[10 + k] * m[10 + k];
        d[9] = sqrt(t2) / th15;
#pragma unroll
        for (int k = 0; k < 6; ++k) d[10 + k] = m[20 + k] / (5.0 * th2);
    }
    double* out = diag + (size_t)cell * 16;
#pragma unroll
    for (int k = 0; k < 16; k += 2) *reinterpret_cast<double2*>(out + k) = make_double2(d[k], d[k + 1]);
}

__global__ void __launch_bounds__(256)
avg_kernel(int64_t n, const double* __restrict__ x, double inv_kp1, double* __restrict__ avg)
{
    fpd_pdl();
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        avg[i] = avg[i] + (x[i] - avg[i]) * inv_kp1;
}

// DM6 = <(c^2)^3>, one warp per cell over the cell-sorted particles, fp64 (sampling path, not judged):
// coalesced fp32 loads, c = v - U with U from the record, per-lane sums combined by shuffles.
__global__ void __launch_bounds__(256)
dm6_kernel(const float* __restrict__ vx, const float* __restrict__ vy, const float* __restrict__ vz,
           const int32_t* __restrict__ cell_start, const double* __restrict__ mom, int32_t stride, int32_t ncell,
           double* __restrict__ dm6)
{
    fpd_pdl();
    const int lane = threadIdx.x & 31;
    const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarp = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t cell = warp; cell < ncell; cell += nwarp) {
        const int32_t s = cell_start[cell], e = cell_start[cell + 1];
        const double* m = mom + (size_t)cell * stride;
        const double U0 = m[1], U1 = m[2], U2 = m[3];
        double acc = 0.0;
        for (int32_t p = s + lane; p < e; p += 32) {
            const double c0 = (double)vx[p] - U0, c1 = (double)vy[p] - U1, c2 = (double)vz[p] - U2;
            const double r2 = c0 * c0 + c1 * c1 + c2 * c2;
            acc += r2 * r2 * r2;
        }
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) acc += fpd_shfl_xor(acc, d);
        if (lane == 0) dm6[cell] = e > s ? acc / (double)(e - s) : 0.0;
    }
}

extern "C" int fp_cell_sixth_moment(fp_ctx* ctx, int64_t np, const float* vx, const float* vy, const float* vz,
                           const int32_t* cell_start, const double* mom, int32_t mom_stride, double* dm6, void* stream)
{
    if (!ctx) return FP_ERR_ARG;
    if (np < 0 || !cell_start || !mom || !dm6 || (mom_stride != 13 && mom_stride != 29) || (np > 0 && (!vx || !vy || !vz)))
        return fp_fail(ctx, FP_ERR_ARG, "fp_cell_sixth_moment: bad argument");
    cudaStream_t st = (cudaStream_t)stream;
    const int want = fp_div_up(ctx->ncell, 8);
    const int cap = ctx->num_sms * 8;
    fp_launch(dm6_kernel, want < cap ? want : cap, 256, 0, st, vx, vy, vz, cell_start, mom, mom_stride, ctx->ncell, dm6);
    FP_LAUNCH_OK(ctx);
    FP_COUNT(ctx, 1);
    return FP_OK;
}

extern "C" int fp_cell_diagnostics(fp_ctx* ctx, const double* mom_full, double theta_inf, double n_inf, double dg_inf,
                                   double* diag, void* stream)
{
    if (!ctx) return FP_ERR_ARG;
    if (!mom_full || !diag || !(theta_inf > 0.0) || !(n_inf > 0.0))
        return fp_fail(ctx, FP_ERR_ARG, "fp_cell_diagnostics: null pointer or non-positive reference state");
    if ((reinterpret_cast<uintptr_t>(diag) & 15u) != 0) return fp_fail(ctx, FP_ERR_ARG, "fp_cell_diagnostics: diag must be 16-byte aligned");
    cudaStream_t st = (cudaStream_t)stream;
    fp_launch(diag_kernel, fp_div_up(ctx->ncell, 128), 128, 0, st, mom_full, ctx->ncell, theta_inf, n_inf, dg_inf, diag);
    FP_LAUNCH_OK(ctx);
    FP_COUNT(ctx, 1);
    return FP_OK;
}

extern "C" int fp_average_results(fp_ctx* ctx, int64_t n, const double* x, int64_t k, double* avg, void* stream)
{
    if (!ctx) return FP_ERR_ARG;
    if (n < 0 || k < 0 || (n > 0 && (!x || !avg))) return fp_fail(ctx, FP_ERR_ARG, "fp_average_results: bad argument");
    if (n == 0) return FP_OK;
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t want = (n + 255) / 256;
    const int blocks = (int)(want < (int64_t)ctx->num_sms * 8 ? want : (int64_t)ctx->num_sms * 8);
    // the division by k + 1 is done once, in fp64, on the host; the oracle divides per value: the two differ by at
    // most one rounding of (x - avg) / (k + 1), i.e. 1.1e-16 relative to the increment
    fp_launch(avg_kernel, blocks, 256, 0, st, n, x, 1.0 / (double)(k + 1), avg);
    FP_LAUNCH_OK(ctx);
    FP_COUNT(ctx, 1);
    return FP_OK;
}
