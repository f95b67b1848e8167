// closure_exact.cu -- a4: exact cubic-FP closure.  Per cell, assemble the 9x9 moment-matching system of
// PAPER.md Eq. 10 (:121) / Table 1 (:130-136) for y = (c11,c12,c13,c22,c23,c33,gamma1,gamma2,gamma3) and solve it
// with partial pivoting.  The blocks the paper does not print (X^T, Z, Q6, R3) and the garbled rows of V are
// derived from the matching condition Eq. 3 (:69) with the drift of Eq. 8 (:102), the diffusion theta/tau and
// Maxwell-molecule relaxation rates 2/tau (stress) and 4/(3 tau) (heat flux, Pr = 2/3 :37, :87) -- DESIGN.md R2:
//   stress rows (i<=j):  c_ik P_kj + c_jk P_ki + gam_i h_j + gam_j h_i = -(2/tau) P_ij + 2 eps2 F_ij
//   heat rows:           c_ik h_k + 2 c_kl t_kli + gam_i (F - 9 theta^2) + 2 gam_k (F_ki - 3 theta P_ki)
//                          = -(4/(3 tau)) h_i + eps2 (3 g_i - 3 theta h_i - 2 P_ik h_k)
// assembled in scaled variables (velocity unit sqrt(theta), time unit tau; R3-a), so all entries are O(1).
//
// Mapping: 16 lanes per cell, lane r < 9 owns row r (9 matrix entries + rhs in registers, fp64).  The system never
// touches HBM: 232 B/cell in, 40 B/cell out.  Pivot search = 4-step butterfly arg-max; the pivot row is
// broadcast by shuffles; rows are never swapped physically (a row remembers the step it was used as pivot).
#include "common.cuh"

#define CE_THREADS 128
#define CE_G 16

__host__ __device__ constexpr int ce_s2(int i, int j) { return i <= j ? i * (5 - i) / 2 + j : j * (5 - j) / 2 + i; }
__host__ __device__ constexpr int ce_s3(int i, int j, int k)
{
    // sort three indices, then 111,112,113,122,123,133,222,223,233,333
    int a = i, b = j, c = k, s = 0;
    if (a > b) { s = a; a = b; b = s; }
    if (b > c) { s = b; b = c; c = s; }
    if (a > b) { s = a; a = b; b = s; }
    return a == 0 ? ce_s2(b, c) : (a == 1 ? 3 + ce_s2(b, c) : 9);
}

struct ce_scaled {   // scaled moments of one cell
    double P[6], t[10], Fij[6], g[3], h[3], F, e2;
};

// row R of the scaled system: a[0..8] matrix entries, a[9] right-hand side
template <int R>
__device__ __forceinline__ void ce_build_row(const ce_scaled& m, double (&a)[10])
{
#pragma unroll
    for (int k = 0; k < 10; ++k) a[k] = 0.0;
    if (R < 6) {
        constexpr int i = R < 3 ? 0 : (R < 5 ? 1 : 2);
        constexpr int j = R < 3 ? R : (R < 5 ? R - 2 : 2);
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            a[ce_s2(i, k)] += m.P[ce_s2(k, j)];
            a[ce_s2(j, k)] += m.P[ce_s2(k, i)];
        }
        a[6 + i] += m.h[j];
        a[6 + j] += m.h[i];
        a[9] = -2.0 * m.P[R] + 2.0 * m.e2 * m.Fij[R];
    } else {
        constexpr int i = R - 6;
#pragma unroll
        for (int k = 0; k < 3; ++k) a[ce_s2(i, k)] += m.h[k];
#pragma unroll
        for (int k = 0; k < 3; ++k)
#pragma unroll
            for (int l = 0; l < 3; ++l) a[ce_s2(k, l)] += 2.0 * m.t[ce_s3(k, l, i)];
        a[6 + i] += m.F - 9.0;
        double Ph = 0.0;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            a[6 + k] += 2.0 * (m.Fij[ce_s2(k, i)] - 3.0 * m.P[ce_s2(k, i)]);
            Ph += m.P[ce_s2(i, k)] * m.h[k];
        }
        a[9] = -(4.0 / 3.0) * m.h[i] + m.e2 * (3.0 * m.g[i] - 3.0 * m.h[i] - 2.0 * Ph);
    }
}

__global__ void __launch_bounds__(CE_THREADS)
closure_exact_kernel(const double* __restrict__ mom, const float* __restrict__ tau_cell, float tau_scalar,
                     float eps2_scale, int32_t min_count, int32_t ncell, float* __restrict__ coef,
                     uint32_t* __restrict__ flags, double* __restrict__ kappa_est)
{
    const int lane = threadIdx.x & 31;
    const int gl = lane & (CE_G - 1);
    const int gbase = lane & ~(CE_G - 1);
    const int64_t cell = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / CE_G;
    const bool have = cell < ncell;
    const double* rec = mom + (size_t)(have ? cell : 0) * 29;
    const double n = rec[0];
    const double tau = (double)(tau_cell ? tau_cell[have ? cell : 0] : tau_scalar);
    double theta = (rec[4] + rec[7] + rec[9]) / 3.0;
    const bool theta_ok = (theta > 0.0) && isfinite(theta);
    const double th = theta_ok ? theta : 1.0;            // keep the arithmetic finite on cells that fall back
    ce_scaled m;
    {
        const double s1 = sqrt(th), s2 = th, s3 = th * s1, s4 = th * th, s5 = s4 * s1;
#pragma unroll
        for (int k = 0; k < 6; ++k) { m.P[k] = rec[4 + k] / s2; m.Fij[k] = rec[20 + k] / s4; }
#pragma unroll
        for (int k = 0; k < 10; ++k) m.t[k] = rec[10 + k] / s3;
#pragma unroll
        for (int k = 0; k < 3; ++k) m.g[k] = rec[26 + k] / s5;
        m.F = 0.0;
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            m.h[i] = 0.0;
#pragma unroll
            for (int k = 0; k < 3; ++k) m.h[i] += m.t[ce_s3(i, k, k)];
            m.F += m.Fij[ce_s2(i, i)];
        }
        // eps2_hat = eps2 tau theta = eps2_scale |det(P/theta - I)|   (R2-e)
        const double a = m.P[0] - 1.0, b = m.P[1], c = m.P[2], d = m.P[3] - 1.0, e = m.P[4], f = m.P[5] - 1.0;
        m.e2 = (double)eps2_scale * fabs(a * (d * f - e * e) - b * (b * f - e * c) + c * (b * e - d * c));
    }
    double a[10];
    switch (gl) {
        case 0: ce_build_row<0>(m, a); break;
        case 1: ce_build_row<1>(m, a); break;
        case 2: ce_build_row<2>(m, a); break;
        case 3: ce_build_row<3>(m, a); break;
        case 4: ce_build_row<4>(m, a); break;
        case 5: ce_build_row<5>(m, a); break;
        case 6: ce_build_row<6>(m, a); break;
        case 7: ce_build_row<7>(m, a); break;
        case 8: ce_build_row<8>(m, a); break;
        default:
#pragma unroll
            for (int k = 0; k < 10; ++k) a[k] = 0.0;
    }
    __syncwarp();
    // norms for the condition estimate: ||A||_inf and ||b||_inf
    double rowsum = 0.0;
#pragma unroll
    for (int k = 0; k < 9; ++k) rowsum += fabs(a[k]);
    double bmax = fabs(a[9]);
#pragma unroll
    for (int d = CE_G / 2; d >= 1; d >>= 1) {
        rowsum = fmax(rowsum, fpd_shfl_xor(rowsum, d));
        bmax = fmax(bmax, fpd_shfl_xor(bmax, d));
    }
    // ---- elimination with partial pivoting, row per lane
    bool used = gl >= 9;
    int piv_lane[9];
    double minpiv = INFINITY, maxpiv = 0.0;
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        double cand = used ? -1.0 : fabs(a[k]);
        if (!(cand >= -1.0)) cand = 0.0;                  // NaN
        double best = cand;
        int bl = gl;
#pragma unroll
        for (int d = CE_G / 2; d >= 1; d >>= 1) {
            const double ob = fpd_shfl_xor(best, d);
            const int ol = __shfl_xor_sync(0xffffffffu, bl, d);
            if (ob > best || (ob == best && ol < bl)) { best = ob; bl = ol; }
        }
        piv_lane[k] = bl;
        minpiv = fmin(minpiv, best);
        maxpiv = fmax(maxpiv, best);
        double pr[10];
#pragma unroll
        for (int j = k; j < 10; ++j) pr[j] = fpd_shfl(a[j], gbase + bl);
        if (gl == bl) used = true;
        else if (!used) {
            const double f = a[k] / pr[k];
#pragma unroll
            for (int j = k + 1; j < 10; ++j) a[j] -= f * pr[j];
            a[k] = 0.0;
        }
    }
    // ---- back substitution: the row used at step k yields y[k]
    double y[9];
#pragma unroll
    for (int k = 8; k >= 0; --k) {
        double s = a[9];
#pragma unroll
        for (int j = k + 1; j < 9; ++j) s -= a[j] * y[j];
        s /= a[k];
        y[k] = fpd_shfl(s, gbase + piv_lane[k]);
    }
    bool finite = true;
    double ymax = 0.0;
#pragma unroll
    for (int k = 0; k < 9; ++k) { finite = finite && isfinite(y[k]); ymax = fmax(ymax, fabs(y[k])); }
    // ---- policy (R3-c) and output
    uint32_t flag = 0;
    double out = 0.0;
    const bool langevin_row = (gl == 0 || gl == 3 || gl == 5);
    const double lang = langevin_row ? -1.0 / tau : 0.0;
    double kap = 0.0;
    if (!(n > 0.0)) { flag = FP_FLAG_EMPTY; out = 0.0; }
    else if (n < (double)min_count) { flag = FP_FLAG_LOWCOUNT; out = lang; }
    else if (!theta_ok) { flag = FP_FLAG_SINGULAR; out = lang; }
    else if (!(minpiv >= 1e-14) || !finite) { flag = FP_FLAG_SINGULAR; out = lang; }
    else {
        const double k1 = bmax > 0.0 ? rowsum * ymax / bmax : 0.0;
        const double k2 = maxpiv / minpiv;
        kap = fmax(k1, k2);
        if (!(kap < 1e8)) flag = FP_FLAG_ILLCOND;
        double yk = 0.0;
#pragma unroll
        for (int k = 0; k < 9; ++k) if (gl == k) yk = y[k];
        out = (gl < 6) ? yk / tau : yk / (tau * sqrt(theta));
    }
    if (have) {
        if (gl < 9) coef[(size_t)cell * 9 + gl] = (float)out;
        if (gl == 0) { flags[cell] = flag; if (kappa_est) kappa_est[cell] = kap; }
    }
}

extern "C" int fp_closure_exact(fp_ctx* ctx, const double* mom_full, const float* tau_cell, float* coef,
                                uint32_t* flags, double* kappa_est, void* stream)
{
    if (!ctx) return FP_ERR_ARG;
    if (!mom_full || !coef || !flags) return fp_fail(ctx, FP_ERR_ARG, "fp_closure_exact: null pointer");
    const int32_t ncell = ctx->ncell;
    const int cells_per_block = CE_THREADS / CE_G;
    const int blocks = fp_div_up(ncell, cells_per_block);
    closure_exact_kernel<<<blocks, CE_THREADS, 0, (cudaStream_t)stream>>>(mom_full, tau_cell, ctx->p.tau, ctx->p.eps2_scale,
                                                                         ctx->p.min_count, ncell, coef, flags, kappa_est);
    FP_LAUNCH_OK(ctx);
    FP_COUNT(ctx, 1);
    return FP_OK;
}
