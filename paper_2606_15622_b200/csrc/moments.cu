// moments.cu -- a3: segmented gather of per-cell velocity moments over cell-sorted particles
// (PAPER.md:124 moment definition, :215-216 M1-M5, :243 LITE, :181 plain 1/N mean; R0).
//
// HBM-bound by design: 12 B/particle read once from DRAM + one record per cell written.
// Layout of the work: a group of G lanes (G = 4..32, chosen from the mean particles per cell) owns one cell, so a
// warp works on 32/G cells at once.  Two passes over the cell's particles (the second pass re-reads L1/L2):
//   pass 1: S = sum (v - v_pivot) in fp32 about the cell's first particle (differences are thermal-sized, so fp32
//           holds them to ~6e-8 of the thermal speed even at Mach 10), reduced across the group in fp64;
//           U = v_pivot + S/N (fp64), m = S/N.
//   pass 2: c = (v - v_pivot) - m in fp32, monomials and per-lane partial sums in fp32 (<= a few tens of terms
//           per lane), then converted to fp64 and reduced across the group with a transposing butterfly that
//           leaves record slot k in lane k*G/32: the store is the record layout itself.
// Cells larger than CHUNK particles are processed chunk by chunk with fp64 accumulation between chunks.
#include "common.cuh"

#define MOM_THREADS 256
#define MOM_CHUNK_PER_LANE 64

template <int G, bool FULL>
__global__ void __launch_bounds__(MOM_THREADS)
moments_kernel(const float* __restrict__ vx, const float* __restrict__ vy, const float* __restrict__ vz,
               const int32_t* __restrict__ cell_start, int32_t ncell, double* __restrict__ mom)
{
    constexpr int NP = FULL ? 32 : 16;          // padded record length
    constexpr int NREC = FULL ? 29 : 13;
    constexpr int PER = NP / G > 0 ? NP / G : 1;  // record slots per lane after the transposing reduction
    static_assert(NP >= G, "group wider than the padded record");
    const int lane = threadIdx.x & 31;
    const int gl = lane & (G - 1);               // lane inside the group
    const int64_t group0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / G;
    const int64_t ngroups = (int64_t)gridDim.x * blockDim.x / G;
    // all groups of a warp iterate together (shuffles need the whole warp): loop bound is warp-uniform
    const int64_t iters = ((int64_t)ncell + ngroups - 1) / ngroups;
    for (int64_t it = 0; it < iters; ++it) {
        const int64_t cell = group0 + it * ngroups;
        const bool have = cell < ncell;
        int32_t s = 0, e = 0;
        if (have) { s = cell_start[cell]; e = cell_start[cell + 1]; }
        const int32_t n = e - s;
        // ---- pass 1: mean about the pivot
        float px = 0.f, py = 0.f, pz = 0.f;
        if (n > 0) { px = vx[s]; py = vy[s]; pz = vz[s]; }
        double S0 = 0.0, S1 = 0.0, S2 = 0.0;
        const int32_t nmax = __reduce_max_sync(0xffffffffu, n);
        for (int32_t c0 = 0; c0 < nmax; c0 += G * MOM_CHUNK_PER_LANE) {
            float a0 = 0.f, a1 = 0.f, a2 = 0.f;
            const int32_t cend = min(n, c0 + G * MOM_CHUNK_PER_LANE);
            for (int32_t j = c0 + gl; j < cend; j += G) {
                a0 += vx[s + j] - px; a1 += vy[s + j] - py; a2 += vz[s + j] - pz;
            }
            S0 += (double)a0; S1 += (double)a1; S2 += (double)a2;
        }
#pragma unroll
        for (int d = G / 2; d >= 1; d >>= 1) {
            S0 += fpd_shfl_xor(S0, d); S1 += fpd_shfl_xor(S1, d); S2 += fpd_shfl_xor(S2, d);
        }
        const double invn = n > 0 ? 1.0 / (double)n : 0.0;
        const double m0d = S0 * invn, m1d = S1 * invn, m2d = S2 * invn;
        const float m0 = (float)m0d, m1 = (float)m1d, m2 = (float)m2d;
        // ---- pass 2: central moments
        double r[NP];
#pragma unroll
        for (int k = 0; k < NP; ++k) r[k] = 0.0;
        for (int32_t c0 = 0; c0 < nmax; c0 += G * MOM_CHUNK_PER_LANE) {
            float P[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
            float t[10], F[6], g[3], h[3];
#pragma unroll
            for (int k = 0; k < 10; ++k) t[k] = 0.f;
#pragma unroll
            for (int k = 0; k < 6; ++k) F[k] = 0.f;
#pragma unroll
            for (int k = 0; k < 3; ++k) { g[k] = 0.f; h[k] = 0.f; }
            const int32_t cend = min(n, c0 + G * MOM_CHUNK_PER_LANE);
            for (int32_t j = c0 + gl; j < cend; j += G) {
                const float cx = (vx[s + j] - px) - m0, cy = (vy[s + j] - py) - m1, cz = (vz[s + j] - pz) - m2;
                const float xx = cx * cx, xy = cx * cy, xz = cx * cz, yy = cy * cy, yz = cy * cz, zz = cz * cz;
                const float c2 = xx + yy + zz;
                P[0] += xx; P[1] += xy; P[2] += xz; P[3] += yy; P[4] += yz; P[5] += zz;
                if (FULL) {
                    t[0] = fmaf(xx, cx, t[0]); t[1] = fmaf(xx, cy, t[1]); t[2] = fmaf(xx, cz, t[2]);
                    t[3] = fmaf(xy, cy, t[3]); t[4] = fmaf(xy, cz, t[4]); t[5] = fmaf(xz, cz, t[5]);
                    t[6] = fmaf(yy, cy, t[6]); t[7] = fmaf(yy, cz, t[7]); t[8] = fmaf(yz, cz, t[8]);
                    t[9] = fmaf(zz, cz, t[9]);
                    F[0] = fmaf(c2, xx, F[0]); F[1] = fmaf(c2, xy, F[1]); F[2] = fmaf(c2, xz, F[2]);
                    F[3] = fmaf(c2, yy, F[3]); F[4] = fmaf(c2, yz, F[4]); F[5] = fmaf(c2, zz, F[5]);
                    const float c4 = c2 * c2;
                    g[0] = fmaf(c4, cx, g[0]); g[1] = fmaf(c4, cy, g[1]); g[2] = fmaf(c4, cz, g[2]);
                } else {
                    h[0] = fmaf(c2, cx, h[0]); h[1] = fmaf(c2, cy, h[1]); h[2] = fmaf(c2, cz, h[2]);
                }
            }
#pragma unroll
            for (int k = 0; k < 6; ++k) r[4 + k] += (double)P[k];
            if (FULL) {
#pragma unroll
                for (int k = 0; k < 10; ++k) r[10 + k] += (double)t[k];
#pragma unroll
                for (int k = 0; k < 6; ++k) r[20 + k] += (double)F[k];
#pragma unroll
                for (int k = 0; k < 3; ++k) r[26 + k] += (double)g[k];
            } else {
#pragma unroll
                for (int k = 0; k < 3; ++k) r[10 + k] += (double)h[k];
            }
        }
        fpd_transpose_reduce<NP, G>(r, gl);
        // lane gl now holds record slots PER*gl .. PER*gl + PER - 1
        if (have) {
            double* rec = mom + (size_t)cell * NREC;
#pragma unroll
            for (int i = 0; i < PER; ++i) {
                const int slot = PER * gl + i;
                double val = r[i] * invn;
                if (slot == 0) val = (double)n;
                else if (slot == 1) val = n > 0 ? (double)px + m0d : 0.0;
                else if (slot == 2) val = n > 0 ? (double)py + m1d : 0.0;
                else if (slot == 3) val = n > 0 ? (double)pz + m2d : 0.0;
                if (slot < NREC) rec[slot] = val;
            }
        }
    }
}

template <int G>
static void launch_moments(fp_ctx* ctx, const float* vx, const float* vy, const float* vz, const int32_t* cell_start,
                           int32_t mode, double* mom, cudaStream_t st)
{
    const int32_t ncell = ctx->ncell;
    const int64_t groups_per_block = MOM_THREADS / G;
    int64_t want = (ncell + groups_per_block - 1) / groups_per_block;
    const int64_t cap = (int64_t)ctx->num_sms * 32;
    const int blocks = (int)(want < cap ? want : cap);
    if (mode) moments_kernel<G, true><<<blocks, MOM_THREADS, 0, st>>>(vx, vy, vz, cell_start, ncell, mom);
    else      moments_kernel<G, false><<<blocks, MOM_THREADS, 0, st>>>(vx, vy, vz, cell_start, ncell, mom);
}

extern "C" int fp_cell_moments(fp_ctx* ctx, int64_t np, const float* vx, const float* vy, const float* vz,
                               const int32_t* cell_start, int32_t mode, double* mom, void* stream)
{
    if (!ctx) return FP_ERR_ARG;
    if (np < 0 || !cell_start || !mom || (mode != 0 && mode != 1)) return fp_fail(ctx, FP_ERR_ARG, "fp_cell_moments: bad argument");
    if (np > 0 && (!vx || !vy || !vz)) return fp_fail(ctx, FP_ERR_ARG, "fp_cell_moments: null velocity pointer");
    cudaStream_t st = (cudaStream_t)stream;
    const double ppc = (double)np / (double)ctx->ncell;
    // group width: about 8-16 particles per lane
    if (ppc >= 192.0)      launch_moments<16>(ctx, vx, vy, vz, cell_start, mode, mom, st);
    else if (ppc >= 48.0)  launch_moments<8>(ctx, vx, vy, vz, cell_start, mode, mom, st);
    else                   launch_moments<4>(ctx, vx, vy, vz, cell_start, mode, mom, st);
    FP_LAUNCH_OK(ctx);
    FP_COUNT(ctx, 1);
    return FP_OK;
}
