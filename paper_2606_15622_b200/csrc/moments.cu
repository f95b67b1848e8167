// moments.cu -- a3: segmented gather of per-cell velocity moments over cell-sorted particles
// (PAPER.md:124 moment definition, :215-216 M1-M5, :243 LITE, :181 plain 1/N mean; R0).
//
// HBM-bound by design: 12 B/particle read once + one record per cell written.
// One CTA per particle tile (tiles.cuh): the tile's vx, vy, vz slices are staged in shared memory by three 1D bulk
// asynchronous copies, then a group of G lanes (G = 4/8/16 by mean particles per cell) owns one cell, so a warp
// works on 32/G cells at once and both passes over a cell read shared memory:
//   pass 1: S = sum (v - v_pivot) in fp32 about the cell's first particle (differences are thermal-sized, so fp32
//           holds them to ~6e-8 of the thermal speed even at Mach 10), reduced across the group in fp64;
//           U = v_pivot + S/N (fp64), m = S/N.
//   pass 2: c = (v - v_pivot) - m in fp32, monomials and per-lane partial sums in fp32 (<= 64 terms per lane and
//           chunk), converted to fp64 and reduced across the group with a transposing butterfly that leaves record
//           slot k in the lane that stores it.
// Cells larger than G*64 particles are processed chunk by chunk with fp64 accumulation between chunks.  A tile that
// does not fit the staging buffer (a huge cell) or unaligned arrays run the same code on global pointers.
#include "tiles.cuh"

#define MOM_THREADS 128
#define MOM_CHUNK_PER_LANE 64

// One cell per group of G lanes.  bx/by/bz may point to shared or global memory; particle p is at b?[p].
template <int G, bool FULL>
__device__ __forceinline__ void mom_cell_group(const float* bx, const float* by, const float* bz, int32_t s, int32_t n,
                                               bool have, int gl, double* __restrict__ rec)
{
    constexpr int NP = FULL ? 32 : 16;          // padded record length
    constexpr int NREC = FULL ? 29 : 13;
    constexpr int PER = NP / G;                 // record slots per lane after the transposing reduction
    static_assert(NP >= G, "group wider than the padded record");
    // ---- pass 1: mean about the pivot
    float px = 0.f, py = 0.f, pz = 0.f;
    if (n > 0) { px = bx[s]; py = by[s]; pz = bz[s]; }
    const int32_t nmax = __reduce_max_sync(0xffffffffu, n);
    double S0 = 0.0, S1 = 0.0, S2 = 0.0;
    for (int32_t c0 = 0; c0 < nmax; c0 += G * MOM_CHUNK_PER_LANE) {
        float a0 = 0.f, a1 = 0.f, a2 = 0.f;
        const int32_t cend = min(n, c0 + G * MOM_CHUNK_PER_LANE);
#pragma unroll 4
        for (int32_t j = c0 + gl; j < cend; j += G) {
            a0 += bx[s + j] - px; a1 += by[s + j] - py; a2 += bz[s + j] - pz;
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
    double tot[PER];
#pragma unroll
    for (int i = 0; i < PER; ++i) tot[i] = 0.0;
    for (int32_t c0 = 0; c0 < nmax; c0 += G * MOM_CHUNK_PER_LANE) {
        float P0 = 0.f, P1 = 0.f, P2 = 0.f, P3 = 0.f, P4 = 0.f, P5 = 0.f;
        float t0 = 0.f, t1 = 0.f, t2 = 0.f, t3 = 0.f, t4 = 0.f, t5 = 0.f, t6 = 0.f, t7 = 0.f, t8 = 0.f, t9 = 0.f;
        float F0 = 0.f, F1 = 0.f, F2 = 0.f, F3 = 0.f, F4 = 0.f, F5 = 0.f;
        float g0 = 0.f, g1 = 0.f, g2 = 0.f;
        const int32_t cend = min(n, c0 + G * MOM_CHUNK_PER_LANE);
#pragma unroll 2
        for (int32_t j = c0 + gl; j < cend; j += G) {
            const float cx = (bx[s + j] - px) - m0, cy = (by[s + j] - py) - m1, cz = (bz[s + j] - pz) - m2;
            const float xx = cx * cx, xy = cx * cy, xz = cx * cz, yy = cy * cy, yz = cy * cz, zz = cz * cz;
            const float c2 = xx + yy + zz;
            P0 += xx; P1 += xy; P2 += xz; P3 += yy; P4 += yz; P5 += zz;
            if (FULL) {
                t0 = fmaf(xx, cx, t0); t1 = fmaf(xx, cy, t1); t2 = fmaf(xx, cz, t2); t3 = fmaf(xy, cy, t3);
                t4 = fmaf(xy, cz, t4); t5 = fmaf(xz, cz, t5); t6 = fmaf(yy, cy, t6); t7 = fmaf(yy, cz, t7);
                t8 = fmaf(yz, cz, t8); t9 = fmaf(zz, cz, t9);
                F0 = fmaf(c2, xx, F0); F1 = fmaf(c2, xy, F1); F2 = fmaf(c2, xz, F2);
                F3 = fmaf(c2, yy, F3); F4 = fmaf(c2, yz, F4); F5 = fmaf(c2, zz, F5);
                const float c4 = c2 * c2;
                g0 = fmaf(c4, cx, g0); g1 = fmaf(c4, cy, g1); g2 = fmaf(c4, cz, g2);
            } else {
                g0 = fmaf(c2, cx, g0); g1 = fmaf(c2, cy, g1); g2 = fmaf(c2, cz, g2);      // h_i = <c^2 c_i>
            }
        }
        double r[NP];
        r[0] = r[1] = r[2] = r[3] = 0.0;
        r[4] = (double)P0; r[5] = (double)P1; r[6] = (double)P2; r[7] = (double)P3; r[8] = (double)P4; r[9] = (double)P5;
        if (FULL) {
            r[10] = (double)t0; r[11] = (double)t1; r[12] = (double)t2; r[13] = (double)t3; r[14] = (double)t4;
            r[15] = (double)t5; r[16] = (double)t6; r[17] = (double)t7; r[18] = (double)t8; r[19] = (double)t9;
            r[20] = (double)F0; r[21] = (double)F1; r[22] = (double)F2; r[23] = (double)F3; r[24] = (double)F4;
            r[25] = (double)F5; r[26] = (double)g0; r[27] = (double)g1; r[28] = (double)g2;
#pragma unroll
            for (int k = 29; k < NP; ++k) r[k] = 0.0;
        } else {
            r[10] = (double)g0; r[11] = (double)g1; r[12] = (double)g2;
#pragma unroll
            for (int k = 13; k < NP; ++k) r[k] = 0.0;
        }
        fpd_transpose_reduce<NP, G>(r, gl);
#pragma unroll
        for (int i = 0; i < PER; ++i) tot[i] += r[i];
    }
    // lane gl holds record slots PER*gl .. PER*gl + PER - 1
    if (have) {
#pragma unroll
        for (int i = 0; i < PER; ++i) {
            const int slot = PER * gl + i;
            double val = tot[i] * invn;
            if (slot == 0) val = (double)n;
            else if (slot == 1) val = n > 0 ? (double)px + m0d : 0.0;
            else if (slot == 2) val = n > 0 ? (double)py + m1d : 0.0;
            else if (slot == 3) val = n > 0 ? (double)pz + m2d : 0.0;
            if (slot < NREC) rec[slot] = val;
        }
    }
}

template <int G, bool FULL>
__global__ void __launch_bounds__(MOM_THREADS)
moments_tile_kernel(const float* __restrict__ vx, const float* __restrict__ vy, const float* __restrict__ vz,
                    const int32_t* __restrict__ cell_start, const int32_t* __restrict__ tile_cell, int32_t ncell,
                    int64_t np, int32_t aligned, double* __restrict__ mom)
{
    constexpr int NREC = FULL ? 29 : 13;
    __shared__ __align__(16) float sx[FPT_CAP], sy[FPT_CAP], sz[FPT_CAP];
    __shared__ __align__(8) uint64_t bar;
    const fpt_tile t = fpt_tile_of_block(tile_cell, cell_start, ncell, np, aligned != 0);
    if (t.c0 >= t.c1) return;
    const float *bx = vx, *by = vy, *bz = vz;
    if (t.staged) {
        const uint32_t bytes = (uint32_t)t.nb * 4u;
        if (threadIdx.x == 0 && bytes > 0) fpt_mbar_init(&bar, 1);
        __syncthreads();
        if (threadIdx.x == 0 && bytes > 0) {
            fpt_mbar_expect_tx(&bar, 3u * bytes);
            fpt_bulk_g2s(sx, vx + t.a0, bytes, &bar);
            fpt_bulk_g2s(sy, vy + t.a0, bytes, &bar);
            fpt_bulk_g2s(sz, vz + t.a0, bytes, &bar);
        }
        // the (at most 3) particles beyond the last multiple of 4 of the whole array
        for (int32_t p = t.a0 + t.nb + (int32_t)threadIdx.x; p < t.s1; p += MOM_THREADS) {
            sx[p - t.a0] = vx[p]; sy[p - t.a0] = vy[p]; sz[p - t.a0] = vz[p];
        }
        if (bytes > 0) fpt_mbar_wait(&bar, 0);
        __syncthreads();
        bx = sx - t.a0; by = sy - t.a0; bz = sz - t.a0;
    }
    const int gl = threadIdx.x & (G - 1);
    const int group = threadIdx.x / G;
    constexpr int NGROUPS = MOM_THREADS / G;
    for (int32_t cb = t.c0; cb < t.c1; cb += NGROUPS) {
        if (cb + (int32_t)((threadIdx.x & ~31) / G) >= t.c1) break;      // this whole warp has no cell left
        const int32_t cell = cb + group;
        const bool have = cell < t.c1;
        int32_t s = 0, n = 0;
        if (have) { s = cell_start[cell]; n = cell_start[cell + 1] - s; }
        mom_cell_group<G, FULL>(bx, by, bz, s, n, have, gl, mom + (size_t)(have ? cell : 0) * NREC);
    }
}

template <int G>
static void launch_moments(fp_ctx* ctx, int64_t np, const float* vx, const float* vy, const float* vz,
                           const int32_t* cell_start, int32_t mode, double* mom, cudaStream_t st)
{
    const int ntiles = fpi_ntiles(np);
    const int aligned = ((((uintptr_t)vx) | ((uintptr_t)vy) | ((uintptr_t)vz)) & 15u) == 0 ? 1 : 0;
    if (mode) moments_tile_kernel<G, true><<<ntiles, MOM_THREADS, 0, st>>>(vx, vy, vz, cell_start, ctx->tile_cell, ctx->ncell, np, aligned, mom);
    else      moments_tile_kernel<G, false><<<ntiles, MOM_THREADS, 0, st>>>(vx, vy, vz, cell_start, ctx->tile_cell, ctx->ncell, np, aligned, mom);
}

// tiles_ready: ctx->tile_cell already holds the table of this (np, cell_start)
int fpi_cell_moments(fp_ctx* ctx, int64_t np, const float* vx, const float* vy, const float* vz,
                     const int32_t* cell_start, int32_t mode, double* mom, bool tiles_ready, cudaStream_t st)
{
    int rc;
    if (!tiles_ready && (rc = fpi_tile_table(ctx, np, cell_start, st)) != FP_OK) return rc;
    const double ppc = (double)np / (double)ctx->ncell;
    // group width: about 8-16 particles per lane
    if (ppc >= 192.0)      launch_moments<16>(ctx, np, vx, vy, vz, cell_start, mode, mom, st);
    else if (ppc >= 48.0)  launch_moments<8>(ctx, np, vx, vy, vz, cell_start, mode, mom, st);
    else                   launch_moments<4>(ctx, np, vx, vy, vz, cell_start, mode, mom, st);
    FP_LAUNCH_OK(ctx);
    FP_COUNT(ctx, 1);
    return FP_OK;
}

extern "C" int fp_cell_moments(fp_ctx* ctx, int64_t np, const float* vx, const float* vy, const float* vz,
                               const int32_t* cell_start, int32_t mode, double* mom, void* stream)
{
    if (!ctx) return FP_ERR_ARG;
    if (np < 0 || !cell_start || !mom || (mode != 0 && mode != 1)) return fp_fail(ctx, FP_ERR_ARG, "fp_cell_moments: bad argument");
    if (np > 0 && (!vx || !vy || !vz)) return fp_fail(ctx, FP_ERR_ARG, "fp_cell_moments: null velocity pointer");
    if (np > ctx->p.max_particles) return fp_fail(ctx, FP_ERR_STATE, "fp_cell_moments: np > max_particles");
    return fpi_cell_moments(ctx, np, vx, vy, vz, cell_start, mode, mom, false, (cudaStream_t)stream);
}
