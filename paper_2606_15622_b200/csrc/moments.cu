// moments.cu -- a3: segmented gather of per-cell velocity moments over cell-sorted particles
// (PAPER.md:124 moment definition, :215-216 M1-M5, :243 LITE, :181 plain 1/N mean; R0).
//
// HBM-bound by design: 12 B/particle read once + one record per cell written.
// A group of G lanes (G = 4/8/16 by mean particles per cell) owns one cell, so a warp works on 32/G consecutive cells
// at once.  Each warp stages the contiguous vx, vy, vz slices of its cells in its own shared-memory buffer with three
// 1D bulk asynchronous copies (tiles.cuh) -- HBM is read once, coalesced, with no block-wide barrier and no
// dependence between warps -- and both passes over a cell read shared memory:
//   pass 1: S = sum (v - v_pivot) in fp32 about the cell's first particle (differences are thermal-sized, so fp32
//           holds them to ~6e-8 of the thermal speed even at Mach 10), reduced across the group in fp64;
//           U = v_pivot + S/N (fp64), m = S/N.
//   pass 2: c = (v - v_pivot) - m in fp32, monomials and per-lane partial sums in fp32 (<= 64 terms per lane and
//           chunk), combined across the group by a balanced fp32 tree (a transposing butterfly that leaves record
//           slot k in the lane that stores it); chunks, the mean and the 1/N normalisation are fp64.
// Cells larger than G*64 particles are processed chunk by chunk with fp64 accumulation between chunks.  A warp whose
// cells do not fit its staging buffer (dense or huge cells), or unaligned arrays, run the same code on global pointers.
#include "tiles.cuh"

#define MOM_THREADS 128
#define MOM_WARPS (MOM_THREADS / 32)
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
#pragma unroll 4
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
        float r[NP];
        r[0] = r[1] = r[2] = r[3] = 0.f;
        r[4] = P0; r[5] = P1; r[6] = P2; r[7] = P3; r[8] = P4; r[9] = P5;
        if (FULL) {
            r[10] = t0; r[11] = t1; r[12] = t2; r[13] = t3; r[14] = t4; r[15] = t5; r[16] = t6; r[17] = t7; r[18] = t8;
            r[19] = t9; r[20] = F0; r[21] = F1; r[22] = F2; r[23] = F3; r[24] = F4; r[25] = F5; r[26] = g0; r[27] = g1;
            r[28] = g2;
#pragma unroll
            for (int k = 29; k < NP; ++k) r[k] = 0.f;
        } else {
            r[10] = g0; r[11] = g1; r[12] = g2;
#pragma unroll
            for (int k = 13; k < NP; ++k) r[k] = 0.f;
        }
        fpd_transpose_reduce<NP, G, float>(r, gl);       // balanced fp32 tree over the group's partial sums
#pragma unroll
        for (int i = 0; i < PER; ++i) tot[i] += (double)r[i];
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

// One warp = one chunk of 32/G consecutive cells, staged and processed independently of the other warps of the CTA.
template <int G, bool FULL>
__global__ void __launch_bounds__(MOM_THREADS)
moments_warp_kernel(const float* __restrict__ vx, const float* __restrict__ vy, const float* __restrict__ vz,
                    const int32_t* __restrict__ cell_start, int32_t ncell, int64_t np, int32_t aligned,
                    double* __restrict__ mom)
{
    constexpr int NREC = FULL ? 29 : 13;
    constexpr int CPW = 32 / G;                          // cells per warp
    extern __shared__ __align__(16) unsigned char fpw_smem[];
    float* stage = reinterpret_cast<float*>(fpw_smem);                                   // [MOM_WARPS][3][FPW_CAP]
    uint64_t* bars = reinterpret_cast<uint64_t*>(fpw_smem + (size_t)MOM_WARPS * 3 * FPW_CAP * sizeof(float));
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int gl = lane & (G - 1), group = lane / G;
    const int64_t cbase = ((int64_t)blockIdx.x * MOM_WARPS + warp) * CPW;
    if (cbase >= ncell) return;
    // the chunk's CPW + 1 cell boundaries in lanes 0..CPW
    const int32_t cs = cell_start[min(cbase + lane, (int64_t)ncell)];
    const fpw_range r = fpw_range_of(__shfl_sync(0xffffffffu, cs, 0), __shfl_sync(0xffffffffu, cs, CPW), np, aligned != 0);
    const int32_t s = __shfl_sync(0xffffffffu, cs, group), e = __shfl_sync(0xffffffffu, cs, group + 1);
    const int64_t cell = cbase + group;
    const bool have = cell < ncell;
    const int32_t n = have ? e - s : 0;
    double* rec = mom + (size_t)(have ? cell : 0) * NREC;
    if (r.staged) {
        float* sx = stage + (size_t)(warp * 3 + 0) * FPW_CAP;
        float* sy = stage + (size_t)(warp * 3 + 1) * FPW_CAP;
        float* sz = stage + (size_t)(warp * 3 + 2) * FPW_CAP;
        const uint32_t bytes = (uint32_t)r.nb * 4u;
        if (bytes > 0) {
            if (lane == 0) {
                fpt_mbar_init(&bars[warp], 1);
                fpt_mbar_expect_tx(&bars[warp], 3u * bytes);
                fpt_bulk_g2s(sx, vx + r.a0, bytes, &bars[warp]);
                fpt_bulk_g2s(sy, vy + r.a0, bytes, &bars[warp]);
                fpt_bulk_g2s(sz, vz + r.a0, bytes, &bars[warp]);
            }
            __syncwarp();
        }
        // the (at most 3) particles beyond the last multiple of 4 of the whole array
        for (int32_t p = r.a0 + r.nb + lane; p < r.s1; p += 32) { sx[p - r.a0] = vx[p]; sy[p - r.a0] = vy[p]; sz[p - r.a0] = vz[p]; }
        if (bytes > 0) fpt_mbar_wait(&bars[warp], 0);
        __syncwarp();
        mom_cell_group<G, FULL>(sx - r.a0, sy - r.a0, sz - r.a0, s, n, have, gl, rec);        // shared-memory loads
    } else {
        mom_cell_group<G, FULL>(vx, vy, vz, s, n, have, gl, rec);                             // global loads
    }
}

template <int G>
static void launch_moments(fp_ctx* ctx, int64_t np, const float* vx, const float* vy, const float* vz,
                           const int32_t* cell_start, int32_t mode, double* mom, cudaStream_t st)
{
    const int cells_per_block = MOM_WARPS * (32 / G);
    const int blocks = fp_div_up(ctx->ncell, cells_per_block);
    const int aligned = ((((uintptr_t)vx) | ((uintptr_t)vy) | ((uintptr_t)vz)) & 15u) == 0 ? 1 : 0;
    const size_t smem = (size_t)MOM_WARPS * 3 * FPW_CAP * sizeof(float) + MOM_WARPS * sizeof(uint64_t);
    static bool attr_set = false;                 // one flag per instantiation (G)
    if (!attr_set) {
        cudaFuncSetAttribute(moments_warp_kernel<G, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        cudaFuncSetAttribute(moments_warp_kernel<G, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        attr_set = true;
    }
    if (mode) moments_warp_kernel<G, true><<<blocks, MOM_THREADS, smem, st>>>(vx, vy, vz, cell_start, ctx->ncell, np, aligned, mom);
    else      moments_warp_kernel<G, false><<<blocks, MOM_THREADS, smem, st>>>(vx, vy, vz, cell_start, ctx->ncell, np, aligned, mom);
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
    if (ppc >= 192.0)      launch_moments<16>(ctx, np, vx, vy, vz, cell_start, mode, mom, st);
    else if (ppc >= 48.0)  launch_moments<8>(ctx, np, vx, vy, vz, cell_start, mode, mom, st);
    else                   launch_moments<4>(ctx, np, vx, vy, vz, cell_start, mode, mom, st);
    FP_LAUNCH_OK(ctx);
    FP_COUNT(ctx, 1);
    return FP_OK;
}
