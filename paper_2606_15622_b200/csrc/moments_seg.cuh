// moments_seg.cuh -- a3 at very high particles per cell (the paper's Couette runs hold 30,000
// particles per cell; cavity sweeps 500-1500, :491-497).  Included by moments.cu only.
//
// One cell per lane group cannot use the device when there are few, huge cells (300 cells x 30,000 particles: 300
// warps).  Here the particle index space is cut into 512-particle slices regardless of cell boundaries: every slice
// is 16-byte aligned (three bulk copies, no ragged staging) and all slices are equal work.  A warp walks the cells
// that intersect its slice; for each it accumulates, in ONE pass, the 28 raw sums of w = v - pivot,
//     S1_i = sum w_i (3), S2_ij = sum w_i w_j (6), S3_ijk = sum w_i w_j w_k (10), S4_ij = sum w^2 w_i w_j (6),
//     S5_i = sum w^4 w_i (3),
// per lane in packed fp32x2 (at most 8 terms per half), across lanes in fp64 (transposing butterfly), and adds them to
// the cell's fp64 accumulators with atomics.  The pivot is the mean of the cell's first min(N, 32) particles (an fp64 sum
// of at most 32 fp32 values is exact, so every slice and the finalising kernel obtain the same fp32 pivot); it is
// within ~0.2 thermal speeds of the mean, which keeps the cancellation of the shift below small.  The contracted
// 4th/5th-order central moments of the record need only these sums: with d = S1/N (the mean of w), A2 = S2/N, ... ,
//     P_ij  = A2_ij - d_i d_j
//     t_ijk = A3_ijk - (d_i A2_jk + d_j A2_ik + d_k A2_ij) + 2 d_i d_j d_k
//     F_ij  = A4_ij - (hw_i d_j + hw_j d_i) + w2 d_i d_j - 2 B_ij + 2 (b_i d_j + b_j d_i) - 2 d2 d_i d_j + d2 (A2_ij - d_i d_j)
//     g_i   = <c^4 w_i> - d_i <c^4>,
//             <c^4 w_i> = A5_i + 4 d_a d_b A3_abi + d2^2 d_i - 4 d_a A4_ai + 2 d2 hw_i - 4 d2 b_i
//             <c^4>     = w4 + 4 d_a d_b A2_ab + d2^2 - 4 d_a hw_a + 2 d2 w2 - 4 d2^2
// (hw_i = A3_iaa, w2 = A2_aa, w4 = A4_aa, B_ij = d_a A3_aij, b_i = d_a A2_ai, d2 = d.d), evaluated per cell in fp64 by
// mom_seg_finalize_kernel.  Used when the mean particles per cell exceed what the staged one-cell-per-group path
// holds (MOM_SEG_MIN) and the arrays are 16-byte aligned.
#pragma once

#ifndef MOM_SEG_MIN
#define MOM_SEG_MIN 448.0
#endif
#define MOM_SEG 512
#define MOM_SEG_WARPS 4

__device__ __forceinline__ int mom_sym3(int i, int j, int k)       // sorted (i<=j<=k) -> 0..9: 111,112,113,122,123,133,222,223,233,333
{
    if (i > j) { int t = i; i = j; j = t; }
    if (j > k) { int t = j; j = k; k = t; }
    if (i > j) { int t = i; i = j; j = t; }
    const int base[3] = {0, 6, 9};
    return base[i] + (i == 0 ? (j == 0 ? k : (j == 1 ? 2 + k : 5)) : (i == 1 ? (j == 1 ? k - 1 : 2) : 0));
}
__device__ __forceinline__ int mom_sym2(int i, int j) { if (i > j) { int t = i; i = j; j = t; } return i == 0 ? j : (i == 1 ? 2 + j : 5); }

// fp32 pivot of a cell: mean of its first min(n, 32) particles, one value per lane, fp64 butterfly (exact)
__device__ __forceinline__ void mom_seg_pivot(const float* __restrict__ vx, const float* __restrict__ vy,
                                              const float* __restrict__ vz, int32_t first, int32_t n, int lane,
                                              float& px, float& py, float& pz)
{
    const int cnt = n < 32 ? n : 32;
    double a = 0.0, b = 0.0, c = 0.0;
    if (lane < cnt) { a = (double)vx[first + lane]; b = (double)vy[first + lane]; c = (double)vz[first + lane]; }
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) { a += fpd_shfl_xor(a, d); b += fpd_shfl_xor(b, d); c += fpd_shfl_xor(c, d); }
    px = (float)(a / (double)cnt); py = (float)(b / (double)cnt); pz = (float)(c / (double)cnt);
}

__global__ void __launch_bounds__(MOM_SEG_WARPS * 32)
mom_seg_kernel(const float* __restrict__ vx, const float* __restrict__ vy, const float* __restrict__ vz,
               const int32_t* __restrict__ cell_start, int32_t ncell, int64_t np, double* __restrict__ acc,
               const uint32_t* __restrict__ err_dev)
{
    fpd_pdl();
    if (*err_dev) return;                                   // cell_start failed fp_cs_check_kernel: touch nothing
    __shared__ __align__(16) float stage[MOM_SEG_WARPS][3][MOM_SEG];
    __shared__ __align__(8) uint64_t bars[MOM_SEG_WARPS];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float* sx = stage[warp][0];
    float* sy = stage[warp][1];
    float* sz = stage[warp][2];
    if (lane == 0) fpt_mbar_init(&bars[warp], 1);
    __syncwarp();
    const int64_t nslices = (np + MOM_SEG - 1) / MOM_SEG;
    uint32_t phase = 0;
    for (int64_t sl = (int64_t)blockIdx.x * MOM_SEG_WARPS + warp; sl < nslices; sl += (int64_t)gridDim.x * MOM_SEG_WARPS) {
        const int32_t a = (int32_t)(sl * MOM_SEG), b = (int32_t)min((int64_t)a + MOM_SEG, np);
        const int32_t nb = (b - a) & ~3;                                   // bulk part; the last slice may end unaligned
        fpt_fence_proxy_async();
        __syncwarp();
        if (lane == 0 && nb > 0) {
            fpt_mbar_expect_tx(&bars[warp], 3u * (uint32_t)nb * 4u);
            fpt_bulk_g2s(sx, vx + a, (uint32_t)nb * 4u, &bars[warp]);
            fpt_bulk_g2s(sy, vy + a, (uint32_t)nb * 4u, &bars[warp]);
            fpt_bulk_g2s(sz, vz + a, (uint32_t)nb * 4u, &bars[warp]);
        }
        for (int32_t p = a + nb + lane; p < b; p += 32) { sx[p - a] = vx[p]; sy[p - a] = vy[p]; sz[p - a] = vz[p]; }
        // first cell that reaches into the slice: largest c with cell_start[c] <= a (binary search, every lane)
        int32_t lo = 0, hi = ncell;                                        // invariant: cell_start[lo] <= a < cell_start[hi] or hi = ncell
        while (hi - lo > 1) {
            const int32_t mid = (lo + hi) >> 1;
            if (cell_start[mid] <= a) lo = mid; else hi = mid;
        }
        if (nb > 0) { fpt_mbar_wait(&bars[warp], phase); phase ^= 1u; }
        __syncwarp();
        for (int32_t c = lo; c < ncell; ++c) {
            const int32_t cs0 = cell_start[c], cs1 = cell_start[c + 1];
            if (cs0 >= b) break;
            const int32_t s = max(cs0, a), e = min(cs1, b);
            if (e <= s) continue;                                          // empty cell, or one that ends at a
            float px, py, pz;
            mom_seg_pivot(vx, vy, vz, cs0, cs1 - cs0, lane, px, py, pz);
            const float2 npx = fpd_dup(-px), npy = fpd_dup(-py), npz = fpd_dup(-pz);
            float2 S1[3], S2[6], S3[10], S4[6], S5[3];
#pragma unroll
            for (int k = 0; k < 3; ++k) { S1[k] = fpd_dup(0.f); S5[k] = fpd_dup(0.f); }
#pragma unroll
            for (int k = 0; k < 6; ++k) { S2[k] = fpd_dup(0.f); S4[k] = fpd_dup(0.f); }
#pragma unroll
            for (int k = 0; k < 10; ++k) S3[k] = fpd_dup(0.f);
            for (int32_t j = s - a + lane; j < e - a; j += 64) {
                const bool two = j + 32 < e - a;
                const int32_t j2 = two ? j + 32 : j;
                float2 wx = fpd_add2(make_float2(sx[j], sx[j2]), npx);
                float2 wy = fpd_add2(make_float2(sy[j], sy[j2]), npy);
                float2 wz = fpd_add2(make_float2(sz[j], sz[j2]), npz);
                if (!two) { wx.y = 0.f; wy.y = 0.f; wz.y = 0.f; }
                const float2 xx = fpd_mul2(wx, wx), xy = fpd_mul2(wx, wy), xz = fpd_mul2(wx, wz);
                const float2 yy = fpd_mul2(wy, wy), yz = fpd_mul2(wy, wz), zz = fpd_mul2(wz, wz);
                const float2 w2 = fpd_add2(fpd_add2(xx, yy), zz);
                S1[0] = fpd_add2(S1[0], wx); S1[1] = fpd_add2(S1[1], wy); S1[2] = fpd_add2(S1[2], wz);
                S2[0] = fpd_add2(S2[0], xx); S2[1] = fpd_add2(S2[1], xy); S2[2] = fpd_add2(S2[2], xz);
                S2[3] = fpd_add2(S2[3], yy); S2[4] = fpd_add2(S2[4], yz); S2[5] = fpd_add2(S2[5], zz);
                S3[0] = fpd_fma2(xx, wx, S3[0]); S3[1] = fpd_fma2(xx, wy, S3[1]); S3[2] = fpd_fma2(xx, wz, S3[2]);
                S3[3] = fpd_fma2(xy, wy, S3[3]); S3[4] = fpd_fma2(xy, wz, S3[4]); S3[5] = fpd_fma2(xz, wz, S3[5]);
                S3[6] = fpd_fma2(yy, wy, S3[6]); S3[7] = fpd_fma2(yy, wz, S3[7]); S3[8] = fpd_fma2(yz, wz, S3[8]);
                S3[9] = fpd_fma2(zz, wz, S3[9]);
                S4[0] = fpd_fma2(w2, xx, S4[0]); S4[1] = fpd_fma2(w2, xy, S4[1]); S4[2] = fpd_fma2(w2, xz, S4[2]);
                S4[3] = fpd_fma2(w2, yy, S4[3]); S4[4] = fpd_fma2(w2, yz, S4[4]); S4[5] = fpd_fma2(w2, zz, S4[5]);
                const float2 w4 = fpd_mul2(w2, w2);
                S5[0] = fpd_fma2(w4, wx, S5[0]); S5[1] = fpd_fma2(w4, wy, S5[1]); S5[2] = fpd_fma2(w4, wz, S5[2]);
            }
            double r[32];
#pragma unroll
            for (int k = 0; k < 3; ++k) { r[k] = (double)S1[k].x + (double)S1[k].y; r[25 + k] = (double)S5[k].x + (double)S5[k].y; }
#pragma unroll
            for (int k = 0; k < 6; ++k) { r[3 + k] = (double)S2[k].x + (double)S2[k].y; r[19 + k] = (double)S4[k].x + (double)S4[k].y; }
#pragma unroll
            for (int k = 0; k < 10; ++k) r[9 + k] = (double)S3[k].x + (double)S3[k].y;
            r[28] = r[29] = r[30] = r[31] = 0.0;
            fpd_transpose_reduce<32, 32, double>(r, lane);                 // lane k: slice total of sum k
            if (lane < 28) atomicAdd(&acc[(size_t)c * 28 + lane], r[0]);
        }
    }
}

template <bool FULL>
__global__ void __launch_bounds__(128)
mom_seg_finalize_kernel(const float* __restrict__ vx, const float* __restrict__ vy, const float* __restrict__ vz,
                        const int32_t* __restrict__ cell_start, int32_t ncell, const double* __restrict__ acc,
                        double* __restrict__ mom, const uint32_t* __restrict__ err_dev)
{
    fpd_pdl();
    if (*err_dev) return;
    constexpr int NREC = FULL ? 29 : 13;
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= ncell) return;
    double* rec = mom + (size_t)cell * NREC;
    const int32_t cs0 = cell_start[cell], n = cell_start[cell + 1] - cs0;
    if (n <= 0) {
#pragma unroll
        for (int k = 0; k < NREC; ++k) rec[k] = 0.0;
        return;
    }
    const int cnt = n < 32 ? n : 32;
    double pa = 0.0, pb = 0.0, pc = 0.0;
    for (int i = 0; i < cnt; ++i) { pa += (double)vx[cs0 + i]; pb += (double)vy[cs0 + i]; pc += (double)vz[cs0 + i]; }
    const float piv[3] = {(float)(pa / (double)cnt), (float)(pb / (double)cnt), (float)(pc / (double)cnt)};
    const double* S = acc + (size_t)cell * 28;
    const double inv = 1.0 / (double)n;
    double d[3], A2[6], A3[10], A4[6], A5[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) { d[k] = S[k] * inv; A5[k] = S[25 + k] * inv; }
#pragma unroll
    for (int k = 0; k < 6; ++k) { A2[k] = S[3 + k] * inv; A4[k] = S[19 + k] * inv; }
#pragma unroll
    for (int k = 0; k < 10; ++k) A3[k] = S[9 + k] * inv;
    const double d2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    const double w2 = A2[0] + A2[3] + A2[5], w4 = A4[0] + A4[3] + A4[5];
    double hw[3], bv[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        hw[i] = A3[mom_sym3(i, 0, 0)] + A3[mom_sym3(i, 1, 1)] + A3[mom_sym3(i, 2, 2)];
        bv[i] = d[0] * A2[mom_sym2(0, i)] + d[1] * A2[mom_sym2(1, i)] + d[2] * A2[mom_sym2(2, i)];
    }
    rec[0] = (double)n;
#pragma unroll
    for (int i = 0; i < 3; ++i) rec[1 + i] = (double)piv[i] + d[i];
    double P[6], t[10];
    {
        int q = 0, q3 = 0;
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = i; j < 3; ++j) {
                P[q] = A2[q] - d[i] * d[j];
                ++q;
#pragma unroll
                for (int k = j; k < 3; ++k) {
                    t[q3] = A3[q3] - (d[i] * A2[mom_sym2(j, k)] + d[j] * A2[mom_sym2(i, k)] + d[k] * A2[mom_sym2(i, j)]) +
                            2.0 * d[i] * d[j] * d[k];
                    ++q3;
                }
            }
    }
#pragma unroll
    for (int k = 0; k < 6; ++k) rec[4 + k] = P[k];
    if (!FULL) {
        rec[10] = t[0] + t[3] + t[5]; rec[11] = t[1] + t[6] + t[8]; rec[12] = t[2] + t[7] + t[9];     // h_i = t_iaa
        return;
    }
#pragma unroll
    for (int k = 0; k < 10; ++k) rec[10 + k] = t[k];
    {
        int q = 0;
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = i; j < 3; ++j) {
                const double Bij = d[0] * A3[mom_sym3(0, i, j)] + d[1] * A3[mom_sym3(1, i, j)] + d[2] * A3[mom_sym3(2, i, j)];
                rec[20 + q] = A4[q] - (hw[i] * d[j] + hw[j] * d[i]) + w2 * d[i] * d[j] - 2.0 * Bij +
                              2.0 * (bv[i] * d[j] + bv[j] * d[i]) - 2.0 * d2 * d[i] * d[j] + d2 * (A2[q] - d[i] * d[j]);
                ++q;
            }
    }
    double ddA2 = 0.0, dhw = 0.0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        dhw += d[a] * hw[a];
#pragma unroll
        for (int b = 0; b < 3; ++b) ddA2 += d[a] * d[b] * A2[mom_sym2(a, b)];
    }
    const double c4 = w4 + 4.0 * ddA2 + d2 * d2 - 4.0 * dhw + 2.0 * d2 * w2 - 4.0 * d2 * d2;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        double ddA3 = 0.0, dA4 = 0.0;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            dA4 += d[a] * A4[mom_sym2(a, i)];
#pragma unroll
            for (int b = 0; b < 3; ++b) ddA3 += d[a] * d[b] * A3[mom_sym3(a, b, i)];
        }
        const double c4wi = A5[i] + 4.0 * ddA3 + d2 * d2 * d[i] - 4.0 * dA4 + 2.0 * d2 * hw[i] - 4.0 * d2 * bv[i];
        rec[26 + i] = c4wi - d[i] * c4;
    }
}
