// update_seg.cuh -- a6 at very high particles per cell (PAPER.md:282 30,000 particles per cell,
// :491-497 500-1500).  Included by update.cu only.
//
// Same arithmetic as upd_giant_cell (pass A in the split form per 512-particle slice with all 32 lanes, per-slice sums
// combined in fp64, fp64 epilogue upd_scales, pass B as a streaming read-modify-write), but spread over the device: the particle index space is
// cut into 512-particle slices regardless of cell boundaries, as in moments_seg.cuh.
//   upd_seg_a_kernel: a warp stages its slice (vx, vy, vz, pid: four aligned bulk copies), runs pass A for every cell
//     that intersects it (w = E1 v + q' over the velocities, seven partial sums), adds the sums to the cell's fp64
//     accumulators with atomics and writes the slice back with bulk stores;
//   upd_seg_b_kernel: a warp walks the cells of its slice again, forms alpha / the recentring mean / the energy scale
//     from the accumulators exactly as upd_giant_cell does, and rewrites its part of the cell.
// A particle beyond its cell's fp32 range (upd_prep.cuh [26]) gets its w recomputed in fp64 while its slice is still in
// shared memory (upd_fix_far_slice); cells of at most UPD_SEG_TINY particles are left to upd_seg_tiny_kernel.
// 52 instead of 28 B per particle, every SM busy: 300 cells x 30,000 particles 1.55 ms -> see DESIGN.md.
#pragma once

#define UPD_SEG 512
#define UPD_SEG_WARPS 4
#define UPD_SEG_TINY 8                 // cells of at most this many particles take the fp64 path (conservation scales of a
                                   // few-particle cell amplify fp32 rounding, see upd_finish)

__device__ __forceinline__ int32_t upd_seg_first_cell(const int32_t* __restrict__ cell_start, int32_t ncell, int32_t a)
{
    int32_t lo = 0, hi = ncell;                                  // largest c with cell_start[c] <= a
    while (hi - lo > 1) {
        const int32_t mid = (lo + hi) >> 1;
        if (cell_start[mid] <= a) lo = mid; else hi = mid;
    }
    return lo;
}

__global__ void __launch_bounds__(UPD_SEG_WARPS * 32)
upd_seg_a_kernel(float* __restrict__ vx, float* __restrict__ vy, float* __restrict__ vz, const uint32_t* __restrict__ pid,
                 const int32_t* __restrict__ cell_start, int64_t np, const float* __restrict__ cellc,
                 double* __restrict__ acc, const uint32_t* __restrict__ err_dev, const __grid_constant__ upd_src R,
                 const __grid_constant__ upd_params Q)
{
    fpd_pdl();
    if (*err_dev) return;                                   // cell_start failed fp_cs_check_kernel: touch nothing
    __shared__ __align__(16) float stage[UPD_SEG_WARPS][4][UPD_SEG];
    __shared__ __align__(8) uint64_t bars[UPD_SEG_WARPS];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float* sx = stage[warp][0];
    float* sy = stage[warp][1];
    float* sz = stage[warp][2];
    uint32_t* sp = reinterpret_cast<uint32_t*>(stage[warp][3]);
    if (lane == 0) fpt_mbar_init(&bars[warp], 1);
    __syncwarp();
    const int64_t nslices = (np + UPD_SEG - 1) / UPD_SEG;
    uint32_t phase = 0;
    for (int64_t sl = (int64_t)blockIdx.x * UPD_SEG_WARPS + warp; sl < nslices; sl += (int64_t)gridDim.x * UPD_SEG_WARPS) {
        const int32_t a = (int32_t)(sl * UPD_SEG), b = (int32_t)min((int64_t)a + UPD_SEG, np);
        const int32_t nb = (b - a) & ~3;
        fpt_fence_proxy_async();
        __syncwarp();
        if (lane == 0 && nb > 0) {
            fpt_mbar_expect_tx(&bars[warp], 4u * (uint32_t)nb * 4u);
            fpt_bulk_g2s(sx, vx + a, (uint32_t)nb * 4u, &bars[warp]);
            fpt_bulk_g2s(sy, vy + a, (uint32_t)nb * 4u, &bars[warp]);
            fpt_bulk_g2s(sz, vz + a, (uint32_t)nb * 4u, &bars[warp]);
            fpt_bulk_g2s(sp, pid + a, (uint32_t)nb * 4u, &bars[warp]);
        }
        for (int32_t p = a + nb + lane; p < b; p += 32) { sx[p - a] = vx[p]; sy[p - a] = vy[p]; sz[p - a] = vz[p]; sp[p - a] = pid[p]; }
        const int32_t c0 = upd_seg_first_cell(cell_start, Q.ncell, a);
        if (nb > 0) { fpt_mbar_wait(&bars[warp], phase); phase ^= 1u; }
        __syncwarp();
        for (int32_t c = c0; c < Q.ncell; ++c) {
            const int32_t cs0 = cell_start[c], cs1 = cell_start[c + 1];
            if (cs0 >= b) break;
            const int32_t s = max(cs0, a), e = min(cs1, b);
            if (e <= s) continue;
            if (cs1 - cs0 <= UPD_SEG_TINY) continue;             // left untouched for the fp64 path in upd_seg_b_kernel
            float k[UPD_NC];
            const float* cc = cellc + (size_t)c * UPD_NC;
#pragma unroll
            for (int q = 0; q < UPD_NC / 4; ++q) {
                const float4 v = reinterpret_cast<const float4*>(cc)[q];
                k[4 * q] = v.x; k[4 * q + 1] = v.y; k[4 * q + 2] = v.z; k[4 * q + 3] = v.w;
            }
            if (k[23] == 0.0f) continue;                         // inactive cell: velocities stay
            const upd_part pa = upd_pass_a<32, true>(sx, sy, sz, sp, s - a, e - s, lane, k, Q);
            double D[7] = {(double)(pa.SNN.x + pa.SNN.y), (double)(pa.SCN.x + pa.SCN.y), (double)(pa.SM0.x + pa.SM0.y),
                           (double)(pa.SM1.x + pa.SM1.y), (double)(pa.SM2.x + pa.SM2.y), (double)(pa.SQ.x + pa.SQ.y),
                           (double)(pa.SCQ.x + pa.SCQ.y)};
            if (__any_sync(0xffffffffu, pa.far > k[27])) {       // particles beyond the cell's fp32 range: their w and their
                __syncwarp();                                    // terms of the sums again, in fp64
                upd_fix_far_slice(vx + s, vy + s, vz + s, pid + s, sx + (s - a), sy + (s - a), sz + (s - a), e - s, lane, R, c,
                                  cc, Q, D);
                __syncwarp();
            }
#pragma unroll
            for (int d = 16; d >= 1; d >>= 1) {
#pragma unroll
                for (int q = 0; q < 7; ++q) D[q] += fpd_shfl_xor(D[q], d);
            }
            if (lane < 7) {
                double mine = D[0];
#pragma unroll
                for (int q = 1; q < 7; ++q) if (lane == q) mine = D[q];
                atomicAdd(&acc[(size_t)c * UPD_ACC + lane], mine);
            }
        }
        // ---- w = E1 v + q' back to global memory: aligned part by bulk stores, the ragged end of the last slice by plain stores
        fpt_fence_proxy_async();
        __syncwarp();
        if (lane == 0 && nb > 0) {
            fpt_bulk_s2g(vx + a, sx, (uint32_t)nb * 4u);
            fpt_bulk_s2g(vy + a, sy, (uint32_t)nb * 4u);
            fpt_bulk_s2g(vz + a, sz, (uint32_t)nb * 4u);
            fpt_bulk_commit_wait();
        }
        for (int32_t p = a + nb + lane; p < b; p += 32) { vx[p] = sx[p - a]; vy[p] = sy[p - a]; vz[p] = sz[p - a]; }
        __syncwarp();
    }
}

__global__ void __launch_bounds__(UPD_SEG_WARPS * 32)
upd_seg_b_kernel(float* __restrict__ vx, float* __restrict__ vy, float* __restrict__ vz,
                 const int32_t* __restrict__ cell_start, int64_t np, const float* __restrict__ cellc,
                 const double* __restrict__ acc, uint32_t* __restrict__ flags, const uint32_t* __restrict__ err_dev,
                 const __grid_constant__ upd_params Q)
{
    fpd_pdl();
    if (*err_dev) return;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t nslices = (np + UPD_SEG - 1) / UPD_SEG;
    for (int64_t sl = (int64_t)blockIdx.x * UPD_SEG_WARPS + warp; sl < nslices; sl += (int64_t)gridDim.x * UPD_SEG_WARPS) {
        const int32_t a = (int32_t)(sl * UPD_SEG), b = (int32_t)min((int64_t)a + UPD_SEG, np);
        const int32_t c0 = upd_seg_first_cell(cell_start, Q.ncell, a);
        for (int32_t c = c0; c < Q.ncell; ++c) {
            const int32_t cs0 = cell_start[c], cs1 = cell_start[c + 1];
            if (cs0 >= b) break;
            const int32_t s = max(cs0, a), e = min(cs1, b);
            if (e <= s) continue;
            if (cs1 - cs0 <= UPD_SEG_TINY) continue;             // upd_seg_tiny_kernel
            float k[UPD_NC];
            const float* cc = cellc + (size_t)c * UPD_NC;
#pragma unroll
            for (int q = 0; q < UPD_NC / 4; ++q) {
                const float4 v = reinterpret_cast<const float4*>(cc)[q];
                k[4 * q] = v.x; k[4 * q + 1] = v.y; k[4 * q + 2] = v.z; k[4 * q + 3] = v.w;
            }
            if (k[23] == 0.0f) continue;
            float sc, f0, f1, f2;
            if (!upd_scales(k, acc + (size_t)c * UPD_ACC, cs1 - cs0, Q.conserve_mode, sc, f0, f1, f2) && lane == 0 && cs0 >= a)
                flags[c] |= FP_FLAG_ALPHA;                        // once per cell
            for (int32_t p = s + lane; p < e; p += 32) {
                vx[p] = fmaf(vx[p], sc, f0);
                vy[p] = fmaf(vy[p], sc, f1);
                vz[p] = fmaf(vz[p], sc, f2);
            }
        }
    }
}

// The cells of at most UPD_SEG_TINY particles, which the two kernels above leave untouched: one warp per 32 cells, each such
// cell redone by the whole warp on the fp64 path (its own kernel: the call would cost upd_seg_b_kernel 88 registers).
__global__ void __launch_bounds__(128)
upd_seg_tiny_kernel(float* __restrict__ vx, float* __restrict__ vy, float* __restrict__ vz, const uint32_t* __restrict__ pid,
                    const int32_t* __restrict__ cell_start, uint32_t* __restrict__ flags, const uint32_t* __restrict__ err_dev,
                    const __grid_constant__ upd_src R, const __grid_constant__ upd_params Q)
{
    fpd_pdl();
    if (*err_dev) return;
    const int lane = threadIdx.x & 31;
    const int32_t c0 = (int32_t)((blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) * 32);
    if (c0 >= Q.ncell) return;
    const int32_t c = c0 + lane;
    const int32_t n = c < Q.ncell ? cell_start[c + 1] - cell_start[c] : 0;
    uint32_t tiny = __ballot_sync(0xffffffffu, n >= 2 && n <= UPD_SEG_TINY);
    while (tiny) {
        const int j = __ffs(tiny) - 1;
        tiny &= tiny - 1;
        upd_far_cell(vx, vy, vz, pid, cell_start, R, flags, c0 + j, Q);
    }
}
