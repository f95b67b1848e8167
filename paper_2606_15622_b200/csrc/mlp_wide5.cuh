// mlp_wide5.cuh -- tcgen05 / TMEM version of the wide surrogate ([13|16]-256-...-256-9, PAPER.md:309; :264, :327,
// :568).  Included by closure_mlp.cu only; same arithmetic contract as mlp_wide.cuh (split-bf16
// "3x" products, fp32 accumulate), but the products run on the 5th-generation tensor cores:
//   * a CTA owns a tile of 128 cells = the M of one tcgen05.mma (cta_group::1, kind::f16, M 128, N 256, K 16); the
//     accumulator D[128 x 256] fp32 lives in TMEM (256 columns), row i = TMEM lane i = cell i of the tile;
//   * A = the tile's activations, shared memory, already split into bf16 hi / lo, in the canonical K-major
//     no-swizzle core-matrix layout (8 rows x 16 bytes per core matrix; SBO = 128 B between 8-row groups, LBO = 2 KB
//     between 8-input slabs), written in place by the previous layer's epilogue (its mma has completed by then);
//   * B = the weights, streamed from L2 through a 4-stage shared-memory ring by one producer lane with 1D bulk
//     copies (cp.async.bulk, mbarrier complete_tx): mlpw5_pack_kernel lays every 16-input chunk out in global
//     memory as the exact byte image of its stage (hi part, lo part, each canonical K-major), so a chunk is one copy;
//   * one elected lane issues, per chunk, A_hi.B_hi, A_lo.B_hi, A_hi.B_lo and commits the stage back to the
//     producer; after the last chunk of a layer it commits to the epilogue's barrier;
//   * 16 epilogue warps: accumulator -> + bias, activation, split -> 16-byte stores of the next layer's A, in
//     32-column blocks; every finished block releases two k-steps of the next layer's mma, which accumulates into
//     the other half of TMEM (2 x 256 columns), so the epilogue of layer l overlaps the mma of layer l + 1; the head
//     (N = 16) ends in the de-standardisation, policy and blend of closure_mlp.cu.
// Roles: warps 0-15 epilogue (warp w: TMEM lanes 32 (w % 4) .., columns 64 (w / 4) ..; warps 0-3 also compute the
// features and finish the head), warp 16 producer, warp 17 mma issuer.  One CTA per SM, persistent over tiles.
#pragma once
#include <cuda_bf16.h>

#define W5_EPI_WARPS 16                           // 4 per TMEM lane quarter, each owns 64 of the 256 columns
#define W5_THREADS ((W5_EPI_WARPS + 2) * 32)
#define W5_M 128
#ifndef W5_STAGES
#define W5_STAGES 4
#endif
#define W5_STAGE_BYTES 16384                      // 256 units x 16 inputs x (hi + lo) bf16
#define W5_A_PART (W5_M * WD_H * 2)               // 64 KB: one part (hi or lo) of the activations

__host__ __device__ inline size_t w5_blob_bytes(int n_layers)
{
    return (size_t)W5_STAGE_BYTES * (1 + (size_t)(n_layers - 2) * (WD_H / 16)) + (size_t)(WD_H / 16) * 1024;
}

__device__ __forceinline__ void w5_wait(uint64_t* bar, uint32_t parity)
{
    uint32_t done = 0;
    unsigned long long t0 = 0;
    while (true) {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(fpt_smem_u32(bar)), "r"(parity) : "memory");
        if (done) break;
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        if (t0 == 0) t0 = t;
        else if (t - t0 > 2000000000ull) __trap();           // 2 s: a protocol error must not hang the device
    }
}
__device__ __forceinline__ void w5_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(fpt_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void w5_commit(uint64_t* bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(fpt_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void w5_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void w5_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// shared-memory matrix descriptor, K-major, no swizzle (cute/arch/mma_sm100_desc.hpp: address, LBO, SBO in 16-byte
// units at bits 0, 16, 32; version 1 at bit 46; layout type 0)
__device__ __forceinline__ uint64_t w5_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes)
{
    return (uint64_t)((saddr >> 4) & 0x3FFFu) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16) |
           ((uint64_t)((sbo_bytes >> 4) & 0x3FFFu) << 32) | (1ull << 46);
}
// instruction descriptor: D fp32, A and B bf16, both K-major, M = 128
__device__ __forceinline__ uint32_t w5_idesc(int n) { return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(W5_M >> 4) << 24); }
__device__ __forceinline__ void w5_mma(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void w5_ld32(uint32_t taddr, uint32_t (&v)[32])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"
                 "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                   "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
                   "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
                   "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
                 : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void w5_ld8(uint32_t taddr, uint32_t (&v)[8])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                 : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void w5_ld16(uint32_t taddr, uint32_t (&v)[16])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                   "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                 : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// Pack the weights as stage images.  Chunk sequence: layer 0 (1 chunk, inputs 0..15), each hidden layer (16 chunks),
// head (16 chunks of N = 16).  A chunk = [hi part | lo part], a part = N x 16 bf16 in canonical K-major order:
// byte(n, k) = (k / 8) * (N / 8) * 128 + (n / 8) * 128 + (n % 8) * 16 + (k % 8) * 2.  One thread per 16-byte unit.
__global__ void mlpw5_pack_kernel(const __grid_constant__ mlp_src S, int32_t n_layers, int32_t nin, uint4* __restrict__ blob)
{
    fpd_pdl();
    const size_t nunits = w5_blob_bytes(n_layers) / 16;
    const size_t big = (size_t)(1 + (n_layers - 2) * (WD_H / 16)) * (W5_STAGE_BYTES / 16);   // units in 16 KB chunks
    for (size_t u = (size_t)blockIdx.x * blockDim.x + threadIdx.x; u < nunits; u += (size_t)gridDim.x * blockDim.x) {
        int l, kc, N;
        size_t r;
        if (u < big) {
            const size_t c = u / (W5_STAGE_BYTES / 16);
            r = u % (W5_STAGE_BYTES / 16);
            N = WD_H;
            if (c == 0) { l = 0; kc = 0; }
            else { l = 1 + (int)((c - 1) / (WD_H / 16)); kc = (int)((c - 1) % (WD_H / 16)); }
        } else {
            const size_t v = u - big;
            l = n_layers - 1; kc = (int)(v / 64); r = v % 64; N = 16;
        }
        const int part = (int)(r / (size_t)(N * 2));            // N * 2 units per part
        const int q = (int)(r % (size_t)(N * 2));
        const int khalf = q / N, n = q % N;                      // unit (khalf, n): n / 8 groups of 8 rows x 16 B
        const int ni = (l == 0) ? nin : WD_H, no = (l == n_layers - 1) ? 9 : WD_H;
        uint32_t w[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int k0 = 16 * kc + 8 * khalf + 2 * i;
            const float a = (n < no && k0 < ni) ? S.W[l][(size_t)n * ni + k0] : 0.0f;
            const float b = (n < no && k0 + 1 < ni) ? S.W[l][(size_t)n * ni + k0 + 1] : 0.0f;
            uint32_t hi, lo;
            wd_split2(a, b, hi, lo);
            w[i] = part == 0 ? hi : lo;
        }
        blob[u] = make_uint4(w[0], w[1], w[2], w[3]);
    }
}

__global__ void __launch_bounds__(W5_THREADS, 1)
mlp_wide5_kernel(const double* __restrict__ mom, const float* __restrict__ tau_cell, const unsigned char* __restrict__ blob,
                 const float* __restrict__ misc, float* __restrict__ coef, uint32_t* __restrict__ flags,
                 const __grid_constant__ wd_params P)
{
    fpd_pdl();
    extern __shared__ __align__(1024) unsigned char w5_smem[];
    unsigned char* a_hi = w5_smem;                                        // [32 slabs][16 groups][8 rows][8 inputs] bf16
    unsigned char* a_lo = a_hi + W5_A_PART;
    unsigned char* bst = a_lo + W5_A_PART;                                // [W5_STAGES][W5_STAGE_BYTES]
    float* ms = reinterpret_cast<float*>(bst + W5_STAGES * W5_STAGE_BYTES);
    const int nmisc = wd_misc_floats(P.n_layers);
    uint64_t* bars = reinterpret_cast<uint64_t*>(ms + ((nmisc + 3) & ~3));
    uint64_t* full = bars;                       // [W5_STAGES] producer -> mma
    uint64_t* empty = bars + W5_STAGES;          // [W5_STAGES] mma -> producer
    uint64_t* a_blk = bars + 2 * W5_STAGES;      // [8] epilogue -> mma: 32-input block b of the next layer's A is written
    uint64_t* d_ready = a_blk + 8;               // mma -> epilogue
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(d_ready + 1);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int L = P.n_layers;
    for (int i = tid; i < nmisc; i += W5_THREADS) ms[i] = misc[i];
    if (tid == 0) {
        for (int s = 0; s < W5_STAGES; ++s) { fpt_mbar_init(&full[s], 1); fpt_mbar_init(&empty[s], 1); }
        for (int b = 0; b < 8; ++b) fpt_mbar_init(&a_blk[b], W5_EPI_WARPS * 32);
        fpt_mbar_init(d_ready, 1);
    }
    if (warp == W5_EPI_WARPS + 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(fpt_smem_u32(tmem_slot)), "r"(512u) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    w5_fence_before();
    __syncthreads();
    w5_fence_after();
    const uint32_t tmem = *tmem_slot;
    const int ntiles = (P.ncell + W5_M - 1) / W5_M;
    const int chunks_per_tile = 1 + (L - 2) * (WD_H / 16) + WD_H / 16;

    if (warp == W5_EPI_WARPS) {
        // ===== producer: one lane streams the chunk sequence of every tile through the ring =====
        if (lane == 0) {
            uint32_t it = 0;
            for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
                size_t off = 0;
                for (int c = 0; c < chunks_per_tile; ++c, ++it) {
                    const uint32_t s = it % W5_STAGES, ph = (it / W5_STAGES) & 1u;
                    const uint32_t bytes = (c < chunks_per_tile - WD_H / 16) ? W5_STAGE_BYTES : 1024u;
                    w5_wait(&empty[s], ph ^ 1u);
                    fpt_mbar_expect_tx(&full[s], bytes);
                    fpt_bulk_g2s(bst + (size_t)s * W5_STAGE_BYTES, blob + off, bytes, &full[s]);
                    off += bytes;
                }
            }
        }
    } else if (warp == W5_EPI_WARPS + 1) {
        // ===== mma issuer =====
        if (lane == 0) {
            uint32_t it = 0, ph0 = 0, ph1 = 0;          // completed phases of a_blk[0] and of a_blk[1..7]
            const uint32_t a_hi_s = fpt_smem_u32(a_hi), a_lo_s = fpt_smem_u32(a_lo), b_s = fpt_smem_u32(bst);
            for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
                for (int l = 0; l < L; ++l) {
                    const int nchunks = (l == 0) ? 1 : WD_H / 16;
                    const int N = (l == L - 1) ? 16 : WD_H;
                    const uint32_t idesc = w5_idesc(N);
                    const uint32_t lbo_b = (uint32_t)(N / 8) * 128u, part_b = (uint32_t)N * 32u;
                    const uint32_t dcol = tmem + (uint32_t)(l & 1) * 256u;     // accumulators alternate between layers
                    for (int c = 0; c < nchunks; ++c, ++it) {
                        if ((c & 1) == 0) {                  // inputs 16c .. 16c+31 = block c/2 of the producer's epilogue
                            w5_wait(&a_blk[c >> 1], (c == 0 ? ph0 : ph1) & 1u);
                            w5_fence_after();
                        }
                        const uint32_t s = it % W5_STAGES, ph = (it / W5_STAGES) & 1u;
                        w5_wait(&full[s], ph);
                        w5_fence_after();
                        const uint32_t bb = b_s + s * W5_STAGE_BYTES;
                        const uint64_t ah = w5_desc(a_hi_s + (uint32_t)c * 4096u, 2048u, 128u);
                        const uint64_t al = w5_desc(a_lo_s + (uint32_t)c * 4096u, 2048u, 128u);
                        const uint64_t bh = w5_desc(bb, lbo_b, 128u);
                        const uint64_t bl = w5_desc(bb + part_b, lbo_b, 128u);
                        w5_mma(dcol, ah, bh, idesc, c > 0 ? 1u : 0u);
                        w5_mma(dcol, al, bh, idesc, 1u);
                        w5_mma(dcol, ah, bl, idesc, 1u);
                        w5_commit(&empty[s]);
                    }
                    ++ph0;
                    if (l > 0) ++ph1;
                    w5_commit(d_ready);
                }
            }
        }
    } else {
        // ===== epilogue warps: row = TMEM lane 32 (warp % 4) + lane, columns 64 (warp / 4) .. + 63 =====
        const int row = 32 * (warp & 3) + lane, cg = warp >> 2;
        const float* hbias = ms + (L - 1) * WD_H;
        const float* xmean = hbias + 16, *xscale = xmean + 16, *ymean = xscale + 16, *yscale = ymean + 16;
        const uint32_t row_off = (uint32_t)(row >> 3) * 128u + (uint32_t)(row & 7) * 16u;   // inside an 8-input slab
        const uint32_t tlane = tmem + ((uint32_t)(32 * (warp & 3)) << 16);
        uint32_t dr = 0;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const int cell = tile * W5_M + row;
            const bool have = cg == 0 && cell < P.ncell;
            double nraw = 0.0, theta = 0.0;
            float tau = P.tau_scalar;
            bool zbad = false;
            if (cg == 0) {
                float x[16];
#pragma unroll
                for (int i = 0; i < 16; ++i) x[i] = 0.0f;
                if (have) {
                    const double* rec = mom + (size_t)cell * P.stride;
                    nraw = rec[0];
                    theta = (rec[4] + rec[7] + rec[9]) / 3.0;
                    if (tau_cell) tau = tau_cell[cell];
                    double h[3];
                    if (P.stride == 13) { h[0] = rec[10]; h[1] = rec[11]; h[2] = rec[12]; }
                    else { h[0] = rec[10] + rec[13] + rec[15]; h[1] = rec[11] + rec[16] + rec[18]; h[2] = rec[12] + rec[17] + rec[19]; }
                    const double n = nraw * (double)P.n_scale;
                    if (P.feature_set == 0) {
                        x[0] = (float)n; x[1] = (float)rec[1]; x[2] = (float)rec[2]; x[3] = (float)rec[3];
                        x[4] = (float)(theta / (double)P.theta_ref);
                        x[5] = (float)(n * (rec[4] - theta)); x[6] = (float)(n * rec[5]); x[7] = (float)(n * rec[6]);
                        x[8] = (float)(n * (rec[7] - theta)); x[9] = (float)(n * rec[8]);
                        x[10] = (float)(0.5 * n * h[0]); x[11] = (float)(0.5 * n * h[1]); x[12] = (float)(0.5 * n * h[2]);
                    } else {
                        x[0] = (float)n; x[1] = (float)(theta / (double)P.theta_ref);
                        x[2] = (float)rec[1]; x[3] = (float)rec[2]; x[4] = (float)rec[3];
#pragma unroll
                        for (int k = 0; k < 6; ++k) x[5 + k] = (float)(n * rec[4 + k]);
                        x[11] = (float)(0.5 * n * h[0]); x[12] = (float)(0.5 * n * h[1]); x[13] = (float)(0.5 * n * h[2]);
                        x[14] = (float)(3.0 * theta);
                        x[15] = (float)(1.0 / (double)tau);
                    }
                }
                uint32_t hi[8], lo[8];
#pragma unroll
                for (int i = 0; i < 16; i += 2) {
                    float z0 = (i < P.nin) ? (x[i] - xmean[i]) / xscale[i] : 0.0f;
                    float z1 = (i + 1 < P.nin) ? (x[i + 1] - xmean[i + 1]) / xscale[i + 1] : 0.0f;
                    if (have && (!isfinite(z0) || !isfinite(z1))) zbad = true;
                    if (!have || !isfinite(z0)) z0 = 0.0f;
                    if (!have || !isfinite(z1)) z1 = 0.0f;
                    wd_split2(z0, z1, hi[i / 2], lo[i / 2]);
                }
                *reinterpret_cast<uint4*>(a_hi + row_off) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
                *reinterpret_cast<uint4*>(a_hi + 2048 + row_off) = make_uint4(hi[4], hi[5], hi[6], hi[7]);
                *reinterpret_cast<uint4*>(a_lo + row_off) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
                *reinterpret_cast<uint4*>(a_lo + 2048 + row_off) = make_uint4(lo[4], lo[5], lo[6], lo[7]);
            }
            fpt_fence_proxy_async();                      // generic-proxy stores -> visible to the tensor core's reads
            w5_arrive(&a_blk[0]);
            // ---- layers 0 .. L-2: accumulator -> bias, activation, split -> next layer's A (in place)
            for (int l = 0; l < L - 1; ++l) {
                w5_wait(d_ready, dr & 1u);
                ++dr;
                w5_fence_after();
                const float* bias = ms + l * WD_H;
                const uint32_t dcol = tlane + (uint32_t)(l & 1) * 256u;
                // 32-column blocks in order; the four warps of a row quarter take 8 columns each, and every finished
                // block releases two k-steps of the next layer's mma (which writes the other accumulator)
#pragma unroll 1
                for (int cb = 0; cb < WD_H / 32; ++cb) {
                    uint32_t v[8];
                    w5_ld8(dcol + (uint32_t)(32 * cb + 8 * cg), v);
                    uint32_t hi[4], lo[4];
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int c0 = 32 * cb + 8 * cg + 2 * i;
                        float s0 = __uint_as_float(v[2 * i]) + bias[c0];
                        float s1 = __uint_as_float(v[2 * i + 1]) + bias[c0 + 1];
                        s0 = (P.act == 0) ? __fdividef(s0, 1.0f + __expf(-s0)) : fmaxf(s0, 0.0f);
                        s1 = (P.act == 0) ? __fdividef(s1, 1.0f + __expf(-s1)) : fmaxf(s1, 0.0f);
                        wd_split2(s0, s1, hi[i], lo[i]);
                    }
                    const uint32_t o = (uint32_t)(4 * cb + cg) * 2048u + row_off;
                    *reinterpret_cast<uint4*>(a_hi + o) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
                    *reinterpret_cast<uint4*>(a_lo + o) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
                    w5_fence_before();                    // the tcgen05.ld above is complete
                    fpt_fence_proxy_async();
                    w5_arrive(&a_blk[cb]);
                }
            }
            // ---- head: 16 accumulator columns -> de-standardise, policy, blend
            w5_wait(d_ready, dr & 1u);
            ++dr;
            w5_fence_after();
            uint32_t yv[16];
            if (cg == 0) w5_ld16(tlane + (uint32_t)((L - 1) & 1) * 256u, yv);
            w5_fence_before();
            if (have) {
                float y[9];
                bool finite = !zbad;
#pragma unroll
                for (int k = 0; k < 9; ++k) {
                    y[k] = fmaf(__uint_as_float(yv[k]) + hbias[k], yscale[k], ymean[k]);
                    finite = finite && isfinite(y[k]);
                }
                float* out = coef + (size_t)cell * 9;
                uint32_t flag = 0;
                if (!(nraw > 0.0)) {
#pragma unroll
                    for (int k = 0; k < 9; ++k) y[k] = 0.0f;
                    flag = FP_FLAG_EMPTY;
                } else {
                    bool langevin = false;
                    if (nraw < (double)P.min_count) { flag = FP_FLAG_LOWCOUNT; langevin = true; }
                    else if (!(theta > 0.0) || !isfinite(theta)) { flag = FP_FLAG_SINGULAR; langevin = true; }
                    else if (!finite) { flag = FP_FLAG_NONFINITE; langevin = true; }
                    if (langevin) {
                        const float d = -1.0f / tau;
                        y[0] = d; y[1] = 0.f; y[2] = 0.f; y[3] = d; y[4] = 0.f; y[5] = d; y[6] = 0.f; y[7] = 0.f; y[8] = 0.f;
                    }
                    if (P.relax_w != 1.0f) {
                        // no history (all nine old coefficients zero: EMPTY last step / zero-initialised first step): no blend (R12)
                        bool history = false;
#pragma unroll
                        for (int k = 0; k < 9; ++k) history = history || out[k] != 0.0f;
                        if (history) {
#pragma unroll
                            for (int k = 0; k < 9; ++k) y[k] = P.relax_w * y[k] + (1.0f - P.relax_w) * out[k];
                        }
                    }
                }
#pragma unroll
                for (int k = 0; k < 9; ++k) out[k] = y[k];
                if (P.cellc)
                    flag |= upd_prep_cell(mom + (size_t)cell * P.stride, P.stride, y, (double)tau, P.dt, P.eps2_scale,
                                          P.cellc + (size_t)cell * UPD_NC);
                flags[cell] = flag;
            }
        }
    }
    // ---- teardown
    w5_fence_before();
    __syncthreads();
    if (warp == W5_EPI_WARPS + 1) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
    }
}
