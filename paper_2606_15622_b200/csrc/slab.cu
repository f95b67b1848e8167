// slab.cu -- SURVEY 8(f) NEXT-4: the device-side pieces of a slab decomposition with one particle exchange per step.
//
// The paper runs one GPU and independent replicas (:668); cutting ONE domain over several devices
// is this build's extension.  The grid is cut into slabs of whole rows; every context is created with the GLOBAL
// geometry (walls, body and the cell-index formula are those of the whole domain) and told which rows it owns
// (fp_set_slab).  A step on a slab is
//     fp_stream_walls                  stream + walls on the slab's particles, global geometry
//     fp_slab_partition                stable partition by destination slab: [to slab 0 | to slab 1 | ...], counts on the device
//     -- exchange (host side: torch.distributed all_to_all over NCCL, or device copies between contexts of one process) --
//        the receive buffer is the concatenation over SOURCE slabs in ascending order, the slab's own stayers in their place
//     fp_collide                       sort by (local) cell -> moments -> closure -> update on the particles now owned
// Because the partition is stable and the receive order is the source order, the array a slab sorts is exactly the
// sub-sequence of the single-domain array that it owns: with the stable cell sort every cell sees its particles in the
// same order as in the uncut run, so the cut run is bit-identical to it (tests/test_gpu_slab.py), not merely close.
#include "common.cuh"

#define SLAB_MAX 64

struct slab_bounds { int32_t n; int32_t row[SLAB_MAX + 1]; };

// destination slab of every particle (the slab whose rows contain the particle's global row) + the tile histogram the
// first (only) radix pass needs
__global__ void __launch_bounds__(SORT_THREADS)
slab_dest_kernel(int64_t np, const float* __restrict__ y, uint32_t* __restrict__ keys, const fp_grid G, const slab_bounds B,
                 uint32_t* __restrict__ block_hist, int nblocks, int bins)
{
    fpd_pdl();
    __shared__ uint32_t h[SORT_MAX_BINS];
    for (int b = threadIdx.x; b < bins; b += SORT_THREADS) h[b] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * SORT_TILE;
#pragma unroll 4
    for (int i = 0; i < SORT_ITEMS; ++i) {
        const int64_t p = base + i * SORT_THREADS + threadIdx.x;
        if (p < np) {
            const int32_t row = G.ny > 1 ? fpd_axis_index(y[p], G.y0, G.inv_dy, G.ny) : 0;
            int d = 0;
            while (d + 1 < B.n && row >= B.row[d + 1]) ++d;
            keys[p] = (uint32_t)d;
            atomicAdd(&h[d], 1u);
        }
    }
    __syncthreads();
    for (int b = threadIdx.x; b < bins; b += SORT_THREADS) block_hist[(size_t)b * nblocks + blockIdx.x] = h[b];
}

extern "C" int fp_set_slab(fp_ctx* ctx, int32_t row0, int32_t nrows)
{
    if (!ctx) return FP_ERR_ARG;
    if (row0 < 0 || nrows < 1 || row0 + nrows > ctx->p.ny) return fp_fail(ctx, FP_ERR_ARG, "fp_set_slab: rows outside the grid");
    ctx->slab_row0 = row0; ctx->slab_rows = nrows;
    ctx->ncell = ctx->p.nx * nrows;
    int bits = 0;
    while (((int64_t)1 << bits) < (int64_t)ctx->ncell) ++bits;
    ctx->key_bits = bits;
    return FP_OK;
}

extern "C" int fp_set_reproducible(fp_ctx* ctx, int32_t on)
{
    if (!ctx) return FP_ERR_ARG;
    ctx->reproducible = on != 0;
    return FP_OK;
}

extern "C" int fp_slab_partition(fp_ctx* ctx, int64_t np,
                                 const float* x, const float* y, const float* vx, const float* vy, const float* vz,
                                 const uint32_t* pid, float* x_out, float* y_out, float* vx_out, float* vy_out, float* vz_out,
                                 uint32_t* pid_out, const int32_t* h_row_bounds, int32_t nslabs, int32_t* slab_start, void* stream)
{
    if (!ctx) return FP_ERR_ARG;
    if (np < 0 || !h_row_bounds || nslabs < 1 || nslabs > SLAB_MAX || !slab_start)
        return fp_fail(ctx, FP_ERR_ARG, "fp_slab_partition: bad argument (1 <= nslabs <= 64)");
    if (np > ctx->p.max_particles) return fp_fail(ctx, FP_ERR_STATE, "fp_slab_partition: np > max_particles");
    if (np > 0 && (!x || !y || !vx || !vy || !vz || !pid || !x_out || !y_out || !vx_out || !vy_out || !vz_out || !pid_out))
        return fp_fail(ctx, FP_ERR_ARG, "fp_slab_partition: null pointer");
    slab_bounds B;
    B.n = nslabs;
    for (int s = 0; s <= nslabs; ++s) {
        B.row[s] = h_row_bounds[s];
        if ((s > 0 && B.row[s] <= B.row[s - 1]) || B.row[s] < 0 || B.row[s] > ctx->p.ny)
            return fp_fail(ctx, FP_ERR_ARG, "fp_slab_partition: row bounds must increase from 0 to ny");
    }
    if (B.row[0] != 0 || B.row[nslabs] != ctx->p.ny) return fp_fail(ctx, FP_ERR_ARG, "fp_slab_partition: row bounds must cover 0 .. ny");
    cudaStream_t st = (cudaStream_t)stream;
    // the partition is the library's stable radix sort with the destination slab as the key: one pass of <= 6 bits
    const int32_t ncell_saved = ctx->ncell, bits_saved = ctx->key_bits;
    int bits = 1;
    while ((1 << bits) < nslabs) ++bits;
    ctx->ncell = nslabs; ctx->key_bits = bits; ctx->sort_slab_keys = true;
    int rc = FP_OK;
    if (np > 0) {
        const int nblocks = fp_div_up(np, SORT_TILE);
        fp_launch(slab_dest_kernel, nblocks, SORT_THREADS, 0, st, np, y, ctx->key_b, fp_grid_of(ctx), B, ctx->block_hist, nblocks,
                  1 << fpi_sort_digit_bits(ctx));
        if (cudaGetLastError() != cudaSuccess) rc = fp_fail(ctx, FP_ERR_CUDA, "fp_slab_partition: launch failed");
        FP_COUNT(ctx, 1);
    }
    if (rc == FP_OK)
        rc = fpi_sort_with_keys(ctx, np, ctx->key_b, np > 0, x, y, vx, vy, vz, pid, x_out, y_out, vx_out, vy_out, vz_out, pid_out,
                                slab_start, nullptr, st);
    ctx->ncell = ncell_saved; ctx->key_bits = bits_saved; ctx->sort_slab_keys = false;
    return rc;
}
