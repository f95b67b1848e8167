// tiles.cu -- the particle-tile table (tiles.cuh): tile_cell[b] = first cell whose first-particle index >= b*FPT_T.
#include "tiles.cuh"

__global__ void __launch_bounds__(128)
tile_table_kernel(const int32_t* __restrict__ cell_start, int32_t ncell, int32_t ntiles, int32_t* __restrict__ tile_cell)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b > ntiles) return;
    if (b == ntiles) { tile_cell[b] = ncell; return; }
    const int64_t target = (int64_t)b * FPT_T;
    int lo = 0, hi = ncell;                      // first c in [0, ncell] with cell_start[c] >= target
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if ((int64_t)cell_start[mid] >= target) hi = mid; else lo = mid + 1;
    }
    tile_cell[b] = lo;
}

int fpi_tile_table(fp_ctx* ctx, int64_t np, const int32_t* cell_start, cudaStream_t st)
{
    if (np > ctx->p.max_particles) return fp_fail(ctx, FP_ERR_STATE, "np > max_particles (tile table scratch)");
    const int ntiles = fpi_ntiles(np);
    tile_table_kernel<<<fp_div_up(ntiles + 1, 128), 128, 0, st>>>(cell_start, ctx->ncell, ntiles, ctx->tile_cell);
    FP_LAUNCH_OK(ctx);
    FP_COUNT(ctx, 1);
    return FP_OK;
}
