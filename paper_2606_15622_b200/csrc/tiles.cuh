// tiles.cuh -- particle tiles for the per-cell kernels (moments, update).
//
// The cell-sorted particle stream is cut into tiles of about FPT_T particles that hold whole cells: tile b owns the
// cells whose first-particle index lies in [b*FPT_T, (b+1)*FPT_T).  One CTA processes one tile: it stages the tile's
// SoA slices in shared memory with 1D bulk asynchronous copies (cp.async.bulk -> UBLKCP, completion on an mbarrier),
// so HBM is read once, fully coalesced, and all later passes over the cell's particles hit shared memory.
// ntiles = np / FPT_T + 1 (the last window also catches trailing empty cells, whose start equals np).
#pragma once
#include "common.cuh"

#define FPT_T 2048                 // particles per tile window
#define FPT_CAP 2560               // staged elements per array: FPT_T - 1 + largest cell that still fits, rounded

#ifdef __CUDACC__

__device__ __forceinline__ uint32_t fpt_smem_u32(const void* p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void fpt_mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(fpt_smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fpt_mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(fpt_smem_u32(bar)), "r"(bytes) : "memory");
}
// 1D bulk copy global -> shared; src, dst 16-byte aligned, bytes a multiple of 16
__device__ __forceinline__ void fpt_bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(fpt_smem_u32(dst)), "l"(src), "r"(bytes), "r"(fpt_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fpt_mbar_wait(uint64_t* bar, uint32_t parity)
{
    uint32_t done = 0;
    while (!done) {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(fpt_smem_u32(bar)), "r"(parity) : "memory");
    }
}
// 1D bulk copy shared -> global (bulk async-group completion)
__device__ __forceinline__ void fpt_bulk_s2g(void* dst, const void* src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(fpt_smem_u32(src)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void fpt_bulk_commit_wait()
{
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}
__device__ __forceinline__ void fpt_fence_proxy_async()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

struct fpt_tile {
    int32_t c0, c1;        // cells [c0, c1)
    int32_t s0, s1;        // particles [s0, s1)
    int32_t a0;            // s0 rounded down to a multiple of 4: staged element k holds particle a0 + k
    int32_t nb;            // elements covered by the bulk copies (multiple of 4), starting at a0
    bool staged;           // false: the tile does not fit (huge cell) or the arrays are not 16-byte aligned
};

__device__ __forceinline__ fpt_tile fpt_tile_of_block(const int32_t* __restrict__ tile_cell,
                                                      const int32_t* __restrict__ cell_start, int32_t ncell,
                                                      int64_t np, bool aligned)
{
    fpt_tile t;
    t.c0 = tile_cell[blockIdx.x];
    t.c1 = min(tile_cell[blockIdx.x + 1], ncell);
    t.s0 = t.s1 = t.a0 = t.nb = 0;
    t.staged = false;
    if (t.c0 >= t.c1) return t;
    t.s0 = cell_start[t.c0];
    t.s1 = cell_start[t.c1];
    t.a0 = t.s0 & ~3;
    const int32_t np4 = (int32_t)(np & ~(int64_t)3);
    const int32_t end4 = min((t.s1 + 3) & ~3, np4);
    t.nb = max(end4 - t.a0, 0);
    t.staged = aligned && (t.s1 - t.a0) <= FPT_CAP && t.s1 > t.s0;
    return t;
}

#endif  // __CUDACC__

// host side (tiles.cu)
int fpi_tile_table(fp_ctx* ctx, int64_t np, const int32_t* cell_start, cudaStream_t st);
static inline int fpi_ntiles(int64_t np) { return (int)(np / FPT_T) + 1; }
