// tiles.cuh -- per-warp staging of contiguous particle slices in shared memory (moments, update).
//
// The per-cell kernels give every warp 32/G consecutive cells.  Their particles are one contiguous slice of each SoA
// array, which the warp copies into its own shared-memory buffer with 1D bulk asynchronous copies (cp.async.bulk ->
// UBLKCP, completion on the warp's own mbarrier): HBM is read once, fully coalesced, and all later passes over the
// cells hit shared memory.  Bulk copies need 16-byte alignment: the slice is widened to multiples of 4 elements,
// the (at most 3) elements past the last multiple of 4 of the whole array are copied by plain loads.
#pragma once
#include "common.cuh"

#define FPW_CAP 512                // staged elements per array, warp and stage (4 cells x 128 particles)
// Lanes per cell G by mean particles per cell: a warp's chunk of 32/G cells has to fit FPW_CAP with room for the
// count fluctuations (at the mean where G changes the chunk holds 7/8 of the buffer); chunks that still do not fit
// are walked cell by cell with all 32 lanes.
#ifndef FPW_G8_MIN
#define FPW_G8_MIN 56.0            // 8 cells x 56 = 448
#endif
#ifndef FPW_G16_MIN
#define FPW_G16_MIN 112.0          // 4 cells x 112 = 448
#endif
#ifndef FPW_G32_MIN
#define FPW_G32_MIN 224.0          // 2 cells x 224 = 448
#endif

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

// Block-wide staging of a contiguous slab (e.g. the moment records of the block's cells): one bulk copy when the
// slab is 16-byte aligned, plain loads for the remainder.  Ends with __syncthreads().  `bar` must be a block-shared
// mbarrier used for nothing else.
__device__ __forceinline__ void fpt_block_stage(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    const bool aligned = ((reinterpret_cast<uintptr_t>(src) | reinterpret_cast<uintptr_t>(dst)) & 15u) == 0;
    const uint32_t bulk = aligned ? (bytes & ~15u) : 0u;
    if (threadIdx.x == 0 && bulk > 0) {
        fpt_mbar_init(bar, 1);
        fpt_mbar_expect_tx(bar, bulk);
        fpt_bulk_g2s(dst, src, bulk, bar);
    }
    for (uint32_t o = bulk + threadIdx.x * 4u; o < bytes; o += blockDim.x * 4u)
        *reinterpret_cast<uint32_t*>(static_cast<unsigned char*>(dst) + o) =
            *reinterpret_cast<const uint32_t*>(static_cast<const unsigned char*>(src) + o);
    __syncthreads();                                     // barrier initialised and visible to every thread
    if (bulk > 0) fpt_mbar_wait(bar, 0);
    __syncthreads();
}

struct fpw_range {
    int32_t s0, s1;        // particles [s0, s1) of the warp's cells
    int32_t a0;            // s0 rounded down to a multiple of 4: staged element k holds particle a0 + k
    int32_t nb;            // elements covered by the bulk copies (multiple of 4), starting at a0
    bool staged;           // false: the slice does not fit FPW_CAP or the arrays are not 16-byte aligned
};

__device__ __forceinline__ fpw_range fpw_range_of(int32_t s0, int32_t s1, int64_t np, bool aligned, int32_t cap = FPW_CAP)
{
    fpw_range r;
    r.s0 = s0; r.s1 = s1;
    r.a0 = s0 & ~3;
    const int32_t np4 = (int32_t)(np & ~(int64_t)3);
    const int32_t end4 = min((s1 + 3) & ~3, np4);
    r.nb = max(end4 - r.a0, 0);
    // (s1 - a0) <= (s1 - s0) + 3: the bound does not depend on where the slice starts, so a chunk takes the same path
    // (staged or walked) wherever its particles sit in the arrays (fp_set_reproducible, slab decompositions)
    r.staged = aligned && s1 > s0 && (s1 - s0) + 3 <= cap;
    return r;
}

#endif  // __CUDACC__

int fpi_velocity_update(fp_ctx* ctx, int64_t np, float* vx, float* vy, float* vz, const uint32_t* pid,
                        const int32_t* cell_start, const double* mom, int32_t mom_stride, const float* coef,
                        const float* tau_cell, uint64_t step, uint32_t* flags, bool prep_done, cudaStream_t st);
