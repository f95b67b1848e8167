// common.cuh -- context, launch helpers and small device utilities shared by the fpcl kernels (sm_100a).
// Product code: shares nothing with oracle/ (test infrastructure).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/fpcl.h"

#define FPCL_MAX_LAYERS 8
// radix sort tiling (sort.cu; the key kernel also produces the first digit histogram per tile)
#define SORT_THREADS 256
#define SORT_WARPS (SORT_THREADS / 32)
#ifndef SORT_ITEMS
#define SORT_ITEMS 16                                    // items per thread
#endif
#define SORT_TILE (SORT_THREADS * SORT_ITEMS)            // 4096 items per block
#define SORT_MAX_BINS 512
#define FPCL_NUM_SMS_DEFAULT 148

// ---------------------------------------------------------------------------------------------------------
// Context.  Owns scratch only (include/fpcl.h "Conventions").
// ---------------------------------------------------------------------------------------------------------
struct fp_mlp_dev {                 // uploaded copy of the caller's MLP (fp_closure_mlp caches it)
    int32_t  n_layers = 0;
    int32_t  dims[FPCL_MAX_LAYERS + 1] = {0};
    int32_t  act = 0, feature_set = 0;
    float    n_scale = 1.f, theta_ref = 0.5f;
    float*   tc_frags = nullptr;    // device: packed 3xTF32 mma fragments + biases/scalers (mlp_tc.cuh)
    float*   wd_frags = nullptr;    // device: packed split-bf16 mma fragments + biases/scalers (mlp_wide.cuh)
    size_t   wd_bytes = 0;
    void*    w5_blob = nullptr;     // device: weights as tcgen05 stage images + biases/scalers (mlp_wide5.cuh)
    size_t   w5_bytes = 0;
    float*   blob = nullptr;        // device: [W0 | b0 | W1 | b1 | ... | x_mean | x_scale | y_mean | y_scale]
    size_t   blob_floats = 0;
    size_t   w_off[FPCL_MAX_LAYERS] = {0}, b_off[FPCL_MAX_LAYERS] = {0};
    size_t   xm_off = 0, xs_off = 0, ym_off = 0, ys_off = 0;
    // identity of the source, to skip re-uploading
    const void* src_W[FPCL_MAX_LAYERS] = {nullptr};
    const void* src_b[FPCL_MAX_LAYERS] = {nullptr};
    const void* src_x_mean = nullptr;
    bool     valid = false;
};

#define SW_TB_CAP 4095               // entries of the reservoir's tie-break list (expected: a handful per step at 20M particles)
#define UPD_ACC 8                  // doubles per cell in upd_acc: seven sums (update.cu: upd_scales), one pad

struct fp_ctx {
    fp_params p;
    int32_t   ncell = 0;
    int32_t   key_bits = 0;         // bits needed for keys in [0, ncell)
    float     inv_dx = 0.f, inv_dy = 0.f;
    float     xmin = 0.f, xmax = 0.f, ymin = 0.f, ymax = 0.f, xmax_in = 0.f, ymax_in = 0.f, Lx = 0.f, Ly = 0.f;
    int       device = 0, num_sms = FPCL_NUM_SMS_DEFAULT;
    bool      reproducible = false;  // fp_set_reproducible
    int32_t   slab_row0 = 0, slab_rows = 0;   // fp_set_slab: this context owns rows row0 .. row0 + rows - 1 (rows = ny by default)
    // sort scratch (sized for max_particles)
    uint32_t *key_a = nullptr, *key_b = nullptr, *idx_a = nullptr, *idx_b = nullptr;
    uint32_t *block_hist = nullptr;  // two tables [bins][nblocks]: even passes use the first, odd passes the second
    bool      sort_no_pack = false;  // FPCL_SORT_UNPACKED=1: always move (key, index) as two arrays (test hook)
    bool      sort_slab_keys = false; // set by fp_slab_partition around its sort: the keys are destination slabs, not cell keys of the positions
    bool      hist0_clean = true;    // the first table is all zero (what the stream kernel's fused histogram needs)
    uint32_t *bin_total = nullptr;   // [bins]
    size_t    block_hist_elems = 0;
    float    *cellc = nullptr;       // [ncell * 28] per-cell constants of the velocity update (update.cu)
    double   *mom_acc = nullptr;     // [ncell * 28] raw-sum accumulators of the high-ppc gather (moments_seg.cuh)
    double   *upd_acc = nullptr;     // [ncell * UPD_ACC] per-cell sums of the high-ppc update (update_seg.cuh)
    // sticky device-side state check (cell_start not a monotone prefix ending at np): one word of mapped pinned host
    // memory that kernels OR into and every entry point reads without synchronising
    uint32_t *h_err = nullptr, *d_err = nullptr;
    uint32_t *d_errdev = nullptr;    // device-memory copy of the word for kernels that must not run on bad boundaries
    uint32_t *d_tiebreak = nullptr;  // [1 + SW_TB_CAP]: count + particle indices whose reservoir accept/reject test was borderline in fp32
    uint32_t *d_deferred = nullptr;  // [1 + max_particles], reservoir grids only: count + indices of the particles that left through a
                                     // freestream face this step (re-inserted by sw_deferred_kernel)
    int       mom_occ[6] = {0, 0, 0, 0, 0, 0};       // resident CTAs per SM of moments_warp_kernel<2^k, *>
    int       mlp_tc_occ = 0, sw_occ[2] = {0, 0}, gather_occ = 0;
    bool      mlp_attr_w5 = false, mlp_attr_wd = false;
    // test / measurement switches read from the environment once, at fp_create
    bool      env_mom_seg = false, env_mom_no_seg = false, env_upd_seg = false, env_upd_no_seg = false;
    bool      upd_attr[4] = {false, false, false, false};   // shared-memory attribute set for update_warp_kernel<4|8|16|32> (per context, i.e. per device)
    // fp_step_host staging (allocated lazily)
    float    *hs_f[2][5] = {{nullptr}};
    uint32_t *hs_pid[2] = {nullptr, nullptr};
    double   *hs_mom = nullptr;
    float    *hs_coef = nullptr;
    uint32_t *hs_flags = nullptr;
    int32_t  *hs_cell_start = nullptr;
    bool      hs_ready = false;
    // fp_step_host overlap: a side stream for the copies that need not sit on the caller's stream, and the two events
    // the payload gather waits on / records (null outside fp_step_host)
    cudaStream_t hs_side = nullptr;
    cudaEvent_t  hs_ev[4] = {nullptr, nullptr, nullptr, nullptr};
    cudaEvent_t  ev_before_gather = nullptr, ev_after_gather = nullptr;
    fp_mlp_dev mlp;
    bool      mlp_force_fp32 = false;   // FPCL_MLP_FP32=1: always use the plain-FMA surrogate kernel
    bool      mlp_wide_mma_sync = false;   // fp_set_mlp_tensor_cores(ctx, 2): wide networks on mma.sync instead of tcgen05
    // measurement hooks
    uint64_t  launches = 0;
    cudaEvent_t* t_ev = nullptr;     // [t_max * (FP_NSTAGES + 1)]
    int32_t   t_max = 0, t_step = 0;
    bool      t_in_step = false;
    char      err[512];
};

// record the stage-boundary event `mark` (0..FP_NSTAGES) of the step being timed, if any
static inline void fp_mark(fp_ctx* ctx, int mark, cudaStream_t st)
{
    if (ctx->t_in_step) cudaEventRecord(ctx->t_ev[(size_t)ctx->t_step * (FP_NSTAGES + 1) + mark], st);
}

static inline int fp_fail(fp_ctx* ctx, int code, const char* msg)
{
    if (ctx) { snprintf(ctx->err, sizeof(ctx->err), "%s", msg); }
    return code;
}

// bits of the device-side state word (fp_ctx::h_err)
#define FP_DEVERR_CELL_START 1u      // cell_start is not a monotone prefix sum ending at np
// read the sticky state word at the entry of a call (no synchronisation: the word lives in mapped host memory)
static inline int fp_state_check(fp_ctx* ctx, const char* who)
{
    if (ctx->h_err && *(volatile uint32_t*)ctx->h_err) {
        snprintf(ctx->err, sizeof(ctx->err), "%s: an earlier call on this context found cell_start not to be a monotone prefix sum "
                 "ending at np; its cells were skipped (call fp_check to clear)", who);
        return FP_ERR_STATE;
    }
    return FP_OK;
}

#define FP_CUDA_OK(ctx, call)                                                                        \
    do {                                                                                             \
        cudaError_t e__ = (call);                                                                    \
        if (e__ != cudaSuccess) {                                                                    \
            if (ctx) snprintf((ctx)->err, sizeof((ctx)->err), "%s:%d %s: %s", __FILE__, __LINE__, #call, \
                              cudaGetErrorString(e__));                                              \
            return FP_ERR_CUDA;                                                                      \
        }                                                                                            \
    } while (0)

#define FP_LAUNCH_OK(ctx) FP_CUDA_OK(ctx, cudaGetLastError())
#define FP_COUNT(ctx, n) ((ctx)->launches += (n))

#ifdef __CUDACC__
// Launch with programmatic dependent launch allowed: the grid is set up while its predecessor on the stream still
// runs and blocks in fpd_pdl() until that predecessor has completed and its writes are visible.  Every kernel of the
// fp_step chain starts with fpd_pdl(); no kernel triggers its dependents early (measured: an early
// griddepcontrol.launch_dependents parks idle blocks on the SMs and costs 55 us per step, the implicit trigger at
// kernel exit saves 18 us of launch gaps per step at 4M particles).
template <typename... KArgs, typename... Args>
static inline cudaError_t fp_launch(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                                    Args&&... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}
// first statement of a kernel launched with fp_launch (a no-op under a plain launch)
__device__ __forceinline__ void fpd_pdl()
{
    asm volatile("griddepcontrol.wait;" ::: "memory");
}
#endif

static inline int fp_div_up(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }


// internal entry points shared between translation units (not exported)
int fpi_sort_digit_bits(const fp_ctx* ctx);           // width of one radix digit for this grid
int fpi_sort_with_keys(fp_ctx* ctx, int64_t np, const uint32_t* keys, bool hist0_ready,
                       const float* x, const float* y, const float* vx, const float* vy, const float* vz,
                       const uint32_t* pid, float* x_out, float* y_out, float* vx_out, float* vy_out,
                       float* vz_out, uint32_t* pid_out, int32_t* cell_start, uint32_t* perm, cudaStream_t st);
int fpi_stream_walls(fp_ctx* ctx, int64_t np, float* x, float* y, float* vx, float* vy, float* vz,
                     const uint32_t* pid, uint64_t step, uint32_t* keys_out /* nullable */,
                     bool with_hist0 /* also the first pass's tile histograms, needs keys_out */, cudaStream_t st);
int fpi_tau_from_counts(fp_ctx* ctx, const int32_t* cell_start, float tau_ref_n, float* tau_cell, cudaStream_t st);
// the closures; with_update_constants: also fill ctx->cellc for the velocity update that follows (upd_prep.cuh)
int fpi_closure_exact(fp_ctx* ctx, const double* mom_full, const float* tau_cell, float* coef, uint32_t* flags,
                      double* kappa_est, bool with_update_constants, cudaStream_t st);
int fpi_closure_mlp(fp_ctx* ctx, const double* mom, int32_t mom_stride, const float* tau_cell, const fp_mlp* h_mlp,
                    float relax_w, float* coef, uint32_t* flags, bool with_update_constants, cudaStream_t st);

// ---------------------------------------------------------------------------------------------------------
// Device helpers
// ---------------------------------------------------------------------------------------------------------
#ifdef __CUDACC__

// Cell index along one axis (R1): clamp(floorf((p - p0) * inv_d), 0, n-1), NaN -> 0.
// (p - p0) * inv_d is a subtract feeding a multiply: no FMA contraction is possible.
__device__ __forceinline__ int32_t fpd_axis_index(float p, float p0, float inv_d, int32_t n)
{
    float t = floorf(__fmul_rn(__fsub_rn(p, p0), inv_d));
    if (!(t >= 0.0f)) return 0;
    if (t >= (float)n) return n - 1;
    return (int32_t)t;
}

// Cell key of a position.  A context that is a slab of the grid (fp_set_slab: rows row0 .. row0 + nrows - 1) numbers its
// cells from its first row; the row itself always comes from the GLOBAL formula, so that a particle gets the same cell
// whether the grid is cut or not.  (nrows = ny, row0 = 0 without a slab.)
struct fp_grid { int32_t nx, ny; float x0, y0, inv_dx, inv_dy; int32_t row0, nrows; };
__device__ __forceinline__ int32_t fpd_cell_key(float x, float y, const fp_grid& g)
{
    const int32_t ix = fpd_axis_index(x, g.x0, g.inv_dx, g.nx);
    int32_t iy = 0;
    if (g.ny > 1) {
        iy = fpd_axis_index(y, g.y0, g.inv_dy, g.ny) - g.row0;
        iy = min(max(iy, 0), g.nrows - 1);                 // rows of other slabs: only if the caller skipped the exchange
    }
    return iy * g.nx + ix;
}

static inline fp_grid fp_grid_of(const fp_ctx* ctx)
{
    fp_grid g;
    g.nx = ctx->p.nx; g.ny = ctx->p.ny; g.x0 = ctx->p.x0; g.y0 = ctx->p.y0; g.inv_dx = ctx->inv_dx; g.inv_dy = ctx->inv_dy;
    g.row0 = ctx->slab_row0; g.nrows = ctx->slab_rows;
    return g;
}

// Philox4x32-10 (Salmon et al., SC'11; R6).  counter (c0..c3), key (k0,k1).
__device__ __forceinline__ uint4 fpd_philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                   uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return make_uint4(c0, c1, c2, c3);
}

// word -> uniform in (0,1): ((w >> 9) + 0.5) * 2^-23, exact in fp32.
// [1,2) mantissa trick: as_float(0x3f800000 | (w>>9)) = 1 + k 2^-23; minus (1 - 2^-24) is exact.
__device__ __forceinline__ float fpd_uniform(uint32_t w)
{
    return __uint_as_float(0x3f800000u | (w >> 9)) - 0.99999994039536f;   // 1 - 2^-24
}

// packed fp32x2 arithmetic (FFMA2 / FADD2 / FMUL2 on sm_100: two fp32 operations per issue slot)
__device__ __forceinline__ float2 fpd_fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 fpd_mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 fpd_add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 fpd_dup(float a) { return make_float2(a, a); }

// The cell boundaries a warp is about to use: lane i holds cell_start[min(c0 + i, ncell)], cells c0 .. c0 + ncells - 1 are the
// warp's.  They must be monotone, lie in [0, np], and cell_start[ncell] must be np.  A violation sets the context's
// state word (FP_ERR_STATE at the next entry point); the caller then treats the cells as empty.
__device__ __forceinline__ bool fpd_cells_ok(int32_t cs, int64_t c0, int ncells, int32_t ncell, int64_t np, int lane,
                                             uint32_t* __restrict__ err)
{
    const int32_t nxt = __shfl_down_sync(0xffffffffu, cs, 1);
    const bool mine = lane <= ncells;
    const bool bad = mine && (cs < 0 || (int64_t)cs > np || (lane < ncells && nxt < cs) ||
                              (c0 + lane >= ncell && (int64_t)cs != np));
    const bool ok = !__any_sync(0xffffffffu, bad);
    if (!ok && lane == 0 && err) atomicOr(err, FP_DEVERR_CELL_START);
    return ok;
}

// Stand-alone version of the same check for the paths that walk cell_start by binary search (moments_seg, update_seg)
static __global__ void fp_cs_check_kernel(const int32_t* __restrict__ cell_start, int32_t ncell, int64_t np, uint32_t* __restrict__ err,
                                          uint32_t* __restrict__ err_dev)
{
    fpd_pdl();
    bool bad = false;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i <= ncell; i += (int64_t)gridDim.x * blockDim.x) {
        const int32_t v = cell_start[i];
        bad |= v < 0 || (int64_t)v > np || (i < ncell && cell_start[i + 1] < v) || (i == ncell && (int64_t)v != np);
    }
    if (bad) { atomicOr(err, FP_DEVERR_CELL_START); atomicOr(err_dev, FP_DEVERR_CELL_START); }
}

// 64-bit shuffle helpers
__device__ __forceinline__ double fpd_shfl_xor(double v, int mask)
{
    int lo = __double2loint(v), hi = __double2hiint(v);
    lo = __shfl_xor_sync(0xffffffffu, lo, mask);
    hi = __shfl_xor_sync(0xffffffffu, hi, mask);
    return __hiloint2double(hi, lo);
}
__device__ __forceinline__ double fpd_shfl(double v, int src)
{
    int lo = __double2loint(v), hi = __double2hiint(v);
    lo = __shfl_sync(0xffffffffu, lo, src);
    hi = __shfl_sync(0xffffffffu, hi, src);
    return __hiloint2double(hi, lo);
}

// Transposing ("multi-value") butterfly over a group of G lanes (G a power of two, groups aligned).
// In:  v[0..NP) per lane (NP a power of two, NP >= G).  Out: v[0..NP/G) of lane L (L = lane index inside the
// group) holds the group sum of original slots (NP/G)*L + i.  (NP - NP/G) 64-bit shuffles instead of NP*log2(G).
__device__ __forceinline__ float fpd_shfl_xor(float v, int mask) { return __shfl_xor_sync(0xffffffffu, v, mask); }

template <int NP, int G, typename T>
__device__ __forceinline__ void fpd_transpose_reduce(T (&v)[NP], int lane_in_group)
{
    static_assert((NP & (NP - 1)) == 0 && (G & (G - 1)) == 0 && NP >= G, "powers of two");
#pragma unroll
    for (int half = G / 2, n = NP; half >= 1; half >>= 1, n >>= 1) {
        const bool up = (lane_in_group & half) != 0;
        const int h = n >> 1;
#pragma unroll
        for (int i = 0; i < h; ++i) {
            const T send = up ? v[i] : v[i + h];
            const T keep = up ? v[i + h] : v[i];
            v[i] = keep + fpd_shfl_xor(send, half);
        }
    }
}

#endif  // __CUDACC__
