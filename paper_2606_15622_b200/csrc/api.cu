// api.cu -- context life cycle and the composition of one step (Algorithm 1 :205-225 and Algorithm 2
// :250-270): stream -> walls -> sort -> moments -> closure -> update, all on one stream with no host
// synchronisation and no allocation inside (scratch lives in fp_ctx).
#include <math.h>
#include <stdlib.h>
#include <new>

#include "tiles.cuh"

static const char* k_version = "fpcl 0.1 (sm_100a)";

extern "C" const char* fp_version(void) { return k_version; }

extern "C" const char* fp_last_error(const fp_ctx* ctx) { return ctx ? ctx->err : "null context"; }

static void fp_free_all(fp_ctx* c)
{
    cudaFree(c->key_a); cudaFree(c->key_b); cudaFree(c->idx_a); cudaFree(c->idx_b);
    cudaFree(c->block_hist); cudaFree(c->bin_total); cudaFree(c->cellc);
    if (c->h_err) cudaFreeHost(c->h_err);
    cudaFree(c->d_errdev); cudaFree(c->d_tiebreak); cudaFree(c->d_deferred);
    for (int s = 0; s < 2; ++s) { for (int k = 0; k < 5; ++k) cudaFree(c->hs_f[s][k]); cudaFree(c->hs_pid[s]); }
    cudaFree(c->hs_mom); cudaFree(c->hs_coef); cudaFree(c->hs_flags); cudaFree(c->hs_cell_start);
    if (c->hs_side) cudaStreamDestroy(c->hs_side);
    for (int k = 0; k < 4; ++k) if (c->hs_ev[k]) cudaEventDestroy(c->hs_ev[k]);
    cudaFree(c->mlp.blob); cudaFree(c->mlp.tc_frags); cudaFree(c->mlp.wd_frags); cudaFree(c->mlp.w5_blob); cudaFree(c->mom_acc); cudaFree(c->upd_acc);
}

static void fp_timing_free(fp_ctx* c);

extern "C" int fp_create(fp_ctx** out, const fp_params* h_params)
{
    if (!out || !h_params) return FP_ERR_ARG;
    *out = nullptr;
    const fp_params& q = *h_params;
    if (q.nx < 1 || q.ny < 1 || !(q.dx > 0.f) || !(q.dy > 0.f) || q.max_particles < 0 ||
        (int64_t)q.nx * q.ny >= ((int64_t)1 << 27) || q.max_particles >= ((int64_t)1 << 31) ||
        !(q.tau > 0.f) || (q.conserve_mode != 0 && q.conserve_mode != 1))
        return FP_ERR_ARG;
    for (int k = 0; k < 4; ++k) {
        if (q.wall[k].kind < 0 || q.wall[k].kind > 3) return FP_ERR_ARG;
        // a freestream face re-inserts at xmin from wall[0]'s freestream, which must flow into the domain
        if (q.wall[k].kind == FP_WALL_INFLOW && (q.wall[0].kind != FP_WALL_INFLOW || !(q.wall[0].ux > 0.f) || !(q.wall[0].theta_w > 0.f)))
            return FP_ERR_ARG;
    }
    fp_ctx* c = new (std::nothrow) fp_ctx();
    if (!c) return FP_ERR_STATE;
    c->err[0] = 0;
    c->p = q;
    { const char* e = getenv("FPCL_MLP_FP32"); c->mlp_force_fp32 = e && e[0] == '1'; }
    { const char* e = getenv("FPCL_SORT_UNPACKED"); c->sort_no_pack = e && e[0] == '1'; }
    c->env_mom_seg = getenv("FPCL_MOM_SEG") != nullptr; c->env_mom_no_seg = getenv("FPCL_MOM_NO_SEG") != nullptr;
    c->env_upd_seg = getenv("FPCL_UPD_SEG") != nullptr; c->env_upd_no_seg = getenv("FPCL_UPD_NO_SEG") != nullptr;
    c->ncell = q.nx * q.ny;
    c->slab_row0 = 0; c->slab_rows = q.ny;
    int bits = 0;
    while (((int64_t)1 << bits) < (int64_t)c->ncell) ++bits;
    c->key_bits = bits;
    // fp32, each operation rounded separately (R1, R7)
    volatile float inv_dx = 1.0f / q.dx, inv_dy = 1.0f / q.dy;
    volatile float wx = (float)q.nx * q.dx, wy = (float)q.ny * q.dy;
    volatile float xmax = q.x0 + wx, ymax = q.y0 + wy;
    c->inv_dx = inv_dx; c->inv_dy = inv_dy;
    c->xmin = q.x0; c->ymin = q.y0; c->xmax = xmax; c->ymax = ymax;
    c->xmax_in = nextafterf(xmax, -INFINITY); c->ymax_in = nextafterf(ymax, -INFINITY);
    volatile float Lx = xmax - q.x0, Ly = ymax - q.y0;
    c->Lx = Lx; c->Ly = Ly;
    if (cudaGetDevice(&c->device) != cudaSuccess) { delete c; return FP_ERR_CUDA; }
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device) == cudaSuccess && sms > 0) c->num_sms = sms;
    const size_t n = (size_t)(q.max_particles > 0 ? q.max_particles : 1);
    const size_t nblocks = (n + SORT_TILE - 1) / SORT_TILE;
    c->block_hist_elems = 512 * nblocks;               // per table; two tables (even / odd radix pass)
    bool ok = cudaMalloc((void**)&c->key_a, n * 4) == cudaSuccess && cudaMalloc((void**)&c->key_b, n * 4) == cudaSuccess &&
              cudaMalloc((void**)&c->idx_a, n * 4) == cudaSuccess && cudaMalloc((void**)&c->idx_b, n * 4) == cudaSuccess &&
              cudaMalloc((void**)&c->block_hist, 2 * c->block_hist_elems * 4) == cudaSuccess &&
              cudaMemset(c->block_hist, 0, 2 * c->block_hist_elems * 4) == cudaSuccess &&
              cudaMalloc((void**)&c->bin_total, 512 * 4) == cudaSuccess &&
              cudaMalloc((void**)&c->cellc, (size_t)c->ncell * 28 * 4) == cudaSuccess &&
              cudaMalloc((void**)&c->mom_acc, (size_t)c->ncell * 28 * sizeof(double)) == cudaSuccess &&
              cudaMalloc((void**)&c->upd_acc, (size_t)c->ncell * UPD_ACC * sizeof(double)) == cudaSuccess &&
              cudaHostAlloc((void**)&c->h_err, sizeof(uint32_t), cudaHostAllocMapped) == cudaSuccess &&
              cudaHostGetDevicePointer((void**)&c->d_err, c->h_err, 0) == cudaSuccess &&
              cudaMalloc((void**)&c->d_errdev, 4) == cudaSuccess && cudaMemset(c->d_errdev, 0, 4) == cudaSuccess &&
              cudaMalloc((void**)&c->d_tiebreak, (1 + SW_TB_CAP) * sizeof(uint32_t)) == cudaSuccess &&
              cudaMemset(c->d_tiebreak, 0, (1 + SW_TB_CAP) * sizeof(uint32_t)) == cudaSuccess;
    if (ok && c->p.wall[0].kind == FP_WALL_INFLOW)       // any freestream face implies wall[0] is one (checked above)
        ok = cudaMalloc((void**)&c->d_deferred, ((size_t)c->p.max_particles + 1) * sizeof(uint32_t)) == cudaSuccess &&
             cudaMemset(c->d_deferred, 0, sizeof(uint32_t)) == cudaSuccess;
    if (ok) *c->h_err = 0;
    if (!ok) { fp_free_all(c); delete c; cudaGetLastError(); return FP_ERR_CUDA; }
    *out = c;
    return FP_OK;
}

extern "C" int fp_destroy(fp_ctx* ctx)
{
    if (!ctx) return FP_ERR_ARG;
    cudaDeviceSynchronize();
    fp_timing_free(ctx);
    fp_free_all(ctx);
    delete ctx;
    return FP_OK;
}

// per-cell tau = tau_ref_n / N (tau = 2 mu / p ~ 1/n for Maxwell molecules); N = 0 -> params.tau
__global__ void tau_kernel(const int32_t* __restrict__ cell_start, int32_t ncell, float tau_ref_n, float tau_default,
                           float* __restrict__ tau_cell)
{
    fpd_pdl();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < ncell) {
        const int32_t n = cell_start[i + 1] - cell_start[i];
        tau_cell[i] = n > 0 ? tau_ref_n / (float)n : tau_default;
    }
}

int fpi_tau_from_counts(fp_ctx* ctx, const int32_t* cell_start, float tau_ref_n, float* tau_cell, cudaStream_t st)
{
    fp_launch(tau_kernel, fp_div_up(ctx->ncell, 256), 256, 0, st, cell_start, ctx->ncell, tau_ref_n, ctx->p.tau, tau_cell);
    FP_LAUNCH_OK(ctx);
    FP_COUNT(ctx, 1);
    return FP_OK;
}

// moments -> closure -> update on cell-sorted particles (the part of Algorithm 1/2 after the sort); shared by fp_step
// and fp_collide
static int fpi_after_sort(fp_ctx* ctx, int64_t np, float* vx_b, float* vy_b, float* vz_b, const uint32_t* pid_b, int32_t closure,
                          const fp_mlp* h_mlp, float relax_w, int32_t tau_mode, float tau_ref_n, float* tau_cell, uint64_t step,
                          double* mom, float* coef, uint32_t* flags, int32_t* cell_start, cudaStream_t st)
{
    int rc;
    const float* tau_use = nullptr;
    if (tau_mode == 1) {
        if ((rc = fpi_tau_from_counts(ctx, cell_start, tau_ref_n, tau_cell, st)) != FP_OK) return rc;
        tau_use = tau_cell;
    }
    // a3
    const int32_t mode = closure == 0 ? 1 : 0;
    const int32_t stride = mode ? 29 : 13;
    if ((rc = fp_cell_moments(ctx, np, vx_b, vy_b, vz_b, cell_start, mode, mom, (void*)st)) != FP_OK) return rc;
    fp_mark(ctx, 4, st);
    // a4 | a5; the closure kernel also writes the per-cell constants of a6 (no separate prep launch)
    if (closure == 0) rc = fpi_closure_exact(ctx, mom, tau_use, coef, flags, nullptr, true, st);
    else              rc = fpi_closure_mlp(ctx, mom, stride, tau_use, h_mlp, relax_w, coef, flags, true, st);
    if (rc != FP_OK) return rc;
    fp_mark(ctx, 5, st);
    // a6
    rc = fpi_velocity_update(ctx, np, vx_b, vy_b, vz_b, pid_b, cell_start, mom, stride, coef, tau_use, step, flags, true, st);
    fp_mark(ctx, 6, st);
    return rc;
}

extern "C" int fp_step(fp_ctx* ctx, int64_t np,
                       float* x_a, float* y_a, float* vx_a, float* vy_a, float* vz_a, uint32_t* pid_a,
                       float* x_b, float* y_b, float* vx_b, float* vy_b, float* vz_b, uint32_t* pid_b,
                       int32_t closure, const fp_mlp* h_mlp, float relax_w,
                       int32_t tau_mode, float tau_ref_n, float* tau_cell,
                       uint64_t step, double* mom, float* coef, uint32_t* flags, int32_t* cell_start, void* stream)
{
    if (!ctx) return FP_ERR_ARG;
    if (np < 0 || !mom || !coef || !flags || !cell_start || (closure != 0 && closure != 1) || (tau_mode != 0 && tau_mode != 1))
        return fp_fail(ctx, FP_ERR_ARG, "fp_step: bad argument");
    if (closure == 1 && !h_mlp) return fp_fail(ctx, FP_ERR_ARG, "fp_step: surrogate closure needs h_mlp");
    if (tau_mode == 1 && !tau_cell) return fp_fail(ctx, FP_ERR_ARG, "fp_step: tau_mode 1 needs tau_cell");
    if (np > ctx->p.max_particles) return fp_fail(ctx, FP_ERR_STATE, "fp_step: np > max_particles");
    if (fp_state_check(ctx, "fp_step") != FP_OK) return FP_ERR_STATE;
    if (np > 0 && (!x_a || !y_a || !vx_a || !vy_a || !vz_a || !pid_a || !x_b || !y_b || !vx_b || !vy_b || !vz_b || !pid_b))
        return fp_fail(ctx, FP_ERR_ARG, "fp_step: null particle pointer");
    cudaStream_t st = (cudaStream_t)stream;
    int rc;
    ctx->t_in_step = ctx->t_ev != nullptr && ctx->t_step < ctx->t_max;
    struct step_guard { fp_ctx* c; ~step_guard() { if (c->t_in_step) { c->t_in_step = false; c->t_step += 1; } } } guard{ctx};
    fp_mark(ctx, 0, st);
    // a0 + a1 (+ cell keys of the streamed positions)
    if ((rc = fpi_stream_walls(ctx, np, x_a, y_a, vx_a, vy_a, vz_a, pid_a, step, ctx->key_b, true, st)) != FP_OK) return rc;
    fp_mark(ctx, 1, st);
    // a2 (records mark 2 between the key sort and the payload gather)
    if ((rc = fpi_sort_with_keys(ctx, np, ctx->key_b, true, x_a, y_a, vx_a, vy_a, vz_a, pid_a, x_b, y_b, vx_b, vy_b, vz_b, pid_b,
                                 cell_start, nullptr, st)) != FP_OK) return rc;
    fp_mark(ctx, 3, st);
    return fpi_after_sort(ctx, np, vx_b, vy_b, vz_b, pid_b, closure, h_mlp, relax_w, tau_mode, tau_ref_n, tau_cell, step, mom, coef,
                          flags, cell_start, st);
}

// Algorithm 1/2 after the move: sort by cell -> moments -> closure -> update, on particles whose positions are final (a slab
// after its exchange, or any caller that streams by itself).  Same arguments as fp_step.
extern "C" int fp_collide(fp_ctx* ctx, int64_t np,
                          const float* x_a, const float* y_a, const float* vx_a, const float* vy_a, const float* vz_a, const uint32_t* pid_a,
                          float* x_b, float* y_b, float* vx_b, float* vy_b, float* vz_b, uint32_t* pid_b,
                          int32_t closure, const fp_mlp* h_mlp, float relax_w,
                          int32_t tau_mode, float tau_ref_n, float* tau_cell,
                          uint64_t step, double* mom, float* coef, uint32_t* flags, int32_t* cell_start, void* stream)
{
    if (!ctx) return FP_ERR_ARG;
    if (np < 0 || !mom || !coef || !flags || !cell_start || (closure != 0 && closure != 1) || (tau_mode != 0 && tau_mode != 1))
        return fp_fail(ctx, FP_ERR_ARG, "fp_collide: bad argument");
    if (closure == 1 && !h_mlp) return fp_fail(ctx, FP_ERR_ARG, "fp_collide: surrogate closure needs h_mlp");
    if (tau_mode == 1 && !tau_cell) return fp_fail(ctx, FP_ERR_ARG, "fp_collide: tau_mode 1 needs tau_cell");
    if (fp_state_check(ctx, "fp_collide") != FP_OK) return FP_ERR_STATE;
    int rc = fp_sort_by_cell(ctx, np, x_a, y_a, vx_a, vy_a, vz_a, pid_a, x_b, y_b, vx_b, vy_b, vz_b, pid_b, cell_start, nullptr, stream);
    if (rc != FP_OK) return rc;
    return fpi_after_sort(ctx, np, vx_b, vy_b, vz_b, pid_b, closure, h_mlp, relax_w, tau_mode, tau_ref_n, tau_cell, step, mom, coef,
                          flags, cell_start, (cudaStream_t)stream);
}

extern "C" uint64_t fp_launch_count(const fp_ctx* ctx) { return ctx ? ctx->launches : 0; }

static void fp_timing_free(fp_ctx* c)
{
    if (c->t_ev) {
        for (size_t i = 0; i < (size_t)c->t_max * (FP_NSTAGES + 1); ++i) if (c->t_ev[i]) cudaEventDestroy(c->t_ev[i]);
        delete[] c->t_ev;
    }
    c->t_ev = nullptr; c->t_max = 0; c->t_step = 0; c->t_in_step = false;
}

extern "C" int fp_timing_enable(fp_ctx* ctx, int32_t max_steps)
{
    if (!ctx || max_steps < 0 || max_steps > 65536) return FP_ERR_ARG;
    fp_timing_free(ctx);
    if (max_steps == 0) return FP_OK;
    const size_t n = (size_t)max_steps * (FP_NSTAGES + 1);
    ctx->t_ev = new (std::nothrow) cudaEvent_t[n]();
    if (!ctx->t_ev) return fp_fail(ctx, FP_ERR_STATE, "fp_timing_enable: out of memory");
    ctx->t_max = max_steps;
    for (size_t i = 0; i < n; ++i) FP_CUDA_OK(ctx, cudaEventCreate(&ctx->t_ev[i]));
    return FP_OK;
}

extern "C" int fp_timing_read(fp_ctx* ctx, float* h_ms, int32_t* h_nsteps)
{
    if (!ctx || !h_ms || !h_nsteps) return FP_ERR_ARG;
    *h_nsteps = 0;
    if (!ctx->t_ev) return fp_fail(ctx, FP_ERR_STATE, "fp_timing_read: timing is not enabled");
    const int n = ctx->t_step;
    if (n > 0) FP_CUDA_OK(ctx, cudaEventSynchronize(ctx->t_ev[(size_t)(n - 1) * (FP_NSTAGES + 1) + FP_NSTAGES]));
    for (int s = 0; s < n; ++s)
        for (int k = 0; k < FP_NSTAGES; ++k) {
            const cudaEvent_t* e = ctx->t_ev + (size_t)s * (FP_NSTAGES + 1);
            FP_CUDA_OK(ctx, cudaEventElapsedTime(&h_ms[s * FP_NSTAGES + k], e[k], e[k + 1]));
        }
    *h_nsteps = n;
    ctx->t_step = 0;
    return FP_OK;
}

static int fp_host_stage_alloc(fp_ctx* c)
{
    if (c->hs_ready) return FP_OK;
    const size_t n = (size_t)(c->p.max_particles > 0 ? c->p.max_particles : 1);
    for (int s = 0; s < 2; ++s) {
        for (int k = 0; k < 5; ++k) FP_CUDA_OK(c, cudaMalloc((void**)&c->hs_f[s][k], n * 4));
        FP_CUDA_OK(c, cudaMalloc((void**)&c->hs_pid[s], n * 4));
    }
    FP_CUDA_OK(c, cudaMalloc((void**)&c->hs_mom, (size_t)c->ncell * 29 * 8));
    FP_CUDA_OK(c, cudaMalloc((void**)&c->hs_coef, (size_t)c->ncell * 9 * 4));
    FP_CUDA_OK(c, cudaMalloc((void**)&c->hs_flags, (size_t)c->ncell * 4));
    FP_CUDA_OK(c, cudaMalloc((void**)&c->hs_cell_start, ((size_t)c->ncell + 1) * 4));
    FP_CUDA_OK(c, cudaStreamCreateWithFlags(&c->hs_side, cudaStreamNonBlocking));
    for (int k = 0; k < 4; ++k) FP_CUDA_OK(c, cudaEventCreateWithFlags(&c->hs_ev[k], cudaEventDisableTiming));
    c->hs_ready = true;
    return FP_OK;
}

int fpi_mlp_reserve(fp_ctx* ctx, const fp_mlp* h_mlp);

extern "C" int fp_reserve(fp_ctx* ctx, const fp_mlp* h_mlp, int32_t host_staging)
{
    if (!ctx) return FP_ERR_ARG;
    int rc = FP_OK;
    if (h_mlp && (rc = fpi_mlp_reserve(ctx, h_mlp)) != FP_OK) return rc;
    if (host_staging && (rc = fp_host_stage_alloc(ctx)) != FP_OK) return rc;
    return FP_OK;
}

extern "C" int fp_check(fp_ctx* ctx, void* stream)
{
    if (!ctx) return FP_ERR_ARG;
    FP_CUDA_OK(ctx, cudaStreamSynchronize((cudaStream_t)stream));
    const uint32_t e = *(volatile uint32_t*)ctx->h_err;
    *(volatile uint32_t*)ctx->h_err = 0;
    FP_CUDA_OK(ctx, cudaMemset(ctx->d_errdev, 0, 4));
    if (e & FP_DEVERR_CELL_START)
        return fp_fail(ctx, FP_ERR_STATE, "fp_check: cell_start was not a monotone prefix sum ending at np in an earlier call; "
                                          "the cells concerned were skipped");
    return FP_OK;
}

extern "C" int fp_step_host(fp_ctx* ctx, int64_t np,
                            float* h_x, float* h_y, float* h_vx, float* h_vy, float* h_vz, uint32_t* h_pid,
                            int32_t closure, const fp_mlp* h_mlp, float relax_w, uint64_t step,
                            float* h_coef, uint32_t* h_flags, int32_t* h_cell_start, void* stream)
{
    if (!ctx) return FP_ERR_ARG;
    if (np < 0 || np > ctx->p.max_particles) return fp_fail(ctx, FP_ERR_STATE, "fp_step_host: np out of range");
    if (np > 0 && (!h_x || !h_y || !h_vx || !h_vy || !h_vz || !h_pid)) return fp_fail(ctx, FP_ERR_ARG, "fp_step_host: null host pointer");
    int rc = fp_host_stage_alloc(ctx);                // no-op after fp_reserve(ctx, ..., 1) or the first call
    if (rc != FP_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    float* hp[5] = {h_x, h_y, h_vx, h_vy, h_vz};
    const size_t nb = (size_t)np * 4;
    cudaStream_t side = ctx->hs_side;
    // host -> device, all on the caller's stream: the stream kernel reads x, y, vx, vy, pid and REWRITES vx, vy, vz of
    // every particle it re-emits at a wall or the body, so no input may still be in flight when it starts
    for (int k = 0; k < 5; ++k) if (nb) FP_CUDA_OK(ctx, cudaMemcpyAsync(ctx->hs_f[0][k], hp[k], nb, cudaMemcpyHostToDevice, st));
    if (nb) FP_CUDA_OK(ctx, cudaMemcpyAsync(ctx->hs_pid[0], h_pid, nb, cudaMemcpyHostToDevice, st));
    ctx->ev_before_gather = nullptr;
    ctx->ev_after_gather = ctx->hs_ev[2];
    rc = fp_step(ctx, np, ctx->hs_f[0][0], ctx->hs_f[0][1], ctx->hs_f[0][2], ctx->hs_f[0][3], ctx->hs_f[0][4], ctx->hs_pid[0],
                 ctx->hs_f[1][0], ctx->hs_f[1][1], ctx->hs_f[1][2], ctx->hs_f[1][3], ctx->hs_f[1][4], ctx->hs_pid[1],
                 closure, h_mlp, relax_w, 0, 0.f, nullptr, step, ctx->hs_mom, ctx->hs_coef, ctx->hs_flags,
                 ctx->hs_cell_start, stream);
    ctx->ev_before_gather = nullptr;
    ctx->ev_after_gather = nullptr;
    if (rc != FP_OK) { cudaStreamSynchronize(side); return rc; }
    // device -> host: positions and ids are final after the gather and go back on the side stream while moments,
    // closure and update run; the velocities and the per-cell outputs follow on the caller's stream
    if (np > 0) {
        FP_CUDA_OK(ctx, cudaStreamWaitEvent(side, ctx->hs_ev[2], 0));
        FP_CUDA_OK(ctx, cudaMemcpyAsync(hp[0], ctx->hs_f[1][0], nb, cudaMemcpyDeviceToHost, side));
        FP_CUDA_OK(ctx, cudaMemcpyAsync(hp[1], ctx->hs_f[1][1], nb, cudaMemcpyDeviceToHost, side));
        FP_CUDA_OK(ctx, cudaMemcpyAsync(h_pid, ctx->hs_pid[1], nb, cudaMemcpyDeviceToHost, side));
    }
    for (int k = 2; k < 5; ++k) if (nb) FP_CUDA_OK(ctx, cudaMemcpyAsync(hp[k], ctx->hs_f[1][k], nb, cudaMemcpyDeviceToHost, st));
    if (h_coef) FP_CUDA_OK(ctx, cudaMemcpyAsync(h_coef, ctx->hs_coef, (size_t)ctx->ncell * 9 * 4, cudaMemcpyDeviceToHost, st));
    if (h_flags) FP_CUDA_OK(ctx, cudaMemcpyAsync(h_flags, ctx->hs_flags, (size_t)ctx->ncell * 4, cudaMemcpyDeviceToHost, st));
    if (h_cell_start) FP_CUDA_OK(ctx, cudaMemcpyAsync(h_cell_start, ctx->hs_cell_start, ((size_t)ctx->ncell + 1) * 4, cudaMemcpyDeviceToHost, st));
    FP_CUDA_OK(ctx, cudaStreamSynchronize(side));
    FP_CUDA_OK(ctx, cudaStreamSynchronize(st));
    return FP_OK;
}
