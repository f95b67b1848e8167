// stream_walls.cu -- a0 + a1: streaming (Eq. 16 :187) and diffuse isothermal walls (:214, :380, :674;
// DESIGN.md R7), fused with the cell-key computation of a2 (R1) when called from fp_step.
//
// One thread per particle, SoA fp32, fully coalesced: 16 B read (x, y, vx, vy; pid is read only by particles that
// hit a wall, vz never), 8 B written (x, y) + 4 B key; wall hits add 12 B of velocity writes.
// Positions follow a fixed fp32 operation sequence (they decide the integer cell index); re-emitted velocities
// are drawn with fp32 logf / sincospif from the Philox uniforms (tolerance 1e-6 relative).
#include "common.cuh"

struct sw_params {
    int32_t nx, ny;
    float x0, y0, inv_dx, inv_dy, dt;
    float xmin, xmax, ymin, ymax, xmax_in, ymax_in, Lx, Ly;
    fp_wall wall[4];
    int32_t body_kind;
    float bcx, bcy, bR, bR_out, bR2, body_theta_w;
    uint32_t k0, k1, step_lo, step_hi;
    fp_grid grid;                    // cell keys (slab-aware)
    float in_mu, in_sg, in_pen;     // freestream reservoir: mode of the flux density, sqrt(theta_inf), fl(U_inf,x * dt)
    uint32_t* tiebreak;              // [0] count, [1..] indices of re-inserted particles with a borderline fp32 accept/reject test
    uint32_t* deferred;              // [0] count, [1..] indices of the particles that left through a freestream face (reservoir grids)
};

// One wall draw (R7): normal component sqrt(-2 theta_w ln u0) into the gas, tangentials
// sqrt(theta_w) * sqrt(-2 ln u1) * (cos, sin)(2 pi u2).
__device__ __forceinline__ void sw_wall_draw(const sw_params& P, uint32_t pid, uint32_t stream, float theta_w,
                                             float& vn, float& t1, float& t2)
{
    const uint4 w = fpd_philox4x32_10(pid, P.step_lo, P.step_hi, stream, P.k0, P.k1);
    const float u0 = fpd_uniform(w.x), u1 = fpd_uniform(w.y), u2 = fpd_uniform(w.z);
    vn = sqrtf(-2.0f * theta_w * logf(u0));
    const float r = sqrtf(theta_w) * sqrtf(-2.0f * logf(u1));
    float s, c;
    sincospif(2.0f * u2, &s, &c);
    t1 = r * c;
    t2 = r * s;
}

// Freestream reservoir (FP_WALL_INFLOW, R11): re-insertion at xmin.  v_x from f(v) ~ v exp(-(v-U)^2/(2 theta)),
// v > 0, by acceptance-rejection about the mode mu (candidate mu + sigma z, accepted iff v > 0 and (v/mu) e^(1 - v/mu) >= u2;
// attempt a uses the Philox stream 16 + a, a < 8; then v = mu); tangentials and the entry position from stream 32.  The
// position follows a fixed fp32 sequence (it decides the cell index).  The accept / reject test DECIDES which attempt's
// candidate the particle gets.  It is evaluated in fp32 here; a particle with a test within 1e-4 of the line (a hundred
// times the fp32 error) is put on a list and sw_tiebreak_kernel repeats its whole draw in fp64, the oracle's precision.
// (An unguarded fp32 test flipped once in ~1e6 draws, found by randomised comparison on 1.2M particles; fp64 arithmetic
// anywhere in this kernel's call tree costs it its 64 registers: 177 -> 300 us at 20M particles.)
__device__ __noinline__ void sw_reinsert(const sw_params& P, uint32_t pid, uint32_t p, bool two_d, float& xp, float& yp, float& v0,
                                         float& v1, float& v2)
{
    float vn = P.in_mu;
    bool borderline = false;
    for (uint32_t a = 0; a < 8u; ++a) {
        const uint4 w = fpd_philox4x32_10(pid, P.step_lo, P.step_hi, 16u + a, P.k0, P.k1);
        float s, c;
        sincospif(2.0f * fpd_uniform(w.y), &s, &c);
        const float cand = fmaf(P.in_sg * sqrtf(-2.0f * logf(fpd_uniform(w.x))), c, P.in_mu);
        const float q = cand / P.in_mu;
        const float lhs = q * expf(1.0f - q), rhs = fpd_uniform(w.z);
        borderline = borderline || fabsf(lhs - rhs) < 1.0e-4f || fabsf(cand) < 1.0e-4f * P.in_sg;
        if (cand > 0.0f && lhs >= rhs) { vn = cand; break; }
    }
    if (borderline) {
        const uint32_t slot = atomicAdd(P.tiebreak, 1u);
        if (slot < SW_TB_CAP) P.tiebreak[1 + slot] = p;
    }
    const uint4 w = fpd_philox4x32_10(pid, P.step_lo, P.step_hi, 32u, P.k0, P.k1);
    const float r = P.in_sg * sqrtf(-2.0f * logf(fpd_uniform(w.x)));
    float s, c;
    sincospif(2.0f * fpd_uniform(w.y), &s, &c);
    v0 = vn; v1 = fmaf(r, c, P.wall[0].uy); v2 = fmaf(r, s, P.wall[0].uz);
    float xn = __fadd_rn(P.xmin, __fmul_rn(fpd_uniform(w.w), P.in_pen));
    if (xn < P.xmin) xn = P.xmin;
    if (xn >= P.xmax) xn = P.xmax_in;
    xp = xn;
    if (two_d) {
        float yn = fmaf(fpd_uniform(w.z), P.Ly, P.ymin);
        if (yn < P.ymin) yn = P.ymin;
        if (yn >= P.ymax) yn = P.ymax_in;
        yp = yn;
    }
}

// One particle: stream, walls, body, key.  pid is read only by particles that hit something.
struct sw_moved { float x, y, v0, v1, v2; uint32_t key; bool redrawn, deferred; };

// INFLOW: 0 = the grid has no freestream face; 1 = a particle that leaves through one is re-inserted here (sw_reinsert);
// 2 = it is only reported (deferred = true, nothing else of the result is valid): the streaming kernel lists it and
// sw_deferred_kernel runs this function again on the untouched inputs with INFLOW = 1.
template <bool WRITE_KEYS, int INFLOW>
__device__ __forceinline__ sw_moved sw_move(const sw_params& P, float xin, float yin, float v0, float v1,
                                            const uint32_t* __restrict__ pid, int64_t p)
{
        float v2 = 0.0f;                           // vz is only ever replaced, never read
        float xp = fmaf(v0, P.dt, xin);
        float yp = fmaf(v1, P.dt, yin);
        bool redrawn = false, reinserted = false;
        // x pair
        {
            const int side = (xp < P.xmin) ? 0 : ((xp >= P.xmax) ? 1 : -1);
            if (side >= 0) {
                const fp_wall w = P.wall[side];
                const float xw = side ? P.xmax : P.xmin;
                if (w.kind == FP_WALL_DIFFUSE) {
                    xp = __fadd_rn(xw, __fsub_rn(xw, xp));
                    if (xp < P.xmin) xp = P.xmin;
                    if (xp >= P.xmax) xp = P.xmax_in;
                    float vn, t1, t2;
                    sw_wall_draw(P, pid[p], 1u, w.theta_w, vn, t1, t2);
                    v0 = side ? -vn : vn; v1 = w.uy + t1; v2 = w.uz + t2; redrawn = true;
                } else if (w.kind == FP_WALL_PERIODIC) {
                    xp = side ? __fsub_rn(xp, P.Lx) : __fadd_rn(xp, P.Lx);
                    if (xp < P.xmin) xp = P.xmin;
                    if (xp >= P.xmax) xp = P.xmax_in;
                } else if (INFLOW == 2 && w.kind == FP_WALL_INFLOW) {
                    sw_moved d; d.x = xin; d.y = yin; d.v0 = v0; d.v1 = v1; d.v2 = 0.0f; d.key = 0u; d.redrawn = false; d.deferred = true;
                    return d;
                } else if (INFLOW == 1 && w.kind == FP_WALL_INFLOW) {
                    sw_reinsert(P, pid[p], (uint32_t)p, P.ny > 1, xp, yp, v0, v1, v2);
                    redrawn = true; reinserted = true;
                }
            }
        }
        // y pair
        if (P.ny > 1 && !reinserted) {
            const int side = (yp < P.ymin) ? 0 : ((yp >= P.ymax) ? 1 : -1);
            if (side >= 0) {
                const fp_wall w = P.wall[2 + side];
                const float yw = side ? P.ymax : P.ymin;
                if (w.kind == FP_WALL_DIFFUSE) {
                    yp = __fadd_rn(yw, __fsub_rn(yw, yp));
                    if (yp < P.ymin) yp = P.ymin;
                    if (yp >= P.ymax) yp = P.ymax_in;
                    float vn, t1, t2;
                    sw_wall_draw(P, pid[p], 2u, w.theta_w, vn, t1, t2);
                    v1 = side ? -vn : vn; v0 = w.ux + t1; v2 = w.uz + t2; redrawn = true;
                } else if (w.kind == FP_WALL_PERIODIC) {
                    yp = side ? __fsub_rn(yp, P.Ly) : __fadd_rn(yp, P.Ly);
                    if (yp < P.ymin) yp = P.ymin;
                    if (yp >= P.ymax) yp = P.ymax_in;
                } else if (INFLOW == 2 && w.kind == FP_WALL_INFLOW) {
                    sw_moved d; d.x = xin; d.y = yin; d.v0 = v0; d.v1 = v1; d.v2 = 0.0f; d.key = 0u; d.redrawn = false; d.deferred = true;
                    return d;
                } else if (INFLOW == 1 && w.kind == FP_WALL_INFLOW) {
                    sw_reinsert(P, pid[p], (uint32_t)p, true, xp, yp, v0, v1, v2);
                    redrawn = true;
                }
            }
        }
        // embedded body: a particle inside the cylinder is moved radially to R (1 + 1e-6) and re-emitted
        if (P.body_kind == 1) {
            const float ddx = __fsub_rn(xp, P.bcx), ddy = __fsub_rn(yp, P.bcy);
            const float r2 = fmaf(ddy, ddy, __fmul_rn(ddx, ddx));
            if (r2 < P.bR2) {
                const float r = sqrtf(r2);
                float nxn, nyn;
                if (r > 0.0f) {
                    const float sc = __fdiv_rn(P.bR_out, r);
                    nxn = ddx / r; nyn = ddy / r;
                    xp = fmaf(ddx, sc, P.bcx); yp = fmaf(ddy, sc, P.bcy);
                } else { nxn = 1.0f; nyn = 0.0f; xp = __fadd_rn(P.bcx, P.bR_out); }
                float vn, t1, t2;
                sw_wall_draw(P, pid[p], 4u, P.body_theta_w, vn, t1, t2);
                v0 = vn * nxn - t1 * nyn; v1 = vn * nyn + t1 * nxn; v2 = t2; redrawn = true;
            }
        }
        sw_moved m;
        m.x = xp; m.y = yp; m.v0 = v0; m.v1 = v1; m.v2 = v2; m.redrawn = redrawn; m.deferred = false; m.key = 0u;
        if (WRITE_KEYS) {
            m.key = (uint32_t)fpd_cell_key(xp, yp, P.grid);
        }
        return m;
}

// first radix digit histogram of the sort tile a warp's particles fall in (sort.cu): lanes with the same digit send
// one aggregated reduction to tile_hist[digit][tile]; the table is zero on entry.  Full-warp collective.
__device__ __forceinline__ void sw_hist(uint32_t* __restrict__ tile_hist, int ntiles, int64_t tile, bool valid,
                                        uint32_t key, uint32_t digit_mask, int lane)
{
    const uint32_t d = valid ? (key & digit_mask) : 0xffffffffu;
    const uint32_t peers = __match_any_sync(0xffffffffu, d);
    if (valid && lane == __ffs(peers) - 1)
        atomicAdd(&tile_hist[(size_t)d * ntiles + (size_t)tile], (uint32_t)__popc(peers));
}

// One particle per thread, grid-stride.  (Four particles per thread with 128-bit accesses was measured slower:
// 37 vs 33 us at 4M particles.)  29 registers without a spill: eight resident blocks, 64 warps per SM (33.1 -> 31.1 us in
// the step at 4M particles against six; loading the next trip's four values before working on the current one is
// slower with six blocks, 33.3 us, and with eight, 35.1 us, spills).
// INFLOW: the grid has freestream faces.  A particle that leaves through one is not re-inserted here -- the call into
// sw_reinsert would cost this kernel its registers (64 instead of 29: four resident blocks, 204 instead of ~165 us at
// 20M particles) -- but put on a list; its arrays stay untouched and sw_deferred_kernel handles it.
#ifndef SW_MINB
#define SW_MINB 8
#endif
template <bool WRITE_KEYS, bool INFLOW>
__global__ void __launch_bounds__(256, SW_MINB)
sw_kernel(int64_t np, float* __restrict__ x, float* __restrict__ y, float* __restrict__ vx,
          float* __restrict__ vy, float* __restrict__ vz, const uint32_t* __restrict__ pid,
          uint32_t* __restrict__ keys, uint32_t* __restrict__ tile_hist, int ntiles, uint32_t digit_mask,
          const __grid_constant__ sw_params P)
{
    fpd_pdl();
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int lane = threadIdx.x & 31;
    // warp-uniform trip count: the histogram is a full-warp collective; a warp's 32 particles lie in one sort tile
    for (int64_t p0 = (int64_t)blockIdx.x * blockDim.x + (threadIdx.x & ~31); p0 < np; p0 += stride) {
        const int64_t p = p0 + lane;
        bool valid = p < np;
        uint32_t key = 0u;
        if (valid) {
            const sw_moved m = sw_move<WRITE_KEYS, INFLOW ? 2 : 0>(P, x[p], y[p], vx[p], vy[p], pid, p);
            if (INFLOW && m.deferred) {
                P.deferred[1u + atomicAdd(P.deferred, 1u)] = (uint32_t)p;     // at most once per particle: the list holds np entries
                valid = false;                                                  // its histogram entry comes with its new position
            } else {
                x[p] = m.x; y[p] = m.y; key = m.key;
                if (m.redrawn) { vx[p] = m.v0; vy[p] = m.v1; vz[p] = m.v2; }
                if (WRITE_KEYS) keys[p] = key;
            }
        }
        if (WRITE_KEYS && tile_hist) sw_hist(tile_hist, ntiles, p0 / SORT_TILE, valid, key, digit_mask, lane);
    }
}

// The particles the streaming kernel listed (they left through a freestream face; ~1e-3 of the ensemble per step):
// the whole move again from their untouched arrays, re-insertion included, then key and histogram entry.
template <bool WRITE_KEYS>
__global__ void __launch_bounds__(128)
sw_deferred_kernel(float* __restrict__ x, float* __restrict__ y, float* __restrict__ vx, float* __restrict__ vy,
                   float* __restrict__ vz, const uint32_t* __restrict__ pid, uint32_t* __restrict__ keys,
                   uint32_t* __restrict__ tile_hist, int ntiles, uint32_t digit_mask, const __grid_constant__ sw_params P)
{
    fpd_pdl();
    const uint32_t n = P.deferred[0];
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const int64_t p = (int64_t)P.deferred[1u + i];
        const sw_moved m = sw_move<WRITE_KEYS, 1>(P, x[p], y[p], vx[p], vy[p], pid, p);
        x[p] = m.x; y[p] = m.y;
        if (m.redrawn) { vx[p] = m.v0; vy[p] = m.v1; vz[p] = m.v2; }
        if (WRITE_KEYS) {
            keys[p] = m.key;
            if (tile_hist) atomicAdd(&tile_hist[(size_t)(m.key & digit_mask) * ntiles + (size_t)(p / SORT_TILE)], 1u);
        }
    }
}

// The listed particles' normal velocity again, every attempt's test in fp64 (as the oracle evaluates it); resets the list.
__device__ __forceinline__ double sw_uniform_f64(uint32_t w) { return ((double)(w >> 9) + 0.5) * (1.0 / 8388608.0); }

__global__ void __launch_bounds__(128)
sw_tiebreak_kernel(float* __restrict__ vx, const uint32_t* __restrict__ pid, const __grid_constant__ sw_params P)
{
    fpd_pdl();
    const uint32_t n = min(P.tiebreak[0], (uint32_t)SW_TB_CAP);
    const double th = (double)P.wall[0].theta_w, U = (double)P.wall[0].ux, sg = sqrt(th), mu = 0.5 * (U + sqrt(U * U + 4.0 * th));
    for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) {
        const uint32_t p = P.tiebreak[1 + i];
        double vn = mu;
        for (uint32_t a = 0; a < 8u; ++a) {
            const uint4 w = fpd_philox4x32_10(pid[p], P.step_lo, P.step_hi, 16u + a, P.k0, P.k1);
            double s, c;
            sincospi(2.0 * sw_uniform_f64(w.y), &s, &c);
            const double cand = mu + sg * sqrt(-2.0 * log(sw_uniform_f64(w.x))) * c;
            const double q = cand / mu;
            if (cand > 0.0 && q * exp(1.0 - q) >= sw_uniform_f64(w.z)) { vn = cand; break; }
        }
        vx[p] = (float)vn;
    }
    __syncthreads();
    if (threadIdx.x == 0) { P.tiebreak[0] = 0u; P.deferred[0] = 0u; }      // both lists are consumed: sw_deferred_kernel ran before
}

int fpi_stream_walls(fp_ctx* ctx, int64_t np, float* x, float* y, float* vx, float* vy, float* vz,
                     const uint32_t* pid, uint64_t step, uint32_t* keys_out, bool with_hist0, cudaStream_t st)
{
    if (np == 0) return FP_OK;
    const fp_params& q = ctx->p;
    const bool inflow = q.wall[0].kind == FP_WALL_INFLOW;      // fp_create: any freestream face implies wall[0] is one
    sw_params P;
    P.nx = q.nx; P.ny = q.ny; P.x0 = q.x0; P.y0 = q.y0; P.inv_dx = ctx->inv_dx; P.inv_dy = ctx->inv_dy; P.dt = q.dt;
    P.xmin = ctx->xmin; P.xmax = ctx->xmax; P.ymin = ctx->ymin; P.ymax = ctx->ymax;
    P.xmax_in = ctx->xmax_in; P.ymax_in = ctx->ymax_in; P.Lx = ctx->Lx; P.Ly = ctx->Ly;
    for (int k = 0; k < 4; ++k) P.wall[k] = q.wall[k];
    P.body_kind = q.body_kind; P.bcx = q.body_cx; P.bcy = q.body_cy; P.bR = q.body_R;
    {   // fp32, two separate roundings (the host compiler targets baseline x86-64: no FMA contraction)
        volatile float rout = q.body_R * 1.000001f; P.bR_out = rout;
        volatile float r2 = q.body_R * q.body_R;    P.bR2 = r2;
    }
    P.body_theta_w = q.body_theta_w;
    P.grid = fp_grid_of(ctx);
    {   // freestream reservoir constants (only read when a face is FP_WALL_INFLOW)
        const double U = q.wall[0].ux, th = q.wall[0].theta_w > 0.f ? q.wall[0].theta_w : 1.0;
        P.in_mu = (float)(0.5 * (U + sqrt(U * U + 4.0 * th)));
        P.in_sg = (float)sqrt(th);
        volatile float pen = q.wall[0].ux * q.dt; P.in_pen = pen;
    }
    P.tiebreak = ctx->d_tiebreak;
    P.deferred = ctx->d_deferred;
    P.k0 = (uint32_t)q.seed; P.k1 = (uint32_t)(q.seed >> 32);
    P.step_lo = (uint32_t)step; P.step_hi = (uint32_t)(step >> 32);
    const int threads = 256;
    const int64_t want = (np + threads - 1) / threads;
    // one resident wave of grid-striding CTAs (a partial extra wave costs up to 8 us at 4M particles)
    int& socc = ctx->sw_occ[inflow ? 1 : 0];
    if (socc == 0) {
        if (inflow) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&socc, sw_kernel<true, true>, threads, 0);
        else        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&socc, sw_kernel<true, false>, threads, 0);
        if (socc < 1) socc = 1;
    }
    const int64_t cap = (int64_t)ctx->num_sms * socc;
    const int blocks = (int)(want < cap ? want : cap);
    if (keys_out) {
        uint32_t* th = nullptr;
        if (with_hist0) {
            th = ctx->block_hist;
            if (!ctx->hist0_clean) FP_CUDA_OK(ctx, cudaMemsetAsync(th, 0, ctx->block_hist_elems * sizeof(uint32_t), st));
            ctx->hist0_clean = false;
        }
        const uint32_t dmask = (1u << fpi_sort_digit_bits(ctx)) - 1u;
        if (inflow) fp_launch(sw_kernel<true, true>, blocks, threads, 0, st, np, x, y, vx, vy, vz, pid, keys_out, th, fp_div_up(np, SORT_TILE), dmask, P);
        else        fp_launch(sw_kernel<true, false>, blocks, threads, 0, st, np, x, y, vx, vy, vz, pid, keys_out, th, fp_div_up(np, SORT_TILE), dmask, P);
    } else {
        if (inflow) fp_launch(sw_kernel<false, true>, blocks, threads, 0, st, np, x, y, vx, vy, vz, pid, nullptr, nullptr, 0, 0u, P);
        else        fp_launch(sw_kernel<false, false>, blocks, threads, 0, st, np, x, y, vx, vy, vz, pid, nullptr, nullptr, 0, 0u, P);
    }
    if (inflow) {
        const int dblocks = 2 * ctx->num_sms;
        if (keys_out) fp_launch(sw_deferred_kernel<true>, dblocks, 128, 0, st, x, y, vx, vy, vz, pid, keys_out,
                                with_hist0 ? ctx->block_hist : nullptr, fp_div_up(np, SORT_TILE), (1u << fpi_sort_digit_bits(ctx)) - 1u, P);
        else          fp_launch(sw_deferred_kernel<false>, dblocks, 128, 0, st, x, y, vx, vy, vz, pid, nullptr, nullptr, 0, 0u, P);
        fp_launch(sw_tiebreak_kernel, 1, 128, 0, st, vx, pid, P);
    }
    FP_LAUNCH_OK(ctx);
    FP_COUNT(ctx, inflow ? 3 : 1);
    return FP_OK;
}

extern "C" int fp_stream_walls(fp_ctx* ctx, int64_t np, float* x, float* y, float* vx, float* vy, float* vz,
                               const uint32_t* pid, uint64_t step, void* stream)
{
    if (!ctx) return FP_ERR_ARG;
    if (np < 0 || (np > 0 && (!x || !y || !vx || !vy || !vz || !pid))) return fp_fail(ctx, FP_ERR_ARG, "fp_stream_walls: null pointer or np < 0");
    return fpi_stream_walls(ctx, np, x, y, vx, vy, vz, pid, step, nullptr, false, (cudaStream_t)stream);
}
