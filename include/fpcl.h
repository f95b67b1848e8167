/*
 * fpcl.h -- C ABI of the B200-native cubic Fokker-Planck closure hot path (arxiv/paper_2606_15622).
 *
 * One library (libfpcl.so, hand-written CUDA for sm_100a) exposes the per-cell, per-time-step closure path of
 * the paper's particle cubic-FP solver: PAPER.md Algorithm 1 (:205-225, physics closure) and Algorithm 2
 * (:250-270, surrogate closure).  Every step of the path runs in this library's kernels; callers only own memory.
 *
 * Conventions
 *  - C99 ABI, no exceptions.  Every call returns FP_OK (0) or a negative FP_ERR_* code; fp_last_error(ctx)
 *    gives a human-readable string for the last failure on that context.
 *  - Pointers are DEVICE pointers unless the name starts with h_ (host).  The caller owns every particle, grid,
 *    coefficient and weight buffer; the library never allocates or frees them.  The library owns only fp_ctx and
 *    its scratch.  Everything whose size follows from fp_params is allocated by fp_create (sort ping-pong buffers,
 *    digit histograms, per-cell update constants, the accumulators of the high-particles-per-cell paths and, on grids
 *    with a freestream face, a list of max_particles + 1 particle indices for the re-insertion pass).  Two
 *    pieces depend on later arguments and are allocated on FIRST USE unless fp_reserve was called: the packed
 *    parameters of a surrogate network (sized by its shape; a differently shaped network re-allocates) and the
 *    device staging buffers of fp_step_host.  A first-use allocation is a cudaMalloc and may stall the stream.
 *  - All calls are asynchronous on the caller's stream (a cudaStream_t passed as void*; NULL = legacy default
 *    stream) and, apart from the first-use allocations above, fp_step_host, fp_timing_read and fp_check, never
 *    synchronise the host.
 *  - cell_start must be a monotone prefix sum over the cells with cell_start[0] >= 0 and cell_start[ncell] == np
 *    (what fp_sort_by_cell writes).  fp_cell_moments and fp_velocity_update verify this ON THE DEVICE while they read it:
 *    cells with bad boundaries are skipped (no out-of-range access) and a sticky state word is set in the context;
 *    because the calls are asynchronous the failing call itself returns FP_OK and every LATER entry point on the
 *    context returns FP_ERR_STATE until fp_check (which synchronises) has reported and cleared it.
 *  - Numerical trouble in a cell is NOT an error code: it sets FP_FLAG_* bits in flags[cell] and the cell gets the
 *    documented fallback (readings R3-c, R5).
 *  - Particle arrays are SoA fp32: x, y, vx, vy, vz [np] and a persistent particle id pid [np] (uint32) that
 *    travels with the particle through the sort and seeds its random stream (R6).
 *  - Moment record per cell, fp64, row-major (R0):
 *      FULL (29): N, U1..3, P11,P12,P13,P22,P23,P33, t111,t112,t113,t122,t123,t133,t222,t223,t233,t333,
 *                 F11,F12,F13,F22,F23,F33 (F_ij = <c^2 c_i c_j>), g1,g2,g3 (g_i = <c^4 c_i>)
 *      LITE (13): N, U1..3, P(6), h1,h2,h3 (h_i = <c^2 c_i>)
 *    with c = v - U and <.> the plain 1/N mean over the cell's particles.
 *  - Coefficient record per cell (9, fp32): c11,c12,c13,c22,c23,c33,gamma1,gamma2,gamma3.
 */
#ifndef FPCL_H
#define FPCL_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* error codes */
#define FP_OK               0
#define FP_ERR_ARG         (-1)   /* null / misaligned pointer, size mismatch, bad enum                  */
#define FP_ERR_STATE       (-2)   /* np > max_particles; cell_start not a sorted prefix (see Conventions)   */
#define FP_ERR_CUDA        (-3)   /* a CUDA runtime call failed; see fp_last_error                        */
#define FP_ERR_UNSUPPORTED (-4)   /* e.g. an MLP wider than the fused kernel supports                     */

/* per-cell flag bits written to flags[cell] */
#define FP_FLAG_EMPTY      1u     /* N == 0: outputs zero                                                 */
#define FP_FLAG_LOWCOUNT   2u     /* N < min_count: Langevin coefficients c = -delta/tau, gamma = 0        */
#define FP_FLAG_SINGULAR   4u     /* theta <= 0, |pivot| < 1e-14 or non-finite solution: Langevin          */
#define FP_FLAG_ILLCOND    8u     /* scaled system ill-conditioned (estimate), solution kept               */
#define FP_FLAG_ALPHA     16u     /* alpha^2 (Eq. 15) non-finite or < 1e-6: alpha := 1                      */
#define FP_FLAG_SKIPPED   32u     /* velocity update skipped: N < 2 or theta <= 0                           */
#define FP_FLAG_NONFINITE 64u     /* surrogate produced a non-finite value: Langevin                        */

/* wall kinds */
#define FP_WALL_NONE     0
#define FP_WALL_DIFFUSE  1        /* diffuse isothermal re-emission                          */
#define FP_WALL_PERIODIC 2
#define FP_WALL_INFLOW   3        /* freestream reservoir (R11): a particle leaving through such a face re-enters
                                     at xmin from the freestream wall[0].{theta_w; ux > 0, uy, uz} with the flux-weighted
                                     half-Maxwellian in v_x; wall[0] must then be FP_WALL_INFLOW too; constant particle count */

typedef struct fp_ctx fp_ctx;

typedef struct {
    int32_t kind;                 /* FP_WALL_*                                                             */
    float   theta_w;              /* wall temperature as k T_w / m                                          */
    float   ux, uy, uz;           /* wall velocity                                                          */
} fp_wall;

/* POD, host memory, copied at fp_create. */
typedef struct {
    int32_t  nx, ny;              /* uniform Cartesian grid; ny = 1 for the 1D Couette case                */
    float    x0, y0, dx, dy;      /* domain origin and cell size (cell index: DESIGN.md R1)                */
    int64_t  max_particles;       /* scratch is sized for this                                              */
    float    dt;                  /* time step                                                              */
    float    tau;                 /* global relaxation time; ignored where a per-cell tau array is given    */
    float    eps2_scale;          /* multiplies the default eps^2 (R2-e); 0 disables the cubic term         */
    int32_t  min_count;           /* exact closure: cells with N < min_count use Langevin (R3-c)            */
    int32_t  min_count_mlp;       /* surrogate closure: same, usually 2                                     */
    int32_t  conserve_mode;       /* 0 = Eq. 13/15 only; 1 = + exact recentre/rescale per cell (R5.5)       */
    uint64_t seed;                /* Philox key                                                             */
    fp_wall  wall[4];             /* xmin, xmax, ymin, ymax                                                 */
    int32_t  body_kind;           /* 0 none, 1 embedded diffuse cylinder                                    */
    float    body_cx, body_cy, body_R, body_theta_w;
} fp_params;

/* MLP surrogate description.  h_dims is a host array of n_layers+1 widths;
 * W[l] / b[l] are host arrays of DEVICE pointers to fp32 weights, row-major [out][in], and biases.
 * x_mean/x_scale [n_in], y_mean/y_scale [9] are DEVICE pointers.  act 0 = SiLU, 1 = ReLU (hidden layers only;
 * the head is linear).  feature_set 0 = 13 inputs (n, U1..3, T, pi11,pi12,pi13,pi22,pi23, q1..3), 1 = the paper's
 * 16 inputs (R4).  n = N * n_scale, T = theta / theta_ref. */
typedef struct {
    int32_t             n_layers;
    const int32_t*      h_dims;
    const float* const* W;
    const float* const* b;
    const float*        x_mean;
    const float*        x_scale;
    const float*        y_mean;
    const float*        y_scale;
    int32_t             act;
    int32_t             feature_set;
    float               n_scale;
    float               theta_ref;
} fp_mlp;

/* Create / destroy a context on the current CUDA device.  fp_create validates h_params (nx, ny >= 1,
 * dx, dy > 0, max_particles >= 0, nx*ny < 2^27) and allocates scratch; fp_destroy frees it. */
int fp_create(fp_ctx** out, const fp_params* h_params);
int fp_destroy(fp_ctx* ctx);
const char* fp_last_error(const fp_ctx* ctx);
/* Library version / build string (static storage). */
const char* fp_version(void);

/* Allocate now what would otherwise be allocated on first use (Conventions): the packed-parameter scratch for a
 * network of h_mlp's shape (h_mlp nullable: skip) and, if host_staging != 0, the device buffers of fp_step_host
 * (6 arrays of max_particles + per-cell outputs, twice).  Synchronous (cudaMalloc).  After it no call on the context
 * allocates, unless a network of another shape is passed. */
int fp_reserve(fp_ctx* ctx, const fp_mlp* h_mlp /* nullable */, int32_t host_staging);
/* Synchronise `stream`, report (FP_ERR_STATE) and clear the sticky device-side state word; FP_OK if it was clear. */
int fp_check(fp_ctx* ctx, void* stream);

/* a2 -- cell index + stable sort (R1).  key = iy*nx + ix with
 * ix = clamp(floorf((x - x0) * (1/dx)), 0, nx-1) in fp32.  Writes the permuted SoA into the *_out arrays (which
 * may not alias the inputs), cell_start[ncell+1] (cell_start[k] = #particles with key < k) and, if non-null,
 * perm[np] with perm[k] = input index of the particle now at position k.  Equal keys keep input order. */
int fp_sort_by_cell(fp_ctx* ctx, int64_t np,
                    const float* x, const float* y, const float* vx, const float* vy, const float* vz,
                    const uint32_t* pid,
                    float* x_out, float* y_out, float* vx_out, float* vy_out, float* vz_out, uint32_t* pid_out,
                    int32_t* cell_start, uint32_t* perm /* nullable */, void* stream);

/* a3 -- segmented gather of the velocity moments over cell-sorted particles.
 * mode 0 = LITE (13 doubles/cell), 1 = FULL (29 doubles/cell).  mom is [ncell * stride] fp64. */
int fp_cell_moments(fp_ctx* ctx, int64_t np, const float* vx, const float* vy, const float* vz,
                    const int32_t* cell_start, int32_t mode, double* mom, void* stream);

/* a3 without a context and WITHOUT ANY ALLOCATION -- for callers that may not call cudaMalloc (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it).  Same operation, arguments and record layout as
 * fp_cell_moments (mode 0 = LITE, 1 = FULL), same fp32-sum / fp64-shift arithmetic as its
 * slice path (moments_seg.cuh): results agree with fp_cell_moments within the moment tolerance (1e-6), not bit for bit.
 * The entry point calls no cudaMalloc, cudaFree or allocating library routine; its only scratch (28 doubles per cell and
 * a status word) is a file-scope __device__ array of FP_STATIC_MAX_CELLS x 28 doubles = 3.5 MiB that every GPU which
 * loads the library holds until the process exits.
 *   - ncell > FP_STATIC_MAX_CELLS, np outside [0, 2^31), mode not 0/1, a null pointer, or vx/vy/vz not 16-byte aligned:
 *     FP_ERR_ARG, nothing launched; the reason is in fp_static_last_error() (thread-local text).
 *   - every call SHARES the one array, which keeps the last call's contents: the call clears what it uses on `stream`
 *     first, so calls in stream order are independent, but calls that overlap on the GPU (other streams, other threads)
 *     race on it and give wrong records.
 *   - cell_start is validated on the device as everywhere else; if it is not a sorted prefix ending at np, `mom` is left
 *     untouched.  d_status (device pointer to one uint32, nullable) receives 0 or the state bits (1 = bad cell_start) in
 *     stream order; there is no context to carry a sticky host-side state.
 *   - the first call on a device resolves the array's device address (cudaGetSymbolAddress) with that device current:
 *     make that call outside stream capture.  Asynchronous on `stream` like every other call. */
#define FP_STATIC_MAX_CELLS 16384
int fp_cell_moments_static(int64_t np, const float* vx, const float* vy, const float* vz,
                           const int32_t* cell_start, int32_t ncell, int32_t mode, double* mom,
                           uint32_t* d_status /* nullable */, void* stream);
const char* fp_static_last_error(void);

/* a4 -- exact cubic-FP closure: assemble and solve the 9x9 moment-matching system per cell (Eq. 10
 * :121, Table 1 :130-136; derivation DESIGN.md R2, scaling and flags R3).  tau_cell nullable (then params.tau).
 * coef [ncell*9] fp32, flags [ncell] (overwritten).  kappa_est nullable: if given receives the library's estimate of
 * the condition number of the scaled system: ||A||_inf times the triangular LINPACK probe of ||U^-1||_inf from the
 * factorisation (also max|pivot|/min|pivot| and ||A|| ||y|| / ||b|| if larger).  Measured against the oracle's exact
 * kappa_1 over condition numbers 1e1 .. 1e16 the estimate stays within a factor 4 either way (observed 0.34 .. 2.9)
 * (tests/test_gpu_parity.py::test_closure_exact_conditioning asserts it), and FP_FLAG_ILLCOND is set at
 * estimate >= 2.5e7, so every cell with kappa_1 >= 1e8 is flagged (a superset; the solution is kept either way). */
int fp_closure_exact(fp_ctx* ctx, const double* mom_full, const float* tau_cell /* nullable */,
                     float* coef, uint32_t* flags, double* kappa_est /* nullable */, void* stream);

/* a5 -- fused MLP surrogate: features -> standardise -> dense layers -> de-standardise (PAPER.md:264, :309,
 * :327).  mom_stride 13 or 29.  relax_w in (0,1]: coef <- w*new + (1-w)*old; 1 overwrites.
 * With relax_w < 1 `coef` is read: it must hold the previous step's coefficients, or zeros before the first step (not
 * uninitialised memory).  A cell whose nine old coefficients are all exactly zero -- it was EMPTY at the previous step,
 * or the array was zero-initialised -- has no history and takes the new values unblended (R12); otherwise
 * a newly populated cell would start at w times its coefficients, i.e. 1/w times too slow a relaxation.
 * The caller's weights (device memory, row-major [out][in]) are re-packed into context scratch by a small
 * kernel on every call, on the same stream: weights changed in place between calls are always picked up. */
int fp_closure_mlp(fp_ctx* ctx, const double* mom, int32_t mom_stride, const float* tau_cell /* nullable */,
                   const fp_mlp* h_mlp, float relax_w, float* coef, uint32_t* flags, void* stream);

/* Surrogate kernel choice.  enable = 1 (default): networks of shape [13|16]-64-64-64-9 run on the tensor cores
 * (mma.sync TF32 with 3xTF32 error compensation; agrees with an fp64 forward pass to ~1e-5 of the output scale --
 * north_star allows 3e-3 for TF32), and networks whose hidden layers are all 256 wide, [13|16]-256-...-256-9 with
 * 1 to 7 hidden layers, e.g. the paper's own 16-256-256-256-256-9, run on the tcgen05 tensor cores
 * with the accumulator in TMEM (bf16 with split operands, three products per useful product, ~3e-5 of the output
 * scale on the test networks, up to 2.5e-4 over 300 random Xavier networks and ensembles; north_star's tensor-core
 * allowance is 3e-3).  enable = 2: as 1, but the wide networks use the mma.sync kernel (same arithmetic, about half the speed;
 * kept for comparison).  enable = 0: every shape runs the plain fp32-FMA kernel (1e-5), as do all other shapes
 * under any setting.  The environment variable FPCL_MLP_FP32=1 sets enable = 0 at fp_create. */
int fp_set_mlp_tensor_cores(fp_ctx* ctx, int32_t enable);

/* Sampling outputs (they run once per sampled step, outside the per-step path).
 * fp_cell_diagnostics: 16 fp64 values per cell from the FULL record (PAPER.md:415 and Eq. 19-23 :632-657; the
 * normalisations are reading R10 of DESIGN.md): theta = P_kk/3; Delta_4 = <c^4> - 15 theta^2; Delta_4/(15 theta^2);
 * D_G = -1/2 log det(P/theta); D_q = |q_hat|^2/5 with q_hat = h/(2 theta^1.5); ds_eq = 3/2 log(theta/theta_inf) -
 * log(N/n_inf); ds_kin,G = ds_eq - (D_G - dg_inf); sigma_norm = |P - theta I|_F/theta; q_norm = |q_hat|;
 * m3_norm = |t|_F/theta^1.5; R_11, R_12, R_13, R_22, R_23, R_33, each <c_i c_j c^2>/(5 theta^2).  Empty or cold
 * (theta <= 0) cell: zeros; singular covariance (N < 4, or det <= 0): D_G = +inf, ds_kin,G = -inf.  DM6 needs a sixth-order
 * sum the record does not carry: fp_cell_sixth_moment.  mom_full [ncell*29], diag [ncell*16] (16-byte aligned),
 * device memory; theta_inf, n_inf > 0 are the upstream reference state (Eq. 20), dg_inf its D_G (Eq. 23).
 * fp_average_results: running time average, avg[i] <- avg[i] + (x[i] - avg[i])/(k + 1) for
 * i < n, k = number of samples already averaged; x, avg device fp64. */
int fp_cell_diagnostics(fp_ctx* ctx, const double* mom_full, double theta_inf, double n_inf, double dg_inf,
                        double* diag, void* stream);
int fp_average_results(fp_ctx* ctx, int64_t n, const double* x, int64_t k, double* avg, void* stream);
/* fp_cell_sixth_moment: DM6 = <(c_k c_k)^3> per cell from the cell-sorted velocities and the means U of the
 * moment record (mom_stride 13 or 29); dm6 [ncell] fp64, 0 for an empty cell.  A Maxwellian has DM6 = 105 theta^3. */
int fp_cell_sixth_moment(fp_ctx* ctx, int64_t np, const float* vx, const float* vy, const float* vz,
                const int32_t* cell_start, const double* mom, int32_t mom_stride, double* dm6, void* stream);

/* a6 -- FP velocity update, in place on cell-sorted vx, vy, vz (Eq. 13-15 :150-181; R5, R6).
 * step is the Philox counter word for time.  flags [ncell] are OR-ed with FP_FLAG_ALPHA / FP_FLAG_SKIPPED.
 * mom, coef and tau_cell must be the arrays the coefficients were computed from and stay valid until the call has run:
 * besides the per-cell constants derived from them, the kernel re-reads them for the cells it redoes in fp64 (cells with a
 * particle beyond the range fp32 arithmetic holds to 1e-6, few-particle cells whose conservation scale cancels; DESIGN.md
 * section 5).  Accuracy: 1e-6 * max(|v|, sqrt(theta_cell)) per component against Eq. 13-15 evaluated in fp64 with the
 * same Philox stream.  Grids of few huge cells (above ~450 particles per cell) run slice kernels that add per-slice sums
 * with fp64 atomics: their results can differ in the last bit from run to run (fp_set_reproducible avoids them). */
int fp_velocity_update(fp_ctx* ctx, int64_t np, float* vx, float* vy, float* vz, const uint32_t* pid,
                       const int32_t* cell_start, const double* mom, int32_t mom_stride, const float* coef,
                       const float* tau_cell /* nullable */, uint64_t step, uint32_t* flags, void* stream);

/* a0 + a1 -- streaming (Eq. 16 :187) and diffuse isothermal walls (:214, :674; R7),
 * in place. */
int fp_stream_walls(fp_ctx* ctx, int64_t np, float* x, float* y, float* vx, float* vy, float* vz,
                    const uint32_t* pid, uint64_t step, void* stream);

/* a7 -- one whole step in the order of Algorithm 1/2: stream -> walls -> sort -> moments -> closure -> update.
 * State is read from (and streamed in place in) the *_a arrays and the cell-sorted, updated state is written to
 * the *_b arrays; the caller swaps a and b between steps.  closure 0 = exact (mom must hold ncell*29 doubles),
 * 1 = surrogate (ncell*13 doubles, LITE gather).  tau_mode 0: params.tau everywhere; 1: per-cell
 * tau = tau_ref_n / N computed on the device from the counts and written to tau_cell [ncell] (must be non-null;
 * PAPER.md:83 tau = 2 mu / p ~ 1/n).  relax_w as in fp_closure_mlp. */
int fp_step(fp_ctx* ctx, int64_t np,
            float* x_a, float* y_a, float* vx_a, float* vy_a, float* vz_a, uint32_t* pid_a,
            float* x_b, float* y_b, float* vx_b, float* vy_b, float* vz_b, uint32_t* pid_b,
            int32_t closure, const fp_mlp* h_mlp, float relax_w,
            int32_t tau_mode, float tau_ref_n, float* tau_cell /* nullable unless tau_mode 1 */,
            uint64_t step, double* mom, float* coef, uint32_t* flags, int32_t* cell_start, void* stream);

/* one domain cut into slabs of whole rows, one particle exchange per step (the paper itself runs one
 * GPU, and independent replicas, :668).  Every slab's context is created with the GLOBAL fp_params (walls,
 * body and the cell-index formula are the whole domain's; max_particles bounds what the slab may hold) and then told its
 * rows: fp_set_slab(ctx, row0, nrows), before any other call; from then on the context has nx*nrows cells, numbered from its
 * first row, and every per-cell array is that long.  A step on a slab: fp_stream_walls -> fp_slab_partition -> exchange
 * (caller: device copies or NCCL) -> fp_collide.
 * fp_slab_partition: stable partition of np particles by destination slab.  h_row_bounds [nslabs+1] (HOST) are the first
 * rows of the slabs, from 0 to ny, 1 <= nslabs <= 64; slab_start [nslabs+1] (DEVICE) receives the offsets: particles
 * slab_start[s] .. slab_start[s+1]-1 of the *_out arrays go to slab s, in input order.  Outputs may not alias inputs.
 * If every receiver concatenates what it gets in ascending source-slab order (its own stayers in their place), fp_collide
 * sees exactly the sub-sequence of the uncut domain's array that the slab owns, and the cut run is bit-identical to the
 * uncut one (tests/test_gpu_slab.py).
 * fp_collide: the part of fp_step after the move -- sort by cell, moments, closure, update -- with fp_step's arguments;
 * positions are read only. */
int fp_set_slab(fp_ctx* ctx, int32_t row0, int32_t nrows);
/* on != 0: every per-cell result (moment record, coefficients, updated velocities) depends only on the cell's own particles
 * in their array order -- not on WHERE in the arrays they sit, on the cell's neighbours, on the context's mean density, nor on
 * the run.  By default the moment gather and the velocity update give a group of 4..32 lanes one cell and pick the group
 * width from the context's mean particles per cell, start each cell at the particle whose shared-memory bank suits the
 * warp, and send ensembles of few huge cells through slice kernels that combine per-slice sums with atomics: all of
 * that changes the fp32 summation ORDER -- not the result beyond rounding -- with the cell's offset and surroundings.
 * Reproducible mode walks every cell on its own with all 32 lanes and never uses the slice kernels (2-3x slower moments
 * and update at 100 particles per cell).  Switch it on (on every slab and on the uncut run) to compare decompositions bit
 * for bit. */
int fp_set_reproducible(fp_ctx* ctx, int32_t on);
int fp_slab_partition(fp_ctx* ctx, int64_t np,
                      const float* x, const float* y, const float* vx, const float* vy, const float* vz, const uint32_t* pid,
                      float* x_out, float* y_out, float* vx_out, float* vy_out, float* vz_out, uint32_t* pid_out,
                      const int32_t* h_row_bounds, int32_t nslabs, int32_t* slab_start, void* stream);
int fp_collide(fp_ctx* ctx, int64_t np,
               const float* x_a, const float* y_a, const float* vx_a, const float* vy_a, const float* vz_a, const uint32_t* pid_a,
               float* x_b, float* y_b, float* vx_b, float* vy_b, float* vz_b, uint32_t* pid_b,
               int32_t closure, const fp_mlp* h_mlp, float relax_w,
               int32_t tau_mode, float tau_ref_n, float* tau_cell /* nullable unless tau_mode 1 */,
               uint64_t step, double* mom, float* coef, uint32_t* flags, int32_t* cell_start, void* stream);

/* Host-buffer convenience used by the end-to-end measurement: uploads the six SoA arrays from host memory
 * (pinned or pageable), runs fp_step on internally held device buffers sized max_particles, and downloads the
 * updated SoA plus cell_start, flags and coef back into the host arrays.  All uploads run on the caller's stream
 * before the first kernel (the stream kernel rewrites vx, vy, vz of re-emitted particles, so none may still be in
 * flight); the download of x, y, pid (final after the gather) runs on a context-owned side stream and overlaps the
 * moment, closure and update kernels; both streams are synchronised before returning.
 * h_* are HOST pointers; h_coef [ncell*9], h_flags [ncell], h_cell_start [ncell+1]. */
int fp_step_host(fp_ctx* ctx, int64_t np,
                 float* h_x, float* h_y, float* h_vx, float* h_vy, float* h_vz, uint32_t* h_pid,
                 int32_t closure, const fp_mlp* h_mlp, float relax_w, uint64_t step,
                 float* h_coef, uint32_t* h_flags, int32_t* h_cell_start, void* stream);

/* Measurement hooks (bench.py).  fp_timing_enable(ctx, max_steps) makes every following fp_step record CUDA events
 * on the caller's stream at its stage boundaries (max_steps = 0 switches it off and frees the events);
 * fp_timing_read waits for the last recorded event and writes, for each recorded step, FP_NSTAGES durations in
 * milliseconds to h_ms (host, [max_steps * FP_NSTAGES]) in the order: stream+walls(+keys), radix sort + cell_start,
 * payload gather, moment gather, closure, velocity update; *h_nsteps receives the number of steps recorded and the
 * recorder is reset.  fp_launch_count returns the number of kernels this context has launched so far. */
#define FP_NSTAGES 6
int fp_timing_enable(fp_ctx* ctx, int32_t max_steps);
int fp_timing_read(fp_ctx* ctx, float* h_ms, int32_t* h_nsteps);
uint64_t fp_launch_count(const fp_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* FPCL_H */
