// closure_mlp.cu -- a5: fused MLP surrogate for the nine closure coefficients (PAPER.md:244, :264 predict_coeffs,
// :309 layer shape, :327 StandardScaler on inputs and outputs, :568 under-relaxation; R4).
//
// One kernel does everything per cell: features from the fp64 moment record -> fp32 -> standardise -> all dense
// layers with the activation -> linear head -> de-standardise -> fallback policy -> optional blend with the
// previous coefficients.  One thread per cell; activations live in shared memory as [unit][cell] (conflict-free),
// weights are repacked once per call into [in][out padded to 8] and kept in shared memory when they fit
// (13-64-64-64-9: 39 KB), otherwise read through L1/L2.  Each thread produces 8 outputs per sweep over the
// inputs, so one activation load and two broadcast 128-bit weight loads feed 8 FMAs.  Plain fp32 FMA pipe
// (tolerance 1e-5); no tensor cores in this kernel.
#include "tiles.cuh"
#include "upd_prep.cuh"

#define MLP_OB 8

struct mlp_desc {
    int32_t n_layers;
    int32_t dims[FPCL_MAX_LAYERS + 1];
    int32_t w_off[FPCL_MAX_LAYERS];     // float offsets into the packed blob: Wt[in][out_pad]
    int32_t b_off[FPCL_MAX_LAYERS];     // bias[out_pad]
    int32_t xm_off, xs_off, ym_off, ys_off;
    int32_t blob_floats, maxw;
    int32_t act, feature_set;
    float n_scale, theta_ref;
};

struct mlp_src {
    const float* W[FPCL_MAX_LAYERS];
    const float* b[FPCL_MAX_LAYERS];
    const float *x_mean, *x_scale, *y_mean, *y_scale;
};

static inline int pad8(int v) { return (v + 7) & ~7; }

#include "mlp_tc.cuh"
#include "mlp_wide.cuh"
#include "mlp_wide5.cuh"

// repack caller weights [out][in] -> blob Wt[in][out_pad], bias[out_pad] (zero padded), scalers appended
__global__ void mlp_pack_kernel(const __grid_constant__ mlp_desc D, const __grid_constant__ mlp_src S,
                                float* __restrict__ blob)
{
    fpd_pdl();
    const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
    for (int l = 0; l < D.n_layers; ++l) {
        const int ni = D.dims[l], no = D.dims[l + 1], nop = (no + 7) & ~7;
        for (int e = tid; e < ni * nop; e += nth) {
            const int i = e / nop, o = e % nop;
            blob[D.w_off[l] + e] = (o < no) ? S.W[l][(size_t)o * ni + i] : 0.0f;
        }
        for (int o = tid; o < nop; o += nth) blob[D.b_off[l] + o] = (o < no) ? S.b[l][o] : 0.0f;
    }
    const int nin = D.dims[0], nout = D.dims[D.n_layers];
    for (int i = tid; i < nin; i += nth) { blob[D.xm_off + i] = S.x_mean[i]; blob[D.xs_off + i] = S.x_scale[i]; }
    for (int i = tid; i < nout; i += nth) { blob[D.ym_off + i] = S.y_mean[i]; blob[D.ys_off + i] = S.y_scale[i]; }
}

template <int CB>
__global__ void __launch_bounds__(CB)
mlp_kernel(const double* __restrict__ mom, int32_t stride, const float* __restrict__ tau_cell, float tau_scalar,
           const float* __restrict__ blob, const __grid_constant__ mlp_desc D, int32_t w_in_smem, int32_t min_count,
           float relax_w, int32_t ncell, float* __restrict__ coef, uint32_t* __restrict__ flags,
           float* __restrict__ cellc, float dt, float eps2_scale)
{
    fpd_pdl();
    extern __shared__ __align__(16) float smem[];
    float* wsm = smem;
    float* act0 = smem + (w_in_smem ? ((D.blob_floats + 3) & ~3) : 0);
    float* act1 = act0 + (size_t)D.maxw * CB;
    const int tid = threadIdx.x;
    if (w_in_smem) {
        for (int e = tid; e < D.blob_floats; e += CB) wsm[e] = blob[e];
    }
    const float* wp = w_in_smem ? wsm : blob;
    const int64_t cell = (int64_t)blockIdx.x * CB + tid;
    const bool have = cell < ncell;
    const double* rec = mom + (size_t)(have ? cell : 0) * stride;
    const double nraw = rec[0];
    const float tau = tau_cell ? tau_cell[have ? cell : 0] : tau_scalar;
    const double theta = (rec[4] + rec[7] + rec[9]) / 3.0;
    // ---- features (R4), fp64 -> fp32
    {
        double h[3];
        if (stride == 13) { h[0] = rec[10]; h[1] = rec[11]; h[2] = rec[12]; }
        else {            // h_i = t_ikk : t111+t122+t133, t112+t222+t233, t113+t223+t333
            h[0] = rec[10] + rec[13] + rec[15]; h[1] = rec[11] + rec[16] + rec[18]; h[2] = rec[12] + rec[17] + rec[19];
        }
        const double n = nraw * (double)D.n_scale;
        float x[16];
        if (D.feature_set == 0) {
            x[0] = (float)n; x[1] = (float)rec[1]; x[2] = (float)rec[2]; x[3] = (float)rec[3];
            x[4] = (float)(theta / (double)D.theta_ref);
            x[5] = (float)(n * (rec[4] - theta)); x[6] = (float)(n * rec[5]); x[7] = (float)(n * rec[6]);
            x[8] = (float)(n * (rec[7] - theta)); x[9] = (float)(n * rec[8]);
            x[10] = (float)(0.5 * n * h[0]); x[11] = (float)(0.5 * n * h[1]); x[12] = (float)(0.5 * n * h[2]);
            x[13] = x[14] = x[15] = 0.f;
        } else {
            x[0] = (float)n; x[1] = (float)(theta / (double)D.theta_ref);
            x[2] = (float)rec[1]; x[3] = (float)rec[2]; x[4] = (float)rec[3];
#pragma unroll
            for (int k = 0; k < 6; ++k) x[5 + k] = (float)(n * rec[4 + k]);
            x[11] = (float)(0.5 * n * h[0]); x[12] = (float)(0.5 * n * h[1]); x[13] = (float)(0.5 * n * h[2]);
            x[14] = (float)(3.0 * theta);
            x[15] = (float)(1.0 / (double)tau);
        }
        __syncthreads();      // weights (and scalers) are in shared memory now
        const int nin = D.dims[0];
#pragma unroll
        for (int i = 0; i < 16; ++i)
            if (i < nin) act0[i * CB + tid] = (x[i] - wp[D.xm_off + i]) / wp[D.xs_off + i];
    }
    // ---- dense layers
    float* ain = act0;
    float* aout = act1;
    for (int l = 0; l < D.n_layers; ++l) {
        const int ni = D.dims[l], no = D.dims[l + 1], nop = (no + 7) & ~7;
        const float* Wt = wp + D.w_off[l];
        const float* bs = wp + D.b_off[l];
        const bool hidden = l < D.n_layers - 1;
        for (int o0 = 0; o0 < nop; o0 += MLP_OB) {
            float acc[MLP_OB];
#pragma unroll
            for (int j = 0; j < MLP_OB; ++j) acc[j] = bs[o0 + j];
            const float* wrow = Wt + o0;
#pragma unroll 4
            for (int i = 0; i < ni; ++i) {
                const float a = ain[i * CB + tid];
                const float4 w0 = *reinterpret_cast<const float4*>(wrow + (size_t)i * nop);
                const float4 w1 = *reinterpret_cast<const float4*>(wrow + (size_t)i * nop + 4);
                acc[0] = fmaf(w0.x, a, acc[0]); acc[1] = fmaf(w0.y, a, acc[1]);
                acc[2] = fmaf(w0.z, a, acc[2]); acc[3] = fmaf(w0.w, a, acc[3]);
                acc[4] = fmaf(w1.x, a, acc[4]); acc[5] = fmaf(w1.y, a, acc[5]);
                acc[6] = fmaf(w1.z, a, acc[6]); acc[7] = fmaf(w1.w, a, acc[7]);
            }
#pragma unroll
            for (int j = 0; j < MLP_OB; ++j) {
                float s = acc[j];
                if (hidden) s = (D.act == 0) ? s / (1.0f + expf(-s)) : fmaxf(s, 0.0f);
                aout[(o0 + j) * CB + tid] = s;
            }
        }
        float* sw = ain; ain = aout; aout = sw;
    }
    // ---- de-standardise, policy, blend
    if (!have) return;
    float y[9];
    bool finite = true;
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        y[k] = fmaf(ain[k * CB + tid], wp[D.ys_off + k], wp[D.ym_off + k]);
        finite = finite && isfinite(y[k]);
    }
    uint32_t flag = 0;
    float* out = coef + (size_t)cell * 9;
    if (!(nraw > 0.0)) {
#pragma unroll
        for (int k = 0; k < 9; ++k) y[k] = 0.0f;
        flag = FP_FLAG_EMPTY;
    } else {
        bool langevin = false;
        if (nraw < (double)min_count) { flag = FP_FLAG_LOWCOUNT; langevin = true; }
        else if (!(theta > 0.0) || !isfinite(theta)) { flag = FP_FLAG_SINGULAR; langevin = true; }
        else if (!finite) { flag = FP_FLAG_NONFINITE; langevin = true; }
        if (langevin) {
            const float d = -1.0f / tau;
            y[0] = d; y[1] = 0.f; y[2] = 0.f; y[3] = d; y[4] = 0.f; y[5] = d; y[6] = 0.f; y[7] = 0.f; y[8] = 0.f;
        }
        if (relax_w != 1.0f) {
            // no history (all nine old coefficients zero: EMPTY last step / zero-initialised first step): no blend (R12)
            bool history = false;
#pragma unroll
            for (int k = 0; k < 9; ++k) history = history || out[k] != 0.0f;
            if (history) {
#pragma unroll
                for (int k = 0; k < 9; ++k) y[k] = relax_w * y[k] + (1.0f - relax_w) * out[k];
            }
        }
    }
#pragma unroll
    for (int k = 0; k < 9; ++k) out[k] = y[k];
    // inside fp_step the velocity update follows: hand it its per-cell constants now (upd_prep.cuh)
    if (cellc) flag |= upd_prep_cell(rec, stride, y, (double)tau, dt, eps2_scale, cellc + (size_t)cell * UPD_NC);
    flags[cell] = flag;
}

extern "C" int fp_set_mlp_tensor_cores(fp_ctx* ctx, int32_t enable)
{
    if (!ctx) return FP_ERR_ARG;
    ctx->mlp_force_fp32 = (enable == 0);
    ctx->mlp_wide_mma_sync = (enable == 2);
    return FP_OK;
}

extern "C" int fp_closure_mlp(fp_ctx* ctx, const double* mom, int32_t mom_stride, const float* tau_cell,
                              const fp_mlp* h_mlp, float relax_w, float* coef, uint32_t* flags, void* stream)
{
    if (!ctx) return FP_ERR_ARG;
    return fpi_closure_mlp(ctx, mom, mom_stride, tau_cell, h_mlp, relax_w, coef, flags, false, (cudaStream_t)stream);
}

// Size every packed-parameter buffer a network of this shape can need (whichever kernel is selected later), now.
// fp_closure_mlp grows the same buffers on first use otherwise; see fp_reserve in include/fpcl.h.
int fpi_mlp_reserve(fp_ctx* ctx, const fp_mlp* h_mlp)
{
    if (!h_mlp || !h_mlp->h_dims || h_mlp->n_layers < 1 || h_mlp->n_layers > FPCL_MAX_LAYERS)
        return fp_fail(ctx, FP_ERR_ARG, "fp_reserve: bad fp_mlp description");
    const fp_mlp& M = *h_mlp;
    fp_mlp_dev& C = ctx->mlp;
    int off = 0;
    for (int l = 0; l <= M.n_layers; ++l)
        if (M.h_dims[l] < 1 || M.h_dims[l] > 1024) return fp_fail(ctx, FP_ERR_UNSUPPORTED, "fp_reserve: layer width must be in [1,1024]");
    for (int l = 0; l < M.n_layers; ++l) off += M.h_dims[l] * pad8(M.h_dims[l + 1]) + pad8(M.h_dims[l + 1]);
    off += 2 * pad8(M.h_dims[0]) + 32;
    auto ensure = [&](void** ptr, size_t* have, size_t need) -> int {
        if (*have >= need) return FP_OK;
        if (*ptr) FP_CUDA_OK(ctx, cudaFree(*ptr));
        *ptr = nullptr; *have = 0;
        FP_CUDA_OK(ctx, cudaMalloc(ptr, need));
        *have = need;
        return FP_OK;
    };
    int rc;
    if (M.n_layers == 4 && M.h_dims[1] == TC_H && M.h_dims[2] == TC_H && M.h_dims[3] == TC_H && !C.tc_frags)
        FP_CUDA_OK(ctx, cudaMalloc((void**)&C.tc_frags, (size_t)TC_FRAGS * sizeof(float4) + (size_t)TC_MISC * sizeof(float)));
    bool wide = M.n_layers >= 2;
    for (int l = 1; l < M.n_layers && wide; ++l) wide = M.h_dims[l] == WD_H;
    if (wide) {
        const size_t mbytes = (size_t)wd_misc_floats(M.n_layers) * sizeof(float);
        if ((rc = ensure(&C.w5_blob, &C.w5_bytes, w5_blob_bytes(M.n_layers) + mbytes)) != FP_OK) return rc;
        if ((rc = ensure((void**)&C.wd_frags, &C.wd_bytes, wd_frag_total(M.n_layers) * sizeof(uint4) + mbytes)) != FP_OK) return rc;
    }
    size_t blob_bytes = C.blob_floats * sizeof(float);
    if ((rc = ensure((void**)&C.blob, &blob_bytes, (size_t)off * sizeof(float))) != FP_OK) return rc;
    C.blob_floats = blob_bytes / sizeof(float);
    return FP_OK;
}

int fpi_closure_mlp(fp_ctx* ctx, const double* mom, int32_t mom_stride, const float* tau_cell, const fp_mlp* h_mlp,
                    float relax_w, float* coef, uint32_t* flags, bool with_update_constants, cudaStream_t st)
{
    float* cellc = with_update_constants ? ctx->cellc : nullptr;
    if (!mom || !h_mlp || !coef || !flags || (mom_stride != 13 && mom_stride != 29))
        return fp_fail(ctx, FP_ERR_ARG, "fp_closure_mlp: null pointer or bad mom_stride");
    const fp_mlp& M = *h_mlp;
    if (M.n_layers < 1 || M.n_layers > FPCL_MAX_LAYERS || !M.h_dims || !M.W || !M.b || !M.x_mean || !M.x_scale ||
        !M.y_mean || !M.y_scale || (M.act != 0 && M.act != 1) || (M.feature_set != 0 && M.feature_set != 1))
        return fp_fail(ctx, FP_ERR_ARG, "fp_closure_mlp: bad fp_mlp description");
    if (!(relax_w > 0.0f && relax_w <= 1.0f)) return fp_fail(ctx, FP_ERR_ARG, "fp_closure_mlp: relax_w must be in (0,1]");
    const int nin_expected = M.feature_set == 0 ? 13 : 16;
    if (M.h_dims[0] != nin_expected || M.h_dims[M.n_layers] != 9)
        return fp_fail(ctx, FP_ERR_ARG, "fp_closure_mlp: input width must match feature_set and output width must be 9");
    mlp_desc D;
    memset(&D, 0, sizeof(D));
    mlp_src S;
    memset(&S, 0, sizeof(S));
    D.n_layers = M.n_layers;
    int off = 0, maxw = 16;
    for (int l = 0; l <= M.n_layers; ++l) {
        if (M.h_dims[l] < 1 || M.h_dims[l] > 1024) return fp_fail(ctx, FP_ERR_UNSUPPORTED, "fp_closure_mlp: layer width must be in [1,1024]");
        D.dims[l] = M.h_dims[l];
        if (pad8(M.h_dims[l]) > maxw) maxw = pad8(M.h_dims[l]);
    }
    for (int l = 0; l < M.n_layers; ++l) {
        if (!M.W[l] || !M.b[l]) return fp_fail(ctx, FP_ERR_ARG, "fp_closure_mlp: null layer pointer");
        S.W[l] = M.W[l]; S.b[l] = M.b[l];
        D.w_off[l] = off; off += D.dims[l] * pad8(D.dims[l + 1]);
        D.b_off[l] = off; off += pad8(D.dims[l + 1]);
    }
    D.xm_off = off; off += pad8(D.dims[0]);
    D.xs_off = off; off += pad8(D.dims[0]);
    D.ym_off = off; off += 16;
    D.ys_off = off; off += 16;
    D.blob_floats = off; D.maxw = maxw;
    D.act = M.act; D.feature_set = M.feature_set; D.n_scale = M.n_scale; D.theta_ref = M.theta_ref;
    S.x_mean = M.x_mean; S.x_scale = M.x_scale; S.y_mean = M.y_mean; S.y_scale = M.y_scale;
    fp_mlp_dev& C = ctx->mlp;
    // ---- tensor-core path for the benchmark shape [13|16]-64-64-64-9
    if (!ctx->mlp_force_fp32 && M.n_layers == 4 && D.dims[1] == TC_H && D.dims[2] == TC_H && D.dims[3] == TC_H) {
        const size_t fbytes = (size_t)TC_FRAGS * sizeof(float4) + (size_t)TC_MISC * sizeof(float);
        if (!C.tc_frags) FP_CUDA_OK(ctx, cudaMalloc((void**)&C.tc_frags, fbytes));
        float4* frags = reinterpret_cast<float4*>(C.tc_frags);
        float* misc = C.tc_frags + (size_t)TC_FRAGS * 4;
        fp_launch(mlp_tc_pack_kernel, 20, 256, 0, st, S, D.dims[0], frags, misc);
        tc_params P;
        P.stride = mom_stride; P.feature_set = M.feature_set; P.act = M.act; P.min_count = ctx->p.min_count_mlp;
        P.ncell = ctx->ncell; P.nin = D.dims[0]; P.tau_scalar = ctx->p.tau; P.n_scale = M.n_scale;
        P.theta_ref = M.theta_ref; P.relax_w = relax_w;
        P.dt = ctx->p.dt; P.eps2_scale = ctx->p.eps2_scale; P.cellc = cellc;
        const size_t smem = fbytes + (size_t)TC_WARPS * 16 * 17 * sizeof(float);
        int& occ = ctx->mlp_tc_occ;
        if (occ == 0) {
            FP_CUDA_OK(ctx, cudaFuncSetAttribute(mlp_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, mlp_tc_kernel, TC_THREADS, smem);
            if (occ < 1) occ = 1;
        }
        const int want = fp_div_up(fp_div_up(ctx->ncell, 16), TC_WARPS);
        const int cap = ctx->num_sms * occ;
        fp_launch(mlp_tc_kernel, want < cap ? want : cap, TC_THREADS, smem, st, mom, tau_cell, frags, misc, coef, flags, P);
        FP_LAUNCH_OK(ctx);
        FP_COUNT(ctx, 2);
        return FP_OK;
    }
    // ---- tensor-core path for wide networks [13|16]-256-...-256-9 (the paper's own shape, mlp_wide.cuh)
    bool wide = !ctx->mlp_force_fp32 && M.n_layers >= 2;
    for (int l = 1; l < M.n_layers && wide; ++l) wide = D.dims[l] == WD_H;
    if (wide && !ctx->mlp_wide_mma_sync) {
        // tcgen05 / TMEM kernel (mlp_wide5.cuh): weights as stage images + biases/scalers
        const size_t bbytes = w5_blob_bytes(M.n_layers);
        const size_t mbytes = (size_t)wd_misc_floats(M.n_layers) * sizeof(float);
        if (C.w5_bytes < bbytes + mbytes) {
            if (C.w5_blob) FP_CUDA_OK(ctx, cudaFree(C.w5_blob));
            C.w5_blob = nullptr; C.w5_bytes = 0;
            FP_CUDA_OK(ctx, cudaMalloc((void**)&C.w5_blob, bbytes + mbytes));
            C.w5_bytes = bbytes + mbytes;
        }
        unsigned char* blob5 = reinterpret_cast<unsigned char*>(C.w5_blob);
        float* misc = reinterpret_cast<float*>(blob5 + bbytes);
        // biases and scalers come from the mma.sync pack kernel's misc section (same layout): pack both
        fp_launch(mlpw5_pack_kernel, 2 * ctx->num_sms, 256, 0, st, S, M.n_layers, D.dims[0], reinterpret_cast<uint4*>(blob5));
        fp_launch(mlpw_misc_kernel, 8, 256, 0, st, S, M.n_layers, D.dims[0], misc);
        wd_params P;
        P.stride = mom_stride; P.feature_set = M.feature_set; P.act = M.act; P.min_count = ctx->p.min_count_mlp;
        P.ncell = ctx->ncell; P.nin = D.dims[0]; P.n_layers = M.n_layers; P.tau_scalar = ctx->p.tau;
        P.n_scale = M.n_scale; P.theta_ref = M.theta_ref; P.relax_w = relax_w;
        P.dt = ctx->p.dt; P.eps2_scale = ctx->p.eps2_scale; P.cellc = cellc;
        const size_t smem = (size_t)2 * W5_A_PART + (size_t)W5_STAGES * W5_STAGE_BYTES +
                            (size_t)((wd_misc_floats(M.n_layers) + 3) & ~3) * sizeof(float) + 16 * sizeof(uint64_t);
        bool& attr5_set = ctx->mlp_attr_w5;
        if (!attr5_set) {
            FP_CUDA_OK(ctx, cudaFuncSetAttribute(mlp_wide5_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024));
            attr5_set = true;
        }
        const int want = fp_div_up(ctx->ncell, W5_M);
        fp_launch(mlp_wide5_kernel, want < ctx->num_sms ? want : ctx->num_sms, W5_THREADS, smem, st, mom, tau_cell,
                  (const unsigned char*)blob5, (const float*)misc, coef, flags, P);
        FP_LAUNCH_OK(ctx);
        FP_COUNT(ctx, 3);
        return FP_OK;
    }
    if (wide) {
        const size_t fbytes = wd_frag_total(M.n_layers) * sizeof(uint4);
        const size_t mbytes = (size_t)wd_misc_floats(M.n_layers) * sizeof(float);
        if (C.wd_bytes < fbytes + mbytes) {
            if (C.wd_frags) FP_CUDA_OK(ctx, cudaFree(C.wd_frags));
            C.wd_frags = nullptr; C.wd_bytes = 0;
            FP_CUDA_OK(ctx, cudaMalloc((void**)&C.wd_frags, fbytes + mbytes));
            C.wd_bytes = fbytes + mbytes;
        }
        uint4* frags = reinterpret_cast<uint4*>(C.wd_frags);
        float* misc = reinterpret_cast<float*>(reinterpret_cast<unsigned char*>(C.wd_frags) + fbytes);
        fp_launch(mlpw_pack_kernel, 2 * ctx->num_sms, 256, 0, st, S, M.n_layers, D.dims[0], frags, misc);
        wd_params P;
        P.stride = mom_stride; P.feature_set = M.feature_set; P.act = M.act; P.min_count = ctx->p.min_count_mlp;
        P.ncell = ctx->ncell; P.nin = D.dims[0]; P.n_layers = M.n_layers; P.tau_scalar = ctx->p.tau;
        P.n_scale = M.n_scale; P.theta_ref = M.theta_ref; P.relax_w = relax_w;
        P.dt = ctx->p.dt; P.eps2_scale = ctx->p.eps2_scale; P.cellc = cellc;
        const size_t smem = (size_t)4 * WD_M * WD_XS * sizeof(__nv_bfloat16) +
                            (size_t)((wd_misc_floats(M.n_layers) + 3) & ~3) * sizeof(float) + (size_t)WD_M * 17 * sizeof(float);
        bool& attr_set = ctx->mlp_attr_wd;
        if (!attr_set) {
            FP_CUDA_OK(ctx, cudaFuncSetAttribute(mlp_wide_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
            attr_set = true;
        }
        const int want = fp_div_up(ctx->ncell, WD_M);
        fp_launch(mlp_wide_kernel, want < ctx->num_sms ? want : ctx->num_sms, WD_THREADS, smem, st, mom, tau_cell,
                  (const uint4*)frags, (const float*)misc, coef, flags, P);
        FP_LAUNCH_OK(ctx);
        FP_COUNT(ctx, 2);
        return FP_OK;
    }
    if (C.blob_floats < (size_t)off) {           // grow the packed-parameter scratch (stream-ordered)
        if (C.blob) FP_CUDA_OK(ctx, cudaFreeAsync(C.blob, st));
        C.blob = nullptr; C.blob_floats = 0;
        FP_CUDA_OK(ctx, cudaMallocAsync((void**)&C.blob, (size_t)off * sizeof(float), st));
        C.blob_floats = (size_t)off;
    }
    fp_launch(mlp_pack_kernel, fp_div_up(off, 256) < 64 ? fp_div_up(off, 256) : 64, 256, 0, st, D, S, C.blob);
    FP_LAUNCH_OK(ctx);
    const int32_t ncell = ctx->ncell;
    const size_t wbytes = (size_t)((off + 3) & ~3) * sizeof(float);
    if (maxw <= 64) {
        constexpr int CB = 128;
        const size_t abytes = (size_t)2 * maxw * CB * sizeof(float);
        const int w_in_smem = (wbytes + abytes <= 200 * 1024) ? 1 : 0;
        const size_t smem = abytes + (w_in_smem ? wbytes : 0);
        FP_CUDA_OK(ctx, cudaFuncSetAttribute(mlp_kernel<CB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        fp_launch(mlp_kernel<CB>, fp_div_up(ncell, CB), CB, smem, st, mom, mom_stride, tau_cell, ctx->p.tau, C.blob, D, w_in_smem,
                                                             ctx->p.min_count_mlp, relax_w, ncell, coef, flags, cellc,
                                                             ctx->p.dt, ctx->p.eps2_scale);
    } else if (maxw <= 512) {
        constexpr int CB = 32;
        const size_t abytes = (size_t)2 * maxw * CB * sizeof(float);
        const int w_in_smem = (wbytes + abytes <= 200 * 1024) ? 1 : 0;
        const size_t smem = abytes + (w_in_smem ? wbytes : 0);
        FP_CUDA_OK(ctx, cudaFuncSetAttribute(mlp_kernel<CB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        fp_launch(mlp_kernel<CB>, fp_div_up(ncell, CB), CB, smem, st, mom, mom_stride, tau_cell, ctx->p.tau, C.blob, D, w_in_smem,
                                                             ctx->p.min_count_mlp, relax_w, ncell, coef, flags, cellc,
                                                             ctx->p.dt, ctx->p.eps2_scale);
    } else {
        return fp_fail(ctx, FP_ERR_UNSUPPORTED, "fp_closure_mlp: hidden width > 512 is not supported");
    }
    FP_LAUNCH_OK(ctx);
    FP_COUNT(ctx, 2);
    return FP_OK;
}
