// mlp_wide.cuh -- tensor-core path of the fused MLP surrogate for wide networks, in particular the paper's own
// 16-256-256-256-256-9 ReLU network (PAPER.md:309, 204,041 parameters; :264 predict_coeffs; :327 StandardScaler;
// :568 under-relaxation).  Included by closure_mlp.cu only.
//
// 0.27 Mflop per cell and 816 KB of fp32 weights: the weights cannot live in shared memory and the work is a dense
// contraction, so this one runs on the tensor cores.  A CTA (8 warps) owns a tile of 64 cells and walks it through
// all layers; the activations of the tile stay in shared memory (ping-pong), the weights stream from L2 in mma
// fragment order (coalesced 16-byte loads, prefetched one k-step ahead in registers), accumulators stay in
// registers (warp tile 32 cells x 64 units).
//   arithmetic: mma.sync.m16n8k16 bf16 inputs, fp32 accumulate, with the "3x" split that keeps fp32-level accuracy:
//   x = x_hi + x_lo (both bf16, 16 mantissa bits together), A.B ~= A_lo.B_hi + A_hi.B_lo + A_hi.B_hi.  A plain
//   bf16 (or TF32) product is outside north_star's 3e-3 on a four-layer network (mlp_tc.cuh measured 7e-3 for
//   TF32 on three layers); the split form measures ~1e-5 of the output scale.
//   layouts: activations are split once, when a layer's epilogue writes them, and stored as two bf16 arrays
//   xh/xl[64][H + 8] (row stride = 16 mod 128 bytes: ldmatrix.x4 rows and the epilogue's 4-byte stores are both
//   conflict free); one ldmatrix.x4 per m-tile, k-step and part delivers the A fragment as an aligned register
//   quad.  The weights are packed in fragment order, already split, one uint4 {b0_hi, b1_hi, b0_lo, b1_lo} per
//   (layer, k-step, n-tile, lane), by mlpw_pack_kernel.
// Features, standardisation, fallback policy, under-relaxation and the update constants are those of the fp32
// kernel (closure_mlp.cu).
#pragma once
#include <cuda_bf16.h>

#define WD_THREADS 256
#define WD_M 64                                   // cells per CTA tile
#define WD_H 256                                  // hidden width served by this kernel

struct wd_params {
    int32_t stride, feature_set, act, min_count, ncell, nin, n_layers;
    float tau_scalar, n_scale, theta_ref, relax_w;
    float dt, eps2_scale;
    float* cellc;
};

// fragments per layer (uint4 units): first layer K = 16 (1 k-step), hidden K = H, head N = 16 (2 n-tiles)
__host__ __device__ inline size_t wd_frag_first() { return (size_t)1 * (WD_H / 8) * 32; }
__host__ __device__ inline size_t wd_frag_hidden() { return (size_t)(WD_H / 16) * (WD_H / 8) * 32; }
__host__ __device__ inline size_t wd_frag_head() { return (size_t)(WD_H / 16) * 2 * 32; }
__host__ __device__ inline size_t wd_frag_total(int n_layers)
{
    return wd_frag_first() + (size_t)(n_layers - 2) * wd_frag_hidden() + wd_frag_head();
}
// misc floats: biases of layers 0..L-2 (H each), head bias (16), x_mean, x_scale, y_mean, y_scale (16 each)
__host__ __device__ inline int wd_misc_floats(int n_layers) { return (n_layers - 1) * WD_H + 16 + 64; }

__device__ __forceinline__ void wd_split2(float x0, float x1, uint32_t& hi, uint32_t& lo)
{
    const __nv_bfloat162 h = __floats2bfloat162_rn(x0, x1);               // .x (low half) = x0
    hi = *reinterpret_cast<const uint32_t*>(&h);
    const float f0 = __uint_as_float(hi << 16), f1 = __uint_as_float(hi & 0xffff0000u);
    const __nv_bfloat162 l = __floats2bfloat162_rn(x0 - f0, x1 - f1);
    lo = *reinterpret_cast<const uint32_t*>(&l);
}
__device__ __forceinline__ void wd_mma(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1)
{
    asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

__device__ __forceinline__ void wd_pack_misc(const mlp_src& S, int n_layers, int nin, float* __restrict__ misc, int tid, int nth)
{
    const int nm = wd_misc_floats(n_layers);
    for (int e = tid; e < nm; e += nth) {
        float v = 0.0f;
        if (e < (n_layers - 1) * WD_H) v = S.b[e / WD_H][e % WD_H];
        else if (e < (n_layers - 1) * WD_H + 16) { const int o = e - (n_layers - 1) * WD_H; v = (o < 9) ? S.b[n_layers - 1][o] : 0.0f; }
        else {
            const int q = (e - (n_layers - 1) * WD_H - 16) / 16, i = (e - (n_layers - 1) * WD_H - 16) % 16;
            if (q == 0) v = (i < nin) ? S.x_mean[i] : 0.0f;
            else if (q == 1) v = (i < nin) ? S.x_scale[i] : 1.0f;
            else if (q == 2) v = (i < 9) ? S.y_mean[i] : 0.0f;
            else v = (i < 9) ? S.y_scale[i] : 0.0f;
        }
        misc[e] = v;
    }
}

// Pack caller weights W[l] ([out][in] row-major) into split bf16 mma B fragments.  Fragment (l, j, n, lane):
// g = lane / 4, t = lane % 4, out = 8 n + g: b0 = inputs (16 j + 2 t, + 1), b1 = inputs (16 j + 2 t + 8, + 9).
__global__ void mlpw_pack_kernel(const __grid_constant__ mlp_src S, int32_t n_layers, int32_t nin,
                                 uint4* __restrict__ frags, float* __restrict__ misc)
{
    fpd_pdl();
    const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (size_t)gridDim.x * blockDim.x;
    const size_t total = wd_frag_total(n_layers);
    for (size_t e = tid; e < total; e += nth) {
        int l;
        size_t r = e;
        if (r < wd_frag_first()) l = 0;
        else {
            r -= wd_frag_first();
            const size_t hl = r / wd_frag_hidden();
            if ((int)hl < n_layers - 2) { l = 1 + (int)hl; r -= hl * wd_frag_hidden(); }
            else { l = n_layers - 1; r -= (size_t)(n_layers - 2) * wd_frag_hidden(); }
        }
        const int NT = (l == n_layers - 1) ? 2 : WD_H / 8;
        const int ni = (l == 0) ? nin : WD_H, no = (l == n_layers - 1) ? 9 : WD_H;
        const int lane = (int)(r & 31), n = (int)((r >> 5) % NT), j = (int)((r >> 5) / NT);
        const int g = lane >> 2, t = lane & 3;
        const int o = 8 * n + g, i0 = 16 * j + 2 * t;
        float w[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int i = i0 + (q & 1) + 8 * (q >> 1);
            w[q] = (o < no && i < ni) ? S.W[l][(size_t)o * ni + i] : 0.0f;
        }
        uint4 f;
        wd_split2(w[0], w[1], f.x, f.z);
        wd_split2(w[2], w[3], f.y, f.w);
        frags[e] = f;
    }
    wd_pack_misc(S, n_layers, nin, misc, (int)tid, (int)nth);
}

// biases and scalers alone (the tcgen05 kernel packs its weights differently, mlp_wide5.cuh)
__global__ void mlpw_misc_kernel(const __grid_constant__ mlp_src S, int32_t n_layers, int32_t nin, float* __restrict__ misc)
{
    fpd_pdl();
    wd_pack_misc(S, n_layers, nin, misc, (int)(blockIdx.x * blockDim.x + threadIdx.x), (int)(gridDim.x * blockDim.x));
}

#define WD_XS (WD_H + 8)                          // activation row stride in bf16 elements (528 bytes)

// A fragment (16 cells x 16 inputs) of the m-tile starting at row r0, k-step j: lane i supplies the address of row
// r0 + (i & 7) + 8 * ((i >> 3) & 1), inputs 16 j + 8 * (i >> 4)
__device__ __forceinline__ void wd_ldmatrix(uint32_t (&a)[4], const __nv_bfloat16* x, int r0, int j, int lane)
{
    const __nv_bfloat16* p = x + (size_t)(r0 + (lane & 7) + 8 * ((lane >> 3) & 1)) * WD_XS + 16 * j + 8 * (lane >> 4);
    const uint32_t addr = (uint32_t)__cvta_generic_to_shared(p);
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(a[0]), "=r"(a[1]), "=r"(a[2]), "=r"(a[3]) : "r"(addr) : "memory");
}

// One dense layer of width H on the CTA's 64-cell tile: warp (wm, wn) computes cells 32 wm .. +31, units 64 wn ..
// +63 (2 m-tiles x 8 n-tiles), KS k-steps of 16 inputs; bias, activation, split and store into the other buffer.
template <int KS>
__device__ __forceinline__ void wd_layer(const __nv_bfloat16* __restrict__ xh, const __nv_bfloat16* __restrict__ xl,
                                         __nv_bfloat16* __restrict__ yh, __nv_bfloat16* __restrict__ yl,
                                         const uint4* __restrict__ wf, const float* __restrict__ bias, int act,
                                         int wm, int wn, int lane)
{
    constexpr int NT = WD_H / 8;
    const int g = lane >> 2, t = lane & 3;
    float acc[2][8][4];
#pragma unroll
    for (int n = 0; n < 8; ++n) {
        const float b0 = bias[64 * wn + 8 * n + 2 * t], b1 = bias[64 * wn + 8 * n + 2 * t + 1];
#pragma unroll
        for (int mt = 0; mt < 2; ++mt) { acc[mt][n][0] = b0; acc[mt][n][1] = b1; acc[mt][n][2] = b0; acc[mt][n][3] = b1; }
    }
    const uint4* wp = wf + (size_t)(8 * wn) * 32 + lane;                 // + (j * NT + n) * 32
    const int row0 = 32 * wm + g;
    auto load_w = [&](uint4 (&w)[8], int j) {
#pragma unroll
        for (int n = 0; n < 8; ++n) w[n] = __ldg(wp + ((size_t)j * NT + n) * 32);
    };
    auto kstep = [&](const uint4 (&w)[8], int j) {
        uint32_t ahi[2][4], alo[2][4];
#pragma unroll
        for (int mt = 0; mt < 2; ++mt) {
            wd_ldmatrix(ahi[mt], xh, 32 * wm + 16 * mt, j, lane);
            wd_ldmatrix(alo[mt], xl, 32 * wm + 16 * mt, j, lane);
        }
        // three sweeps over the 16 independent accumulator tiles (small terms first), so that consecutive mma
        // instructions never depend on one another
#pragma unroll
        for (int n = 0; n < 8; ++n)
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) wd_mma(acc[mt][n], alo[mt], w[n].x, w[n].y);
#pragma unroll
        for (int n = 0; n < 8; ++n)
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) wd_mma(acc[mt][n], ahi[mt], w[n].z, w[n].w);
#pragma unroll
        for (int n = 0; n < 8; ++n)
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) wd_mma(acc[mt][n], ahi[mt], w[n].x, w[n].y);
    };
    // weights of the next k-step are in flight while this one is multiplied: two register buffers, no copies
    uint4 w0[8], w1[8];
    load_w(w0, 0);
#pragma unroll
    for (int j = 0; j < KS; j += 2) {
        if (j + 1 < KS) load_w(w1, j + 1);
        kstep(w0, j);
        if (j + 2 < KS) load_w(w0, j + 2);
        if (j + 1 < KS) kstep(w1, j + 1);
    }
    // epilogue: activation, split, store (c0, c1) -> row g, (c2, c3) -> row g + 8, columns 8n + 2t, +1
#pragma unroll
    for (int mt = 0; mt < 2; ++mt) {
        const int r = row0 + 16 * mt;
#pragma unroll
        for (int n = 0; n < 8; ++n) {
            float v[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const float s = acc[mt][n][q];
                v[q] = (act == 0) ? __fdividef(s, 1.0f + __expf(-s)) : fmaxf(s, 0.0f);
            }
            const int col = 64 * wn + 8 * n + 2 * t;
            uint32_t h, l;
            wd_split2(v[0], v[1], h, l);
            *reinterpret_cast<uint32_t*>(yh + (size_t)r * WD_XS + col) = h;
            *reinterpret_cast<uint32_t*>(yl + (size_t)r * WD_XS + col) = l;
            wd_split2(v[2], v[3], h, l);
            *reinterpret_cast<uint32_t*>(yh + (size_t)(r + 8) * WD_XS + col) = h;
            *reinterpret_cast<uint32_t*>(yl + (size_t)(r + 8) * WD_XS + col) = l;
        }
    }
}

__global__ void __launch_bounds__(WD_THREADS, 1)
mlp_wide_kernel(const double* __restrict__ mom, const float* __restrict__ tau_cell, const uint4* __restrict__ frags,
                const float* __restrict__ misc, float* __restrict__ coef, uint32_t* __restrict__ flags,
                const __grid_constant__ wd_params P)
{
    fpd_pdl();
    extern __shared__ __align__(16) unsigned char wd_smem[];
    constexpr size_t XB = (size_t)WD_M * WD_XS;                           // bf16 elements per activation array
    __nv_bfloat16* xh0 = reinterpret_cast<__nv_bfloat16*>(wd_smem);
    __nv_bfloat16* xl0 = xh0 + XB;
    __nv_bfloat16* xh1 = xl0 + XB;
    __nv_bfloat16* xl1 = xh1 + XB;
    float* ms = reinterpret_cast<float*>(xl1 + XB);                       // [wd_misc_floats]
    const int nmisc = wd_misc_floats(P.n_layers);
    float* yout = ms + ((nmisc + 3) & ~3);                                // [64][17] head outputs
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int g = lane >> 2, t = lane & 3, wm = warp >> 2, wn = warp & 3;
    for (int i = tid; i < nmisc; i += WD_THREADS) ms[i] = misc[i];
    __syncthreads();
    const int L = P.n_layers;
    const float* hbias = ms + (L - 1) * WD_H;
    const float* xmean = hbias + 16, *xscale = xmean + 16, *ymean = xscale + 16, *yscale = ymean + 16;
    const uint4* f_hidden = frags + wd_frag_first();
    const uint4* f_head = f_hidden + (size_t)(L - 2) * wd_frag_hidden();
    const int ntiles = (P.ncell + WD_M - 1) / WD_M;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int cell0 = tile * WD_M;
        // ---- features of cell cell0 + tid (threads 0..63), standardised, split, into buffer 0 columns 0..15
        double nraw = 0.0, theta = 0.0;
        float tau = P.tau_scalar;
        bool zbad = false;
        const int cell = cell0 + tid;
        const bool have = tid < WD_M && cell < P.ncell;
        if (tid < WD_M) {
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
            float z[16];
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                z[i] = (i < P.nin) ? (x[i] - xmean[i]) / xscale[i] : 0.0f;
                if (have && !isfinite(z[i])) zbad = true;
                if (!have || !isfinite(z[i])) z[i] = 0.0f;
            }
#pragma unroll
            for (int i = 0; i < 16; i += 2) {
                uint32_t h, l;
                wd_split2(z[i], z[i + 1], h, l);
                *reinterpret_cast<uint32_t*>(xh0 + (size_t)tid * WD_XS + i) = h;
                *reinterpret_cast<uint32_t*>(xl0 + (size_t)tid * WD_XS + i) = l;
            }
        }
        __syncthreads();
        // ---- layer 0 (K = 16), hidden layers (K = H): buffers alternate
        wd_layer<1>(xh0, xl0, xh1, xl1, frags, ms, P.act, wm, wn, lane);
        __syncthreads();
        int cur = 1;
        for (int l = 1; l < L - 1; ++l) {
            const uint4* wf = f_hidden + (size_t)(l - 1) * wd_frag_hidden();
            if (cur) wd_layer<WD_H / 16>(xh1, xl1, xh0, xl0, wf, ms + l * WD_H, P.act, wm, wn, lane);
            else     wd_layer<WD_H / 16>(xh0, xl0, xh1, xl1, wf, ms + l * WD_H, P.act, wm, wn, lane);
            __syncthreads();
            cur ^= 1;
        }
        // ---- head (N = 16): warp w owns m-tile w & 3, n-tile w >> 2
        {
            const __nv_bfloat16* xh = cur ? xh1 : xh0;
            const __nv_bfloat16* xl = cur ? xl1 : xl0;
            const int mt = warp & 3, nt = warp >> 2;
            float c[4];
            c[0] = c[2] = hbias[8 * nt + 2 * t];
            c[1] = c[3] = hbias[8 * nt + 2 * t + 1];
            const int r = 16 * mt + g;
#pragma unroll 4
            for (int j = 0; j < WD_H / 16; ++j) {
                const uint4 w = __ldg(f_head + ((size_t)j * 2 + nt) * 32 + lane);
                uint32_t ahi[4], alo[4];
                wd_ldmatrix(ahi, xh, 16 * mt, j, lane);
                wd_ldmatrix(alo, xl, 16 * mt, j, lane);
                wd_mma(c, alo, w.x, w.y);
                wd_mma(c, ahi, w.z, w.w);
                wd_mma(c, ahi, w.x, w.y);
            }
            yout[r * 17 + 8 * nt + 2 * t] = c[0]; yout[r * 17 + 8 * nt + 2 * t + 1] = c[1];
            yout[(r + 8) * 17 + 8 * nt + 2 * t] = c[2]; yout[(r + 8) * 17 + 8 * nt + 2 * t + 1] = c[3];
        }
        __syncthreads();
        // ---- de-standardise, policy, blend: thread tid < 64 owns cell cell0 + tid
        if (have) {
            float y[9];
            bool finite = !zbad;
#pragma unroll
            for (int k = 0; k < 9; ++k) {
                y[k] = fmaf(yout[tid * 17 + k], yscale[k], ymean[k]);
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
        __syncthreads();                                  // yout and the activation buffers are reused by the next tile
    }
}
