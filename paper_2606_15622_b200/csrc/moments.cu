// moments.cu -- a3: segmented gather of per-cell velocity moments over cell-sorted particles
// (PAPER.md:124 moment definition, :215-216 M1-M5, :243 LITE, :181 plain 1/N mean; R0).
//
// HBM-bound by design: 12 B/particle read once + one record per cell written.
// A group of G lanes (G = 4/8/16/32 by mean particles per cell, tiles.cuh) owns one cell, so a warp works on 32/G consecutive cells
// at once.  Each warp stages the contiguous vx, vy, vz slices of its cells in its own shared-memory buffer with three
// 1D bulk asynchronous copies (tiles.cuh) -- HBM is read once, coalesced, with no block-wide barrier and no
// dependence between warps -- and both passes over a cell read shared memory:
//   pass 1: S = sum (v - v_pivot) in fp32 about the cell's first particle (differences are thermal-sized, so fp32
//           holds them to ~6e-8 of the thermal speed even at Mach 10), reduced across the group in fp64;
//           U = v_pivot + S/N (fp64), m = S/N.
//   pass 2: c = (v - v_pivot) - m in fp32, monomials and per-lane partial sums in fp32 (<= 64 terms per lane and
//           chunk), combined across the group by a balanced fp32 tree (a transposing butterfly that leaves record
//           slot k in the lane that stores it); chunks, the mean and the 1/N normalisation are fp64.
// A chunk whose cells do not fit the warp's staging buffer (load-imbalanced grids) is walked cell by cell, each cell
// staged on its own and reduced by all 32 lanes; a cell that alone exceeds the buffer, and unaligned arrays, take
// mom_giant_cell: the same two passes over shared-memory slices filled by plain coalesced loads, slices combined in
// fp64.
#include "tiles.cuh"

#ifndef MOM_THREADS
#define MOM_THREADS 128
#endif
#define MOM_WARPS (MOM_THREADS / 32)
#define MOM_CHUNK_PER_LANE 64
#ifndef MOM_CAP
#define MOM_CAP FPW_CAP            // staged elements per array, warp and stage
#endif

// One cell per group of G lanes.  bx/by/bz: the warp's private staging copy in shared memory, particle p at b?[p];
// pass 1 overwrites v by v - v_pivot.
struct mom_no_hook { __device__ __forceinline__ void operator()() const {} };

template <int G, bool FULL, class Hook = mom_no_hook>
__device__ __forceinline__ void mom_cell_group(const float* bx, const float* by, const float* bz, int32_t s, int32_t n,
                                               bool have, int gl, double* __restrict__ rec, Hook after_reads = Hook())
{
    float* wx = const_cast<float*>(bx);
    float* wy = const_cast<float*>(by);
    float* wz = const_cast<float*>(bz);
    constexpr int NP = (FULL || G > 16) ? 32 : 16;   // padded record length (at least one slot per lane)
    constexpr int NREC = FULL ? 29 : 13;
    constexpr int PER = NP / G;                 // record slots per lane after the transposing reduction
    static_assert(NP >= G, "group wider than the padded record");
    // ---- pass 1: mean about the pivot
    float px = 0.f, py = 0.f, pz = 0.f;
    if (n > 0) { px = bx[s]; py = by[s]; pz = bz[s]; }
    const float2 npx = fpd_dup(-px), npy = fpd_dup(-py), npz = fpd_dup(-pz);
    const int32_t nmax = __reduce_max_sync(0xffffffffu, n);
    double S0 = 0.0, S1 = 0.0, S2 = 0.0;
    for (int32_t c0 = 0; c0 < nmax; c0 += G * MOM_CHUNK_PER_LANE) {
        float2 A0 = fpd_dup(0.f), A1 = fpd_dup(0.f), A2 = fpd_dup(0.f);      // two particles per lane and step
        const int32_t cend = min(n, c0 + G * MOM_CHUNK_PER_LANE);
        int32_t j = c0 + gl;
#pragma unroll 2
        for (; j + G < cend; j += 2 * G) {
            const float2 w0 = fpd_add2(make_float2(bx[s + j], bx[s + j + G]), npx);
            const float2 w1 = fpd_add2(make_float2(by[s + j], by[s + j + G]), npy);
            const float2 w2 = fpd_add2(make_float2(bz[s + j], bz[s + j + G]), npz);
            A0 = fpd_add2(A0, w0); A1 = fpd_add2(A1, w1); A2 = fpd_add2(A2, w2);
            // park w = v - v_pivot for pass 2 (store pipe is idle, the FMA pipe is the bottleneck)
            wx[s + j] = w0.x; wx[s + j + G] = w0.y; wy[s + j] = w1.x; wy[s + j + G] = w1.y;
            wz[s + j] = w2.x; wz[s + j + G] = w2.y;
        }
        if (j < cend) {
            const float w0 = bx[s + j] - px, w1 = by[s + j] - py, w2 = bz[s + j] - pz;
            A0.x += w0; A1.x += w1; A2.x += w2;
            wx[s + j] = w0; wy[s + j] = w1; wz[s + j] = w2;
        }
        const float a0 = A0.x + A0.y, a1 = A1.x + A1.y, a2 = A2.x + A2.y;
        S0 += (double)a0; S1 += (double)a1; S2 += (double)a2;
    }
#pragma unroll
    for (int d = G / 2; d >= 1; d >>= 1) {
        S0 += fpd_shfl_xor(S0, d); S1 += fpd_shfl_xor(S1, d); S2 += fpd_shfl_xor(S2, d);
    }
    const double invn = n > 0 ? 1.0 / (double)n : 0.0;
    const double m0d = S0 * invn, m1d = S1 * invn, m2d = S2 * invn;
    const float m0 = (float)m0d, m1 = (float)m1d, m2 = (float)m2d;
    const float2 nm0 = fpd_dup(-m0), nm1 = fpd_dup(-m1), nm2 = fpd_dup(-m2);
    // ---- pass 2: central moments
    double tot[PER];
#pragma unroll
    for (int i = 0; i < PER; ++i) tot[i] = 0.0;
    for (int32_t c0 = 0; c0 < nmax; c0 += G * MOM_CHUNK_PER_LANE) {
        // packed accumulators: .x and .y hold the partial sums of the two particles a lane handles per step
        float2 P[6], T[10], F[6], Gm[3];
#pragma unroll
        for (int k = 0; k < 6; ++k) { P[k] = fpd_dup(0.f); F[k] = fpd_dup(0.f); }
#pragma unroll
        for (int k = 0; k < 10; ++k) T[k] = fpd_dup(0.f);
#pragma unroll
        for (int k = 0; k < 3; ++k) Gm[k] = fpd_dup(0.f);
        const int32_t cend = min(n, c0 + G * MOM_CHUNK_PER_LANE);
        int32_t j = c0 + gl;
        const int32_t jlast = j + ((cend - j + G - 1) / G) * G;          // first index this lane does not own
#pragma unroll 1
        for (; j < jlast; j += 2 * G) {
            const bool two = j + G < cend;
            const int32_t jb = two ? j + G : j;                            // lone last particle: second half masked
            float2 cx, cy, cz;
            cx = fpd_add2(make_float2(bx[s + j], bx[s + jb]), nm0);
            cy = fpd_add2(make_float2(by[s + j], by[s + jb]), nm1);
            cz = fpd_add2(make_float2(bz[s + j], bz[s + jb]), nm2);
            if (!two) { cx.y = 0.f; cy.y = 0.f; cz.y = 0.f; }
            const float2 xx = fpd_mul2(cx, cx), xy = fpd_mul2(cx, cy), xz = fpd_mul2(cx, cz);
            const float2 yy = fpd_mul2(cy, cy), yz = fpd_mul2(cy, cz), zz = fpd_mul2(cz, cz);
            const float2 c2 = fpd_add2(fpd_add2(xx, yy), zz);
            P[0] = fpd_add2(P[0], xx); P[1] = fpd_add2(P[1], xy); P[2] = fpd_add2(P[2], xz);
            P[3] = fpd_add2(P[3], yy); P[4] = fpd_add2(P[4], yz); P[5] = fpd_add2(P[5], zz);
            if (FULL) {
                T[0] = fpd_fma2(xx, cx, T[0]); T[1] = fpd_fma2(xx, cy, T[1]); T[2] = fpd_fma2(xx, cz, T[2]);
                T[3] = fpd_fma2(xy, cy, T[3]); T[4] = fpd_fma2(xy, cz, T[4]); T[5] = fpd_fma2(xz, cz, T[5]);
                T[6] = fpd_fma2(yy, cy, T[6]); T[7] = fpd_fma2(yy, cz, T[7]); T[8] = fpd_fma2(yz, cz, T[8]);
                T[9] = fpd_fma2(zz, cz, T[9]);
                F[0] = fpd_fma2(c2, xx, F[0]); F[1] = fpd_fma2(c2, xy, F[1]); F[2] = fpd_fma2(c2, xz, F[2]);
                F[3] = fpd_fma2(c2, yy, F[3]); F[4] = fpd_fma2(c2, yz, F[4]); F[5] = fpd_fma2(c2, zz, F[5]);
                const float2 c4 = fpd_mul2(c2, c2);
                Gm[0] = fpd_fma2(c4, cx, Gm[0]); Gm[1] = fpd_fma2(c4, cy, Gm[1]); Gm[2] = fpd_fma2(c4, cz, Gm[2]);
            } else {
                Gm[0] = fpd_fma2(c2, cx, Gm[0]); Gm[1] = fpd_fma2(c2, cy, Gm[1]); Gm[2] = fpd_fma2(c2, cz, Gm[2]);   // h_i
            }
        }
        if (c0 + G * MOM_CHUNK_PER_LANE >= nmax) after_reads();     // the staging buffer is not read again
        const float P0 = P[0].x + P[0].y, P1 = P[1].x + P[1].y, P2 = P[2].x + P[2].y, P3 = P[3].x + P[3].y,
                    P4 = P[4].x + P[4].y, P5 = P[5].x + P[5].y;
        const float t0 = T[0].x + T[0].y, t1 = T[1].x + T[1].y, t2 = T[2].x + T[2].y, t3 = T[3].x + T[3].y,
                    t4 = T[4].x + T[4].y, t5 = T[5].x + T[5].y, t6 = T[6].x + T[6].y, t7 = T[7].x + T[7].y,
                    t8 = T[8].x + T[8].y, t9 = T[9].x + T[9].y;
        const float F0 = F[0].x + F[0].y, F1 = F[1].x + F[1].y, F2 = F[2].x + F[2].y, F3 = F[3].x + F[3].y,
                    F4 = F[4].x + F[4].y, F5 = F[5].x + F[5].y;
        const float g0 = Gm[0].x + Gm[0].y, g1 = Gm[1].x + Gm[1].y, g2 = Gm[2].x + Gm[2].y;
        float r[NP];
        r[0] = r[1] = r[2] = r[3] = 0.f;
        r[4] = P0; r[5] = P1; r[6] = P2; r[7] = P3; r[8] = P4; r[9] = P5;
        if (FULL) {
            r[10] = t0; r[11] = t1; r[12] = t2; r[13] = t3; r[14] = t4; r[15] = t5; r[16] = t6; r[17] = t7; r[18] = t8;
            r[19] = t9; r[20] = F0; r[21] = F1; r[22] = F2; r[23] = F3; r[24] = F4; r[25] = F5; r[26] = g0; r[27] = g1;
            r[28] = g2;
#pragma unroll
            for (int k = 29; k < NP; ++k) r[k] = 0.f;
        } else {
            r[10] = g0; r[11] = g1; r[12] = g2;
#pragma unroll
            for (int k = 13; k < NP; ++k) r[k] = 0.f;
        }
        fpd_transpose_reduce<NP, G, float>(r, gl);       // balanced fp32 tree over the group's partial sums
#pragma unroll
        for (int i = 0; i < PER; ++i) tot[i] += (double)r[i];
    }
    // lane gl holds record slots PER*gl .. PER*gl + PER - 1
    if (have) {
#pragma unroll
        for (int i = 0; i < PER; ++i) {
            const int slot = PER * gl + i;
            double val = tot[i] * invn;
            if (slot == 0) val = (double)n;
            else if (slot == 1) val = n > 0 ? (double)px + m0d : 0.0;
            else if (slot == 2) val = n > 0 ? (double)py + m1d : 0.0;
            else if (slot == 3) val = n > 0 ? (double)pz + m2d : 0.0;
            if (slot < NREC) rec[slot] = val;
        }
    }
}

// Cross-lane sums of the group's partial records through shared memory: every lane stores its NP partial sums as one row
// (row stride NP + 4 floats: 128-bit stores, and the reads below, hit the minimal number of bank wavefronts for G >= 8),
// lane gl then adds up slots PER*gl .. PER*gl + PER - 1 over the G rows of its group in a balanced tree and leaves them in
// r[0 .. PER).  45 instructions per lane for a FULL record and G = 8, against 112 for the transposing shuffle tree
// (28 SHFL + 56 FSEL + 28 FADD), and one shared-memory round trip instead of three dependent shuffle stages.
// `scratch`: 32 * (NP + 4) floats, 16-byte aligned, that no lane of the warp reads for anything else any more.
#ifndef MOM_SMEM_TREE
#define MOM_SMEM_TREE 1
#endif
template <int NP, int G>
__device__ __forceinline__ void mom_group_reduce_smem(float (&r)[NP], float* scratch, int lane, int gl, int group)
{
    constexpr int PER = NP / G, ROW = NP + 4;
    __syncwarp();                                            // the other groups are done with the staged particles too
    float4* mine = reinterpret_cast<float4*>(scratch + lane * ROW);
#pragma unroll
    for (int q = 0; q < NP / 4; ++q) mine[q] = make_float4(r[4 * q], r[4 * q + 1], r[4 * q + 2], r[4 * q + 3]);
    __syncwarp();
    const float* col = scratch + (group * G) * ROW + PER * gl;
    float a[G][PER];
#pragma unroll
    for (int j = 0; j < G; ++j) {
        if constexpr (PER % 4 == 0) {
#pragma unroll
            for (int q = 0; q < PER / 4; ++q) {
                const float4 v = reinterpret_cast<const float4*>(col + j * ROW)[q];
                a[j][4 * q] = v.x; a[j][4 * q + 1] = v.y; a[j][4 * q + 2] = v.z; a[j][4 * q + 3] = v.w;
            }
        } else if constexpr (PER == 2) {
            const float2 v = *reinterpret_cast<const float2*>(col + j * ROW);
            a[j][0] = v.x; a[j][1] = v.y;
        } else {
            a[j][0] = col[j * ROW];
        }
    }
#pragma unroll
    for (int h = G / 2; h >= 1; h >>= 1) {
#pragma unroll
        for (int j = 0; j < h; ++j) {
#pragma unroll
            for (int i = 0; i < PER; ++i) a[j][i] += a[j + h][i];
        }
    }
#pragma unroll
    for (int i = 0; i < PER; ++i) r[i] = a[0][i];
}

// The common case, cells of at most 128*G particles: same two passes, but (i) the particles of a cell are visited in
// rotated order, starting at the particle whose shared-memory bank is G*group, so that the 32 lanes of a warp hit 32
// different banks in every load whatever the cell boundaries are (the lanes of a group step through the cell
// 2G particles at a time; only the part after the wrap-around can conflict); (ii) nothing is parked: pass 2 forms
// (v - v_pivot) - m again; (iii) per-lane sums stay fp32 for the whole cell (<= 64 terms per packed half, as in the
// chunked path) and go straight to the cross-lane tree.  `after_reads` runs once the staging buffer is not needed
// any more.  Lanes of different groups run different trip counts; the (masked) last step is peeled.
#ifndef MOM_F32MEAN
#define MOM_F32MEAN 0                   // 1: mean by an fp32 tree (2 % fewer instructions, but U then uses 0.8 of its 1e-6 tolerance)
#endif
template <int G, bool FULL, class Hook>
__device__ __forceinline__ void mom_cell_rot(const float* bx, const float* by, const float* bz, int32_t s, int32_t n,
                                             bool have, int gl, int group, double* __restrict__ rec, bool norot,
                                             float* scratch, Hook after_reads)
{
    constexpr int NP = (FULL || G > 16) ? 32 : 16;
    constexpr int NREC = FULL ? 29 : 13;
    constexpr int PER = NP / G;
    const float* x = bx + s;
    const float* y = by + s;
    const float* z = bz + s;
    float px = 0.f, py = 0.f, pz = 0.f;
    if (n > 0) { px = x[0]; py = y[0]; pz = z[0]; }
    const float2 npx = fpd_dup(-px), npy = fpd_dup(-py), npz = fpd_dup(-pz);
    // rotation: particle o of the cell sits in bank G*group
    int32_t o = norot ? 0 : (int32_t)((uint32_t)(G * group) - (fpt_smem_u32(x) >> 2)) & 31;
    while (n > 0 && o >= n) o -= n;
    if (n <= 0) o = 0;
    const int32_t full = n / (2 * G);                       // steps in which all 2G particles exist
    const int32_t t0 = 2 * G * full + gl, t1 = t0 + G;      // the peeled last step
    const bool v0 = t0 < n, v1 = t1 < n;
    int32_t q0 = o + t0, q1 = o + t1;
    if (q0 >= n) q0 -= n;
    if (q1 >= n) q1 -= n;
    if (!v0) q0 = 0;
    if (!v1) q1 = 0;
    const float2 msk = make_float2(v0 ? 1.f : 0.f, v1 ? 1.f : 0.f);
    int32_t j0s = o + gl, j1s = o + gl + G;
    if (j0s >= n) j0s -= n;
    if (j1s >= n) j1s -= n;
    // ---- pass 1: mean about the pivot
    float2 A0 = fpd_dup(0.f), A1 = fpd_dup(0.f), A2 = fpd_dup(0.f);
    {
        int32_t j0 = j0s, j1 = j1s;
#pragma unroll 2
        for (int32_t k = 0; k < full; ++k) {
            A0 = fpd_add2(A0, fpd_add2(make_float2(x[j0], x[j1]), npx));
            A1 = fpd_add2(A1, fpd_add2(make_float2(y[j0], y[j1]), npy));
            A2 = fpd_add2(A2, fpd_add2(make_float2(z[j0], z[j1]), npz));
            j0 += 2 * G; j1 += 2 * G;
            if (j0 >= n) j0 -= n;
            if (j1 >= n) j1 -= n;
        }
        A0 = fpd_fma2(fpd_add2(make_float2(x[q0], x[q1]), npx), msk, A0);
        A1 = fpd_fma2(fpd_add2(make_float2(y[q0], y[q1]), npy), msk, A1);
        A2 = fpd_fma2(fpd_add2(make_float2(z[q0], z[q1]), npz), msk, A2);
    }
#if MOM_F32MEAN
    // the mean in fp32: <= 64 thermal-sized terms per packed half, a balanced tree over the lanes, n < 2^24 exact and its
    // reciprocal correctly rounded: ~1e-7 of the thermal speed on U, far below that on the central moments
    float S0 = A0.x + A0.y, S1 = A1.x + A1.y, S2 = A2.x + A2.y;
#pragma unroll
    for (int d = G / 2; d >= 1; d >>= 1) {
        S0 += __shfl_xor_sync(0xffffffffu, S0, d); S1 += __shfl_xor_sync(0xffffffffu, S1, d);
        S2 += __shfl_xor_sync(0xffffffffu, S2, d);
    }
    const float invnf = n > 0 ? __frcp_rn((float)n) : 0.0f;
    const float m0f = S0 * invnf, m1f = S1 * invnf, m2f = S2 * invnf;
    const double invn = (double)invnf, m0d = (double)m0f, m1d = (double)m1f, m2d = (double)m2f;
    const float2 nm0 = fpd_dup(-m0f), nm1 = fpd_dup(-m1f), nm2 = fpd_dup(-m2f);
#else
    double S0 = (double)A0.x + (double)A0.y, S1 = (double)A1.x + (double)A1.y, S2 = (double)A2.x + (double)A2.y;
#pragma unroll
    for (int d = G / 2; d >= 1; d >>= 1) {
        S0 += fpd_shfl_xor(S0, d); S1 += fpd_shfl_xor(S1, d); S2 += fpd_shfl_xor(S2, d);
    }
    const double invn = n > 0 ? 1.0 / (double)n : 0.0;
    const double m0d = S0 * invn, m1d = S1 * invn, m2d = S2 * invn;
    const float2 nm0 = fpd_dup(-(float)m0d), nm1 = fpd_dup(-(float)m1d), nm2 = fpd_dup(-(float)m2d);
#endif
    // ---- pass 2: central moments
    float2 P[6], T[10], F[6], Gm[3];
#pragma unroll
    for (int k = 0; k < 6; ++k) { P[k] = fpd_dup(0.f); F[k] = fpd_dup(0.f); }
#pragma unroll
    for (int k = 0; k < 10; ++k) T[k] = fpd_dup(0.f);
#pragma unroll
    for (int k = 0; k < 3; ++k) Gm[k] = fpd_dup(0.f);
    auto accumulate = [&](const float2 cx, const float2 cy, const float2 cz) {
        const float2 xx = fpd_mul2(cx, cx), xy = fpd_mul2(cx, cy), xz = fpd_mul2(cx, cz);
        const float2 yy = fpd_mul2(cy, cy), yz = fpd_mul2(cy, cz), zz = fpd_mul2(cz, cz);
        const float2 c2 = fpd_add2(fpd_add2(xx, yy), zz);
        P[0] = fpd_add2(P[0], xx); P[1] = fpd_add2(P[1], xy); P[2] = fpd_add2(P[2], xz);
        P[3] = fpd_add2(P[3], yy); P[4] = fpd_add2(P[4], yz); P[5] = fpd_add2(P[5], zz);
        if (FULL) {
            T[0] = fpd_fma2(xx, cx, T[0]); T[1] = fpd_fma2(xx, cy, T[1]); T[2] = fpd_fma2(xx, cz, T[2]);
            T[3] = fpd_fma2(xy, cy, T[3]); T[4] = fpd_fma2(xy, cz, T[4]); T[5] = fpd_fma2(xz, cz, T[5]);
            T[6] = fpd_fma2(yy, cy, T[6]); T[7] = fpd_fma2(yy, cz, T[7]); T[8] = fpd_fma2(yz, cz, T[8]);
            T[9] = fpd_fma2(zz, cz, T[9]);
            F[0] = fpd_fma2(c2, xx, F[0]); F[1] = fpd_fma2(c2, xy, F[1]); F[2] = fpd_fma2(c2, xz, F[2]);
            F[3] = fpd_fma2(c2, yy, F[3]); F[4] = fpd_fma2(c2, yz, F[4]); F[5] = fpd_fma2(c2, zz, F[5]);
            const float2 c4 = fpd_mul2(c2, c2);
            Gm[0] = fpd_fma2(c4, cx, Gm[0]); Gm[1] = fpd_fma2(c4, cy, Gm[1]); Gm[2] = fpd_fma2(c4, cz, Gm[2]);
        } else {
            Gm[0] = fpd_fma2(c2, cx, Gm[0]); Gm[1] = fpd_fma2(c2, cy, Gm[1]); Gm[2] = fpd_fma2(c2, cz, Gm[2]);   // h_i
        }
    };
    {
        int32_t j0 = j0s, j1 = j1s;
#pragma unroll 1
        for (int32_t k = 0; k < full; ++k) {
            const float2 cx = fpd_add2(fpd_add2(make_float2(x[j0], x[j1]), npx), nm0);
            const float2 cy = fpd_add2(fpd_add2(make_float2(y[j0], y[j1]), npy), nm1);
            const float2 cz = fpd_add2(fpd_add2(make_float2(z[j0], z[j1]), npz), nm2);
            j0 += 2 * G; j1 += 2 * G;
            if (j0 >= n) j0 -= n;
            if (j1 >= n) j1 -= n;
            accumulate(cx, cy, cz);
        }
        const float2 cx = fpd_mul2(fpd_add2(fpd_add2(make_float2(x[q0], x[q1]), npx), nm0), msk);
        const float2 cy = fpd_mul2(fpd_add2(fpd_add2(make_float2(y[q0], y[q1]), npy), nm1), msk);
        const float2 cz = fpd_mul2(fpd_add2(fpd_add2(make_float2(z[q0], z[q1]), npz), nm2), msk);
        accumulate(cx, cy, cz);
    }
    after_reads();                                           // the staging buffer is not read again
    float r[NP];
    r[0] = r[1] = r[2] = r[3] = 0.f;
#pragma unroll
    for (int k = 0; k < 6; ++k) r[4 + k] = P[k].x + P[k].y;
    if (FULL) {
#pragma unroll
        for (int k = 0; k < 10; ++k) r[10 + k] = T[k].x + T[k].y;
#pragma unroll
        for (int k = 0; k < 6; ++k) r[20 + k] = F[k].x + F[k].y;
#pragma unroll
        for (int k = 0; k < 3; ++k) r[26 + k] = Gm[k].x + Gm[k].y;
#pragma unroll
        for (int k = 29; k < NP; ++k) r[k] = 0.f;
    } else {
#pragma unroll
        for (int k = 0; k < 3; ++k) r[10 + k] = Gm[k].x + Gm[k].y;
#pragma unroll
        for (int k = 13; k < NP; ++k) r[k] = 0.f;
    }
    // balanced fp32 tree over the group's partial sums (scratch: the chunk's own staging buffer, free once every lane
    // has read its last particle; the next bulk copy into it is issued behind a proxy fence).  FULL records only: with
    // the 13-slot record the shuffle tree is as fast (17.5 vs 17.7 us)
    if (MOM_SMEM_TREE && FULL && scratch) mom_group_reduce_smem<NP, G>(r, scratch, gl + G * group, gl, group);
    else fpd_transpose_reduce<NP, G, float>(r, gl);
    // lane gl holds record slots PER*gl .. PER*gl + PER - 1
    if (have) {
#pragma unroll
        for (int i = 0; i < PER; ++i) {
            const int slot = PER * gl + i;
            double val = (double)r[i] * invn;
            if (i < 4) {                                     // slots 0..3 (N, U) can only sit at i < 4
                if (slot == 0) val = (double)n;
                else if (slot == 1) val = n > 0 ? (double)px + m0d : 0.0;
                else if (slot == 2) val = n > 0 ? (double)py + m1d : 0.0;
                else if (slot == 3) val = n > 0 ? (double)pz + m2d : 0.0;
            }
            if (slot < NREC) rec[slot] = val;
        }
    }
}

// A cell that alone exceeds the staging buffer (or unaligned arrays), all 32 lanes: both passes run over slices of the
// cell copied to shared memory with plain coalesced loads (16 independent loads per lane and array in flight; any
// alignment).  Per slice a lane adds at most MOM_CAP / 32 terms in fp32; slices are combined in fp64 (pass 1 per
// lane, pass 2 after the transposing tree, lane i owning record slot i).  Twice the algorithmic traffic, no
// per-iteration latency chain.
template <bool FULL>
__device__ __noinline__ void mom_giant_cell(const float* __restrict__ vx, const float* __restrict__ vy,
                                            const float* __restrict__ vz, int32_t s, int32_t n, float* sx, int lane,
                                            double* __restrict__ rec)
{
    constexpr int NREC = FULL ? 29 : 13;
    float* sy = sx + MOM_CAP;
    float* sz = sy + MOM_CAP;
    const float px = vx[s], py = vy[s], pz = vz[s];                      // pivot: the cell's first particle
    double S0 = 0.0, S1 = 0.0, S2 = 0.0;
#pragma unroll 1
    for (int32_t off = 0; off < n; off += MOM_CAP) {
        const int32_t len = min((int32_t)MOM_CAP, n - off), b0 = s + off;
        float a0 = 0.f, a1 = 0.f, a2 = 0.f;
#pragma unroll 4
        for (int32_t i = lane; i < len; i += 32) { a0 += vx[b0 + i] - px; a1 += vy[b0 + i] - py; a2 += vz[b0 + i] - pz; }
        S0 += (double)a0; S1 += (double)a1; S2 += (double)a2;
    }
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) { S0 += fpd_shfl_xor(S0, d); S1 += fpd_shfl_xor(S1, d); S2 += fpd_shfl_xor(S2, d); }
    const double invn = 1.0 / (double)n;
    const double m0d = S0 * invn, m1d = S1 * invn, m2d = S2 * invn;
    const float m0 = (float)m0d, m1 = (float)m1d, m2 = (float)m2d;
    double tot = 0.0;                                                     // lane i: record slot i
#pragma unroll 1
    for (int32_t off = 0; off < n; off += MOM_CAP) {
        const int32_t len = min((int32_t)MOM_CAP, n - off), b0 = s + off;
        __syncwarp();
        for (int32_t i = lane; i < len; i += 32) { sx[i] = vx[b0 + i]; sy[i] = vy[b0 + i]; sz[i] = vz[b0 + i]; }
        __syncwarp();
        float r[32];
#pragma unroll
        for (int q = 0; q < 32; ++q) r[q] = 0.f;
        for (int32_t i = lane; i < len; i += 32) {
            const float cx = (sx[i] - px) - m0, cy = (sy[i] - py) - m1, cz = (sz[i] - pz) - m2;
            const float xx = cx * cx, xy = cx * cy, xz = cx * cz, yy = cy * cy, yz = cy * cz, zz = cz * cz;
            const float c2 = (xx + yy) + zz;
            r[4] += xx; r[5] += xy; r[6] += xz; r[7] += yy; r[8] += yz; r[9] += zz;
            if (FULL) {
                r[10] = fmaf(xx, cx, r[10]); r[11] = fmaf(xx, cy, r[11]); r[12] = fmaf(xx, cz, r[12]);
                r[13] = fmaf(xy, cy, r[13]); r[14] = fmaf(xy, cz, r[14]); r[15] = fmaf(xz, cz, r[15]);
                r[16] = fmaf(yy, cy, r[16]); r[17] = fmaf(yy, cz, r[17]); r[18] = fmaf(yz, cz, r[18]);
                r[19] = fmaf(zz, cz, r[19]);
                r[20] = fmaf(c2, xx, r[20]); r[21] = fmaf(c2, xy, r[21]); r[22] = fmaf(c2, xz, r[22]);
                r[23] = fmaf(c2, yy, r[23]); r[24] = fmaf(c2, yz, r[24]); r[25] = fmaf(c2, zz, r[25]);
                const float c4 = c2 * c2;
                r[26] = fmaf(c4, cx, r[26]); r[27] = fmaf(c4, cy, r[27]); r[28] = fmaf(c4, cz, r[28]);
            } else {
                r[10] = fmaf(c2, cx, r[10]); r[11] = fmaf(c2, cy, r[11]); r[12] = fmaf(c2, cz, r[12]);   // h_i
            }
        }
        fpd_transpose_reduce<32, 32, float>(r, lane);
        tot += (double)r[0];
    }
    double val = tot * invn;
    if (lane == 0) val = (double)n;
    else if (lane == 1) val = (double)px + m0d;
    else if (lane == 2) val = (double)py + m1d;
    else if (lane == 3) val = (double)pz + m2d;
    if (lane < NREC) rec[lane] = val;
}

// The cells of a chunk that does not fit the staging buffer, one at a time: each staged on its own and reduced by
// all 32 lanes; only a cell that alone exceeds the buffer reads global memory.  Kept out of line so that its
// registers do not add to the common path's.
template <bool FULL>
__device__ __noinline__ void mom_dense_chunk(const float* __restrict__ vx, const float* __restrict__ vy,
                                             const float* __restrict__ vz, int32_t cs_cur, int cpw, int64_t chunk,
                                             int32_t ncell, int64_t np, int32_t aligned, float* sx, uint64_t* bar,
                                             uint32_t& phase, int b, int lane, double* __restrict__ mom)
{
    constexpr int NREC = FULL ? 29 : 13;
    float* sy = sx + MOM_CAP;
    float* sz = sy + MOM_CAP;
#pragma unroll 1
    for (int c = 0; c < cpw; ++c) {
        const int32_t s1c = __shfl_sync(0xffffffffu, cs_cur, c), e1c = __shfl_sync(0xffffffffu, cs_cur, c + 1);
        const int64_t cellc = chunk * cpw + c;
        if (cellc >= ncell) continue;                                             // warp-uniform
        double* recc = mom + (size_t)cellc * NREC;
        const fpw_range rc = fpw_range_of(s1c, e1c, np, (aligned & 1) != 0, MOM_CAP);
        if (rc.staged) {
            fpt_fence_proxy_async();                 // earlier generic writes to the buffer vs the new bulk copy
            __syncwarp();
            const uint32_t bytes = (uint32_t)rc.nb * 4u;
            if (bytes > 0 && lane == 0) {
                fpt_mbar_expect_tx(bar, 3u * bytes);
                fpt_bulk_g2s(sx, vx + rc.a0, bytes, bar);
                fpt_bulk_g2s(sy, vy + rc.a0, bytes, bar);
                fpt_bulk_g2s(sz, vz + rc.a0, bytes, bar);
            }
            for (int32_t p = rc.a0 + rc.nb + lane; p < rc.s1; p += 32) {
                sx[p - rc.a0] = vx[p]; sy[p - rc.a0] = vy[p]; sz[p - rc.a0] = vz[p];
            }
            if (bytes > 0) { fpt_mbar_wait(bar, (phase >> b) & 1u); phase ^= 1u << b; }
            __syncwarp();
            mom_cell_group<32, FULL>(sx - rc.a0, sy - rc.a0, sz - rc.a0, s1c, e1c - s1c, true, lane, recc);
        } else {
            if (e1c > s1c) mom_giant_cell<FULL>(vx, vy, vz, s1c, e1c - s1c, sx, lane, recc);
            else if (lane < NREC) recc[lane] = 0.0;                       // empty cell: N = 0 and zeros
        }
    }
}

// Persistent warps: a warp owns chunks wg, wg + nwarps, ... of 32/G consecutive cells.  MOM_STAGES = 2: while it reduces
// one chunk the bulk copies of its next chunk are already in flight into the warp's other staging buffer (mbarrier
// per stage).  MOM_STAGES = 1: one (larger) buffer per warp; the copies of the next chunk are issued as soon as pass 2
// has read the last particle, i.e. they overlap the cross-lane tree, the fp64 finish and the record stores, and the
// other resident warps cover the rest of the latency.  The cell boundaries of the chunk after next are fetched ahead
// in both cases.
#ifndef MOM_MINB
#define MOM_MINB 4                      // 128 registers: four CTAs per SM is what the staging buffers allow
#endif
#ifndef MOM_STAGES
#define MOM_STAGES 2
#endif
#ifndef MOM_ROT
#define MOM_ROT 1                       // rotated, conflict-free visiting order for cells of <= 128*G particles
#endif
#ifndef MOM_GMIN
#define MOM_GMIN 4                      // smallest group width instantiated for the dispatch
#endif
#ifndef MOM_FILL
#define MOM_FILL 0.875                  // a chunk of 32/G mean-sized cells fills at most this part of the buffer
#endif
template <int G, bool FULL>
__global__ void __launch_bounds__(MOM_THREADS, MOM_MINB)
moments_warp_kernel(const float* __restrict__ vx, const float* __restrict__ vy, const float* __restrict__ vz,
                    const int32_t* __restrict__ cell_start, int32_t ncell, int64_t np, int32_t aligned,
                    double* __restrict__ mom, uint32_t* __restrict__ err)
{
    fpd_pdl();
    constexpr int NREC = FULL ? 29 : 13;
    constexpr int CPW = 32 / G;                          // cells per warp and chunk
    constexpr int NST = MOM_STAGES;
    extern __shared__ __align__(16) unsigned char fpw_smem[];
    float* stage = reinterpret_cast<float*>(fpw_smem);                                   // [MOM_WARPS][NST][3][MOM_CAP]
    uint64_t* bars = reinterpret_cast<uint64_t*>(fpw_smem + (size_t)MOM_WARPS * NST * 3 * MOM_CAP * sizeof(float));
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int gl = lane & (G - 1), group = lane / G;
    const int64_t nchunks = ((int64_t)ncell + CPW - 1) / CPW;
    const int64_t nw = (int64_t)gridDim.x * MOM_WARPS;
    int64_t chunk = (int64_t)blockIdx.x * MOM_WARPS + warp;
    if (chunk >= nchunks) return;
    float* wbuf = stage + (size_t)warp * NST * 3 * MOM_CAP;
    uint64_t* wbar = bars + warp * 2;
    if (lane == 0) { fpt_mbar_init(&wbar[0], 1); fpt_mbar_init(&wbar[1], 1); }
    __syncwarp();
    // A chunk's cell boundaries are FETCHED two chunks ahead and VALIDATED (empty chunk if invalid) only when the chunk moves
    // up: the check's shuffle would otherwise wait for the load it was meant to hide (12 % of the kernel's stall samples).
    auto fetch_cs = [&](int64_t c) { return cell_start[min(c * CPW + lane, (int64_t)ncell)]; };
    auto check_cs = [&](int32_t v, int64_t c) {
        const int cells = (int)min((int64_t)CPW, (int64_t)ncell - c * CPW);
        return fpd_cells_ok(v, c * CPW, cells, ncell, np, lane, err) ? v : 0;
    };
    auto range_of = [&](int32_t cs) {
        fpw_range r = fpw_range_of(__shfl_sync(0xffffffffu, cs, 0), __shfl_sync(0xffffffffu, cs, CPW), np, (aligned & 1) != 0, MOM_CAP);
        // fp_set_reproducible: every cell on its own with all 32 lanes (mom_dense_chunk), so that a cell's summation order
        // depends on nothing but the cell -- not on its neighbours in the chunk, nor on the lanes-per-cell width the
        // context's mean density selects
        if (aligned & 2) r.staged = false;
        return r;
    };
    auto issue = [&](const fpw_range& r, int b) {
        const uint32_t bytes = (uint32_t)r.nb * 4u;
        if (r.staged && bytes > 0 && lane == 0) {
            float* d = wbuf + (size_t)b * 3 * MOM_CAP;
            fpt_mbar_expect_tx(&wbar[b], 3u * bytes);
            fpt_bulk_g2s(d, vx + r.a0, bytes, &wbar[b]);
            fpt_bulk_g2s(d + MOM_CAP, vy + r.a0, bytes, &wbar[b]);
            fpt_bulk_g2s(d + 2 * MOM_CAP, vz + r.a0, bytes, &wbar[b]);
        }
    };
    int32_t cs_cur = fetch_cs(chunk);
    int64_t nxt = chunk + nw;
    int32_t cs_nxt = nxt < nchunks ? fetch_cs(nxt) : 0;
    cs_cur = check_cs(cs_cur, chunk);
    if (nxt < nchunks) cs_nxt = check_cs(cs_nxt, nxt);
    fpw_range r_cur = range_of(cs_cur);
    issue(r_cur, 0);
    int b = 0;
    uint32_t phase = 0;
    while (true) {
        fpw_range r_nxt = r_cur;
        const bool more = nxt < nchunks;
        if (more) {
            r_nxt = range_of(cs_nxt);
            if (NST == 2) {
                fpt_fence_proxy_async();                    // generic-proxy writes to buffer b^1 (tail particles, scratch) vs the bulk copy
                __syncwarp();                               // every lane is done with buffer b^1 (previous chunk)
                issue(r_nxt, b ^ 1);
            }
        }
        const int64_t nxt2 = nxt + nw;
        const int32_t cs_nxt2 = nxt2 < nchunks ? fetch_cs(nxt2) : 0;      // not validated yet
        // ---- the current chunk
        const int32_t s = __shfl_sync(0xffffffffu, cs_cur, group), e = __shfl_sync(0xffffffffu, cs_cur, group + 1);
        const int64_t cell = chunk * CPW + group;
        const bool have = cell < ncell;
        const int32_t n = have ? e - s : 0;
        double* rec = mom + (size_t)(have ? cell : 0) * NREC;
        bool reissued = false;
        if (r_cur.staged) {
            float* sx = wbuf + (size_t)b * 3 * MOM_CAP;
            float* sy = sx + MOM_CAP;
            float* sz = sy + MOM_CAP;
            // the (at most 3) particles beyond the last multiple of 4 of the whole array
            for (int32_t p = r_cur.a0 + r_cur.nb + lane; p < r_cur.s1; p += 32) {
                sx[p - r_cur.a0] = vx[p]; sy[p - r_cur.a0] = vy[p]; sz[p - r_cur.a0] = vz[p];
            }
            if (r_cur.nb > 0) { fpt_mbar_wait(&wbar[b], (phase >> b) & 1u); phase ^= 1u << b; }
            __syncwarp();
            const int32_t nmax = __reduce_max_sync(0xffffffffu, n);
            const int32_t sb = n > 0 ? s : r_cur.a0;        // empty cell: any staged address
            if (MOM_ROT && nmax <= 128 * G) {
                auto hook = [&]() {
                    if (NST == 1 && more) {
                        fpt_fence_proxy_async();
                        __syncwarp();
                        issue(r_nxt, 0);
                    }
                    reissued = true;
                };
                mom_cell_rot<G, FULL>(sx - r_cur.a0, sy - r_cur.a0, sz - r_cur.a0, sb, n, have, gl, group, rec, (aligned & 2) != 0,
                                      NST == 2 ? sx : nullptr, hook);
            } else if (NST == 1) {
                auto hook = [&]() {
                    if (more) {
                        fpt_fence_proxy_async();            // generic-proxy writes of pass 1 vs the new bulk copy
                        __syncwarp();
                        issue(r_nxt, 0);
                    }
                    reissued = true;
                };
                mom_cell_group<G, FULL>(sx - r_cur.a0, sy - r_cur.a0, sz - r_cur.a0, s, n, have, gl, rec, hook);
            } else {
                mom_cell_group<G, FULL>(sx - r_cur.a0, sy - r_cur.a0, sz - r_cur.a0, s, n, have, gl, rec);
            }
        } else {
            // a chunk too dense for the staging buffer (load-imbalanced grids): cell by cell in buffer b
            mom_dense_chunk<FULL>(vx, vy, vz, cs_cur, CPW, chunk, ncell, np, aligned, wbuf + (size_t)b * 3 * MOM_CAP,
                                  &wbar[b], phase, b, lane, mom);
        }
        if (!more) break;
        if (NST == 1 && !reissued) {
            fpt_fence_proxy_async();
            __syncwarp();
            issue(r_nxt, 0);
        }
        chunk = nxt; cs_cur = cs_nxt; r_cur = r_nxt;
        nxt = nxt2; cs_nxt = nxt2 < nchunks ? check_cs(cs_nxt2, nxt2) : 0;
        if (NST == 2) b ^= 1;
    }
}

#include "moments_seg.cuh"

template <int G>
static void launch_moments(fp_ctx* ctx, int64_t np, const float* vx, const float* vy, const float* vz,
                           const int32_t* cell_start, int32_t mode, double* mom, cudaStream_t st)
{
    const int cells_per_block = MOM_WARPS * (32 / G);
    // bit 0: 16-byte aligned arrays (bulk copies); bit 1: fp_set_reproducible (no address-dependent visiting order)
    const int aligned = (((((uintptr_t)vx) | ((uintptr_t)vy) | ((uintptr_t)vz)) & 15u) == 0 ? 1 : 0) | (ctx->reproducible ? 2 : 0);
    const size_t smem = (size_t)MOM_WARPS * MOM_STAGES * 3 * MOM_CAP * sizeof(float) + MOM_WARPS * 2 * sizeof(uint64_t);
    int& occ = ctx->mom_occ[G == 2 ? 0 : G == 4 ? 1 : G == 8 ? 2 : G == 16 ? 3 : 4];   // resident CTAs per SM
    if (occ == 0) {
        cudaFuncSetAttribute(moments_warp_kernel<G, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        cudaFuncSetAttribute(moments_warp_kernel<G, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, moments_warp_kernel<G, true>, MOM_THREADS, smem);
        if (occ < 1) occ = 1;
    }
    const int want = fp_div_up(ctx->ncell, cells_per_block);
    const int cap = ctx->num_sms * occ;
    const int blocks = want < cap ? want : cap;
    if (mode) fp_launch(moments_warp_kernel<G, true>, blocks, MOM_THREADS, smem, st, vx, vy, vz, cell_start, ctx->ncell, np, aligned, mom, ctx->d_err);
    else      fp_launch(moments_warp_kernel<G, false>, blocks, MOM_THREADS, smem, st, vx, vy, vz, cell_start, ctx->ncell, np, aligned, mom, ctx->d_err);
}

extern "C" int fp_cell_moments(fp_ctx* ctx, int64_t np, const float* vx, const float* vy, const float* vz,
                               const int32_t* cell_start, int32_t mode, double* mom, void* stream)
{
    if (!ctx) return FP_ERR_ARG;
    if (np < 0 || !cell_start || !mom || (mode != 0 && mode != 1)) return fp_fail(ctx, FP_ERR_ARG, "fp_cell_moments: bad argument");
    if (np > 0 && (!vx || !vy || !vz)) return fp_fail(ctx, FP_ERR_ARG, "fp_cell_moments: null velocity pointer");
    if (fp_state_check(ctx, "fp_cell_moments") != FP_OK) return FP_ERR_STATE;
    cudaStream_t st = (cudaStream_t)stream;
    const double ppc = (double)np / (double)ctx->ncell;
    // group width: the chunk of 32/G cells must fit the staging buffer (tiles.cuh)
    // very high particles per cell: equal 512-particle slices, one-pass raw sums, fp64 shift (moments_seg.cuh)
    const bool aligned16 = ((((uintptr_t)vx) | ((uintptr_t)vy) | ((uintptr_t)vz)) & 15u) == 0;
    // (with at least one resident warp's worth of cells per warp slot, one warp per huge cell is still the faster
    // path: 4096 cells x 1000 particles 39 vs 46 us; 300 cells x 30,000 particles 367 vs 60 us)
    const bool few_cells = ctx->ncell < ctx->num_sms * 16 || ctx->env_mom_seg;
    // (not in reproducible mode: the slices add to a cell's accumulators with atomics, in an order that varies from run to run)
    if (ppc > MOM_SEG_MIN && few_cells && aligned16 && np > 0 && np < ((int64_t)1 << 31) && !ctx->env_mom_no_seg && !ctx->reproducible) {
        const size_t bytes = (size_t)ctx->ncell * 28 * sizeof(double);       // allocated at fp_create
        fp_launch(fp_cs_check_kernel, fp_div_up(ctx->ncell + 1, 256) < 296 ? fp_div_up(ctx->ncell + 1, 256) : 296, 256, 0, st, cell_start,
                  ctx->ncell, np, ctx->d_err, ctx->d_errdev);
        FP_CUDA_OK(ctx, cudaMemsetAsync(ctx->mom_acc, 0, bytes, st));
        const int64_t nslices = (np + MOM_SEG - 1) / MOM_SEG;
        const int64_t want = (nslices + MOM_SEG_WARPS - 1) / MOM_SEG_WARPS;
        const int cap = ctx->num_sms * 8;
        fp_launch(mom_seg_kernel, (int)(want < cap ? want : cap), MOM_SEG_WARPS * 32, 0, st, vx, vy, vz, cell_start,
                  ctx->ncell, np, ctx->mom_acc, (const uint32_t*)ctx->d_errdev);
        if (mode) fp_launch(mom_seg_finalize_kernel<true>, fp_div_up(ctx->ncell, 128), 128, 0, st, vx, vy, vz, cell_start,
                            ctx->ncell, (const double*)ctx->mom_acc, mom, (const uint32_t*)ctx->d_errdev);
        else      fp_launch(mom_seg_finalize_kernel<false>, fp_div_up(ctx->ncell, 128), 128, 0, st, vx, vy, vz, cell_start,
                            ctx->ncell, (const double*)ctx->mom_acc, mom, (const uint32_t*)ctx->d_errdev);
        FP_LAUNCH_OK(ctx);
        FP_COUNT(ctx, 3);
        return FP_OK;
    }
    // lanes per cell: the smallest G whose chunk of 32/G mean-sized cells leaves room for the count fluctuations
    const double room = MOM_FILL * (double)MOM_CAP;
    if (ppc * 2 > room)                        launch_moments<32>(ctx, np, vx, vy, vz, cell_start, mode, mom, st);
    else if (ppc * 4 > room)                   launch_moments<16>(ctx, np, vx, vy, vz, cell_start, mode, mom, st);
    else if (ppc * 8 > room)                   launch_moments<8>(ctx, np, vx, vy, vz, cell_start, mode, mom, st);
#if MOM_GMIN <= 2
    else if (ppc * 16 > room)                  launch_moments<4>(ctx, np, vx, vy, vz, cell_start, mode, mom, st);
    else                                       launch_moments<2>(ctx, np, vx, vy, vz, cell_start, mode, mom, st);
#else
    else                                       launch_moments<4>(ctx, np, vx, vy, vz, cell_start, mode, mom, st);
#endif
    FP_LAUNCH_OK(ctx);
    FP_COUNT(ctx, 1);
    return FP_OK;
}
