// sort.cu -- a2: cell key + STABLE sort by key + payload permute + cell_start (
// DESIGN.md R1).  Integer work: results are bit-exact and unique (equal keys keep input order).
//
// Least-significant-digit radix sort on (key, index) pairs, digit width <= 9 bits so that a 2^18-cell grid sorts
// in two passes.  Each pass = per-tile digit histogram -> per-digit scan over tiles -> stable scatter; the histogram
// of a pass is produced by whoever writes that pass's input (key_kernel / the stream kernel for the first pass, the
// previous scatter for the later ones), hist_kernel only serves callers that bring their own keys.  Stability
// inside a tile comes from warp-striped item order plus __match_any_sync ranking (no atomics decide an order).
// The payload (x, y, vx, vy, vz, pid) is gathered once at the end through the final permutation.  Two-pass sorts whose
// index and high digit fit one 32-bit word (4M particles x 40k cells: 22 + 8 bits) move that single word between the
// passes instead of a key and an index, and do not store sorted keys at all (the gather recomputes a particle's key
// from the positions it reads anyway): 16 B/particle less traffic and one register array less in the scatter.
#include "common.cuh"

// cell keys of tile blockIdx.x plus the tile's histogram of the first radix digit
__global__ void __launch_bounds__(SORT_THREADS)
key_kernel(int64_t np, const float* __restrict__ x, const float* __restrict__ y, uint32_t* __restrict__ keys,
           const fp_grid G, uint32_t* __restrict__ block_hist, int nblocks, int bins)
{
    __shared__ uint32_t h[SORT_MAX_BINS];
    for (int b = threadIdx.x; b < bins; b += SORT_THREADS) h[b] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * SORT_TILE;
    const uint32_t mask = (uint32_t)bins - 1u;
#pragma unroll 4
    for (int i = 0; i < SORT_ITEMS; ++i) {
        const int64_t p = base + i * SORT_THREADS + threadIdx.x;
        const bool valid = p < np;
        uint32_t key = 0;
        if (valid) {
            key = (uint32_t)fpd_cell_key(x[p], y[p], G);
            keys[p] = key;
        }
        if (valid) atomicAdd(&h[key & mask], 1u);
    }
    __syncthreads();
    for (int b = threadIdx.x; b < bins; b += SORT_THREADS) block_hist[(size_t)b * nblocks + blockIdx.x] = h[b];
}

// per-tile digit histogram: block_hist[bin * nblocks + block]
__global__ void __launch_bounds__(SORT_THREADS)
hist_kernel(int64_t np, const uint32_t* __restrict__ keys, uint32_t* __restrict__ block_hist, int nblocks,
            int shift, int bins)
{
    __shared__ uint32_t h[SORT_MAX_BINS];
    for (int b = threadIdx.x; b < bins; b += SORT_THREADS) h[b] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * SORT_TILE;
    const uint32_t mask = (uint32_t)bins - 1u;
#pragma unroll
    for (int i = 0; i < SORT_ITEMS; ++i) {
        const int64_t p = base + i * SORT_THREADS + threadIdx.x;
        if (p < np) atomicAdd(&h[(keys[p] >> shift) & mask], 1u);
    }
    __syncthreads();
    for (int b = threadIdx.x; b < bins; b += SORT_THREADS) block_hist[(size_t)b * nblocks + blockIdx.x] = h[b];
}

// one block per digit value: exclusive scan of that digit's counts over tiles (in place) and the digit total;
// also zeroes the same row of the other table
__global__ void __launch_bounds__(256)
scan_rows_kernel(uint32_t* __restrict__ block_hist, uint32_t* __restrict__ bin_total, int nblocks,
                 uint32_t* __restrict__ other_table)
{
    fpd_pdl();
    // the other pass's table is free now: clear this digit's row for the reductions that fill it next
    for (int i = threadIdx.x; i < nblocks; i += 256) other_table[(size_t)blockIdx.x * nblocks + i] = 0u;
    __shared__ uint32_t wsum[8];
    uint32_t* row = block_hist + (size_t)blockIdx.x * nblocks;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int per = (nblocks + 255) / 256;
    const int beg = min(tid * per, nblocks), end = min(beg + per, nblocks);
    constexpr int KEEP = 8;                       // counts held in registers (up to 2048 tiles = 8M particles) ...
    uint32_t keep[KEEP];
    uint32_t sum = 0;
    if (per <= KEEP) {
#pragma unroll
        for (int q = 0; q < KEEP; ++q) { keep[q] = (beg + q < end) ? row[beg + q] : 0u; sum += keep[q]; }
    } else {                                      // ... re-read from global memory beyond that
        for (int i = beg; i < end; ++i) sum += row[i];
    }
    uint32_t incl = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += t; }
    if (lane == 31) wsum[warp] = incl;
    __syncthreads();
    uint32_t wbase = 0, total = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) { if (w < warp) wbase += wsum[w]; total += wsum[w]; }
    uint32_t run = wbase + incl - sum;
    if (per <= KEEP) {
#pragma unroll
        for (int q = 0; q < KEEP; ++q) { if (beg + q < end) row[beg + q] = run; run += keep[q]; }
    } else {
        for (int i = beg; i < end; ++i) { const uint32_t v = row[i]; row[i] = run; run += v; }
    }
    if (tid == 0) bin_total[blockIdx.x] = total;
}

__device__ __forceinline__ int dbits_of(int bins) { return 31 - __clz(bins); }

// What a scatter pass reads and writes.  PLAIN: (key, index) pairs in two arrays.  With two passes and
// index bits + high-digit bits <= 32 the pair travels as one word between the passes: PACK_OUT (first pass) writes
// (high digit << pack_bits) | index into keys_out, PACK_IN (second pass) reads that word, ranks by its digit and
// writes only the index; the sorted keys are not stored (the gather recomputes them from the positions).
// LATER_NOKEYS: the last pass of a two-array sort whose keys are cell keys: only the index is written, the gather recomputes
// the keys from the positions (as after a packed sort).
enum { SORT_FIRST = 0, SORT_LATER = 1, SORT_PACK_OUT = 2, SORT_PACK_IN = 3, SORT_LATER_NOKEYS = 4 };

// The items of one tile: load, rank, scatter.  FULLT: every item of the tile exists (no bounds checks).
template <int MODE, bool FULLT>
__device__ __forceinline__ void scatter_items(int64_t np, const uint32_t* __restrict__ keys_in,
                                              const uint32_t* __restrict__ idx_in, uint32_t* __restrict__ keys_out,
                                              uint32_t* __restrict__ idx_out, int nblocks, int shift, int bins,
                                              int pack_bits, uint32_t* __restrict__ next_hist,
                                              uint32_t (*cnt)[SORT_MAX_BINS], const uint32_t* bin_base)
{
    constexpr bool FIRST_PASS = (MODE == SORT_FIRST || MODE == SORT_PACK_OUT);
    constexpr bool HAS_IDX = (MODE == SORT_LATER || MODE == SORT_LATER_NOKEYS);       // a separate index array comes in
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t mask = (uint32_t)bins - 1u;
    const int64_t wbase = (int64_t)blockIdx.x * SORT_TILE + warp * (32 * SORT_ITEMS) + lane;   // this lane's first item
    const uint32_t* kp = keys_in + wbase;
    const uint32_t* ip = HAS_IDX ? idx_in + wbase : nullptr;
    uint32_t key[SORT_ITEMS], idx[SORT_ITEMS], rank[SORT_ITEMS];   // PACK_IN: key[] holds the packed word, idx[] is unused
    bool valid[SORT_ITEMS];
#pragma unroll
    for (int i = 0; i < SORT_ITEMS; ++i) {
        valid[i] = FULLT ? true : (wbase + i * 32 < np);
        key[i] = valid[i] ? kp[i * 32] : 0xffffffffu;
        idx[i] = FIRST_PASS ? (uint32_t)wbase + (uint32_t)(i * 32) : ((HAS_IDX && valid[i]) ? ip[i * 32] : 0u);
    }
    // rank inside the warp's sub-tile, round by round (stable)
#pragma unroll
    for (int i = 0; i < SORT_ITEMS; ++i) {
        const uint32_t d = (key[i] >> shift) & mask;
        const uint32_t act = FULLT ? 0xffffffffu : __ballot_sync(0xffffffffu, valid[i]);
        uint32_t r = 0;
        if (valid[i]) {
            const uint32_t peers = __match_any_sync(act, d);   // (a ballot-per-bit search measured slower: 111 vs 99 us)
            const int leader = __ffs(peers) - 1;
            const uint32_t before = __popc(peers & ((1u << lane) - 1u));
            uint32_t c = 0;
            if (lane == leader) { c = cnt[warp][d]; cnt[warp][d] = c + __popc(peers); }
            c = __shfl_sync(peers, c, leader);
            r = c + before;
        }
        rank[i] = r;
        __syncwarp();
    }
    __syncthreads();
    // per digit value: exclusive scan over the warps -> base of (warp, digit) inside the tile's digit run
    for (int b = threadIdx.x; b < bins; b += SORT_THREADS) {
        uint32_t run = 0;
#pragma unroll
        for (int w = 0; w < SORT_WARPS; ++w) { const uint32_t c = cnt[w][b]; cnt[w][b] = run; run += c; }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < SORT_ITEMS; ++i) {
        uint32_t code = 0xffffffffu;               // (next digit, next tile) of this item
        if (valid[i]) {
            const uint32_t d = (key[i] >> shift) & mask;
            const uint32_t dst = bin_base[d] + cnt[warp][d] + rank[i];
            if (MODE == SORT_PACK_OUT) keys_out[dst] = ((key[i] >> (shift + dbits_of(bins))) << pack_bits) | idx[i];
            else if (MODE == SORT_PACK_IN) idx_out[dst] = key[i] & ((1u << pack_bits) - 1u);
            else if (MODE == SORT_LATER_NOKEYS) idx_out[dst] = idx[i];
            else { keys_out[dst] = key[i]; idx_out[dst] = idx[i]; }
            code = (((key[i] >> shift) >> dbits_of(bins)) & mask) << 20 | (dst / SORT_TILE);
        }
        // the next pass's tile histograms: the tile an item lands in is known here, so lanes that agree on
        // (next digit, next tile) send one aggregated reduction to the (zeroed) table of the next pass
        if (next_hist) {
            const uint32_t peers = __match_any_sync(0xffffffffu, code);
            if (valid[i] && lane == __ffs(peers) - 1)
                atomicAdd(&next_hist[(size_t)(code >> 20) * nblocks + (code & 0xfffffu)], (uint32_t)__popc(peers));
        }
    }
}

// stable scatter of one tile.  Warp w owns items [w*256, (w+1)*256) of the tile in warp-striped order
// (round i, lane l -> w*256 + i*32 + l), so (tile, warp, round, lane) order is input order.
#ifndef SORT_SCATTER_MINB
#define SORT_SCATTER_MINB 4                               // 64 registers: four tiles per SM hide the latency phases
#endif
template <int MODE>
__global__ void __launch_bounds__(SORT_THREADS, SORT_SCATTER_MINB)
scatter_kernel(int64_t np, const uint32_t* __restrict__ keys_in, const uint32_t* __restrict__ idx_in,
               uint32_t* __restrict__ keys_out, uint32_t* __restrict__ idx_out,
               const uint32_t* __restrict__ block_hist, const uint32_t* __restrict__ bin_total, int nblocks,
               int shift, int bins, int pack_bits, uint32_t* __restrict__ next_hist)
{
    fpd_pdl();
    __shared__ uint32_t cnt[SORT_WARPS][SORT_MAX_BINS];   // per-warp running digit counts, then bases
    __shared__ uint32_t bin_base[SORT_MAX_BINS];          // global start of each digit value + this tile's offset
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t mask = (uint32_t)bins - 1u;
    for (int b = threadIdx.x; b < bins; b += SORT_THREADS) {          // bins is a power of two <= SORT_MAX_BINS
#pragma unroll
        for (int w = 0; w < SORT_WARPS; ++w) cnt[w][b] = 0;
    }
    // exclusive scan of the digit totals (bins <= 512 = 8 warps x 32 lanes x 2 consecutive bins): every thread fetches
    // its two totals and its two tile offsets at once (one global latency), warps scan, warp totals go through smem
    {
        __shared__ uint32_t wtot[SORT_WARPS];
        const int b0 = 2 * (int)threadIdx.x, b1 = b0 + 1;
        const uint32_t v0 = (b0 < bins) ? bin_total[b0] : 0u, v1 = (b1 < bins) ? bin_total[b1] : 0u;
        const uint32_t h0 = (b0 < bins) ? block_hist[(size_t)b0 * nblocks + blockIdx.x] : 0u;
        const uint32_t h1 = (b1 < bins) ? block_hist[(size_t)b1 * nblocks + blockIdx.x] : 0u;
        uint32_t incl = v0 + v1;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += t; }
        if (lane == 31) wtot[warp] = incl;
        __syncthreads();
        uint32_t wb = 0;
#pragma unroll
        for (int w = 0; w < SORT_WARPS; ++w) if (w < warp) wb += wtot[w];
        const uint32_t e = wb + incl - (v0 + v1);
        if (b0 < bins) bin_base[b0] = e + h0;
        if (b1 < bins) bin_base[b1] = e + v0 + h1;
    }
    __syncthreads();
    if ((int64_t)(blockIdx.x + 1) * SORT_TILE <= np)       // block-uniform: all but the last tile are full
        scatter_items<MODE, true>(np, keys_in, idx_in, keys_out, idx_out, nblocks, shift, bins, pack_bits, next_hist, cnt, bin_base);
    else
        scatter_items<MODE, false>(np, keys_in, idx_in, keys_out, idx_out, nblocks, shift, bins, pack_bits, next_hist, cnt, bin_base);
}

// payload permute fused with cell_start from the sorted keys: cell_start[k] = first position whose key >= k,
// cell_start[ncell] = np.  Thread k owns the boundary between positions k-1 and k (and the last one also np).
// FROM_POS (packed sort): the sorted keys were not stored; a particle's key is recomputed from the positions this
// kernel gathers anyway (the same function of the same numbers as the key that was sorted), the left neighbour's
// key comes from the lane below or, for lane 0, from the neighbour's positions.
typedef fp_grid gather_grid;

template <bool FROM_POS>
#ifndef GATHER_MINB
#define GATHER_MINB 6
#endif
__global__ void __launch_bounds__(256, GATHER_MINB)         // 40 registers: all eight gathers of a trip in flight
gather_kernel(int64_t np, const uint32_t* __restrict__ perm, const uint32_t* __restrict__ skeys, int32_t ncell,
              int32_t* __restrict__ cell_start,
              const float* __restrict__ x, const float* __restrict__ y, const float* __restrict__ vx,
              const float* __restrict__ vy, const float* __restrict__ vz, const uint32_t* __restrict__ pid,
              float* __restrict__ xo, float* __restrict__ yo, float* __restrict__ vxo, float* __restrict__ vyo,
              float* __restrict__ vzo, uint32_t* __restrict__ pido, const __grid_constant__ gather_grid Gd)
{
    fpd_pdl();
    // cell_start is int32, so np < 2^31 and every index fits 32 bits
    const int n = (int)np, stride = (int)(gridDim.x * blockDim.x);
    const int lane = threadIdx.x & 31;
    const int kfirst = (int)(blockIdx.x * blockDim.x + (threadIdx.x & ~31));
    uint32_t s_pref = (kfirst + lane < n) ? perm[kfirst + lane] : 0u;      // the permutation entry is fetched one trip ahead
    // lane 0 also needs the key of position k0 - 1 (its left neighbour belongs to another warp): that entry is fetched one
    // trip ahead too, and its positions are gathered together with the trip's own (as a dependent chain after them --
    // perm[k0 - 1], then x and y -- it made the whole warp wait twice more per trip: 11 % of the kernel's stall samples)
    uint32_t l_pref = (FROM_POS && lane == 0 && kfirst > 0 && kfirst < n) ? perm[kfirst - 1] : 0u;
    for (int k0 = kfirst; k0 < n; k0 += stride) {                           // warp-uniform
        const int k = k0 + lane;
        const bool valid = k < n;
        int key = 0, lo = 0;
        float px = 0.f, py = 0.f, pvx = 0.f, pvy = 0.f, pvz = 0.f, lx = 0.f, ly = 0.f;
        uint32_t ppid = 0u;
        const uint32_t s = s_pref, sl = l_pref;
        if ((int64_t)k + stride < n) s_pref = perm[k + stride];
        if (FROM_POS && lane == 0 && (int64_t)k0 + stride < n) l_pref = perm[k0 + stride - 1];
        if (valid) {
            // every gather of the trip is issued before the first use
            px = x[s]; py = y[s]; pvx = vx[s]; pvy = vy[s]; pvz = vz[s]; ppid = pid[s];
            if (FROM_POS && lane == 0 && k > 0) { lx = x[sl]; ly = y[sl]; }
            if (FROM_POS) {
                key = fpd_cell_key(px, py, Gd);
            } else {
                key = (int)skeys[k];
                lo = (k == 0) ? 0 : (int)skeys[k - 1] + 1;
            }
        }
        if (FROM_POS) {
            int prev = __shfl_up_sync(0xffffffffu, key, 1);
            if (lane == 0 && k > 0 && valid) prev = fpd_cell_key(lx, ly, Gd);
            lo = (k == 0) ? 0 : prev + 1;
        }
        if (valid) {
            xo[k] = px; yo[k] = py; vxo[k] = pvx; vyo[k] = pvy; vzo[k] = pvz; pido[k] = ppid;
            for (int c = lo; c <= key; ++c) cell_start[c] = k;
            if (k == n - 1) for (int c = key + 1; c <= ncell; ++c) cell_start[c] = n;
        }
    }
}

__global__ void zero_i32_kernel(int32_t* a, int64_t n)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) a[i] = 0;
}

int fpi_sort_digit_bits(const fp_ctx* ctx)
{
    const int bits = ctx->key_bits < 1 ? 1 : ctx->key_bits;
    const int passes = (bits + 8) / 9;
    return (bits + passes - 1) / passes;                 // <= 9
}

int fpi_sort_with_keys(fp_ctx* ctx, int64_t np, const uint32_t* keys, bool hist0_ready,
                       const float* x, const float* y, const float* vx, const float* vy, const float* vz,
                       const uint32_t* pid, float* x_out, float* y_out, float* vx_out, float* vy_out,
                       float* vz_out, uint32_t* pid_out, int32_t* cell_start, uint32_t* perm, cudaStream_t st)
{
    const int32_t ncell = ctx->ncell;
    if (np == 0) {
        zero_i32_kernel<<<fp_div_up(ncell + 1, 256), 256, 0, st>>>(cell_start, (int64_t)ncell + 1);
        FP_LAUNCH_OK(ctx);
        FP_COUNT(ctx, 1);
        fp_mark(ctx, 2, st);
        return FP_OK;
    }
    const int nblocks = fp_div_up(np, SORT_TILE);
    const int bits = ctx->key_bits < 1 ? 1 : ctx->key_bits;
    const int passes = (bits + 8) / 9;
    const int dbits = fpi_sort_digit_bits(ctx);
    const int bins = 1 << dbits;
    if ((size_t)bins * nblocks > ctx->block_hist_elems) return fp_fail(ctx, FP_ERR_STATE, "sort scratch too small");
    // two passes and (index, high digit) fit one word: the pair travels packed between the passes
    int idx_bits = 1;
    while (idx_bits < 32 && ((int64_t)1 << idx_bits) < np) ++idx_bits;
    const bool packed = !ctx->sort_no_pack && passes == 2 && idx_bits + (bits - dbits) <= 32;
    // two-array sorts of cell keys (20M particles: index + high digit do not fit one word) need not store the sorted keys either
    const bool nokeys_last = !packed && passes >= 2 && !ctx->sort_slab_keys;
    const uint32_t* kin = keys;
    const uint32_t* iin = nullptr;
    uint32_t* kout = ctx->key_a;
    uint32_t* iout = ctx->idx_a;
    for (int pass = 0; pass < passes; ++pass) {
        const int shift = pass * dbits;
        uint32_t* table = ctx->block_hist + (size_t)(pass & 1) * ctx->block_hist_elems;
        uint32_t* other = ctx->block_hist + (size_t)((pass + 1) & 1) * ctx->block_hist_elems;
        if (pass == 0 && !hist0_ready) {              // later passes: the previous scatter filled the table
            hist_kernel<<<nblocks, SORT_THREADS, 0, st>>>(np, kin, table, nblocks, shift, bins);
            FP_COUNT(ctx, 1);
        }
        fp_launch(scan_rows_kernel, bins, 256, 0, st, table, ctx->bin_total, nblocks, other);
        uint32_t* next = (pass + 1 < passes) ? other : nullptr;
        if (packed && pass == 0)
            fp_launch(scatter_kernel<SORT_PACK_OUT>, nblocks, SORT_THREADS, 0, st, np, kin, iin, kout, iout, table, ctx->bin_total, nblocks, shift, bins, idx_bits, next);
        else if (packed)                              // the digit sits above the index bits of the packed word
            fp_launch(scatter_kernel<SORT_PACK_IN>, nblocks, SORT_THREADS, 0, st, np, kin, iin, kout, iout, table, ctx->bin_total, nblocks, idx_bits, bins, idx_bits, next);
        else if (pass == 0)
            fp_launch(scatter_kernel<SORT_FIRST>, nblocks, SORT_THREADS, 0, st, np, kin, iin, kout, iout, table, ctx->bin_total, nblocks, shift, bins, 0, next);
        else if (nokeys_last && pass + 1 == passes)
            fp_launch(scatter_kernel<SORT_LATER_NOKEYS>, nblocks, SORT_THREADS, 0, st, np, kin, iin, kout, iout, table, ctx->bin_total, nblocks, shift, bins, 0, next);
        else
            fp_launch(scatter_kernel<SORT_LATER>, nblocks, SORT_THREADS, 0, st, np, kin, iin, kout, iout, table, ctx->bin_total, nblocks, shift, bins, 0, next);
        FP_LAUNCH_OK(ctx);
        FP_COUNT(ctx, 2);
        kin = kout; iin = iout;
        kout = (kout == ctx->key_a) ? ctx->key_b : ctx->key_a;
        iout = (iout == ctx->idx_a) ? ctx->idx_b : ctx->idx_a;
    }
    ctx->hist0_clean = (passes & 1) == 0;             // the last scan zeroed the table the last pass did not use
    fp_mark(ctx, 2, st);
    // one resident wave of grid-striding CTAs (a partial second wave costs 4 us at 4M particles)
    int& gocc = ctx->gather_occ;
    if (gocc == 0) {
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&gocc, gather_kernel<true>, 256, 0);
        if (gocc < 1) gocc = 1;
    }
    const int64_t cap = (int64_t)ctx->num_sms * gocc;
    const int64_t want = (np + 255) / 256;
    const int gblocks = (int)(want < cap ? want : cap);
    const gather_grid Gd = fp_grid_of(ctx);
    if (ctx->ev_before_gather) FP_CUDA_OK(ctx, cudaStreamWaitEvent(st, ctx->ev_before_gather, 0));
    if (packed || nokeys_last)
        fp_launch(gather_kernel<true>, gblocks, 256, 0, st, np, iin, kin, ncell, cell_start, x, y, vx, vy, vz, pid,
                  x_out, y_out, vx_out, vy_out, vz_out, pid_out, Gd);
    else
        fp_launch(gather_kernel<false>, gblocks, 256, 0, st, np, iin, kin, ncell, cell_start, x, y, vx, vy, vz, pid,
                  x_out, y_out, vx_out, vy_out, vz_out, pid_out, Gd);
    FP_LAUNCH_OK(ctx);
    FP_COUNT(ctx, 1);
    if (ctx->ev_after_gather) FP_CUDA_OK(ctx, cudaEventRecord(ctx->ev_after_gather, st));
    if (perm) FP_CUDA_OK(ctx, cudaMemcpyAsync(perm, iin, (size_t)np * sizeof(uint32_t), cudaMemcpyDeviceToDevice, st));
    return FP_OK;
}

extern "C" int fp_sort_by_cell(fp_ctx* ctx, int64_t np,
                               const float* x, const float* y, const float* vx, const float* vy, const float* vz,
                               const uint32_t* pid,
                               float* x_out, float* y_out, float* vx_out, float* vy_out, float* vz_out,
                               uint32_t* pid_out, int32_t* cell_start, uint32_t* perm, void* stream)
{
    if (!ctx) return FP_ERR_ARG;
    if (np < 0 || !cell_start) return fp_fail(ctx, FP_ERR_ARG, "fp_sort_by_cell: np < 0 or null cell_start");
    if (np > ctx->p.max_particles) return fp_fail(ctx, FP_ERR_STATE, "fp_sort_by_cell: np > max_particles");
    if (np > 0 && (!x || !y || !vx || !vy || !vz || !pid || !x_out || !y_out || !vx_out || !vy_out || !vz_out || !pid_out))
        return fp_fail(ctx, FP_ERR_ARG, "fp_sort_by_cell: null pointer");
    if (np > 0 && (x == x_out || y == y_out || vx == vx_out || vy == vy_out || vz == vz_out || pid == pid_out))
        return fp_fail(ctx, FP_ERR_ARG, "fp_sort_by_cell: outputs may not alias inputs");
    cudaStream_t st = (cudaStream_t)stream;
    if (np > 0) {
        const int nblocks = fp_div_up(np, SORT_TILE);
        key_kernel<<<nblocks, SORT_THREADS, 0, st>>>(np, x, y, ctx->key_b, fp_grid_of(ctx), ctx->block_hist, nblocks,
                                                    1 << fpi_sort_digit_bits(ctx));
        FP_LAUNCH_OK(ctx);
        FP_COUNT(ctx, 1);
    }
    // keys live in key_b; the first pass writes key_a, so the ping-pong never overwrites its own input
    return fpi_sort_with_keys(ctx, np, ctx->key_b, np > 0, x, y, vx, vy, vz, pid, x_out, y_out, vx_out, vy_out, vz_out,
                              pid_out, cell_start, perm, st);
}
