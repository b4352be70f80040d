// sort.cu -- hand-written device primitives for the tree build and the interaction lists:
// a stable LSD radix sort of (u64 key, u32 value) pairs and an exclusive scan of int32.
// Integer work only; HBM-bound (tree / lists).
#include "fmm_internal.cuh"

// ----------------------------------------------------------------------------------------
// exclusive scan of int32 (three launches: tile sums, scan of the sums by one block, tile scan)
// ----------------------------------------------------------------------------------------
#define SCAN_THREADS 256
#define SCAN_ITEMS 8
#define SCAN_TILE (SCAN_THREADS * SCAN_ITEMS)

__device__ __forceinline__ int block_exclusive_scan_256(int v, int *total, int *smem /* [8] */)
{
    // exclusive scan of one int per thread over a 256-thread block; *total = block sum
    int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) smem[warp] = inc;
    __syncthreads();
    int wsum = (lane < 8) ? smem[lane] : 0;
    int winc = wsum;
#pragma unroll
    for (int o = 1; o < 8; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, winc, o);
        if (lane >= o) winc += t;
    }
    int wbase = __shfl_sync(0xffffffffu, winc - wsum, warp);
    *total = __shfl_sync(0xffffffffu, winc, 7);
    __syncthreads();
    return wbase + inc - v;
}

__global__ void __launch_bounds__(SCAN_THREADS) scan_tile_sums(const int32_t *__restrict__ in, int32_t *__restrict__ sums, int64_t n)
{
    __shared__ int sm[8];
    int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    int s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k)
        if (base + k < n) s += in[base + k];
    int total;
    block_exclusive_scan_256(s, &total, sm);
    if (threadIdx.x == 0) sums[blockIdx.x] = total;
}

__global__ void __launch_bounds__(SCAN_THREADS) scan_single_block(int32_t *__restrict__ a, int64_t n)
{
    // in-place exclusive scan of a short array by one block, chunk by chunk with a carry
    __shared__ int sm[8];
    int carry = 0;
    for (int64_t c0 = 0; c0 < n; c0 += SCAN_TILE) {
        int64_t base = c0 + (int64_t)threadIdx.x * SCAN_ITEMS;
        int v[SCAN_ITEMS], s = 0;
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; ++k) {
            v[k] = (base + k < n) ? a[base + k] : 0;
            s += v[k];
        }
        int total;
        int ex = block_exclusive_scan_256(s, &total, sm) + carry;
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; ++k) {
            if (base + k < n) a[base + k] = ex;
            ex += v[k];
        }
        carry += total;
    }
}

__global__ void __launch_bounds__(SCAN_THREADS) scan_tiles(const int32_t *__restrict__ in, int32_t *__restrict__ out,
                                                           const int32_t *__restrict__ sums, int64_t n)
{
    __shared__ int sm[8];
    int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    int v[SCAN_ITEMS], s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        v[k] = (base + k < n) ? in[base + k] : 0;
        s += v[k];
    }
    int total;
    int ex = block_exclusive_scan_256(s, &total, sm) + sums[blockIdx.x];
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        if (base + k < n) out[base + k] = ex;
        ex += v[k];
    }
}

static int scan_rec(fmm_ctx *c, const int32_t *in, int32_t *out, int64_t n)
{
    if (n <= 0) return FMM_OK;
    int64_t tiles = (n + SCAN_TILE - 1) / SCAN_TILE;
    if (tiles == 1) {
        if (in != out) FMM_CUDA(c, cudaMemcpyAsync(out, in, sizeof(int32_t) * n, cudaMemcpyDeviceToDevice, c->stream));
        scan_single_block<<<1, SCAN_THREADS, 0, c->stream>>>(out, n);
        FMM_LAUNCH_CHECK(c, "scan_single_block");
        return FMM_OK;
    }
    int32_t *sums = (int32_t *)ctx_alloc(c, sizeof(int32_t) * tiles);
    if (!sums) return FMM_ENOMEM;
    scan_tile_sums<<<(unsigned)tiles, SCAN_THREADS, 0, c->stream>>>(in, sums, n);
    FMM_LAUNCH_CHECK(c, "scan_tile_sums");
    if (tiles <= 64 * SCAN_TILE) {
        scan_single_block<<<1, SCAN_THREADS, 0, c->stream>>>(sums, tiles);
        FMM_LAUNCH_CHECK(c, "scan_single_block");
    } else {
        FMM_TRY(scan_rec(c, sums, sums, tiles));
    }
    scan_tiles<<<(unsigned)tiles, SCAN_THREADS, 0, c->stream>>>(in, out, sums, n);
    FMM_LAUNCH_CHECK(c, "scan_tiles");
    ctx_free(c, sums);  // stream-ordered reuse: the caller's allocator is stream-aware or the pool is ours
    return FMM_OK;
}

int scan_exclusive_i32(fmm_ctx *c, const int32_t *in, int32_t *out, int64_t n) { return scan_rec(c, in, out, n); }

// ----------------------------------------------------------------------------------------
// radix sort, 8 bits per pass
// ----------------------------------------------------------------------------------------
#define RS_THREADS 256
#define RS_WARPS 8

// lanes of the warp whose 8-bit digit equals this lane's (dead lanes match only dead lanes).  Eight ballots instead of
// MATCH.ANY: the match instruction walks the distinct values of the warp one by one (about 300 cycles per call with
// random digits, measured in profiles/r02_tree.md), the ballots are single-issue.
__device__ __forceinline__ unsigned digit_peers(int d, bool ok)
{
    unsigned m = __ballot_sync(0xffffffffu, ok);
    m = ok ? m : ~m;
#pragma unroll
    for (int b = 0; b < 8; ++b) {
        const unsigned bal = __ballot_sync(0xffffffffu, (d >> b) & 1);
        m &= ((d >> b) & 1) ? bal : ~bal;
    }
    return m;
}
#define RS_ROUNDS 8                       // keys per thread
#define RS_TILE (RS_THREADS * RS_ROUNDS)  // 2048 keys per block
#define RS_RADIX 256

// Warp w of a block owns the contiguous chunk [w*256, (w+1)*256) of the tile and walks it in 8 rounds
// of 32 consecutive keys, so that (warp, round, lane) order == input order: the sort is stable.
__global__ void __launch_bounds__(RS_THREADS) rs_histogram(const uint64_t *__restrict__ keys, int64_t n, int shift,
                                                           int32_t *__restrict__ table, int nblocks)
{
    __shared__ int cnt[RS_RADIX];
    cnt[threadIdx.x] = 0;
    __syncthreads();
    keys += (int64_t)blockIdx.y * n;                       // batch segment
    table += (int64_t)blockIdx.y * RS_RADIX * nblocks;
    int64_t base = (int64_t)blockIdx.x * RS_TILE;
#pragma unroll
    for (int r = 0; r < RS_ROUNDS; ++r) {
        int64_t i = base + (int64_t)r * RS_THREADS + threadIdx.x;
        if (i < n) atomicAdd(&cnt[(int)((keys[i] >> shift) & 0xff)], 1);
    }
    __syncthreads();
    table[(int64_t)threadIdx.x * nblocks + blockIdx.x] = cnt[threadIdx.x];
}

__global__ void __launch_bounds__(RS_THREADS) rs_scatter(const uint64_t *__restrict__ keys, const uint32_t *__restrict__ vals,
                                                         uint64_t *__restrict__ okeys, uint32_t *__restrict__ ovals,
                                                         int64_t n, int shift, const int32_t *__restrict__ table, int nblocks)
{
    __shared__ int cnt[RS_WARPS][RS_RADIX];  // per-warp running digit counts, then per-warp bases
    int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int k = threadIdx.x; k < RS_WARPS * RS_RADIX; k += RS_THREADS) (&cnt[0][0])[k] = 0;
    __syncthreads();
    // batch segment: the scan ran over the concatenated tables, so segment b's positions start at b * n
    const int64_t seg = (int64_t)blockIdx.y * n;
    keys += seg; okeys += seg;
    if (vals) { vals += seg; ovals += seg; }
    table += (int64_t)blockIdx.y * RS_RADIX * nblocks;
    const int seg_base = (int)seg;
    int64_t wbase = (int64_t)blockIdx.x * RS_TILE + (int64_t)warp * (RS_TILE / RS_WARPS);
    uint64_t key[RS_ROUNDS];
    int rank[RS_ROUNDS];
    unsigned lt = (1u << lane) - 1u;
#pragma unroll
    for (int r = 0; r < RS_ROUNDS; ++r) {
        int64_t i = wbase + r * 32 + lane;
        bool ok = i < n;
        key[r] = ok ? keys[i] : ~0ull;
        int d = ok ? (int)((key[r] >> shift) & 0xff) : 0;
        unsigned m = digit_peers(d, ok);
        int leader = __ffs(m) - 1;
        int prior = 0;
        if (ok && lane == leader) {
            prior = cnt[warp][d];
            cnt[warp][d] = prior + __popc(m);
        }
        prior = __shfl_sync(0xffffffffu, prior, leader);
        rank[r] = prior + __popc(m & lt);
        __syncwarp();
    }
    __syncthreads();
    {  // digit d = threadIdx.x: exclusive prefix over warps + global base of this block
        int d = threadIdx.x;
        int run = table[(int64_t)d * nblocks + blockIdx.x] - seg_base;
#pragma unroll
        for (int w = 0; w < RS_WARPS; ++w) {
            int t = cnt[w][d];
            cnt[w][d] = run;
            run += t;
        }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < RS_ROUNDS; ++r) {
        int64_t i = wbase + r * 32 + lane;
        if (i < n) {
            int d = (int)((key[r] >> shift) & 0xff);
            int64_t pos = (int64_t)cnt[warp][d] + rank[r];
            okeys[pos] = key[r];
            if (vals) ovals[pos] = vals[i];
        }
    }
}

int sort_pairs_u64(fmm_ctx *c, uint64_t *keys, uint32_t *vals, uint64_t *tmp_keys, uint32_t *tmp_vals,
                   int64_t n, int bit_lo, int bit_hi)
{
    return sort_pairs_u64_batched(c, keys, vals, tmp_keys, tmp_vals, n, 1, bit_lo, bit_hi);
}

// `batch` independent sorts of equal length n laid out back to back (segment b = [b n, (b+1) n)), one launch per pass
// for all of them (grid.y = batch): the passes of a 1M-key sort are latency-bound, so three sorts cost little more than one.
int sort_pairs_u64_batched(fmm_ctx *c, uint64_t *keys, uint32_t *vals, uint64_t *tmp_keys, uint32_t *tmp_vals,
                           int64_t n, int batch, int bit_lo, int bit_hi)
{
    if (n <= 1 || bit_hi <= bit_lo || batch < 1) return FMM_OK;
    if (n * batch >= (int64_t)1 << 31) return FMM_EOVERFLOW;
    int nblocks = (int)((n + RS_TILE - 1) / RS_TILE);
    int64_t tlen = (int64_t)RS_RADIX * nblocks * batch;
    int32_t *table = (int32_t *)ctx_alloc(c, sizeof(int32_t) * tlen);
    if (!table) return FMM_ENOMEM;
    uint64_t *ki = keys, *ko = tmp_keys;
    uint32_t *vi = vals, *vo = tmp_vals;
    for (int shift = bit_lo; shift < bit_hi; shift += 8) {
        rs_histogram<<<dim3(nblocks, batch), RS_THREADS, 0, c->stream>>>(ki, n, shift, table, nblocks);
        FMM_LAUNCH_CHECK(c, "rs_histogram");
        FMM_TRY(scan_exclusive_i32(c, table, table, tlen));
        rs_scatter<<<dim3(nblocks, batch), RS_THREADS, 0, c->stream>>>(ki, vi, ko, vo, n, shift, table, nblocks);
        FMM_LAUNCH_CHECK(c, "rs_scatter");
        uint64_t *tk = ki; ki = ko; ko = tk;
        uint32_t *tv = vi; vi = vo; vo = tv;
    }
    if (ki != keys) {
        FMM_CUDA(c, cudaMemcpyAsync(keys, ki, sizeof(uint64_t) * n * batch, cudaMemcpyDeviceToDevice, c->stream));
        if (vals) FMM_CUDA(c, cudaMemcpyAsync(vals, vi, sizeof(uint32_t) * n * batch, cudaMemcpyDeviceToDevice, c->stream));
    }
    ctx_free(c, table);
    return FMM_OK;
}

// ----------------------------------------------------------------------------------------
// radix sort of (u32 key, u32 value) pairs, 8 bits per pass, for the KD build (quantised coordinates).  Same ranking
// as above (stable); the scatter first reorders the tile in shared memory so that the keys of one digit leave the
// block as one contiguous run (coalesced stores instead of one sector per key).
// ----------------------------------------------------------------------------------------
#define RS32_ROUNDS 16
#define RS32_TILE (RS_THREADS * RS32_ROUNDS)  // 4096 keys per block

__global__ void __launch_bounds__(RS_THREADS) rs32_histogram(const uint32_t *__restrict__ keys, int64_t n, int shift,
                                                             int32_t *__restrict__ table, int nblocks)
{
    __shared__ int cnt[RS_RADIX];
    cnt[threadIdx.x] = 0;
    __syncthreads();
    keys += (int64_t)blockIdx.y * n;
    table += (int64_t)blockIdx.y * RS_RADIX * nblocks;
    const int64_t base = (int64_t)blockIdx.x * RS32_TILE;
    uint32_t k[RS32_ROUNDS];
#pragma unroll
    for (int r = 0; r < RS32_ROUNDS; ++r) {  // all loads first: one memory round trip per thread
        const int64_t i = base + (int64_t)r * RS_THREADS + threadIdx.x;
        k[r] = (i < n) ? keys[i] : 0u;
    }
#pragma unroll
    for (int r = 0; r < RS32_ROUNDS; ++r) {
        const int64_t i = base + (int64_t)r * RS_THREADS + threadIdx.x;
        if (i < n) atomicAdd(&cnt[(k[r] >> shift) & 0xffu], 1);
    }
    __syncthreads();
    table[(int64_t)threadIdx.x * nblocks + blockIdx.x] = cnt[threadIdx.x];
}

__global__ void __launch_bounds__(RS_THREADS) rs32_scatter(const uint32_t *__restrict__ keys, const uint32_t *__restrict__ vals,
                                                           uint32_t *__restrict__ okeys, uint32_t *__restrict__ ovals, int64_t n, int shift,
                                                           const int32_t *__restrict__ table, int nblocks)
{
    __shared__ int cnt[RS_WARPS][RS_RADIX];  // per-warp running digit counts, then per-warp bases inside the tile
    __shared__ int dbase[RS_RADIX];          // first tile position of a digit
    __shared__ int gbase[RS_RADIX];          // global position of a digit's first key of this block
    __shared__ uint32_t skey[RS32_TILE], sval[RS32_TILE];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int k = threadIdx.x; k < RS_WARPS * RS_RADIX; k += RS_THREADS) (&cnt[0][0])[k] = 0;
    __syncthreads();
    const int64_t seg = (int64_t)blockIdx.y * n;
    keys += seg; okeys += seg; vals += seg; ovals += seg;
    table += (int64_t)blockIdx.y * RS_RADIX * nblocks;
    const int64_t tile0 = (int64_t)blockIdx.x * RS32_TILE;
    const int64_t wbase = tile0 + (int64_t)warp * (RS32_TILE / RS_WARPS);
    const int live = (int)((n - tile0 < RS32_TILE) ? (n - tile0) : RS32_TILE);
    uint32_t key[RS32_ROUNDS];
    int rank[RS32_ROUNDS];
    const unsigned lt = (1u << lane) - 1u;
#pragma unroll
    for (int r = 0; r < RS32_ROUNDS; ++r) {  // warp w walks its contiguous chunk in rounds of 32: (warp, round, lane) order == input order
        const int64_t i = wbase + r * 32 + lane;
        const bool ok = i < n;
        key[r] = ok ? keys[i] : 0xffffffffu;
        const int d = ok ? (int)((key[r] >> shift) & 0xffu) : 0;
        const unsigned m = digit_peers(d, ok);
        const int leader = __ffs(m) - 1;
        int prior = 0;
        if (ok && lane == leader) {
            prior = cnt[warp][d];
            cnt[warp][d] = prior + __popc(m);
        }
        prior = __shfl_sync(0xffffffffu, prior, leader);
        rank[r] = prior + __popc(m & lt);
        __syncwarp();
    }
    __syncthreads();
    {  // digit d = threadIdx.x: exclusive prefix over warps, then over digits
        const int d = threadIdx.x;
        int run = 0;
#pragma unroll
        for (int w = 0; w < RS_WARPS; ++w) {
            const int t = cnt[w][d];
            cnt[w][d] = run;
            run += t;
        }
        // exclusive scan of the digit totals over the block (256 threads)
        int inc = run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        __shared__ int wsum[RS_WARPS];
        if (lane == 31) wsum[warp] = inc;
        __syncthreads();
        int wb = 0;
        for (int w = 0; w < warp; ++w) wb += wsum[w];
        dbase[d] = wb + inc - run;
        gbase[d] = table[(int64_t)d * nblocks + blockIdx.x] - (int)seg;
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < RS32_ROUNDS; ++r) {
        const int64_t i = wbase + r * 32 + lane;
        if (i < n) {
            const int d = (int)((key[r] >> shift) & 0xffu);
            const int pos = dbase[d] + cnt[warp][d] + rank[r];
            skey[pos] = key[r];
            sval[pos] = vals[i];
        }
    }
    __syncthreads();
    for (int q = threadIdx.x; q < live; q += RS_THREADS) {
        const uint32_t k = skey[q];
        const int d = (int)((k >> shift) & 0xffu);
        const int64_t pos = (int64_t)gbase[d] + (q - dbase[d]);
        okeys[pos] = k;
        ovals[pos] = sval[q];
    }
}

// `batch` independent sorts of length n laid out back to back on all 32 key bits; the result ends in keys / vals
int sort_pairs_u32_batched(fmm_ctx *c, uint32_t *keys, uint32_t *vals, uint32_t *tmp_keys, uint32_t *tmp_vals, int64_t n, int batch)
{
    if (n <= 1 || batch < 1) return FMM_OK;
    if (n * batch >= (int64_t)1 << 31) return FMM_EOVERFLOW;
    const int nblocks = (int)((n + RS32_TILE - 1) / RS32_TILE);
    const int64_t tlen = (int64_t)RS_RADIX * nblocks * batch;
    int32_t *table = (int32_t *)ctx_alloc(c, sizeof(int32_t) * tlen);
    if (!table) return FMM_ENOMEM;
    uint32_t *ki = keys, *ko = tmp_keys, *vi = vals, *vo = tmp_vals;
    for (int shift = 0; shift < 32; shift += 8) {  // (an even number of passes: the result is back in keys / vals)
        rs32_histogram<<<dim3(nblocks, batch), RS_THREADS, 0, c->stream>>>(ki, n, shift, table, nblocks);
        FMM_LAUNCH_CHECK(c, "rs32_histogram");
        FMM_TRY(scan_exclusive_i32(c, table, table, tlen));
        rs32_scatter<<<dim3(nblocks, batch), RS_THREADS, 0, c->stream>>>(ki, vi, ko, vo, n, shift, table, nblocks);
        FMM_LAUNCH_CHECK(c, "rs32_scatter");
        uint32_t *tk = ki; ki = ko; ko = tk;
        uint32_t *tv = vi; vi = vo; vo = tv;
    }
    ctx_free(c, table);
    return FMM_OK;
}
