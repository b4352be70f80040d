// kernels_kd.cu -- step a1, mode KD: the particle order of the balanced cluster tree of Alg 5.1 / 5.2
// (App. B) on the array tree of section 8.
//
// Exactly the paper's tree (readings T-1 .. T-3, G7 - G9): every node splits at the median rank along the axis of
// largest stretched extent, members ranked by (coordinate, original index), the first ceil(size/2) go left, ties of
// the axis choice to the first maximiser, ascending original index inside a leaf.  Built without recursion:
//   1. three index lists LX, LY, LZ sorted by (coordinate, index) and the index-ordered list LI.  The sort key is a
//      monotone 32-bit quantisation of the coordinate (4 radix passes instead of 8 on the 64-bit pattern); runs of
//      equal keys are then put into exact (coordinate, index) order by kd_find_runs / kd_fix_runs, which report the (pathological)
//      inputs they cannot repair locally so that the build falls back to the exact 64-bit keys;
//   2. per level: mark the left members in a bit mask (the first ceil(size/2) entries of the node's segment in the list
//      of its split axis; the node's box is read off the segment ends of the three sorted lists), then split every
//      segment of all four lists stably (left members first).  One kernel each: the running count of a node that spans
//      several tiles is looked up from the tiles before it (every tile publishes its count before it looks back, so
//      nothing waits on a chain), node ranges are closed-form (T-2);
//   3. once a node holds at most KD_LOCAL particles one block finishes all its remaining levels in shared memory.  The
//      index-ordered list LI is only needed there (ascending index inside a leaf), and a node's part of LI is just the
//      sorted ids of its members: the block sorts them itself (kdl_sort_ids), so the level kernels of step 2 split three
//      lists, not four (all four only when the leaves are larger than KD_LOCAL and step 3 does not run).
// Integer / compare work only: HBM-, L2- and launch-latency-bound.
#include "fmm_internal.cuh"

#include <stdlib.h>

#define KD_TILE 2048     // list entries per block of the level kernels (256 threads x 8)
#define KD_LOCAL 4096    // nodes of at most this many particles are finished by one block
#define KDL_THREADS 512
#define KDL_ITEMS 8      // KDL_THREADS x KDL_ITEMS = KD_LOCAL

// node [lo, hi) at `level` that contains list position pos (T-2: the left child gets ceil(size / 2))
__device__ __forceinline__ int kd_range_of(int N, int level, int pos, int &lo, int &hi)  // returns the node's index in its level
{
    lo = 0;
    hi = N;
    int k = 0;
    for (int l = 0; l < level; ++l) {
        const int mid = lo + (hi - lo + 1) / 2;
        k <<= 1;
        if (pos < mid) hi = mid; else { lo = mid; k |= 1; }
    }
    return k;
}

// Alg 5.1: split axis = first maximiser of s_k (b_k - a_k) (reading G9).  The lists are sorted by
// coordinate inside every node segment, so the bounding box is read off the segment ends.
__device__ __forceinline__ int kd_axis(double gamma_bar, double x0, double x1, double y0, double y1, double z0, double z1)
{
    const double ex = __dmul_rn(1.0, __dsub_rn(x1, x0));
    const double ey = __dmul_rn(1.0, __dsub_rn(y1, y0));
    const double ez = __dmul_rn(gamma_bar, __dsub_rn(z1, z0));
    int a = 0;
    double best = ex;
    if (ey > best) { best = ey; a = 1; }
    if (ez > best) { best = ez; a = 2; }
    return a;
}

// ---------------------------------------------------------------------------------------
// sort keys
// ---------------------------------------------------------------------------------------
// total order of doubles as unsigned keys; -0.0 == +0.0 (the oracle compares with <, so they tie)
__device__ __forceinline__ uint64_t sortable_key(double v)
{
    v = v + 0.0;  // -0.0 -> +0.0
    uint64_t b = (uint64_t)__double_as_longlong(v);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}

__global__ void kd_keys64(int N, const double *__restrict__ x, const double *__restrict__ y, const double *__restrict__ z,
                          uint64_t *__restrict__ keys /* [3 N] */, uint32_t *__restrict__ lists /* [4 N] */)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    keys[i] = sortable_key(x[i]);
    keys[(size_t)N + i] = sortable_key(y[i]);
    keys[2 * (size_t)N + i] = sortable_key(z[i]);
#pragma unroll
    for (int a = 0; a < 4; ++a) lists[(size_t)a * N + i] = (uint32_t)i;
}

// q = min(floor((c - lo) * 2^32 / (hi - lo)), 2^32 - 1): every step is monotone in c, so c1 <= c2 implies q1 <= q2
__global__ void kd_keys32(int N, const double *__restrict__ x, const double *__restrict__ y, const double *__restrict__ z,
                          const fmm_hdr *__restrict__ hdr, uint32_t *__restrict__ keys /* [3 N] */, uint32_t *__restrict__ lists /* [4 N] */)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double c[3] = {x[i], y[i], z[i]};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double lo = hdr->mm[a], ext = hdr->mm[3 + a] - lo;
        const double scale = (ext > 0.0) ? 4294967296.0 / ext : 0.0;
        double f = floor((c[a] - lo) * scale);
        f = fmin(f, 4294967295.0);
        keys[(size_t)a * N + i] = (f > 0.0) ? (uint32_t)f : 0u;  // (NaN / negative -> 0; non-finite inputs are refused later)
        lists[(size_t)a * N + i] = (uint32_t)i;
    }
    lists[3 * (size_t)N + i] = (uint32_t)i;
}

// After the stable sort by the quantised key a run of equal keys is in index order; the tree wants (coordinate, index).
// kd_find_runs (read-only): the thread at the FIRST out-of-order position of a run records the run; kd_fix_runs: one thread
// per recorded run puts it in order (insertion sort on the indices, at most KD_RUN entries).  Longer runs that are out of
// order raise hdr->kd_fallback (the build is redone with exact keys).
#define KD_RUN 64
__global__ void kd_find_runs(int N, const double *__restrict__ x, const double *__restrict__ y, const double *__restrict__ z,
                             const uint32_t *__restrict__ keys /* [3 N] sorted */, const uint32_t *__restrict__ lists,
                             fmm_hdr *__restrict__ hdr, unsigned int *__restrict__ nruns, uint2 *__restrict__ runs /* (axis N + head, end) */)
{
    const int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= 3 * (int64_t)N) return;
    const int a = (int)(g / N), j = (int)(g - (int64_t)a * N);
    if (j == 0) return;
    const uint32_t *K = keys + (size_t)a * N;
    const uint32_t *V = lists + (size_t)a * N;
    const double *coord = (a == 0) ? x : (a == 1) ? y : z;
    const uint32_t q = K[j];
    if (K[j - 1] != q) return;
    if (!(coord[V[j]] < coord[V[j - 1]])) return;  // in order here
    // first violation of its run?  walk back to the head of the run
    int h = j - 1;
    while (h > 0 && K[h - 1] == q) {
        if (j - h > KD_RUN) { hdr->kd_fallback = 1; return; }
        if (coord[V[h]] < coord[V[h - 1]]) return;  // an earlier violation: that thread records the run
        --h;
    }
    int e = j + 1;
    while (e < N && K[e] == q) {
        if (e - h > KD_RUN) { hdr->kd_fallback = 1; return; }
        ++e;
    }
    const unsigned int slot = atomicAdd(nruns, 1u);
    runs[slot] = make_uint2((unsigned int)a * (unsigned int)N + (unsigned int)h, (unsigned int)a * (unsigned int)N + (unsigned int)e);
}

__global__ void kd_fix_runs(int N, const double *__restrict__ x, const double *__restrict__ y, const double *__restrict__ z,
                            const unsigned int *__restrict__ nruns, const uint2 *__restrict__ runs, uint32_t *__restrict__ lists)
{
    const unsigned int n = *nruns;
    for (unsigned int r = blockIdx.x * blockDim.x + threadIdx.x; r < n; r += gridDim.x * blockDim.x) {
        const uint2 run = runs[r];
        const int a = (int)(run.x / (unsigned int)N);
        const double *coord = (a == 0) ? x : (a == 1) ? y : z;
        uint32_t *V = lists;
        for (unsigned int k = run.x + 1; k < run.y; ++k) {  // [head, k) is in (coordinate, index) order; equals keep ascending index
            const uint32_t v = V[k];
            const double cv = coord[v];
            unsigned int m = k;
            while (m > run.x && cv < coord[V[m - 1]]) { V[m] = V[m - 1]; --m; }
            V[m] = v;
        }
    }
}

// ---------------------------------------------------------------------------------------
// small bunches (N <= KD_LOCAL): the three sorts in one launch, one block per axis, bitonic network on the exact
// (coordinate key, index) pairs -- the 4-pass radix sort is 16 launches, which at N = 4,096 is most of the tree time.
// A thread keeps four consecutive elements in registers: partner distances 1 and 2 are exchanged in registers, 4 .. 64
// by warp shuffles (the partner thread is in the same warp), and only distances >= 128 go through shared memory with
// block barriers (15 of the 78 stages at 4,096 elements).
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ bool kss_greater(uint64_t ka, uint32_t va, uint64_t kb, uint32_t vb)  // (coordinate, index): a total order
{
    return ka > kb || (ka == kb && va > vb);
}

__global__ void __launch_bounds__(1024) kd_sort_small(int N, int npow2 /* >= 128 */, const double *__restrict__ x, const double *__restrict__ y,
                                                      const double *__restrict__ z, uint32_t *__restrict__ lists /* [4 N] */)
{
    extern __shared__ __align__(16) unsigned char kss_raw[];
    uint64_t *skey = reinterpret_cast<uint64_t *>(kss_raw);          // [npow2]
    uint32_t *sval = reinterpret_cast<uint32_t *>(skey + npow2);     // [npow2]
    const int a = blockIdx.x, t = threadIdx.x;
    const bool active = 4 * t < npow2;  // (whole warps: npow2 / 4 is a multiple of 32)
    const double *coord = (a == 0) ? x : (a == 1) ? y : z;
    uint64_t key[4];
    uint32_t val[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const int i = 4 * t + e;
        key[e] = (i < N) ? sortable_key(coord[i]) : ~0ull;  // padding sorts last (index beyond every particle)
        val[e] = (uint32_t)i;
    }
    if (a == 0)
        for (int i = t; i < N; i += blockDim.x) lists[3 * (size_t)N + i] = (uint32_t)i;
    for (int k = 2; k <= npow2; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            if (j >= 128) {  // the partner thread t ^ (j / 4) sits in another warp
                if (active) {
#pragma unroll
                    for (int e = 0; e < 4; ++e) { skey[4 * t + e] = key[e]; sval[4 * t + e] = val[e]; }
                }
                __syncthreads();
                if (active) {
                    const int pt = t ^ (j >> 2);
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const int i = 4 * t + e;
                        const uint64_t pk = skey[4 * pt + e];
                        const uint32_t pv = sval[4 * pt + e];
                        const bool g = kss_greater(key[e], val[e], pk, pv);
                        const bool want_min = ((i & j) == 0) == ((i & k) == 0);
                        if (want_min == g) { key[e] = pk; val[e] = pv; }
                    }
                }
                __syncthreads();
            } else if (j >= 4) {  // same warp: lane ^ (j / 4)
                if (active) {
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const int i = 4 * t + e;
                        const uint64_t pk = __shfl_xor_sync(0xffffffffu, key[e], j >> 2);
                        const uint32_t pv = __shfl_xor_sync(0xffffffffu, val[e], j >> 2);
                        const bool g = kss_greater(key[e], val[e], pk, pv);
                        const bool want_min = ((i & j) == 0) == ((i & k) == 0);
                        if (want_min == g) { key[e] = pk; val[e] = pv; }
                    }
                }
            } else {  // both elements in this thread's registers (k >= 4: one direction for the thread's four elements)
                const bool asc = ((4 * t) & k) == 0;
#define KSS_CX(E, F, UP)                                                     \
    if (kss_greater(key[E], val[E], key[F], val[F]) == (UP)) {               \
        const uint64_t tk = key[E]; key[E] = key[F]; key[F] = tk;            \
        const uint32_t tv = val[E]; val[E] = val[F]; val[F] = tv;            \
    }
                if (j == 2) { KSS_CX(0, 2, asc) KSS_CX(1, 3, asc) }
                else if (k > 2) { KSS_CX(0, 1, asc) KSS_CX(2, 3, asc) }
                else { KSS_CX(0, 1, true) KSS_CX(2, 3, false) }
#undef KSS_CX
            }
        }
    }
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const int i = 4 * t + e;
        if (i < N) lists[(size_t)a * N + i] = val[e];
    }
}

// ---------------------------------------------------------------------------------------
// one level on the whole lists (nodes larger than KD_LOCAL: a tile of KD_TILE entries meets at most two nodes)
// ---------------------------------------------------------------------------------------
// Alg 5.2 (readings G7, G8): in the list of the split axis the first ceil(size/2) members of the
// node (ranked by (coordinate, index)) go to the left child: their bits are set.
__global__ void __launch_bounds__(256) kd_mark(int N, int level, int stop_level, int N0, const double *__restrict__ x, const double *__restrict__ y,
                                               const double *__restrict__ z, const uint32_t *__restrict__ lists,
                                               const fmm_hdr *__restrict__ hdr, uint32_t *__restrict__ bits,
                                               uint8_t *__restrict__ node_axis /* [2^level] */)
{
    __shared__ int s_lo[2], s_hi[2], s_axis[2], s_node[2];
    __shared__ double s_ext[2][6];
    const int start = blockIdx.x * KD_TILE, end = min(N, start + KD_TILE);
    if (start >= N) return;
    if (threadIdx.x < 12) {  // the (at most two) nodes of this tile: six segment ends each, fetched by twelve threads at once
        const int k = threadIdx.x / 6, e = threadIdx.x - 6 * k, a = e >> 1;
        int lo, hi;
        const int node = kd_range_of(N, level, k == 0 ? start : end - 1, lo, hi);
        const double *coord = (a == 0) ? x : (a == 1) ? y : z;
        s_ext[k][e] = coord[lists[(size_t)a * N + ((e & 1) ? hi - 1 : lo)]];
        if (e == 0) { s_lo[k] = lo; s_hi[k] = hi; s_node[k] = node; }
    }
    __syncthreads();
    if (threadIdx.x < 2) {
        const double *v = s_ext[threadIdx.x];
        s_axis[threadIdx.x] = kd_axis(hdr->gamma_bar, v[0], v[1], v[2], v[3], v[4], v[5]);
        node_axis[s_node[threadIdx.x]] = (uint8_t)s_axis[threadIdx.x];  // (every tile of a node writes the same value)
    }
    __syncthreads();
    for (int i = start + threadIdx.x; i < end; i += 256) {
        const int k = (i >= s_hi[0]) ? 1 : 0;
        const int lo = s_lo[k], hi = s_hi[k];
        const int mid = fmm_split_mid(lo, hi, level, stop_level, N0);
        if (i < mid) {
            const uint32_t p = lists[(size_t)s_axis[k] * N + i];
            atomicOr(&bits[p >> 5], 1u << (p & 31));
        }
    }
}

__device__ __forceinline__ int kd_block_scan_256(int v, int *total, int *sm /* [8] */)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    __syncthreads();
    if (lane == 31) sm[warp] = inc;
    __syncthreads();
    int wb = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) {
        const int t = sm[w];
        if (w < warp) wb += t;
        tot += t;
    }
    *total = tot;
    return wb + inc - v;
}

// stable split of every node segment of the four lists: left members first.  Single pass with a decoupled look-back: a
// tile publishes the number of left members of its last node (as a final running count if that node starts inside the
// tile), a tile whose first node began earlier walks back over the published words until it meets a running count, and
// then publishes its own.  In the list of a node's split axis the left members are simply the first ceil(size/2)
// entries: no look-up in the bit mask there.
#define KD_PUB_AGG 1ull
#define KD_PUB_RUN 2ull
__device__ __forceinline__ unsigned long long kd_pub_word(int level, unsigned long long status, int value)
{
    return ((unsigned long long)(level + 1) << 40) | (status << 32) | (unsigned long long)(unsigned int)value;
}

__global__ void __launch_bounds__(256, 6) kd_split(int N, int level, int stop_level, int N0, int tiles_per_list, const uint32_t *__restrict__ bits,
                                                   const uint8_t *__restrict__ node_axis, const uint32_t *__restrict__ cur,
                                                   uint32_t *__restrict__ nxt, unsigned long long *pub /* [4 tiles_per_list] */)
{
    __shared__ int sm[8];
    __shared__ int s_carry;
    __shared__ uint32_t stage[KD_TILE];
    // tile = block index: a tile only waits for tiles with smaller indices, and blocks of a 1-D grid start in index
    // order, so the tiles it waits for are running or done (the assumption of every single-pass look-back scan).
    // The tiles of list li are shifted by sh entries so that a thread's eight entries are two aligned 16-byte words.
    const int li = blockIdx.y, t = blockIdx.x, tile = li * tiles_per_list + t;
    const int sh = (int)(((size_t)li * (size_t)N) & 3);
    const int start = max(0, t * KD_TILE - sh), end = min(N, (t + 1) * KD_TILE - sh);
    if (start >= end) {  // (only the last tile of a list can be empty)
        if (threadIdx.x == 0) atomicExch(&pub[tile], kd_pub_word(level, KD_PUB_RUN, 0));
        return;
    }
    int loA, hiA, hiB;
    const int nodeA = kd_range_of(N, level, start, loA, hiA);
    hiB = hiA;
    if (hiA < end) {
        int lo2;
        kd_range_of(N, level, hiA, lo2, hiB);
    }
    const int midA = fmm_split_mid(loA, hiA, level, stop_level, N0), midB = fmm_split_mid(hiA, hiB, level, stop_level, N0);
    const bool axisA = node_axis[nodeA] == li, axisB = (hiA < end) && node_axis[nodeA + 1] == li;
    const uint32_t *L = cur + (size_t)li * N;
    uint32_t *O = nxt + (size_t)li * N;
    const int i0 = t * KD_TILE - sh + threadIdx.x * 8;
    uint32_t part[8];
    if (i0 >= 0 && i0 + 8 <= N) {
        const uint4 v0 = *reinterpret_cast<const uint4 *>(L + i0), v1 = *reinterpret_cast<const uint4 *>(L + i0 + 4);
        part[0] = v0.x; part[1] = v0.y; part[2] = v0.z; part[3] = v0.w;
        part[4] = v1.x; part[5] = v1.y; part[6] = v1.z; part[7] = v1.w;
    } else {
#pragma unroll
        for (int k = 0; k < 8; ++k) part[k] = (i0 + k >= 0 && i0 + k < N) ? L[i0 + k] : 0u;
    }
    unsigned int flags = 0;
    int s = 0, sA = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const int i = i0 + k;
        unsigned int f = 0;
        if (i >= start && i < end) {
            const bool inA = i < hiA;
            if (inA ? axisA : axisB) f = (unsigned int)(i < (inA ? midA : midB));
            else f = (__ldg(&bits[part[k] >> 5]) >> (part[k] & 31)) & 1u;
        }
        flags |= f << k;
        s += (int)f;
        sA += (int)(f && i < hiA);
    }
    int both;  // one scan for both counts: left members in the low half, those of node A in the high half (each <= 2048)
    const int ex = kd_block_scan_256(s | (sA << 16), &both, sm) & 0xffff;
    const int total = both & 0xffff, cA = both >> 16;
    const bool hasB = hiA < end, startsA = loA >= start;
    if (threadIdx.x == 0) {
        if (hasB) atomicExch(&pub[tile], kd_pub_word(level, KD_PUB_RUN, total - cA));          // node B starts here
        else atomicExch(&pub[tile], kd_pub_word(level, startsA ? KD_PUB_RUN : KD_PUB_AGG, total));
    }
    // The tile's entries leave in four runs: left / right members of node A, then of node B.  They are collected in
    // shared memory first so that every run is written with coalesced stores.
    const int endA = min(end, hiA);
    const int nAL = cA, nAR = (endA - start) - cA, nBL = total - cA;
    {
        int running = ex;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int i = i0 + k;
            if (i >= start && i < end) {
                const unsigned int f = (flags >> k) & 1u;
                int slot;
                if (i < hiA) slot = f ? running : nAL + (i - start - running);
                else slot = nAL + nAR + (f ? (running - cA) : nBL + (i - hiA - (running - cA)));
                stage[slot] = part[k];
                running += (int)f;
            }
        }
    }
    // left members of node A in the tiles before this one: warp 0 walks back, 32 tiles per round, to the nearest running count
    if (!startsA && threadIdx.x < 32) {
        const int lane = threadIdx.x;
        const unsigned long long tag = (unsigned long long)(level + 1);
        int carry = 0;
        for (int j = tile - 1;; j -= 32) {
            unsigned long long w = kd_pub_word(level, KD_PUB_RUN, 0);  // (lanes that would leave the list: nothing before it)
            if (j - lane >= li * tiles_per_list) {
                do { w = *((volatile unsigned long long *)&pub[j - lane]); } while ((w >> 40) != tag);
            }
            const unsigned int runs = __ballot_sync(0xffffffffu, ((w >> 32) & 0xffull) == KD_PUB_RUN);
            const int stop = runs ? __ffs(runs) - 1 : 32;  // the nearest tile whose count is final
            int v = (lane <= stop) ? (int)(unsigned int)w : 0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            carry += v;
            if (runs) break;
        }
        if (lane == 0) {
            s_carry = carry;
            if (!hasB) atomicExch(&pub[tile], kd_pub_word(level, KD_PUB_RUN, carry + total));  // node A goes on: its running count
        }
    }
    __syncthreads();
    const int carry = startsA ? 0 : s_carry;
    const int gAL = loA + carry, gAR = midA + (start - loA - carry), gBL = hiA, gBR = midB;
    const int b1 = nAL, b2 = nAL + nAR, b3 = nAL + nAR + nBL, cnt = end - start;
    for (int q = threadIdx.x; q < cnt; q += 256) {
        const int dest = (q < b1) ? gAL + q : (q < b2) ? gAR + (q - b1) : (q < b3) ? gBL + (q - b2) : gBR + (q - b3);
        O[dest] = stage[q];
    }
}

// ---------------------------------------------------------------------------------------
// all remaining levels of one node of at most KD_LOCAL particles in one block
// ---------------------------------------------------------------------------------------
// The node's members are renamed 0 .. m-1 by ascending original index (their order in LI); the three sorted lists and LI
// become arrays of 16-bit local names in shared memory, the left flags a byte array.  Output: the node's part of the
// final particle order (leaves in heap order, ascending index inside, reading T-3).
struct __align__(16) kdl_smem {
    uint32_t ids[KD_LOCAL];          // local name -> particle
    uint16_t L[2][4][KD_LOCAL];      // ping-pong: LX, LY, LZ, LI in local names
    uint16_t F[KD_LOCAL + 8];        // exclusive scan of the flags along one list
    uint8_t flag[KD_LOCAL];
    uint8_t axis[KD_LOCAL];          // split axis per sub-node of the current level
    int scan[KDL_THREADS / 32];
};

__device__ __forceinline__ int kdl_block_scan(int v, int *total, int *sm)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    __syncthreads();
    if (lane == 31) sm[warp] = inc;
    __syncthreads();
    int wb = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < KDL_THREADS / 32; ++w) {
        const int t = sm[w];
        if (w < warp) wb += t;
        tot += t;
    }
    *total = tot;
    return wb + inc - v;
}

// sub-node of [lo, hi) `depth` levels further down that contains position pos; k = its index among the 2^depth sub-nodes
__device__ __forceinline__ void kdl_sub_of(int lo, int hi, int depth, int pos, int &slo, int &shi, int &k)
{
    slo = lo;
    shi = hi;
    k = 0;
    for (int l = 0; l < depth; ++l) {
        const int mid = slo + (shi - slo + 1) / 2;
        k <<= 1;
        if (pos < mid) shi = mid; else { slo = mid; k |= 1; }
    }
}

// ascending sort of the block's m <= KD_LOCAL member ids: thread t holds elements 8 t .. 8 t + 7; a bitonic network with
// partner distances 1, 2, 4 in registers, 8 .. 128 by warp shuffles (partner lane = lane ^ (j / 8)) and >= 256 through `buf`
// (shared memory, block barriers).  Padding (0xffffffff) sorts last.  All KDL_THREADS threads call it.
__device__ __forceinline__ void kdl_sort_ids(uint32_t (&v)[KDL_ITEMS], int npow2 /* >= 256, power of two */, uint32_t *buf)
{
    const int t = threadIdx.x;
    const bool active = KDL_ITEMS * t < npow2;  // (whole warps: npow2 / 8 is a multiple of 32)
    for (int k = 2; k <= npow2; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            if (j >= 32 * KDL_ITEMS) {  // the partner thread t ^ (j / 8) sits in another warp
                if (active) {
#pragma unroll
                    for (int e = 0; e < KDL_ITEMS; ++e) buf[KDL_ITEMS * t + e] = v[e];
                }
                __syncthreads();
                if (active) {
                    const int pt = t ^ (j / KDL_ITEMS);
#pragma unroll
                    for (int e = 0; e < KDL_ITEMS; ++e) {
                        const int i = KDL_ITEMS * t + e;
                        const uint32_t pv = buf[KDL_ITEMS * pt + e];
                        const bool want_min = ((i & j) == 0) == ((i & k) == 0);
                        if (want_min == (v[e] > pv)) v[e] = pv;
                    }
                }
                __syncthreads();
            } else if (j >= KDL_ITEMS) {  // same warp
                if (active) {
#pragma unroll
                    for (int e = 0; e < KDL_ITEMS; ++e) {
                        const int i = KDL_ITEMS * t + e;
                        const uint32_t pv = __shfl_xor_sync(0xffffffffu, v[e], j / KDL_ITEMS);
                        const bool want_min = ((i & j) == 0) == ((i & k) == 0);
                        if (want_min == (v[e] > pv)) v[e] = pv;
                    }
                }
            } else {  // both elements in this thread's registers (compile-time register indices)
                static_assert(KDL_ITEMS == 8, "kdl_sort_ids is written for eight elements per thread");
                const int base = KDL_ITEMS * t;
#define KDL_CX(E, F)                                             \
    {                                                            \
        const bool up = ((base + E) & k) == 0;                   \
        const uint32_t a = v[E], b = v[F];                       \
        if ((a > b) == up) { v[E] = b; v[F] = a; }               \
    }
                if (j == 4) { KDL_CX(0, 4) KDL_CX(1, 5) KDL_CX(2, 6) KDL_CX(3, 7) }
                else if (j == 2) { KDL_CX(0, 2) KDL_CX(1, 3) KDL_CX(4, 6) KDL_CX(5, 7) }
                else { KDL_CX(0, 1) KDL_CX(2, 3) KDL_CX(4, 5) KDL_CX(6, 7) }
#undef KDL_CX
            }
        }
    }
}

__global__ void __launch_bounds__(KDL_THREADS) kd_local(int N, int level0, int kappa, int stop_level, int N0, int li_global, const double *__restrict__ x, const double *__restrict__ y,
                                                        const double *__restrict__ z, const fmm_hdr *__restrict__ hdr,
                                                        const uint32_t *__restrict__ lists, uint16_t *names /* [N] scratch */,
                                                        uint32_t *__restrict__ order)
{
    extern __shared__ __align__(16) unsigned char kdl_raw[];
    kdl_smem &S = *reinterpret_cast<kdl_smem *>(kdl_raw);
    int lo = 0, hi = N;
    for (int b = level0 - 1; b >= 0; --b) {  // node blockIdx.x of level0
        const int mid = lo + (hi - lo + 1) / 2;
        if ((blockIdx.x >> b) & 1) lo = mid; else hi = mid;
    }
    const int m = hi - lo;
    if (m <= 0) return;
    const double gamma_bar = hdr->gamma_bar;
    // local name of a particle = its rank in the node's (ascending) part of LI; the map particle -> name goes through a
    // global scratch array (written and read by this block only; read past L1, which may hold a neighbour's stale line)
    // (the node's part of LI = its member ids in ascending order: taken from the x list and sorted here)
    {
        int npow2 = 32 * KDL_ITEMS;
        while (npow2 < m) npow2 <<= 1;
        uint32_t v[KDL_ITEMS];
#pragma unroll
        for (int e = 0; e < KDL_ITEMS; ++e) {
            const int i = KDL_ITEMS * threadIdx.x + e;
            // li_global: the level kernels carried LI along (small bunches, where sorting here costs more than a fourth list there)
            v[e] = (i < m) ? (li_global ? lists[3 * (size_t)N + lo + i] : lists[lo + i]) : 0xffffffffu;
        }
        if (!li_global) kdl_sort_ids(v, npow2, S.ids);
#pragma unroll
        for (int e = 0; e < KDL_ITEMS; ++e) {
            const int r = KDL_ITEMS * threadIdx.x + e;
            if (r < m) {
                S.ids[r] = v[e];
                S.L[0][3][r] = (uint16_t)r;
                names[v[e]] = (uint16_t)r;
            }
        }
    }
    __syncthreads();
    for (int q = threadIdx.x; q < 3 * m; q += KDL_THREADS) {
        const int a = q / m, i = q - a * m;
        S.L[0][a][i] = __ldcg(&names[lists[(size_t)a * N + lo + i]]);
    }
    __syncthreads();
    int cb = 0;
    for (int level = level0; level < kappa; ++level) {
        const int depth = level - level0, nsub = 1 << depth;
        uint16_t(*Lc)[KD_LOCAL] = S.L[cb];
        uint16_t(*Ln)[KD_LOCAL] = S.L[cb ^ 1];
        // split axis of every sub-node (Alg 5.1) from the ends of its segments
        for (int k = threadIdx.x; k < nsub; k += KDL_THREADS) {
            int slo = lo, shi = hi;
            for (int b = depth - 1; b >= 0; --b) {
                const int mid = slo + (shi - slo + 1) / 2;
                if ((k >> b) & 1) slo = mid; else shi = mid;
            }
            int ax = 0;
            if (shi > slo) {
                const int a0 = slo - lo, a1 = shi - 1 - lo;
                ax = kd_axis(gamma_bar, x[S.ids[Lc[0][a0]]], x[S.ids[Lc[0][a1]]], y[S.ids[Lc[1][a0]]], y[S.ids[Lc[1][a1]]],
                             z[S.ids[Lc[2][a0]]], z[S.ids[Lc[2][a1]]]);
            }
            S.axis[k] = (uint8_t)ax;
        }
        __syncthreads();
        // this thread's positions: KDL_ITEMS consecutive entries; their sub-nodes are the same in all four lists
        const int i0 = threadIdx.x * KDL_ITEMS;
        int slo[KDL_ITEMS], smid[KDL_ITEMS];
        {
            union { uint4 v; uint16_t h[KDL_ITEMS]; } n3[3];  // the thread's entries of LX, LY, LZ (three LDS.128)
#pragma unroll
            for (int a = 0; a < 3; ++a) n3[a].v = *reinterpret_cast<const uint4 *>(&Lc[a][i0]);
#pragma unroll
            for (int k = 0; k < KDL_ITEMS; ++k) {
                const int i = i0 + k;
                slo[k] = smid[k] = 0;
                if (i < m) {
                    int a, b, sk;
                    kdl_sub_of(lo, hi, depth, lo + i, a, b, sk);
                    slo[k] = a - lo;
                    smid[k] = fmm_split_mid(a, b, level, stop_level, N0) - lo;  // (a cluster that stays a leaf keeps its order)
                    const int ax = S.axis[sk];
                    const uint16_t name = (ax == 0) ? n3[0].h[k] : (ax == 1) ? n3[1].h[k] : n3[2].h[k];
                    S.flag[name] = (uint8_t)(i < smid[k]);  // Alg 5.2: the first ceil(size/2) along the split axis go left
                }
            }
        }
        __syncthreads();
        for (int a = 0; a < 4; ++a) {
            // the thread's KDL_ITEMS = 8 consecutive 16-bit names are one 16-byte word: LDS.128 / STS.128 without bank conflicts
            union { uint4 v; uint16_t h[KDL_ITEMS]; } rr, ff;
            rr.v = *reinterpret_cast<const uint4 *>(&Lc[a][i0]);
            uint16_t r[KDL_ITEMS];
            unsigned int fl = 0;
            int s = 0;
#pragma unroll
            for (int k = 0; k < KDL_ITEMS; ++k) {
                const int i = i0 + k;
                r[k] = (i < m) ? rr.h[k] : (uint16_t)0;
                const unsigned int f = (i < m) ? S.flag[r[k]] : 0u;
                fl |= f << k;
                s += (int)f;
            }
            int total;
            int run = kdl_block_scan(s, &total, S.scan);
#pragma unroll
            for (int k = 0; k < KDL_ITEMS; ++k) {
                ff.h[k] = (uint16_t)run;
                run += (int)((fl >> k) & 1u);
            }
            *reinterpret_cast<uint4 *>(&S.F[i0]) = ff.v;  // (entries beyond m are never read)
            __syncthreads();
#pragma unroll
            for (int k = 0; k < KDL_ITEMS; ++k) {
                const int i = i0 + k;
                if (i < m) {
                    const int before = (int)ff.h[k] - (int)S.F[slo[k]];  // left members of the sub-node before entry i
                    const unsigned int f = (fl >> k) & 1u;
                    Ln[a][f ? (slo[k] + before) : (smid[k] + (i - slo[k] - before))] = r[k];
                }
            }
            __syncthreads();
        }
        cb ^= 1;
    }
    for (int i = threadIdx.x; i < m; i += KDL_THREADS) order[lo + i] = S.ids[S.L[cb][3][i]];
}

// ---------------------------------------------------------------------------------------
// host: particle order of the KD tree into `order` ([N], scratch from the arena)
// ---------------------------------------------------------------------------------------
int kd_build_order(fmm_plan *p, const fmm_particles_t *in, uint32_t **order_out)
{
    fmm_ctx *c = &p->ctx;
    cudaStream_t st = c->stream;
    const int N = (int)p->N, T = 256, gN = (N + T - 1) / T;
    uint32_t *lists = (uint32_t *)ctx_alloc(c, sizeof(uint32_t) * 4 * (size_t)N);  // LX, LY, LZ, LI
    uint32_t *lists2 = (uint32_t *)ctx_alloc(c, sizeof(uint32_t) * 4 * (size_t)N);
    if (!lists || !lists2) return FMM_ENOMEM;
    if (p->kappa == 0) {  // the root is a leaf: index order
        uint32_t *k32 = (uint32_t *)ctx_alloc(c, sizeof(uint32_t) * 3 * (size_t)N);
        if (!k32) return FMM_ENOMEM;
        kd_keys32<<<gN, T, 0, st>>>(N, in->x, in->y, in->z, p->hdr, k32, lists);
        FMM_LAUNCH_CHECK(c, "kd_keys32");
        *order_out = lists + 3 * (size_t)N;
        return FMM_OK;
    }
    if (N <= KD_LOCAL) {  // one launch for the three sorts
        int npow2 = 128;  // (four elements per thread, whole warps)
        while (npow2 < N) npow2 <<= 1;
        const size_t smem = (size_t)npow2 * 12;
        if (smem > 40 * 1024) FMM_CUDA(c, cudaFuncSetAttribute((const void *)kd_sort_small, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kd_sort_small<<<3, 1024, smem, st>>>(N, npow2, in->x, in->y, in->z, lists);
        FMM_LAUNCH_CHECK(c, "kd_sort_small");
    } else if (p->kd_exact) {  // exact 64-bit keys: 8 radix passes
        uint64_t *keys = (uint64_t *)ctx_alloc(c, sizeof(uint64_t) * 3 * (size_t)N);
        uint64_t *tkeys = (uint64_t *)ctx_alloc(c, sizeof(uint64_t) * 3 * (size_t)N);
        if (!keys || !tkeys) return FMM_ENOMEM;
        kd_keys64<<<gN, T, 0, st>>>(N, in->x, in->y, in->z, keys, lists);
        FMM_LAUNCH_CHECK(c, "kd_keys64");
        FMM_TRY(sort_pairs_u64_batched(c, keys, lists, tkeys, lists2, N, 3, 0, 64));
        ctx_free(c, tkeys);
        ctx_free(c, keys);
    } else {
        uint32_t *k32 = (uint32_t *)ctx_alloc(c, sizeof(uint32_t) * 3 * (size_t)N);
        uint32_t *t32 = (uint32_t *)ctx_alloc(c, sizeof(uint32_t) * 3 * (size_t)N);
        if (!k32 || !t32) return FMM_ENOMEM;
        kd_keys32<<<gN, T, 0, st>>>(N, in->x, in->y, in->z, p->hdr, k32, lists);
        FMM_LAUNCH_CHECK(c, "kd_keys32");
        FMM_TRY(sort_pairs_u32_batched(c, k32, lists, t32, lists2, N, 3));
        // (3 N <= 2^32 - 1: positions axis N + j fit 32 bits because sort_pairs_u32_batched requires 3 N < 2^31)
        unsigned int *nruns = (unsigned int *)ctx_alloc(c, sizeof(unsigned int) * 2 + sizeof(uint2) * (3 * (size_t)N / 2 + 2));
        if (!nruns) return FMM_ENOMEM;
        uint2 *runs = reinterpret_cast<uint2 *>(nruns + 2);
        FMM_CUDA(c, cudaMemsetAsync(nruns, 0, sizeof(unsigned int) * 2, st));
        kd_find_runs<<<(unsigned)((3 * (int64_t)N + T - 1) / T), T, 0, st>>>(N, in->x, in->y, in->z, k32, lists, p->hdr, nruns, runs);
        FMM_LAUNCH_CHECK(c, "kd_find_runs");
        kd_fix_runs<<<FMM_SM_COUNT, 128, 0, st>>>(N, in->x, in->y, in->z, nruns, runs, lists);
        FMM_LAUNCH_CHECK(c, "kd_fix_runs");
        ctx_free(c, nruns);
        ctx_free(c, t32);
        ctx_free(c, k32);
    }
    // levels on the whole lists while a node holds more than KD_LOCAL particles ...
    int level0 = 0;
    while (level0 < p->kappa && (((int64_t)N + ((int64_t)1 << level0) - 1) >> level0) > KD_LOCAL) ++level0;
    // LI through the level kernels, or rebuilt by kd_local from its members (one shared-memory sort per block): the sort pays
    // from about 2^19 particles on (N = 2^20: a0-a2 0.725 -> 0.710 ms, N = 2.56e7: 15.3 -> 14.4 ms; N = 65,536: +25 us)
    // (FMM_TEST_KD_SORT_LI: the tests take the sorting route on small bunches too)
    const int li_global = (level0 == p->kappa || level0 == 0 || (N < (1 << 19) && !getenv("FMM_TEST_KD_SORT_LI"))) ? 1 : 0;
    uint32_t *cur = lists, *nxt = lists2;
    if (level0 > 0) {
        const int tiles = (N + 3 + KD_TILE - 1) / KD_TILE;  // (tiles of a list are shifted by up to three entries, see kd_split)
        const size_t nbits = ((size_t)N + 31) / 32;
        uint32_t *bits = (uint32_t *)ctx_alloc(c, sizeof(uint32_t) * nbits);
        unsigned long long *pub = (unsigned long long *)ctx_alloc(c, sizeof(unsigned long long) * 4 * (size_t)tiles);
        uint8_t *node_axis = (uint8_t *)ctx_alloc(c, (size_t)1 << level0);
        if (!bits || !pub || !node_axis) return FMM_ENOMEM;
        FMM_CUDA(c, cudaMemsetAsync(pub, 0, sizeof(unsigned long long) * 4 * (size_t)tiles, st));
        for (int level = 0; level < level0; ++level) {
            FMM_CUDA(c, cudaMemsetAsync(bits, 0, sizeof(uint32_t) * nbits, st));
            kd_mark<<<tiles, 256, 0, st>>>(N, level, p->stop_level, p->N0, in->x, in->y, in->z, cur, p->hdr, bits, node_axis);
            FMM_LAUNCH_CHECK(c, "kd_mark");
            kd_split<<<dim3(tiles, li_global ? 4 : 3), 256, 0, st>>>(N, level, p->stop_level, p->N0, tiles, bits, node_axis, cur, nxt, pub);
            FMM_LAUNCH_CHECK(c, "kd_split");
            uint32_t *t = cur; cur = nxt; nxt = t;
        }
    }
    // ... then one block per node for the rest
    if (level0 < p->kappa) {
        const size_t smem = sizeof(kdl_smem);
        FMM_CUDA(c, cudaFuncSetAttribute((const void *)kd_local, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        uint32_t *order = nxt;  // (the other list buffer is free now: [0, N) takes the order, the rest the name map)
        uint16_t *names = reinterpret_cast<uint16_t *>(nxt + (size_t)N);
        kd_local<<<1u << level0, KDL_THREADS, smem, st>>>(N, level0, p->kappa, p->stop_level, p->N0, li_global, in->x, in->y, in->z, p->hdr, cur, names, order);
        FMM_LAUNCH_CHECK(c, "kd_local");
        *order_out = order;
    } else {
        *order_out = cur + 3 * (size_t)N;  // the index-ordered list: leaves in heap order, ascending index inside (T-3)
    }
    return FMM_OK;
}
