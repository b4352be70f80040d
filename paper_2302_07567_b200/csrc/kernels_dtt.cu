// kernels_dtt.cu -- step a3: dual tree traversal (Alg 9.1; same logic as Alg 5.11,
// PAPER.md:400-435) with the stretched admissibility condition of Alg 5.6-5.8 (PAPER.md:337-366,
// eq. (4.3)), emitting the two interaction lists in CSR form sorted by
// (target, source) (readings D-4, G20).
//
// The recursion runs in two kernels: one block expands the pair (root, root) breadth-first (classify every pair of
// the frontier as P2P / M2L / split, block barrier, next frontier) until the frontier holds a few thousand pairs;
// then every such pair is walked depth-first by one warp with a stack in shared memory.  Pairs are emitted through INTEGER
// atomic counters and count into their target's row length.  The order of emission is irrelevant: rows are laid out
// from the scanned row lengths and then sorted by source, so the lists are unique and bit-reproducible.  One host
// wait per build, at its very end (list lengths, gamma_bar, the input check).
#include "fmm_internal.cuh"

#include <stdlib.h>

#include <cooperative_groups.h>
namespace cg = cooperative_groups;

struct dtt_counters {           // device
    unsigned int n_p2p, n_m2l, overflow, pad;
    unsigned int n_front[72];   // frontier sizes per step (at most 2*kappa+2 steps)
    unsigned long long evals;   // particle pairs of the whole P2P list
    unsigned long long max_row; // particle pairs of the heaviest target leaf
};

struct dtt_args {
    int nsteps, leaves, key_shift, treecode_leaves;
    int early_first, N0;        // FMM_TREE_STOP_AT_N0: a node >= early_first (level kappa-1) with at most N0 particles is a leaf (else INT_MAX)
    unsigned int roots;         // breadth-first until the frontier holds this many pairs, then one depth-first walk per pair
    double theta2;
    const fmm_hdr *hdr;
    const int32_t *node_lo, *node_hi;
    const double *geo;
    uint64_t *front0, *front1, *p2p, *m2l;
    unsigned int cap;
    int32_t *rows;              // [2][rows_len] row lengths: P2P by target leaf id, then M2L by target node id
    int32_t *row_work;          // [leaves] sum of the source leaf sizes of a target leaf's row
    int rows_len;
    dtt_counters *cnt;
};


// one pair of Alg 9.1: 0 = nothing (empty cluster), 1 = P2P, 2 = M2L, 3 = split the target, 4 = split the source
__device__ __forceinline__ int dtt_decide(const dtt_args &a, double gamma_bar, int i, int j, int *nj_out)
{
    const int ni = a.node_hi[i] - a.node_lo[i], nj = a.node_hi[j] - a.node_lo[j];
    *nj_out = nj;
    if (ni <= 0 || nj <= 0) return 0;
    // children(S) empty (Alg 5.2): level kappa, or a cluster of level kappa-1 that was not split (FMM_TREE_STOP_AT_N0)
    const bool leaf_i = i >= a.leaves || (i >= a.early_first && ni <= a.N0), leaf_j = j >= a.leaves || (j >= a.early_first && nj <= a.N0);
    if (leaf_i && leaf_j) return 1;  // D-1: leaf-leaf -> P2P, no admissibility test
    // D-2: Alg 5.6-5.8 squared; every product and sum rounded separately, in this order
    const double *gi = a.geo + 4 * (int64_t)i, *gj = a.geo + 4 * (int64_t)j;
    const double ri = gi[0], rj = gj[0];
    const double ex = __dmul_rn(1.0, __dsub_rn(gi[1], gj[1]));
    const double ey = __dmul_rn(1.0, __dsub_rn(gi[2], gj[2]));
    const double ez = __dmul_rn(gamma_bar, __dsub_rn(gi[3], gj[3]));
    const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(ex, ex), __dmul_rn(ey, ey)), __dmul_rn(ez, ez));
    const double rmax = (ri > rj) ? ri : rj;
    if (rmax < __dmul_rn(a.theta2, d2)) return 2;  // admissible -> M2L
    // D-3: which side to split
    return (leaf_i ? false : (leaf_j ? true : (ri > rj))) ? 3 : 4;
}

// slot in a pair buffer: one atomic per group of threads that arrive together (the counter is a single hot address)
__device__ __forceinline__ unsigned int dtt_slot(unsigned int *counter)
{
    cg::coalesced_group g = cg::coalesced_threads();
    unsigned int base = 0;
    if (g.thread_rank() == 0) base = atomicAdd(counter, (unsigned int)g.size());
    return g.shfl(base, 0) + g.thread_rank();
}

__device__ __forceinline__ void dtt_emit(const dtt_args &a, int kind, int i, int j, int nj)
{
    dtt_counters *cnt = a.cnt;
    if (kind == 1) {
        // a leaf S of level kappa-1 goes by the name of its slot 2S on level kappa, which holds the same particles (fmm_internal.cuh)
        if (i < a.leaves) i *= 2;
        if (j < a.leaves) j *= 2;
        const unsigned int pos = dtt_slot(&cnt->n_p2p);
        if (pos < a.cap) a.p2p[pos] = ((uint64_t)i << a.key_shift) | (uint64_t)j; else cnt->overflow = 1;
        atomicAdd(&a.rows[i], 1);
        atomicAdd(&a.row_work[i - a.leaves], nj);
    } else {
        const unsigned int pos = dtt_slot(&cnt->n_m2l);
        if (pos < a.cap) a.m2l[pos] = ((uint64_t)i << a.key_shift) | (uint64_t)j; else cnt->overflow = 1;
        atomicAdd(&a.rows[a.rows_len + i], 1);
    }
}

// Top of the traversal by ONE block (block barriers between the steps): resets the counters and the row lengths, seeds the
// frontier -- FMM: (root, root); treecode (FMM_METHOD_TREECODE): (t, root) for every leaf t, so the target is never split
// and the "m2l" list becomes the particle-cluster list -- and expands it breadth-first until it holds a.roots pairs.
__global__ void __launch_bounds__(1024) dtt_top(dtt_args a)
{
    __shared__ unsigned int n_in, n_out;
    dtt_counters *cnt = a.cnt;
    const int tid = threadIdx.x, nth = blockDim.x;
    if (tid == 0) {
        cnt->n_p2p = cnt->n_m2l = cnt->overflow = cnt->pad = 0;
        cnt->evals = cnt->max_row = 0ull;
        n_in = a.treecode_leaves > 0 ? (unsigned)a.treecode_leaves : 1u;
        if (a.treecode_leaves <= 0) a.front0[0] = (1ull << 32) | 1ull;
        n_out = 0;
    }
    for (int k = tid; k < 72; k += nth) cnt->n_front[k] = 0;
    for (int k = tid; k < a.treecode_leaves; k += nth) a.front0[k] = ((uint64_t)(a.treecode_leaves + k) << 32) | 1ull;
    for (int k = tid; k < 2 * a.rows_len; k += nth) a.rows[k] = 0;
    for (int k = tid; k < a.leaves; k += nth) a.row_work[k] = 0;
    __threadfence();
    __syncthreads();
    int step = 0;
    if (!a.hdr->nonfinite) {  // NaN / Inf in the inputs: no lists (FMM_ENONFINITE after the read-back)
        const double gamma_bar = a.hdr->gamma_bar;
        for (; step < a.nsteps; ++step) {
            const unsigned int nin = n_in;
            if (nin == 0 || nin >= a.roots || nin > a.cap) break;
            const uint64_t *front_in = (step & 1) ? a.front1 : a.front0;
            uint64_t *front_out = (step & 1) ? a.front0 : a.front1;
            for (unsigned int k = tid; k < nin; k += nth) {
                const uint64_t pr = front_in[k];
                const int i = (int)(pr >> 32), j = (int)(pr & 0xffffffffu);  // i = target, j = source
                int nj;
                const int kind = dtt_decide(a, gamma_bar, i, j, &nj);
                if (kind == 1 || kind == 2) dtt_emit(a, kind, i, j, nj);
                if (kind >= 3) {
                    const unsigned int pos = atomicAdd(&n_out, 2u);
                    if (pos + 1 < a.cap) {
                        front_out[pos] = (kind == 3) ? (((uint64_t)(2 * i) << 32) | (uint64_t)j) : (((uint64_t)i << 32) | (uint64_t)(2 * j));
                        front_out[pos + 1] = (kind == 3) ? (((uint64_t)(2 * i + 1) << 32) | (uint64_t)j) : (((uint64_t)i << 32) | (uint64_t)(2 * j + 1));
                    } else {
                        cnt->overflow = 1;
                    }
                }
            }
            __syncthreads();
            if (tid == 0) { n_in = n_out; n_out = 0; }
            __syncthreads();
        }
    }
    if (tid == 0) {  // what is left for the walks: n_front[0] pairs in buffer (n_front[1] & 1)
        cnt->n_front[0] = a.hdr->nonfinite ? 0u : (n_in > a.cap ? a.cap : n_in);
        cnt->n_front[1] = (unsigned)step;
    }
}

// Rest of the traversal: every pair the top left over is the root of a walk by one WARP.  The warp keeps a stack of pairs
// in shared memory, takes up to 32 pairs off its top per round (one per lane), classifies them and pushes the children of
// the pairs that split: depth-first in blocks of 32, so the stack stays short while all lanes have work.  A stack that
// would overflow hands the children to a global buffer instead, which a second launch walks the same way.
#define DTT_WALK_WARPS 4
#define DTT_WSTACK 512
__global__ void __launch_bounds__(32 * DTT_WALK_WARPS) dtt_walk(dtt_args a, int pass, int wstack /* <= DTT_WSTACK */)
{
    __shared__ uint64_t stk_all[DTT_WALK_WARPS][DTT_WSTACK];
    dtt_counters *cnt = a.cnt;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint64_t *stk = stk_all[warp];
    // pass 0: roots left by dtt_top in buffer (n_front[1] & 1), spill into the other buffer counted by n_front[2];
    // pass 1: walks that spill; anything it would spill again is reported as an overflow (larger buffers, new traversal)
    const int rb = (int)(cnt->n_front[1] & 1) ^ pass;
    const unsigned int nroots = pass == 0 ? cnt->n_front[0] : (cnt->n_front[2] > a.cap ? a.cap : cnt->n_front[2]);
    const uint64_t *roots = rb ? a.front1 : a.front0;
    uint64_t *spill = rb ? a.front0 : a.front1;
    if (nroots == 0) return;
    const double gamma_bar = a.hdr->gamma_bar;
    const unsigned int lt = (1u << lane) - 1u;
    // the sub-trees differ a lot in size: warps take the next root from a counter instead of a fixed share
    for (;;) {
        unsigned int r = 0;
        if (lane == 0) r = atomicAdd(&cnt->n_front[4 + pass], 1u);
        r = __shfl_sync(0xffffffffu, r, 0);
        if (r >= nroots) break;
        int top = 1;
        if (lane == 0) stk[0] = roots[r];
        __syncwarp();
        while (top > 0) {
            const int take = top < 32 ? top : 32;
            top -= take;
            const uint64_t pr = lane < take ? stk[top + lane] : 0ull;
            __syncwarp();
            const int i = (int)(pr >> 32), j = (int)(pr & 0xffffffffu);  // i = target, j = source
            int kind = 0, nj = 0;
            if (lane < take) kind = dtt_decide(a, gamma_bar, i, j, &nj);
            if (kind == 1 || kind == 2) dtt_emit(a, kind, i, j, nj);
            const unsigned int splits = __ballot_sync(0xffffffffu, kind >= 3);
            const int nsplit = __popc(splits);
            if (kind >= 3) {
                const uint64_t c0 = (kind == 3) ? (((uint64_t)(2 * i) << 32) | (uint64_t)j) : (((uint64_t)i << 32) | (uint64_t)(2 * j));
                const uint64_t c1 = (kind == 3) ? (((uint64_t)(2 * i + 1) << 32) | (uint64_t)j) : (((uint64_t)i << 32) | (uint64_t)(2 * j + 1));
                if (top + 2 * nsplit <= wstack) {
                    const int at = top + 2 * __popc(splits & lt);
                    stk[at] = c0;
                    stk[at + 1] = c1;
                } else {  // (warp-uniform condition)
                    const unsigned int pos = atomicAdd(&cnt->n_front[2 + pass], 2u);
                    if (pass == 0 && pos + 1 < a.cap) { spill[pos] = c0; spill[pos + 1] = c1; }
                    else cnt->overflow = 1;
                }
            }
            if (top + 2 * nsplit <= wstack) top += 2 * nsplit;
            __syncwarp();
        }
    }
}

// particle pairs of the P2P list and of its heaviest row (the near-field kernels choose their row split from these)
__global__ void __launch_bounds__(256) dtt_totals(dtt_args a)
{
    const int gtid = blockIdx.x * blockDim.x + threadIdx.x, gsize = gridDim.x * blockDim.x;
    unsigned long long sum = 0, mx = 0;
    for (int k = gtid; k < a.leaves; k += gsize) {
        const int t = a.leaves + k;
        const unsigned long long w = (unsigned long long)(a.node_hi[t] - a.node_lo[t]) * (unsigned long long)a.row_work[k];
        sum += w;
        mx = w > mx ? w : mx;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        sum += __shfl_down_sync(0xffffffffu, sum, o);
        const unsigned long long m2 = __shfl_down_sync(0xffffffffu, mx, o);
        mx = m2 > mx ? m2 : mx;
    }
    if ((threadIdx.x & 31) == 0 && sum) {
        atomicAdd(&a.cnt->evals, sum);
        atomicMax(&a.cnt->max_row, mx);
    }
}

// rows of both lists from the scanned row lengths: offsets, then every emitted pair takes a slot of its target's row
__global__ void csr_offsets(int rows_len, const int32_t *__restrict__ scan /* [2 rows_len] */, int32_t *__restrict__ p2p_off,
                            int32_t *__restrict__ m2l_off)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= rows_len) return;
    p2p_off[k] = scan[k];
    m2l_off[k] = scan[rows_len + k] - scan[rows_len];
}

__global__ void csr_fill(const dtt_counters *__restrict__ cnt, const uint64_t *__restrict__ kp2p, const uint64_t *__restrict__ km2l, int key_shift,
                         int rows_len, const int32_t *__restrict__ p2p_off, const int32_t *__restrict__ m2l_off,
                         int32_t *__restrict__ rows /* remaining slots per row, counted down */, int32_t *__restrict__ p2p_tmp,
                         int32_t *__restrict__ m2l_tmp)
{
    if (cnt->overflow) return;  // (the host enlarges the buffers and runs the traversal again)
    const int64_t n_p2p = cnt->n_p2p, n_all = n_p2p + (int64_t)cnt->n_m2l;
    const uint64_t mask = (1ull << key_shift) - 1ull;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n_all; k += (int64_t)gridDim.x * blockDim.x) {
        if (k < n_p2p) {
            const uint64_t key = kp2p[k];
            const int t = (int)(key >> key_shift);
            const int slot = atomicSub(&rows[t], 1) - 1;
            p2p_tmp[p2p_off[t] + slot] = (int32_t)(key & mask);
        } else {
            const uint64_t key = km2l[k - n_p2p];
            const int t = (int)(key >> key_shift);
            const int slot = atomicSub(&rows[rows_len + t], 1) - 1;
            m2l_tmp[m2l_off[t] + slot] = (int32_t)(key & mask);
        }
    }
}

// One block per row: ascending source ids (the sources of a row are distinct, so the rank of an entry is the number of
// smaller ones).  Rows are short (tens of entries with the KD tree, at most a few thousand with MORTON_MEDIAN).
#define ROWSORT_THREADS 64
__global__ void __launch_bounds__(ROWSORT_THREADS) csr_sort_rows(const dtt_counters *__restrict__ cnt, int first_p2p, int n_rows_p2p, int first_m2l, const int32_t *__restrict__ p2p_off,
                                                                 const int32_t *__restrict__ m2l_off, const int32_t *__restrict__ p2p_tmp,
                                                                 const int32_t *__restrict__ m2l_tmp, int32_t *__restrict__ p2p_src,
                                                                 int32_t *__restrict__ m2l_src, int32_t *__restrict__ p2p_tgt)
{
    __shared__ int32_t sm[1024];
    if (cnt->overflow) return;
    const bool is_p2p = (int)blockIdx.x < n_rows_p2p;
    const int t = is_p2p ? first_p2p + blockIdx.x : first_m2l + (blockIdx.x - n_rows_p2p);
    const int32_t *off = is_p2p ? p2p_off : m2l_off;
    const int a = off[t], m = off[t + 1] - a;
    if (m <= 0) return;
    const int32_t *in = (is_p2p ? p2p_tmp : m2l_tmp) + a;
    int32_t *out = (is_p2p ? p2p_src : m2l_src) + a;
    const bool staged = m <= 1024;
    if (staged) {
        for (int k = threadIdx.x; k < m; k += ROWSORT_THREADS) sm[k] = in[k];
        __syncthreads();
    }
    const int32_t *row = staged ? sm : in;
    for (int k = threadIdx.x; k < m; k += ROWSORT_THREADS) {
        const int32_t v = row[k];
        int rank = 0;
        for (int q = 0; q < m; ++q) rank += row[q] < v;
        out[rank] = v;
        if (is_p2p && p2p_tgt) p2p_tgt[a + rank] = t;
    }
}

// ---------------------------------------------------------------------------------------
// Mutual near field ("P2P"): the kernel of eq. (3.2) depends on the pair only through x_i - x_j and
// gamma_bar, so g(x_j, x_i) = -g(x_i, x_j): when the P2P list holds both (t, s) and (s, t), one block evaluates
// D^{-3/2} once per particle pair and forms both sums.  Entry kinds, per list entry e = (t, s):
//   dst[e] = -1  one-sided: s == t, or (s, t) is not in the list (possible after a radius tie in Alg 5.11, reading D-3)
//   dst[e] >= 0  t owns the pair {t, s}: its block also sums the reaction on the particles of s and writes it to the
//                partial segment [dst[e], dst[e] + |s|) that the entry (s, t) receives
//   dst[e] = -2  s owns the pair: nothing to do for block t; recv[e] >= 0 is the segment holding the sums for t's particles
// Ownership alternates with the parity of t + s so that every leaf owns about half of its row.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ int p2p_pair_owner(int t, int s)
{
    const int lo = t < s ? t : s, hi = t < s ? s : t;
    return ((lo + hi) & 1) ? hi : lo;
}

__global__ void p2p_mates(const dtt_counters *__restrict__ cnt, int64_t cap, const int32_t *__restrict__ off, const int32_t *__restrict__ src,
                          const int32_t *__restrict__ tgt, const int32_t *__restrict__ node_lo, const int32_t *__restrict__ node_hi,
                          int32_t *__restrict__ mate, int32_t *__restrict__ len /* [cap], zero beyond the list */)
{
    const int64_t n = cnt->overflow ? 0 : (int64_t)cnt->n_p2p;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < cap; e += (int64_t)gridDim.x * blockDim.x) {
        if (e >= n) { len[e] = 0; continue; }
        const int t = tgt[e], s = src[e];
        int m = -1;
        if (s != t) {  // row s is sorted by source: binary search for t
            int a = off[s], b = off[s + 1];
            while (a < b) {
                int mid = (a + b) >> 1;
                int v = src[mid];
                if (v < t) a = mid + 1; else b = mid;
            }
            if (a < off[s + 1] && src[a] == t) m = a;
        }
        mate[e] = m;
        len[e] = (m >= 0 && p2p_pair_owner(t, s) != t) ? (node_hi[t] - node_lo[t]) : 0;  // non-empty clusters only reach the list
    }
}

__global__ void p2p_segments(const dtt_counters *__restrict__ cnt, const int32_t *__restrict__ mate, const int32_t *__restrict__ len,
                             const int32_t *__restrict__ scan, int32_t *__restrict__ dst, int32_t *__restrict__ recv)
{
    const int64_t n = cnt->overflow ? 0 : (int64_t)cnt->n_p2p;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
        const int m = mate[e];
        recv[e] = len[e] > 0 ? scan[e] : -1;
        dst[e] = (m < 0) ? -1 : (len[e] > 0 ? -2 : scan[m]);
    }
}

// LPT block order: targets by descending work.  The order only needs a coarse, deterministic ranking: an 8-bit monotone
// code of the work (5-bit exponent, 3-bit mantissa), so the sort is a single radix pass.
__global__ void list_work_keys(const dtt_counters *__restrict__ cnt, int first, int count, const int32_t *__restrict__ off, const int32_t *__restrict__ src,
                               const int32_t *__restrict__ node_lo, const int32_t *__restrict__ node_hi, int by_size,
                               const int32_t *__restrict__ dst /* P2P entry kinds, or NULL */,
                               uint64_t *__restrict__ keys, uint32_t *__restrict__ vals)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= count) return;
    int t = first + k;
    unsigned long long work = 0;
    if (cnt->overflow) {
        work = 0;
    } else if (by_size) {
        // block work in FP64 instructions per particle pair: 25 one-sided, 34 for an owned mutual pair, 0 if the mate owns it
        for (int e = off[t]; e < off[t + 1]; ++e)
            work += (unsigned long long)(node_hi[src[e]] - node_lo[src[e]]) * (unsigned long long)(!dst ? 25 : (dst[e] >= 0 ? 34 : (dst[e] == -1 ? 25 : 0)));
    } else {
        work = (unsigned long long)(off[t + 1] - off[t]);
    }
    unsigned int wq = 0;
    if (work > 0) {
        int e = 63 - __clzll((long long)work);
        if (e > 30) e = 30;
        unsigned long long mant = (e >= 3) ? (work >> (e - 3)) : (work << (3 - e));  // 1.xxx
        if (mant > 15) mant = 15;
        wq = ((unsigned int)e << 3) | (unsigned int)(mant & 7ull);
        wq += 1;  // keep 0 for "no work"
    }
    keys[k] = 0xffull - (unsigned long long)wq;  // ascending sort of this = descending work
    vals[k] = (uint32_t)t;
}

// The same order by ONE block (counting sort on the 8-bit code) for small lists (up to LIST_ORDER_SMALL targets; slower than the sort beyond): five launches less per
// list.  Targets of equal code come out in arbitrary order: the order only schedules blocks, it never enters the arithmetic.
#define LIST_ORDER_SMALL 1024
__global__ void __launch_bounds__(1024) list_order_small(const dtt_counters *__restrict__ cnt, int first, int count, const int32_t *__restrict__ off,
                                                         const int32_t *__restrict__ src, const int32_t *__restrict__ node_lo,
                                                         const int32_t *__restrict__ node_hi, int by_size, const int32_t *__restrict__ dst,
                                                         int32_t *__restrict__ order)
{
    __shared__ int hist[256], cursor[256];
    for (int k = threadIdx.x; k < 256; k += blockDim.x) hist[k] = 0;
    __syncthreads();
    const bool bad = cnt->overflow != 0;
    auto code = [&](int t) -> int {
        unsigned long long work = 0;
        if (bad) {
            work = 0;
        } else if (by_size) {
            for (int e = off[t]; e < off[t + 1]; ++e)
                work += (unsigned long long)(node_hi[src[e]] - node_lo[src[e]]) * (unsigned long long)(!dst ? 25 : (dst[e] >= 0 ? 34 : (dst[e] == -1 ? 25 : 0)));
        } else {
            work = (unsigned long long)(off[t + 1] - off[t]);
        }
        unsigned int wq = 0;
        if (work > 0) {
            int e = 63 - __clzll((long long)work);
            if (e > 30) e = 30;
            unsigned long long mant = (e >= 3) ? (work >> (e - 3)) : (work << (3 - e));
            if (mant > 15) mant = 15;
            wq = (((unsigned int)e << 3) | (unsigned int)(mant & 7ull)) + 1;
        }
        return 255 - (int)wq;  // ascending code = descending work
    };
    for (int k = threadIdx.x; k < count; k += blockDim.x) atomicAdd(&hist[code(first + k)], 1);
    __syncthreads();
    if (threadIdx.x == 0) {
        int run = 0;
        for (int d = 0; d < 256; ++d) { cursor[d] = run; run += hist[d]; }
    }
    __syncthreads();
    for (int k = threadIdx.x; k < count; k += blockDim.x) {
        const int t = first + k;
        order[atomicAdd(&cursor[code(t)], 1)] = t;
    }
}

__global__ void copy_u32_to_i32(int n, const uint32_t *__restrict__ a, int32_t *__restrict__ b)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) b[k] = (int32_t)a[k];
}

static int make_order(fmm_plan *p, const dtt_counters *cnt, int first, int count, const int32_t *off, const int32_t *src, int by_size,
                      const int32_t *dst, int32_t *order_out)
{
    fmm_ctx *c = &p->ctx;
    if (count <= LIST_ORDER_SMALL) {
        list_order_small<<<1, 1024, 0, c->stream>>>(cnt, first, count, off, src, p->node_lo, p->node_hi, by_size, dst, order_out);
        FMM_LAUNCH_CHECK(c, "list_order_small");
        return FMM_OK;
    }
    uint64_t *keys = (uint64_t *)ctx_alloc(c, sizeof(uint64_t) * count);
    uint64_t *tkeys = (uint64_t *)ctx_alloc(c, sizeof(uint64_t) * count);
    uint32_t *vals = (uint32_t *)ctx_alloc(c, sizeof(uint32_t) * count);
    uint32_t *tvals = (uint32_t *)ctx_alloc(c, sizeof(uint32_t) * count);
    if (!keys || !tkeys || !vals || !tvals) return FMM_ENOMEM;
    list_work_keys<<<(count + 255) / 256, 256, 0, c->stream>>>(cnt, first, count, off, src, p->node_lo, p->node_hi, by_size, dst, keys, vals);
    FMM_LAUNCH_CHECK(c, "list_work_keys");
    FMM_TRY(sort_pairs_u64(c, keys, vals, tkeys, tvals, count, 0, 8));
    copy_u32_to_i32<<<(count + 255) / 256, 256, 0, c->stream>>>(count, vals, order_out);
    FMM_LAUNCH_CHECK(c, "copy_u32_to_i32");
    ctx_free(c, keys); ctx_free(c, tkeys); ctx_free(c, vals); ctx_free(c, tvals);
    return FMM_OK;
}

// (re)size one of the plan's list buffers; they keep their capacity from build to build
static int ensure_list(fmm_ctx *c, int32_t **buf, int64_t have, int64_t want)
{
    if (*buf && have >= want) return FMM_OK;
    if (*buf) ctx_free(c, *buf);
    *buf = (int32_t *)ctx_alloc_keep(c, sizeof(int32_t) * (size_t)want);
    return *buf ? FMM_OK : FMM_ENOMEM;
}

// Lists kept across a refit (fmm_plan_refit_keep_lists): the two lists still cover every pair of leaves exactly once --
// that is a property of the tree's index ranges alone -- but the boxes have moved, so a kept far pair may no longer meet
// eq. (4.3).  One pass over the M2L list with the new boxes: the largest max(r_t^2, r_s^2) / d^2 (Alg 5.6-5.8 squared, same
// rounding order as the traversal), kept as the bit pattern of a non-negative double (monotone as an integer).
__global__ void __launch_bounds__(256) m2l_ratio_max(int nodes, const fmm_hdr *__restrict__ hdr, const double *__restrict__ geo,
                                                     const int32_t *__restrict__ m2l_off, const int32_t *__restrict__ m2l_src,
                                                     unsigned long long *__restrict__ out)
{
    const double gamma_bar = hdr->gamma_bar;
    double worst = 0.0;
    for (int t = blockIdx.x * blockDim.x + threadIdx.x + 1; t <= nodes; t += gridDim.x * blockDim.x) {
        const int a = m2l_off[t], b = m2l_off[t + 1];
        if (b <= a) continue;
        const double *gi = geo + 4 * (int64_t)t;
        for (int k = a; k < b; ++k) {
            const double *gj = geo + 4 * (int64_t)m2l_src[k];
            const double ex = __dmul_rn(1.0, __dsub_rn(gi[1], gj[1]));
            const double ey = __dmul_rn(1.0, __dsub_rn(gi[2], gj[2]));
            const double ez = __dmul_rn(gamma_bar, __dsub_rn(gi[3], gj[3]));
            const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(ex, ex), __dmul_rn(ey, ey)), __dmul_rn(ez, ez));
            const double rmax = (gi[0] > gj[0]) ? gi[0] : gj[0];
            double ratio = __ddiv_rn(rmax, d2);  // (d2 = 0: +inf, or NaN for two point clusters at one place -> reported as +inf)
            if (ratio != ratio) ratio = INFINITY;
            worst = ratio > worst ? ratio : worst;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double v = __shfl_xor_sync(0xffffffffu, worst, o);
        worst = v > worst ? v : worst;
    }
    if ((threadIdx.x & 31) == 0 && worst > 0.0) atomicMax(out, (unsigned long long)__double_as_longlong(worst));
}

// a3 of a refit that keeps the lists: no traversal; the admissibility ratio of the kept far pairs and the build's one host wait
int dtt_keep_lists(fmm_plan *p, double *eta_eff /* host */)
{
    fmm_ctx *c = &p->ctx;
    cudaStream_t st = c->stream;
    unsigned long long *slot = (unsigned long long *)ctx_alloc(c, sizeof(unsigned long long));
    if (!slot) return FMM_ENOMEM;
    FMM_CUDA(c, cudaMemsetAsync(slot, 0, sizeof(unsigned long long), st));
    const int blocks = (int)((p->nodes + 255) / 256 < 4 * FMM_SM_COUNT ? (p->nodes + 255) / 256 : 4 * FMM_SM_COUNT);
    m2l_ratio_max<<<blocks, 256, 0, st>>>((int)p->nodes, p->hdr, p->node_geo, p->m2l_off, p->m2l_src, slot);
    FMM_LAUNCH_CHECK(c, "m2l_ratio_max");
    unsigned long long bits = 0;
    fmm_hdr hh;
    FMM_CUDA(c, cudaMemcpyAsync(&bits, slot, sizeof(bits), cudaMemcpyDeviceToHost, st));
    FMM_CUDA(c, cudaMemcpyAsync(&hh, p->hdr, sizeof(hh), cudaMemcpyDeviceToHost, st));
    FMM_CUDA(c, cudaEventRecord(p->ev_plan[2], st));
    FMM_TRY(plan_upward(p));  // (as in a build: the GPU works on the moments while the host waits)
    FMM_CUDA(c, cudaEventSynchronize(p->ev_plan[2]));
    ctx_free(c, slot);
    p->gamma_bar = hh.gamma_bar;
    p->kd_retry = 0;
    if (hh.nonfinite) {
        snprintf(c->err, sizeof(c->err), "%u non-finite values among the positions, momenta and charges (or gamma_bar is not finite)", hh.nonfinite);
        return FMM_ENONFINITE;
    }
    double r2;
    memcpy(&r2, &bits, sizeof(r2));
    if (eta_eff) *eta_eff = sqrt(r2);
    return FMM_OK;
}

int dtt_build_lists(fmm_plan *p)
{
    fmm_ctx *c = &p->ctx;
    cudaStream_t st = c->stream;
    const int key_shift = p->kappa + 2;  // node ids < 2^(kappa+1)
    const int nsteps = 2 * p->kappa + 1;
    const int rows_len = (int)p->nodes + 2;
    const int64_t maxleaf = p->maxleaf;
    // the mean-gamma kernel is antisymmetric in the pair, the source-momentum kernel (D depends on p_j) is not
    const bool mutual = !(p->flags & FMM_KERNEL_SOURCE_MOMENTUM) && maxleaf <= FMM_MUTUAL_MAX_LEAF && maxleaf >= FMM_MUTUAL_MIN_LEAF;
    dtt_counters h;
    fmm_hdr hh;
    int64_t cap = p->leaves * 128;  // first guess; enlarged until nothing overflows, and kept by the plan
    if (cap < 4096) cap = 4096;
    if (cap < p->list_cap) cap = p->list_cap;
    for (int attempt = 0;; ++attempt) {
        if (cap >= ((int64_t)1 << 31)) return FMM_EOVERFLOW;
        // the lists themselves (kept by the plan) ...
        const int64_t have = p->list_cap;
        FMM_TRY(ensure_list(c, &p->p2p_src, have, cap));
        FMM_TRY(ensure_list(c, &p->m2l_src, have, cap));
        if (mutual) {
            FMM_TRY(ensure_list(c, &p->p2p_dst, have, cap));
            FMM_TRY(ensure_list(c, &p->p2p_recv, have, cap));
        }
        p->list_cap = cap;
        // ... and the scratch of this build (arena)
        dtt_counters *cnt = (dtt_counters *)ctx_alloc(c, sizeof(dtt_counters));
        int32_t *rows = (int32_t *)ctx_alloc(c, sizeof(int32_t) * 2 * (size_t)rows_len);
        int32_t *row_work = (int32_t *)ctx_alloc(c, sizeof(int32_t) * (size_t)p->leaves);
        int32_t *scan = (int32_t *)ctx_alloc(c, sizeof(int32_t) * 2 * (size_t)rows_len);
        uint64_t *f0 = (uint64_t *)ctx_alloc(c, sizeof(uint64_t) * cap);
        uint64_t *f1 = (uint64_t *)ctx_alloc(c, sizeof(uint64_t) * cap);
        uint64_t *kp2p = (uint64_t *)ctx_alloc(c, sizeof(uint64_t) * cap);
        uint64_t *km2l = (uint64_t *)ctx_alloc(c, sizeof(uint64_t) * cap);
        int32_t *p2p_tmp = (int32_t *)ctx_alloc(c, sizeof(int32_t) * cap);
        int32_t *m2l_tmp = (int32_t *)ctx_alloc(c, sizeof(int32_t) * cap);
        if (!cnt || !rows || !row_work || !scan || !f0 || !f1 || !kp2p || !km2l || !p2p_tmp || !m2l_tmp) return FMM_ENOMEM;
        int32_t *tgt = NULL, *mate = NULL, *len = NULL, *seg = NULL;
        if (mutual) {
            tgt = (int32_t *)ctx_alloc(c, sizeof(int32_t) * cap);
            mate = (int32_t *)ctx_alloc(c, sizeof(int32_t) * cap);
            len = (int32_t *)ctx_alloc(c, sizeof(int32_t) * cap);
            seg = (int32_t *)ctx_alloc(c, sizeof(int32_t) * cap);
            if (!tgt || !mate || !len || !seg) return FMM_ENOMEM;
        }
        dtt_args a;
        a.nsteps = nsteps; a.leaves = (int)p->leaves; a.key_shift = key_shift;
        a.early_first = p->stop_level >= 0 ? (int)(p->leaves / 2) : 0x7fffffff; a.N0 = p->N0;
        a.treecode_leaves = (p->flags & FMM_METHOD_TREECODE) ? (int)p->leaves : 0;
        a.theta2 = p->theta * p->theta;
        a.roots = (unsigned int)(p->leaves / 4 < 4096 ? 4096 : (p->leaves / 4 > 65536 ? 65536 : p->leaves / 4));
        a.hdr = p->hdr; a.node_lo = p->node_lo; a.node_hi = p->node_hi; a.geo = p->node_geo;
        a.front0 = f0; a.front1 = f1; a.p2p = kp2p; a.m2l = km2l; a.cap = (unsigned)cap;
        a.rows = rows; a.row_work = row_work; a.rows_len = rows_len; a.cnt = cnt;
        dtt_top<<<1, 1024, 0, st>>>(a);
        FMM_LAUNCH_CHECK(c, "dtt_top");
        // (FMM_TEST_WALK_STACK shrinks the walk's stack so that the tests reach the spill path)
        const char *ws = getenv("FMM_TEST_WALK_STACK");
        int wstack = ws ? atoi(ws) : DTT_WSTACK;
        if (wstack < 64 || wstack > DTT_WSTACK) wstack = DTT_WSTACK;
        dtt_walk<<<12 * FMM_SM_COUNT, 32 * DTT_WALK_WARPS, 0, st>>>(a, 0, wstack);
        FMM_LAUNCH_CHECK(c, "dtt_walk");
        dtt_walk<<<2 * FMM_SM_COUNT, 32 * DTT_WALK_WARPS, 0, st>>>(a, 1, DTT_WSTACK);  // (walks that spilled: normally none)
        FMM_LAUNCH_CHECK(c, "dtt_walk");
        dtt_totals<<<(unsigned)((p->leaves + 255) / 256 < 2 * FMM_SM_COUNT ? (p->leaves + 255) / 256 : 2 * FMM_SM_COUNT), 256, 0, st>>>(a);
        FMM_LAUNCH_CHECK(c, "dtt_totals");
        // rows -> CSR without waiting for the host (the list lengths are read on the device; every kernel below does
        // nothing if the traversal overflowed its buffers): offsets from the scanned row lengths, entries dealt to their
        // rows, rows sorted by source, then pair ownership and the reaction segments, then the block orders
        FMM_TRY(scan_exclusive_i32(c, rows, scan, 2 * (int64_t)rows_len));
        csr_offsets<<<(rows_len + 255) / 256, 256, 0, st>>>(rows_len, scan, p->p2p_off, p->m2l_off);
        FMM_LAUNCH_CHECK(c, "csr_offsets");
        csr_fill<<<4 * FMM_SM_COUNT, 256, 0, st>>>(cnt, kp2p, km2l, key_shift, rows_len, p->p2p_off, p->m2l_off, rows, p2p_tmp, m2l_tmp);
        FMM_LAUNCH_CHECK(c, "csr_fill");
        csr_sort_rows<<<(unsigned)(p->leaves + p->nodes), ROWSORT_THREADS, 0, st>>>(cnt, (int)p->leaves, (int)p->leaves, 1, p->p2p_off, p->m2l_off,
                                                                                   p2p_tmp, m2l_tmp, p->p2p_src, p->m2l_src, tgt);
        FMM_LAUNCH_CHECK(c, "csr_sort_rows");
        if (mutual) {
            p2p_mates<<<4 * FMM_SM_COUNT, 256, 0, st>>>(cnt, cap, p->p2p_off, p->p2p_src, tgt, p->node_lo, p->node_hi, mate, len);
            FMM_LAUNCH_CHECK(c, "p2p_mates");
            FMM_TRY(scan_exclusive_i32(c, len, seg, cap));  // segment starts, in particles
            p2p_segments<<<4 * FMM_SM_COUNT, 256, 0, st>>>(cnt, mate, len, seg, p->p2p_dst, p->p2p_recv);
            FMM_LAUNCH_CHECK(c, "p2p_segments");
        }
        FMM_TRY(make_order(p, cnt, (int)p->leaves, (int)p->leaves, p->p2p_off, p->p2p_src, 1, mutual ? p->p2p_dst : NULL, p->p2p_order));
        FMM_TRY(make_order(p, cnt, 1, (int)p->nodes, p->m2l_off, p->m2l_src, 0, NULL, p->m2l_order));
        FMM_CUDA(c, cudaMemcpyAsync(&h, cnt, sizeof(h), cudaMemcpyDeviceToHost, st));
        FMM_CUDA(c, cudaMemcpyAsync(&hh, p->hdr, sizeof(hh), cudaMemcpyDeviceToHost, st));
        // the one host wait of a build (list lengths, gamma_bar, the input check) is on an event behind those copies; the
        // upward pass is enqueued first, so that the GPU has work while the host reads them and returns to the caller
        FMM_CUDA(c, cudaEventRecord(p->ev_plan[2], st));
        FMM_TRY(plan_upward(p));
        FMM_CUDA(c, cudaEventSynchronize(p->ev_plan[2]));
        ctx_free(c, seg); ctx_free(c, len); ctx_free(c, mate); ctx_free(c, tgt);
        ctx_free(c, m2l_tmp); ctx_free(c, p2p_tmp); ctx_free(c, km2l); ctx_free(c, kp2p); ctx_free(c, f1); ctx_free(c, f0);
        ctx_free(c, scan); ctx_free(c, row_work); ctx_free(c, rows); ctx_free(c, cnt);
        p->gamma_bar = hh.gamma_bar;
        p->kd_retry = (hh.kd_fallback && !p->kd_exact) ? 1 : 0;
        if (p->kd_retry) return FMM_OK;  // (plan_build runs the whole build again with exact sort keys)
        if (hh.nonfinite) {
            snprintf(c->err, sizeof(c->err), "%u non-finite values among the positions, momenta and charges (or gamma_bar is not finite)", hh.nonfinite);
            return FMM_ENONFINITE;
        }
        if (!h.overflow) break;
        int64_t need = (int64_t)h.n_p2p;  // the counters kept counting past the capacity: they say how much was needed so far
        if ((int64_t)h.n_m2l > need) need = h.n_m2l;
        if ((int64_t)h.n_front[0] > need) need = h.n_front[0];
        if ((int64_t)h.n_front[2] > need) need = h.n_front[2];
        cap = (need + need / 8 > 2 * cap) ? need + need / 8 : 2 * cap;
    }
    p->n_p2p = h.n_p2p;
    p->n_m2l = h.n_m2l;
    p->p2p_pairs = (int64_t)h.evals;
    p->p2p_max_row = (int64_t)h.max_row;
    p->m2l_pairs = (p->flags & FMM_METHOD_TREECODE) ? p->n_m2l * (int64_t)p->P * ((p->N + p->leaves - 1) / p->leaves)  // particle-proxy pairs (full leaves)
                                                    : p->n_m2l * (int64_t)p->P * (int64_t)p->P;
    // the reaction segments hold at most one leaf per pair of mated entries (segment offsets are 32-bit)
    p->p2p_mutual = (mutual && p->n_p2p > 0 && (p->n_p2p / 2) * maxleaf < ((int64_t)1 << 31)) ? 1 : 0;
    p->p2p_react = p->p2p_mutual ? (p->n_p2p / 2) * maxleaf : 0;
    return FMM_OK;
}
