// kernels_dtt.cu -- step a3: dual tree traversal (Alg 9.1; same logic as Alg 5.11,
// PAPER.md:400-435) with the stretched admissibility condition of Alg 5.6-5.8 (PAPER.md:337-366,
// eq. (4.3)), emitting the two interaction lists, then sorting them by
// (target, source) into CSR form (readings D-4, G20).
//
// The recursion is run level-synchronously: a frontier of (target, source) node pairs is
// classified by one kernel per step (P2P / M2L / split), children are appended to the next frontier
// through INTEGER atomic counters (order inside a frontier is irrelevant: the lists are sorted
// afterwards, so the result is unique and bit-reproducible).  No host round trip until the final
// list lengths are read back.
#include "fmm_internal.cuh"

struct dtt_counters {           // device
    unsigned int n_p2p, n_m2l, overflow, pad;
    unsigned int n_front[72];   // frontier sizes per step (at most 2*kappa+2 steps)
};

__global__ void dtt_init(dtt_counters *cnt, uint64_t *front0, int treecode_leaves)
{
    // FMM: the traversal starts at (root, root).  Treecode (FMM_METHOD_TREECODE): at (t, root) for every leaf t, so
    // the target is never split and the "m2l" list becomes the particle-cluster list.
    int k0 = blockIdx.x * blockDim.x + threadIdx.x;
    if (k0 == 0) {
        cnt->n_p2p = cnt->n_m2l = cnt->overflow = cnt->pad = 0;
        for (int k = 0; k < 72; ++k) cnt->n_front[k] = 0;
        cnt->n_front[0] = treecode_leaves > 0 ? (unsigned)treecode_leaves : 1u;
        if (treecode_leaves <= 0) front0[0] = (1ull << 32) | 1ull;  // (root, root)
    }
    if (k0 < treecode_leaves) front0[k0] = ((uint64_t)(treecode_leaves + k0) << 32) | 1ull;  // (leaf, root)
}

__global__ void __launch_bounds__(256) dtt_step(int step, int leaves, const fmm_hdr *__restrict__ hdr, double theta2,
                                                const int32_t *__restrict__ node_lo, const int32_t *__restrict__ node_hi,
                                                const double *__restrict__ geo, const uint64_t *__restrict__ front_in,
                                                uint64_t *__restrict__ front_out, unsigned int cap_front,
                                                uint64_t *__restrict__ p2p, unsigned int cap_p2p,
                                                uint64_t *__restrict__ m2l, unsigned int cap_m2l,
                                                int key_shift, dtt_counters *cnt)
{
    if (hdr->nonfinite) return;  // NaN / Inf in the inputs: no lists (FMM_ENONFINITE after the read-back)
    const double gamma_bar = hdr->gamma_bar;
    unsigned int nin = cnt->n_front[step];
    if (nin > cap_front) nin = cap_front;
    for (unsigned int k = blockIdx.x * blockDim.x + threadIdx.x; k < nin; k += gridDim.x * blockDim.x) {
        uint64_t pr = front_in[k];
        int i = (int)(pr >> 32), j = (int)(pr & 0xffffffffu);  // i = target, j = source
        if (node_hi[i] <= node_lo[i] || node_hi[j] <= node_lo[j]) continue;  // empty cluster
        bool leaf_i = i >= leaves, leaf_j = j >= leaves;
        if (leaf_i && leaf_j) {  // D-1: leaf-leaf -> P2P, no admissibility test
            unsigned int pos = atomicAdd(&cnt->n_p2p, 1u);
            if (pos < cap_p2p) p2p[pos] = ((uint64_t)i << key_shift) | (uint64_t)j; else cnt->overflow = 1;
            continue;
        }
        // D-2: Alg 5.6-5.8 squared; every product and sum rounded separately, in this order
        const double *gi = geo + 4 * (int64_t)i, *gj = geo + 4 * (int64_t)j;
        double ri = gi[0], rj = gj[0];
        double ex = __dmul_rn(1.0, __dsub_rn(gi[1], gj[1]));
        double ey = __dmul_rn(1.0, __dsub_rn(gi[2], gj[2]));
        double ez = __dmul_rn(gamma_bar, __dsub_rn(gi[3], gj[3]));
        double d2 = __dadd_rn(__dadd_rn(__dmul_rn(ex, ex), __dmul_rn(ey, ey)), __dmul_rn(ez, ez));
        double rmax = (ri > rj) ? ri : rj;
        if (rmax < __dmul_rn(theta2, d2)) {  // admissible -> M2L
            unsigned int pos = atomicAdd(&cnt->n_m2l, 1u);
            if (pos < cap_m2l) m2l[pos] = ((uint64_t)i << key_shift) | (uint64_t)j; else cnt->overflow = 1;
            continue;
        }
        // D-3: which side to split
        bool split_target = leaf_i ? false : (leaf_j ? true : (ri > rj));
        unsigned int pos = atomicAdd(&cnt->n_front[step + 1], 2u);
        if (pos + 1 < cap_front) {
            if (split_target) {
                front_out[pos] = ((uint64_t)(2 * i) << 32) | (uint64_t)j;
                front_out[pos + 1] = ((uint64_t)(2 * i + 1) << 32) | (uint64_t)j;
            } else {
                front_out[pos] = ((uint64_t)i << 32) | (uint64_t)(2 * j);
                front_out[pos + 1] = ((uint64_t)i << 32) | (uint64_t)(2 * j + 1);
            }
        } else {
            cnt->overflow = 1;
        }
    }
}

// sorted keys (target << shift | source) -> CSR: off[t] = first position with target >= t
__global__ void csr_from_sorted(const uint64_t *__restrict__ keys, int64_t n, int key_shift, int nodes,
                                int32_t *__restrict__ off /* [nodes+2] */, int32_t *__restrict__ src, int32_t *__restrict__ tgt /* or NULL */)
{
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k > n) return;
    uint64_t mask = (1ull << key_shift) - 1ull;
    int t_prev = (k == 0) ? -1 : (int)(keys[k - 1] >> key_shift);
    int t_cur = (k == n) ? nodes + 1 : (int)(keys[k] >> key_shift);
    for (int t = t_prev + 1; t <= t_cur; ++t) off[t] = (int32_t)k;
    if (k < n) {
        src[k] = (int32_t)(keys[k] & mask);
        if (tgt) tgt[k] = t_cur;
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

__global__ void p2p_mates(int64_t n, const int32_t *__restrict__ off, const int32_t *__restrict__ src, const int32_t *__restrict__ tgt,
                          const int32_t *__restrict__ node_lo, const int32_t *__restrict__ node_hi, int32_t *__restrict__ mate,
                          int32_t *__restrict__ len)
{
    int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
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

__global__ void p2p_segments(int64_t n, const int32_t *__restrict__ src, const int32_t *__restrict__ tgt, const int32_t *__restrict__ mate,
                             const int32_t *__restrict__ len, const int32_t *__restrict__ scan, int32_t *__restrict__ dst,
                             int32_t *__restrict__ recv, unsigned long long *__restrict__ total /* [2] = reaction particles */)
{
    int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    const int m = mate[e];
    recv[e] = len[e] > 0 ? scan[e] : -1;
    dst[e] = (m < 0) ? -1 : (len[e] > 0 ? -2 : scan[m]);
    if (e == n - 1) total[2] = (unsigned long long)scan[e] + (unsigned long long)len[e];
}

// LPT block order: targets by descending work (number of source clusters x their sizes)
__global__ void list_work_keys(int first, int count, const int32_t *__restrict__ off, const int32_t *__restrict__ src,
                               const int32_t *__restrict__ node_lo, const int32_t *__restrict__ node_hi, int by_size,
                               const int32_t *__restrict__ dst /* P2P entry kinds, or NULL */,
                               uint64_t *__restrict__ keys, uint32_t *__restrict__ vals, unsigned long long *__restrict__ total)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= count) return;
    int t = first + k;
    unsigned long long work = 0;
    if (by_size) {
        unsigned long long nt = (unsigned long long)(node_hi[t] - node_lo[t]), evals = 0;
        for (int e = off[t]; e < off[t + 1]; ++e) {
            const unsigned long long pairs = nt * (unsigned long long)(node_hi[src[e]] - node_lo[src[e]]);
            evals += pairs;
            // block work in FP64 instructions per particle pair: 25 one-sided, 34 for an owned mutual pair, 0 if the mate owns it
            work += pairs * (unsigned long long)(!dst ? 25 : (dst[e] >= 0 ? 34 : (dst[e] == -1 ? 25 : 0)));
        }
        work /= 25;
        atomicAdd(total, evals);      // kernel evaluations of the whole list (the algorithmic count)
        atomicMax(total + 1, work);   // heaviest row, in one-sided pair units
        atomicAdd(total + 3, work);
    } else {
        work = (unsigned long long)(off[t + 1] - off[t]);
    }
    // block order only needs a coarse, deterministic ranking: a 16-bit monotone code of the work (6-bit exponent,
    // 10-bit mantissa: 0.1 % resolution over the whole 64-bit range), so the sort takes 2 radix passes
    unsigned long long wq = 0;
    if (work > 0) {
        int e = 63 - __clzll((long long)work);
        unsigned long long mant = (e >= 10) ? (work >> (e - 10)) : (work << (10 - e));  // 1.xxxxxxxxxx
        wq = ((unsigned long long)e << 10) | (mant & 0x3ffull);
        wq += 1;  // keep 0 for "no work"
    }
    keys[k] = 0xffffull - wq;  // ascending sort of this = descending work
    vals[k] = (uint32_t)t;
}

__global__ void copy_u32_to_i32(int n, const uint32_t *__restrict__ a, int32_t *__restrict__ b)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) b[k] = (int32_t)a[k];
}

static int make_order(fmm_plan *p, int first, int count, const int32_t *off, const int32_t *src, int by_size, const int32_t *dst,
                      int32_t *order_out, unsigned long long *total_dev)
{
    fmm_ctx *c = &p->ctx;
    uint64_t *keys = (uint64_t *)ctx_alloc(c, sizeof(uint64_t) * count);
    uint64_t *tkeys = (uint64_t *)ctx_alloc(c, sizeof(uint64_t) * count);
    uint32_t *vals = (uint32_t *)ctx_alloc(c, sizeof(uint32_t) * count);
    uint32_t *tvals = (uint32_t *)ctx_alloc(c, sizeof(uint32_t) * count);
    if (!keys || !tkeys || !vals || !tvals) return FMM_ENOMEM;
    list_work_keys<<<(count + 255) / 256, 256, 0, c->stream>>>(first, count, off, src, p->node_lo, p->node_hi, by_size, dst, keys, vals, total_dev);
    FMM_LAUNCH_CHECK(c, "list_work_keys");
    FMM_TRY(sort_pairs_u64(c, keys, vals, tkeys, tvals, count, 0, 16));
    copy_u32_to_i32<<<(count + 255) / 256, 256, 0, c->stream>>>(count, vals, order_out);
    FMM_LAUNCH_CHECK(c, "copy_u32_to_i32");
    ctx_free(c, keys); ctx_free(c, tkeys); ctx_free(c, vals); ctx_free(c, tvals);
    return FMM_OK;
}

int dtt_build_lists(fmm_plan *p)
{
    fmm_ctx *c = &p->ctx;
    cudaStream_t st = c->stream;
    const int key_shift = p->kappa + 2;  // node ids < 2^(kappa+1)
    const int nsteps = 2 * p->kappa + 1;
    dtt_counters *cnt = (dtt_counters *)ctx_alloc(c, sizeof(dtt_counters) + 4 * sizeof(unsigned long long));
    if (!cnt) return FMM_ENOMEM;
    unsigned long long *total_dev = (unsigned long long *)(cnt + 1);
    dtt_counters h;
    int64_t cap = p->leaves * 128;  // first guess; doubled until nothing overflows
    if (cap < 4096) cap = 4096;
    uint64_t *f0 = NULL, *f1 = NULL, *kp2p = NULL, *km2l = NULL;
    for (int attempt = 0;; ++attempt) {
        if (cap >= ((int64_t)1 << 31)) return FMM_EOVERFLOW;
        f0 = (uint64_t *)ctx_alloc(c, sizeof(uint64_t) * cap);
        f1 = (uint64_t *)ctx_alloc(c, sizeof(uint64_t) * cap);
        kp2p = (uint64_t *)ctx_alloc(c, sizeof(uint64_t) * cap);
        km2l = (uint64_t *)ctx_alloc(c, sizeof(uint64_t) * cap);
        if (!f0 || !f1 || !kp2p || !km2l) return FMM_ENOMEM;
        const int tc_leaves = (p->flags & FMM_METHOD_TREECODE) ? (int)p->leaves : 0;
        dtt_init<<<tc_leaves > 0 ? (tc_leaves + 255) / 256 : 1, 256, 0, st>>>(cnt, f0, tc_leaves);
        FMM_LAUNCH_CHECK(c, "dtt_init");
        uint64_t *fin = f0, *fout = f1;
        for (int step = 0; step < nsteps; ++step) {
            dtt_step<<<2 * FMM_SM_COUNT, 256, 0, st>>>(step, (int)p->leaves, p->hdr, p->theta * p->theta, p->node_lo, p->node_hi,
                                                       p->node_geo, fin, fout, (unsigned)cap, kp2p, (unsigned)cap, km2l, (unsigned)cap,
                                                       key_shift, cnt);
            FMM_LAUNCH_CHECK(c, "dtt_step");
            uint64_t *t = fin; fin = fout; fout = t;
        }
        fmm_hdr hh;
        FMM_CUDA(c, cudaMemcpyAsync(&h, cnt, sizeof(h), cudaMemcpyDeviceToHost, st));
        FMM_CUDA(c, cudaMemcpyAsync(&hh, p->hdr, sizeof(hh), cudaMemcpyDeviceToHost, st));
        FMM_CUDA(c, cudaStreamSynchronize(st));  // the one host wait of a build: list lengths, gamma_bar, the input check
        p->gamma_bar = hh.gamma_bar;
        if (hh.nonfinite) {
            ctx_free(c, f0); ctx_free(c, f1); ctx_free(c, kp2p); ctx_free(c, km2l); ctx_free(c, cnt);
            snprintf(c->err, sizeof(c->err), "%u non-finite values among the positions, momenta and charges (or gamma_bar is not finite)", hh.nonfinite);
            return FMM_ENONFINITE;
        }
        ctx_free(c, f0); ctx_free(c, f1);
        if (!h.overflow) break;
        ctx_free(c, kp2p); ctx_free(c, km2l);
        cap *= 4;
    }
    p->n_p2p = h.n_p2p;
    p->n_m2l = h.n_m2l;

    // sort by (target, source), then CSR
    int64_t nmax = (p->n_p2p > p->n_m2l) ? p->n_p2p : p->n_m2l;
    uint64_t *tkeys = (uint64_t *)ctx_alloc(c, sizeof(uint64_t) * (nmax > 0 ? nmax : 1));
    if (!tkeys) return FMM_ENOMEM;
    if (p->p2p_src) ctx_free(c, p->p2p_src);
    if (p->m2l_src) ctx_free(c, p->m2l_src);
    if (p->p2p_dst) ctx_free(c, p->p2p_dst);
    if (p->p2p_recv) ctx_free(c, p->p2p_recv);
    p->p2p_dst = p->p2p_recv = NULL;
    p->p2p_src = (int32_t *)ctx_alloc(c, sizeof(int32_t) * (p->n_p2p > 0 ? p->n_p2p : 1));
    p->m2l_src = (int32_t *)ctx_alloc(c, sizeof(int32_t) * (p->n_m2l > 0 ? p->n_m2l : 1));
    if (!p->p2p_src || !p->m2l_src) return FMM_ENOMEM;
    // the mean-gamma kernel is antisymmetric in the pair, the source-momentum kernel (D depends on p_j) is not
    const bool mutual = !(p->flags & FMM_KERNEL_SOURCE_MOMENTUM) && p->n_p2p > 0;
    int32_t *tgt = NULL, *mate = NULL, *len = NULL, *seg = NULL;
    if (mutual) {
        p->p2p_dst = (int32_t *)ctx_alloc(c, sizeof(int32_t) * p->n_p2p);
        p->p2p_recv = (int32_t *)ctx_alloc(c, sizeof(int32_t) * p->n_p2p);
        tgt = (int32_t *)ctx_alloc(c, sizeof(int32_t) * p->n_p2p);
        mate = (int32_t *)ctx_alloc(c, sizeof(int32_t) * p->n_p2p);
        len = (int32_t *)ctx_alloc(c, sizeof(int32_t) * p->n_p2p);
        seg = (int32_t *)ctx_alloc(c, sizeof(int32_t) * p->n_p2p);
        if (!p->p2p_dst || !p->p2p_recv || !tgt || !mate || !len || !seg) return FMM_ENOMEM;
    }
    FMM_TRY(sort_pairs_u64(c, kp2p, NULL, tkeys, NULL, p->n_p2p, 0, 2 * key_shift));
    FMM_TRY(sort_pairs_u64(c, km2l, NULL, tkeys, NULL, p->n_m2l, 0, 2 * key_shift));
    csr_from_sorted<<<(unsigned)((p->n_p2p + 256) / 256), 256, 0, st>>>(kp2p, p->n_p2p, key_shift, (int)p->nodes, p->p2p_off, p->p2p_src, tgt);
    FMM_LAUNCH_CHECK(c, "csr_from_sorted");
    csr_from_sorted<<<(unsigned)((p->n_m2l + 256) / 256), 256, 0, st>>>(km2l, p->n_m2l, key_shift, (int)p->nodes, p->m2l_off, p->m2l_src, NULL);
    FMM_LAUNCH_CHECK(c, "csr_from_sorted");
    ctx_free(c, tkeys); ctx_free(c, kp2p); ctx_free(c, km2l);
    FMM_CUDA(c, cudaMemsetAsync(total_dev, 0, 4 * sizeof(unsigned long long), st));
    if (mutual) {  // pair ownership and the reaction segments
        const unsigned g = (unsigned)((p->n_p2p + 255) / 256);
        p2p_mates<<<g, 256, 0, st>>>(p->n_p2p, p->p2p_off, p->p2p_src, tgt, p->node_lo, p->node_hi, mate, len);
        FMM_LAUNCH_CHECK(c, "p2p_mates");
        FMM_TRY(scan_exclusive_i32(c, len, seg, p->n_p2p));  // segment starts, in particles
        p2p_segments<<<g, 256, 0, st>>>(p->n_p2p, p->p2p_src, tgt, mate, len, seg, p->p2p_dst, p->p2p_recv, total_dev);
        FMM_LAUNCH_CHECK(c, "p2p_segments");
        ctx_free(c, tgt); ctx_free(c, mate); ctx_free(c, len); ctx_free(c, seg);
    }

    // block orders (descending work) and evaluation counts
    FMM_TRY(make_order(p, (int)p->leaves, (int)p->leaves, p->p2p_off, p->p2p_src, 1, p->p2p_dst, p->p2p_order, total_dev));
    FMM_TRY(make_order(p, 1, (int)p->nodes, p->m2l_off, p->m2l_src, 0, NULL, p->m2l_order, total_dev));
    unsigned long long total_h2[4] = {0, 0, 0, 0};
    FMM_CUDA(c, cudaMemcpyAsync(total_h2, total_dev, sizeof(total_h2), cudaMemcpyDeviceToHost, st));
    FMM_CUDA(c, cudaStreamSynchronize(st));
    p->p2p_pairs = (int64_t)total_h2[0];
    p->p2p_max_row = (int64_t)total_h2[1];
    p->p2p_react = (int64_t)total_h2[2];
    p->p2p_work = (int64_t)total_h2[3];
    p->m2l_pairs = (p->flags & FMM_METHOD_TREECODE) ? p->n_m2l * (int64_t)p->P * ((p->N + p->leaves - 1) / p->leaves)  // particle-proxy pairs (full leaves)
                                                    : p->n_m2l * (int64_t)p->P * (int64_t)p->P;
    ctx_free(c, cnt);
    return FMM_OK;
}
