// fmm_internal.cuh -- plan layout, launch bookkeeping and device helpers shared by the
// kernels of libfmm_b200.so (include/fmm.h).  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
#include <atomic>
#include <vector>

#include "../../include/fmm.h"

#define FMM_SM_COUNT 148           // B200: 2 dies x 74 SMs (grids are sized in multiples of this)
#define FMM_EPS0 8.8541878128e-12  // F/m, CODATA 2018 (eq. (3.1))
#define FMM_C0 299792458.0         // m/s
#define FMM_PI 3.14159265358979323846

extern std::atomic<int64_t> g_fmm_launches;
#define FMM_COUNT_LAUNCH() (g_fmm_launches.fetch_add(1, std::memory_order_relaxed))

struct fmm_ctx {  // allocator + stream + error text, shared by plans and plan-less calls
    fmm_alloc_fn alloc;
    fmm_free_fn free_;
    void *user;
    cudaStream_t stream;
    char err[256];
    int64_t bytes;
    std::vector<void *> owned;
    std::vector<size_t> owned_bytes;
    // Scratch arena of a plan: one block from the caller's allocator that serves every temporary of a build (bump
    // pointer, reset per build), so that a build costs no allocator calls in steady state (each call through the Python
    // binding is a callback into torch, ~10 us of host time with the GPU idle).  Stream-ordered like everything else.
    char *arena;
    size_t arena_cap, arena_top, arena_need;
    int arena_on;
    std::vector<size_t> arena_marks;  // start offsets of the arena blocks handed out, for last-in-first-out reuse
    std::vector<char> arena_live;
};

void *ctx_alloc(fmm_ctx *c, size_t bytes);       // NULL on failure (err set); from the arena while a build is running
void *ctx_alloc_keep(fmm_ctx *c, size_t bytes);  // always from the caller's allocator (buffers that outlive the build)
void ctx_free(fmm_ctx *c, void *p);
void ctx_free_keep(fmm_ctx *c, void *p);
int ctx_arena_begin(fmm_ctx *c, size_t estimate);
void ctx_arena_end(fmm_ctx *c);
void ctx_free_all(fmm_ctx *c);
int ctx_cuda_fail(fmm_ctx *c, cudaError_t e, const char *what);

// T-2: position that separates the children of the cluster [lo, hi) of `level`: the left child gets ceil(size / 2);
// a cluster of level stop_level with at most N0 particles is not split (FMM_TREE_STOP_AT_N0): everything stays left.
__host__ __device__ __forceinline__ int fmm_split_mid(int lo, int hi, int level, int stop_level, int N0)
{
    return (level == stop_level && hi - lo <= N0) ? hi : lo + (hi - lo + 1) / 2;
}
#define FMM_CUDA(c, call)                                                  \
    do {                                                                   \
        cudaError_t e__ = (call);                                          \
        if (e__ != cudaSuccess) return ctx_cuda_fail((c), e__, #call);     \
    } while (0)
#define FMM_LAUNCH_CHECK(c, name)                                          \
    do {                                                                   \
        FMM_COUNT_LAUNCH();                                                \
        cudaError_t e__ = cudaGetLastError();                              \
        if (e__ != cudaSuccess) return ctx_cuda_fail((c), e__, name);      \
    } while (0)
#define FMM_TRY(expr)                    \
    do {                                 \
        int rc__ = (expr);               \
        if (rc__ != FMM_OK) return rc__; \
    } while (0)

// Device-resident scalars of one plan build (step a0), read by every kernel that needs them, so that the build
// never waits for the host between a0 and the traversal.
struct fmm_hdr {
    double gamma_bar;        // sqrt(1 + pbar.pbar), or the caller's value
    double g2;               // gamma_bar * gamma_bar (one rounding), the stretch of eq. (3.2)
    double mm[6];            // min x, y, z / max x, y, z of the positions
    unsigned int nonfinite;  // number of NaN / Inf values among x, y, z, px, py, pz, q (saturating) + 1 if gamma_bar is not finite
    unsigned int kd_fallback; // the quantised sort keys of the KD build left a long run out of order: rebuild with exact keys
};

enum { EV_P2M = 0, EV_M2M, EV_UPEND, EV_M2L, EV_L2L, EV_P2P, EV_L2P, EV_END, EV_COUNT };

struct fmm_plan {
    fmm_ctx ctx;
    int64_t N;
    int n, n1, P, N0, kappa;
    int64_t nodes, leaves;
    // FMM_TREE_STOP_AT_N0 (Alg 5.2 as printed): a cluster of level stop_level = kappa-1 that holds at most N0 particles is a
    // leaf.  In this library such a leaf S keeps its two slots: slot 2S holds all its particles (same range, same box), slot
    // 2S+1 is empty, so that every kernel that works on "the leaves" still works on level kappa; the transfer matrices between
    // S and 2S are identities (equal boxes, exact-hit rule I-4), so M_S and L_2S are exact copies.  Only the traversal knows:
    // it treats S as a leaf and names it 2S in the P2P list; fmm_plan_export translates back.  -1: no such cluster.
    int stop_level, early_leaves;
    int maxleaf;            // largest leaf: N0 with early leaves, else ceil(N / 2^kappa)
#define FMM_MUTUAL_MAX_LEAF 2048  // the mutual near field holds a leaf's targets in registers: 1024 per pass, at most two passes
#define FMM_MUTUAL_MIN_LEAF 24    // below that (one target per lane, lanes idle) the gather of many tiny reaction segments in L2P costs more
                                  // than the shared evaluations save: N = 1.28e6, leaves of 20: P2P + L2P 3.54 ms mutual, 3.26 ms one-sided
                                  // (leaves of 10: 4.68 / 3.99; leaves of 39: 3.48 / 4.42)
    double theta, gamma_bar, gamma_bar_param;
    fmm_hdr *hdr;           // device
    int ranges_done;        // node_lo / node_hi are filled (they depend on N and N0 only)
    int kd_exact;           // KD build with the exact 64-bit sort keys (set once the quantised keys were not enough)
    int kd_retry;           // the last build asked for that
    int valid;              // 0 after a failed build: fmm_eval refuses the plan until an update / refit succeeds
    uint32_t flags;
    // particles in tree order (SoA), source weights w0 = q gamma, w1..3 = q p
    double *tx, *ty, *tz, *w0, *w1, *w2, *w3;
    double *pmx, *pmy, *pmz;  // plain momenta in tree order, only with FMM_KERNEL_SOURCE_MOMENTUM (else NULL)
    int32_t *perm;          // [N] tree position -> caller index
    // nodes, heap index 1..nodes (entry 0 unused)
    int32_t *node_lo;       // [nodes+2] range start; node_hi(i) stored separately
    int32_t *node_hi;
    double *bbox;           // [nodes+1][6]
    double *node_geo;       // [nodes+1][4] : r^2 (Alg 5.6 squared), cx, cy, cz (box centres)
    double *node_T;         // [nodes+2][3 (n+1)^2 rounded up to even] 1-D transfer matrices child <- parent, filled per build
    int *xfer_sync;         // [2][nodes+2] M2M arrival counters (zero between evaluations), L2L stamps
    int xfer_stamp;         // stamp of the last L2L launch
    double *node_xi;        // [nodes+1][3][16] : proxy points per axis (I-3), filled by pairs_m2l
    // interaction lists, CSR by target node id (offset arrays indexed by node id, length nodes+2)
    int32_t *p2p_off, *p2p_src, *m2l_off, *m2l_src;
    // mutual near field (kernels_dtt.cu "p2p_mates"): per P2P entry, dst >= 0: the target's block owns the pair and writes the
    // reaction on the source leaf to partial segment dst; dst = -1: one-sided; dst = -2: the mate's block does the work and
    // recv >= 0 is the segment holding the sums for this entry's target particles.  NULL with FMM_KERNEL_SOURCE_MOMENTUM.
    int32_t *p2p_dst, *p2p_recv;
    int p2p_mutual;         // the lists of the last build carry pair ownership (dst / recv) that the near-field kernel may use
    int64_t list_cap;       // entries allocated for p2p_src, m2l_src, p2p_dst, p2p_recv
    int64_t p2p_react;      // upper bound of the particles in all reaction segments
    double *react;          // [6][p2p_react] reaction sums (E, B components as planes), rewritten by every fmm_eval
    int64_t react_cap;
    int react_used;         // the last pairs_p2p ran the mutual kernel (L2P then subtracts the reaction segments)
    int64_t n_p2p, n_m2l, cap_p2p, cap_m2l;
    int64_t p2p_pairs, m2l_pairs;
    int64_t p2p_max_row;    // particle pairs of the heaviest target leaf row
    int p2p_split;          // P2P row split K: block (t, k) sums chunk k of t's row into near_[k]; L2P adds the K partials in order
    int64_t near_cap;       // doubles allocated for near_
    int m2l_split;          // M2L row split (small trees): chunk kc > 0 of a row goes to Lpart[kc-1], combined into L in order
    double *Lpart;          // [m2l_split-1][nodes+2][P][6]
    int64_t lpart_cap;
    int32_t *p2p_order, *m2l_order;  // target ids sorted by descending work (LPT block order)
    int32_t n_p2p_targets, n_m2l_targets;
    // expansions
    double *M;              // [nodes+1][P][4]
    double *L;              // [nodes+1][P][6]
    double *near_;          // [p2p_split][6][N] tree order, P2P partial results
    // timing
    int timing;
    cudaEvent_t ev[EV_COUNT];
    cudaEvent_t ev_plan[3];
    // near / far overlap: P2P runs on `side` while the upward pass, M2L and L2L run on the caller's stream
    cudaStream_t side;
    cudaEvent_t ev_fork, ev_join;
    int overlap;
    int ev_valid;
    int upward_done;        // P2M + M2M of the current tree are enqueued already (plan_upward: at the end of a build, behind the host wait)
    int plan_ms_pending;    // ms_tree / ms_lists of the last build have not been read from ev_plan yet
    float ms_tree, ms_lists;
};

// ---- kernels_tree.cu ----------------------------------------------------------------
int tree_gamma_bar(fmm_ctx *c, int64_t N, const double *px, const double *py, const double *pz,
                   double *gamma_bar_out /* host */);  // plan-less calls (fmm_direct): synchronises
int tree_scan_inputs(fmm_plan *p, const fmm_particles_t *in);  // a0 into p->hdr, enqueue only
int tree_build(fmm_plan *p, const fmm_particles_t *in);
int kd_build_order(fmm_plan *p, const fmm_particles_t *in, uint32_t **order_out);  // kernels_kd.cu
int tree_boxes(fmm_plan *p);
int tree_refit(fmm_plan *p, const fmm_particles_t *in);  // keeps the particle order of the last build
// ---- kernels_dtt.cu -----------------------------------------------------------------
int dtt_build_lists(fmm_plan *p);
int dtt_keep_lists(fmm_plan *p, double *eta_eff /* host */);  // refit without a traversal: checks the kept far pairs
// ---- kernels_interp.cu --------------------------------------------------------------
int interp_transfer_tables(fmm_plan *p);  // after the boxes of a build
int plan_upward(fmm_plan *p);  // a4 + a5 once per build (fmm_api.cu)
int interp_p2m(fmm_plan *p);
int interp_m2m(fmm_plan *p);
int interp_l2l(fmm_plan *p);
int interp_l2p_finalize(fmm_plan *p, /* treecode: no far interpolation, near_ has one more partial */ double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz);
// ---- kernels_pairs.cu ---------------------------------------------------------------
int pairs_p2p(fmm_plan *p);
int pairs_p2p_prepare(fmm_plan *p);
int pairs_m2l_prepare(fmm_plan *p);
int pairs_proxy_points(fmm_plan *p);  // after the boxes of a build (a2): per-axis proxy points of every node
int pairs_m2l(fmm_plan *p);
int pairs_pc(fmm_plan *p);   // treecode: particle-cluster sums
int pairs_direct(fmm_ctx *c, int64_t N, const double *x, const double *y, const double *z,
                 const double *w0, const double *w1, const double *w2, const double *w3,
                 const double *px, const double *py, const double *pz /* non-NULL: source-momentum kernel */,
                 double gamma_bar, int raw, int64_t nt, const int64_t *tidx,
                 double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz);
int pairs_direct_noalloc(fmm_ctx *c, const fmm_particles_t *in, bool sm, double gamma_bar, int raw, int64_t nt, const int64_t *tidx,
                         double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz);  // scratch in a static device array
int pairs_source_weights(fmm_ctx *c, int64_t N, const double *px, const double *py, const double *pz,
                         const double *q, double q_scalar, double *w0, double *w1, double *w2, double *w3);
// ---- sort.cu --------------------------------------------------------------------------
// Stable LSD radix sort of (key, value) pairs on bits [bit_lo, bit_hi) of the key.  keys/vals are
// overwritten with the sorted sequence; tmp_* are scratch of the same length.
int sort_pairs_u64(fmm_ctx *c, uint64_t *keys, uint32_t *vals, uint64_t *tmp_keys, uint32_t *tmp_vals,
                   int64_t n, int bit_lo, int bit_hi);
int sort_pairs_u64_batched(fmm_ctx *c, uint64_t *keys, uint32_t *vals, uint64_t *tmp_keys, uint32_t *tmp_vals,
                           int64_t n, int batch, int bit_lo, int bit_hi);  // `batch` segments of length n, back to back
int sort_pairs_u32_batched(fmm_ctx *c, uint32_t *keys, uint32_t *vals, uint32_t *tmp_keys, uint32_t *tmp_vals, int64_t n, int batch);
int scan_exclusive_i32(fmm_ctx *c, const int32_t *in, int32_t *out, int64_t n);  // out may alias in

#ifdef __CUDACC__
// ---- device helpers -------------------------------------------------------------------

// w = D^{-3/2}.  Reading G17 (a coincident pair contributes nothing, which also removes i == j) is met without a test: every
// D is built as FMM_TINY_D + dx^2 + ..., so a coincident pair gets the finite w = 1e300 and g = w d = 0 exactly, while
// D + 1e-200 == D for every D > 1e-184 (distances above 1e-92 in the caller's unit).  One MUFU.RSQ64H seed y0 (relative error
// ~2^-20) and one cubic correction of y0^3:  D y0^2 = 1 - e  =>  D^{-3/2} = y0^3 (1-e)^{-3/2} = y0^3 (1 + 3/2 e + 15/8 e^2 + O(e^3)),
// truncation 35/16 e^3 < 1e-17 relative.  6 FP64 instructions, no integer ones.
#define FMM_TINY_D 1e-200
__device__ __forceinline__ double inv_r3(double D)
{
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(D));
    double t = y0 * y0;
    double e = fma(-D, t, 1.0);
    double c = y0 * t;
    double p = fma(1.875, e, 1.5);
    double pe = p * e;
    return fma(c, pe, c);
}

#endif
