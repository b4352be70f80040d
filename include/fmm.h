/*
 * fmm.h -- C ABI of libfmm_b200.so: the B200 (sm_100a, FP64) hot path of the
 * interpolation-based fast multipole method for the lab-frame relativistic space-charge
 * field (arXiv 2302.07567; citations are PAPER.md:<line> + equation / algorithm, or a
 * DESIGN.md reading where the paper is silent or garbled).
 *
 * Problem (eq. (3.1)-(3.2)): N particles with positions x_i, normalised
 * momenta p_i = gamma_i beta_i and charges q_i.  Wanted at every particle:
 *     E_i = 1/(4 pi eps0)    * sum_{j != i} q_j gamma_j g(x_i, x_j)
 *     B_i = 1/(4 pi eps0 c0) * sum_{j != i} q_j p_j x g(x_i, x_j)
 *     g(x_i, x_j) = (x_i - x_j) / (dx^2 + dy^2 + gamma_bar^2 dz^2)^{3/2},
 *     gamma_j = sqrt(1 + p_j.p_j),  gamma_bar^2 = 1 + pbar.pbar,  pbar = mean momentum.
 * Method (Alg 5.12): cluster tree (Alg 5.1/5.2) -> dual tree traversal
 * with the stretched admissibility condition (Alg 5.6-5.8, Alg 9.1) -> P2M/M2M (Alg 5.3-5.5)
 * -> M2L (Alg 5.9) + P2P (Alg 5.10) -> L2L/L2P (Alg 5.13-5.15).
 *
 * Conventions
 *   Pointers   every array pointer is a DEVICE pointer unless the name of the call ends in
 *              _host.  Arrays are structure-of-arrays FP64 of length N, caller-owned; inputs
 *              are read-only and need not outlive the call that takes them.
 *   Workspace  every byte of device workspace is obtained through the caller's allocator
 *              (fmm_alloc_fn / fmm_free_fn, e.g. PyTorch's caching allocator).  If both are
 *              NULL the library uses cudaMallocAsync / cudaFreeAsync on `cuda_stream`.  The
 *              allocator must be STREAM-ORDERED on `cuda_stream`: the library hands scratch
 *              back (free_) right after enqueueing the kernels that use it, while they may
 *              still be pending, so a block may be handed out again only to work that is
 *              enqueued on the same stream (PyTorch's allocator behaves like this for the
 *              stream that was current at allocation; the Python binding therefore runs every
 *              call of a plan under the stream the plan was created on).  A plan frees its
 *              remaining workspace in fmm_plan_destroy.
 *   Memory     a plan keeps about 110 N bytes of particle data, 80 P bytes per tree node for
 *              the moments and local fields (P = (n+1)^3), the two lists (4 to 16 bytes per
 *              entry) and, with the mean-gamma kernel, the reaction segments of the mutual
 *              near field: 48 bytes x ceil(N / leaves) per PAIR of P2P entries (0.9 GB at
 *              N = 2^20 with leaves of 256, 18 GB at N = 2.56e7 with leaves of 78; reported
 *              as fmm_stats_t.react_particles).  If the allocator refuses that block the plan
 *              falls back to the one-sided near field (same results to rounding, about 1.3x
 *              the P2P time) instead of failing.  A build needs 120 to 230 N bytes of scratch
 *              on top, returned before the call ends.
 *   Stream     all work is enqueued on `cuda_stream` (a cudaStream_t passed as void*; NULL =
 *              the legacy default stream).  fmm_plan_create / fmm_plan_update / fmm_plan_refit
 *              wait for the stream ONCE, after the traversal (the interaction-list lengths
 *              must be read back to size the lists; gamma_bar and the input check come with
 *              them), and return with the rest of the build enqueued; the inputs are no
 *              longer read after that wait.  The upward pass (P2M, M2M: Alg 5.3-5.5), which
 *              depends on the tree and the particles only, is enqueued by the build behind
 *              the copies it waits for, so that the device works on it while the host reads
 *              the lengths and returns to the caller; fmm_eval reuses those moments (they are
 *              recomputed inside fmm_eval only after fmm_plan_set_timing, so that the stage
 *              timers bracket them).  fmm_eval and fmm_direct only enqueue and return.
 *   Errors     0 on success, a negative FMM_E* code otherwise; no exceptions, no exit().
 *              Outputs are unspecified after an error.  A plan whose fmm_plan_update /
 *              fmm_plan_refit failed is marked invalid: fmm_eval returns FMM_EINVAL for it
 *              until a later update / refit succeeds (or destroy it).
 *   Globals    the library keeps three process-wide items, none of which carries results from
 *              one call to another: the launch counter behind fmm_launch_count, one side
 *              stream per device (fmm_plan_set_overlap), and a per-device flag that the table
 *              of Chebyshev points has been uploaded to constant memory.  Plans are otherwise
 *              independent; one plan must not be used from two threads at once.  The only
 *              environment variables read are FMM_TEST_WALK_STACK (a smaller traversal stack,
 *              used by the tests to reach the spill path) and FMM_TEST_KD_SORT_LI (the KD build
 *              takes its large-N route on small bunches); results do not depend on either.
 *   Order      outputs are in the caller's particle order.
 *   Units      SI; eps0 = 8.8541878128e-12 F/m, c0 = 299792458 m/s (CODATA 2018), unless
 *              FMM_RAW_SUMS is set (then the bare sums without prefactors are returned).
 *   Determinism  accumulation is target-owned (every target gathers over its own list in a
 *              fixed order); there are no floating-point atomics: identical inputs give
 *              bit-identical outputs run to run.
 */
#ifndef FMM_B200_H
#define FMM_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FMM_MAX_ORDER 12            /* interpolation degree n <= 12 (P = (n+1)^3 <= 2197)        */

/* flags word of fmm_params_t / fmm_direct */
#define FMM_TREE_KD            0u   /* Alg 5.2: median split along the axis of
                                       largest stretched extent (default)                        */
#define FMM_TREE_MORTON_MEDIAN 1u   /* particle order = 63-bit Morton key of the stretched, cube-
                                       normalised coordinates, same closed-form ranges (DESIGN T-3') */
#define FMM_TREE_MASK          1u
#define FMM_TREE_STOP_AT_N0    32u  /* non-balanced tree: Alg 5.2 as printed
                                       splits a cluster only while |S| > N0, so a cluster of exactly N0 particles on level
                                       kappa-1 stays a leaf; leaves then sit on levels kappa-1 and kappa of the same array
                                       tree and the two slots below such a leaf are unused.  It differs
                                       from the default (every node of level kappa is a leaf) only when
                                       floor(N / 2^(kappa-1)) == N0; either tree order.  In the export the unused slots
                                       have the range [0, 0), a zero box and zero expansions.              */
#define FMM_RAW_SUMS           4u   /* skip the prefactors of eq. (3.1)                          */
#define FMM_KERNEL_MEAN_GAMMA      0u  /* eq. (3.2) with gamma_bar in near and far field (default)    */
#define FMM_KERNEL_SOURCE_MOMENTUM 8u  /* alternative reading of Alg 5.10 (PAPER.md:393-394 write
                                          g(x_i, x_j, p_j); G6): the NEAR field (P2P, fmm_direct)
                                          of source j is stretched along j's own momentum,
                                          D = |d|^2 + (p_j . d)^2, the exact field of a uniformly moving
                                          charge; the far field (M2L) keeps eq. (3.2) with gamma_bar      */

#define FMM_METHOD_FMM      0u      /* Alg 5.12: dual tree traversal, M2L, L2L, L2P (default)              */
#define FMM_METHOD_TREECODE 16u     /* particle-cluster variant (Fig. 1a): Alg 9.1
                                       with the target held at a leaf; admissible clusters act on the target PARTICLES
                                       through their proxy points (no M2L / L2L / L2P).  In the statistics and the export
                                       the "m2l" list is then the particle-cluster list (target leaf, source cluster). */

#define FMM_OK          0
#define FMM_EINVAL     -1           /* bad argument: N < 1, order out of range, leaf_size < 1,
                                       theta <= 0 or non-finite, NULL pointer                    */
#define FMM_ENOMEM     -2           /* the allocator returned NULL                               */
#define FMM_ECUDA      -3           /* a CUDA call failed; text in fmm_last_error                */
#define FMM_ENONFINITE -4           /* NaN or Inf among x, y, z, px, py, pz, q (one fused scan in
                                       step a0), or the caller's gamma_bar is not finite          */
#define FMM_EOVERFLOW  -5           /* an interaction list exceeds 2^31-1 entries                */

typedef struct fmm_plan fmm_plan_t; /* opaque; owns its device workspace                          */

typedef void *(*fmm_alloc_fn)(size_t bytes, void *user); /* returns a device pointer (256-B aligned) or NULL */
typedef void (*fmm_free_fn)(void *ptr, void *user);

typedef struct {
    int64_t N;                      /* number of particles, >= 1                                 */
    const double *x, *y, *z;        /* positions [m]                                             */
    const double *px, *py, *pz;     /* normalised momenta gamma*beta [1]        */
    const double *q;                /* charges [C], or NULL: every particle carries q_scalar      */
    double q_scalar;
} fmm_particles_t;

typedef struct {
    int order_n;                    /* interpolation degree n, 1 <= n <= FMM_MAX_ORDER           */
    int leaf_size;                  /* N0 >= 1: maximum particles per leaf (Alg 5.2)             */
    double theta;                   /* admissibility parameter eta > 0 (eq. (4.3)) */
    double gamma_bar;               /* <= 0: computed from the mean momentum;
                                       > 0: use this value                                       */
    uint32_t flags;                 /* FMM_TREE_* | FMM_RAW_SUMS | FMM_KERNEL_* | FMM_METHOD_* */
} fmm_params_t;

/* Per-stage device times are CUDA-event times of the last fmm_plan_create/_update (tree, lists)
 * and of the last fmm_eval that ran with timing switched on (fmm_plan_set_timing). */
typedef struct {
    int64_t N;
    int32_t order_n, P, leaf_size, kappa;   /* P = (n+1)^3; kappa = tree depth     */
    int64_t nodes, leaves;                  /* 2^{kappa+1}-1, 2^kappa              */
    int64_t n_p2p, n_m2l;                   /* lengths of the two interaction lists (Alg 9.1)     */
    int64_t p2p_pairs, m2l_pairs;           /* kernel evaluations: particle pairs, proxy pairs    */
    double gamma_bar, theta;
    uint32_t flags;
    int32_t timing_valid;                   /* 1 if the eval times below were measured            */
    float ms_tree;                          /* a0-a2: gamma_bar, order, permute, bounding boxes    */
    float ms_lists;                         /* a3: traversal, sort, CSR                            */
    float ms_p2m, ms_m2m, ms_m2l, ms_l2l, ms_p2p, ms_l2p;  /* a4-a10 (l2p includes finalise)      */
    int64_t workspace_bytes;                /* device bytes currently held by the plan            */
    int32_t p2p_split, m2l_split;           /* row chunks per target of the near / far pair kernels (partial sums added in order) */
    int32_t p2p_mutual;                     /* 1: the near field evaluates every mated pair of leaves once for both directions   */
    int32_t early_leaves;                   /* FMM_TREE_STOP_AT_N0: leaves on level kappa-1 (0 otherwise)                        */
    int64_t react_particles;                /* particles in the reaction segments of the mutual near field (6 doubles each)       */
} fmm_stats_t;

/* Copies of the plan's integer structures and (optionally) expansions, for bit-exact
 * comparison with the oracle.  Every non-NULL field is a HOST pointer to caller memory of the
 * stated length; NULL fields are skipped.  Node ids are heap indices, root = 1
 * (PAPER.md:578-584); row i-1 describes node i. */
typedef struct {
    int64_t *perm;      /* [N]         tree position -> caller index                              */
    int64_t *node_lo;   /* [nodes]     half-open range [lo, hi) of tree positions                 */
    int64_t *node_hi;   /* [nodes]                                                                */
    double *bbox;       /* [nodes][6]  ax ay az bx by bz (tight)                  */
    int32_t *p2p_off;   /* [nodes+1]   CSR by target node (row i-1 = node i), P2P list            */
    int32_t *p2p_src;   /* [n_p2p]     source leaf ids, ascending within a target                 */
    int32_t *m2l_off;   /* [nodes+1]   CSR by target node, M2L list                               */
    int32_t *m2l_src;   /* [n_m2l]                                                                */
    double *M;          /* [nodes][P][4]  multipole moments (q gamma, q px, q py, q pz) after the
                                          upward pass of the last fmm_eval; nu = (nu1*(n+1)+nu2)*(n+1)+nu3 */
    double *L;          /* [nodes][P][6]  local fields (E, B sums) after the downward pass         */
} fmm_export_t;

/* a0-a3: mean momentum -> gamma_bar, tree order, bounding boxes, dual tree traversal, CSR lists.
 * Waits for the stream once (see "Stream" above).  *out is NULL on error. */
int fmm_plan_create(fmm_plan_t **out, const fmm_particles_t *particles, const fmm_params_t *params,
                    fmm_alloc_fn alloc, fmm_free_fn free_, void *user, void *cuda_stream);

/* Same N and parameters, new positions / momenta / charges: rebuilds tree and lists in place,
 * reusing the workspace where sizes allow. */
int fmm_plan_update(fmm_plan_t *plan, const fmm_particles_t *particles);

/* Refit for time stepping (the paper leaves the tracker outside): same N and
 * parameters, particles have moved a little.  The particle ORDER of the last fmm_plan_create / fmm_plan_update is kept
 * (no sort): the new positions / momenta / charges are gathered through it, gamma_bar, the tight bounding boxes and both
 * interaction lists are rebuilt on the new boxes.  Any partition into contiguous ranges is a valid cluster tree for
 * Alg 5.11 and the admissibility condition is evaluated on the actual boxes, so the result is a correct FMM of the same
 * order of accuracy; it is no longer the median split of the NEW positions.  Waits for the stream once. */
int fmm_plan_refit(fmm_plan_t *plan, const fmm_particles_t *particles);

/* Refit that also keeps BOTH INTERACTION LISTS of the last build ("reuse lists while particles move
 * little"): no sort and no traversal; gamma_bar, the source weights, the tight boxes and what hangs on them (transfer
 * matrices, proxy points, moments) are recomputed.  The kept lists still cover every ordered pair of leaves exactly once
 * (Alg 5.11 decides that on index ranges, which have not changed), so the result is a complete sum; what can degrade is the
 * accuracy of a kept far pair whose boxes no longer meet eq. (4.3).  *eta_eff (HOST pointer, may be NULL)
 * receives the largest max(diam S_t, diam S_s) / dist(S_t, S_s) (Alg 5.6-5.8 with the new gamma_bar) over the kept M2L list:
 * eta_eff < theta means every kept far pair is still admissible; the caller rebuilds (fmm_plan_refit / fmm_plan_update) when
 * it has grown past what it accepts (+inf if two clusters of a kept pair now share their centre; 0 with an empty M2L list).
 * Right after a traversal the largest ratio of the list sits just below theta, so any motion pushes it over: build the plan
 * with a margin (say theta = 0.42) and keep the lists while eta_eff <= the eta whose accuracy is wanted (say 0.5).  Past 0.5 the
 * boxes of a "far" pair may overlap (reading G11) and the error grows at once (measured: x5 at eta_eff = 0.506).
 * Needs a valid plan; FMM_EINVAL with FMM_METHOD_TREECODE.  Waits for the stream once; errors as fmm_plan_refit. */
int fmm_plan_refit_keep_lists(fmm_plan_t *plan, const fmm_particles_t *particles, double *eta_eff);

/* a4-a10: P2M, M2M, M2L, P2P, L2L, L2P, prefactors, scatter to caller order.  Enqueue only.
 * Ex..Bz: device arrays of length N, overwritten. */
int fmm_eval(fmm_plan_t *plan, double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz);

/* a11: direct O(N * n_targets) summation (Alg 5.10 with S_t = S_s = S).
 * target_idx: device array of n_targets particle indices, or NULL = all N particles in order
 * (then n_targets must be N).  gamma_bar <= 0: computed from the mean momentum.
 * Outputs: device arrays of length n_targets.  Enqueue only (synchronises only if gamma_bar <= 0). */
int fmm_direct(const fmm_particles_t *particles, double gamma_bar, uint32_t flags,
               int64_t n_targets, const int64_t *target_idx,
               double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz,
               fmm_alloc_fn alloc, fmm_free_fn free_, void *user, void *cuda_stream);

/* a11 for callers that must not allocate (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc):
 * the same sums as fmm_direct, computed by the same kernels, with NO allocation of any kind -- no allocator arguments, no
 * cudaMalloc / cudaFree / cudaMallocAsync; kernel launches only, enqueue only.  The scratch (source weights, partial sums)
 * is a fixed 8 MiB device array inside the library that every GPU which loads the library holds until the process exits.
 *   Limits     N <= FMM_NOALLOC_MAX_N and n_targets <= FMM_NOALLOC_MAX_N, else FMM_EINVAL (text in fmm_last_error(NULL)).
 *              gamma_bar must be given (> 0) unless FMM_KERNEL_SOURCE_MOMENTUM is set: computing it would need a host wait.
 *   Sharing    every call on a device uses the same array, which keeps the last call's contents (a call writes all it
 *              reads, so nothing needs clearing).  Calls that overlap on the GPU -- different streams or threads -- RACE on
 *              it: issue one call at a time per device, or order them on one stream.
 *   Accuracy   same kernels and summation scheme as fmm_direct's target-subset route; against fmm_direct the results agree
 *              to rounding (the number of source slices, and for all-targets calls the pair-sharing kernel, may differ).
 * Arguments as fmm_direct: device pointers, outputs of length n_targets, target_idx NULL = all N particles. */
#define FMM_NOALLOC_MAX_N 32768
int fmm_direct_noalloc(const fmm_particles_t *particles, double gamma_bar, uint32_t flags,
                       int64_t n_targets, const int64_t *target_idx,
                       double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz, void *cuda_stream);

/* Whole of Alg 5.12 from HOST memory: copies the particles to the device, fmm_plan_create,
 * fmm_eval, copies E and B back, destroys the plan.  All pointers in `particles` and the six
 * outputs are HOST pointers (pinned memory makes the copies asynchronous).  Returns after the
 * results are in host memory.  stats (may be NULL) receives the plan's statistics. */
int fmm_field_host(const fmm_particles_t *particles_host, const fmm_params_t *params,
                   double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz,
                   fmm_stats_t *stats,
                   fmm_alloc_fn alloc, fmm_free_fn free_, void *user, void *cuda_stream);

/* on != 0: fmm_eval brackets every stage with CUDA events (adds a few microseconds) and
 * fmm_plan_stats synchronises on the last one. */
int fmm_plan_set_timing(fmm_plan_t *plan, int on);

/* on != 0 (default is 0): fmm_eval runs P2P (a7) on a second stream of the plan, concurrently with P2M, M2M, M2L and L2L on
 * the caller's stream (a7 is independent of a4-a6, a8; PAPER.md:562-566 runs them as separate kernels too); the second
 * stream is forked from and joined into the caller's stream with events, so the call still behaves as work enqueued on
 * `cuda_stream`.  Results are bit-identical either way.  Stage timing (fmm_plan_set_timing) forces the serial order.
 * Measured on B200: 2 % faster at N = 2^20, n = 6 (the small upward / downward kernels hide behind P2P), but P2P itself
 * runs up to 45 % slower whenever other grids are resident beside it, so this is opt-in for far-field-heavy settings. */
int fmm_plan_set_overlap(fmm_plan_t *plan, int on);
int fmm_plan_stats(fmm_plan_t *plan, fmm_stats_t *stats);
int fmm_plan_export(fmm_plan_t *plan, fmm_export_t *out);  /* synchronises the stream */
void fmm_plan_destroy(fmm_plan_t *plan);

/* Number of kernel launches the library has enqueued in this process (bench.py's gpu_launches). */
int64_t fmm_launch_count(void);

const char *fmm_strerror(int code);
const char *fmm_last_error(const fmm_plan_t *plan);  /* plan may be NULL: last error of a plan-less call */
const char *fmm_version(void);

#ifdef __cplusplus
}
#endif
#endif /* FMM_B200_H */
