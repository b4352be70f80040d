/*
 * fmm_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU (FP64) statement of what the hot path of
 * arXiv 2302.07567 computes.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call this.  It shares no
 * code, header, table or helper with the CUDA path under
 * paper_2302_07567_b200/csrc/, and includes nothing from it.
 *
 * Two parts:
 *   O1  direct O(N^2) summation of eq. (3.1)-(3.2)   (Alg 5.10
 *       PAPER.md:386-398 with S_t = S_s = S)
 *   O2  the serial FMM of Alg 5.12, step by step: Alg 5.1/5.2
 *       tree, Alg 5.3-5.5 upward pass, Alg 9.1 dual tree traversal with the
 *       stretched admissibility of Alg 5.6-5.8, Alg 5.9 M2L, Alg 5.10 P2P,
 *       Alg 5.13-5.15 downward pass.
 *
 * Pins (tests/test_oracle_*.py, all "-m not gpu"): closed-form field of a uniformly
 * moving charge, Coulomb limit, B = beta x E / c0, symmetry, Theorem 1 polynomial
 * reproduction, moment conservation, M2M == P2M at the parent, Lemma 1, empty far
 * list => FMM == direct, brute-force coverage of the leaf x leaf matrix, tree
 * invariants, convergence in n and eta; the traversal's split rule (Alg 5.11: target iff
 * diam(S_t) > diam(S_s), ties split the source) by a plain-Python restatement of Alg 5.11 whose
 * lists must equal these exactly, incl. mirror-symmetric inputs with bit-identical radii and a
 * hand-worked example; Alg 5.1's first-maximiser rule by two- and three-way non-zero ties
 * (tests/test_oracle_traversal_pins.py); the non-balanced option ORC_TREE_STOP_AT_N0 by Alg 5.1 / 5.2 / 5.11 restated on
 * plain index sets, Alg 5.2's invariants and brute-force coverage (tests/test_oracle_nonbalanced_pins.py); list reuse
 * (orc_plan_set_lists, orc_plan_eta_eff) by list exchange between plans, the all-near list == direct sum and a numpy
 * restatement of Alg 5.6-5.8 (tests/test_oracle_kept_lists_pins.py).  The ABSOLUTE FMM-vs-direct error values
 * are "parity unpinned" by the paper (Fig. 2 is an image): only their trend is pinned.
 *
 * All pointers are HOST pointers.  Arrays are caller-owned unless stated.
 */
#ifndef FMM_ORACLE_H
#define FMM_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORC_TREE_KD            0  /* Alg 5.2, reading T-3   */
#define ORC_TREE_MORTON_MEDIAN 1  /* DESIGN.md reading T-3' (north_star's Morton order)  */
#define ORC_TREE_GIVEN         2  /* particle order supplied by the caller (orc_plan_create_given_order) */

/* flags word passed as `raw`: */
#define ORC_RAW_SUMS               1  /* no SI prefactors                                                  */
#define ORC_KERNEL_SOURCE_MOMENTUM 2  /* near field (P2P, direct) stretched along the source's own momentum,
                                         D = |d|^2 + (p_j.d)^2 (alternative reading of Alg 5.10, G6);
                                         the far field keeps eq. (3.2) with gamma_bar                      */
#define ORC_TREE_STOP_AT_N0        4  /* Alg 5.2 as printed: a cluster is split only while |S| > N0,
                                         so a cluster of exactly N0 particles one level above kappa stays a leaf and the
                                         tree is not balanced (leaves on levels kappa-1 and kappa).
                                         It sits in the same array of section 8: the slots below such
                                         a leaf are unused (range [0,0), zero box).  Default (flag clear): reading T-1,
                                         every node of level kappa is a leaf.                              */

typedef struct orc_plan orc_plan_t;

/* gamma_bar^2 = 1 + pbar.pbar, pbar = plain mean momentum (reading G16). */
double orc_gamma_bar(int64_t N, const double *px, const double *py, const double *pz);

/* Reference interpolation nodes on [-1,1] (reading I-1) and 1-D Lagrange basis on [a,b]
 * in barycentric form with the exact-hit rule (readings I-2..I-4). ell has n+1 entries. */
void orc_cheb_nodes(int n, double *c);
void orc_basis_1d(int n, double a, double b, double x, double *ell);

/* O1. Direct sum at the targets tidx[0..nt) (NULL = all N, in order).
 * q == NULL -> every particle has charge q_scalar.  raw != 0 -> no SI prefactors.
 * Outputs have length nt (or N).  Returns 0. */
int orc_direct(int64_t N, const double *x, const double *y, const double *z,
               const double *px, const double *py, const double *pz,
               const double *q, double q_scalar, double gamma_bar, int raw,
               int64_t nt, const int64_t *tidx,
               double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz);

/* O2. Build tree + interaction lists (Alg 5.2, Alg 9.1). gamma_bar <= 0 -> orc_gamma_bar. */
orc_plan_t *orc_plan_create(int64_t N, const double *x, const double *y, const double *z,
                            const double *px, const double *py, const double *pz,
                            const double *q, double q_scalar,
                            int n, int N0, double theta, double gamma_bar,
                            int tree_mode, int raw);
/* Same, over a particle order supplied by the caller (perm[N]: tree position -> particle index, a permutation):
 * closed-form node ranges (T-2) over that order, tight boxes, same traversal.  Refit of an existing partition. */
orc_plan_t *orc_plan_create_given_order(int64_t N, const double *x, const double *y, const double *z,
                                        const double *px, const double *py, const double *pz,
                                        const double *q, double q_scalar,
                                        int n, int N0, double theta, double gamma_bar, int raw, const int64_t *perm);
void orc_plan_destroy(orc_plan_t *);

/* sizes: out[0]=kappa out[1]=nodes out[2]=leaves out[3]=P out[4]=len(p2p) out[5]=len(m2l) */
void   orc_plan_sizes(const orc_plan_t *, int64_t *out);
double orc_plan_gamma_bar(const orc_plan_t *);
/* perm[N]: tree position -> original particle index */
void orc_plan_perm(const orc_plan_t *, int64_t *perm);
/* node i = 1..nodes (heap index): lo[i-1], hi[i-1] (half-open), bbox[(i-1)*6 + {ax,ay,az,bx,by,bz}] */
void orc_plan_nodes(const orc_plan_t *, int64_t *lo, int64_t *hi, double *bbox);
/* leaf[i-1] = 1 if heap node i is a leaf, 0 if it has children, 2 if the slot is unused (below a leaf of level
 * kappa-1, ORC_TREE_STOP_AT_N0 only) */
void orc_plan_leaf_flags(const orc_plan_t *, int8_t *leaf);
/* lists sorted by (target, source); node ids are heap indices (root = 1). */
void orc_plan_lists(const orc_plan_t *, int32_t *p2p_t, int32_t *p2p_s, int32_t *m2l_t, int32_t *m2l_s);

/* Lists kept from an earlier traversal (refit with list reuse): replaces both lists of the plan
 * by the caller's pairs (heap ids; every target / source of the P2P list must be a leaf of this plan), sorted by
 * (target, source) here.  Alg 5.12 is then evaluated over them exactly as over its own.  Returns 0, or -1 for a bad id. */
int orc_plan_set_lists(orc_plan_t *, int64_t np2p, const int32_t *p2p_t, const int32_t *p2p_s,
                       int64_t nm2l, const int32_t *m2l_t, const int32_t *m2l_s);
/* The largest max(diam S_t, diam S_s) / dist(S_t, S_s) (Alg 5.6-5.8) over the plan's M2L list, with
 * the plan's boxes and gamma_bar: below theta for lists the plan's own traversal made (Alg 5.8); 0 for an empty list. */
double orc_plan_eta_eff(const orc_plan_t *);

/* Upward pass (Alg 5.5). M_out (may be NULL) receives [nodes][P][4] = (q*gamma, q*px, q*py, q*pz)
 * moments, node i at row i-1, proxy nu = (nu1*(n+1)+nu2)*(n+1)+nu3. */
void orc_upward(orc_plan_t *, double *M_out);
/* P2M evaluated directly at an arbitrary node from its member particles (eq. (2.4)) - pin P7. */
void orc_p2m_node(const orc_plan_t *, int64_t node, double *M_node /* [P][4] */);

/* Full evaluation (Alg 5.12 after subdivide): upward, M2L+P2P over the lists, downward.
 * nsel > 0: only the target leaves sel[0..nsel) (heap ids) are evaluated; outputs of other
 * particles are left untouched.  Outputs are length N in CALLER order.
 * L_out (may be NULL): [nodes][P][6] cumulative local fields after the downward pass
 * (only meaningful for nodes on a selected root-leaf chain).
 * near_only/far_only: 1 -> only P2P part / only far (L2P) part is written (pins P8, P9). */
int orc_eval(orc_plan_t *, int64_t nsel, const int64_t *sel, int part /*0 all,1 near,2 far*/,
             double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz,
             double *L_out);

/* Treecode variant (particle-cluster; Fig. 1a): Alg 9.1 started at (t, root) for
 * every target leaf t -> PP list (leaf, leaf: direct sum) and PC list (leaf, admissible cluster: the leaf's particles
 * evaluate the kernel at the cluster's proxy points with its moments).  Lists sorted by (target, source). */
void orc_treecode_sizes(orc_plan_t *, int64_t *out /* [2]: len(pp), len(pc) */);
void orc_treecode_lists(orc_plan_t *, int32_t *pp_t, int32_t *pp_s, int32_t *pc_t, int32_t *pc_s);
int  orc_eval_treecode(orc_plan_t *, double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz);

/* M2L sums only (before any L2L): L_raw[nodes][P][6]. Pin P8 (Lemma 1). */
void orc_m2l_raw(orc_plan_t *, double *L_raw);

int orc_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
