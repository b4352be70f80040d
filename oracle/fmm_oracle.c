/*
 * fmm_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.  See fmm_oracle.h.
 *
 * Plain C99, FP64, compiled with -O2 -ffp-contract=off (no FMA contraction: the
 * admissibility test of Alg 5.8 must round every product and sum separately so
 * that the GPU can reproduce the interaction lists bit for bit).
 * OpenMP is used only over independent targets (particles / target nodes); the
 * summation order inside one target is the order written here.
 *
 * Citations are PAPER.md:<line> (+ the equation / algorithm) or a DESIGN.md reading
 * (G*, T*, I*, D*) where the paper is silent or garbled.
 */
#define _GNU_SOURCE
#include "fmm_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_EPS0 8.8541878128e-12 /* F/m, CODATA 2018 */
#define ORC_C0 299792458.0        /* m/s */
#define ORC_PI 3.14159265358979323846

struct orc_plan {
    int64_t N;
    int n, n1, P, N0, kappa, tree_mode, raw;
    int64_t nodes, leaves;
    double theta, gamma_bar;
    double s[3];
    double *x, *y, *z;    /* caller order */
    double *w;            /* [N][4] source weights q*gamma, q*px, q*py, q*pz, caller order */
    double *pm;           /* [N][3] plain momenta px, py, pz, caller order (source-momentum near field) */
    int64_t *perm;        /* tree position -> caller index */
    int64_t *lo, *hi;     /* [nodes+1], heap index, half open */
    signed char *leaf;    /* [nodes+1]: 1 leaf, 0 has children, 2 unused slot below a leaf of level kappa-1 */
    double *bbox;         /* [nodes+1][6] ax ay az bx by bz */
    int64_t np2p, nm2l, cap_p2p, cap_m2l;
    int32_t *p2p, *m2l;   /* pairs (t,s) interleaved */
    int64_t ntcpp, ntcpc, cap_tcpp, cap_tcpc;
    int32_t *tcpp, *tcpc; /* treecode lists: (target leaf, source leaf) and (target leaf, source cluster) */
    double *M;            /* [nodes+1][P][4] */
    int have_M;
    double cheb[64];
};

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------- */
/* gamma_bar^2 = 1 + pbar.pbar, pbar = average momentum (G16: plain mean). */
double orc_gamma_bar(int64_t N, const double *px, const double *py, const double *pz)
{
    double sx = 0.0, sy = 0.0, sz = 0.0;
    for (int64_t j = 0; j < N; ++j) {
        sx += px[j];
        sy += py[j];
        sz += pz[j];
    }
    double mx = sx / (double)N, my = sy / (double)N, mz = sz / (double)N;
    return sqrt(1.0 + (mx * mx + my * my + mz * mz));
}

/* eq. (3.2): g = d / (dx^2 + dy^2 + gamma_bar^2 dz^2)^{3/2};
 * G17: the contribution is 0 iff D == 0 (covers i == j). */
static inline double kernel_w(double dx, double dy, double dz, double g2)
{
    double D = dx * dx + dy * dy + g2 * dz * dz;
    return (D > 0.0) ? 1.0 / (D * sqrt(D)) : 0.0;
}

/* One source (weights m = q*gamma, q*p) acting on one target: eq. (3.1) without the
 * prefactor, E += gamma_j g ; B += p_j x g   (Alg 5.10 lines PAPER.md:393-394, reading G6). */
static inline void accumulate(double dx, double dy, double dz, double g2, const double *m, double *acc)
{
    double w = kernel_w(dx, dy, dz, g2);
    double gx = w * dx, gy = w * dy, gz = w * dz;
    acc[0] += m[0] * gx;
    acc[1] += m[0] * gy;
    acc[2] += m[0] * gz;
    acc[3] += m[2] * gz - m[3] * gy; /* (p x g)_x = py gz - pz gy */
    acc[4] += m[3] * gx - m[1] * gz; /* (p x g)_y = pz gx - px gz */
    acc[5] += m[1] * gy - m[2] * gx; /* (p x g)_z = px gy - py gx */
}

/* Alternative reading of Alg 5.10 (PAPER.md:393-394 write g(x_i, x_j, p_j); G6):
 * the NEAR field of source j is stretched along j's own momentum, D = |d|^2 + (p_j . d)^2 with p_j = gamma_j beta_j.
 * For p_j = (0, 0, p) this is dx^2 + dy^2 + (1 + p^2) dz^2 = dx^2 + dy^2 + gamma_j^2 dz^2: eq. (3.2) with the
 * source's own gamma, i.e. the exact field of a uniformly moving charge.  pj = plain momentum of the source. */
static inline void accumulate_sm(double dx, double dy, double dz, const double *pj, const double *m, double *acc)
{
    double pd = pj[0] * dx + pj[1] * dy + pj[2] * dz;
    double D = (dx * dx + dy * dy + dz * dz) + pd * pd;
    double w = (D > 0.0) ? 1.0 / (D * sqrt(D)) : 0.0;
    double gx = w * dx, gy = w * dy, gz = w * dz;
    acc[0] += m[0] * gx;
    acc[1] += m[0] * gy;
    acc[2] += m[0] * gz;
    acc[3] += m[2] * gz - m[3] * gy;
    acc[4] += m[3] * gx - m[1] * gz;
    acc[5] += m[1] * gy - m[2] * gx;
}

/* `raw` is a flags word: bit 0 = no SI prefactors, bit 1 = source-momentum near field (ORC_KERNEL_SOURCE_MOMENTUM). */
static void prefactors(int raw, double *cE, double *cB)
{
    if (raw & 1) {
        *cE = 1.0;
        *cB = 1.0;
    } else {
        *cE = 1.0 / (4.0 * ORC_PI * ORC_EPS0);          /* eq. (3.1) */
        *cB = 1.0 / (4.0 * ORC_PI * ORC_EPS0 * ORC_C0); /* eq. (3.1) */
    }
}

/* O1 ---------------------------------------------------------------------- */
int orc_direct(int64_t N, const double *x, const double *y, const double *z,
               const double *px, const double *py, const double *pz,
               const double *q, double q_scalar, double gamma_bar, int raw,
               int64_t nt, const int64_t *tidx,
               double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz)
{
    double g2 = gamma_bar * gamma_bar;
    double cE, cB;
    prefactors(raw, &cE, &cB);
    double *w = (double *)malloc(sizeof(double) * 4 * (size_t)N);
    for (int64_t j = 0; j < N; ++j) {
        double qj = q ? q[j] : q_scalar;
        double gam = sqrt(1.0 + (px[j] * px[j] + py[j] * py[j] + pz[j] * pz[j]));
        w[4 * j + 0] = qj * gam;
        w[4 * j + 1] = qj * px[j];
        w[4 * j + 2] = qj * py[j];
        w[4 * j + 3] = qj * pz[j];
    }
    int64_t T = tidx ? nt : N;
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < T; ++k) {
        int64_t i = tidx ? tidx[k] : k;
        double acc[6] = {0, 0, 0, 0, 0, 0};
        if (raw & 2) {
            for (int64_t j = 0; j < N; ++j) {
                double pj[3] = {px[j], py[j], pz[j]};
                accumulate_sm(x[i] - x[j], y[i] - y[j], z[i] - z[j], pj, &w[4 * j], acc);
            }
        } else {
            for (int64_t j = 0; j < N; ++j)
                accumulate(x[i] - x[j], y[i] - y[j], z[i] - z[j], g2, &w[4 * j], acc);
        }
        Ex[k] = cE * acc[0];
        Ey[k] = cE * acc[1];
        Ez[k] = cE * acc[2];
        Bx[k] = cB * acc[3];
        By[k] = cB * acc[4];
        Bz[k] = cB * acc[5];
    }
    free(w);
    return 0;
}

/* Interpolation ----------------------------------------------------------- */
/* I-1: c_k = cos(k pi / n) written as sin(pi (n-2k) / (2n)) so that c_k = -c_{n-k}. */
void orc_cheb_nodes(int n, double *c)
{
    for (int k = 0; k <= n; ++k)
        c[k] = sin(ORC_PI * (double)(n - 2 * k) / (double)(2 * n));
    c[0] = 1.0;
    c[n] = -1.0;
}

static void node_points(int n, const double *cheb, double a, double b, double *xi)
{
    double mid = (a + b) * 0.5, half = (b - a) * 0.5; /* I-3 */
    for (int k = 0; k <= n; ++k)
        xi[k] = mid + half * cheb[k];
}

static void basis_1d_c(int n, const double *cheb, double a, double b, double x, double *ell)
{
    double xi[64], t[64];
    node_points(n, cheb, a, b, xi);
    for (int k = 0; k <= n; ++k) {
        if (x == xi[k]) { /* I-4 exact hit: first such k */
            for (int m = 0; m <= n; ++m)
                ell[m] = 0.0;
            ell[k] = 1.0;
            return;
        }
    }
    double S = 0.0;
    for (int k = 0; k <= n; ++k) {
        double wk = (k == 0 || k == n) ? 0.5 : 1.0; /* I-2 */
        if (k & 1)
            wk = -wk;
        t[k] = wk / (x - xi[k]);
        S += t[k];
    }
    for (int k = 0; k <= n; ++k)
        ell[k] = t[k] / S;
}

void orc_basis_1d(int n, double a, double b, double x, double *ell)
{
    double c[64];
    orc_cheb_nodes(n, c);
    basis_1d_c(n, c, a, b, x, ell);
}

/* Tree ---------------------------------------------------------------------- */
typedef struct {
    const double *coord;
} sort_ctx;

static int cmp_coord_idx(const void *pa, const void *pb, void *vctx)
{
    const sort_ctx *ctx = (const sort_ctx *)vctx;
    int64_t a = *(const int64_t *)pa, b = *(const int64_t *)pb;
    double ca = ctx->coord[a], cb = ctx->coord[b];
    if (ca < cb) return -1;
    if (ca > cb) return 1;
    return (a < b) ? -1 : (a > b);
}

static int cmp_idx(const void *pa, const void *pb)
{
    int64_t a = *(const int64_t *)pa, b = *(const int64_t *)pb;
    return (a < b) ? -1 : (a > b);
}

static void tight_bbox(const orc_plan_t *p, int64_t lo, int64_t hi, double *bb)
{
    /* a_g = min, b_g = max over the members. Empty node: zeros. */
    if (hi <= lo) {
        for (int k = 0; k < 6; ++k) bb[k] = 0.0;
        return;
    }
    int64_t j0 = p->perm[lo];
    bb[0] = bb[3] = p->x[j0];
    bb[1] = bb[4] = p->y[j0];
    bb[2] = bb[5] = p->z[j0];
    for (int64_t k = lo + 1; k < hi; ++k) {
        int64_t j = p->perm[k];
        if (p->x[j] < bb[0]) bb[0] = p->x[j];
        if (p->x[j] > bb[3]) bb[3] = p->x[j];
        if (p->y[j] < bb[1]) bb[1] = p->y[j];
        if (p->y[j] > bb[4]) bb[4] = p->y[j];
        if (p->z[j] < bb[2]) bb[2] = p->z[j];
        if (p->z[j] > bb[5]) bb[5] = p->z[j];
    }
}

/* Alg 5.2 on the array tree of section 8,
 * readings T-1..T-4, G7-G9, G13. */
static void subdivide(orc_plan_t *p, int64_t node, int64_t lo, int64_t hi, int level)
{
    p->lo[node] = lo;
    p->hi[node] = hi;
    double *bb = &p->bbox[6 * node];
    tight_bbox(p, lo, hi, bb);
    /* T-1: every node of level kappa is a leaf.  ORC_TREE_STOP_AT_N0: Alg 5.2 as printed,
     * "if |S| > N0 then split ... else children(S) = {}" -- a node of at most N0 particles is a leaf wherever it is
     * (a node of level kappa never holds more than N0). */
    if (level == p->kappa || ((p->raw & ORC_TREE_STOP_AT_N0) && hi - lo <= p->N0)) {
        p->leaf[node] = 1; /* canonical order inside a leaf = ascending original index (T-3) */
        if (p->tree_mode == ORC_TREE_KD)
            qsort(p->perm + lo, (size_t)(hi - lo), sizeof(int64_t), cmp_idx);
        return;
    }
    p->leaf[node] = 0;
    int64_t mid = lo + (hi - lo + 1) / 2; /* T-2: left child gets ceil(size/2) */
    if (p->tree_mode == ORC_TREE_KD && hi > lo) {
        /* Alg 5.1: k = argmax s_k (b_k - a_k); G9: first maximiser */
        int axis = 0;
        double best = p->s[0] * (bb[3] - bb[0]);
        for (int k = 1; k < 3; ++k) {
            double e = p->s[k] * (bb[3 + k] - bb[k]);
            if (e > best) {
                best = e;
                axis = k;
            }
        }
        sort_ctx ctx;
        ctx.coord = (axis == 0) ? p->x : (axis == 1) ? p->y : p->z;
        /* G8: total order (coordinate, original index) decides membership */
        qsort_r(p->perm + lo, (size_t)(hi - lo), sizeof(int64_t), cmp_coord_idx, &ctx);
    }
    subdivide(p, 2 * node, lo, mid, level + 1);
    subdivide(p, 2 * node + 1, mid, hi, level + 1);
}

/* T-3': 63-bit Morton key of the stretched, cube-normalised coordinates. */
typedef struct {
    uint64_t key;
    int64_t idx;
} mkey_t;

static int cmp_mkey(const void *pa, const void *pb)
{
    const mkey_t *a = (const mkey_t *)pa, *b = (const mkey_t *)pb;
    if (a->key < b->key) return -1;
    if (a->key > b->key) return 1;
    return (a->idx < b->idx) ? -1 : (a->idx > b->idx);
}

static void morton_order(orc_plan_t *p)
{
    int64_t N = p->N;
    double lo[3], hi[3];
    for (int k = 0; k < 3; ++k) {
        const double *c = (k == 0) ? p->x : (k == 1) ? p->y : p->z;
        lo[k] = hi[k] = p->s[k] * c[0];
        for (int64_t j = 1; j < N; ++j) {
            double u = p->s[k] * c[j];
            if (u < lo[k]) lo[k] = u;
            if (u > hi[k]) hi[k] = u;
        }
    }
    double L = hi[0] - lo[0];
    if (hi[1] - lo[1] > L) L = hi[1] - lo[1];
    if (hi[2] - lo[2] > L) L = hi[2] - lo[2];
    mkey_t *keys = (mkey_t *)malloc(sizeof(mkey_t) * (size_t)N);
    for (int64_t j = 0; j < N; ++j) {
        uint64_t qk[3];
        for (int k = 0; k < 3; ++k) {
            const double *c = (k == 0) ? p->x : (k == 1) ? p->y : p->z;
            double u = p->s[k] * c[j];
            double f = (L > 0.0) ? floor((u - lo[k]) / L * 2097152.0) : 0.0;
            if (f > 2097151.0) f = 2097151.0;
            if (f < 0.0) f = 0.0;
            qk[k] = (uint64_t)f;
        }
        uint64_t key = 0; /* bit b of x -> 3b, of y -> 3b+1, of z -> 3b+2 (z most significant) */
        for (int b = 0; b < 21; ++b) {
            key |= ((qk[0] >> b) & 1ull) << (3 * b);
            key |= ((qk[1] >> b) & 1ull) << (3 * b + 1);
            key |= ((qk[2] >> b) & 1ull) << (3 * b + 2);
        }
        keys[j].key = key;
        keys[j].idx = j;
    }
    qsort(keys, (size_t)N, sizeof(mkey_t), cmp_mkey);
    for (int64_t j = 0; j < N; ++j)
        p->perm[j] = keys[j].idx;
    free(keys);
}

/* Dual tree traversal --------------------------------------------------------- */
/* Alg 5.6 squared: r^2 = || s o (b - a)/2 ||^2 (reading D-2: no sqrt, no division). */
static double diam2(const orc_plan_t *p, int64_t i)
{
    const double *bb = &p->bbox[6 * i];
    double hx = (bb[3] - bb[0]) * 0.5, hy = (bb[4] - bb[1]) * 0.5, hz = (bb[5] - bb[2]) * 0.5;
    double ex = p->s[0] * hx, ey = p->s[1] * hy, ez = p->s[2] * hz;
    return (ex * ex + ey * ey) + ez * ez;
}

/* Alg 5.7 squared: d^2 = || s o (c_i - c_j) ||^2 with c = (a + b)/2. */
static double dist2(const orc_plan_t *p, int64_t i, int64_t j)
{
    const double *bi = &p->bbox[6 * i], *bj = &p->bbox[6 * j];
    double cix = (bi[0] + bi[3]) * 0.5, ciy = (bi[1] + bi[4]) * 0.5, ciz = (bi[2] + bi[5]) * 0.5;
    double cjx = (bj[0] + bj[3]) * 0.5, cjy = (bj[1] + bj[4]) * 0.5, cjz = (bj[2] + bj[5]) * 0.5;
    double ex = p->s[0] * (cix - cjx), ey = p->s[1] * (ciy - cjy), ez = p->s[2] * (ciz - cjz);
    return (ex * ex + ey * ey) + ez * ez;
}

static void push_pair(int32_t **list, int64_t *n, int64_t *cap, int64_t t, int64_t s)
{
    if (*n == *cap) {
        *cap = *cap ? 2 * *cap : 1024;
        *list = (int32_t *)realloc(*list, sizeof(int32_t) * 2 * (size_t)*cap);
    }
    (*list)[2 * *n] = (int32_t)t;
    (*list)[2 * *n + 1] = (int32_t)s;
    ++*n;
}

/* Alg 9.1, i = target, j = source; readings D-1..D-3, G12, G22. */
static void dualtraversefillitl(orc_plan_t *p, int64_t i, int64_t j)
{
    if (p->hi[i] == p->lo[i] || p->hi[j] == p->lo[j])
        return; /* an empty cluster has nothing to receive or to send */
    int leaf_i = (p->leaf[i] == 1), leaf_j = (p->leaf[j] == 1);
    if (leaf_i && leaf_j) {
        push_pair(&p->p2p, &p->np2p, &p->cap_p2p, i, j);
        return;
    }
    double ri = diam2(p, i), rj = diam2(p, j), d2 = dist2(p, i, j);
    double rmax = (ri > rj) ? ri : rj;
    int adm = rmax < (p->theta * p->theta) * d2; /* Alg 5.8 squared */
    if (adm) {
        push_pair(&p->m2l, &p->nm2l, &p->cap_m2l, i, j);
    } else if (leaf_i) {
        dualtraversefillitl(p, i, 2 * j);
        dualtraversefillitl(p, i, 2 * j + 1);
    } else if (leaf_j) {
        dualtraversefillitl(p, 2 * i, j);
        dualtraversefillitl(p, 2 * i + 1, j);
    } else if (ri > rj) {
        dualtraversefillitl(p, 2 * i, j);
        dualtraversefillitl(p, 2 * i + 1, j);
    } else {
        dualtraversefillitl(p, i, 2 * j);
        dualtraversefillitl(p, i, 2 * j + 1);
    }
}

static int cmp_pair(const void *pa, const void *pb)
{
    const int32_t *a = (const int32_t *)pa, *b = (const int32_t *)pb;
    if (a[0] != b[0]) return (a[0] < b[0]) ? -1 : 1;
    return (a[1] < b[1]) ? -1 : (a[1] > b[1]);
}

/* Plan ------------------------------------------------------------------------ */
static orc_plan_t *plan_create(int64_t N, const double *x, const double *y, const double *z,
                               const double *px, const double *py, const double *pz,
                               const double *q, double q_scalar,
                               int n, int N0, double theta, double gamma_bar,
                               int tree_mode, int raw, const int64_t *given_perm);

orc_plan_t *orc_plan_create(int64_t N, const double *x, const double *y, const double *z,
                            const double *px, const double *py, const double *pz,
                            const double *q, double q_scalar,
                            int n, int N0, double theta, double gamma_bar,
                            int tree_mode, int raw)
{
    if (tree_mode != ORC_TREE_KD && tree_mode != ORC_TREE_MORTON_MEDIAN)
        return NULL;
    return plan_create(N, x, y, z, px, py, pz, q, q_scalar, n, N0, theta, gamma_bar, tree_mode, raw, NULL);
}

/* Cluster tree over a GIVEN particle order (refit of an existing partition): node ranges are the
 * closed-form ranges of T-2 over perm, bounding boxes are tight (T-4), lists come from the same traversal.  Any
 * partition into contiguous ranges is a valid cluster tree for Alg 5.11 (PAPER.md:253 only asks for a partition);
 * the admissibility condition is evaluated on the actual bounding boxes. */
orc_plan_t *orc_plan_create_given_order(int64_t N, const double *x, const double *y, const double *z,
                                        const double *px, const double *py, const double *pz,
                                        const double *q, double q_scalar,
                                        int n, int N0, double theta, double gamma_bar, int raw, const int64_t *perm)
{
    if (!perm) return NULL;
    return plan_create(N, x, y, z, px, py, pz, q, q_scalar, n, N0, theta, gamma_bar, ORC_TREE_GIVEN, raw, perm);
}

static orc_plan_t *plan_create(int64_t N, const double *x, const double *y, const double *z,
                               const double *px, const double *py, const double *pz,
                               const double *q, double q_scalar,
                               int n, int N0, double theta, double gamma_bar,
                               int tree_mode, int raw, const int64_t *given_perm)
{
    if (N < 1 || n < 1 || n > 31 || N0 < 1 || !(theta > 0.0))
        return NULL;
    orc_plan_t *p = (orc_plan_t *)calloc(1, sizeof(orc_plan_t));
    p->N = N;
    p->n = n;
    p->n1 = n + 1;
    p->P = (n + 1) * (n + 1) * (n + 1);
    p->N0 = N0;
    p->theta = theta;
    p->tree_mode = tree_mode;
    p->raw = raw;
    p->gamma_bar = (gamma_bar > 0.0) ? gamma_bar : orc_gamma_bar(N, px, py, pz);
    p->s[0] = 1.0;
    p->s[1] = 1.0;
    p->s[2] = p->gamma_bar;
    /* T-1: smallest kappa with N0 * 2^kappa >= N */
    int kappa = 0;
    while (((int64_t)N0 << kappa) < N)
        ++kappa;
    p->kappa = kappa;
    p->leaves = (int64_t)1 << kappa;
    p->nodes = ((int64_t)2 << kappa) - 1;
    orc_cheb_nodes(n, p->cheb);

    size_t sz = sizeof(double) * (size_t)N;
    p->x = (double *)malloc(sz);
    p->y = (double *)malloc(sz);
    p->z = (double *)malloc(sz);
    memcpy(p->x, x, sz);
    memcpy(p->y, y, sz);
    memcpy(p->z, z, sz);
    p->w = (double *)malloc(4 * sz);
    for (int64_t j = 0; j < N; ++j) {
        double qj = q ? q[j] : q_scalar;
        double gam = sqrt(1.0 + (px[j] * px[j] + py[j] * py[j] + pz[j] * pz[j]));
        p->w[4 * j + 0] = qj * gam;
        p->w[4 * j + 1] = qj * px[j];
        p->w[4 * j + 2] = qj * py[j];
        p->w[4 * j + 3] = qj * pz[j];
    }
    p->pm = (double *)malloc(3 * sz);
    for (int64_t j = 0; j < N; ++j) {
        p->pm[3 * j + 0] = px[j];
        p->pm[3 * j + 1] = py[j];
        p->pm[3 * j + 2] = pz[j];
    }
    p->perm = (int64_t *)malloc(sizeof(int64_t) * (size_t)N);
    for (int64_t j = 0; j < N; ++j)
        p->perm[j] = given_perm ? given_perm[j] : j;
    p->lo = (int64_t *)calloc((size_t)p->nodes + 1, sizeof(int64_t));
    p->hi = (int64_t *)calloc((size_t)p->nodes + 1, sizeof(int64_t));
    p->bbox = (double *)calloc(6 * ((size_t)p->nodes + 1), sizeof(double));
    p->leaf = (signed char *)malloc((size_t)p->nodes + 1);
    memset(p->leaf, 2, (size_t)p->nodes + 1); /* slots that subdivide never reaches stay unused */
    if (tree_mode == ORC_TREE_MORTON_MEDIAN)
        morton_order(p);
    subdivide(p, 1, 0, N, 0);

    dualtraversefillitl(p, 1, 1);
    qsort(p->p2p, (size_t)p->np2p, 2 * sizeof(int32_t), cmp_pair); /* D-4, G20 */
    qsort(p->m2l, (size_t)p->nm2l, 2 * sizeof(int32_t), cmp_pair);
    p->M = NULL;
    p->have_M = 0;
    return p;
}

void orc_plan_destroy(orc_plan_t *p)
{
    if (!p) return;
    free(p->x); free(p->y); free(p->z); free(p->w); free(p->pm); free(p->perm);
    free(p->lo); free(p->hi); free(p->leaf); free(p->bbox); free(p->p2p); free(p->m2l); free(p->tcpp); free(p->tcpc); free(p->M);
    free(p);
}

void orc_plan_sizes(const orc_plan_t *p, int64_t *out)
{
    out[0] = p->kappa;
    out[1] = p->nodes;
    out[2] = p->leaves;
    out[3] = p->P;
    out[4] = p->np2p;
    out[5] = p->nm2l;
}

double orc_plan_gamma_bar(const orc_plan_t *p) { return p->gamma_bar; }

void orc_plan_perm(const orc_plan_t *p, int64_t *perm)
{
    memcpy(perm, p->perm, sizeof(int64_t) * (size_t)p->N);
}

void orc_plan_nodes(const orc_plan_t *p, int64_t *lo, int64_t *hi, double *bbox)
{
    for (int64_t i = 1; i <= p->nodes; ++i) {
        lo[i - 1] = p->lo[i];
        hi[i - 1] = p->hi[i];
        memcpy(&bbox[6 * (i - 1)], &p->bbox[6 * i], 6 * sizeof(double));
    }
}

int orc_plan_set_lists(orc_plan_t *p, int64_t np2p, const int32_t *p2p_t, const int32_t *p2p_s,
                       int64_t nm2l, const int32_t *m2l_t, const int32_t *m2l_s)
{
    for (int64_t k = 0; k < np2p; ++k) {
        if (p2p_t[k] < 1 || p2p_t[k] > p->nodes || p2p_s[k] < 1 || p2p_s[k] > p->nodes) return -1;
        if (p->leaf[p2p_t[k]] != 1 || p->leaf[p2p_s[k]] != 1) return -1;
    }
    for (int64_t k = 0; k < nm2l; ++k)
        if (m2l_t[k] < 1 || m2l_t[k] > p->nodes || m2l_s[k] < 1 || m2l_s[k] > p->nodes ||
            p->leaf[m2l_t[k]] == 2 || p->leaf[m2l_s[k]] == 2)
            return -1;
    p->np2p = p->nm2l = 0;
    for (int64_t k = 0; k < np2p; ++k) push_pair(&p->p2p, &p->np2p, &p->cap_p2p, p2p_t[k], p2p_s[k]);
    for (int64_t k = 0; k < nm2l; ++k) push_pair(&p->m2l, &p->nm2l, &p->cap_m2l, m2l_t[k], m2l_s[k]);
    qsort(p->p2p, (size_t)p->np2p, 2 * sizeof(int32_t), cmp_pair);
    qsort(p->m2l, (size_t)p->nm2l, 2 * sizeof(int32_t), cmp_pair);
    return 0;
}

double orc_plan_eta_eff(const orc_plan_t *p)
{
    double worst = 0.0;
    for (int64_t k = 0; k < p->nm2l; ++k) {
        int64_t i = p->m2l[2 * k], j = p->m2l[2 * k + 1];
        double ri = diam2(p, i), rj = diam2(p, j), d2 = dist2(p, i, j);
        double ratio = ((ri > rj) ? ri : rj) / d2; /* Alg 5.8 squared: admissible iff ratio < theta^2 */
        if (ratio != ratio) ratio = INFINITY;      /* two point clusters at one place */
        if (ratio > worst) worst = ratio;
    }
    return sqrt(worst);
}

void orc_plan_leaf_flags(const orc_plan_t *p, int8_t *leaf)
{
    for (int64_t i = 1; i <= p->nodes; ++i)
        leaf[i - 1] = (int8_t)p->leaf[i];
}

void orc_plan_lists(const orc_plan_t *p, int32_t *p2p_t, int32_t *p2p_s, int32_t *m2l_t, int32_t *m2l_s)
{
    for (int64_t k = 0; k < p->np2p; ++k) {
        p2p_t[k] = p->p2p[2 * k];
        p2p_s[k] = p->p2p[2 * k + 1];
    }
    for (int64_t k = 0; k < p->nm2l; ++k) {
        m2l_t[k] = p->m2l[2 * k];
        m2l_s[k] = p->m2l[2 * k + 1];
    }
}

/* Upward pass --------------------------------------------------------------- */
/* Alg 5.3 / eq. (2.4): M_{S,nu} = sum_j l_{S,nu}(x_j) m_j */
static void p2m_node(const orc_plan_t *p, int64_t node, double *M)
{
    int n = p->n, n1 = p->n1;
    const double *bb = &p->bbox[6 * node];
    double lx[64], ly[64], lz[64];
    memset(M, 0, sizeof(double) * 4 * (size_t)p->P);
    for (int64_t k = p->lo[node]; k < p->hi[node]; ++k) {
        int64_t j = p->perm[k];
        basis_1d_c(n, p->cheb, bb[0], bb[3], p->x[j], lx);
        basis_1d_c(n, p->cheb, bb[1], bb[4], p->y[j], ly);
        basis_1d_c(n, p->cheb, bb[2], bb[5], p->z[j], lz);
        const double *m = &p->w[4 * j];
        for (int a = 0; a < n1; ++a)
            for (int b = 0; b < n1; ++b)
                for (int c = 0; c < n1; ++c) {
                    double l = lx[a] * ly[b] * lz[c];
                    double *Mv = &M[4 * ((a * n1 + b) * n1 + c)];
                    Mv[0] += l * m[0];
                    Mv[1] += l * m[1];
                    Mv[2] += l * m[2];
                    Mv[3] += l * m[3];
                }
    }
}

void orc_p2m_node(const orc_plan_t *p, int64_t node, double *M_node) { p2m_node(p, node, M_node); }

/* 1-D transfer matrix T[k][k'] = l_{S,k}(xi_{S',k'}) on one axis (used by M2M and L2L). */
static void transfer_1d(const orc_plan_t *p, double aS, double bS, double aC, double bC, double *T)
{
    int n = p->n, n1 = p->n1;
    double xi[64], col[64];
    node_points(n, p->cheb, aC, bC, xi);
    for (int kc = 0; kc < n1; ++kc) {
        basis_1d_c(n, p->cheb, aS, bS, xi[kc], col);
        for (int k = 0; k < n1; ++k)
            T[k * n1 + kc] = col[k];
    }
}

/* Alg 5.4 / eq. (2.9) (G4): M_S += sum_nu' l_{S,nu}(xi_{S',nu'}) M_{S',nu'} */
static void m2m(const orc_plan_t *p, int64_t S, int64_t C, double *M)
{
    if (p->hi[C] == p->lo[C]) return;
    int n1 = p->n1, P = p->P;
    const double *bS = &p->bbox[6 * S], *bC = &p->bbox[6 * C];
    double Tx[1024], Ty[1024], Tz[1024];
    transfer_1d(p, bS[0], bS[3], bC[0], bC[3], Tx);
    transfer_1d(p, bS[1], bS[4], bC[1], bC[4], Ty);
    transfer_1d(p, bS[2], bS[5], bC[2], bC[5], Tz);
    double *MS = &M[4 * (size_t)P * S];
    const double *MC = &M[4 * (size_t)P * C];
    for (int a = 0; a < n1; ++a)
        for (int b = 0; b < n1; ++b)
            for (int c = 0; c < n1; ++c) {
                double acc[4] = {0, 0, 0, 0};
                for (int a2 = 0; a2 < n1; ++a2)
                    for (int b2 = 0; b2 < n1; ++b2)
                        for (int c2 = 0; c2 < n1; ++c2) {
                            double l = Tx[a * n1 + a2] * Ty[b * n1 + b2] * Tz[c * n1 + c2];
                            const double *mc = &MC[4 * ((a2 * n1 + b2) * n1 + c2)];
                            acc[0] += l * mc[0];
                            acc[1] += l * mc[1];
                            acc[2] += l * mc[2];
                            acc[3] += l * mc[3];
                        }
                double *ms = &MS[4 * ((a * n1 + b) * n1 + c)];
                ms[0] += acc[0];
                ms[1] += acc[1];
                ms[2] += acc[2];
                ms[3] += acc[3];
            }
}

/* Alg 5.5, done level by level as PAPER.md:125 describes. */
static void upward(orc_plan_t *p)
{
    if (p->have_M) return;
    size_t P4 = 4 * (size_t)p->P;
    p->M = (double *)calloc(P4 * ((size_t)p->nodes + 1), sizeof(double));
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 1; i <= p->nodes; ++i)
        if (p->leaf[i] == 1) p2m_node(p, i, &p->M[P4 * i]); /* Alg 5.5: P2M where children(S) is empty */
    for (int level = p->kappa - 1; level >= 0; --level) {
        int64_t first = (int64_t)1 << level;
#pragma omp parallel for schedule(dynamic, 1)
        for (int64_t i = first; i < 2 * first; ++i) {
            if (p->leaf[i] != 0) continue; /* a leaf or an unused slot has no children */
            m2m(p, i, 2 * i, p->M);
            m2m(p, i, 2 * i + 1, p->M);
        }
    }
    p->have_M = 1;
}

void orc_upward(orc_plan_t *p, double *M_out)
{
    upward(p);
    if (M_out)
        memcpy(M_out, &p->M[4 * (size_t)p->P], sizeof(double) * 4 * (size_t)p->P * (size_t)p->nodes);
}

/* Interaction phase ----------------------------------------------------------- */
static void proxy_points(const orc_plan_t *p, int64_t node, double *xi /* [3][64] */)
{
    const double *bb = &p->bbox[6 * node];
    node_points(p->n, p->cheb, bb[0], bb[3], xi);
    node_points(p->n, p->cheb, bb[1], bb[4], xi + 64);
    node_points(p->n, p->cheb, bb[2], bb[5], xi + 128);
}

/* Alg 5.9 (G5 "+="), eq. (2.5):
 * E_{t,mu} += sum_nu gamma_{s,nu} g(xi_{t,mu}, xi_{s,nu});  B_{t,mu} += sum_nu p_{s,nu} x g */
static void m2l(const orc_plan_t *p, int64_t t, int64_t s, double *Lt)
{
    int n1 = p->n1;
    double g2 = p->gamma_bar * p->gamma_bar;
    double xt[192], xs[192];
    proxy_points(p, t, xt);
    proxy_points(p, s, xs);
    const double *Ms = &p->M[4 * (size_t)p->P * s];
    for (int a = 0; a < n1; ++a)
        for (int b = 0; b < n1; ++b)
            for (int c = 0; c < n1; ++c) {
                double *acc = &Lt[6 * ((a * n1 + b) * n1 + c)];
                for (int a2 = 0; a2 < n1; ++a2)
                    for (int b2 = 0; b2 < n1; ++b2)
                        for (int c2 = 0; c2 < n1; ++c2)
                            accumulate(xt[a] - xs[a2], xt[64 + b] - xs[64 + b2], xt[128 + c] - xs[128 + c2],
                                       g2, &Ms[4 * ((a2 * n1 + b2) * n1 + c2)], acc);
            }
}

/* Alg 5.13 / eq. (2.11): L_{S',mu'} += sum_mu l_{S,mu}(xi_{S',mu'}) L_{S,mu} */
static void l2l(const orc_plan_t *p, int64_t C, int64_t S, double *L)
{
    if (p->hi[C] == p->lo[C]) return;
    int n1 = p->n1, P = p->P;
    const double *bS = &p->bbox[6 * S], *bC = &p->bbox[6 * C];
    double Tx[1024], Ty[1024], Tz[1024];
    transfer_1d(p, bS[0], bS[3], bC[0], bC[3], Tx);
    transfer_1d(p, bS[1], bS[4], bC[1], bC[4], Ty);
    transfer_1d(p, bS[2], bS[5], bC[2], bC[5], Tz);
    const double *LS = &L[6 * (size_t)P * S];
    double *LC = &L[6 * (size_t)P * C];
    for (int a2 = 0; a2 < n1; ++a2)
        for (int b2 = 0; b2 < n1; ++b2)
            for (int c2 = 0; c2 < n1; ++c2) {
                double acc[6] = {0, 0, 0, 0, 0, 0};
                for (int a = 0; a < n1; ++a)
                    for (int b = 0; b < n1; ++b)
                        for (int c = 0; c < n1; ++c) {
                            double l = Tx[a * n1 + a2] * Ty[b * n1 + b2] * Tz[c * n1 + c2];
                            const double *ls = &LS[6 * ((a * n1 + b) * n1 + c)];
                            for (int f = 0; f < 6; ++f)
                                acc[f] += l * ls[f];
                        }
                double *lc = &LC[6 * ((a2 * n1 + b2) * n1 + c2)];
                for (int f = 0; f < 6; ++f)
                    lc[f] += acc[f];
            }
}

/* Alg 5.14 / eq. (2.10): f_i += sum_mu l_{S,mu}(x_i) L_{S,mu} */
static void l2p(const orc_plan_t *p, int64_t leaf, const double *L, double *far /* [N][6] tree order */)
{
    int n = p->n, n1 = p->n1;
    const double *bb = &p->bbox[6 * leaf];
    const double *LS = &L[6 * (size_t)p->P * leaf];
    double lx[64], ly[64], lz[64];
    for (int64_t k = p->lo[leaf]; k < p->hi[leaf]; ++k) {
        int64_t j = p->perm[k];
        basis_1d_c(n, p->cheb, bb[0], bb[3], p->x[j], lx);
        basis_1d_c(n, p->cheb, bb[1], bb[4], p->y[j], ly);
        basis_1d_c(n, p->cheb, bb[2], bb[5], p->z[j], lz);
        double acc[6] = {0, 0, 0, 0, 0, 0};
        for (int a = 0; a < n1; ++a)
            for (int b = 0; b < n1; ++b)
                for (int c = 0; c < n1; ++c) {
                    double l = lx[a] * ly[b] * lz[c];
                    const double *ls = &LS[6 * ((a * n1 + b) * n1 + c)];
                    for (int f = 0; f < 6; ++f)
                        acc[f] += l * ls[f];
                }
        for (int f = 0; f < 6; ++f)
            far[6 * k + f] += acc[f];
    }
}

/* Alg 5.10 for one (target leaf, source leaf) pair. */
static void p2p(const orc_plan_t *p, int64_t t, int64_t s, double *near /* [N][6] tree order */)
{
    double g2 = p->gamma_bar * p->gamma_bar;
    for (int64_t ki = p->lo[t]; ki < p->hi[t]; ++ki) {
        int64_t i = p->perm[ki];
        double *acc = &near[6 * ki];
        for (int64_t kj = p->lo[s]; kj < p->hi[s]; ++kj) {
            int64_t j = p->perm[kj];
            if (p->raw & 2)
                accumulate_sm(p->x[i] - p->x[j], p->y[i] - p->y[j], p->z[i] - p->z[j], &p->pm[3 * j], &p->w[4 * j], acc);
            else
                accumulate(p->x[i] - p->x[j], p->y[i] - p->y[j], p->z[i] - p->z[j], g2, &p->w[4 * j], acc);
        }
    }
}

static void csr_offsets(const int32_t *pairs, int64_t npairs, int64_t nodes, int64_t *off /* [nodes+2] */)
{
    for (int64_t i = 0; i <= nodes + 1; ++i) off[i] = 0;
    for (int64_t k = 0; k < npairs; ++k) off[pairs[2 * k] + 1]++;
    for (int64_t i = 1; i <= nodes + 1; ++i) off[i] += off[i - 1];
}

/* M2L over the whole list for the nodes flagged in need[] (NULL = all). L is [nodes+1][P][6], zeroed. */
static void m2l_all(orc_plan_t *p, const char *need, double *L)
{
    int64_t *off = (int64_t *)malloc(sizeof(int64_t) * ((size_t)p->nodes + 2));
    csr_offsets(p->m2l, p->nm2l, p->nodes, off);
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t t = 1; t <= p->nodes; ++t) {
        if (need && !need[t]) continue;
        for (int64_t k = off[t]; k < off[t + 1]; ++k)
            m2l(p, t, p->m2l[2 * k + 1], &L[6 * (size_t)p->P * t]);
    }
    free(off);
}

void orc_m2l_raw(orc_plan_t *p, double *L_raw)
{
    upward(p);
    size_t P6 = 6 * (size_t)p->P;
    double *L = (double *)calloc(P6 * ((size_t)p->nodes + 1), sizeof(double));
    m2l_all(p, NULL, L);
    memcpy(L_raw, &L[P6], sizeof(double) * P6 * (size_t)p->nodes);
    free(L);
}

/* Treecode variant (particle-cluster, Fig. 1a, ref [16]) -------------------------
 * The traversal is Alg 9.1 with the target held at a leaf: for every target leaf t, dualtraverse(t, root).  With a
 * leaf target Alg 9.1 never splits the target, so: both leaves -> direct sum (PP list); admissible (Alg 5.8) ->
 * particle-cluster interaction (PC list): the target PARTICLES evaluate the kernel at the source's proxy points,
 *   E_i += sum_nu gamma_{s,nu} g(x_i, xi_{s,nu}),  B_i += sum_nu p_{s,nu} x g(x_i, xi_{s,nu})   (eq. (2.5) with the
 * target side not interpolated); otherwise the source is split.  Needs P2M / M2M only; no L2L / L2P. */
static void treecode_lists(orc_plan_t *p)
{
    if (p->tcpp || p->tcpc) return;
    /* reuse dualtraversefillitl with temporarily swapped list buffers */
    int32_t *sp2p = p->p2p, *sm2l = p->m2l;
    int64_t np2p = p->np2p, nm2l = p->nm2l, cp2p = p->cap_p2p, cm2l = p->cap_m2l;
    p->p2p = NULL; p->m2l = NULL; p->np2p = p->nm2l = p->cap_p2p = p->cap_m2l = 0;
    for (int64_t t = 1; t <= p->nodes; ++t)
        if (p->leaf[t] == 1) dualtraversefillitl(p, t, 1);
    qsort(p->p2p, (size_t)p->np2p, 2 * sizeof(int32_t), cmp_pair);
    qsort(p->m2l, (size_t)p->nm2l, 2 * sizeof(int32_t), cmp_pair);
    p->tcpp = p->p2p; p->ntcpp = p->np2p; p->cap_tcpp = p->cap_p2p;
    p->tcpc = p->m2l; p->ntcpc = p->nm2l; p->cap_tcpc = p->cap_m2l;
    if (!p->tcpp) p->tcpp = (int32_t *)malloc(8);
    if (!p->tcpc) p->tcpc = (int32_t *)malloc(8);
    p->p2p = sp2p; p->m2l = sm2l; p->np2p = np2p; p->nm2l = nm2l; p->cap_p2p = cp2p; p->cap_m2l = cm2l;
}

void orc_treecode_sizes(orc_plan_t *p, int64_t *out /* [2]: len(pp), len(pc) */)
{
    treecode_lists(p);
    out[0] = p->ntcpp;
    out[1] = p->ntcpc;
}

void orc_treecode_lists(orc_plan_t *p, int32_t *pp_t, int32_t *pp_s, int32_t *pc_t, int32_t *pc_s)
{
    treecode_lists(p);
    for (int64_t k = 0; k < p->ntcpp; ++k) { pp_t[k] = p->tcpp[2 * k]; pp_s[k] = p->tcpp[2 * k + 1]; }
    for (int64_t k = 0; k < p->ntcpc; ++k) { pc_t[k] = p->tcpc[2 * k]; pc_s[k] = p->tcpc[2 * k + 1]; }
}

/* particle-cluster interaction of target leaf t with source cluster s (far field with the mean gamma_bar, eq. (3.2)) */
static void pc(const orc_plan_t *p, int64_t t, int64_t s, double *far /* [N][6] tree order */)
{
    int n1 = p->n1;
    double g2 = p->gamma_bar * p->gamma_bar;
    double xs[192];
    proxy_points(p, s, xs);
    const double *Ms = &p->M[4 * (size_t)p->P * s];
    for (int64_t ki = p->lo[t]; ki < p->hi[t]; ++ki) {
        int64_t i = p->perm[ki];
        double *acc = &far[6 * ki];
        for (int a2 = 0; a2 < n1; ++a2)
            for (int b2 = 0; b2 < n1; ++b2)
                for (int c2 = 0; c2 < n1; ++c2)
                    accumulate(p->x[i] - xs[a2], p->y[i] - xs[64 + b2], p->z[i] - xs[128 + c2], g2,
                               &Ms[4 * ((a2 * n1 + b2) * n1 + c2)], acc);
    }
}

int orc_eval_treecode(orc_plan_t *p, double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz)
{
    int64_t N = p->N;
    treecode_lists(p);
    upward(p);
    double *near = (double *)calloc(6 * (size_t)N, sizeof(double));
    double *far = (double *)calloc(6 * (size_t)N, sizeof(double));
    int64_t *offp = (int64_t *)malloc(sizeof(int64_t) * ((size_t)p->nodes + 2));
    int64_t *offc = (int64_t *)malloc(sizeof(int64_t) * ((size_t)p->nodes + 2));
    csr_offsets(p->tcpp, p->ntcpp, p->nodes, offp);
    csr_offsets(p->tcpc, p->ntcpc, p->nodes, offc);
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t t = 1; t <= p->nodes; ++t) { /* (only leaves have rows) */
        for (int64_t k = offp[t]; k < offp[t + 1]; ++k) p2p(p, t, p->tcpp[2 * k + 1], near);
        for (int64_t k = offc[t]; k < offc[t + 1]; ++k) pc(p, t, p->tcpc[2 * k + 1], far);
    }
    double cE, cB;
    prefactors(p->raw, &cE, &cB);
    for (int64_t k = 0; k < N; ++k) {
        int64_t i = p->perm[k];
        Ex[i] = cE * (near[6 * k + 0] + far[6 * k + 0]); /* fixed order: near + far */
        Ey[i] = cE * (near[6 * k + 1] + far[6 * k + 1]);
        Ez[i] = cE * (near[6 * k + 2] + far[6 * k + 2]);
        Bx[i] = cB * (near[6 * k + 3] + far[6 * k + 3]);
        By[i] = cB * (near[6 * k + 4] + far[6 * k + 4]);
        Bz[i] = cB * (near[6 * k + 5] + far[6 * k + 5]);
    }
    free(near); free(far); free(offp); free(offc);
    return 0;
}

/* Alg 5.12 after subdivide. */
int orc_eval(orc_plan_t *p, int64_t nsel, const int64_t *sel, int part,
             double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz,
             double *L_out)
{
    int64_t N = p->N;
    size_t P6 = 6 * (size_t)p->P;
    char *need = NULL;
    if (nsel > 0) { /* only the chains root -> selected leaf */
        need = (char *)calloc((size_t)p->nodes + 1, 1);
        for (int64_t k = 0; k < nsel; ++k) {
            if (sel[k] < 1 || sel[k] > p->nodes || p->leaf[sel[k]] != 1) {
                free(need);
                return -1;
            }
            for (int64_t i = sel[k]; i >= 1; i /= 2) need[i] = 1;
        }
    }
    double *near = (double *)calloc(6 * (size_t)N, sizeof(double)); /* E_i = B_i = 0 */
    double *far = (double *)calloc(6 * (size_t)N, sizeof(double));
    double *L = NULL;

    if (part != 1) {
        upward(p); /* Alg 5.5 */
        L = (double *)calloc(P6 * ((size_t)p->nodes + 1), sizeof(double));
        m2l_all(p, need, L); /* Alg 5.9 over m2l_itl */
    }
    if (part != 2) { /* Alg 5.10 over p2p_itl, grouped by target */
        int64_t *off = (int64_t *)malloc(sizeof(int64_t) * ((size_t)p->nodes + 2));
        csr_offsets(p->p2p, p->np2p, p->nodes, off);
#pragma omp parallel for schedule(dynamic, 1)
        for (int64_t t = 1; t <= p->nodes; ++t) { /* (only leaves have rows) */
            if (need && !need[t]) continue;
            for (int64_t k = off[t]; k < off[t + 1]; ++k)
                p2p(p, t, p->p2p[2 * k + 1], near);
        }
        free(off);
    }
    if (part != 1) { /* Alg 5.15: L2L level by level (pre-order), then L2P at the leaves */
        for (int level = 1; level <= p->kappa; ++level) {
            int64_t first = (int64_t)1 << level;
#pragma omp parallel for schedule(dynamic, 1)
            for (int64_t c = first; c < 2 * first; ++c) {
                if (need && !need[c]) continue;
                if (p->leaf[c] == 2) continue; /* unused slot: its parent is a leaf */
                l2l(p, c, c / 2, L);
            }
        }
#pragma omp parallel for schedule(dynamic, 1)
        for (int64_t t = 1; t <= p->nodes; ++t) {
            if (p->leaf[t] != 1 || (need && !need[t])) continue;
            l2p(p, t, L, far);
        }
        if (L_out)
            memcpy(L_out, &L[P6], sizeof(double) * P6 * (size_t)p->nodes);
    }
    double cE, cB;
    prefactors(p->raw, &cE, &cB);
    for (int64_t t = 1; t <= p->nodes; ++t) {
        if (p->leaf[t] != 1 || (need && !need[t])) continue;
        for (int64_t k = p->lo[t]; k < p->hi[t]; ++k) {
            int64_t i = p->perm[k];
            double v[6];
            for (int f = 0; f < 6; ++f)
                v[f] = near[6 * k + f] + far[6 * k + f]; /* fixed order: near + far */
            Ex[i] = cE * v[0];
            Ey[i] = cE * v[1];
            Ez[i] = cE * v[2];
            Bx[i] = cB * v[3];
            By[i] = cB * v[4];
            Bz[i] = cB * v[5];
        }
    }
    free(near);
    free(far);
    free(L);
    free(need);
    return 0;
}
