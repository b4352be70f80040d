// kernels_interp.cu -- the interpolation passes of the hot path:
//   a4  P2M  Alg 5.3 / eq. (2.4)
//   a5  M2M  Alg 5.4 / eq. (2.9), level by level upward (Alg 5.5)
//   a8  L2L  Alg 5.13 / eq. (2.11), level by level downward (Alg 5.15)
//   a9  L2P  Alg 5.14 / eq. (2.10)  + a10 prefactors of eq. (3.1) and the
//       scatter back to the caller's particle order
// Barycentric Lagrange basis on Chebyshev points of the second kind (readings I-1..I-5).
// M2M / L2L use the tensor-product structure: three 1-D contractions with (n+1)x(n+1) transfer
// matrices instead of the (n+1)^6 form.  All of it is < 2 % of the run time; the passes are
// HBM / launch-latency-bound (M2M, L2L) or small FP64 loops (P2M, L2P).
#include "fmm_internal.cuh"

struct cheb_t {
    double c[FMM_MAX_ORDER + 1];
};

static cheb_t host_cheb(int n)
{
    cheb_t t;
    memset(&t, 0, sizeof(t));
    for (int k = 0; k <= n; ++k) t.c[k] = sin(FMM_PI * (double)(n - 2 * k) / (double)(2 * n));  // I-1
    t.c[0] = 1.0;
    t.c[n] = -1.0;
    return t;
}

// I-3: xi_k = (a+b)/2 + (b-a)/2 c_k, product and sum rounded separately
__device__ __forceinline__ double node_point(double mid, double half, double ck) { return __dadd_rn(mid, __dmul_rn(half, ck)); }

// I-2, I-4: l_k(x) = (w_k/(x-xi_k)) / sum_m (w_m/(x-xi_m)), w_k = (-1)^k delta_k, delta_0 = delta_n = 1/2;
// exact hit x == xi_k: l_k = 1 for the first such k, 0 elsewhere.  out has stride `stride`.
__device__ __forceinline__ void basis_1d(int n, const cheb_t &ch, double a, double b, double x, double *out, int stride)
{
    double mid = __dmul_rn(__dadd_rn(a, b), 0.5), half = __dmul_rn(__dsub_rn(b, a), 0.5);
    int hit = -1;
    double S = 0.0;
    for (int k = 0; k <= n; ++k) {
        double xi = node_point(mid, half, ch.c[k]);
        double d = x - xi;
        if (d == 0.0 && hit < 0) hit = k;
        double wk = (k == 0 || k == n) ? 0.5 : 1.0;
        if (k & 1) wk = -wk;
        double t = wk / d;
        out[k * stride] = t;
        S += t;
    }
    if (hit >= 0) {
        for (int k = 0; k <= n; ++k) out[k * stride] = (k == hit) ? 1.0 : 0.0;
    } else {
        const double rS = 1.0 / S;  // (one division; l_k = t_k / S to one more rounding)
        for (int k = 0; k <= n; ++k) out[k * stride] = out[k * stride] * rS;
    }
}

// ---------------------------------------------------------------------------------------
// a4: P2M.  One block per leaf.  A thread owns one (nu1, nu2) column of the proxy grid and keeps the
// 4 x (n+1) moments of that column in registers:  M[nu1,nu2,:][k] += (l_x l_y m_k) l_z[:]  per particle.
// The block's threads form G = THREADS / (n+1)^2 groups that take the particles of a chunk round-robin;
// the groups' partial sums are then added in group order (fixed order: deterministic, no atomics).
// 1-D basis values and weights of a chunk of particles are staged in shared memory.
// ---------------------------------------------------------------------------------------
#define P2M_THREADS 256
#define P2M_CHUNK 64

template <int N1>
struct p2m_cfg {
    static constexpr int COLS = N1 * N1;
    static constexpr int G0 = P2M_THREADS / COLS;
    static constexpr int G = G0 > 8 ? 8 : (G0 < 1 ? 1 : G0);
    static constexpr int P = N1 * N1 * N1;
    static constexpr size_t SMEM = sizeof(double) * (3 * N1 * P2M_CHUNK + 4 * P2M_CHUNK + (G > 1 ? G * 4 * P : 0));
};

template <int N1>
__global__ void __launch_bounds__(P2M_THREADS, (N1 <= 7) ? 3 : 1) p2m_kernel(cheb_t ch, int leaves, const int32_t *__restrict__ node_lo,
                                                          const int32_t *__restrict__ node_hi, const double *__restrict__ bbox,
                                                          const double *__restrict__ tx, const double *__restrict__ ty,
                                                          const double *__restrict__ tz, const double *__restrict__ w0,
                                                          const double *__restrict__ w1, const double *__restrict__ w2,
                                                          const double *__restrict__ w3, double *__restrict__ M)
{
    constexpr int COLS = p2m_cfg<N1>::COLS, G = p2m_cfg<N1>::G, P = p2m_cfg<N1>::P, n = N1 - 1;
    extern __shared__ __align__(16) double sm[];
    double *bas = sm;                                  // [3][P2M_CHUNK][N1]
    double *wts = sm + 3 * N1 * P2M_CHUNK;             // [P2M_CHUNK][4]
    double *red = wts + 4 * P2M_CHUNK;                 // [P][4] (only if G > 1)
    const int node = leaves + blockIdx.x;
    const int lo = node_lo[node], hi = node_hi[node];
    const double *bb = bbox + 6 * (int64_t)node;
    double *Mn = M + 4 * (int64_t)P * node;
    const int grp = threadIdx.x / COLS, col = threadIdx.x - grp * COLS;
    const bool active = grp < G;
    const int a = col / N1, b = col - a * N1;
    double acc[4][N1];
#pragma unroll
    for (int k = 0; k < 4; ++k)
#pragma unroll
        for (int c = 0; c < N1; ++c) acc[k][c] = 0.0;
    for (int j0 = lo; j0 < hi; j0 += P2M_CHUNK) {
        const int cnt = min(P2M_CHUNK, hi - j0);
        __syncthreads();
        for (int t = threadIdx.x; t < 3 * cnt; t += P2M_THREADS) {
            int g = t / cnt, jj = t - g * cnt;
            const double *coord = (g == 0) ? tx : (g == 1) ? ty : tz;
            basis_1d(n, ch, bb[g], bb[3 + g], coord[j0 + jj], bas + ((size_t)g * P2M_CHUNK + jj) * N1, 1);
        }
        for (int t = threadIdx.x; t < cnt; t += P2M_THREADS) {
            wts[4 * t + 0] = w0[j0 + t];
            wts[4 * t + 1] = w1[j0 + t];
            wts[4 * t + 2] = w2[j0 + t];
            wts[4 * t + 3] = w3[j0 + t];
        }
        __syncthreads();
        if (active) {
            for (int jj = grp; jj < cnt; jj += G) {
                const double lab = bas[(size_t)jj * N1 + a] * bas[((size_t)P2M_CHUNK + jj) * N1 + b];
                const double *lc = bas + ((size_t)2 * P2M_CHUNK + jj) * N1;
                const double t0 = lab * wts[4 * jj], t1 = lab * wts[4 * jj + 1], t2 = lab * wts[4 * jj + 2], t3 = lab * wts[4 * jj + 3];
#pragma unroll
                for (int c = 0; c < N1; ++c) {
                    const double l = lc[c];
                    acc[0][c] = fma(t0, l, acc[0][c]);
                    acc[1][c] = fma(t1, l, acc[1][c]);
                    acc[2][c] = fma(t2, l, acc[2][c]);
                    acc[3][c] = fma(t3, l, acc[3][c]);
                }
            }
        }
    }
    // M[nu][k], nu = (a N1 + b) N1 + c
    if (G == 1) {
        if (active)
#pragma unroll
            for (int c = 0; c < N1; ++c) {
                double *m = Mn + 4 * (int64_t)(col * N1 + c);
                m[0] = acc[0][c]; m[1] = acc[1][c]; m[2] = acc[2][c]; m[3] = acc[3][c];
            }
    } else {
        // every group leaves its partial sums in its own slab; they are then added in group order (two barriers instead of G)
        __syncthreads();
        if (active)
#pragma unroll
            for (int c = 0; c < N1; ++c) {
                double *r = red + (size_t)grp * 4 * P + 4 * (col * N1 + c);
                *reinterpret_cast<double2 *>(r) = make_double2(acc[0][c], acc[1][c]);
                *reinterpret_cast<double2 *>(r + 2) = make_double2(acc[2][c], acc[3][c]);
            }
        __syncthreads();
        for (int e = threadIdx.x; e < 4 * P; e += P2M_THREADS) {
            double v = red[e];
#pragma unroll
            for (int g = 1; g < G; ++g) v += red[(size_t)g * 4 * P + e];
            Mn[e] = v;
        }
    }
}

// ---------------------------------------------------------------------------------------
// 1-D transfer matrices T_g[k][k'] = l_{S,k}(xi_{S',k'}) on the three axes (S = parent, S' = child)
// ---------------------------------------------------------------------------------------
// T of every child node C (parent S = C / 2), stride XFER_T per node, computed once per plan build (the boxes do not change
// between evaluations): M2M and L2L then only load 3 (n+1)^2 doubles instead of running 3 (n+1) barycentric evaluations
// with their divisions at the head of every level's dependency chain.
__global__ void transfer_tables_kernel(int n, cheb_t ch, int nodes, int stride, const int32_t *__restrict__ node_lo,
                                       const int32_t *__restrict__ node_hi, const double *__restrict__ bbox, double *__restrict__ tab)
{
    const int n1 = n + 1;
    const int q = blockIdx.x * blockDim.x + threadIdx.x;  // (child, axis, column)
    const int C = 2 + q / (3 * n1);
    if (C > nodes) return;
    if (node_hi[C] <= node_lo[C]) return;
    const int r = q - (C - 2) * 3 * n1, g = r / n1, kc = r - g * n1;
    const double *bS = bbox + 6 * (int64_t)(C >> 1), *bC = bbox + 6 * (int64_t)C;
    const double mid = __dmul_rn(__dadd_rn(bC[g], bC[3 + g]), 0.5), half = __dmul_rn(__dsub_rn(bC[3 + g], bC[g]), 0.5);
    const double xi = node_point(mid, half, ch.c[kc]);
    basis_1d(n, ch, bS[g], bS[3 + g], xi, tab + (size_t)C * stride + (size_t)g * n1 * n1 + kc, n1);  // column kc
}

int interp_transfer_tables(fmm_plan *p)
{
    fmm_ctx *c = &p->ctx;
    if (p->nodes < 2) return FMM_OK;
    const cheb_t ch = host_cheb(p->n);
    const int stride = (3 * p->n1 * p->n1 + 1) & ~1;
    const int64_t count = (int64_t)(p->nodes - 1) * 3 * p->n1;
    transfer_tables_kernel<<<(unsigned)((count + 127) / 128), 128, 0, c->stream>>>(p->n, ch, (int)p->nodes, stride, p->node_lo, p->node_hi, p->bbox,
                                                                                 p->node_T);
    FMM_LAUNCH_CHECK(c, "transfer_tables_kernel");
    return FMM_OK;
}

// ---------------------------------------------------------------------------------------
// a5: M2M for one level.  One block per parent; for each non-empty child three 1-D contractions:
//   M_S[a,b,c] += sum_{a',b',c'} Tx[a][a'] Ty[b][b'] Tz[c][c'] M_S'[a',b',c']
// ---------------------------------------------------------------------------------------
// threads of a transfer block: one per proxy point (in whole warps) up to 512, so the two inner phases are one pass
template <int N1>
struct xfer_cfg {
    static constexpr int P = N1 * N1 * N1;
    static constexpr int THREADS = ((P + 31) / 32 * 32 <= 512) ? ((P + 31) / 32 * 32 < 64 ? 64 : (P + 31) / 32 * 32) : 512;
};

// The whole upward pass is ONE launch: a block starts at a parent of two leaves; when a node is finished the block counts
// itself into the node's parent, and the second of the two siblings to arrive (both children are then complete) goes on with
// the parent.  No grid barrier, no launch per level: the dependency chain of the kappa levels costs a few microseconds per
// level.  The result does not depend on which sibling arrives last (child 0 is always added before child 1).
template <int N1>
__global__ void __launch_bounds__(xfer_cfg<N1>::THREADS) m2m_kernel(int first, const int32_t *__restrict__ node_lo,
                                                           const int32_t *__restrict__ node_hi, const double *__restrict__ tab,
                                                           double *M, int *arrive /* [nodes + 2], zero between evaluations */)
{
    extern __shared__ __align__(16) double sm[];
    __shared__ int s_prev;
    constexpr int n1 = N1, P = n1 * n1 * n1, P4 = 4 * P, TS = (3 * n1 * n1 + 1) & ~1;  // compile-time order: index arithmetic without integer division
    constexpr int XFER_THREADS = xfer_cfg<N1>::THREADS;
    double *T = sm;                              // [3][n1][n1]
    double *A = sm + TS;                         // [P][4], 16-byte aligned
    double *B = A + P4;                          // [P][4]
    for (int S = first + blockIdx.x; S >= 1; S >>= 1) {
    double *MS = M + (int64_t)P4 * S;
    // parent accumulators live in registers across the two children: element e = threadIdx.x + k*blockDim
    for (int e0 = 0; e0 < P4; e0 += XFER_THREADS * 8) {
        // (P4 <= 8788; with 256 threads at most 35 elements per thread -> process in slabs of 8 per thread)
        double acc[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) acc[k] = 0.0;
        for (int child = 0; child < 2; ++child) {
            int C = 2 * S + child;
            if (node_hi[C] <= node_lo[C]) continue;  // uniform per block
            __syncthreads();
            for (int e = threadIdx.x; e < 3 * n1 * n1; e += XFER_THREADS) T[e] = tab[(size_t)C * TS + e];
            const double *MC = M + (int64_t)P4 * C;
            for (int e = threadIdx.x; e < P4; e += XFER_THREADS) A[e] = __ldcg(MC + e);  // (written by another block of this launch: past L1)
            __syncthreads();
            const double *Tx = T, *Ty = T + n1 * n1, *Tz = T + 2 * n1 * n1;
            // z: B[a',b',c] = sum_c' Tz[c][c'] A[a',b',c']   (a thread takes a proxy point with its four moments: the moments
            // come as two 16-byte words, a matrix entry is loaded once for four products)
            for (int nu = threadIdx.x; nu < P; nu += XFER_THREADS) {
                const int c3 = nu % n1, ab = nu / n1;
                double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
#pragma unroll
                for (int k = 0; k < n1; ++k) {
                    const double t = Tz[c3 * n1 + k];
                    const double2 v01 = *reinterpret_cast<const double2 *>(&A[4 * (ab * n1 + k)]);
                    const double2 v23 = *reinterpret_cast<const double2 *>(&A[4 * (ab * n1 + k) + 2]);
                    s0 = fma(t, v01.x, s0); s1 = fma(t, v01.y, s1); s2 = fma(t, v23.x, s2); s3 = fma(t, v23.y, s3);
                }
                *reinterpret_cast<double2 *>(&B[4 * nu]) = make_double2(s0, s1);
                *reinterpret_cast<double2 *>(&B[4 * nu + 2]) = make_double2(s2, s3);
            }
            __syncthreads();
            // y: A[a',b,c] = sum_b' Ty[b][b'] B[a',b',c]
            for (int nu = threadIdx.x; nu < P; nu += XFER_THREADS) {
                const int c3 = nu % n1, b = (nu / n1) % n1, a = nu / (n1 * n1);
                double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
#pragma unroll
                for (int k = 0; k < n1; ++k) {
                    const double t = Ty[b * n1 + k];
                    const int q = 4 * ((a * n1 + k) * n1 + c3);
                    const double2 v01 = *reinterpret_cast<const double2 *>(&B[q]);
                    const double2 v23 = *reinterpret_cast<const double2 *>(&B[q + 2]);
                    s0 = fma(t, v01.x, s0); s1 = fma(t, v01.y, s1); s2 = fma(t, v23.x, s2); s3 = fma(t, v23.y, s3);
                }
                *reinterpret_cast<double2 *>(&A[4 * nu]) = make_double2(s0, s1);
                *reinterpret_cast<double2 *>(&A[4 * nu + 2]) = make_double2(s2, s3);
            }
            __syncthreads();
            // x: out[a,b,c] = sum_a' Tx[a][a'] A[a',b,c]
#pragma unroll
            for (int k8 = 0; k8 < 8; ++k8) {
                int e = e0 + threadIdx.x + k8 * XFER_THREADS;
                if (e < P4) {
                    int f = e & 3, nu = e >> 2, bc = nu % (n1 * n1), a = nu / (n1 * n1);
                    double s = 0.0;
                    for (int k = 0; k < n1; ++k) s = fma(Tx[a * n1 + k], A[4 * (k * n1 * n1 + bc) + f], s);
                    acc[k8] += s;
                }
            }
        }
#pragma unroll
        for (int k8 = 0; k8 < 8; ++k8) {
            int e = e0 + threadIdx.x + k8 * XFER_THREADS;
            if (e < P4) MS[e] = acc[k8];
        }
    }
    // node S is complete: make it visible, then count into the parent; the first sibling to arrive stops here
    if (S == 1) break;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const int prev = atomicAdd(&arrive[S >> 1], 1);
        if (prev == 1) arrive[S >> 1] = 0;  // (both are here: leave the counter clean for the next evaluation)
        __threadfence();
        s_prev = prev;
    }
    __syncthreads();
    if (s_prev == 0) break;
    }
}

// ---------------------------------------------------------------------------------------
// a8: L2L for one level.  One block per child S' (parent S = S'/2):
//   L_S'[a',b',c'] += sum_{a,b,c} Tx[a][a'] Ty[b][b'] Tz[c][c'] L_S[a,b,c]
// ---------------------------------------------------------------------------------------
// The whole downward pass is ONE launch over the nodes 2 .. nodes in heap order: a block waits until its parent carries this
// evaluation's stamp, adds the parent's field and stamps its own node.  A block only ever waits for a block with a smaller
// index, and the blocks of a 1-D grid start in index order, so the block it waits for is running or done.
template <int N1>
__global__ void __launch_bounds__(xfer_cfg<N1>::THREADS) l2l_kernel(int first, int leaves, int stamp, const int32_t *__restrict__ node_lo,
                                                           const int32_t *__restrict__ node_hi, const double *__restrict__ tab,
                                                           double *L, int *ready /* [nodes + 2] */)
{
    extern __shared__ __align__(16) double sm[];
    constexpr int n1 = N1, P = n1 * n1 * n1, P6 = 6 * P, TS = (3 * n1 * n1 + 1) & ~1;
    constexpr int XFER_THREADS = xfer_cfg<N1>::THREADS;
    double *T = sm;
    double *A = sm + TS;  // [P][6], 16-byte aligned
    double *B = A + P6;
    int C = first + blockIdx.x, S = C >> 1;
    if (node_hi[C] <= node_lo[C]) return;  // (its descendants are empty too: nobody waits for it)
    for (int e = threadIdx.x; e < 3 * n1 * n1; e += XFER_THREADS) T[e] = tab[(size_t)C * TS + e];
    if (S > 1) {
        if (threadIdx.x == 0) {
            while (*((volatile int *)&ready[S]) != stamp) {}
            __threadfence();
        }
        __syncthreads();
    }
    const double *LS = L + (int64_t)P6 * S;
    double *LC = L + (int64_t)P6 * C;
    for (int e = threadIdx.x; e < P6; e += XFER_THREADS) A[e] = __ldcg(LS + e);  // (written by another block of this launch: past L1)
    __syncthreads();
    const double *Tx = T, *Ty = T + n1 * n1, *Tz = T + 2 * n1 * n1;
    // z: B[a,b,c'] = sum_c Tz[c][c'] A[a,b,c]   (a thread takes a proxy point with its six field components: three 16-byte
    // words per term, a matrix entry is loaded once for six products)
    for (int nu = threadIdx.x; nu < P; nu += XFER_THREADS) {
        const int c3 = nu % n1, ab = nu / n1;
        double s[6] = {0, 0, 0, 0, 0, 0};
#pragma unroll
        for (int k = 0; k < n1; ++k) {
            const double t = Tz[k * n1 + c3];
            const double2 *v = reinterpret_cast<const double2 *>(&A[6 * (ab * n1 + k)]);
            const double2 v0 = v[0], v1 = v[1], v2 = v[2];
            s[0] = fma(t, v0.x, s[0]); s[1] = fma(t, v0.y, s[1]); s[2] = fma(t, v1.x, s[2]);
            s[3] = fma(t, v1.y, s[3]); s[4] = fma(t, v2.x, s[4]); s[5] = fma(t, v2.y, s[5]);
        }
        double2 *o = reinterpret_cast<double2 *>(&B[6 * nu]);
        o[0] = make_double2(s[0], s[1]); o[1] = make_double2(s[2], s[3]); o[2] = make_double2(s[4], s[5]);
    }
    __syncthreads();
    // y: A[a,b',c'] = sum_b Ty[b][b'] B[a,b,c']
    for (int nu = threadIdx.x; nu < P; nu += XFER_THREADS) {
        const int c3 = nu % n1, b = (nu / n1) % n1, a = nu / (n1 * n1);
        double s[6] = {0, 0, 0, 0, 0, 0};
#pragma unroll
        for (int k = 0; k < n1; ++k) {
            const double t = Ty[k * n1 + b];
            const double2 *v = reinterpret_cast<const double2 *>(&B[6 * ((a * n1 + k) * n1 + c3)]);
            const double2 v0 = v[0], v1 = v[1], v2 = v[2];
            s[0] = fma(t, v0.x, s[0]); s[1] = fma(t, v0.y, s[1]); s[2] = fma(t, v1.x, s[2]);
            s[3] = fma(t, v1.y, s[3]); s[4] = fma(t, v2.x, s[4]); s[5] = fma(t, v2.y, s[5]);
        }
        double2 *o = reinterpret_cast<double2 *>(&A[6 * nu]);
        o[0] = make_double2(s[0], s[1]); o[1] = make_double2(s[2], s[3]); o[2] = make_double2(s[4], s[5]);
    }
    __syncthreads();
    // x: L_S'[a',b',c'] += sum_a Tx[a][a'] A[a,b',c']
    for (int e = threadIdx.x; e < P6; e += XFER_THREADS) {
        int f = e % 6, nu = e / 6, bc = nu % (n1 * n1), a = nu / (n1 * n1);
        double s = 0.0;
        for (int k = 0; k < n1; ++k) s = fma(Tx[k * n1 + a], A[6 * (k * n1 * n1 + bc) + f], s);
        LC[e] += s;
    }
    if (C < leaves) {  // an inner node: its children wait for this stamp
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0) *((volatile int *)&ready[C]) = stamp;
    }
}

// ---------------------------------------------------------------------------------------
// a9 + a10: L2P, add the near field, prefactors, scatter to caller order.  One block per leaf, one thread
// per particle; the leaf's local fields sit in shared memory and are read as broadcasts.
// ---------------------------------------------------------------------------------------
#define L2P_THREADS 128
#define L2P_SEGS 256

template <int N1>
__global__ void __launch_bounds__(L2P_THREADS) l2p_kernel(cheb_t ch, int leaves, int N, const int32_t *__restrict__ node_lo,
                                                          const int32_t *__restrict__ node_hi, const double *__restrict__ bbox,
                                                          const double *__restrict__ tx, const double *__restrict__ ty,
                                                          const double *__restrict__ tz, const double *__restrict__ L,
                                                          const double *__restrict__ near_, int K, int skip_far, const int32_t *__restrict__ perm,
                                                          const int32_t *__restrict__ p2p_off, const int32_t *__restrict__ p2p_recv,
                                                          const double *__restrict__ react, size_t rstride,
                                                          double cE, double cB, double *__restrict__ Ex, double *__restrict__ Ey,
                                                          double *__restrict__ Ez, double *__restrict__ Bx, double *__restrict__ By,
                                                          double *__restrict__ Bz)
{
    extern __shared__ __align__(16) double sm[];
    __shared__ int seg[L2P_SEGS];    // reaction segments of this leaf's row, in list order
    __shared__ int nseg_s;
    constexpr int n = N1 - 1, n1 = N1, P = n1 * n1 * n1, P6 = 6 * P;
    double *Ls = sm;                 // [P][6]
    double *bas = sm + P6;           // [3][n1][L2P_THREADS]
    int node = leaves + blockIdx.x;
    int lo = node_lo[node], hi = node_hi[node];
    const double *bb = bbox + 6 * (int64_t)node;
    const double *Ln = L + (int64_t)P6 * node;
    if (!skip_far) {  // the leaf's local field: all loads of a thread first (one memory round trip), 16-byte words
        constexpr int W2 = P6 / 2, PER = (W2 + L2P_THREADS - 1) / L2P_THREADS;  // (6 P doubles: an even number)
        const double2 *src2 = reinterpret_cast<const double2 *>(Ln);
        double2 *dst2 = reinterpret_cast<double2 *>(Ls);
        double2 v[PER];
#pragma unroll
        for (int k = 0; k < PER; ++k) {
            const int e = threadIdx.x + k * L2P_THREADS;
            if (e < W2) v[k] = src2[e];
        }
#pragma unroll
        for (int k = 0; k < PER; ++k) {
            const int e = threadIdx.x + k * L2P_THREADS;
            if (e < W2) dst2[e] = v[k];
        }
    }
    // mutual near field: the segments holding the pairs a neighbour's block evaluated (g(x_j, x_i) = -g(x_i, x_j)); warp 0
    // compacts the row's valid entries in list order, so that the gather below runs on independent loads
    const int row0 = p2p_recv ? p2p_off[node] : 0, rowlen = p2p_recv ? p2p_off[node + 1] - row0 : 0;
    if (threadIdx.x < 32) {
        int count = 0;
        for (int e0 = 0; e0 < rowlen; e0 += 32) {
            const int e = e0 + threadIdx.x;
            const int r = (e < rowlen) ? p2p_recv[row0 + e] : -1;
            const unsigned int m = __ballot_sync(0xffffffffu, r >= 0);
            const int at = count + __popc(m & ((1u << threadIdx.x) - 1u));
            if (r >= 0 && at < L2P_SEGS) seg[at] = r;
            count += __popc(m);
        }
        if (threadIdx.x == 0) nseg_s = count;
    }
    __syncthreads();
    const int nseg = nseg_s;  // (> L2P_SEGS: the row is walked entry by entry instead)
    for (int k = lo + threadIdx.x; k < hi; k += L2P_THREADS) {
        double *lx = bas + threadIdx.x, *ly = lx + n1 * L2P_THREADS, *lz = ly + n1 * L2P_THREADS;
        basis_1d(n, ch, bb[0], bb[3], tx[k], lx, L2P_THREADS);
        basis_1d(n, ch, bb[1], bb[4], ty[k], ly, L2P_THREADS);
        basis_1d(n, ch, bb[2], bb[5], tz[k], lz, L2P_THREADS);
        double fx[6] = {0, 0, 0, 0, 0, 0};
        for (int a = 0; a < (skip_far ? 0 : n1); ++a) {
            double fy[6] = {0, 0, 0, 0, 0, 0};
            for (int b = 0; b < n1; ++b) {
                double fz[6] = {0, 0, 0, 0, 0, 0};
                const double *row = Ls + 6 * (size_t)((a * n1 + b) * n1);
                for (int c3 = 0; c3 < n1; ++c3) {
                    double l = lz[c3 * L2P_THREADS];
                    const double2 *v = reinterpret_cast<const double2 *>(row + 6 * c3);  // (three 16-byte broadcasts)
                    const double2 v0 = v[0], v1 = v[1], v2 = v[2];
                    fz[0] = fma(l, v0.x, fz[0]); fz[1] = fma(l, v0.y, fz[1]); fz[2] = fma(l, v1.x, fz[2]);
                    fz[3] = fma(l, v1.y, fz[3]); fz[4] = fma(l, v2.x, fz[4]); fz[5] = fma(l, v2.y, fz[5]);
                }
                double l = ly[b * L2P_THREADS];
#pragma unroll
                for (int f = 0; f < 6; ++f) fy[f] = fma(l, fz[f], fy[f]);
            }
            double l = lx[a * L2P_THREADS];
#pragma unroll
            for (int f = 0; f < 6; ++f) fx[f] = fma(l, fy[f], fx[f]);
        }
        int i = perm[k];
        // fixed order: near + far, then the prefactors of eq. (3.1)
        double nr[6];  // near field: the K row chunks of P2P, added in chunk order
#pragma unroll
        for (int f = 0; f < 6; ++f) nr[f] = near_[f * (size_t)N + k];
        if (K > 1)
            for (int kc = 1; kc < K; ++kc)
#pragma unroll
                for (int f = 0; f < 6; ++f) nr[f] += near_[((size_t)kc * 6 + f) * (size_t)N + k];
        if (nseg <= L2P_SEGS) {
#pragma unroll 8
            for (int q = 0; q < nseg; ++q) {
                const double *rp = react + (size_t)seg[q] + (size_t)(k - lo);
#pragma unroll
                for (int f = 0; f < 6; ++f) nr[f] -= rp[f * rstride];
            }
        } else {
            for (int e = row0; e < row0 + rowlen; ++e) {
                const int r = p2p_recv[e];
                if (r < 0) continue;
                const double *rp = react + (size_t)r + (size_t)(k - lo);
#pragma unroll
                for (int f = 0; f < 6; ++f) nr[f] -= rp[f * rstride];
            }
        }
        Ex[i] = cE * (nr[0] + fx[0]);
        Ey[i] = cE * (nr[1] + fx[1]);
        Ez[i] = cE * (nr[2] + fx[2]);
        Bx[i] = cB * (nr[3] + fx[3]);
        By[i] = cB * (nr[4] + fx[4]);
        Bz[i] = cB * (nr[5] + fx[5]);
    }
}

// ---------------------------------------------------------------------------------------
static int set_smem(fmm_ctx *c, const void *fn, size_t bytes)
{
    // (dynamic + static shared memory count against the 48 KB default: opt in a little below it)
    if (bytes > 40 * 1024) FMM_CUDA(c, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return FMM_OK;
}

template <int N1>
static int launch_p2m(fmm_plan *p, const cheb_t &ch)
{
    fmm_ctx *c = &p->ctx;
    const size_t smem = p2m_cfg<N1>::SMEM;
    FMM_TRY(set_smem(c, (const void *)p2m_kernel<N1>, smem));
    p2m_kernel<N1><<<(unsigned)p->leaves, P2M_THREADS, smem, c->stream>>>(ch, (int)p->leaves, p->node_lo, p->node_hi, p->bbox, p->tx, p->ty,
                                                                        p->tz, p->w0, p->w1, p->w2, p->w3, p->M);
    FMM_LAUNCH_CHECK(c, "p2m_kernel");
    return FMM_OK;
}

int interp_p2m(fmm_plan *p)
{
    cheb_t ch = host_cheb(p->n);
    switch (p->n1) {
        case 2: return launch_p2m<2>(p, ch);
        case 3: return launch_p2m<3>(p, ch);
        case 4: return launch_p2m<4>(p, ch);
        case 5: return launch_p2m<5>(p, ch);
        case 6: return launch_p2m<6>(p, ch);
        case 7: return launch_p2m<7>(p, ch);
        case 8: return launch_p2m<8>(p, ch);
        case 9: return launch_p2m<9>(p, ch);
        case 10: return launch_p2m<10>(p, ch);
        case 11: return launch_p2m<11>(p, ch);
        case 12: return launch_p2m<12>(p, ch);
        case 13: return launch_p2m<13>(p, ch);
    }
    return FMM_EINVAL;
}

// kernels templated on N1 = n + 1: dispatch on the plan's order
#include <type_traits>
template <typename F>
static int dispatch_n1(int n1, F &&f)
{
    switch (n1) {
#define INTERP_CASE(K) case K: return f(std::integral_constant<int, K>{});
        INTERP_CASE(2) INTERP_CASE(3) INTERP_CASE(4) INTERP_CASE(5) INTERP_CASE(6) INTERP_CASE(7) INTERP_CASE(8)
        INTERP_CASE(9) INTERP_CASE(10) INTERP_CASE(11) INTERP_CASE(12) INTERP_CASE(13)
#undef INTERP_CASE
    }
    return FMM_EINVAL;
}

int interp_m2m(fmm_plan *p)
{
    fmm_ctx *c = &p->ctx;
    if (p->kappa < 1) return FMM_OK;
    size_t smem = sizeof(double) * (3 * (size_t)p->n1 * p->n1 + 1 + 8 * (size_t)p->P);
    FMM_TRY(dispatch_n1(p->n1, [&](auto k) { return set_smem(c, (const void *)m2m_kernel<decltype(k)::value>, smem); }));
    const int first = 1 << (p->kappa - 1);  // one block per parent of two leaves; it climbs as long as it is the second to arrive
    FMM_TRY(dispatch_n1(p->n1, [&](auto k) {
        m2m_kernel<decltype(k)::value><<<first, xfer_cfg<decltype(k)::value>::THREADS, smem, c->stream>>>(first, p->node_lo, p->node_hi, p->node_T, p->M, p->xfer_sync);
        return FMM_OK;
    }));
    FMM_LAUNCH_CHECK(c, "m2m_kernel");
    return FMM_OK;
}

int interp_l2l(fmm_plan *p)
{
    fmm_ctx *c = &p->ctx;
    if (p->kappa < 1) return FMM_OK;
    size_t smem = sizeof(double) * (3 * (size_t)p->n1 * p->n1 + 1 + 12 * (size_t)p->P);
    FMM_TRY(dispatch_n1(p->n1, [&](auto k) { return set_smem(c, (const void *)l2l_kernel<decltype(k)::value>, smem); }));
    p->xfer_stamp = (p->xfer_stamp >= (1 << 30)) ? 1 : p->xfer_stamp + 1;
    int *ready = p->xfer_sync + (p->nodes + 2);
    FMM_TRY(dispatch_n1(p->n1, [&](auto k) {
        l2l_kernel<decltype(k)::value><<<(unsigned)(p->nodes - 1), xfer_cfg<decltype(k)::value>::THREADS, smem, c->stream>>>(2, (int)p->leaves, p->xfer_stamp, p->node_lo, p->node_hi,
                                                                                                   p->node_T, p->L, ready);
        return FMM_OK;
    }));
    FMM_LAUNCH_CHECK(c, "l2l_kernel");
    return FMM_OK;
}

int interp_l2p_finalize(fmm_plan *p, double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz)
{
    fmm_ctx *c = &p->ctx;
    cheb_t ch = host_cheb(p->n);
    double cE = 1.0, cB = 1.0;
    if (!(p->flags & FMM_RAW_SUMS)) {  // eq. (3.1)
        cE = 1.0 / (4.0 * FMM_PI * FMM_EPS0);
        cB = 1.0 / (4.0 * FMM_PI * FMM_EPS0 * FMM_C0);
    }
    size_t smem = sizeof(double) * (6 * (size_t)p->P + 3 * (size_t)p->n1 * L2P_THREADS);
    FMM_TRY(dispatch_n1(p->n1, [&](auto k) { return set_smem(c, (const void *)l2p_kernel<decltype(k)::value>, smem); }));
    const int nparts = p->p2p_split + ((p->flags & FMM_METHOD_TREECODE) ? 1 : 0);
    const int skip_far = (p->flags & FMM_METHOD_TREECODE) ? 1 : 0;
    FMM_TRY(dispatch_n1(p->n1, [&](auto k) {
        l2p_kernel<decltype(k)::value><<<(unsigned)p->leaves, L2P_THREADS, smem, c->stream>>>(
            ch, (int)p->leaves, (int)p->N, p->node_lo, p->node_hi, p->bbox, p->tx, p->ty, p->tz, p->L, p->near_, nparts, skip_far, p->perm,
            p->p2p_off, p->react_used ? p->p2p_recv : NULL, p->react, (size_t)(p->react_cap > 0 ? p->react_cap : 1), cE, cB, Ex, Ey, Ez, Bx, By, Bz);
        return FMM_OK;
    }));
    FMM_LAUNCH_CHECK(c, "l2p_kernel");
    return FMM_OK;
}
