// kernels_pairs.cu -- the two FP64-bound stages of the hot path and the all-pairs ceiling kernel:
//   a7   P2P  Alg 5.10 (eq. (2.7)) over the P2P list
//   a6   M2L  Alg 5.9  (eq. (2.5)) over the M2L list
//   a11  direct summation
// Kernel of eq. (3.2) with the mean gamma_bar everywhere (reading G6).
// Accumulation is target-owned: one block owns one target cluster and walks its CSR row in order;
// no floating-point atomics anywhere.
// These are not contractions (the kernel is not separable): plain FP64 pipe, no tensor cores.
#include "fmm_internal.cuh"

// ---------------------------------------------------------------------------------------
// source weights (a0): w0 = q gamma, (w1,w2,w3) = q p, gamma = sqrt(1 + p.p)
// ---------------------------------------------------------------------------------------
__global__ void source_weights_kernel(int64_t N, const double *__restrict__ px, const double *__restrict__ py,
                                      const double *__restrict__ pz, const double *__restrict__ q, double q_scalar,
                                      double *__restrict__ w0, double *__restrict__ w1, double *__restrict__ w2, double *__restrict__ w3)
{
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    double ax = px[j], ay = py[j], az = pz[j];
    double qj = q ? q[j] : q_scalar;
    double gam = sqrt(1.0 + (ax * ax + ay * ay + az * az));
    w0[j] = qj * gam;
    w1[j] = qj * ax;
    w2[j] = qj * ay;
    w3[j] = qj * az;
}

int pairs_source_weights(fmm_ctx *c, int64_t N, const double *px, const double *py, const double *pz,
                         const double *q, double q_scalar, double *w0, double *w1, double *w2, double *w3)
{
    source_weights_kernel<<<(unsigned)((N + 255) / 256), 256, 0, c->stream>>>(N, px, py, pz, q, q_scalar, w0, w1, w2, w3);
    FMM_LAUNCH_CHECK(c, "source_weights_kernel");
    return FMM_OK;
}

// ---------------------------------------------------------------------------------------
// shared-memory source tile: 4 x double2 per source = (x,y) (z,m0) (m1,m2) (m3,-), read as
// warp-wide broadcasts (every thread of a warp reads the same source): 4 LDS.128 per evaluation-warp.
// ---------------------------------------------------------------------------------------
#define PAIR_TILE 256

__device__ __forceinline__ void stage_tile(double2 *tile, int count, const double *__restrict__ x, const double *__restrict__ y,
                                           const double *__restrict__ z, const double *__restrict__ w0, const double *__restrict__ w1,
                                           const double *__restrict__ w2, const double *__restrict__ w3, int64_t base)
{
    for (int j = threadIdx.x; j < count; j += blockDim.x) {
        tile[4 * j + 0] = make_double2(x[base + j], y[base + j]);
        tile[4 * j + 1] = make_double2(z[base + j], w0[base + j]);
        tile[4 * j + 2] = make_double2(w1[base + j], w2[base + j]);
        tile[4 * j + 3] = make_double2(w3[base + j], 0.0);
    }
}

__device__ __forceinline__ void tile_interact(const double2 *tile, int count, double xt, double yt, double zt, double g2,
                                              double &ex, double &ey, double &ez, double &bx, double &by, double &bz)
{
#pragma unroll 4
    for (int j = 0; j < count; ++j) {
        double2 a = tile[4 * j + 0], b = tile[4 * j + 1], c = tile[4 * j + 2], d = tile[4 * j + 3];
        pair_accumulate(xt, yt, zt, g2, a.x, a.y, b.x, b.y, c.x, c.y, d.x, ex, ey, ez, bx, by, bz);
    }
}

// ---------------------------------------------------------------------------------------
// a7: P2P.  One block per target leaf (blocks issued in descending-work order); one thread per
// target particle; the source leaves of the CSR row are staged tile by tile.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) p2p_kernel(int N, double g2, const int32_t *__restrict__ order, const int32_t *__restrict__ off,
                                                  const int32_t *__restrict__ src, const int32_t *__restrict__ node_lo,
                                                  const int32_t *__restrict__ node_hi, const double *__restrict__ tx,
                                                  const double *__restrict__ ty, const double *__restrict__ tz,
                                                  const double *__restrict__ w0, const double *__restrict__ w1,
                                                  const double *__restrict__ w2, const double *__restrict__ w3, double *__restrict__ near_)
{
    __shared__ double2 tile[4 * PAIR_TILE];
    const int t = order[blockIdx.x];
    const int tlo = node_lo[t], thi = node_hi[t];
    const int e0 = off[t], e1 = off[t + 1];
    for (int i0 = tlo; i0 < thi; i0 += blockDim.x) {
        int i = i0 + threadIdx.x;
        bool live = i < thi;
        double xt = live ? tx[i] : 0.0, yt = live ? ty[i] : 0.0, zt = live ? tz[i] : 0.0;
        double ex = 0, ey = 0, ez = 0, bx = 0, by = 0, bz = 0;
        for (int e = e0; e < e1; ++e) {
            int s = src[e];
            int slo = node_lo[s], shi = node_hi[s];
            for (int j0 = slo; j0 < shi; j0 += PAIR_TILE) {
                int count = min(PAIR_TILE, shi - j0);
                __syncthreads();
                stage_tile(tile, count, tx, ty, tz, w0, w1, w2, w3, j0);
                __syncthreads();
                tile_interact(tile, count, xt, yt, zt, g2, ex, ey, ez, bx, by, bz);
            }
        }
        if (live) {
            near_[i] = ex;
            near_[(size_t)N + i] = ey;
            near_[2 * (size_t)N + i] = ez;
            near_[3 * (size_t)N + i] = bx;
            near_[4 * (size_t)N + i] = by;
            near_[5 * (size_t)N + i] = bz;
        }
    }
}

int pairs_p2p(fmm_plan *p)
{
    fmm_ctx *c = &p->ctx;
    int maxleaf = (int)((p->N + p->leaves - 1) / p->leaves);
    int threads = ((maxleaf + 31) / 32) * 32;
    if (threads > 256) threads = 256;
    if (threads < 32) threads = 32;
    p2p_kernel<<<(unsigned)p->leaves, threads, 0, c->stream>>>((int)p->N, p->gamma_bar * p->gamma_bar, p->p2p_order, p->p2p_off, p->p2p_src,
                                                               p->node_lo, p->node_hi, p->tx, p->ty, p->tz, p->w0, p->w1, p->w2, p->w3,
                                                               p->near_);
    FMM_LAUNCH_CHECK(c, "p2p_kernel");
    return FMM_OK;
}

// ---------------------------------------------------------------------------------------
// a11: direct summation.  grid = (target blocks, source splits); each block sums its slice of the
// sources for 256 targets; the slices are then added in a fixed order by direct_reduce.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) direct_kernel(int64_t N, double g2, int64_t nt, const int64_t *__restrict__ tidx,
                                                     int64_t chunk, const double *__restrict__ x, const double *__restrict__ y,
                                                     const double *__restrict__ z, const double *__restrict__ w0,
                                                     const double *__restrict__ w1, const double *__restrict__ w2,
                                                     const double *__restrict__ w3, double *__restrict__ part /* [splits][6][nt] */)
{
    __shared__ double2 tile[4 * PAIR_TILE];
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool live = k < nt;
    int64_t i = live ? (tidx ? tidx[k] : k) : 0;
    double xt = live ? x[i] : 0.0, yt = live ? y[i] : 0.0, zt = live ? z[i] : 0.0;
    double ex = 0, ey = 0, ez = 0, bx = 0, by = 0, bz = 0;
    int64_t s0 = (int64_t)blockIdx.y * chunk, s1 = s0 + chunk;
    if (s1 > N) s1 = N;
    for (int64_t j0 = s0; j0 < s1; j0 += PAIR_TILE) {
        int count = (int)((s1 - j0 < PAIR_TILE) ? (s1 - j0) : PAIR_TILE);
        __syncthreads();
        stage_tile(tile, count, x, y, z, w0, w1, w2, w3, j0);
        __syncthreads();
        tile_interact(tile, count, xt, yt, zt, g2, ex, ey, ez, bx, by, bz);
    }
    if (live) {
        double *o = part + (size_t)blockIdx.y * 6 * nt + k;
        o[0] = ex; o[nt] = ey; o[2 * nt] = ez; o[3 * nt] = bx; o[4 * nt] = by; o[5 * nt] = bz;
    }
}

__global__ void direct_reduce(int64_t nt, int splits, const double *__restrict__ part, double cE, double cB,
                              double *__restrict__ Ex, double *__restrict__ Ey, double *__restrict__ Ez,
                              double *__restrict__ Bx, double *__restrict__ By, double *__restrict__ Bz)
{
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nt) return;
    double a[6] = {0, 0, 0, 0, 0, 0};
    for (int s = 0; s < splits; ++s)
#pragma unroll
        for (int f = 0; f < 6; ++f) a[f] += part[((size_t)s * 6 + f) * nt + k];
    Ex[k] = cE * a[0]; Ey[k] = cE * a[1]; Ez[k] = cE * a[2];
    Bx[k] = cB * a[3]; By[k] = cB * a[4]; Bz[k] = cB * a[5];
}

int pairs_direct(fmm_ctx *c, int64_t N, const double *x, const double *y, const double *z,
                 const double *w0, const double *w1, const double *w2, const double *w3,
                 double gamma_bar, int raw, int64_t nt, const int64_t *tidx,
                 double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz)
{
    int64_t tblocks = (nt + 255) / 256;
    // enough blocks for ~8 waves of 148 SMs x 4 resident blocks, source slices in whole tiles
    int64_t want = 8 * 4 * FMM_SM_COUNT;
    int64_t splits = (want + tblocks - 1) / tblocks;
    int64_t tiles = (N + PAIR_TILE - 1) / PAIR_TILE;
    if (splits > tiles) splits = tiles;
    if (splits > 65535) splits = 65535;
    if (splits < 1) splits = 1;
    int64_t chunk = ((tiles + splits - 1) / splits) * PAIR_TILE;
    splits = (N + chunk - 1) / chunk;
    double *part = (double *)ctx_alloc(c, sizeof(double) * 6 * (size_t)nt * (size_t)splits);
    if (!part) return FMM_ENOMEM;
    dim3 grid((unsigned)tblocks, (unsigned)splits);
    direct_kernel<<<grid, 256, 0, c->stream>>>(N, gamma_bar * gamma_bar, nt, tidx, chunk, x, y, z, w0, w1, w2, w3, part);
    FMM_LAUNCH_CHECK(c, "direct_kernel");
    double cE = 1.0, cB = 1.0;
    if (!raw) {
        cE = 1.0 / (4.0 * FMM_PI * FMM_EPS0);
        cB = 1.0 / (4.0 * FMM_PI * FMM_EPS0 * FMM_C0);
    }
    direct_reduce<<<(unsigned)tblocks, 256, 0, c->stream>>>(nt, (int)splits, part, cE, cB, Ex, Ey, Ez, Bx, By, Bz);
    FMM_LAUNCH_CHECK(c, "direct_reduce");
    ctx_free(c, part);
    return FMM_OK;
}

// ---------------------------------------------------------------------------------------
// a6: M2L.  One block per target node (descending-work order), one thread per target proxy point
// mu = (a,b,c).  The proxy grids are tensor products, so the differences separate per axis:
//   D = (xt_a - xs_a')^2 + (yt_b - ys_b')^2 + gamma_bar^2 (zt_c - zs_c')^2
// The thread keeps dz and gamma_bar^2 dz^2 for its c against all c' in registers, builds dx^2 + dy^2
// in the two outer loops and runs the innermost loop over c'.  Inside it only the sums
//   A_k = sum_c' m_k w   (k = 0..3)   and   Z_k = sum_c' m_k w dz   (k = 0..2)
// are formed (dx, dy are constant there):  E += (A0 dx, A0 dy, Z0),
//   B += (Z2 - A3 dy, A3 dx - Z1, A1 dy - A2 dx).   15 FP64 instructions per evaluation + 9 per (a',b').
// ---------------------------------------------------------------------------------------
template <int N1>
struct m2l_cfg {
    static constexpr int P = N1 * N1 * N1;
    static constexpr int BATCHES = (P + 1023) / 1024;
    static constexpr int PER = (P + BATCHES - 1) / BATCHES;
    static constexpr int THREADS = ((PER + 31) / 32) * 32;
};

struct cheb13 {
    double c[FMM_MAX_ORDER + 1];
};

template <int N1>
__global__ void __launch_bounds__(m2l_cfg<N1>::THREADS) m2l_kernel(cheb13 ch, double g2, const int32_t *__restrict__ order,
                                                                   const int32_t *__restrict__ off, const int32_t *__restrict__ src,
                                                                   const double *__restrict__ bbox, const double *__restrict__ M,
                                                                   double *__restrict__ L)
{
    constexpr int P = m2l_cfg<N1>::P;
    constexpr int THREADS = m2l_cfg<N1>::THREADS;
    extern __shared__ double2 m2l_smem[];
    double2 *Ms = m2l_smem;                                                    // (m0,m1) (m2,m3) per source proxy
    double(*xs)[N1 + 1] = reinterpret_cast<double(*)[N1 + 1]>(m2l_smem + 2 * P);  // source proxy coordinates per axis
    const int t = order[blockIdx.x];
    const int e0 = off[t], e1 = off[t + 1];
    double *Lt = L + 6 * (size_t)P * t;
    if (e0 == e1) {  // no far-field sources: the local expansion starts at zero (L2L adds into it)
        for (int k = threadIdx.x; k < 6 * P; k += THREADS) Lt[k] = 0.0;
        return;
    }
    const double *bt = bbox + 6 * (size_t)t;
    for (int mu0 = 0; mu0 < P; mu0 += THREADS) {
        const int mu = mu0 + threadIdx.x;
        const bool live = mu < P;
        const int a = live ? mu / (N1 * N1) : 0, b = live ? (mu / N1) % N1 : 0, c3 = live ? mu % N1 : 0;
        // I-3: xi = (a+b)/2 + (b-a)/2 c_k, rounded as the sequence mul, mul, add
        const double xt = __dadd_rn(__dmul_rn(__dadd_rn(bt[0], bt[3]), 0.5), __dmul_rn(__dmul_rn(__dsub_rn(bt[3], bt[0]), 0.5), ch.c[a]));
        const double yt = __dadd_rn(__dmul_rn(__dadd_rn(bt[1], bt[4]), 0.5), __dmul_rn(__dmul_rn(__dsub_rn(bt[4], bt[1]), 0.5), ch.c[b]));
        const double zt = __dadd_rn(__dmul_rn(__dadd_rn(bt[2], bt[5]), 0.5), __dmul_rn(__dmul_rn(__dsub_rn(bt[5], bt[2]), 0.5), ch.c[c3]));
        double ex = 0, ey = 0, ez = 0, bx = 0, by = 0, bz = 0;
        for (int e = e0; e < e1; ++e) {
            const int s = src[e];
            __syncthreads();
            {
                const double2 *Mg = reinterpret_cast<const double2 *>(M + 4 * (size_t)P * s);
                for (int k = threadIdx.x; k < 2 * P; k += THREADS) Ms[k] = Mg[k];
                if (threadIdx.x < 3 * N1) {
                    int g = threadIdx.x / N1, k = threadIdx.x - g * N1;
                    const double *bs = bbox + 6 * (size_t)s;
                    xs[g][k] = __dadd_rn(__dmul_rn(__dadd_rn(bs[g], bs[3 + g]), 0.5),
                                         __dmul_rn(__dmul_rn(__dsub_rn(bs[3 + g], bs[g]), 0.5), ch.c[k]));
                }
            }
            __syncthreads();
            double dz[N1], gz2[N1];
#pragma unroll
            for (int k = 0; k < N1; ++k) {
                dz[k] = zt - xs[2][k];
                gz2[k] = (g2 * dz[k]) * dz[k];
            }
            for (int a2 = 0; a2 < N1; ++a2) {
                const double dx = xt - xs[0][a2];
                const double dx2 = dx * dx;
#pragma unroll 1
                for (int b2 = 0; b2 < N1; ++b2) {
                    const double dy = yt - xs[1][b2];
                    const double s2 = fma(dy, dy, dx2);
                    const double2 *row = Ms + 2 * ((a2 * N1 + b2) * N1);
                    double A0 = 0, A1 = 0, A2 = 0, A3 = 0, Z0 = 0, Z1 = 0, Z2 = 0;
#pragma unroll
                    for (int c2 = 0; c2 < N1; ++c2) {
                        const double w = inv_r3(s2 + gz2[c2]);
                        const double2 m01 = row[2 * c2], m23 = row[2 * c2 + 1];
                        const double wz = w * dz[c2];
                        A0 = fma(m01.x, w, A0);
                        A1 = fma(m01.y, w, A1);
                        A2 = fma(m23.x, w, A2);
                        A3 = fma(m23.y, w, A3);
                        Z0 = fma(m01.x, wz, Z0);
                        Z1 = fma(m01.y, wz, Z1);
                        Z2 = fma(m23.x, wz, Z2);
                    }
                    ex = fma(A0, dx, ex);
                    ey = fma(A0, dy, ey);
                    ez += Z0;
                    bx = fma(-A3, dy, bx + Z2);
                    by = fma(A3, dx, by - Z1);
                    bz = fma(A1, dy, fma(-A2, dx, bz));
                }
            }
        }
        if (live) {
            double *o = Lt + 6 * (size_t)mu;
            o[0] = ex; o[1] = ey; o[2] = ez; o[3] = bx; o[4] = by; o[5] = bz;
        }
    }
}

template <int N1>
static int launch_m2l(fmm_plan *p, const cheb13 &ch)
{
    fmm_ctx *c = &p->ctx;
    const size_t smem = sizeof(double2) * 2 * m2l_cfg<N1>::P + sizeof(double) * 3 * (N1 + 1);
    if (smem > 48 * 1024)
        FMM_CUDA(c, cudaFuncSetAttribute((const void *)m2l_kernel<N1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    m2l_kernel<N1><<<(unsigned)p->nodes, m2l_cfg<N1>::THREADS, smem, c->stream>>>(ch, p->gamma_bar * p->gamma_bar, p->m2l_order, p->m2l_off,
                                                                               p->m2l_src, p->bbox, p->M, p->L);
    FMM_LAUNCH_CHECK(c, "m2l_kernel");
    return FMM_OK;
}

int pairs_m2l(fmm_plan *p)
{
    cheb13 ch;
    memset(&ch, 0, sizeof(ch));
    for (int k = 0; k <= p->n; ++k) ch.c[k] = sin(FMM_PI * (double)(p->n - 2 * k) / (double)(2 * p->n));  // I-1
    ch.c[0] = 1.0;
    ch.c[p->n] = -1.0;
    switch (p->n1) {
        case 2: return launch_m2l<2>(p, ch);
        case 3: return launch_m2l<3>(p, ch);
        case 4: return launch_m2l<4>(p, ch);
        case 5: return launch_m2l<5>(p, ch);
        case 6: return launch_m2l<6>(p, ch);
        case 7: return launch_m2l<7>(p, ch);
        case 8: return launch_m2l<8>(p, ch);
        case 9: return launch_m2l<9>(p, ch);
        case 10: return launch_m2l<10>(p, ch);
        case 11: return launch_m2l<11>(p, ch);
        case 12: return launch_m2l<12>(p, ch);
        case 13: return launch_m2l<13>(p, ch);
    }
    return FMM_EINVAL;
}
