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

// SM (FMM_KERNEL_SOURCE_MOMENTUM): a fifth double2 carries the source's plain momentum, (m3,px) (py,pz).
template <bool SM>
__device__ __forceinline__ void stage_tile(double2 *tile, int count, const double *__restrict__ x, const double *__restrict__ y,
                                           const double *__restrict__ z, const double *__restrict__ w0, const double *__restrict__ w1,
                                           const double *__restrict__ w2, const double *__restrict__ w3, const double *__restrict__ px,
                                           const double *__restrict__ py, const double *__restrict__ pz, int64_t base)
{
    constexpr int ST = SM ? 5 : 4;
    for (int j = threadIdx.x; j < count; j += blockDim.x) {
        tile[ST * j + 0] = make_double2(x[base + j], y[base + j]);
        tile[ST * j + 1] = make_double2(z[base + j], w0[base + j]);
        tile[ST * j + 2] = make_double2(w1[base + j], w2[base + j]);
        tile[ST * j + 3] = make_double2(w3[base + j], SM ? px[base + j] : 0.0);
        if (SM) tile[ST * j + 4] = make_double2(py[base + j], pz[base + j]);
    }
}

// One staged tile acting on the thread's NT targets: the tile is read once from shared memory for NT evaluations
// (4 LDS.128 per source), and the accumulate-FMAs of the NT targets that share a source weight are adjacent.
template <int NT, bool SM>
__device__ __forceinline__ void tile_interact(const double2 *tile, int count, const double (&xt)[NT], const double (&yt)[NT],
                                              const double (&zt)[NT], double gb, double (&ex)[NT], double (&ey)[NT], double (&ez)[NT],
                                              double (&bx)[NT], double (&by)[NT], double (&bz)[NT])
{
#pragma unroll 2
    for (int j = 0; j < count; ++j) {
        constexpr int ST = SM ? 5 : 4;
        double2 a = tile[ST * j + 0], b = tile[ST * j + 1], c = tile[ST * j + 2], d = tile[ST * j + 3];
        double2 pyz = SM ? tile[ST * j + (SM ? 4 : 0)] : make_double2(0.0, 0.0);
        double gx[NT], gy[NT], gz[NT];
#pragma unroll
        for (int k = 0; k < NT; ++k) {
            double dx = xt[k] - a.x, dy = yt[k] - a.y, dz = zt[k] - b.x;
            double D = fma(dx, dx, FMM_TINY_D);  // (> 0 also for a coincident pair: see inv_r3)
            D = fma(dy, dy, D);
            if (SM) {  // D = |d|^2 + (p_j . d)^2 (G6 alternative)
                D = fma(dz, dz, D);
                double pd = fma(pyz.y, dz, fma(pyz.x, dy, d.y * dx));
                D = fma(pd, pd, D);
            } else {   // eq. (3.2): D = dx^2 + dy^2 + (gamma_bar dz)^2; squaring the scaled difference keeps the
                       // DFMA at two register operands (full FP64 issue rate)
                const double sz = gb * dz;
                D = fma(sz, sz, D);
            }
            double w = inv_r3(D);
            gx[k] = w * dx; gy[k] = w * dy; gz[k] = w * dz;
        }
        const double m0 = b.y, m1 = c.x, m2 = c.y, m3 = d.x;
#pragma unroll
        for (int k = 0; k < NT; ++k) { ex[k] = fma(m0, gx[k], ex[k]); ey[k] = fma(m0, gy[k], ey[k]); ez[k] = fma(m0, gz[k], ez[k]); }
#pragma unroll
        for (int k = 0; k < NT; ++k) { bx[k] = fma(m2, gz[k], bx[k]); bz[k] = fma(-m2, gx[k], bz[k]); }
#pragma unroll
        for (int k = 0; k < NT; ++k) { by[k] = fma(m3, gx[k], by[k]); bx[k] = fma(-m3, gy[k], bx[k]); }
#pragma unroll
        for (int k = 0; k < NT; ++k) { bz[k] = fma(m1, gy[k], bz[k]); by[k] = fma(-m1, gz[k], by[k]); }
    }
}

// ---------------------------------------------------------------------------------------
// a7: P2P.  One block per target leaf (blocks issued in descending-work order); NT target particles per
// thread; the source leaves of the CSR row are staged tile by tile.
// ---------------------------------------------------------------------------------------
template <int NT, bool SM, bool SPLIT>
__global__ void __launch_bounds__(256) p2p_kernel(int N, double gb, const int32_t *__restrict__ order, const int32_t *__restrict__ off,
                                                  const int32_t *__restrict__ src, const int32_t *__restrict__ node_lo,
                                                  const int32_t *__restrict__ node_hi, const double *__restrict__ tx,
                                                  const double *__restrict__ ty, const double *__restrict__ tz,
                                                  const double *__restrict__ w0, const double *__restrict__ w1,
                                                  const double *__restrict__ w2, const double *__restrict__ w3,
                                                  const double *__restrict__ pmx, const double *__restrict__ pmy,
                                                  const double *__restrict__ pmz, int K, double *__restrict__ near_)
{
    __shared__ double2 tile[(SM ? 5 : 4) * PAIR_TILE];
    // block (t, k): chunk k of the K contiguous chunks of target t's row; its sums go to partial buffer k
    const int t = SPLIT ? order[blockIdx.x / K] : order[blockIdx.x], kc = SPLIT ? blockIdx.x % K : 0;
    const int tlo = node_lo[t], thi = node_hi[t];
    const int r0 = off[t], rl = off[t + 1] - r0;
    const int e0 = SPLIT ? r0 + (int)(((int64_t)rl * kc) / K) : r0, e1 = SPLIT ? r0 + (int)(((int64_t)rl * (kc + 1)) / K) : r0 + rl;
    for (int i0 = tlo; i0 < thi; i0 += NT * blockDim.x) {
        double xt[NT], yt[NT], zt[NT], ex[NT], ey[NT], ez[NT], bx[NT], by[NT], bz[NT];
#pragma unroll
        for (int k = 0; k < NT; ++k) {
            int i = i0 + k * blockDim.x + threadIdx.x;
            bool live = i < thi;
            xt[k] = live ? tx[i] : 0.0; yt[k] = live ? ty[i] : 0.0; zt[k] = live ? tz[i] : 0.0;
            ex[k] = ey[k] = ez[k] = bx[k] = by[k] = bz[k] = 0.0;
        }
        for (int e = e0; e < e1; ++e) {
            int s = src[e];
            int slo = node_lo[s], shi = node_hi[s];
            for (int j0 = slo; j0 < shi; j0 += PAIR_TILE) {
                int count = min(PAIR_TILE, shi - j0);
                __syncthreads();
                stage_tile<SM>(tile, count, tx, ty, tz, w0, w1, w2, w3, pmx, pmy, pmz, j0);
                __syncthreads();
                tile_interact<NT, SM>(tile, count, xt, yt, zt, gb, ex, ey, ez, bx, by, bz);
            }
        }
#pragma unroll
        for (int k = 0; k < NT; ++k) {
            int i = i0 + k * blockDim.x + threadIdx.x;
            if (i < thi) {
                double *o = near_ + (SPLIT ? (size_t)kc * 6 * (size_t)N : (size_t)0) + i;
                o[0] = ex[k];
                o[(size_t)N] = ey[k];
                o[2 * (size_t)N] = ez[k];
                o[3 * (size_t)N] = bx[k];
                o[4 * (size_t)N] = by[k];
                o[5 * (size_t)N] = bz[k];
            }
        }
    }
}


// ---------------------------------------------------------------------------------------
// a7, mutual form (mean-gamma kernel only).  g(x_j, x_i) = -g(x_i, x_j) for the kernel of eq. (3.2), so for a pair of
// leaves {t, s} that sits in the P2P list in both directions the owner's block evaluates D^{-3/2} once per particle
// pair and forms both sums: 34 FP64 instructions per particle pair = 17 per kernel evaluation instead of 25.
//   * targets: NT particles per thread in registers (positions, their own source weights, six sums), as in p2p_kernel;
//   * sources: the owned source leaves of the row are streamed through a shared-memory tile (structure of arrays) in
//     batches of 32; at step k of a batch lane l works on source (l + k) mod 32, so every lane reads its own source
//     (conflict-free LDS.64) and every target / source pair of the batch is visited once in 32 steps;
//   * reaction: the six sums of a source travel with it from lane to lane (SHFL, one rotation per step) and are back in
//     the source's home lane after 32 steps holding the contribution of this warp's 32 NT targets; the warps of the
//     block are then added in warp order (shared memory) and the result is stored to the partial segment of the
//     entry (s, t), which L2P subtracts from s's own sums in list order.  One writer per segment, fixed orders: no atomics.
// Entries without a mate (and t's own leaf) go through the one-sided loop.  Dead lanes / padded sources carry zero
// weights (they add exact zeros) and their own results are dropped.
// ---------------------------------------------------------------------------------------
#define MUT_TILE 256

template <int NT>
struct mut_targets {
    double x[NT], y[NT], z[NT], q0[NT], q1[NT], q2[NT], q3[NT];
    double ex[NT], ey[NT], ez[NT], bx[NT], by[NT], bz[NT];
};

struct mut_tile {
    double x[MUT_TILE], y[MUT_TILE], z[MUT_TILE], m0[MUT_TILE], m1[MUT_TILE], m2[MUT_TILE], m3[MUT_TILE];
    int dst[MUT_TILE];
};

// NL <= NT: the first NL of the thread's NT target slots are worked on (a warp whose last slot holds no particle of a ragged
// leaf runs the NL = NT - 1 instantiation, see p2p_mutual_kernel)
template <int NT, int NL = NT>
__device__ __forceinline__ void mut_pair_terms(const mut_targets<NT> &T, double gb, double xs, double ys, double zs,
                                               double (&gx)[NT], double (&gy)[NT], double (&gz)[NT])
{
#pragma unroll
    for (int k = 0; k < NL; ++k) {
        const double dx = T.x[k] - xs, dy = T.y[k] - ys, dz = T.z[k] - zs;
        double D = fma(dx, dx, FMM_TINY_D);  // (> 0 also for a coincident pair: see inv_r3)
        D = fma(dy, dy, D);
        const double sz = gb * dz;
        D = fma(sz, sz, D);
        const double w = inv_r3(D);
        gx[k] = w * dx; gy[k] = w * dy; gz[k] = w * dz;
    }
}

template <int NT, int NL = NT>
__device__ __forceinline__ void mut_target_sums(mut_targets<NT> &T, double m0, double m1, double m2, double m3,
                                                const double (&gx)[NT], const double (&gy)[NT], const double (&gz)[NT])
{
#pragma unroll
    for (int k = 0; k < NL; ++k) { T.ex[k] = fma(m0, gx[k], T.ex[k]); T.ey[k] = fma(m0, gy[k], T.ey[k]); T.ez[k] = fma(m0, gz[k], T.ez[k]); }
#pragma unroll
    for (int k = 0; k < NL; ++k) { T.bx[k] = fma(m2, gz[k], T.bx[k]); T.bz[k] = fma(-m2, gx[k], T.bz[k]); }
#pragma unroll
    for (int k = 0; k < NL; ++k) { T.by[k] = fma(m3, gx[k], T.by[k]); T.bx[k] = fma(-m3, gy[k], T.bx[k]); }
#pragma unroll
    for (int k = 0; k < NL; ++k) { T.bz[k] = fma(m1, gy[k], T.bz[k]); T.by[k] = fma(-m1, gz[k], T.by[k]); }
}

// one step of a batch: lane l works on source b0 + (l + k2) mod 32 with its first NL target slots, then the six reaction sums
// move on to the lane that takes this source next
template <int NT, int NL>
__device__ __forceinline__ void mut_step(mut_targets<NT> &T, const mut_tile &S, int b0, int lane, int k2, double gb, double &rex,
                                         double &rey, double &rez, double &rbx, double &rby, double &rbz)
{
    const int j = b0 + ((lane + k2) & 31);
    const double xs = S.x[j], ys = S.y[j], zs = S.z[j], m0 = S.m0[j], m1 = S.m1[j], m2 = S.m2[j], m3 = S.m3[j];
    double gx[NT], gy[NT], gz[NT];
    mut_pair_terms<NT, NL>(T, gb, xs, ys, zs, gx, gy, gz);
    mut_target_sums<NT, NL>(T, m0, m1, m2, m3, gx, gy, gz);
#pragma unroll
    for (int k = 0; k < NL; ++k) {
        rex = fma(T.q0[k], gx[k], rex); rey = fma(T.q0[k], gy[k], rey); rez = fma(T.q0[k], gz[k], rez);
        rbx = fma(T.q2[k], gz[k], rbx); rbz = fma(-T.q2[k], gx[k], rbz);
        rby = fma(T.q3[k], gx[k], rby); rbx = fma(-T.q3[k], gy[k], rbx);
        rbz = fma(T.q1[k], gy[k], rbz); rby = fma(-T.q1[k], gz[k], rby);
    }
    const int from = (lane + 1) & 31;  // the source this lane takes next was with lane + 1
    rex = __shfl_sync(0xffffffffu, rex, from); rey = __shfl_sync(0xffffffffu, rey, from); rez = __shfl_sync(0xffffffffu, rez, from);
    rbx = __shfl_sync(0xffffffffu, rbx, from); rby = __shfl_sync(0xffffffffu, rby, from); rbz = __shfl_sync(0xffffffffu, rbz, from);
}

// `cnt` staged sources (a multiple of 32), both directions: this warp's part (no block barrier in here) ...
// HALF (W = 1): the last target slot holds the leaf's 1 .. 15 tail particles TWICE, in lanes l and l + MUT_HALF_OFF (odd), and is
// worked on at the even steps only: lane l then meets the sources of l's parity, lane l + MUT_HALF_OFF the others, so every
// (tail target, source) pair is still visited exactly once while the slot costs 16 steps of a batch instead of 32.
#define MUT_HALF_OFF 17
template <int NT, int NL, int W, bool ACCUM, bool HALF = false>  // ACCUM: add to the segment instead of overwriting it (all-pairs kernel)
__device__ __forceinline__ void mut_batches(mut_targets<NT> &T, const mut_tile &S, int cnt, double gb, double *red,
                                            double *__restrict__ react, size_t rstride)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int b0 = 0; b0 < cnt; b0 += 32) {
        double rex = 0, rey = 0, rez = 0, rbx = 0, rby = 0, rbz = 0;  // sum_i q_i (x) g(x_i, x_j) for the source travelling through this lane
        if (HALF) {
#pragma unroll 1
            for (int k2 = 0; k2 < 32; k2 += 2) {
                mut_step<NT, NL>(T, S, b0, lane, k2, gb, rex, rey, rez, rbx, rby, rbz);
                mut_step<NT, (NL > 1 ? NL - 1 : 1)>(T, S, b0, lane, k2 + 1, gb, rex, rey, rez, rbx, rby, rbz);
            }
        } else {
#pragma unroll 1
            for (int k2 = 0; k2 < 32; ++k2) mut_step<NT, NL>(T, S, b0, lane, k2, gb, rex, rey, rez, rbx, rby, rbz);
        }
        // lane l now holds the sums for source b0 + l over this warp's targets
        if (W == 1) {
            const int d = S.dst[b0 + lane];
            if (d >= 0) {
                const double r6[6] = {rex, rey, rez, rbx, rby, rbz};
#pragma unroll
                for (int f = 0; f < 6; ++f) react[f * rstride + d] = ACCUM ? react[f * rstride + d] + r6[f] : r6[f];
            }
        } else {
            double *r = red + (size_t)warp * (6 * MUT_TILE) + b0 + lane;
            r[0] = rex; r[MUT_TILE] = rey; r[2 * MUT_TILE] = rez; r[3 * MUT_TILE] = rbx; r[4 * MUT_TILE] = rby; r[5 * MUT_TILE] = rbz;
        }
    }
}

// ... and, once per tile, the warps' sums added in warp order and stored (W > 1; the caller's barrier follows)
template <int W, bool ACCUM>
__device__ __forceinline__ void mut_reduce_tile(const mut_tile &S, int cnt, double *red, double *__restrict__ react, size_t rstride)
{
    if (W > 1) {
        __syncthreads();
        for (int q = threadIdx.x; q < 6 * MUT_TILE; q += 32 * W) {
            const int j = q & (MUT_TILE - 1);
            if (j < cnt) {
                const int d = S.dst[j];
                double v = red[q];
#pragma unroll
                for (int w = 1; w < W; ++w) v += red[(size_t)w * (6 * MUT_TILE) + q];
                if (d >= 0) {
                    double *o = react + (size_t)(q / MUT_TILE) * rstride + d;
                    *o = ACCUM ? *o + v : v;
                }
            }
        }
    }
}

template <int NT, int W, bool ACCUM = false>
__device__ __forceinline__ void mut_process_mutual(mut_targets<NT> &T, const mut_tile &S, int cnt, double gb, double *red,
                                                   double *__restrict__ react, size_t rstride)
{
    mut_batches<NT, NT, W, ACCUM>(T, S, cnt, gb, red, react, rstride);
    mut_reduce_tile<W, ACCUM>(S, cnt, red, react, rstride);
}

// `cnt` staged sources acting on the targets only (broadcast reads)
template <int NT, int NL = NT>
__device__ __forceinline__ void mut_process_onesided(mut_targets<NT> &T, const mut_tile &S, int cnt, double gb)
{
#pragma unroll 2
    for (int j = 0; j < cnt; ++j) {
        double gx[NT], gy[NT], gz[NT];
        mut_pair_terms<NT, NL>(T, gb, S.x[j], S.y[j], S.z[j], gx, gy, gz);
        mut_target_sums<NT, NL>(T, S.m0[j], S.m1[j], S.m2[j], S.m3[j], gx, gy, gz);
    }
}

// resident warps per SM the register budget is sized for: 216 registers at NT = 4 schedule the four dependency chains of a
// step with the fewest stalls (profiles/r02_p2p_mutual.md), the smaller shapes fit more warps
template <int NT, int W>
struct mut_cfg {
    static constexpr int WARPS = (NT == 4) ? 8 : (NT == 3) ? ((W == 8) ? 8 : 12) : (NT == 2) ? 16 : 32;
    static constexpr int MINB = (WARPS / W) > 0 ? (WARPS / W) : 1;
};

// RAGGED (W > 1, leaves that leave at least one whole warp-slot of the block's 32 W NT target slots empty, e.g. 313 particles
// in 4 x 32 x 3 slots): the warps whose last slot is empty run the NL = NT - 1 instantiation of the loops, and the slot
// assignment is rotated by the block index.  Warp w of every block sits on SM sub-partition w mod 4, so without the rotation
// the lighter warps would always share the same sub-partitions and the heavier ones would still set the pace; with it every
// sub-partition sees the mix and the block's FP64 work drops from W NT to ceil(leaf / 32) warp-slots.
// Used at W = 8 only (one block per SM, so every sub-partition holds exactly one longer and one shorter warp): leaves of 625,
// n = 8 of the paper's grid, 37.9 -> 34.7 ms.  At W = 4 (three blocks per SM) the block barriers keep every block at the pace
// of its longer warps and the second copy of the loops only costs instruction fetches: leaves of 313, 17.7 -> 18.1 ms, not used.
// TP = 2 (leaves of 1025 .. 2048 particles, W = 8): the block walks its row twice, for the first 32 W NT targets and for the
// rest; the second walk ADDS its reaction sums to the segments the first one wrote (the same thread owns the same words).
// HALF (W = 1, NT >= 2, leaves whose last slot holds at most 15 particles, e.g. 78 = 32 + 32 + 14): see mut_batches.
template <int NT, int W, bool SPLIT, bool RAGGED = false, int TP = 1, bool HALF = false>
__global__ void __launch_bounds__(32 * W, mut_cfg<NT, W>::MINB) p2p_mutual_kernel(int N, double gb, const int32_t *__restrict__ order, const int32_t *__restrict__ off,
                                                         const int32_t *__restrict__ src, const int32_t *__restrict__ dst,
                                                         const int32_t *__restrict__ node_lo, const int32_t *__restrict__ node_hi,
                                                         const double *__restrict__ tx, const double *__restrict__ ty,
                                                         const double *__restrict__ tz, const double *__restrict__ w0,
                                                         const double *__restrict__ w1, const double *__restrict__ w2,
                                                         const double *__restrict__ w3, int K, double *__restrict__ near_,
                                                         double *__restrict__ react, size_t rstride)
{
    __shared__ mut_tile S;
    extern __shared__ double mut_red[];  // [W][6][MUT_TILE] reaction sums of the current tile, per warp (W > 1)
    const int t = SPLIT ? order[blockIdx.x / K] : order[blockIdx.x], kc = SPLIT ? blockIdx.x % K : 0;
    const int tlo0 = node_lo[t], thi0 = node_hi[t];
    const int r0 = off[t], rl = off[t + 1] - r0;
    const int e0 = SPLIT ? r0 + (int)(((int64_t)rl * kc) / K) : r0, e1 = SPLIT ? r0 + (int)(((int64_t)rl * (kc + 1)) / K) : r0 + rl;
#pragma unroll 1
    for (int tp = 0; tp < TP; ++tp) {
    int tlo, thi;  // the targets of this walk over the row
    if (TP > 1 && HALF) {  // (TP = 2) the two halves of the leaf
        const int half = (thi0 - tlo0 + 1) / 2;
        tlo = tlo0 + tp * half;
        thi = (tp + 1 < TP) ? tlo0 + half : thi0;
    } else {
        tlo = tlo0 + tp * (32 * W * NT);
        thi = (TP > 1 && tp + 1 < TP) ? min(thi0, tlo + 32 * W * NT) : thi0;
    }
    if (TP > 1 && tp > 0) __syncthreads();  // (the tile of the walk before is no longer read)
    mut_targets<NT> T;
    // slot k of this thread holds target tlo + k blockDim + vt; vt = the thread index, rotated by whole warps when RAGGED
    const int vt = RAGGED ? (int)((threadIdx.x + 32u * (blockIdx.x % W)) & (32u * W - 1u)) : (int)threadIdx.x;
    bool short_warp = false;  // (warp-uniform) the warp's last slot holds no particle at all
    if (RAGGED) short_warp = (NT > 1) && (tlo + (NT - 1) * (int)blockDim.x + (vt & ~31) >= thi);
    // HALF: every warp takes an equal, contiguous share [wlo, whi) of the targets (slot k of lane l = wlo + 32 k + l), so that all
    // warps of the block have the same short last slot; the second copy of its tail particle l sits in lane l + MUT_HALF_OFF
    const int lane = threadIdx.x & 31;
    int wlo = tlo, whi = thi, tstride = blockDim.x, tpos = vt;
    if (HALF) {
        const int share = (max(thi - tlo, 0) + W - 1) / W;
        wlo = min(thi, tlo + (int)(threadIdx.x >> 5) * share);
        whi = min(thi, wlo + share);
        tstride = 32;
        tpos = lane;
    }
    const int tail = HALF ? max(0, whi - (wlo + (NT - 1) * 32)) : 0;  // (at most 15 by the choice of the shape)
    const bool copy_b = HALF && lane >= MUT_HALF_OFF && lane - MUT_HALF_OFF < tail;
#pragma unroll
    for (int k = 0; k < NT; ++k) {
        int i = wlo + k * tstride + tpos;
        if (HALF && k == NT - 1 && copy_b) i -= MUT_HALF_OFF;
        const bool live = i < whi;
        T.x[k] = live ? tx[i] : 0.0; T.y[k] = live ? ty[i] : 0.0; T.z[k] = live ? tz[i] : 0.0;
        T.q0[k] = live ? w0[i] : 0.0; T.q1[k] = live ? w1[i] : 0.0; T.q2[k] = live ? w2[i] : 0.0; T.q3[k] = live ? w3[i] : 0.0;
        T.ex[k] = T.ey[k] = T.ez[k] = T.bx[k] = T.by[k] = T.bz[k] = 0.0;
    }
    double keep[6] = {0, 0, 0, 0, 0, 0};  // HALF: the second copy's sums while the one-sided pass (all sources, every step) runs
    // the row is walked twice: first the owned mutual entries (pass 0), then the one-sided ones (pass 1); the sources of a
    // pass form one stream that fills the tile across entry boundaries, so only the last tile of a pass is ragged
    for (int pass = 0; pass < 2; ++pass) {
        int fill = 0;
        if (HALF && pass == 1) {  // the one-sided loops visit every source in every lane: only the first copy may count them
            keep[0] = T.ex[NT - 1]; keep[1] = T.ey[NT - 1]; keep[2] = T.ez[NT - 1];
            keep[3] = T.bx[NT - 1]; keep[4] = T.by[NT - 1]; keep[5] = T.bz[NT - 1];
        }
        for (int e = e0; e <= e1; ++e) {
            int slo = 0, shi = 0, d = -1;
            const bool flush = (e == e1);
            if (!flush) {
                d = dst[e];
                if (pass == 0 ? (d < 0) : (d != -1)) continue;
                const int s = src[e];
                slo = node_lo[s]; shi = node_hi[s];
            }
            int j0 = slo;
            while (j0 < shi || (flush && fill > 0)) {
                if (!flush) {
                    const int n = min(shi - j0, MUT_TILE - fill);
                    for (int j = threadIdx.x; j < n; j += blockDim.x) {
                        const int a = fill + j, g = j0 + j;
                        S.x[a] = tx[g]; S.y[a] = ty[g]; S.z[a] = tz[g];
                        S.m0[a] = w0[g]; S.m1[a] = w1[g]; S.m2[a] = w2[g]; S.m3[a] = w3[g];
                        S.dst[a] = d + (g - slo);
                    }
                    fill += n; j0 += n;
                    if (fill < MUT_TILE) break;  // (this entry is exhausted)
                } else if (pass == 0) {
                    const int padded = (fill + 31) & ~31;  // dead sources: zero weights, nowhere to store
                    for (int a = fill + threadIdx.x; a < padded; a += blockDim.x) {
                        S.x[a] = S.y[a] = S.z[a] = S.m0[a] = S.m1[a] = S.m2[a] = S.m3[a] = 0.0;
                        S.dst[a] = -1;
                    }
                    fill = padded;
                }
                __syncthreads();
                if (pass == 0) {
                    if (RAGGED && short_warp) mut_batches<NT, (NT > 1 ? NT - 1 : 1), W, false>(T, S, fill, gb, mut_red, react, rstride);
                    else mut_batches<NT, NT, W, false, HALF>(T, S, fill, gb, mut_red, react, rstride);
                    // (all warps meet at its barrier; the second walk over the row adds to what the first one stored)
                    if (TP > 1 && tp > 0) mut_reduce_tile<W, true>(S, fill, mut_red, react, rstride);
                    else mut_reduce_tile<W, false>(S, fill, mut_red, react, rstride);
                } else {
                    if (RAGGED && short_warp) mut_process_onesided<NT, (NT > 1 ? NT - 1 : 1)>(T, S, fill, gb);
                    else mut_process_onesided<NT>(T, S, fill, gb);
                }
                __syncthreads();
                fill = 0;
            }
        }
    }
    if (HALF) {  // the tail particle's sums = first copy (mutual + one-sided entries) + second copy (its share of the mutual ones)
        double *s6[6] = {&T.ex[NT - 1], &T.ey[NT - 1], &T.ez[NT - 1], &T.bx[NT - 1], &T.by[NT - 1], &T.bz[NT - 1]};
#pragma unroll
        for (int f = 0; f < 6; ++f) {
            const double mine = copy_b ? keep[f] : *s6[f];
            const double other = __shfl_sync(0xffffffffu, mine, (lane + MUT_HALF_OFF) & 31);
            *s6[f] = (lane < tail) ? mine + other : mine;
        }
    }
#pragma unroll
    for (int k = 0; k < NT; ++k) {
        const int i = wlo + k * tstride + tpos;
        if (i < whi) {
            double *o = near_ + (SPLIT ? (size_t)kc * 6 * (size_t)N : (size_t)0) + i;
            o[0] = T.ex[k];
            o[(size_t)N] = T.ey[k];
            o[2 * (size_t)N] = T.ez[k];
            o[3 * (size_t)N] = T.bx[k];
            o[4 * (size_t)N] = T.by[k];
            o[5 * (size_t)N] = T.bz[k];
        }
    }
    }  // tp
}

// Targets per thread: the NT <= 4 that wastes the fewest lanes, ties to the larger NT (a leaf of 78 particles fills 3 x 32 slots at NT = 3 but only 78 of 128 at NT = 4).
// Mutual kernel (mutual != 0): a whole leaf in one pass, the fewest warps W in {1, 2, 4, 8} with NT <= 4, then the smallest NT;
// the travelling reaction sums cost the same per step whatever NT is, so NT is kept high (NT >= 3 whenever W > 1).
static void p2p_shape(int64_t leaves, int maxleaf, int64_t pairs, int64_t max_row, int *nt_out, int *threads_out, int *split_out,
                      int mutual = 0)
{
    int best_nt = 1, best_threads = 32;
    double best_score = -1.0;
    if (mutual && maxleaf <= FMM_MUTUAL_MAX_LEAF) {
        // (leaves of more than 1024 particles: two target passes of eight warps, the shape is that of half a leaf)
        if (maxleaf > 1024) maxleaf = (maxleaf + 1) / 2;
        // W a power of two: the resident warps of an SM then split evenly over its four sub-partitions (three warps per
        // block left one sub-partition with 3 of 9 warps: 46 % instead of 59 % of peak at leaves of 312, profiles/r02_sweep_paper.md)
        int W = 1;
        while (32 * 4 * W < maxleaf) W *= 2;
        best_threads = 32 * W;
        best_nt = (maxleaf + best_threads - 1) / best_threads;
        if (best_nt < 1) best_nt = 1;
        best_score = 1.0;
    }
    for (int nt = 1; nt <= 4 && best_score < 0.0; ++nt) {
        int per = (maxleaf + nt - 1) / nt;
        int threads = ((per + 31) / 32) * 32;
        if (threads > 256) threads = 256;
        int passes = (maxleaf + nt * threads - 1) / (nt * threads);
        double eff = (double)maxleaf / ((double)passes * nt * threads);
        double score = eff * (1.0 + 0.02 * nt);  // ties: more targets per thread (the row split K restores the block count)
        if (score > best_score) { best_score = score; best_nt = nt; best_threads = threads; }
    }
    *nt_out = best_nt;
    *threads_out = best_threads;
    // Row split K: (a) enough warps in flight when there are few leaves, (b) no single row longer than a quarter of an
    // SM's fair share of the whole near field (the tail leaves of a Gaussian bunch have rows of several hundred leaves).
    double warps = (double)leaves * (best_threads / 32);
    // four waves of resident warps: with few leaves (N = 65,536: 512 one-warp blocks) the last wave otherwise runs a third
    // empty (P2P 48 % -> 62 % of peak there, profiles/r02_bench_configs.md)
    const double K_FILL_WAVES = 4.0;
    int k_fill = (int)((K_FILL_WAVES * 8.0 * FMM_SM_COUNT + warps - 1) / warps);
    double fair = (double)pairs / (4.0 * FMM_SM_COUNT);
    int k_bal = (fair > 0.0) ? (int)((double)max_row / fair + 0.999) : 1;
    int K = k_fill > k_bal ? k_fill : k_bal;
    if (K > 8) K = 8;
    if (K < 1) K = 1;
    *split_out = K;
}

int pairs_m2l_prepare(fmm_plan *p)  // after the lists: M2L row split for small trees
{
    fmm_ctx *c = &p->ctx;
    int K = 1;
    if (!(p->flags & FMM_METHOD_TREECODE) && p->n_m2l > 0) {
        // two resident blocks per SM; aim at four waves of blocks.  Only trees with few nodes need it, and the partial
        // buffers stay below 256 MB.
        int64_t want = 4 * 2 * FMM_SM_COUNT;
        K = (int)((want + p->nodes - 1) / p->nodes);
        if (K > 8) K = 8;
        if (K < 1) K = 1;
        while (K > 1 && (int64_t)(K - 1) * 48 * p->P * (p->nodes + 2) > ((int64_t)256 << 20)) --K;
    }
    p->m2l_split = K;
    int64_t need = (int64_t)(K - 1) * 6 * p->P * (p->nodes + 2);
    if (need > p->lpart_cap) {
        if (p->Lpart) ctx_free(c, p->Lpart);
        p->Lpart = (double *)ctx_alloc_keep(c, sizeof(double) * (size_t)need);
        if (!p->Lpart) return FMM_ENOMEM;
        p->lpart_cap = need;
    }
    return FMM_OK;
}

// the mutual kernel keeps a whole target leaf in one pass of NT x blockDim registers
static bool p2p_use_mutual(const fmm_plan *p, int maxleaf) { return p->p2p_mutual && p->p2p_dst != NULL && maxleaf <= FMM_MUTUAL_MAX_LEAF; }

int pairs_p2p_prepare(fmm_plan *p)  // after the lists: choose the row split and size the partial buffers
{
    fmm_ctx *c = &p->ctx;
    int maxleaf = p->maxleaf;
    int nt, threads, K;
    if (p2p_use_mutual(p, maxleaf) && p->p2p_react > p->react_cap) {
        if (p->react) ctx_free(c, p->react);
        p->react_cap = 0;
        p->react = (double *)ctx_alloc_keep(c, sizeof(double) * 6 * (size_t)p->p2p_react);
        if (p->react) {
            p->react_cap = p->p2p_react;
        } else {  // no room for the reaction segments (48 bytes per particle of half the list): the one-sided kernel needs none
            p->p2p_mutual = 0;
            c->err[0] = 0;
        }
    }
    p2p_shape(p->leaves, maxleaf, p->p2p_pairs, p->p2p_max_row, &nt, &threads, &K, p2p_use_mutual(p, maxleaf));
    p->p2p_split = K;
    int64_t need = (int64_t)(K + ((p->flags & FMM_METHOD_TREECODE) ? 1 : 0)) * 6 * p->N;  // treecode: + the particle-cluster sums
    if (need > p->near_cap) {
        if (p->near_) ctx_free(c, p->near_);
        p->near_ = (double *)ctx_alloc_keep(c, sizeof(double) * (size_t)need);
        if (!p->near_) return FMM_ENOMEM;
        p->near_cap = need;
    }
    return FMM_OK;
}

int pairs_p2p(fmm_plan *p)
{
    fmm_ctx *c = &p->ctx;
    int maxleaf = p->maxleaf;
    int nt, threads, K;
    p2p_shape(p->leaves, maxleaf, p->p2p_pairs, p->p2p_max_row, &nt, &threads, &K, p2p_use_mutual(p, maxleaf));
    K = p->p2p_split;
    const bool sm = (p->flags & FMM_KERNEL_SOURCE_MOMENTUM) != 0;
    p->react_used = p2p_use_mutual(p, maxleaf) ? 1 : 0;
    if (p->react_used) {
        const size_t rstride = (size_t)(p->react_cap > 0 ? p->react_cap : 1);
#define MUT_LAUNCH_R(NT, W, R, TP, H)                                                                                                     \
    {                                                                                                                                     \
        const size_t red_bytes = (W > 1) ? sizeof(double) * 6 * MUT_TILE * W : 0;                                                         \
        if (red_bytes + sizeof(mut_tile) > 48 * 1024) {                                                                                   \
            FMM_CUDA(c, cudaFuncSetAttribute((const void *)p2p_mutual_kernel<NT, W, true, R, TP, H>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)red_bytes));  \
            FMM_CUDA(c, cudaFuncSetAttribute((const void *)p2p_mutual_kernel<NT, W, false, R, TP, H>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)red_bytes)); \
        }                                                                                                                                 \
        if (K > 1)                                                                                                                        \
            p2p_mutual_kernel<NT, W, true, R, TP, H><<<(unsigned)(p->leaves * K), 32 * W, red_bytes, c->stream>>>(                        \
                (int)p->N, p->gamma_bar, p->p2p_order, p->p2p_off, p->p2p_src, p->p2p_dst, p->node_lo, p->node_hi, p->tx, p->ty, p->tz, p->w0, \
                p->w1, p->w2, p->w3, K, p->near_, p->react, rstride);                                                                     \
        else                                                                                                                              \
            p2p_mutual_kernel<NT, W, false, R, TP, H><<<(unsigned)p->leaves, 32 * W, red_bytes, c->stream>>>(                             \
                (int)p->N, p->gamma_bar, p->p2p_order, p->p2p_off, p->p2p_src, p->p2p_dst, p->node_lo, p->node_hi, p->tx, p->ty, p->tz, p->w0, \
                p->w1, p->w2, p->w3, K, p->near_, p->react, rstride);                                                                     \
    }
#define MUT_LAUNCH(NT, W) MUT_LAUNCH_R(NT, W, false, 1, false)
// one warp per block: the last slot at half rate when it holds at most 15 particles of the largest leaf
#define MUT_LAUNCH_1(NT)                                                          \
    if (maxleaf - 32 * (NT - 1) <= 15) MUT_LAUNCH_R(NT, 1, false, 1, true) else MUT_LAUNCH_R(NT, 1, false, 1, false)
// eight warps per block: two target passes for leaves of more than 1024 particles; else the ragged variant when at least one
// whole warp-slot of the block stays empty
#define MUT_LAUNCH_W(NT, W)                                                       \
    if (maxleaf > 1024) {                                                         \
        if (MUT_HALF_OK(NT, W)) MUT_LAUNCH_R(NT, W, false, 2, true) else MUT_LAUNCH_R(NT, W, true, 2, false)            \
    } else if (MUT_HALF_OK(NT, W)) MUT_LAUNCH_R(NT, W, false, 1, true)            \
    else if (32 * W * NT - maxleaf >= 32) MUT_LAUNCH_R(NT, W, true, 1, false) else MUT_LAUNCH_R(NT, W, false, 1, false)
// two or four warps per block: the half-rate last slot when every warp's share of the largest leaf ends in 1 .. 15 particles
#define MUT_LAUNCH_H(NT, W)                                                       \
    if (MUT_HALF_OK(NT, W)) MUT_LAUNCH_R(NT, W, false, 1, true) else MUT_LAUNCH_R(NT, W, false, 1, false)
// (the share of a warp: the largest leaf, or its larger half when the block walks its row twice, divided by the warps)
#define MUT_SHARE(W) (((maxleaf > 1024 ? (maxleaf + 1) / 2 : maxleaf) + W - 1) / W)
#define MUT_HALF_OK(NT, W) ((MUT_SHARE(W) + 31) / 32 == NT && MUT_SHARE(W) - 32 * (NT - 1) >= 1 && MUT_SHARE(W) - 32 * (NT - 1) <= 15)
        const int W = threads / 32;
        if (nt == 1) { MUT_LAUNCH(1, 1); }
        else if (nt == 2) { MUT_LAUNCH_1(2); }
        else if (nt == 3 && W == 1) { MUT_LAUNCH_1(3); }
        else if (nt == 3 && W == 2) { MUT_LAUNCH_H(3, 2); }
        else if (nt == 3 && W == 4) { MUT_LAUNCH_H(3, 4); }
        else if (nt == 3) { MUT_LAUNCH_W(3, 8); }
        else if (W == 1) { MUT_LAUNCH_1(4); }
        else if (W == 2) { MUT_LAUNCH_H(4, 2); }
        else if (W == 4) { MUT_LAUNCH_H(4, 4); }
        else { MUT_LAUNCH_W(4, 8); }
#undef MUT_LAUNCH
#undef MUT_LAUNCH_1
#undef MUT_LAUNCH_H
#undef MUT_SHARE
#undef MUT_HALF_OK
#undef MUT_LAUNCH_W
#undef MUT_LAUNCH_R
        FMM_LAUNCH_CHECK(c, "p2p_mutual_kernel");
        return FMM_OK;
    }
#define P2P_LAUNCH(NT, SM)                                                                                                               \
    if (K > 1)                                                                                                                           \
        p2p_kernel<NT, SM, true><<<(unsigned)(p->leaves * K), threads, 0, c->stream>>>((int)p->N, p->gamma_bar, p->p2p_order, p->p2p_off, \
                                                                       p->p2p_src, p->node_lo, p->node_hi, p->tx, p->ty, p->tz, p->w0,   \
                                                                       p->w1, p->w2, p->w3, p->pmx, p->pmy, p->pmz, K, p->near_);        \
    else                                                                                                                                 \
    p2p_kernel<NT, SM, false><<<(unsigned)(p->leaves * K), threads, 0, c->stream>>>((int)p->N, p->gamma_bar, p->p2p_order, p->p2p_off, \
                                                                       p->p2p_src, p->node_lo, p->node_hi, p->tx, p->ty, p->tz, p->w0,   \
                                                                       p->w1, p->w2, p->w3, p->pmx, p->pmy, p->pmz, K, p->near_)
    switch (nt) {
        case 1: if (sm) P2P_LAUNCH(1, true); else P2P_LAUNCH(1, false); break;
        case 2: if (sm) P2P_LAUNCH(2, true); else P2P_LAUNCH(2, false); break;
        case 3: if (sm) P2P_LAUNCH(3, true); else P2P_LAUNCH(3, false); break;
        default: if (sm) P2P_LAUNCH(4, true); else P2P_LAUNCH(4, false); break;
    }
#undef P2P_LAUNCH
    FMM_LAUNCH_CHECK(c, "p2p_kernel");
    return FMM_OK;
}

// ---------------------------------------------------------------------------------------
// a11: direct summation.  grid = (target blocks, source splits); each block sums its slice of the sources for
// DIRECT_NT x 128 targets; the slices are then added in a fixed order by direct_reduce.
// ---------------------------------------------------------------------------------------
#define DIRECT_NT 4
#define DIRECT_THREADS 128
#define DIRECT_TARGETS (DIRECT_NT * DIRECT_THREADS)
template <bool SM>
__global__ void __launch_bounds__(DIRECT_THREADS) direct_kernel(int64_t N, double gb, int64_t nt, const int64_t *__restrict__ tidx,
                                                                int64_t chunk, const double *__restrict__ x, const double *__restrict__ y,
                                                                const double *__restrict__ z, const double *__restrict__ w0,
                                                                const double *__restrict__ w1, const double *__restrict__ w2,
                                                                const double *__restrict__ w3, const double *__restrict__ px,
                                                                const double *__restrict__ py, const double *__restrict__ pz,
                                                                double *__restrict__ part /* [splits][6][nt] */)
{
    __shared__ double2 tile[(SM ? 5 : 4) * PAIR_TILE];
    double xt[DIRECT_NT], yt[DIRECT_NT], zt[DIRECT_NT], ex[DIRECT_NT], ey[DIRECT_NT], ez[DIRECT_NT], bx[DIRECT_NT], by[DIRECT_NT], bz[DIRECT_NT];
#pragma unroll
    for (int k = 0; k < DIRECT_NT; ++k) {
        int64_t q = (int64_t)blockIdx.x * DIRECT_TARGETS + k * DIRECT_THREADS + threadIdx.x;
        bool live = q < nt;
        int64_t i = live ? (tidx ? tidx[q] : q) : 0;
        xt[k] = live ? x[i] : 0.0; yt[k] = live ? y[i] : 0.0; zt[k] = live ? z[i] : 0.0;
        ex[k] = ey[k] = ez[k] = bx[k] = by[k] = bz[k] = 0.0;
    }
    int64_t s0 = (int64_t)blockIdx.y * chunk, s1 = s0 + chunk;
    if (s1 > N) s1 = N;
    for (int64_t j0 = s0; j0 < s1; j0 += PAIR_TILE) {
        int count = (int)((s1 - j0 < PAIR_TILE) ? (s1 - j0) : PAIR_TILE);
        __syncthreads();
        stage_tile<SM>(tile, count, x, y, z, w0, w1, w2, w3, px, py, pz, j0);
        __syncthreads();
        tile_interact<DIRECT_NT, SM>(tile, count, xt, yt, zt, gb, ex, ey, ez, bx, by, bz);
    }
#pragma unroll
    for (int k = 0; k < DIRECT_NT; ++k) {
        int64_t q = (int64_t)blockIdx.x * DIRECT_TARGETS + k * DIRECT_THREADS + threadIdx.x;
        if (q < nt) {
            double *o = part + (size_t)blockIdx.y * 6 * nt + q;
            o[0] = ex[k]; o[nt] = ey[k]; o[2 * nt] = ez[k]; o[3 * nt] = bx[k]; o[4 * nt] = by[k]; o[5 * nt] = bz[k];
        }
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

// ---------------------------------------------------------------------------------------
// a11, mutual form (all targets, mean-gamma kernel): the particles are cut into tiles of 256 and the tiles into super-tiles of
// G; block (a, b), a <= b, lets every tile I of super-tile a act on every tile J of super-tile b and back (J >= I on the
// diagonal, I == J one-sided) with the same inner loops as the mutual near field.  The sums of the targets of I go to
// tpart[block][I], the reaction on J is added to rpart[block][J] in the fixed order of the I loop (one block owns the
// segment: no atomics); direct_mutual_reduce adds a particle's partials over the blocks of its row and column.
// ---------------------------------------------------------------------------------------
#define DM_NT 4
#define DM_W 2
__global__ void __launch_bounds__(32 * DM_W, mut_cfg<DM_NT, DM_W>::MINB) direct_mutual_kernel(
    int64_t N, double gb, int G, int S, const double *__restrict__ x, const double *__restrict__ y, const double *__restrict__ z,
    const double *__restrict__ w0, const double *__restrict__ w1, const double *__restrict__ w2, const double *__restrict__ w3,
    double *__restrict__ tpart, double *__restrict__ rpart /* [blocks][6][G * 256] each */)
{
    __shared__ mut_tile St;
    __shared__ double red[DM_W * 6 * MUT_TILE];
    // block -> (a, b), a <= b: row a holds S - a blocks
    int a = 0, rem = blockIdx.x;
    while (rem >= S - a) { rem -= S - a; ++a; }
    const int b = a + rem;
    const size_t plane = (size_t)G * MUT_TILE;
    double *tp = tpart + (size_t)blockIdx.x * 6 * plane, *rp = rpart + (size_t)blockIdx.x * 6 * plane;
    for (int il = 0; il < G; ++il) {
        const int64_t i0 = ((int64_t)a * G + il) * MUT_TILE;
        mut_targets<DM_NT> T;
#pragma unroll
        for (int k = 0; k < DM_NT; ++k) {
            const int64_t i = i0 + k * (32 * DM_W) + threadIdx.x;
            const bool live = i < N;
            T.x[k] = live ? x[i] : 0.0; T.y[k] = live ? y[i] : 0.0; T.z[k] = live ? z[i] : 0.0;
            T.q0[k] = live ? w0[i] : 0.0; T.q1[k] = live ? w1[i] : 0.0; T.q2[k] = live ? w2[i] : 0.0; T.q3[k] = live ? w3[i] : 0.0;
            T.ex[k] = T.ey[k] = T.ez[k] = T.bx[k] = T.by[k] = T.bz[k] = 0.0;
        }
        if (i0 < N) {
            for (int jl = (a == b ? il : 0); jl < G; ++jl) {
                const int64_t j0 = ((int64_t)b * G + jl) * MUT_TILE;
                if (j0 >= N) break;
                __syncthreads();
                for (int j = threadIdx.x; j < MUT_TILE; j += 32 * DM_W) {  // (dead sources: zero weights)
                    const int64_t g = j0 + j;
                    const bool live = g < N;
                    St.x[j] = live ? x[g] : 0.0; St.y[j] = live ? y[g] : 0.0; St.z[j] = live ? z[g] : 0.0;
                    St.m0[j] = live ? w0[g] : 0.0; St.m1[j] = live ? w1[g] : 0.0; St.m2[j] = live ? w2[g] : 0.0; St.m3[j] = live ? w3[g] : 0.0;
                    St.dst[j] = jl * MUT_TILE + j;
                }
                __syncthreads();
                // the reaction segment of J is written by the first tile I that meets it (il == 0) and added to afterwards
                if (a == b && il == jl) mut_process_onesided<DM_NT>(T, St, MUT_TILE, gb);
                else if (il == 0) mut_process_mutual<DM_NT, DM_W, false>(T, St, MUT_TILE, gb, red, rp, plane);
                else mut_process_mutual<DM_NT, DM_W, true>(T, St, MUT_TILE, gb, red, rp, plane);
            }
        }
#pragma unroll
        for (int k = 0; k < DM_NT; ++k) {
            const int q = il * MUT_TILE + k * (32 * DM_W) + threadIdx.x;
            tp[q] = T.ex[k]; tp[plane + q] = T.ey[k]; tp[2 * plane + q] = T.ez[k];
            tp[3 * plane + q] = T.bx[k]; tp[4 * plane + q] = T.by[k]; tp[5 * plane + q] = T.bz[k];
        }
    }
}

__global__ void direct_mutual_reduce(int64_t N, int G, int S, const double *__restrict__ tpart, const double *__restrict__ rpart, double cE,
                                     double cB, double *__restrict__ Ex, double *__restrict__ Ey, double *__restrict__ Ez,
                                     double *__restrict__ Bx, double *__restrict__ By, double *__restrict__ Bz)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const size_t plane = (size_t)G * MUT_TILE;
    const int s = (int)(i / (int64_t)plane);
    const size_t q = (size_t)(i - (int64_t)s * (int64_t)plane);
    auto block_of = [&](int a, int b) { return (size_t)a * S - (size_t)a * (a - 1) / 2 + (size_t)(b - a); };
    double acc[6] = {0, 0, 0, 0, 0, 0};
    for (int b = s; b < S; ++b) {  // this particle as a target: blocks (s, b)
        const double *p = tpart + block_of(s, b) * 6 * plane + q;
#pragma unroll
        for (int f = 0; f < 6; ++f) acc[f] += p[f * plane];
    }
    // ... and as a source: the reaction sums of blocks (c, s), g(x_j, x_i) = -g(x_i, x_j).  On the diagonal block the first tile
    // of the super-tile receives nothing (its segment is never written): tiles J > I only.
    for (int c = 0; c <= s; ++c) {
        if (c == s && q < MUT_TILE) continue;
        const double *p = rpart + block_of(c, s) * 6 * plane + q;
#pragma unroll
        for (int f = 0; f < 6; ++f) acc[f] -= p[f * plane];
    }
    Ex[i] = cE * acc[0]; Ey[i] = cE * acc[1]; Ez[i] = cE * acc[2];
    Bx[i] = cB * acc[3]; By[i] = cB * acc[4]; Bz[i] = cB * acc[5];
}

int pairs_direct(fmm_ctx *c, int64_t N, const double *x, const double *y, const double *z,
                 const double *w0, const double *w1, const double *w2, const double *w3,
                 const double *px, const double *py, const double *pz,
                 double gamma_bar, int raw, int64_t nt, const int64_t *tidx,
                 double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz)
{
    double cE = 1.0, cB = 1.0;
    if (!raw) {
        cE = 1.0 / (4.0 * FMM_PI * FMM_EPS0);
        cB = 1.0 / (4.0 * FMM_PI * FMM_EPS0 * FMM_C0);
    }
    if (!px && !tidx && nt == N && N >= 8 * MUT_TILE) {  // all targets, kernel of eq. (3.2): every pair once for both directions
        const int64_t tiles = (N + MUT_TILE - 1) / MUT_TILE;
        int G = (int)(tiles / 128);  // (about 8,000 blocks: enough to level the half-size diagonal blocks out)
        if (G < 1) G = 1;
        if (G > 32) G = 32;
        const int S = (int)((tiles + G - 1) / G);
        const int64_t blocks = (int64_t)S * (S + 1) / 2;
        const size_t bytes = sizeof(double) * 6 * (size_t)G * MUT_TILE * (size_t)blocks;
        if (2 * bytes <= ((size_t)8 << 30) && blocks < ((int64_t)1 << 31)) {
            double *tp = (double *)ctx_alloc(c, bytes), *rp = (double *)ctx_alloc(c, bytes);
            if (!tp || !rp) return FMM_ENOMEM;
            direct_mutual_kernel<<<(unsigned)blocks, 32 * DM_W, 0, c->stream>>>(N, gamma_bar, G, S, x, y, z, w0, w1, w2, w3, tp, rp);
            FMM_LAUNCH_CHECK(c, "direct_mutual_kernel");
            direct_mutual_reduce<<<(unsigned)((N + 255) / 256), 256, 0, c->stream>>>(N, G, S, tp, rp, cE, cB, Ex, Ey, Ez, Bx, By, Bz);
            FMM_LAUNCH_CHECK(c, "direct_mutual_reduce");
            ctx_free(c, rp);
            ctx_free(c, tp);
            return FMM_OK;
        }
    }
    int64_t tblocks = (nt + DIRECT_TARGETS - 1) / DIRECT_TARGETS;
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
    if (px)
        direct_kernel<true><<<grid, DIRECT_THREADS, 0, c->stream>>>(N, gamma_bar, nt, tidx, chunk, x, y, z, w0, w1, w2, w3, px, py, pz, part);
    else
        direct_kernel<false><<<grid, DIRECT_THREADS, 0, c->stream>>>(N, gamma_bar, nt, tidx, chunk, x, y, z, w0, w1, w2, w3, px, py, pz, part);
    FMM_LAUNCH_CHECK(c, "direct_kernel");
    direct_reduce<<<(unsigned)((nt + 255) / 256), 256, 0, c->stream>>>(nt, (int)splits, part, cE, cB, Ex, Ey, Ez, Bx, By, Bz);
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
#ifndef M2L_NT
#define M2L_NT 1
#endif
    static constexpr int NT = M2L_NT;                      // target proxy points per thread
    static constexpr int BATCHES = (P + 992 * NT - 1) / (992 * NT);  // 992 + the 32 producer threads = 1024 per block
    static constexpr int PER = (P + BATCHES - 1) / BATCHES;
    static constexpr int THREADS = (((PER + NT - 1) / NT + 31) / 32) * 32;
    // two resident blocks per SM while 2 x THREADS x 88 registers fit the register file (the dependent
    // seed -> series chain of inv_r3 needs >= 5 warps per sub-partition to keep the FP64 pipe fed)
#ifndef M2L_MINB
#define M2L_MINB 2
#endif
    static constexpr int MINB = (THREADS + 32 <= 400) ? M2L_MINB : 1;
    // pipeline depth: as many stages of (M tile + proxy coordinates) as fit 227 KB, at most 3
    static constexpr int STAGE_BYTES = 32 * P + 3 * 16 * 8;
    static constexpr int FIT = (227 * 1024 - 64) / STAGE_BYTES;
    static constexpr int STAGES = FIT >= 3 ? 3 : (FIT >= 2 ? 2 : 1);
    // Helper warp: WARPS consumer warps with WARPS % 4 == 3 (11 at n = 6) cannot be spread evenly over the four SM
    // sub-partitions.  One more consumer warp takes, for source e, the target group e mod (WARPS + 1) off its owner
    // (nothing when that is WARPS), so all WARPS + 1 warps do the same (WARPS / (WARPS + 1)) share of the work.
    static constexpr bool HELP = (NT == 1) && (BATCHES == 1) && ((THREADS / 32) % 4 == 3);
    static constexpr int CWARPS = THREADS / 32 + (HELP ? 1 : 0);       // consumer warps
    static constexpr int BLOCK = 32 * CWARPS + (HELP ? 0 : 32);        // + a producer warp (with a helper, the helper also refills the ring)
};

struct cheb13 {
    double c[FMM_MAX_ORDER + 1];
};

// ---- 1-D bulk TMA copy (global -> shared, completion on an mbarrier) ----------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}

__device__ __forceinline__ bool mbar_test(uint64_t *bar, uint32_t parity)  // non-blocking
{
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// Per-node tables for M2L, filled once per build (pairs_proxy_points):
//   xi[node][g][k]  proxy points per axis (reading I-3), row stride M2L_XI_STRIDE.  Row 2 (z) holds the points
//                   RELATIVE to the box centre z0 = (a_z + b_z)/2, and z0 itself sits in xi[node][2][15].
//                   xi[node][2][14] = h_z = (b_z - a_z)/2, so that zrel_k = h_z c_k up to one rounding of the proxy point.
// With z relative to the source box centre,  sum_nu m_k w dz = (zt - z0) sum_nu m_k w - h_z sum_nu m_k (c_{nu3} w):
// the innermost loop needs no dz array; the Chebyshev points c_k are compile-time-indexed constant-bank operands
// (m2l_cheb_c), so the extra product u = c_k w costs no register and vanishes for c_k = +-1 and 0.
#define M2L_XI_STRIDE 16
__constant__ double m2l_cheb_c[FMM_MAX_ORDER + 2][M2L_XI_STRIDE];  // [n1][k] = cos(k pi / (n1 - 1)) (reading I-1)
#define M2L_XI_BYTES (3 * M2L_XI_STRIDE * 8)
__global__ void m2l_proxy_points(int nodes, int n1, cheb13 ch, const double *__restrict__ bbox, double *__restrict__ xi)
{
    int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= (nodes + 1) * 3 * M2L_XI_STRIDE) return;
    int k = q % M2L_XI_STRIDE, g = (q / M2L_XI_STRIDE) % 3, i = q / (3 * M2L_XI_STRIDE);
    const double *bs = bbox + 6 * (size_t)i;
    double v = 0.0;
    if (i >= 1) {
        const double mid = __dmul_rn(__dadd_rn(bs[g], bs[3 + g]), 0.5);
        if (k < n1) {  // xi = (a+b)/2 + (b-a)/2 c_k, rounded as the sequence mul, mul, add
            v = __dadd_rn(mid, __dmul_rn(__dmul_rn(__dsub_rn(bs[3 + g], bs[g]), 0.5), ch.c[k]));
            if (g == 2) v = __dsub_rn(v, mid);
        } else if (g == 2 && k == M2L_XI_STRIDE - 1) {
            v = mid;
        } else if (g == 2 && k == M2L_XI_STRIDE - 2) {
            v = __dmul_rn(__dsub_rn(bs[3 + g], bs[g]), 0.5);
        }
    }
    xi[q] = v;
}

// Shared memory of one block: m2l_cfg::STAGES stages, each = the source node's moments (P x 4 doubles, one contiguous
// 32 P byte tile of M) + its proxy coordinates per axis, both fetched by 1-D bulk TMA copies that complete on the
// stage's `full` mbarrier.  There is no block-wide barrier in the source loop: every warp walks the CSR row at its
// own pace, waits on full[stage], and releases the stage on empty[stage] (one arrival per warp); an extra producer
// warp refills a stage as soon as all consumer warps have left it, so warps may drift up to STAGES-1 sources apart.
// one source node (stage in shared memory) acting on one target proxy point per thread
struct m2l_no_poll {
    __device__ __forceinline__ void operator()() const {}
};
template <int N1, typename Poll>
__device__ __forceinline__ void m2l_source(const double2 *__restrict__ Ms, const double *__restrict__ xs, double g2, double xt, double yt,
                                           double zt, double &ex, double &ey, double &ez, double &bx, double &by, double &bz, Poll poll)
{
    const double ztr = zt - xs[2 * M2L_XI_STRIDE + M2L_XI_STRIDE - 1];  // target z relative to the source box centre
    double gz2[N1];
#pragma unroll
    for (int c = 0; c < N1; ++c) {
        const double dz = ztr - xs[2 * M2L_XI_STRIDE + c];
        gz2[c] = (g2 * dz) * dz;
    }
    double S0 = 0, S1 = 0, S2 = 0;  // sum over this source of m_k (c_{nu3} w)
    for (int a2 = 0; a2 < N1; ++a2) {
        poll();  // (helper warp: refill a released stage; nothing for the other warps)
        const double dx = xt - xs[a2];
        const double dx2 = fma(dx, dx, FMM_TINY_D);  // (keeps D > 0 should two proxy points coincide: see inv_r3)
#pragma unroll 1
        for (int b2 = 0; b2 < N1; ++b2) {
            const double2 *row = Ms + 2 * ((a2 * N1 + b2) * N1);
            const double dy = yt - xs[M2L_XI_STRIDE + b2];
            const double s2 = fma(dy, dy, dx2);
            double A0 = 0, A1 = 0, A2 = 0, A3 = 0;
#pragma unroll
            for (int c2 = 0; c2 < N1; ++c2) {
                const double2 m01 = row[2 * c2], m23 = row[2 * c2 + 1];
                const double w = inv_r3(s2 + gz2[c2]);
                A0 = fma(m01.x, w, A0);
                A1 = fma(m01.y, w, A1);
                A2 = fma(m23.x, w, A2);
                A3 = fma(m23.y, w, A3);
                if (c2 == 0 || c2 == N1 - 1 || 2 * c2 != N1 - 1) {  // c_k = 0 at the middle point of an even order
                    const double u = (c2 == 0) ? w : (c2 == N1 - 1) ? -w : w * m2l_cheb_c[N1][c2];
                    S0 = fma(m01.x, u, S0);
                    S1 = fma(m01.y, u, S1);
                    S2 = fma(m23.x, u, S2);
                }
            }
            // sum m_k w dz = ztr sum m_k w - h_z sum m_k c w:  E_z += Z0,  B_x += Z2,  B_y -= Z1
            ex = fma(A0, dx, ex);
            ey = fma(A0, dy, ey);
            ez = fma(A0, ztr, ez);
            bx = fma(-A3, dy, fma(A2, ztr, bx));
            by = fma(A3, dx, fma(-A1, ztr, by));
            bz = fma(A1, dy, fma(-A2, dx, bz));
        }
    }
    const double hz = xs[2 * M2L_XI_STRIDE + M2L_XI_STRIDE - 2];
    ez = fma(-hz, S0, ez);
    bx = fma(-hz, S2, bx);
    by = fma(hz, S1, by);
}

template <int N1, bool SPLIT>
__global__ void __launch_bounds__(m2l_cfg<N1>::BLOCK, m2l_cfg<N1>::MINB) m2l_kernel(double g2, const int32_t *__restrict__ order,
                                                                                  const int32_t *__restrict__ off, const int32_t *__restrict__ src,
                                                                                  const double *__restrict__ xi, const double *__restrict__ M, double *__restrict__ L,
                                                                                  int K, double *__restrict__ Lpart, size_t lstride)
{
    constexpr int P = m2l_cfg<N1>::P;
    constexpr int THREADS = m2l_cfg<N1>::THREADS;   // threads that own target proxy points
    constexpr int WARPS = THREADS / 32;
    constexpr bool HELP = m2l_cfg<N1>::HELP;
    constexpr int CWARPS = m2l_cfg<N1>::CWARPS;
    constexpr int CTHREADS = 32 * CWARPS;
    constexpr int S = m2l_cfg<N1>::STAGES;
    constexpr uint32_t TILE_BYTES = 32u * P;
    constexpr uint32_t STAGE_BYTES = TILE_BYTES + M2L_XI_BYTES;
    extern __shared__ __align__(128) unsigned char m2l_smem_raw[];
    uint64_t *full = reinterpret_cast<uint64_t *>(m2l_smem_raw + S * STAGE_BYTES);
    uint64_t *empty = full + S;
    double *hacc = reinterpret_cast<double *>(m2l_smem_raw + S * STAGE_BYTES + 2 * S * sizeof(uint64_t));  // [THREADS][6], HELP only
    // block (t, kc): chunk kc of the K contiguous chunks of target t's row (K > 1 only for small trees, to fill the GPU);
    // chunk 0 writes L, chunk kc > 0 the partial buffer kc - 1, added to L in chunk order by m2l_combine
    const int t = SPLIT ? order[blockIdx.x / K] : order[blockIdx.x], kc = SPLIT ? blockIdx.x % K : 0;
    const int r0 = off[t], rl = off[t + 1] - r0;
    const int e0 = SPLIT ? r0 + (int)(((int64_t)rl * kc) / K) : r0, e1 = SPLIT ? r0 + (int)(((int64_t)rl * (kc + 1)) / K) : r0 + rl;
    double *Lt = ((!SPLIT || kc == 0) ? L : Lpart + (size_t)(kc - 1) * lstride) + 6 * (size_t)P * t;
    if (e0 == e1) {  // no far-field sources: the local expansion starts at zero (L2L adds into it)
        for (int k = threadIdx.x; k < 6 * P; k += m2l_cfg<N1>::BLOCK) Lt[k] = 0.0;
        return;
    }
    if (threadIdx.x == 0) {
        for (int k = 0; k < S; ++k) {
            mbar_init(&full[k], 1);
            mbar_init(&empty[k], CWARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const int ne = e1 - e0;
    const int total = m2l_cfg<N1>::BATCHES * ne;  // loads in the order they are consumed
    if (!HELP && threadIdx.x >= CTHREADS) {  // producer warp: one lane keeps the stages filled, then the warp retires
        if (threadIdx.x == CTHREADS)
            for (int q = 0; q < total; ++q) {
                const int st = q % S;
                if (q >= S) mbar_wait(&empty[st], (uint32_t)((q / S - 1) & 1));  // all consumer warps left that stage
                const int sn = src[e0 + q % ne];
                unsigned char *dst = m2l_smem_raw + (size_t)st * STAGE_BYTES;
                mbar_expect_tx(&full[st], STAGE_BYTES);
                bulk_g2s(dst, M + 4 * (size_t)P * sn, TILE_BYTES, &full[st]);
                bulk_g2s(dst + TILE_BYTES, xi + (size_t)sn * 3 * M2L_XI_STRIDE, M2L_XI_BYTES, &full[st]);
            }
        return;
    }
    const double *xt3 = xi + (size_t)t * 3 * M2L_XI_STRIDE;
    const int wi = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // release of a stage: order this thread's generic-proxy reads before the next bulk copy into it (async proxy);
    // without the fence a warp occasionally saw part of the NEXT source's tile (cross-proxy write-after-read hazard)
    auto release = [&](int st) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[st]);
    };
    auto target_point = [&](int mu, double &xt, double &yt, double &zt) {  // z = centre + relative part (mid + half c_k)
        const bool live = mu < P;
        const int a = live ? mu / (N1 * N1) : 0, b = live ? (mu / N1) % N1 : 0, c3 = live ? mu % N1 : 0;
        xt = xt3[a];
        yt = xt3[M2L_XI_STRIDE + b];
        zt = __dadd_rn(xt3[2 * M2L_XI_STRIDE + M2L_XI_STRIDE - 1], xt3[2 * M2L_XI_STRIDE + c3]);
    };
    if (HELP && wi == WARPS) {
        // helper warp: for source e it works for target group e mod CWARPS (sums kept in hacc), and its lane 0 keeps the
        // ring filled: it polls the `empty` barriers between slices of its own work and only blocks when the next
        // source it needs itself has not been requested yet
        for (int k = lane; k < 6 * THREADS; k += 32) hacc[k] = 0.0;
        int q = 0;  // loads issued so far (lane 0)
        auto issue = [&]() {
            const int st = q % S;
            const int sn = src[e0 + q];
            unsigned char *dst = m2l_smem_raw + (size_t)st * STAGE_BYTES;
            mbar_expect_tx(&full[st], STAGE_BYTES);
            bulk_g2s(dst, M + 4 * (size_t)P * sn, TILE_BYTES, &full[st]);
            bulk_g2s(dst + TILE_BYTES, xi + (size_t)sn * 3 * M2L_XI_STRIDE, M2L_XI_BYTES, &full[st]);
            ++q;
        };
        auto poll = [&]() {
            if (lane == 0 && q < ne && (q < S || mbar_test(&empty[q % S], (uint32_t)((q / S - 1) & 1)))) issue();
        };
        if (lane == 0)
            while (q < ne && q < S) issue();
        __syncwarp();
        for (int e = 0; e < ne; ++e) {
            const int st = e % S, g = e % CWARPS;
            if (lane == 0)
                while (q <= e) {  // source e itself must be on its way before anybody can wait for it
                    if (q >= S) mbar_wait(&empty[q % S], (uint32_t)((q / S - 1) & 1));
                    issue();
                }
            __syncwarp();
            mbar_wait(&full[st], (uint32_t)((e / S) & 1));  // (also when idle: see the note at the other consumer loop)
            if (g < WARPS) {
                double xt, yt, zt, ex = 0, ey = 0, ez = 0, bx = 0, by = 0, bz = 0;
                target_point(g * 32 + lane, xt, yt, zt);
                m2l_source<N1>(reinterpret_cast<const double2 *>(m2l_smem_raw + (size_t)st * STAGE_BYTES),
                               reinterpret_cast<const double *>(m2l_smem_raw + (size_t)st * STAGE_BYTES + TILE_BYTES), g2, xt, yt, zt, ex,
                               ey, ez, bx, by, bz, poll);
                double *h = hacc + 6 * (g * 32 + lane);
                h[0] += ex; h[1] += ey; h[2] += ez; h[3] += bx; h[4] += by; h[5] += bz;
            }
            release(st);
            poll();
        }
        asm volatile("bar.sync 1, %0;" ::"n"(CTHREADS) : "memory");  // hacc complete (consumer warps only)
        return;
    }
    int i = 0;  // consumed loads so far
    for (int mu0 = 0; mu0 < P; mu0 += THREADS) {
        const int mu = mu0 + threadIdx.x;
        double xt, yt, zt, ex = 0, ey = 0, ez = 0, bx = 0, by = 0, bz = 0;
        target_point(mu, xt, yt, zt);
        for (int e = 0; e < ne; ++e, ++i) {
            const int st = i % S;
            // every warp waits for the stage even when it skips the source: arrivals on `empty` are anonymous, and an
            // early second arrival would complete the PREVIOUS phase while a slower warp is still reading the stage
            mbar_wait(&full[st], (uint32_t)((i / S) & 1));
            if (!(HELP && (e % CWARPS) == wi)) {  // (with a helper: the helper takes this group's source e)
                m2l_source<N1>(reinterpret_cast<const double2 *>(m2l_smem_raw + (size_t)st * STAGE_BYTES),
                               reinterpret_cast<const double *>(m2l_smem_raw + (size_t)st * STAGE_BYTES + TILE_BYTES), g2, xt, yt, zt, ex,
                               ey, ez, bx, by, bz, m2l_no_poll());
            }
            release(st);
        }
        if (HELP) {  // own sums + the helper's, in this fixed order
            asm volatile("bar.sync 1, %0;" ::"n"(CTHREADS) : "memory");
            const double *h = hacc + 6 * threadIdx.x;
            ex += h[0]; ey += h[1]; ez += h[2]; bx += h[3]; by += h[4]; bz += h[5];
        }
        if (mu < P) {
            double *o = Lt + 6 * (size_t)mu;
            o[0] = ex; o[1] = ey; o[2] = ez; o[3] = bx; o[4] = by; o[5] = bz;
        }
    }
}

// L += partial buffers of the row chunks 1 .. K-1, in chunk order
__global__ void m2l_combine(size_t count, int K, size_t lstride, const double *__restrict__ Lpart, double *__restrict__ L)
{
    size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= count) return;
    double v = L[k];
    for (int kc = 1; kc < K; ++kc) v += Lpart[(size_t)(kc - 1) * lstride + k];
    L[k] = v;
}

template <int N1>
static int launch_m2l(fmm_plan *p)
{
    fmm_ctx *c = &p->ctx;
    const size_t smem = m2l_cfg<N1>::STAGES * ((size_t)32 * m2l_cfg<N1>::P + M2L_XI_BYTES) + 2 * m2l_cfg<N1>::STAGES * sizeof(uint64_t) +
                        (m2l_cfg<N1>::HELP ? sizeof(double) * 6 * m2l_cfg<N1>::THREADS : 0);
    if (smem > 48 * 1024)
    {
        FMM_CUDA(c, cudaFuncSetAttribute((const void *)m2l_kernel<N1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        FMM_CUDA(c, cudaFuncSetAttribute((const void *)m2l_kernel<N1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    }
    // the default carveout leaves room for one block only; ask for enough shared memory for every resident block
    FMM_CUDA(c, cudaFuncSetAttribute((const void *)m2l_kernel<N1, false>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    FMM_CUDA(c, cudaFuncSetAttribute((const void *)m2l_kernel<N1, true>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    const int K = p->m2l_split;
    const size_t lstride = 6 * (size_t)m2l_cfg<N1>::P * (size_t)(p->nodes + 2);
    if (K > 1)
        m2l_kernel<N1, true><<<(unsigned)(p->nodes * K), m2l_cfg<N1>::BLOCK, smem, c->stream>>>(p->gamma_bar * p->gamma_bar, p->m2l_order, p->m2l_off,
                                                                                               p->m2l_src, p->node_xi, p->M, p->L, K, p->Lpart, lstride);
    else
        m2l_kernel<N1, false><<<(unsigned)p->nodes, m2l_cfg<N1>::BLOCK, smem, c->stream>>>(p->gamma_bar * p->gamma_bar, p->m2l_order, p->m2l_off,
                                                                                          p->m2l_src, p->node_xi, p->M, p->L, K, p->Lpart, lstride);
    FMM_LAUNCH_CHECK(c, "m2l_kernel");
    if (K > 1) {
        const size_t count = 6 * (size_t)m2l_cfg<N1>::P * (size_t)(p->nodes + 1);
        m2l_combine<<<(unsigned)((count + 255) / 256), 256, 0, c->stream>>>(count, K, lstride, p->Lpart, p->L);
        FMM_LAUNCH_CHECK(c, "m2l_combine");
    }
    return FMM_OK;
}

// ---------------------------------------------------------------------------------------
// Treecode variant (FMM_METHOD_TREECODE): particle-cluster interaction.  One block per target leaf, NT target
// particles per thread as in P2P; the "source particles" of a cluster are its (n+1)^3 proxy points with the moments
// M as weights (eq. (2.5) with the target side not interpolated; mean-gamma kernel of eq. (3.2)).  The sums go to
// partial buffer `slot` of near_, which L2P adds to the P2P partials in a fixed order.
// ---------------------------------------------------------------------------------------
template <int NT>
__global__ void __launch_bounds__(256) pc_kernel(int N, int n1, double gb, const int32_t *__restrict__ order, const int32_t *__restrict__ off,
                                                 const int32_t *__restrict__ src, const int32_t *__restrict__ node_lo,
                                                 const int32_t *__restrict__ node_hi, const double *__restrict__ tx,
                                                 const double *__restrict__ ty, const double *__restrict__ tz,
                                                 const double *__restrict__ xi, const double *__restrict__ M, int slot, int leaves,
                                                 double *__restrict__ near_)
{
    __shared__ double2 tile[4 * PAIR_TILE];
    const int t = order[blockIdx.x];
    if (t < leaves) return;  // only leaves are targets
    const int tlo = node_lo[t], thi = node_hi[t];
    const int e0 = off[t], e1 = off[t + 1];
    const int P = n1 * n1 * n1;
    for (int i0 = tlo; i0 < thi; i0 += NT * blockDim.x) {
        double xt[NT], yt[NT], zt[NT], ex[NT], ey[NT], ez[NT], bx[NT], by[NT], bz[NT];
#pragma unroll
        for (int k = 0; k < NT; ++k) {
            int i = i0 + k * blockDim.x + threadIdx.x;
            bool live = i < thi;
            xt[k] = live ? tx[i] : 0.0; yt[k] = live ? ty[i] : 0.0; zt[k] = live ? tz[i] : 0.0;
            ex[k] = ey[k] = ez[k] = bx[k] = by[k] = bz[k] = 0.0;
        }
        for (int e = e0; e < e1; ++e) {
            const int s = src[e];
            const double *xs = xi + (size_t)s * 3 * M2L_XI_STRIDE;
            const double z0 = xs[2 * M2L_XI_STRIDE + M2L_XI_STRIDE - 1];
            const double2 *Ms = reinterpret_cast<const double2 *>(M + 4 * (size_t)P * s);
            for (int j0 = 0; j0 < P; j0 += PAIR_TILE) {
                const int count = min(PAIR_TILE, P - j0);
                __syncthreads();
                for (int j = threadIdx.x; j < count; j += blockDim.x) {  // proxy nu = (a n1 + b) n1 + c as a source particle
                    const int nu = j0 + j, a = nu / (n1 * n1), b = (nu / n1) % n1, c = nu % n1;
                    const double2 m01 = Ms[2 * nu], m23 = Ms[2 * nu + 1];
                    tile[4 * j + 0] = make_double2(xs[a], xs[M2L_XI_STRIDE + b]);
                    tile[4 * j + 1] = make_double2(__dadd_rn(z0, xs[2 * M2L_XI_STRIDE + c]), m01.x);
                    tile[4 * j + 2] = make_double2(m01.y, m23.x);
                    tile[4 * j + 3] = make_double2(m23.y, 0.0);
                }
                __syncthreads();
                tile_interact<NT, false>(tile, count, xt, yt, zt, gb, ex, ey, ez, bx, by, bz);
            }
        }
#pragma unroll
        for (int k = 0; k < NT; ++k) {
            int i = i0 + k * blockDim.x + threadIdx.x;
            if (i < thi) {
                double *o = near_ + (size_t)slot * 6 * (size_t)N + i;
                o[0] = ex[k];
                o[(size_t)N] = ey[k];
                o[2 * (size_t)N] = ez[k];
                o[3 * (size_t)N] = bx[k];
                o[4 * (size_t)N] = by[k];
                o[5 * (size_t)N] = bz[k];
            }
        }
    }
}

static int m2l_upload_cheb(fmm_ctx *c)
{
    static std::atomic<int> done_on[64];  // __constant__ memory is per device
    int dev = 0;
    FMM_CUDA(c, cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return FMM_EINVAL;
    std::atomic<int> &done = done_on[dev];
    if (done.load(std::memory_order_acquire)) return FMM_OK;
    double tab[FMM_MAX_ORDER + 2][M2L_XI_STRIDE];
    memset(tab, 0, sizeof(tab));
    for (int n1 = 2; n1 <= FMM_MAX_ORDER + 1; ++n1) {
        const int n = n1 - 1;
        for (int k = 0; k <= n; ++k) tab[n1][k] = sin(FMM_PI * (double)(n - 2 * k) / (double)(2 * n));  // I-1
        tab[n1][0] = 1.0;
        tab[n1][n] = -1.0;
    }
    FMM_CUDA(c, cudaMemcpyToSymbol(m2l_cheb_c, tab, sizeof(tab)));  // identical bytes from every caller
    done.store(1, std::memory_order_release);
    return FMM_OK;
}

// proxy points of every node (m2l_proxy_points): part of a2, called by the build after the boxes
int pairs_proxy_points(fmm_plan *p)
{
    fmm_ctx *c = &p->ctx;
    FMM_TRY(m2l_upload_cheb(c));
    cheb13 ch;
    memset(&ch, 0, sizeof(ch));
    for (int k = 0; k <= p->n; ++k) ch.c[k] = sin(FMM_PI * (double)(p->n - 2 * k) / (double)(2 * p->n));  // I-1
    ch.c[0] = 1.0;
    ch.c[p->n] = -1.0;
    int count = (int)(p->nodes + 1) * 3 * M2L_XI_STRIDE;
    m2l_proxy_points<<<(count + 255) / 256, 256, 0, c->stream>>>((int)p->nodes, p->n1, ch, p->bbox, p->node_xi);
    FMM_LAUNCH_CHECK(c, "m2l_proxy_points");
    return FMM_OK;
}

int pairs_m2l(fmm_plan *p)
{
    switch (p->n1) {
        case 2: return launch_m2l<2>(p);
        case 3: return launch_m2l<3>(p);
        case 4: return launch_m2l<4>(p);
        case 5: return launch_m2l<5>(p);
        case 6: return launch_m2l<6>(p);
        case 7: return launch_m2l<7>(p);
        case 8: return launch_m2l<8>(p);
        case 9: return launch_m2l<9>(p);
        case 10: return launch_m2l<10>(p);
        case 11: return launch_m2l<11>(p);
        case 12: return launch_m2l<12>(p);
        case 13: return launch_m2l<13>(p);
    }
    return FMM_EINVAL;
}

int pairs_pc(fmm_plan *p)  // treecode: particle-cluster sums into partial buffer p2p_split
{
    fmm_ctx *c = &p->ctx;
    int maxleaf = p->maxleaf;
    int nt, threads, K;
    p2p_shape(p->leaves, maxleaf, p->p2p_pairs, p->p2p_max_row, &nt, &threads, &K);
#define PC_LAUNCH(NT)                                                                                                            \
    pc_kernel<NT><<<(unsigned)p->nodes, threads, 0, c->stream>>>((int)p->N, p->n1, p->gamma_bar, p->m2l_order, p->m2l_off, p->m2l_src, \
                                                                 p->node_lo, p->node_hi, p->tx, p->ty, p->tz, p->node_xi, p->M,  \
                                                                 p->p2p_split, (int)p->leaves, p->near_)
    switch (nt) {
        case 1: PC_LAUNCH(1); break;
        case 2: PC_LAUNCH(2); break;
        case 3: PC_LAUNCH(3); break;
        default: PC_LAUNCH(4); break;
    }
#undef PC_LAUNCH
    FMM_LAUNCH_CHECK(c, "pc_kernel");
    return FMM_OK;
}

// ---------------------------------------------------------------------------------------
// a11 for callers that cannot allocate (fmm_direct_noalloc, include/fmm.h): the same three kernels as the target-subset
// route of pairs_direct -- source weights, one-sided direct sums per (target block, source slice), fixed-order reduction --
// with their scratch (4 N weights + 6 n_targets partial sums per source slice) in ONE file-scope device array instead of
// the caller's allocator.  Every GPU that loads the library holds these 8 MiB until the process exits.
//   * No cudaMalloc / cudaFree / stream-ordered allocation anywhere on this route; kernel launches only.
//   * In host code `g_noalloc_scratch` is a host-side stand-in, not a device address: the kernels get the pointer that
//     cudaGetSymbolAddress returned for the CURRENT device (looked up once per device, kept).
//   * Every call uses the same array and finds the last call's contents in it.  Nothing has to start at zero: the weights of
//     all N sources and the partial sums of every (slice, target) the reduction reads are written by this call before they
//     are read, so there is nothing to clear.  For the same reason two calls that overlap on the GPU (different streams, or
//     different host threads) race on the array: one call at a time per device.
// ---------------------------------------------------------------------------------------
#include <mutex>

#define NOALLOC_SCRATCH_DOUBLES ((size_t)1 << 20)                  // 8 MiB
#define NOALLOC_WEIGHT_DOUBLES (4 * (size_t)FMM_NOALLOC_MAX_N)      // w0..w3 at a stride of FMM_NOALLOC_MAX_N (256-B aligned planes)
static __device__ __align__(256) double g_noalloc_scratch[NOALLOC_SCRATCH_DOUBLES];
static_assert(NOALLOC_WEIGHT_DOUBLES + 6 * (size_t)FMM_NOALLOC_MAX_N <= NOALLOC_SCRATCH_DOUBLES, "scratch too small for one source slice");

static int noalloc_scratch_of_current_device(fmm_ctx *c, double **out)
{
    static std::mutex mu;
    static double *addr[64] = {};
    int dev = -1;
    FMM_CUDA(c, cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return ctx_cuda_fail(c, cudaErrorInvalidDevice, "fmm_direct_noalloc: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        double *p = NULL;
        FMM_CUDA(c, cudaGetSymbolAddress((void **)&p, g_noalloc_scratch));  // the array's address on the current device
        if (!p) return ctx_cuda_fail(c, cudaErrorInvalidSymbol, "fmm_direct_noalloc: cudaGetSymbolAddress returned NULL");
        addr[dev] = p;
    }
    *out = addr[dev];
    return FMM_OK;
}

int pairs_direct_noalloc(fmm_ctx *c, const fmm_particles_t *in, bool sm, double gamma_bar, int raw, int64_t nt, const int64_t *tidx,
                         double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz)
{
    const int64_t N = in->N;
    if (N > FMM_NOALLOC_MAX_N || nt > FMM_NOALLOC_MAX_N) return FMM_EINVAL;  // (the entry point has said why)
    double *scratch = NULL;
    FMM_TRY(noalloc_scratch_of_current_device(c, &scratch));
    double *w0 = scratch, *w1 = w0 + FMM_NOALLOC_MAX_N, *w2 = w1 + FMM_NOALLOC_MAX_N, *w3 = w2 + FMM_NOALLOC_MAX_N;
    double *part = scratch + NOALLOC_WEIGHT_DOUBLES;
    double cE = 1.0, cB = 1.0;
    if (!raw) {
        cE = 1.0 / (4.0 * FMM_PI * FMM_EPS0);
        cB = 1.0 / (4.0 * FMM_PI * FMM_EPS0 * FMM_C0);
    }
    source_weights_kernel<<<(unsigned)((N + 255) / 256), 256, 0, c->stream>>>(N, in->px, in->py, in->pz, in->q, in->q_scalar, w0, w1, w2, w3);
    FMM_LAUNCH_CHECK(c, "source_weights_kernel");
    // source slices as in pairs_direct, but no more than the partial sums the array has room for
    const int64_t tblocks = (nt + DIRECT_TARGETS - 1) / DIRECT_TARGETS;
    int64_t splits = (8 * 4 * FMM_SM_COUNT + tblocks - 1) / tblocks;
    const int64_t tiles = (N + PAIR_TILE - 1) / PAIR_TILE;
    const int64_t room = (int64_t)((NOALLOC_SCRATCH_DOUBLES - NOALLOC_WEIGHT_DOUBLES) / (6 * (size_t)nt));
    if (splits > tiles) splits = tiles;
    if (splits > room) splits = room;
    if (splits < 1) splits = 1;
    const int64_t chunk = ((tiles + splits - 1) / splits) * PAIR_TILE;
    splits = (N + chunk - 1) / chunk;
    const dim3 grid((unsigned)tblocks, (unsigned)splits);
    if (sm)
        direct_kernel<true><<<grid, DIRECT_THREADS, 0, c->stream>>>(N, gamma_bar, nt, tidx, chunk, in->x, in->y, in->z, w0, w1, w2, w3, in->px, in->py, in->pz, part);
    else
        direct_kernel<false><<<grid, DIRECT_THREADS, 0, c->stream>>>(N, gamma_bar, nt, tidx, chunk, in->x, in->y, in->z, w0, w1, w2, w3, NULL, NULL, NULL, part);
    FMM_LAUNCH_CHECK(c, "direct_kernel");
    direct_reduce<<<(unsigned)((nt + 255) / 256), 256, 0, c->stream>>>(nt, (int)splits, part, cE, cB, Ex, Ey, Ez, Bx, By, Bz);
    FMM_LAUNCH_CHECK(c, "direct_reduce");
    return FMM_OK;
}
