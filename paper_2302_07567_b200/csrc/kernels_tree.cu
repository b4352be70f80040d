// kernels_tree.cu -- steps a0-a2 of the hot path:
//   a0  mean momentum -> gamma_bar, source weights q gamma, q p
//   a1  particle order of the balanced cluster tree: mode KD = Alg 5.1/5.2 in kernels_kd.cu;
//       mode MORTON_MEDIAN = 63-bit Morton order of the stretched coordinates (DESIGN T-3') here
//   a2  tight bounding boxes, stretched radii and centres (Alg 5.6/5.7)
// Everything here is integer / compare / min-max work: HBM- and launch-latency-bound.
#include "fmm_internal.cuh"

// ---------------------------------------------------------------------------------------
// closed-form node ranges (DESIGN T-2): root [0,N); left child gets ceil(size/2)
// ---------------------------------------------------------------------------------------
__global__ void node_ranges_kernel(int N, int kappa, int nodes, int stop_level, int N0, int32_t *__restrict__ node_lo,
                                   int32_t *__restrict__ node_hi)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x + 1;  // heap id
    if (i > nodes) return;
    int level = 31 - __clz(i);
    int lo = 0, hi = N;
    for (int b = level - 1; b >= 0; --b) {
        int mid = fmm_split_mid(lo, hi, level - 1 - b, stop_level, N0);
        if ((i >> b) & 1) lo = mid; else hi = mid;
    }
    node_lo[i] = lo;
    node_hi[i] = hi;
}

// ---------------------------------------------------------------------------------------
// a0: deterministic mean momentum (fixed grid, fixed reduction tree)
// ---------------------------------------------------------------------------------------
#define RED_BLOCKS (2 * FMM_SM_COUNT)
#define RED_THREADS 256

__device__ __forceinline__ double block_sum_256(double v, double *sm /* [8] */)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) sm[warp] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < RED_THREADS / 32; ++w) t += sm[w];
    return t;  // valid in thread 0
}

__global__ void __launch_bounds__(RED_THREADS) momentum_partial(int64_t N, const double *__restrict__ px, const double *__restrict__ py,
                                                                const double *__restrict__ pz, double *__restrict__ partial)
{
    __shared__ double sm[8];
    double sx = 0.0, sy = 0.0, sz = 0.0;
    for (int64_t j = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; j < N; j += (int64_t)RED_BLOCKS * RED_THREADS) {
        sx += px[j];
        sy += py[j];
        sz += pz[j];
    }
    sx = block_sum_256(sx, sm);
    sy = block_sum_256(sy, sm);
    sz = block_sum_256(sz, sm);
    if (threadIdx.x == 0) {
        partial[3 * blockIdx.x + 0] = sx;
        partial[3 * blockIdx.x + 1] = sy;
        partial[3 * blockIdx.x + 2] = sz;
    }
}

__global__ void momentum_final(int64_t N, const double *__restrict__ partial, double *__restrict__ out)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    double sx = 0.0, sy = 0.0, sz = 0.0;
    for (int b = 0; b < RED_BLOCKS; ++b) {
        sx += partial[3 * b + 0];
        sy += partial[3 * b + 1];
        sz += partial[3 * b + 2];
    }
    double mx = sx / (double)N, my = sy / (double)N, mz = sz / (double)N;
    out[0] = sqrt(1.0 + (mx * mx + my * my + mz * mz));  // gamma_bar^2 = 1 + pbar.pbar
}

int tree_gamma_bar(fmm_ctx *c, int64_t N, const double *px, const double *py, const double *pz, double *gamma_bar_out)
{
    double *partial = (double *)ctx_alloc(c, sizeof(double) * (3 * RED_BLOCKS + 1));
    if (!partial) return FMM_ENOMEM;
    momentum_partial<<<RED_BLOCKS, RED_THREADS, 0, c->stream>>>(N, px, py, pz, partial);
    FMM_LAUNCH_CHECK(c, "momentum_partial");
    momentum_final<<<1, 32, 0, c->stream>>>(N, partial, partial + 3 * RED_BLOCKS);
    FMM_LAUNCH_CHECK(c, "momentum_final");
    FMM_CUDA(c, cudaMemcpyAsync(gamma_bar_out, partial + 3 * RED_BLOCKS, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    FMM_CUDA(c, cudaStreamSynchronize(c->stream));
    ctx_free(c, partial);
    return FMM_OK;
}

// ---------------------------------------------------------------------------------------
// a0 for a plan: one pass over the inputs gives the momentum sums (same fixed grid and reduction tree as above), the
// coordinate ranges (Morton keys, sort keys) and the number of non-finite input values (FMM_ENONFINITE); the result
// stays on the device (fmm_hdr).
// ---------------------------------------------------------------------------------------
#define A0_STRIDE 10  // per block: 3 momentum sums, 3 minima, 3 maxima, non-finite count

__global__ void __launch_bounds__(RED_THREADS) a0_scan_partial(int64_t N, const double *__restrict__ x, const double *__restrict__ y,
                                                               const double *__restrict__ z, const double *__restrict__ px,
                                                               const double *__restrict__ py, const double *__restrict__ pz,
                                                               const double *__restrict__ q, double *__restrict__ partial)
{
    __shared__ double sm[8];
    __shared__ double smm[6][8];
    __shared__ int sbad[8];
    double sx = 0.0, sy = 0.0, sz = 0.0;
    double lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    int bad = 0;
    for (int64_t j = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; j < N; j += (int64_t)RED_BLOCKS * RED_THREADS) {
        const double ax = px[j], ay = py[j], az = pz[j], vx = x[j], vy = y[j], vz = z[j];
        sx += ax; sy += ay; sz += az;
        lo[0] = fmin(lo[0], vx); hi[0] = fmax(hi[0], vx);
        lo[1] = fmin(lo[1], vy); hi[1] = fmax(hi[1], vy);
        lo[2] = fmin(lo[2], vz); hi[2] = fmax(hi[2], vz);
        bad += !isfinite(ax) + !isfinite(ay) + !isfinite(az) + !isfinite(vx) + !isfinite(vy) + !isfinite(vz);
        if (q) bad += !isfinite(q[j]);
    }
    sx = block_sum_256(sx, sm);
    sy = block_sum_256(sy, sm);
    sz = block_sum_256(sz, sm);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lo[k] = fmin(lo[k], __shfl_down_sync(0xffffffffu, lo[k], o));
            hi[k] = fmax(hi[k], __shfl_down_sync(0xffffffffu, hi[k], o));
        }
        if (lane == 0) { smm[k][warp] = lo[k]; smm[3 + k][warp] = hi[k]; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) bad += __shfl_down_sync(0xffffffffu, bad, o);
    if (lane == 0) sbad[warp] = bad;
    __syncthreads();
    double *out = partial + (size_t)A0_STRIDE * blockIdx.x;
    if (threadIdx.x == 0) {
        out[0] = sx; out[1] = sy; out[2] = sz;
        int b = 0;
        for (int w = 0; w < 8; ++w) b += sbad[w];
        out[9] = (double)b;
    }
    if (threadIdx.x < 6) {
        double v = smm[threadIdx.x][0];
        for (int w = 1; w < 8; ++w) v = (threadIdx.x < 3) ? fmin(v, smm[threadIdx.x][w]) : fmax(v, smm[threadIdx.x][w]);
        out[3 + threadIdx.x] = v;
    }
}

// one warp: lane l adds the blocks l, l + 32, ... in order, then the lanes are added by a fixed shuffle tree
__global__ void a0_scan_final(int64_t N, double gamma_bar_param, const double *__restrict__ partial, fmm_hdr *__restrict__ hdr)
{
    const int lane = threadIdx.x;
    double s[3] = {0.0, 0.0, 0.0}, lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY}, bad = 0.0;
    for (int b = lane; b < RED_BLOCKS; b += 32) {
        const double *pb = partial + (size_t)A0_STRIDE * b;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            s[k] += pb[k];
            lo[k] = fmin(lo[k], pb[3 + k]);
            hi[k] = fmax(hi[k], pb[6 + k]);
        }
        bad += pb[9];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            s[k] += __shfl_down_sync(0xffffffffu, s[k], o);
            lo[k] = fmin(lo[k], __shfl_down_sync(0xffffffffu, lo[k], o));
            hi[k] = fmax(hi[k], __shfl_down_sync(0xffffffffu, hi[k], o));
        }
        bad += __shfl_down_sync(0xffffffffu, bad, o);
    }
    if (lane == 0) {
        double gb = gamma_bar_param;
        if (!(gb > 0.0)) {
            const double mx = s[0] / (double)N, my = s[1] / (double)N, mz = s[2] / (double)N;
            gb = sqrt(1.0 + (mx * mx + my * my + mz * mz));  // gamma_bar^2 = 1 + pbar.pbar
        }
        hdr->gamma_bar = gb;
        hdr->g2 = __dmul_rn(gb, gb);
#pragma unroll
        for (int k = 0; k < 3; ++k) { hdr->mm[k] = lo[k]; hdr->mm[3 + k] = hi[k]; }
        unsigned int nb = bad > 4.0e9 ? 4000000000u : (unsigned int)bad;
        if (!isfinite(gb)) nb += 1u;
        hdr->nonfinite = nb;
        hdr->kd_fallback = 0;
    }
}

int tree_scan_inputs(fmm_plan *p, const fmm_particles_t *in)
{
    fmm_ctx *c = &p->ctx;
    double *partial = (double *)ctx_alloc(c, sizeof(double) * A0_STRIDE * RED_BLOCKS);
    if (!partial) return FMM_ENOMEM;
    a0_scan_partial<<<RED_BLOCKS, RED_THREADS, 0, c->stream>>>(p->N, in->x, in->y, in->z, in->px, in->py, in->pz, in->q, partial);
    FMM_LAUNCH_CHECK(c, "a0_scan_partial");
    a0_scan_final<<<1, 32, 0, c->stream>>>(p->N, p->gamma_bar_param, partial, p->hdr);
    FMM_LAUNCH_CHECK(c, "a0_scan_final");
    ctx_free(c, partial);
    return FMM_OK;
}

// ---------------------------------------------------------------------------------------
// a1', mode MORTON_MEDIAN (DESIGN T-3')
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ uint64_t spread3(uint64_t v)  // 21 bits -> every third bit
{
    v &= 0x1fffffull;
    v = (v | (v << 32)) & 0x1f00000000ffffull;
    v = (v | (v << 16)) & 0x1f0000ff0000ffull;
    v = (v | (v << 8)) & 0x100f00f00f00f00full;
    v = (v | (v << 4)) & 0x10c30c30c30c30c3ull;
    v = (v | (v << 2)) & 0x1249249249249249ull;
    return v;
}

__global__ void morton_keys(int N, const double *__restrict__ x, const double *__restrict__ y, const double *__restrict__ z,
                            const fmm_hdr *__restrict__ hdr /* min xyz, max xyz of the raw coordinates, gamma_bar */,
                            uint64_t *__restrict__ keys, uint32_t *__restrict__ vals)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double *mm = hdr->mm;
    const double gamma_bar = hdr->gamma_bar;
    // u = s o x; s > 0 so min/max commute with the scaling (every operation rounded separately)
    double s[3] = {1.0, 1.0, gamma_bar};
    double lo[3], L = 0.0;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        lo[k] = __dmul_rn(s[k], mm[k]);
        double ext = __dsub_rn(__dmul_rn(s[k], mm[3 + k]), lo[k]);
        if (k == 0 || ext > L) L = ext;
    }
    double c[3] = {x[i], y[i], z[i]};
    uint64_t q[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        double u = __dmul_rn(s[k], c[k]);
        double f = (L > 0.0) ? floor(__dmul_rn(__ddiv_rn(__dsub_rn(u, lo[k]), L), 2097152.0)) : 0.0;
        if (f > 2097151.0) f = 2097151.0;
        if (f < 0.0) f = 0.0;
        q[k] = (uint64_t)f;
    }
    keys[i] = spread3(q[0]) | (spread3(q[1]) << 1) | (spread3(q[2]) << 2);  // z most significant
    vals[i] = (uint32_t)i;
}

// ---------------------------------------------------------------------------------------
// a1 end: physical permutation into tree order + source weights (a0)
// ---------------------------------------------------------------------------------------
__global__ void permute_particles(int N, const uint32_t *__restrict__ order, const double *__restrict__ x, const double *__restrict__ y,
                                  const double *__restrict__ z, const double *__restrict__ px, const double *__restrict__ py,
                                  const double *__restrict__ pz, const double *__restrict__ q, double q_scalar,
                                  int32_t *__restrict__ perm, double *__restrict__ tx, double *__restrict__ ty, double *__restrict__ tz,
                                  double *__restrict__ w0, double *__restrict__ w1, double *__restrict__ w2, double *__restrict__ w3,
                                  double *__restrict__ pmx, double *__restrict__ pmy, double *__restrict__ pmz)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    uint32_t j = order[k];
    if (perm) perm[k] = (int32_t)j;
    tx[k] = x[j];
    ty[k] = y[j];
    tz[k] = z[j];
    double ax = px[j], ay = py[j], az = pz[j];
    double qj = q ? q[j] : q_scalar;
    double gam = sqrt(1.0 + (ax * ax + ay * ay + az * az));  // gamma_j = sqrt(1 + p.p)
    w0[k] = qj * gam;
    w1[k] = qj * ax;
    w2[k] = qj * ay;
    w3[k] = qj * az;
    if (pmx) {  // FMM_KERNEL_SOURCE_MOMENTUM: the near field needs the plain momenta of the sources
        pmx[k] = ax;
        pmy[k] = ay;
        pmz[k] = az;
    }
}

// Large N (the seven input arrays no longer fit the L2): a random 8-byte read drags a 32-byte sector out of DRAM, 7 x 32 B per
// particle.  The inputs are therefore first packed into 64-byte records with streaming reads and writes, and the permutation
// then reads one record (two sectors) per particle: 2.5 instead of 3.3 ms at N = 2.56e7.
__global__ void pack_particles(int N, const double *__restrict__ x, const double *__restrict__ y, const double *__restrict__ z,
                               const double *__restrict__ px, const double *__restrict__ py, const double *__restrict__ pz,
                               const double *__restrict__ q, double q_scalar, double4 *__restrict__ rec /* [N][2] */)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    rec[2 * (size_t)j] = make_double4(x[j], y[j], z[j], q ? q[j] : q_scalar);
    rec[2 * (size_t)j + 1] = make_double4(px[j], py[j], pz[j], 0.0);
}

__global__ void permute_packed(int N, const uint32_t *__restrict__ order, const double4 *__restrict__ rec, int32_t *__restrict__ perm,
                               double *__restrict__ tx, double *__restrict__ ty, double *__restrict__ tz, double *__restrict__ w0,
                               double *__restrict__ w1, double *__restrict__ w2, double *__restrict__ w3, double *__restrict__ pmx,
                               double *__restrict__ pmy, double *__restrict__ pmz)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const uint32_t j = order[k];
    if (perm) perm[k] = (int32_t)j;
    const double4 a = rec[2 * (size_t)j], b = rec[2 * (size_t)j + 1];
    tx[k] = a.x;
    ty[k] = a.y;
    tz[k] = a.z;
    const double gam = sqrt(1.0 + (b.x * b.x + b.y * b.y + b.z * b.z));  // gamma_j = sqrt(1 + p.p)
    w0[k] = a.w * gam;
    w1[k] = a.w * b.x;
    w2[k] = a.w * b.y;
    w3[k] = a.w * b.z;
    if (pmx) {
        pmx[k] = b.x;
        pmy[k] = b.y;
        pmz[k] = b.z;
    }
}

// the physical permutation, by either route
static int permute_into_tree_order(fmm_plan *p, const fmm_particles_t *in, const uint32_t *order, int32_t *perm_out)
{
    fmm_ctx *c = &p->ctx;
    const int N = (int)p->N, T = 256, gN = (N + T - 1) / T;
    if (p->N >= ((int64_t)1 << 21)) {  // 7 x 8 N bytes >= 117 MB: past the L2
        double4 *rec = (double4 *)ctx_alloc(c, sizeof(double4) * 2 * (size_t)N);
        if (!rec) return FMM_ENOMEM;
        pack_particles<<<gN, T, 0, c->stream>>>(N, in->x, in->y, in->z, in->px, in->py, in->pz, in->q, in->q_scalar, rec);
        FMM_LAUNCH_CHECK(c, "pack_particles");
        permute_packed<<<gN, T, 0, c->stream>>>(N, order, rec, perm_out, p->tx, p->ty, p->tz, p->w0, p->w1, p->w2, p->w3, p->pmx, p->pmy, p->pmz);
        FMM_LAUNCH_CHECK(c, "permute_packed");
        ctx_free(c, rec);
        return FMM_OK;
    }
    permute_particles<<<gN, T, 0, c->stream>>>(N, order, in->x, in->y, in->z, in->px, in->py, in->pz, in->q, in->q_scalar, perm_out, p->tx, p->ty,
                                               p->tz, p->w0, p->w1, p->w2, p->w3, p->pmx, p->pmy, p->pmz);
    FMM_LAUNCH_CHECK(c, "permute_particles");
    return FMM_OK;
}

// ---------------------------------------------------------------------------------------
// a2: bounding boxes
// ---------------------------------------------------------------------------------------
// one warp per leaf: tight min/max over its members (exact, order-free)
__global__ void leaf_bbox(int leaves, const int32_t *__restrict__ node_lo, const int32_t *__restrict__ node_hi,
                          const double *__restrict__ tx, const double *__restrict__ ty, const double *__restrict__ tz,
                          double *__restrict__ bbox)
{
    int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (w >= leaves) return;
    int node = leaves + w;
    int lo = node_lo[node], hi = node_hi[node];
    double a[3] = {INFINITY, INFINITY, INFINITY}, b[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (int k = lo + lane; k < hi; k += 32) {
        double vx = tx[k], vy = ty[k], vz = tz[k];
        a[0] = fmin(a[0], vx); b[0] = fmax(b[0], vx);
        a[1] = fmin(a[1], vy); b[1] = fmax(b[1], vy);
        a[2] = fmin(a[2], vz); b[2] = fmax(b[2], vz);
    }
#pragma unroll
    for (int k = 0; k < 3; ++k)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            a[k] = fmin(a[k], __shfl_xor_sync(0xffffffffu, a[k], o));
            b[k] = fmax(b[k], __shfl_xor_sync(0xffffffffu, b[k], o));
        }
    if (lane == 0) {
        double *bb = bbox + 6 * (int64_t)node;
        bool empty = hi <= lo;  // empty cluster: zeros (it takes part in nothing)
        for (int k = 0; k < 3; ++k) {
            bb[k] = empty ? 0.0 : a[k];
            bb[3 + k] = empty ? 0.0 : b[k];
        }
    }
}

// Parents = union of the non-empty children (an empty cluster has a zero box and takes part in nothing).  One warp takes
// 32 consecutive nodes of level `lc` and forms their ancestors on up to five levels with shuffles (min / max are exact and
// order-free), so the whole upward pass is ceil(kappa / 5) small launches instead of kappa block barriers.
__global__ void __launch_bounds__(256) bbox_up_warp(int lc, int steps, const int32_t *__restrict__ node_lo, const int32_t *__restrict__ node_hi,
                                                    double *__restrict__ bbox)
{
    const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    const int first = 1 << lc, count = 1 << lc;
    const int k = w * 32 + lane;
    if (w * 32 >= count) return;
    const bool live = k < count;
    const int node = first + (live ? k : 0);
    bool empty = !live || node_hi[node] <= node_lo[node];
    double b[6];
#pragma unroll
    for (int q = 0; q < 6; ++q) b[q] = empty ? 0.0 : bbox[6 * (int64_t)node + q];
    for (int s = 1; s <= steps; ++s) {
        const int o = 1 << (s - 1);
        const bool e2 = __shfl_down_sync(0xffffffffu, empty, o);
        double c[6];
#pragma unroll
        for (int q = 0; q < 6; ++q) c[q] = __shfl_down_sync(0xffffffffu, b[q], o);
        if ((lane & ((1 << s) - 1)) == 0) {  // this lane holds the left child, lane + o the right one
#pragma unroll
            for (int q = 0; q < 3; ++q) {
                b[q] = empty ? c[q] : (e2 ? b[q] : fmin(b[q], c[q]));
                b[3 + q] = empty ? c[3 + q] : (e2 ? b[3 + q] : fmax(b[3 + q], c[3 + q]));
            }
            empty = empty && e2;
            if (live) {
                double *bb = bbox + 6 * (int64_t)(node >> s);
#pragma unroll
                for (int q = 0; q < 6; ++q) bb[q] = empty ? 0.0 : b[q];
            }
        }
    }
}

// the stretched squared radius (Alg 5.6) and the box centre (Alg 5.7) of every node, each product
// and sum rounded separately (reading D-2) so that the traversal is bit-reproducible
__global__ void node_geometry(int nodes, const fmm_hdr *__restrict__ hdr, const double *__restrict__ bbox, double *__restrict__ geo)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x + 1;
    if (i > nodes) return;
    const double gamma_bar = hdr->gamma_bar;
    const double *bb = bbox + 6 * (int64_t)i;
    double hx = __dmul_rn(__dsub_rn(bb[3], bb[0]), 0.5), hy = __dmul_rn(__dsub_rn(bb[4], bb[1]), 0.5),
           hz = __dmul_rn(__dsub_rn(bb[5], bb[2]), 0.5);
    double ex = __dmul_rn(1.0, hx), ey = __dmul_rn(1.0, hy), ez = __dmul_rn(gamma_bar, hz);
    double *g = geo + 4 * (int64_t)i;
    g[0] = __dadd_rn(__dadd_rn(__dmul_rn(ex, ex), __dmul_rn(ey, ey)), __dmul_rn(ez, ez));
    g[1] = __dmul_rn(__dadd_rn(bb[0], bb[3]), 0.5);
    g[2] = __dmul_rn(__dadd_rn(bb[1], bb[4]), 0.5);
    g[3] = __dmul_rn(__dadd_rn(bb[2], bb[5]), 0.5);
}

// ---------------------------------------------------------------------------------------
int tree_build(fmm_plan *p, const fmm_particles_t *in)
{
    fmm_ctx *c = &p->ctx;
    cudaStream_t st = c->stream;
    const int N = (int)p->N;
    const int T = 256;
    const int gN = (N + T - 1) / T;

    if (!p->ranges_done) {  // closed-form ranges (T-2): they depend on (N, N0) only
        node_ranges_kernel<<<(unsigned)((p->nodes + T - 1) / T), T, 0, st>>>(N, p->kappa, (int)p->nodes, p->stop_level, p->N0, p->node_lo, p->node_hi);
        FMM_LAUNCH_CHECK(c, "node_ranges_kernel");
        p->ranges_done = 1;
    }

    uint32_t *order = NULL;
    if ((p->flags & FMM_TREE_MASK) == FMM_TREE_KD) {
        FMM_TRY(kd_build_order(p, in, &order));  // kernels_kd.cu
    } else {
        uint64_t *keys = (uint64_t *)ctx_alloc(c, sizeof(uint64_t) * N);
        uint64_t *tkeys = (uint64_t *)ctx_alloc(c, sizeof(uint64_t) * N);
        uint32_t *tvals = (uint32_t *)ctx_alloc(c, sizeof(uint32_t) * N);
        order = (uint32_t *)ctx_alloc(c, sizeof(uint32_t) * (size_t)N);
        if (!keys || !tkeys || !tvals || !order) return FMM_ENOMEM;
        morton_keys<<<gN, T, 0, st>>>(N, in->x, in->y, in->z, p->hdr, keys, order);
        FMM_LAUNCH_CHECK(c, "morton_keys");
        FMM_TRY(sort_pairs_u64(c, keys, order, tkeys, tvals, N, 0, 64));
    }
    FMM_TRY(permute_into_tree_order(p, in, order, p->perm));
    return tree_boxes(p);  // (the scratch goes back with the arena of the build)
}

// a2 on the particles as they sit in tree order
int tree_boxes(fmm_plan *p)
{
    fmm_ctx *c = &p->ctx;
    const int T = 256;
    leaf_bbox<<<(unsigned)((p->leaves * 32 + T - 1) / T), T, 0, c->stream>>>((int)p->leaves, p->node_lo, p->node_hi, p->tx, p->ty, p->tz, p->bbox);
    FMM_LAUNCH_CHECK(c, "leaf_bbox");
    for (int lc = p->kappa; lc > 0; lc -= 5) {
        const int steps = lc < 5 ? lc : 5;
        const int64_t threads = (int64_t)1 << lc;
        bbox_up_warp<<<(unsigned)((threads + T - 1) / T), T, 0, c->stream>>>(lc, steps, p->node_lo, p->node_hi, p->bbox);
        FMM_LAUNCH_CHECK(c, "bbox_up_warp");
    }
    node_geometry<<<(unsigned)((p->nodes + T - 1) / T), T, 0, c->stream>>>((int)p->nodes, p->hdr, p->bbox, p->node_geo);
    FMM_LAUNCH_CHECK(c, "node_geometry");
    FMM_TRY(interp_transfer_tables(p));  // M2M / L2L matrices of the new boxes (kernels_interp.cu)
    FMM_TRY(pairs_proxy_points(p));      // proxy points of the new boxes for M2L and the treecode (kernels_pairs.cu)
    return FMM_OK;
}

// Refit: the particle order of the last build is kept; the new positions / momenta are
// gathered through it and only the bounding boxes are recomputed.  Node ranges (T-2) depend on (N, N0) alone.
int tree_refit(fmm_plan *p, const fmm_particles_t *in)
{
    FMM_TRY(permute_into_tree_order(p, in, reinterpret_cast<const uint32_t *>(p->perm), NULL));
    return tree_boxes(p);
}
