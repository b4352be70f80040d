// probe_fp64.cu -- libfmm_probe.so: micro-benchmarks of the FP64 pipe of the device, used by bench.py for the
// roofline denominator (MEASURED_PEAKS.json has no FP64 entry) and by `bench.py --probe-fp64` for the operand-pattern
// table in profiles/ (why an accumulate-type DFMA costs more than two issue cycles).  Measurement tooling only: it is
// not part of the boundary (include/fmm.h) and libfmm_b200.so does not contain it.
//
//   int fmm_probe_fp64(int pattern, double *inst_per_s, double *ms, void *cuda_stream)
//     pattern 0  DFMA v = fma(v, a, b), a and b kernel parameters        (one register source)
//             1  DFMA v_k = fma(x_k, y_k, v_k), all registers distinct    (three register sources)
//             2  DFMA v_k = fma(x_0, y_k, v_k), x_0 shared by neighbours  (three sources, one repeated: operand reuse)
//             3  DMUL / DADD alternating, two distinct register sources
//             4  MUFU.RSQ64H (rsqrt.approx.ftz.f64)
//             5  the one-sided near-field evaluation (25 FP64 instructions, kernels_pairs.cu tile_interact)
//             6  the mutual near-field evaluation of a pair (34 FP64 instructions)
//     inst_per_s = thread-level instructions (patterns 5, 6: kernel evaluations) per second, best of 3 launches.
#include <cuda_runtime.h>
#include <stdint.h>

#define PROBE_BLOCKS (148 * 8)
#define PROBE_THREADS 256
#define PROBE_ITERS 4000

__device__ __forceinline__ double probe_inv_r3(double D)
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

template <int PATTERN>
__global__ void __launch_bounds__(PROBE_THREADS) probe_kernel(int iters, double a, double b, const double *__restrict__ in, double *__restrict__ out)
{
    double v[8], x[8], y[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        v[k] = in[(threadIdx.x + k) & 255];
        x[k] = in[(threadIdx.x + 8 + 3 * k) & 255];
        y[k] = in[(threadIdx.x + 40 + 5 * k) & 255];
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (PATTERN == 0) {
#pragma unroll
                for (int k = 0; k < 8; ++k) v[k] = fma(v[k], a, b);
            } else if (PATTERN == 1) {
#pragma unroll
                for (int k = 0; k < 8; ++k) v[k] = fma(x[k], y[k], v[k]);
            } else if (PATTERN == 2) {
#pragma unroll
                for (int k = 0; k < 8; ++k) v[k] = fma(x[0], y[k], v[k]);
            } else if (PATTERN == 3) {
#pragma unroll
                for (int k = 0; k < 8; ++k) v[k] = (k & 1) ? v[k] * x[k] : v[k] + y[k];
            } else if (PATTERN == 4) {
#pragma unroll
                for (int k = 0; k < 8; ++k) asm volatile("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(v[k]) : "d"(v[k]));
            }
        }
        if (PATTERN == 5 || PATTERN == 6) {
            // four targets (x, y, v as positions), one source per iteration; sums in v / y like the real kernels
            double gx[4], gy[4], gz[4];
            const double xs = a * (double)it, ys = b, zs = a, m0 = x[4], m1 = x[5], m2 = x[6], m3 = x[7];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const double dx = x[k] - xs, dy = y[k] - ys, dz = in[k] - zs;
                double D = fma(dx, dx, 1e-200);
                D = fma(dy, dy, D);
                const double sz = a * dz;
                D = fma(sz, sz, D);
                const double w = probe_inv_r3(D);
                gx[k] = w * dx; gy[k] = w * dy; gz[k] = w * dz;
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                v[k] = fma(m0, gx[k], v[k]); v[4 + k] = fma(m0, gy[k], v[4 + k]); y[4 + k] = fma(m0, gz[k], y[4 + k]);
                v[k] = fma(m2, gz[k], v[k]); v[k] = fma(-m3, gy[k], v[k]);
                v[4 + k] = fma(m3, gx[k], v[4 + k]); v[4 + k] = fma(-m1, gz[k], v[4 + k]);
                y[4 + k] = fma(m1, gy[k], y[4 + k]); y[4 + k] = fma(-m2, gx[k], y[4 + k]);
            }
            if (PATTERN == 6) {
                double r0 = 0, r1 = 0, r2 = 0;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    r0 = fma(y[k], gx[k], r0); r1 = fma(y[k], gy[k], r1); r2 = fma(y[k], gz[k], r2);
                    r0 = fma(x[k], gz[k], r0); r0 = fma(-v[4 + k], gy[k], r0);
                    r1 = fma(v[4 + k], gx[k], r1); r1 = fma(-x[k], gz[k], r1);
                    r2 = fma(x[k], gy[k], r2); r2 = fma(-y[k], gx[k], r2);
                }
                x[4] += r0 * 1e-300; x[5] += r1 * 1e-300; x[6] += r2 * 1e-300;
            }
        }
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += v[k] + x[k] + y[k];
    if (s == 123.456) out[0] = s;  // keeps the chains alive without a store in practice
}

template <int PATTERN>
static int run_pattern(double *inst_per_s, double *ms_out, cudaStream_t st)
{
    double *buf = NULL;
    if (cudaMalloc(&buf, sizeof(double) * 512) != cudaSuccess) return -2;
    double h[256];
    for (int k = 0; k < 256; ++k) h[k] = 0.5 + 1e-3 * k;
    cudaMemcpyAsync(buf, h, sizeof(h), cudaMemcpyHostToDevice, st);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int iters = (PATTERN >= 5) ? PROBE_ITERS * 4 : PROBE_ITERS;
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, st);
        probe_kernel<PATTERN><<<PROBE_BLOCKS, PROBE_THREADS, 0, st>>>(iters, 0.999999, 1e-9, buf, buf + 256);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) return -3;
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(buf);
    const double per_thread = (PATTERN >= 5) ? 4.0 * iters : 32.0 * iters;  // patterns 5, 6: evaluations (6: four pairs = eight evaluations)
    double count = per_thread * (double)PROBE_THREADS * (double)PROBE_BLOCKS;
    if (PATTERN == 6) count *= 2.0;
    *inst_per_s = count / ((double)best * 1e-3);
    if (ms_out) *ms_out = best;
    return cudaGetLastError() == cudaSuccess ? 0 : -3;
}

extern "C" int fmm_probe_fp64(int pattern, double *inst_per_s, double *ms, void *cuda_stream)
{
    if (!inst_per_s) return -1;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    switch (pattern) {
        case 0: return run_pattern<0>(inst_per_s, ms, st);
        case 1: return run_pattern<1>(inst_per_s, ms, st);
        case 2: return run_pattern<2>(inst_per_s, ms, st);
        case 3: return run_pattern<3>(inst_per_s, ms, st);
        case 4: return run_pattern<4>(inst_per_s, ms, st);
        case 5: return run_pattern<5>(inst_per_s, ms, st);
        case 6: return run_pattern<6>(inst_per_s, ms, st);
    }
    return -1;
}
