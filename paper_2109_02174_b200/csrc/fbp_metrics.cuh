// fbp_metrics.cuh -- PSNR (eq. 3) and global-statistics SSIM (eq. 4)
// of an image pair as a deterministic device-side reduction.
//
//   MSE = (1/n) sum (x-y)^2,  PSNR = 20 log10(MAX / sqrt(MSE))   (+inf when MSE = 0)
//   SSIM = (2 mu_x mu_y + C1)(2 s_xy + C2) / ((mu_x^2 + mu_y^2 + C1)(s_x^2 + s_y^2 + C2)),
//   mu = mean, s^2 / s_xy = population (co)variances over the whole image (the paper gives no window).
//
// ONE pass over the two arrays (the kernel is HBM-bound: 2 n sizeof(T) bytes): shifted moments.  With the
// shifts a = x[0], b = y[0] (any value near the data does) every thread accumulates, in fp64,
//   sum u, sum v, sum u^2, sum v^2, sum u v, sum (x-y)^2,      u = x - a, v = y - b,
// and the last CTA turns them into  mu_x = a + S_u/n,  s_x^2 = (S_uu - S_u^2/n)/n,  s_xy = (S_uv - S_u S_v/n)/n.
// The shift keeps S_u^2/n small against S_uu (no catastrophic cancellation when the mean is large against the
// spread), so the result agrees with the two-pass definition to a few ulp of fp64; x = y gives u = v term by
// term, hence MSE = 0 and SSIM = 1 exactly.  Determinism: a fixed grid, every thread walks a fixed strided index
// set, lanes are combined with a fixed shuffle tree, warps and CTAs in index order -- no atomics on data (one
// ticket per CTA orders the finish), so repeated runs give the same bits (the paper's parallel versions did not,
// PAPER.md:218).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

namespace fbp {

constexpr int kMetricThreads = 256;
constexpr int kMetricSums = 6;
constexpr int kMetricU = 4;      // 16-byte vectors per array, thread and pipeline stage

// partial: [gridDim.x][6] doubles.  ticket: zero-initialised, self re-arming.  out: 8 doubles.
template <typename T>
__global__ void __launch_bounds__(kMetricThreads)
metrics_kernel(const T* __restrict__ x, const T* __restrict__ y, long long n, double* __restrict__ partial,
               unsigned* __restrict__ ticket, double max_val, double c1, double c2, double* __restrict__ out)
{
    const double sa = (double)__ldg(x), sb = (double)__ldg(y);
    double s[kMetricSums] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    auto add = [&](double a, double b) {
        const double u = a - sa, v = b - sb, e = a - b;
        s[0] += u; s[1] += v;
        s[2] = fma(u, u, s[2]); s[3] = fma(v, v, s[3]); s[4] = fma(u, v, s[4]); s[5] = fma(e, e, s[5]);
    };
    // 16-byte loads; the element -> thread map is fixed by (n, grid)
    constexpr int V = 16 / (int)sizeof(T);
    const bool vec = ((reinterpret_cast<uintptr_t>(x) | reinterpret_cast<uintptr_t>(y)) & 15u) == 0;
    const long long nvec = vec ? n / V : 0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const uint4* xv = reinterpret_cast<const uint4*>(x);
    const uint4* yv = reinterpret_cast<const uint4*>(y);
    // software pipeline: the loads of the next group of kMetricU vectors per array are in flight while the current
    // group is accumulated (a warp that computes after waiting for its loads leaves HBM idle a third of the time);
    // the accumulation order of a thread -- ascending index -- does not depend on the grouping
    constexpr int U = kMetricU;
    uint4 a[U], b[U];
    long long i = t0;
    auto load = [&](long long at) {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const long long k = at + u * stride;
            if (k < nvec) { a[u] = __ldg(xv + k); b[u] = __ldg(yv + k); }
        }
    };
    if (i < nvec) load(i);
    while (i < nvec) {
        uint4 ca[U], cb[U];
#pragma unroll
        for (int u = 0; u < U; ++u) { ca[u] = a[u]; cb[u] = b[u]; }
        const long long nxt = i + U * stride;
        if (nxt < nvec) load(nxt);
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (i + u * stride < nvec) {
                const T* pa = reinterpret_cast<const T*>(&ca[u]);
                const T* pb = reinterpret_cast<const T*>(&cb[u]);
#pragma unroll
                for (int e = 0; e < V; ++e) add((double)pa[e], (double)pb[e]);
            }
        }
        i = nxt;
    }
    for (long long k = nvec * V + t0; k < n; k += stride) add((double)x[k], (double)y[k]);   // tail / unaligned
#pragma unroll
    for (int q = 0; q < kMetricSums; ++q)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s[q] += __shfl_down_sync(0xffffffffu, s[q], o);
    __shared__ double red[kMetricSums][kMetricThreads / 32];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0)
        for (int q = 0; q < kMetricSums; ++q) red[q][warp] = s[q];
    __syncthreads();
    if (threadIdx.x < kMetricSums) {
        double t = 0.0;
        for (int w = 0; w < kMetricThreads / 32; ++w) t += red[threadIdx.x][w];
        partial[(size_t)kMetricSums * blockIdx.x + threadIdx.x] = t;
    }
    // The CTA that draws the last ticket (ordering only, never data) adds the CTA partials in index order --
    // the same order whichever CTA that is -- and writes the eight outputs.
    __shared__ bool s_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned t = atomicAdd(ticket, 1u);
        s_last = (t == gridDim.x - 1);
        if (s_last) *ticket = 0u;                 // re-arm for the next call
    }
    __syncthreads();
    if (!s_last || threadIdx.x >= 32) return;
    __threadfence();
    double f[kMetricSums] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    for (int c = threadIdx.x; c < (int)gridDim.x; c += 32)
#pragma unroll
        for (int q = 0; q < kMetricSums; ++q) f[q] += __ldcg(partial + (size_t)kMetricSums * c + q);
#pragma unroll
    for (int q = 0; q < kMetricSums; ++q)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) f[q] += __shfl_down_sync(0xffffffffu, f[q], o);
    if (threadIdx.x != 0) return;
    const double inv_n = 1.0 / (double)n;
    const double du = f[0] * inv_n, dv = f[1] * inv_n;                 // mean offsets from the shifts
    const double mx = sa + du, my = sb + dv, mse = f[5] * inv_n;
    const double vx = fma(-f[0], du, f[2]) * inv_n, vy = fma(-f[1], dv, f[3]) * inv_n, cxy = fma(-f[0], dv, f[4]) * inv_n;
    out[0] = mse;
    out[1] = mse > 0.0 ? 20.0 * log10(max_val / sqrt(mse)) : __longlong_as_double(0x7ff0000000000000ll);
    out[2] = ((2.0 * mx * my + c1) * (2.0 * cxy + c2)) / ((mx * mx + my * my + c1) * (vx + vy + c2));
    out[3] = mx; out[4] = my; out[5] = vx; out[6] = vy; out[7] = cxy;
}

}  // namespace fbp
