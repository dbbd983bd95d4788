// fbp_metrics.cuh -- PSNR (eq. 3) and global-statistics SSIM (eq. 4)
// of an image pair as deterministic device-side reductions.
//
//   MSE = (1/n) sum (x-y)^2,  PSNR = 20 log10(MAX / sqrt(MSE))   (+inf when MSE = 0)
//   SSIM = (2 mu_x mu_y + C1)(2 s_xy + C2) / ((mu_x^2 + mu_y^2 + C1)(s_x^2 + s_y^2 + C2)),
//   mu = mean, s^2 / s_xy = population (co)variances over the whole image (the paper gives no window).
//
// Two passes (two launches), like the definition: pass 0 sums x, y, (x-y)^2 and its last CTA turns them into the
// means; pass 1 sums the centred products (x-mu_x)^2, (y-mu_y)^2, (x-mu_x)(y-mu_y).  All sums are
// fp64 whatever the image dtype.  Determinism: a fixed grid, every thread walks a fixed strided
// index set, lanes are combined with a fixed shuffle tree, warps and CTAs in index order -- no
// atomics, so repeated runs give the same bits (the paper's parallel versions did not).
// HBM-bound: 2 passes x 2 images x n x sizeof(T) bytes.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

namespace fbp {

constexpr int kMetricThreads = 256;

// Run by the first warp of the last CTA: CTA partials are added in index order by lane-strided sums + the shuffle tree.
// PASS 0: mid[0..2] = (mu_x, mu_y, MSE).   PASS 1: out[0..7] = MSE, PSNR, SSIM, mu_x, mu_y, s_x^2, s_y^2, s_xy.
template <int PASS>
__device__ __forceinline__ void metrics_finish(const double* partial, int n_partial, long long n, double* mid,
                                               double max_val, double c1, double c2, double* out)
{
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
    for (int i = threadIdx.x; i < n_partial; i += 32) {
        s0 += __ldcg(partial + 3 * i + 0); s1 += __ldcg(partial + 3 * i + 1); s2 += __ldcg(partial + 3 * i + 2);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        s0 += __shfl_down_sync(0xffffffffu, s0, o);
        s1 += __shfl_down_sync(0xffffffffu, s1, o);
        s2 += __shfl_down_sync(0xffffffffu, s2, o);
    }
    if (threadIdx.x != 0) return;
    const double inv_n = 1.0 / (double)n;
    if (PASS == 0) {
        mid[0] = s0 * inv_n; mid[1] = s1 * inv_n; mid[2] = s2 * inv_n;
    } else {
        const double mx = mid[0], my = mid[1], mse = mid[2];
        const double vx = s0 * inv_n, vy = s1 * inv_n, cxy = s2 * inv_n;
        out[0] = mse;
        out[1] = mse > 0.0 ? 20.0 * log10(max_val / sqrt(mse)) : __longlong_as_double(0x7ff0000000000000ll);
        out[2] = ((2.0 * mx * my + c1) * (2.0 * cxy + c2)) / ((mx * mx + my * my + c1) * (vx + vy + c2));
        out[3] = mx; out[4] = my; out[5] = vx; out[6] = vy; out[7] = cxy;
    }
}

// partial: [gridDim.x][3] doubles.  PASS 0: (sum x, sum y, sum (x-y)^2);  PASS 1: centred, means from `mid`.
template <typename T, int PASS>
__global__ void __launch_bounds__(kMetricThreads)
metrics_partial_kernel(const T* __restrict__ x, const T* __restrict__ y, long long n,
                       double* __restrict__ mid, double* __restrict__ partial, unsigned* __restrict__ ticket,
                       double max_val, double c1, double c2, double* __restrict__ out)
{
    double mx = 0.0, my = 0.0;
    if (PASS == 1) { mx = mid[0]; my = mid[1]; }
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
    auto add = [&](double a, double b) {
        if (PASS == 0) {
            const double e = a - b;
            s0 += a; s1 += b; s2 = fma(e, e, s2);
        } else {
            const double u = a - mx, v = b - my;
            s0 = fma(u, u, s0); s1 = fma(v, v, s1); s2 = fma(u, v, s2);
        }
    };
    // 16-byte loads, four in flight per array and thread; the element -> thread map is fixed by (n, grid)
    constexpr int V = 16 / (int)sizeof(T);
    const bool vec = ((reinterpret_cast<uintptr_t>(x) | reinterpret_cast<uintptr_t>(y)) & 15u) == 0;
    const long long nvec = vec ? n / V : 0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const uint4* xv = reinterpret_cast<const uint4*>(x);
    const uint4* yv = reinterpret_cast<const uint4*>(y);
    long long i = t0;
    for (; i + 3 * stride < nvec; i += 4 * stride) {
        uint4 a[4], b[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) { a[u] = __ldg(xv + i + u * stride); b[u] = __ldg(yv + i + u * stride); }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const T* pa = reinterpret_cast<const T*>(&a[u]);
            const T* pb = reinterpret_cast<const T*>(&b[u]);
#pragma unroll
            for (int e = 0; e < V; ++e) add((double)pa[e], (double)pb[e]);
        }
    }
    for (; i < nvec; i += stride) {
        const uint4 a = __ldg(xv + i), b = __ldg(yv + i);
        const T* pa = reinterpret_cast<const T*>(&a);
        const T* pb = reinterpret_cast<const T*>(&b);
#pragma unroll
        for (int e = 0; e < V; ++e) add((double)pa[e], (double)pb[e]);
    }
    for (long long k = nvec * V + t0; k < n; k += stride) add((double)x[k], (double)y[k]);   // tail / unaligned
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        s0 += __shfl_down_sync(0xffffffffu, s0, o);
        s1 += __shfl_down_sync(0xffffffffu, s1, o);
        s2 += __shfl_down_sync(0xffffffffu, s2, o);
    }
    __shared__ double red[3][kMetricThreads / 32];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { red[0][warp] = s0; red[1][warp] = s1; red[2][warp] = s2; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double t0 = 0.0, t1 = 0.0, t2 = 0.0;
        for (int w = 0; w < kMetricThreads / 32; ++w) { t0 += red[0][w]; t1 += red[1][w]; t2 += red[2][w]; }
        partial[3 * blockIdx.x + 0] = t0;
        partial[3 * blockIdx.x + 1] = t1;
        partial[3 * blockIdx.x + 2] = t2;
    }
    // The CTA that draws the last ticket (ordering only, never data) adds the CTA partials in index order --
    // the same order whichever CTA that is -- and finishes the pass: means (pass 0) or the eight outputs (pass 1).
    __shared__ bool s_last;
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned t = atomicAdd(ticket, 1u);
        s_last = (t == gridDim.x - 1);
        if (s_last) *ticket = 0u;                 // re-arm for the next pass / call
    }
    __syncthreads();
    if (!s_last || threadIdx.x >= 32) return;
    __threadfence();
    metrics_finish<PASS>(partial, (int)gridDim.x, n, mid, max_val, c1, c2, out);
}

}  // namespace fbp
