// fbp_stack.cuh -- a volume from a stack of reconstructed slices by linear interpolation along the
// stack axis ("interpolation of a stack of 2D images").
//
// Output slice m of n_out sits at z_m = m (n_in - 1)/(n_out - 1); k = floor(z_m) clamped to n_in - 2,
// t = z_m - k (fp64, per CTA); out[m][p] = (1 - t) in[k][p] + t in[k+1][p] in the working precision.
// The paper names no interpolation rule; linear is the reading taken (R4).
// Elementwise and HBM-bound: every output element is written once by one thread (deterministic),
// with 16-byte loads and stores when the slices are 16-byte aligned.  Grid (chunks of a slice, n_out).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

namespace fbp {

constexpr int kStackThreads = 256;
constexpr int kStackVecPerThread = 4;   // 16-byte vectors per thread

template <typename T>
__global__ void __launch_bounds__(kStackThreads)
interpolate_stack_kernel(const T* __restrict__ in, int n_in, T* __restrict__ out, int n_out, long long n_pix)
{
    const int m = blockIdx.y;
    const double z = n_out > 1 ? (double)m * (double)(n_in - 1) / (double)(n_out - 1) : 0.0;
    long long k = (long long)floor(z);
    if (k > n_in - 2) k = n_in - 2;
    if (k < 0) k = 0;
    const T t = n_in > 1 ? (T)(z - (double)k) : T(0);
    const T omt = T(1) - t;
    const T* a = in + (size_t)k * n_pix;
    const T* b = in + (size_t)(n_in > 1 ? k + 1 : k) * n_pix;
    T* o = out + (size_t)m * n_pix;

    constexpr int V = 16 / (int)sizeof(T);
    const bool vec = (((reinterpret_cast<uintptr_t>(a) | reinterpret_cast<uintptr_t>(b) | reinterpret_cast<uintptr_t>(o)) & 15u) == 0);
    const long long nvec = vec ? n_pix / V : 0;
    const long long base = (long long)blockIdx.x * kStackThreads * kStackVecPerThread + threadIdx.x;
    uint4 va[kStackVecPerThread], vb[kStackVecPerThread];
#pragma unroll
    for (int u = 0; u < kStackVecPerThread; ++u) {
        const long long i = base + (long long)u * kStackThreads;
        if (i < nvec) {
            va[u] = __ldg(reinterpret_cast<const uint4*>(a) + i);
            vb[u] = __ldg(reinterpret_cast<const uint4*>(b) + i);
        }
    }
#pragma unroll
    for (int u = 0; u < kStackVecPerThread; ++u) {
        const long long i = base + (long long)u * kStackThreads;
        if (i < nvec) {
            uint4 r;
            const T* pa = reinterpret_cast<const T*>(&va[u]);
            const T* pb = reinterpret_cast<const T*>(&vb[u]);
            T* pr = reinterpret_cast<T*>(&r);
#pragma unroll
            for (int e = 0; e < V; ++e) pr[e] = fma(t, pb[e], omt * pa[e]);
            reinterpret_cast<uint4*>(o)[i] = r;
        }
    }
    // tail (or everything, when a slice is not 16-byte aligned): the first CTA row walks it
    if (blockIdx.x == 0)
        for (long long p = nvec * V + threadIdx.x; p < n_pix; p += kStackThreads) o[p] = fma(t, b[p], omt * a[p]);
}

}  // namespace fbp
