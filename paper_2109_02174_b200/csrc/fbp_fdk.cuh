// fbp_fdk.cuh -- cone-beam reconstruction by the algorithm of Feldkamp, Davis and Kress (the
// continuation the paper announces, ref [20] at PAPER.md:259).  Textbook FDK (Kak & Slaney ch. 3.6,
// ref [8] PAPER.md:247) in the conventions of the 2-D path; the readings are listed in include/fbp.h
// (fbp_fdk_reconstruct) and DESIGN.md:
//   1. pre-weight  p'[m][i][j] = p[m][i][j] * sad / sqrt(sad^2 + a_j^2 + b_i^2)                (fdk_weight_kernel)
//   2. row filter  Q[m][i][:] = (1/d_a) h * p'[m][i][:]  -- the plan's row filter, on K * n_rows rows (fbp_fft.cuh)
//   3. voxel r = (x, y, z):  t = r.e_a, s = r.e_s, U = sad + s,  e_a = (cos, sin, 0), e_s = (-sin, cos, 0);
//      f(r) = (pi/K) sum_m (sad/U)^2 bilinear(Q[m]; sad t/(U d_a) + c_a, sad z/(U d_b) + c_b)   (fdk_backproject_kernel)
// Back-projection is a gather with one owner thread per voxel column and a fixed angle order: deterministic, no
// atomics (the paper's parallel versions were not).  For a fixed (x, y, angle) the detector column
// and the weight do not depend on z and the detector row is affine in z: a thread owns ZT voxels of one (x, y)
// column and pays the per-angle work once for all of them.
#pragma once
#include <cuda_runtime.h>

#include "fbp_backproject.cuh"  // Magic<T>: floor by adding 1.5 * 2^23 | 2^52

namespace fbp {

struct FdkParams {
    int n_angles, n_a, n_b;      // K, detector columns, detector rows
    int image_n, n_z;
    double sad_a;                // sad / d_a: source-axis distance in detector-column units
    double rz;                   // voxel_z / d_b
    double c_n, c_z, c_a, c_b;   // (N-1)/2, (n_z-1)/2, (n_a-1)/2, (n_b-1)/2
    double scale;                // pi / K
};

// p, out: [K][n_b][n_a].  One thread per element.
template <typename T>
__global__ void __launch_bounds__(256)
fdk_weight_kernel(const T* __restrict__ p, T* __restrict__ out, long long n, int n_a, int n_b, double d_a, double d_b, double sad)
{
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    const int j = (int)(e % n_a), i = (int)((e / n_a) % n_b);
    const double a = ((double)j - 0.5 * (double)(n_a - 1)) * d_a, b = ((double)i - 0.5 * (double)(n_b - 1)) * d_b;
    out[e] = (T)((double)p[e] * (sad * rsqrt(sad * sad + a * a + b * b)));
}

constexpr int kFdkZT = 8;        // voxels per thread along z

// Q: [K][n_b][n_a] filtered, weighted projections.  cs2: [K] (cos, sin) * pix/d_a (fp64).  vol: [n_z][N][N].
// Grid (ceil(N/32), ceil(N/4), ceil(n_z/ZT)), block (32, 4): thread = one (x, y) and ZT consecutive z.
template <typename T>
__global__ void __launch_bounds__(128)
fdk_backproject_kernel(const T* __restrict__ Q, T* __restrict__ vol, const double2* __restrict__ cs2, FdkParams prm)
{
    const int c = blockIdx.x * 32 + threadIdx.x, r = blockIdx.y * 4 + threadIdx.y, k0 = blockIdx.z * kFdkZT;
    const int N = prm.image_n, n_a = prm.n_a, n_b = prm.n_b;
    if (c >= N || r >= N) return;
    const double xi = (double)c - prm.c_n, yi = (double)r - prm.c_n;
    const T M = Magic<T>::m();
    T zk[kFdkZT], acc[kFdkZT];
#pragma unroll
    for (int z = 0; z < kFdkZT; ++z) { zk[z] = (T)(((double)(k0 + z) - prm.c_z) * prm.rz); acc[z] = T(0); }
    const size_t plane = (size_t)n_b * n_a;
    for (int m = 0; m < prm.n_angles; ++m) {
        const double2 cs = cs2[m];
        // per (x, y, angle), in fp64 (shared by the ZT voxels): column coordinate and magnification
        const double t = xi * cs.x + yi * cs.y, s = yi * cs.x - xi * cs.y;
        const double mag = prm.sad_a / (prm.sad_a + s);
        const double ua = mag * t + prm.c_a;
        const double fa = floor(ua);
        const int ja = (int)fa;
        const T wa = (T)(ua - fa), w2 = (T)(mag * mag), mg = (T)mag, cb = (T)prm.c_b;
        const T* Qm = Q + (size_t)m * plane;
        const bool in0 = ja >= 0 && ja < n_a, in1 = ja + 1 >= 0 && ja + 1 < n_a;
        if (!in0 && !in1) continue;
#pragma unroll
        for (int z = 0; z < kFdkZT; ++z) {
            const T ub = fma(mg, zk[z], cb);
            const T tb = ub + M;
            const int ib = (int)(Magic<T>::bits(tb) - Magic<T>::kBits) - (tb - M > ub ? 1 : 0);   // floor(ub)
            const T wb = ub - (T)ib;
            const T* row0 = Qm + (size_t)ib * n_a + ja;
            const bool r0 = ib >= 0 && ib < n_b, r1 = ib + 1 >= 0 && ib + 1 < n_b;
            const T q00 = (r0 && in0) ? __ldg(row0) : T(0), q01 = (r0 && in1) ? __ldg(row0 + 1) : T(0);
            const T q10 = (r1 && in0) ? __ldg(row0 + n_a) : T(0), q11 = (r1 && in1) ? __ldg(row0 + n_a + 1) : T(0);
            const T v0 = fma(wa, q01 - q00, q00), v1 = fma(wa, q11 - q10, q10);
            acc[z] = fma(w2, fma(wb, v1 - v0, v0), acc[z]);
        }
    }
    const T sc = (T)prm.scale;
#pragma unroll
    for (int z = 0; z < kFdkZT; ++z)
        if (k0 + z < prm.n_z) vol[((size_t)(k0 + z) * N + r) * N + c] = acc[z] * sc;
}

}  // namespace fbp
