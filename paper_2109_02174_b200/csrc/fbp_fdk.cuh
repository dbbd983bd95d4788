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
// column and pays the per-angle work once for all of them.  Between 2 and 3 the filtered projections are re-packed
// into zero-bordered 2 x 2 quads (fdk_quads_kernel) so that a bilinear sample is one aligned load without bounds tests.
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


// The back-projector's operands: 2 x 2 neighbourhoods ("quads") of the filtered projections with zero borders,
//   P4[m][i'][j'] = ( Q~[i][j], Q~[i][j+1], Q~[i+1][j], Q~[i+1][j+1] ),  i = i'-1, j = j'-1,
//   i' in [0, n_b+2), j' in [0, n_a+2),  Q~ = 0 outside the detector,
// so that a bilinear sample at (ua, ub) clamped to [-1, n_a] x [-1, n_b] is ONE aligned 16-byte load (fp32; two in
// fp64) at one address, with no bounds test: whatever lies outside the detector reads as zero.  Four times the bytes
// of the plain projections; per angle they are read by every CTA at about the same time and stay in L2.
template <typename T> struct alignas(4 * sizeof(T)) FdkQuad { T q00, q01, q10, q11; };

// One thread per quad.
template <typename T>
__global__ void __launch_bounds__(256)
fdk_quads_kernel(const T* __restrict__ Q, FdkQuad<T>* __restrict__ P4, long long n, int n_a, int n_b)
{
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    const int pa = n_a + 2, pb = n_b + 2;
    const int jp = (int)(e % pa), ip = (int)((e / pa) % pb);
    const long long m = e / ((long long)pa * pb);
    const int i = ip - 1, j = jp - 1;
    auto at = [&](int ii, int jj) -> T {
        return (ii >= 0 && ii < n_b && jj >= 0 && jj < n_a) ? Q[((size_t)m * n_b + ii) * n_a + jj] : T(0);
    };
    FdkQuad<T> v;
    v.q00 = at(i, j); v.q01 = at(i, j + 1); v.q10 = at(i + 1, j); v.q11 = at(i + 1, j + 1);
    P4[e] = v;
}

__device__ __forceinline__ FdkQuad<float> ldg_quad(const FdkQuad<float>* p)
{
    const float4 v = __ldg(reinterpret_cast<const float4*>(p));
    return FdkQuad<float>{v.x, v.y, v.z, v.w};
}
__device__ __forceinline__ FdkQuad<double> ldg_quad(const FdkQuad<double>* p)
{
    const double2 a = __ldg(reinterpret_cast<const double2*>(p)), b = __ldg(reinterpret_cast<const double2*>(p) + 1);
    return FdkQuad<double>{a.x, a.y, b.x, b.y};
}

// P4: the quads above.  cs2: [K] (cos, sin) * pix/d_a (fp64).  vol: [n_z][N][N].
// Grid (ceil(N/32), ceil(N/4), ceil(n_z/ZT)), block (32, 4): thread = one (x, y) and ZT consecutive z (ZT = 16, or 8 for
// thin volumes).  Per (x, y, angle), in fp64 and shared by the ZT voxels: column coordinate ua (clamped, floor by the round-down add of
// 1.5 * 2^52), magnification, weight.  Per voxel, in the working precision: ub = mag z + c_b clamped to [-1, n_b], floor
// and fraction by the same trick (no F2I / I2F: those run at a quarter of the issue rate), one quad load, three lerps.
template <typename T, int ZT>
__global__ void __launch_bounds__(128)
fdk_backproject_kernel(const FdkQuad<T>* __restrict__ P4, T* __restrict__ vol, const double2* __restrict__ cs2, FdkParams prm)
{
    const int c = blockIdx.x * 32 + threadIdx.x, r = blockIdx.y * 4 + threadIdx.y, k0 = blockIdx.z * ZT;
    const int N = prm.image_n, n_a = prm.n_a, n_b = prm.n_b;
    if (c >= N || r >= N) return;
    const double xi = (double)c - prm.c_n, yi = (double)r - prm.c_n;
    const T M = Magic<T>::m();
    const double M64 = Magic<double>::m();
    T acc[ZT];
#pragma unroll
    for (int z = 0; z < ZT; ++z) acc[z] = T(0);
    const T zk0 = (T)(((double)k0 - prm.c_z) * prm.rz), rz = (T)prm.rz;     // z of voxel k0 + z: zk0 + z rz (detector rows)
    const int pa = n_a + 2;
    const unsigned plane = (unsigned)(n_b + 2) * (unsigned)pa;      // quads per angle (< 2^31: checked by the caller)
    const T ub_hi = (T)n_b, cb = (T)prm.c_b;
    const double ua_hi = (double)n_a;
    for (int m = 0; m < prm.n_angles; ++m) {
        const double2 cs = cs2[m];
        const double t = xi * cs.x + yi * cs.y, s = yi * cs.x - xi * cs.y;
        const double mag = prm.sad_a / (prm.sad_a + s);
        const double ua = fmin(fmax(mag * t + prm.c_a, -1.0), ua_hi);
        const double ta = __dadd_rd(ua, M64);
        const int ja = __double2loint(ta);                           // floor(ua) in [-1, n_a]
        const T wa = (T)(ua - (ta - M64)), w2 = (T)(mag * mag), mg = (T)mag;
        // quads of column ja (buffer rows: detector row i is row i + 1, so the row index floor(ub) + 1 is in [0, n_b + 1])
        const FdkQuad<T>* col = P4 + (size_t)m * plane + (unsigned)(ja + 1);
        const T ub0 = fma(mg, zk0, cb), du = mg * rz;
#pragma unroll
        for (int z = 0; z < ZT; ++z) {
            const T ub = fmin(fmax(fma((T)z, du, ub0), T(-1)), ub_hi);
            const T tb = add_rd(ub, M);
            const unsigned ibp = Magic<T>::bits(tb) - (Magic<T>::kBits - 1u);   // floor(ub) + 1
            const T wb = ub - (tb - M);
            const FdkQuad<T> q = ldg_quad(col + (size_t)(ibp * (unsigned)pa));
            const T v0 = fma(wa, q.q01 - q.q00, q.q00), v1 = fma(wa, q.q11 - q.q10, q.q10);
            acc[z] = fma(w2, fma(wb, v1 - v0, v0), acc[z]);
        }
    }
    const T sc = (T)prm.scale;
#pragma unroll
    for (int z = 0; z < ZT; ++z)
        if (k0 + z < prm.n_z) vol[((size_t)(k0 + z) * N + r) * N + c] = acc[z] * sc;
}

}  // namespace fbp
