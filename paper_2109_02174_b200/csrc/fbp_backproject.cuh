// fbp_backproject.cuh -- pixel-driven gather back-projection for sm_100a (eq. 2).
//
// f[r][c] = (pi/K) sum_i lerp(Q~_i, u_i),  u_i = (x cos_i + y sin_i)/d + (D-1)/2.
//
// A CTA owns a tile of 32 x (WY*R) pixels and a contiguous range of angles (angle split s of
// S).  Angles are processed in chunks: for each angle of the chunk the CTA stages the
// segment of Q_i the tile projects onto into shared memory as (mid, slope) pairs
//   mid[e] = (Q~[j]+Q~[j+1])/2,  slope[e] = Q~[j+1]-Q~[j],  j = j0 + e,
// plus a per-angle record (cos, sin, b) with b = u(tile origin) - j0 - 1/2 computed in fp64
// (tile-local coordinates keep fp32 detector coordinates below 64, ulp <= 3.8e-6).
// A thread owns R pixels of one column (register accumulators).  Per update:
//   u' = b + lx cos + ly sin;  t = u' + M (M = 1.5*2^23 or 1.5*2^52) rounds to nearest;
//   e = bits(t) - bits(M);  w' = u' - (t - M) in [-1/2, 1/2];  acc += mid[e] + w' slope[e]
// which equals (1-w) Q~[j] + w Q~[j+1] (the interpolant is continuous, so a tie in the
// rounding picks either neighbour interval with the same value).
// One owner per pixel, angles in ascending order, no atomics => bit-identical runs.
// With S > 1 the S partial images are written to scratch and summed in fixed order s=0..S-1
// by reduce_kernel.
#pragma once
#include <cuda_runtime.h>

namespace fbp {

struct BpParams {
    int n_angles, n_det, image_n;
    int tiles_x, tiles_y;
    int n_splits;        // S
    int chunk;           // angles staged per chunk (A)
    int seg_len;         // L entries per angle
    double c_n, c_d;     // (N-1)/2, (D-1)/2
    double scale;        // pi / K
};

template <typename T> struct Magic;
template <> struct Magic<float> {
    __device__ static float m() { return 12582912.0f; }  // 1.5 * 2^23
    __device__ static int idx(float t) { return __float_as_int(t) - 0x4B400000; }
};
template <> struct Magic<double> {
    __device__ static double m() { return 6755399441055744.0; }  // 1.5 * 2^52
    __device__ static int idx(double t) { return __double2loint(t); }
};

template <typename T> struct alignas(2 * sizeof(T)) Pair { T mid, slope; };
template <typename T> struct alignas(4 * sizeof(T)) AngleRec { T c, s, b, pad; };

// cs2: [K] pairs (cos*pix/d, sin*pix/d) in fp64.  out: image (S == 1, scaled) or partial
// buffer [S][batch][N][N] (S > 1, unscaled).
template <typename T, int R, int WY>
__global__ void __launch_bounds__(32 * WY)
backproject_kernel(const T* __restrict__ Q, T* __restrict__ out, const double2* __restrict__ cs2,
                   BpParams prm, int batch)
{
    constexpr int TH = WY * R;
    constexpr int NT = 32 * WY;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    AngleRec<T>* rec = reinterpret_cast<AngleRec<T>*>(smem_raw);
    Pair<T>* seg = reinterpret_cast<Pair<T>*>(rec + prm.chunk);
    int* j0s = reinterpret_cast<int*>(seg + (size_t)prm.chunk * prm.seg_len);

    const int tid = threadIdx.x, lane = tid & 31, wy = tid >> 5;
    const int tile = blockIdx.x;
    const int ty = tile / prm.tiles_x, tx = tile - ty * prm.tiles_x;
    const int split = blockIdx.y, b = blockIdx.z;
    const int K = prm.n_angles, D = prm.n_det, N = prm.image_n, L = prm.seg_len;

    const int per = (K + prm.n_splits - 1) / prm.n_splits;
    const int a_begin = split * per;
    const int a_end = min(K, a_begin + per);

    const double x0 = (double)(tx * 32) - prm.c_n;
    const double y0 = (double)(ty * TH) - prm.c_n;
    const T* Qb = Q + (size_t)b * K * D;

    T acc[R];
#pragma unroll
    for (int r = 0; r < R; ++r) acc[r] = T(0);
    const T lx = (T)lane, ly = (T)(wy * R);

    for (int a0 = a_begin; a0 < a_end; a0 += prm.chunk) {
        const int na = min(prm.chunk, a_end - a0);
        __syncthreads();  // previous chunk fully consumed
        for (int a = tid; a < na; a += NT) {
            const double2 cs = cs2[a0 + a];
            const double ub = x0 * cs.x + y0 * cs.y + prm.c_d;
            const double umin = ub + fmin(0.0, 31.0 * cs.x) + fmin(0.0, (double)(TH - 1) * cs.y);
            const double fl = floor(umin) - 1.0;
            AngleRec<T> r;
            if (fabs(fl) < 1.0e9) {
                j0s[a] = (int)fl;
                r.c = (T)cs.x; r.s = (T)cs.y; r.b = (T)(ub - fl - 0.5);
            } else {
                // absurd geometry: the tile projects > 1e9 bins off the detector.  Stage a
                // segment that is entirely outside [0, D) (all zeros) and pin every pixel to
                // entry 1 of it, so no index can leave the staged range.
                j0s[a] = -(1 << 30);
                r.c = T(0); r.s = T(0); r.b = T(1);
            }
            r.pad = T(0);
            rec[a] = r;
        }
        __syncthreads();
        for (int idx = tid; idx < na * L; idx += NT) {
            const int a = idx / L, e = idx - a * L;
            const long long j = (long long)j0s[a] + e;
            const T* row = Qb + (size_t)(a0 + a) * D;
            const T q0 = (j >= 0 && j < D) ? row[j] : T(0);
            const T q1 = (j + 1 >= 0 && j + 1 < D) ? row[j + 1] : T(0);
            Pair<T> pr;
            pr.mid = T(0.5) * (q0 + q1);
            pr.slope = q1 - q0;
            seg[(size_t)a * L + e] = pr;
        }
        __syncthreads();

        const T M = Magic<T>::m();
#pragma unroll 2
        for (int a = 0; a < na; ++a) {
            const AngleRec<T> rc = rec[a];
            const Pair<T>* sg = seg + (size_t)a * L;
            const T u0 = fma(lx, rc.c, fma(ly, rc.s, rc.b));
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const T u = fma((T)r, rc.s, u0);
                const T t = u + M;
                const T w = u - (t - M);
                const int e = Magic<T>::idx(t);  // in [0, L-1] by construction of j0 and L
                const Pair<T> pr = sg[e];
                acc[r] += fma(w, pr.slope, pr.mid);
            }
        }
    }

    const int c = tx * 32 + lane;
    if (c < N) {
        const size_t img = (size_t)N * N;
        T* o = out + ((size_t)split * batch + b) * img;
        const T sc = (prm.n_splits == 1) ? (T)prm.scale : T(1);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int row = ty * TH + wy * R + r;
            if (row < N) o[(size_t)row * N + c] = acc[r] * sc;
        }
    }
}

// image[p] = scale * (part[0][p] + part[1][p] + ... + part[S-1][p]), fixed order.
template <typename T>
__global__ void reduce_kernel(const T* __restrict__ part, T* __restrict__ image, size_t n,
                              int n_splits, T scale)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        T s = part[i];
        for (int k = 1; k < n_splits; ++k) s += part[(size_t)k * n + i];
        image[i] = s * scale;
    }
}

}  // namespace fbp
