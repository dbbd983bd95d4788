// fbp_project.cuh -- the matched forward projector R = B^T of the pixel-driven, linearly
// interpolating back-projector (rays x cos + y sin = t):
//
//   y[i][j] = sum over pixels (r,c) of hat(u_i(r,c) - j) * x[r][c],   hat(s) = max(0, 1 - |s|),
//   u_i(r,c) = ((c - c_N) cos_i + (r - c_N) sin_i) * pix/d + c_D,
//
// i.e. exactly the transpose of "read Q at u with weights (1-w, w)": a pixel with floor(u) = j gives
// 1-w to bin j and w to bin j+1, and both are hat(u - bin).  The scatter form of that sum has many
// writers per bin -- the read-modify-write race the paper reports as noise.  Here it
// is a GATHER: one thread owns one bin (i, j) and walks the image in a fixed order (lines ascending,
// pixels ascending within a line), so the result is deterministic and needs no atomics.
//
// Along the image axis on which u changes fastest (x when |cos| >= |sin|, else y), each line has a
// short run of pixels with |u - j| < 1 around p* = the position where u = j: p* is affine in the line
// index and is evaluated in fp64 (so fp32 weights see only the small offset p - p*, never a
// coordinate of size N); the run is round(p*) + e, |e| <= E, with E = ceil(d/(pix max(|cos|,|sin|)) + 1/2) - 1.
// Lanes are consecutive bins, hence consecutive-ish pixels of the same line: coalesced reads.  For
// y-major angles the same code runs on a transposed copy of the image (transpose_kernel), with the
// roles of cos and sin swapped, so those reads are coalesced too.
#pragma once
#include <cuda_runtime.h>

#include "fbp_backproject.cuh"  // Magic<T>: round-to-nearest by adding 1.5 * 2^23 | 2^52

namespace fbp {

struct ProjParams {
    int n_angles, n_det, image_n;
    double c_n, c_d;
};

// xt[b][c][r] = x[b][r][c]; 32x32 tiles through shared memory.  Grid (ceil(N/32), ceil(N/32), batch).
template <typename T>
__global__ void __launch_bounds__(256)
transpose_kernel(const T* __restrict__ x, T* __restrict__ xt, int n)
{
    __shared__ T tile[32][33];
    const size_t off = (size_t)blockIdx.z * n * n;
    const int c0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
    for (int k = threadIdx.y; k < 32; k += 8) {
        const int r = r0 + k, c = c0 + threadIdx.x;
        if (r < n && c < n) tile[k][threadIdx.x] = x[off + (size_t)r * n + c];
    }
    __syncthreads();
    for (int k = threadIdx.y; k < 32; k += 8) {
        const int c = c0 + k, r = r0 + threadIdx.x;
        if (r < n && c < n) xt[off + (size_t)c * n + r] = tile[threadIdx.x][k];
    }
}

// cs2: [K] (cos, sin) * pix/d in fp64.  Grid (ceil(D/128), K, batch), block 128: thread = bin j.
// x: image [batch][N][N]; xt: its transpose (read for y-major angles).  y: [batch][K][D], fully written.
template <typename T>
__global__ void __launch_bounds__(128)
project_kernel(const T* __restrict__ x, const T* __restrict__ xt, T* __restrict__ y,
               const double2* __restrict__ cs2, ProjParams prm)
{
    const int j = blockIdx.x * 128 + threadIdx.x;
    const int i = blockIdx.y, b = blockIdx.z;
    const int N = prm.image_n;
    const double2 cs = cs2[i];
    const bool xmajor = fabs(cs.x) >= fabs(cs.y);
    const double cf = xmajor ? cs.x : cs.y;      // change of u per pixel along a line (fast axis)
    const double cl = xmajor ? cs.y : cs.x;      // change of u per line
    const T* img = (xmajor ? x : xt) + (size_t)b * N * N;
    if (j >= prm.n_det) return;
    if (cf == 0.0) {                             // cannot happen (cos^2 + sin^2 = (pix/d)^2 > 0); guards the division
        y[((size_t)b * prm.n_angles + i) * prm.n_det + j] = T(0);
        return;
    }
    // u(line l, pixel p) = c_D + (p - c_N) cf + (l - c_N) cl;   u = j  <=>  p = p*(l) = A + Bl * l
    const double inv = 1.0 / cf;
    const double A = prm.c_n + ((double)j - prm.c_d + prm.c_n * cl) * inv;
    const double Bl = -cl * inv;
    const T acf = (T)fabs(cf);
    // |e - d0| < 1/|cf| with |d0| <= 1/2  =>  |e| < 1/|cf| + 1/2:  E = 1 whenever pix >= d (1/|cf| <= sqrt 2)
    const int E = (int)ceil(fabs(inv) + 0.5) - 1;
    const T BlT = (T)Bl;
    const unsigned inner = N > 2 ? (unsigned)(N - 2) : 0u;   // columns 1 .. N-2 have both neighbours
    T acc = T(0);
    // Lines in blocks of 32: p*(l0) in fp64 once per block, split into an integer part and a fraction;
    // inside the block the fraction advances in the working precision (|.| < 34: ulp <= 4e-6 in fp32)
    // and is rounded with the add-magic-constant trick (no conversion instructions in the loop).
    for (int l0 = 0; l0 < N; l0 += 32) {
        const double base = fma(Bl, (double)l0, A);
        if (!(base > -1.0e9 && base < 1.0e9)) continue;                         // far outside: nothing to add
        const double bfl = floor(base);
        const int pb = (int)bfl;
        const T fb = (T)(base - bfl);
        const int l1 = min(32, N - l0);
        const T* line = img + (size_t)l0 * N;
        for (int q = 0; q < l1; ++q, line += N) {
            const T ps = fma(BlT, (T)q, fb);                                    // p* - pb
            const T tm = ps + Magic<T>::m();
            const int p0 = pb + (int)(Magic<T>::bits(tm) - Magic<T>::kBits);    // round(p*)
            const T d0 = ps - (tm - Magic<T>::m());                             // p* - round(p*), in [-1/2, 1/2]
            if (E == 1) {
                if ((unsigned)(p0 - 1) < inner) {                                // 1 <= p0 <= N-2: no edge in the run
                    const T* c = line + p0;
                    const T vm = __ldg(c - 1), v0 = __ldg(c), vp = __ldg(c + 1);
                    const T wm = fmax(fma(-acf, T(1) + d0, T(1)), T(0));         // e = -1: |e - d0| = 1 + d0
                    const T w0 = fmax(fma(-acf, fabs(d0), T(1)), T(0));
                    const T wp = fmax(fma(-acf, T(1) - d0, T(1)), T(0));
                    acc = fma(wm, vm, acc); acc = fma(w0, v0, acc); acc = fma(wp, vp, acc);
                    continue;
                }
                if (p0 < -1 || p0 > N) continue;                                 // the run misses the line
            }
            for (int e = -E; e <= E; ++e) {
                const int pp = p0 + e;
                const T w = T(1) - fabs((T)e - d0) * acf;                        // hat(u - j) = 1 - |p - p*| |cf|
                if (w > T(0) && pp >= 0 && pp < N) acc = fma(w, __ldg(line + pp), acc);
            }
        }
    }
    y[((size_t)b * prm.n_angles + i) * prm.n_det + j] = acc;
}

}  // namespace fbp
