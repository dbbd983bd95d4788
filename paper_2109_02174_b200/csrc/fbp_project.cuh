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
// Lanes are consecutive bins, hence consecutive-ish pixels of the same line: coalesced reads.  The image
// is first staged (stage_image_kernel) into a copy with zero columns on both sides of every line and, for
// y-major angles, a transposed copy of the same form (roles of cos and sin swapped), so that the inner loop
// has no bounds checks and no divergence; each thread visits only the lines its ray can touch.
#pragma once
#include <cuda_runtime.h>

#include "fbp_backproject.cuh"  // Magic<T>: round-to-nearest by adding 1.5 * 2^23 | 2^52

namespace fbp {

struct ProjParams {
    int n_angles, n_det, image_n;
    int pad;             // zero columns on each side of a staged line (>= 2 E_max + 1, multiple of 4)
    double c_n, c_d;
};

// Staging: xp[b][r][pad + c] = x[b][r][c] and xtp[b][c][pad + r] = x[b][r][c], both with `pad` zero columns on
// each side of every line (pitch = N + 2 pad), so that the projector's runs never need a bounds check.
// 32x32 tiles through shared memory; the CTAs of the first tile column/row also write the zero pads.
// Grid (ceil(N/32), ceil(N/32), batch), block (32, 8).
template <typename T>
__global__ void __launch_bounds__(256)
stage_image_kernel(const T* __restrict__ x, T* __restrict__ xp, T* __restrict__ xtp, int n, int pad)
{
    __shared__ T tile[32][33];
    const int pitch = n + 2 * pad;
    const size_t off = (size_t)blockIdx.z * n * n, offp = (size_t)blockIdx.z * n * pitch;
    const int c0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
    for (int k = threadIdx.y; k < 32; k += 8) {
        const int r = r0 + k, c = c0 + threadIdx.x;
        if (r < n && c < n) {
            const T v = x[off + (size_t)r * n + c];
            tile[k][threadIdx.x] = v;
            xp[offp + (size_t)r * pitch + pad + c] = v;
        }
    }
    __syncthreads();
    for (int k = threadIdx.y; k < 32; k += 8) {
        const int c = c0 + k, r = r0 + threadIdx.x;
        if (r < n && c < n) xtp[offp + (size_t)c * pitch + pad + r] = tile[threadIdx.x][k];
    }
    // zero pads: lines r0..r0+31 of xp by the CTAs with blockIdx.x == 0, lines c0..c0+31 of xtp by blockIdx.y == 0
    const int t = threadIdx.y * 32 + threadIdx.x;
    if (blockIdx.x == 0)
        for (int i = t; i < 32 * 2 * pad; i += 256) {
            const int r = r0 + i / (2 * pad), q = i % (2 * pad);
            if (r < n) xp[offp + (size_t)r * pitch + (q < pad ? q : n + q)] = T(0);
        }
    if (blockIdx.y == 0)
        for (int i = t; i < 32 * 2 * pad; i += 256) {
            const int c = c0 + i / (2 * pad), q = i % (2 * pad);
            if (c < n) xtp[offp + (size_t)c * pitch + (q < pad ? q : n + q)] = T(0);
        }
}

// Point symmetry (as in the back-projector): the mirror pixel (N-1-l, N-1-p) has u' = (D-1) - u, so it meets the
// mirror bin D-1-j with the SAME weight hat(u - j).  A thread therefore owns bin j < ceil(D/2) and its mirror bin
// and computes the run and its weights once for both.
// cs2: [K] (cos, sin) * pix/d in fp64.  Grid (bin_blocks * K, 1, batch), bin_blocks = ceil(ceil(D/2)/128), block 128: thread = bin j.
// xp / xtp: the padded image and its padded transpose (stage_image_kernel).  y: [batch][K][D], fully written.
template <typename T>
__global__ void __launch_bounds__(128)
project_kernel(const T* __restrict__ xp, const T* __restrict__ xtp, T* __restrict__ y,
               const double2* __restrict__ cs2, ProjParams prm, int bin_blocks)
{
    const int i = blockIdx.x / bin_blocks, b = blockIdx.z;
    const int j = (blockIdx.x - i * bin_blocks) * 128 + threadIdx.x;
    const int N = prm.image_n, pitch = N + 2 * prm.pad;
    if (j >= (prm.n_det + 1) / 2) return;
    const int jm = prm.n_det - 1 - j;            // mirror bin (== j for the middle bin of an odd detector)
    const double2 cs = cs2[i];
    const bool xmajor = fabs(cs.x) >= fabs(cs.y);
    const double cf = xmajor ? cs.x : cs.y;      // change of u per pixel along a line (fast axis); |cf| > 0
    const double cl = xmajor ? cs.y : cs.x;      // change of u per line
    const T* img = (xmajor ? xp : xtp) + (size_t)b * N * pitch + prm.pad;
    // u(line l, pixel p) = c_D + (p - c_N) cf + (l - c_N) cl;   u = j  <=>  p = p*(l) = A + Bl * l
    const double inv = 1.0 / cf;
    const double A = prm.c_n + ((double)j - prm.c_d + prm.c_n * cl) * inv;
    const double Bl = -cl * inv;
    const T acf = (T)fabs(cf);
    // |e - d0| < 1/|cf| with |d0| <= 1/2  =>  |e| < 1/|cf| + 1/2:  E = 1 whenever pix >= d (1/|cf| <= sqrt 2)
    const int E = (int)ceil(fabs(inv) + 0.5) - 1;
    // lines on which the run can touch the image: p*(l) in [-(E+1), N+E]; p* is affine in l, so an interval
    const double plo = -(double)(E + 1), phi = (double)(N + E);
    int l_lo = 0, l_hi = N - 1;
    if (Bl != 0.0) {
        const double t0 = (plo - A) / Bl, t1 = (phi - A) / Bl;
        const double tl = fmax(fmin(t0, t1), -1.0), th = fmin(fmax(t0, t1), (double)N);
        l_lo = max(0, (int)ceil(tl));
        l_hi = min(N - 1, (int)floor(th));
    } else if (!(A >= plo && A <= phi)) {
        l_hi = -1;
    }
    const T BlT = (T)Bl;
    const int cmin = -(E + 1), cmax = N + E;     // clamp of round(p*): the run stays inside the zero pads
    T acc = T(0), accm = T(0);
    const T* imgm = img + (size_t)(N - 1) * pitch + (N - 1);       // mirror of (line 0, pixel 0)
    // Lines in blocks of 32: p*(l0) in fp64 once per block, split into an integer part and a fraction; inside
    // the block the fraction advances in the working precision (|.| < 34: ulp <= 4e-6 in fp32) and is rounded
    // with the add-magic-constant trick.  No bounds checks: out-of-image pixels of a run read the zero pads.
    for (int l0 = l_lo; l0 <= l_hi; l0 += 32) {
        const double base = fma(Bl, (double)l0, A);
        const double bfl = floor(base);
        const int pb = (int)bfl;
        const T fb = (T)(base - bfl);
        const int l1 = min(32, l_hi - l0 + 1);
        const T* line = img + (size_t)l0 * pitch;
        const T* linem = imgm - (size_t)l0 * pitch;
        if (E == 1) {
#pragma unroll 4
            for (int q = 0; q < l1; ++q) {
                const T ps = fma(BlT, (T)q, fb);                                    // p* - pb
                const T tm = ps + Magic<T>::m();
                const int p0 = min(max(pb + (int)(Magic<T>::bits(tm) - Magic<T>::kBits), cmin), cmax);   // round(p*)
                const T d0 = ps - (tm - Magic<T>::m());                             // p* - round(p*), in [-1/2, 1/2]
                const T* c = line + (size_t)q * pitch + p0;
                const T* cm = linem - (size_t)q * pitch - p0;                       // mirror pixel of (line, p0)
                const T vm = __ldg(c - 1), v0 = __ldg(c), vp = __ldg(c + 1);
                const T um = __ldg(cm + 1), u0 = __ldg(cm), up = __ldg(cm - 1);
                const T wm = fmax(fma(-acf, T(1) + d0, T(1)), T(0));                // e = -1: |e - d0| = 1 + d0
                const T w0 = fmax(fma(-acf, fabs(d0), T(1)), T(0));
                const T wp = fmax(fma(-acf, T(1) - d0, T(1)), T(0));
                acc = fma(wm, vm, acc); acc = fma(w0, v0, acc); acc = fma(wp, vp, acc);
                accm = fma(wm, um, accm); accm = fma(w0, u0, accm); accm = fma(wp, up, accm);
            }
        } else {
            for (int q = 0; q < l1; ++q) {
                const T ps = fma(BlT, (T)q, fb);
                const T tm = ps + Magic<T>::m();
                const int p0 = min(max(pb + (int)(Magic<T>::bits(tm) - Magic<T>::kBits), cmin), cmax);
                const T d0 = ps - (tm - Magic<T>::m());
                const T* c = line + (size_t)q * pitch + p0;
                const T* cm = linem - (size_t)q * pitch - p0;
                for (int e = -E; e <= E; ++e) {
                    const T w = fmax(fma(-acf, fabs((T)e - d0), T(1)), T(0));       // hat(u - j)
                    acc = fma(w, __ldg(c + e), acc);
                    accm = fma(w, __ldg(cm - e), accm);
                }
            }
        }
    }
    T* yrow = y + ((size_t)b * prm.n_angles + i) * prm.n_det;
    yrow[j] = acc;
    if (jm != j) yrow[jm] = accm;
}

}  // namespace fbp
