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
// Lanes are consecutive bins, hence consecutive-ish pixels of the same line.  The image is first staged
// (stage_image_kernel) into zero-padded lines of (pixel, mirror pixel) pairs and, for y-major angles, a
// transposed copy of the same form (roles of cos and sin swapped); the projector moves each line's window
// of a CTA's bins into shared memory with one TMA bulk copy and gathers from there (see project_kernel):
// no bounds checks, and each thread visits only the lines its ray can touch.
#pragma once
#include <cuda_runtime.h>

#include "fbp_backproject.cuh"  // Magic<T>: round-to-nearest by adding 1.5 * 2^23 | 2^52
#include "fbp_ptx.cuh"          // mbarrier, TMA 1-D bulk copy

namespace fbp {

template <typename T> __device__ __forceinline__ T lds(unsigned addr);
template <> __device__ __forceinline__ float lds<float>(unsigned addr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
template <> __device__ __forceinline__ double lds<double>(unsigned addr)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}

struct ProjParams {
    int n_angles, n_det, image_n;
    int pad;             // zero columns left of every staged line (a multiple of 4, >= E_max + 2, and wide enough for a window)
    int pitch;           // elements per staged line (a multiple of 4): pad + N + right pad
    int win;             // W: elements of a staged window (a multiple of 4)
    int lb;              // LB: lines staged per block (<= 16)
    double c_n, c_d;
};

template <typename T> struct ProjPair;
template <> struct ProjPair<float> { using type = float2; };
template <> struct ProjPair<double> { using type = double2; };

// Staging: two padded copies of the image, interleaved with their point mirrors, every line `pitch` pairs with zero
// pads on both sides:
//   xi [b][r][pad + c] = ( x[b][r][c], x[b][N-1-r][N-1-c] )        xti[b][c][pad + r] = ( x[b][r][c], x[b][N-1-r][N-1-c] )
// (xti: the transpose, for the angles whose fast axis is y).  A projector window is then ONE aligned row segment that
// carries, for every pixel, the pixel and its mirror pixel.  32x32 tiles through shared memory; the CTAs of the first
// tile column also write the pads.  Grid (ceil(N/32), ceil(N/32), batch), block (32, 8).
template <typename T>
__global__ void __launch_bounds__(256)
stage_image_kernel(const T* __restrict__ x, typename ProjPair<T>::type* __restrict__ xi, typename ProjPair<T>::type* __restrict__ xti,
                   int n, int pad, int pitch)
{
    __shared__ T tile[32][33];
    const size_t off = (size_t)blockIdx.z * n * n, offp = (size_t)blockIdx.z * n * pitch;
    const int c0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
    for (int k = threadIdx.y; k < 32; k += 8) {
        const int r = r0 + k, c = c0 + threadIdx.x;
        if (r < n && c < n) {
            const T v = x[off + (size_t)r * n + c];
            tile[k][threadIdx.x] = v;
            xi[offp + (size_t)r * pitch + pad + c].x = v;
            xi[offp + (size_t)(n - 1 - r) * pitch + pad + (n - 1 - c)].y = v;
        }
    }
    __syncthreads();
    for (int k = threadIdx.y; k < 32; k += 8) {
        const int c = c0 + k, r = r0 + threadIdx.x;
        if (r < n && c < n) {
            const T v = tile[threadIdx.x][k];
            xti[offp + (size_t)c * pitch + pad + r].x = v;
            xti[offp + (size_t)(n - 1 - c) * pitch + pad + (n - 1 - r)].y = v;
        }
    }
    // zero pads (pad pairs on the left, pitch - pad - n on the right) of lines r0..r0+31 of both copies, by the CTAs of
    // the first tile column
    const int t = threadIdx.y * 32 + threadIdx.x, npad = pitch - n;
    typename ProjPair<T>::type zero;
    zero.x = T(0); zero.y = T(0);
    if (blockIdx.x == 0)
        for (int i = t; i < 32 * npad; i += 256) {
            const int r = r0 + i / npad, q = i % npad;
            if (r < n) {
                const size_t e = offp + (size_t)r * pitch + (q < pad ? q : n + q);
                xi[e] = zero; xti[e] = zero;
            }
        }
}

// Point symmetry (as in the back-projector): the mirror pixel (N-1-l, N-1-p) has u' = (D-1) - u, so it meets the
// mirror bin D-1-j with the SAME weight hat(u - j).  A thread therefore owns bin j < ceil(D/2) and its mirror bin
// and computes the run and its weights once for both.
//
// Shared-memory staging.  A CTA owns 128 consecutive bins of ONE angle.  On line l their runs lie in a window of
// W >= 127/|cf| + 2E + 7 pixels starting at ps(l) = floor(min_j p*(j, l)) - E - 1 rounded down to a multiple of 4 (and
// clamped into the padded line: a run that matters never leaves [-(E+2), N+E+2]).  Lines are processed in blocks of LB:
// lane q of the producer warp (warp 4) issues ONE TMA bulk copy of the window of line q -- W (pixel, mirror pixel)
// pairs -- into a two-stage ring (full / empty mbarriers, no block-wide barrier), and the four consumer warps read a
// run and its mirror run with one LDS.64 per pixel.  Why: read straight from global memory, a warp's load of 32
// neighbouring runs touches 2-3 cache lines and costs ~5 cycles of the L1 tag stage (ncu: 80 % of the stall samples waited
// for these loads, issue-active 32 %); the same load from shared memory is one or two wavefronts.
// cs2: [K] (cos, sin) * pix/d in fp64.  Grid (bin_blocks * K, 1, batch), bin_blocks = ceil(ceil(D/2)/128), block 160:
// thread t < 128 = bin j0 + t.  xi / xti: the interleaved padded copies of stage_image_kernel.  y: [batch][K][D], fully written.
// Dynamic shared memory: full[2], empty[2] mbarriers (32 B) | int ps[2][16] | pair seg[2][LB][W].
template <typename T> struct ProjAcc;
template <> struct ProjAcc<float> {          // (bin, mirror bin) sums in one 64-bit register: packed FFMA2 with a scalar weight
    unsigned long long v = 0ull;
    __device__ __forceinline__ void add(float w, unsigned addr)
    {
        unsigned long long q, w2;
        asm volatile("ld.shared.b64 %0, [%1];" : "=l"(q) : "r"(addr));
        asm("mov.b64 %0, {%1, %1};" : "=l"(w2) : "f"(w));
        asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(v) : "l"(q), "l"(w2));
    }
    __device__ __forceinline__ float a() const { return __uint_as_float((unsigned)(v & 0xffffffffull)); }
    __device__ __forceinline__ float b() const { return __uint_as_float((unsigned)(v >> 32)); }
};
template <> struct ProjAcc<double> {
    double va = 0.0, vb = 0.0;
    __device__ __forceinline__ void add(double w, unsigned addr)
    {
        double qa, qb;
        asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(qa), "=d"(qb) : "r"(addr));
        va = fma(w, qa, va); vb = fma(w, qb, vb);
    }
    __device__ __forceinline__ double a() const { return va; }
    __device__ __forceinline__ double b() const { return vb; }
};

template <typename T>
__global__ void __launch_bounds__(160)
project_kernel(const typename ProjPair<T>::type* __restrict__ xi, const typename ProjPair<T>::type* __restrict__ xti,
               T* __restrict__ y, const double2* __restrict__ cs2, ProjParams prm, int bin_blocks)
{
    using Pair = typename ProjPair<T>::type;
    extern __shared__ __align__(16) unsigned char proj_smem[];
    const unsigned bar_full = smem_u32(proj_smem), bar_empty = bar_full + 16u;
    int* ps_s = reinterpret_cast<int*>(proj_smem + 32);            // [2][16]
    const unsigned seg_u = smem_u32(proj_smem + 32 + 128);
    __shared__ int s_lo, s_hi;

    const int i = blockIdx.x / bin_blocks, b = blockIdx.z;
    const int j0 = (blockIdx.x - i * bin_blocks) * 128;
    const int tid = threadIdx.x, lane = tid & 31;
    const bool producer = tid >= 128;
    const int j = j0 + tid;
    const int N = prm.image_n, pitch = prm.pitch, W = prm.win, LB = prm.lb;
    const int half = (prm.n_det + 1) / 2;
    const bool live = !producer && j < half;
    const int jm = prm.n_det - 1 - j;            // mirror bin (== j for the middle bin of an odd detector)
    const double2 cs = cs2[i];
    const bool xmajor = fabs(cs.x) >= fabs(cs.y);
    const double cf = xmajor ? cs.x : cs.y;      // change of u per pixel along a line (fast axis); |cf| > 0
    const double cl = xmajor ? cs.y : cs.x;      // change of u per line
    const Pair* img = (xmajor ? xi : xti) + (size_t)b * N * pitch + prm.pad;
    // u(line l, pixel p) = c_D + (p - c_N) cf + (l - c_N) cl;   u = j  <=>  p = p*(l) = A + Bl * l
    const double inv = 1.0 / cf;
    const double A0 = prm.c_n + ((double)j0 - prm.c_d + prm.c_n * cl) * inv;     // bin j0
    const double A = A0 + (double)tid * inv;
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
    if (!live || l_lo > l_hi) { l_lo = N; l_hi = -1; }

    // the CTA's line range (a min / max of integers: the order of the atomics does not matter)
    if (tid == 0) {
        s_lo = N; s_hi = -1;
        for (int st = 0; st < 2; ++st) { mbar_init(bar_full + 8u * st, 1); mbar_init(bar_empty + 8u * st, 4); }
        fence_mbar_init();
    }
    __syncthreads();
    if (l_lo <= l_hi) { atomicMin(&s_lo, l_lo); atomicMax(&s_hi, l_hi); }
    __syncthreads();
    const int lo = s_lo, hi = s_hi;
    const int n_blocks = lo <= hi ? (hi - lo) / LB + 1 : 0;
    const unsigned pair_bytes = 2u * (unsigned)sizeof(T);
    const unsigned line_bytes = (unsigned)W * pair_bytes, buf_bytes = (unsigned)LB * line_bytes;
    ProjAcc<T> acc;
    if (producer) {
        // window start of a line: the smallest p* among the CTA's live bins is at bin j0 or at the last one
        const int jl = min(127, half - 1 - j0);
        const double Amin = fmin(A0, A0 + (double)jl * inv);
        const int ps_min = -prm.pad, ps_max = pitch - prm.pad - W;         // the window stays inside the padded line
        for (int k = 0; k < n_blocks; ++k) {
            const int buf = k & 1, l0 = lo + k * LB;
            const int nl = min(LB, hi - l0 + 1);
            const Pair* src = img;
            int ps = 0;
            if (lane < nl) {
                double f = floor(fma(Bl, (double)(l0 + lane), Amin)) - (double)(E + 1);
                f = fmin(fmax(f, -1.0e6), 1.0e6);
                ps = (int)f;
                ps = (ps >= 0 ? ps : ps - 3) / 4 * 4;                      // down to a multiple of 4
                ps = min(max(ps, ps_min), ps_max);
                src = img + (size_t)(l0 + lane) * pitch + ps;
            }
            if (k >= 2) mbar_wait(bar_empty + 8u * buf, (unsigned)(((k >> 1) - 1) & 1));   // the consumers released the stage
            if (lane < nl) {
                ps_s[buf * 16 + lane] = ps;
                tma_load_1d(seg_u + buf * buf_bytes + lane * line_bytes, src, line_bytes, bar_full + 8u * buf);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive_expect_tx(bar_full + 8u * buf, (unsigned)nl * line_bytes);
        }
    } else {
        const T BlT = (T)Bl;
        const int cmin = -(E + 1), cmax = N + E;     // clamp of round(p*)
        for (int k = 0; k < n_blocks; ++k) {
            const int buf = k & 1, l0 = lo + k * LB;
            mbar_wait(bar_full + 8u * buf, (unsigned)((k >> 1) & 1));
            // p*(l0) in fp64 once per block, split into an integer part and a fraction; inside the block the fraction
            // advances in the working precision (|.| < 18: ulp <= 2e-6 in fp32) and is rounded by adding 1.5 * 2^23 | 2^52
            const double base = fma(Bl, (double)l0, A);
            const double bfl = floor(fmin(fmax(base, -1.0e6), 1.0e6));
            const int pb = (int)bfl;
            const T fb = (T)(base - bfl);
            const int q_lo = max(0, l_lo - l0), q_hi = min(LB - 1, l_hi - l0);   // this thread's lines of the block
            const unsigned seg_b = seg_u + buf * buf_bytes;
            const int* psb = ps_s + buf * 16;
            T qf = (T)q_lo;
            if (E == 1) {
#pragma unroll 4
                for (int q = q_lo; q <= q_hi; ++q) {
                    const T ps = fma(BlT, qf, fb);                                      // p* - pb
                    const T tm = ps + Magic<T>::m();
                    const int p0 = min(max(pb + (int)(Magic<T>::bits(tm) - Magic<T>::kBits), cmin), cmax);   // round(p*)
                    const T d0 = ps - (tm - Magic<T>::m());                             // p* - round(p*), in [-1/2, 1/2]
                    const unsigned a = seg_b + (unsigned)q * line_bytes + (unsigned)(p0 - 1 - psb[q]) * pair_bytes;
                    const T wm = fmax(fma(-acf, T(1) + d0, T(1)), T(0));                // e = -1: |e - d0| = 1 + d0
                    const T w0 = fmax(fma(-acf, fabs(d0), T(1)), T(0));
                    const T wp = fmax(fma(-acf, T(1) - d0, T(1)), T(0));
                    acc.add(wm, a); acc.add(w0, a + pair_bytes); acc.add(wp, a + 2u * pair_bytes);
                    qf += T(1);
                }
            } else {
                for (int q = q_lo; q <= q_hi; ++q) {
                    const T ps = fma(BlT, qf, fb);
                    const T tm = ps + Magic<T>::m();
                    const int p0 = min(max(pb + (int)(Magic<T>::bits(tm) - Magic<T>::kBits), cmin), cmax);
                    const T d0 = ps - (tm - Magic<T>::m());
                    const unsigned a = seg_b + (unsigned)q * line_bytes + (unsigned)(p0 - psb[q]) * pair_bytes;
                    for (int e = -E; e <= E; ++e)
                        acc.add(fmax(fma(-acf, fabs((T)e - d0), T(1)), T(0)), a + e * (int)pair_bytes);   // hat(u - j)
                    qf += T(1);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_empty + 8u * buf);       // this warp is done with the stage
        }
    }
    if (!live) return;
    T* yrow = y + ((size_t)b * prm.n_angles + i) * prm.n_det;
    yrow[j] = acc.a();
    if (jm != j) yrow[jm] = acc.b();
}

}  // namespace fbp
