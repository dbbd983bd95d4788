// fbp_fft.cuh -- FFT form of the row filter for sm_100a (Q = P * H), hand-written, in shared memory.
//
// Q[n] = (1/d) sum_{k=0}^{D-1} h[n-k] P[k] is the same linear ("same", zero-extended) convolution the direct
// form computes (fbp_filter3.cuh); here it is evaluated as a circular convolution of length N = 2^p >= 2D:
//
//   summation by parts   Q[n] = (1/d) sum_{k=0}^{D} g[n-k] (P[k] - P[k-1]),   P[-1] = P[D] = 0,
//                        g[l] = sum_{m <= l} h[m]   (the taps' running sum; h is even with sum_m h[m] = 0, so
//                        g[-1] = -h[0]/2 and every g[l] is a FINITE sum of the closed-form taps)
//   circular kernel      c[l mod N] = g[l] / (d N)  for l = -D .. D-1, 0 elsewhere;   G = DFT_N(c)   (host, long double)
//   device               z = dP_a + i dP_b  (two rows per transform: the kernel is real, so the real and imaginary
//                        parts stay the two rows' results);  Z = DFT_N(z);  Z *= G;  y = N IDFT_N(Z) (the 1/N is in G);
//                        Q_a[n] = Re y[n], Q_b[n] = Im y[n], n = 0 .. D-1.
//
// Why first differences: 1/4 P[n] cancels against sum |h[m]| P[n-m]; an fp32 FFT of P itself would carry a
// rounding error proportional to |P| (hundreds) into a result of size |Q| (units).  The differences are as small
// as the result, so the error is eps * sqrt(log N) relative to Q: smaller than the direct form's.
// The taps are the same closed-form taps as the direct form's (their DFT, not a sampled |w|: SURVEY.md G2);
// apodised windows only change the table.
//
// Transform: Stockham autosort, radix 16 / 8 / 4 passes in registers (16 points per thread and pass), data in
// shared memory in place (two barriers per pass).  Twiddles come from a per-pass table laid out in the order the
// lanes read it ([pass][r][k] = exp(-2 pi i k r / (NS R)), rounded from long double), followed by the kernel's DFT G;
// when the table fits beside the data it is staged once per CTA by one TMA bulk copy (a 2048-point fp32 plan: 32 KB),
// otherwise it is read through L1.  The first pass reads the rows from global memory and takes the differences; the first inverse pass multiplies by G as it reads; the last inverse pass drops its outputs straight into the two row buffers from which the plain
// rows and the back-projector's entries (fbp_entries.cuh) are written.  Shared-memory index i lives at
// i + (i >> S) (one pad element per 32 fp32 / 16 fp64 complex): the radix-16 stores of the first pass, whose lane
// stride is 16 elements, would otherwise all hit the same banks.
// Rows are paired within a slice only (a slice with an odd number of angles filters its last row alone), so a
// slice's bytes do not depend on its neighbours in the batch.  One owner per output, fixed order: deterministic.
#pragma once
#include <cuda_runtime.h>

#include "fbp_entries.cuh"
#include "fbp_ptx.cuh"

namespace fbp {

struct FftParams {
    int n_slices, n_angles, n_det;   // batch, K, D
    int pairs_per_slice;             // ceil(K / 2)
    int ent_pitch, ent_guard;
    int buf_bytes;                   // bytes of the transform / row buffer region (a multiple of 16)
    const void* warm;                // a table of the NEXT kernel (the back-projector's cos/sin) to start into L2, or NULL
    int warm_bytes;
    unsigned long long* trace;
};

template <typename T> struct Cx { T x, y; };
template <typename T> __device__ __forceinline__ Cx<T> operator+(Cx<T> a, Cx<T> b) { return {a.x + b.x, a.y + b.y}; }
template <typename T> __device__ __forceinline__ Cx<T> operator-(Cx<T> a, Cx<T> b) { return {a.x - b.x, a.y - b.y}; }
// a * b, or a * conj(b)
template <bool CONJ, typename T> __device__ __forceinline__ Cx<T> cmul(Cx<T> a, Cx<T> b)
{
    if (CONJ) return {fma(a.y, b.y, a.x * b.x), fma(a.y, b.x, -(a.x * b.y))};
    return {fma(-a.y, b.y, a.x * b.x), fma(a.y, b.x, a.x * b.y)};
}

// d * exp(-/+ 2 pi i t / LEN) for the constants a radix-16 network needs (INV: + sign)
template <int LEN, int t, bool INV, typename T> __device__ __forceinline__ Cx<T> mul_root(Cx<T> d)
{
    constexpr int e = (16 / LEN) * t;                  // sixteenths of a turn, 0 .. 7
    const T h = T(0.70710678118654752440), c1 = T(0.92387953251128675613), s1 = T(0.38268343236508977173);
    if (e == 0) return d;
    if (e == 4) return INV ? Cx<T>{-d.y, d.x} : Cx<T>{d.y, -d.x};
    if (e == 2) return INV ? Cx<T>{(d.x - d.y) * h, (d.x + d.y) * h} : Cx<T>{(d.x + d.y) * h, (d.y - d.x) * h};
    if (e == 6) return INV ? Cx<T>{(-d.x - d.y) * h, (d.x - d.y) * h} : Cx<T>{(d.y - d.x) * h, (-d.x - d.y) * h};
    const T c = (e == 1) ? c1 : (e == 3) ? s1 : (e == 5) ? -s1 : -c1;
    const T s = (e == 1 || e == 7) ? s1 : c1;
    return cmul<!INV>(d, Cx<T>{c, s});                  // forward: d * (c - i s)
}

// in-register DFT of R points, decimation in frequency: v[i] holds X[bitrev_R(i)] on return
template <int LEN, bool INV, typename T> struct DifStage {
    __device__ __forceinline__ static void run(Cx<T>* v)
    {
        constexpr int H = LEN / 2;
        dif<0>(v);
        DifStage<H, INV, T>::run(v);
        DifStage<H, INV, T>::run(v + H);
    }
    template <int t> __device__ __forceinline__ static void dif(Cx<T>* v)
    {
        constexpr int H = LEN / 2;
        if constexpr (t < H) {
            const Cx<T> a = v[t], b = v[t + H];
            v[t] = a + b;
            v[t + H] = mul_root<LEN, t, INV, T>(a - b);
            dif<t + 1>(v);
        }
    }
};
template <bool INV, typename T> struct DifStage<1, INV, T> { __device__ __forceinline__ static void run(Cx<T>*) {} };

__host__ __device__ constexpr int bitrev(int i, int r) { int o = 0; for (int b = 1; b < r; b <<= 1) { o = (o << 1) | (i & 1); i >>= 1; } return o; }

// pass radices of a 2^p-point transform; the first is always 16 (p >= 6)
__host__ __device__ constexpr int fft_n_passes(int p) { return p <= 8 ? 2 : (p <= 12 ? 3 : 4); }
__host__ __device__ constexpr int fft_radix(int p, int pass)
{
    // p: 6 16.4  7 16.8  8 16.16  9 16.8.4  10 16.8.8  11 16.16.8  12 16.16.16  13 16.8.8.8
    if (pass == 0) return 16;
    if (p == 6) return 4;
    if (p == 7) return 8;
    if (p == 8) return 16;
    if (p == 9) return pass == 1 ? 8 : 4;
    if (p == 10) return 8;
    if (p == 11) return pass == 1 ? 16 : 8;
    if (p == 12) return 16;
    return 8;
}

template <typename T> struct FftSkew { static constexpr int shift = sizeof(T) == 4 ? 5 : 4; };
template <typename T> __device__ __forceinline__ int skew(int i) { return i + (i >> FftSkew<T>::shift); }

// offset (in complex elements) of pass `pass`'s twiddles in the table, and the table's total twiddle count
__host__ __device__ constexpr int fft_tw_offset(int p, int pass)
{
    int off = 0, ns = 16;
    for (int q = 1; q < pass; ++q) { off += (fft_radix(p, q) - 1) * ns; ns *= fft_radix(p, q); }
    return off;
}
__host__ __device__ constexpr int fft_tw_total(int p) { return fft_tw_offset(p, fft_n_passes(p)); }

// One Stockham pass of radix R over N = 2^P points held in `buf` (skewed), in place: every thread first reads its
// 16 points -- multiplying each, as it arrives, by its twiddle Wp[(r-1) NS + k] (and, PREMUL, by the kernel's DFT
// Gt[i]: the point-wise product is taken on the way into the first inverse pass) -- then all threads meet, transform
// and write.  NS = product of the radices of earlier passes.  FIRST: the points come from `loader(i)` (global
// memory) instead of buf.  SINK: outputs go to sink(i, value) (the row buffers) instead of buf.
// (Measured and rejected: one copy of the code per radix with run-time NS / flags, to shrink the 45 KB of
// straight-line instructions a CTA runs once -- 1.7x slower at every size.)
template <typename T, int P, int R, int NS, bool INV, bool FIRST, bool PREMUL, bool SINK, typename Loader, typename Sink>
__device__ __forceinline__ void fft_pass(Cx<T>* buf, const Cx<T>* __restrict__ Wp, const Cx<T>* __restrict__ Gt,
                                         int tid, int nthr, Loader loader, Sink sink)
{
    constexpr int N = 1 << P, B = 16 / R, NB = N / R;      // butterflies per thread, butterflies per pass
    Cx<T> v[16];
#pragma unroll
    for (int b = 0; b < B; ++b) {
        const int j = tid + b * nthr;
        if (j < NB) {
            const int k = j & (NS - 1);
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int i = j + r * NB;
                Cx<T> x = FIRST ? loader(i) : buf[skew<T>(i)];
                if (PREMUL) x = cmul<false>(x, Gt[i]);
                if (NS > 1 && r > 0) x = cmul<INV>(x, Wp[(r - 1) * NS + k]);
                v[b * R + r] = x;
            }
        }
    }
    if (!FIRST) __syncthreads();                             // everyone has read: the buffer may be overwritten
#pragma unroll
    for (int b = 0; b < B; ++b) {
        const int j = tid + b * nthr;
        if (j < NB) {
            const int k = j & (NS - 1);
            DifStage<R, INV, T>::run(v + b * R);
            const int j0 = (j - k) * R + k;
#pragma unroll
            for (int q = 0; q < R; ++q) {
                const int i = j0 + bitrev(q, R) * NS;         // v[q] holds output bitrev(q)
                if (SINK) sink(i, v[b * R + q]);
                else buf[skew<T>(i)] = v[b * R + q];
            }
        }
    }
    __syncthreads();
}

// Registers: 16 complex points per thread are 32 (fp32) / 64 (fp64) registers, and left alone the compiler hoists
// the table loads of a whole pass and takes 220+.  What a cap buys depends on the block size:
//   - N <= 2048 (blocks of <= 128 threads; configs 3 and 4): no cap.  Shared memory already limits these to <= 4
//     CTAs per SM, a config-3 launch is 180 CTAs on 148 SMs, and every cap measured on B200 lost to none: the
//     96-register build spilled 212 bytes in the passes (136-byte stack) and took 14.8 us for the config-3 filter,
//     128 registers 13.2 us (still spilling), 255 registers 12.6 us with no local memory at all (whole step 42.3 ->
//     40.1 us); the config-4 stack went 431 -> 413 us with half the resident warps.
//   - longer transforms (256 / 512 threads) keep the caps below: 512 threads cannot have more than 128 registers.
#ifndef FBP_FFT_REGS32
#define FBP_FFT_REGS32 96
#endif
#ifndef FBP_FFT_REGS64
#define FBP_FFT_REGS64 168
#endif
template <typename T, int P> struct FftLaunch {
    static constexpr int threads = (1 << P) / 16 < 32 ? 32 : (1 << P) / 16;
    static constexpr int regs = threads <= 128 ? 255 : (sizeof(T) == 4 ? FBP_FFT_REGS32 : FBP_FFT_REGS64);
    static constexpr int min_blocks = 65536 / (regs * threads) < 1 ? 1 : (65536 / (regs * threads) > 32 ? 32 : 65536 / (regs * threads));
};

// Tab: [fft_tw_total(P)] per-pass twiddles, then [N] DFT of the circular kernel (includes 1/(d N)).  TSMEM: the
// table is staged in shared memory behind the transform buffer.  Pin: [batch][K][D].  Q (plain rows) and/or E
// (entries) may be NULL.  wrow: per-row entry multipliers or NULL.
// Block: max(32, N / 16) threads.  Grid: persistent over batch * ceil(K / 2) row pairs.
template <typename T, int P, bool TSMEM>
__global__ void __launch_bounds__(FftLaunch<T, P>::threads, FftLaunch<T, P>::min_blocks)
fft_filter_kernel(const T* __restrict__ Pin, T* __restrict__ Q, uint4* __restrict__ E, const Cx<T>* __restrict__ Tab,
                  const T* __restrict__ wrow, FftParams prm)
{
    constexpr int N = 1 << P, NTW = fft_tw_total(P);
    extern __shared__ __align__(16) unsigned char fft_smem_raw[];
    // layout: bar (16 B) | transform buffer, later the two row buffers (buf_bytes) | table (TSMEM)
    Cx<T>* buf = reinterpret_cast<Cx<T>*>(fft_smem_raw + 16);     // skewed N points
    const int D = prm.n_det, K = prm.n_angles, pitch = prm.ent_pitch, guard = prm.ent_guard;
    T* yza = reinterpret_cast<T*>(fft_smem_raw + 16);              // yz[k] = Q~[k - 1 - guard], k in [0, pitch + 2)
    T* yzb = yza + (pitch + 2);
    const int tid = threadIdx.x, nthr = blockDim.x;
    const Cx<T>* Wp = Tab;
    const Cx<T>* Gt = Tab + NTW;

    pdl_launch_dependents();
    trace_mark(prm.trace, blockIdx.x, 0);
    // the back-projector's first instruction after its grid dependency is a read of its cos/sin table, which nothing
    // has touched since the caller's last use of the plan: one CTA starts it on its way into L2 now
    if (blockIdx.x == 0 && prm.warm != nullptr)
        for (int i = tid * 128; i < prm.warm_bytes; i += nthr * 128)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(static_cast<const char*>(prm.warm) + i));
    if (TSMEM) {
        // one bulk copy brings the whole table in while the first pass reads the rows
        const unsigned bar = smem_u32(fft_smem_raw);
        Cx<T>* tab_s = reinterpret_cast<Cx<T>*>(fft_smem_raw + 16 + prm.buf_bytes);
        if (tid == 0) {
            mbar_init(bar, 1);
            fence_mbar_init();
            const unsigned bytes = (unsigned)((NTW + N) * sizeof(Cx<T>));
            mbar_arrive_expect_tx(bar, bytes);
            tma_load_1d(smem_u32(tab_s), Tab, bytes, bar);
        }
        __syncthreads();
        Wp = tab_s;
        Gt = tab_s + NTW;
    }
    const long long n_work = (long long)prm.n_slices * prm.pairs_per_slice;
    for (long long w = blockIdx.x; w < n_work; w += gridDim.x) {
        const int slice = (int)(w / prm.pairs_per_slice), pr = (int)(w - (long long)slice * prm.pairs_per_slice);
        const int ra = 2 * pr, rb = 2 * pr + 1;
        const bool has_b = rb < K;
        const T* pa = Pin + ((size_t)slice * K + ra) * D;
        const T* pb = pa + D;
        // z[i] = dP_a[i] + i dP_b[i],  dP[i] = P[i] - P[i-1] with P[-1] = P[D] = 0;  zero for i > D.
        // The loads are unconditional (clamped addresses) and the zeros selected afterwards: behind a branch
        // the compiler cannot hoist them and a thread's points arrive one memory round trip after the other.
        const T* pbb = has_b ? pb : pa;
        auto loader = [&](int i) -> Cx<T> {
            const int i1 = min(i, D - 1), i0 = min(max(i - 1, 0), D - 1);
            const T a1 = __ldg(pa + i1), a0 = __ldg(pa + i0), b1 = __ldg(pbb + i1), b0 = __ldg(pbb + i0);
            Cx<T> z;
            z.x = (i < D ? a1 : T(0)) - (i > 0 && i <= D ? a0 : T(0));
            z.y = has_b ? (i < D ? b1 : T(0)) - (i > 0 && i <= D ? b0 : T(0)) : T(0);
            return z;
        };
        auto to_buf = [](int, Cx<T>) {};
        auto to_rows = [&](int i, Cx<T> o) {
            if (i < D) { yza[i + 1 + guard] = o.x; yzb[i + 1 + guard] = o.y; }
        };
        constexpr int NP = fft_n_passes(P);
        constexpr int R1 = fft_radix(P, 1), R2 = NP > 2 ? fft_radix(P, 2) : 1, R3 = NP > 3 ? fft_radix(P, 3) : 1;
        constexpr int O1 = fft_tw_offset(P, 1), O2 = fft_tw_offset(P, 2), O3 = fft_tw_offset(P, 3);
        // ---- forward ----
        fft_pass<T, P, 16, 1, false, true, false, false>(buf, Wp, Gt, tid, nthr, loader, to_buf);
        if (w == blockIdx.x) {
            trace_mark(prm.trace, blockIdx.x, 1);              // rows read, first pass done
            if (TSMEM) mbar_wait(smem_u32(fft_smem_raw), 0u);  // the table has landed
        }
        fft_pass<T, P, R1, 16, false, false, false, false>(buf, Wp + O1, Gt, tid, nthr, loader, to_buf);
        if (NP > 2) fft_pass<T, P, R2, 16 * R1, false, false, false, false>(buf, Wp + O2, Gt, tid, nthr, loader, to_buf);
        if (NP > 3) fft_pass<T, P, R3, 16 * R1 * R2, false, false, false, false>(buf, Wp + O3, Gt, tid, nthr, loader, to_buf);
        if (w == blockIdx.x) trace_mark(prm.trace, blockIdx.x, 2);   // spectrum ready
        // ---- inverse (conjugate twiddles): the first pass multiplies by the kernel's DFT as it reads, the last
        // one writes the two rows over the transform buffer ----
        fft_pass<T, P, 16, 1, true, false, true, false>(buf, Wp, Gt, tid, nthr, loader, to_buf);
        if (NP == 2) {
            fft_pass<T, P, R1, 16, true, false, false, true>(buf, Wp + O1, Gt, tid, nthr, loader, to_rows);
        } else if (NP == 3) {
            fft_pass<T, P, R1, 16, true, false, false, false>(buf, Wp + O1, Gt, tid, nthr, loader, to_buf);
            fft_pass<T, P, R2, 16 * R1, true, false, false, true>(buf, Wp + O2, Gt, tid, nthr, loader, to_rows);
        } else {
            fft_pass<T, P, R1, 16, true, false, false, false>(buf, Wp + O1, Gt, tid, nthr, loader, to_buf);
            fft_pass<T, P, R2, 16 * R1, true, false, false, false>(buf, Wp + O2, Gt, tid, nthr, loader, to_buf);
            fft_pass<T, P, R3, 16 * R1 * R2, true, false, false, true>(buf, Wp + O3, Gt, tid, nthr, loader, to_rows);
        }
        // zero guards of the two row buffers (k <= guard and k >= guard + 1 + D); disjoint from the sink's writes
        for (int k = tid; k < 2 * (guard + 1); k += nthr) {
            const int kk = k <= guard ? k : D + k;             // 0 .. guard, then guard + 1 + D .. pitch + 1
            yza[kk] = T(0); yzb[kk] = T(0);
        }
        __syncthreads();
        if (w == blockIdx.x) trace_mark(prm.trace, blockIdx.x, 3);   // rows back in shared memory
        // ---- stores: plain rows and/or entries j = -1 .. D-1 of both rows (guards beyond stay zero in E) ----
        const int n_rows_here = has_b ? 2 : 1;
        for (int h = 0; h < n_rows_here; ++h) {
            const T* yz = h ? yzb : yza;
            const size_t row = (size_t)slice * K + ra + h;
            if (Q) {
                T* q = Q + row * D;
                for (int n = tid; n < D; n += nthr) q[n] = yz[n + 1 + guard];
            }
            if (E) {
                uint4* erow = E + row * pitch;
                const bool scaled = wrow != nullptr;
                const T m = scaled ? wrow[ra + h] : T(1);
                for (int i = guard - 1 + tid; i <= guard + D - 1; i += nthr) {
                    T a0 = yz[i + 1], a1 = yz[i + 2];
                    T b0 = yz[pitch - 1 - i], b1 = yz[pitch - i];
                    if (scaled) { a0 *= m; a1 *= m; b0 *= m; b1 *= m; }
                    store_entry(erow, i, a0, a1, b0, b1);
                }
            }
        }
        __syncthreads();                                       // the row buffers are the next pair's transform buffer
    }
    trace_mark(prm.trace, blockIdx.x, 4);
}

}  // namespace fbp
