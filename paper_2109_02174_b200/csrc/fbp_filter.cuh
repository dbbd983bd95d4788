// fbp_filter.cuh -- Ram-Lak row filter for sm_100a (Q_theta = P_theta * H).
//
// Q[i][n] = (1/d) * ( h[0] P[i][n] + sum_{odd m} h[m] P[i][n-m] ),  h[0] = 1/4,
// h[m] = -1/(pi^2 m^2) for odd m, 0 for even m != 0 (include/fbp.h).
//
// Polyphase form.  Only odd taps are non-zero, so an output of parity p reads inputs of
// parity 1-p only.  With n = 2a + p, k = 2b + (1-p), m = n - k = 2q + 1:
//   q = a - b - (1-p),   g[q] := h[2q+1] = -1/(pi^2 (2q+1)^2).
// A thread owns R consecutive same-parity outputs a0..a0+R-1 and walks inputs b:
//   acc[r] += g[a0 + r - b - (1-p)] * (X[b] - c)
// The R taps needed at step b form a window that slides by one per step; it lives in
// registers (rotating through an R-times unrolled body): per step one tap load (lanes own
// consecutive output blocks => stride R words, R odd => conflict-free), one broadcast input
// load, one subtract and R FMAs.
//
// Conditioning.  1/4 P[n] cancels against sum_m |h[m]| P[n-m] ~ 1/4 P[n]; summed naively in
// fp32 the rounding error scales with P, not with Q.  Filtering is linear, so each thread
// subtracts a constant c (the input at the centre of its output block) from every input and
// adds c * rho[n] back at the end, rho[n] = 1/4 + sum_b g[a - b - (1-p)] over the (padded)
// input range, computed in fp64 on the host.  The running sums then hold differences of
// neighbouring samples times taps instead of two large cancelling numbers.
//
// Work decomposition.  One CTA filters one row.  Warp (p, ob, sb) owns parity p, output block
// ob (32*R outputs) and slice sb of the input range (SB slices, so that one 512^2-sized
// sinogram still fills 148 SMs).  Partial sums go to shared memory and are added in fixed
// order sb = 0..SB-1 by one owner thread per output: no atomics, deterministic.
// The epilogue writes the plain row Q[i][:] (fbp_filter) and/or the back-projector's
// interleaved entries (fbp_reconstruct; see fbp_backproject.cuh "BpEntry").
#pragma once
#include <cuda_runtime.h>

namespace fbp {

#ifdef FBP_TRACE   // phase timestamps for _work experiments (never defined in the product build)
__device__ unsigned long long g_trace[16 * 4096];
__device__ __forceinline__ unsigned long long trace_now()
{
    unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t;
}
#endif

struct FilterParams {
    int n_rows;            // batch * K
    int n_det;             // D
    int de, dn;            // ceil(D/2) even-indexed samples, floor(D/2) odd-indexed samples
    int de_pad, dn_pad;    // padded to a multiple of SB*R (zero filled)
    int n_ob;              // output blocks of 32*R per parity
    int n_sb;              // input slices SB
    int tab_off;           // tap table: G[q + tab_off] = g[q]
    int tab_cnt;           // taps staged per parity: max(de_pad, dn_pad) + n_ob*32*R + R + 1
    int x_pitch;           // elements per staged input array
    // entry output (0 = none): row pitch in entries and left guard, see BpEntry
    int ent_pitch, ent_guard;
};

// ---- entries: the back-projector's operands (fbp_backproject.cuh) -------------------------
// For detector interval j (between bins j and j+1 of the zero-extended row Q~) and its mirror
// interval D-2-j:   mid_a = (Q~[j]+Q~[j+1])/2, mid_b = (Q~[D-2-j]+Q~[D-1-j])/2,
//                   slope_a = Q~[j+1]-Q~[j],   nslope_b = Q~[D-2-j]-Q~[D-1-j].
// Row layout in 16-byte units, index i = j + guard, i in [0, pitch), pitch = D + 2*guard:
//   fp32: one plane   [pitch] of (mid_a, mid_b, slope_a, nslope_b)
//   fp64: two planes  [pitch] of (mid_a, mid_b)  then  [pitch] of (slope_a, nslope_b)
// `yz` is the row with one extra leading zero and the guards: yz[k] = Q~[k - 1 - guard],
// k in [0, pitch + 2).  Then the mirror interval of i starts at yz[pitch - 1 - i].
template <typename T> struct EntryPlanes { static constexpr int value = (int)sizeof(T) / 4; };

__device__ __forceinline__ void store_entry(uint4* erow, int /*pitch*/, int i, float ma, float mb, float sa, float sb)
{
    erow[i] = make_uint4(__float_as_uint(ma), __float_as_uint(mb), __float_as_uint(sa), __float_as_uint(sb));
}
__device__ __forceinline__ void store_entry(uint4* erow, int pitch, int i, double ma, double mb, double sa, double sb)
{
    reinterpret_cast<double2*>(erow)[i] = make_double2(ma, mb);
    reinterpret_cast<double2*>(erow)[pitch + i] = make_double2(sa, sb);
}

template <typename T>
__device__ __forceinline__ void store_entries(const T* yz, uint4* erow, int pitch, int tid, int nthr,
                                              const T* wmul = nullptr)
{
    // wmul: this row's angle weight divided by pi/K (fbp_set_angle_weights); NULL = the uniform pi/K
    const bool scaled = wmul != nullptr;
    const T m = scaled ? *wmul : T(1);
    for (int i = tid; i < pitch; i += nthr) {
        T a0 = yz[i + 1], a1 = yz[i + 2];
        T b0 = yz[pitch - 1 - i], b1 = yz[pitch - i];
        if (scaled) { a0 *= m; a1 *= m; b0 *= m; b1 *= m; }
        store_entry(erow, pitch, i, T(0.5) * (a0 + a1), T(0.5) * (b0 + b1), a1 - a0, b0 - b1);
    }
}

template <typename T, int R>
__global__ void __launch_bounds__(512)
filter_kernel(const T* __restrict__ P, T* __restrict__ Q, uint4* __restrict__ E,
              const T* __restrict__ G_gmem, const T* __restrict__ rho, FilterParams prm, T inv_d)
{
    extern __shared__ __align__(16) unsigned char filt_smem_raw[];
    // layout: G0[tab_cnt] G1[tab_cnt] X0[x_pitch] X1[x_pitch] C[2*n_ob*32] Y[y_pitch] part[...]
    T* G0 = reinterpret_cast<T*>(filt_smem_raw);
    T* X0 = G0 + 2 * prm.tab_cnt;
    T* X1 = X0 + prm.x_pitch;
    T* Cs = X1 + prm.x_pitch;
    const int blk = 32 * R;
    const int y_pitch = 2 * prm.n_ob * blk;
    T* Y = Cs + 2 * prm.n_ob * 32;          // Y[p][ob*blk + o] : filtered outputs by parity
    T* part = Y + y_pitch;                  // part[sb][p][ob*blk + o]

    const int tid = threadIdx.x, nthr = blockDim.x;
    const int row = blockIdx.x;
    const int D = prm.n_det;
    const T* prow = P + (size_t)row * D;

    // ---- stage: inputs de-interleaved by parity (zero padded), taps of both parities ----
    for (int k = tid; k < 2 * prm.x_pitch; k += nthr) {
        const T v = k < D ? prow[k] : T(0);
        if (k & 1) X1[k >> 1] = v; else X0[k >> 1] = v;
    }
    // parity p uses taps q = a - b - (1-p), a in [0, n_ob*blk + R), b in [0, din_pad):
    // local index = a - b + din_pad(p)  =>  global q = local - din_pad(p) - (1-p)
    for (int i = tid; i < 2 * prm.tab_cnt; i += nthr) {
        const int p = i >= prm.tab_cnt;
        const int l = i - p * prm.tab_cnt;
        const int din_pad = p ? prm.de_pad : prm.dn_pad;
        G0[i] = G_gmem[l - din_pad - (1 - p) + prm.tab_off];
    }
    __syncthreads();

    // ---- compute: warp -> (parity, output block, input slice) ----
    const int warp = tid >> 5, lane = tid & 31;
    {
        const int sb = warp % prm.n_sb;
        const int pob = warp / prm.n_sb;
        const int p = pob / prm.n_ob, ob = pob - p * prm.n_ob;
        const int count = p ? prm.dn : prm.de;            // outputs of this parity
        const int din_pad = p ? prm.de_pad : prm.dn_pad;  // inputs have parity 1-p
        const T* Xin = p ? X0 : X1;
        const T* Xown = p ? X1 : X0;
        const T* G = G0 + p * prm.tab_cnt;
        const int a0 = ob * blk + lane * R;
        const int ac = min(a0 + R / 2, max(count - 1, 0));
        const T c = Xown[ac];
        if (sb == 0) Cs[pob * 32 + lane] = c;
        const int per = din_pad / prm.n_sb;               // multiple of R
        const int b_begin = sb * per, b_end = b_begin + per;
        const T* Gw = G + (a0 + din_pad);                 // Gw[r - b] = g[a0 + r - b - (1-p)]

        T acc[R], W[R];
#pragma unroll
        for (int r = 0; r < R; ++r) { acc[r] = T(0); W[r] = Gw[r - b_begin]; }
        for (int b0 = b_begin; b0 < b_end; b0 += R) {
#pragma unroll
            for (int s = 0; s < R; ++s) {
                if (s > 0) W[R - s] = Gw[-(b0 + s)];
                const T x = Xin[b0 + s] - c;
#pragma unroll
                for (int r = 0; r < R; ++r) acc[r] = fma(W[(r - s + R) % R], x, acc[r]);
            }
            W[0] = Gw[-(b0 + R)];
        }
        T* pp = part + (size_t)sb * y_pitch + pob * blk + lane * R;
#pragma unroll
        for (int r = 0; r < R; ++r) pp[r] = acc[r];
    }
    __syncthreads();

    // ---- fixed-order reduction over input slices, centre tap, conditioning term, scale ----
    for (int o = tid; o < y_pitch; o += nthr) {
        const int pob = o / blk;
        const int p = pob / prm.n_ob;
        const int a = o - p * prm.n_ob * blk;
        const int count = p ? prm.dn : prm.de;
        if (a < count) {
            T s = part[o];
            for (int k = 1; k < prm.n_sb; ++k) s += part[(size_t)k * y_pitch + o];
            const int n = 2 * a + p;
            const T c = Cs[pob * 32 + (o - pob * blk) / R];
            const T xn = (p ? X1 : X0)[a];
            Y[o] = (s + T(0.25) * (xn - c) + c * rho[n]) * inv_d;
        }
    }
    __syncthreads();

    // ---- stores: plain row and/or interleaved entries, coalesced ----
    // yz[k] = Q~[k - 1 - guard]: the row in natural order with zero guards (see store_entries)
    T* yz = part + (size_t)prm.n_sb * y_pitch;
    for (int k = tid; k < prm.ent_pitch + 2; k += nthr) {
        const int n = k - 1 - prm.ent_guard;
        yz[k] = (n >= 0 && n < D) ? Y[(n & 1) * prm.n_ob * blk + (n >> 1)] : T(0);
    }
    __syncthreads();
    if (Q) {
        T* q = Q + (size_t)row * D;
        const T* yn = yz + 1 + prm.ent_guard;
        for (int n = tid; n < D; n += nthr) q[n] = yn[n];
    }
    if (E) store_entries<T>(yz, E + (size_t)row * EntryPlanes<T>::value * prm.ent_pitch, prm.ent_pitch, tid, nthr);
}

// Plain filtered rows -> interleaved entries (fbp_backproject's first step); same arithmetic
// as the filter epilogue, so fbp_reconstruct == fbp_backproject(fbp_filter) bit for bit.
template <typename T>
__global__ void __launch_bounds__(256)
entries_kernel(const T* __restrict__ Q, uint4* __restrict__ E, int n_det, int ent_pitch, int ent_guard,
               const T* __restrict__ wrow, int n_angles)
{
    extern __shared__ __align__(16) unsigned char ent_smem_raw[];
    T* yz = reinterpret_cast<T*>(ent_smem_raw);
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // the back-projector may start its prologue
    const int row = blockIdx.x;
    const T* q = Q + (size_t)row * n_det;
    for (int k = threadIdx.x; k < ent_pitch + 2; k += blockDim.x) {
        const int n = k - 1 - ent_guard;
        yz[k] = (n >= 0 && n < n_det) ? q[n] : T(0);
    }
    __syncthreads();
    store_entries<T>(yz, E + (size_t)row * EntryPlanes<T>::value * ent_pitch, ent_pitch, threadIdx.x, blockDim.x,
                     wrow ? wrow + row % n_angles : nullptr);
}

}  // namespace fbp
