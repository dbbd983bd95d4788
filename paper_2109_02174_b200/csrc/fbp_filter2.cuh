// fbp_filter2.cuh -- Ram-Lak row filter for sm_100a, paired-parity form (Q = P * H).
//
// Q[i][n] = (1/d) ( h[0] P[i][n] + sum_{odd m} h[m] P[i][n-m] ),  h[0] = 1/4, h[m] = -1/(pi^2 m^2).
// With g[q] := h[2q+1] (any integer q), an output pair (n = 2a+1, n = 2a) and an input pair
// (k = 2b, k = 2b+1):      Q[2a+1] += g[a-b]   * P[2b]        (odd output  <- even input)
//                           Q[2a]   += g[a-b-1] * P[2b+1]      (even output <- odd input)
// i.e. ONE packed multiply-add of the tap pair (g[a-b], g[a-b-1]) with the input pair as it lies
// in memory.  A thread owns R consecutive output pairs a0..a0+R-1 and walks b; the R tap pairs it
// needs slide by one pair per step and live in registers (rotating through an R-times unrolled
// body).  Per step: one tap-pair load, one broadcast input-pair load, one packed subtract and R
// packed FMAs (fp32: FFMA2 = fma.rn.f32x2, which leaves issue slots free for the loads; fp64:
// two DFMA).  Tap pairs start at alternating word parity, so the reversed table U[j] = g[J0 - j]
// is staged twice, UA[j] = U[j] and UB[j] = U[j+1]; both copies are then read with aligned
// 2-element loads, lane stride R elements (R = 2 mod 4 => conflict-free).
//
// Conditioning (fp32 accuracy): 1/4 P[n] cancels against sum |h[m]| P[n-m]; each thread
// subtracts c (the input at the centre of its outputs) from every input and the epilogue adds
// c * rho[n] back, rho = the filter's response to a constant row over the padded input range
// (host, fp64).  The running sums then hold differences of neighbouring samples times taps.
//
// Work decomposition.  Persistent CTAs loop over rows (taps staged once per CTA, the next row
// prefetched with cp.async while the current one is filtered).  Warp (ob, sb) owns output block
// ob (32*R output pairs) and slice sb of the input pairs; the SB partial sums are added in fixed
// order by one owner thread per output: no atomics, deterministic.  The epilogue writes the plain
// row (fbp_filter) and/or the back-projector's entries (fbp_reconstruct; fbp_filter.cuh).
#pragma once
#include <cuda_runtime.h>

#include "fbp_filter.cuh"  // store_entries, EntryPlanes

namespace fbp {

struct Filter2Params {
    int n_rows;            // batch * K
    int n_det;             // D
    int n_ob;              // output blocks of 32*R pairs
    int n_sb;              // input slices SB
    int a_tot;             // n_ob * 32 * R output pairs (padded)
    int n_chunks;          // ceil(ceil(D/2) / R) chunks of R input pairs
    int b_pad;             // n_chunks * R input pairs (zero padded)
    int tab_len;           // elements per tap-table copy (multiple of 4); gmem holds UA | UB
    int ent_pitch, ent_guard;
};

// ---- a pair of T with packed arithmetic --------------------------------------------------
template <typename T> struct Pair2;
template <> struct Pair2<float> {
    unsigned long long v;
    __device__ __forceinline__ static Pair2 load(const float* p)
    {
        Pair2 r; r.v = *reinterpret_cast<const unsigned long long*>(p); return r;
    }
    __device__ __forceinline__ static Pair2 splat(float c)
    {
        Pair2 r; asm("mov.b64 %0, {%1, %1};" : "=l"(r.v) : "f"(c)); return r;
    }
    __device__ __forceinline__ static Pair2 zero() { Pair2 r; r.v = 0ull; return r; }
    __device__ __forceinline__ void fma(Pair2 a, Pair2 b) { asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(v) : "l"(a.v), "l"(b.v)); }
    __device__ __forceinline__ Pair2 plus(Pair2 b) const { Pair2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(v), "l"(b.v)); return r; }
    __device__ __forceinline__ float lo() const { return __uint_as_float((unsigned)(v & 0xffffffffull)); }
    __device__ __forceinline__ float hi() const { return __uint_as_float((unsigned)(v >> 32)); }
};
template <> struct Pair2<double> {
    double x, y;
    __device__ __forceinline__ static Pair2 load(const double* p)
    {
        const double2 t = *reinterpret_cast<const double2*>(p); Pair2 r; r.x = t.x; r.y = t.y; return r;
    }
    __device__ __forceinline__ static Pair2 splat(double c) { Pair2 r; r.x = c; r.y = c; return r; }
    __device__ __forceinline__ static Pair2 zero() { Pair2 r; r.x = 0.0; r.y = 0.0; return r; }
    __device__ __forceinline__ void fma(Pair2 a, Pair2 b) { x = ::fma(a.x, b.x, x); y = ::fma(a.y, b.y, y); }
    __device__ __forceinline__ Pair2 plus(Pair2 b) const { Pair2 r; r.x = x + b.x; r.y = y + b.y; return r; }
    __device__ __forceinline__ double lo() const { return x; }
    __device__ __forceinline__ double hi() const { return y; }
};

// ---- cp.async (LDGSTS): element-sized for unaligned rows, 16 bytes for the tap tables ----
template <int BYTES>
__device__ __forceinline__ void cp_async(void* smem_dst, const void* gmem_src)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    if (BYTES == 16)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
    else
        asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(d), "l"(gmem_src), "n"(BYTES) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// programmatic dependent launch: let the next kernel of the stream start its prologue
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

#ifdef FBP_TRACE
#define FBP_TRACE_MARK(slot) do { if (threadIdx.x == 0 && blockIdx.x < 4096) g_trace[blockIdx.x * 16 + (slot)] = trace_now(); } while (0)
#else
#define FBP_TRACE_MARK(slot) do { } while (0)
#endif

// U_gmem: [tab_copies][2][tab_len] = UA | UB (see above), U[j] = g[a_tot - 1 - j]; CTAs read replica
// blockIdx % tab_copies (every CTA stages the same table at the same moment: one copy is an L2 hot spot).  rho: [D].
// Block = n_ob * n_sb warps.  Grid <= number of co-resident CTAs (persistent).
//
// DENSE = true is the general form for apodised windows (every tap non-zero; SURVEY.md 8(f) row 1,
// the paper's H is generic): input k (splat) meets the tap pair (H[2a+1-k], H[2a-k])
// of output pair a, U[j] = H[2 a_tot - j], pair index j = 2 a_tot - 1 - 2a + k.  The pairs of even and
// of odd k form two register windows that each slide by one slot every second step; lane stride
// is 2R words, so R is odd.  Twice the multiply-adds of the Ram-Lak form (twice the taps).
// wrow: per-row multipliers of the entries (fbp_set_angle_weights), NULL = none.
template <typename T, int R, bool DENSE>
__global__ void __launch_bounds__(512)
filter2_kernel(const T* __restrict__ P, T* __restrict__ Q, uint4* __restrict__ E,
               const T* __restrict__ U_gmem, const T* __restrict__ rho, const T* __restrict__ wrow,
               int n_angles, Filter2Params prm, T inv_d, int tab_copies)
{
    static_assert(DENSE ? (R % 2 == 1) : (R % 4 == 2), "lane stride (R or 2R words) must be 2 mod 4: conflict-free pair loads");
    using P2 = Pair2<T>;
    extern __shared__ __align__(16) unsigned char f2_smem_raw[];
    // layout: UA[tab_len] UB[tab_len] X[2][2*b_pad] C[n_ob*32] part[n_sb][2*a_tot] yz[ent_pitch+2] rho[D]
    T* UA = reinterpret_cast<T*>(f2_smem_raw);
    T* UB = UA + prm.tab_len;
    T* X0 = UB + prm.tab_len;
    const int x_len = 2 * prm.b_pad;
    T* Cs = X0 + 2 * x_len;
    T* part = Cs + prm.n_ob * 32;
    const int y_len = 2 * prm.a_tot;
    T* yz = part + (size_t)prm.n_sb * y_len;
    T* rho_s = yz + prm.ent_pitch + 2;

    pdl_launch_dependents();   // every CTA of this grid is resident: dependents may take what is left
    FBP_TRACE_MARK(0);

    const int tid = threadIdx.x, nthr = blockDim.x;
    const int D = prm.n_det;
    const int warp = tid >> 5, lane = tid & 31;
    const int sb = warp % prm.n_sb, ob = warp / prm.n_sb;

    // ---- once per CTA: tap tables, zero padding of both input buffers, first row ----
    {
        const T* Ug = U_gmem + (size_t)(blockIdx.x % tab_copies) * 2 * prm.tab_len;
        for (int i = tid * (16 / (int)sizeof(T)); i < 2 * prm.tab_len; i += nthr * (16 / (int)sizeof(T)))
            cp_async<16>(UA + i, Ug + i);
    }
    for (int k = D + tid; k < x_len; k += nthr) { X0[k] = T(0); X0[x_len + k] = T(0); }
#ifdef FBP_TRACE
    cp_async_commit();         // tables in their own group, to time them apart from the row
#endif
    int row = blockIdx.x;
    if (row < prm.n_rows) {
        const T* prow = P + (size_t)row * D;
        for (int k = tid; k < D; k += nthr) cp_async<(int)sizeof(T)>(X0 + k, prow + k);
    }
    cp_async_commit();
    // the conditioning term is needed only by the reduction: its own group, waited for there
    for (int k = tid; k < D; k += nthr) cp_async<(int)sizeof(T)>(rho_s + k, rho + k);
    cp_async_commit();

    // per-thread constants
    const int a0 = (ob * 32 + lane) * R;                 // first output pair of this thread
    const int cl = (DENSE ? 2 * prm.a_tot - 1 - 2 * a0    // odd: U index of (a0, k = 0)
                          : prm.a_tot - 1 - a0);          // odd: U index of (a0, b = 0)
    const T* ua = UA + cl;                               // pair at even U index j: ua[j - cl]
    const T* ub = UB + cl - 1;                           // pair at odd  U index j: ub[j - cl]
    const int a_max = (D - 1) >> 1;
    const int ac = min(a0 + R / 2, a_max);
    const int ch_begin = (int)(((long long)sb * prm.n_chunks) / prm.n_sb);
    const int ch_end = (int)(((long long)(sb + 1) * prm.n_chunks) / prm.n_sb);

    for (int it = 0; row < prm.n_rows; row += gridDim.x, ++it) {
        T* X = X0 + (it & 1) * x_len;
        {   // prefetch the next row of this CTA into the other buffer
            const int nxt = row + gridDim.x;
            if (nxt < prm.n_rows) {
                T* Xn = X0 + ((it + 1) & 1) * x_len;
                const T* prow = P + (size_t)nxt * D;
                for (int k = tid; k < D; k += nthr) cp_async<(int)sizeof(T)>(Xn + k, prow + k);
            }
            cp_async_commit();
        }
#ifdef FBP_TRACE
        if (it == 0) { cp_async_wait<3>(); __syncthreads(); FBP_TRACE_MARK(5); }
#endif
        if (it == 0) cp_async_wait<2>();   // taps and row 0 (rho and the prefetch may still be in flight)
        else cp_async_wait<1>();           // everything but the prefetch just issued has landed
        __syncthreads();
        FBP_TRACE_MARK(1);

        // ---- compute: R output pairs x this warp's slice of the inputs (chunks of 2R inputs) ----
        {
            const T c = X[2 * ac];
            if (sb == 0) Cs[ob * 32 + lane] = c;
            const P2 nc = P2::splat(-c);
            P2 acc[R];
#pragma unroll
            for (int r = 0; r < R; ++r) acc[r] = P2::zero();
            if (!DENSE) {
                P2 W[R];
                const int b_begin = ch_begin * R;
#pragma unroll
                for (int r = 0; r < R; ++r)   // U index cl - r + b_begin: even for odd r (UA), odd for even r (UB)
                    W[r] = (r & 1) ? P2::load(ua + (b_begin - r)) : P2::load(ub + (b_begin - r));
                for (int ch = ch_begin; ch < ch_end; ++ch) {
                    const int b0 = ch * R;
#pragma unroll
                    for (int s = 0; s < R; ++s) {
                        // the pair of (r = 0, b = b0 + s): U index cl + b0 + s, even iff s odd
                        if (s > 0) W[R - s] = (s & 1) ? P2::load(ua + (b0 + s)) : P2::load(ub + (b0 + s));
                        const P2 x = P2::load(X + 2 * (b0 + s)).plus(nc);
#pragma unroll
                        for (int r = 0; r < R; ++r) acc[r].fma(W[(r - s + R) % R], x);
                    }
                    W[0] = P2::load(ub + (b0 + R));
                }
            } else {
                P2 WE[R], WO[R];
                const int k_begin = ch_begin * 2 * R;
#pragma unroll
                for (int r = 0; r < R; ++r) {     // U index cl - 2r + k: odd for even k (UB), even for odd k (UA)
                    WE[r] = P2::load(ub + (k_begin - 2 * r));
                    WO[r] = P2::load(ua + (k_begin + 1 - 2 * r));
                }
                for (int ch = ch_begin; ch < ch_end; ++ch) {
                    const int k0 = ch * 2 * R;
#pragma unroll
                    for (int s = 0; s < R; ++s) {
                        if (s > 0) {
                            WE[R - s] = P2::load(ub + (k0 + 2 * s));
                            WO[R - s] = P2::load(ua + (k0 + 2 * s + 1));
                        }
                        const P2 x = P2::load(X + (k0 + 2 * s)).plus(nc);
                        const P2 xe = P2::splat(x.lo()), xo = P2::splat(x.hi());
#pragma unroll
                        for (int r = 0; r < R; ++r) acc[r].fma(WE[(r - s + R) % R], xe);
#pragma unroll
                        for (int r = 0; r < R; ++r) acc[r].fma(WO[(r - s + R) % R], xo);
                    }
                    WE[0] = P2::load(ub + (k0 + 2 * R));
                    WO[0] = P2::load(ua + (k0 + 2 * R + 1));
                }
            }
            // natural order: n = 2(a0+r) is the even output (hi), n+1 the odd output (lo)
            T* pp = part + (size_t)sb * y_len + 2 * a0;
#pragma unroll
            for (int r = 0; r < R; ++r) { pp[2 * r] = acc[r].hi(); pp[2 * r + 1] = acc[r].lo(); }
        }
        if (it == 0) cp_async_wait<1>();   // rho
        __syncthreads();
        FBP_TRACE_MARK(2);

        // ---- fixed-order reduction over input slices, centre tap, conditioning term, scale ----
        // yz[k] = Q~[k - 1 - guard]: the row in natural order with zero guards (store_entries)
        for (int k = tid; k < prm.ent_pitch + 2; k += nthr) {
            const int n = k - 1 - prm.ent_guard;
            T y = T(0);
            if (n >= 0 && n < D) {
                T s = part[n];
                for (int q = 1; q < prm.n_sb; ++q) s += part[(size_t)q * y_len + n];
                const T c = Cs[(n >> 1) / R];
                y = DENSE ? (s + c * rho_s[n]) * inv_d                      // the centre tap is in the sum
                          : (s + T(0.25) * (X[n] - c) + c * rho_s[n]) * inv_d;
            }
            yz[k] = y;
        }
        __syncthreads();
        FBP_TRACE_MARK(3);

        // ---- stores: plain row and/or interleaved entries, coalesced ----
        if (Q) {
            T* q = Q + (size_t)row * D;
            const T* yn = yz + 1 + prm.ent_guard;
            for (int n = tid; n < D; n += nthr) q[n] = yn[n];
        }
        if (E) store_entries<T>(yz, E + (size_t)row * EntryPlanes<T>::value * prm.ent_pitch, prm.ent_pitch, tid, nthr,
                                wrow ? wrow + row % n_angles : nullptr);
    }
    cp_async_wait<0>();
    __syncthreads();
    FBP_TRACE_MARK(4);
}

}  // namespace fbp
