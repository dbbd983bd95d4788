// fbp_filter3.cuh -- direct-form row filter for sm_100a in "mirrored units" (Q = P * H).
//
// Q[i][n] = (1/d) sum_k h[n-k] P[i][k].  Ram-Lak (h[0] = 1/4, h[odd m] = -1/(pi^2 m^2), else 0) runs the
// paired-parity form: with g[q] := h[2q+1], an output pair (2a+1, 2a) and an input pair (2b, 2b+1),
//     Q[2a+1] += g[a-b] * P[2b]          Q[2a] += g[a-b-1] * P[2b+1]
// is ONE packed multiply-add (fp32: FFMA2) of the tap pair (g[a-b], g[a-b-1]) with the input pair as it
// lies in memory.  A thread owns R consecutive output pairs ("a group") and walks b; its R tap pairs slide
// by one pair per step and live in registers (rotating through an R-times unrolled body): per step one
// tap-pair load, one broadcast input-pair load, one packed subtract, R packed FMAs.  Tap pairs start at
// alternating word parity, so the reversed table U[j] = g[a_hi - 1 - j] is staged twice (UA[j] = U[j],
// UB[j] = U[j+1]) and both are read with aligned 2-element loads; lane stride R elements, R = 2 mod 4,
// is conflict-free within each half-warp.  DENSE = true is the general form for apodised windows (every tap
// non-zero; fbp_set_window): input k (splat) meets the tap pair (H[2a+1-k], H[2a-k]), U[j] = H[2 a_hi - j].
//
// Work decomposition: one CTA filters one UNIT of a row at a time; its SB warps split the input range and
// their partial sums are added in fixed order (no atomics, deterministic).  A unit is one warp-width of
// output groups chosen so that everything the back-projector's entries need is local to the CTA:
//   - groups are cut on two grids: the LEFT grid from output 0 upward, [2R g, 2R (g+1)), used for outputs
//     n < M, and the RIGHT grid from D' = D rounded up to a multiple of 4 downward, [D' - 2R (g+1), D' - 2R g), used
//     for n >= M (M even, about D/2).  Every output has ONE canonical group, hence one conditioning
//     constant and one summation order, whichever unit computes it: units may recompute a neighbour's
//     group and get the same bits.
//   - lanes 0..15 of unit u take left groups 15u .. 15u+15, lanes 16..31 right groups 15u+15 .. 15u
//     (ascending outputs).  An outer unit owns 15 groups per side and recomputes one neighbour group per
//     side (the entry of detector interval j needs Q[j], Q[j+1] and, for the mirror pixel of the
//     back-projector, Q[D-2-j], Q[D-1-j]); the innermost unit owns all 16 per side and contains M.
// So a row is U = 1 + ceil(max(0, M - 32R) / 30R) independent units (2 at D = 725, R = 6): 720 CTAs of 4
// warps for one 360-row sinogram, 4.9 per SM, instead of 360 whole-row CTAs (2.4 per SM, 3 on the busiest).
//
// Conditioning (fp32 accuracy): 1/4 P[n] cancels against sum |h[m]| P[n-m]; each thread subtracts c (the
// input at the centre of its group) from every input and the epilogue adds c * rho[n] back, rho = the
// filter's response to a constant row over the padded input range (host, fp64).
//
// Outputs: the plain row (fbp_filter) and/or the back-projector's entries (fbp_reconstruct;
// fbp_entries.cuh).
//
// Staging.  Tables and rows arrive by TMA bulk copies (cp.async.bulk, completion on an mbarrier) issued by one
// thread: three instructions per CTA instead of ~60 warp-level cp.async.  That matters for a small launch
// (one 360-row sinogram is a single wave of 720 CTAs, five per SM): with per-thread cp.async the load/store
// unit, which the arithmetic loop of the CTAs that are already computing keeps busy with shared-memory loads,
// let the last CTA of every SM finish issuing its loads only when the others were done (fbp_set_trace:
// staged after 5.1 us instead of 1.8).  A row starts at any multiple of the element size, a bulk copy at a
// multiple of 16 bytes: the 16-byte-aligned superset of the row lands in XB and is moved down to X (whose
// pairs must be aligned) by a shared-to-shared copy; elements that the aligned superset would take from
// beyond the end of the sinogram are fetched with plain loads.  A persistent CTA prefetches its next row into
// the other XB buffer while it filters the current one.
#pragma once
#include <cuda_runtime.h>

#include "fbp_entries.cuh"
#include "fbp_ptx.cuh"

namespace fbp {

struct Filter3Params {
    int n_rows;            // batch * K
    int n_det;             // D
    int d_even;            // D' = D rounded up to a multiple of 4 (right-grid groups start at even pairs)
    int m_split;           // M: outputs n < M belong to the left grid, n >= M to the right grid (even)
    int n_units;           // U units per row
    int n_sb;              // SB warps per CTA = input slices
    int n_chunks;          // chunks of R input pairs (sparse) / 2R inputs (dense)
    int b_pad;             // n_chunks * R input pairs (zero padded)
    int a_hi;              // pair index bound: U index of (pair a, input 0) is a_hi - 1 - a (dense: 2 a_hi - 1 - 2a)
    int tab_len;           // elements per tap-table copy (multiple of 4); gmem holds UA | UB
    int ent_pitch, ent_guard;
    unsigned long long* trace;   // fbp_set_trace: [grid][8] %globaltimer marks of each CTA's first unit, or NULL
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

// U_gmem: [2][tab_len] = UA | UB.  rho: [D rounded up to 16 bytes].  wrow: per-row multipliers of the entries (fbp_set_angle_weights) or NULL.
// Block = 32 * n_sb threads.  Grid <= number of co-resident CTAs (persistent loop over units).
template <typename T, int R, bool DENSE>
__global__ void __launch_bounds__(256)
filter3_kernel(const T* __restrict__ P, T* __restrict__ Q, uint4* __restrict__ E,
               const T* __restrict__ U_gmem, const T* __restrict__ rho, const T* __restrict__ wrow,
               int n_angles, Filter3Params prm, T inv_d)
{
    static_assert(DENSE ? (R % 2 == 1) : (R % 4 == 2), "lane stride (R or 2R words) must be 2 mod 4: conflict-free pair loads");
    using P2 = Pair2<T>;
    constexpr int W2 = 2 * R;            // outputs per group
    constexpr int HALF = 16 * W2;        // outputs per side of a unit
    extern __shared__ __align__(16) unsigned char f3_smem_raw[];
    // layout: bar[2] (16 B) | UA[tab_len] UB[tab_len] | rho[D4] | XB[2][xb_len] | X[x_len] | part[n_sb][2 HALF] | Qs[2 HALF] | Cs[32]
    constexpr int V = 16 / (int)sizeof(T);           // elements per 16 bytes
    const int D = prm.n_det, D4 = (D + V - 1) / V * V;
    const int xb_len = D4 + 2 * V;                    // the aligned superset of a row: up to V-1 elements before, V after
    const int x_len = 2 * prm.b_pad;
    const unsigned bar0 = smem_u32(f3_smem_raw);
    T* UA = reinterpret_cast<T*>(f3_smem_raw + 16);
    T* UB = UA + prm.tab_len;
    T* rho_s = UB + prm.tab_len;
    T* XB = rho_s + D4;
    T* X = XB + 2 * xb_len;
    T* part = X + x_len;
    T* Qs = part + (size_t)prm.n_sb * 2 * HALF;
    T* Cs = Qs + 2 * HALF;

    pdl_launch_dependents();   // every CTA of this grid is resident: dependents may take what is left
    trace_mark(prm.trace, blockIdx.x, 0);

    const int tid = threadIdx.x, nthr = blockDim.x;
    const int Uu = prm.n_units, M = prm.m_split;
    const int sb = tid >> 5, lane = tid & 31;
    const long long n_work = (long long)prm.n_rows * Uu;
    const uintptr_t p_end = reinterpret_cast<uintptr_t>(P) + (size_t)prm.n_rows * D * sizeof(T);   // one past the sinogram

    // One thread issues the bulk copy of row `r` into landing buffer `buf`; `extra` more bytes (the tables) are
    // expected on the same barrier.  The copy covers [row start rounded down to 16 B, row end rounded up), cut
    // at the last 16-byte boundary inside the sinogram.
    auto issue_row = [&](int r, int buf, unsigned extra) {
        const uintptr_t beg = reinterpret_cast<uintptr_t>(P + (size_t)r * D);
        const uintptr_t al = beg & ~(uintptr_t)15;
        uintptr_t end = (beg + (size_t)D * sizeof(T) + 15) & ~(uintptr_t)15;
        if (end > p_end) end = p_end & ~(uintptr_t)15;
        const unsigned bytes = end > al ? (unsigned)(end - al) : 0u;
        mbar_arrive_expect_tx(bar0 + 8u * buf, bytes + extra);
        if (bytes) tma_load_1d(smem_u32(XB + (size_t)buf * xb_len), reinterpret_cast<const void*>(al), bytes, bar0 + 8u * buf);
    };

    // ---- once per CTA: barriers, tap tables, conditioning term, first row; zero padding of X ----
    long long unit = blockIdx.x;
    if (tid == 0) {
        mbar_init(bar0, 1);
        mbar_init(bar0 + 8u, 1);
        fence_mbar_init();
        const unsigned tab_bytes = 2u * prm.tab_len * sizeof(T), rho_bytes = (unsigned)D4 * sizeof(T);
        if (unit < n_work) issue_row((int)(unit / Uu), 0, tab_bytes + rho_bytes);
        else mbar_arrive_expect_tx(bar0, tab_bytes + rho_bytes);
        tma_load_1d(smem_u32(UA), U_gmem, tab_bytes, bar0);
        tma_load_1d(smem_u32(rho_s), rho, rho_bytes, bar0);
    }
    for (int k = D + tid; k < x_len; k += nthr) X[k] = T(0);
    __syncthreads();           // barrier init visible to the waiters

    const int a_max = (D - 1) >> 1;
    const int ch_begin = (int)(((long long)sb * prm.n_chunks) / prm.n_sb);
    const int ch_end = (int)(((long long)(sb + 1) * prm.n_chunks) / prm.n_sb);

    for (int it = 0; unit < n_work; unit += gridDim.x, ++it) {
        const int row = (int)(unit / Uu), u = (int)(unit - (long long)row * Uu);
        const int buf = it & 1;
        // prefetch the row of this CTA's next unit into the other landing buffer (its last reader, the move
        // below in iteration it - 1, is behind a __syncthreads)
        if (tid == 0 && unit + gridDim.x < n_work) issue_row((int)((unit + gridDim.x) / Uu), buf ^ 1, 0u);
        mbar_wait(bar0 + 8u * buf, (unsigned)((it >> 1) & 1));
        {   // landing buffer -> X: the row starts `mis` elements into the aligned superset
            const uintptr_t beg = reinterpret_cast<uintptr_t>(P + (size_t)row * D);
            const int mis = (int)((beg & 15) / sizeof(T));
            uintptr_t end = (beg + (size_t)D * sizeof(T) + 15) & ~(uintptr_t)15;
            if (end > p_end) end = p_end & ~(uintptr_t)15;
            const long long got = ((long long)end - (long long)(beg & ~(uintptr_t)15)) / (long long)sizeof(T) - mis;   // elements of the row that landed
            const int covered = (int)(got < 0 ? 0 : (got > D ? D : got));
            const T* xb = XB + (size_t)buf * xb_len + mis;
            for (int k = tid; k < covered; k += nthr) X[k] = xb[k];
            const T* prow = P + (size_t)row * D;
            for (int k = covered + tid; k < D; k += nthr) X[k] = prow[k];
        }
        // first outputs of the two blocks of this unit (both even) and this thread's first pair
        const int nL0 = 15 * W2 * u, nR0 = prm.d_even - 15 * W2 * u - HALF;
        const int a0 = (lane < 16 ? nL0 + lane * W2 : nR0 + (lane - 16) * W2) / 2;   // exact: all terms even; may be < 0
        const int cl = DENSE ? 2 * prm.a_hi - 1 - 2 * a0 : prm.a_hi - 1 - a0;         // odd U index of (a0, input 0)
        const T* ua = UA + cl;                               // pair at even U index j: ua[j - cl]
        const T* ub = UB + cl - 1;                           // pair at odd  U index j: ub[j - cl]
        const int ac = min(max(a0 + R / 2, 0), a_max);
        __syncthreads();
        if (it == 0) trace_mark(prm.trace, blockIdx.x, 1);     // tables and row staged

        // ---- compute: R output pairs x this warp's slice of the inputs ----
        {
            const T c = X[2 * ac];
            if (sb == 0) Cs[lane] = c;
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
            T* pp = part + (size_t)sb * 2 * HALF + lane * W2;
#pragma unroll
            for (int r = 0; r < R; ++r) { pp[2 * r] = acc[r].hi(); pp[2 * r + 1] = acc[r].lo(); }
        }
        __syncthreads();
        if (it == 0) trace_mark(prm.trace, blockIdx.x, 2);     // partial sums done

        // ---- fixed-order reduction over input slices, centre tap, conditioning term, scale ----
        // Qs[o]: o < HALF is output nL0 + o (canonical iff below M), else output nR0 + o - HALF (iff >= M)
        for (int o = tid; o < 2 * HALF; o += nthr) {
            const bool left = o < HALF;
            const int n = left ? nL0 + o : nR0 + (o - HALF);
            T y = T(0);
            if (n >= 0 && n < D && (left ? n < M : n >= M)) {
                T s = part[o];
                for (int q = 1; q < prm.n_sb; ++q) s += part[(size_t)q * 2 * HALF + o];
                const T c = Cs[o / W2];
                y = DENSE ? (s + c * rho_s[n]) * inv_d                                // the centre tap is in the sum
                          : (s + T(0.25) * (X[n] - c) + c * rho_s[n]) * inv_d;
            }
            Qs[o] = y;
        }
        __syncthreads();
        if (it == 0) trace_mark(prm.trace, blockIdx.x, 3);     // row reduced

        // ---- stores: owned outputs of the plain row and/or owned entries ----
        const bool inner = (u == Uu - 1);
        if (Q) {
            T* q = Q + (size_t)row * D;
            const int l_end = inner ? M : nL0 + 15 * W2;            // left outputs [nL0, l_end)
            const int r_beg = inner ? M : nR0 + W2;                  // right outputs [r_beg, nR0 + HALF)
            for (int o = tid; o < 2 * HALF; o += nthr) {
                const bool left = o < HALF;
                const int n = left ? nL0 + o : nR0 + (o - HALF);
                if (n < D && (left ? n < l_end : n >= r_beg)) q[n] = Qs[o];
            }
        }
        if (E) {
            // zero-extended row through the two blocks: canonical side by M
            auto q_at = [&](int n) -> T {
                if (n < 0 || n >= D) return T(0);
                return n < M ? Qs[n - nL0] : Qs[HALF + n - nR0];
            };
            // intervals j = -1 .. D-1 pair up as (j, D-2-j); this unit owns the left members
            // j in [j_beg, j_end) and writes both entries of each pair
            const int j_beg = u == 0 ? -1 : nL0;
            const int j_end = inner ? D / 2 : nL0 + 15 * W2;        // floor(D/2) = number of left members >= 0
            uint4* erow = E + (size_t)row * prm.ent_pitch;
            const bool scaled = wrow != nullptr;
            const T m = scaled ? wrow[row % n_angles] : T(1);
            for (int j = j_beg + tid; j < j_end; j += nthr) {
                const int jm = D - 2 - j;
                T a0v = q_at(j), a1v = q_at(j + 1), b0v = q_at(jm), b1v = q_at(jm + 1);
                if (scaled) { a0v *= m; a1v *= m; b0v *= m; b1v *= m; }
                store_entry(erow, j + prm.ent_guard, a0v, a1v, b0v, b1v);
                if (jm != j) store_entry(erow, jm + prm.ent_guard, b0v, b1v, a0v, a1v);
            }
        }
    }
    trace_mark(prm.trace, blockIdx.x, 4);                      // last unit stored
}

}  // namespace fbp
