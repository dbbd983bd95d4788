// fbp_filter.cuh -- Ram-Lak row filter for sm_100a (Q_theta = P_theta * H).
//
// Q[i][n] = (1/d) * ( h[0] P[i][n] + sum_{odd m} h[m] P[i][n-m] ),  h[0] = 1/4,
// h[m] = -1/(pi^2 m^2) for odd m, 0 for even m != 0 (include/fbp.h).
//
// Only odd taps are non-zero, so an output of parity p reads inputs of parity 1-p only:
// the row splits into two half-size dense Toeplitz products (polyphase form).  With
//   n = 2a + p,  k = 2b + (1-p),  m = n - k = 2q + 1,  q = a - b - (1-p),
//   g[q] := h[2q+1] = -1/(pi^2 (2q+1)^2)
// a thread owns R consecutive same-parity outputs a0..a0+R-1 and walks b = 0..Din-1:
//   acc[r] += g[a0 + r - b - (1-p)] * X[b].
// The R taps it needs at step b are a window that slides by one per step, so the window
// lives in registers (rotating through an R-times unrolled body): one new tap load + one
// broadcast input load per R FMAs.  Lanes of a warp own consecutive output blocks, so the
// tap loads of a warp have stride R words: R is odd => conflict-free.  The input load is
// the same address for the whole warp (broadcast).
//
// One CTA filters `rows_per_cta` rows; each row is served by wpr0 warps for even outputs
// and wpr1 warps for odd outputs.  Rows are staged to shared memory de-interleaved by
// parity (coalesced global reads), results go through a shared row buffer so the global
// stores are coalesced too.  No atomics; every output has one owner; fixed order.
#pragma once
#include <cuda_runtime.h>

namespace fbp {

struct FilterParams {
    int n_rows;        // batch * K
    int n_det;         // D
    int rows_per_cta;
    int wpr0, wpr1;    // warps per row for even / odd outputs
    int de, dn;        // ceil(D/2) even-indexed samples, floor(D/2) odd-indexed samples
    int de_pad, dn_pad;  // padded to a multiple of R (zero filled)
    int tab_len, tab_off;  // tap table: G[idx] = g[idx - tab_off]
    int y_pitch;       // elements per staged output row
};

template <typename T, int R>
__global__ void __launch_bounds__(512)
filter_kernel(const T* __restrict__ P, T* __restrict__ Q, const T* __restrict__ G_gmem,
              FilterParams prm, T inv_d)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* G = reinterpret_cast<T*>(smem_raw);
    const int row_words = prm.de_pad + prm.dn_pad + prm.y_pitch;
    T* rows_base = G + prm.tab_len;

    const int tid = threadIdx.x;
    const int nthr = blockDim.x;
    const int row0 = blockIdx.x * prm.rows_per_cta;
    const int D = prm.n_det;

    // ---- stage taps and rows (coalesced), zero the padding ----
    for (int i = tid; i < prm.tab_len; i += nthr) G[i] = G_gmem[i];
    for (int rl = 0; rl < prm.rows_per_cta; ++rl) {
        const int row = row0 + rl;
        T* X0 = rows_base + (size_t)rl * row_words;   // even-indexed inputs
        T* X1 = X0 + prm.de_pad;                      // odd-indexed inputs
        const bool live = row < prm.n_rows;
        const T* p = P + (size_t)row * D;
        const int span = 2 * (prm.de_pad > prm.dn_pad ? prm.de_pad : prm.dn_pad);
        for (int k = tid; k < span; k += nthr) {
            T v = (live && k < D) ? p[k] : T(0);
            const int b = k >> 1;
            if (k & 1) { if (b < prm.dn_pad) X1[b] = v; }
            else       { if (b < prm.de_pad) X0[b] = v; }
        }
    }
    __syncthreads();

    // ---- compute: warp -> (row slot, parity, block of 32*R outputs) ----
    const int warp = tid >> 5, lane = tid & 31;
    const int wpr = prm.wpr0 + prm.wpr1;
    const int rl = warp / wpr;
    const int wr = warp - rl * wpr;
    if (rl < prm.rows_per_cta && row0 + rl < prm.n_rows) {
        const int p = (wr >= prm.wpr0) ? 1 : 0;
        const int tp = (wr - p * prm.wpr0) * 32 + lane;
        const int count = p ? prm.dn : prm.de;        // outputs of this parity
        const int din_pad = p ? prm.de_pad : prm.dn_pad;  // inputs have parity 1-p
        T* X0 = rows_base + (size_t)rl * row_words;
        T* X1 = X0 + prm.de_pad;
        T* Y = X1 + prm.dn_pad;
        const T* Xin = p ? X0 : X1;
        const T* Xown = p ? X1 : X0;
        const bool active = tp * R < count;
        const int a0 = active ? tp * R : 0;
        // tap index of (r, b): a0 + r - b - (1-p) + tab_off
        const T* Gw = G + (a0 - (1 - p) + prm.tab_off);

        T acc[R], W[R];
#pragma unroll
        for (int r = 0; r < R; ++r) { acc[r] = T(0); W[r] = Gw[r]; }

        for (int b0 = 0; b0 < din_pad; b0 += R) {
#pragma unroll
            for (int s = 0; s < R; ++s) {
                if (s > 0) W[R - s] = Gw[-(b0 + s)];
                const T x = Xin[b0 + s];
#pragma unroll
                for (int r = 0; r < R; ++r) acc[r] = fma(W[(r - s + R) % R], x, acc[r]);
            }
            W[0] = Gw[-(b0 + R)];
        }
        if (active) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int a = a0 + r;
                if (a < count) Y[2 * a + p] = (acc[r] + T(0.25) * Xown[a]) * inv_d;
            }
        }
    }
    __syncthreads();

    // ---- coalesced store ----
    for (int rl2 = 0; rl2 < prm.rows_per_cta; ++rl2) {
        const int row = row0 + rl2;
        if (row >= prm.n_rows) break;
        const T* Y = rows_base + (size_t)rl2 * row_words + prm.de_pad + prm.dn_pad;
        T* q = Q + (size_t)row * D;
        for (int n = tid; n < D; n += nthr) q[n] = Y[n];
    }
}

}  // namespace fbp
