// fbp_backproject.cuh -- pixel-driven gather back-projection for sm_100a (eq. 2).
//
// f[r][c] = (pi/K) sum_i lerp(Q~_i, u_i),  u_i = (x cos_i + y sin_i)/d + (D-1)/2.
//
// Point symmetry.  The image grid and the detector are both centred, so the pixel (-x,-y)
// has u' = (D-1) - u at every angle: if u = j + 1/2 + w (w in [-1/2,1/2]) then the mirror
// pixel reads interval D-2-j with offset -w.  One thread therefore owns R pixels of the top
// half of the image AND their R mirror pixels, computes (j, w) once, and fetches both
// interpolation operands with ONE 16-byte (fp32) shared-memory load of the entry
//   E[i][j] = ( mid[j], mid[D-2-j], slope[j], -slope[D-2-j] ),
//   mid[j] = (Q~[j]+Q~[j+1])/2,  slope[j] = Q~[j+1]-Q~[j],  Q~ = 0 outside [0, D-1]
// so that  value = mid_a + w slope_a  and  mirror value = mid_b + w nslope_b.
// The entries are produced by the filter epilogue (fbp_reconstruct) or entries_kernel
// (fbp_backproject) into a plan-owned buffer [batch][K][pitch] with >= L+1 zero guard
// entries on both sides.
//
// A CTA owns a tile of 32 x (WY*R) primary pixels and a contiguous range of angles (split s
// of S).  Angles are processed in chunks; for each angle of a chunk lane a of warp 0
// computes, in fp64, the tile-local base b = u(tile origin) - j0 - 1/2 (fp32 coordinates
// stay below 64: ulp <= 3.8e-6) and issues one TMA bulk copy (cp.async.bulk, completion on an
// mbarrier) of the L entries starting at j0 into shared memory.
// Per update pair:  u' = b + lx cos + ly sin;  t = u' + M (M = 1.5*2^23 | 1.5*2^52, round to
// nearest);  e = bits(t) - bits(M);  w = u' - (t - M);  one LDS.128;  2 FMA + 2 ADD.
// A tie in the rounding picks either neighbouring interval with the same interpolated value.
// One owner per pixel, ascending angles, no atomics => bit-identical runs.  With S > 1 the S
// partial images go to scratch and reduce_kernel adds them in fixed order s = 0..S-1.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

#include "fbp_filter.cuh"  // BpEntry

namespace fbp {

struct BpParams {
    int n_angles, n_det, image_n;
    int half_rows;       // ceil(N/2): rows of the primary (top) half
    int tiles_x, tiles_y;
    int n_splits;        // S
    int chunk;           // angles staged per chunk (A)
    int seg_len;         // L entries per angle
    int ent_pitch, ent_guard;
    double c_n, c_d;     // (N-1)/2, (D-1)/2
    double scale;        // pi / K
};

template <typename T> struct Magic;
template <> struct Magic<float> {
    __device__ static float m() { return 12582912.0f; }  // 1.5 * 2^23
    __device__ static unsigned bits(float t) { return __float_as_uint(t); }
    static constexpr unsigned kBits = 0x4B400000u;
};
template <> struct Magic<double> {
    __device__ static double m() { return 6755399441055744.0; }  // 1.5 * 2^52
    __device__ static unsigned bits(double t) { return (unsigned)__double2loint(t); }
    static constexpr unsigned kBits = 0u;
};

template <typename T> struct alignas(4 * sizeof(T)) AngleRec { T c, s, b, pad; };

// ---- PTX wrappers: shared-space addresses, mbarrier, TMA 1-D bulk copy ----------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void fence_mbar_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_1d(unsigned dst, const void* src, unsigned bytes, unsigned bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

template <typename T> struct EntryLoad;
template <> struct EntryLoad<float> {
    __device__ static void ld(unsigned addr, float& ma, float& mb, float& sa, float& sb)
    {
        asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(ma), "=f"(mb), "=f"(sa), "=f"(sb) : "r"(addr));
    }
};
template <> struct EntryLoad<double> {
    __device__ static void ld(unsigned addr, double& ma, double& mb, double& sa, double& sb)
    {
        asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(ma), "=d"(mb) : "r"(addr));
        asm volatile("ld.shared.v2.f64 {%0,%1}, [%2+16];" : "=d"(sa), "=d"(sb) : "r"(addr));
    }
};

// cs2: [K] pairs (cos*pix/d, sin*pix/d) in fp64.  E: entries [batch][K][ent_pitch].
// out: image (S == 1, scaled) or partial buffer [S][batch][N][N] (S > 1, unscaled).
template <typename T, int R, int WY>
__global__ void __launch_bounds__(32 * WY)
backproject_kernel(const BpEntry<T>* __restrict__ E, T* __restrict__ out, const double2* __restrict__ cs2,
                   BpParams prm, int batch)
{
    constexpr int TH = WY * R;
    constexpr int ESZ = (int)sizeof(BpEntry<T>);
    extern __shared__ __align__(128) unsigned char bp_smem_raw[];
    // layout: mbarrier (16 B) | rec[chunk] | seg[chunk][L]
    const unsigned bar = smem_u32(bp_smem_raw);
    AngleRec<T>* rec = reinterpret_cast<AngleRec<T>*>(bp_smem_raw + 16);
    unsigned char* seg_ptr = bp_smem_raw + 16 + (size_t)prm.chunk * sizeof(AngleRec<T>);
    seg_ptr += (128 - (reinterpret_cast<uintptr_t>(seg_ptr) & 127)) & 127;
    const unsigned seg = smem_u32(seg_ptr);

    const int tid = threadIdx.x, lane = tid & 31, wy = tid >> 5;
    const int tile = blockIdx.x;
    const int ty = tile / prm.tiles_x, tx = tile - ty * prm.tiles_x;
    const int split = blockIdx.y, b = blockIdx.z;
    const int K = prm.n_angles, N = prm.image_n, L = prm.seg_len;

    const int per = (K + prm.n_splits - 1) / prm.n_splits;
    const int a_begin = split * per;
    const int a_end = min(K, a_begin + per);

    if (tid == 0) { mbar_init(bar, 1); fence_mbar_init(); }
    __syncthreads();

    const double x0 = (double)(tx * 32) - prm.c_n;
    const double y0 = (double)(ty * TH) - prm.c_n;
    const BpEntry<T>* Eb = E + (size_t)b * K * prm.ent_pitch;

    T acc_a[R], acc_b[R];
#pragma unroll
    for (int r = 0; r < R; ++r) { acc_a[r] = T(0); acc_b[r] = T(0); }
    const T lx = (T)lane, ly = (T)(wy * R);
    unsigned phase = 0;

    for (int a0 = a_begin; a0 < a_end; a0 += prm.chunk) {
        const int na = min(prm.chunk, a_end - a0);
        __syncthreads();  // every warp is done reading the previous chunk
        if (wy == 0) {
            if (lane == 0) mbar_arrive_expect_tx(bar, (unsigned)(na * L * ESZ));
            for (int a = lane; a < na; a += 32) {
                const double2 cs = cs2[a0 + a];
                const double ub = x0 * cs.x + y0 * cs.y + prm.c_d;
                const double umin = ub + fmin(0.0, 31.0 * cs.x) + fmin(0.0, (double)(TH - 1) * cs.y);
                const double fl = floor(umin) - 1.0;
                AngleRec<T> rc;
                long long j0;
                // the window [j0, j0+L) must lie inside the guarded row [-guard, pitch-guard)
                if (fl >= -(double)prm.ent_guard && fl <= (double)(prm.ent_pitch - prm.ent_guard - L)) {
                    j0 = (long long)fl;
                    rc.c = (T)cs.x; rc.s = (T)cs.y; rc.b = (T)(ub - fl - 0.5);
                } else {
                    // the tile projects entirely off the detector at this angle: stage the
                    // all-zero left guard and pin every pixel to entry 1 of it
                    j0 = -(long long)prm.ent_guard;
                    rc.c = T(0); rc.s = T(0); rc.b = T(1);
                }
                rc.pad = T(0);
                rec[a] = rc;
                const BpEntry<T>* src = Eb + (size_t)(a0 + a) * prm.ent_pitch + (j0 + prm.ent_guard);
                tma_load_1d(seg + (unsigned)(a * L * ESZ), src, (unsigned)(L * ESZ), bar);
            }
        }
        __syncthreads();        // rec[] visible to all warps
        mbar_wait(bar, phase);  // all bulk copies of this chunk have landed
        phase ^= 1u;

        const T M = Magic<T>::m();
#pragma unroll 2
        for (int a = 0; a < na; ++a) {
            const AngleRec<T> rc = rec[a];
            // address of entry e: seg + a*L*ESZ + (bits(t) - bits(M)) * ESZ, bits(M) folded in
            const unsigned rowbase = seg + (unsigned)(a * L * ESZ) - Magic<T>::kBits * (unsigned)ESZ;
            const T u0 = fma(lx, rc.c, fma(ly, rc.s, rc.b));
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const T u = fma((T)r, rc.s, u0);
                const T t = u + M;
                const T w = u - (t - M);
                T ma, mb, sa, sb;
                EntryLoad<T>::ld(rowbase + Magic<T>::bits(t) * (unsigned)ESZ, ma, mb, sa, sb);
                acc_a[r] += fma(w, sa, ma);
                acc_b[r] += fma(w, sb, mb);
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
            if (row < prm.half_rows) {
                o[(size_t)row * N + c] = acc_a[r] * sc;
                const int mrow = N - 1 - row;
                if (mrow >= prm.half_rows) o[(size_t)mrow * N + (N - 1 - c)] = acc_b[r] * sc;
            }
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
