// fbp_backproject.cuh -- pixel-driven gather back-projection for sm_100a (eq. 2).
//
// f[r][c] = (pi/K) sum_i lerp(Q~_i, u_i),  u_i = (x cos_i + y sin_i)/d + (D-1)/2.
//
// Point symmetry.  The image grid and the detector are both centred, so the pixel (-x,-y)
// has u' = (D-1) - u at every angle: if u = j + 1/2 + w (w in [-1/2,1/2]) then the mirror
// pixel reads interval D-2-j with offset -w.  One thread therefore owns R pixels of the top
// half of the image AND their R mirror pixels, computes (j, w) once, and in fp32 fetches both
// interpolation operands with ONE 16-byte shared-memory load of the entry
//   E[i][j] = ( mid[j], mid[D-2-j], slope[j], -slope[D-2-j] ),
//   mid[j] = (Q~[j]+Q~[j+1])/2,  slope[j] = Q~[j+1]-Q~[j],  Q~ = 0 outside [0, D-1]
// so that  value = mid_a + w slope_a  and  mirror value = mid_b + w nslope_b; in fp32 that is
// one packed FFMA2 + one packed FADD2 on the (pixel, mirror) accumulator pair.
// In fp64 the 16-byte unit of interval j holds the NEAR end points (Q~[j], Q~[D-1-j]) of the interval and
// of its mirror; the far end points are the next unit:  value = near (1-w) + far w,  w = u - floor(u) in [0,1).
// A thread's R pixels step by s = sin(theta) pix/d along its column; where 0 <= s <= 1 - 2^-40 (every angle of
// [0, pi] at pix <= d) consecutive pixels fall into the same or the next interval, so the thread WALKS: it keeps
// `near` in registers (the previous pixel's near or far, one select) and loads only `far` -- one LDS.128 per
// pixel pair instead of two, 8 instead of 16 bytes of shared-memory operands per update.  Angles outside that
// range (the producer flags every staged chunk) load both end points.  (In fp32 the same walk is slower than
// the (mid, slope) entry: the selects and the extra subtract cost more issue slots than the saved wavefronts --
// measured.)
// The entries are produced by the filter epilogue (fbp_reconstruct) or entries_kernel
// (fbp_backproject) into a plan-owned buffer [batch][K][pitch] with >= L+1 zero
// guard entries on both sides (fbp_entries.cuh).
//
// A CTA owns a tile of 32 x (WY*R) primary pixels and a contiguous range of angles (split s
// of S).  Its warps form WA groups of WY warps; group g takes every WA-th angle, so one small
// tile still keeps 4-8 warps busy, and the WA partial sums are added in fixed order g = 0..WA-1
// through shared memory at the end.  Angles are staged in chunks through a two-stage ring:
// while the CTA works on chunk k, lane a of warp 0 computes for each angle of chunk k+1, in
// fp64, the tile-local base b = u(tile origin) - j0 - 1/2 (fp32 coordinates stay below 64:
// ulp <= 3.8e-6) and issues one TMA bulk copy (cp.async.bulk, completion on an mbarrier) of
// the L entries starting at j0 into the other stage.
// Per update pair, fp32:  u' = b + lx cos + ly sin;  t = u' + M (M = 1.5*2^23, round to nearest);
// e = bits(t) - bits(M);  w = u' - (t - M);  one LDS.128;  2 FMA + 2 ADD.  A tie in the rounding picks
// either neighbouring interval with the same interpolated value.  fp64: b carries no -1/2 and the add
// rounds DOWN (M = 1.5*2^52), so e = floor(u'), w = u' - e in [0, 1).
// One owner per pixel, ascending angles => bit-identical runs.  With S > 1 (one small slice
// would otherwise leave most of the 148 SMs idle) the S CTAs of a tile each write their
// partial tile to a scratch image [S][batch][N][N] and take a ticket (one atomicAdd per CTA on
// a per-tile counter -- ordering only, never data); the CTA that draws the last ticket adds the
// S partials in fixed order s = 0..S-1, scales by pi/K and stores the final pixels.  The sum
// order does not depend on which CTA arrives last, so the output bytes do not either.
// (A thread-block cluster + DSMEM reduction was measured first: clusters of 8 leave whole SMs
// without work on B200 -- sm__cycles_active.min = 0 -- and ran 20 % slower.)
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

#include "fbp_entries.cuh"  // entry layout
#include "fbp_ptx.cuh"      // mbarrier, TMA bulk copy, trace_mark

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
    unsigned long long* trace;   // fbp_set_trace: [CTAs][8] %globaltimer marks, or NULL
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

// a + b rounded toward -infinity: with b = Magic::m() the floor of a (|a| < 2^22 | 2^51) lands in the low mantissa bits
__device__ __forceinline__ float add_rd(float a, float b) { return __fadd_rd(a, b); }
__device__ __forceinline__ double add_rd(double a, double b) { return __dadd_rd(a, b); }

template <typename T> struct alignas(4 * sizeof(T)) AngleRec { T c, s, b, pad; };
// ---- the per-update arithmetic: (pixel, mirror pixel) accumulator pair ---------------------
// fp32: packed pair in one 64-bit register; LDS.128 -> (mids, slopes) as two packed pairs;
//       t = slopes * (w, w) + mids  (FFMA2, scalar w broadcast);  acc += t  (FADD2).
// fp64: near/far end points (two LDS.128, or one when walking); 1 DADD + 4 DFMA per pixel pair.
template <typename T> struct PairAcc;
template <> struct PairAcc<float> {
    unsigned long long v;
    __device__ __forceinline__ void zero() { v = 0ull; }
    __device__ __forceinline__ void update(unsigned addr, float w)
    {
#ifndef FBP_SCALAR_PAIR
        unsigned long long m2, s2, w2, t;
        asm volatile("ld.shared.v2.b64 {%0,%1}, [%2];" : "=l"(m2), "=l"(s2) : "r"(addr));
        asm("mov.b64 %0, {%1, %1};" : "=l"(w2) : "f"(w));
        asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(t) : "l"(s2), "l"(w2), "l"(m2));
        asm("add.rn.f32x2 %0, %0, %1;" : "+l"(v) : "l"(t));
#else
        float ma, mb, sa, sb;
        asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(ma), "=f"(mb), "=f"(sa), "=f"(sb) : "r"(addr));
        const float na = a() + fmaf(w, sa, ma), nb = b() + fmaf(w, sb, mb);
        v = (unsigned long long)__float_as_uint(na) | ((unsigned long long)__float_as_uint(nb) << 32);
#endif
    }
    __device__ __forceinline__ float a() const { return __uint_as_float((unsigned)(v & 0xffffffffull)); }
    __device__ __forceinline__ float b() const { return __uint_as_float((unsigned)(v >> 32)); }
};
template <> struct PairAcc<double> {
    double va, vb;
    __device__ __forceinline__ void zero() { va = 0.0; vb = 0.0; }
    // near (1-w) + far w for the pixel and its mirror
    __device__ __forceinline__ void lerp(double na, double nb, double fa, double fb, double w)
    {
        const double omw = 1.0 - w;
        va = fma(na, omw, va); vb = fma(nb, omw, vb);
        va = fma(fa, w, va);   vb = fma(fb, w, vb);
    }
    __device__ __forceinline__ double a() const { return va; }
    __device__ __forceinline__ double b() const { return vb; }
};
__device__ __forceinline__ void lds_f64x2(double& x, double& y, unsigned addr)
{
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(x), "=d"(y) : "r"(addr));
}

// cs2: [K] pairs (cos*pix/d, sin*pix/d) in fp64.  E: 16-byte entry units [batch][K][pitch].
// Grid (tiles, S, batch).  image: [batch][N][N], fully written, scaled by pi/K.
// part: scratch [S][batch][N][N] and tickets: [batch][tiles] zero-initialised counters (S > 1 only).
// TRACE: the instantiation launched while fbp_set_trace is on (the marks are compiled out of the other one: under its
// 64-register cap even predicated-off stores cost the main loop 1.5 us at config 3).
// Registers per thread the occupancy bound aims at.  fp32: 64 for the small-tile variants (6 CTAs of 160 threads per SM),
// 72 for the 32x32 tile (R = 8, WY = 4: at 64 the 16 packed accumulators spill 48 bytes; measured 1.84 -> 1.78 ms at
// config 5, 2.88 -> 2.84 ms at config 4).  fp64: 96, and 112 for the 32x32 tile (3.60 -> 3.52 ms at config 5).
#ifndef FBP_BP_REGCAP64
#define FBP_BP_REGCAP64 ((R == 8 && WY == 4 && WA == 1) ? 112 : 96)
#endif
#ifndef FBP_BP_REGCAP
#define FBP_BP_REGCAP (sizeof(T) == 4 ? ((R == 8 && WY == 4 && WA == 1) ? 72 : 64) : FBP_BP_REGCAP64)
#endif
#ifndef FBP_BP_STAGES
#define FBP_BP_STAGES 3
#endif
constexpr int kBpStages = FBP_BP_STAGES;

template <typename T, int R, int WY, int WA, bool TRACE>
__global__ void __launch_bounds__(32 * (WY * WA + 1), 65536 / (FBP_BP_REGCAP * 32 * (WY * WA + 1)))
backproject_kernel(const uint4* __restrict__ E, T* __restrict__ image, const double2* __restrict__ cs2,
                   T* __restrict__ part, int* __restrict__ tickets, BpParams prm)
{
    constexpr int TH = WY * R;
    constexpr int NW = WY * WA;          // consumer warps; warp NW is the producer
    constexpr int NS = kBpStages;
    extern __shared__ __align__(128) unsigned char bp_smem_raw[];
    // layout: full[NS], empty[NS] mbarriers, walk[NS] flags (64 B) | rec[NS][chunk] | pad to 128 |
    //         seg[NS stages][chunk][L] x 16 B
    const unsigned bar_full = smem_u32(bp_smem_raw);
    const unsigned bar_empty = bar_full + 8u * NS;
    static_assert(16 * NS + 4 * NS <= 64, "barriers and flags share the 64-byte header");
    volatile int* walk_flag = reinterpret_cast<volatile int*>(bp_smem_raw + 16 * NS);   // fp64: every angle of the stage may be walked
    AngleRec<T>* rec = reinterpret_cast<AngleRec<T>*>(bp_smem_raw + 64);
    unsigned char* seg_ptr = bp_smem_raw + 64 + NS * (size_t)prm.chunk * sizeof(AngleRec<T>);
    seg_ptr += (128 - (reinterpret_cast<uintptr_t>(seg_ptr) & 127)) & 127;
    const unsigned seg = smem_u32(seg_ptr);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned cta_id = blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z);
    if (TRACE) {
        trace_mark(prm.trace, cta_id, 0);                       // CTA resident
        if (prm.trace != nullptr && threadIdx.x == 0) {         // slot 7: the SM this CTA runs on (placement and fairness studies)
            unsigned smid;
            asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
            prm.trace[(size_t)cta_id * 8 + 7] = smid;
        }
    }
    const bool producer = warp == NW;
    const int wy = warp % WY, wa = producer ? WA : warp / WY;
    const int tile = blockIdx.x;
    const int ty = tile / prm.tiles_x, tx = tile - ty * prm.tiles_x;
    const int split = blockIdx.y, b = blockIdx.z;
    const int K = prm.n_angles, N = prm.image_n, L = prm.seg_len, S = prm.n_splits;
    const unsigned stage_stride = (unsigned)(prm.chunk * L * 16);

    const int per = (K + S - 1) / S;
    const int a_begin = split * per;
    const int a_end = min(K, a_begin + per);
    const int n_chunks = a_end > a_begin ? (a_end - a_begin + prm.chunk - 1) / prm.chunk : 0;

    if (tid == 0) {
        for (int st = 0; st < NS; ++st) {
            mbar_init(bar_full + 8u * st, 1);     // the producer's expect_tx arrival
            mbar_init(bar_empty + 8u * st, NW);   // one arrival per consumer warp
        }
        fence_mbar_init();
    }
    __syncthreads();
    // programmatic dependent launch: everything above overlapped the tail of the kernel that writes
    // E.  Every thread blocks here (consumers would otherwise spin on their mbarriers and take issue
    // slots from that kernel); a no-op when launched without the attribute.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (TRACE) trace_mark(prm.trace, cta_id, 1);               // past the grid dependency

    PairAcc<T> acc[R];
#pragma unroll
    for (int r = 0; r < R; ++r) acc[r].zero();

    if (producer) {
        // ---- producer warp: per angle, the tile-local record (fp64) and one TMA bulk copy ----
        const double x0 = (double)(tx * 32) - prm.c_n;
        const double y0 = (double)(ty * TH) - prm.c_n;
        const uint4* Eb = E + (size_t)b * K * prm.ent_pitch;
        for (int k = 0; k < n_chunks; ++k) {
            const int st = k % NS;
            const int a0 = a_begin + k * prm.chunk;
            const int na = min(prm.chunk, a_end - a0);
            const unsigned bar = bar_full + 8u * st;
            // lane a's record and source address are computed BEFORE waiting for the stage to be released:
            // the table read and the fp64 arithmetic overlap the consumers' work on the chunks in flight
            // (chunk <= 32: one angle per lane)
            AngleRec<T> rc;
            const uint4* src = Eb;
            bool walk_ok = true;
            if (lane < na) {
                long long off;            // first staged entry of this angle's row, in entries from the row start
                const double2 cs = cs2[a0 + lane];
                const double ub = x0 * cs.x + y0 * cs.y + prm.c_d;
                const double umin = ub + fmin(0.0, 31.0 * cs.x) + fmin(0.0, (double)(TH - 1) * cs.y);
                const double fl = floor(umin) - 1.0;
                // the window [j0, j0+L) must lie inside the guarded row [-guard, pitch-guard)
                if (fl >= -(double)prm.ent_guard && fl <= (double)(prm.ent_pitch - prm.ent_guard - L)) {
                    off = (long long)fl + prm.ent_guard;
                    rc.c = (T)cs.x; rc.s = (T)cs.y;
                    rc.b = sizeof(T) == 4 ? (T)(ub - fl - 0.5) : (T)(ub - fl);
                } else {
                    // the tile projects entirely off the detector at this angle: stage the
                    // all-zero left guard and pin every pixel to entry 1 of it
                    off = 0;
                    rc.c = T(0); rc.s = T(0); rc.b = T(1);
                }
                rc.pad = T(0);
                src = Eb + (size_t)(a0 + lane) * prm.ent_pitch + off;
                // fp64: may the consumers walk along their column at this angle?  (0 <= step < 1 with a margin far
                // above the rounding of fma(r, s, u0): the interval index then never moves by more than 1)
                walk_ok = cs.y >= 0.0 && cs.y <= 1.0 - 0x1p-40;
            }
            if (sizeof(T) == 8) walk_ok = __all_sync(0xffffffffu, walk_ok);
            if (k >= NS) mbar_wait(bar_empty + 8u * st, (unsigned)((k / NS - 1) & 1));  // stage released
            if (lane < na) {
                rec[st * prm.chunk + lane] = rc;
                tma_load_1d(seg + st * stage_stride + (unsigned)(lane * L * 16), src, (unsigned)(L * 16), bar);
            }
            if (sizeof(T) == 8 && lane == 0) walk_flag[st] = walk_ok ? 1 : 0;
            // every lane's records are written before lane 0's (releasing) arrival, so a warp
            // that sees the phase complete also sees the records
            __syncwarp();
            if (lane == 0) mbar_arrive_expect_tx(bar, (unsigned)(na * L * 16));
        }
    } else {
        // ---- consumer warps: no block-wide barrier, only data (full) waits ----
        const T lx = (T)lane, ly = (T)(wy * R);
        const T M = Magic<T>::m();
        for (int k = 0; k < n_chunks; ++k) {
            const int st = k % NS;
            const int na = min(prm.chunk, a_end - (a_begin + k * prm.chunk));
            mbar_wait(bar_full + 8u * st, (unsigned)((k / NS) & 1));  // chunk k has landed
            if (TRACE && k == 0) trace_mark(prm.trace, cta_id, 2);   // first chunk landed (thread 0 is a consumer)
            const AngleRec<T>* rk = rec + st * prm.chunk;
            const unsigned segk = seg + st * stage_stride - Magic<T>::kBits * 16u;  // bits(M) folded in
            if constexpr (sizeof(T) == 4) {
#pragma unroll 2
                for (int a = wa; a < na; a += WA) {
                    const AngleRec<T> rc = rk[a];
                    const unsigned rowbase = segk + (unsigned)(a * L * 16);
                    const T u0 = fma(lx, rc.c, fma(ly, rc.s, rc.b));
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const T u = fma((T)r, rc.s, u0);
                        const T t = u + M;
                        const T w = u - (t - M);
                        acc[r].update(rowbase + Magic<T>::bits(t) * 16u, w);
                    }
                }
            } else if (walk_flag[st] != 0) {
                // walk: `near` of pixel r is the previous pixel's near (same interval) or far (next interval)
#pragma unroll 4
                for (int a = wa; a < na; a += WA) {
                    const AngleRec<T> rc = rk[a];
                    const unsigned rowbase = segk + (unsigned)(a * L * 16);
                    const double u0 = fma(lx, rc.c, fma(ly, rc.s, rc.b));
                    double na_ = 0.0, nb_ = 0.0, pa = 0.0, pb = 0.0;
                    unsigned pe = 0u;
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const double u = fma((double)r, rc.s, u0);
                        const double t = __dadd_rd(u, M);
                        const double w = u - (t - M);
                        const unsigned e = Magic<T>::bits(t);
                        const unsigned addr = rowbase + e * 16u;
                        double fa, fb;
                        lds_f64x2(fa, fb, addr + 16u);
                        if (r == 0) {
                            lds_f64x2(na_, nb_, addr);
                        } else {
                            const bool moved = e != pe;
                            na_ = moved ? pa : na_;
                            nb_ = moved ? pb : nb_;
                        }
                        acc[r].lerp(na_, nb_, fa, fb, w);
                        pe = e; pa = fa; pb = fb;
                    }
                }
            } else {
#pragma unroll 2
                for (int a = wa; a < na; a += WA) {
                    const AngleRec<T> rc = rk[a];
                    const unsigned rowbase = segk + (unsigned)(a * L * 16);
                    const double u0 = fma(lx, rc.c, fma(ly, rc.s, rc.b));
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const double u = fma((double)r, rc.s, u0);
                        const double t = __dadd_rd(u, M);
                        const double w = u - (t - M);
                        const unsigned addr = rowbase + Magic<T>::bits(t) * 16u;
                        double na_, nb_, fa, fb;
                        lds_f64x2(na_, nb_, addr);
                        lds_f64x2(fa, fb, addr + 16u);
                        acc[r].lerp(na_, nb_, fa, fb, w);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_empty + 8u * st);   // this warp is done with stage st
        }
    }

    if (TRACE) trace_mark(prm.trace, cta_id, 3);               // main loop done
    // ---- in-CTA reduction over the WA angle groups, fixed order g = 0..WA-1 ----
    T va[R], vb[R];
#pragma unroll
    for (int r = 0; r < R; ++r) { va[r] = acc[r].a(); vb[r] = acc[r].b(); }
    if (WA > 1) {
        __syncthreads();  // the last chunk has been consumed: the seg region can be reused
        T* red = reinterpret_cast<T*>(seg_ptr);   // [WA-1][2R][32*WY]
        const int lt = wy * 32 + lane;
        if (wa > 0 && !producer) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                red[((wa - 1) * 2 * R + r) * (32 * WY) + lt] = va[r];
                red[((wa - 1) * 2 * R + R + r) * (32 * WY) + lt] = vb[r];
            }
        }
        __syncthreads();
        if (wa == 0) {
            for (int g = 1; g < WA; ++g) {
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    va[r] += red[((g - 1) * 2 * R + r) * (32 * WY) + lt];
                    vb[r] += red[((g - 1) * 2 * R + R + r) * (32 * WY) + lt];
                }
            }
        }
    }
    const bool owner = (wa == 0);   // group 0 (never the producer warp) holds the tile's sums and does every store below

    const int c = tx * 32 + lane;
    T* img = image + (size_t)b * N * N;
    const T sc = (T)prm.scale;
    // pixel offsets of this thread: primary rows (base_a + r*N) and their mirrors (base_b - r*N)
    const int row0 = ty * TH + wy * R;
    const long long base_a = (long long)row0 * N + c;
    const long long base_b = (long long)(N - 1 - row0) * N + (N - 1 - c);
    auto ok_a = [&](int r) { return owner && c < N && row0 + r < prm.half_rows; };
    auto ok_b = [&](int r) { return ok_a(r) && (N - 1 - row0 - r) >= prm.half_rows; };

    if (S == 1) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (ok_a(r)) img[base_a + (long long)r * N] = va[r] * sc;
            if (ok_b(r)) img[base_b - (long long)r * N] = vb[r] * sc;
        }
        if (TRACE) trace_mark(prm.trace, cta_id, 4);           // pixels stored
        return;
    }

    // ---- S > 1: partial tile -> scratch, ticket, last arriver reduces in fixed order ----
    const size_t img_elems = (size_t)N * N;
    const size_t split_stride = (size_t)gridDim.z * img_elems;      // [S][batch][N][N]
    T* mine = part + (size_t)split * split_stride + (size_t)b * img_elems;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        if (ok_a(r)) mine[base_a + (long long)r * N] = va[r];
        if (ok_b(r)) mine[base_b - (long long)r * N] = vb[r];
    }
    __threadfence();
    __syncthreads();
    __shared__ int s_last;
    if (tid == 0) {
        int* tk = tickets + (size_t)b * gridDim.x + tile;
        const int t = atomicAdd(tk, 1);
        s_last = (t == S - 1);
        if (t == S - 1) *tk = 0;   // every CTA of the tile has arrived: re-arm for the next launch
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    const T* p0 = part + (size_t)b * img_elems;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        va[r] = ok_a(r) ? __ldcg(p0 + base_a + (long long)r * N) : T(0);
        vb[r] = ok_b(r) ? __ldcg(p0 + base_b - (long long)r * N) : T(0);
    }
#pragma unroll 1
    for (int s = 1; s < S; ++s) {
        const T* ps = p0 + (size_t)s * split_stride;
        T ta[R], tb[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            ta[r] = ok_a(r) ? __ldcg(ps + base_a + (long long)r * N) : T(0);
            tb[r] = ok_b(r) ? __ldcg(ps + base_b - (long long)r * N) : T(0);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) { va[r] += ta[r]; vb[r] += tb[r]; }
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        if (ok_a(r)) img[base_a + (long long)r * N] = va[r] * sc;
        if (ok_b(r)) img[base_b - (long long)r * N] = vb[r] * sc;
    }
}

}  // namespace fbp
