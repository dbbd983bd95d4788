// ubench_bp_inner.cu -- micro-benchmark of the back-projector's inner loop: which operand scheme
// does a B200 SM run fastest?  NOT part of libfbp: a stand-alone program, built and run by
// `python -m paper_2109_02174_b200.ubench`; its table is profiles/r2b_ubench_bp_inner.txt.
//
// Every variant does the arithmetic of eq. 2 for R pixels of a column and their point-mirror pixels
// per angle -- coordinate, floor, fraction, linear interpolation, accumulate -- on a synthetic staged segment that
// stays in shared memory (no producer, no TMA, no global traffic in the loop): 4 warps per CTA, warp g takes every
// 4th angle, NB CTAs per SM, as the config-3 launch of the product.  What differs is how the two interpolation
// operands reach the registers:
//   fp32  V0  (mid, slope) entry of the interval and its mirror: one LDS.128 per pixel pair        [the product]
//         V1  near and far end points (Q[j], Q[D-1-j]), (Q[j+1], Q[D-2-j]): two LDS.64
//         V2  walk: near = the previous pixel's near or far (one select), only far is loaded: one LDS.64
//         V3  V2 with the coordinates of two pixels per packed FFMA2 / FADD2
//   fp64  V0  two-plane (mid, slope) entries: two LDS.128 per pixel pair                           [the product until r2]
//         V1  near and far: two LDS.128                                  [the product where an angle cannot be walked]
//         V3  walk, one LDS.128, value = near (1-w) + far w                                         [the product]
// Findings on B200 (profiles/r2b_ubench_bp_inner.txt): fp32 V0 runs at 0.92 of the shared-memory bound of 16
// updates/clk/SM (4 wavefronts per pair); V2/V3 halve the wavefronts but need 15-17 issue slots per pair instead of
// 10-11 (a packed FFMA2/FADD2 saves an instruction, not an issue cycle: its 64-bit operands take two) and land at the
// same ~14.3 updates/clk/SM -- issue-bound.  In fp64 the walk wins: 8.7 against 7.5 updates/clk/SM.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <vector>

#ifndef NB
#define NB 4          // CTAs per SM
#endif
typedef unsigned long long u64;
constexpr int L = 36, CH = 16, R = 7;
struct Rec { float c, s, b, pad; };
struct RecD { double c, s, b, pad; };

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

template <int V>
__global__ void __launch_bounds__(128, NB) k32(const Rec* __restrict__ recs, int K, int reps, float* out)
{
    extern __shared__ __align__(128) unsigned char sm[];
    Rec* rec = reinterpret_cast<Rec*>(sm);                     // [K]
    float* seg = reinterpret_cast<float*>(sm + 16 * 512);      // [CH][L] entries
    constexpr int ESZ = V == 0 ? 4 : 2;                        // floats per entry
    for (int i = threadIdx.x; i < K; i += blockDim.x) rec[i] = recs[i];
    for (int i = threadIdx.x; i < CH * L * ESZ; i += blockDim.x) seg[i] = (float)((i * 2654435761u) >> 20) * 1e-3f;
    __syncthreads();
    const int lane = threadIdx.x & 31, wa = threadIdx.x >> 5;
    const float lx = (float)lane, ly = 0.f, M = 12582912.0f;
    u64 acc[R];
#pragma unroll
    for (int r = 0; r < R; ++r) acc[r] = 0ull;
    unsigned segb = smem_u32(seg) - 0x4B400000u * (unsigned)(ESZ * 4);   // bits(M) folded into the base
    asm volatile("mov.u32 %0, %0;" : "+r"(segb));                        // opaque: keep the fold
    for (int rep = 0; rep < reps; ++rep) {
#pragma unroll 2
        for (int a = wa; a < K; a += 4) {
            const Rec rc = rec[a];
            const unsigned rowbase = segb + (unsigned)((a & (CH - 1)) * L * ESZ * 4);
            const float u0 = fmaf(lx, rc.c, fmaf(ly, rc.s, rc.b));
            if (V == 0) {
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const float u = fmaf((float)r, rc.s, u0);
                    const float t = u + M;
                    const float w = u - (t - M);
                    const unsigned addr = rowbase + __float_as_uint(t) * 16u;
                    u64 m2, s2, w2, tt;
                    asm volatile("ld.shared.v2.b64 {%0,%1}, [%2];" : "=l"(m2), "=l"(s2) : "r"(addr));
                    asm("mov.b64 %0, {%1, %1};" : "=l"(w2) : "f"(w));
                    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(tt) : "l"(s2), "l"(w2), "l"(m2));
                    asm("add.rn.f32x2 %0, %0, %1;" : "+l"(acc[r]) : "l"(tt));
                }
            } else if (V == 1) {
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const float u = fmaf((float)r, rc.s, u0);
                    float t; asm("add.rm.f32 %0, %1, %2;" : "=f"(t) : "f"(u), "f"(M));
                    const float w = u - (t - M);
                    const unsigned addr = rowbase + __float_as_uint(t) * 8u;
                    u64 nr, fr, w2, d;
                    asm volatile("ld.shared.b64 %0, [%1];" : "=l"(nr) : "r"(addr));
                    asm volatile("ld.shared.b64 %0, [%1+8];" : "=l"(fr) : "r"(addr));
                    asm("mov.b64 %0, {%1, %1};" : "=l"(w2) : "f"(w));
                    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(fr), "l"(nr));
                    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc[r]) : "l"(d), "l"(w2));
                    asm("add.rn.f32x2 %0, %0, %1;" : "+l"(acc[r]) : "l"(nr));
                }
            } else if (V == 3) {
                u64 nr = 0, frp = 0; unsigned pb = 0;
                u64 s2, u02;
                asm("mov.b64 %0, {%1, %1};" : "=l"(s2) : "f"(rc.s));
                asm("mov.b64 %0, {%1, %1};" : "=l"(u02) : "f"(u0));
                const u64 M2 = 0x4B4000004B400000ull, NM2 = 0xCB400000CB400000ull;
#pragma unroll
                for (int m = 0; m < (R + 1) / 2; ++m) {
                    const u64 k2 = (u64)__float_as_uint((float)(2 * m)) | ((u64)__float_as_uint((float)(2 * m + 1)) << 32);
                    u64 u2, t2, tm2, w2p;
                    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(u2) : "l"(s2), "l"(k2), "l"(u02));
                    asm("add.rm.f32x2 %0, %1, %2;" : "=l"(t2) : "l"(u2), "l"(M2));
                    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(tm2) : "l"(t2), "l"(NM2));
                    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(w2p) : "l"(u2), "l"(tm2));
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const int r = 2 * m + h;
                        if (r < R) {
                            const unsigned bt = h ? (unsigned)(t2 >> 32) : (unsigned)t2;
                            const float w = __uint_as_float(h ? (unsigned)(w2p >> 32) : (unsigned)w2p);
                            const unsigned addr = rowbase + bt * 8u;
                            u64 fr, w2, d;
                            asm volatile("ld.shared.b64 %0, [%1+8];" : "=l"(fr) : "r"(addr));
                            if (r == 0) { asm volatile("ld.shared.b64 %0, [%1];" : "=l"(nr) : "r"(addr)); }
                            else { nr = (bt != pb) ? frp : nr; }
                            asm("mov.b64 %0, {%1, %1};" : "=l"(w2) : "f"(w));
                            asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(fr), "l"(nr));
                            asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc[r]) : "l"(d), "l"(w2));
                            asm("add.rn.f32x2 %0, %0, %1;" : "+l"(acc[r]) : "l"(nr));
                            pb = bt; frp = fr;
                        }
                    }
                }
            } else {
                u64 nr = 0, frp = 0; unsigned pb = 0;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const float u = fmaf((float)r, rc.s, u0);
                    float t; asm("add.rm.f32 %0, %1, %2;" : "=f"(t) : "f"(u), "f"(M));
                    const float w = u - (t - M);
                    const unsigned bt = __float_as_uint(t);
                    const unsigned addr = rowbase + bt * 8u;
                    u64 fr, w2, d;
                    asm volatile("ld.shared.b64 %0, [%1+8];" : "=l"(fr) : "r"(addr));
                    if (r == 0) { asm volatile("ld.shared.b64 %0, [%1];" : "=l"(nr) : "r"(addr)); }
                    else { nr = (bt != pb) ? frp : nr; }
                    asm("mov.b64 %0, {%1, %1};" : "=l"(w2) : "f"(w));
                    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(fr), "l"(nr));
                    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc[r]) : "l"(d), "l"(w2));
                    asm("add.rn.f32x2 %0, %0, %1;" : "+l"(acc[r]) : "l"(nr));
                    pb = bt; frp = fr;
                }
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int r = 0; r < R; ++r) s += __uint_as_float((unsigned)acc[r]) + __uint_as_float((unsigned)(acc[r] >> 32));
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <int V>
__global__ void __launch_bounds__(128, NB) k64(const RecD* __restrict__ recs, int K, int reps, double* out)
{
    extern __shared__ __align__(128) unsigned char sm[];
    RecD* rec = reinterpret_cast<RecD*>(sm);                    // [K]
    double* seg = reinterpret_cast<double*>(sm + 32 * 512);
    constexpr int ESZ = V == 0 ? 4 : 2;
    for (int i = threadIdx.x; i < K; i += blockDim.x) rec[i] = recs[i];
    for (int i = threadIdx.x; i < CH * L * ESZ; i += blockDim.x) seg[i] = (double)((i * 2654435761u) >> 20) * 1e-3;
    __syncthreads();
    const int lane = threadIdx.x & 31, wa = threadIdx.x >> 5;
    const double lx = (double)lane, ly = 0., M = 6755399441055744.0;
    double aa[R], ab[R];
#pragma unroll
    for (int r = 0; r < R; ++r) { aa[r] = 0; ab[r] = 0; }
    const unsigned segb = smem_u32(seg);
    const unsigned plane = CH * L * 16;
    for (int rep = 0; rep < reps; ++rep) {
#pragma unroll 2
        for (int a = wa; a < K; a += 4) {
            const RecD rc = rec[a];
            const unsigned rowbase = segb + (unsigned)((a & (CH - 1)) * L * 16);
            const double u0 = fma(lx, rc.c, fma(ly, rc.s, rc.b));
            if (V == 0) {
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const double u = fma((double)r, rc.s, u0);
                    const double t = u + M;
                    const double w = u - (t - M);
                    const unsigned addr = rowbase + (unsigned)__double2loint(t) * 16u;
                    double ma, mb, sa, sb;
                    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(ma), "=d"(mb) : "r"(addr));
                    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(sa), "=d"(sb) : "r"(addr + plane));
                    aa[r] += fma(w, sa, ma); ab[r] += fma(w, sb, mb);
                }
            } else {
                double na = 0, nb = 0, fpa = 0, fpb = 0; unsigned pb = 0;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const double u = fma((double)r, rc.s, u0);
                    const double t = __dadd_rd(u, M);
                    const double w = u - (t - M);
                    const unsigned bt = (unsigned)__double2loint(t);
                    const unsigned addr = rowbase + bt * 16u;
                    double fa, fb;
                    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2+16];" : "=d"(fa), "=d"(fb) : "r"(addr));
                    if (r == 0 || V == 1) { asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(na), "=d"(nb) : "r"(addr)); }
                    else { const bool p = bt != pb; na = p ? fpa : na; nb = p ? fpb : nb; }
                    const double omw = 1.0 - w;
                    aa[r] = fma(na, omw, aa[r]); ab[r] = fma(nb, omw, ab[r]);
                    aa[r] = fma(fa, w, aa[r]);   ab[r] = fma(fb, w, ab[r]);
                    pb = bt; fpa = fa; fpb = fb;
                }
            }
        }
    }
    double s = 0;
#pragma unroll
    for (int r = 0; r < R; ++r) s += aa[r] + ab[r];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <typename F>
static float best_ms(F f, int n = 5)
{
    cudaEvent_t a, b;
    cudaEventCreate(&a); cudaEventCreate(&b);
    f(); cudaDeviceSynchronize();
    float best = 1e9f;
    for (int i = 0; i < n; ++i) {
        cudaEventRecord(a); f(); cudaEventRecord(b); cudaEventSynchronize(b);
        float ms; cudaEventElapsedTime(&ms, a, b);
        if (ms < best) best = ms;
    }
    return best;
}

int main()
{
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, 0) != cudaSuccess) { fprintf(stderr, "no CUDA device\n"); return 1; }
    int khz = 0;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0);
    const int sms = prop.multiProcessorCount;
    const double clk = 1e3 * khz;
    const int K = 360, reps = 20, grid = sms * NB;
    std::vector<Rec> h(K); std::vector<RecD> hd(K);
    for (int i = 0; i < K; ++i) {       // the records of a tile at the image centre, angles i pi / K
        const double th = M_PI * i / K, c = cos(th), s = sin(th);
        const double b = 1.3 + fmax(0.0, -31.0 * c);
        h[i] = {(float)c, (float)s, (float)b, 0.f}; hd[i] = {c, s, b, 0.};
    }
    Rec* dr; RecD* drd; float* o; double* od;
    cudaMalloc(&dr, sizeof(Rec) * K); cudaMalloc(&drd, sizeof(RecD) * K);
    cudaMalloc(&o, 4 * (size_t)grid * 128); cudaMalloc(&od, 8 * (size_t)grid * 128);
    cudaMemcpy(dr, h.data(), sizeof(Rec) * K, cudaMemcpyHostToDevice);
    cudaMemcpy(drd, hd.data(), sizeof(RecD) * K, cudaMemcpyHostToDevice);
    const int smem32 = 16 * 512 + CH * L * 16, smem64 = 32 * 512 + CH * L * 32;
    const double updates = (double)grid * 32 * R * 2 * K * reps;
    printf("%s, %d SMs, %.0f MHz (max), %d CTAs x 128 threads per SM, R = %d, %d angles x %d repetitions\n",
           prop.name, sms, clk * 1e-6, NB, R, K, reps);
    printf("%-6s %-8s %10s %12s %14s\n", "dtype", "variant", "ms", "Gupdates/s", "updates/clk/SM");
#define RUN32(V) { auto kf = k32<V>; cudaFuncSetAttribute(kf, cudaFuncAttributeMaxDynamicSharedMemorySize, smem32); \
    const float ms = best_ms([&] { kf<<<grid, 128, smem32>>>(dr, K, reps, o); }); \
    printf("%-6s V%-7d %10.3f %12.1f %14.2f   %s\n", "f32", V, ms, updates / ms * 1e-6, updates / (ms * 1e-3) / sms / clk, cudaGetErrorString(cudaGetLastError())); }
#define RUN64(V) { auto kf = k64<V>; cudaFuncSetAttribute(kf, cudaFuncAttributeMaxDynamicSharedMemorySize, smem64); \
    const float ms = best_ms([&] { kf<<<grid, 128, smem64>>>(drd, K, reps, od); }); \
    printf("%-6s V%-7d %10.3f %12.1f %14.2f   %s\n", "f64", V, ms, updates / ms * 1e-6, updates / (ms * 1e-3) / sms / clk, cudaGetErrorString(cudaGetLastError())); }
    RUN32(0) RUN32(1) RUN32(2) RUN32(3) RUN64(0) RUN64(1) RUN64(3)
    return 0;
}
