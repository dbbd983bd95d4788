// fbp.cu -- libfbp: plan, launch configuration and the C ABI of include/fbp.h.
// Kernels: fbp_filter.cuh and fbp_backproject.cuh (eq. 2).
// This library has no CPU path and shares nothing with oracle/ (the test oracle).
#include "../../include/fbp.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "fbp_backproject.cuh"
#include "fbp_filter.cuh"
#include "fbp_filter2.cuh"
#include "fbp_metrics.cuh"
#include "fbp_stack.cuh"
#include "fbp_project.cuh"

namespace {

constexpr double kPi = 3.14159265358979323846264338327950288;
constexpr int kNumSm = 148;  // B200
constexpr int kMetricGrid = 8 * kNumSm;
constexpr int kTabCopies = 1;    // replicas of the filter tap table in global memory; 16 measured no faster than 1 (no L2 hot spot)

thread_local std::string g_create_error;

int env_int(const char* name, int dflt)
{
    const char* v = std::getenv(name);
    if (!v || !*v) return dflt;
    return std::atoi(v);
}

}  // namespace

struct fbp_plan {
    fbp_dtype dtype = FBP_F32;
    int K = 0, D = 0, N = 0, max_batch = 0, device = 0;
    double d = 1.0, pix = 1.0;
    size_t esize = 4;

    // device tables / scratch
    double2* d_cs2 = nullptr;   // [K] (cos, sin) * pix/d, fp64
    void* d_taps = nullptr;     // [tab_len] dtype: G[q + tab_off] = g[q]
    void* d_rho = nullptr;      // [D] dtype: conditioning term of the filter (fbp_filter.cuh)
    void* d_ent = nullptr;      // [max_batch][K][ent_pitch] BpEntry: back-projector operands
    void* d_recs = nullptr;     // [tiles][K] AngleRec: per (tile, angle) records of the back-projector (or NULL)
    void* d_part = nullptr;     // [S][max_batch][N][N] partial images when S > 1
    int* d_tickets = nullptr;   // [max_batch][tiles] arrival counters when S > 1 (self re-arming)
    void* d_hsino = nullptr;    // host-path staging (lazy)
    void* d_himg = nullptr;

    // back-projection configuration
    int bp_variant = 0;         // index into kBpVariants: (R, WY, WA)
    int bp_tw = 32, bp_th = 32, bp_r = 8, bp_threads = 128;
    int bp_splits = 1, bp_chunk = 1, bp_seg = 0, bp_smem = 0;
    fbp::BpParams bp{};

    // filter configuration
    int f_r = 9, f_threads = 0, f_smem = 0, f_tab_len = 0;
    fbp::FilterParams fp{};

    // paired-parity filter (fbp_filter2.cuh); filter_v = 1 selects the older one-parity kernel
    int filter_v = 2;
    int f2_r = 6, f2_threads = 0, f2_smem = 0, f2_grid_cap = 0;
    fbp::Filter2Params f2{};
    void* d_u = nullptr;        // [2][tab_len] dtype: UA | UB, U[j] = g[a_tot - 1 - j]
    void* d_rho2 = nullptr;     // [D] dtype: conditioning term of the paired-parity filter
    // apodised windows (fbp_set_window): the dense form of the same kernel; window 0 = Ram-Lak
    int window = 0;
    int f2d_r = 7, f2d_threads = 0, f2d_smem = 0, f2d_grid_cap = 0;
    fbp::Filter2Params f2d{};
    void* d_ud = nullptr;       // [2][tab_len] dtype: UA | UB of the dense table, U[j] = H[2 a_tot - j]
    void* d_rhod = nullptr;     // [D] dtype
    void* d_xt = nullptr;       // 2 x [max_batch][N][N + 2 pad] dtype: padded image and padded transpose for fbp_project
    void* d_wrow = nullptr;     // [K] dtype: angle weight / (pi/K) (fbp_set_angle_weights); NULL = uniform

    double* d_mscratch = nullptr;   // fbp_metrics: [kMetricGrid][3] CTA partials, then mid[3]
    bool use_pdl = true;
    bool host_zero_copy = true;   // fbp_reconstruct_host: store results straight into pinned host memory
    // batch pipeline (run_pipelined): filter of slice group g+1 overlaps back-projection of group g
    static constexpr int kMaxGroups = 16;
    int pipe_min_batch = 8, pipe_group = 0;
    cudaStream_t st_f = nullptr, st_b[2] = {nullptr, nullptr};
    cudaEvent_t ev_fork = nullptr, ev_f[kMaxGroups] = {}, ev_b[2] = {nullptr, nullptr};
    bool profiling = false;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    bool ran_filter = false, ran_bp = false;

    std::string err;
};

namespace {

fbp_status fail(fbp_plan* p, fbp_status st, const std::string& msg)
{
    if (p) p->err = msg; else g_create_error = msg;
    return st;
}

fbp_status cuda_fail(fbp_plan* p, cudaError_t e, const char* what)
{
    std::string m = std::string(what) + ": " + cudaGetErrorString(e);
    cudaGetLastError();  // clear non-sticky error state
    return fail(p, e == cudaErrorMemoryAllocation ? FBP_ENOMEM : FBP_ECUDA, m);
}

#define FBP_CUDA(plan, call)                                        \
    do {                                                            \
        cudaError_t e__ = (call);                                   \
        if (e__ != cudaSuccess) return cuda_fail(plan, e__, #call); \
    } while (0)

// RAII device switch: the plan's device is made current for the call and restored after.
struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; cudaGetLastError(); return; }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) { ok = false; cudaGetLastError(); }
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

int round_up(int v, int m) { return (v + m - 1) / m * m; }

// The dynamic shared-memory limit is an attribute of the KERNEL (per context), not of a plan: plans with
// different geometries share the instantiations, so each one is opened up once to the device maximum
// (227 KB on sm_100, less the kernel's static shared memory) instead of to whatever the first plan needed.
constexpr int kMaxDynSmem = 227 * 1024;
constexpr int kMaxDevices = 64;
template <typename Kern>
cudaError_t allow_max_smem(Kern kern, bool (&done)[kMaxDevices], int device)
{
    const bool tracked = device >= 0 && device < kMaxDevices;
    if (tracked && done[device]) return cudaSuccess;
    cudaFuncAttributes fa{};
    cudaError_t e = cudaFuncGetAttributes(&fa, kern);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem - (int)fa.sharedSizeBytes);
    if (e == cudaSuccess && tracked) done[device] = true;
    return e;
}

// ---- filter launch configuration -------------------------------------------------
// One CTA per row; warps = 2 parities x n_ob output blocks (32*R outputs) x n_sb input slices.
void configure_filter(fbp_plan* p)
{
    const int D = p->D;
    const int de = (D + 1) / 2, dn = D / 2;
    static const int cand[] = {5, 7, 9, 11, 13, 15};
    int best_r = 9;
    double best = -1.0;
    const int forced = env_int("FBP_FILTER_R", 0);
    for (int R : cand) {
        const int n_ob = (de + 32 * R - 1) / (32 * R);
        const double util = (double)de / ((double)n_ob * 32 * R);
        const double score = util * R / (R + 3.0);
        if (forced == R) { best_r = R; break; }
        if (score > best) { best = score; best_r = R; }
    }
    const int R = best_r;
    p->f_r = R;
    fbp::FilterParams& f = p->fp;
    f.n_det = D;
    f.de = de; f.dn = dn;
    f.n_ob = (de + 32 * R - 1) / (32 * R);
    // input slices: enough warps to fill 148 SMs with ~16 warps each, at most 16 warps per CTA
    int sb = env_int("FBP_FILTER_SB", 0);
    if (sb <= 0) {
        sb = (int)std::ceil(16.0 * kNumSm / ((double)p->K * 2 * f.n_ob));
        if (sb < 2) sb = 2;
        if (sb > 8) sb = 8;
    }
    while (sb > 1 && 2 * f.n_ob * sb > 16) --sb;
    f.n_sb = sb;
    f.de_pad = round_up(de, sb * R);
    f.dn_pad = round_up(dn, sb * R);
    const int din_max = f.de_pad > f.dn_pad ? f.de_pad : f.dn_pad;
    f.tab_off = din_max + 1;
    f.tab_cnt = din_max + f.n_ob * 32 * R + R + 1;
    p->f_tab_len = f.tab_off + f.tab_cnt + 2;
    f.x_pitch = round_up(din_max, 4);
    p->f_threads = 2 * f.n_ob * sb * 32;
    const size_t words = 2 * (size_t)f.tab_cnt + 2 * (size_t)f.x_pitch + 2 * (size_t)f.n_ob * 32 +
                         (size_t)(1 + sb) * 2 * f.n_ob * 32 * R + (size_t)(p->bp.ent_pitch + 2);
    p->f_smem = (int)(words * p->esize + 16);
}

// Paired-parity filter: R output pairs per thread (R = 2 mod 4), warps = n_ob output blocks x SB
// input slices, persistent CTAs.
void configure_filter2(fbp_plan* p)
{
    const int D = p->D;
    const int na = (D + 1) / 2;                        // output pairs = input pairs
    static const int cand[] = {6, 10, 14};
    const int forced = env_int("FBP_FILTER_R", 0);
    int best_r = 6;
    double best = -1.0;
    for (int R : cand) {
        const int n_ob = (na + 32 * R - 1) / (32 * R);
        if (n_ob > 16) continue;
        if (p->dtype == FBP_F64 && R > 6) continue;   // 4R fp64 registers of accumulators and taps: R = 10 spills
        const double util = (double)na / ((double)n_ob * 32 * R);
        const double score = util * (2.0 * R) / (2.0 * R + 2.5);
        if (forced == R) { best_r = R; best = 1e9; }
        if (score > best) { best = score; best_r = R; }
    }
    const int R = best_r;
    p->f2_r = R;
    fbp::Filter2Params& f = p->f2;
    f.n_det = D;
    f.n_ob = (na + 32 * R - 1) / (32 * R);
    f.a_tot = f.n_ob * 32 * R;
    f.n_chunks = (na + R - 1) / R;
    f.b_pad = f.n_chunks * R;
    int sb = env_int("FBP_FILTER_SB", 0);
    if (sb <= 0) {
        // warps per CTA: few when rows are plentiful (less reduction work per row), more when one launch
        // has only a few rows per SM or a row needs many output blocks (measured on B200)
        const double rows_per_sm = (double)p->max_batch * p->K / kNumSm;
        const int target = rows_per_sm >= 64.0 ? 4 : (f.n_ob >= 4 ? 16 : 8);
        sb = (target + f.n_ob / 2) / f.n_ob;
        if (sb < 1) sb = 1;
    }
    if (sb > 8) sb = 8;
    if (sb > f.n_chunks) sb = f.n_chunks;
    while (sb > 1 && f.n_ob * sb > 16) --sb;
    if (sb < 1) sb = 1;
    f.n_sb = sb;
    f.tab_len = round_up(f.a_tot + f.b_pad + 2, 4);
    f.ent_pitch = p->bp.ent_pitch; f.ent_guard = p->bp.ent_guard;
    p->f2_threads = f.n_ob * sb * 32;
    const size_t elems = 2 * (size_t)f.tab_len + 4 * (size_t)f.b_pad + (size_t)f.n_ob * 32 +
                         (size_t)sb * 2 * f.a_tot + (size_t)(f.ent_pitch + 2) + (size_t)D;
    p->f2_smem = (int)(elems * p->esize + 16);
}

// Dense form (apodised windows): R odd, chunks of 2R inputs, same warp layout.
void configure_filter2_dense(fbp_plan* p)
{
    const int D = p->D;
    const int na = (D + 1) / 2;
    static const int cand[] = {5, 7, 9};
    int best_r = 5;
    double best = -1.0;
    for (int R : cand) {
        const int n_ob = (na + 32 * R - 1) / (32 * R);
        if (n_ob > 16) continue;
        if (p->dtype == FBP_F64 && R > 5) continue;    // 6R fp64 registers of accumulators and taps
        const double util = (double)na / ((double)n_ob * 32 * R);
        const double score = util * (2.0 * R) / (2.0 * R + 2.0);
        if (score > best) { best = score; best_r = R; }
    }
    const int R = best_r;
    p->f2d_r = R;
    fbp::Filter2Params& f = p->f2d;
    f.n_det = D;
    f.n_ob = (na + 32 * R - 1) / (32 * R);
    f.a_tot = f.n_ob * 32 * R;
    f.n_chunks = (D + 2 * R - 1) / (2 * R);
    f.b_pad = f.n_chunks * R;
    const double rows_per_sm = (double)p->max_batch * p->K / kNumSm;
    const int target = rows_per_sm >= 64.0 ? 4 : (f.n_ob >= 4 ? 16 : 8);
    int sb = (target + f.n_ob / 2) / f.n_ob;
    if (sb < 1) sb = 1;
    if (sb > 8) sb = 8;
    if (sb > f.n_chunks) sb = f.n_chunks;
    while (sb > 1 && f.n_ob * sb > 16) --sb;
    f.n_sb = sb;
    f.tab_len = round_up(2 * f.a_tot + 2 * f.b_pad + 4, 4);
    f.ent_pitch = p->bp.ent_pitch; f.ent_guard = p->bp.ent_guard;
    p->f2d_threads = f.n_ob * sb * 32;
    const size_t elems = 2 * (size_t)f.tab_len + 4 * (size_t)f.b_pad + (size_t)f.n_ob * 32 +
                         (size_t)sb * 2 * f.a_tot + (size_t)(f.ent_pitch + 2) + (size_t)D;
    p->f2d_smem = (int)(elems * p->esize + 16);
}

// One tap of the apodised ramp |f| W(f), |f| <= 1/2: h_W[m] = 2 int_0^{1/2} f W(f) cos(2 pi f m) df in closed
// form (include/fbp.h, fbp_set_window; derivations in DESIGN.md "Windows").  Any integer m.
double window_tap(int window, long long m)
{
    auto ramlak = [](long long q) -> double {
        if (q == 0) return 0.25;
        if (q % 2 == 0) return 0.0;
        return -1.0 / (kPi * kPi * (double)q * (double)q);
    };
    auto half_moment = [](double a) { return std::sin(0.5 * a) / (2.0 * a) + (std::cos(0.5 * a) - 1.0) / (a * a); };
    const double md = (double)m;
    switch (window) {
        case FBP_WINDOW_SHEPP_LOGAN: return -2.0 / (kPi * kPi * (4.0 * md * md - 1.0));
        case FBP_WINDOW_COSINE: return half_moment(kPi * (2.0 * md + 1.0)) + half_moment(kPi * (2.0 * md - 1.0));
        case FBP_WINDOW_HAMMING: return 0.54 * ramlak(m) + 0.23 * (ramlak(m + 1) + ramlak(m - 1));
        case FBP_WINDOW_HANN: return 0.5 * ramlak(m) + 0.25 * (ramlak(m + 1) + ramlak(m - 1));
        default: return ramlak(m);
    }
}

// ---- back-projection launch configuration ------------------------------------------
// (R, WY, WA) instantiations of backproject_kernel, see launch_bp
constexpr int kNumBpVariants = 11;
constexpr int kBpVariants[kNumBpVariants][3] = {
    {8, 4, 1}, {4, 4, 1}, {4, 1, 4}, {5, 1, 4}, {6, 1, 4}, {7, 1, 4}, {8, 1, 4},
    {4, 1, 8}, {6, 1, 8}, {7, 1, 8}, {8, 1, 8}};
void configure_bp(fbp_plan* p, const std::vector<double>& cs)
{
    const int N = p->N, K = p->K;
    const int half_rows = (N + 1) / 2;  // primary (top) half; the mirror pixels come for free
    const int tiles_x = (N + p->bp_tw - 1) / p->bp_tw;
    // variant = (R rows per thread, WY warps along y, WA angle groups): tile 32 x (R*WY) primary pixels
    int v = env_int("FBP_BP_VARIANT", -1);
    if (v < 0 || v >= kNumBpVariants) {
        // Small launches (one 512^2 slice is 16 column strips x 256 primary rows) are chosen to fill
        // 148 SMs evenly: short tiles of R rows with 4 angle groups, R picked so that the number of
        // CTAs is as close as possible to a whole number of waves.  Large launches take the 32x32
        // tile (a third of the L2->shared staging traffic per update).
        const long big = (long)tiles_x * ((half_rows + 31) / 32) * p->max_batch;
        if (big >= 8L * kNumSm) {
            v = 0;
        } else {
            double best = -1.0;
            v = 3;
            for (int cand = 2; cand <= 6; ++cand) {
                const int th = kBpVariants[cand][0] * kBpVariants[cand][1];
                const long ctas = (long)tiles_x * ((half_rows + th - 1) / th) * p->max_batch;
                const long waves = (ctas + 4L * kNumSm - 1) / (4L * kNumSm);   // 4 CTAs of 4 warps per SM
                const double fill = (double)ctas / (double)(waves * 4L * kNumSm);
                const double waste = (double)half_rows / (double)(((half_rows + th - 1) / th) * th);
                const double score = fill * waste * (1.0 - 0.15 / th);         // taller tiles stage less
                if (score > best) { best = score; v = cand; }
            }
        }
    }
    p->bp_variant = v;
    p->bp_r = kBpVariants[v][0];
    p->bp_th = kBpVariants[v][0] * kBpVariants[v][1];
    p->bp_threads = 32 * (kBpVariants[v][1] * kBpVariants[v][2] + 1);   // + the producer warp
    const int tiles_y = (half_rows + p->bp_th - 1) / p->bp_th;
    double ext = 0.0;
    for (int i = 0; i < K; ++i) {
        const double e = (p->bp_tw - 1) * std::fabs(cs[2 * i]) + (p->bp_th - 1) * std::fabs(cs[2 * i + 1]);
        if (e > ext) ext = e;
    }
    p->bp_seg = (int)std::ceil(ext) + 4;

    // angle splits: fill 148 SMs evenly when one launch has few tiles
    const long tiles = (long)tiles_x * tiles_y * p->max_batch;
    int S = env_int("FBP_BP_SPLITS", 0);
    if (S <= 0) {
        const int s_max = K / 16 > 1 ? (K / 16 < 16 ? K / 16 : 16) : 1;
        double best = -1.0;
        S = 1;
        for (int s = 1; s <= s_max; ++s) {
            const long ctas = tiles * s;
            const long waves = (ctas + kNumSm - 1) / kNumSm;
            double eff = (double)ctas / (double)(waves * kNumSm);
            if (ctas < 4L * kNumSm) eff *= 0.5 + 0.5 * (double)ctas / (4.0 * kNumSm);
            eff -= 0.01 * (s - 1);  // splitting is not free: prefer fewer splits on ties
            if (eff > best) { best = eff; S = s; }
        }
    }
    if (S > K) S = K;
    if (S > 64) S = 64;
    if (S < 1) S = 1;
    p->bp_splits = S;
    const int per = (K + S - 1) / S;

    const size_t entry = 4 * p->esize, rec = 4 * p->esize;
    const size_t per_angle = (size_t)p->bp_seg * entry + rec;
    // A small launch (c CTAs per SM on average, c <= 5) is placed evenly only if no SM can hold more
    // than c of its CTAs: with programmatic dependent launch the CTAs arrive while the filter is
    // still draining and would otherwise pile up (up to 6 per SM) on the SMs that free up first.
    // Sizing the dynamic shared memory so that c + 1 CTAs do not fit caps the residency at c; the
    // extra room goes to longer chunks (fewer chunk boundaries: 33.6 -> 33.3 us at config 3).
    int even_smem = 0;
    {
        const long ctas = tiles * S;
        const int cps = (int)((ctas + kNumSm - 1) / kNumSm);
        const int smem_sm = 228 * 1024, reserve = 1024;
        if (cps >= 1 && cps <= 5 && env_int("FBP_BP_EVEN", 1)) {
            const int want = smem_sm / (cps + 1) - reserve + 256;
            if ((long)cps * (want + reserve) <= smem_sm) even_smem = want;
        }
    }
    const int wa = kBpVariants[v][2];
    int budget = env_int("FBP_BP_SMEM", even_smem > 36 * 1024 ? even_smem - 512 : 36 * 1024);
    int chunk = env_int("FBP_BP_CHUNK", 0);
    if (chunk <= 0) {
        chunk = (int)(budget / (fbp::kBpStages * per_angle));
        if (chunk > 32) chunk = 32;                       // one producer lane per angle of a chunk
        if (chunk > wa) chunk -= chunk % wa;              // equal work for the angle groups
    }
    if (chunk > per) chunk = per;
    if (chunk < 1) chunk = 1;
    p->bp_chunk = chunk;
    size_t seg_bytes = fbp::kBpStages * (size_t)p->bp_seg * entry * chunk;
    const size_t red_bytes = (size_t)(wa - 1) * 2 * p->bp_r * (32 * kBpVariants[v][1]) * p->esize;
    if (seg_bytes < red_bytes) seg_bytes = red_bytes;          // in-CTA reduction reuses the stages
    p->bp_smem = (int)(64 + fbp::kBpStages * rec * chunk + 128 + seg_bytes);
    if (even_smem > p->bp_smem) p->bp_smem = even_smem;

    fbp::BpParams& b = p->bp;
    b.n_angles = K; b.n_det = p->D; b.image_n = N;
    b.tiles_x = tiles_x; b.tiles_y = tiles_y;
    b.n_splits = S; b.chunk = chunk; b.seg_len = p->bp_seg;
    b.half_rows = half_rows;
    b.ent_guard = p->bp_seg + 1;                       // >= L+1 zero entries on both sides
    b.ent_pitch = p->D + 2 * b.ent_guard;
    p->fp.ent_guard = b.ent_guard; p->fp.ent_pitch = b.ent_pitch;
    b.c_n = 0.5 * (N - 1); b.c_d = 0.5 * (p->D - 1);
    b.scale = kPi / K;
}

}  // namespace

// ---- kernel launchers ---------------------------------------------------------------
namespace {

template <typename T, int R>
cudaError_t launch_filter_r(const fbp_plan* p, const void* sino, void* filt, void* ent, int batch, cudaStream_t st)
{
    fbp::FilterParams f = p->fp;
    f.n_rows = batch * p->K;
    auto kern = fbp::filter_kernel<T, R>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, p->f_smem);
    if (e != cudaSuccess) return e;
    kern<<<f.n_rows, p->f_threads, p->f_smem, st>>>(static_cast<const T*>(sino), static_cast<T*>(filt),
                                                     static_cast<uint4*>(ent),
                                                     static_cast<const T*>(p->d_taps),
                                                     static_cast<const T*>(p->d_rho), f, (T)(1.0 / p->d));
    return cudaGetLastError();
}

// filt and/or ent may be NULL: plain rows (fbp_filter) and/or interleaved entries (fbp_reconstruct)
template <typename T>
cudaError_t launch_filter(const fbp_plan* p, const void* sino, void* filt, void* ent, int batch, cudaStream_t st)
{
    switch (p->f_r) {
        case 5: return launch_filter_r<T, 5>(p, sino, filt, ent, batch, st);
        case 7: return launch_filter_r<T, 7>(p, sino, filt, ent, batch, st);
        case 9: return launch_filter_r<T, 9>(p, sino, filt, ent, batch, st);
        case 11: return launch_filter_r<T, 11>(p, sino, filt, ent, batch, st);
        case 13: return launch_filter_r<T, 13>(p, sino, filt, ent, batch, st);
        default: return launch_filter_r<T, 15>(p, sino, filt, ent, batch, st);
    }
}

template <typename T, int R, bool DENSE>
cudaError_t launch_filter2_r(fbp_plan* p, const void* sino, void* filt, void* ent, int batch, cudaStream_t st)
{
    fbp::Filter2Params f = DENSE ? p->f2d : p->f2;
    f.n_rows = batch * p->K;
    const int threads = DENSE ? p->f2d_threads : p->f2_threads, smem = DENSE ? p->f2d_smem : p->f2_smem;
    int& cap = DENSE ? p->f2d_grid_cap : p->f2_grid_cap;
    auto kern = fbp::filter2_kernel<T, R, DENSE>;
    static bool smem_open[kMaxDevices] = {};
    if (cudaError_t e = allow_max_smem(kern, smem_open, p->device); e != cudaSuccess) return e;
    if (cap == 0) {
        int per_sm = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, smem);
        if (e != cudaSuccess) return e;
        if (per_sm < 1) return cudaErrorLaunchOutOfResources;
        cap = per_sm * kNumSm;
    }
    // A whole number of CTAs per SM: with 360 rows on 148 SMs the 64 CTAs of a third, partial round were starved
    // of issue slots by the two FMA-bound CTAs already computing on their SM (measured with %globaltimer: their
    // tables "landed" 4.6 us late and the kernel ended at 10.5 us); with 296 persistent CTAs, 64 of which take a
    // second row, every CTA on an SM reaches its compute phase together.
    int grid = f.n_rows < cap ? f.n_rows : cap;
    if (grid > kNumSm && env_int("FBP_FILTER_WHOLE_WAVES", 1)) grid -= grid % kNumSm;
    kern<<<grid, threads, smem, st>>>(static_cast<const T*>(sino), static_cast<T*>(filt), static_cast<uint4*>(ent),
                                      static_cast<const T*>(DENSE ? p->d_ud : p->d_u),
                                      static_cast<const T*>(DENSE ? p->d_rhod : p->d_rho2),
                                      static_cast<const T*>(p->d_wrow), p->K, f, (T)(1.0 / p->d), kTabCopies);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_filter2(fbp_plan* p, const void* sino, void* filt, void* ent, int batch, cudaStream_t st)
{
    if (p->window != 0) {
        switch (p->f2d_r) {
            case 5: return launch_filter2_r<T, 5, true>(p, sino, filt, ent, batch, st);
            case 7: return launch_filter2_r<T, 7, true>(p, sino, filt, ent, batch, st);
            default: return launch_filter2_r<T, 9, true>(p, sino, filt, ent, batch, st);
        }
    }
    switch (p->f2_r) {
        case 6: return launch_filter2_r<T, 6, false>(p, sino, filt, ent, batch, st);
        case 10: return launch_filter2_r<T, 10, false>(p, sino, filt, ent, batch, st);
        default: return launch_filter2_r<T, 14, false>(p, sino, filt, ent, batch, st);
    }
}

template <typename T>
cudaError_t launch_entries(fbp_plan* p, const void* filt, int batch, cudaStream_t st)
{
    const size_t smem = (size_t)(p->bp.ent_pitch + 2) * sizeof(T);
    auto kern = fbp::entries_kernel<T>;
    static bool smem_open[kMaxDevices] = {};
    if (cudaError_t e = allow_max_smem(kern, smem_open, p->device); e != cudaSuccess) return e;
    kern<<<batch * p->K, 256, smem, st>>>(static_cast<const T*>(filt), static_cast<uint4*>(p->d_ent), p->D,
                                          p->bp.ent_pitch, p->bp.ent_guard, static_cast<const T*>(p->d_wrow), p->K);
    return cudaGetLastError();
}

template <typename T, int R, int WY, int WA>
cudaError_t launch_bp_v(fbp_plan* p, void* image, int batch, cudaStream_t st, int slice0)
{
    auto kern = fbp::backproject_kernel<T, R, WY, WA>;
    static bool smem_open[kMaxDevices] = {};     // per instantiation and device
    if (cudaError_t e = allow_max_smem(kern, smem_open, p->device); e != cudaSuccess) return e;
    // programmatic dependent launch: the CTAs may become resident and run their prologue while the
    // kernel that writes the entries (filter / entries_kernel) drains; the producer warp executes
    // griddepcontrol.wait before its first read of the entries
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(p->bp.tiles_x * p->bp.tiles_y, p->bp_splits, batch);
    cfg.blockDim = dim3(32 * (WY * WA + 1));
    cfg.dynamicSmemBytes = (size_t)p->bp_smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = p->use_pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    // slice0: first slice of this launch within the plan's entry buffer (`image` already points at it)
    const uint4* ent = static_cast<const uint4*>(p->d_ent) +
                       (size_t)slice0 * p->K * fbp::EntryPlanes<T>::value * p->bp.ent_pitch;
    return cudaLaunchKernelEx(&cfg, kern, ent, static_cast<T*>(image),
                              static_cast<const double2*>(p->d_cs2), static_cast<T*>(p->d_part), p->d_tickets, p->bp);
}

// back-projection of the plan's entry buffer into `image`
template <typename T>
cudaError_t launch_bp(fbp_plan* p, void* image, int batch, cudaStream_t st, int slice0 = 0)
{
    switch (p->bp_variant) {
        case 0: return launch_bp_v<T, 8, 4, 1>(p, image, batch, st, slice0);
        case 1: return launch_bp_v<T, 4, 4, 1>(p, image, batch, st, slice0);
        case 2: return launch_bp_v<T, 4, 1, 4>(p, image, batch, st, slice0);
        case 3: return launch_bp_v<T, 5, 1, 4>(p, image, batch, st, slice0);
        case 4: return launch_bp_v<T, 6, 1, 4>(p, image, batch, st, slice0);
        case 5: return launch_bp_v<T, 7, 1, 4>(p, image, batch, st, slice0);
        case 6: return launch_bp_v<T, 8, 1, 4>(p, image, batch, st, slice0);
        case 7: return launch_bp_v<T, 4, 1, 8>(p, image, batch, st, slice0);
        case 8: return launch_bp_v<T, 6, 1, 8>(p, image, batch, st, slice0);
        case 9: return launch_bp_v<T, 7, 1, 8>(p, image, batch, st, slice0);
        default: return launch_bp_v<T, 8, 1, 8>(p, image, batch, st, slice0);
    }
}

bool aligned16(const void* q) { return (reinterpret_cast<uintptr_t>(q) & 15u) == 0; }

fbp_status check_call(fbp_plan* p, const void* a, const void* b, int batch)
{
    if (!p) return FBP_EINVAL;
    if (!a || !b) return fail(p, FBP_EINVAL, "NULL device pointer");
    if (!aligned16(a) || !aligned16(b)) return fail(p, FBP_EINVAL, "device pointers must be 16-byte aligned");
    if (batch < 1 || batch > p->max_batch) return fail(p, FBP_EINVAL, "batch must be in [1, max_batch]");
    return FBP_OK;
}

fbp_status run_filter(fbp_plan* p, const void* sino, void* filt, void* ent, int batch, cudaStream_t st)
{
    if (p->profiling) FBP_CUDA(p, cudaEventRecord(p->ev[0], st));
    cudaError_t e;
    if (p->filter_v == 2)
        e = p->dtype == FBP_F32 ? launch_filter2<float>(p, sino, filt, ent, batch, st)
                                : launch_filter2<double>(p, sino, filt, ent, batch, st);
    else
        e = p->dtype == FBP_F32 ? launch_filter<float>(p, sino, filt, ent, batch, st)
                                : launch_filter<double>(p, sino, filt, ent, batch, st);
    if (e != cudaSuccess) return cuda_fail(p, e, "filter launch");
    if (p->profiling) FBP_CUDA(p, cudaEventRecord(p->ev[1], st));
    p->ran_filter = true;
    return FBP_OK;
}

// filt != NULL: convert plain filtered rows to entries first (fbp_backproject);
// filt == NULL: the entry buffer was already written by the filter (fbp_reconstruct).
fbp_status run_bp(fbp_plan* p, const void* filt, void* image, int batch, cudaStream_t st)
{
    cudaError_t e = cudaSuccess;
    if (filt) {
        e = p->dtype == FBP_F32 ? launch_entries<float>(p, filt, batch, st) : launch_entries<double>(p, filt, batch, st);
        if (e != cudaSuccess) return cuda_fail(p, e, "entries launch");
    }
    if (p->profiling) FBP_CUDA(p, cudaEventRecord(p->ev[2], st));
    e = p->dtype == FBP_F32 ? launch_bp<float>(p, image, batch, st) : launch_bp<double>(p, image, batch, st);
    if (e != cudaSuccess) return cuda_fail(p, e, "back-projection launch");
    if (p->profiling) FBP_CUDA(p, cudaEventRecord(p->ev[3], st));
    p->ran_bp = true;
    return FBP_OK;
}

// fbp_reconstruct for a stack of slices: the filter is FMA-pipe bound and the back-projector
// shared-memory bound, so they run well side by side.  The batch is cut into groups; group g+1 is
// filtered on a plan-owned high-priority stream while group g is back-projected on one of two other
// plan-owned streams (two, so that the tail of one launch overlaps the head of the next).  The
// caller's stream forks into them and joins at the end: still enqueue-only, no host wait.  Same
// kernels on the same data as the sequential path, hence the same bytes.
fbp_status run_pipelined(fbp_plan* p, const void* sino, void* image, int batch, cudaStream_t s,
                         const void* h_sino = nullptr)
{
    int group = p->pipe_group > 0 ? p->pipe_group : (batch + 3) / 4;   // 4 groups measured best at 64 slices
    const int min_group = (batch + fbp_plan::kMaxGroups - 1) / fbp_plan::kMaxGroups;
    if (group < min_group) group = min_group;
    const int n_groups = (batch + group - 1) / group;
    const size_t sino_slice = p->esize * (size_t)p->K * p->D, img_slice = p->esize * (size_t)p->N * p->N;
    const size_t ent_slice = 4 * p->esize * (size_t)p->K * p->bp.ent_pitch;
    FBP_CUDA(p, cudaEventRecord(p->ev_fork, s));
    FBP_CUDA(p, cudaStreamWaitEvent(p->st_f, p->ev_fork, 0));
    FBP_CUDA(p, cudaStreamWaitEvent(p->st_b[0], p->ev_fork, 0));
    FBP_CUDA(p, cudaStreamWaitEvent(p->st_b[1], p->ev_fork, 0));
    for (int g = 0; g < n_groups; ++g) {
        const int g0 = g * group, nb = batch - g0 < group ? batch - g0 : group;
        const char* sg = static_cast<const char*>(sino) + (size_t)g0 * sino_slice;
        char* eg = static_cast<char*>(p->d_ent) + (size_t)g0 * ent_slice;
        // host source (fbp_reconstruct_host): this group's copy rides the filter stream, so it overlaps the
        // back-projection of the previous group on the copy engine
        if (h_sino)
            FBP_CUDA(p, cudaMemcpyAsync(const_cast<char*>(sg), static_cast<const char*>(h_sino) + (size_t)g0 * sino_slice,
                                        (size_t)nb * sino_slice, cudaMemcpyHostToDevice, p->st_f));
        cudaError_t e = p->dtype == FBP_F32 ? launch_filter2<float>(p, sg, nullptr, eg, nb, p->st_f)
                                            : launch_filter2<double>(p, sg, nullptr, eg, nb, p->st_f);
        if (e != cudaSuccess) return cuda_fail(p, e, "filter launch");
        FBP_CUDA(p, cudaEventRecord(p->ev_f[g], p->st_f));
        cudaStream_t sb = p->st_b[g & 1];
        FBP_CUDA(p, cudaStreamWaitEvent(sb, p->ev_f[g], 0));
        char* ig = static_cast<char*>(image) + (size_t)g0 * img_slice;
        e = p->dtype == FBP_F32 ? launch_bp<float>(p, ig, nb, sb, g0) : launch_bp<double>(p, ig, nb, sb, g0);
        if (e != cudaSuccess) return cuda_fail(p, e, "back-projection launch");
    }
    for (int i = 0; i < 2; ++i) {
        FBP_CUDA(p, cudaEventRecord(p->ev_b[i], p->st_b[i]));
        FBP_CUDA(p, cudaStreamWaitEvent(s, p->ev_b[i], 0));
    }
    p->ran_filter = p->ran_bp = false;
    return FBP_OK;
}

bool use_pipeline(const fbp_plan* p, int batch)
{
    return p->st_f && !p->profiling && p->filter_v == 2 && p->bp_splits == 1 && batch >= p->pipe_min_batch;
}

}  // namespace

// ---- C ABI ----------------------------------------------------------------------------
extern "C" {

fbp_status fbp_create(fbp_plan** out, int n_angles, int n_det, const double* angles_rad,
                      double det_spacing, int image_n, double pixel_size, fbp_dtype dtype,
                      int max_batch, int device)
{
    if (!out) return fail(nullptr, FBP_EINVAL, "out is NULL");
    *out = nullptr;
    if (!angles_rad) return fail(nullptr, FBP_EINVAL, "angles_rad is NULL");
    if (n_angles < 1 || n_angles > (1 << 20)) return fail(nullptr, FBP_EINVAL, "n_angles must be in [1, 2^20]");
    if (n_det < 2 || n_det > (1 << 20)) return fail(nullptr, FBP_EINVAL, "n_det must be in [2, 2^20]");
    if (image_n < 1 || image_n > (1 << 16)) return fail(nullptr, FBP_EINVAL, "image_n must be in [1, 65536]");
    if (!(det_spacing > 0.0) || !std::isfinite(det_spacing)) return fail(nullptr, FBP_EINVAL, "det_spacing must be finite and > 0");
    if (!std::isfinite(pixel_size)) return fail(nullptr, FBP_EINVAL, "pixel_size must be finite");
    if (dtype != FBP_F32 && dtype != FBP_F64) return fail(nullptr, FBP_EINVAL, "unknown dtype");
    if (max_batch < 1 || max_batch > 65535) return fail(nullptr, FBP_EINVAL, "max_batch must be in [1, 65535]");
    for (int i = 0; i < n_angles; ++i)
        if (!std::isfinite(angles_rad[i])) return fail(nullptr, FBP_EINVAL, "non-finite angle");
    const double pix = pixel_size > 0.0 ? pixel_size : det_spacing;

    int ndev = 0;
    cudaError_t ce = cudaGetDeviceCount(&ndev);
    if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "cudaGetDeviceCount");
    if (device < 0) {
        ce = cudaGetDevice(&device);
        if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "cudaGetDevice");
    }
    if (device >= ndev) return fail(nullptr, FBP_EINVAL, "no such CUDA device");
    cudaDeviceProp prop;
    ce = cudaGetDeviceProperties(&prop, device);
    if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "cudaGetDeviceProperties");
    if (prop.major != 10)
        return fail(nullptr, FBP_EUNSUPPORTED, "libfbp is built for sm_100a (B200) only; no fallback path");

    fbp_plan* p = new (std::nothrow) fbp_plan();
    if (!p) return fail(nullptr, FBP_ENOMEM, "host allocation failed");
    p->dtype = dtype; p->K = n_angles; p->D = n_det; p->N = image_n; p->max_batch = max_batch;
    p->device = device; p->d = det_spacing; p->pix = pix;
    p->esize = dtype == FBP_F32 ? 4 : 8;

    // host tables in fp64: (cos, sin) * pix/d  (A0 of SURVEY.md 8(a))
    std::vector<double> cs(2 * (size_t)n_angles);
    const double ratio = pix / det_spacing;
    for (int i = 0; i < n_angles; ++i) {
        cs[2 * i] = std::cos(angles_rad[i]) * ratio;
        cs[2 * i + 1] = std::sin(angles_rad[i]) * ratio;
    }
    configure_bp(p, cs);
    configure_filter(p);   // after configure_bp: needs the entry pitch
    configure_filter2(p);
    configure_filter2_dense(p);
    p->filter_v = env_int("FBP_FILTER_V", 2) == 1 ? 1 : 2;
    p->use_pdl = env_int("FBP_PDL", 1) != 0;
    p->host_zero_copy = env_int("FBP_HOST_ZERO_COPY", 1) != 0;

    auto bail = [&](fbp_status st) { std::string m = p->err; fbp_destroy(p); g_create_error = m; return st; };
    if (p->filter_v == 2 && (p->f2_threads > 512 || p->f2_smem > 220 * 1024)) p->filter_v = 1;
    if (p->filter_v == 1 && p->f_threads > 512) { p->err = "n_det too large for the row filter (more than 512 threads per row)"; return bail(FBP_EUNSUPPORTED); }
    if (p->filter_v == 1 && p->f_smem > 220 * 1024) { p->err = "n_det too large for the shared-memory row filter"; return bail(FBP_EUNSUPPORTED); }
    if (p->bp_smem > 220 * 1024) { p->err = "pixel_size/det_spacing too large for the staged segment"; return bail(FBP_EUNSUPPORTED); }

    DeviceGuard guard(device);
    if (!guard.ok) { p->err = "cudaSetDevice failed"; return bail(FBP_ECUDA); }

    // taps g[q] = h[2q+1] = -1/(pi^2 (2q+1)^2), index = q + tab_off, rounded once to dtype
    const int tl = p->f_tab_len;
    std::vector<double> g64(tl);
    for (int i = 0; i < tl; ++i) {
        const double m = 2.0 * (double)(i - p->fp.tab_off) + 1.0;
        g64[i] = -1.0 / (kPi * kPi * m * m);
    }
    // conditioning term rho[n] = 1/4 + sum_{b=0}^{din_pad(p)-1} g[a - b - (1-p)], n = 2a + p:
    // what filtering a constant row (padding included) gives; fp64, smallest terms first
    std::vector<double> rho64(n_det);
    for (int n = 0; n < n_det; ++n) {
        const int par = n & 1, a = n >> 1;
        const int din_pad = par ? p->fp.de_pad : p->fp.dn_pad;
        std::vector<double> terms(din_pad);
        for (int b = 0; b < din_pad; ++b) {
            const double m = 2.0 * (double)(a - b - (1 - par)) + 1.0;
            terms[b] = 1.0 / (kPi * kPi * m * m);
        }
        std::sort(terms.begin(), terms.end());
        double ssum = 0.0;
        for (double t : terms) ssum += t;
        rho64[n] = 0.25 - ssum;
    }
    // paired-parity filter tables: U[j] = g[a_tot - 1 - j] as UA | UB (UB[j] = U[j+1]); rho2[n] = 1/4 +
    // sum_{b < b_pad} g[a - b - (1 - p)], n = 2a + p  (constant-row response, smallest terms first)
    const int tl2 = p->f2.tab_len;
    std::vector<double> u64(2 * (size_t)tl2), rho2_64(n_det);
    auto gq = [](long long q) { const double m = 2.0 * (double)q + 1.0; return -1.0 / (kPi * kPi * m * m); };
    for (int j = 0; j < tl2; ++j) {
        u64[j] = gq((long long)p->f2.a_tot - 1 - j);
        u64[tl2 + j] = gq((long long)p->f2.a_tot - 2 - j);
    }
    for (int n = 0; n < n_det; ++n) {
        const int par = n & 1, a = n >> 1;
        std::vector<double> terms(p->f2.b_pad);
        for (int b = 0; b < p->f2.b_pad; ++b) terms[b] = -gq((long long)a - b - (1 - par));
        std::sort(terms.begin(), terms.end());
        double ssum = 0.0;
        for (double t : terms) ssum += t;
        rho2_64[n] = 0.25 - ssum;
    }
    std::vector<float> u32, rho2_32;
    const void* usrc = u64.data();
    const void* r2src = rho2_64.data();
    if (dtype == FBP_F32) {
        u32.assign(u64.begin(), u64.end()); usrc = u32.data();
        rho2_32.assign(rho2_64.begin(), rho2_64.end()); r2src = rho2_32.data();
    }
    std::vector<float> g32, rho32;
    const void* gsrc = g64.data();
    const void* rsrc = rho64.data();
    if (dtype == FBP_F32) {
        g32.assign(g64.begin(), g64.end()); gsrc = g32.data();
        rho32.assign(rho64.begin(), rho64.end()); rsrc = rho32.data();
    }

#define FBP_TRY(call)                                                            \
    do {                                                                         \
        cudaError_t e__ = (call);                                                \
        if (e__ != cudaSuccess) return bail(cuda_fail(p, e__, #call));           \
    } while (0)
    FBP_TRY(cudaMalloc(&p->d_cs2, sizeof(double2) * (size_t)n_angles));
    FBP_TRY(cudaMemcpy(p->d_cs2, cs.data(), sizeof(double2) * (size_t)n_angles, cudaMemcpyHostToDevice));
    FBP_TRY(cudaMalloc(&p->d_taps, p->esize * (size_t)tl));
    FBP_TRY(cudaMemcpy(p->d_taps, gsrc, p->esize * (size_t)tl, cudaMemcpyHostToDevice));
    FBP_TRY(cudaMalloc(&p->d_rho, p->esize * (size_t)n_det));
    FBP_TRY(cudaMemcpy(p->d_rho, rsrc, p->esize * (size_t)n_det, cudaMemcpyHostToDevice));
    FBP_TRY(cudaMalloc(&p->d_u, p->esize * 2 * (size_t)tl2 * kTabCopies));
    for (int c = 0; c < kTabCopies; ++c)
        FBP_TRY(cudaMemcpy(static_cast<char*>(p->d_u) + (size_t)c * p->esize * 2 * tl2, usrc, p->esize * 2 * (size_t)tl2,
                           cudaMemcpyHostToDevice));
    FBP_TRY(cudaMalloc(&p->d_rho2, p->esize * (size_t)n_det));
    FBP_TRY(cudaMemcpy(p->d_rho2, r2src, p->esize * (size_t)n_det, cudaMemcpyHostToDevice));
    // Optional (FBP_BP_RECS=1): back-projector records per (tile, angle) computed here in fp64 with the formulas of
    // the kernel's own path, so that the producer warp only copies them.  Measured on B200: no change in fp32
    // (the producer is not the limiter: cfg3 33.2 us either way) and slower in fp64 (32-byte records: 56 -> 73 us),
    // so it is off by default.
    {
        const size_t n_tiles = (size_t)p->bp.tiles_x * p->bp.tiles_y;
        const size_t bytes = n_tiles * n_angles * 4 * p->esize;
        if (bytes <= ((size_t)128 << 20) && env_int("FBP_BP_RECS", 0)) {
            std::vector<unsigned char> host(bytes);
            const int TH = p->bp_th, L = p->bp_seg;
            for (size_t t = 0; t < n_tiles; ++t) {
                const int ty = (int)(t / p->bp.tiles_x), tx = (int)(t % p->bp.tiles_x);
                const double x0 = (double)(tx * 32) - p->bp.c_n, y0 = (double)(ty * TH) - p->bp.c_n;
                for (int i = 0; i < n_angles; ++i) {
                    const double cx = cs[2 * i], sy = cs[2 * i + 1];
                    const double ub = x0 * cx + y0 * sy + p->bp.c_d;
                    const double umin = ub + std::fmin(0.0, 31.0 * cx) + std::fmin(0.0, (double)(TH - 1) * sy);
                    const double fl = std::floor(umin) - 1.0;
                    const bool on = fl >= -(double)p->bp.ent_guard && fl <= (double)(p->bp.ent_pitch - p->bp.ent_guard - L);
                    const int off = on ? (int)fl + p->bp.ent_guard : 0;
                    const size_t idx = t * n_angles + i;
                    if (dtype == FBP_F32) {
                        fbp::AngleRec<float> rc;
                        rc.c = on ? (float)cx : 0.f; rc.s = on ? (float)sy : 0.f; rc.b = on ? (float)(ub - fl - 0.5) : 1.f;
                        rc.pad = fbp::RecOffset<float>::put(off);
                        std::memcpy(host.data() + idx * sizeof(rc), &rc, sizeof(rc));
                    } else {
                        fbp::AngleRec<double> rc;
                        rc.c = on ? cx : 0.0; rc.s = on ? sy : 0.0; rc.b = on ? ub - fl - 0.5 : 1.0;
                        rc.pad = fbp::RecOffset<double>::put(off);
                        std::memcpy(host.data() + idx * sizeof(rc), &rc, sizeof(rc));
                    }
                }
            }
            FBP_TRY(cudaMalloc(&p->d_recs, bytes));
            FBP_TRY(cudaMemcpy(p->d_recs, host.data(), bytes, cudaMemcpyHostToDevice));
        }
        p->bp.recs = p->d_recs;
    }
    FBP_TRY(cudaMalloc(&p->d_ent, 4 * p->esize * (size_t)max_batch * n_angles * p->bp.ent_pitch));
    if (p->bp_splits > 1) {
        const size_t nt = (size_t)max_batch * p->bp.tiles_x * p->bp.tiles_y;
        FBP_TRY(cudaMalloc(&p->d_part, p->esize * (size_t)p->bp_splits * max_batch * image_n * image_n));
        FBP_TRY(cudaMalloc(&p->d_tickets, sizeof(int) * nt));
        FBP_TRY(cudaMemset(p->d_tickets, 0, sizeof(int) * nt));
    }
    FBP_TRY(cudaMalloc(&p->d_mscratch, sizeof(double) * (3 * kMetricGrid + 4)));
    FBP_TRY(cudaMemset(p->d_mscratch, 0, sizeof(double) * (3 * kMetricGrid + 4)));
    for (int i = 0; i < 4; ++i) FBP_TRY(cudaEventCreate(&p->ev[i]));
    p->pipe_min_batch = env_int("FBP_PIPE_MIN_BATCH", 8);
    p->pipe_group = env_int("FBP_PIPE_GROUP", 0);
    if (env_int("FBP_PIPE", 1) && max_batch >= p->pipe_min_batch) {
        int prio_lo = 0, prio_hi = 0;
        FBP_TRY(cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
        FBP_TRY(cudaStreamCreateWithPriority(&p->st_f, cudaStreamNonBlocking, prio_hi));
        for (int i = 0; i < 2; ++i) FBP_TRY(cudaStreamCreateWithPriority(&p->st_b[i], cudaStreamNonBlocking, prio_lo));
        FBP_TRY(cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming));
        for (int i = 0; i < fbp_plan::kMaxGroups; ++i) FBP_TRY(cudaEventCreateWithFlags(&p->ev_f[i], cudaEventDisableTiming));
        for (int i = 0; i < 2; ++i) FBP_TRY(cudaEventCreateWithFlags(&p->ev_b[i], cudaEventDisableTiming));
    }
#undef FBP_TRY
    *out = p;
    return FBP_OK;
}

void fbp_destroy(fbp_plan* p)
{
    if (!p) return;
    {
        DeviceGuard guard(p->device);
        cudaFree(p->d_cs2); cudaFree(p->d_taps); cudaFree(p->d_rho); cudaFree(p->d_ent); cudaFree(p->d_part); cudaFree(p->d_tickets);
        cudaFree(p->d_hsino); cudaFree(p->d_himg); cudaFree(p->d_u); cudaFree(p->d_rho2); cudaFree(p->d_mscratch);
        cudaFree(p->d_recs); cudaFree(p->d_ud); cudaFree(p->d_rhod); cudaFree(p->d_wrow); cudaFree(p->d_xt);
        for (int i = 0; i < 4; ++i) if (p->ev[i]) cudaEventDestroy(p->ev[i]);
        if (p->st_f) { cudaStreamSynchronize(p->st_f); cudaStreamDestroy(p->st_f); }
        for (int i = 0; i < 2; ++i) if (p->st_b[i]) { cudaStreamSynchronize(p->st_b[i]); cudaStreamDestroy(p->st_b[i]); }
        if (p->ev_fork) cudaEventDestroy(p->ev_fork);
        for (int i = 0; i < fbp_plan::kMaxGroups; ++i) if (p->ev_f[i]) cudaEventDestroy(p->ev_f[i]);
        for (int i = 0; i < 2; ++i) if (p->ev_b[i]) cudaEventDestroy(p->ev_b[i]);
        cudaGetLastError();
    }
    delete p;
}

const char* fbp_last_error(const fbp_plan* p) { return p ? p->err.c_str() : g_create_error.c_str(); }

}  // extern "C"

extern "C" {

fbp_status fbp_filter(fbp_plan* p, const void* d_sino, void* d_filtered, int batch, void* stream)
{
    fbp_status st = check_call(p, d_sino, d_filtered, batch);
    if (st != FBP_OK) return st;
    if (d_sino == d_filtered) return fail(p, FBP_EINVAL, "fbp_filter: input and output may not alias");
    DeviceGuard guard(p->device);
    p->ran_filter = p->ran_bp = false;
    return run_filter(p, d_sino, d_filtered, nullptr, batch, static_cast<cudaStream_t>(stream));
}

fbp_status fbp_backproject(fbp_plan* p, const void* d_filtered, void* d_image, int batch, void* stream)
{
    fbp_status st = check_call(p, d_filtered, d_image, batch);
    if (st != FBP_OK) return st;
    DeviceGuard guard(p->device);
    p->ran_filter = p->ran_bp = false;
    return run_bp(p, d_filtered, d_image, batch, static_cast<cudaStream_t>(stream));
}

fbp_status fbp_reconstruct(fbp_plan* p, const void* d_sino, void* d_image, int batch, void* stream)
{
    fbp_status st = check_call(p, d_sino, d_image, batch);
    if (st != FBP_OK) return st;
    DeviceGuard guard(p->device);
    p->ran_filter = p->ran_bp = false;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (use_pipeline(p, batch)) return run_pipelined(p, d_sino, d_image, batch, s);
    st = run_filter(p, d_sino, nullptr, p->d_ent, batch, s);
    if (st != FBP_OK) return st;
    return run_bp(p, nullptr, d_image, batch, s);
}

fbp_status fbp_reconstruct_host(fbp_plan* p, const void* h_sino, void* h_image, int batch, void* stream)
{
    if (!p) return FBP_EINVAL;
    if (!h_sino || !h_image) return fail(p, FBP_EINVAL, "NULL host pointer");
    if (batch < 1 || batch > p->max_batch) return fail(p, FBP_EINVAL, "batch must be in [1, max_batch]");
    DeviceGuard guard(p->device);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const size_t sino_bytes = p->esize * (size_t)p->K * p->D, img_bytes = p->esize * (size_t)p->N * p->N;
    if (!p->d_hsino) FBP_CUDA(p, cudaMalloc(&p->d_hsino, sino_bytes * p->max_batch));
    // Result: if h_image is pinned (device-accessible) host memory, the back-projector stores its pixels straight
    // into it -- coalesced 128-byte posted writes over PCIe that overlap the kernel -- instead of a device image
    // followed by a copy.  Pageable memory takes the staged path.
    void* img_target = nullptr;
    {
        cudaPointerAttributes attr{};
        if (cudaPointerGetAttributes(&attr, h_image) == cudaSuccess && attr.type == cudaMemoryTypeHost &&
            attr.devicePointer != nullptr && aligned16(attr.devicePointer) && p->host_zero_copy)
            img_target = attr.devicePointer;
        cudaGetLastError();
    }
    const bool staged = img_target == nullptr;
    if (staged) {
        if (!p->d_himg) FBP_CUDA(p, cudaMalloc(&p->d_himg, img_bytes * p->max_batch));
        img_target = p->d_himg;
    }
    p->ran_filter = p->ran_bp = false;
    fbp_status st;
    if (use_pipeline(p, batch)) {
        st = run_pipelined(p, p->d_hsino, img_target, batch, s, h_sino);
    } else {
        // Small pinned sinograms are read by the filter straight from host memory (each row once, by cp.async):
        // the rows stream in over PCIe while earlier rows are already being filtered, and one copy operation with
        // its launch gap disappears.  Large or pageable ones are copied first.
        const void* sino_src = p->d_hsino;
        {
            cudaPointerAttributes attr{};
            const int in_mode = env_int("FBP_HOST_ZERO_COPY_IN", 1);
            if (in_mode && p->host_zero_copy && sino_bytes * batch <= ((size_t)8 << 20) &&
                cudaPointerGetAttributes(&attr, h_sino) == cudaSuccess && attr.type == cudaMemoryTypeHost &&
                attr.devicePointer != nullptr && aligned16(attr.devicePointer))
                sino_src = attr.devicePointer;
            cudaGetLastError();
        }
        if (sino_src == p->d_hsino)
            FBP_CUDA(p, cudaMemcpyAsync(p->d_hsino, h_sino, sino_bytes * batch, cudaMemcpyHostToDevice, s));
        st = run_filter(p, sino_src, nullptr, p->d_ent, batch, s);
        if (st != FBP_OK) return st;
        st = run_bp(p, nullptr, img_target, batch, s);
    }
    if (st != FBP_OK) return st;
    if (staged) FBP_CUDA(p, cudaMemcpyAsync(h_image, p->d_himg, img_bytes * batch, cudaMemcpyDeviceToHost, s));
    FBP_CUDA(p, cudaStreamSynchronize(s));
    return FBP_OK;
}

}  // extern "C"

template <typename T>
static cudaError_t launch_metrics(fbp_plan* p, const void* x, const void* y, long long n, double max_val,
                                  double c1, double c2, double* d_out, cudaStream_t st)
{
    double* partial = p->d_mscratch;
    double* mid = p->d_mscratch + 3 * kMetricGrid;
    // at least 32 elements per thread: small inputs get few CTAs (fewer partials, fewer tickets on one counter)
    long long want = (n + 32LL * fbp::kMetricThreads - 1) / (32LL * fbp::kMetricThreads);
    const int grid = (int)(want < kMetricGrid ? (want < 1 ? 1 : want) : kMetricGrid);
    const T* a = static_cast<const T*>(x);
    const T* b = static_cast<const T*>(y);
    unsigned* ticket = reinterpret_cast<unsigned*>(mid + 3);      // zero-initialised at fbp_create, self re-arming
    fbp::metrics_partial_kernel<T, 0><<<grid, fbp::kMetricThreads, 0, st>>>(a, b, n, mid, partial, ticket, max_val, c1, c2, d_out);
    fbp::metrics_partial_kernel<T, 1><<<grid, fbp::kMetricThreads, 0, st>>>(a, b, n, mid, partial, ticket, max_val, c1, c2, d_out);
    return cudaGetLastError();
}

extern "C" {

fbp_status fbp_metrics(fbp_plan* p, const void* d_x, const void* d_y, long long n, double max_val, double c1,
                       double c2, double* d_out8, void* stream)
{
    if (!p) return FBP_EINVAL;
    if (!d_x || !d_y || !d_out8) return fail(p, FBP_EINVAL, "NULL device pointer");
    if (n < 1) return fail(p, FBP_EINVAL, "n must be >= 1");
    if (!(max_val > 0.0) || !std::isfinite(max_val)) return fail(p, FBP_EINVAL, "max_val must be finite and > 0");
    if ((reinterpret_cast<uintptr_t>(d_out8) & 7u) != 0) return fail(p, FBP_EINVAL, "d_out8 must be 8-byte aligned");
    if (c1 < 0.0) c1 = (0.01 * max_val) * (0.01 * max_val);
    if (c2 < 0.0) c2 = (0.03 * max_val) * (0.03 * max_val);
    DeviceGuard guard(p->device);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    cudaError_t e = p->dtype == FBP_F32 ? launch_metrics<float>(p, d_x, d_y, n, max_val, c1, c2, d_out8, s)
                                        : launch_metrics<double>(p, d_x, d_y, n, max_val, c1, c2, d_out8, s);
    if (e != cudaSuccess) return cuda_fail(p, e, "metrics launch");
    return FBP_OK;
}

fbp_status fbp_project(fbp_plan* p, const void* d_image, void* d_sino, int batch, void* stream)
{
    fbp_status st = check_call(p, d_image, d_sino, batch);
    if (st != FBP_OK) return st;
    if (d_image == d_sino) return fail(p, FBP_EINVAL, "fbp_project: input and output may not alias");
    DeviceGuard guard(p->device);
    // zero pad of the staged lines: the widest run is 2 E + 1 pixels, E <= ceil(sqrt(2) d/pix + 1/2) - 1
    const int e_max = (int)std::ceil(std::sqrt(2.0) * p->d / p->pix + 0.5) - 1;
    const int pad = round_up(2 * e_max + 2, 4);            // round(p*) is clamped to [-(E+1), N+E], the run adds +-E
    const size_t plane = (size_t)p->N * (p->N + 2 * pad);
    if (!p->d_xt) FBP_CUDA(p, cudaMalloc(&p->d_xt, p->esize * 2 * (size_t)p->max_batch * plane));
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    fbp::ProjParams prm{p->K, p->D, p->N, pad, 0.5 * (p->N - 1), 0.5 * (p->D - 1)};
    const dim3 tgrid((p->N + 31) / 32, (p->N + 31) / 32, batch), tblock(32, 8);
    const dim3 pgrid(((p->D + 1) / 2 + 127) / 128, p->K, batch);     // a thread owns a bin and its mirror bin
    if (p->dtype == FBP_F32) {
        float* xp = static_cast<float*>(p->d_xt);
        float* xtp = xp + (size_t)p->max_batch * plane;
        fbp::stage_image_kernel<float><<<tgrid, tblock, 0, s>>>(static_cast<const float*>(d_image), xp, xtp, p->N, pad);
        fbp::project_kernel<float><<<pgrid, 128, 0, s>>>(xp, xtp, static_cast<float*>(d_sino), p->d_cs2, prm);
    } else {
        double* xp = static_cast<double*>(p->d_xt);
        double* xtp = xp + (size_t)p->max_batch * plane;
        fbp::stage_image_kernel<double><<<tgrid, tblock, 0, s>>>(static_cast<const double*>(d_image), xp, xtp, p->N, pad);
        fbp::project_kernel<double><<<pgrid, 128, 0, s>>>(xp, xtp, static_cast<double*>(d_sino), p->d_cs2, prm);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(p, e, "projector launch");
    return FBP_OK;
}

fbp_status fbp_interpolate_stack(fbp_plan* p, const void* d_stack, int n_in, void* d_out, int n_out, void* stream)
{
    if (!p) return FBP_EINVAL;
    if (!d_stack || !d_out) return fail(p, FBP_EINVAL, "NULL device pointer");
    if (n_in < 1 || n_out < 1 || n_out > 65535) return fail(p, FBP_EINVAL, "n_in >= 1 and 1 <= n_out <= 65535 required");
    if (d_stack == d_out) return fail(p, FBP_EINVAL, "fbp_interpolate_stack: input and output may not alias");
    if ((reinterpret_cast<uintptr_t>(d_stack) | reinterpret_cast<uintptr_t>(d_out)) & (p->esize - 1))
        return fail(p, FBP_EINVAL, "device pointers must be aligned to the element size");
    DeviceGuard guard(p->device);
    const long long n_pix = (long long)p->N * p->N;
    const long long per_cta = (long long)fbp::kStackThreads * fbp::kStackVecPerThread * (16 / (long long)p->esize);
    dim3 grid((unsigned)((n_pix + per_cta - 1) / per_cta), (unsigned)n_out);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (p->dtype == FBP_F32)
        fbp::interpolate_stack_kernel<float><<<grid, fbp::kStackThreads, 0, s>>>(static_cast<const float*>(d_stack), n_in,
                                                                               static_cast<float*>(d_out), n_out, n_pix);
    else
        fbp::interpolate_stack_kernel<double><<<grid, fbp::kStackThreads, 0, s>>>(static_cast<const double*>(d_stack), n_in,
                                                                                static_cast<double*>(d_out), n_out, n_pix);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(p, e, "stack interpolation launch");
    return FBP_OK;
}

fbp_status fbp_set_window(fbp_plan* p, fbp_window window)
{
    if (!p) return FBP_EINVAL;
    if ((int)window < 0 || (int)window > (int)FBP_WINDOW_HANN) return fail(p, FBP_EINVAL, "unknown window");
    if (window == FBP_WINDOW_RAMLAK) { p->window = 0; return FBP_OK; }
    if (p->filter_v != 2 || p->f2d_threads > 512 || p->f2d_smem > 220 * 1024)
        return fail(p, FBP_EUNSUPPORTED, "n_det too large for the dense (windowed) row filter");
    DeviceGuard guard(p->device);
    FBP_CUDA(p, cudaDeviceSynchronize());          // nothing of this plan may be in flight while its tables change
    const fbp::Filter2Params& f = p->f2d;
    const int tl = f.tab_len, D = p->D, x_len = 2 * f.b_pad;
    std::vector<double> u64(2 * (size_t)tl), rho64(D);
    for (int j = 0; j < tl; ++j) {
        u64[j] = window_tap((int)window, 2LL * f.a_tot - j);
        u64[tl + j] = window_tap((int)window, 2LL * f.a_tot - j - 1);
    }
    // conditioning term: the dense filter's response to a constant row over the padded inputs,
    // rho[n] = sum_{k < x_len} H[n - k], summed smallest magnitudes first
    for (int n = 0; n < D; ++n) {
        std::vector<double> terms(x_len);
        for (int k = 0; k < x_len; ++k) terms[k] = window_tap((int)window, (long long)n - k);
        std::sort(terms.begin(), terms.end(), [](double a, double b) { return std::fabs(a) < std::fabs(b); });
        double ssum = 0.0;
        for (double t : terms) ssum += t;
        rho64[n] = ssum;
    }
    std::vector<float> u32, rho32;
    const void* usrc = u64.data();
    const void* rsrc = rho64.data();
    if (p->dtype == FBP_F32) {
        u32.assign(u64.begin(), u64.end()); usrc = u32.data();
        rho32.assign(rho64.begin(), rho64.end()); rsrc = rho32.data();
    }
    if (!p->d_ud) FBP_CUDA(p, cudaMalloc(&p->d_ud, p->esize * 2 * (size_t)tl * kTabCopies));
    if (!p->d_rhod) FBP_CUDA(p, cudaMalloc(&p->d_rhod, p->esize * (size_t)D));
    for (int c = 0; c < kTabCopies; ++c)
        FBP_CUDA(p, cudaMemcpy(static_cast<char*>(p->d_ud) + (size_t)c * p->esize * 2 * tl, usrc, p->esize * 2 * (size_t)tl,
                               cudaMemcpyHostToDevice));
    FBP_CUDA(p, cudaMemcpy(p->d_rhod, rsrc, p->esize * (size_t)D, cudaMemcpyHostToDevice));
    p->window = (int)window;
    return FBP_OK;
}

fbp_status fbp_set_angle_weights(fbp_plan* p, const double* h_weights)
{
    if (!p) return FBP_EINVAL;
    DeviceGuard guard(p->device);
    FBP_CUDA(p, cudaDeviceSynchronize());
    if (!h_weights) {
        cudaFree(p->d_wrow);
        p->d_wrow = nullptr;
        return FBP_OK;
    }
    if (p->filter_v != 2) return fail(p, FBP_EUNSUPPORTED, "angle weights need the paired-parity filter");
    for (int i = 0; i < p->K; ++i)
        if (!std::isfinite(h_weights[i])) return fail(p, FBP_EINVAL, "non-finite angle weight");
    // the back-projector keeps its pi/K factor: the entries of row i carry w_i / (pi/K)
    std::vector<double> m64(p->K);
    for (int i = 0; i < p->K; ++i) m64[i] = h_weights[i] * (double)p->K / kPi;
    std::vector<float> m32;
    const void* src = m64.data();
    if (p->dtype == FBP_F32) { m32.assign(m64.begin(), m64.end()); src = m32.data(); }
    if (!p->d_wrow) FBP_CUDA(p, cudaMalloc(&p->d_wrow, p->esize * (size_t)p->K));
    FBP_CUDA(p, cudaMemcpy(p->d_wrow, src, p->esize * (size_t)p->K, cudaMemcpyHostToDevice));
    return FBP_OK;
}

int fbp_plan_info(const fbp_plan* p, int* out, int n)
{
    if (!p) return 0;
    // kernels launched by fbp_reconstruct at batch = max_batch: filter + back-projection, per slice group when
    // the batch pipeline is on
    int launches = 2;
    if (use_pipeline(p, p->max_batch)) {
        int group = p->pipe_group > 0 ? p->pipe_group : (p->max_batch + 3) / 4;
        const int min_group = (p->max_batch + fbp_plan::kMaxGroups - 1) / fbp_plan::kMaxGroups;
        if (group < min_group) group = min_group;
        launches = 2 * ((p->max_batch + group - 1) / group);
    }
    const int v[14] = {p->bp_tw, p->bp_th, p->bp_r, p->bp_splits, p->bp_chunk, p->bp_seg,
                       p->bp.tiles_x * p->bp.tiles_y * p->bp_splits, p->bp_threads, p->bp_smem,
                       p->filter_v == 2 ? 2 * p->f2_r : p->f_r, p->filter_v == 2 ? p->f2_threads : p->f_threads,
                       p->filter_v == 2 ? p->f2.n_sb : p->fp.n_sb, p->filter_v == 2 ? p->f2_smem : p->f_smem,
                       launches};
    if (out) for (int i = 0; i < n && i < 14; ++i) out[i] = v[i];
    return 14;
}

fbp_status fbp_set_profiling(fbp_plan* p, int enable)
{
    if (!p) return FBP_EINVAL;
    p->profiling = enable != 0;
    p->ran_filter = p->ran_bp = false;
    return FBP_OK;
}

fbp_status fbp_get_kernel_ms(fbp_plan* p, float* filter_ms, float* backproject_ms)
{
    if (!p) return FBP_EINVAL;
    if (!p->profiling) return fail(p, FBP_EINVAL, "profiling is off (fbp_set_profiling)");
    DeviceGuard guard(p->device);
    float f = 0.f, b = 0.f;
    if (p->ran_filter) {
        FBP_CUDA(p, cudaEventSynchronize(p->ev[1]));
        FBP_CUDA(p, cudaEventElapsedTime(&f, p->ev[0], p->ev[1]));
    }
    if (p->ran_bp) {
        FBP_CUDA(p, cudaEventSynchronize(p->ev[3]));
        FBP_CUDA(p, cudaEventElapsedTime(&b, p->ev[2], p->ev[3]));
    }
    if (filter_ms) *filter_ms = f;
    if (backproject_ms) *backproject_ms = b;
    return FBP_OK;
}

}  // extern "C"

#ifdef FBP_TRACE
extern "C" int fbp_debug_read_trace(unsigned long long* out, int n)
{
    return (int)cudaMemcpyFromSymbol(out, fbp::g_trace, sizeof(unsigned long long) * (size_t)n);
}
#endif
