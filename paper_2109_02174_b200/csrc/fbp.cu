// fbp.cu -- libfbp: plan, launch configuration and the C ABI of include/fbp.h.
// Kernels: fbp_filter3.cuh / fbp_fft.cuh and fbp_backproject.cuh (eq. 2).
// This library has no CPU path and shares nothing with oracle/ (the test oracle).
// Nothing here reads the environment: behaviour depends on the arguments only (fbp_create_tuned).
#include "../../include/fbp.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "fbp_backproject.cuh"
#include "fbp_filter3.cuh"
#include "fbp_fft.cuh"
#include "fbp_metrics.cuh"
#include "fbp_stack.cuh"
#include "fbp_project.cuh"
#include "fbp_fdk.cuh"

namespace {

constexpr double kPi = 3.14159265358979323846264338327950288;
constexpr long double kPiL = 3.14159265358979323846264338327950288L;
constexpr int kMetricGridMax = 8 * 192;   // scratch for the CTA partials of fbp_metrics (grid = 8 per SM)

thread_local std::string g_create_error;

// Options of fbp_create_tuned (include/fbp.h); every field defaults to "the library's choice".
struct Tuning {
    int bp_variant = -1, bp_splits = 0, bp_chunk = 0;
    int filter_r = 0, filter_sb = 0, filter_kind = 0;
    int pipeline = -1, pipe_group = 0, pipe_min_batch = 8;
    int pdl = -1, host_zero_copy = -1, bp_even = -1;
};

}  // namespace

struct fbp_plan {
    fbp_dtype dtype = FBP_F32;
    int K = 0, D = 0, N = 0, max_batch = 0, device = 0, num_sm = 148;
    double d = 1.0, pix = 1.0;
    size_t esize = 4;
    Tuning tune;

    // device tables / scratch
    double2* d_cs2 = nullptr;   // [K] (cos, sin) * pix/d, fp64
    void* d_ent = nullptr;      // [max_batch][K][ent_pitch] 16-byte entries: back-projector operands (fbp_entries.cuh)
    void* d_part = nullptr;     // [S][max_batch][N][N] partial images when S > 1
    int* d_tickets = nullptr;   // [max_batch][tiles] arrival counters when S > 1 (self re-arming)
    void* d_hsino = nullptr;    // host-path staging (lazy)
    void* d_himg = nullptr;

    // back-projection configuration
    int bp_variant = 0;         // index into kBpVariants: (R, WY, WA)
    int bp_tw = 32, bp_th = 32, bp_r = 8, bp_threads = 128;
    int bp_splits = 1, bp_chunk = 1, bp_seg = 0, bp_smem = 0;
    fbp::BpParams bp{};

    // direct-form filter (fbp_filter3.cuh): [0] Ram-Lak (paired parity), [1] dense (apodised windows)
    struct F3 {
        bool ok = false;        // the geometry fits this kernel's shared-memory layout
        int r = 6, threads = 0, smem = 0, grid_cap = 0, a_lo = 0;
        fbp::Filter3Params prm{};
        void* d_u = nullptr;    // [2][tab_len] dtype: UA | UB
        void* d_rho = nullptr;  // [D] dtype: conditioning term
    } f3[2];
    // FFT-form filter (fbp_fft.cuh)
    struct Fft {
        bool ok = false;        // 2D <= 8192: the transform fits the kernel's instantiations
        int p = 0, threads = 0, smem = 0, buf_bytes = 0, grid_cap = 0;
        bool tab_smem = false;  // the table is staged in shared memory (it fits beside the transform buffer)
        void* d_tab = nullptr;  // complex dtype: per-pass twiddles [fft_tw_total(p)], then [N] the DFT of the circular
                                // kernel of the current window, / (d N)
    } fft;
    int filter_kind = 1;        // 1 direct form, 2 FFT form
    int window = 0;             // fbp_set_window; 0 = Ram-Lak
    void* d_xt = nullptr;       // 2 x [max_batch][N][pitch] pairs: padded image and padded transpose, each interleaved with its point mirror (fbp_project)
    void* d_fdk = nullptr;      // fbp_fdk_reconstruct: weighted | filtered cone-beam projections [K][n_rows][n_det], then the
                                // back-projector's zero-bordered 2 x 2 quads [K][n_rows + 2][n_det + 2][4]
    size_t fdk_elems = 0;
    void* d_wrow = nullptr;     // [K] dtype: angle weight / (pi/K) (fbp_set_angle_weights); NULL = uniform

    double* d_mscratch = nullptr;   // fbp_metrics: [kMetricGridMax][6] CTA partials, then the ticket
    int metric_ctas_per_sm = 0;     // co-resident CTAs of metrics_kernel per SM (occupancy query, first call)
    bool use_pdl = true;
    bool host_zero_copy = true;   // fbp_reconstruct_host: store results straight into pinned host memory
    // batch pipeline (run_pipelined): filter of slice group g+1 overlaps back-projection of group g
    static constexpr int kMaxGroups = 16;
    cudaStream_t st_f = nullptr, st_b[2] = {nullptr, nullptr};
    cudaEvent_t ev_fork = nullptr, ev_f[kMaxGroups] = {}, ev_b[2] = {nullptr, nullptr};
    unsigned long long* d_trace = nullptr;   // fbp_set_trace (caller-owned)
    long long trace_cap = 0;
    bool trace_launch = false;               // set by run_filter / run_bp around their own launch only: the batch pipeline's
                                             // groups and the cone-beam path's K x n_rows filter launch would overwrite or overrun
                                             // the records (include/fbp.h: "fbp_filter, fbp_backproject, fbp_reconstruct only")
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

// The trace buffer as THIS launch sees it: NULL unless tracing is on and the launch comes from run_filter / run_bp.
unsigned long long* trace_of(const fbp_plan* p) { return p->trace_launch ? p->d_trace : nullptr; }
struct TraceScope {
    fbp_plan* p;
    explicit TraceScope(fbp_plan* plan) : p(plan) { p->trace_launch = true; }
    ~TraceScope() { p->trace_launch = false; }
};

// The dynamic shared-memory limit is an attribute of the KERNEL (per context), not of a plan: plans with
// different geometries share the instantiations, so each one is opened up once per device to the device
// maximum (227 KB on sm_100, less the kernel's static shared memory).  One mutex serialises the
// bookkeeping: plans may be created and used from several host threads.
constexpr int kMaxDynSmem = 227 * 1024;
constexpr int kMaxDevices = 64;
std::mutex g_attr_mutex;
template <typename Kern>
cudaError_t allow_max_smem(Kern kern, bool (&done)[kMaxDevices], int device)
{
    std::lock_guard<std::mutex> lock(g_attr_mutex);
    const bool tracked = device >= 0 && device < kMaxDevices;
    if (tracked && done[device]) return cudaSuccess;
    cudaFuncAttributes fa{};
    cudaError_t e = cudaFuncGetAttributes(&fa, kern);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem - (int)fa.sharedSizeBytes);
    if (e == cudaSuccess && tracked) done[device] = true;
    return e;
}

// ---- taps (host, fp64 / long double) ------------------------------------------------------
// One tap of the apodised ramp |f| W(f), |f| <= 1/2: h_W[m] = 2 int_0^{1/2} f W(f) cos(2 pi f m) df in closed
// form (include/fbp.h, fbp_set_window; derivations in DESIGN.md "Windows").  Any integer m.
long double window_tap(int window, long long m)
{
    auto ramlak = [](long long q) -> long double {
        if (q == 0) return 0.25L;
        if (q % 2 == 0) return 0.0L;
        return -1.0L / (kPiL * kPiL * (long double)q * (long double)q);
    };
    auto half_moment = [](long double a) { return std::sin(0.5L * a) / (2.0L * a) + (std::cos(0.5L * a) - 1.0L) / (a * a); };
    const long double md = (long double)m;
    switch (window) {
        case FBP_WINDOW_SHEPP_LOGAN: return -2.0L / (kPiL * kPiL * (4.0L * md * md - 1.0L));
        case FBP_WINDOW_COSINE: return half_moment(kPiL * (2.0L * md + 1.0L)) + half_moment(kPiL * (2.0L * md - 1.0L));
        case FBP_WINDOW_HAMMING: return 0.54L * ramlak(m) + 0.23L * (ramlak(m + 1) + ramlak(m - 1));
        case FBP_WINDOW_HANN: return 0.5L * ramlak(m) + 0.25L * (ramlak(m + 1) + ramlak(m - 1));
        default: return ramlak(m);
    }
}

// ---- direct-form filter configuration (fbp_filter3.cuh) ------------------------------------
// A row is cut into U units of one warp-width (32 groups of R output pairs) on two grids that meet at M.
void configure_filter3(fbp_plan* p, bool dense)
{
    fbp_plan::F3& c = p->f3[dense ? 1 : 0];
    const int D = p->D;
    const int d_even = round_up(D, 4), M = d_even / 2;
    static const int cand_sparse[] = {6, 10, 14}, cand_dense[] = {5, 7, 9};
    const int* cand = dense ? cand_dense : cand_sparse;
    int best_r = cand[0];
    double best = -1.0;
    for (int i = 0; i < 3; ++i) {
        const int R = cand[i];
        // fp64: accumulators and the tap window take 4R (sparse) / 6R (dense) registers: larger R spills
        if (p->dtype == FBP_F64 && i > 0) continue;
        const int half = 32 * R;
        const int U = 1 + (std::max(0, M - half) + 30 * R - 1) / (30 * R);
        const double util = (double)D / ((double)U * 2 * half);
        const double score = util * (2.0 * R) / (2.0 * R + (dense ? 2.0 : 2.5));
        if (p->tune.filter_r == R) { best_r = R; best = 1e9; }
        if (score > best) { best = score; best_r = R; }
    }
    const int R = best_r, half = 32 * R;
    c.r = R;
    fbp::Filter3Params& f = c.prm;
    f.n_det = D; f.d_even = d_even; f.m_split = M;
    f.n_units = 1 + (std::max(0, M - half) + 30 * R - 1) / (30 * R);
    f.n_chunks = dense ? (D + 2 * R - 1) / (2 * R) : ((D + 1) / 2 + R - 1) / R;
    f.b_pad = f.n_chunks * R;
    // pair indices used: left blocks end at 15 R (U-1) + 16 R, the right grid ends at D'/2 and starts (innermost
    // unit) at (D' - 30 R (U-1) - 32 R) / 2, which is negative for short rows
    const int left_end = 15 * R * (f.n_units - 1) + 16 * R;
    f.a_hi = round_up(std::max(left_end, d_even / 2), 2);
    c.a_lo = std::min(0, d_even / 2 - left_end);
    f.tab_len = dense ? round_up(2 * (f.a_hi - c.a_lo) + 2 * f.b_pad + 4, 4) : round_up(f.a_hi - c.a_lo + f.b_pad + 2, 4);
    int sb = p->tune.filter_sb > 0 ? p->tune.filter_sb : 4;
    if (sb > 8) sb = 8;
    if (sb > f.n_chunks) sb = f.n_chunks;
    if (sb < 1) sb = 1;
    f.n_sb = sb;
    f.ent_pitch = p->bp.ent_pitch; f.ent_guard = p->bp.ent_guard;
    c.threads = 32 * sb;
    const int vec = 16 / (int)p->esize, d4 = round_up(D, vec);
    const size_t elems = 2 * (size_t)f.tab_len + (size_t)d4 + 2 * (size_t)(d4 + 2 * vec) + 2 * (size_t)f.b_pad +
                         (size_t)(sb + 1) * 2 * half + 32;
    c.smem = (int)(elems * p->esize + 16 + 16);
    c.ok = c.smem <= 200 * 1024;
    c.grid_cap = 0;
}

// ---- FFT-form filter configuration and tables (fbp_fft.cuh) -------------------------------
void configure_fft(fbp_plan* p)
{
    fbp_plan::Fft& c = p->fft;
    int pw = 6;
    while ((1 << pw) < 2 * p->D && pw < 20) ++pw;          // N = 2^pw >= 2 D (no wrap-around of the lags -D .. D-1), >= 64
    c.p = pw;
    c.ok = pw <= 13;
    if (!c.ok) return;
    const int n = 1 << pw, shift = p->dtype == FBP_F32 ? 5 : 4;
    c.threads = std::max(32, n / 16);
    const size_t fft_bytes = (size_t)(n + (n >> shift)) * 2 * p->esize;
    const size_t row_bytes = 2 * (size_t)(p->bp.ent_pitch + 2) * p->esize;
    c.buf_bytes = (int)((std::max(fft_bytes, row_bytes) + 15) / 16 * 16);
    const size_t tab_bytes = (size_t)(fbp::fft_tw_total(pw) + n) * 2 * p->esize;
    c.tab_smem = 16 + c.buf_bytes + tab_bytes <= 110 * 1024;     // at least two CTAs per SM
    c.smem = 16 + c.buf_bytes + (c.tab_smem ? (int)tab_bytes : 0);
    c.grid_cap = 0;
    if (c.smem > 200 * 1024) c.ok = false;
}

// in-place radix-2 FFT in long double (host; N a power of two): the kernel's DFT is computed once per window
void host_fft(std::vector<long double>& re, std::vector<long double>& im)
{
    const size_t n = re.size();
    for (size_t i = 1, j = 0; i < n; ++i) {
        size_t bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { std::swap(re[i], re[j]); std::swap(im[i], im[j]); }
    }
    for (size_t len = 2; len <= n; len <<= 1) {
        for (size_t k = 0; k < len / 2; ++k) {
            const long double ang = -2.0L * kPiL * (long double)k / (long double)len;
            const long double wr = std::cos(ang), wi = std::sin(ang);
            for (size_t i = k; i < n; i += len) {
                const size_t j = i + len / 2;
                const long double tr = re[j] * wr - im[j] * wi, ti = re[j] * wi + im[j] * wr;
                re[j] = re[i] - tr; im[j] = im[i] - ti;
                re[i] += tr; im[i] += ti;
            }
        }
    }
}

// Per-pass twiddles (once) and the DFT of the circular kernel c[l mod N] = g[l] / (d N), l = -D .. D-1, where
// g[l] = sum_{m <= l} h_W[m]: h_W is even and sums to zero (|f| W(f) vanishes at f = 0), so g[-1] = -h_W[0]/2 and
// every other g[l] follows by adding or subtracting finitely many closed-form taps.
template <typename T>
cudaError_t upload_fft_tables(fbp_plan* p, int window, bool twiddles)
{
    fbp_plan::Fft& c = p->fft;
    const int n = 1 << c.p, D = p->D, ntw = fbp::fft_tw_total(c.p);
    cudaError_t e;
    if (!c.d_tab && (e = cudaMalloc(&c.d_tab, sizeof(T) * 2 * (size_t)(ntw + n))) != cudaSuccess) return e;
    if (twiddles) {
        // [pass][r - 1][k] = exp(-2 pi i k r / (NS R)): the order in which the lanes of a pass read them
        std::vector<T> w(2 * (size_t)ntw);
        size_t o = 0;
        int ns = 16;
        for (int pass = 1; pass < fbp::fft_n_passes(c.p); ++pass) {
            const int R = fbp::fft_radix(c.p, pass);
            for (int r = 1; r < R; ++r)
                for (int k = 0; k < ns; ++k) {
                    const long double ang = 2.0L * kPiL * (long double)k * (long double)r / ((long double)ns * (long double)R);
                    w[o++] = (T)std::cos(ang); w[o++] = (T)(-std::sin(ang));
                }
            ns *= R;
        }
        if ((e = cudaMemcpy(c.d_tab, w.data(), sizeof(T) * w.size(), cudaMemcpyHostToDevice)) != cudaSuccess) return e;
    }
    std::vector<long double> re((size_t)n, 0.0L), im((size_t)n, 0.0L);
    const long double scale = 1.0L / ((long double)p->d * (long double)n);
    long double g = -0.5L * window_tap(window, 0);           // g[-1]
    re[(size_t)(n - 1)] = g * scale;
    for (long long l = -2; l >= -(long long)D; --l) { g -= window_tap(window, l + 1); re[(size_t)(n + l)] = g * scale; }
    g = -0.5L * window_tap(window, 0);
    for (long long l = 0; l <= (long long)D - 1; ++l) { g += window_tap(window, l); re[(size_t)l] = g * scale; }
    host_fft(re, im);
    std::vector<T> gt(2 * (size_t)n);
    for (int k = 0; k < n; ++k) { gt[2 * k] = (T)re[k]; gt[2 * k + 1] = (T)im[k]; }
    return cudaMemcpy(static_cast<T*>(c.d_tab) + 2 * (size_t)ntw, gt.data(), sizeof(T) * 2 * (size_t)n, cudaMemcpyHostToDevice);
}

// ---- back-projection launch configuration ------------------------------------------
// (R, WY, WA) instantiations of backproject_kernel, see launch_bp
constexpr int kNumBpVariants = 11;
constexpr int kBpVariants[kNumBpVariants][3] = {
    {8, 4, 1}, {4, 4, 1}, {4, 1, 4}, {5, 1, 4}, {6, 1, 4}, {7, 1, 4}, {8, 1, 4},
    {4, 1, 8}, {6, 1, 8}, {7, 1, 8}, {8, 1, 8}};
void configure_bp(fbp_plan* p, const std::vector<double>& cs)
{
    const int N = p->N, K = p->K, num_sm = p->num_sm;
    const int half_rows = (N + 1) / 2;  // primary (top) half; the mirror pixels come for free
    const int tiles_x = (N + p->bp_tw - 1) / p->bp_tw;
    // variant = (R rows per thread, WY warps along y, WA angle groups): tile 32 x (R*WY) primary pixels
    int v = p->tune.bp_variant;
    if (v < 0 || v >= kNumBpVariants) {
        // Small launches (one 512^2 slice is 16 column strips x 256 primary rows) are chosen to fill
        // the SMs evenly: short tiles of R rows with 4 angle groups, R picked so that the number of
        // CTAs is as close as possible to a whole number of waves.  Large launches take the 32x32
        // tile (a third of the L2->shared staging traffic per update).
        const long big = (long)tiles_x * ((half_rows + 31) / 32) * p->max_batch;
        if (big >= 8L * num_sm) {
            v = 0;
        } else {
            double best = -1.0;
            v = 3;
            for (int cand = 2; cand <= 6; ++cand) {
                const int th = kBpVariants[cand][0] * kBpVariants[cand][1];
                const long ctas = (long)tiles_x * ((half_rows + th - 1) / th) * p->max_batch;
                const long waves = (ctas + 4L * num_sm - 1) / (4L * num_sm);   // 4 CTAs of 4 warps per SM
                const double fill = (double)ctas / (double)(waves * 4L * num_sm);
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

    // angle splits: fill the SMs evenly when one launch has few tiles
    const long tiles = (long)tiles_x * tiles_y * p->max_batch;
    int S = p->tune.bp_splits;
    if (S <= 0) {
        const int s_max = K / 16 > 1 ? (K / 16 < 16 ? K / 16 : 16) : 1;
        double best = -1.0;
        S = 1;
        for (int s = 1; s <= s_max; ++s) {
            const long ctas = tiles * s;
            const long waves = (ctas + num_sm - 1) / num_sm;
            double eff = (double)ctas / (double)(waves * num_sm);
            if (ctas < 4L * num_sm) eff *= 0.5 + 0.5 * (double)ctas / (4.0 * num_sm);
            eff -= 0.01 * (s - 1);  // splitting is not free: prefer fewer splits on ties
            if (eff > best) { best = eff; S = s; }
        }
    }
    if (S > K) S = K;
    if (S > 64) S = 64;
    if (S < 1) S = 1;
    p->bp_splits = S;
    const int per = (K + S - 1) / S;

    const size_t entry = 16, rec = 4 * p->esize;
    const size_t per_angle = (size_t)p->bp_seg * entry + rec;
    // A small launch (c CTAs per SM on average, c <= 5) is placed evenly only if no SM can hold more
    // than c of its CTAs: with programmatic dependent launch the CTAs arrive while the filter is
    // still draining and would otherwise pile up (up to 6 per SM) on the SMs that free up first.
    // Sizing the dynamic shared memory so that c + 1 CTAs do not fit caps the residency at c; the
    // extra room goes to longer chunks (fewer chunk boundaries: 33.6 -> 33.3 us at config 3).
    int even_smem = 0;
    {
        const long ctas = tiles * S;
        const int cps = (int)((ctas + num_sm - 1) / num_sm);
        const int smem_sm = 228 * 1024, reserve = 1024;
        if (cps >= 1 && cps <= 5 && p->tune.bp_even != 0) {
            const int want = smem_sm / (cps + 1) - reserve + 256;
            if ((long)cps * (want + reserve) <= smem_sm) even_smem = want;
        }
    }
    const int wa = kBpVariants[v][2];
    const int budget = even_smem > 36 * 1024 ? even_smem - 512 : 36 * 1024;
    int chunk = p->tune.bp_chunk;
    if (chunk <= 0) {
        chunk = (int)(budget / (fbp::kBpStages * per_angle));
        if (chunk > 32) chunk = 32;                       // one producer lane per angle of a chunk
        if (chunk > wa) chunk -= chunk % wa;              // equal work for the angle groups
    }
    if (chunk > 32) chunk = 32;
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
    b.c_n = 0.5 * (N - 1); b.c_d = 0.5 * (p->D - 1);
    b.scale = kPi / K;
    b.trace = nullptr;
}

// ---- host tables of the direct-form filter ---------------------------------------------------
// U tables (UA | UB) and the conditioning term rho[n] = the filter's response to a constant row over the
// padded input range.  rho comes from long-double prefix sums of the taps over the lag axis (O(D), no
// sorting: |error| ~ D * 2^-64 * max|h|, far below fp64 rounding of the table itself).
template <typename T>
cudaError_t upload_filter3_tables(fbp_plan* p, bool dense, int window)
{
    fbp_plan::F3& c = p->f3[dense ? 1 : 0];
    const fbp::Filter3Params& f = c.prm;
    const int tl = f.tab_len, D = p->D;
    std::vector<T> u(2 * (size_t)tl), rho((size_t)round_up(D, 4), T(0));   // rho padded to 16 bytes (bulk copy)
    if (!dense) {
        auto gq = [](long long q) -> long double { const long double m = 2.0L * (long double)q + 1.0L; return -1.0L / (kPiL * kPiL * m * m); };
        for (int j = 0; j < tl; ++j) {
            u[j] = (T)gq((long long)f.a_hi - 1 - j);
            u[tl + j] = (T)gq((long long)f.a_hi - 2 - j);
        }
        // rho[n] = 1/4 + sum_{b < b_pad} g[a - b - (1 - par)], n = 2a + par: prefix sums G(q) = sum_{t <= q} g[t], t >= q_min
        const long long q_min = -(long long)f.b_pad - 2, q_max = D / 2 + 2;
        std::vector<long double> G((size_t)(q_max - q_min + 1));
        long double run = 0.0L;
        for (long long q = q_min; q <= q_max; ++q) { run += gq(q); G[(size_t)(q - q_min)] = run; }
        for (int n = 0; n < D; ++n) {
            const long long q0 = (n >> 1) - (1 - (n & 1));
            rho[n] = (T)(0.25L + G[(size_t)(q0 - q_min)] - G[(size_t)(q0 - f.b_pad - q_min)]);
        }
    } else {
        for (int j = 0; j < tl; ++j) {
            u[j] = (T)window_tap(window, 2LL * f.a_hi - j);
            u[tl + j] = (T)window_tap(window, 2LL * f.a_hi - j - 1);
        }
        // rho[n] = sum_{k < 2 b_pad} H[n - k]: prefix sums C(L) = sum_{m <= L} H[m], m >= m_min
        const long long x_len = 2LL * f.b_pad, m_min = -x_len - 1, m_max = D;
        std::vector<long double> C((size_t)(m_max - m_min + 1));
        long double run = 0.0L;
        for (long long m = m_min; m <= m_max; ++m) { run += window_tap(window, m); C[(size_t)(m - m_min)] = run; }
        for (int n = 0; n < D; ++n) rho[n] = (T)(C[(size_t)(n - m_min)] - C[(size_t)(n - x_len - m_min)]);
    }
    cudaError_t e;
    if (!c.d_u && (e = cudaMalloc(&c.d_u, sizeof(T) * 2 * (size_t)tl)) != cudaSuccess) return e;
    if (!c.d_rho && (e = cudaMalloc(&c.d_rho, sizeof(T) * rho.size())) != cudaSuccess) return e;
    if ((e = cudaMemcpy(c.d_u, u.data(), sizeof(T) * 2 * (size_t)tl, cudaMemcpyHostToDevice)) != cudaSuccess) return e;
    return cudaMemcpy(c.d_rho, rho.data(), sizeof(T) * rho.size(), cudaMemcpyHostToDevice);
}

// ---- kernel launchers ---------------------------------------------------------------
// filt and/or ent may be NULL: plain rows (fbp_filter) and/or entries (fbp_reconstruct)
// rows: rows per slice (the plan's K, or K * n_rows for the cone-beam path, whose rows carry no entries)
template <typename T, int R, bool DENSE>
cudaError_t launch_filter3_r(fbp_plan* p, const void* sino, void* filt, void* ent, int batch, cudaStream_t st, int rows)
{
    fbp_plan::F3& c = p->f3[DENSE ? 1 : 0];
    fbp::Filter3Params f = c.prm;
    f.n_rows = batch * rows;
    f.trace = nullptr;
    auto kern = fbp::filter3_kernel<T, R, DENSE>;
    static bool smem_open[kMaxDevices] = {};
    if (cudaError_t e = allow_max_smem(kern, smem_open, p->device); e != cudaSuccess) return e;
    if (c.grid_cap == 0) {
        int per_sm = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, c.threads, c.smem);
        if (e != cudaSuccess) return e;
        if (per_sm < 1) return cudaErrorLaunchOutOfResources;
        c.grid_cap = per_sm * p->num_sm;
    }
    // persistent: never more CTAs than are co-resident (tables staged once per CTA)
    const long long work = (long long)f.n_rows * f.n_units;
    const int grid = (int)std::min<long long>(work, c.grid_cap);
    if (trace_of(p) && 8LL * grid <= p->trace_cap) f.trace = trace_of(p);
    kern<<<grid, c.threads, c.smem, st>>>(static_cast<const T*>(sino), static_cast<T*>(filt), static_cast<uint4*>(ent),
                                          static_cast<const T*>(c.d_u), static_cast<const T*>(c.d_rho),
                                          static_cast<const T*>(p->d_wrow), p->K, f, (T)(1.0 / p->d));
    return cudaGetLastError();
}

template <typename T, int P, bool TSMEM>
cudaError_t launch_fft_p(fbp_plan* p, const void* sino, void* filt, void* ent, int batch, cudaStream_t st, int rows)
{
    fbp_plan::Fft& c = p->fft;
    auto kern = fbp::fft_filter_kernel<T, P, TSMEM>;
    static bool smem_open[kMaxDevices] = {};
    if (cudaError_t e = allow_max_smem(kern, smem_open, p->device); e != cudaSuccess) return e;
    if (c.grid_cap == 0) {
        int per_sm = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, c.threads, c.smem);
        if (e != cudaSuccess) return e;
        if (per_sm < 1) return cudaErrorLaunchOutOfResources;
        c.grid_cap = per_sm * p->num_sm;
    }
    fbp::FftParams f{batch, rows, p->D, (rows + 1) / 2, p->bp.ent_pitch, p->bp.ent_guard, c.buf_bytes,
                     ent ? p->d_cs2 : nullptr, (int)(sizeof(double2) * (size_t)p->K), nullptr};
    const long long work = (long long)batch * f.pairs_per_slice;
    const int grid = (int)std::min<long long>(work, c.grid_cap);
    if (trace_of(p) && 8LL * grid <= p->trace_cap) f.trace = trace_of(p);
    kern<<<grid, c.threads, c.smem, st>>>(static_cast<const T*>(sino), static_cast<T*>(filt), static_cast<uint4*>(ent),
                                          static_cast<const fbp::Cx<T>*>(c.d_tab), static_cast<const T*>(p->d_wrow), f);
    return cudaGetLastError();
}

template <typename T, bool TSMEM>
cudaError_t launch_fft_t(fbp_plan* p, const void* sino, void* filt, void* ent, int batch, cudaStream_t st, int rows)
{
    switch (p->fft.p) {
        case 6: return launch_fft_p<T, 6, TSMEM>(p, sino, filt, ent, batch, st, rows);
        case 7: return launch_fft_p<T, 7, TSMEM>(p, sino, filt, ent, batch, st, rows);
        case 8: return launch_fft_p<T, 8, TSMEM>(p, sino, filt, ent, batch, st, rows);
        case 9: return launch_fft_p<T, 9, TSMEM>(p, sino, filt, ent, batch, st, rows);
        case 10: return launch_fft_p<T, 10, TSMEM>(p, sino, filt, ent, batch, st, rows);
        case 11: return launch_fft_p<T, 11, TSMEM>(p, sino, filt, ent, batch, st, rows);
        case 12: return launch_fft_p<T, 12, TSMEM>(p, sino, filt, ent, batch, st, rows);
        default: return launch_fft_p<T, 13, TSMEM>(p, sino, filt, ent, batch, st, rows);
    }
}
template <typename T>
cudaError_t launch_fft(fbp_plan* p, const void* sino, void* filt, void* ent, int batch, cudaStream_t st, int rows)
{
    return p->fft.tab_smem ? launch_fft_t<T, true>(p, sino, filt, ent, batch, st, rows)
                           : launch_fft_t<T, false>(p, sino, filt, ent, batch, st, rows);
}

template <typename T>
cudaError_t launch_filter(fbp_plan* p, const void* sino, void* filt, void* ent, int batch, cudaStream_t st, int rows = 0)
{
    if (rows <= 0) rows = p->K;
    if (p->filter_kind == 2) return launch_fft<T>(p, sino, filt, ent, batch, st, rows);
    if (p->window != 0) {
        switch (p->f3[1].r) {
            case 5: return launch_filter3_r<T, 5, true>(p, sino, filt, ent, batch, st, rows);
            case 7: return launch_filter3_r<T, 7, true>(p, sino, filt, ent, batch, st, rows);
            default: return launch_filter3_r<T, 9, true>(p, sino, filt, ent, batch, st, rows);
        }
    }
    switch (p->f3[0].r) {
        case 6: return launch_filter3_r<T, 6, false>(p, sino, filt, ent, batch, st, rows);
        case 10: return launch_filter3_r<T, 10, false>(p, sino, filt, ent, batch, st, rows);
        default: return launch_filter3_r<T, 14, false>(p, sino, filt, ent, batch, st, rows);
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

// filter CTAs per launch at batch = max_batch (plan_info[16]); 0 until the filter has run once
long long filter_ctas(const fbp_plan* p)
{
    if (p->filter_kind == 2)
        return p->fft.grid_cap > 0 ? std::min<long long>((long long)p->max_batch * ((p->K + 1) / 2), p->fft.grid_cap) : 0;
    const fbp_plan::F3& f = p->f3[p->window != 0 ? 1 : 0];
    return f.grid_cap > 0 ? std::min<long long>((long long)p->max_batch * p->K * f.prm.n_units, f.grid_cap) : 0;
}

template <typename T, int R, int WY, int WA, bool TRACE>
cudaError_t launch_bp_t(fbp_plan* p, void* image, int batch, cudaStream_t st, int slice0)
{
    auto kern = fbp::backproject_kernel<T, R, WY, WA, TRACE>;
    static bool smem_open[kMaxDevices] = {};     // per instantiation and device
    if (cudaError_t e = allow_max_smem(kern, smem_open, p->device); e != cudaSuccess) return e;
    // programmatic dependent launch: the CTAs may become resident and run their prologue while the
    // kernel that writes the entries (filter / entries_kernel) drains; they block in griddepcontrol.wait
    // before the first read of the entries
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
                       (size_t)slice0 * p->K * p->bp.ent_pitch;
    fbp::BpParams prm = p->bp;
    // trace records of the back-projector follow the filter's (fbp_set_trace)
    prm.trace = nullptr;
    if (trace_of(p)) {
        const long long f_ctas = filter_ctas(p);   // plan_info[16]
        const long long b_ctas = (long long)cfg.gridDim.x * cfg.gridDim.y * cfg.gridDim.z;
        if (8 * (f_ctas + b_ctas) <= p->trace_cap) prm.trace = p->d_trace + 8 * f_ctas;
    }
    return cudaLaunchKernelEx(&cfg, kern, ent, static_cast<T*>(image),
                              static_cast<const double2*>(p->d_cs2), static_cast<T*>(p->d_part), p->d_tickets, prm);
}

template <typename T, int R, int WY, int WA>
cudaError_t launch_bp_v(fbp_plan* p, void* image, int batch, cudaStream_t st, int slice0)
{
    return trace_of(p) ? launch_bp_t<T, R, WY, WA, true>(p, image, batch, st, slice0)
                      : launch_bp_t<T, R, WY, WA, false>(p, image, batch, st, slice0);
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
    TraceScope traced(p);
    cudaError_t e = p->dtype == FBP_F32 ? launch_filter<float>(p, sino, filt, ent, batch, st)
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
    TraceScope traced(p);
    e = p->dtype == FBP_F32 ? launch_bp<float>(p, image, batch, st) : launch_bp<double>(p, image, batch, st);
    if (e != cudaSuccess) return cuda_fail(p, e, "back-projection launch");
    if (p->profiling) FBP_CUDA(p, cudaEventRecord(p->ev[3], st));
    p->ran_bp = true;
    return FBP_OK;
}

int pipe_group_size(const fbp_plan* p, int batch)
{
    int group = p->tune.pipe_group > 0 ? p->tune.pipe_group : (batch + 3) / 4;   // 4 groups measured best at 64 slices
    const int min_group = (batch + fbp_plan::kMaxGroups - 1) / fbp_plan::kMaxGroups;
    return group < min_group ? min_group : group;
}

// fbp_reconstruct for a stack of slices, group by group.  The batch is cut into groups; group g+1 is filtered on a
// plan-owned high-priority stream while group g is back-projected on one of two other plan-owned streams (two, so
// that the tail of one launch overlaps the head of the next).  The caller's stream forks into them and joins at the
// end: still enqueue-only, no host wait.  Same kernels on the same data as the sequential path, hence the same bytes.
// What it buys, measured on B200 at config 4 (64 slices): with HOST buffers (fbp_reconstruct_host) each group's
// host-to-device copy rides the filter stream under the previous group's back-projection -- that is the case it is
// kept for.  With device-resident data the FFT-form filter (shared-memory and latency bound, ~12 % of the step) and
// the back-projector (shared-memory operand bound) compete for the same SMs and the step is within 1 % of the two
// launches in sequence (profiles/r3_bench.md); it stays on there only so that both entry points run one code path.
fbp_status run_pipelined(fbp_plan* p, const void* sino, void* image, int batch, cudaStream_t s,
                         const void* h_sino = nullptr)
{
    const int group = pipe_group_size(p, batch);
    const int n_groups = (batch + group - 1) / group;
    const size_t sino_slice = p->esize * (size_t)p->K * p->D, img_slice = p->esize * (size_t)p->N * p->N;
    const size_t ent_slice = 16 * (size_t)p->K * p->bp.ent_pitch;
    FBP_CUDA(p, cudaEventRecord(p->ev_fork, s));
    FBP_CUDA(p, cudaStreamWaitEvent(p->st_f, p->ev_fork, 0));
    FBP_CUDA(p, cudaStreamWaitEvent(p->st_b[0], p->ev_fork, 0));
    FBP_CUDA(p, cudaStreamWaitEvent(p->st_b[1], p->ev_fork, 0));
    // a failure below must not leave the plan's streams forked off the caller's: they are always joined
    // back before returning, so whatever was enqueued still completes in stream order
    cudaError_t err = cudaSuccess;
    const char* what = "";
    for (int g = 0; g < n_groups && err == cudaSuccess; ++g) {
        const int g0 = g * group, nb = batch - g0 < group ? batch - g0 : group;
        const char* sg = static_cast<const char*>(sino) + (size_t)g0 * sino_slice;
        char* eg = static_cast<char*>(p->d_ent) + (size_t)g0 * ent_slice;
        // host source (fbp_reconstruct_host): this group's copy rides the filter stream, so it overlaps the
        // back-projection of the previous group on the copy engine
        if (h_sino) {
            err = cudaMemcpyAsync(const_cast<char*>(sg), static_cast<const char*>(h_sino) + (size_t)g0 * sino_slice,
                                  (size_t)nb * sino_slice, cudaMemcpyHostToDevice, p->st_f);
            if (err != cudaSuccess) { what = "host-to-device copy"; break; }
        }
        err = p->dtype == FBP_F32 ? launch_filter<float>(p, sg, nullptr, eg, nb, p->st_f)
                                  : launch_filter<double>(p, sg, nullptr, eg, nb, p->st_f);
        if (err != cudaSuccess) { what = "filter launch"; break; }
        if ((err = cudaEventRecord(p->ev_f[g], p->st_f)) != cudaSuccess) { what = "cudaEventRecord"; break; }
        cudaStream_t sb = p->st_b[g & 1];
        if ((err = cudaStreamWaitEvent(sb, p->ev_f[g], 0)) != cudaSuccess) { what = "cudaStreamWaitEvent"; break; }
        char* ig = static_cast<char*>(image) + (size_t)g0 * img_slice;
        err = p->dtype == FBP_F32 ? launch_bp<float>(p, ig, nb, sb, g0) : launch_bp<double>(p, ig, nb, sb, g0);
        if (err != cudaSuccess) { what = "back-projection launch"; break; }
    }
    cudaEventRecord(p->ev_fork, p->st_f);             // (its earlier waiters captured the earlier record)
    cudaStreamWaitEvent(s, p->ev_fork, 0);
    for (int i = 0; i < 2; ++i) {
        const cudaError_t e1 = cudaEventRecord(p->ev_b[i], p->st_b[i]);
        const cudaError_t e2 = cudaStreamWaitEvent(s, p->ev_b[i], 0);
        if (err == cudaSuccess && (e1 != cudaSuccess || e2 != cudaSuccess)) { err = e1 != cudaSuccess ? e1 : e2; what = "stream join"; }
    }
    p->ran_filter = p->ran_bp = false;
    if (err != cudaSuccess) return cuda_fail(p, err, what);
    return FBP_OK;
}

bool use_pipeline(const fbp_plan* p, int batch)
{
    return p->st_f && !p->profiling && p->bp_splits == 1 && batch >= p->tune.pipe_min_batch;
}

fbp_status create_impl(fbp_plan** out, int n_angles, int n_det, const double* angles_rad, double det_spacing,
                       int image_n, double pixel_size, fbp_dtype dtype, int max_batch, int device, const Tuning& tune)
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
    // FBP_OPT_FILTER_R names a group size of the direct-form filter: 6, 10, 14 (Ram-Lak, sparse taps) or 5, 7, 9
    // (windowed, dense taps); fp64 plans have the smallest of each only (larger ones spill).  A value the plan
    // cannot honour is an error, not a silent fallback to the library's choice.
    if (tune.filter_r != 0) {
        const int r = tune.filter_r;
        const bool known = r == 5 || r == 6 || r == 7 || r == 9 || r == 10 || r == 14;
        if (!known) return fail(nullptr, FBP_EINVAL, "FBP_OPT_FILTER_R must be one of 6, 10, 14 (Ram-Lak) or 5, 7, 9 (windowed)");
        if (dtype == FBP_F64 && r != 5 && r != 6)
            return fail(nullptr, FBP_EINVAL, "FBP_OPT_FILTER_R: fp64 plans run the direct-form filter with R = 6 (Ram-Lak) or 5 (windowed) only");
    }
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
    p->num_sm = prop.multiProcessorCount > 0 ? prop.multiProcessorCount : 148;   // grids are sized from the device, not from a constant
    p->tune = tune;

    // host tables in fp64: (cos, sin) * pix/d  (A0 of SURVEY.md 8(a))
    std::vector<double> cs(2 * (size_t)n_angles);
    const double ratio = pix / det_spacing;
    for (int i = 0; i < n_angles; ++i) {
        cs[2 * i] = std::cos(angles_rad[i]) * ratio;
        cs[2 * i + 1] = std::sin(angles_rad[i]) * ratio;
    }
    configure_bp(p, cs);
    configure_filter3(p, false);   // after configure_bp: needs the entry pitch
    configure_filter3(p, true);
    configure_fft(p);
    // FFT form where the transform has 2048 .. 8192 points (it does ~D / (10 log2 D) times less work than the direct
    // form and is better conditioned in fp32); the direct form for longer rows, on request, and for short rows
    // (2 D <= 1024), where a transform is one or two warps and latency-bound: measured 8.6 vs 18.9 us at D = 91 and
    // 9.4 vs 12.7 us at D = 363 for one sinogram
    const bool fft_pays = p->fft.ok && p->fft.p >= 11;
    p->filter_kind = tune.filter_kind == 1 ? 1 : (tune.filter_kind == 2 ? 2 : (fft_pays ? 2 : 1));
    if (p->filter_kind == 2 && !p->fft.ok) p->filter_kind = p->f3[0].ok ? 1 : 2;
    if (p->filter_kind == 1 && !p->f3[0].ok && p->fft.ok) p->filter_kind = 2;
    p->use_pdl = tune.pdl != 0;
    p->host_zero_copy = tune.host_zero_copy != 0;

    auto bail = [&](fbp_status st) { std::string m = p->err; fbp_destroy(p); g_create_error = m; return st; };
    if (!p->f3[0].ok && !p->fft.ok) { p->err = "n_det too large for the shared-memory row filter"; return bail(FBP_EUNSUPPORTED); }
    if (p->bp_smem > 220 * 1024) { p->err = "pixel_size/det_spacing too large for the staged segment"; return bail(FBP_EUNSUPPORTED); }

    DeviceGuard guard(device);
    if (!guard.ok) { p->err = "cudaSetDevice failed"; return bail(FBP_ECUDA); }

#define FBP_TRY(call)                                                            \
    do {                                                                         \
        cudaError_t e__ = (call);                                                \
        if (e__ != cudaSuccess) return bail(cuda_fail(p, e__, #call));           \
    } while (0)
    FBP_TRY(cudaMalloc(&p->d_cs2, sizeof(double2) * (size_t)n_angles));
    FBP_TRY(cudaMemcpy(p->d_cs2, cs.data(), sizeof(double2) * (size_t)n_angles, cudaMemcpyHostToDevice));
    if (p->filter_kind == 1)
        FBP_TRY(dtype == FBP_F32 ? upload_filter3_tables<float>(p, false, 0) : upload_filter3_tables<double>(p, false, 0));
    else
        FBP_TRY(dtype == FBP_F32 ? upload_fft_tables<float>(p, 0, true) : upload_fft_tables<double>(p, 0, true));
    // entries: zero-filled once, so that the guard entries (never written by the filter) read as zeros
    const size_t ent_bytes = 16 * (size_t)max_batch * n_angles * p->bp.ent_pitch;
    FBP_TRY(cudaMalloc(&p->d_ent, ent_bytes));
    FBP_TRY(cudaMemset(p->d_ent, 0, ent_bytes));
    if (p->bp_splits > 1) {
        const size_t nt = (size_t)max_batch * p->bp.tiles_x * p->bp.tiles_y;
        FBP_TRY(cudaMalloc(&p->d_part, p->esize * (size_t)p->bp_splits * max_batch * image_n * image_n));
        FBP_TRY(cudaMalloc(&p->d_tickets, sizeof(int) * nt));
        FBP_TRY(cudaMemset(p->d_tickets, 0, sizeof(int) * nt));
    }
    FBP_TRY(cudaMalloc(&p->d_mscratch, sizeof(double) * (fbp::kMetricSums * kMetricGridMax + 8)));
    FBP_TRY(cudaMemset(p->d_mscratch, 0, sizeof(double) * (fbp::kMetricSums * kMetricGridMax + 8)));
    for (int i = 0; i < 4; ++i) FBP_TRY(cudaEventCreate(&p->ev[i]));
    if (tune.pipeline != 0 && max_batch >= tune.pipe_min_batch) {
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

}  // namespace

// ---- C ABI ----------------------------------------------------------------------------
extern "C" {

fbp_status fbp_create(fbp_plan** out, int n_angles, int n_det, const double* angles_rad,
                      double det_spacing, int image_n, double pixel_size, fbp_dtype dtype,
                      int max_batch, int device)
{
    return create_impl(out, n_angles, n_det, angles_rad, det_spacing, image_n, pixel_size, dtype, max_batch, device, Tuning{});
}

fbp_status fbp_create_tuned(fbp_plan** out, int n_angles, int n_det, const double* angles_rad,
                            double det_spacing, int image_n, double pixel_size, fbp_dtype dtype,
                            int max_batch, int device, const int* h_options, int n_options)
{
    Tuning t;
    if (out) *out = nullptr;
    if (n_options < 0 || (n_options > 0 && !h_options)) return fail(nullptr, FBP_EINVAL, "bad option list");
    for (int i = 0; i < n_options; ++i) {
        const int key = h_options[2 * i], val = h_options[2 * i + 1];
        switch (key) {
            case FBP_OPT_BP_VARIANT: t.bp_variant = val; break;
            case FBP_OPT_BP_SPLITS: t.bp_splits = val; break;
            case FBP_OPT_BP_CHUNK: t.bp_chunk = val; break;
            case FBP_OPT_FILTER_R: t.filter_r = val; break;
            case FBP_OPT_FILTER_SB: t.filter_sb = val; break;
            case FBP_OPT_FILTER_KIND: t.filter_kind = val; break;
            case FBP_OPT_PIPELINE: t.pipeline = val; break;
            case FBP_OPT_PIPE_GROUP: t.pipe_group = val; break;
            case FBP_OPT_PIPE_MIN_BATCH: t.pipe_min_batch = val < 1 ? 1 : val; break;
            case FBP_OPT_PDL: t.pdl = val; break;
            case FBP_OPT_HOST_ZERO_COPY: t.host_zero_copy = val; break;
            case FBP_OPT_BP_EVEN: t.bp_even = val; break;
            default: return fail(nullptr, FBP_EINVAL, "unknown option key");
        }
    }
    return create_impl(out, n_angles, n_det, angles_rad, det_spacing, image_n, pixel_size, dtype, max_batch, device, t);
}

void fbp_destroy(fbp_plan* p)
{
    if (!p) return;
    {
        DeviceGuard guard(p->device);
        cudaFree(p->d_cs2); cudaFree(p->d_ent); cudaFree(p->d_part); cudaFree(p->d_tickets);
        cudaFree(p->d_hsino); cudaFree(p->d_himg); cudaFree(p->d_mscratch); cudaFree(p->d_wrow); cudaFree(p->d_xt); cudaFree(p->d_fdk);
        for (int i = 0; i < 2; ++i) { cudaFree(p->f3[i].d_u); cudaFree(p->f3[i].d_rho); }
        cudaFree(p->fft.d_tab);
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
        // Small pinned sinograms whose rows are one filter unit each are read by the filter straight from host
        // memory (each row once, by cp.async): the rows stream in over PCIe while earlier rows are already being
        // filtered, and one copy operation with its launch gap disappears.  Rows of several units (each unit
        // would fetch the row again over PCIe), large or pageable sinograms are copied first.
        const void* sino_src = p->d_hsino;
        {
            cudaPointerAttributes attr{};
            if (p->host_zero_copy && sino_bytes * batch <= ((size_t)8 << 20) && p->filter_kind == 1 && p->f3[p->window != 0 ? 1 : 0].prm.n_units == 1 &&
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
    unsigned* ticket = reinterpret_cast<unsigned*>(p->d_mscratch + fbp::kMetricSums * kMetricGridMax);   // zero-initialised at fbp_create
    // one wave: as many CTAs as are co-resident (the kernel is register-limited to 4 per SM; a grid of 8 per SM ran
    // as two waves with a ragged tail: 44 us instead of 31 us for the 2 x 67 MB of the config-4 stack)
    if (p->metric_ctas_per_sm == 0) {
        int per_sm = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fbp::metrics_kernel<T>, fbp::kMetricThreads, 0);
        if (e != cudaSuccess) return e;
        p->metric_ctas_per_sm = per_sm < 1 ? 1 : per_sm;
    }
    const int grid_max = std::min(p->metric_ctas_per_sm * p->num_sm, kMetricGridMax);
    // at least 32 elements per thread: small inputs get few CTAs (fewer partials, fewer tickets on one counter)
    long long want = (n + 32LL * fbp::kMetricThreads - 1) / (32LL * fbp::kMetricThreads);
    const int grid = (int)(want < grid_max ? (want < 1 ? 1 : want) : grid_max);
    fbp::metrics_kernel<T><<<grid, fbp::kMetricThreads, 0, st>>>(static_cast<const T*>(x), static_cast<const T*>(y), n, partial,
                                                                 ticket, max_val, c1, c2, d_out);
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
    if ((reinterpret_cast<uintptr_t>(d_x) | reinterpret_cast<uintptr_t>(d_y)) & (p->esize - 1))
        return fail(p, FBP_EINVAL, "d_x and d_y must be aligned to the element size");
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
    // geometry of the staged copies and of the projector's windows (fbp_project.cuh): the widest run is 2 E + 1 pixels,
    // E <= ceil(sqrt(2) d/pix + 1/2) - 1; a CTA's 128 bins span at most 127 sqrt(2) d/pix pixels of a line
    const double inv_max = std::sqrt(2.0) * p->d / p->pix;
    const int e_max = (int)std::ceil(inv_max + 0.5) - 1;
    const int win = round_up((int)std::ceil(127.0 * inv_max) + 2 * e_max + 8, 4);
    const int pad = std::max(round_up(2 * e_max + 2, 4), round_up((win - p->N + 1) / 2 + 1, 4));
    const int pitch = round_up(p->N + 2 * pad, 4);
    // lines per staged block: as many (<= 16) as keep two stages within 48 KB, so that several CTAs share an SM
    int lb = 16;
    while (lb > 1 && 2 * (size_t)lb * 2 * win * p->esize > 48 * 1024) lb /= 2;
    const size_t proj_smem = 32 + 128 + 2 * (size_t)lb * 2 * win * p->esize;
    if (proj_smem > (size_t)kMaxDynSmem) return fail(p, FBP_EUNSUPPORTED, "fbp_project: det_spacing / pixel_size too large for the staged windows");
    const size_t plane = (size_t)p->N * pitch;
    if (!p->d_xt) FBP_CUDA(p, cudaMalloc(&p->d_xt, p->esize * 4 * (size_t)p->max_batch * plane));   // two copies of pairs
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    fbp::ProjParams prm{p->K, p->D, p->N, pad, pitch, win, lb, 0.5 * (p->N - 1), 0.5 * (p->D - 1)};
    const dim3 tgrid((p->N + 31) / 32, (p->N + 31) / 32, batch), tblock(32, 8);
    // a thread owns a bin and its mirror bin; (bin block, angle) pairs are folded into grid.x (K may exceed 65535)
    const int bin_blocks = ((p->D + 1) / 2 + 127) / 128;
    if ((long long)bin_blocks * p->K > 0x7fffffffLL) return fail(p, FBP_EUNSUPPORTED, "n_det x n_angles too large for fbp_project");
    const dim3 pgrid((unsigned)(bin_blocks * p->K), 1, batch);
    const size_t copy = (size_t)p->max_batch * plane;
    if (p->dtype == FBP_F32) {
        float2* xi = static_cast<float2*>(p->d_xt);
        static bool smem_open[kMaxDevices] = {};
        if (cudaError_t e0 = allow_max_smem(fbp::project_kernel<float>, smem_open, p->device); e0 != cudaSuccess) return cuda_fail(p, e0, "projector setup");
        fbp::stage_image_kernel<float><<<tgrid, tblock, 0, s>>>(static_cast<const float*>(d_image), xi, xi + copy, p->N, pad, pitch);
        fbp::project_kernel<float><<<pgrid, 160, proj_smem, s>>>(xi, xi + copy, static_cast<float*>(d_sino), p->d_cs2, prm, bin_blocks);
    } else {
        double2* xi = static_cast<double2*>(p->d_xt);
        static bool smem_open[kMaxDevices] = {};
        if (cudaError_t e0 = allow_max_smem(fbp::project_kernel<double>, smem_open, p->device); e0 != cudaSuccess) return cuda_fail(p, e0, "projector setup");
        fbp::stage_image_kernel<double><<<tgrid, tblock, 0, s>>>(static_cast<const double*>(d_image), xi, xi + copy, p->N, pad, pitch);
        fbp::project_kernel<double><<<pgrid, 160, proj_smem, s>>>(xi, xi + copy, static_cast<double*>(d_sino), p->d_cs2, prm, bin_blocks);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(p, e, "projector launch");
    return FBP_OK;
}

fbp_status fbp_fdk_reconstruct(fbp_plan* p, const void* d_proj, void* d_volume, int n_rows, double row_spacing, double sad,
                               int n_z, double voxel_z, void* stream)
{
    if (!p) return FBP_EINVAL;
    if (!d_proj || !d_volume) return fail(p, FBP_EINVAL, "NULL device pointer");
    if (!aligned16(d_proj) || !aligned16(d_volume)) return fail(p, FBP_EINVAL, "device pointers must be 16-byte aligned");
    if (n_rows < 1 || n_rows > (1 << 16) || n_z < 1 || n_z > (1 << 16)) return fail(p, FBP_EINVAL, "n_rows and n_z must be in [1, 65536]");
    if (!(row_spacing > 0.0) || !std::isfinite(row_spacing) || !(voxel_z > 0.0) || !std::isfinite(voxel_z))
        return fail(p, FBP_EINVAL, "row_spacing and voxel_z must be finite and > 0");
    // every voxel must lie strictly inside the source orbit: U = sad + s > 0 with |s| <= (N-1)/2 sqrt(2) pix
    const double reach = 0.5 * (p->N - 1) * std::sqrt(2.0) * p->pix;
    if (!std::isfinite(sad) || !(sad > reach)) return fail(p, FBP_EINVAL, "sad must be finite and exceed the half-diagonal of the image");
    const long long rows = (long long)p->K * n_rows;
    if (rows > 0x7fffffffLL / 2) return fail(p, FBP_EINVAL, "too many projection rows");
    DeviceGuard guard(p->device);
    const size_t elems = (size_t)rows * p->D;
    // the back-projector's operands: zero-bordered 2 x 2 quads [K][n_rows + 2][D + 2] (fbp_fdk.cuh)
    const size_t pairs_per_angle = (size_t)(n_rows + 2) * (size_t)(p->D + 2);
    if (pairs_per_angle > 0x7fffffffULL) return fail(p, FBP_EINVAL, "detector too large");
    const size_t pairs = pairs_per_angle * p->K;
    // the two elementwise kernels run one thread per element / quad in a one-dimensional grid
    if ((elems + 255) / 256 > 0x7fffffffULL || (pairs + 255) / 256 > 0x7fffffffULL)
        return fail(p, FBP_EINVAL, "projection set too large (more than 2^31 x 256 elements)");
    const size_t need = 2 * elems + 4 + 4 * pairs;   // elements: weighted | filtered | (pad to a quad) | quads
    if (need > p->fdk_elems) {                       // first call (or a taller detector): synchronous, like fbp_project
        FBP_CUDA(p, cudaDeviceSynchronize());
        cudaFree(p->d_fdk);
        p->d_fdk = nullptr; p->fdk_elems = 0;
        FBP_CUDA(p, cudaMalloc(&p->d_fdk, need * p->esize));
        p->fdk_elems = need;
    }
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    void* weighted = p->d_fdk;
    void* filtered = static_cast<char*>(p->d_fdk) + elems * p->esize;
    void* pair_buf = static_cast<char*>(p->d_fdk) + (2 * elems + 3) / 4 * 4 * p->esize;   // aligned to a quad (4 esize)
    const unsigned wgrid = (unsigned)((elems + 255) / 256), pgrid = (unsigned)((pairs + 255) / 256);
    fbp::FdkParams prm{p->K, p->D, n_rows, p->N, n_z, sad / p->d, voxel_z / row_spacing,
                       0.5 * (p->N - 1), 0.5 * (n_z - 1), 0.5 * (p->D - 1), 0.5 * (n_rows - 1), kPi / p->K};
    const int zt = 8;                                // voxels per thread along z (16 measured slower: 6.8 vs 6.2 ms at 64 x 512^2)
    const dim3 bgrid((p->N + 31) / 32, (p->N + 3) / 4, (n_z + zt - 1) / zt), bblock(32, 4);
    cudaError_t e;
    if (p->dtype == FBP_F32) {
        fbp::fdk_weight_kernel<float><<<wgrid, 256, 0, s>>>(static_cast<const float*>(d_proj), static_cast<float*>(weighted),
                                                            (long long)elems, p->D, n_rows, p->d, row_spacing, sad);
        e = launch_filter<float>(p, weighted, filtered, nullptr, 1, s, (int)rows);
        if (e == cudaSuccess) {
            fbp::fdk_quads_kernel<float><<<pgrid, 256, 0, s>>>(static_cast<const float*>(filtered), static_cast<fbp::FdkQuad<float>*>(pair_buf),
                                                               (long long)pairs, p->D, n_rows);
            if (zt == 16)
                fbp::fdk_backproject_kernel<float, 16><<<bgrid, bblock, 0, s>>>(static_cast<const fbp::FdkQuad<float>*>(pair_buf),
                                                                                static_cast<float*>(d_volume), p->d_cs2, prm);
            else
                fbp::fdk_backproject_kernel<float, 8><<<bgrid, bblock, 0, s>>>(static_cast<const fbp::FdkQuad<float>*>(pair_buf),
                                                                               static_cast<float*>(d_volume), p->d_cs2, prm);
        }
    } else {
        fbp::fdk_weight_kernel<double><<<wgrid, 256, 0, s>>>(static_cast<const double*>(d_proj), static_cast<double*>(weighted),
                                                             (long long)elems, p->D, n_rows, p->d, row_spacing, sad);
        e = launch_filter<double>(p, weighted, filtered, nullptr, 1, s, (int)rows);
        if (e == cudaSuccess) {
            fbp::fdk_quads_kernel<double><<<pgrid, 256, 0, s>>>(static_cast<const double*>(filtered), static_cast<fbp::FdkQuad<double>*>(pair_buf),
                                                                (long long)pairs, p->D, n_rows);
            if (zt == 16)
                fbp::fdk_backproject_kernel<double, 16><<<bgrid, bblock, 0, s>>>(static_cast<const fbp::FdkQuad<double>*>(pair_buf),
                                                                                 static_cast<double*>(d_volume), p->d_cs2, prm);
            else
                fbp::fdk_backproject_kernel<double, 8><<<bgrid, bblock, 0, s>>>(static_cast<const fbp::FdkQuad<double>*>(pair_buf),
                                                                                static_cast<double*>(d_volume), p->d_cs2, prm);
        }
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(p, e, "FDK launch");
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
    if (p->filter_kind == 2) {
        // the FFT form treats every window alike: only the kernel's DFT changes
        DeviceGuard guard(p->device);
        FBP_CUDA(p, cudaDeviceSynchronize());      // nothing of this plan may be in flight while its tables change
        cudaError_t e = p->dtype == FBP_F32 ? upload_fft_tables<float>(p, (int)window, false)
                                            : upload_fft_tables<double>(p, (int)window, false);
        if (e != cudaSuccess) return cuda_fail(p, e, "window tables");
        p->window = (int)window;
        return FBP_OK;
    }
    if (window == FBP_WINDOW_RAMLAK) { p->window = 0; return FBP_OK; }
    if (!p->f3[1].ok) return fail(p, FBP_EUNSUPPORTED, "n_det too large for the dense (windowed) row filter");
    DeviceGuard guard(p->device);
    FBP_CUDA(p, cudaDeviceSynchronize());          // nothing of this plan may be in flight while its tables change
    cudaError_t e = p->dtype == FBP_F32 ? upload_filter3_tables<float>(p, true, (int)window)
                                        : upload_filter3_tables<double>(p, true, (int)window);
    if (e != cudaSuccess) return cuda_fail(p, e, "window tables");
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
        const int group = pipe_group_size(p, p->max_batch);
        launches = 2 * ((p->max_batch + group - 1) / group);
    }
    const fbp_plan::F3& f = p->f3[p->window != 0 ? 1 : 0];
    const bool fft = p->filter_kind == 2;
    const int v[19] = {p->bp_tw, p->bp_th, p->bp_r, p->bp_splits, p->bp_chunk, p->bp_seg,
                       p->bp.tiles_x * p->bp.tiles_y * p->bp_splits, p->bp_threads, p->bp_smem,
                       fft ? 16 : 2 * f.r, fft ? p->fft.threads : f.threads, fft ? 0 : f.prm.n_sb, fft ? p->fft.smem : f.smem, launches,
                       fft ? 1 : f.prm.n_units, p->num_sm, (int)filter_ctas(p), p->filter_kind, fft ? 1 << p->fft.p : 0};
    if (out) for (int i = 0; i < n && i < 19; ++i) out[i] = v[i];
    return 19;
}

fbp_status fbp_set_trace(fbp_plan* p, unsigned long long* d_marks, long long capacity)
{
    if (!p) return FBP_EINVAL;
    if (d_marks && (capacity < 8 || (reinterpret_cast<uintptr_t>(d_marks) & 7u))) return fail(p, FBP_EINVAL, "bad trace buffer");
    p->d_trace = d_marks;
    p->trace_cap = d_marks ? capacity : 0;
    return FBP_OK;
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

// ---- fbp_metrics_static: the metrics reduction for callers that may not allocate -----------------------------
// fbp_metrics needs a plan, and making a plan calls cudaMalloc.  Some users of this library never get to do
// that: a process whose device memory was handed, all of it, to a pool or caching allocator at start-up (a
// cudaMalloc from a library underneath it fails or eats into what the pool counts as its own); a control loop
// with a latency bound (cudaMalloc and cudaFree wait for the whole device); a process held to a fixed memory
// budget in which every allocation is accounted for up front.  For them the CTA partial sums and the finish
// ticket of metrics_kernel live in the array below, which is part of the library image: the driver places it
// when the library's device code is loaded on a GPU, and it stays there, on every GPU that loads the library,
// until the process exits.  Size: 1536 CTA records of six doubles + one 256-byte line for the ticket = 73 984
// bytes.
//
// `g_metrics_static_scratch` is a device symbol.  Device code may name it; in HOST code the name is only a
// stand-in handle for the runtime -- not a device address -- so nothing below ever hands `g_metrics_static_scratch`
// itself to a kernel: the address is asked for once per device with cudaGetSymbolAddress, with that device
// current, and the pointer it returns is what the kernel gets.
namespace {
constexpr int kStaticMetricCtas = kMetricGridMax;                              // CTA records the array holds
constexpr int kStaticTicketAt = fbp::kMetricSums * kStaticMetricCtas;          // in doubles: byte 73 728, a multiple of 256
constexpr long long kStaticMetricMaxN = 1LL << 31;                             // FBP_METRICS_STATIC_MAX_N of fbp.h
static_assert(kStaticMetricMaxN == FBP_METRICS_STATIC_MAX_N, "fbp.h and fbp.cu disagree on the limit");
static_assert(kStaticMetricCtas == FBP_METRICS_STATIC_MAX_CTAS, "fbp.h and fbp.cu disagree on the scratch size");
static_assert((kStaticTicketAt * sizeof(double)) % 256 == 0, "the ticket sits on its own 256-byte line");
}  // namespace

static __device__ __align__(256) double g_metrics_static_scratch[kStaticTicketAt + 256 / sizeof(double)];

namespace {

struct StaticMetricsDevice {
    bool ready = false;
    double* scratch = nullptr;     // device address of g_metrics_static_scratch ON THIS DEVICE
    int grid_max[2] = {0, 0};      // one wave of metrics_kernel<float> / <double>, as launch_metrics sizes it
};
StaticMetricsDevice g_static_metrics[kMaxDevices];
std::mutex g_static_metrics_mutex;

// Once per device, with that device current (the caller's: this entry point never switches devices).
fbp_status static_metrics_setup(int device, StaticMetricsDevice& out)
{
    std::lock_guard<std::mutex> lock(g_static_metrics_mutex);
    StaticMetricsDevice& sd = g_static_metrics[device];
    if (!sd.ready) {
        int major = 0, sms = 0;
        cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device);
        if (e != cudaSuccess) return cuda_fail(nullptr, e, "fbp_metrics_static: cudaDeviceGetAttribute");
        if (major != 10)
            return fail(nullptr, FBP_EUNSUPPORTED, "libfbp is built for sm_100a (B200) only; no fallback path");
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
        if (e != cudaSuccess) return cuda_fail(nullptr, e, "fbp_metrics_static: cudaDeviceGetAttribute");
        if (sms < 1) sms = 148;
        int per_sm[2] = {0, 0};
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm[0], fbp::metrics_kernel<float>, fbp::kMetricThreads, 0);
        if (e != cudaSuccess) return cuda_fail(nullptr, e, "fbp_metrics_static: occupancy query");
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm[1], fbp::metrics_kernel<double>, fbp::kMetricThreads, 0);
        if (e != cudaSuccess) return cuda_fail(nullptr, e, "fbp_metrics_static: occupancy query");
        double* ptr = nullptr;
        e = cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_metrics_static_scratch);
        if (e != cudaSuccess) return cuda_fail(nullptr, e, "fbp_metrics_static: cudaGetSymbolAddress");
        if (!ptr) return fail(nullptr, FBP_ECUDA, "fbp_metrics_static: cudaGetSymbolAddress returned no address");
        sd.scratch = ptr;
        for (int t = 0; t < 2; ++t) sd.grid_max[t] = std::min(std::max(per_sm[t], 1) * sms, kStaticMetricCtas);
        sd.ready = true;
    }
    out = sd;
    return FBP_OK;
}

}  // namespace

extern "C" {

fbp_status fbp_metrics_static(fbp_dtype dtype, const void* d_x, const void* d_y, long long n, double max_val,
                              double c1, double c2, double* d_out8, void* stream)
{
    if (dtype != FBP_F32 && dtype != FBP_F64) return fail(nullptr, FBP_EINVAL, "fbp_metrics_static: unknown dtype");
    if (!d_x || !d_y || !d_out8) return fail(nullptr, FBP_EINVAL, "fbp_metrics_static: NULL device pointer");
    if (n < 1) return fail(nullptr, FBP_EINVAL, "fbp_metrics_static: n must be >= 1");
    if (n > kStaticMetricMaxN) {
        char msg[200];
        std::snprintf(msg, sizeof msg, "fbp_metrics_static: n = %lld exceeds FBP_METRICS_STATIC_MAX_N = %lld elements; "
                      "use fbp_metrics on a plan for larger inputs", n, kStaticMetricMaxN);
        return fail(nullptr, FBP_EINVAL, msg);
    }
    if (!(max_val > 0.0) || !std::isfinite(max_val))
        return fail(nullptr, FBP_EINVAL, "fbp_metrics_static: max_val must be finite and > 0");
    if ((reinterpret_cast<uintptr_t>(d_out8) & 7u) != 0)
        return fail(nullptr, FBP_EINVAL, "fbp_metrics_static: d_out8 must be 8-byte aligned");
    const size_t esize = dtype == FBP_F32 ? 4 : 8;
    if ((reinterpret_cast<uintptr_t>(d_x) | reinterpret_cast<uintptr_t>(d_y)) & (esize - 1))
        return fail(nullptr, FBP_EINVAL, "fbp_metrics_static: d_x and d_y must be aligned to the element size");
    if (c1 < 0.0) c1 = (0.01 * max_val) * (0.01 * max_val);
    if (c2 < 0.0) c2 = (0.03 * max_val) * (0.03 * max_val);

    int device = -1;
    cudaError_t e = cudaGetDevice(&device);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "fbp_metrics_static: cudaGetDevice");
    if (device < 0 || device >= kMaxDevices)
        return fail(nullptr, FBP_EUNSUPPORTED, "fbp_metrics_static: device ordinal beyond the 64 this entry point keeps state for");
    StaticMetricsDevice sd;
    fbp_status st = static_metrics_setup(device, sd);
    if (st != FBP_OK) return st;

    // the same grid rule as launch_metrics, so the sums are added in the same order as on a plan
    const int t = dtype == FBP_F32 ? 0 : 1;
    const long long want = (n + 32LL * fbp::kMetricThreads - 1) / (32LL * fbp::kMetricThreads);
    const int grid = (int)(want < sd.grid_max[t] ? want : sd.grid_max[t]);
    double* partial = sd.scratch;
    unsigned* ticket = reinterpret_cast<unsigned*>(sd.scratch + kStaticTicketAt);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    // The array is shared by every call and keeps what the last one left.  Partials: each CTA of this launch
    // overwrites its own record before anyone reads it, records of a larger earlier grid are never read.  The
    // ticket must be 0 when the kernel starts; the kernel re-arms it as it finishes, but a launch that died
    // half-way would leave it counting, so it is cleared here, on the caller's stream, every time.
    e = cudaMemsetAsync(ticket, 0, sizeof(unsigned), s);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "fbp_metrics_static: clearing the ticket");
    if (dtype == FBP_F32)
        fbp::metrics_kernel<float><<<grid, fbp::kMetricThreads, 0, s>>>(static_cast<const float*>(d_x), static_cast<const float*>(d_y),
                                                                        n, partial, ticket, max_val, c1, c2, d_out8);
    else
        fbp::metrics_kernel<double><<<grid, fbp::kMetricThreads, 0, s>>>(static_cast<const double*>(d_x), static_cast<const double*>(d_y),
                                                                         n, partial, ticket, max_val, c1, c2, d_out8);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "fbp_metrics_static: launch");
    return FBP_OK;
}

}  // extern "C"

// ---- fbp_measure_issue_rate: the denominator of the back-projector's roofline, measured ----------------------
// Eight independent FMA chains per thread, 64 FMAs per loop trip, two CTAs of 1024 threads on every SM: nothing but
// the FP32 (FFMA) or FP64 (DFMA) pipe limits it, so lane-instructions per second of this kernel is the issue peak
// that bench.py's "alu" roofline is stated against ("builder measures with an FMA micro-benchmark").
namespace fbp {
template <typename T>
__global__ void __launch_bounds__(1024) fma_rate_kernel(T* out, int iters, T a, T b)
{
    T x[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) x[q] = a + T(threadIdx.x + q);
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
#pragma unroll
            for (int q = 0; q < 8; ++q) x[q] = fma(x[q], a, b);
    }
    T s = T(0);
#pragma unroll
    for (int q = 0; q < 8; ++q) s += x[q];
    if (s == T(-1)) out[0] = s;          // never true (a, b > 0): keeps the chains alive without a store per thread
}
}  // namespace fbp

extern "C" fbp_status fbp_measure_issue_rate(fbp_dtype dtype, double* h_lane_instr_per_s)
{
    if (!h_lane_instr_per_s || (dtype != FBP_F32 && dtype != FBP_F64)) return fail(nullptr, FBP_EINVAL, "fbp_measure_issue_rate: bad arguments");
    *h_lane_instr_per_s = 0.0;
    int device = 0, sms = 0, major = 0;
    cudaError_t e = cudaGetDevice(&device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "fbp_measure_issue_rate: device query");
    if (major != 10) return fail(nullptr, FBP_EUNSUPPORTED, "libfbp is built for sm_100a (B200) only; no fallback path");
    void* d_out = nullptr;
    cudaEvent_t ev[2] = {nullptr, nullptr};
    e = cudaMalloc(&d_out, 16);
    if (e == cudaSuccess) e = cudaEventCreate(&ev[0]);
    if (e == cudaSuccess) e = cudaEventCreate(&ev[1]);
    const int grid = 2 * sms, iters = dtype == FBP_F32 ? 8192 : 4096;
    float best_ms = 0.f;
    for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {          // rep 0 warms up (clocks, code)
        e = cudaEventRecord(ev[0], nullptr);
        if (e != cudaSuccess) break;
        if (dtype == FBP_F32) fbp::fma_rate_kernel<float><<<grid, 1024>>>(static_cast<float*>(d_out), iters, 1.0000001f, 1e-7f);
        else fbp::fma_rate_kernel<double><<<grid, 1024>>>(static_cast<double*>(d_out), iters, 1.0000001, 1e-7);
        e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaEventRecord(ev[1], nullptr);
        if (e == cudaSuccess) e = cudaEventSynchronize(ev[1]);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, ev[0], ev[1]);
        if (e == cudaSuccess && rep > 0 && (best_ms == 0.f || ms < best_ms)) best_ms = ms;
    }
    if (ev[0]) cudaEventDestroy(ev[0]);
    if (ev[1]) cudaEventDestroy(ev[1]);
    cudaFree(d_out);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "fbp_measure_issue_rate");
    if (!(best_ms > 0.f)) return fail(nullptr, FBP_ECUDA, "fbp_measure_issue_rate: no time measured");
    *h_lane_instr_per_s = (double)grid * 1024.0 * (double)iters * 64.0 / ((double)best_ms * 1e-3);
    return FBP_OK;
}
