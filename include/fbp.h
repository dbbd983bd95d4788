/*
 * fbp.h -- C ABI of libfbp: 2-D parallel-beam filtered back-projection on one B200 (sm_100a).
 *
 * The operation is the one the paper states (arxiv 2109.02174, "PAPER.md"):
 *   PAPER.md:55   a ray is  x cos(theta) + y sin(theta) = t;  the projections P_theta(t)
 *                 indexed by (angle, detector offset) form the sinogram.
 *   PAPER.md:61   Q_theta(t) = P_theta(t) * H(t)               -- the filter step
 *   PAPER.md:59   f(x,y) = sum_i Q_theta_i( x cos theta_i + y sin theta_i )   (eq. 2)
 * The paper leaves the filter, the interpolation and the scale factors open; the readings
 * taken are:
 *   taps   h[0] = 1/4,  h[m] = -1/(pi^2 m^2) for odd m,  0 for even m != 0      (Ram-Lak)
 *   filter Q[i][n] = (1/d) * sum_{k=0}^{D-1} h[n-k] P[i][k]      (linear, "same", zero-extended)
 *   pixel  x = (c - (N-1)/2) * pix,  y = (r - (N-1)/2) * pix     (column <-> +x, row <-> +y)
 *   coord  u = (x cos theta_i + y sin theta_i)/d + (D-1)/2 ;  j = floor(u) ;  w = u - j
 *   interp q_i = (1-w) Q~[i][j] + w Q~[i][j+1],   Q~ = 0 outside [0, D-1]
 *   image  f[r][c] = (pi/K) * sum_{i=0}^{K-1} q_i                (every angle weighted pi/K)
 *
 * Conventions common to every entry point
 *   - Arrays are dense, row-major, element type = the plan's dtype (float or double):
 *       sinogram / filtered sinogram  [batch][n_angles][n_det]
 *       image                         [batch][image_n][image_n]
 *   - "d_" arguments are DEVICE pointers (16-byte aligned), "h_" arguments are HOST pointers.
 *     The caller owns them; inputs are never written; outputs are fully overwritten.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *     Device-pointer calls only enqueue work on that stream: no host synchronisation, no
 *     allocation.  A plan must not be used from two streams at once (it owns scratch
 *     buffers); different plans are independent.
 *   - Determinism: every output element has one owner thread and a fixed summation order
 *     (no atomics, no read-modify-write between threads -- the defect PAPER.md:218 reports
 *     for its parallel versions).  Same plan parameters + same input bytes => same output
 *     bytes on every run.
 *   - Errors: a non-zero fbp_status is returned, nothing is enqueued and no output is
 *     touched.  FBP_EINVAL: NULL / misaligned pointers, sizes out of range, non-finite
 *     geometry, batch < 1 or > max_batch.  FBP_ENOMEM: allocation failure.
 *     FBP_EUNSUPPORTED: the device is not compute capability 10.x (there is no fallback
 *     path by design).  FBP_ECUDA: any CUDA runtime error (text via fbp_last_error).
 *     Nothing throws across this boundary and nothing calls exit/abort.
 */
#ifndef FBP_H_
#define FBP_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fbp_plan fbp_plan; /* opaque; owned by the library */

typedef enum { FBP_F32 = 0, FBP_F64 = 1 } fbp_dtype;

typedef enum {
    FBP_OK = 0,
    FBP_EINVAL = 1,
    FBP_ENOMEM = 2,
    FBP_ECUDA = 3,
    FBP_EUNSUPPORTED = 4
} fbp_status;

/*
 * fbp_create -- build a plan for one geometry (rays x cos + y sin = t).
 *   out          receives the plan (HOST pointer to a pointer); NULL on failure
 *   n_angles     K >= 1;  n_det  D >= 2
 *   angles_rad   HOST pointer, K finite values theta_i in radians; copied
 *   det_spacing  d > 0; the detector is centred: t_j = (j - (D-1)/2) * d
 *   image_n      N >= 1;  pixel_size > 0, or <= 0 meaning "= det_spacing"
 *   dtype        arithmetic and storage type of every array passed to this plan
 *   max_batch    >= 1; sizes the plan-owned filtered-sinogram scratch used by fbp_reconstruct
 *   device       CUDA ordinal, or -1 for the current device
 * Host work happens here only: the Ram-Lak taps and the cos/sin table are computed in fp64
 * on the host and uploaded; scratch buffers are allocated.  Synchronous.
 */
fbp_status fbp_create(fbp_plan **out, int n_angles, int n_det, const double *angles_rad,
                      double det_spacing, int image_n, double pixel_size, fbp_dtype dtype,
                      int max_batch, int device);

/*
 * fbp_create_tuned -- fbp_create with explicit launch-configuration overrides, for tests, A/B measurements and
 * bench.py.  h_options: HOST array of n_options (key, value) int pairs; keys not listed keep the library's
 * choice; an unknown key is FBP_EINVAL.  The library never reads the environment: a plan's behaviour depends
 * on these arguments only.  Options change launch shapes and summation grouping (hence possibly the last
 * bits of a result), never the definition of what is computed; each plan stays bit-reproducible.
 *   FBP_OPT_BP_VARIANT      index of the back-projection tile variant (R rows/thread, warps in y, angle groups)
 *   FBP_OPT_BP_SPLITS       angle splits S per tile (>= 1)        FBP_OPT_BP_CHUNK   angles staged per chunk (<= 32)
 *   FBP_OPT_FILTER_R        output pairs per thread of the direct-form filter (6, 10, 14; dense 5, 7, 9; fp64 plans: 6 or 5
 *                           only); any other value, or one the plan's dtype does not have, is FBP_EINVAL
 *   FBP_OPT_FILTER_SB       warps (input slices) per filter CTA (1..8)
 *   FBP_OPT_FILTER_KIND     0 = library's choice, 1 = direct form, 2 = FFT form
 *   FBP_OPT_PIPELINE        0 = no batch pipeline; FBP_OPT_PIPE_GROUP slices per pipeline group;
 *   FBP_OPT_PIPE_MIN_BATCH  smallest batch that takes the pipeline (default 8)
 *   FBP_OPT_PDL             0 = no programmatic dependent launch between filter and back-projector
 *   FBP_OPT_HOST_ZERO_COPY  0 = fbp_reconstruct_host always stages through device buffers
 *   FBP_OPT_BP_EVEN         0 = do not size shared memory for even CTA placement of small launches
 */
typedef enum {
    FBP_OPT_BP_VARIANT = 1,
    FBP_OPT_BP_SPLITS = 2,
    FBP_OPT_BP_CHUNK = 3,
    FBP_OPT_FILTER_R = 4,
    FBP_OPT_FILTER_SB = 5,
    FBP_OPT_FILTER_KIND = 6,
    FBP_OPT_PIPELINE = 7,
    FBP_OPT_PIPE_GROUP = 8,
    FBP_OPT_PIPE_MIN_BATCH = 9,
    FBP_OPT_PDL = 10,
    FBP_OPT_HOST_ZERO_COPY = 11,
    FBP_OPT_BP_EVEN = 13
} fbp_option;
fbp_status fbp_create_tuned(fbp_plan **out, int n_angles, int n_det, const double *angles_rad,
                            double det_spacing, int image_n, double pixel_size, fbp_dtype dtype,
                            int max_batch, int device, const int *h_options, int n_options);

/*
 * fbp_filter -- Q = (1/d) h * P along the detector axis of every row.
 *   d_sino [batch][K][D] in, d_filtered [batch][K][D] out (may not alias).
 */
fbp_status fbp_filter(fbp_plan *plan, const void *d_sino, void *d_filtered, int batch,
                      void *cuda_stream);

/*
 * fbp_backproject -- f = (pi/K) sum_i lerp(Q_i, u_i(x,y)) for every pixel (eq. 2).
 *   d_filtered [batch][K][D] in, d_image [batch][N][N] out.  Includes the pi/K weight.
 */
fbp_status fbp_backproject(fbp_plan *plan, const void *d_filtered, void *d_image, int batch,
                           void *cuda_stream);

/*
 * fbp_reconstruct -- fbp_backproject(fbp_filter(sino)) through the plan-owned scratch;
 * bit-identical to calling the two entry points in sequence.
 */
fbp_status fbp_reconstruct(fbp_plan *plan, const void *d_sino, void *d_image, int batch,
                           void *cuda_stream);

/*
 * fbp_reconstruct_host -- the same reconstruction for HOST buffers: h_sino [batch][K][D] in, h_image
 * [batch][N][N] out, then waits for the stream.  This is the end-to-end path bench.py's "e2e" leg times
 * (transfers inside the timed region).  The sinogram is copied to a plan-owned device buffer (for stacks
 * of >= 8 slices group by group, overlapping the previous group's back-projection).  If h_image is pinned
 * (page-locked, device-accessible) memory the back-projector stores its pixels straight into it over PCIe,
 * overlapped with the kernel; pageable memory takes a device image and a copy.  Same bytes either way.
 */
fbp_status fbp_reconstruct_host(fbp_plan *plan, const void *h_sino, void *h_image, int batch,
                                void *cuda_stream);

/*
 * fbp_metrics -- the paper's image-similarity measures of one image pair:
 *   PSNR = 20 log10(MAX / sqrt(MSE))                                        (eq. 3)
 *   SSIM = (2 mu_x mu_y + C1)(2 s_xy + C2) / ((mu_x^2 + mu_y^2 + C1)(s_x^2 + s_y^2 + C2))
 *                                                                            (eq. 4)
 * with statistics over all n elements (the paper names no window): mu = mean, s^2 and s_xy =
 * population variance and covariance.  d_x, d_y: DEVICE arrays of n elements of the plan's dtype
 * (any shape, e.g. one image or a whole stack).  max_val = MAX > 0.  c1, c2 < 0 select the customary
 * (0.01 MAX)^2 and (0.03 MAX)^2 (the paper does not state its constants).  d_out8: DEVICE array of
 * 8 doubles, written on the stream: MSE, PSNR (+inf when MSE = 0), SSIM, mu_x, mu_y,
 * s_x^2, s_y^2, s_xy.  One pass over the two arrays (shifted fp64 moments), sums in a fixed order: repeated calls give
 * the same bits.  Enqueue-only;
 * uses plan-owned scratch, so not concurrently with other calls on the same plan.
 */
fbp_status fbp_metrics(fbp_plan *plan, const void *d_x, const void *d_y, long long n, double max_val,
                       double c1, double c2, double *d_out8, void *cuda_stream);

/*
 * fbp_metrics_static -- fbp_metrics for callers that must not allocate device memory: no plan, no cudaMalloc,
 * no cudaFree, no allocating library routine, on any call.  Same definition (eq. 3 and 4), same
 * kernel, same grid rule and summation order as fbp_metrics, hence the same eight outputs for the same inputs.
 *
 * Who needs it.  Every other compute entry point takes a plan, and fbp_create allocates.  That rules the
 * library out for a caller that gave ALL device memory to its own pool or caching allocator at start-up (a
 * cudaMalloc from underneath such a pool fails, or takes memory the pool believes it owns), for a loop with a
 * latency bound (cudaMalloc / cudaFree wait for the whole device to go idle), and for a process that must account
 * for every device byte before it starts.  Those callers compare two reconstructions with this call instead: they
 * pass the two arrays and the result buffer, and the kernel's work area (one 48-byte partial-sum record per CTA and
 * the finish ticket) is a fixed array inside the library image instead of plan-owned memory.
 *
 * The price, and the limits:
 *   - The work area is FBP_METRICS_STATIC_MAX_CTAS (1536) records + one 256-byte line = 73 984 bytes of device
 *     memory, held by EVERY GPU on which the library's device code gets loaded, from that moment until the
 *     process exits, whether or not this call is ever made there.
 *   - n <= FBP_METRICS_STATIC_MAX_N (2^31 elements per array).  A larger n is refused with FBP_EINVAL and a message
 *     naming the limit (fbp_last_error(NULL)); nothing is enqueued.  fbp_metrics on a plan has no such limit.
 *   - It runs on the CURRENT device (the one d_x, d_y and d_out8 belong to) and never switches devices.
 *   - First call on each device: the library looks up where the work area sits on that device and how many CTAs
 *     fit one wave (two occupancy queries), under a mutex, and keeps the answers.  That first call may also be what
 *     makes the CUDA runtime load the library's device code.  Make it once per device during start-up, BEFORE any
 *     stream capture begins on that device; later calls only enqueue a 4-byte memset and one kernel.
 *   - All calls on a device share the one work area, and it keeps the previous call's contents (the call clears the
 *     one word that has to start at zero).  Two calls may therefore not overlap on the GPU: issue them on one
 *     stream, or order them with events.  Calls on different streams with nothing between them race on the
 *     records and the ticket and return garbage without any error.  Plans are not affected (they own their scratch).
 * Arguments as fbp_metrics, with `dtype` in place of the plan: d_x, d_y DEVICE arrays of n elements of `dtype`
 * (aligned to the element size; 16-byte alignment takes the vector path), d_out8 DEVICE array of 8 doubles written
 * on the stream.  Errors: FBP_EINVAL (arguments, n beyond the limit), FBP_EUNSUPPORTED (not a compute-capability-10
 * device, or a device ordinal >= 64), FBP_ECUDA; text through fbp_last_error(NULL) on the calling thread.
 */
#define FBP_METRICS_STATIC_MAX_N (1LL << 31)
#define FBP_METRICS_STATIC_MAX_CTAS 1536
fbp_status fbp_metrics_static(fbp_dtype dtype, const void *d_x, const void *d_y, long long n, double max_val,
                              double c1, double c2, double *d_out8, void *cuda_stream);

/*
 * fbp_set_window -- choose the reconstruction filter H of PAPER.md:61 ("Q = P * H"; the paper names
 * no particular H).  The taps are the inverse DTFT of |f| W(f) on |f| <= 1/2 cycles per sample,
 *   h_W[m] = 2 * integral_0^{1/2} f W(f) cos(2 pi f m) df   (closed forms, computed in fp64 on the host):
 *   FBP_WINDOW_RAMLAK       W = 1  (default; the only window with zero even taps)
 *   FBP_WINDOW_SHEPP_LOGAN  W = sin(pi f)/(pi f)      h[m] = -2 / (pi^2 (4 m^2 - 1))
 *   FBP_WINDOW_COSINE       W = cos(pi f)
 *   FBP_WINDOW_HAMMING      W = 0.54 + 0.46 cos(2 pi f)
 *   FBP_WINDOW_HANN         W = 0.5 + 0.5 cos(2 pi f)
 * Applies to fbp_filter and fbp_reconstruct from the next call on.  Synchronous: waits for the device,
 * rebuilds and uploads the tap tables (FFT form: the DFT of the taps' running sum).  FBP_EUNSUPPORTED if the
 * plan runs the direct form and the row is too long for its dense kernel.
 */
typedef enum {
    FBP_WINDOW_RAMLAK = 0,
    FBP_WINDOW_SHEPP_LOGAN = 1,
    FBP_WINDOW_COSINE = 2,
    FBP_WINDOW_HAMMING = 3,
    FBP_WINDOW_HANN = 4
} fbp_window;
fbp_status fbp_set_window(fbp_plan *plan, fbp_window window);

/*
 * fbp_set_angle_weights -- per-angle weights for non-uniform angle sets: f = sum_i w_i q_i instead of
 * (pi/K) sum_i q_i (eq. 2, which carries no weight at all).
 * h_weights: HOST pointer to K finite values, copied; NULL restores pi/K for every angle.  Applies to
 * fbp_backproject and fbp_reconstruct from the next call on.  Synchronous.
 */
fbp_status fbp_set_angle_weights(fbp_plan *plan, const double *h_weights);

/*
 * fbp_project -- the matched forward projector R = B^T of fbp_backproject WITHOUT its pi/K weight
 * (rays x cos + y sin = t):
 *   y[i][j] = sum over pixels (r,c) of max(0, 1 - |u_i(r,c) - j|) * x[r][c],  u_i as in fbp.h's header,
 * so that <R x, y> = <x, B y> for the unweighted B.  d_image [batch][N][N] in, d_sino [batch][K][D] out
 * (fully overwritten; may not alias).  A gather with one owner thread per bin and a fixed pixel order:
 * deterministic, no atomics.  The first call allocates a plan-owned transposed-image scratch
 * (synchronous); later calls only enqueue.  Angle weights and windows do not apply.
 */
fbp_status fbp_project(fbp_plan *plan, const void *d_image, void *d_sino, int batch, void *cuda_stream);

/*
 * fbp_fdk_reconstruct -- cone-beam reconstruction by the algorithm of Feldkamp, Davis and Kress, the continuation the
 * paper announces (ref [20]: it "uses the filtered backprojection algorithm in the reconstruction of
 * three-dimensional images obtained by projections of a cone beam").  The paper gives no
 * formula; this is the textbook algorithm (Kak & Slaney ch. 3.6, ref [8]) in the plan's 2-D conventions.  Readings
 * (DESIGN.md "FDK"): circular source orbit of radius `sad` about the z axis in the plane z = 0, source at
 * -sad * e_s(beta), e_s = (-sin beta, cos beta, 0); flat VIRTUAL detector through the axis spanned by
 * e_a = (cos beta, sin beta, 0) (columns: the plan's n_det bins of det_spacing, centred) and e_z (n_rows rows of
 * row_spacing, centred); angles = the plan's (meant to cover [0, 2 pi) uniformly); x, y grid = the plan's image grid,
 * z_k = (k - (n_z-1)/2) voxel_z.
 *   1. p'[m][i][j] = p[m][i][j] * sad / sqrt(sad^2 + a_j^2 + b_i^2)
 *   2. Q[m][i][:]  = the plan's row filter applied to every detector row (fbp_filter's operation; fbp_set_window applies)
 *   3. f[k][r][c]  = (pi/K) sum_m (sad/U)^2 bilinear(Q[m]; sad t/(U d_a) + (n_det-1)/2, sad z_k/(U d_b) + (n_rows-1)/2),
 *                    t = x cos + y sin,  U = sad - x sin + y cos,  zero outside the detector.
 * d_proj [K][n_rows][n_det] in, d_volume [n_z][N][N] out (DEVICE, plan dtype, 16-byte aligned).  sad must exceed the
 * image's half-diagonal (FBP_EINVAL otherwise).  The first call (and any call with more rows than before) allocates
 * plan-owned scratch (synchronous); later calls only enqueue.  That scratch is about SIX times the projection set --
 * the weighted copy, the filtered copy and the zero-bordered 2 x 2 quads, 4 (n_rows + 2)(n_det + 2) K elements -- and
 * is kept until fbp_destroy.  A projection set of more than 2^31 x 256 elements is FBP_EINVAL.  One owner thread per
 * voxel, fixed order: deterministic.  Angle weights do not apply.
 */
fbp_status fbp_fdk_reconstruct(fbp_plan *plan, const void *d_proj, void *d_volume, int n_rows, double row_spacing,
                               double sad, int n_z, double voxel_z, void *cuda_stream);

/*
 * fbp_interpolate_stack -- a volume from a stack of reconstructed slices (3-D images
 * "through the interpolation of a stack of 2D images"; the paper names no rule, LINEAR is the reading
 * taken, R4).  d_stack [n_in][N][N] in, d_out [n_out][N][N] out (DEVICE, plan dtype, may not
 * alias).  Output slice m sits at z_m = m (n_in - 1)/(n_out - 1) (z = 0 when n_out = 1):
 *   k = floor(z_m) clamped to n_in - 2,  t = z_m - k,  out[m] = (1 - t) stack[k] + t stack[k+1];
 * n_in = 1 copies the slice.  Enqueue-only, one owner thread per output element.
 */
fbp_status fbp_interpolate_stack(fbp_plan *plan, const void *d_stack, int n_in, void *d_out, int n_out,
                                 void *cuda_stream);

/* fbp_destroy -- free the plan, its tables and scratch.  NULL-safe.  Synchronous. */
void fbp_destroy(fbp_plan *plan);

/*
 * fbp_last_error -- text of the last error on this plan (plan-owned, never freed by the
 * caller; "" if none).  NULL plan: the last error, on the calling thread, of the calls that take no plan
 * (fbp_create, fbp_create_tuned, fbp_metrics_static).
 */
const char *fbp_last_error(const fbp_plan *plan);

/*
 * fbp_plan_info -- launch configuration chosen by fbp_create, for tests, bench.py and
 * DESIGN.md tables.  Writes up to `n` ints into `out` (HOST) and returns how many it has:
 *   [0] back-projection tile width   [1] tile height   [2] pixels per thread (register tile)
 *   [3] angle splits S (deterministic fixed-order reduction when > 1)
 *   [4] angles staged per shared-memory chunk   [5] staged segment length (entries per angle)
 *   [6] back-projection CTAs per slice   [7] back-projection threads per CTA
 *   [8] back-projection dynamic shared memory bytes per CTA
 *   [9] filter outputs per thread (direct form) / points per thread and pass (FFT form)   [10] filter threads per CTA
 *   [11] filter input slices per row (SB; 0 for the FFT form)
 *   [12] filter dynamic shared memory bytes per CTA   [13] kernels launched by fbp_reconstruct at batch = max_batch
 *   [14] filter units per row (a row is cut into independent units of one warp-width of outputs; 1 for the FFT form)
 *   [15] SMs of the plan's device
 *   [16] filter CTAs per launch at batch = max_batch (0 until the filter has run once: it comes from the occupancy query)
 *   [17] filter kind (1 direct, 2 FFT)   [18] transform length N of the FFT form (0 for the direct form)
 */
int fbp_plan_info(const fbp_plan *plan, int *out, int n);

/*
 * fbp_set_trace -- optional in-kernel timeline (profiles/: where the microseconds of a step go).  d_marks: DEVICE
 * array of `capacity` 64-bit words (caller-owned, zero it first), or NULL to switch tracing off.  While set, thread 0
 * of every CTA of the filter and of the back-projector stores %globaltimer (ns) into its 8-word record:
 *   filter CTA c          -> d_marks[8 c + s],  direct form: s = 0 start, 1 tables and first row staged, 2 partial sums
 *                            done, 3 row reduced, 4 last unit stored (1-3: the CTA's first unit only);
 *                            FFT form: s = 0 start, 1 row pair read and first pass done, 2 spectrum ready (forward passes
 *                            done, before the product with the kernel's DFT), 3 rows back in shared memory (inverse
 *                            passes done), 4 last row pair stored (1-3: the CTA's first row pair only)
 *   back-projector CTA c  -> d_marks[8 (F + c) + s],  F = plan_info[16],  s = 0 CTA resident, 1 past the grid
 *                            dependency, 2 first chunk landed, 3 main loop done, 4 pixels stored,
 *                            7 the SM the CTA ran on (%smid, not a time)
 * A kernel whose records would not fit in `capacity` is not traced.  The filters carry the marks as predicated
 * stores; the back-projector runs a second instantiation of the same source with the marks compiled in (under its
 * register cap even predicated-off marks cost the main loop).  Traced launches are those of fbp_filter,
 * fbp_backproject, fbp_reconstruct and fbp_reconstruct_host when they run one filter launch and one back-projector
 * launch; the batch pipeline's per-group launches (which would overwrite each other's records) and the launches of
 * fbp_fdk_reconstruct (whose filter grid is sized for K x n_rows rows) never write marks.
 */
fbp_status fbp_set_trace(fbp_plan *plan, unsigned long long *d_marks, long long capacity);

/*
 * fbp_set_profiling / fbp_get_kernel_ms -- optional per-kernel timing of the LAST compute
 * call, with CUDA events recorded on the caller's stream around each kernel group.
 * fbp_get_kernel_ms waits for those events (host sync) and returns milliseconds; a group
 * that did not run in the last call reports 0.  Off by default (no events recorded).
 */
fbp_status fbp_set_profiling(fbp_plan *plan, int enable);
fbp_status fbp_get_kernel_ms(fbp_plan *plan, float *filter_ms, float *backproject_ms);

/*
 * fbp_measure_issue_rate -- the FP32 (FFMA) or FP64 (DFMA) issue peak of the current device, measured: a kernel of
 * independent FMA chains at full occupancy (two CTAs of 1024 threads per SM, 64 FMAs per loop trip), best of three
 * timed launches after a warm-up, in lane-instructions per second (one FMA on one lane = 1).  This is the
 * denominator bench.py states the back-projector's "alu" roofline against next to the figure derived from SM count,
 * lanes and clock.  A measurement aid, not part of the reconstruction path:
 * synchronous, runs on the legacy default stream, allocates and frees 16 bytes.  h_lane_instr_per_s: HOST pointer.
 */
fbp_status fbp_measure_issue_rate(fbp_dtype dtype, double *h_lane_instr_per_s);

#ifdef __cplusplus
}
#endif
#endif /* FBP_H_ */
