/*
 * fbp_oracle.c -- the ORACLE: a plain, slow, obviously-correct CPU implementation of
 * 2-D parallel-beam filtered back-projection, written from the paper, in fp64.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It
 * shares no code, header, table or constant with the CUDA library in
 * paper_2109_02174_b200/csrc/, and neither includes the other.
 *
 * What it computes (arxiv 2109.02174, "PAPER.md"):
 *   eq. 2, PAPER.md:59      f(x,y) = sum_i Q_theta_i( x cos(theta_i) + y sin(theta_i) )
 *   PAPER.md:61             Q_theta(t) = P_theta(t) * H(t)       (filter convolution)
 *   PAPER.md:55             a ray is  x cos(theta) + y sin(theta) = t
 * The paper leaves the filter, the interpolation rule, the scale factors and the axis
 * conventions open; the readings taken are those of SURVEY.md section 8(c) (G1-G12) and
 * are listed in DESIGN.md section "Readings":
 *   O1  Ram-Lak taps  h[0] = 1/4,  h[m] = -1/(pi^2 m^2) for odd m,  0 for even m != 0
 *       (inverse DTFT of |f| band-limited to 1/2 cycle per sample; Kak & Slaney ch. 3,
 *       ref [8] PAPER.md:247; BASELINE.json north_star item 2).
 *   O2  Q[i][n] = (1/d) * sum_{k=0}^{D-1} h[n-k] * P[i][k],  n = 0..D-1: linear ("same")
 *       convolution, zero extension, full 2D-1 tap support, no window, no FFT (G2-G4).
 *   O3  per pixel (r,c): x = (c-(N-1)/2)*pix, y = (r-(N-1)/2)*pix; per angle i:
 *       t = x cos + y sin;  u = t/d + (D-1)/2;  j = floor(u);  w = u - j;
 *       q_i = (1-w) Qz[i][j] + w Qz[i][j+1],  Qz = 0 outside [0, D-1];
 *       f[r][c] = (pi/K) * sum_i q_i                                   (G1, G5-G8, G10).
 *   O4  the adjoint pair used only for self-checking: B = O3 without the pi/K weight,
 *       and R = B^T written independently as a SCATTER.
 *
 * Arithmetic: IEEE fp64 for every product; every long sum is carried in long double
 * (x87 80-bit on this platform) so that the oracle's own rounding is far below the
 * 1e-12 bar the fp64 CUDA path is held to.  No blocking, no fusion, no reordering.
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): P1-P12 of SURVEY.md 8(c):
 * tap closed forms, numpy.convolve / Toeplitz, continuous ramp-filtered disk, impulse
 * -> pi/(4d), partition of unity -> pi, numpy.interp at theta = 0 and pi/2, dense-matrix
 * brute force on 8x8, adjoint identity, linearity, uniform-disk reconstruction, ellipse
 * region means, symmetries.  Nothing here is "parity unpinned".
 *
 * Layouts (all dense row-major, fp64): P, Q: [batch][K][D];  f: [batch][N][N] with
 * row <-> +y and column <-> +x.  `threads` <= 0 means "all cores OpenMP reports".
 */
#include <math.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static const double ORACLE_PI = 3.14159265358979323846264338327950288;

int fbp_oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static int pick_threads(int threads)
{
    int m = fbp_oracle_max_threads();
    if (threads <= 0 || threads > m) return m;
    return threads;
}

/* O1: one Ram-Lak tap. */
static double ramlak_tap(long m)
{
    if (m == 0) return 0.25;
    if (m % 2 == 0) return 0.0;
    return -1.0 / (ORACLE_PI * ORACLE_PI * (double)m * (double)m);
}

/* O1: h_out[m + (D-1)] = h[m], m = -(D-1) .. D-1   (2D-1 values). */
void fbp_oracle_taps(int n_det, double *h_out)
{
    for (long m = -(long)(n_det - 1); m <= (long)(n_det - 1); ++m)
        h_out[m + (n_det - 1)] = ramlak_tap(m);
}

/* O2: direct O(D^2) filter of every row. */
void fbp_oracle_filter(const double *P, double *Q, int batch, int n_angles, int n_det,
                       double det_spacing, int threads)
{
    long rows = (long)batch * n_angles;
    int nt = pick_threads(threads);
    (void)nt;
#pragma omp parallel for schedule(static) num_threads(nt)
    for (long row = 0; row < rows; ++row) {
        const double *p = P + row * n_det;
        double *q = Q + row * n_det;
        for (int n = 0; n < n_det; ++n) {
            long double acc = 0.0L;
            for (int k = 0; k < n_det; ++k)
                acc += (long double)(ramlak_tap((long)n - (long)k) * p[k]);
            q[n] = (double)(acc / (long double)det_spacing);
        }
    }
}

/* Qz: Q extended by zero outside the detector (G5). */
static double q_at(const double *qrow, int n_det, long j)
{
    if (j < 0 || j >= n_det) return 0.0;
    return qrow[j];
}

/* O3 for one pixel of one slice; `scaled` != 0 applies the pi/K weight (G1). */
static double backproject_pixel(const double *Q, int n_angles, int n_det, const double *angles,
                                double det_spacing, int image_n, double pixel_size,
                                int r, int c, int scaled)
{
    double c_n = 0.5 * (double)(image_n - 1);
    double c_d = 0.5 * (double)(n_det - 1);
    double x = ((double)c - c_n) * pixel_size;
    double y = ((double)r - c_n) * pixel_size;
    long double acc = 0.0L;
    for (int i = 0; i < n_angles; ++i) {
        double t = x * cos(angles[i]) + y * sin(angles[i]);
        double u = t / det_spacing + c_d;
        double fl = floor(u);
        long j = (long)fl;
        double w = u - fl;
        const double *qrow = Q + (size_t)i * n_det;
        double q = (1.0 - w) * q_at(qrow, n_det, j) + w * q_at(qrow, n_det, j + 1);
        acc += (long double)q;                                 /* PAPER.md:59, eq. 2 */
    }
    if (scaled) acc *= (long double)ORACLE_PI / (long double)n_angles;
    return (double)acc;
}

/* O3 over whole images. */
void fbp_oracle_backproject(const double *Q, double *f, int batch, int n_angles, int n_det,
                            const double *angles, double det_spacing, int image_n,
                            double pixel_size, int scaled, int threads)
{
    long rows = (long)batch * image_n;
    int nt = pick_threads(threads);
    (void)nt;
#pragma omp parallel for schedule(static) num_threads(nt)
    for (long br = 0; br < rows; ++br) {
        long b = br / image_n;
        int r = (int)(br % image_n);
        const double *Qb = Q + (size_t)b * n_angles * n_det;
        double *fb = f + (size_t)b * image_n * image_n;
        for (int c = 0; c < image_n; ++c)
            fb[(size_t)r * image_n + c] = backproject_pixel(Qb, n_angles, n_det, angles, det_spacing,
                                                            image_n, pixel_size, r, c, scaled);
    }
}

/* O3 on a list of pixels of slice 0 (sampled parity at sizes where a whole image is slow). */
void fbp_oracle_backproject_pixels(const double *Q, const int *rows, const int *cols, long n_pix,
                                   double *out, int n_angles, int n_det, const double *angles,
                                   double det_spacing, int image_n, double pixel_size, int threads)
{
    int nt = pick_threads(threads);
    (void)nt;
#pragma omp parallel for schedule(static) num_threads(nt)
    for (long p = 0; p < n_pix; ++p)
        out[p] = backproject_pixel(Q, n_angles, n_det, angles, det_spacing, image_n, pixel_size,
                                   rows[p], cols[p], 1);
}

/* O2 on a list of rows (sampled parity for the filter at large sizes). */
void fbp_oracle_filter_rows(const double *P, const int *row_ids, long n_rows, double *Q_rows,
                            int n_det, double det_spacing, int threads)
{
    int nt = pick_threads(threads);
    (void)nt;
#pragma omp parallel for schedule(static) num_threads(nt)
    for (long s = 0; s < n_rows; ++s) {
        const double *p = P + (size_t)row_ids[s] * n_det;
        double *q = Q_rows + (size_t)s * n_det;
        for (int n = 0; n < n_det; ++n) {
            long double acc = 0.0L;
            for (int k = 0; k < n_det; ++k)
                acc += (long double)(ramlak_tap((long)n - (long)k) * p[k]);
            q[n] = (double)(acc / (long double)det_spacing);
        }
    }
}

/*
 * O4: forward projector R := B^T as a scatter, one slice, sequential (its bins have many
 * writers, which is exactly the read-modify-write hazard of PAPER.md:218, so it is kept
 * single-threaded).  y[i][j] += (1-w) x[p],  y[i][j+1] += w x[p], bins outside the
 * detector skipped.  `y` is overwritten.
 */
void fbp_oracle_forward_scatter(const double *x_img, double *y_sino, int n_angles, int n_det,
                                const double *angles, double det_spacing, int image_n,
                                double pixel_size)
{
    double c_n = 0.5 * (double)(image_n - 1);
    double c_d = 0.5 * (double)(n_det - 1);
    for (size_t e = 0; e < (size_t)n_angles * n_det; ++e) y_sino[e] = 0.0;
    for (int i = 0; i < n_angles; ++i) {
        double cs = cos(angles[i]), sn = sin(angles[i]);
        double *yrow = y_sino + (size_t)i * n_det;
        for (int r = 0; r < image_n; ++r)
            for (int c = 0; c < image_n; ++c) {
                double px = ((double)c - c_n) * pixel_size;
                double py = ((double)r - c_n) * pixel_size;
                double u = (px * cs + py * sn) / det_spacing + c_d;
                double fl = floor(u);
                long j = (long)fl;
                double w = u - fl;
                double v = x_img[(size_t)r * image_n + c];
                if (j >= 0 && j < n_det) yrow[j] += (1.0 - w) * v;
                if (j + 1 >= 0 && j + 1 < n_det) yrow[j + 1] += w * v;
            }
    }
}

/* eq. 2 end to end: O2 then O3 (scaled).  `Q_work` is caller-provided scratch [batch][K][D]. */
void fbp_oracle_reconstruct(const double *P, double *Q_work, double *f, int batch, int n_angles,
                            int n_det, const double *angles, double det_spacing, int image_n,
                            double pixel_size, int threads)
{
    fbp_oracle_filter(P, Q_work, batch, n_angles, n_det, det_spacing, threads);
    fbp_oracle_backproject(Q_work, f, batch, n_angles, n_det, angles, det_spacing, image_n,
                           pixel_size, 1, threads);
}
