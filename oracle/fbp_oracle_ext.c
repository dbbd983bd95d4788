/*
 * fbp_oracle_ext.c -- ORACLE, continued: the rows SURVEY.md 8(f) marks "next".
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as fbp_oracle.c: only tests/,
 * smoke() and bench.py's cpu_baseline / --impl reference legs may use it; it shares nothing
 * with paper_2109_02174_b200/csrc/).  Plain fp64 with long-double sums, no blocking, no fusion.
 *
 * W1  Apodised reconstruction filters.  The paper's filter is a generic H (PAPER.md:61,
 *     "Q_theta = P_theta * H"); the taps are the inverse DTFT of |f| W(f) on |f| <= 1/2
 *     cycles per sample (Kak & Slaney ch. 3 = ref [8]):
 *         h_W[m] = 2 * integral_0^{1/2} f W(f) cos(2 pi f m) df .
 *     window 0 Ram-Lak       W = 1                       (BASELINE.json north_star item 2)
 *            1 Shepp-Logan   W = sin(pi f) / (pi f)
 *            2 cosine        W = cos(pi f)
 *            3 Hamming       W = 0.54 + 0.46 cos(2 pi f)
 *            4 Hann          W = 0.5  + 0.5  cos(2 pi f)
 *     The integrals have closed forms, written out below; tests/test_oracle_ext.py pins each
 *     against numerical quadrature of the defining integral (scipy), against the DTFT of the
 *     taps, and against the Ram-Lak taps of fbp_oracle.c for window 0.
 * W2  Per-angle weights (non-uniform angle sets): f = sum_i w_i q_i with
 *     caller-supplied w_i instead of pi/K each (eq. 2, weighted).  Pinned in
 *     tests/test_oracle_ext.py: uniform weights == the core back-projector; one-hot e_i == the core
 *     back-projector on the sinogram with every row but i zeroed (x K/pi); random weights == the
 *     dense brute-force matrix of P7 with the columns of angle i scaled by w_i (the last two fix
 *     WHICH weight goes with WHICH angle).
 * M1  PSNR (eq. 3) and the global-statistics SSIM (eq. 4).
 */
#include <math.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static const double EXT_PI = 3.14159265358979323846264338327950288;

static int ext_threads(int threads)
{
#ifdef _OPENMP
    int m = omp_get_max_threads();
#else
    int m = 1;
#endif
    if (threads <= 0 || threads > m) return m;
    return threads;
}

/* W = 1:  h[0] = 1/4,  h[odd m] = -1/(pi^2 m^2),  h[even m != 0] = 0. */
static double tap_ramlak(long m)
{
    if (m == 0) return 0.25;
    if (m % 2 == 0) return 0.0;
    return -1.0 / (EXT_PI * EXT_PI * (double)m * (double)m);
}

/* integral_0^{1/2} f cos(a f) df = sin(a/2)/(2a) + (cos(a/2) - 1)/a^2   (a != 0). */
static double int_f_cos(double a)
{
    return sin(0.5 * a) / (2.0 * a) + (cos(0.5 * a) - 1.0) / (a * a);
}

/* W1: one tap of window `window`; returns NaN for an unknown window. */
double fbp_oracle_window_tap(int window, long m)
{
    switch (window) {
    case 0:
        return tap_ramlak(m);
    case 1:
        /* 2 int f sin(pi f)/(pi f) cos(2 pi f m) = (1/pi) int [sin(pi f (1+2m)) + sin(pi f (1-2m))]
         * = (1/pi^2) [1/(1+2m) + 1/(1-2m)]   (cos(pi/2 + pi m) = 0)  = -2 / (pi^2 (4 m^2 - 1)) */
        return -2.0 / (EXT_PI * EXT_PI * (4.0 * (double)m * (double)m - 1.0));
    case 2:
        /* 2 f cos(pi f) cos(2 pi f m) = f [cos(pi f (2m+1)) + cos(pi f (2m-1))] */
        return int_f_cos(EXT_PI * (2.0 * (double)m + 1.0)) + int_f_cos(EXT_PI * (2.0 * (double)m - 1.0));
    case 3:
    case 4: {
        /* cos(2 pi f) cos(2 pi f m) = (1/2)[cos(2 pi f (m+1)) + cos(2 pi f (m-1))] */
        double alpha = window == 3 ? 0.54 : 0.5, beta = 1.0 - alpha;
        return alpha * tap_ramlak(m) + 0.5 * beta * (tap_ramlak(m + 1) + tap_ramlak(m - 1));
    }
    default:
        return NAN;
    }
}

/* h_out[m + (D-1)] = h_W[m], m = -(D-1) .. D-1. */
void fbp_oracle_window_taps(int n_det, int window, double *h_out)
{
    for (long m = -(long)(n_det - 1); m <= (long)(n_det - 1); ++m)
        h_out[m + (n_det - 1)] = fbp_oracle_window_tap(window, m);
}

/* Q[i][n] = (1/d) sum_k h_W[n-k] P[i][k]: the filter step of PAPER.md:61 with window W. */
void fbp_oracle_filter_window(const double *P, double *Q, int batch, int n_angles, int n_det,
                              double det_spacing, int window, int threads)
{
    long rows = (long)batch * n_angles;
    int nt = ext_threads(threads);
    (void)nt;
#pragma omp parallel for schedule(static) num_threads(nt)
    for (long row = 0; row < rows; ++row) {
        const double *p = P + row * n_det;
        double *q = Q + row * n_det;
        for (int n = 0; n < n_det; ++n) {
            long double acc = 0.0L;
            for (int k = 0; k < n_det; ++k)
                acc += (long double)(fbp_oracle_window_tap(window, (long)n - (long)k) * p[k]);
            q[n] = (double)(acc / (long double)det_spacing);
        }
    }
}

/* W2: f[r][c] = sum_i w_i * lerp(Q~_i, u_i)  (eq. 2, with per-angle weights). */
void fbp_oracle_backproject_weighted(const double *Q, double *f, int batch, int n_angles, int n_det,
                                     const double *angles, const double *weights,
                                     double det_spacing, int image_n, double pixel_size, int threads)
{
    long rows = (long)batch * image_n;
    int nt = ext_threads(threads);
    double c_n = 0.5 * (double)(image_n - 1), c_d = 0.5 * (double)(n_det - 1);
    (void)nt;
#pragma omp parallel for schedule(static) num_threads(nt)
    for (long br = 0; br < rows; ++br) {
        long b = br / image_n;
        int r = (int)(br % image_n);
        const double *Qb = Q + (size_t)b * n_angles * n_det;
        for (int c = 0; c < image_n; ++c) {
            double x = ((double)c - c_n) * pixel_size, y = ((double)r - c_n) * pixel_size;
            long double acc = 0.0L;
            for (int i = 0; i < n_angles; ++i) {
                double u = (x * cos(angles[i]) + y * sin(angles[i])) / det_spacing + c_d;
                double fl = floor(u);
                long j = (long)fl;
                double w = u - fl;
                const double *qrow = Qb + (size_t)i * n_det;
                double q0 = (j >= 0 && j < n_det) ? qrow[j] : 0.0;
                double q1 = (j + 1 >= 0 && j + 1 < n_det) ? qrow[j + 1] : 0.0;
                acc += (long double)(weights[i] * ((1.0 - w) * q0 + w * q1));
            }
            f[(size_t)b * image_n * image_n + (size_t)r * image_n + c] = (double)acc;
        }
    }
}

/*
 * M1: image-similarity metrics of the paper, over all n pixels of one image pair.
 *   eq. 3:  PSNR = 20 log10( MAX / sqrt(MSE) ),  MSE = (1/n) sum (x - y)^2;
 *       MSE = 0 gives +infinity ("the images are the same").
 *   eq. 4:  SSIM = (2 mu_x mu_y + C1)(2 s_xy + C2) / ((mu_x^2 + mu_y^2 + C1)(s_x^2 + s_y^2 + C2))
 *       with global statistics over the whole image (the paper gives no window; SURVEY.md 2, item
 *       14): mu = mean, s_x^2, s_y^2 = population variances (divide by n), s_xy = population
 *       covariance.  Readings: MAX and the constants are caller-supplied; the
 *       customary C1 = (0.01 MAX)^2, C2 = (0.03 MAX)^2 are the binding's defaults, not the paper's.
 * Two passes (means first, then centred moments), long-double sums.
 * out[0] = MSE, out[1] = PSNR, out[2] = SSIM, out[3] = mu_x, out[4] = mu_y, out[5] = s_x^2,
 * out[6] = s_y^2, out[7] = s_xy.
 */
void fbp_oracle_metrics(const double *x, const double *y, long n, double max_val, double c1,
                        double c2, double *out)
{
    long double sx = 0.0L, sy = 0.0L, se = 0.0L;
    for (long i = 0; i < n; ++i) {
        sx += (long double)x[i];
        sy += (long double)y[i];
        long double e = (long double)x[i] - (long double)y[i];
        se += e * e;
    }
    long double mx = sx / (long double)n, my = sy / (long double)n;
    long double vx = 0.0L, vy = 0.0L, cxy = 0.0L;
    for (long i = 0; i < n; ++i) {
        long double a = (long double)x[i] - mx, b = (long double)y[i] - my;
        vx += a * a;
        vy += b * b;
        cxy += a * b;
    }
    vx /= (long double)n;
    vy /= (long double)n;
    cxy /= (long double)n;
    long double mse = se / (long double)n;
    out[0] = (double)mse;
    out[1] = mse > 0.0L ? 20.0 * log10(max_val / sqrt((double)mse)) : INFINITY;
    out[2] = (double)(((2.0L * mx * my + c1) * (2.0L * cxy + c2)) /
                      ((mx * mx + my * my + c1) * (vx + vy + c2)));
    out[3] = (double)mx;
    out[4] = (double)my;
    out[5] = (double)vx;
    out[6] = (double)vy;
    out[7] = (double)cxy;
}

/*
 * S1: a 3-D volume from a stack of reconstructed 2-D slices by interpolation along the stack axis
 * ("3D computed tomography images ... through the interpolation of a stack of 2D images";
 * PAPER.md:222).  The paper does not say which interpolation (its ref [21] is a PDE method that it
 * does not describe); reading taken (R4): LINEAR interpolation between the two neighbouring
 * slices, output slice m of n_out at stack coordinate z_m = m (n_in - 1)/(n_out - 1) (z_0 = 0 when
 * n_out = 1), k = floor(z_m) clamped to n_in - 2, t = z_m - k:
 *     out[m][p] = (1 - t) in[k][p] + t in[k+1][p]          (n_in = 1: out[m] = in[0]).
 * `n_pix` = pixels per slice.
 */
void fbp_oracle_interpolate_stack(const double *in, int n_in, double *out, int n_out, long n_pix)
{
    for (int m = 0; m < n_out; ++m) {
        double z = n_out > 1 ? (double)m * (double)(n_in - 1) / (double)(n_out - 1) : 0.0;
        long k = (long)floor(z);
        if (k > n_in - 2) k = n_in - 2;
        if (k < 0) k = 0;
        double t = n_in > 1 ? z - (double)k : 0.0;
        const double *a = in + (size_t)k * n_pix;
        const double *b = in + (size_t)(n_in > 1 ? k + 1 : k) * n_pix;
        double *o = out + (size_t)m * n_pix;
        for (long p = 0; p < n_pix; ++p) o[p] = (1.0 - t) * a[p] + t * b[p];
    }
}
