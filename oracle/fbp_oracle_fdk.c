/*
 * fbp_oracle_fdk.c -- ORACLE for the cone-beam algorithm of Feldkamp, Davis and Kress (FDK), the continuation
 * the paper announces (ref [20] at PAPER.md:259: "uses the filtered backprojection algorithm
 * in the reconstruction of three-dimensional images obtained by projections of a cone beam").
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as fbp_oracle.c: only tests/, smoke() and bench.py's
 * oracle legs may use it; it shares nothing with paper_2109_02174_b200/csrc/).  Plain fp64, long-double sums,
 * no blocking, no fusion, the textbook order: weight, filter, back-project.
 *
 * The paper gives no formula for FDK; what follows is the textbook algorithm (Kak & Slaney ch. 3.6 = ref [8],
 * PAPER.md:247; Feldkamp et al. 1984) in the conventions of fbp_oracle.c.  Every choice is a reading, listed in
 * DESIGN.md ("FDK readings" C1-C7):
 *   C1  circular orbit of radius `sad` (source to rotation axis) in the plane z = 0.  With e_a = (cos b, sin b, 0)
 *       and e_s = (-sin b, cos b, 0) (b = the angle; e_a is the detector axis of the parallel-beam code, rays of
 *       PAPER.md:55 run along e_s), the source sits at -sad * e_s.
 *   C2  flat VIRTUAL detector through the rotation axis, spanned by e_a (columns, spacing d_a) and e_z (rows,
 *       spacing d_b), centred:  a_j = (j - (n_a-1)/2) d_a,  b_i = (i - (n_b-1)/2) d_b.
 *       p[beta][i][j] = line integral from the source through (a_j, b_i).
 *   C3  pre-weight   p'[beta][i][j] = p[beta][i][j] * sad / sqrt(sad^2 + a_j^2 + b_i^2).
 *   C4  row filter   Q[beta][i][:] = (1/d_a) h * p'[beta][i][:]  along the columns, h = the Ram-Lak taps of
 *       fbp_oracle.c (O1, O2) -- the same filter as the 2-D method; the factor 1/2 of the fan-beam filter
 *       g = h/2 is carried by the angular weight below.
 *   C5  back-projection of voxel r = (x, y, z):  t = r.e_a,  s = r.e_s,  U = sad + s,
 *         a' = sad t / U,   b' = sad z / U,   weight (sad / U)^2,
 *         f(r) = (pi / K) * sum_beta (sad/U)^2 * bilinear(Q[beta]; a'/d_a + (n_a-1)/2, b'/d_b + (n_b-1)/2),
 *       bilinear = linear in each detector coordinate, zero outside the detector.  pi/K = (1/2)(2 pi / K): the
 *       angles are meant to cover [0, 2 pi) uniformly (C6); as sad -> infinity this is the 2-D method with the
 *       K angles spread over 2 pi.
 *   C6  angles: caller-supplied radians, K values.
 *   C7  volume grid: x = (c - (N-1)/2) pix, y = (r - (N-1)/2) pix as in 2-D (row <-> +y), z_k = (k - (n_z-1)/2) vz;
 *       layout f[n_z][N][N].
 *
 * Pins (tests/test_oracle_fdk.py): the parallel limit (sad = 1e9 N: every detector row is an independent 2-D
 * problem and the result must equal fbp_oracle.c's, itself pinned by P1-P12); the mid-plane of a centred and of
 * an off-centre ball from ANALYTIC cone-beam line integrals (fan-beam FBP is exact there up to discretisation:
 * catches a wrong power of sad/U, a wrong sign of s, a missing pre-weight); a dense brute-force matrix on a
 * 4 x 4 x 3 volume built by an independent loop; the pre-weight's closed form; linearity; z-symmetry.
 */
#include <math.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static const double FDK_PI = 3.14159265358979323846264338327950288;

static int fdk_threads(int threads)
{
#ifdef _OPENMP
    int m = omp_get_max_threads();
#else
    int m = 1;
#endif
    if (threads <= 0 || threads > m) return m;
    return threads;
}

/* C3: out[beta][i][j] = p[beta][i][j] * sad / sqrt(sad^2 + a_j^2 + b_i^2). */
void fbp_oracle_fdk_weight(const double *p, double *out, int n_angles, int n_b, int n_a, double d_a, double d_b,
                           double sad)
{
    for (int k = 0; k < n_angles; ++k)
        for (int i = 0; i < n_b; ++i)
            for (int j = 0; j < n_a; ++j) {
                double a = ((double)j - 0.5 * (double)(n_a - 1)) * d_a;
                double b = ((double)i - 0.5 * (double)(n_b - 1)) * d_b;
                size_t e = ((size_t)k * n_b + i) * n_a + j;
                out[e] = p[e] * sad / sqrt(sad * sad + a * a + b * b);
            }
}

static double q_at2(const double *Q, int n_b, int n_a, long i, long j)
{
    if (i < 0 || i >= n_b || j < 0 || j >= n_a) return 0.0;
    return Q[(size_t)i * n_a + j];
}

/* C5: f[n_z][N][N] from the filtered, weighted projections Q[K][n_b][n_a]. */
void fbp_oracle_fdk_backproject(const double *Q, double *f, int n_angles, int n_b, int n_a, const double *angles,
                                double d_a, double d_b, double sad, int image_n, double pixel_size, int n_z,
                                double voxel_z, int threads)
{
    int nt = fdk_threads(threads);
    double c_n = 0.5 * (double)(image_n - 1), c_z = 0.5 * (double)(n_z - 1);
    double c_a = 0.5 * (double)(n_a - 1), c_b = 0.5 * (double)(n_b - 1);
    long rows = (long)n_z * image_n;
    (void)nt;
#pragma omp parallel for schedule(static) num_threads(nt)
    for (long kr = 0; kr < rows; ++kr) {
        int k = (int)(kr / image_n), r = (int)(kr % image_n);
        double z = ((double)k - c_z) * voxel_z, y = ((double)r - c_n) * pixel_size;
        for (int c = 0; c < image_n; ++c) {
            double x = ((double)c - c_n) * pixel_size;
            long double acc = 0.0L;
            for (int m = 0; m < n_angles; ++m) {
                double cb = cos(angles[m]), sb = sin(angles[m]);
                double t = x * cb + y * sb;            /* r . e_a */
                double s = -x * sb + y * cb;           /* r . e_s */
                double U = sad + s;
                double ua = (sad * t / U) / d_a + c_a;
                double ub = (sad * z / U) / d_b + c_b;
                double fa = floor(ua), fb = floor(ub);
                long ja = (long)fa, ib = (long)fb;
                double wa = ua - fa, wb = ub - fb;
                const double *Qm = Q + (size_t)m * n_b * n_a;
                double v = (1.0 - wb) * ((1.0 - wa) * q_at2(Qm, n_b, n_a, ib, ja) + wa * q_at2(Qm, n_b, n_a, ib, ja + 1)) +
                           wb * ((1.0 - wa) * q_at2(Qm, n_b, n_a, ib + 1, ja) + wa * q_at2(Qm, n_b, n_a, ib + 1, ja + 1));
                double w = sad / U;
                acc += (long double)(w * w * v);
            }
            f[((size_t)k * image_n + r) * image_n + c] = (double)(acc * (long double)FDK_PI / (long double)n_angles);
        }
    }
}
