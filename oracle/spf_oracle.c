/*
 * spf_oracle.c -- the ORACLE for the M-TIP slicing + orientation-matching path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It
 * shares no code, header, table or helper with the CUDA path under
 * paper_2109_05339_b200/ and neither side includes the other.
 *
 * What it is: the plain definition of what the path computes, written out slowly in
 * fp64 (PAPER.md gives no formulas, so the definitions are the readings recorded in
 * SURVEY.md section 8(c) / DESIGN.md "Readings"):
 *
 *   slicing   (section 2.1: "M 2D model images ... computed via the
 *              type-2 (uniform to nonuniform, a.k.a. 'forward') NUFFT of the
 *              autocorrelation"): the exact transform a type-2 NUFFT approximates is
 *              the nonuniform DFT
 *                  c(x) = sum_n A[n] exp(-i n.x),  n = (i1,i2,i3) - floor(N/2),
 *              evaluated at x = R(quat) q_pixel.  No kernel, no fine grid, no FFT.
 *   matching  (section 2.2: "compared to all of the M model images ...
 *              closest in the Euclidean distance metric"): d[i][m] = sum_j mask_j
 *              (I[i][j] - S[m][j])^2 as a sum of squared differences, then argmin over
 *              m with the lowest index winning exact ties.
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): Gaussian-blob closed form
 * with an off-centre, axis-distinct centre (sign, centring, axis order, normalisation);
 * equality with numpy.fft.fftn at x = 2 pi k / N; Friedel symmetry; real-even => real;
 * rotation conventions (identity, q vs -q, 90 degrees about z, composition, isotropy);
 * linearity; distances == scipy cdist 'sqeuclidean'; planted / permuted / tied argmin.
 * No function here is "parity unpinned".
 *
 * Two evaluations of the same NUDFT are kept on purpose: oracle_nudft_direct() is the
 * un-factored triple loop with one complex exponential per voxel (obviously the
 * definition, affordable on Tiny only); oracle_nudft() groups the same sum by axis
 * (sum_n1 e1 sum_n2 e2 sum_n3 A e3), which is the same definition with the factor
 * exp(-i n.x) = e1 e2 e3 pulled out of inner sums -- tests check one against the other.
 *
 * Build: gcc -O2 -fopenmp -fPIC -shared spf_oracle.c -o liboracle.so -lm   (oracle/build.py)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* number of threads the parallel loops will use (reported by bench.py as "cores") */
int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * Rotation matrix of a quaternion (w,x,y,z), normalised first.  Reading s2:
 * Hamilton convention, ACTIVE rotation, x_rot = R q.  Rows as in SURVEY.md 8(c) item 2.
 * quat: 4 floats (the same fp32 values the GPU gets), R: 9 doubles row-major.
 */
void oracle_rotation_matrix(const float *quat, double *R) {
    double w = quat[0], x = quat[1], y = quat[2], z = quat[3];
    double nrm = sqrt(w * w + x * x + y * y + z * z);
    w /= nrm; x /= nrm; y /= nrm; z /= nrm;
    R[0] = 1.0 - 2.0 * (y * y + z * z); R[1] = 2.0 * (x * y - w * z);       R[2] = 2.0 * (x * z + w * y);
    R[3] = 2.0 * (x * y + w * z);       R[4] = 1.0 - 2.0 * (x * x + z * z); R[5] = 2.0 * (y * z - w * x);
    R[6] = 2.0 * (x * z - w * y);       R[7] = 2.0 * (y * z + w * x);       R[8] = 1.0 - 2.0 * (x * x + y * y);
}

/* x[3] = R q, q given as 3 floats (widened), all arithmetic fp64 */
static void rotate_point(const double *R, const float *q, double *x) {
    double q0 = q[0], q1 = q[1], q2 = q[2];
    x[0] = R[0] * q0 + R[1] * q1 + R[2] * q2;
    x[1] = R[3] * q0 + R[4] * q1 + R[5] * q2;
    x[2] = R[6] * q0 + R[7] * q1 + R[8] * q2;
}

/*
 * Un-factored nonuniform DFT: c = sum over ALL voxels of A[n] * exp(-i n.x).
 * model: [N][N][N] C-order fp32 (axis order (x,y,z) = (i1,i2,i3)); x: npts x 3 doubles
 * (radians per voxel); out: npts x 2 doubles (re, im).  Sign: reading s1, exponent -i.
 */
void oracle_nudft_direct(const float *model, int N, const double *x, int64_t npts, double *out) {
    const int c = N / 2; /* floor(N/2): for odd N the centre voxel is n = 0 */
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t p = 0; p < npts; ++p) {
        double re = 0.0, im = 0.0;
        for (int i1 = 0; i1 < N; ++i1)
            for (int i2 = 0; i2 < N; ++i2)
                for (int i3 = 0; i3 < N; ++i3) {
                    double a = model[((size_t)i1 * N + i2) * N + i3];
                    double ph = (double)(i1 - c) * x[3 * p + 0] + (double)(i2 - c) * x[3 * p + 1] +
                                (double)(i3 - c) * x[3 * p + 2];
                    re += a * cos(ph);
                    im -= a * sin(ph);
                }
        out[2 * p + 0] = re;
        out[2 * p + 1] = im;
    }
}

/*
 * The same sum grouped by axis:  c = sum_n1 e1[n1] ( sum_n2 e2[n2] ( sum_n3 A[n] e3[n3] ) ),
 * e_d[n] = exp(-i (n - c) x_d), each phase from its own cos/sin (no recurrences).
 */
void oracle_nudft(const float *model, int N, const double *x, int64_t npts, double *out) {
    const int c = N / 2;
#pragma omp parallel
    {
        double *e = (double *)malloc(sizeof(double) * 6 * (size_t)N);
        double *e1r = e, *e1i = e + N, *e2r = e + 2 * N, *e2i = e + 3 * N, *e3r = e + 4 * N, *e3i = e + 5 * N;
#pragma omp for schedule(dynamic, 1)
        for (int64_t p = 0; p < npts; ++p) {
            for (int n = 0; n < N; ++n) {
                double k = (double)(n - c);
                e1r[n] = cos(k * x[3 * p + 0]); e1i[n] = -sin(k * x[3 * p + 0]);
                e2r[n] = cos(k * x[3 * p + 1]); e2i[n] = -sin(k * x[3 * p + 1]);
                e3r[n] = cos(k * x[3 * p + 2]); e3i[n] = -sin(k * x[3 * p + 2]);
            }
            double cr = 0.0, ci = 0.0;
            for (int i1 = 0; i1 < N; ++i1) {
                double t2r = 0.0, t2i = 0.0;
                for (int i2 = 0; i2 < N; ++i2) {
                    const float *row = model + ((size_t)i1 * N + i2) * N;
                    double t3r = 0.0, t3i = 0.0;
                    for (int i3 = 0; i3 < N; ++i3) {
                        double a = row[i3];
                        t3r += a * e3r[i3];
                        t3i += a * e3i[i3];
                    }
                    t2r += t3r * e2r[i2] - t3i * e2i[i2];
                    t2i += t3r * e2i[i2] + t3i * e2r[i2];
                }
                cr += t2r * e1r[i1] - t2i * e1i[i1];
                ci += t2r * e1i[i1] + t2i * e1r[i1];
            }
            out[2 * p + 0] = cr;
            out[2 * p + 1] = ci;
        }
        free(e);
    }
}

/*
 * Slices at selected (orientation, pixel) pairs: x = R(quats[m]) pix_q[j], c = NUDFT(x).
 * sel_m / sel_j: nsel index pairs; pass sel_m = sel_j = NULL for the full M x P set
 * (then nsel must be M*P and out is [M][P][2]).  direct != 0 selects the un-factored loop.
 */
void oracle_slice(const float *model, int N, const float *quats, int64_t M, const float *pix_q, int64_t P,
                  const int64_t *sel_m, const int64_t *sel_j, int64_t nsel, int direct, double *out) {
    double *x = (double *)malloc(sizeof(double) * 3 * (size_t)nsel);
    for (int64_t s = 0; s < nsel; ++s) {
        int64_t m = sel_m ? sel_m[s] : s / P;
        int64_t j = sel_j ? sel_j[s] : s % P;
        double R[9];
        oracle_rotation_matrix(quats + 4 * m, R);
        rotate_point(R, pix_q + 3 * j, x + 3 * s);
    }
    (void)M;
    if (direct) oracle_nudft_direct(model, N, x, nsel, out);
    else        oracle_nudft(model, N, x, nsel, out);
    free(x);
}

/*
 * Squared Euclidean distances as a sum of squared differences (NOT the expanded form):
 * d[i][m] = sum_{j: mask[j] != 0} (I[i][j] - S[m][j])^2.   PAPER.md:72, readings s7, s8.
 * images [n_img][P] fp32, slices [M][P] fp32 (the same fp32 arrays spf_match gets),
 * mask [P] bytes or NULL (= all pixels used); dist [n_img][M] doubles.
 */
void oracle_distances(const float *images, int64_t n_img, const float *slices, int64_t M, int64_t P,
                      const uint8_t *mask, double *dist) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < n_img; ++i) {
        const float *I = images + (size_t)i * P;
        for (int64_t m = 0; m < M; ++m) {
            const float *S = slices + (size_t)m * P;
            double d = 0.0;
            for (int64_t j = 0; j < P; ++j) {
                if (mask && !mask[j]) continue;
                double t = (double)I[j] - (double)S[j];
                d += t * t;
            }
            dist[(size_t)i * M + m] = d;
        }
    }
}

/* the same with fp64 slices (oracle slices fed straight to the oracle matcher) */
void oracle_distances_f64(const float *images, int64_t n_img, const double *slices, int64_t M, int64_t P,
                          const uint8_t *mask, double *dist) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < n_img; ++i) {
        const float *I = images + (size_t)i * P;
        for (int64_t m = 0; m < M; ++m) {
            const double *S = slices + (size_t)m * P;
            double d = 0.0;
            for (int64_t j = 0; j < P; ++j) {
                if (mask && !mask[j]) continue;
                double t = (double)I[j] - S[j];
                d += t * t;
            }
            dist[(size_t)i * M + m] = d;
        }
    }
}

/*
 * Argmin over m of each row of dist [n_img][M]: lowest index wins exact ties (reading s9).
 * Also returns the runner-up (second smallest distance, over m != best) so that callers
 * can list near-ties; second_dist = +inf when M == 1.
 */
void oracle_argmin(const double *dist, int64_t n_img, int64_t M, int64_t *best_idx, double *best_dist,
                   double *second_dist) {
    for (int64_t i = 0; i < n_img; ++i) {
        const double *d = dist + (size_t)i * M;
        int64_t b = 0;
        for (int64_t m = 1; m < M; ++m)
            if (d[m] < d[b]) b = m;
        double s = INFINITY;
        for (int64_t m = 0; m < M; ++m)
            if (m != b && d[m] < s) s = d[m];
        best_idx[i] = b;
        best_dist[i] = d[b];
        second_dist[i] = s;
    }
}
