// tests/hostsim: the interpolation arithmetic of libspf compiled for the HOST from the very header the
// CUDA kernels include (paper_2109_05339_b200/csrc/spf_slice_math.cuh), so that tests can compare it
// with the oracle on a machine without a GPU.  TEST INFRASTRUCTURE ONLY: nothing in the product loads
// this library and it is not a CPU fallback.  The per-point sequence below mirrors one thread of
// k_slice (spf_slice.cu): rotate in fp64 -> cell + fraction -> 3 w weights -> gather.
//
// Build: g++ -O2 -fopenmp -fPIC -shared -std=c++17 -ffp-contract=off spf_hostsim.cpp -o libspf_hostsim.so
#include "../../paper_2109_05339_b200/csrc/spf_slice_math.cuh"

extern "C" {

void hostsim_deapod(int N, int nf, int w, double *out) {
    std::vector<double> p;
    spfm::deapodisation_factors(N, nf, w, 2.30 * w, p);
    for (int i = 0; i < N; ++i) out[i] = p[i];
}

int hostsim_fit(int w, float *coef /*[SPF_MAX_W][SPF_MAX_DEG+1]*/, double *worst) {
    return spfm::fit_kernel_polys(w, 2.30 * w, reinterpret_cast<float(*)[SPF_MAX_DEG + 1]>(coef), worst);
}

// grid: centred padded grid [np][np][sz] fp32 (is_real) or interleaved complex; out: [M][P] complex (re, im)
void hostsim_slice(const float *grid, int is_real, int np, int sz, int nf, int halo, int w, const float *quats, long M,
                   const float *pix, long P, int use_poly, float *out) {
    static float coef[SPF_MAX_W][SPF_MAX_DEG + 1];
    const double beta = 2.30 * w;
    const int deg = spfm::fit_kernel_polys(w, beta, coef);
    const double kPi = 3.14159265358979323846;
    const double xi_scale = (double)nf / (2.0 * kPi), inv_nf = 1.0 / (double)nf;
    const int off = nf / 2 + halo;
#pragma omp parallel for schedule(static)
    for (long m = 0; m < M; ++m) {
        double R[9];
        spfm::quat_to_R(quats + 4 * m, R);
        for (long j = 0; j < P; ++j) {
            const double q0 = pix[3 * j], q1 = pix[3 * j + 1], q2 = pix[3 * j + 2];
            int px, py, pz;
            float fx, fy, fz;
            spfm::cell_and_fraction(R[0] * q0 + R[1] * q1 + R[2] * q2, xi_scale, inv_nf, nf, off, np, w, px, fx);
            spfm::cell_and_fraction(R[3] * q0 + R[4] * q1 + R[5] * q2, xi_scale, inv_nf, nf, off, np, w, py, fy);
            spfm::cell_and_fraction(R[6] * q0 + R[7] * q1 + R[8] * q2, xi_scale, inv_nf, nf, off, np, w, pz, fz);
            float wx[SPF_MAX_W], wy[SPF_MAX_W], wz[SPF_MAX_W];
            if (use_poly) {
                spfm::weights_poly<SPF_MAX_W>(fx, w, coef, deg, wx); spfm::weights_poly<SPF_MAX_W>(fy, w, coef, deg, wy);
                spfm::weights_poly<SPF_MAX_W>(fz, w, coef, deg, wz);
            } else {
                spfm::weights_direct<SPF_MAX_W>(fx, w, (float)beta, wx); spfm::weights_direct<SPF_MAX_W>(fy, w, (float)beta, wy);
                spfm::weights_direct<SPF_MAX_W>(fz, w, (float)beta, wz);
            }
            const int E = is_real ? 1 : 2;
            const float *base = grid + ((size_t)((size_t)px * np + py) * sz + pz) * E;
            spfm::c2 c = is_real ? spfm::gather<SPF_MAX_W, true>(base, np * sz, sz, w, wx, wy, wz)
                                 : spfm::gather<SPF_MAX_W, false>(base, np * sz, sz, w, wx, wy, wz);
            out[2 * (m * P + j)] = c.x;
            out[2 * (m * P + j) + 1] = c.y;
        }
    }
}

// cell index and fraction of one coordinate, for the index-range tests
void hostsim_cell(double x, int nf, int halo, int w, int *p, float *f) {
    const double kPi = 3.14159265358979323846;
    spfm::cell_and_fraction(x, (double)nf / (2.0 * kPi), 1.0 / (double)nf, nf, nf / 2 + halo, nf + 2 * halo, w, *p, *f);
}

}  // extern "C"
