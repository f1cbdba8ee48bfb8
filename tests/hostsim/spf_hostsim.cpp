// tests/hostsim: the interpolation arithmetic of libspf compiled for the HOST from the very header the
// CUDA kernels include (paper_2109_05339_b200/csrc/spf_slice_math.cuh), so that tests can compare it
// with the oracle on a machine without a GPU.  TEST INFRASTRUCTURE ONLY: nothing in the product loads
// this library and it is not a CPU fallback.  The per-point sequence below mirrors one thread of
// k_slice (spf_slice.cu): rotate in fp64 -> cell + fraction -> 3 w weights -> gather.
//
// Build: g++ -O2 -fopenmp -fPIC -shared -std=c++17 -ffp-contract=off spf_hostsim.cpp -o libspf_hostsim.so
#include <limits.h>

#include <algorithm>
#include <cmath>

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

// Replay of one k_slice<COOP | GCOOP> launch on the CPU, block by block (spf_slice.cu): patch table ->
// per-point cell + fraction -> block bounding box -> tile_geom -> the tile image TMA would write (one
// (by x bz) box per x-plane at pitch S1, zeros outside the padded grid) -> gather from the tile, lane by
// lane as a warp does it (coop = 1; coop = 2 is variant 3, the same
// walk with no tile, straight from the grid: weights parked in the
// 28-float layout, groups of 8 points, partial sums added by the multi-value butterfly).  Everything the tile image
// does NOT receive from a copy is NaN, so a read outside the staged box poisons the result even
// where its weight is zero.  stats: [0] blocks staged, [1] blocks not staged (global gather),
// [2] largest tile in bytes.
void hostsim_slice_blocks(const float *grid, int is_real, int np, int sz, int nf, int halo, int w, const float *quats, long M,
                          const float *pix, long P, const int *patch, long n_patches, int coop, unsigned cap_bytes,
                          float *out, long *stats) {
    static float coef[SPF_MAX_W][SPF_MAX_DEG + 1];
    const double beta = 2.30 * w;
    const int deg = spfm::fit_kernel_polys(w, beta, coef);
    const double kPi = 3.14159265358979323846;
    const double xi_scale = (double)nf / (2.0 * kPi), inv_nf = 1.0 / (double)nf;
    const int off = nf / 2 + halo;
    const int E = is_real ? 1 : 2, CELL = 4 * E;
    const int PATCH = 128;
    long n_staged = 0, n_global = 0, max_tile = 0;
#pragma omp parallel for schedule(dynamic) reduction(+ : n_staged, n_global) reduction(max : max_tile)
    for (long blk = 0; blk < M * n_patches; ++blk) {
        const long m = blk / n_patches, pt = blk % n_patches;
        double R[9];
        spfm::quat_to_R(quats + 4 * m, R);
        int px[PATCH], py[PATCH], pz[PATCH];
        long jj[PATCH];
        float wx[PATCH][SPF_MAX_W], wy[PATCH][SPF_MAX_W], wz[PATCH][SPF_MAX_W];
        int lo[3] = {INT_MAX, INT_MAX, INT_MAX}, hi[3] = {INT_MIN, INT_MIN, INT_MIN};
        for (int t = 0; t < PATCH; ++t) {
            const long j = patch[pt * PATCH + t];
            jj[t] = j;
            if (j < 0) continue;
            const double q0 = pix[3 * j], q1 = pix[3 * j + 1], q2 = pix[3 * j + 2];
            float fx, fy, fz;
            spfm::cell_and_fraction(R[0] * q0 + R[1] * q1 + R[2] * q2, xi_scale, inv_nf, nf, off, np, w, px[t], fx);
            spfm::cell_and_fraction(R[3] * q0 + R[4] * q1 + R[5] * q2, xi_scale, inv_nf, nf, off, np, w, py[t], fy);
            spfm::cell_and_fraction(R[6] * q0 + R[7] * q1 + R[8] * q2, xi_scale, inv_nf, nf, off, np, w, pz[t], fz);
            spfm::weights_poly<SPF_MAX_W>(fx, w, coef, deg, wx[t]); spfm::weights_poly<SPF_MAX_W>(fy, w, coef, deg, wy[t]);
            spfm::weights_poly<SPF_MAX_W>(fz, w, coef, deg, wz[t]);
            lo[0] = std::min(lo[0], px[t]); hi[0] = std::max(hi[0], px[t]);
            lo[1] = std::min(lo[1], py[t]); hi[1] = std::max(hi[1], py[t]);
            lo[2] = std::min(lo[2], pz[t]); hi[2] = std::max(hi[2], pz[t]);
        }
        const bool any = hi[0] >= lo[0];
        const int Lx = any ? hi[0] - lo[0] + w : 0, Ly = any ? hi[1] - lo[1] + w : 0, Lz = any ? hi[2] - lo[2] + w : 0;
        spfm::TileGeom g = spfm::tile_geom(Lx, Ly, Lz, w, CELL, cap_bytes);
        if (coop == 2) g.ok = false;        // variant 3: no tile at all (tile_geom itself refuses w > 8)
        std::vector<float> tile;
        if (g.ok) {
            n_staged++;
            max_tile = std::max(max_tile, (long)Lx * g.S1 * CELL);
            tile.assign((size_t)(cap_bytes / 4) + 8192, std::nanf(""));   // slack: a stray read must find NaN, not crash
            for (int x = 0; x < Lx; ++x)          // one TMA copy per x-plane: box (bz*E floats, by rows, 1 plane)
                for (int y = 0; y < g.by; ++y)
                    for (int z = 0; z < g.bz * E; ++z) {
                        const long gx = lo[0] + x, gy = lo[1] + y, gz = (long)lo[2] * E + z;
                        const bool in = gx < np && gy < np && gz < (long)sz * E;   // TMA fills out-of-range elements with zeros
                        tile[(size_t)x * g.S1 * E + (size_t)y * g.bz * E + z] = in ? grid[((size_t)gx * np + gy) * sz * E + gz] : 0.0f;
                    }
        } else {
            n_global++;
        }
        spfm::c2 res[PATCH];
        {
            // weights parked in the 28-float layout (slots of empty lanes hold NaN: they must never be read)
            const bool wide = w > 8;                 // variant 3 at w = 10: 16-cell window, 44-float weight sets
            const int wstride = wide ? SPF_COOPW_STRIDE : SPF_COOP_STRIDE;
            std::vector<float> wts((size_t)PATCH * wstride, std::nanf(""));
            for (int t = 0; t < PATCH; ++t) {
                if (wide) {
                    float pk[44];
                    spfm::coop_pack_weights_wide<SPF_MAX_W>(pk, w, wx[t], wy[t], wz[t]);
                    for (int v = 0; v < 44; ++v) wts[(size_t)t * wstride + v] = jj[t] >= 0 ? pk[v] : std::nanf("");
                } else {
                    float pk[24];
                    spfm::coop_pack_weights<SPF_MAX_W>(pk, w, wx[t], wy[t], wz[t]);
                    for (int v = 0; v < 24; ++v) wts[(size_t)t * wstride + v] = jj[t] >= 0 ? pk[v] : std::nanf("");
                }
            }
            // one lane's partial sum for point t: from the staged tile, or (variant 3, and blocks of variant 2
            // whose box does not fit) straight from the padded grid with the y / z clamp of the kernel
            auto lane_part = [&](int t, int lane) {
                const float *wt = &wts[(size_t)t * wstride];
                if (wide) {      // exactly the w x w taps: no clamp
                    const long long cell = ((long long)px[t] * np + py[t]) * sz + pz[t];
                    return is_real ? spfm::gather_coop_lane_wide<true, long long>(grid, cell, np * sz, sz, w, wt, lane)
                                   : spfm::gather_coop_lane_wide<false, long long>(grid, cell, np * sz, sz, w, wt, lane);
                }
                if (g.ok) {
                    const int cell = (px[t] - lo[0]) * g.S1 + (py[t] - lo[1]) * g.bz + (pz[t] - lo[2]);
                    return is_real ? spfm::gather_coop_lane<true, 0, int>(tile.data(), cell, g.S1, g.bz, w, wt, lane >> 3, lane & 7)
                                   : spfm::gather_coop_lane<false, 0, int>(tile.data(), cell, g.S1, g.bz, w, wt, lane >> 3, lane & 7);
                }
                const int qy = std::min(py[t], np - 8), qz = std::min(pz[t], np - 8);
                const long long cell = ((long long)px[t] * np + qy) * sz + qz;
                return is_real ? spfm::gather_coop_lane<true, 0, long long>(grid, cell, np * sz, sz, w, wt, lane >> 3, lane & 7)
                               : spfm::gather_coop_lane<false, 0, long long>(grid, cell, np * sz, sz, w, wt, lane >> 3, lane & 7);
            };
            // warp by warp, points in groups of MR8, exactly as coop_sweep (spf_slice.cu) walks them
            for (int wv = 0; wv < PATCH / 32; ++wv)
                for (int g0 = 0; g0 < 32; g0 += spfm::MR8) {
                    float pr[32][spfm::MR8], pi[32][spfm::MR8];
                    for (int u = 0; u < spfm::MR8; ++u) {
                        const int t = wv * 32 + g0 + u;
                        for (int lane = 0; lane < 32; ++lane) {
                            spfm::c2 c; c.x = c.y = 0.0f;
                            if (jj[t] >= 0) c = lane_part(t, lane);
                            pr[lane][u] = c.x; pi[lane][u] = c.y;
                        }
                    }
                    for (int o = 16, n = spfm::MR8 / 2; n >= 1; o >>= 1, n >>= 1) {      // exchange steps: all lanes read, then all write
                        float nr[32][spfm::MR8], ni[32][spfm::MR8];
                        for (int lane = 0; lane < 32; ++lane) {
                            const bool upper = (lane & o) != 0, pupper = ((lane ^ o) & o) != 0;
                            for (int v = 0; v < n; ++v) {
                                const float keep_r = upper ? pr[lane][v + n] : pr[lane][v], keep_i = upper ? pi[lane][v + n] : pi[lane][v];
                                const float recv_r = pupper ? pr[lane ^ o][v] : pr[lane ^ o][v + n], recv_i = pupper ? pi[lane ^ o][v] : pi[lane ^ o][v + n];
                                nr[lane][v] = keep_r + recv_r; ni[lane][v] = keep_i + recv_i;
                            }
                        }
                        for (int lane = 0; lane < 32; ++lane)
                            for (int v = 0; v < n; ++v) { pr[lane][v] = nr[lane][v]; pi[lane][v] = ni[lane][v]; }
                    }
                    for (int o = 2; o >= 1; o >>= 1) {
                        float nr[32], ni[32];
                        for (int lane = 0; lane < 32; ++lane) { nr[lane] = pr[lane][0] + pr[lane ^ o][0]; ni[lane] = pi[lane][0] + pi[lane ^ o][0]; }
                        for (int lane = 0; lane < 32; ++lane) { pr[lane][0] = nr[lane]; pi[lane][0] = ni[lane]; }
                    }
                    for (int u = 0; u < spfm::MR8; ++u) {         // owner lane g0 + u fetches from mr8_result_lane(u)
                        const int t = wv * 32 + g0 + u;
                        res[t].x = pr[spfm::mr8_result_lane(u)][0]; res[t].y = pi[spfm::mr8_result_lane(u)][0];
                    }
                }
        }
        for (int t = 0; t < PATCH; ++t)
            if (jj[t] >= 0) { out[2 * (m * P + jj[t])] = res[t].x; out[2 * (m * P + jj[t]) + 1] = res[t].y; }
    }
    stats[0] = n_staged; stats[1] = n_global; stats[2] = max_tile;
}

// the patch table spf_slice builds (spf_slice_math.cuh); returns the number of entries, fills out if it is large enough
long hostsim_patch_table(int panels, int rows, int cols, long P, int *out, long cap) {
    std::vector<int32_t> tab;
    spfm::build_patch_table(panels, rows, cols, P, tab);
    if ((long)tab.size() <= cap)
        for (size_t i = 0; i < tab.size(); ++i) out[i] = tab[i];
    return (long)tab.size();
}

// spf_prepare_model's two index kernels replayed with the header's maps: k_deapod_pad (model -> zeroed fine grid,
// complex64 interleaved) and k_relayout (fine grid after the FFT -> centred padded grid [np][np][sz], zeros in the
// z padding beyond np)
void hostsim_scatter_model(const float *A, const float *p32, int N, int nf, float *fine /*[nf^3][2], zeroed*/) {
    for (int i1 = 0; i1 < N; ++i1)
        for (int i2 = 0; i2 < N; ++i2)
            for (int i3 = 0; i3 < N; ++i3) {
                const size_t l = ((size_t)spfm::fine_index_of_voxel(i1, N, nf) * nf + spfm::fine_index_of_voxel(i2, N, nf)) * nf +
                                 spfm::fine_index_of_voxel(i3, N, nf);
                fine[2 * l] = spfm::deapodised(A[((size_t)i1 * N + i2) * N + i3], p32[i1], p32[i2], p32[i3]);
                fine[2 * l + 1] = 0.0f;
            }
}
void hostsim_relayout(const float *fine /*[nf^3][2]*/, int nf, int np, int sz, int off, float *gc /*[np][np][sz][2]*/) {
#pragma omp parallel for schedule(static)
    for (int px = 0; px < np; ++px)
        for (int py = 0; py < np; ++py)
            for (int pz = 0; pz < sz; ++pz) {
                const size_t o = ((size_t)px * np + py) * sz + pz;
                float re = 0.0f, im = 0.0f;
                if (pz < np) {
                    const size_t l = ((size_t)spfm::fine_index_of_padded(px, off, nf) * nf + spfm::fine_index_of_padded(py, off, nf)) * nf +
                                     spfm::fine_index_of_padded(pz, off, nf);
                    re = fine[2 * l]; im = fine[2 * l + 1];
                }
                gc[2 * o] = re; gc[2 * o + 1] = im;
            }
}

// k_check_even replayed: number of voxels that break A[n] == A[-n]
long hostsim_count_uneven(const float *A, int N) {
    long bad = 0;
    for (int i1 = 0; i1 < N; ++i1)
        for (int i2 = 0; i2 < N; ++i2)
            for (int i3 = 0; i3 < N; ++i3) bad += spfm::voxel_breaks_evenness(A, N, i1, i2, i3) ? 1 : 0;
    return bad;
}

// tile geometry alone, for the menu / capacity tests
void hostsim_tile_geom(int Lx, int Ly, int Lz, int w, int cell_bytes, unsigned cap, int *out4) {
    const spfm::TileGeom g = spfm::tile_geom(Lx, Ly, Lz, w, cell_bytes, cap);
    out4[0] = g.by; out4[1] = g.bz; out4[2] = g.S1; out4[3] = g.ok ? 1 : 0;
}

// cell index and fraction of one coordinate, for the index-range tests
void hostsim_cell(double x, int nf, int halo, int w, int *p, float *f) {
    const double kPi = 3.14159265358979323846;
    spfm::cell_and_fraction(x, (double)nf / (2.0 * kPi), 1.0 / (double)nf, nf, nf / 2 + halo, nf + 2 * halo, w, *p, *f);
}

}  // extern "C"
