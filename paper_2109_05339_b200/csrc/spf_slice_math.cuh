// Arithmetic of the type-2 NUFFT interpolation (steps a3-a5; PAPER.md:66-68,
// reading s10), written once for both compilers: nvcc uses these functions inside k_slice and
// spf_create; tests/hostsim compiles the very same header with g++ so the arithmetic can be checked
// against the oracle on a box without a GPU.  It is NOT a CPU fallback: nothing in the library's
// ABI reaches the host versions.
//
//   kernel        phi(z) = exp(beta (sqrt(1 - z^2) - 1)) on |z| <= 1,  beta = 2.30 w
//   point         xi = x n_f / (2 pi) folded into [-n_f/2, n_f/2],  i0 = ceil(xi - w/2),  f = i0 - xi
//   weights       phi_d[t] = phi(2 (f_d + t) / w),  t = 0..w-1
//   value         c = sum_{t1,t2,t3} b[i0 + t] phi_1[t1] phi_2[t2] phi_3[t3]
//   deapodisation p(n) = 2 / (w phihat(pi w n / n_f)),  phihat(xi) = 2 int_0^1 phi(z) cos(xi z) dz
#pragma once
#include <math.h>
#include <stddef.h>
#include <stdint.h>

#include <vector>

#if defined(__CUDACC__)
#define SPF_HD __host__ __device__ __forceinline__
#else
#define SPF_HD inline
#endif

#ifndef SPF_MAX_W
#define SPF_MAX_W 16
#endif
#define SPF_MAX_DEG 12

// Menu of TMA box sizes of the staged slicing kernels: {SPF_BOX_MIN, +SPF_BOX_STEP, ..., SPF_BOX_MAX}
// cells along z and along y, one x-plane deep; one tensor map per (by, bz) pair.
#define SPF_BOX_MIN 8
#define SPF_BOX_MAX 40
#define SPF_BOX_STEP 4
#define SPF_BOX_N ((SPF_BOX_MAX - SPF_BOX_MIN) / SPF_BOX_STEP + 1)  // 9

namespace spfm {

struct alignas(8) c2 { float x, y; };

// Index maps of spf_prepare_model (steps a1-a2), shared by the kernels and the CPU replay:
//   model voxel index i (0..N-1), n = i - floor(N/2)      ->  fine-grid index n mod n_f          (deapodise + pad)
//   padded index p of the centred grid with its periodic halo ->  fine-grid index (p - off) mod n_f (relayout),
//   off = n_f/2 + halo, so padded index p holds fine cell l = p - off, l in [-off, n_f/2 + halo)
SPF_HD int fine_index_of_voxel(int i, int N, int nf) {
    const int l = i - N / 2;
    return l < 0 ? l + nf : l;
}
SPF_HD int fine_index_of_padded(int p, int off, int nf) {
    const int l = (p - off) % nf;
    return l < 0 ? l + nf : l;
}
// Evenness test of the model (k_check_even): the voxel at -n has index 2 floor(N/2) - i; for even N the
// index-0 planes have no partner (the result is N) and must be exactly zero for the fine grid to be real.
SPF_HD int mirror_voxel(int i, int N) { return 2 * (N / 2) - i; }
SPF_HD bool voxel_breaks_evenness(const float *A, int N, int i1, int i2, int i3) {
    const int j1 = mirror_voxel(i1, N), j2 = mirror_voxel(i2, N), j3 = mirror_voxel(i3, N);
    const float a = A[((size_t)i1 * N + i2) * N + i3];
    if (j1 >= N || j2 >= N || j3 >= N) return a != 0.0f;
    return a != A[((size_t)j1 * N + j2) * N + j3];
}
// deapodised value of one voxel, in the kernel's operand order (fp32)
SPF_HD float deapodised(float a, float p1, float p2, float p3) { return a * (p1 * p2) * p3; }

// rotation matrix of the normalised quaternion, fp64 (reading s2: (w,x,y,z), Hamilton, active)
SPF_HD void quat_to_R(const float *q4, double *R) {
    double w = q4[0], x = q4[1], y = q4[2], z = q4[3];
    const double inv = 1.0 / sqrt(w * w + x * x + y * y + z * z);
    w *= inv; x *= inv; y *= inv; z *= inv;
    R[0] = 1.0 - 2.0 * (y * y + z * z); R[1] = 2.0 * (x * y - w * z);       R[2] = 2.0 * (x * z + w * y);
    R[3] = 2.0 * (x * y + w * z);       R[4] = 1.0 - 2.0 * (x * x + z * z); R[5] = 2.0 * (y * z - w * x);
    R[6] = 2.0 * (x * z - w * y);       R[7] = 2.0 * (y * z + w * x);       R[8] = 1.0 - 2.0 * (x * x + y * y);
}

// One axis: rotated coordinate (radians) -> first padded cell index p and fraction f = i0 - xi in
// [-w/2, -w/2 + 1).  `off` = n_f/2 + halo maps fine cell l to padded index l + off.  The result is
// clamped to [0, np - w] so that no input (NaN, inf) can index outside the padded grid; for finite
// input the clamp never acts (lowest index 2, highest n_f + 2).
SPF_HD void cell_and_fraction(double x, double xi_scale, double inv_nf, int nf, int off, int np, int w, int &p, float &f) {
    double xi = x * xi_scale;
    xi -= (double)nf * rint(xi * inv_nf);  // 2 pi-periodic: fold into [-n_f/2, n_f/2]
    const double c = ceil(xi - 0.5 * (double)w);
    double fr = c - xi;
    if (!(fr >= -0.5 * (double)w - 1.0 && fr <= 1.0)) fr = 0.0;   // NaN / inf input
    double pc = c + (double)off;
    if (!(pc >= 0.0)) pc = 0.0;
    if (pc > (double)(np - w)) pc = (double)(np - w);
    p = (int)pc;
    f = (float)fr;
}

// weights by the definition: exp(beta (sqrt(1-z^2) - 1)) written as exp(-beta z^2 / (1 + sqrt(1-z^2)))
template <int WMAX>
SPF_HD void weights_direct(float f, int w, float beta, float (&wt)[WMAX]) {
    const float s2w = 2.0f / (float)w;
#pragma unroll
    for (int t = 0; t < WMAX; ++t) {
        if (t < w) {
            const float z = (f + (float)t) * s2w;
            const float om = fmaxf(fmaf(-z, z, 1.0f), 0.0f);
            wt[t] = expf(-beta * z * z / (1.0f + sqrtf(om)));
        }
    }
}

// weights by per-tap polynomials in u = 2 (f + w/2) - 1 in [-1, 1) (Horner, FMA pipe only);
// coef[t][k] from fit_kernel_polys
template <int WMAX>
SPF_HD void weights_poly(float f, int w, const float (*coef)[SPF_MAX_DEG + 1], int deg, float (&wt)[WMAX]) {
    const float u = fmaf(2.0f, f, (float)w - 1.0f);
#pragma unroll
    for (int t = 0; t < WMAX; ++t) {
        if (t < w) {
            float p = coef[t][deg];
            for (int k = deg - 1; k >= 0; --k) p = fmaf(p, u, coef[t][k]);
            wt[t] = p;
        }
    }
}

// sum over the w^3 neighbours; `base` points at cell (i0x, i0y, i0z); sx, sy strides in cells
template <int WMAX, bool REAL>
SPF_HD c2 gather(const float *base, int sx, int sy, int w, const float (&wx)[WMAX], const float (&wy)[WMAX],
                 const float (&wz)[WMAX]) {
    float accr = 0.0f, acci = 0.0f;
    constexpr int E = REAL ? 1 : 2;
    // the outer tap loop is unrolled for the compile-time widths up to 8 (wx[] then stays in registers);
    // for wider or run-time widths it stays a loop and wx[] is indexed in local memory
#pragma unroll(WMAX <= 8 ? WMAX : 1)
    for (int t1 = 0; t1 < (WMAX <= 8 ? WMAX : w); ++t1) {
        if (WMAX <= 8 && t1 >= w) break;
        float pr = 0.0f, pi = 0.0f;
#pragma unroll
        for (int t2 = 0; t2 < WMAX; ++t2) {
            if (t2 < w) {
                const float *row = base + (size_t)(t1 * sx + t2 * sy) * E;
                float rr = 0.0f, ri = 0.0f;
#pragma unroll
                for (int t3 = 0; t3 < WMAX; ++t3) {
                    if (t3 < w) {
                        if (REAL) rr = fmaf(wz[t3], row[t3], rr);
                        else {
                            const c2 v = *reinterpret_cast<const c2 *>(row + 2 * t3);  // one 64-bit load
                            rr = fmaf(wz[t3], v.x, rr);
                            ri = fmaf(wz[t3], v.y, ri);
                        }
                    }
                }
                pr = fmaf(wy[t2], rr, pr);
                if (!REAL) pi = fmaf(wy[t2], ri, pi);
            }
        }
        accr = fmaf(wx[t1], pr, accr);
        if (!REAL) acci = fmaf(wx[t1], pi, acci);
    }
    c2 r; r.x = accr; r.y = acci;
    return r;
}

// ------------------------------------------------------------------------------------------
// shared-memory tile of the staged kernel (k_slice, slice_impl 2) and the cooperative gather
// ------------------------------------------------------------------------------------------
// A block's points touch the box [lo, hi + w) of padded cells; L = hi - lo + w per axis.  The box is
// staged one x-plane per TMA copy with a (by x bz)-cell box taken from a fixed menu (one tensor map
// per size), rows written densely (row pitch = bz cells), planes S1 cells apart (128-byte aligned).
// A warp's lanes read rows t2 = h, h + 4 (h = lane >> 3) and cells t3 = lane & 7 of every x-plane, i.e.
// an 8 x 8 window per point (w <= 8), so the box needs 8 - w spare rows and cells; bz is 8, 24 or 40
// (bz = 8 mod 16), which puts the four rows a warp reads at once (offsets 0, bz, 2 bz, 3 bz) into four
// disjoint groups of 8 banks: no conflicts.
struct TileGeom { int by, bz, S1; bool ok; };
SPF_HD TileGeom tile_geom(int Lx, int Ly, int Lz, int w, int cell_bytes, uint32_t cap_bytes) {
    TileGeom g;
    const int ey = Ly + 8 - w, ez = Lz + 8 - w;
    g.by = (ey + SPF_BOX_STEP - 1) / SPF_BOX_STEP * SPF_BOX_STEP;
    if (g.by < SPF_BOX_MIN) g.by = SPF_BOX_MIN;
    g.bz = ez <= 8 ? 8 : (ez <= 24 ? 24 : 40);
    const int per128 = 128 / cell_bytes;
    g.S1 = (g.by * g.bz + per128 - 1) / per128 * per128;
    g.ok = w <= 8 && Lx > 0 && g.by <= SPF_BOX_MAX && g.bz <= SPF_BOX_MAX && ez <= SPF_BOX_MAX &&
           (uint64_t)Lx * (uint64_t)g.S1 * (uint64_t)cell_bytes <= (uint64_t)cap_bytes;
    return g;
}
SPF_HD int tile_map_index(int by, int bz) { return ((by - SPF_BOX_MIN) / SPF_BOX_STEP) * SPF_BOX_N + (bz - SPF_BOX_MIN) / SPF_BOX_STEP; }

// One point's 3 w weights as the cooperative gather reads them (SPF_COOP_STRIDE floats per point; the
// stride of 28 keeps the owners' 16-byte stores and the warp's loads free of bank conflicts):
//   [0,8)   wz[0..7]                       (0 beyond w)
//   [8,16)  wy[0],wy[4],wy[1],wy[5],wy[2],wy[6],wy[3],wy[7]   (pairs read as one 8-byte load)
//   [16,24) wx[0..7]
#define SPF_COOP_STRIDE 28
template <int WMAX>
SPF_HD void coop_pack_weights(float (&out)[24], int w, const float (&wx)[WMAX], const float (&wy)[WMAX], const float (&wz)[WMAX]) {
#pragma unroll
    for (int t = 0; t < 8; ++t) {
        float vx = 0.0f, vy = 0.0f, vz = 0.0f;
        if (t < WMAX) {
            if (t < w) { vx = wx[t < WMAX ? t : 0]; vy = wy[t < WMAX ? t : 0]; vz = wz[t < WMAX ? t : 0]; }
        }
        out[t] = vz;
        out[8 + 2 * (t & 3) + (t >> 2)] = vy;
        out[16 + t] = vx;
    }
}

// Partial sum of lane (h, k) for one point: tile = staged box, cell = the point's first cell inside the
// box (x-plane pitch S1, row pitch bz), wts = the point's weights as stored above.
//   sum_t1 wx[t1] (wy[h] wz[k] b[t1][h][k] + wy[h+4] wz[k] b[t1][h+4][k])
// BZ > 0 fixes the row pitch at compile time (the row offsets become immediates); BZ = 0 uses bz.
// IDX: int for a shared-memory tile, long long when `tile` is the whole padded grid in global memory.
template <bool REAL, int BZ, typename IDX = int>
SPF_HD c2 gather_coop_lane(const float *tile, IDX cell, int S1, int bz, int w, const float *wts, int h, int k) {
    constexpr int E = REAL ? 1 : 2;
    const int rp = BZ ? BZ : bz;
    const float wzk = wts[k];
    const float cA = wts[8 + 2 * h] * wzk, cB = wts[9 + 2 * h] * wzk;
    const float *p0 = tile + (size_t)(cell + (IDX)(h * rp + k)) * E;
    const size_t row4 = (size_t)(4 * rp) * E, plane = (size_t)S1 * E;
    float ar = 0.0f, ai = 0.0f, br = 0.0f, bi = 0.0f;
#pragma unroll 8
    for (int t1 = 0; t1 < w; ++t1) {
        const float wxt = wts[16 + t1];
        if (REAL) {
            ar = fmaf(wxt, p0[0], ar);
            br = fmaf(wxt, p0[row4], br);
        } else {
            const c2 v0 = *reinterpret_cast<const c2 *>(p0), v1 = *reinterpret_cast<const c2 *>(p0 + row4);
            ar = fmaf(wxt, v0.x, ar); ai = fmaf(wxt, v0.y, ai);
            br = fmaf(wxt, v1.x, br); bi = fmaf(wxt, v1.y, bi);
        }
        p0 += plane;
    }
    c2 r;
    r.x = fmaf(cA, ar, cB * br);
    r.y = REAL ? 0.0f : fmaf(cA, ai, cB * bi);
    return r;
}

// The warp-per-point gather for 8 < w <= 16 (variant 3 at w = 10, Slicing-heavy): the window is 16 cells wide
// (lanes with k >= w stay idle and load nothing), so a warp covers 2 rows per load and needs ceil(w / 2) loads
// per x-plane: rows h, h + 2, h + 4, ...  Weight layout per point (SPF_COOPW_STRIDE floats; 44 = 12 mod 32 keeps
// the owners' 16-byte stores conflict-free):
//   [0,16)  wz[0..15]            [16,32) wy[h + 2 i] at 16 + 8 h + i  (h = 0, 1; i = 0..7)            [32,48) wx[0..15]
// only the first 44 are stored (wx[12..15] are never read: w <= 12 for this layout; w = 10 is what is built).
#define SPF_COOPW_STRIDE 44
template <int WMAX>
SPF_HD void coop_pack_weights_wide(float (&out)[44], int w, const float (&wx)[WMAX], const float (&wy)[WMAX], const float (&wz)[WMAX]) {
#pragma unroll
    for (int v = 0; v < 44; ++v) out[v] = 0.0f;
#pragma unroll
    for (int t = 0; t < 12; ++t) {
        if (t < WMAX) {
            if (t < w) {
                out[t] = wz[t < WMAX ? t : 0];
                out[16 + 8 * (t & 1) + (t >> 1)] = wy[t < WMAX ? t : 0];
                out[32 + t] = wx[t < WMAX ? t : 0];
            }
        }
    }
}

// lane = (h, k), h = lane >> 4 in {0, 1}, k = lane & 15; NPASS = ceil(w / 2) <= 6 loads per x-plane
template <bool REAL, typename IDX>
SPF_HD c2 gather_coop_lane_wide(const float *grid, IDX cell, int S1, int rp, int w, const float *wts, int lane) {
    constexpr int E = REAL ? 1 : 2;
    constexpr int MAXPASS = 6;
    c2 r; r.x = r.y = 0.0f;
    const int h = lane >> 4, k = lane & 15;
    if (k >= w) return r;
    const int npass = (w + 1) >> 1;
    const float *p0 = grid + (size_t)(cell + (IDX)(h * rp + k)) * E;
    const size_t row2 = (size_t)(2 * rp) * E, plane = (size_t)S1 * E;
    float ar[MAXPASS], ai[MAXPASS];
#pragma unroll
    for (int i = 0; i < MAXPASS; ++i) ar[i] = ai[i] = 0.0f;
    for (int t1 = 0; t1 < w; ++t1) {
        const float wxt = wts[32 + t1];
#pragma unroll
        for (int i = 0; i < MAXPASS; ++i) {
            if (i < npass && h + 2 * i < w) {
                if (REAL) ar[i] = fmaf(wxt, p0[i * row2], ar[i]);
                else {
                    const c2 v = *reinterpret_cast<const c2 *>(p0 + i * row2);
                    ar[i] = fmaf(wxt, v.x, ar[i]); ai[i] = fmaf(wxt, v.y, ai[i]);
                }
            }
        }
        p0 += plane;
    }
    float sr = 0.0f, si = 0.0f;
#pragma unroll
    for (int i = 0; i < MAXPASS; ++i) {
        if (i < npass) {
            const float wyi = wts[16 + 8 * h + i];
            sr = fmaf(wyi, ar[i], sr); si = fmaf(wyi, ai[i], si);
        }
    }
    r.x = wts[k] * sr;
    r.y = REAL ? 0.0f : wts[k] * si;
    return r;
}

// Multi-value warp reduction used by the cooperative gather: every lane holds MR8 = 8 partial sums (one
// per point of a group).  Exchange step with lane offset o = 16, 8, 4 and n = 4, 2, 1 values: a lane whose
// bit o is set keeps values [n, 2n) and sends [0, n), the others the opposite, and adds what it receives;
// after the three steps a lane holds ONE value, the partial sum of point u = 4 bit4 + 2 bit3 + bit2 of
// its lane number over 4 lanes' worth of partials; two plain butterfly steps (o = 2, 1) finish the sum.
// 9 exchanges for 8 points instead of 40.
constexpr int MR8 = 8;
SPF_HD int mr8_result_lane(int u) { return u << 2; }   // a lane that ends with point u's total (bits 1,0 are free)

// ------------------------------------------------------------------------------------------
// host side (fp64): kernel, polynomial fit of the weights, deapodisation factors
// ------------------------------------------------------------------------------------------
// pixel -> patch table of spf_slice: SPF_PATCH_PIXELS pixels per thread block.  Under a detector layout promise
// (panels x rows x cols == P) a patch is an 8 x 16 lattice tile of one panel (ragged tiles at the panel edges
// are padded with -1); otherwise patches are runs of consecutive pixels.  Every pixel appears exactly once.
#define SPF_PATCH_PIXELS 128
inline void build_patch_table(int panels, int rows, int cols, int64_t P, std::vector<int32_t> &tab) {
    tab.clear();
    const bool lattice = panels > 0 && rows > 0 && cols > 0 && (int64_t)panels * rows * cols == P;
    if (lattice) {
        const int TR = 8, TC = SPF_PATCH_PIXELS / TR;
        for (int p = 0; p < panels; ++p)
            for (int r0 = 0; r0 < rows; r0 += TR)
                for (int c0 = 0; c0 < cols; c0 += TC)
                    for (int t = 0; t < SPF_PATCH_PIXELS; ++t) {
                        const int r = r0 + t / TC, c = c0 + t % TC;
                        tab.push_back((r < rows && c < cols) ? (int32_t)(((int64_t)p * rows + r) * cols + c) : -1);
                    }
    } else {
        const int64_t n = (P + SPF_PATCH_PIXELS - 1) / SPF_PATCH_PIXELS;
        tab.resize((size_t)n * SPF_PATCH_PIXELS);
        for (int64_t i = 0; i < n * SPF_PATCH_PIXELS; ++i) tab[(size_t)i] = i < P ? (int32_t)i : -1;
    }
}

inline double es_phi(double z, double beta) { return fabs(z) <= 1.0 ? exp(beta * (sqrt(1.0 - z * z) - 1.0)) : 0.0; }

// Per-tap Chebyshev interpolants of phi on the fraction interval, converted to monomials in u.
// Returns the degree used: the lowest in [6, SPF_MAX_DEG] whose worst error over all taps is < 1e-7.
inline int fit_kernel_polys(int w, double beta, float coef[SPF_MAX_W][SPF_MAX_DEG + 1], double *worst_out = nullptr) {
    const double kPi = 3.14159265358979323846;
    for (int deg = 6; deg <= SPF_MAX_DEG; ++deg) {
        const int n = deg + 1;
        double worst = 0.0;
        std::vector<std::vector<double>> mono(w, std::vector<double>(n, 0.0));
        for (int t = 0; t < w; ++t) {
            auto g = [&](double u) { return es_phi(((u + 1.0) * 0.5 - 0.5 * w + t) * 2.0 / w, beta); };
            std::vector<double> cheb(n, 0.0);
            for (int jn = 0; jn < n; ++jn) {
                double s = 0.0;
                for (int k = 0; k < n; ++k) {
                    const double th = kPi * (k + 0.5) / n;
                    s += g(cos(th)) * cos(jn * th);
                }
                cheb[jn] = s * (jn == 0 ? 1.0 : 2.0) / n;
            }
            // Chebyshev -> monomial: T0 = 1, T1 = u, T_{k+1} = 2 u T_k - T_{k-1}
            std::vector<double> Tkm1(n, 0.0), Tk(n, 0.0), Tn(n, 0.0);
            Tkm1[0] = 1.0;
            for (int i = 0; i < n; ++i) mono[t][i] += cheb[0] * Tkm1[i];
            if (n > 1) {
                Tk[1] = 1.0;
                for (int i = 0; i < n; ++i) mono[t][i] += cheb[1] * Tk[i];
            }
            for (int k = 2; k < n; ++k) {
                for (int i = 0; i < n; ++i) Tn[i] = (i ? 2.0 * Tk[i - 1] : 0.0) - Tkm1[i];
                for (int i = 0; i < n; ++i) mono[t][i] += cheb[k] * Tn[i];
                Tkm1 = Tk; Tk = Tn;
            }
            for (int s = 0; s < 400; ++s) {
                const double u = -1.0 + 2.0 * (s + 0.5) / 400.0;
                double p = mono[t][n - 1];
                for (int k = n - 2; k >= 0; --k) p = p * u + mono[t][k];
                worst = fmax(worst, fabs(p - g(u)));
            }
        }
        if (worst < 1e-7 || deg == SPF_MAX_DEG) {
            for (int t = 0; t < w; ++t)
                for (int k = 0; k <= SPF_MAX_DEG; ++k) coef[t][k] = k < n ? (float)mono[t][k] : 0.0f;
            if (worst_out) *worst_out = worst;
            return deg;
        }
    }
    return SPF_MAX_DEG;
}

inline void gauss_legendre(int n, std::vector<double> &x, std::vector<double> &wgt) {
    const double kPi = 3.14159265358979323846;
    x.resize(n); wgt.resize(n);
    for (int i = 0; i < (n + 1) / 2; ++i) {
        double z = cos(kPi * (i + 0.75) / (n + 0.5)), pp = 0.0;
        for (int it = 0; it < 100; ++it) {
            double p1 = 1.0, p2 = 0.0;
            for (int j = 0; j < n; ++j) { double p3 = p2; p2 = p1; p1 = ((2.0 * j + 1.0) * z * p2 - j * p3) / (j + 1.0); }
            pp = n * (z * p1 - p2) / (z * z - 1.0);
            double dz = p1 / pp;
            z -= dz;
            if (fabs(dz) < 1e-16) break;
        }
        x[i] = -z; x[n - 1 - i] = z;
        wgt[i] = wgt[n - 1 - i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
}

// phihat(xi) = 2 int_0^1 exp(beta (sqrt(1-z^2) - 1)) cos(xi z) dz; with z = sin(theta) the integrand is analytic:
//            = 2 int_0^{pi/2} exp(beta (cos(theta) - 1)) cos(xi sin(theta)) cos(theta) dtheta
inline double es_kernel_ft(double xi, double beta, const std::vector<double> &gx, const std::vector<double> &gw) {
    const double kPi = 3.14159265358979323846;
    double s = 0.0;
    for (size_t k = 0; k < gx.size(); ++k) {
        double th = 0.25 * kPi * (gx[k] + 1.0);
        s += gw[k] * exp(beta * (cos(th) - 1.0)) * cos(xi * sin(th)) * cos(th);
    }
    return 2.0 * s * 0.25 * kPi;
}

// p(n) for n = i - floor(N/2), i = 0..N-1
inline void deapodisation_factors(int N, int nf, int w, double beta, std::vector<double> &out) {
    const double kPi = 3.14159265358979323846;
    std::vector<double> gx, gw;
    gauss_legendre(96, gx, gw);
    out.resize(N);
    const double alpha = kPi * w / nf;
    for (int i = 0; i < N; ++i) out[i] = 2.0 / (w * es_kernel_ft(alpha * (double)(i - N / 2), beta, gx, gw));
}

}  // namespace spfm
