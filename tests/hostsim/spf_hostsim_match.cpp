// tests/hostsim: the data path of spf_match replayed on the HOST from the very header the CUDA kernels
// include (paper_2109_05339_b200/csrc/spf_match_math.cuh).  TEST INFRASTRUCTURE ONLY: nothing in the
// product loads this library and it is not a CPU fallback.
//
// What is replayed, kernel by kernel (spf_match.cu):
//   k_common_vector       c = mean of up to 1,024 evenly spaced slices (the conditioning vector)
//   k_absmax / k_split    abs-max over unmasked pixels -> power-of-two rescale -> two fp16 planes per
//                         operand (raw images; slices minus c; zero in masked pixels and in the K padding),
//                         fp64-accumulated a_i = sum (I - c)^2 and b_m = sum S' (S' + 2 c)
//   k_match_gemm          persistent tile loop (tile_coords, cluster stride), per K block the TMA boxes
//                         of every CTA of the group written into a byte image of its shared-memory
//                         stage (128-byte swizzle, zero fill outside the tensor), the tcgen05.mma
//                         operand reads through SWIZZLE_128B descriptors with the +32-byte K advance,
//                         fp32 accumulation product by product in issue order, the epilogue's norm add
//                         and running argmin per TMEM lane, packed 64-bit keys merged with min
//   k_match_finalize      key -> (index, distance)
//   k_match_refine        the winner's distance recomputed as sum (I - S)^2
// What is NOT modelled: the tensor core's internal summation order inside one K = 16 instruction (here:
// sequential fp32), barriers, phases, timing.  So this checks index arithmetic, layouts, the operand
// split and the error budget -- not the hardware.
//
// Build: g++ -O2 -fopenmp -fPIC -shared -std=c++17 -ffp-contract=off spf_hostsim_match.cpp -o libspf_hostsim_match.so
#include <string.h>

#include <vector>

#include "../../paper_2109_05339_b200/csrc/spf_match_math.cuh"

namespace {

using namespace spfmm;

// cp.async.bulk.tensor.2d with CU_TENSOR_MAP_SWIZZLE_128B, box {BK, box_rows} of fp16 at element
// coordinates (c0, c1) of a [rows][Ppad] tensor: rows outside the tensor are zero-filled
void tma_load_2d(uint8_t *tile, const uint16_t *plane, long rows, long Ppad, int box_rows, long c0, long c1) {
    for (int r = 0; r < box_rows; ++r)
        for (int ch = 0; ch < 8; ++ch) {
            uint16_t v[8] = {0, 0, 0, 0, 0, 0, 0, 0};
            const long gr = c1 + r, gc = c0 + ch * 8;
            if (gr >= 0 && gr < rows)
                for (int k = 0; k < 8; ++k)
                    if (gc + k < Ppad) v[k] = plane[gr * Ppad + gc + k];
            memcpy(tile + sw128_offset((uint32_t)r, (uint32_t)ch), v, 16);
        }
}

// what tcgen05.mma reads for logical element (row, k) of a K-major SWIZZLE_128B operand whose
// descriptor start address is tile + start_off (start_off = 32 bytes per K = 16 step), SBO = 1024:
// linear address start + (row / 8) * 1024 + (row % 8) * 128 + 2 k, then address bits [4,7) ^= bits [7,10)
float umma_read(const uint8_t *tile, uint32_t start_off, int row, int k) {
    uint32_t a = start_off + (uint32_t)(row >> 3) * 1024u + (uint32_t)(row & 7) * 128u + (uint32_t)k * 2u;
    a ^= ((a >> 7) & 7u) << 4;
    uint16_t h;
    memcpy(&h, tile + a, 2);
    return f16_bits_to_f32(h);
}

float round_toward_zero(double x) {
    float f = (float)x;   // nearest
    if (fabs((double)f) > fabs(x)) f = nextafterf(f, 0.0f);
    return f;
}

struct Planes {
    std::vector<uint16_t> h;   // [2][rows][Ppad]
    std::vector<double> term;  // [rows]: a_i (images) or b_m (slices)
    int e = 0;
    bool two = false;
};

// k_common_vector: c[j] = mean over rows 0, step, 2 step, ... of the slices (fp32 sum in ascending row order),
// 0 in masked pixels and in the K padding; all zero when conditioning is off
std::vector<float> common_vector(const float *slices, long M, long P, long Ppad, const uint8_t *mask, bool condition) {
    std::vector<float> c((size_t)Ppad, 0.0f);
    if (!condition) return c;
    const long step = common_step(M);
    const float inv = 1.0f / (float)common_count(M);
    for (long j = 0; j < P; ++j) {
        if (mask && !mask[j]) continue;
        float sum = 0.0f;
        for (long m = 0; m < M; m += step) sum += slices[m * P + j];
        c[(size_t)j] = sum * inv;
    }
    return c;
}

// k_absmax + k_split.  which = 0: images (planes of the RAW values, term = a_i = sum (I - c)^2);
// which = 1: slices (planes of S' = fl(S - c), term = b_m = sum S' (S' + 2 c)).
Planes prepare(const float *x, long rows, long P, long Ppad, const uint8_t *mask, const std::vector<float> &c, int which) {
    Planes out;
    uint32_t mx = 0;   // k_absmax
    for (long r = 0; r < rows; ++r)
        for (long j = 0; j < P; ++j) {
            if (mask && !mask[j]) continue;
            const float val = which ? conditioned(x[r * P + j], c[(size_t)j]) : x[r * P + j];
            union { float f; uint32_t u; } v; v.f = fabsf(val);
            if (v.u > mx) mx = v.u;
        }
    out.e = scale_exponent(mx);
    const float sc = ldexpf(1.0f, out.e);
    out.h.assign((size_t)2 * rows * Ppad, 0);
    out.term.assign(rows, 0.0);
    for (long r = 0; r < rows; ++r) {   // k_split
        double acc = 0.0;
        for (long j = 0; j < Ppad; ++j) {
            float v = 0.0f;
            if (j < P && (!mask || mask[j])) {
                const float raw = x[r * P + j];
                if (which) { v = conditioned(raw, c[(size_t)j]); acc += slice_term(v, c[(size_t)j]); }
                else { v = raw; acc += image_term(raw, c[(size_t)j]); }
            }
            uint16_t a, b;
            out.two |= split_fp16(v, sc, a, b);
            out.h[(size_t)r * Ppad + j] = a;
            out.h[(size_t)(rows + r) * Ppad + j] = b;
        }
        out.term[r] = acc;
    }
    return out;
}

}  // namespace

extern "C" {

// fp16 conversion of the header's host path, for the pin against numpy.float16
void hostsim_f16_roundtrip(const float *x, long n, uint16_t *bits, float *back) {
    for (long i = 0; i < n; ++i) { bits[i] = f32_to_f16_bits(x[i]); back[i] = f16_bits_to_f32(bits[i]); }
}

int hostsim_chunk_kb(void) { return CHUNK_KB; }

void hostsim_tile_coords(int n_ib, int n_mb, int *ib, int *mb) {
    for (int t = 0; t < n_ib * n_mb; ++t) tile_coords(t, n_ib, n_mb, ib[t], mb[t]);
}

int hostsim_stage_layout(int cg, int ni, int *out /*[5]: stage_bytes, stages, off_a1, off_b0, off_b1*/) {
    out[0] = stage_bytes(cg, ni); out[1] = stages(cg, ni); out[2] = off_a(1); out[3] = off_b(cg, ni, 0); out[4] = off_b(cg, ni, 1);
    return out[0] * out[1] + SMEM_AUX + 1024;
}

// returns the number of products per K step (2 or 3); cta_group = 1 or 2; n_clusters = persistent clusters.
// acc_rz = 1 models a tensor core whose accumulator additions round toward zero (what the literature reports
// for earlier generations) instead of to nearest; chunk_kblocks = the kernel's CHUNK_KB (K blocks summed in
// TMEM before the epilogue warps add the chunk into their fp32 registers with round-to-nearest), 0 = whole K.
// condition = 1: the conditioned expansion (common vector subtracted from the slices), 0: c = 0 (the plain expansion).
// refine = 1: best_dist is recomputed in the difference form (k_match_refine), 0: the epilogue's own value is returned.
int hostsim_match(const float *images, long n_img, const float *slices, long M, long P, const uint8_t *mask, int cta_group,
                  int n_clusters, int acc_rz, int chunk_kblocks, int condition, int refine, int32_t *best_idx, float *best_dist) {
    const int CG = cta_group;
    const long Ppad = (P + BK - 1) / BK * BK;
    const std::vector<float> c = common_vector(slices, M, P, Ppad, mask, condition != 0);
    Planes I = prepare(images, n_img, P, Ppad, mask, c, 0), S = prepare(slices, M, P, Ppad, mask, c, 1);
    const int NI = I.two ? 2 : 1;
    const int kblocks = (int)(Ppad / BK);
    const int n_ib = (int)((n_img + TILE_ROWS * CG - 1) / (TILE_ROWS * CG)), n_mb = (int)((M + BN - 1) / BN);
    const int n_tiles = n_ib * n_mb;
    if (n_clusters > n_tiles) n_clusters = n_tiles;
    std::vector<unsigned long long> keys(n_img, ~0ull);
    const float neg2sc = cross_scale(I.e, S.e);
    const int ST = stages(CG, NI), SB = stage_bytes(CG, NI), BR = b_rows(CG);
    const uint16_t *I1 = I.h.data(), *I2 = I1 + (size_t)n_img * Ppad, *S1 = S.h.data(), *S2 = S1 + (size_t)M * Ppad;

#pragma omp parallel for schedule(dynamic, 1)
    for (int cluster = 0; cluster < n_clusters; ++cluster) {
        std::vector<uint8_t> smem[2];
        for (int r = 0; r < CG; ++r) smem[r].assign((size_t)ST * SB, 0xAB);   // poison: unwritten bytes must never be read
        std::vector<float> tmem((size_t)CG * TILE_ROWS * BN);                // [rank][lane][column] of one accumulator stage
        std::vector<float> regs((size_t)CG * TILE_ROWS * BN);                // the epilogue threads' running sums
        std::vector<float> Ar((size_t)CG * TILE_ROWS * 16), Br((size_t)BN * 16);
        int s = 0;
        for (int t = cluster; t < n_tiles; t += n_clusters) {
            int ib, mb;
            tile_coords(t, n_ib, n_mb, ib, mb);
            const int CH = chunk_kblocks > 0 ? chunk_kblocks : kblocks;
            for (size_t z = 0; z < regs.size(); ++z) regs[z] = 0.0f;
            for (int kb = 0; kb < kblocks; ++kb) {
                // ---- TMA producer of every CTA of the group
                for (int rank = 0; rank < CG; ++rank) {
                    uint8_t *st = smem[rank].data() + (size_t)s * SB;
                    const long rowA = (long)ib * (TILE_ROWS * CG) + (long)rank * TILE_ROWS, rowB = (long)mb * BN + (long)rank * BR;
                    const long kc = (long)kb * BK;
                    tma_load_2d(st, I1, n_img, Ppad, TILE_ROWS, kc, rowA);
                    if (NI == 2) tma_load_2d(st + off_a(1), I2, n_img, Ppad, TILE_ROWS, kc, rowA);
                    tma_load_2d(st + off_b(CG, NI, 0), S1, M, Ppad, BR, kc, rowB);
                    tma_load_2d(st + off_b(CG, NI, 1), S2, M, Ppad, BR, kc, rowB);
                }
                // ---- MMA issuer: per K = 16 step the products in issue order (A0.B0, A0.B1, A1.B0)
                for (int k4 = 0; k4 < BK / 16; ++k4) {
                    const uint32_t ko = (uint32_t)k4 * 32u;
                    const int prod_a[3] = {0, 0, 1}, prod_b[3] = {0, 1, 0};
                    for (int pr = 0; pr < (NI == 2 ? 3 : 2); ++pr) {
                        const bool accumulate = !(pr == 0 && kb % CH == 0 && k4 == 0);   // a chunk starts on a cleared accumulator
                        for (int row = 0; row < CG * TILE_ROWS; ++row) {   // UMMA M rows: CTA `rank` supplies rows rank*128..
                            const uint8_t *st = smem[row / TILE_ROWS].data() + (size_t)s * SB;
                            for (int k = 0; k < 16; ++k) Ar[(size_t)row * 16 + k] = umma_read(st + off_a(prod_a[pr]), ko, row % TILE_ROWS, k);
                        }
                        for (int n = 0; n < BN; ++n) {                      // UMMA N rows: CTA `rank` supplies rows rank*BR..
                            const uint8_t *st = smem[n / BR].data() + (size_t)s * SB;
                            for (int k = 0; k < 16; ++k) Br[(size_t)n * 16 + k] = umma_read(st + off_b(CG, NI, prod_b[pr]), ko, n % BR, k);
                        }
                        for (int row = 0; row < CG * TILE_ROWS; ++row) {
                            float *acc = tmem.data() + (size_t)row * BN;
                            const float *ar = Ar.data() + (size_t)row * 16;
                            for (int n = 0; n < BN; ++n) {
                                const float *br = Br.data() + (size_t)n * 16;
                                if (!acc_rz) {
                                    float p = 0.0f;
                                    for (int k = 0; k < 16; ++k) p += ar[k] * br[k];
                                    acc[n] = accumulate ? acc[n] + p : p;
                                } else {
                                    double p = accumulate ? (double)acc[n] : 0.0;   // exact 16-term sum, one truncation
                                    for (int k = 0; k < 16; ++k) p += (double)ar[k] * (double)br[k];
                                    acc[n] = round_toward_zero(p);
                                }
                            }
                        }
                    }
                }
                if (++s == ST) s = 0;
                if ((kb + 1) % CH == 0 || kb == kblocks - 1)      // epilogue warps: registers += chunk (fp32, round to nearest)
                    for (size_t z = 0; z < regs.size(); ++z) regs[z] += tmem[z];
            }
            // ---- epilogue of every CTA: TMEM lane = image row of the CTA's tile, columns = slices
            for (int rank = 0; rank < CG; ++rank)
                for (int lane = 0; lane < TILE_ROWS; ++lane) {
                    const long i = (long)ib * (TILE_ROWS * CG) + (long)rank * TILE_ROWS + lane;
                    const double aI = (i < n_img) ? I.term[i] : 0.0;
                    float best = INFINITY;
                    uint32_t bm = 0xffffffffu;
                    const long m0 = (long)mb * BN;
                    for (int c = 0; c < BN; ++c) {
                        if (m0 + c >= M) break;
                        const float d = distance(aI, S.term[m0 + c], neg2sc, regs[((size_t)rank * TILE_ROWS + lane) * BN + c]);
                        if (d < best) { best = d; bm = (uint32_t)(m0 + c); }
                    }
                    if (i < n_img && bm != 0xffffffffu) {
                        const unsigned long long key = pack_key(best, bm);
#pragma omp critical
                        if (key < keys[i]) keys[i] = key;
                    }
                }
        }
    }
    for (long i = 0; i < n_img; ++i) {   // k_match_finalize
        const unsigned long long k = keys[i];
        best_idx[i] = (int32_t)(uint32_t)(k & 0xffffffffull);
        union { uint32_t u; float f; } nan; nan.u = 0x7fc00000u;
        best_dist[i] = (k == ~0ull) ? nan.f : unorderable((uint32_t)(k >> 32));
        if (refine && k != ~0ull) {   // k_match_refine: the winner's distance in the difference form, fp64 sum, rounded once
            const float *Ir = images + i * P, *Sr = slices + (long)best_idx[i] * P;
            double acc = 0.0;
            for (long j = 0; j < P; ++j) {
                if (mask && !mask[j]) continue;
                const double t = (double)Ir[j] - (double)Sr[j];
                acc += t * t;
            }
            best_dist[i] = (float)acc;
        }
    }
    return NI == 2 ? 3 : 2;
}

}  // extern "C"
