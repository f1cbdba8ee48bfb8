// Arithmetic and index logic of spf_match (steps a6-a8), written
// once for both compilers: nvcc uses these functions inside k_absmax / k_split / k_match_gemm,
// tests/hostsim compiles the very same header with g++ and replays the kernels' data path on the CPU
// (operand split, shared-memory tile images as TMA writes them, descriptor-addressed UMMA reads, fp32
// accumulation, norm add, packed argmin keys) against the oracle.  It is NOT a CPU fallback: nothing
// in the library's ABI reaches the host versions.
//
// Conditioned expansion (SURVEY.md section 7 "Split precision vs cancellation").  With one
// common vector c (the mean of up to 1,024 evenly spaced slices; any c gives the same d in exact arithmetic) and
// S'_m = fl(S_m - c):
//   d[i][m] = sum_j (I_ij - S_mj)^2 = sum_j ((I_ij - c_j) - S'_mj)^2 = a_i + b_m - 2 G_im
//   a_i  = sum_j (I_ij - c_j)^2                 per image, fp64
//   b_m  = sum_j S'_mj (S'_mj + 2 c_j)          per slice, fp64   ( = ||S'||^2 + 2 c . S' )
//   G_im = sum_j I_ij S'_mj                     the contraction (tensor cores); the images stay RAW, so photon
//                                               counts remain exact in one fp16 plane
// Everything the slices have in common (the radial fall-off of a diffraction pattern) is gone from G, so the
// terms that cancel are the size of ||I - c||^2 + ||S'||^2, not of ||I||^2 + ||S||^2, and the accumulator's
// rounding acts on a signed sum instead of a monotone one.  a_i + b_m - 2 G is added in fp64 (once per pair per
// tile: free), and the winner's distance is recomputed in the difference form (k_match_refine) so that best_dist
// never carries the expansion's cancellation error.
//   I_i . S'_m = 2^-(eI+eS) (I1 + I2) . (S1 + S2)
//   x 2^e = h1 + h2 + r,  h1 = fp16(x 2^e), h2 = fp16(x 2^e - h1), |r| <= 2^-22 |x 2^e| (or 2^-25 absolute)
//   products kept: I1.S1 + I1.S2 (+ I2.S1 when some image value is not exact in one fp16 term)
#pragma once
#include <math.h>
#include <stdint.h>

#if defined(__CUDACC__)
#include <cuda_fp16.h>
#define SPF_MHD __host__ __device__ __forceinline__
#else
#define SPF_MHD inline
#endif

namespace spfmm {

constexpr int BK = 64;          // fp16 elements per K block: 128 bytes, one swizzle row
constexpr int BN = 256;         // slices per tile (UMMA N)
constexpr int TILE_ROWS = 128;  // image rows per CTA (UMMA M = 128 * CG)
constexpr int TILE_GROUP = 8;   // image blocks whose tiles are scheduled together (L2 reuse of slice rows)
// K blocks summed inside the tensor core's accumulator (TMEM) before the epilogue warps add that chunk
// to their own fp32 registers with round-to-nearest FADDs (run-time option "match_chunk_kblocks"; this is its
// default, 0 = the whole of K in TMEM).  Tensor-core accumulators have been measured to round toward zero on
// earlier generations; whether sm_100a's do is not known yet (no hardware run), so the default is chosen from
// the CPU replay under BOTH roundings (tests/test_hostsim_match.py, Paper-scale statistics, P = 65,536, worst
// relative error of any winning distance before k_match_refine):
//   truncating accumulator, conditioned:  whole K 1.9e-4 | 64 blocks 1.8e-5 | 4 blocks 1.6e-6
//   truncating accumulator, plain:        whole K 3.7e-4 | 64 blocks 3.2e-5 | 4 blocks 6.1e-6
//   round to nearest (either form):       <= 5e-6 at any chunk size
// 32 blocks (2,048 pixels) keeps the truncating case an order of magnitude inside the 1e-4 bar and drains the
// 128 x 256 accumulator 32 times per tile at P = 65,536 (it was 256 times at the round-1 value of 4): one drain
// (128 KB of TMEM reads) per 32,768 tensor-pipe cycles, hidden behind the other accumulator stage.
constexpr int CHUNK_KB = 32;
constexpr int COMMON_ROWS = 1024;   // slices averaged into the common vector c (evenly spaced over M)

// ---------------------------------------------------------------- shared-memory stage layout
// One pipeline stage of CTA `rank` of a CG-CTA group holds, in this order: NI image tiles
// (TILE_ROWS x BK fp16 each: plane 1, then plane 2 when NI == 2), then the two slice tiles
// (BN / CG rows x BK fp16 each: plane 1, plane 2).  Every tile is a multiple of 1024 bytes.
constexpr int A_TILE_BYTES = TILE_ROWS * BK * 2;   // 16 KB
constexpr int SMEM_AUX = 1024;                     // barriers + tmem pointer + abort word
constexpr int SMEM_BUDGET = 227 * 1024;
constexpr int b_rows(int cg) { return BN / cg; }
constexpr int b_tile_bytes(int cg) { return b_rows(cg) * BK * 2; }
constexpr int stage_bytes(int cg, int ni) { return ni * A_TILE_BYTES + 2 * b_tile_bytes(cg); }
constexpr int stages(int cg, int ni) {
    return (SMEM_BUDGET - SMEM_AUX - 1024) / stage_bytes(cg, ni) > 6 ? 6 : (SMEM_BUDGET - SMEM_AUX - 1024) / stage_bytes(cg, ni);
}
constexpr int off_a(int plane) { return plane * A_TILE_BYTES; }                                   // plane 0 or 1
constexpr int off_b(int cg, int ni, int plane) { return ni * A_TILE_BYTES + plane * b_tile_bytes(cg); }

// ---------------------------------------------------------------- fp16 conversion
// round-to-nearest-even fp32 -> fp16 bits and back.  The device uses the hardware conversion; the
// host version is plain integer arithmetic (tests pin it to numpy.float16).
SPF_MHD uint16_t f32_to_f16_bits(float x) {
#if defined(__CUDA_ARCH__)
    return __half_as_ushort(__float2half_rn(x));
#else
    union { float f; uint32_t u; } v; v.f = x;
    const uint32_t sign = (v.u >> 16) & 0x8000u;
    const uint32_t absu = v.u & 0x7fffffffu;
    if (absu >= 0x7f800000u) return (uint16_t)(sign | (absu > 0x7f800000u ? 0x7e00u : 0x7c00u));  // NaN / inf
    if (absu >= 0x477ff000u) return (uint16_t)(sign | 0x7c00u);                                   // rounds to inf (>= 65520)
    if (absu < 0x33000001u) return (uint16_t)sign;                                                // <= 2^-25: rounds to 0
    int e = (int)(absu >> 23) - 127;
    uint32_t man = (absu & 0x7fffffu) | 0x800000u;   // 24-bit significand
    int shift;                                       // bits dropped from the significand
    uint32_t base;
    if (e >= -14) { shift = 13; base = (uint32_t)(e + 15) << 10; }
    else { shift = 13 + (-14 - e); base = 0; }       // subnormal result
    uint32_t kept = man >> shift;
    const uint32_t rem = man & ((1u << shift) - 1u), half = 1u << (shift - 1);
    if (rem > half || (rem == half && (kept & 1u))) kept++;
    // normal: kept has the implicit bit at position 10; adding base - (1 << 10) + kept lets a carry roll into the exponent
    return (uint16_t)(sign | (e >= -14 ? (base + kept - 0x400u) : kept));
#endif
}

SPF_MHD float f16_bits_to_f32(uint16_t h) {
#if defined(__CUDA_ARCH__)
    return __half2float(__ushort_as_half(h));
#else
    const uint32_t sign = (uint32_t)(h & 0x8000u) << 16;
    const uint32_t e = (h >> 10) & 0x1fu, m = h & 0x3ffu;
    union { float f; uint32_t u; } v;
    if (e == 0) {
        if (m == 0) { v.u = sign; return v.f; }
        const float sub = (float)m * 5.9604644775390625e-8f;   // m * 2^-24, exact
        return sign ? -sub : sub;
    }
    if (e == 31) { v.u = sign | 0x7f800000u | (m << 13); return v.f; }
    v.u = sign | ((e + 112u) << 23) | (m << 13);
    return v.f;
#endif
}

// ---------------------------------------------------------------- a6: rescale and split
// exponent e with 2^e * max|x| in [2^14, 2^15): fp16 holds it with 11 significant bits and the
// products stay far from overflow.  absmax_bits = bit pattern of max |x| (a non-negative float).
SPF_MHD int scale_exponent(uint32_t absmax_bits) {
    union { uint32_t u; float f; } v; v.u = absmax_bits;
    const float mx = v.f;
    if (!(mx > 0.0f) || isinf(mx) || isnan(mx)) return 0;
    int k;
    frexpf(mx, &k);  // mx = f * 2^k, f in [0.5, 1)
    int e = 15 - k;
    if (e < -100) e = -100;
    if (e > 100) e = 100;
    return e;
}

// x * sc = h1 + h2 (+ residual below fp16 resolution); returns true when h2 != 0 is needed (residual non-zero)
SPF_MHD bool split_fp16(float x, float sc, uint16_t &h1, uint16_t &h2) {
    const float vs = x * sc;
    h1 = f32_to_f16_bits(vs);
    const float r = vs - f16_bits_to_f32(h1);
    h2 = f32_to_f16_bits(r);
    return r != 0.0f;
}

// ---------------------------------------------------------------- a6: conditioning
// rows of the slice array averaged into c: m = 0, step, 2 step, ... (at most COMMON_ROWS of them)
SPF_MHD long common_step(long M) { return M <= COMMON_ROWS ? 1 : (M + COMMON_ROWS - 1) / COMMON_ROWS; }
SPF_MHD long common_count(long M) { const long st = common_step(M); return (M + st - 1) / st; }
// the conditioned slice value S' = fl(S - c), one fp32 subtraction; everything downstream (planes, b_m) uses S'
SPF_MHD float conditioned(float s, float c) { return s - c; }
// per-pixel terms of a_i and b_m (fp64)
SPF_MHD double image_term(float x, float c) { const double t = (double)x - (double)c; return t * t; }
SPF_MHD double slice_term(float sp, float c) { return (double)sp * ((double)sp + 2.0 * (double)c); }

// ---------------------------------------------------------------- a8: epilogue
// factor that undoes both rescales and carries the -2 of the cross term
SPF_MHD float cross_scale(int eI, int eS) { return ldexpf(-2.0f, -(eI + eS)); }

// d = a_i + b_m - 2 G in fp64, rounded once; neg2sc * acc is exact in fp32 (a power-of-two scaling)
SPF_MHD float distance(double aI, double bS, float neg2sc, float acc) { return (float)(aI + bS + (double)(neg2sc * acc)); }

// fp32 -> uint32 that orders like the float (negative values below positive ones)
SPF_MHD uint32_t orderable(float d) {
    union { float f; uint32_t u; } v; v.f = d;
    return (v.u & 0x80000000u) ? ~v.u : (v.u | 0x80000000u);
}
SPF_MHD float unorderable(uint32_t u) {
    union { uint32_t u; float f; } v;
    v.u = (u & 0x80000000u) ? (u & 0x7fffffffu) : ~u;
    return v.f;
}
// running-argmin key: smaller distance wins, then the lower orientation index
SPF_MHD unsigned long long pack_key(float d, uint32_t m) { return ((unsigned long long)orderable(d) << 32) | m; }

// ---------------------------------------------------------------- tile schedule
// tile t -> (image block ib, slice block mb): groups of TILE_GROUP image blocks, within a group the
// image block runs fastest, so tiles running at the same time share slice rows in L2.
SPF_MHD void tile_coords(int t, int n_ib, int n_mb, int &ib, int &mb) {
    const int per_group = TILE_GROUP * n_mb;
    const int g = t / per_group, r = t - g * per_group;
    const int left = n_ib - g * TILE_GROUP;
    const int gsz = left < TILE_GROUP ? left : TILE_GROUP;
    ib = g * TILE_GROUP + r % gsz;
    mb = r / gsz;
}

// ---------------------------------------------------------------- shared-memory operand tiles
// Byte offset, inside a 1024-byte-aligned K-major tile of 128-byte rows, of the 16-byte chunk
// `chunk` (0..7) of row `row` under the 128-byte swizzle: the chunk index is XORed with row mod 8.
// This is where TMA (CU_TENSOR_MAP_SWIZZLE_128B) writes it and where tcgen05.mma, given a
// SWIZZLE_128B descriptor with stride-byte-offset 1024, reads it.
SPF_MHD uint32_t sw128_offset(uint32_t row, uint32_t chunk) { return row * 128u + ((chunk ^ (row & 7u)) << 4); }

}  // namespace spfmm
