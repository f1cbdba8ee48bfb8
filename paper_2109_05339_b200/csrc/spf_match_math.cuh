// Arithmetic and index logic of spf_match (steps a6-a8), written
// once for both compilers: nvcc uses these functions inside k_absmax / k_split / k_match_gemm,
// tests/hostsim compiles the very same header with g++ and replays the kernels' data path on the CPU
// (operand split, shared-memory tile images as TMA writes them, descriptor-addressed UMMA reads, fp32
// accumulation, norm add, packed argmin keys) against the oracle.  It is NOT a CPU fallback: nothing
// in the library's ABI reaches the host versions.
//
//   d[i][m] = ||I_i||^2 + ||S_m||^2 - 2 I_i . S_m,   I_i . S_m = 2^-(eI+eS) (I1 + I2) . (S1 + S2)
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
// to their own fp32 registers with round-to-nearest FADDs.  Tensor-core accumulators have been measured
// to round toward zero on earlier generations; over K = 65,536 that is a bias of ~1e-4 of the cross
// term, i.e. up to 1e-3 of the distance (tests/test_hostsim_match.py reproduces it), ten times the parity
// bar.  With chunks of 4 x 64 the bias stays below 2e-5 of the distance under either rounding.
constexpr int CHUNK_KB = 4;

// ---------------------------------------------------------------- shared-memory stage layout
// One pipeline stage of CTA `rank` of a CG-CTA group holds, in this order: NI image tiles
// (TILE_ROWS x BK fp16 each: plane 1, then plane 2 when NI == 2), then the two slice tiles
// (BN / CG rows x BK fp16 each: plane 1, plane 2).  Every tile is a multiple of 1024 bytes.
constexpr int A_TILE_BYTES = TILE_ROWS * BK * 2;   // 16 KB
constexpr int SMEM_AUX = 6144;                     // 1 KB barriers + tmem pointer + abort word; 4 KB per-warp ||S||^2 tiles
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

// ---------------------------------------------------------------- a8: epilogue
// factor that undoes both rescales and carries the -2 of the cross term
SPF_MHD float cross_scale(int eI, int eS) { return ldexpf(-2.0f, -(eI + eS)); }

SPF_MHD float distance(float nI, float nS, float neg2sc, float acc) { return nI + fmaf(neg2sc, acc, nS); }

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
