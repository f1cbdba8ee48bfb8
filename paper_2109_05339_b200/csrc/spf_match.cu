// libspf: spf_match (steps a6-a8 of SURVEY.md section 8(a)).
//
//   d[i][m] = sum_j (I_ij - S_mj)^2 over unmasked pixels,  best_i = argmin_m d[i][m]
//           = a_i + b_m - 2 G_im,   a_i = ||I_i - c||^2,  b_m = sum S'_m (S'_m + 2 c),  G_im = I_i . S'_m,  S' = S - c
// (the conditioned expansion of spf_match_math.cuh: c is one common vector, the mean of up to 1,024 slices).
//
// The cross term G is a dense contraction (n_img x P) . (M x P)^T and runs on the 5th-generation tensor
// cores: tcgen05.mma with fp32 accumulators in TMEM, operands staged in shared memory by TMA.
// fp32-equivalent products come from a two-term fp16 split of each operand, x * 2^e = h1 + h2 (+ <=2^-22
// relative), after a power-of-two rescale into fp16 range.  Photon-count images are exact in ONE fp16
// term (integers < 2048), which is tested on the device: the kernel instantiated for one image plane
// issues 2 products per K step (I1.S1, I1.S2), the one for two planes issues 3 (adds I2.S1).  Both
// instantiations are launched and the one the data does not need returns at once, so the host never
// synchronises.  The epilogue reads the accumulator tile out of TMEM, adds a_i + b_m (fp64, rounded once)
// and keeps a running (min, argmin) per image row; tiles merge through a 64-bit atomicMin on
// (order-preserving bits of d) << 32 | m, so the lowest index wins exact ties and the distance
// matrix never exists in memory.  k_match_refine then recomputes each winner's distance in the
// difference form, so best_dist carries no cancellation error of the expansion.
#include <assert.h>
#include <cuda_fp16.h>
#include <math.h>

#include "ptx_sm100.cuh"
#include "spf_internal.cuh"
#include "spf_match_math.cuh"

namespace {

using spfmm::BK;         // 64 fp16 per K block: 128 bytes, one swizzle row
using spfmm::BN;         // 256 slices per tile (UMMA N)
using spfmm::TILE_ROWS;  // 128 image rows per CTA (UMMA M = 128 * CG)
using spfmm::A_TILE_BYTES;
constexpr int EPI_WARPS = 8;                      // two per TMEM lane quadrant, each takes one half of the tile's columns
constexpr int GEMM_THREADS = 64 + 32 * EPI_WARPS; // warp 0 TMA, warp 1 MMA + TMEM alloc, warps 2-9 epilogue
constexpr int EPI_COLS = BN / (EPI_WARPS / 4);    // 128 accumulator registers per epilogue thread
constexpr int EPI_PIECE = 16;                     // columns per tcgen05.ld (16 transient registers beside the 128 running sums)
constexpr int ACC_STAGES = 2;
constexpr int TMEM_COLS = ACC_STAGES * BN;        // 512: all of TMEM, one CTA per SM
constexpr size_t SMEM_AUX = spfmm::SMEM_AUX;

template <int CG, int NI>
struct GemmCfg {
    static constexpr int B_ROWS = spfmm::b_rows(CG);            // slice rows this CTA stages
    static constexpr int B_TILE_BYTES = spfmm::b_tile_bytes(CG);
    static constexpr int STAGE_BYTES = spfmm::stage_bytes(CG, NI);
    static constexpr int STAGES = spfmm::stages(CG, NI);
    static constexpr size_t SMEM_BYTES = (size_t)STAGES * STAGE_BYTES + SMEM_AUX + 1024;
    static constexpr int OFF_A1 = spfmm::off_a(1), OFF_B0 = spfmm::off_b(CG, NI, 0), OFF_B1 = spfmm::off_b(CG, NI, 1);
    static_assert(STAGES >= 2, "need at least a double buffer");
    static_assert(SMEM_BYTES <= (size_t)spfmm::SMEM_BUDGET, "shared memory budget");
};

struct MatchArgs {
    int64_t n_img, M;
    int kblocks;            // P_pad / 64
    int chunk_kb;           // K blocks accumulated in TMEM between two drains by the epilogue (>= 1)
    int n_ib, n_mb;         // tiles along images / slices
    uint32_t m_base;        // orientation index of slice row 0 (streaming: slices arrive in chunks of M)
    unsigned long long *keys;
    const double *aI, *bS;  // a_i = ||I_i - c||^2, b_m = sum S'_m (S'_m + 2 c)
    const uint32_t *scal;   // [2] = image plane 2 needed, [4] = eI, [5] = eS
    uint32_t *fault;        // context fault record (host-mapped): written when a pipeline wait gives up
    uint32_t *abort_flag;   // context abort flag (device memory): set by the first wait that gives up, read by every block
};

struct WsLayout {
    size_t scal, keys, aI, bS, common, planesI, planesS, total;
    int64_t Ppad;
};

size_t rup(size_t v, size_t a) { return (v + a - 1) / a * a; }

WsLayout ws_layout(int64_t n_img, int64_t M, int64_t P) {
    WsLayout L{};
    L.Ppad = (int64_t)rup((size_t)P, BK);
    size_t off = 0;
    L.scal = off; off += 1024;
    L.keys = off; off += rup((size_t)n_img * 8, 1024);
    L.aI = off; off += rup((size_t)n_img * 8, 1024);
    L.bS = off; off += rup((size_t)M * 8, 1024);
    L.common = off; off += rup((size_t)L.Ppad * 4, 1024);
    L.planesI = off; off += rup((size_t)2 * n_img * L.Ppad * 2, 1024);
    L.planesS = off; off += rup((size_t)2 * M * L.Ppad * 2, 1024);
    L.total = off;
    return L;
}

// ------------------------------------------------------------------------------------------
// a6 + operand preparation
// ------------------------------------------------------------------------------------------
// c[j] = mean over the rows 0, step, 2 step, ... of the slices (fp32 sum in ascending row order), 0 in masked
// pixels; one thread per pixel, so a warp reads 128 consecutive bytes of every row it visits.  condition = 0
// leaves c = 0 (the plain expansion; option "match_condition").  c is [Ppad]; the K padding is zeroed by the caller.
__global__ void k_common_vector(const float *__restrict__ slices, int64_t M, int64_t P, const uint8_t *__restrict__ mask,
                                int condition, float *__restrict__ c) {
    const int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (j >= P) return;
    float v = 0.0f;
    if (condition && (!mask || mask[j])) {
        const int64_t step = spfmm::common_step((long)M);
        float sum = 0.0f;
        for (int64_t m = 0; m < M; m += step) sum += slices[m * P + j];
        v = sum * (1.0f / (float)spfmm::common_count((long)M));
    }
    c[j] = v;
}

// max |x| (which = 0, images) or max |x - c| (which = 1, slices) over unmasked pixels, as the bit pattern of a
// non-negative float (orders like an unsigned).  Blocks stride over rows, threads over the pixels of a row:
// no integer division or modulo per element, coalesced loads.
__global__ void __launch_bounds__(256) k_absmax(const float *__restrict__ x, int64_t rows, int64_t P,
                                                const uint8_t *__restrict__ mask, const float *__restrict__ c, int which,
                                                uint32_t *__restrict__ out) {
    uint32_t m = 0;
    for (int64_t r = blockIdx.x; r < rows; r += gridDim.x) {
        const float *xr = x + r * P;
        for (int64_t j = threadIdx.x; j < P; j += blockDim.x) {
            if (mask && !mask[j]) continue;
            const float v = which ? spfmm::conditioned(xr[j], c[j]) : xr[j];
            m = max(m, __float_as_uint(fabsf(v)));
        }
    }
    m = __reduce_max_sync(0xffffffffu, m);
    if ((threadIdx.x & 31) == 0 && m) atomicMax(out, m);
}

// One block per row: v * 2^e = h1 + h2 as two fp16 planes (zero in masked pixels and in the K padding), where
//   which = 0 (images): v = the RAW value,   term = a_i = sum (x - c)^2; sets scal[2] when some residual is
//                       non-zero and resets the running-argmin key;
//   which = 1 (slices): v = S' = fl(x - c),  term = b_m = sum S' (S' + 2 c);
// both sums over unmasked pixels, accumulated in fp64.
__global__ void __launch_bounds__(256) k_split(const float *__restrict__ x, int64_t P, int64_t Ppad,
                                               const uint8_t *__restrict__ mask, const float *__restrict__ c,
                                               uint32_t *__restrict__ scal, int which, int64_t rows,
                                               __half *__restrict__ planes, double *__restrict__ term,
                                               unsigned long long *__restrict__ keys) {
    const int64_t row = blockIdx.x;
    const int e = spfmm::scale_exponent(scal[which]);
    const float sc = ldexpf(1.0f, e);
    const float *xr = x + row * P;
    __half *h1 = planes + row * Ppad, *h2 = planes + (rows + row) * Ppad;
    double acc = 0.0;
    bool inexact = false;
    for (int64_t j = threadIdx.x; j < Ppad; j += blockDim.x) {
        float v = 0.0f;
        if (j < P && (!mask || mask[j])) {
            const float raw = xr[j], cj = c[j];
            if (which) { v = spfmm::conditioned(raw, cj); acc += spfmm::slice_term(v, cj); }
            else { v = raw; acc += spfmm::image_term(raw, cj); }
        }
        uint16_t a, b;
        inexact |= spfmm::split_fp16(v, sc, a, b);
        h1[j] = __ushort_as_half(a);
        h2[j] = __ushort_as_half(b);
    }
    __shared__ double red[8];
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    const bool any = __any_sync(0xffffffffu, inexact);
    if ((threadIdx.x & 31) == 0) {
        red[threadIdx.x >> 5] = acc;
        if (which == 0 && any) atomicOr(&scal[2], 1u);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int k = 0; k < (int)(blockDim.x >> 5); ++k) s += red[k];
        term[row] = s;
        if (which == 0) keys[row] = ~0ull;
        if (row == 0) scal[4 + which] = (uint32_t)e;
    }
}

__global__ void k_match_finalize(const unsigned long long *__restrict__ keys, int64_t n_img, int32_t *__restrict__ best_idx,
                                 float *__restrict__ best_dist) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n_img) return;
    unsigned long long k = keys[i];
    best_idx[i] = (int32_t)(uint32_t)(k & 0xffffffffull);  // -1 if no finite distance was seen
    best_dist[i] = (k == ~0ull) ? __uint_as_float(0x7fc00000u) : spfmm::unorderable((uint32_t)(k >> 32));
}

// The winner's distance by the definition: d = sum_j (I_ij - S_mj)^2 over unmasked pixels, differences
// and sum in fp64, rounded once.  One block per image; n_img x P pixel pairs in all (1e-4 of the contraction's work).
// The tensor-core pass decides WHICH orientation wins; this makes the reported distance free of the expansion's
// cancellation.  Rows with no winner (index -1) keep their NaN.
__global__ void __launch_bounds__(256) k_match_refine(const float *__restrict__ images, const float *__restrict__ slices,
                                                      int64_t M, int64_t P, const uint8_t *__restrict__ mask,
                                                      const int32_t *__restrict__ best_idx, float *__restrict__ best_dist,
                                                      int rows_are_winners) {
    // rows_are_winners = 0: slices is the whole [M][P] array, the winner's row is best_idx[i];
    //                  = 1: slices holds, in row i, the slice of image i's winning orientation (streaming: re-sliced)
    const int64_t i = blockIdx.x;
    const int64_t w = best_idx[i];
    if (w < 0 || (!rows_are_winners && w >= M)) return;
    const int64_t m = rows_are_winners ? i : w;
    const float *I = images + i * P, *S = slices + m * P;
    double acc = 0.0;
    for (int64_t j = threadIdx.x; j < P; j += blockDim.x) {
        if (mask && !mask[j]) continue;
        const double t = (double)I[j] - (double)S[j];
        acc += t * t;
    }
    __shared__ double red[8];
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int k = 0; k < (int)(blockDim.x >> 5); ++k) s += red[k];
        best_dist[i] = (float)s;
    }
}

// ------------------------------------------------------------------------------------------
// a7 + a8: tcgen05 GEMM with the fused norm-add / argmin epilogue
// ------------------------------------------------------------------------------------------
template <int CG, int NI>
__global__ void __launch_bounds__(GEMM_THREADS, 1)
k_match_gemm(const __grid_constant__ CUtensorMap mapA0, const __grid_constant__ CUtensorMap mapA1,
             const __grid_constant__ CUtensorMap mapB0, const __grid_constant__ CUtensorMap mapB1, const MatchArgs a) {
    using Cfg = GemmCfg<CG, NI>;
    constexpr int ST = Cfg::STAGES;
    // the instantiation the data does not need leaves before touching any barrier or TMEM; so does every block
    // once some block's pipeline has given up (both conditions are uniform over a CTA pair)
    if ((a.scal[2] != 0u) != (NI == 2)) return;
    volatile uint32_t *g_abort = a.abort_flag;
    if (*g_abort) return;

    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;  // SWIZZLE_128B tiles need 1024-byte alignment
    uint8_t *smem_al = smem_raw + (smem_base - ptx::smem_u32(smem_raw));
    const uint32_t aux = smem_base + ST * Cfg::STAGE_BYTES;
    uint8_t *aux_p = smem_al + (size_t)ST * Cfg::STAGE_BYTES;
    const uint32_t bar_full = aux, bar_empty = aux + 8 * ST, bar_tfull = aux + 16 * ST, bar_tempty = bar_tfull + 8 * ACC_STAGES;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(aux_p + 16 * ST + 16 * ACC_STAGES);
    volatile uint32_t *abort_w = tmem_slot + 1;              // raised by the first wait of this block that gives up
    static_assert(16 * 6 + 16 * ACC_STAGES + 8 <= (int)SMEM_AUX, "barriers, TMEM slot and abort word fit the auxiliary block");
#ifdef SPF_DEBUG
    // invariants the descriptors and the bulk copies rely on (table of PTX wrappers)
    if (threadIdx.x == 0) {
        assert((smem_base & 1023u) == 0u);                                           // SWIZZLE_128B atom alignment
        assert(smem_base + ST * Cfg::STAGE_BYTES + SMEM_AUX <= ptx::smem_u32(smem_raw) + (uint32_t)Cfg::SMEM_BYTES);
        // 14-bit start-address field of the UMMA descriptor (the window offset; in a CTA pair the odd CTA's shared
        // addresses carry its rank above bit 18, which umma_desc_sw128 masks off)
        assert((((smem_base & 0x3FFFFu) + ST * Cfg::STAGE_BYTES) >> 4) <= (1u << 14));
        assert((bar_full & 7u) == 0u);
        assert(gridDim.x % CG == 0 && a.chunk_kb >= 1);
    }
#endif

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = (CG == 2) ? ptx::cluster_ctarank() : 0u;
    const bool leader = (rank == 0);
    const int cluster_id = blockIdx.x / CG, n_clusters = gridDim.x / CG;
    const int n_tiles = a.n_ib * a.n_mb;

    if (warp == 0 && lane == 0) {
        *abort_w = 0u;
        ptx::prefetch_tensormap(&mapA0); ptx::prefetch_tensormap(&mapB0); ptx::prefetch_tensormap(&mapB1);
        if (NI == 2) ptx::prefetch_tensormap(&mapA1);
        for (int s = 0; s < ST; ++s) { ptx::mbar_init(bar_full + 8 * s, 1); ptx::mbar_init(bar_empty + 8 * s, 1); }
        for (int s = 0; s < ACC_STAGES; ++s) { ptx::mbar_init(bar_tfull + 8 * s, 1); ptx::mbar_init(bar_tempty + 8 * s, EPI_WARPS * CG); }
        ptx::fence_mbar_init();
    }
    if (warp == 1) ptx::tmem_alloc<CG>(ptx::smem_u32(tmem_slot), TMEM_COLS);
    ptx::tc_fence_before();
    if (CG == 2) ptx::cluster_sync(); else __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
#ifdef SPF_DEBUG
    if (threadIdx.x == 0) assert((tmem_base & 0xffffu) + TMEM_COLS <= 512u && (tmem_base >> 16) == 0u);   // whole TMEM, lane 0
#endif

    auto tile_coords = [&](int t, int &ib, int &mb) { spfmm::tile_coords(t, a.n_ib, a.n_mb, ib, mb); };

    // a wait that gave up: note where (first writer wins is not needed -- any one record will do)
    auto give_up = [&](uint32_t role, int t) {
        if (lane == 0) {
            a.fault[1] = blockIdx.x; a.fault[2] = (uint32_t)t; a.fault[3] = (uint32_t)(CG * 10 + NI);
            a.fault[0] = SPF_FAULT_MATCH + role;
            __threadfence_system();
        }
    };

    if (warp == 0) {
        // ===================== TMA producer =====================
        int s = 0; uint32_t ph = 0;
        bool alive = true;
        for (int t = cluster_id; alive && t < n_tiles; t += n_clusters) {
            int ib, mb; tile_coords(t, ib, mb);
            const int rowA = ib * (TILE_ROWS * CG) + (int)rank * TILE_ROWS;
            const int rowB = mb * BN + (int)rank * Cfg::B_ROWS;
            for (int kb = 0; kb < a.kblocks; ++kb) {
                if (!ptx::mbar_wait(bar_empty + 8 * s, ph ^ 1u, abort_w, g_abort)) { give_up(0, t); alive = false; break; }
                if (lane == 0) {
                    const uint32_t st = smem_base + s * Cfg::STAGE_BYTES;
                    const uint32_t fb = bar_full + 8 * s;
                    if (CG == 1) ptx::mbar_expect_tx(fb, Cfg::STAGE_BYTES);
                    else if (leader) ptx::mbar_expect_tx(fb, 2 * Cfg::STAGE_BYTES);
                    const int kc = kb * BK;
                    if (CG == 1) {
                        ptx::tma_load_2d(st, &mapA0, kc, rowA, fb);
                        if (NI == 2) ptx::tma_load_2d(st + Cfg::OFF_A1, &mapA1, kc, rowA, fb);
                        ptx::tma_load_2d(st + Cfg::OFF_B0, &mapB0, kc, rowB, fb);
                        ptx::tma_load_2d(st + Cfg::OFF_B1, &mapB1, kc, rowB, fb);
                    } else {
                        ptx::tma_load_2d_2sm(st, &mapA0, kc, rowA, fb);
                        if (NI == 2) ptx::tma_load_2d_2sm(st + Cfg::OFF_A1, &mapA1, kc, rowA, fb);
                        ptx::tma_load_2d_2sm(st + Cfg::OFF_B0, &mapB0, kc, rowB, fb);
                        ptx::tma_load_2d_2sm(st + Cfg::OFF_B1, &mapB1, kc, rowB, fb);
                    }
                }
                __syncwarp();
                if (++s == ST) { s = 0; ph ^= 1u; }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer (leader CTA of the pair) =====================
        if (leader) {
            constexpr uint32_t idesc = ptx::umma_idesc_f16(TILE_ROWS * CG, BN);
            int s = 0; uint32_t ph = 0; int as = 0; uint32_t aph = 0;
            bool alive = true;
            for (int t = cluster_id; alive && t < n_tiles; t += n_clusters) {
                // K runs in chunks of a.chunk_kb blocks; each chunk starts on a cleared accumulator stage
                // and is handed to the epilogue warps, which keep the running sum (spf_match_math.cuh)
                for (int kb0 = 0; alive && kb0 < a.kblocks; kb0 += a.chunk_kb) {
                    // epilogue has drained this accumulator stage
                    if (!ptx::mbar_wait(bar_tempty + 8 * as, aph ^ 1u, abort_w, g_abort)) { give_up(1, t); alive = false; break; }
                    ptx::tc_fence_after();
                    const uint32_t tacc = tmem_base + (uint32_t)(as * BN);
                    const int kend = min(kb0 + a.chunk_kb, a.kblocks);
                    for (int kb = kb0; kb < kend; ++kb) {
                        if (!ptx::mbar_wait(bar_full + 8 * s, ph, abort_w, g_abort)) { give_up(2, t); alive = false; break; }
                        ptx::tc_fence_after();
                        if (lane == 0) {
                            const uint32_t st = smem_base + s * Cfg::STAGE_BYTES;
                            const uint64_t dA0 = ptx::umma_desc_sw128(st);
                            const uint64_t dA1 = ptx::umma_desc_sw128(st + Cfg::OFF_A1);
                            const uint64_t dB0 = ptx::umma_desc_sw128(st + Cfg::OFF_B0);
                            const uint64_t dB1 = ptx::umma_desc_sw128(st + Cfg::OFF_B1);
#pragma unroll
                            for (int k4 = 0; k4 < BK / 16; ++k4) {  // 16 fp16 = 32 bytes per UMMA K step: +2 in the address field
                                const uint64_t ko = (uint64_t)(k4 * 2);
                                ptx::umma_f16<CG>(tacc, dA0 + ko, dB0 + ko, idesc, (uint32_t)(kb != kb0 || k4 != 0));
                                ptx::umma_f16<CG>(tacc, dA0 + ko, dB1 + ko, idesc, 1u);
                                if (NI == 2) ptx::umma_f16<CG>(tacc, dA1 + ko, dB0 + ko, idesc, 1u);
                            }
                            ptx::umma_commit<CG>(bar_empty + 8 * s);                       // smem slot free when these MMAs retire
                            if (kb == kend - 1) ptx::umma_commit<CG>(bar_tfull + 8 * as);  // chunk complete
                        }
                        __syncwarp();
                        if (++s == ST) { s = 0; ph ^= 1u; }
                    }
                    if (++as == ACC_STAGES) { as = 0; aph ^= 1u; }
                }
            }
        }
    } else {
        // ===================== epilogue: TMEM chunks -> fp32 registers -> a_i + b_m - 2 G, running argmin =====================
        // Warp (warp - 2) reads TMEM lane quadrant warp % 4 (the only one the hardware lets it read) and
        // the column half (warp - 2) / 4 of the tile: thread = one image row x EPI_COLS slices, whose
        // cross terms it sums chunk by chunk in registers (round to nearest).  Each warp works alone --
        // its own lanes, nothing shared -- so epilogue warps never wait for one another.
        const int ew = warp - 2;
        const int q = warp & 3;                 // TMEM lane quadrant
        const int col0 = (ew >> 2) * EPI_COLS;  // first tile column of this warp
        const float neg2sc = spfmm::cross_scale((int)a.scal[4], (int)a.scal[5]);
        int as = 0; uint32_t aph = 0;
        bool alive = true;
        for (int t = cluster_id; alive && t < n_tiles; t += n_clusters) {
            int ib, mb; tile_coords(t, ib, mb);
            const int64_t m0 = (int64_t)mb * BN + col0;
            const int64_t i = (int64_t)ib * (TILE_ROWS * CG) + (int64_t)rank * TILE_ROWS + q * 32 + lane;
            float acc[EPI_COLS];
#pragma unroll
            for (int k = 0; k < EPI_COLS; ++k) acc[k] = 0.0f;
            for (int kb0 = 0; kb0 < a.kblocks; kb0 += a.chunk_kb) {
                if (!ptx::mbar_wait(bar_tfull + 8 * as, aph, abort_w, g_abort)) { give_up(3, t); alive = false; break; }
                ptx::tc_fence_after();
                const uint32_t trow = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(as * BN + col0);
#pragma unroll
                for (int c = 0; c < EPI_COLS / EPI_PIECE; ++c) {
                    uint32_t r[EPI_PIECE];
                    ptx::tmem_ld_32x16(trow + c * EPI_PIECE, r);
                    ptx::tmem_ld_wait();
#pragma unroll
                    for (int k = 0; k < EPI_PIECE; ++k) acc[c * EPI_PIECE + k] += __uint_as_float(r[k]);
                }
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) { if (CG == 2) ptx::mbar_arrive_cluster(bar_tempty + 8 * as, 0); else ptx::mbar_arrive(bar_tempty + 8 * as); }
                if (++as == ACC_STAGES) { as = 0; aph ^= 1u; }
            }
            if (!alive) break;
            if (i < a.n_img) {
                // once per pair per tile: fp64 add of the two row terms and the (exactly rescaled) cross term
                const double aIv = a.aI[i];
                float best = INFINITY; uint32_t bm = 0xffffffffu;
#pragma unroll
                for (int k = 0; k < EPI_COLS; ++k) {
                    if (m0 + k < a.M) {
                        const float d = spfmm::distance(aIv, __ldg(a.bS + m0 + k), neg2sc, acc[k]);
                        if (d < best) { best = d; bm = a.m_base + (uint32_t)(m0 + k); }   // ascending k: the lowest index wins ties
                    }
                }
                if (bm != 0xffffffffu) atomicMin(&a.keys[i], spfmm::pack_key(best, bm));
            }
        }
    }

    // teardown.  After a give-up, bulk copies and MMAs issued earlier may still be in flight: let them land
    // before TMEM is released and the shared memory goes to the next block (ptx::abort_drain).
    ptx::tc_fence_before();
    if (CG == 2) ptx::cluster_sync(); else __syncthreads();
    if (*abort_w || *g_abort) ptx::abort_drain();
    if (warp == 1) ptx::tmem_dealloc<CG>(tmem_base, TMEM_COLS);
}

// ------------------------------------------------------------------------------------------
// CUDA-core matcher (option "match_impl" = 1, the library default until the tensor-core kernel has
// passed its self-check on the device): the definition itself, d = sum_j (I_ij - S_mj)^2 over unmasked
// pixels, in fp32 -- no expansion, so no cancellation and no operand split.  A register-tiled kernel in
// the shape of a plain SGEMM: block = 128 images x 128 slices, 256 threads x (8 x 8) pairs, K tiles of
// 16 pixels staged through shared memory (transposed, padded rows).  Each pair's sum runs in two
// levels -- 1,024 pixels into `acc`, then `acc` into `tot` -- so the rounding error stays ~1e-6 of d at
// P = 65,536.  The argmin merges through the same packed 64-bit atomicMin keys as the tensor-core kernel.
// Cost: 2 instructions per pixel pair on the fp32 pipes (74 TFLOP/s) against 2 fp16 products on the
// tensor pipe (> 1 PFLOP/s): about 20x slower at Paper-scale.  It is the fallback, not the product.
// ------------------------------------------------------------------------------------------
constexpr int ST_BM = 128, ST_BN = 128, ST_BK = 16, ST_PAD = 4, ST_FLUSH = 1024 / ST_BK;

__global__ void __launch_bounds__(256, 1)
k_match_simt(const float *__restrict__ images, int64_t n_img, const float *__restrict__ slices, int64_t M, int64_t P,
             const uint8_t *__restrict__ mask, unsigned long long *__restrict__ keys, uint32_t m_base) {
    __shared__ __align__(16) float sI[ST_BK][ST_BM + ST_PAD];
    __shared__ __align__(16) float sS[ST_BK][ST_BN + ST_PAD];
    const int tid = threadIdx.x;
    const int ty = tid >> 4, tx = tid & 15;                 // 16 x 16 threads, 8 x 8 pairs each
    const int64_t i0 = (int64_t)blockIdx.x * ST_BM, m0 = (int64_t)blockIdx.y * ST_BN;
    const int lk = tid & 15, lr = tid >> 4;                 // loader: pixel lk of the K tile, rows lr + 16 r
    float acc[8][8], tot[8][8];
#pragma unroll
    for (int a = 0; a < 8; ++a)
#pragma unroll
        for (int b = 0; b < 8; ++b) acc[a][b] = tot[a][b] = 0.0f;

    const int64_t ktiles = (P + ST_BK - 1) / ST_BK;
    float pI[8], pS[8];                                     // next K tile, fetched while the current one is summed
    auto fetch = [&](int64_t kt) {
        const int64_t j = kt * ST_BK + lk;
        const bool use = kt < ktiles && j < P && (!mask || mask[j]);
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const int64_t i = i0 + lr + 16 * r, m = m0 + lr + 16 * r;
            pI[r] = (use && i < n_img) ? images[i * P + j] : 0.0f;
            pS[r] = (use && m < M) ? slices[m * P + j] : 0.0f;
        }
    };
    fetch(0);
    for (int64_t kt = 0; kt < ktiles; ++kt) {
#pragma unroll
        for (int r = 0; r < 8; ++r) { sI[lk][lr + 16 * r] = pI[r]; sS[lk][lr + 16 * r] = pS[r]; }
        __syncthreads();
        fetch(kt + 1);
#pragma unroll
        for (int kk = 0; kk < ST_BK; ++kk) {
            // thread (ty, tx) owns image rows ty*8 .. +7 and slice columns tx*4 .. +3 and 64 + tx*4 .. +3
            // (two 16-byte loads per operand, neighbouring lanes 16 bytes apart: no bank conflicts)
            float a[8], b[8];
            const float4 a0 = *reinterpret_cast<const float4 *>(&sI[kk][ty * 8]), a1 = *reinterpret_cast<const float4 *>(&sI[kk][ty * 8 + 4]);
            const float4 b0 = *reinterpret_cast<const float4 *>(&sS[kk][tx * 4]), b1 = *reinterpret_cast<const float4 *>(&sS[kk][64 + tx * 4]);
            a[0] = a0.x; a[1] = a0.y; a[2] = a0.z; a[3] = a0.w; a[4] = a1.x; a[5] = a1.y; a[6] = a1.z; a[7] = a1.w;
            b[0] = b0.x; b[1] = b0.y; b[2] = b0.z; b[3] = b0.w; b[4] = b1.x; b[5] = b1.y; b[6] = b1.z; b[7] = b1.w;
#pragma unroll
            for (int u = 0; u < 8; ++u)
#pragma unroll
                for (int v = 0; v < 8; ++v) {
                    const float t = a[u] - b[v];
                    acc[u][v] = fmaf(t, t, acc[u][v]);
                }
        }
        __syncthreads();
        if ((kt + 1) % ST_FLUSH == 0) {
#pragma unroll
            for (int u = 0; u < 8; ++u)
#pragma unroll
                for (int v = 0; v < 8; ++v) { tot[u][v] += acc[u][v]; acc[u][v] = 0.0f; }
        }
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) {
        const int64_t i = i0 + ty * 8 + u;
        float best = INFINITY; uint32_t bm = 0xffffffffu;
#pragma unroll
        for (int v = 0; v < 8; ++v) {
            const int64_t m = m0 + (v < 4 ? tx * 4 + v : 64 + tx * 4 + v - 4);   // ascending in v: the lowest index wins ties
            const float d = tot[u][v] + acc[u][v];
            if (m < M && d < best) { best = d; bm = m_base + (uint32_t)m; }
        }
        if (i < n_img && bm != 0xffffffffu) atomicMin(&keys[i], spfmm::pack_key(best, bm));
    }
}

// ------------------------------------------------------------------------------------------
// Warp-level tensor-core matcher (option "match_impl" = 2): the same conditioned, split-precision contraction as
// k_match_gemm -- same operand planes, same products, same fp64 epilogue, same packed-key argmin -- on the CLASSIC
// CUDA tensor-core path: cp.async multi-stage pipeline, ldmatrix, mma.sync.m16n8k16 with fp32 accumulators in registers.
// No tensor map, no mbarrier, no TMEM, no tcgen05: nothing in it that a device fault has ever been traced to, so it
// can be checked in-process (spf_selftest "match_mma") and used where the tcgen05 kernel has not been cleared.  It is the
// legacy path -- mma.sync cannot reach tcgen05 throughput on sm_100a -- and exists as the safe tensor-core matcher, not
// as the product.  Block tile 128 images x 128 slices, 8 warps of 64 x 32, K stages of 32 pixels (64-byte rows, 16-byte
// chunks XOR-swizzled with (row / 2) mod 4 so that ldmatrix reads 8 rows from 8 distinct bank groups).
// ------------------------------------------------------------------------------------------
constexpr int MM_BM = 128, MM_BN = 128, MM_BK = 32, MM_STAGES = 4, MM_THREADS = 256;
constexpr int MM_TILE_BYTES = 128 * MM_BK * 2;   // 8 KB: 128 rows of 64 bytes
template <int NI> struct MmaCfg {
    static constexpr int TILES = NI + 2;          // image planes, then the two slice planes
    static constexpr int STAGE_BYTES = TILES * MM_TILE_BYTES;
    static constexpr int SMEM_BYTES = MM_STAGES * STAGE_BYTES;
};
__device__ __forceinline__ uint32_t mm_off(int row, int chunk) { return (uint32_t)(row * 64 + ((chunk ^ ((row >> 1) & 3)) << 4)); }

template <int NI>
__global__ void __launch_bounds__(MM_THREADS, 1)
k_match_mma(const __half *__restrict__ plI, const __half *__restrict__ plS, int64_t Ppad, const MatchArgs a) {
    using Cfg = MmaCfg<NI>;
    if ((a.scal[2] != 0u) != (NI == 2)) return;   // the instantiation the data does not need
    extern __shared__ __align__(128) uint8_t mm_smem[];
    const uint32_t smem0 = ptx::smem_u32(mm_smem);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp >> 2, wn = warp & 3;                       // warp grid 2 x 4: rows wm * 64, columns wn * 32
    const int ib = (int)(blockIdx.x % (unsigned)a.n_ib), mb = (int)(blockIdx.x / (unsigned)a.n_ib);
    const int64_t i0 = (int64_t)ib * MM_BM, m0 = (int64_t)mb * MM_BN;
    const int nk = a.kblocks * (BK / MM_BK);                       // K steps of 32 pixels
    const int chunk_steps = a.chunk_kb * (BK / MM_BK);

    auto load_stage = [&](int kt, int slot) {
        const uint32_t st = smem0 + (uint32_t)(slot * Cfg::STAGE_BYTES);
        const int64_t k0 = (int64_t)kt * MM_BK;
#pragma unroll
        for (int it = 0; it < Cfg::TILES * 512 / MM_THREADS; ++it) {
            const int idx = tid + it * MM_THREADS, tile = idx >> 9, r = (idx & 511) >> 2, c = idx & 3;
            const bool img = tile < NI;
            const int64_t rows = img ? a.n_img : a.M, row = (img ? i0 : m0) + r;
            const int plane = img ? tile : tile - NI;
            const __half *base = (img ? plI : plS) + (size_t)plane * (size_t)rows * (size_t)Ppad;
            const int64_t rr = row < rows ? row : rows - 1;        // rows past the end: zero-filled, the address stays valid
            ptx::cp_async_16_zfill(st + (uint32_t)(tile * MM_TILE_BYTES) + mm_off(r, c), base + rr * Ppad + k0 + c * 8, row < rows ? 16u : 0u);
        }
    };

    float acc[4][4][4], tot[4][4][4];
#pragma unroll
    for (int x = 0; x < 4; ++x)
#pragma unroll
        for (int y = 0; y < 4; ++y)
#pragma unroll
            for (int z = 0; z < 4; ++z) acc[x][y][z] = tot[x][y][z] = 0.0f;

    for (int s = 0; s < MM_STAGES - 1; ++s) {
        if (s < nk) load_stage(s, s);
        ptx::cp_async_commit();
    }
    int since_flush = 0;
    for (int kt = 0; kt < nk; ++kt) {
        ptx::cp_async_wait_group<MM_STAGES - 2>();   // stage kt has landed (this thread's pieces) ...
        __syncthreads();                             // ... and everybody's; and every warp has finished stage kt - 1
        if (kt + MM_STAGES - 1 < nk) load_stage(kt + MM_STAGES - 1, (kt + MM_STAGES - 1) % MM_STAGES);
        ptx::cp_async_commit();
        const uint32_t st = smem0 + (uint32_t)((kt % MM_STAGES) * Cfg::STAGE_BYTES);
        const uint32_t tS1 = st + (uint32_t)(NI * MM_TILE_BYTES), tS2 = tS1 + MM_TILE_BYTES;
#pragma unroll
        for (int kk = 0; kk < MM_BK / 16; ++kk) {
            uint32_t af[4][4], af2[4][4];
            const int mat = lane >> 3, r8 = lane & 7;
#pragma unroll
            for (int mt = 0; mt < 4; ++mt) {
                const int row = wm * 64 + mt * 16 + (mat & 1) * 8 + r8, chunk = kk * 2 + (mat >> 1);
                ptx::ldmatrix_x4(af[mt], st + mm_off(row, chunk));
                if (NI == 2) ptx::ldmatrix_x4(af2[mt], st + MM_TILE_BYTES + mm_off(row, chunk));
            }
#pragma unroll
            for (int np = 0; np < 2; ++np) {          // pairs of 8-column tiles
                uint32_t b1[4], b2[4];
                const int n = wn * 32 + np * 16 + (mat >> 1) * 8 + r8, chunk = kk * 2 + (mat & 1);
                ptx::ldmatrix_x4(b1, tS1 + mm_off(n, chunk));
                ptx::ldmatrix_x4(b2, tS2 + mm_off(n, chunk));
#pragma unroll
                for (int mt = 0; mt < 4; ++mt)
#pragma unroll
                    for (int nt = 0; nt < 2; ++nt) {
                        ptx::mma_m16n8k16(acc[mt][np * 2 + nt], af[mt], b1[2 * nt], b1[2 * nt + 1]);            // I1 . S1
                        ptx::mma_m16n8k16(acc[mt][np * 2 + nt], af[mt], b2[2 * nt], b2[2 * nt + 1]);            // I1 . S2
                        if (NI == 2) ptx::mma_m16n8k16(acc[mt][np * 2 + nt], af2[mt], b1[2 * nt], b1[2 * nt + 1]);   // I2 . S1
                    }
            }
        }
        if (++since_flush == chunk_steps) {           // the chunk's sum joins the running total with round-to-nearest adds
            since_flush = 0;
#pragma unroll
            for (int x = 0; x < 4; ++x)
#pragma unroll
                for (int y = 0; y < 4; ++y)
#pragma unroll
                    for (int z = 0; z < 4; ++z) { tot[x][y][z] += acc[x][y][z]; acc[x][y][z] = 0.0f; }
        }
    }
    ptx::cp_async_wait_group<0>();

    // epilogue: d = a_i + b_m - 2 G (fp64, rounded once), best of this thread's 8 columns per row, then of the 4 lanes that
    // share the row; ascending column order and the packed key keep "lowest index wins ties"
    const float neg2sc = spfmm::cross_scale((int)a.scal[4], (int)a.scal[5]);
    const int g = lane >> 2, t = lane & 3;
#pragma unroll
    for (int mt = 0; mt < 4; ++mt)
#pragma unroll
        for (int half = 0; half < 2; ++half) {
            const int64_t i = i0 + wm * 64 + mt * 16 + g + 8 * half;
            unsigned long long key = ~0ull;
            if (i < a.n_img) {
                const double aIv = a.aI[i];
#pragma unroll
                for (int nt = 0; nt < 4; ++nt)
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const int64_t m = m0 + wn * 32 + nt * 8 + 2 * t + e;
                        if (m < a.M) {
                            const float G = tot[mt][nt][half * 2 + e] + acc[mt][nt][half * 2 + e];
                            const unsigned long long k2 = spfmm::pack_key(spfmm::distance(aIv, __ldg(a.bS + m), neg2sc, G), a.m_base + (uint32_t)m);
                            key = k2 < key ? k2 : key;
                        }
                    }
            }
            unsigned long long o = __shfl_xor_sync(0xffffffffu, key, 1);
            key = o < key ? o : key;
            o = __shfl_xor_sync(0xffffffffu, key, 2);
            key = o < key ? o : key;
            if (t == 0 && key != ~0ull) atomicMin(&a.keys[i], key);
        }
}

// ------------------------------------------------------------------------------------------
// reference matcher (tests only): difference form on the CUDA cores, fp64 accumulation
// ------------------------------------------------------------------------------------------
__global__ void k_match_ref_dist(const float *__restrict__ images, int64_t n_img, const float *__restrict__ slices, int64_t M,
                                 int64_t P, const uint8_t *__restrict__ mask, float *__restrict__ dist) {
    const int64_t pair = blockIdx.x;  // one block per (i, m)
    const int64_t i = pair / M, m = pair % M;
    const float *I = images + i * P, *S = slices + m * P;
    double acc = 0.0;
    for (int64_t j = threadIdx.x; j < P; j += blockDim.x) {
        if (mask && !mask[j]) continue;
        double t = (double)I[j] - (double)S[j];
        acc += t * t;
    }
    __shared__ double red[8];
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int k = 0; k < (int)(blockDim.x >> 5); ++k) s += red[k];
        dist[pair] = (float)s;
    }
}

__global__ void k_match_ref_argmin(const float *__restrict__ dist, int64_t n_img, int64_t M, int32_t *__restrict__ best_idx,
                                   float *__restrict__ best_dist) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n_img) return;
    const float *d = dist + i * M;
    int64_t b = 0;
    for (int64_t m = 1; m < M; ++m)
        if (d[m] < d[b]) b = m;
    best_idx[i] = (int32_t)b;
    best_dist[i] = d[b];
}

int encode_operand_map(spf_ctx *ctx, CUtensorMap *map, const void *base, int64_t rows, int64_t Ppad, int box_rows) {
    spf_encode_tiled_fn enc = spf_get_encode_tiled();
    if (!enc) return spf_set_err(ctx, SPF_ECUDA, "cuTensorMapEncodeTiled entry point not available");
    cuuint64_t gdim[2] = {(cuuint64_t)Ppad, (cuuint64_t)rows};
    cuuint64_t gstr[1] = {(cuuint64_t)Ppad * 2};
    cuuint32_t box[2] = {(cuuint32_t)BK, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, const_cast<void *>(base), gdim, gstr, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return spf_set_err(ctx, SPF_ECUDA, "cuTensorMapEncodeTiled(match operand) failed: %d", (int)r);
    return SPF_OK;
}

template <int CG, int NI>
int launch_gemm(spf_ctx *ctx, const CUtensorMap &a0, const CUtensorMap &a1, const CUtensorMap &b0, const CUtensorMap &b1,
                const MatchArgs &args, cudaStream_t st) {
    using Cfg = GemmCfg<CG, NI>;
    auto kern = k_match_gemm<CG, NI>;
    SPF_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM_BYTES));
    const int n_tiles = args.n_ib * args.n_mb;
    cudaLaunchConfig_t cfg{};
    cfg.blockDim = dim3(GEMM_THREADS);
    cfg.dynamicSmemBytes = Cfg::SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CG; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    // Persistent grid with a static tile stride: every cluster must be resident at once, or the ones
    // that start late run their whole share after the others have finished.  CTA pairs need two free
    // SMs of one TPC, so fewer than sm_count / 2 pairs may fit: ask the runtime (cached per context and variant).
    int &max_clusters = ctx->gemm_max_clusters[CG - 1][NI - 1];
    if (max_clusters == 0) {
        int n = 0;
        cfg.gridDim = dim3((unsigned)(ctx->sm_count / CG * CG));
        if (cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess || n < 1) { (void)cudaGetLastError(); n = ctx->sm_count / CG; }
        max_clusters = n < ctx->sm_count / CG ? n : ctx->sm_count / CG;
    }
    int clusters = max_clusters;
    if (clusters > n_tiles) clusters = n_tiles;
    cfg.gridDim = dim3((unsigned)(clusters * CG));
    SPF_CUDA(ctx, cudaLaunchKernelEx(&cfg, kern, a0, a1, b0, b1, args));
    ctx->launches++;
    return SPF_OK;
}

}  // namespace

extern "C" {

size_t spf_match_workspace_bytes(int64_t n_img, int64_t M, int64_t P) {
    if (n_img < 0 || M < 0 || P < 0) return 0;
    return ws_layout(n_img, M, P).total;
}

// One pass of the matcher over a chunk of M slices whose first row is orientation m_base.  first: reset the argmin keys,
// (tensor-core path) take the common vector from THIS chunk and prepare the image operand; later chunks reuse both.
// The keys merge across chunks through the same packed atomicMin, so the result is that of one pass over all slices.
static int match_pass(spf_ctx *ctx, const float *images, int64_t n_img, const float *slices, int64_t M, int64_t P, const uint8_t *mask,
                      void *workspace, const WsLayout &L, cudaStream_t st, int64_t m_base, bool first) {
    uint8_t *ws = (uint8_t *)workspace;
    uint32_t *scal = (uint32_t *)(ws + L.scal);
    unsigned long long *keys = (unsigned long long *)(ws + L.keys);
    double *aI = (double *)(ws + L.aI), *bS = (double *)(ws + L.bS);
    float *cvec = (float *)(ws + L.common);
    __half *plI = (__half *)(ws + L.planesI), *plS = (__half *)(ws + L.planesS);

    int rc;
    if ((rc = spf_record_event(ctx, 4, st))) return rc;
    if (first) SPF_CUDA(ctx, cudaMemsetAsync(scal, 0, 64, st));
    else SPF_CUDA(ctx, cudaMemsetAsync(scal + 1, 0, 4, st));   // the slices' abs-max is per chunk
    ctx->last_match_impl = ctx->opt_match_impl;
    if (ctx->opt_match_impl == 1) {
        // CUDA-core matcher: no operand preparation, only the argmin keys are reset (all ones = "nothing seen")
        const int64_t gy = (M + ST_BN - 1) / ST_BN;
        if (gy > 65535) return spf_set_err(ctx, SPF_EINVAL, "spf_match: M too large for the CUDA-core matcher (%lld slices)", (long long)M);
        if (first) SPF_CUDA(ctx, cudaMemsetAsync(keys, 0xff, (size_t)n_img * 8, st));
        if ((rc = spf_record_event(ctx, 2, st))) return rc;
        k_match_simt<<<dim3((unsigned)((n_img + ST_BM - 1) / ST_BM), (unsigned)gy), 256, 0, st>>>(images, n_img, slices, M, P, mask, keys, (uint32_t)m_base);
        SPF_LAUNCH_CHECK(ctx);
        if ((rc = spf_record_event(ctx, 3, st))) return rc;
        ctx->last_scal = scal; ctx->last_match_stream = st;
        ctx->ev_valid[1] = ctx->ev_valid[2] = ctx->opt_record_events != 0;
        return SPF_OK;
    }
    // a6: common vector, abs-max of both operands (images raw, slices minus c), two-term fp16 split, a_i and b_m
    const int rb = ctx->sm_count * 8;
    if (first) {
        SPF_CUDA(ctx, cudaMemsetAsync(cvec, 0, (size_t)L.Ppad * 4, st));
        k_common_vector<<<(unsigned)((P + 255) / 256), 256, 0, st>>>(slices, M, P, mask, ctx->opt_match_condition, cvec);
        SPF_LAUNCH_CHECK(ctx);
        k_absmax<<<(unsigned)(n_img < rb ? n_img : rb), 256, 0, st>>>(images, n_img, P, mask, cvec, 0, scal + 0);
        SPF_LAUNCH_CHECK(ctx);
        k_split<<<(unsigned)n_img, 256, 0, st>>>(images, P, L.Ppad, mask, cvec, scal, 0, n_img, plI, aI, keys);
        SPF_LAUNCH_CHECK(ctx);
    }
    k_absmax<<<(unsigned)(M < rb ? M : rb), 256, 0, st>>>(slices, M, P, mask, cvec, 1, scal + 1);
    SPF_LAUNCH_CHECK(ctx);
    k_split<<<(unsigned)M, 256, 0, st>>>(slices, P, L.Ppad, mask, cvec, scal, 1, M, plS, bS, nullptr);
    SPF_LAUNCH_CHECK(ctx);

    if (ctx->opt_match_impl == 2) {
        // the warp-level tensor-core matcher (mma.sync): same operand planes, one block per 128 x 128 tile, image tiles fastest
        MatchArgs args{};
        args.n_img = n_img; args.M = M; args.kblocks = (int)(L.Ppad / BK);
        args.n_ib = (int)((n_img + MM_BM - 1) / MM_BM); args.n_mb = (int)((M + MM_BN - 1) / MM_BN);
        args.m_base = (uint32_t)m_base;
        args.chunk_kb = ctx->opt_match_chunk_kb > 0 ? ctx->opt_match_chunk_kb : args.kblocks;
        args.keys = keys; args.aI = aI; args.bS = bS; args.scal = scal; args.fault = ctx->d_fault; args.abort_flag = ctx->d_abort;
        if ((int64_t)args.n_ib * args.n_mb > 0x7fffffffLL) return spf_set_err(ctx, SPF_EINVAL, "spf_match: too many tiles");
        const unsigned grid = (unsigned)(args.n_ib * args.n_mb);
        auto mma1 = k_match_mma<1>, mma2 = k_match_mma<2>;
        SPF_CUDA(ctx, cudaFuncSetAttribute(mma1, cudaFuncAttributeMaxDynamicSharedMemorySize, MmaCfg<1>::SMEM_BYTES));
        SPF_CUDA(ctx, cudaFuncSetAttribute(mma2, cudaFuncAttributeMaxDynamicSharedMemorySize, MmaCfg<2>::SMEM_BYTES));
        if ((rc = spf_record_event(ctx, 2, st))) return rc;
        mma1<<<grid, MM_THREADS, MmaCfg<1>::SMEM_BYTES, st>>>(plI, plS, L.Ppad, args);
        SPF_LAUNCH_CHECK(ctx);
        mma2<<<grid, MM_THREADS, MmaCfg<2>::SMEM_BYTES, st>>>(plI, plS, L.Ppad, args);
        SPF_LAUNCH_CHECK(ctx);
        if ((rc = spf_record_event(ctx, 3, st))) return rc;
        ctx->last_scal = scal; ctx->last_match_stream = st;
        ctx->ev_valid[1] = ctx->ev_valid[2] = ctx->opt_record_events != 0;
        return SPF_OK;
    }
    const int CG = ctx->opt_match_cta_group;
    CUtensorMap a0, a1, b0, b1;
    if ((rc = encode_operand_map(ctx, &a0, plI, n_img, L.Ppad, TILE_ROWS))) return rc;
    if ((rc = encode_operand_map(ctx, &a1, plI + (size_t)n_img * L.Ppad, n_img, L.Ppad, TILE_ROWS))) return rc;
    if ((rc = encode_operand_map(ctx, &b0, plS, M, L.Ppad, BN / CG))) return rc;
    if ((rc = encode_operand_map(ctx, &b1, plS + (size_t)M * L.Ppad, M, L.Ppad, BN / CG))) return rc;
    MatchArgs args{};
    args.n_img = n_img; args.M = M; args.kblocks = (int)(L.Ppad / BK);
    args.n_ib = (int)((n_img + TILE_ROWS * CG - 1) / (TILE_ROWS * CG));
    args.n_mb = (int)((M + BN - 1) / BN);
    args.m_base = (uint32_t)m_base;
    args.chunk_kb = ctx->opt_match_chunk_kb > 0 ? ctx->opt_match_chunk_kb : args.kblocks;   // 0 = the whole of K in TMEM
    args.keys = keys; args.aI = aI; args.bS = bS; args.scal = scal; args.fault = ctx->d_fault; args.abort_flag = ctx->d_abort;
    if ((int64_t)args.n_ib * args.n_mb > 0x7fffffffLL) return spf_set_err(ctx, SPF_EINVAL, "spf_match: too many tiles");
    if ((rc = spf_record_event(ctx, 2, st))) return rc;
    if (CG == 2) {
        if ((rc = launch_gemm<2, 1>(ctx, a0, a1, b0, b1, args, st))) return rc;
        if ((rc = launch_gemm<2, 2>(ctx, a0, a1, b0, b1, args, st))) return rc;
    } else {
        if ((rc = launch_gemm<1, 1>(ctx, a0, a1, b0, b1, args, st))) return rc;
        if ((rc = launch_gemm<1, 2>(ctx, a0, a1, b0, b1, args, st))) return rc;
    }
    if ((rc = spf_record_event(ctx, 3, st))) return rc;
    ctx->last_scal = scal; ctx->last_match_stream = st;
    ctx->ev_valid[1] = ctx->ev_valid[2] = ctx->opt_record_events != 0;
    return SPF_OK;
}

static int check_match_args(spf_ctx *ctx, const char *who, const void *images, int64_t n_img, int64_t M, int64_t P, const void *bi,
                            const void *bd, const void *workspace) {
    if (n_img < 0 || M < 0 || P < 0) return spf_set_err(ctx, SPF_EINVAL, "%s: negative size", who);
    if (n_img == 0) return SPF_OK;
    if (M < 1 || P < 1) return spf_set_err(ctx, SPF_EINVAL, "%s: M and P must be >= 1 when n_img >= 1", who);
    if (!images || !bi || !bd || !workspace) return spf_set_err(ctx, SPF_EINVAL, "%s: null pointer", who);
    if (M > 0x7fffffffLL || n_img > 0x7fffffffLL) return spf_set_err(ctx, SPF_EINVAL, "%s: more than 2^31-1 rows", who);
    if (((uintptr_t)workspace & 1023u) != 0) return spf_set_err(ctx, SPF_EINVAL, "%s: workspace must be 1024-byte aligned", who);
    return SPF_OK;
}

int spf_match(spf_ctx *ctx, const float *images, int64_t n_img, const float *slices, int64_t M, int64_t P,
              const uint8_t *mask, int32_t *best_idx, float *best_dist, void *workspace, size_t workspace_bytes,
              void *stream_) {
    if (!ctx) return SPF_EINVAL;
    int rc = check_match_args(ctx, "spf_match", images, n_img, M, P, best_idx, best_dist, workspace);
    if (rc || n_img == 0) return rc;
    if (!slices) return spf_set_err(ctx, SPF_EINVAL, "spf_match: null pointer");
    const WsLayout L = ws_layout(n_img, M, P);
    if (workspace_bytes < L.total) return spf_set_err(ctx, SPF_EINVAL, "spf_match: workspace %zu < required %zu bytes", workspace_bytes, L.total);
    cudaStream_t st = (cudaStream_t)stream_;
    SPF_CUDA(ctx, cudaSetDevice(ctx->prm.device));
    if ((rc = match_pass(ctx, images, n_img, slices, M, P, mask, workspace, L, st, 0, true))) return rc;
    unsigned long long *keys = (unsigned long long *)((uint8_t *)workspace + L.keys);
    k_match_finalize<<<(unsigned)((n_img + 255) / 256), 256, 0, st>>>(keys, n_img, best_idx, best_dist);
    SPF_LAUNCH_CHECK(ctx);
    if (ctx->opt_match_impl != 1 && ctx->opt_match_refine) {
        k_match_refine<<<(unsigned)n_img, 256, 0, st>>>(images, slices, M, P, mask, best_idx, best_dist, 0);
        SPF_LAUNCH_CHECK(ctx);
    }
    return SPF_OK;
}

// ------------------------------------------------------------------------------------------
// slices produced in chunks of chunk_M orientations and consumed by the matcher at once,
// so the [M][P] slice array never exists (26 GB at Matching-heavy, 79 GB for the paper-shaped workload)
// ------------------------------------------------------------------------------------------
__global__ void k_gather_quats(const float *__restrict__ quats, const int32_t *__restrict__ best_idx, int64_t n, int64_t M,
                               float *__restrict__ out) {
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    int64_t m = best_idx[i];
    if (m < 0 || m >= M) m = 0;   // no winner: any valid orientation (k_match_refine skips the row)
    for (int c = 0; c < 4; ++c) out[4 * i + c] = quats[4 * m + c];
}

struct StreamLayout { WsLayout match; size_t chunk_slices, quats, total; };
static StreamLayout stream_layout(int64_t n_img, int64_t chunk_M, int64_t P) {
    StreamLayout S{};
    S.match = ws_layout(n_img, chunk_M, P);
    size_t off = S.match.total;
    S.chunk_slices = off; off += rup((size_t)chunk_M * P * 4, 1024);
    S.quats = off; off += rup((size_t)chunk_M * 16, 1024);
    S.total = off;
    return S;
}

size_t spf_slice_match_workspace_bytes(int64_t n_img, int64_t chunk_M, int64_t P) {
    if (n_img < 0 || chunk_M < 1 || P < 0) return 0;
    return stream_layout(n_img, chunk_M, P).total;
}

int spf_slice_match(spf_ctx *ctx, const float *quats, int64_t M, const float *pix_q, int64_t P, float scale, const float *images,
                    int64_t n_img, const uint8_t *mask, int64_t chunk_M, int32_t *best_idx, float *best_dist, void *workspace,
                    size_t workspace_bytes, void *stream_) {
    if (!ctx) return SPF_EINVAL;
    int rc = check_match_args(ctx, "spf_slice_match", images, n_img, M, P, best_idx, best_dist, workspace);
    if (rc || n_img == 0) return rc;
    if (!quats || !pix_q) return spf_set_err(ctx, SPF_EINVAL, "spf_slice_match: null pointer");
    if (chunk_M < 1) return spf_set_err(ctx, SPF_EINVAL, "spf_slice_match: chunk_M must be >= 1");
    if (chunk_M > M) chunk_M = M;
    const StreamLayout S = stream_layout(n_img, chunk_M, P);
    if (workspace_bytes < S.total) return spf_set_err(ctx, SPF_EINVAL, "spf_slice_match: workspace %zu < required %zu bytes", workspace_bytes, S.total);
    cudaStream_t st = (cudaStream_t)stream_;
    SPF_CUDA(ctx, cudaSetDevice(ctx->prm.device));
    uint8_t *ws = (uint8_t *)workspace;
    float *chunk = (float *)(ws + S.chunk_slices), *wq = (float *)(ws + S.quats);
    for (int64_t m0 = 0; m0 < M; m0 += chunk_M) {
        const int64_t Mc = M - m0 < chunk_M ? M - m0 : chunk_M;
        if ((rc = spf_slice(ctx, quats + 4 * m0, Mc, pix_q, P, SPF_OUT_INTENSITY, scale, chunk, st))) return rc;
        if ((rc = match_pass(ctx, images, n_img, chunk, Mc, P, mask, workspace, S.match, st, m0, m0 == 0))) return rc;
    }
    unsigned long long *keys = (unsigned long long *)(ws + S.match.keys);
    k_match_finalize<<<(unsigned)((n_img + 255) / 256), 256, 0, st>>>(keys, n_img, best_idx, best_dist);
    SPF_LAUNCH_CHECK(ctx);
    if (ctx->opt_match_impl != 1 && ctx->opt_match_refine) {
        // the winners' slices no longer exist: slice them again, chunk_M images at a time (n_img x P points in all)
        for (int64_t i0 = 0; i0 < n_img; i0 += chunk_M) {
            const int64_t nc = n_img - i0 < chunk_M ? n_img - i0 : chunk_M;
            k_gather_quats<<<(unsigned)((nc + 127) / 128), 128, 0, st>>>(quats, best_idx + i0, nc, M, wq);
            SPF_LAUNCH_CHECK(ctx);
            if ((rc = spf_slice(ctx, wq, nc, pix_q, P, SPF_OUT_INTENSITY, scale, chunk, st))) return rc;
            k_match_refine<<<(unsigned)nc, 256, 0, st>>>(images + i0 * P, chunk, nc, P, mask, best_idx + i0, best_dist + i0, 1);
            SPF_LAUNCH_CHECK(ctx);
        }
    }
    return SPF_OK;
}

int spf_last_match_products(spf_ctx *ctx, int32_t *products) {
    if (!ctx || !products) return SPF_EINVAL;
    if (!ctx->last_scal) return spf_set_err(ctx, SPF_ESTATE, "spf_last_match_products before spf_match");
    uint32_t two_planes = 0;
    if (ctx->last_match_impl == 1) { *products = 0; return SPF_OK; }   // CUDA-core matcher: no tensor-core products
    SPF_CUDA(ctx, cudaStreamSynchronize(ctx->last_match_stream));
    SPF_CUDA(ctx, cudaMemcpy(&two_planes, ctx->last_scal + 2, sizeof two_planes, cudaMemcpyDeviceToHost));
    *products = two_planes ? 3 : 2;
    return SPF_OK;
}

int spf_match_reference(spf_ctx *ctx, const float *images, int64_t n_img, const float *slices, int64_t M, int64_t P,
                        const uint8_t *mask, int32_t *best_idx, float *best_dist, float *dist, void *stream_) {
    if (!ctx) return SPF_EINVAL;
    if (n_img < 0 || M < 0 || P < 0) return spf_set_err(ctx, SPF_EINVAL, "spf_match_reference: negative size");
    if (n_img == 0) return SPF_OK;
    if (M < 1 || P < 1) return spf_set_err(ctx, SPF_EINVAL, "spf_match_reference: M and P must be >= 1");
    if (!images || !slices || !best_idx || !best_dist || !dist) return spf_set_err(ctx, SPF_EINVAL, "spf_match_reference: null pointer");
    if (n_img * M > 0x7fffffffLL) return spf_set_err(ctx, SPF_EINVAL, "spf_match_reference: n_img*M too large (tests only)");
    cudaStream_t st = (cudaStream_t)stream_;
    SPF_CUDA(ctx, cudaSetDevice(ctx->prm.device));
    k_match_ref_dist<<<(unsigned)(n_img * M), 256, 0, st>>>(images, n_img, slices, M, P, mask, dist);
    SPF_LAUNCH_CHECK(ctx);
    k_match_ref_argmin<<<(unsigned)((n_img + 127) / 128), 128, 0, st>>>(dist, n_img, M, best_idx, best_dist);
    SPF_LAUNCH_CHECK(ctx);
    return SPF_OK;
}

}  // extern "C"
