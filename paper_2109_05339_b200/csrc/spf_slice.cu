// libspf: spf_slice (steps a3-a5 of SURVEY.md section 8(a)).
//
//   c_{m,j} ~= sum_{t1,t2,t3 < w} b[i0 + t] phi1[t1] phi2[t2] phi3[t3],   x = R(quat_m) q_j,  xi = x n_f / 2 pi,
//   i0 = ceil(xi - w/2),  phi_d[t] = phi(2 (i0_d + t - xi_d) / w),  phi(z) = exp(beta (sqrt(1 - z^2) - 1))
//
// One thread block = one orientation x one compact patch of SPF_PATCH detector pixels (an 8 x 16
// lattice tile when the caller promised a panel layout).  The rotated patch is a small tilted
// piece of a plane in the fine grid, so its axis-aligned bounding box is a small regular 3-D
// tile: the block finds the box with a min/max reduction, one warp issues one TMA tensor copy per
// x-plane of the box into shared memory, and while those are in flight every thread evaluates
// its 3 w kernel weights (piecewise polynomials, Horner).  The gather then reads shared memory
// only.  The stored grid is centred with a periodic halo (spf_prepare_model), so there is no
// modulo anywhere, and it is real fp32 when the model is even -- half the bytes per neighbour.
// Coordinates (rotation, scaling to cells, split into integer cell + fraction) are fp64: an fp32
// error of one ulp at |xi| ~ 150 cells is 1.5e-5 cells, which a model that fills the grid turns
// into a 1e-5 relative error, the whole parity budget.
#include <assert.h>
#include <limits.h>
#include <math.h>

#include <type_traits>
#include <vector>

#include "ptx_sm100.cuh"
#include "spf_internal.cuh"
#include "spf_slice_math.cuh"

namespace {

struct SliceArgs {
    const float *quats, *pix_q;
    const int32_t *patch;   // [n_patches][SPF_PATCH]
    int64_t M, P, n_patches;
    void *out;
    float scale;
    const float *grid;      // centred padded grid, fp32 (REAL) or interleaved complex
    int np, sz, off, nf, w, deg;
    double xi_scale;        // n_f / (2 pi)
    double inv_nf;
    float beta;
    uint32_t cap_bytes;     // dynamic shared memory available for the tile
    int stage_mode;         // IMPL_COOP: 0 = tile staged by TMA (bulk tensor copies + mbarrier), 1 = by cp.async (classic CUDA)
    uint32_t *fault;        // context fault record (host-mapped): written when the tile wait gives up
    uint32_t *abort_flag;   // context abort flag (device memory): set by the first wait that gives up, read by every block
    float coef[SPF_MAX_W][SPF_MAX_DEG + 1];  // phi at tap t as a polynomial in u = 2 (f + w/2) - 1
    SliceMaps maps;
};

template <int OUTK>
__device__ __forceinline__ void store_out(const SliceArgs &a, int64_t m, int64_t j, spfm::c2 c) {
    if (OUTK == SPF_OUT_COMPLEX) reinterpret_cast<float2 *>(a.out)[m * a.P + j] = make_float2(c.x, c.y);
    else reinterpret_cast<float *>(a.out)[m * a.P + j] = a.scale * c.x;
}

// Kernel variants (option "slice_impl"):
//   IMPL_GLOBAL  1  one thread per point, w^3 loads straight from the grid in global memory (L1/L2): the
//                   reference gather (the definition written out), and the library's starting variant
//   IMPL_COOP    2  tile staged by TMA, a WARP gathers each point: lane (h, k) reads rows h, h + 4 and
//                   cell k of the point's 8 x 8 window in every x-plane -- 32 consecutive-bank words per
//                   load, no bank conflicts (spf_slice_math.cuh) -- and a shuffle tree adds the 32
//                   partial sums: 14 conflict-free loads + 4 weight loads per point.  Blocks whose box does
//                   not fit the tile, and every block at w > 8, walk the grid in global memory instead
//                   (the IMPL_GCOOP path below).
//   IMPL_GCOOP   3  the same warp-per-point walk straight from the grid in global memory: no TMA, no
//                   mbarrier, no tile -- each load is four 32-byte row segments instead of 32 scattered words
// (A TMA-staged one-thread-per-point form existed in round 1 as variant 0.  With one thread per point the 32 lanes
// of a warp are scattered over the tile and every load replays ~3.8 times on bank conflicts -- 41 wavefronts per
// point against 18 here, tests/test_hostsim_slice_math.py::test_bank_conflicts... -- so it could not reach half of
// the shared-memory roofline by construction and was deleted.)
//   IMPL_COOP_LD 4  IMPL_COOP's kernel with the tile staged by cp.async (16-byte pieces, every thread copies) instead of
//                   TMA: Ampere-style classic CUDA, no tensor map, no mbarrier -- the staged gather for a device on which
//                   the TMA path has not been cleared.  The box starts at a multiple of 4 cells along z (16-byte pieces).
enum { IMPL_GLOBAL = 1, IMPL_COOP = 2, IMPL_GCOOP = 3, IMPL_COOP_LD = 4 };
#define SPF_COOP_WTS_BYTES (SPF_PATCH * SPF_COOP_STRIDE * 4)   // 14,336 = 112 x 128

// The cooperative gather of one warp over its 32 points (variants 2 and 3).  `tile` is the staged box in
// shared memory (IDX = int, BZ = its row pitch) or the whole padded grid in global memory (IDX = long
// long, BZ = 0: row pitch `bz` at run time); `cell` is this lane's own point's first cell (< 0: none);
// `wts_warp` the warp's 32 parked weight sets.  Points go in groups of 8: eight independent gathers in
// flight per lane, then ONE multi-value butterfly (spf_slice_math.cuh: 4 + 2 + 1 exchanges halve the
// value count while halving the lane group, 2 more finish) instead of eight 5-step reductions; lane
// 4 u ends with point u's sum and the owner lanes fetch theirs.
template <bool REAL, int BZ, typename IDX, bool WIDE = false>
__device__ __forceinline__ void coop_sweep(const float *tile, IDX cell, int S1, int bz, int w, const float *wts_warp, int lane,
                                           spfm::c2 &c) {
    constexpr int STRIDE = WIDE ? SPF_COOPW_STRIDE : SPF_COOP_STRIDE;
    const int h = lane >> 3, k = lane & 7;
    for (int g0 = 0; g0 < 32; g0 += spfm::MR8) {
        float pr[spfm::MR8], pi[spfm::MR8];
#pragma unroll
        for (int u = 0; u < spfm::MR8; ++u) {
            const IDX cell_p = __shfl_sync(0xffffffffu, cell, g0 + u);
            spfm::c2 part; part.x = part.y = 0.0f;
            if (cell_p >= 0) {  // warp-uniform: skips an empty slot of a ragged patch
                if (WIDE) part = spfm::gather_coop_lane_wide<REAL, IDX>(tile, cell_p, S1, bz, w, wts_warp + (g0 + u) * STRIDE, lane);
                else part = spfm::gather_coop_lane<REAL, BZ, IDX>(tile, cell_p, S1, bz, w, wts_warp + (g0 + u) * STRIDE, h, k);
            }
            pr[u] = part.x; pi[u] = part.y;
        }
#pragma unroll
        for (int o = 16, n = spfm::MR8 / 2; n >= 1; o >>= 1, n >>= 1) {
            const bool upper = (lane & o) != 0;
#pragma unroll
            for (int v = 0; v < n; ++v) {
                const float keep_r = upper ? pr[v + n] : pr[v], send_r = upper ? pr[v] : pr[v + n];
                pr[v] = keep_r + __shfl_xor_sync(0xffffffffu, send_r, o);
                if (!REAL) {
                    const float keep_i = upper ? pi[v + n] : pi[v], send_i = upper ? pi[v] : pi[v + n];
                    pi[v] = keep_i + __shfl_xor_sync(0xffffffffu, send_i, o);
                }
            }
        }
#pragma unroll
        for (int o = 2; o >= 1; o >>= 1) {
            pr[0] += __shfl_xor_sync(0xffffffffu, pr[0], o);
            if (!REAL) pi[0] += __shfl_xor_sync(0xffffffffu, pi[0], o);
        }
        // the lanes g0 .. g0 + 7 own these points; point u's sum sits in lane mr8_result_lane(u)
        const float vr = __shfl_sync(0xffffffffu, pr[0], spfm::mr8_result_lane(lane & (spfm::MR8 - 1)));
        const float vi = REAL ? 0.0f : __shfl_sync(0xffffffffu, pi[0], spfm::mr8_result_lane(lane & (spfm::MR8 - 1)));
        if ((lane & ~(spfm::MR8 - 1)) == g0) { c.x = vr; c.y = vi; }
    }
}

// W = 0: runtime kernel width (any w <= SPF_MAX_W), else compile-time.
template <int W, bool REAL, int OUTK, int IMPL>
__global__ void __launch_bounds__(SPF_PATCH, (IMPL == IMPL_GLOBAL || IMPL == IMPL_GCOOP) ? 4 : 3) k_slice(const __grid_constant__ SliceArgs a) {
    constexpr bool STAGED = (IMPL == IMPL_COOP);
    constexpr bool COOP = (IMPL == IMPL_COOP);
    constexpr bool GCOOP = (IMPL == IMPL_GCOOP);
    constexpr bool WIDE = GCOOP && W > 8;      // 16-cell window, global memory only (spf_slice_math.cuh)
    static_assert(!COOP || (W >= 2 && W <= 8), "the staged cooperative gather reads an 8 x 8 window per x-plane");
    static_assert(!GCOOP || (W >= 2 && W <= 12), "the cooperative gather handles 2 <= w <= 12");
    constexpr int WSTRIDE = WIDE ? SPF_COOPW_STRIDE : SPF_COOP_STRIDE;
    constexpr int WMAX = W ? W : SPF_MAX_W;
    constexpr int E = REAL ? 1 : 2;            // floats per cell
    constexpr int CELL = 4 * E;                // bytes per cell
    const int w = W ? W : a.w;
    const int tid = threadIdx.x;
    // one stalled tile costs one time-out, not one per block: blocks that start after a give-up leave at once
    if (STAGED && *reinterpret_cast<volatile uint32_t *>(a.abort_flag)) return;
    const int64_t m = blockIdx.x / a.n_patches;
    const int64_t patch = blockIdx.x - m * a.n_patches;

    __shared__ double sR[9];
    __shared__ int s_lo[3], s_hi[3];
    __shared__ __align__(8) unsigned long long s_bar;
    __shared__ uint32_t s_abort;
    extern __shared__ __align__(128) uint8_t s_dyn[];
    // cooperative variant: the first SPF_COOP_WTS_BYTES of dynamic shared memory hold the points' weights
    uint8_t *s_tile = s_dyn + (COOP ? SPF_COOP_WTS_BYTES : 0);

    if (tid == 0) {
        spfm::quat_to_R(a.quats + 4 * m, sR);
        s_lo[0] = s_lo[1] = s_lo[2] = INT_MAX;
        s_hi[0] = s_hi[1] = s_hi[2] = INT_MIN;
        if (STAGED) { s_abort = 0u; ptx::mbar_init(ptx::smem_u32(&s_bar), 1); ptx::fence_mbar_init(); }
    }
    __syncthreads();

    const int64_t j = a.patch[patch * SPF_PATCH + tid];
    const bool active = (j >= 0);
    int px = 0, py = 0, pz = 0;
    float fx = 0.f, fy = 0.f, fz = 0.f;
    if (active) {
        const double q0 = a.pix_q[3 * j + 0], q1 = a.pix_q[3 * j + 1], q2 = a.pix_q[3 * j + 2];
        spfm::cell_and_fraction(sR[0] * q0 + sR[1] * q1 + sR[2] * q2, a.xi_scale, a.inv_nf, a.nf, a.off, a.np, w, px, fx);
        spfm::cell_and_fraction(sR[3] * q0 + sR[4] * q1 + sR[5] * q2, a.xi_scale, a.inv_nf, a.nf, a.off, a.np, w, py, fy);
        spfm::cell_and_fraction(sR[6] * q0 + sR[7] * q1 + sR[8] * q2, a.xi_scale, a.inv_nf, a.nf, a.off, a.np, w, pz, fz);
    }

    bool staged = false;
    int lox = 0, loy = 0, loz = 0, bz = 0, S1 = 0;
    if (STAGED) {
        const int lx = __reduce_min_sync(0xffffffffu, active ? px : INT_MAX), hx = __reduce_max_sync(0xffffffffu, active ? px : INT_MIN);
        const int ly = __reduce_min_sync(0xffffffffu, active ? py : INT_MAX), hy = __reduce_max_sync(0xffffffffu, active ? py : INT_MIN);
        const int lz = __reduce_min_sync(0xffffffffu, active ? pz : INT_MAX), hz = __reduce_max_sync(0xffffffffu, active ? pz : INT_MIN);
        if ((tid & 31) == 0) {
            atomicMin(&s_lo[0], lx); atomicMax(&s_hi[0], hx);
            atomicMin(&s_lo[1], ly); atomicMax(&s_hi[1], hy);
            atomicMin(&s_lo[2], lz); atomicMax(&s_hi[2], hz);
        }
        __syncthreads();
        lox = s_lo[0]; loy = s_lo[1]; loz = s_lo[2];
        // cp.async staging copies 16-byte pieces: the box starts at a multiple of 4 cells along z (rows of the padded grid
        // are 16-byte aligned: sz is a multiple of 4), at most 3 cells wider than the tight box
        if (a.stage_mode == 1) loz &= ~3;
        // a patch with no pixel at all (cannot happen with the tables build_patches makes) has lo > hi: not staged
        const bool any = s_hi[0] >= lox;
        const int Lx = any ? s_hi[0] - lox + w : 0, Ly = any ? s_hi[1] - loy + w : 0, Lz = any ? s_hi[2] - loz + w : 0;
        const spfm::TileGeom g = spfm::tile_geom(Lx, Ly, Lz, w, CELL, a.cap_bytes);
        bz = g.bz; S1 = g.S1;
        staged = g.ok;
#ifdef SPF_DEBUG
        // invariants of the bulk tensor copies: 128-byte aligned destinations, the box
        // inside the tile capacity, a box size that is on the tensor-map menu, transaction bytes below 2^20
        if (staged && tid == 0) {
            assert((ptx::smem_u32(s_tile) & 127u) == 0u && ((uint32_t)(S1 * CELL) & 127u) == 0u);
            assert((uint32_t)(Lx * S1 * CELL) <= a.cap_bytes && (uint32_t)(Lx * g.by * bz * CELL) < (1u << 20));
            assert(g.by >= SPF_BOX_MIN && g.by <= SPF_BOX_MAX && bz >= SPF_BOX_MIN && bz <= SPF_BOX_MAX);
            assert(g.by % SPF_BOX_STEP == 0 && bz % SPF_BOX_STEP == 0 && g.by * bz <= S1);
            assert(lox >= 0 && loy >= 0 && loz >= 0 && lox + Lx <= a.np && loy + Ly <= a.np && loz + Lz <= a.sz);
        }
#endif
        if (staged && a.stage_mode == 1) {
            // classic staging: every thread copies 16-byte pieces of the box, row by row (a warp covers 512 consecutive
            // bytes of a row or of neighbouring rows); pieces beyond the grid (rows >= np, cells >= sz) are zero-filled,
            // which is what the TMA path's out-of-bounds fill gives
            const int q_per_row = bz * E / 4, pieces = Lx * g.by * q_per_row;
            const uint32_t dst0 = ptx::smem_u32(s_tile);
            for (int idx = tid; idx < pieces; idx += SPF_PATCH) {
                const int q = idx % q_per_row, y = (idx / q_per_row) % g.by, x = idx / (q_per_row * g.by);
                const uint32_t dst = dst0 + (uint32_t)(((x * S1 + y * bz) * E + 4 * q) * 4);
                const int gy = loy + y, gz4 = loz * E + 4 * q;
                if (gy < a.np && gz4 + 3 < a.sz * E)
                    ptx::cp_async_16(dst, a.grid + ((size_t)((size_t)(lox + x) * a.np + gy) * a.sz) * E + gz4);
                else
                    *reinterpret_cast<float4 *>(s_tile + (dst - dst0)) = make_float4(0.f, 0.f, 0.f, 0.f);
            }
        } else if (staged && tid < 32) {
            const uint32_t bar = ptx::smem_u32(&s_bar);
            if (tid == 0) ptx::mbar_expect_tx(bar, (uint32_t)(Lx * g.by * bz * CELL));
            __syncwarp();
            const CUtensorMap *map = &a.maps.m[spfm::tile_map_index(g.by, bz)];
            const uint32_t dst = ptx::smem_u32(s_tile);
            for (int x = tid; x < Lx; x += 32)
                ptx::tma_load_3d(dst + (uint32_t)(x * S1 * CELL), map, loz * E, loy, lox + x, bar);
        }
    }

    // kernel weights while the tile is in flight
    float wx[WMAX], wy[WMAX], wz[WMAX];
    if (STAGED || GCOOP) {
        spfm::weights_poly<WMAX>(fx, w, a.coef, a.deg, wx); spfm::weights_poly<WMAX>(fy, w, a.coef, a.deg, wy);
        spfm::weights_poly<WMAX>(fz, w, a.coef, a.deg, wz);
    } else {
        spfm::weights_direct<WMAX>(fx, w, a.beta, wx); spfm::weights_direct<WMAX>(fy, w, a.beta, wy);
        spfm::weights_direct<WMAX>(fz, w, a.beta, wz);
    }

    spfm::c2 c;
    c.x = c.y = 0.0f;
    const int lane = tid & 31;
    const float *wts_warp = reinterpret_cast<const float *>(s_dyn) + (tid & ~31) * WSTRIDE;
    if (COOP || GCOOP) {
        // every lane parks its point's weights where its warp will read them back
        float4 *dst4 = reinterpret_cast<float4 *>(reinterpret_cast<float *>(s_dyn) + tid * WSTRIDE);
        if (WIDE) {
            float pk[44];
            spfm::coop_pack_weights_wide<WMAX>(pk, w, wx, wy, wz);
#pragma unroll
            for (int v = 0; v < 11; ++v) dst4[v] = make_float4(pk[4 * v], pk[4 * v + 1], pk[4 * v + 2], pk[4 * v + 3]);
        } else {
            float pk[24];
            spfm::coop_pack_weights<WMAX>(pk, w, wx, wy, wz);
#pragma unroll
            for (int v = 0; v < 6; ++v) dst4[v] = make_float4(pk[4 * v], pk[4 * v + 1], pk[4 * v + 2], pk[4 * v + 3]);
        }
        __syncwarp();
    }
    if (STAGED && staged && a.stage_mode == 1) {
        ptx::cp_async_wait_all();
        __syncthreads();          // every thread's pieces have landed
    }
    if (STAGED && staged) {
        if (a.stage_mode == 0 && !ptx::mbar_wait(ptx::smem_u32(&s_bar), 0, &s_abort, a.abort_flag)) {
            if (tid == 0) {
                a.fault[1] = blockIdx.x; a.fault[2] = (uint32_t)patch; a.fault[3] = (uint32_t)(W * 10 + (REAL ? 1 : 0) + 100 * IMPL);
                a.fault[0] = SPF_FAULT_SLICE;
                __threadfence_system();
            }
            ptx::abort_drain();   // bulk copies still in flight must land before this shared memory goes to the next block
            return;
        }
        const float *tile = reinterpret_cast<const float *>(s_tile);
        const int cell = active ? (px - lox) * S1 + (py - loy) * bz + (pz - loz) : -1;
        // bz is 8, 24 or 40 (tile_geom): one loop per value, so the row offsets are immediates
        if (bz == 24) coop_sweep<REAL, 24, int>(tile, cell, S1, bz, w, wts_warp, lane, c);
        else if (bz == 8) coop_sweep<REAL, 8, int>(tile, cell, S1, bz, w, wts_warp, lane, c);
        else coop_sweep<REAL, 40, int>(tile, cell, S1, bz, w, wts_warp, lane, c);
        if (!active) return;
    } else if (COOP || GCOOP) {
        // the same warp-per-point walk straight from the padded grid (L1/L2): variant 3, and the blocks of
        // variant 2 whose box does not fit the tile.  The 8 x 8 window reads one row and one cell past the
        // w taps (weight 0): for finite input the last first-cell is np - 8 (spf_slice_math.cuh), so the
        // window ends at np - 1; the clamp only acts on the NaN / inf inputs cell_and_fraction parks at np - w.
        // The wide form (w > 8) reads exactly the w x w taps: no clamp needed.
        const int qy = WIDE ? py : min(py, a.np - 8), qz = WIDE ? pz : min(pz, a.np - 8);
        const long long cell = active ? ((long long)px * a.np + qy) * a.sz + qz : -1;
        coop_sweep<REAL, 0, long long, WIDE>(a.grid, cell, a.np * a.sz, a.sz, w, wts_warp, lane, c);
        if (!active) return;
    } else {
        if (!active) return;
        const float *base = a.grid + ((size_t)((size_t)px * a.np + py) * a.sz + pz) * E;
        c = spfm::gather<WMAX, REAL>(base, a.np * a.sz, a.sz, w, wx, wy, wz);
    }
    store_out<OUTK>(a, m, j, c);
}

// ------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------
// pixel -> patch table: 8 x 16 lattice tiles per panel under a layout promise, else runs of SPF_PATCH pixels
int build_patches(spf_ctx *ctx, int64_t P) {
    const bool lattice = ctx->lay_panels > 0 && (int64_t)ctx->lay_panels * ctx->lay_rows * ctx->lay_cols == P;
    const int key[3] = {lattice ? ctx->lay_panels : 0, lattice ? ctx->lay_rows : 0, lattice ? ctx->lay_cols : 0};
    if (ctx->d_patch && ctx->patch_P == P && !memcmp(key, ctx->patch_key, sizeof key)) return SPF_OK;
    static_assert(SPF_PATCH == SPF_PATCH_PIXELS, "block size = pixels per patch");
    std::vector<int32_t> tab;
    spfm::build_patch_table(key[0], key[1], key[2], P, tab);
    if (ctx->d_patch) { cudaFree(ctx->d_patch); ctx->d_patch = nullptr; }
    SPF_CUDA(ctx, cudaMalloc(&ctx->d_patch, tab.size() * sizeof(int32_t)));
    SPF_CUDA(ctx, cudaMemcpy(ctx->d_patch, tab.data(), tab.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
    ctx->n_patches = (int64_t)(tab.size() / SPF_PATCH);
    ctx->patch_P = P;
    memcpy(ctx->patch_key, key, sizeof key);
    return SPF_OK;
}

template <int W, bool REAL, int OUTK, int IMPL>
int launch_slice(spf_ctx *ctx, SliceArgs &args, cudaStream_t st) {
    auto kern = k_slice<W, REAL, OUTK, IMPL>;
    // shared-memory tile capacity: 3 blocks per SM on the real grid, 2 on the complex grid (w = 8)
    uint32_t smem = 0;
    args.cap_bytes = 0;
    if (IMPL == IMPL_GCOOP) smem = W > 8 ? (uint32_t)(SPF_PATCH * SPF_COOPW_STRIDE * 4) : (uint32_t)SPF_COOP_WTS_BYTES;   // the parked weights only
    if (IMPL == IMPL_COOP) {
        args.cap_bytes = 48u * 1024u * (REAL ? 1u : 2u);
        smem = args.cap_bytes + (uint32_t)SPF_COOP_WTS_BYTES;
        SPF_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        // three (real grid) or two (complex grid) blocks per SM only fit with the largest shared-memory carve-out
        SPF_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared));
    }
    const int64_t blocks = args.n_patches * args.M;
    if (blocks > 0x7fffffffLL) return spf_set_err(ctx, SPF_EINVAL, "spf_slice: M * patches exceeds 2^31-1 blocks; split M");
    int rc = spf_record_event(ctx, 0, st);
    if (rc) return rc;
    kern<<<(unsigned)blocks, SPF_PATCH, smem, st>>>(args);
    SPF_LAUNCH_CHECK(ctx);
    if ((rc = spf_record_event(ctx, 1, st))) return rc;
    ctx->ev_valid[0] = ctx->opt_record_events != 0;
    return SPF_OK;
}

template <bool REAL, int OUTK>
int launch_slice_w(spf_ctx *ctx, SliceArgs &args, int impl, cudaStream_t st) {
    switch (ctx->w) {
        case 8:    // eps = 1e-6: the 8 x 8 window is exactly the kernel's footprint
            if (impl == IMPL_COOP || impl == IMPL_COOP_LD) return launch_slice<8, REAL, OUTK, IMPL_COOP>(ctx, args, st);
            if (impl == IMPL_GCOOP) return launch_slice<8, REAL, OUTK, IMPL_GCOOP>(ctx, args, st);
            return launch_slice<8, REAL, OUTK, IMPL_GLOBAL>(ctx, args, st);
        case 10:   // 10 x 10 window: the staged 8 x 8 form does not apply, variants 2 and 3 both walk global memory (16-cell window)
            if (impl == IMPL_COOP || impl == IMPL_COOP_LD || impl == IMPL_GCOOP) return launch_slice<10, REAL, OUTK, IMPL_GCOOP>(ctx, args, st);
            return launch_slice<10, REAL, OUTK, IMPL_GLOBAL>(ctx, args, st);
        default: return launch_slice<0, REAL, OUTK, IMPL_GLOBAL>(ctx, args, st);  // any other width: runtime-w global gather
    }
}

}  // namespace

extern "C" int spf_slice(spf_ctx *ctx, const float *quats, int64_t M, const float *pix_q, int64_t P, int32_t out_kind,
                         float scale, void *out, void *stream_) {
    if (!ctx) return SPF_EINVAL;
    if (M < 0 || P < 0) return spf_set_err(ctx, SPF_EINVAL, "spf_slice: negative size");
    if (out_kind != SPF_OUT_COMPLEX && out_kind != SPF_OUT_INTENSITY) return spf_set_err(ctx, SPF_EINVAL, "spf_slice: bad out_kind %d", out_kind);
    if (!ctx->prepared) return spf_set_err(ctx, SPF_ESTATE, "spf_slice before spf_prepare_model");
    if (M == 0 || P == 0) return SPF_OK;
    if (!quats || !pix_q || !out) return spf_set_err(ctx, SPF_EINVAL, "spf_slice: null pointer");
    if (P > 0x7fffffffLL) return spf_set_err(ctx, SPF_EINVAL, "spf_slice: P too large");
    cudaStream_t st = (cudaStream_t)stream_;
    SPF_CUDA(ctx, cudaSetDevice(ctx->prm.device));
    int rc = build_patches(ctx, P);
    if (rc) return rc;

    const bool real = ctx->grid_is_real && !ctx->opt_force_complex;
    static thread_local SliceArgs args;  // 11 KB: keep it off the stack
    args.quats = quats; args.pix_q = pix_q; args.patch = ctx->d_patch;
    args.M = M; args.P = P; args.n_patches = ctx->n_patches;
    args.out = out; args.scale = scale;
    args.grid = real ? ctx->d_gridr : reinterpret_cast<const float *>(ctx->d_gridc);
    args.np = ctx->np; args.sz = ctx->sz; args.off = ctx->nf / 2 + ctx->halo; args.nf = ctx->nf; args.w = ctx->w;
    args.xi_scale = (double)ctx->nf / (2.0 * M_PI);
    args.inv_nf = 1.0 / (double)ctx->nf;
    args.beta = (float)ctx->beta;
    args.deg = spfm::fit_kernel_polys(ctx->w, ctx->beta, args.coef);
    args.maps = real ? ctx->maps_r : ctx->maps_c;
    args.fault = ctx->d_fault; args.abort_flag = ctx->d_abort;
    args.stage_mode = ctx->opt_slice_impl == IMPL_COOP_LD ? 1 : 0;
    const int impl = ctx->opt_slice_impl;
    if (impl == IMPL_COOP && ctx->w <= 8 && !ctx->maps_ok)
        return spf_set_err(ctx, SPF_ECUDA, "spf_slice: slice_impl %d needs the TMA tensor maps, which could not be encoded: %s", impl,
                           ctx->maps_err.c_str());
    if (real) {
        return out_kind == SPF_OUT_COMPLEX ? launch_slice_w<true, SPF_OUT_COMPLEX>(ctx, args, impl, st)
                                           : launch_slice_w<true, SPF_OUT_INTENSITY>(ctx, args, impl, st);
    }
    return out_kind == SPF_OUT_COMPLEX ? launch_slice_w<false, SPF_OUT_COMPLEX>(ctx, args, impl, st)
                                       : launch_slice_w<false, SPF_OUT_INTENSITY>(ctx, args, impl, st);
}
