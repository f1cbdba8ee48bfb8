// Internal declarations of libspf (not part of the ABI).  sm_100a only.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cufft.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include <string>
#include <vector>

#include "../../include/spf.h"

#define SPF_MAX_W 16

#include "spf_slice_math.cuh"  // SPF_BOX_*: the menu of TMA box sizes (one tensor map per (by, bz) pair)
#include "spf_match_math.cuh"  // CHUNK_KB: default of option "match_chunk_kblocks"

struct SliceMaps {
    CUtensorMap m[SPF_BOX_N * SPF_BOX_N];  // [iy * SPF_BOX_N + iz]
};

struct spf_ctx {
    spf_params prm{};
    int n = 0, nf = 0, w = 0, halo = 0, np = 0;  // np: padded edge (x and y); sz: z pitch (>= np, multiple of 4)
    int sz = 0;
    double beta = 0.0;
    int sm_count = 0;
    bool prepared = false;
    bool grid_is_real = false;
    int opt_slice_impl = 1;       // conservative defaults until a variant has been checked on the device (spf.h)
    int opt_force_complex = 0;
    int opt_match_cta_group = 1;
    int opt_match_impl = 1;       // 1 = CUDA-core difference-form matcher, 0 = tcgen05 GEMM (spf.h)
    int last_match_impl = 1;
    int opt_match_chunk_kb = spfmm::CHUNK_KB;   // K blocks per accumulator drain of k_match_gemm (0 = whole K)
    int opt_match_condition = 1;                // 1 = subtract the common vector from the slices (spf_match_math.cuh)
    int opt_match_refine = 1;                   // 1 = recompute the winner's distance in the difference form
    int gemm_max_clusters[2][2] = {{0, 0}, {0, 0}};  // [CG - 1][NI - 1]: co-resident clusters of k_match_gemm, 0 = not asked yet
    int opt_record_events = 0;
    int opt_selftest_small = 0;                 // 1 = spf_selftest uses its small cases (quick checks, the emulator)
    float selftest_slice_ms = 0.f;              // time of the fastest slicer spf_selftest has verified and switched on (0: none yet)
    int64_t launches = 0;
    // CUDA events around the dominant kernels (option "record_events"): [0,1] slice kernel,
    // [2,3] match GEMM, [4] start of the match operand preparation (which ends at [2])
    cudaEvent_t ev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    bool ev_valid[3] = {false, false, false};
    const uint32_t *last_scal = nullptr;  // scalars block of the last spf_match's workspace (caller-owned memory)
    cudaStream_t last_match_stream = nullptr;

    std::vector<double> deapod;  // host, n entries
    float *d_deapod = nullptr;   // device fp32 copy (n)
    float2 *d_fft = nullptr;     // n_fine^3 complex, natural order (FFT in place)
    float2 *d_gridc = nullptr;   // np*np*sz complex, centred + halo
    float *d_gridr = nullptr;    // np*np*sz real, centred + halo (valid when grid_is_real)
    int *d_flag = nullptr;       // 1 int: model-not-even counter
    cufftHandle plan = 0;
    bool plan_ok = false;
    void *d_fft_work = nullptr;
    size_t fft_work_bytes = 0;

    // detector layout promise
    int lay_panels = 0, lay_rows = 0, lay_cols = 0;
    int32_t *d_patch = nullptr;  // [n_patches][SPF_PATCH] pixel indices, -1 = empty
    int64_t patch_P = -1;        // P the patch table was built for
    int patch_key[3] = {-1, -1, -1};
    int64_t n_patches = 0;

    SliceMaps maps_c{}, maps_r{};
    bool maps_ok = false;
    std::string maps_err;         // why the slice tensor maps could not be encoded (then only slice_impl 1 / 3 run)

    // host-buffer entry point: cached device buffers
    struct HostBufs {
        float *model = nullptr, *quats = nullptr, *pix = nullptr, *images = nullptr, *slices = nullptr, *bdist = nullptr;
        uint8_t *mask = nullptr;
        int32_t *bidx = nullptr;
        void *ws = nullptr;
        size_t cap_model = 0, cap_quats = 0, cap_pix = 0, cap_images = 0, cap_slices = 0, cap_mask = 0, cap_bi = 0, cap_bd = 0, cap_ws = 0;
        cudaStream_t s_main = nullptr, s_copy = nullptr;
        cudaEvent_t ev_img = nullptr;
    } hb;

    // watchdog fault record: 4 words of pinned, device-mapped host memory
    // [0] code (0 = none), [1] block, [2] tile / patch, [3] kernel variant
    volatile uint32_t *h_fault = nullptr;
    uint32_t *d_fault = nullptr;
    // device-global abort flag (device memory, 1 word): raised by the first pipeline wait that gives up, read by
    // every block at entry and inside every bounded wait; cleared by spf_check_fault
    uint32_t *d_abort = nullptr;

    std::string err;
};

#define SPF_FAULT_SLICE 16u  // k_slice: tile wait gave up
#define SPF_FAULT_MATCH 32u  // k_match_gemm: + 0 producer, 1 MMA (accumulator), 2 MMA (operands), 3 epilogue

#define SPF_PATCH 128  // threads per slicing block = pixels per patch

int spf_set_err(spf_ctx *ctx, int code, const char *fmt, ...);

#define SPF_CUDA(ctx, call)                                                                      \
    do {                                                                                         \
        cudaError_t e_ = (call);                                                                 \
        if (e_ != cudaSuccess)                                                                   \
            return spf_set_err((ctx), e_ == cudaErrorMemoryAllocation ? SPF_ENOMEM : SPF_ECUDA, \
                               "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

#define SPF_LAUNCH_CHECK(ctx)                                                                                   \
    do {                                                                                                        \
        cudaError_t e_ = cudaGetLastError();                                                                    \
        if (e_ != cudaSuccess)                                                                                  \
            return spf_set_err((ctx), SPF_ECUDA, "kernel launch failed: %s (%s:%d)", cudaGetErrorString(e_), __FILE__, \
                               __LINE__);                                                                       \
        (ctx)->launches++;                                                                                      \
    } while (0)

// driver entry point for cuTensorMapEncodeTiled fetched through the runtime (no -lcuda needed)
typedef CUresult (*spf_encode_tiled_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                        const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                        CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                        CUtensorMapFloatOOBfill);
spf_encode_tiled_fn spf_get_encode_tiled();

// implemented in spf_prepare.cu / spf_slice.cu / spf_match.cu
int spf_build_slice_maps(spf_ctx *ctx);
// records ctx->ev[i] on `st` when option "record_events" is on (creates the events on first use)
int spf_record_event(spf_ctx *ctx, int i, cudaStream_t st);
