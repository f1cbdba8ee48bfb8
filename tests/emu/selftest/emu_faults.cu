// tests/emu/selftest: deliberately BROKEN little kernels, written against the same wrappers the library's kernels use
// (csrc/ptx_sm100.cuh), to show that the emulator notices the classes of mistake it is relied on to notice
// (tests/test_emu_selftest.py).  Each entry point runs one kernel and returns; the test reads spf_emu_last_fault().
// TEST INFRASTRUCTURE ONLY.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "ptx_sm100.cuh"
#include "spf_internal.cuh"

namespace {

struct Args { const CUtensorMap *map; float *out; int mode; };

// mode 0: correct (expect_tx, copy, wait, read); 1: reads the tile WITHOUT waiting; 2: misaligned destination;
// 3: waits on a barrier that was never initialised; 4: forgets expect_tx and the copy, so the wait can never complete
__global__ void k_tma_cases(const __grid_constant__ CUtensorMap map, float *out, int mode, uint32_t *abort_flag) {
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ __align__(8) unsigned long long bar;
    __shared__ uint32_t s_abort;
    const uint32_t b = ptx::smem_u32(&bar), dst = ptx::smem_u32(smem) + (mode == 2 ? 64u : 0u);
    if (threadIdx.x == 0) {
        s_abort = 0u;
        if (mode != 3) { ptx::mbar_init(b, 1); ptx::fence_mbar_init(); }
    }
    __syncthreads();
    if (threadIdx.x == 0 && mode != 4) {
        ptx::mbar_expect_tx(b, 8 * 8 * 4);
        ptx::tma_load_3d(dst, &map, 0, 0, 0, b);
    }
    __syncthreads();
    bool ok = true;
    if (mode != 1) ok = ptx::mbar_wait(b, 0, &s_abort, abort_flag);
    const float *tile = reinterpret_cast<const float *>(smem + (mode == 2 ? 64 : 0));
    out[threadIdx.x] = ok ? tile[threadIdx.x] : -777.0f;
}

// mode 0: correct alloc / ld of own quadrant / dealloc; 1: warp 1 reads warp 0's lane quadrant; 2: exits without
// dealloc; 3: reads beyond the allocated columns
__global__ void k_tmem_cases(float *out, int mode) {
    __shared__ uint32_t slot;
    const int warp = threadIdx.x >> 5;
    if (warp == 0) ptx::tmem_alloc<1>(ptx::smem_u32(&slot), 32);
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t base = slot;
    uint32_t r[16];
    const uint32_t quadrant = (mode == 1 && warp == 1) ? 0u : (uint32_t)(warp & 3);
    ptx::tmem_ld_32x16(base + ((quadrant * 32u) << 16) + (mode == 3 ? 24u : 0u), r);
    ptx::tmem_ld_wait();
    out[threadIdx.x] = __uint_as_float(r[0]);
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 0 && mode != 2) ptx::tmem_dealloc<1>(base, 32);
}

}  // namespace

extern "C" __attribute__((visibility("default"))) int emu_fault_case(const char *family, int mode, float *out128) {
    float *grid = nullptr, *d_out = nullptr;
    uint32_t *d_abort = nullptr;
    cudaMalloc(&grid, 16 * 16 * 16 * 4); cudaMalloc(&d_out, 128 * 4); cudaMalloc(&d_abort, 4);
    cudaMemset(d_abort, 0, 4);
    for (int i = 0; i < 16 * 16 * 16; ++i) grid[i] = (float)i;     // host-visible under the emulator
    if (family[0] == 't' && family[1] == 'm' && family[2] == 'a') {
        CUtensorMap map;
        cuuint64_t gdim[3] = {16, 16, 16}, gstr[2] = {64, 1024};
        cuuint32_t box[3] = {8, 8, 1}, estr[3] = {1, 1, 1};
        spf_encode_tiled_fn enc = spf_get_encode_tiled();
        if (!enc || enc(&map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, grid, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                        CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) return -1;
        k_tma_cases<<<1, 64, 1024, 0>>>(map, d_out, mode, d_abort);
    } else {
        k_tmem_cases<<<1, 128, 0, 0>>>(d_out, mode);
    }
    cudaMemcpy(out128, d_out, 128 * 4, cudaMemcpyDeviceToHost);
    cudaFree(grid); cudaFree(d_out); cudaFree(d_abort);
    return 0;
}
