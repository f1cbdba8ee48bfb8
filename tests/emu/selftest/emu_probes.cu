// tests/emu/selftest: one-instruction probe kernels, written against the wrappers of csrc/ptx_sm100.cuh, through which
// tests/test_cutlass_pins.py compares the EMULATOR's model of an instruction (tests/emu/ptx_emu.cuh, emu_runtime.cpp)
// with the tables CuTe publishes for it (tests/cutlass_pin/cutlass_tables.cu): fragment layouts of mma.sync.m16n8k16
// and ldmatrix.x4, the byte position of element (row, k) in a 128-byte-swizzled K-major tile as TMA writes it and as
// tcgen05.mma reads it through the kernels' own descriptor builder, the +32-byte K advance, tcgen05.ld's lane / column
// mapping.  These kernels only ever run under the emulator (they omit the proxy fence a generic-proxy write to an MMA
// operand needs on hardware).  TEST INFRASTRUCTURE ONLY.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

#include "ptx_sm100.cuh"
#include "spf_internal.cuh"

namespace {

// in: [32][6] words (a0..a3, b0, b1) per lane; out: [32][4] floats (d0..d3), accumulators start at zero
__global__ void k_probe_mma(const uint32_t *in, float *out) {
    const int l = threadIdx.x;
    uint32_t a[4] = {in[l * 6 + 0], in[l * 6 + 1], in[l * 6 + 2], in[l * 6 + 3]};
    float d[4] = {0.0f, 0.0f, 0.0f, 0.0f};
    ptx::mma_m16n8k16(d, a, in[l * 6 + 4], in[l * 6 + 5]);
    for (int o = 0; o < 4; ++o) out[l * 4 + o] = d[o];
}

// rows: 32 rows of 16 bytes; lane l supplies the address of row perm[l]; out: [32][4] words
__global__ void k_probe_ldsm(const uint8_t *rows, const int *perm, uint32_t *out) {
    extern __shared__ __align__(16) uint8_t tile[];
    const int l = threadIdx.x;
    for (int i = 0; i < 16; ++i) tile[l * 16 + i] = rows[l * 16 + i];
    __syncthreads();
    uint32_t r[4];
    ptx::ldmatrix_x4(r, ptx::smem_u32(tile) + 16u * (uint32_t)perm[l]);
    for (int j = 0; j < 4; ++j) out[l * 4 + j] = r[j];
}

// one [16 rows][64 fp16] box of a [16][64] fp16 tensor through a SWIZZLE_128B tensor map; out: the 2,048 bytes of the tile
__global__ void k_probe_tma(const __grid_constant__ CUtensorMap map, uint8_t *out, uint32_t *abort_flag) {
    extern __shared__ __align__(1024) uint8_t smem[];
    __shared__ __align__(8) unsigned long long bar;
    __shared__ uint32_t s_abort;
    const uint32_t base = (ptx::smem_u32(smem) + 1023u) & ~1023u, b = ptx::smem_u32(&bar);
    uint8_t *tile = smem + (base - ptx::smem_u32(smem));
    if (threadIdx.x == 0) { s_abort = 0u; ptx::mbar_init(b, 1); ptx::fence_mbar_init(); }
    __syncthreads();
    if (threadIdx.x == 0) { ptx::mbar_expect_tx(b, 16 * 128); ptx::tma_load_2d(base, &map, 0, 0, b); }
    __syncthreads();
    const bool ok = ptx::mbar_wait(b, 0, &s_abort, abort_flag);
    for (int i = threadIdx.x; i < 2048; i += blockDim.x) out[i] = ok ? tile[i] : (uint8_t)0xEE;
}

// imgA: 16 KB byte image of a [128][64] fp16 K-major SW128 tile; imgB: 8 KB image of a [64][64] tile; one
// tcgen05.mma (M 128, N 64, K 16) at K step kk of the 64-wide block, exactly as k_match_gemm forms its operands
// (umma_desc_sw128(base) + 2 kk); out: [128][64] fp32 = A[:, 16kk:16kk+16] . B[:, 16kk:16kk+16]^T
__global__ void k_probe_umma(const uint8_t *imgA, const uint8_t *imgB, int kk, float *out, uint32_t *abort_flag) {
    extern __shared__ __align__(1024) uint8_t smem[];
    __shared__ __align__(8) unsigned long long bar;
    __shared__ uint32_t slot, s_abort;
    const uint32_t base = (ptx::smem_u32(smem) + 1023u) & ~1023u, b = ptx::smem_u32(&bar);
    uint8_t *tileA = smem + (base - ptx::smem_u32(smem)), *tileB = tileA + 16384;
    const int warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < 16384; i += blockDim.x) tileA[i] = imgA[i];
    for (int i = threadIdx.x; i < 8192; i += blockDim.x) tileB[i] = imgB[i];
    if (threadIdx.x == 0) { s_abort = 0u; ptx::mbar_init(b, 1); ptx::fence_mbar_init(); }
    if (warp == 0) ptx::tmem_alloc<1>(ptx::smem_u32(&slot), 64);
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tacc = slot;
    if (threadIdx.x == 0) {
        const uint64_t ko = (uint64_t)(kk * 2);
        ptx::umma_f16<1>(tacc, ptx::umma_desc_sw128(base) + ko, ptx::umma_desc_sw128(base + 16384u) + ko, ptx::umma_idesc_f16(128, 64), 0u);
        ptx::umma_commit<1>(b);
    }
    const bool ok = ptx::mbar_wait(b, 0, &s_abort, abort_flag);
    ptx::tc_fence_after();
    for (int c = 0; c < 64; c += 16) {
        uint32_t r[16];
        ptx::tmem_ld_32x16(tacc + ((uint32_t)(warp * 32) << 16) + (uint32_t)c, r);
        ptx::tmem_ld_wait();
        for (int j = 0; j < 16; ++j) out[threadIdx.x * 64 + c + j] = ok ? __uint_as_float(r[j]) : -777.0f;
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 0) ptx::tmem_dealloc<1>(tacc, 64);
}

// the same on a CTA pair (cta_group::2, M 256, N 64): each CTA holds its own 128 rows of A and 32 rows of B at the same
// shared-memory offsets, the leader issues ONE instruction, the commit is multicast to both CTAs' barriers, and each CTA
// reads its own 128 x 64 half of D from its own TMEM -- set up and torn down as k_match_gemm<2, .> does it
__global__ void k_probe_umma_pair(const uint8_t *imgA, const uint8_t *imgB, int kk, float *out, uint32_t *abort_flag) {
    extern __shared__ __align__(1024) uint8_t smem[];
    __shared__ __align__(8) unsigned long long bar;
    __shared__ uint32_t slot, s_abort;
    const uint32_t base = (ptx::smem_u32(smem) + 1023u) & ~1023u, b = ptx::smem_u32(&bar);
    uint8_t *tileA = smem + (base - ptx::smem_u32(smem)), *tileB = tileA + 16384;
    const int warp = threadIdx.x >> 5;
    const uint32_t rank = ptx::cluster_ctarank();
    for (int i = threadIdx.x; i < 16384; i += blockDim.x) tileA[i] = imgA[rank * 16384 + i];
    for (int i = threadIdx.x; i < 4096; i += blockDim.x) tileB[i] = imgB[rank * 4096 + i];
    if (threadIdx.x == 0) { s_abort = 0u; ptx::mbar_init(b, 1); ptx::fence_mbar_init(); }
    if (warp == 1) ptx::tmem_alloc<2>(ptx::smem_u32(&slot), 64);
    ptx::tc_fence_before();
    ptx::cluster_sync();
    ptx::tc_fence_after();
    const uint32_t tacc = slot;
    if (rank == 0 && threadIdx.x == 32) {
        const uint64_t ko = (uint64_t)(kk * 2);
        ptx::umma_f16<2>(tacc, ptx::umma_desc_sw128(base) + ko, ptx::umma_desc_sw128(base + 16384u) + ko, ptx::umma_idesc_f16(256, 64), 0u);
        ptx::umma_commit<2>(b);
    }
    const bool ok = ptx::mbar_wait(b, 0, &s_abort, abort_flag);
    ptx::tc_fence_after();
    for (int c = 0; c < 64; c += 16) {
        uint32_t r[16];
        ptx::tmem_ld_32x16(tacc + ((uint32_t)(warp * 32) << 16) + (uint32_t)c, r);
        ptx::tmem_ld_wait();
        for (int j = 0; j < 16; ++j) out[(rank * 128 + threadIdx.x) * 64 + c + j] = ok ? __uint_as_float(r[j]) : -777.0f;
    }
    ptx::tc_fence_before();
    ptx::cluster_sync();
    if (warp == 1) ptx::tmem_dealloc<2>(tacc, 64);
}

}  // namespace

#define EMU_EXPORT extern "C" __attribute__((visibility("default")))

// the product's descriptor builders, as compiled (unchanged) into the emulator build
EMU_EXPORT unsigned long long emu_probe_smem_desc(unsigned smem_addr) { return ptx::umma_desc_sw128(smem_addr); }
EMU_EXPORT unsigned emu_probe_idesc(int M, int N) { return ptx::umma_idesc_f16(M, N); }

EMU_EXPORT int emu_probe_mma(const uint32_t *in, float *out) {
    uint32_t *d_in; float *d_out;
    cudaMalloc(&d_in, 32 * 6 * 4); cudaMalloc(&d_out, 32 * 4 * 4);
    cudaMemcpy(d_in, in, 32 * 6 * 4, cudaMemcpyHostToDevice);
    k_probe_mma<<<1, 32, 0, 0>>>(d_in, d_out);
    cudaMemcpy(out, d_out, 32 * 4 * 4, cudaMemcpyDeviceToHost);
    cudaFree(d_in); cudaFree(d_out);
    return 0;
}

EMU_EXPORT int emu_probe_ldsm(const uint8_t *rows, const int *perm, uint32_t *out) {
    uint8_t *d_rows; int *d_perm; uint32_t *d_out;
    cudaMalloc(&d_rows, 512); cudaMalloc(&d_perm, 128); cudaMalloc(&d_out, 512);
    cudaMemcpy(d_rows, rows, 512, cudaMemcpyHostToDevice); cudaMemcpy(d_perm, perm, 128, cudaMemcpyHostToDevice);
    k_probe_ldsm<<<1, 32, 512, 0>>>(d_rows, d_perm, d_out);
    cudaMemcpy(out, d_out, 512, cudaMemcpyDeviceToHost);
    cudaFree(d_rows); cudaFree(d_perm); cudaFree(d_out);
    return 0;
}

EMU_EXPORT int emu_probe_tma(const uint16_t *tensor16x64, uint8_t *out2048) {
    uint16_t *d_t; uint8_t *d_out; uint32_t *d_abort;
    cudaMalloc(&d_t, 16 * 64 * 2); cudaMalloc(&d_out, 2048); cudaMalloc(&d_abort, 4);
    cudaMemcpy(d_t, tensor16x64, 16 * 64 * 2, cudaMemcpyHostToDevice); cudaMemset(d_abort, 0, 4);
    CUtensorMap map;
    cuuint64_t gdim[2] = {64, 16}, gstr[1] = {128};
    cuuint32_t box[2] = {64, 16}, estr[2] = {1, 1};
    spf_encode_tiled_fn enc = spf_get_encode_tiled();
    if (!enc || enc(&map, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, d_t, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) return -1;
    k_probe_tma<<<1, 64, 2048 + 1024, 0>>>(map, d_out, d_abort);
    cudaMemcpy(out2048, d_out, 2048, cudaMemcpyDeviceToHost);
    cudaFree(d_t); cudaFree(d_out); cudaFree(d_abort);
    return 0;
}

EMU_EXPORT int emu_probe_umma(const uint8_t *imgA, const uint8_t *imgB, int kk, float *out) {
    uint8_t *d_a, *d_b; float *d_out; uint32_t *d_abort;
    cudaMalloc(&d_a, 16384); cudaMalloc(&d_b, 8192); cudaMalloc(&d_out, 128 * 64 * 4); cudaMalloc(&d_abort, 4);
    cudaMemcpy(d_a, imgA, 16384, cudaMemcpyHostToDevice); cudaMemcpy(d_b, imgB, 8192, cudaMemcpyHostToDevice); cudaMemset(d_abort, 0, 4);
    k_probe_umma<<<1, 128, 16384 + 8192 + 1024, 0>>>(d_a, d_b, kk, d_out, d_abort);
    cudaMemcpy(out, d_out, 128 * 64 * 4, cudaMemcpyDeviceToHost);
    cudaFree(d_a); cudaFree(d_b); cudaFree(d_out); cudaFree(d_abort);
    return 0;
}

EMU_EXPORT int emu_probe_umma_pair(const uint8_t *imgA, const uint8_t *imgB, int kk, float *out) {
    uint8_t *d_a, *d_b; float *d_out; uint32_t *d_abort;
    cudaMalloc(&d_a, 2 * 16384); cudaMalloc(&d_b, 2 * 4096); cudaMalloc(&d_out, 256 * 64 * 4); cudaMalloc(&d_abort, 4);
    cudaMemcpy(d_a, imgA, 2 * 16384, cudaMemcpyHostToDevice); cudaMemcpy(d_b, imgB, 2 * 4096, cudaMemcpyHostToDevice); cudaMemset(d_abort, 0, 4);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(2); cfg.blockDim = dim3(128); cfg.dynamicSmemBytes = 16384 + 4096 + 1024; cfg.stream = 0;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, k_probe_umma_pair, (const uint8_t *)d_a, (const uint8_t *)d_b, kk, d_out, d_abort);
    cudaMemcpy(out, d_out, 256 * 64 * 4, cudaMemcpyDeviceToHost);
    cudaFree(d_a); cudaFree(d_b); cudaFree(d_out); cudaFree(d_abort);
    return e == cudaSuccess ? 0 : -1;
}
