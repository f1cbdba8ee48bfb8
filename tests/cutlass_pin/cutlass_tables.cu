// tests/cutlass_pin: prints, as one JSON object, what the CUTLASS / CuTe headers vendored in this image say about the
// instruction-level facts this repository's kernels and its emulator rely on.  HOST program (nothing is launched);
// it only evaluates CuTe's own layout algebra and descriptor unions.  TEST INFRASTRUCTURE ONLY: the product does not
// include CUTLASS; tests/test_cutlass_pins.py compares these tables with csrc/ptx_sm100.cuh's descriptor builders and
// with the emulator's models of tcgen05.mma, TMA swizzling, mma.sync and ldmatrix (tests/emu/ptx_emu.cuh).
//
// Build: nvcc -std=c++17 -I<cutlass/include> -gencode arch=compute_100a,code=sm_100a cutlass_tables.cu -o cutlass_tables
#include <cstdint>
#include <cstdio>

#include <cute/tensor.hpp>
#include <cute/arch/mma_sm100_desc.hpp>
#include <cute/atom/copy_traits_sm75.hpp>
#include <cute/atom/copy_traits_sm100.hpp>
#include <cute/atom/mma_traits_sm100.hpp>
#include <cute/atom/mma_traits_sm80.hpp>

using namespace cute;

template <int M, int N>
static uint32_t idesc() {
    return (uint32_t)UMMA::make_instr_desc<half_t, half_t, float, M, N, UMMA::Major::K, UMMA::Major::K>();
}

int main() {
    printf("{\n");
    // (1) kind::f16 instruction descriptors, fp16 x fp16 -> fp32, both operands K-major
    printf(" \"idesc\": {\"128x64\": %u, \"128x128\": %u, \"128x256\": %u, \"256x64\": %u, \"256x128\": %u, \"256x256\": %u},\n",
           idesc<128, 64>(), idesc<128, 128>(), idesc<128, 256>(), idesc<256, 64>(), idesc<256, 128>(), idesc<256, 256>());

    // (2) shared-memory descriptor of a K-major [128 rows][64 fp16] tile in the 128-byte-swizzle atom
    auto layout = tile_to_shape(UMMA::Layout_K_SW128_Atom<half_t>{}, Shape<_128, _64>{});
    alignas(1024) static half_t buf[128 * 64];
    Tensor sA = make_tensor(make_smem_ptr(buf), layout);
    UMMA::SmemDescriptor d = UMMA::make_umma_desc<UMMA::Major::K>(sA);      // on the host the start address is 0 (CuTe prints one ERROR line about it, which the test drops)
    printf(" \"smem_desc\": {\"lbo\": %u, \"sbo\": %u, \"version\": %u, \"layout_type\": %u, \"base_offset\": %u, \"lbo_mode\": %u, \"hi\": %u},\n",
           (unsigned)d.leading_byte_offset_, (unsigned)d.stride_byte_offset_, (unsigned)d.version_, (unsigned)d.layout_type_,
           (unsigned)d.base_offset_, (unsigned)d.lbo_mode_, (unsigned)d.hi);

    // (3) where element (row, k) of that tile lives, in bytes from the tile's (1024-byte aligned) base
    printf(" \"sw128_byte_offset\": [");
    for (int r = 0; r < 128; ++r) {
        printf("%s[", r ? "," : "");
        for (int k = 0; k < 64; ++k) printf("%s%d", k ? "," : "", (int)((const char *)&sA(r, k) - (const char *)buf));
        printf("]");
    }
    printf("],\n");

    // (4) mma.sync.m16n8k16 f16 x f16 -> f32 fragments: (thread, value) -> matrix coordinates
    using T = MMA_Traits<SM80_16x8x16_F32F16F16F32_TN>;
    printf(" \"mma_A\": [");
    for (int t = 0; t < 32; ++t) { printf("%s[", t ? "," : ""); for (int v = 0; v < 8; ++v) { int i = (int)typename T::ALayout{}(t, v); printf("%s[%d,%d]", v ? "," : "", i % 16, i / 16); } printf("]"); }
    printf("],\n \"mma_B\": [");
    for (int t = 0; t < 32; ++t) { printf("%s[", t ? "," : ""); for (int v = 0; v < 4; ++v) { int i = (int)typename T::BLayout{}(t, v); printf("%s[%d,%d]", v ? "," : "", i % 8, i / 8); } printf("]"); }
    printf("],\n \"mma_C\": [");
    for (int t = 0; t < 32; ++t) { printf("%s[", t ? "," : ""); for (int v = 0; v < 4; ++v) { int i = (int)typename T::CLayout{}(t, v); printf("%s[%d,%d]", v ? "," : "", i % 16, i / 16); } printf("]"); }
    printf("],\n");

    // (5) ldmatrix.x4 (non-transposed): register j of thread t <- 32 bits at this bit index of the 32 x 128-bit source,
    //     where source thread s supplies bits [128 s, 128 s + 128) (its row address)
    using L = Copy_Traits<SM75_U32x4_LDSM_N>;
    printf(" \"ldsm_dst_bit\": [");
    for (int t = 0; t < 32; ++t) { printf("%s[", t ? "," : ""); for (int j = 0; j < 4; ++j) printf("%s%d", j ? "," : "", (int)typename L::DstLayout{}(t, make_coord(0, j))); printf("]"); }
    printf("],\n \"ldsm_src_bit\": [");
    for (int t = 0; t < 32; ++t) printf("%s%d", t ? "," : "", (int)typename L::SrcLayout{}(t, 0));
    printf("],\n");

    // (5b) tcgen05.mma cta_group::2, M 256 x N 64: which rows of A, B and D CTA v of the pair holds (v, (row, k)) -> row
    using P = MMA_Traits<SM100_MMA_F16BF16_2x1SM_SS<half_t, half_t, float, 256, 64, UMMA::Major::K, UMMA::Major::K>>;
    printf(" \"pair_256x64\": {\"A_row\": [[%d,%d],[%d,%d]], \"B_row\": [[%d,%d],[%d,%d]], \"D_row\": [[%d,%d],[%d,%d]]},\n",
           (int)typename P::ALayout{}(0, make_coord(0, 0)) % 256, (int)typename P::ALayout{}(0, make_coord(127, 0)) % 256,
           (int)typename P::ALayout{}(1, make_coord(0, 0)) % 256, (int)typename P::ALayout{}(1, make_coord(127, 0)) % 256,
           (int)typename P::BLayout{}(0, make_coord(0, 0)) % 64, (int)typename P::BLayout{}(0, make_coord(31, 0)) % 64,
           (int)typename P::BLayout{}(1, make_coord(0, 0)) % 64, (int)typename P::BLayout{}(1, make_coord(31, 0)) % 64,
           (int)typename P::CLayout{}(0, make_coord(0, 0)) % 256, (int)typename P::CLayout{}(0, make_coord(127, 0)) % 256,
           (int)typename P::CLayout{}(1, make_coord(0, 0)) % 256, (int)typename P::CLayout{}(1, make_coord(127, 0)) % 256);

    // (6) tcgen05.ld 32x32b.x16: thread t <- 512 consecutive bits (16 fp32 columns) of data path (lane) t;
    //     one lane step in TMEM address bits
    using M = Copy_Traits<SM100::TMEM::LOAD::SM100_TMEM_LOAD_32dp32b16x>;
    printf(" \"tmem_ld_dst_bit\": [%d, %d, %d], \"tmem_dp_bits\": %d\n",
           (int)typename M::DstLayout{}(0, 0), (int)typename M::DstLayout{}(1, 0), (int)typename M::DstLayout{}(0, 511), (int)TMEM::DP_b{});
    printf("}\n");
    return 0;
}
