// tests/emu: functional stand-ins for the inline-PTX wrappers of csrc/ptx_sm100.cuh (same names, same
// signatures, namespace ptx).  build_emu.py strips every asm-bodied function from a copy of ptx_sm100.cuh and
// includes this file in their place; the wrappers that are plain C++ there (mbar_wait, abort_drain, the
// descriptor builders) are compiled UNCHANGED.  TEST INFRASTRUCTURE ONLY.
//
// Semantics stated here (what the emulator assumes the hardware does):
//   mbarrier      phase bit + pending-arrival count + transaction-byte count; a phase completes when both reach
//                 zero; try_wait.parity(p) is true once the phase of parity p has completed; using a barrier that
//                 was never initialised is a fault
//   TMA           a bulk tensor copy is DEFERRED: it lands some scheduler steps after it was issued, writes the box
//                 row by row at the destination (zero fill outside the tensor; with SWIZZLE_128B the 16-byte chunk
//                 index is XORed with address bits [7,10)), then completes box-bytes on the barrier -- for the
//                 cta_group::2 form on the barrier at the same offset in the even CTA of the pair
//   tcgen05.mma   DEFERRED and in issue order; reads both operands through SWIZZLE_128B K-major descriptors at
//                 execution time (so a stage recycled too early is read as poison); D[m][n] (+)= sum_k A[m][k] B[n][k]
//                 in fp32; cta_group::2: rows 0-127 of A and of D belong to the even CTA, rows 128-255 to the odd one,
//                 the first N/2 rows of B come from the even CTA's shared memory, the rest from the odd one's
//   tcgen05.commit  deferred behind the MMAs issued before it; arrives once (cta_group::2: on both CTAs' barriers)
//   tcgen05.ld    32 lanes x 16 columns; a warp may only address the lane quadrant 32 * (warp mod 4)
//   TMEM          128 lanes x 512 columns per CTA, NaN after allocation; leaving a block with columns allocated is a fault
#pragma once
#include <unordered_map>

#include "cuda_emu.h"

namespace emu {
struct MBar { int phase = 0, pending = 0, expected = 0; long tx = 0; };
std::unordered_map<uint32_t, MBar> &mbar_table();   // keyed by shared address; cleared per cluster (emu_ptx.cpp)
MBar *mbar_at(uint32_t addr, const char *what);
void mbar_check(MBar *m);
void tma_copy(uint32_t dst, const CUtensorMap *map, int nd, const int *crd, uint32_t bar);
void drain_all_async();
void umma(int cg, uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate);
}  // namespace emu

namespace ptx {

inline void mbar_init(uint32_t bar, uint32_t count) {
    if (bar & 7u) emu::fault("mbarrier.init at unaligned shared address 0x%x", bar);
    emu::MBar m; m.pending = m.expected = (int)count;
    emu::mbar_table()[bar] = m;
}
inline void fence_mbar_init() {}
inline void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    emu::MBar *m = emu::mbar_at(bar, "arrive.expect_tx");
    if (!m) return;
    if (bytes >= (1u << 20)) emu::fault("expect_tx of %u bytes exceeds the transaction-count range", bytes);
    m->tx += bytes; m->pending--; emu::mbar_check(m);
}
inline void mbar_arrive(uint32_t bar) {
    emu::MBar *m = emu::mbar_at(bar, "arrive");
    if (m) { m->pending--; emu::mbar_check(m); }
}
inline void mbar_arrive_cluster(uint32_t bar, uint32_t rank) {
    if ((int)rank >= emu::g_cluster_size) { emu::fault("mapa to CTA rank %u of a cluster of %d", rank, emu::g_cluster_size); return; }
    mbar_arrive((bar & 0x00ffffffu) | (rank << 24));
}
inline bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    emu::MBar *m = emu::mbar_at(bar, "try_wait");
    const bool ready = m && (uint32_t)m->phase != (parity & 1u);
    if (!ready) emu::yield();
    return ready;
}

// cp.async: deferred like every other asynchronous copy; wait_all drains the queue (all threads' copies: a superset)
inline void cp_async_16(uint32_t dst, const void *src) {
    if ((dst & 15u) || ((uintptr_t)src & 15u)) emu::fault("cp.async 16: unaligned address (shared 0x%x, global %p)", dst, src);
    emu::note_cp_async16(dst);
    emu::async_push([=]() { void *d = emu::shared_ptr(dst); if (d) memcpy(d, src, 16); });
}
inline void cp_async_wait_all() { emu::drain_all_async(); }
inline void cp_async_16_zfill(uint32_t dst, const void *src, uint32_t src_bytes) {
    if ((dst & 15u) || ((uintptr_t)src & 15u) || (src_bytes != 0u && src_bytes != 16u)) emu::fault("cp.async 16 (zfill %u): bad operands (shared 0x%x, global %p)", src_bytes, dst, src);
    emu::note_cp_async16(dst);
    emu::async_push([=]() { uint8_t *d = (uint8_t *)emu::shared_ptr(dst); if (!d) return; memset(d, 0, 16); if (src_bytes) memcpy(d, src, src_bytes); });
}
inline void cp_async_commit() {}
template <int N> inline void cp_async_wait_group() { emu::drain_all_async(); }   // a superset of what the hardware guarantees

// ldmatrix / mma.sync: the fragment layouts of the PTX ISA, written out (the comments in ptx_sm100.cuh state them)
inline void ldmatrix_x4(uint32_t (&r)[4], uint32_t row_addr) {
    if (row_addr & 15u) emu::fault("ldmatrix: row address 0x%x not 16-byte aligned", row_addr);
    const uint64_t *all = emu::warp_collective((uint64_t)row_addr);
    const int lane = emu::lane();
    if (lane == 0) emu::note_ldmatrix(all);
    for (int j = 0; j < 4; ++j) {
        const uint8_t *row = (const uint8_t *)emu::shared_ptr((uint32_t)all[8 * j + (lane >> 2)]);
        if (!row) { r[j] = 0xffffffffu; continue; }
        memcpy(&r[j], row + 4 * (lane & 3), 4);
    }
    emu::warp_collective(0);   // nobody's deposited address is overwritten before everyone has read it
}
namespace emu_detail {
inline float h2f(uint16_t h) {
    const uint32_t sign = (uint32_t)(h & 0x8000u) << 16, e = (h >> 10) & 0x1fu, m = h & 0x3ffu;
    uint32_t u;
    if (e == 0) { const float sub = (float)m * 5.9604644775390625e-8f; return sign ? -sub : sub; }
    if (e == 31) u = sign | 0x7f800000u | (m << 13); else u = sign | ((e + 112u) << 23) | (m << 13);
    float f; memcpy(&f, &u, 4); return f;
}
}  // namespace emu_detail
inline void mma_m16n8k16(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    // three exchange rounds collect every lane's A and B registers; each lane then computes its own four outputs
    uint32_t A[32][4], B[32][2];
    const uint64_t *s = emu::warp_collective((uint64_t)a[0] | ((uint64_t)a[1] << 32));
    for (int l = 0; l < 32; ++l) { A[l][0] = (uint32_t)s[l]; A[l][1] = (uint32_t)(s[l] >> 32); }
    s = emu::warp_collective((uint64_t)a[2] | ((uint64_t)a[3] << 32));
    for (int l = 0; l < 32; ++l) { A[l][2] = (uint32_t)s[l]; A[l][3] = (uint32_t)(s[l] >> 32); }
    s = emu::warp_collective((uint64_t)b0 | ((uint64_t)b1 << 32));
    for (int l = 0; l < 32; ++l) { B[l][0] = (uint32_t)s[l]; B[l][1] = (uint32_t)(s[l] >> 32); }
    auto Ael = [&](int row, int k) {   // A[row][k], row < 16, k < 16
        const int l = (row & 7) * 4 + ((k & 7) >> 1), reg = (row >> 3) + 2 * (k >> 3);
        return emu_detail::h2f((uint16_t)(A[l][reg] >> (16 * (k & 1))));
    };
    auto Bel = [&](int k, int n) {     // B[k][n], k < 16, n < 8
        const int l = n * 4 + ((k & 7) >> 1), reg = k >> 3;
        return emu_detail::h2f((uint16_t)(B[l][reg] >> (16 * (k & 1))));
    };
    const int lane = emu::lane(), g = lane >> 2, t = lane & 3;
    for (int o = 0; o < 4; ++o) {
        const int row = g + 8 * (o >> 1), col = 2 * t + (o & 1);
        float p = 0.0f;
        for (int k = 0; k < 16; ++k) p += Ael(row, k) * Bel(k, col);
        d[o] += p;
    }
}

inline void prefetch_tensormap(const void *) {}
inline void tma_load_2d(uint32_t dst, const void *map, int c0, int c1, uint32_t bar) {
    const int crd[3] = {c0, c1, 0};
    emu::tma_copy(dst, (const CUtensorMap *)map, 2, crd, bar);
}
inline void tma_load_2d_2sm(uint32_t dst, const void *map, int c0, int c1, uint32_t bar) {
    if (emu::g_cluster_size != 2) emu::fault("cta_group::2 bulk copy outside a CTA pair");
    const int crd[3] = {c0, c1, 0};
    emu::tma_copy(dst, (const CUtensorMap *)map, 2, crd, bar & 0xFEFFFFFFu);
}
inline void tma_load_3d(uint32_t dst, const void *map, int c0, int c1, int c2, uint32_t bar) {
    const int crd[3] = {c0, c1, c2};
    emu::tma_copy(dst, (const CUtensorMap *)map, 3, crd, bar);
}

inline uint32_t cluster_ctarank() { return (uint32_t)emu::cur_cta->rank; }
inline void cluster_sync() { emu::cluster_barrier(); }

template <int CG>
inline void tmem_alloc(uint32_t dst_smem, uint32_t ncols) {
    if (CG != emu::g_cluster_size && CG == 2) emu::fault("tcgen05.alloc.cta_group::2 outside a CTA pair");
    if (emu::lane() == 0) {
        emu::Cta *c = emu::cur_cta;
        if (ncols < 32 || ncols > 512 || (ncols & (ncols - 1))) emu::fault("tcgen05.alloc of %u columns (power of two in [32,512])", ncols);
        if (c->tmem_cols + (int)ncols > 512) emu::fault("tcgen05.alloc: %u columns requested with %d in use (the hardware would block)", ncols, c->tmem_cols);
        if (!c->tmem) c->tmem = (float *)malloc(sizeof(float) * 128 * 512);
        for (int i = 0; i < 128 * 512; ++i) c->tmem[i] = NAN;
        uint32_t *slot = (uint32_t *)emu::shared_ptr(dst_smem);
        if (slot) *slot = (uint32_t)c->tmem_cols;
        c->tmem_cols += (int)ncols;
    }
    emu::warp_collective(0);   // .sync.aligned: the whole warp executes it
}
template <int CG>
inline void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
    if (emu::lane() == 0) {
        emu::Cta *c = emu::cur_cta;
        if ((taddr >> 16) != 0 || (int)((taddr & 0xffffu) + ncols) > 512 || c->tmem_cols < (int)ncols) emu::fault("tcgen05.dealloc(0x%x, %u) does not match an allocation", taddr, ncols);
        c->tmem_cols -= (int)ncols;
    }
    emu::warp_collective(0);
}
inline void tc_fence_before() {}
inline void tc_fence_after() {}

template <int CG>
inline void umma_f16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    if (CG == 2 && emu::cur_cta->rank != 0) emu::fault("cta_group::2 MMA issued by the odd CTA of the pair");
    emu::async_push([=]() { emu::umma(CG, tmem_d, adesc, bdesc, idesc, accumulate); });
}
template <int CG>
inline void umma_commit(uint32_t bar) {
    const int rank = emu::cur_cta->rank;
    emu::async_push([=]() {
        if (CG == 1) mbar_arrive((bar & 0x00ffffffu) | ((uint32_t)rank << 24));
        else { mbar_arrive(bar & 0x00ffffffu); mbar_arrive((bar & 0x00ffffffu) | (1u << 24)); }   // multicast mask 0b11
    });
}
inline void tmem_ld_32x16(uint32_t taddr, uint32_t (&r)[16]) {
    emu::Cta *c = emu::cur_cta;
    const int warp = emu::cur_tid() >> 5, lane0 = (int)(taddr >> 16), col = (int)(taddr & 0xffffu);
    if (lane0 != 32 * (warp & 3)) emu::fault("tcgen05.ld: warp %d addresses TMEM lane %d (its quadrant starts at %d)", warp, lane0, 32 * (warp & 3));
    if (!c->tmem || col + 16 > c->tmem_cols) { emu::fault("tcgen05.ld: columns %d..%d outside the %d allocated", col, col + 15, c->tmem_cols); return; }
    const float *row = c->tmem + (size_t)(lane0 + emu::lane()) * 512 + col;
    for (int k = 0; k < 16; ++k) memcpy(&r[k], &row[k], 4);
}
inline void tmem_ld_wait() {}

}  // namespace ptx
