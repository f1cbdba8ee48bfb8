// tests/emu: scheduler, barriers, warp collectives, deferred asynchronous engines, shared-address map,
// tensor-map encoder and the DFT behind the cuFFT stub.  See cuda_emu.h for the model.  TEST INFRASTRUCTURE ONLY.
#include <stdarg.h>
#include <setjmp.h>
#include <ucontext.h>

#include <array>
#include <deque>
#include <string>
#include <vector>

#include "cuda_emu.h"
#include "ptx_emu.cuh"

dim3 threadIdx, blockIdx, blockDim, gridDim;

#include <chrono>
double emu_now_ms() { return std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now().time_since_epoch()).count(); }

namespace emu {

// Fiber switches: a fiber is entered the first time with swapcontext (which installs its stack) and from then on with
// _setjmp / _longjmp, which do not save the signal mask -- glibc's swapcontext makes a system call per switch, and the
// emulator makes millions of switches.  Under AddressSanitizer (which tracks stacks through swapcontext) every switch
// stays a swapcontext.
#if defined(__SANITIZE_ADDRESS__)
#define EMU_FAST_SWITCH 0
#else
#define EMU_FAST_SWITCH 1
#endif

struct Fiber {
    ucontext_t ctx;
    jmp_buf jb;
    bool started = false;
    char *stack = nullptr;
    bool done = true;
    int cta = 0, tid = 0;
    long cp_seq = 0;          // how many cp.async.16 this thread has issued in this block (lanes of a warp issue them in step)
    dim3 t3;
};

Fiber *cur = nullptr;
Cta *cur_cta = nullptr;
int g_cluster_size = 1;
long long g_ticks = 0;
int g_sm_count = 4;
long g_smem_counters[4] = {0, 0, 0, 0};
long g_counters[4] = {0, 0, 0, 0};   // [0] bulk tensor copies, [1] tcgen05.mma, [2] kernel launches, [3] fiber switches

namespace {
constexpr size_t STACK_BYTES = 256 * 1024;
ucontext_t sched_ctx;
jmp_buf sched_jb;
std::vector<Fiber> fibers;
std::vector<Cta> ctas;
std::vector<uint8_t *> dyn_store;      // 1024-byte aligned, one per CTA of the cluster
std::vector<size_t> dyn_cap;
const std::function<void()> *body_fn = nullptr;
int cluster_alive = 0, cluster_arrived = 0;
unsigned cluster_gen = 0;
struct AsyncOp { long ready; std::function<void()> fn; };
std::deque<AsyncOp> async_q;        // FIFO: an operation lands no earlier than `ready` (in fiber switches) and never before its predecessors
std::string g_fault;
uint32_t rng_state = 12345u;
std::vector<const void *> static_shared;   // static __shared__ objects whose address was taken (mbarriers of k_slice)
constexpr uint32_t WINDOW = 0x00000400u;     // shared-window offset of the dynamic block inside a CTA (1024-aligned, keeps addresses < 256 KB)
constexpr uint32_t STATIC_BASE = 0x00800000u;

// cp.async.16 destinations of the running block: [cta * 32 + warp][sequence number][lane] (0 = no access)
std::vector<std::vector<std::array<uint32_t, 32>>> cp_log;

// wavefronts a group of up to 8 sixteen-byte accesses takes: the busiest of the 8 bank groups, equal addresses merged
int wavefronts16(const uint32_t *addr, int n) {
    int worst = 0;
    for (int g = 0; g < 8; ++g) {
        uint32_t seen[8]; int ns = 0;
        for (int i = 0; i < n; ++i) {
            if (!addr[i] || (int)((addr[i] >> 4) & 7u) != g) continue;
            bool dup = false;
            for (int k = 0; k < ns; ++k) dup = dup || seen[k] == addr[i];
            if (!dup) seen[ns++] = addr[i];
        }
        worst = ns > worst ? ns : worst;
    }
    return worst;
}
void flush_cp_log() {
    for (auto &w : cp_log)
        for (auto &ins : w)
            for (int q = 0; q < 4; ++q) {
                const int wf = wavefronts16(&ins[(size_t)q * 8], 8);
                if (wf) { g_smem_counters[2]++; g_smem_counters[3] += wf; }
            }
    cp_log.clear();
}

uint32_t rnd() { rng_state = rng_state * 1664525u + 1013904223u; return rng_state >> 8; }

void fiber_entry() {
    (*body_fn)();
    Fiber *f = cur;
    Cta &c = ctas[f->cta];
    f->done = true;
    // an exited thread no longer takes part in barriers: complete the ones it was the last to be missing from
    Warp &w = c.warps[f->tid >> 5];
    w.alive--;
    if (w.alive > 0 && w.arrived == w.alive) { w.arrived = 0; w.gen++; }
    c.alive--;
    if (c.alive > 0 && c.bar_arrived == c.alive) { c.bar_arrived = 0; c.bar_gen++; }
    cluster_alive--;
    if (cluster_alive > 0 && cluster_arrived == cluster_alive) { cluster_arrived = 0; cluster_gen++; }
#if EMU_FAST_SWITCH
    _longjmp(sched_jb, 1);
#else
    swapcontext(&f->ctx, &sched_ctx);
#endif
}

void drain_async(bool all) {
    // deferred operations land in issue order, each no earlier than its own latency after it was issued (a few hundred to
    // a few thousand fiber switches): a consumer that does not wait for the barrier reads poison, not data
    while (!async_q.empty() && (all || async_q.front().ready <= g_counters[3])) {
        std::function<void()> op = std::move(async_q.front().fn);
        async_q.pop_front();
        op();
    }
}
}  // namespace

void fault(const char *fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (g_fault.empty()) g_fault = buf;
    fprintf(stderr, "[emu] FAULT: %s\n", buf);
}
const char *last_fault() { return g_fault.c_str(); }
void clear_fault() { g_fault.clear(); }

void yield() {
    ++g_ticks;
    ++g_counters[3];
    Fiber *f = cur;
#if EMU_FAST_SWITCH
    if (!_setjmp(f->jb)) _longjmp(sched_jb, 1);
#else
    swapcontext(&f->ctx, &sched_ctx);
#endif
}

int cur_tid() { return cur->tid; }
void note_ldmatrix(const uint64_t *addr32) {
    for (int j = 0; j < 4; ++j) {
        uint32_t a[8];
        for (int i = 0; i < 8; ++i) a[i] = (uint32_t)addr32[8 * j + i] | 0x80000000u;    // never 0 ("no access")
        g_smem_counters[0]++;
        g_smem_counters[1] += wavefronts16(a, 8);
    }
}
void note_cp_async16(uint32_t dst) {
    const size_t w = (size_t)cur->cta * 32 + (size_t)(cur->tid >> 5);
    if (cp_log.size() <= w) cp_log.resize(w + 1);
    const size_t seq = (size_t)cur->cp_seq++;
    if (cp_log[w].size() <= seq) cp_log[w].resize(seq + 1, std::array<uint32_t, 32>{});
    cp_log[w][seq][(size_t)(cur->tid & 31)] = dst | 0x80000000u;
}
Cta *cta_of_rank(int rank) {
    if (rank < 0 || rank >= (int)ctas.size()) { fault("CTA rank %d outside the cluster of %zu", rank, ctas.size()); return &ctas[0]; }
    return &ctas[rank];
}
void *dyn_smem() { return cur_cta->dyn; }

void block_barrier() {
    Cta &c = *cur_cta;
    const unsigned g = c.bar_gen;
    if (++c.bar_arrived == c.alive) { c.bar_arrived = 0; c.bar_gen++; return; }
    while (c.bar_gen == g) yield();
}
void cluster_barrier() {
    const unsigned g = cluster_gen;
    if (++cluster_arrived == cluster_alive) { cluster_arrived = 0; cluster_gen++; return; }
    while (cluster_gen == g) yield();
}
int warp_alive_mask() {
    // lanes of the running warp that have not exited
    const int w = cur->tid >> 5, base = cur->cta * (int)(blockDim.x * blockDim.y * blockDim.z) + (w << 5);
    int m = 0;
    for (int l = 0; l < 32; ++l)
        if (base + l < (int)fibers.size() && fibers[base + l].cta == cur->cta && !fibers[base + l].done) m |= 1 << l;
    return m;
}
const uint64_t *warp_collective(uint64_t v) {
    Warp &w = cur_cta->warps[cur->tid >> 5];
    const unsigned g = w.gen;
    w.vals[g & 1][cur->tid & 31] = v;
    if (++w.arrived == w.alive) { w.arrived = 0; w.gen++; }
    else while (w.gen == g) yield();
    return w.vals[g & 1];
}

void drain_all_async() { drain_async(true); }
void async_push(std::function<void()> op) { async_q.push_back(AsyncOp{g_counters[3] + 300 + (long)(rnd() % 3000u), std::move(op)}); }

uint32_t shared_addr(const void *p) {
    const uint8_t *b = (const uint8_t *)p;
    for (size_t r = 0; r < ctas.size(); ++r)
        if (b >= ctas[r].dyn && b < ctas[r].dyn + ctas[r].dyn_bytes + 1)
            return WINDOW + (uint32_t)(b - ctas[r].dyn) + ((uint32_t)r << 24);
    for (size_t i = 0; i < static_shared.size(); ++i)
        if (static_shared[i] == p) return STATIC_BASE + (uint32_t)i * 64u + ((uint32_t)cur_cta->rank << 24);
    static_shared.push_back(p);
    return STATIC_BASE + (uint32_t)(static_shared.size() - 1) * 64u + ((uint32_t)cur_cta->rank << 24);
}
void *shared_ptr(uint32_t addr) {
    const int rank = (int)(addr >> 24);
    const uint32_t off = addr & 0x00ffffffu;
    if (off >= STATIC_BASE) {
        const uint32_t i = (off - STATIC_BASE) / 64u, rem = (off - STATIC_BASE) % 64u;
        if (i >= static_shared.size()) { fault("shared address 0x%x names no static __shared__ object", addr); return nullptr; }
        return (uint8_t *)static_shared[i] + rem;
    }
    Cta *c = cta_of_rank(rank);
    if (off < WINDOW || off - WINDOW > c->dyn_bytes) { fault("shared address 0x%x outside the %zu dynamic bytes of CTA %d", addr, c->dyn_bytes, rank); return nullptr; }
    return c->dyn + (off - WINDOW);
}

void run_grid(dim3 grid, dim3 block, size_t dyn_bytes, int cluster, const std::function<void()> &body) {
    g_counters[2]++;
    const int T = (int)(block.x * block.y * block.z);
    const long nblocks = (long)grid.x * grid.y * grid.z;
    if (cluster < 1 || grid.x % (unsigned)cluster != 0) { fault("grid %u not a multiple of the cluster size %d", grid.x, cluster); return; }
    if (T % 32 != 0 || T > 1024) { fault("block of %d threads", T); return; }
    blockDim = block; gridDim = grid; g_cluster_size = cluster;
    body_fn = &body;
    if ((int)fibers.size() < T * cluster) fibers.resize((size_t)T * cluster);
    for (auto &f : fibers)
        if (!f.stack) f.stack = (char *)malloc(STACK_BYTES);
    ctas.assign((size_t)cluster, Cta());
    dyn_store.resize((size_t)cluster, nullptr);
    dyn_cap.resize((size_t)cluster, 0);
    for (int r = 0; r < cluster; ++r)
        if (dyn_cap[(size_t)r] < dyn_bytes + 64) {
            free(dyn_store[(size_t)r]);
            void *q = nullptr;
            if (posix_memalign(&q, 1024, dyn_bytes + 1024)) { fault("out of host memory"); return; }
            dyn_store[(size_t)r] = (uint8_t *)q; dyn_cap[(size_t)r] = dyn_bytes + 1024;
        }
    for (long b0 = 0; b0 < nblocks; b0 += cluster) {
        async_q.clear();
        mbar_table().clear();
        cluster_alive = T * cluster; cluster_arrived = 0;
        for (int r = 0; r < cluster; ++r) {
            Cta &c = ctas[(size_t)r];
            float *keep_tmem = c.tmem;
            c = Cta();
            c.tmem = keep_tmem;
            c.rank = r;
            const long b = b0 + r;
            c.bid = dim3((unsigned)(b % grid.x), (unsigned)((b / grid.x) % grid.y), (unsigned)(b / ((long)grid.x * grid.y)));
            memset(dyn_store[(size_t)r], 0xFF, dyn_bytes + 64);   // poison: NaN as float, 0xFFFF as fp16 (NaN too)
            c.dyn = dyn_store[(size_t)r];
            c.dyn_bytes = dyn_bytes;
            c.alive = T;
            for (int w = 0; w < T / 32; ++w) c.warps[w].alive = 32;
            for (int t = 0; t < T; ++t) {
                Fiber &f = fibers[(size_t)r * T + t];
                f.done = false; f.started = false; f.cta = r; f.tid = t; f.cp_seq = 0;
                f.t3 = dim3((unsigned)(t % block.x), (unsigned)((t / block.x) % block.y), (unsigned)(t / (block.x * block.y)));
                getcontext(&f.ctx);
                f.ctx.uc_stack.ss_sp = f.stack;
                f.ctx.uc_stack.ss_size = STACK_BYTES;
                f.ctx.uc_link = nullptr;
                makecontext(&f.ctx, fiber_entry, 0);
            }
        }
        int live = T * cluster;
        while (live > 0) {
            live = 0;
            for (int i = 0; i < T * cluster; ++i) {
                Fiber &f = fibers[(size_t)i];
                if (f.done) continue;
                cur = &f; cur_cta = &ctas[(size_t)f.cta];
                threadIdx = f.t3; blockIdx = cur_cta->bid;
#if EMU_FAST_SWITCH
                if (!_setjmp(sched_jb)) {
                    if (f.started) _longjmp(f.jb, 1);
                    f.started = true;
                    swapcontext(&sched_ctx, &f.ctx);   // first entry: installs the fiber's stack (never returns here)
                }
#else
                swapcontext(&sched_ctx, &f.ctx);
#endif
                if (!f.done) live++;
                drain_async(false);
            }
        }
        drain_async(true);
        flush_cp_log();
        for (int r = 0; r < cluster; ++r)
            if (ctas[(size_t)r].tmem_cols != 0) fault("block %ld exited with %d TMEM columns still allocated", b0 + r, ctas[(size_t)r].tmem_cols);
    }
    cur = nullptr; cur_cta = nullptr;
}

// ------------------------------------------------------------------------------------------ mbarrier
std::unordered_map<uint32_t, MBar> &mbar_table() { static std::unordered_map<uint32_t, MBar> t; return t; }
MBar *mbar_at(uint32_t addr, const char *what) {
    auto it = mbar_table().find(addr);
    if (it == mbar_table().end()) { fault("mbarrier.%s on shared address 0x%x that was never initialised", what, addr); return nullptr; }
    return &it->second;
}
void mbar_check(MBar *m) {
    if (m->pending < 0) fault("mbarrier received more arrivals than its count");
    if (m->pending == 0 && m->tx == 0) { m->phase ^= 1; m->pending = m->expected; }
}

// ------------------------------------------------------------------------------------------ TMA (deferred)
void tma_copy(uint32_t dst, const CUtensorMap *map, int nd, const int *crd, uint32_t bar) {
    TensorMap m;
    memcpy(&m, map, sizeof m);
    g_counters[0]++;
    if (m.magic != 0x454d55544d4150ull || (int)m.rank != nd) { fault("bulk tensor copy through something that is not a %d-d tensor map", nd); return; }
    const bool sw128 = m.swizzle == (uint32_t)CU_TENSOR_MAP_SWIZZLE_128B;
    if (dst & (sw128 ? 1023u : 127u)) fault("bulk tensor copy to shared address 0x%x (needs %d-byte alignment)", dst, sw128 ? 1024 : 128);
    const int c0 = crd[0], c1 = crd[1], c2 = crd[2];
    async_push([=]() {
        const uint32_t row_bytes = m.box[0] * m.elem_bytes;
        uint32_t lin = 0;
        for (uint32_t z = 0; z < m.box[2]; ++z)
            for (uint32_t y = 0; y < m.box[1]; ++y)
                for (uint32_t xb = 0; xb < row_bytes; xb += m.elem_bytes, lin += m.elem_bytes) {
                    const long gx = (long)c0 + xb / m.elem_bytes, gy = (long)c1 + y, gz = (long)c2 + z;
                    const bool in = gx >= 0 && gy >= 0 && gz >= 0 && (uint64_t)gx < m.dim[0] && (uint64_t)gy < m.dim[1] && (uint64_t)gz < m.dim[2];
                    uint32_t a = dst + lin;
                    if (sw128) a ^= ((a >> 7) & 7u) << 4;
                    uint8_t *d = (uint8_t *)shared_ptr(a);
                    if (!d) return;
                    if (in) memcpy(d, m.base + (uint64_t)gx * m.elem_bytes + (uint64_t)gy * m.stride_bytes[1] + (uint64_t)gz * m.stride_bytes[2], m.elem_bytes);
                    else memset(d, 0, m.elem_bytes);
                }
        MBar *b = mbar_at(bar, "complete_tx");
        if (b) { b->tx -= (long)lin; mbar_check(b); }
    });
}

// ------------------------------------------------------------------------------------------ tcgen05.mma kind::f16 (deferred)
namespace {
float f16_to_f32(uint16_t h) {
    const uint32_t sign = (uint32_t)(h & 0x8000u) << 16, e = (h >> 10) & 0x1fu, mnt = h & 0x3ffu;
    uint32_t u;
    if (e == 0) { const float sub = (float)mnt * 5.9604644775390625e-8f; return sign ? -sub : sub; }
    if (e == 31) u = sign | 0x7f800000u | (mnt << 13);
    else u = sign | ((e + 112u) << 23) | (mnt << 13);
    float f; memcpy(&f, &u, 4); return f;
}
// element (row, k) of a K-major SWIZZLE_128B operand: linear address start + (row / 8) SBO + (row % 8) 128 + 2 k,
// then address bits [4,7) ^= bits [7,10)
float operand(int rank, uint64_t desc, int row, int k) {
    const uint32_t start = (uint32_t)(desc & 0x3FFFu) << 4, sbo = (uint32_t)((desc >> 32) & 0x3FFFu) << 4;
    uint32_t a = start + (uint32_t)(row >> 3) * sbo + (uint32_t)(row & 7) * 128u + (uint32_t)k * 2u;
    a ^= ((a >> 7) & 7u) << 4;
    const uint8_t *p = (const uint8_t *)shared_ptr(a | ((uint32_t)rank << 24));
    if (!p) return NAN;
    uint16_t h; memcpy(&h, p, 2);
    return f16_to_f32(h);
}
}  // namespace
void umma(int cg, uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    g_counters[1]++;
    const int M = (int)((idesc >> 24) & 31u) << 4, N = (int)((idesc >> 17) & 63u) << 3;
    const bool fmt_ok = ((idesc >> 4) & 3u) == 1u && ((idesc >> 7) & 7u) == 0u && ((idesc >> 10) & 7u) == 0u && ((idesc >> 15) & 3u) == 0u;
    if (!fmt_ok || M != 128 * cg || N < 16 || N > 256 || N % 16) { fault("tcgen05.mma: instruction descriptor 0x%x (M %d, N %d) for cta_group::%d", idesc, M, N, cg); return; }
    for (uint64_t d : {adesc, bdesc})
        if (((d >> 61) & 7u) != 2u || ((d >> 46) & 3u) != 1u || (((uint32_t)(d & 0x3FFFu) << 4) & 1023u) > 96u)
            { fault("tcgen05.mma: shared-memory descriptor 0x%llx is not a 1024-aligned SWIZZLE_128B tile (+ K advance)", (unsigned long long)d); return; }
    const int col = (int)(tmem_d & 0xffffu);
    if ((tmem_d >> 16) != 0u) { fault("tcgen05.mma: accumulator address 0x%x not at lane 0", tmem_d); return; }
    static float A[256][16], B[256][16];
    for (int m = 0; m < M; ++m)
        for (int k = 0; k < 16; ++k) A[m][k] = operand(m / 128, adesc, m % 128, k);
    const int brows = N / cg;
    for (int n = 0; n < N; ++n)
        for (int k = 0; k < 16; ++k) B[n][k] = operand(n / brows, bdesc, n % brows, k);
    for (int m = 0; m < M; ++m) {
        Cta *c = cta_of_rank(m / 128);
        if (!c->tmem || col + N > c->tmem_cols) { fault("tcgen05.mma: accumulator columns %d..%d outside the %d allocated", col, col + N - 1, c->tmem_cols); return; }
        float *d = c->tmem + (size_t)(m % 128) * 512 + col;
        for (int n = 0; n < N; ++n) {
            float p = 0.0f;
            for (int k = 0; k < 16; ++k) p += A[m][k] * B[n][k];
            d[n] = accumulate ? d[n] + p : p;
        }
    }
}

// ------------------------------------------------------------------------------------------ tensor maps
CUresult encode_tiled(CUtensorMap *out, CUtensorMapDataType dt, cuuint32_t rank, void *base, const cuuint64_t *gdim, const cuuint64_t *gstride,
                      const cuuint32_t *box, const cuuint32_t *estride, CUtensorMapInterleave, CUtensorMapSwizzle sw, CUtensorMapL2promotion,
                      CUtensorMapFloatOOBfill) {
    // the driver's documented argument checks (the ones a wrong call would trip)
    const uint32_t eb = dt == CU_TENSOR_MAP_DATA_TYPE_FLOAT32 ? 4 : (dt == CU_TENSOR_MAP_DATA_TYPE_FLOAT16 ? 2 : 1);
    if (rank < 1 || rank > 3 || ((uintptr_t)base & 15u)) return 1;
    for (cuuint32_t d = 0; d < rank; ++d) {
        if (box[d] < 1 || box[d] > 256 || estride[d] != 1 || gdim[d] < 1) return 1;
        if (d + 1 < rank && (gstride[d] % 16 != 0)) return 1;
    }
    if (((uint64_t)box[0] * eb) % 16 != 0) return 1;
    if (sw == CU_TENSOR_MAP_SWIZZLE_128B && (uint64_t)box[0] * eb > 128) return 1;
    TensorMap m{};
    m.magic = 0x454d55544d4150ull;
    m.base = (const uint8_t *)base; m.elem_bytes = eb; m.rank = rank; m.swizzle = (uint32_t)sw;
    for (cuuint32_t d = 0; d < 3; ++d) {
        m.box[d] = d < rank ? box[d] : 1;
        m.dim[d] = d < rank ? gdim[d] : 1;
        m.stride_bytes[d] = d == 0 ? eb : (d < rank ? gstride[d - 1] : 0);
    }
    memset(out, 0, sizeof *out);
    memcpy(out, &m, sizeof m);
    return CUDA_SUCCESS;
}

}  // namespace emu

// ------------------------------------------------------------------------------------------ cuFFT stub: per-axis DFT, fp64
namespace {
struct Plan { int n[3]; bool used; };
std::vector<Plan> plans;

// forward DFT of one line by recursive decimation in time on the smallest prime factor (any length; fine-grid edges are
// 2-3-5-7-smooth, so this is O(n log n)); x has n complex entries at stride 1, tw[k] = exp(-2 pi i k / n0) for the top length n0
template <class R>
void fft_rec(const R *xr, const R *xi, long stride, int n, R *yr, R *yi, const R *twr, const R *twi, int tw_step) {
    if (n == 1) { yr[0] = xr[0]; yi[0] = xi[0]; return; }
    int p = n;
    for (int q = 2; q * q <= n; ++q)
        if (n % q == 0) { p = q; break; }
    const int m = n / p;
    std::vector<R> sr((size_t)n), si((size_t)n);
    for (int r = 0; r < p; ++r)   // sub-transform of the entries r, r + p, r + 2p, ...
        fft_rec(xr + r * stride, xi + r * stride, stride * p, m, sr.data() + (size_t)r * m, si.data() + (size_t)r * m, twr, twi, tw_step * p);
    for (int k = 0; k < n; ++k) {
        R ar = 0, ai = 0;
        const int km = k % m;
        for (int r = 0; r < p; ++r) {
            const long t = ((long)r * k % n) * tw_step;          // exp(-2 pi i r k / n)
            const R cr = twr[t], ci = twi[t], vr = sr[(size_t)r * m + km], vi = si[(size_t)r * m + km];
            ar += vr * cr - vi * ci;
            ai += vr * ci + vi * cr;
        }
        yr[k] = ar; yi[k] = ai;
    }
}

template <class R>
void dft_axis(std::vector<R> &re, std::vector<R> &im, const int n[3], int axis) {
    const int len = n[axis];
    std::vector<R> cs((size_t)len), sn((size_t)len), lr((size_t)len), li((size_t)len), tr((size_t)len), ti((size_t)len);
    for (int k = 0; k < len; ++k) { cs[(size_t)k] = (R)cos(2.0 * M_PI * k / len); sn[(size_t)k] = (R)-sin(2.0 * M_PI * k / len); }   // forward: exp(-i ...)
    const long stride = axis == 2 ? 1 : (axis == 1 ? n[2] : (long)n[1] * n[2]);
    const long total = (long)n[0] * n[1] * n[2];
    for (long base = 0; base < total; ++base) {
        const long idx_axis = (base / stride) % len;
        if (idx_axis != 0) continue;   // one pass per line
        for (int j = 0; j < len; ++j) { lr[(size_t)j] = re[(size_t)(base + j * stride)]; li[(size_t)j] = im[(size_t)(base + j * stride)]; }
        fft_rec(lr.data(), li.data(), 1, len, tr.data(), ti.data(), cs.data(), sn.data(), 1);
        for (int k = 0; k < len; ++k) { re[(size_t)(base + k * stride)] = tr[(size_t)k]; im[(size_t)(base + k * stride)] = ti[(size_t)k]; }
    }
}
}  // namespace

cufftResult cufftPlan3d(cufftHandle *plan, int nx, int ny, int nz, int) {
    plans.push_back(Plan{{nx, ny, nz}, true});
    *plan = (int)plans.size() - 1;
    return CUFFT_SUCCESS;
}
cufftResult cufftSetStream(cufftHandle, cudaStream_t) { return CUFFT_SUCCESS; }
cufftResult cufftDestroy(cufftHandle) { return CUFFT_SUCCESS; }
cufftResult cufftExecC2C(cufftHandle plan, cufftComplex *in, cufftComplex *out, int dir) {
    if (plan < 0 || plan >= (int)plans.size() || dir != CUFFT_FORWARD) return 1;
    const int *n = plans[(size_t)plan].n;
    const size_t total = (size_t)n[0] * n[1] * n[2];
    // fp64 by default (the stub then adds no error of its own); SPF_EMU_FFT32=1 runs the same transform in fp32, the
    // arithmetic cuFFT uses, to see what an fp32 FFT's rounding does to the slices (tests/test_emu_kernels.py)
    const char *f32 = getenv("SPF_EMU_FFT32");
    if (f32 && f32[0] == '1') {
        std::vector<float> re(total), im(total);
        for (size_t i = 0; i < total; ++i) { re[i] = in[i].x; im[i] = in[i].y; }
        for (int axis = 0; axis < 3; ++axis) dft_axis<float>(re, im, n, axis);
        for (size_t i = 0; i < total; ++i) { out[i].x = re[i]; out[i].y = im[i]; }
        return CUFFT_SUCCESS;
    }
    std::vector<double> re(total), im(total);
    for (size_t i = 0; i < total; ++i) { re[i] = in[i].x; im[i] = in[i].y; }
    for (int axis = 0; axis < 3; ++axis) dft_axis<double>(re, im, n, axis);
    for (size_t i = 0; i < total; ++i) { out[i].x = (float)re[i]; out[i].y = (float)im[i]; }
    return CUFFT_SUCCESS;
}

// ------------------------------------------------------------------------------------------ test hooks (C ABI)
extern "C" {
__attribute__((visibility("default"))) const char *spf_emu_last_fault(void) { return emu::last_fault(); }
__attribute__((visibility("default"))) void spf_emu_counters(long *out4, int reset) {
    for (int i = 0; i < 4; ++i) { out4[i] = emu::g_counters[i]; if (reset) emu::g_counters[i] = 0; }
}
__attribute__((visibility("default"))) void spf_emu_smem_counters(long *out4, int reset) {
    for (int i = 0; i < 4; ++i) { out4[i] = emu::g_smem_counters[i]; if (reset) emu::g_smem_counters[i] = 0; }
}
__attribute__((visibility("default"))) void spf_emu_clear_fault(void) { emu::clear_fault(); }
__attribute__((visibility("default"))) void spf_emu_set_sm_count(int n) { emu::g_sm_count = n > 0 ? n : 1; }
}
