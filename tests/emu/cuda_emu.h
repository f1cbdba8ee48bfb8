// tests/emu: a small FUNCTIONAL emulator of the CUDA constructs libspf's kernels use, so that the kernels'
// own source (paper_2109_05339_b200/csrc/*.cu, unchanged except for the mechanical rewrite done by
// build_emu.py) can be compiled with g++ and executed on a box without a GPU.
//
// TEST INFRASTRUCTURE ONLY.  Nothing in the product loads the library built from this (libspf_emu.so);
// it is not a CPU fallback, it is how `-m "not gpu"` tests execute the kernel source against the oracle
// when no B200 can be had.  It shows that the kernels' index arithmetic, barriers,
// pipelines and descriptors are self-consistent under the programming model as this file states it; it
// cannot show that the hardware agrees with that statement, and it says nothing about speed.
//
// Model
//   * a launch runs cluster by cluster (cluster = 1 or 2 consecutive blocks), one cluster at a time, on
//     one OS thread; every CUDA thread of the cluster is a fiber (ucontext) scheduled round-robin;
//   * a fiber runs until it blocks: __syncthreads, a warp collective (__shfl*_sync, __reduce_*_sync,
//     __any/__all_sync, __syncwarp), a cluster barrier, or a failed mbarrier.try_wait (ptx_emu.cuh);
//   * `__shared__` variables are statics (blocks of one launch run one after another), dynamic shared
//     memory is a per-CTA buffer poisoned with NaN bit patterns before every block;
//   * asynchronous engines (TMA copies, tcgen05.mma, tcgen05.commit) are a FIFO of deferred operations
//     drained a few at a time between fiber switches, so a consumer that forgets to wait on the
//     barrier reads poison instead of data;
//   * atomics are plain read-modify-writes (one OS thread);
//   * the runtime API is a set of stubs over malloc / memcpy; cuFFT is a direct per-axis DFT in fp64.
#pragma once
#include <assert.h>
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <functional>
#include <tuple>
#include <type_traits>
#include <utility>

// ------------------------------------------------------------------------------------------ qualifiers
#define __global__
#define __device__
#define __host__
#define __forceinline__ inline
#define __shared__ static
#define __grid_constant__
#define __launch_bounds__(...)
#define __align__(n) __attribute__((aligned(n)))

// ------------------------------------------------------------------------------------------ vector types
struct dim3 {
    unsigned x = 1, y = 1, z = 1;
    dim3() = default;
    dim3(unsigned x_, unsigned y_ = 1, unsigned z_ = 1) : x(x_), y(y_), z(z_) {}
};
struct alignas(8) float2 { float x, y; };
struct alignas(16) float4 { float x, y, z, w; };
inline float2 make_float2(float x, float y) { float2 r; r.x = x; r.y = y; return r; }
inline float4 make_float4(float x, float y, float z, float w) { float4 r; r.x = x; r.y = y; r.z = z; r.w = w; return r; }
struct __half { uint16_t x; };
inline __half __ushort_as_half(uint16_t u) { __half h; h.x = u; return h; }
inline uint16_t __half_as_ushort(__half h) { return h.x; }

// ------------------------------------------------------------------------------------------ the scheduler
namespace emu {

struct Warp {
    unsigned gen = 0;
    int arrived = 0, alive = 0;
    uint64_t vals[2][32];
};

struct Cta {
    int rank = 0;                 // rank inside the cluster
    dim3 bid;
    uint8_t *dyn = nullptr;       // dynamic shared memory
    size_t dyn_bytes = 0;
    int alive = 0, bar_arrived = 0;
    unsigned bar_gen = 0;
    Warp warps[32];
    float *tmem = nullptr;        // [128 lanes][512 columns], allocated on first tcgen05.alloc
    int tmem_cols = 0;
};

struct Fiber;
extern Fiber *cur;                // running fiber
extern Cta *cur_cta;
extern int g_cluster_size;
extern long long g_ticks;         // clock64(): advances at every fiber switch and every call
extern int g_sm_count;            // multiprocessors the emulated device reports (small: persistent loops take several tiles)

void yield();                                             // give the other fibers of the cluster a turn
void run_grid(dim3 grid, dim3 block, size_t dyn_smem, int cluster, const std::function<void()> &body);
Cta *cta_of_rank(int rank);                               // CTA `rank` of the running cluster
int cur_tid();                                            // linear thread index inside the block
void block_barrier();
void cluster_barrier();
const uint64_t *warp_collective(uint64_t my_value);       // returns the 32 deposited values
void async_push(std::function<void()> op);                // deferred (TMA / tensor-core) operation
uint32_t shared_addr(const void *p);                      // 32-bit shared-window address (CTA rank in bit 24)
void *shared_ptr(uint32_t addr);                          // and back (any CTA of the running cluster)
void *dyn_smem();
const char *last_fault();                                 // non-empty after an emulator assertion (bad address, ...)
void fault(const char *fmt, ...);
void clear_fault();
extern long g_counters[4];
// shared-memory wavefront accounting of the 16-byte-granular instructions (a MODEL: 8 x 16-byte bank groups per 128-byte
// wavefront, a warp-wide access served quarter-warp by quarter-warp, equal addresses merged)
extern long g_smem_counters[4];      // [0] ldmatrix 8-row phases, [1] wavefronts they take, [2] cp.async.16 quarter-warp groups, [3] wavefronts
void note_ldmatrix(const uint64_t *addr32);
void note_cp_async16(uint32_t dst);

template <class... KA, class... A>
void launch(void (*kern)(KA...), dim3 grid, dim3 block, size_t dyn_smem, int cluster, A &&...a) {
    std::tuple<std::decay_t<KA>...> args(std::forward<A>(a)...);
    run_grid(grid, block, dyn_smem, cluster, [&]() { std::apply(kern, args); });
}

}  // namespace emu

// the built-in index variables: plain globals the scheduler rewrites at every fiber switch
extern dim3 threadIdx, blockIdx, blockDim, gridDim;

// ------------------------------------------------------------------------------------------ device intrinsics
inline void __syncthreads() { emu::block_barrier(); }
inline void __syncwarp(unsigned = 0xffffffffu) { emu::warp_collective(0); }
inline void __threadfence() {}
inline void __threadfence_system() {}
inline void __threadfence_block() {}
inline long long clock64() { return ++emu::g_ticks; }
template <class T> inline T __ldg(const T *p) { return *p; }
template <class T> inline T __ldcg(const T *p) { return *p; }
inline uint32_t __float_as_uint(float f) { uint32_t u; memcpy(&u, &f, 4); return u; }
inline float __uint_as_float(uint32_t u) { float f; memcpy(&f, &u, 4); return f; }
inline size_t __cvta_generic_to_shared(const void *p) { return emu::shared_addr(p); }

namespace emu {
template <class T> inline uint64_t to_bits(T v) { uint64_t u = 0; static_assert(sizeof(T) <= 8, ""); memcpy(&u, &v, sizeof(T)); return u; }
template <class T> inline T from_bits(uint64_t u) { T v; memcpy(&v, &u, sizeof(T)); return v; }
inline int lane() { return cur_tid() & 31; }
}  // namespace emu

template <class T> inline T __shfl_sync(unsigned, T v, int src) { return emu::from_bits<T>(emu::warp_collective(emu::to_bits(v))[src & 31]); }
template <class T> inline T __shfl_xor_sync(unsigned, T v, int m) { const int l = emu::lane(); return emu::from_bits<T>(emu::warp_collective(emu::to_bits(v))[(l ^ m) & 31]); }
// reductions and votes run over the lanes that are still alive (a full-mask collective with exited lanes is
// undefined in CUDA; the kernels never do that, and the emulator asserts it)
namespace emu {
int warp_alive_mask();
template <class T, class F> inline T warp_reduce(T v, F f) {
    const uint64_t *s = warp_collective(to_bits(v));
    const int mask = warp_alive_mask();
    bool first = true; T r = v;
    for (int l = 0; l < 32; ++l)
        if (mask >> l & 1) { const T x = from_bits<T>(s[l]); r = first ? x : f(r, x); first = false; }
    return r;
}
}  // namespace emu
inline int __reduce_min_sync(unsigned, int v) { return emu::warp_reduce(v, [](int a, int b) { return a < b ? a : b; }); }
inline int __reduce_max_sync(unsigned, int v) { return emu::warp_reduce(v, [](int a, int b) { return a > b ? a : b; }); }
inline int __reduce_add_sync(unsigned, int v) { return emu::warp_reduce(v, [](int a, int b) { return a + b; }); }
inline unsigned __reduce_min_sync(unsigned, unsigned v) { return emu::warp_reduce(v, [](unsigned a, unsigned b) { return a < b ? a : b; }); }
inline unsigned __reduce_max_sync(unsigned, unsigned v) { return emu::warp_reduce(v, [](unsigned a, unsigned b) { return a > b ? a : b; }); }
inline unsigned __reduce_add_sync(unsigned, unsigned v) { return emu::warp_reduce(v, [](unsigned a, unsigned b) { return a + b; }); }
inline int __any_sync(unsigned, int p) { return emu::warp_reduce(p != 0 ? 1 : 0, [](int a, int b) { return a | b; }); }
inline int __all_sync(unsigned, int p) { return emu::warp_reduce(p != 0 ? 1 : 0, [](int a, int b) { return a & b; }); }

template <class T> inline T atomicAdd(T *p, T v) { T o = *p; *p = o + v; return o; }
template <class T> inline T atomicMin(T *p, T v) { T o = *p; if (v < o) *p = v; return o; }
template <class T> inline T atomicMax(T *p, T v) { T o = *p; if (v > o) *p = v; return o; }
template <class T> inline T atomicOr(T *p, T v) { T o = *p; *p = o | v; return o; }
template <class T> inline T atomicExch(T *p, T v) { T o = *p; *p = v; return o; }

template <class T> inline T min(T a, T b) { return a < b ? a : b; }
template <class T> inline T max(T a, T b) { return a > b ? a : b; }

// ------------------------------------------------------------------------------------------ runtime API
typedef int cudaError_t;
enum { cudaSuccess = 0, cudaErrorMemoryAllocation = 2, cudaErrorInvalidValue = 1 };
typedef struct emuStream *cudaStream_t;
typedef struct emuEvent *cudaEvent_t;
enum cudaMemcpyKind { cudaMemcpyHostToHost, cudaMemcpyHostToDevice, cudaMemcpyDeviceToHost, cudaMemcpyDeviceToDevice };
enum { cudaStreamNonBlocking = 1, cudaEventDisableTiming = 2, cudaHostAllocMapped = 2, cudaEnableDefault = 0 };
enum cudaFuncAttribute { cudaFuncAttributeMaxDynamicSharedMemorySize = 8, cudaFuncAttributePreferredSharedMemoryCarveout = 9 };
enum { cudaSharedmemCarveoutMaxShared = 100 };
enum cudaDriverEntryPointQueryResult { cudaDriverEntryPointSuccess = 0, cudaDriverEntryPointSymbolNotFound = 1 };
struct cudaDeviceProp { int major, minor, multiProcessorCount; };

inline const char *cudaGetErrorString(cudaError_t e) { return e == cudaSuccess ? "no error" : (e == cudaErrorMemoryAllocation ? "out of memory" : "emulator error"); }
inline cudaError_t cudaGetLastError() { return cudaSuccess; }
inline cudaError_t cudaSetDevice(int) { return cudaSuccess; }
inline cudaError_t cudaGetDeviceCount(int *n) { *n = 1; return cudaSuccess; }
inline cudaError_t cudaGetDeviceProperties(cudaDeviceProp *p, int) { p->major = 10; p->minor = 0; p->multiProcessorCount = emu::g_sm_count; return cudaSuccess; }
inline cudaError_t cudaDeviceSynchronize() { return cudaSuccess; }
template <class T> inline cudaError_t cudaMalloc(T **p, size_t n) {
    void *q = nullptr;
    if (posix_memalign(&q, 1024, n ? n : 16)) return cudaErrorMemoryAllocation;
    memset(q, 0xFF, n);   // device memory is not zeroed: poison it (NaN bit patterns)
    *p = (T *)q;
    return cudaSuccess;
}
inline cudaError_t cudaFree(void *p) { free(p); return cudaSuccess; }
inline cudaError_t cudaHostAlloc(void **p, size_t n, unsigned) { *p = calloc(1, n); return *p ? cudaSuccess : cudaErrorMemoryAllocation; }
inline cudaError_t cudaHostGetDevicePointer(void **d, void *h, unsigned) { *d = h; return cudaSuccess; }
inline cudaError_t cudaFreeHost(void *p) { free(p); return cudaSuccess; }
inline cudaError_t cudaMemcpy(void *d, const void *s, size_t n, cudaMemcpyKind) { memmove(d, s, n); return cudaSuccess; }
inline cudaError_t cudaMemcpyAsync(void *d, const void *s, size_t n, cudaMemcpyKind, cudaStream_t = nullptr) { memmove(d, s, n); return cudaSuccess; }
inline cudaError_t cudaMemset(void *d, int v, size_t n) { memset(d, v, n); return cudaSuccess; }
inline cudaError_t cudaMemsetAsync(void *d, int v, size_t n, cudaStream_t = nullptr) { memset(d, v, n); return cudaSuccess; }
inline cudaError_t cudaStreamCreateWithFlags(cudaStream_t *s, unsigned) { *s = (cudaStream_t)malloc(8); return cudaSuccess; }
inline cudaError_t cudaStreamDestroy(cudaStream_t s) { free(s); return cudaSuccess; }
inline cudaError_t cudaStreamSynchronize(cudaStream_t) { return cudaSuccess; }
inline cudaError_t cudaStreamWaitEvent(cudaStream_t, cudaEvent_t, unsigned) { return cudaSuccess; }
// events carry the host clock at record time (launches are synchronous here), so elapsed times are positive
struct emuEvent { double t_ms; };
double emu_now_ms();
inline cudaError_t cudaEventCreate(cudaEvent_t *e) { *e = (cudaEvent_t)calloc(1, sizeof(emuEvent)); return cudaSuccess; }
inline cudaError_t cudaEventCreateWithFlags(cudaEvent_t *e, unsigned) { return cudaEventCreate(e); }
inline cudaError_t cudaEventDestroy(cudaEvent_t e) { free(e); return cudaSuccess; }
inline cudaError_t cudaEventRecord(cudaEvent_t e, cudaStream_t = nullptr) { e->t_ms = emu_now_ms(); return cudaSuccess; }
inline cudaError_t cudaEventSynchronize(cudaEvent_t) { return cudaSuccess; }
inline cudaError_t cudaEventElapsedTime(float *ms, cudaEvent_t a, cudaEvent_t b) { *ms = (float)fmax(b->t_ms - a->t_ms, 1e-3); return cudaSuccess; }
template <class K> inline cudaError_t cudaFuncSetAttribute(K, cudaFuncAttribute, int) { return cudaSuccess; }

enum cudaLaunchAttributeID { cudaLaunchAttributeClusterDimension = 4 };
struct cudaLaunchAttribute {
    cudaLaunchAttributeID id;
    struct { struct { unsigned x, y, z; } clusterDim; } val;
};
struct cudaLaunchConfig_t {
    dim3 gridDim, blockDim;
    size_t dynamicSmemBytes = 0;
    cudaStream_t stream = nullptr;
    cudaLaunchAttribute *attrs = nullptr;
    unsigned numAttrs = 0;
};
inline int emu_cluster_of(const cudaLaunchConfig_t *cfg) {
    for (unsigned i = 0; i < cfg->numAttrs; ++i)
        if (cfg->attrs[i].id == cudaLaunchAttributeClusterDimension) return (int)cfg->attrs[i].val.clusterDim.x;
    return 1;
}
template <class K> inline cudaError_t cudaOccupancyMaxActiveClusters(int *n, K, const cudaLaunchConfig_t *cfg) {
    *n = emu::g_sm_count / emu_cluster_of(cfg);
    return cudaSuccess;
}
template <class... KA, class... A>
inline cudaError_t cudaLaunchKernelEx(const cudaLaunchConfig_t *cfg, void (*kern)(KA...), A &&...a) {
    emu::launch(kern, cfg->gridDim, cfg->blockDim, cfg->dynamicSmemBytes, emu_cluster_of(cfg), std::forward<A>(a)...);
    return cudaSuccess;
}

// ------------------------------------------------------------------------------------------ driver API: tensor maps
typedef int CUresult;
enum { CUDA_SUCCESS = 0 };
typedef uint64_t cuuint64_t;
typedef uint32_t cuuint32_t;
enum CUtensorMapDataType { CU_TENSOR_MAP_DATA_TYPE_UINT8 = 0, CU_TENSOR_MAP_DATA_TYPE_FLOAT16 = 6, CU_TENSOR_MAP_DATA_TYPE_FLOAT32 = 7 };
enum CUtensorMapInterleave { CU_TENSOR_MAP_INTERLEAVE_NONE = 0 };
enum CUtensorMapSwizzle { CU_TENSOR_MAP_SWIZZLE_NONE = 0, CU_TENSOR_MAP_SWIZZLE_32B, CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_SWIZZLE_128B };
enum CUtensorMapL2promotion { CU_TENSOR_MAP_L2_PROMOTION_NONE = 0, CU_TENSOR_MAP_L2_PROMOTION_L2_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B };
enum CUtensorMapFloatOOBfill { CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE = 0 };
struct alignas(64) CUtensorMap { uint64_t opaque[16]; };
namespace emu {
struct TensorMap {   // what the emulator keeps inside the 128 opaque bytes
    uint64_t magic;
    const uint8_t *base;
    uint32_t elem_bytes, rank, swizzle;
    uint32_t box[3];
    uint64_t dim[3], stride_bytes[3];   // stride_bytes[0] = elem_bytes
};
static_assert(sizeof(TensorMap) <= sizeof(CUtensorMap), "tensor-map record fits the opaque blob");
CUresult encode_tiled(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                      const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
}  // namespace emu
inline cudaError_t cudaGetDriverEntryPoint(const char *name, void **fn, unsigned, cudaDriverEntryPointQueryResult *q) {
    if (!strcmp(name, "cuTensorMapEncodeTiled")) { *fn = (void *)&emu::encode_tiled; *q = cudaDriverEntryPointSuccess; return cudaSuccess; }
    *q = cudaDriverEntryPointSymbolNotFound;
    return cudaErrorInvalidValue;
}

// ------------------------------------------------------------------------------------------ cuFFT (3-D C2C, forward)
typedef int cufftHandle;
typedef int cufftResult;
typedef float2 cufftComplex;
enum { CUFFT_SUCCESS = 0, CUFFT_ALLOC_FAILED = 2, CUFFT_C2C = 0x29, CUFFT_FORWARD = -1 };
cufftResult cufftPlan3d(cufftHandle *plan, int nx, int ny, int nz, int type);
cufftResult cufftSetStream(cufftHandle, cudaStream_t);
cufftResult cufftExecC2C(cufftHandle plan, cufftComplex *in, cufftComplex *out, int dir);
cufftResult cufftDestroy(cufftHandle);
