// libspf: spf_microbench -- the two SM-side denominators SURVEY.md section 8(d) says must be MEASURED, not taken from a data
// sheet: the aggregate shared-memory load bandwidth (what k_slice's "smem" roofline divides by)
// and the L2 -> SM bandwidth (what bounds k_match_gemm's operand traffic), plus a plain HBM copy as a sanity check
// against MEASURED_PEAKS.json.  bench.py calls it before the timed region and reports the figures in `peaks`.
#include "spf_internal.cuh"

namespace {

constexpr int MB_THREADS = 512;
constexpr int MB_WORDS = 8192;      // 32 KB of shared memory per block: 2-4 blocks per SM

// Every lane loads consecutive 4-byte words: one conflict-free wavefront (128 bytes) per warp instruction.  Eight
// independent accumulators keep eight loads in flight per thread; the volatile pointer keeps every load in the SASS.
__global__ void __launch_bounds__(MB_THREADS) k_mb_lds32(int iters, float *out) {
    __shared__ float s[MB_WORDS];
    for (int i = threadIdx.x; i < MB_WORDS; i += MB_THREADS) s[i] = (float)(i & 7);
    __syncthreads();
    const volatile float *v = s;
    float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    int base = threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) acc[u] += v[(base + u * MB_THREADS) & (MB_WORDS - 1)];
        base = (base + 8 * MB_THREADS + 32) & (MB_WORDS - 1);
    }
    float t = 0.f;
    for (int u = 0; u < 8; ++u) t += acc[u];
    if (t == -1.0f) out[0] = t;   // never true: keeps the loop alive without a store per thread
}

// The same with 16-byte loads (a quarter-warp per wavefront): the form a staged gather with vector loads would use.
__global__ void __launch_bounds__(MB_THREADS) k_mb_lds128(int iters, float *out) {
    __shared__ __align__(16) float s[MB_WORDS];
    for (int i = threadIdx.x; i < MB_WORDS; i += MB_THREADS) s[i] = (float)(i & 7);
    __syncthreads();
    const float4 *v = reinterpret_cast<const float4 *>(s);
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    int base = threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const float4 *p = &v[(base + u * MB_THREADS) & (MB_WORDS / 4 - 1)];
            float4 q;
#if defined(__CUDA_ARCH__)
            // one 16-byte shared load that the compiler can neither split, hoist nor drop
            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(q.x), "=f"(q.y), "=f"(q.z), "=f"(q.w) : "r"((uint32_t)__cvta_generic_to_shared(p)));
#else
            q = *p;
#endif
            acc[u] += q.x + q.y + q.z + q.w;
        }
        base = (base + 4 * MB_THREADS + 8) & (MB_WORDS / 4 - 1);
    }
    const float t = acc[0] + acc[1] + acc[2] + acc[3];
    if (t == -1.0f) out[0] = t;
}

// Streams `n4` float4 through every SM `passes` times with loads that bypass L1 (ld.global.cg): with a buffer that
// fits L2 (48 MB of 126) the later passes measure L2 -> SM; with a buffer far beyond L2 they measure HBM reads.
__global__ void __launch_bounds__(256) k_mb_read(const float4 *__restrict__ buf, size_t n4, int passes, float *out) {
    float acc = 0.f;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (int p = 0; p < passes; ++p) {
        size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
        for (; i + 3 * stride < n4; i += 4 * stride) {   // four independent 16-byte loads in flight per thread
            const float4 a = __ldcg(buf + i), b = __ldcg(buf + i + stride), c = __ldcg(buf + i + 2 * stride), d = __ldcg(buf + i + 3 * stride);
            acc += (a.x + a.y + a.z + a.w) + (b.x + b.y + b.z + b.w) + (c.x + c.y + c.z + c.w) + (d.x + d.y + d.z + d.w);
        }
        for (; i < n4; i += stride) { const float4 a = __ldcg(buf + i); acc += a.x + a.y + a.z + a.w; }
    }
    if (acc == -1.0f) out[0] = acc;
}

__global__ void __launch_bounds__(256) k_mb_copy(const float4 *__restrict__ src, float4 *__restrict__ dst, size_t n4) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) dst[i] = src[i];
}

}  // namespace

extern "C" int spf_microbench(spf_ctx *ctx, const char *what, double *gb_per_s, void *stream_) {
    if (!ctx || !what || !gb_per_s) return SPF_EINVAL;
    *gb_per_s = 0.0;
    cudaStream_t st = (cudaStream_t)stream_;
    SPF_CUDA(ctx, cudaSetDevice(ctx->prm.device));
    const bool small = ctx->opt_selftest_small != 0;   // quick functional run (the emulator): tiny sizes, the number means nothing
    cudaEvent_t e0, e1;
    SPF_CUDA(ctx, cudaEventCreate(&e0)); SPF_CUDA(ctx, cudaEventCreate(&e1));
    float *d_out = nullptr, *buf = nullptr, *buf2 = nullptr;
    double bytes = 0.0;
    float best_ms = 1e30f;
    int rc = SPF_OK;
    auto fail = [&](cudaError_t e, const char *call) { rc = spf_set_err(ctx, SPF_ECUDA, "%s failed: %s", call, cudaGetErrorString(e)); };
    cudaError_t e = cudaMalloc(&d_out, 64);
    if (e != cudaSuccess) fail(e, "cudaMalloc");
    const bool lds32 = !strcmp(what, "lds32"), lds128 = !strcmp(what, "lds128"), l2 = !strcmp(what, "l2"), hbm_r = !strcmp(what, "hbm_read"),
               hbm_c = !strcmp(what, "hbm_copy");
    if (rc == SPF_OK && !(lds32 || lds128 || l2 || hbm_r || hbm_c))
        rc = spf_set_err(ctx, SPF_EINVAL, "spf_microbench: unknown measurement %s (lds32, lds128, l2, hbm_read, hbm_copy)", what);
    if (rc == SPF_OK && (lds32 || lds128)) {
        const int iters = small ? 4 : 20000, blocks = ctx->sm_count * (small ? 1 : 4);
        bytes = (double)blocks * MB_THREADS * iters * (lds32 ? 8 * 4 : 4 * 16);
        for (int rep = 0; rep < (small ? 1 : 4); ++rep) {   // first repetition is the warm-up
            cudaEventRecord(e0, st);
            if (lds32) k_mb_lds32<<<blocks, MB_THREADS, 0, st>>>(iters, d_out);
            else k_mb_lds128<<<blocks, MB_THREADS, 0, st>>>(iters, d_out);
            cudaEventRecord(e1, st);
            if ((e = cudaEventSynchronize(e1)) != cudaSuccess) { fail(e, "k_mb_lds"); break; }
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 || small) best_ms = ms < best_ms ? ms : best_ms;
            ctx->launches++;
        }
    }
    if (rc == SPF_OK && (l2 || hbm_r || hbm_c)) {
        const size_t n4 = small ? 4096 : (l2 ? (48u << 20) : (1024u << 20)) / 16;   // 48 MB inside L2; 1 GB far beyond it
        const int passes = small ? 1 : (l2 ? 20 : 2), blocks = ctx->sm_count * (small ? 1 : 16);
        if ((e = cudaMalloc(&buf, n4 * 16)) != cudaSuccess) fail(e, "cudaMalloc");
        if (rc == SPF_OK && hbm_c && (e = cudaMalloc(&buf2, n4 * 16)) != cudaSuccess) fail(e, "cudaMalloc");
        if (rc == SPF_OK) {
            cudaMemsetAsync(buf, 0, n4 * 16, st);
            bytes = hbm_c ? 2.0 * n4 * 16 : (double)n4 * 16 * passes;
            for (int rep = 0; rep < (small ? 1 : 4); ++rep) {
                cudaEventRecord(e0, st);
                if (hbm_c) k_mb_copy<<<blocks, 256, 0, st>>>((const float4 *)buf, (float4 *)buf2, n4);
                else k_mb_read<<<blocks, 256, 0, st>>>((const float4 *)buf, n4, passes, d_out);
                cudaEventRecord(e1, st);
                if ((e = cudaEventSynchronize(e1)) != cudaSuccess) { fail(e, "k_mb_read"); break; }
                float ms = 0.f;
                cudaEventElapsedTime(&ms, e0, e1);
                if (rep > 0 || small) best_ms = ms < best_ms ? ms : best_ms;
                ctx->launches++;
            }
        }
    }
    cudaFree(d_out); cudaFree(buf); cudaFree(buf2);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (rc != SPF_OK) return rc;
    *gb_per_s = bytes / (best_ms * 1e-3) / 1e9;
    return SPF_OK;
}
