// libspf: context creation and spf_prepare_model (steps a1-a2 of SURVEY.md section 8(a)).
//
// Type-2 NUFFT set-up (Barnett, Magland, af Klinteberg 2019 -- PAPER.md ref [8]; reading s10):
//   kernel   phi(z) = exp(beta (sqrt(1 - z^2) - 1)) on |z| <= 1,  beta = 2.30 w
//   fine grid b_l = sum_n A[n] p(n1) p(n2) p(n3) exp(-i n.l h),  h = 2 pi / n_fine
//   deapodisation  p(n) = 2 / (w phihat(pi w n / n_fine)),  phihat(xi) = 2 int_0^1 phi(z) cos(xi z) dz
// so that  c(x) ~= sum_l b_l phi(2 (x/h - l) / w)  over the w^3 nearest fine cells (spf_slice).
#include <math.h>

#include <new>

#include "spf_internal.cuh"
#include "spf_slice_math.cuh"

// ------------------------------------------------------------------------------------------
// device kernels
// ------------------------------------------------------------------------------------------
// Counts voxels that break A[n] == A[-n] (n = index - floor(N/2)); for even N the unpaired
// index-0 planes must be exactly zero for the fine grid to be real.
__global__ void k_check_even(const float *__restrict__ A, int N, int *__restrict__ bad) {
    const size_t total = (size_t)N * N * N;
    int local = 0;
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        int i3 = (int)(idx % N), i2 = (int)((idx / N) % N), i1 = (int)(idx / ((size_t)N * N));
        local += spfm::voxel_breaks_evenness(A, N, i1, i2, i3) ? 1 : 0;
    }
    local = __reduce_add_sync(0xffffffffu, local);
    if ((threadIdx.x & 31) == 0 && local) atomicAdd(bad, local);
}

// a1: deapodise and scatter into the (already zeroed) n_fine^3 complex grid at index n mod n_fine
__global__ void k_deapod_pad(const float *__restrict__ A, const float *__restrict__ p, int N, int nf,
                             float2 *__restrict__ fine) {
    const size_t total = (size_t)N * N * N;
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        int i3 = (int)(idx % N), i2 = (int)((idx / N) % N), i1 = (int)(idx / ((size_t)N * N));
        const int l1 = spfm::fine_index_of_voxel(i1, N, nf), l2 = spfm::fine_index_of_voxel(i2, N, nf), l3 = spfm::fine_index_of_voxel(i3, N, nf);
        const float v = spfm::deapodised(A[idx], p[i1], p[i2], p[i3]);
        fine[((size_t)l1 * nf + l2) * nf + l3] = make_float2(v, 0.0f);
    }
}

// after the FFT: centred layout with a periodic halo; padded index p <-> fine cell l = p - off (mod n_fine).
// One thread per padded cell; z is the fastest index so both sides are coalesced along z.
__global__ void k_relayout(const float2 *__restrict__ fine, int nf, int np, int sz, int off, float2 *__restrict__ gc,
                           float *__restrict__ gr) {
    const size_t total = (size_t)np * np * sz;
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        int pz = (int)(idx % sz), py = (int)((idx / sz) % np), px = (int)(idx / ((size_t)sz * np));
        float2 v = make_float2(0.f, 0.f);
        if (pz < np) {
            const int l1 = spfm::fine_index_of_padded(px, off, nf), l2 = spfm::fine_index_of_padded(py, off, nf), l3 = spfm::fine_index_of_padded(pz, off, nf);
            v = fine[((size_t)l1 * nf + l2) * nf + l3];
        }
        gc[idx] = v;
        gr[idx] = v.x;
    }
}

// ------------------------------------------------------------------------------------------
// TMA tensor maps for the slicing kernel's tile loads
// ------------------------------------------------------------------------------------------
int spf_build_slice_maps(spf_ctx *ctx) {
    spf_encode_tiled_fn enc = spf_get_encode_tiled();
    if (!enc) return spf_set_err(ctx, SPF_ECUDA, "cuTensorMapEncodeTiled entry point not available");
    for (int real = 0; real < 2; ++real) {
        const int epc = real ? 1 : 2;  // fp32 elements per cell
        for (int iy = 0; iy < SPF_BOX_N; ++iy)
            for (int iz = 0; iz < SPF_BOX_N; ++iz) {
                cuuint64_t gdim[3] = {(cuuint64_t)ctx->sz * epc, (cuuint64_t)ctx->np, (cuuint64_t)ctx->np};
                cuuint64_t gstr[2] = {(cuuint64_t)ctx->sz * epc * 4, (cuuint64_t)ctx->sz * epc * 4 * ctx->np};
                cuuint32_t box[3] = {(cuuint32_t)((SPF_BOX_MIN + SPF_BOX_STEP * iz) * epc),
                                     (cuuint32_t)(SPF_BOX_MIN + SPF_BOX_STEP * iy), 1u};
                cuuint32_t estr[3] = {1, 1, 1};
                void *base = real ? (void *)ctx->d_gridr : (void *)ctx->d_gridc;
                CUtensorMap *dst = real ? &ctx->maps_r.m[iy * SPF_BOX_N + iz] : &ctx->maps_c.m[iy * SPF_BOX_N + iz];
                CUresult r = enc(dst, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, base, gdim, gstr, box, estr,
                                 CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                 CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
                if (r != CUDA_SUCCESS)
                    return spf_set_err(ctx, SPF_ECUDA, "cuTensorMapEncodeTiled(slice tile %d,%d,%d) failed: %d", real, iy, iz, (int)r);
            }
    }
    ctx->maps_ok = true;
    return SPF_OK;
}

// ------------------------------------------------------------------------------------------
// ABI
// ------------------------------------------------------------------------------------------
extern "C" {

void spf_destroy(spf_ctx *ctx) {
    if (!ctx) return;
    cudaSetDevice(ctx->prm.device);
    if (ctx->plan_ok) cufftDestroy(ctx->plan);
    cudaFree(ctx->d_deapod); cudaFree(ctx->d_fft); cudaFree(ctx->d_gridc); cudaFree(ctx->d_gridr);
    cudaFree(ctx->d_flag); cudaFree(ctx->d_patch); cudaFree(ctx->d_abort);
    if (ctx->h_fault) cudaFreeHost((void *)ctx->h_fault);
    auto &b = ctx->hb;
    cudaFree(b.model); cudaFree(b.quats); cudaFree(b.pix); cudaFree(b.images); cudaFree(b.slices);
    cudaFree(b.mask); cudaFree(b.bidx); cudaFree(b.bdist); cudaFree(b.ws);
    if (b.s_main) cudaStreamDestroy(b.s_main);
    if (b.s_copy) cudaStreamDestroy(b.s_copy);
    if (b.ev_img) cudaEventDestroy(b.ev_img);
    for (int k = 0; k < 5; ++k)
        if (ctx->ev[k]) cudaEventDestroy(ctx->ev[k]);
    delete ctx;
}

static int create_impl(spf_ctx *ctx, const spf_params *p) {
    ctx->prm = *p;
    if (p->n < 2 || p->n > 1024) return spf_set_err(ctx, SPF_EINVAL, "n must be in [2, 1024], got %d", p->n);
    ctx->w = spf_plan_kernel_width(p->eps);
    if (ctx->w < 0) return spf_set_err(ctx, SPF_EINVAL, "eps must be in (0, 0.1], got %g", p->eps);
    if (!(p->upsampfac >= 2.0) || p->upsampfac > 4.0)
        return spf_set_err(ctx, SPF_EINVAL, "upsampfac must be in [2, 4], got %g", p->upsampfac);
    ctx->n = p->n;
    ctx->nf = p->n_fine ? p->n_fine : spf_plan_n_fine(p->n, p->upsampfac);
    if (ctx->nf < 2 * p->n) return spf_set_err(ctx, SPF_EINVAL, "n_fine must be >= 2 n, got %d", ctx->nf);
    if (ctx->nf < 2 * ctx->w) return spf_set_err(ctx, SPF_EINVAL, "n_fine %d too small for kernel width %d", ctx->nf, ctx->w);
    ctx->beta = 2.30 * ctx->w;
    ctx->halo = (ctx->w + 1) / 2 + 1;
    ctx->np = ctx->nf + 2 * ctx->halo;
    ctx->sz = (ctx->np + 3) & ~3;

    int ndev = 0;
    SPF_CUDA(ctx, cudaGetDeviceCount(&ndev));
    if (p->device < 0 || p->device >= ndev) return spf_set_err(ctx, SPF_EINVAL, "device %d out of range (%d devices)", p->device, ndev);
    SPF_CUDA(ctx, cudaSetDevice(p->device));
    cudaDeviceProp prop;
    SPF_CUDA(ctx, cudaGetDeviceProperties(&prop, p->device));
    if (prop.major != 10)
        return spf_set_err(ctx, SPF_ECUDA, "libspf is built for sm_100a only; device %d is sm_%d%d", p->device, prop.major, prop.minor);
    ctx->sm_count = prop.multiProcessorCount;

    // deapodisation factors, fp64 on the host
    spfm::deapodisation_factors(ctx->n, ctx->nf, ctx->w, ctx->beta, ctx->deapod);
    std::vector<float> p32(ctx->n);
    for (int i = 0; i < ctx->n; ++i) p32[i] = (float)ctx->deapod[i];
    const size_t nf3 = (size_t)ctx->nf * ctx->nf * ctx->nf, ng = (size_t)ctx->np * ctx->np * ctx->sz;
    SPF_CUDA(ctx, cudaMalloc(&ctx->d_deapod, sizeof(float) * ctx->n));
    SPF_CUDA(ctx, cudaMemcpy(ctx->d_deapod, p32.data(), sizeof(float) * ctx->n, cudaMemcpyHostToDevice));
    SPF_CUDA(ctx, cudaMalloc(&ctx->d_fft, sizeof(float2) * nf3));
    SPF_CUDA(ctx, cudaMalloc(&ctx->d_gridc, sizeof(float2) * ng));
    SPF_CUDA(ctx, cudaMalloc(&ctx->d_gridr, sizeof(float) * ng));
    SPF_CUDA(ctx, cudaMalloc(&ctx->d_flag, sizeof(int)));
    void *hf = nullptr;
    SPF_CUDA(ctx, cudaHostAlloc(&hf, 4 * sizeof(uint32_t), cudaHostAllocMapped));
    memset(hf, 0, 4 * sizeof(uint32_t));
    ctx->h_fault = (volatile uint32_t *)hf;
    SPF_CUDA(ctx, cudaHostGetDevicePointer((void **)&ctx->d_fault, hf, 0));
    SPF_CUDA(ctx, cudaMalloc(&ctx->d_abort, sizeof(uint32_t)));
    SPF_CUDA(ctx, cudaMemset(ctx->d_abort, 0, sizeof(uint32_t)));
    cufftResult fr = cufftPlan3d(&ctx->plan, ctx->nf, ctx->nf, ctx->nf, CUFFT_C2C);
    if (fr != CUFFT_SUCCESS) return spf_set_err(ctx, fr == CUFFT_ALLOC_FAILED ? SPF_ENOMEM : SPF_ECUDA, "cufftPlan3d(%d^3) failed: %d", ctx->nf, (int)fr);
    ctx->plan_ok = true;
    // The tensor maps serve the TMA-staged slicing variants only: if the driver refuses one, the context is
    // still good for the variants that do not use TMA, and spf_slice reports the reason when asked for a staged one.
    if (spf_build_slice_maps(ctx) != SPF_OK) { ctx->maps_err = ctx->err; ctx->err.clear(); }
    SPF_CUDA(ctx, cudaDeviceSynchronize());
    return SPF_OK;
}

int spf_create(spf_ctx **out, const spf_params *p) {
    if (!out || !p) return spf_set_err(nullptr, SPF_EINVAL, "spf_create: null argument");
    *out = nullptr;
    spf_ctx *ctx = new (std::nothrow) spf_ctx();
    if (!ctx) return spf_set_err(nullptr, SPF_ENOMEM, "spf_create: out of host memory");
    int rc = create_impl(ctx, p);
    if (rc) {
        spf_set_err(nullptr, rc, "%s", ctx->err.c_str());
        spf_destroy(ctx);
        return rc;
    }
    *out = ctx;
    return SPF_OK;
}

int spf_prepare_model(spf_ctx *ctx, const float *model, void *stream_) {
    if (!ctx) return SPF_EINVAL;
    if (!model) return spf_set_err(ctx, SPF_EINVAL, "spf_prepare_model: null model");
    cudaStream_t st = (cudaStream_t)stream_;
    SPF_CUDA(ctx, cudaSetDevice(ctx->prm.device));
    const size_t nf3 = (size_t)ctx->nf * ctx->nf * ctx->nf;
    const int blocks = ctx->sm_count * 8;
    SPF_CUDA(ctx, cudaMemsetAsync(ctx->d_flag, 0, sizeof(int), st));
    k_check_even<<<blocks, 256, 0, st>>>(model, ctx->n, ctx->d_flag);
    SPF_LAUNCH_CHECK(ctx);
    SPF_CUDA(ctx, cudaMemsetAsync(ctx->d_fft, 0, sizeof(float2) * nf3, st));
    k_deapod_pad<<<blocks, 256, 0, st>>>(model, ctx->d_deapod, ctx->n, ctx->nf, ctx->d_fft);
    SPF_LAUNCH_CHECK(ctx);
    cufftResult fr = cufftSetStream(ctx->plan, st);
    if (fr == CUFFT_SUCCESS) fr = cufftExecC2C(ctx->plan, (cufftComplex *)ctx->d_fft, (cufftComplex *)ctx->d_fft, CUFFT_FORWARD);
    if (fr != CUFFT_SUCCESS) return spf_set_err(ctx, SPF_ECUDA, "cufftExecC2C failed: %d", (int)fr);
    // (cuFFT's own kernels are not counted in spf_launch_count: it counts this library's kernels only)
    k_relayout<<<blocks, 256, 0, st>>>(ctx->d_fft, ctx->nf, ctx->np, ctx->sz, ctx->nf / 2 + ctx->halo, ctx->d_gridc, ctx->d_gridr);
    SPF_LAUNCH_CHECK(ctx);
    int bad = 1;
    SPF_CUDA(ctx, cudaMemcpyAsync(&bad, ctx->d_flag, sizeof(int), cudaMemcpyDeviceToHost, st));
    SPF_CUDA(ctx, cudaStreamSynchronize(st));
    ctx->grid_is_real = (bad == 0);
    ctx->prepared = true;
    return SPF_OK;
}

int spf_debug_deapodisation(const spf_ctx *ctx, double *out_host) {
    if (!ctx || !out_host) return SPF_EINVAL;
    memcpy(out_host, ctx->deapod.data(), sizeof(double) * ctx->n);
    return SPF_OK;
}

int spf_debug_fine_grid(spf_ctx *ctx, float *out_dev_complex, void *stream_) {
    if (!ctx || !out_dev_complex) return SPF_EINVAL;
    if (!ctx->prepared) return spf_set_err(ctx, SPF_ESTATE, "spf_debug_fine_grid before spf_prepare_model");
    cudaStream_t st = (cudaStream_t)stream_;
    const size_t nf3 = (size_t)ctx->nf * ctx->nf * ctx->nf;
    SPF_CUDA(ctx, cudaMemcpyAsync(out_dev_complex, ctx->d_fft, sizeof(float2) * nf3, cudaMemcpyDeviceToDevice, st));
    SPF_CUDA(ctx, cudaStreamSynchronize(st));
    return SPF_OK;
}

}  // extern "C"
