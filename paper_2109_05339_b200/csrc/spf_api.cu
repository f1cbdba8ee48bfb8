// libspf: context life cycle, errors, options, and the host-buffer entry point.
#include <math.h>
#include <stdarg.h>

#include "spf_internal.cuh"

static std::string g_create_err;

int spf_set_err(spf_ctx *ctx, int code, const char *fmt, ...) {
    char buf[1024];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (ctx) ctx->err = buf;
    else g_create_err = buf;
    return code;
}

// ------------------------------------------------------------------------------------------
// host-buffer entry point
// ------------------------------------------------------------------------------------------
template <typename T>
static int grow(spf_ctx *ctx, T **p, size_t *cap, size_t bytes) {
    if (bytes <= *cap && *p) return SPF_OK;
    if (*p) { cudaFree(*p); *p = nullptr; *cap = 0; }
    if (bytes == 0) bytes = 16;
    SPF_CUDA(ctx, cudaMalloc((void **)p, bytes));
    *cap = bytes;
    return SPF_OK;
}

extern "C" {

const char *spf_version(void) { return "libspf 0.1 (sm_100a)"; }

const char *spf_status_string(int s) {
    switch (s) {
        case SPF_OK: return "SPF_OK";
        case SPF_EINVAL: return "SPF_EINVAL";
        case SPF_ENOMEM: return "SPF_ENOMEM";
        case SPF_ECUDA: return "SPF_ECUDA";
        case SPF_ESTATE: return "SPF_ESTATE";
        case SPF_EFAULT: return "SPF_EFAULT";
        default: return "SPF_UNKNOWN";
    }
}

const char *spf_last_error(const spf_ctx *ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

// Kernel width for a requested tolerance: w = ceil(log10(1/eps)) + 2, at most 10 (reading s10b).
// The usual rule is "+ 1" (w = 7 at eps = 1e-6).  On the models of this path -- non-negative autocorrelations that fill
// the grid, whose transform has a central peak sum(A) hundreds of times the rms of what the detector sees -- every
// mode's kernel error adds coherently near q = 0 and the relative L2 error OVER THE DETECTOR PIXELS is 0.6 - 1.8e-5 at
// w = 7 (evaluated in fp64, so it is the kernel's own error, not an implementation artefact): it straddles the 1e-5
// parity bar.  One more cell per axis brings it to 1e-6 (7e-7 measured through the fp32 kernel at Paper-scale).
// Beyond w = 10 fp32 arithmetic gains nothing, so eps < 1e-8 keeps w = 10 (the Slicing-heavy configuration).
int32_t spf_plan_kernel_width(double eps) {
    if (!(eps > 0.0) || eps > 0.1) return -1;
    int w = (int)ceil(log10(1.0 / eps) - 1e-9) + 2;
    if (w < 3) w = 3;
    if (w > 10) w = 10;
    return w;
}

static bool smooth2357(int v) {
    for (int p : {2, 3, 5, 7})
        while (v % p == 0) v /= p;
    return v == 1;
}

// smallest even 2-3-5-7-smooth integer >= upsampfac * n: cuFFT then needs no Bluestein pass
// (2 * 151 = 302 has the prime factor 151; the next smooth even size is 320)
int32_t spf_plan_n_fine(int32_t n, double upsampfac) {
    if (n < 2 || !(upsampfac >= 2.0)) return -1;
    int v = (int)ceil(upsampfac * n - 1e-9);
    if (v % 2) ++v;
    while (!smooth2357(v)) v += 2;
    return v;
}

int spf_get_info(const spf_ctx *ctx, spf_info *out) {
    if (!ctx || !out) return SPF_EINVAL;
    out->n = ctx->n; out->n_fine = ctx->nf; out->w = ctx->w; out->beta = ctx->beta;
    out->n_padded = ctx->np; out->grid_is_real = ctx->grid_is_real ? 1 : 0;
    out->prepared = ctx->prepared ? 1 : 0; out->sm_count = ctx->sm_count;
    return SPF_OK;
}

int spf_set_detector_layout(spf_ctx *ctx, int32_t n_panels, int32_t rows, int32_t cols) {
    if (!ctx) return SPF_EINVAL;
    if (n_panels == 0) { ctx->lay_panels = ctx->lay_rows = ctx->lay_cols = 0; return SPF_OK; }
    if (n_panels < 0 || rows <= 0 || cols <= 0) return spf_set_err(ctx, SPF_EINVAL, "detector layout sizes must be positive");
    ctx->lay_panels = n_panels; ctx->lay_rows = rows; ctx->lay_cols = cols;
    return SPF_OK;
}

int spf_set_option(spf_ctx *ctx, const char *key, int64_t value) {
    if (!ctx || !key) return SPF_EINVAL;
    if (!strcmp(key, "slice_impl") && value >= 1 && value <= 4) { ctx->opt_slice_impl = (int)value; return SPF_OK; }
    if (!strcmp(key, "force_complex_grid") && (value == 0 || value == 1)) { ctx->opt_force_complex = (int)value; return SPF_OK; }
    if (!strcmp(key, "match_cta_group") && (value == 1 || value == 2)) { ctx->opt_match_cta_group = (int)value; return SPF_OK; }
    if (!strcmp(key, "match_impl") && value >= 0 && value <= 2) { ctx->opt_match_impl = (int)value; return SPF_OK; }
    if (!strcmp(key, "match_chunk_kblocks") && value >= 0 && value <= (1 << 20)) { ctx->opt_match_chunk_kb = (int)value; return SPF_OK; }
    if (!strcmp(key, "match_condition") && (value == 0 || value == 1)) { ctx->opt_match_condition = (int)value; return SPF_OK; }
    if (!strcmp(key, "match_refine") && (value == 0 || value == 1)) { ctx->opt_match_refine = (int)value; return SPF_OK; }
    if (!strcmp(key, "selftest_small") && (value == 0 || value == 1)) { ctx->opt_selftest_small = (int)value; return SPF_OK; }
    if (!strcmp(key, "record_events") && (value == 0 || value == 1)) { ctx->opt_record_events = (int)value; return SPF_OK; }
    return spf_set_err(ctx, SPF_EINVAL, "unknown option %s=%lld", key, (long long)value);
}

int spf_get_option(const spf_ctx *ctx, const char *key, int64_t *value) {
    if (!ctx || !key || !value) return SPF_EINVAL;
    const struct { const char *k; int v; } tab[] = {
        {"slice_impl", ctx->opt_slice_impl}, {"force_complex_grid", ctx->opt_force_complex}, {"match_cta_group", ctx->opt_match_cta_group},
        {"match_impl", ctx->opt_match_impl}, {"match_chunk_kblocks", ctx->opt_match_chunk_kb}, {"match_condition", ctx->opt_match_condition},
        {"match_refine", ctx->opt_match_refine}, {"selftest_small", ctx->opt_selftest_small}, {"record_events", ctx->opt_record_events}};
    for (const auto &e : tab)
        if (!strcmp(key, e.k)) { *value = e.v; return SPF_OK; }
    return SPF_EINVAL;
}

int spf_check_fault(spf_ctx *ctx, void *stream_) {
    if (!ctx) return SPF_EINVAL;
    SPF_CUDA(ctx, cudaSetDevice(ctx->prm.device));
    SPF_CUDA(ctx, cudaStreamSynchronize((cudaStream_t)stream_));
    if (!ctx->h_fault || ctx->h_fault[0] == 0u) return SPF_OK;
    const uint32_t code = ctx->h_fault[0], block = ctx->h_fault[1], unit = ctx->h_fault[2], variant = ctx->h_fault[3];
    ctx->h_fault[0] = ctx->h_fault[1] = ctx->h_fault[2] = ctx->h_fault[3] = 0u;
    SPF_CUDA(ctx, cudaMemset(ctx->d_abort, 0, sizeof(uint32_t)));   // later launches run again
    if (code >= SPF_FAULT_MATCH) {
        static const char *role[4] = {"TMA producer (slot never freed)", "MMA issuer (accumulator never drained)",
                                      "MMA issuer (operands never arrived)", "epilogue (accumulator never completed)"};
        return spf_set_err(ctx, SPF_EFAULT, "watchdog: k_match_gemm<CG=%u,NI=%u> %s, block %u, tile %u", variant / 10, variant % 10,
                           role[(code - SPF_FAULT_MATCH) & 3u], block, unit);
    }
    return spf_set_err(ctx, SPF_EFAULT, "watchdog: k_slice (variant %u) tile never arrived, block %u", variant, block);
}

int64_t spf_launch_count(const spf_ctx *ctx) { return ctx ? ctx->launches : 0; }

int spf_last_kernel_ms(spf_ctx *ctx, int32_t which, float *ms) {
    if (!ctx || !ms) return SPF_EINVAL;
    if (which < 0 || which > 2) return spf_set_err(ctx, SPF_EINVAL, "spf_last_kernel_ms: which must be 0, 1 or 2");
    if (!ctx->ev_valid[which]) return spf_set_err(ctx, SPF_ESTATE, "spf_last_kernel_ms: nothing recorded (set option record_events=1 first)");
    const int a = which == 0 ? 0 : (which == 1 ? 2 : 4), b = which == 0 ? 1 : (which == 1 ? 3 : 2);
    SPF_CUDA(ctx, cudaEventSynchronize(ctx->ev[b]));
    SPF_CUDA(ctx, cudaEventElapsedTime(ms, ctx->ev[a], ctx->ev[b]));
    return SPF_OK;
}

int spf_orientation_match_host(spf_ctx *ctx, const float *model, const float *quats, int64_t M, const float *pix_q,
                               int64_t P, float scale, const float *images, int64_t n_img, const uint8_t *mask,
                               int32_t *best_idx, float *best_dist, float *slices_out) {
    if (!ctx) return SPF_EINVAL;
    if (!model || !quats || !pix_q || !images || !best_idx || !best_dist || M < 1 || P < 1 || n_img < 1)
        return spf_set_err(ctx, SPF_EINVAL, "spf_orientation_match_host: null pointer or non-positive size");
    SPF_CUDA(ctx, cudaSetDevice(ctx->prm.device));
    auto &b = ctx->hb;
    if (!b.s_main) {
        SPF_CUDA(ctx, cudaStreamCreateWithFlags(&b.s_main, cudaStreamNonBlocking));
        SPF_CUDA(ctx, cudaStreamCreateWithFlags(&b.s_copy, cudaStreamNonBlocking));
        SPF_CUDA(ctx, cudaEventCreateWithFlags(&b.ev_img, cudaEventDisableTiming));
    }
    const size_t n3 = (size_t)ctx->n * ctx->n * ctx->n;
    const size_t ws_bytes = spf_match_workspace_bytes(n_img, M, P);
    int rc;
    if ((rc = grow(ctx, &b.model, &b.cap_model, n3 * 4))) return rc;
    if ((rc = grow(ctx, &b.quats, &b.cap_quats, (size_t)M * 16))) return rc;
    if ((rc = grow(ctx, &b.pix, &b.cap_pix, (size_t)P * 12))) return rc;
    if ((rc = grow(ctx, &b.images, &b.cap_images, (size_t)n_img * P * 4))) return rc;
    if ((rc = grow(ctx, &b.slices, &b.cap_slices, (size_t)M * P * 4))) return rc;
    if ((rc = grow(ctx, &b.mask, &b.cap_mask, (size_t)P))) return rc;
    if ((rc = grow(ctx, &b.bidx, &b.cap_bi, (size_t)n_img * 4))) return rc;
    if ((rc = grow(ctx, &b.bdist, &b.cap_bd, (size_t)n_img * 4))) return rc;
    if ((rc = grow(ctx, &b.ws, &b.cap_ws, ws_bytes))) return rc;

    // images (the large input) upload on the copy stream, underneath prepare + slice
    SPF_CUDA(ctx, cudaMemcpyAsync(b.images, images, (size_t)n_img * P * 4, cudaMemcpyHostToDevice, b.s_copy));
    SPF_CUDA(ctx, cudaEventRecord(b.ev_img, b.s_copy));
    SPF_CUDA(ctx, cudaMemcpyAsync(b.model, model, n3 * 4, cudaMemcpyHostToDevice, b.s_main));
    SPF_CUDA(ctx, cudaMemcpyAsync(b.quats, quats, (size_t)M * 16, cudaMemcpyHostToDevice, b.s_main));
    SPF_CUDA(ctx, cudaMemcpyAsync(b.pix, pix_q, (size_t)P * 12, cudaMemcpyHostToDevice, b.s_main));
    if (mask) SPF_CUDA(ctx, cudaMemcpyAsync(b.mask, mask, (size_t)P, cudaMemcpyHostToDevice, b.s_main));
    if ((rc = spf_prepare_model(ctx, b.model, b.s_main))) return rc;
    if ((rc = spf_slice(ctx, b.quats, M, b.pix, P, SPF_OUT_INTENSITY, scale, b.slices, b.s_main))) return rc;
    SPF_CUDA(ctx, cudaStreamWaitEvent(b.s_main, b.ev_img, 0));
    if ((rc = spf_match(ctx, b.images, n_img, b.slices, M, P, mask ? b.mask : nullptr, b.bidx, b.bdist, b.ws, ws_bytes,
                        b.s_main)))
        return rc;
    SPF_CUDA(ctx, cudaMemcpyAsync(best_idx, b.bidx, (size_t)n_img * 4, cudaMemcpyDeviceToHost, b.s_main));
    SPF_CUDA(ctx, cudaMemcpyAsync(best_dist, b.bdist, (size_t)n_img * 4, cudaMemcpyDeviceToHost, b.s_main));
    if (slices_out)
        SPF_CUDA(ctx, cudaMemcpyAsync(slices_out, b.slices, (size_t)M * P * 4, cudaMemcpyDeviceToHost, b.s_main));
    return spf_check_fault(ctx, b.s_main);
}

}  // extern "C"

int spf_record_event(spf_ctx *ctx, int i, cudaStream_t st) {
    if (!ctx->opt_record_events) return SPF_OK;
    if (!ctx->ev[0])
        for (int k = 0; k < 5; ++k) SPF_CUDA(ctx, cudaEventCreate(&ctx->ev[k]));
    SPF_CUDA(ctx, cudaEventRecord(ctx->ev[i], st));
    return SPF_OK;
}

spf_encode_tiled_fn spf_get_encode_tiled() {
    static spf_encode_tiled_fn fn = nullptr;
    if (fn) return fn;
    void *p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess)
        return nullptr;
    fn = (spf_encode_tiled_fn)p;
    return fn;
}
