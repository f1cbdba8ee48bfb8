// libspf: spf_selftest -- the library's own check of a kernel variant against its reference kernels on the device at
// hand, and the switch that turns a verified variant on (the verified-variant choice lives in the C
// library, not in the Python binding).
//
// This is a CONSISTENCY check between two CUDA paths of this library on seeded inputs -- the warp-per-point gathers
// against the one-thread-per-point reference gather, the tcgen05 matcher against the CUDA-core difference-form
// reference (k_match_ref_dist) -- not parity: parity against the oracle is what tests/ does, and nothing here touches
// oracle/.  It runs IN THE CALLING PROCESS: a kernel that raises an SM exception poisons the caller's CUDA context.
// A caller that wants containment runs it in a child process first (paper_2109_05339_b200/selfcheck.py does).
#include <math.h>
#include <stdarg.h>

#include <vector>

#include "spf_internal.cuh"

namespace {

struct Lcg {   // the inputs are data, not method arithmetic: a plain 64-bit LCG, the same on every platform
    uint64_t s;
    explicit Lcg(uint64_t seed) : s(seed * 2862933555777941757ull + 3037000493ull) {}
    uint32_t next() { s = s * 6364136223846793005ull + 1442695040888963407ull; return (uint32_t)(s >> 33); }
    float uni() { return (float)(next() & 0xffffff) / 16777216.0f; }
    float gauss() { float a = 0.f; for (int i = 0; i < 12; ++i) a += uni(); return a - 6.0f; }
};

struct DevBuf {
    void *p = nullptr;
    ~DevBuf() { if (p) cudaFree(p); }
    cudaError_t alloc(size_t n) { return cudaMalloc(&p, n ? n : 16); }
    template <class T> T *as() { return (T *)p; }
};

void say(spf_selftest_report *r, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(r->detail, sizeof r->detail, fmt, ap);
    va_end(ap);
}

float elapsed_ms(cudaEvent_t a, cudaEvent_t b) { float ms = 0.f; cudaEventSynchronize(b); cudaEventElapsedTime(&ms, a, b); return ms; }

// ------------------------------------------------------------------------------------------ slicing variants
// The caller's own prepared model is sliced (read-only) at 64 seeded orientations x a 128 x 128-pixel flat detector (1 M points, 8,192 blocks: long enough to time; 3 x 24 x 24
// with option "selftest_small") on
// the Ewald sphere (8 x 16 lattice patches with the layout promise, 0.9 Nyquist), once with the reference gather and
// once with `impl`; complex output.  Bar: relative L2 difference <= 3e-6 (the two differ in how the kernel weights are
// evaluated -- polynomial fit vs exp / sqrt -- and in summation order), every value finite.
int selftest_slice(spf_ctx *ctx, int impl, spf_selftest_report *rep, cudaStream_t st) {
    if (!ctx->prepared) return spf_set_err(ctx, SPF_ESTATE, "spf_selftest(slice variant) slices the caller's model: call spf_prepare_model first");
    const int edge = ctx->opt_selftest_small ? 24 : 128, P = edge * edge, M = ctx->opt_selftest_small ? 3 : 64;
    std::vector<float> pix((size_t)P * 3), quats((size_t)M * 4);
    double qmax = 0.0;
    for (int r = 0; r < edge; ++r)
        for (int c = 0; c < edge; ++c) {
            const double u = (c + 0.5 - edge / 2.0) / edge, v = (r + 0.5 - edge / 2.0) / edge, nrm = sqrt(u * u + v * v + 1.0);
            const double q[3] = {u / nrm, v / nrm, 1.0 / nrm - 1.0};
            qmax = fmax(qmax, sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2]));
            for (int d = 0; d < 3; ++d) pix[(size_t)(r * edge + c) * 3 + d] = (float)q[d];
        }
    for (auto &v : pix) v = (float)(v * 0.9 * M_PI / qmax);
    Lcg g(11);
    for (auto &v : quats) v = g.gauss();
    DevBuf dq, dp, o_ref, o_var;
    SPF_CUDA(ctx, dq.alloc(quats.size() * 4)); SPF_CUDA(ctx, dp.alloc(pix.size() * 4));
    SPF_CUDA(ctx, o_ref.alloc((size_t)M * P * 8)); SPF_CUDA(ctx, o_var.alloc((size_t)M * P * 8));
    SPF_CUDA(ctx, cudaMemcpyAsync(dq.p, quats.data(), quats.size() * 4, cudaMemcpyHostToDevice, st));
    SPF_CUDA(ctx, cudaMemcpyAsync(dp.p, pix.data(), pix.size() * 4, cudaMemcpyHostToDevice, st));
    const int keep_impl = ctx->opt_slice_impl, keep_lay[3] = {ctx->lay_panels, ctx->lay_rows, ctx->lay_cols};
    ctx->lay_panels = 1; ctx->lay_rows = edge; ctx->lay_cols = edge;
    cudaEvent_t ev[2];
    SPF_CUDA(ctx, cudaEventCreate(&ev[0])); SPF_CUDA(ctx, cudaEventCreate(&ev[1]));
    int rc = SPF_OK;
    float ms[2] = {0.f, 0.f};
    for (int which = 0; which < 2 && rc == SPF_OK; ++which) {
        ctx->opt_slice_impl = which ? impl : 1;
        void *out = which ? o_var.p : o_ref.p;
        for (int rep_i = 0; rep_i < 2 && rc == SPF_OK; ++rep_i) {   // the second run is the timed one
            cudaEventRecord(ev[0], st);
            rc = spf_slice(ctx, dq.as<float>(), M, dp.as<float>(), P, SPF_OUT_COMPLEX, 1.0f, out, st);
            cudaEventRecord(ev[1], st);
            if (rc == SPF_OK) rc = spf_check_fault(ctx, st);
        }
        if (rc == SPF_OK) ms[which] = elapsed_ms(ev[0], ev[1]);
    }
    cudaEventDestroy(ev[0]); cudaEventDestroy(ev[1]);
    ctx->opt_slice_impl = keep_impl;
    ctx->lay_panels = keep_lay[0]; ctx->lay_rows = keep_lay[1]; ctx->lay_cols = keep_lay[2];
    if (rc != SPF_OK) return rc;
    std::vector<float> a((size_t)M * P * 2), b((size_t)M * P * 2);
    SPF_CUDA(ctx, cudaMemcpy(a.data(), o_ref.p, a.size() * 4, cudaMemcpyDeviceToHost));
    SPF_CUDA(ctx, cudaMemcpy(b.data(), o_var.p, b.size() * 4, cudaMemcpyDeviceToHost));
    double num = 0.0, den = 0.0;
    bool finite = true;
    for (size_t i = 0; i < a.size(); ++i) {
        finite = finite && isfinite(b[i]) && isfinite(a[i]);
        num += ((double)b[i] - a[i]) * ((double)b[i] - a[i]);
        den += (double)a[i] * a[i];
    }
    rep->worst_rel = den > 0.0 ? sqrt(num / den) : (num > 0.0 ? INFINITY : 0.0);
    rep->ms_reference = ms[0]; rep->ms_variant = ms[1];
    rep->passed = finite && rep->worst_rel <= 3e-6;
    say(rep, "slice_impl %d vs reference gather: relative L2 %.2e on %d x %d points (w = %d, %s grid), %.3f ms vs %.3f ms", impl,
        rep->worst_rel, M, P, ctx->w, (ctx->grid_is_real && !ctx->opt_force_complex) ? "real" : "complex", ms[1], ms[0]);
    return SPF_OK;
}

// ------------------------------------------------------------------------------------------ tensor-core matcher
// Two seeded cases that span several tiles and ragged tails, each with and without a mask:
//   300 photon-count images x 513 slices x 2,048 pixels (one fp16 image plane, 2 products per K step)
//   130 non-integer, nearly noise-free images x 257 slices x 200 pixels (two image planes, 3 products)
// against spf_match_reference (difference form, fp64 accumulation).  With the refinement (the library's result): distances
// within 1e-4 d.  Without it (the contraction's own a_i + b_m - 2 G): within 1e-4 d + 2e-6 of the norms, the expansion's
// fp32 floor.  Argmin: equal, or the reference's own margin between the two candidates is inside that tolerance.
int selftest_match(spf_ctx *ctx, int impl, int cta_group, spf_selftest_report *rep, cudaStream_t st) {
    const int keep[5] = {ctx->opt_match_impl, ctx->opt_match_cta_group, ctx->opt_match_refine, ctx->opt_record_events, ctx->last_match_impl};
    ctx->opt_match_impl = impl; ctx->opt_match_cta_group = cta_group;
    const char *name = impl == 2 ? "mma.sync matcher" : (cta_group == 2 ? "tcgen05 matcher cta_group::2" : "tcgen05 matcher cta_group::1");
    struct Case { int n_img, M, P; bool counts; } cases[2] = {{300, 513, 2048, true}, {130, 257, 200, false}};
    if (ctx->opt_selftest_small) { cases[0] = Case{140, 18, 320, true}; cases[1] = Case{12, 260, 100, false}; }   // option "selftest_small"
    int rc = SPF_OK;
    bool ok = true;
    double worst = 0.0;
    float ms_var = 0.f, ms_ref = 0.f;
    char why[96] = "";
    cudaEvent_t ev[2];
    SPF_CUDA(ctx, cudaEventCreate(&ev[0])); SPF_CUDA(ctx, cudaEventCreate(&ev[1]));
    Lcg g(5 + (uint64_t)cta_group);
    for (int ci = 0; ci < 2 && rc == SPF_OK && ok; ++ci) {
        const Case c = cases[ci];
        std::vector<float> S((size_t)c.M * c.P), I((size_t)c.n_img * c.P);
        std::vector<uint8_t> mask((size_t)c.P);
        for (int m = 0; m < c.M; ++m) {
            const float bright = 3.0f * g.uni();
            for (int j = 0; j < c.P; ++j) S[(size_t)m * c.P + j] = bright * g.uni();
        }
        for (int i = 0; i < c.n_img; ++i) {
            const int m = (int)(g.next() % (uint32_t)c.M);
            for (int j = 0; j < c.P; ++j) {
                const float lam = S[(size_t)m * c.P + j];
                float v;
                if (c.counts) {   // Poisson by inversion (lam <= 3)
                    float pr = expf(-lam), cum = pr, u = g.uni();
                    int k = 0;
                    while (u > cum && k < 40) { ++k; pr *= lam / (float)k; cum += pr; }
                    v = (float)k;
                } else v = lam + 0.1f * g.uni();
                I[(size_t)i * c.P + j] = v;
            }
        }
        for (auto &b : mask) b = g.uni() > 0.2f ? 1 : 0;
        const size_t ws_bytes = spf_match_workspace_bytes(c.n_img, c.M, c.P);
        DevBuf dS, dI, dm, ws, bi, bd, ri, rd, dist;
        SPF_CUDA(ctx, dS.alloc(S.size() * 4)); SPF_CUDA(ctx, dI.alloc(I.size() * 4)); SPF_CUDA(ctx, dm.alloc(mask.size()));
        SPF_CUDA(ctx, ws.alloc(ws_bytes + 1024));
        SPF_CUDA(ctx, bi.alloc((size_t)c.n_img * 4)); SPF_CUDA(ctx, bd.alloc((size_t)c.n_img * 4));
        SPF_CUDA(ctx, ri.alloc((size_t)c.n_img * 4)); SPF_CUDA(ctx, rd.alloc((size_t)c.n_img * 4));
        SPF_CUDA(ctx, dist.alloc((size_t)c.n_img * c.M * 4));
        SPF_CUDA(ctx, cudaMemcpyAsync(dS.p, S.data(), S.size() * 4, cudaMemcpyHostToDevice, st));
        SPF_CUDA(ctx, cudaMemcpyAsync(dI.p, I.data(), I.size() * 4, cudaMemcpyHostToDevice, st));
        SPF_CUDA(ctx, cudaMemcpyAsync(dm.p, mask.data(), mask.size(), cudaMemcpyHostToDevice, st));
        void *wsp = (void *)(((uintptr_t)ws.p + 1023) & ~(uintptr_t)1023);
        for (int masked = 0; masked < 2 && rc == SPF_OK && ok; ++masked) {
            const uint8_t *mk = masked ? dm.as<uint8_t>() : nullptr;
            cudaEventRecord(ev[0], st);
            rc = spf_match_reference(ctx, dI.as<float>(), c.n_img, dS.as<float>(), c.M, c.P, mk, ri.as<int32_t>(), rd.as<float>(), dist.as<float>(), st);
            cudaEventRecord(ev[1], st);
            if (rc != SPF_OK) break;
            std::vector<float> h_rd((size_t)c.n_img), h_dist((size_t)c.n_img * c.M);
            std::vector<int32_t> h_ri((size_t)c.n_img);
            SPF_CUDA(ctx, cudaMemcpy(h_rd.data(), rd.p, h_rd.size() * 4, cudaMemcpyDeviceToHost));
            SPF_CUDA(ctx, cudaMemcpy(h_ri.data(), ri.p, h_ri.size() * 4, cudaMemcpyDeviceToHost));
            SPF_CUDA(ctx, cudaMemcpy(h_dist.data(), dist.p, h_dist.size() * 4, cudaMemcpyDeviceToHost));
            if (ci == 0 && !masked) ms_ref = elapsed_ms(ev[0], ev[1]);
            std::vector<double> nrm((size_t)c.n_img, 0.0);
            for (int i = 0; i < c.n_img; ++i)
                for (int j = 0; j < c.P; ++j)
                    if (!masked || mask[(size_t)j]) {
                        const double a = I[(size_t)i * c.P + j], b = S[(size_t)h_ri[(size_t)i] * c.P + j];
                        nrm[(size_t)i] += a * a + b * b;
                    }
            for (int refine = 1; refine >= 0 && rc == SPF_OK && ok; --refine) {
                ctx->opt_match_refine = refine;
                cudaEventRecord(ev[0], st);
                rc = spf_match(ctx, dI.as<float>(), c.n_img, dS.as<float>(), c.M, c.P, mk, bi.as<int32_t>(), bd.as<float>(), wsp, ws_bytes, st);
                cudaEventRecord(ev[1], st);
                if (rc == SPF_OK) rc = spf_check_fault(ctx, st);
                if (rc != SPF_OK) break;
                if (ci == 0 && !masked && refine) ms_var = elapsed_ms(ev[0], ev[1]);
                std::vector<float> h_bd((size_t)c.n_img);
                std::vector<int32_t> h_bi((size_t)c.n_img);
                SPF_CUDA(ctx, cudaMemcpy(h_bd.data(), bd.p, h_bd.size() * 4, cudaMemcpyDeviceToHost));
                SPF_CUDA(ctx, cudaMemcpy(h_bi.data(), bi.p, h_bi.size() * 4, cudaMemcpyDeviceToHost));
                for (int i = 0; i < c.n_img && ok; ++i) {
                    const double r = h_rd[(size_t)i], tol = 1e-4 * r + (refine ? 0.0 : 2e-6 * nrm[(size_t)i]);
                    const int m = h_bi[(size_t)i];
                    if (m < 0 || m >= c.M || !isfinite(h_bd[(size_t)i])) { ok = false; snprintf(why, sizeof why, "image %d: index %d / distance not finite", i, m); break; }
                    const double err = fabs((double)h_bd[(size_t)i] - r);
                    if (refine && r > 0.0) worst = fmax(worst, err / r);
                    if (err > tol) { ok = false; snprintf(why, sizeof why, "image %d (refine %d): distance off by %.2e of d", i, refine, err / fmax(r, 1e-30)); }
                    else if (m != h_ri[(size_t)i] && (double)h_dist[(size_t)i * c.M + m] - r > tol) { ok = false; snprintf(why, sizeof why, "image %d (refine %d): argmin %d vs %d", i, refine, m, h_ri[(size_t)i]); }
                }
            }
        }
    }
    cudaEventDestroy(ev[0]); cudaEventDestroy(ev[1]);
    ctx->opt_match_impl = keep[0]; ctx->opt_match_cta_group = keep[1]; ctx->opt_match_refine = keep[2]; ctx->opt_record_events = keep[3];
    ctx->last_match_impl = keep[4];
    ctx->last_scal = nullptr;   // the workspace of the check is gone
    if (rc != SPF_OK) return rc;
    rep->passed = ok; rep->worst_rel = worst; rep->ms_variant = ms_var; rep->ms_reference = ms_ref;
    if (ok) say(rep, "%s vs CUDA-core reference: distances to %.1e, argmin equal outside near-ties, %.3f ms vs %.3f ms", name, worst, ms_var, ms_ref);
    else say(rep, "%s FAILED: %s", name, why);
    return SPF_OK;
}

}  // namespace

extern "C" int spf_selftest(spf_ctx *ctx, const char *variant, spf_selftest_report *report, void *stream_) {
    if (!ctx || !variant || !report) return SPF_EINVAL;
    memset(report, 0, sizeof *report);
    cudaStream_t st = (cudaStream_t)stream_;
    SPF_CUDA(ctx, cudaSetDevice(ctx->prm.device));
    int rc;
    if (!strcmp(variant, "slice_gcoop") || !strcmp(variant, "slice_coop") || !strcmp(variant, "slice_coop_ld")) {
        const int impl = !strcmp(variant, "slice_coop") ? 2 : (!strcmp(variant, "slice_coop_ld") ? 4 : 3);
        if ((rc = selftest_slice(ctx, impl, report, st))) return rc;
        if (report->passed) {
            // among the verified slicers the one this check timed fastest is switched on (never a slower one)
            const float best = ctx->selftest_slice_ms > 0.f ? ctx->selftest_slice_ms : report->ms_reference;
            if (report->ms_variant > 0.f && report->ms_variant < best) { ctx->opt_slice_impl = impl; ctx->selftest_slice_ms = report->ms_variant; }
        }
        return SPF_OK;
    }
    if (!strcmp(variant, "match_mma")) {
        if ((rc = selftest_match(ctx, 2, 1, report, st))) return rc;
        if (report->passed && ctx->opt_match_impl == 1) ctx->opt_match_impl = 2;   // never replaces a verified tcgen05 matcher
        return SPF_OK;
    }
    if (!strcmp(variant, "match_cg1") || !strcmp(variant, "match_cg2")) {
        const int cg = variant[8] == '2' ? 2 : 1;
        if ((rc = selftest_match(ctx, 0, cg, report, st))) return rc;
        if (report->passed) {   // pairs supersede the single-CTA form; the single-CTA form never replaces verified pairs
            if (ctx->opt_match_impl != 0 || cg == 2) ctx->opt_match_cta_group = cg;   // (also supersedes the mma.sync matcher)
            ctx->opt_match_impl = 0;
        }
        return SPF_OK;
    }
    return spf_set_err(ctx, SPF_EINVAL, "spf_selftest: unknown variant %s (slice_gcoop, slice_coop_ld, slice_coop, match_mma, match_cg1, match_cg2)", variant);
}
