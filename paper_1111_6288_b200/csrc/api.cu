// C ABI entry points (include/ov.h): argument checks, context lifetime, workspaces.
#include <cmath>
#include <cstring>

#include "ov_internal.h"

namespace ov {

int fail(const ov_ctx* ctx, int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (ctx) ctx->err = buf;
    return code;
}

int cuda_fail(const ov_ctx* ctx, cudaError_t e, const char* what) {
    return fail(ctx, e == cudaErrorMemoryAllocation ? OV_ENOMEM : OV_ECUDA, "CUDA error '%s' in %s",
                cudaGetErrorString(e), what);
}

int workspace(ov_ctx* ctx, int i, double2** out) {
    if (!ctx->ws[i]) OV_CUDA(ctx, cudaMalloc(&ctx->ws[i], spinor_elems(ctx) * sizeof(double2)));
    *out = ctx->ws[i];
    return OV_OK;
}

int workspace_f32(ov_ctx* ctx, int i, float2** out) {
    if (!ctx->wsf[i]) OV_CUDA(ctx, cudaMalloc(&ctx->wsf[i], spinor_elems(ctx) * sizeof(float2)));
    *out = ctx->wsf[i];
    return OV_OK;
}

int ensure_reduction_buffers(ov_ctx* ctx, size_t partial_elems, size_t result_elems) {
    if (partial_elems > ctx->partial_cap) {
        OV_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        if (ctx->d_partial) cudaFree(ctx->d_partial);
        ctx->d_partial = nullptr;
        ctx->partial_cap = 0;
        OV_CUDA(ctx, cudaMalloc(&ctx->d_partial, partial_elems * sizeof(double2)));
        ctx->partial_cap = partial_elems;
    }
    if (result_elems > ctx->result_cap) {
        OV_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        if (ctx->d_result) cudaFree(ctx->d_result);
        if (ctx->h_result) cudaFreeHost(ctx->h_result);
        ctx->d_result = nullptr;
        ctx->h_result = nullptr;
        ctx->result_cap = 0;
        const size_t cap = result_elems < 1024 ? 1024 : result_elems;
        OV_CUDA(ctx, cudaMalloc(&ctx->d_result, cap * sizeof(double2)));
        OV_CUDA(ctx, cudaMallocHost(&ctx->h_result, cap * sizeof(double2)));
        ctx->result_cap = cap;
    }
    return OV_OK;
}

static bool tma_usable(const ov_ctx* ctx) { return ctx->tma_ok && !ctx->blocked && tma_eligible(ctx->lat); }

int effective_variant(const ov_ctx* ctx) {
    if (ctx->dslash_variant == 1) return 1;
    if (ctx->dslash_variant == 2) return 2;
    return tma_usable(ctx) ? 2 : 1;
}

// Automatic choice (variant 0): the TMA-staged kernel wherever it applies (planes layout, X % 8 == Y % 4 == Z % 4 == 0),
// for launches with and without fused axpy operands (measured: DESIGN.md section 10); the gather kernel otherwise.
// An explicit variant 1 or 2 sends every single-right-hand-side launch to that kernel.
int launch_wilson(ov_ctx* ctx, const double2* in, double2* out, const Epilogue& ep) {
    if (ctx->dslash_variant == 2 || (ctx->dslash_variant == 0 && tma_usable(ctx)))
        return launch_wilson_tma(ctx, in, out, ep);
    return launch_wilson_gather(ctx, in, out, ep);
}

Span::Span(ov_ctx* c, int phase) : ctx(c) {
    if (!c->timing) return;
    if (2 * c->ev_used + 2 > c->ev_pool.size()) {
        cudaEvent_t a, b;
        if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return;
        c->ev_pool.push_back(a);
        c->ev_pool.push_back(b);
        c->ev_phase.push_back(0);
        c->ev_launches.push_back(0);
    }
    slot = (int)c->ev_used++;
    c->ev_phase[slot] = phase;
    launches0 = c->launches;
    cudaEventRecord(c->ev_pool[2 * slot], c->stream);
}
Span::~Span() {
    if (slot < 0) return;
    cudaEventRecord(ctx->ev_pool[2 * slot + 1], ctx->stream);
    ctx->ev_launches[slot] = ctx->launches - launches0;
}

static bool overlaps(const ov_ctx* ctx, const void* a, const void* b, int nrhs) {
    const char* pa = (const char*)a;
    const char* pb = (const char*)b;
    const size_t n = spinor_elems(ctx) * sizeof(double2) * (size_t)nrhs;
    return pa < pb + n && pb < pa + n;
}

static int check_apply(ov_ctx* ctx, const void* in, void* out, int nrhs) {
    if (!ctx) return OV_EINVAL;
    if (!in || !out || nrhs < 1) return fail(ctx, OV_EINVAL, "null pointer or nrhs < 1");
    if (overlaps(ctx, in, out, nrhs)) return fail(ctx, OV_EINVAL, "in and out overlap (the operator is a stencil)");
    return OV_OK;
}

}  // namespace ov

using namespace ov;

extern "C" {

int ov_create(ov_ctx** out, const int dims[4], double kappa, const void* gauge_dev, int recon, void* cuda_stream) {
    return ov_create_ex(out, dims, kappa, gauge_dev, recon, cuda_stream, nullptr);
}

int ov_create_ex(ov_ctx** out, const int dims[4], double kappa, const void* gauge_dev, int recon, void* cuda_stream,
                 const ov_options* options) {
    if (!out) return OV_EINVAL;
    ov_options opt{};
    if (options) opt = *options;
    if (opt.layout < 0 || opt.layout > 2 || opt.t_boundary < 0 || opt.t_boundary > 2) return OV_EINVAL;
    if (opt.reserved != 0 || opt.wall_mask < 0 || opt.wall_mask > 7 || opt.field < 0 || opt.field > 3) return OV_EINVAL;
    if (opt.field != 0 && !std::isfinite(opt.field_qE)) return OV_EINVAL;
    *out = nullptr;
    if (!dims || !gauge_dev) return OV_EINVAL;
    if (recon != 18 && recon != 12) return OV_EINVAL;
    for (int d = 0; d < 4; d++)
        if (dims[d] < 2) return OV_EINVAL;
    if (!(kappa > 0.0) || !std::isfinite(kappa)) return OV_EINVAL;  // the kernel forms in/kappa (own term first)
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return OV_ECUDA;  // no CPU fallback
    ov_ctx* ctx = new ov_ctx();
    ctx->lat.X = dims[0]; ctx->lat.Y = dims[1]; ctx->lat.Z = dims[2]; ctx->lat.T = dims[3];
    ctx->lat.V = (long long)dims[0] * dims[1] * dims[2] * dims[3];
    ctx->kappa = kappa;
    ctx->recon = recon;
    if (opt.layout == 1 && ctx->lat.V % 32 != 0) { delete ctx; return OV_EINVAL; }
    ctx->blocked = opt.layout == 1 || (opt.layout == 0 && ctx->lat.V % 32 == 0 && !tma_eligible(ctx->lat));
    ctx->t_phase = opt.t_boundary == OV_BC_PERIODIC ? 1.0 : opt.t_boundary == OV_BC_OPEN ? 0.0 : -1.0;
    ctx->field_dir = opt.field - 1;
    ctx->field_qE = opt.field_qE;
    ctx->field_origin = opt.field_origin;
    ctx->stream = (cudaStream_t)cuda_stream;
    const size_t gbytes = gauge_elems(ctx->lat.V, recon) * sizeof(double2);
    cudaError_t e = cudaMalloc(&ctx->gauge, gbytes);
    if (e != cudaSuccess) { delete ctx; return e == cudaErrorMemoryAllocation ? OV_ENOMEM : OV_ECUDA; }
    // the planes layout was chosen for the TMA-staged kernel: make sure tensor maps can actually be built here, and if
    // not (driver entry point missing, encode refused, OV_NO_TMA) fall back NOW, while the layout can still change, to
    // what a non-eligible lattice gets -- the gather kernel on the blocked layout -- instead of failing at every launch
    if (!ctx->blocked && tma_eligible(ctx->lat) && !tma_probe(ctx)) {
        ctx->tma_ok = false;
        if (opt.layout == 0 && ctx->lat.V % 32 == 0) ctx->blocked = true;
    }
    int rc = OV_OK;
    if (recon == 12) {   // rows 0-1 only make sense if row 2 really is conj(row0 x row1)
        double defect = 0.0;
        rc = gauge_su3_defect(ctx, (const double2*)gauge_dev, &defect);
        if (rc == OV_OK && !(defect <= 1e-9)) rc = OV_EINVAL;
    }
    GaugeMods mods{};
    mods.wall_mask = opt.wall_mask;
    mods.field_dir = opt.field - 1;
    mods.qE = opt.field_qE;
    mods.origin = opt.field_origin;
    if (rc == OV_OK) rc = launch_gauge_relayout(ctx, (const double2*)gauge_dev, &mods);
    if (rc == OV_OK && cudaStreamSynchronize(ctx->stream) != cudaSuccess) rc = OV_ECUDA;
    if (rc == OV_OK) rc = ensure_reduction_buffers(ctx, 1, 1024);
    if (rc != OV_OK) { ov_destroy(ctx); return rc; }
    *out = ctx;
    return OV_OK;
}

void ov_destroy(ov_ctx* ctx) {
    if (!ctx) return;
    cudaStreamSynchronize(ctx->stream);
    cudaFree(ctx->gauge);
    for (auto& w : ctx->ws) cudaFree(w);
    for (auto& w : ctx->wsf) cudaFree(w);
    cudaFree(ctx->gauge_f);
    cudaFree(ctx->wsb);
    cudaFree(ctx->d_partial);
    cudaFree(ctx->d_result);
    if (ctx->h_result) cudaFreeHost(ctx->h_result);
    cudaFree(ctx->d_sgn);
    cudaFree(ctx->d_coef);
    cudaFree(ctx->d_coefb);
    {
        HostPipe& hp = ctx->host_pipe;
        if (hp.h2d) { cudaStreamSynchronize(hp.h2d); cudaStreamDestroy(hp.h2d); }
        if (hp.d2h) { cudaStreamSynchronize(hp.d2h); cudaStreamDestroy(hp.d2h); }
        for (int b = 0; b < 2; b++) {
            cudaFree(hp.cin[b]); cudaFree(hp.cout[b]);
            if (hp.in_ready[b]) cudaEventDestroy(hp.in_ready[b]);
            if (hp.in_free[b]) cudaEventDestroy(hp.in_free[b]);
            if (hp.out_ready[b]) cudaEventDestroy(hp.out_ready[b]);
            if (hp.out_free[b]) cudaEventDestroy(hp.out_free[b]);
        }
        cudaFree(hp.abi_in); cudaFree(hp.abi_out);
        if (hp.start) cudaEventDestroy(hp.start);
    }
    for (auto e : ctx->ev_pool) cudaEventDestroy(e);
    tma_state_free(ctx);
    delete ctx;
}

const char* ov_last_error(const ov_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }
size_t ov_spinor_bytes(const ov_ctx* ctx) { return ctx ? spinor_elems(ctx) * sizeof(double2) : 0; }
long long ov_volume(const ov_ctx* ctx) { return ctx ? ctx->lat.V : 0; }
int ov_spinor_layout(const ov_ctx* ctx) { return ctx && ctx->blocked ? 1 : 0; }
long long ov_launch_count(const ov_ctx* ctx) { return ctx ? ctx->launches : 0; }

int ov_timing_enable(ov_ctx* ctx, int on) {
    if (!ctx) return OV_EINVAL;
    OV_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->timing = on != 0;
    ctx->ev_used = 0;
    return OV_OK;
}

int ov_timing_read(ov_ctx* ctx, double* out_host) {
    if (!ctx) return OV_EINVAL;
    if (!out_host) return fail(ctx, OV_EINVAL, "null pointer");
    OV_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    double ms[2] = {0, 0}, launches[2] = {0, 0};
    for (size_t i = 0; i < ctx->ev_used; i++) {
        float t = 0.f;
        OV_CUDA(ctx, cudaEventElapsedTime(&t, ctx->ev_pool[2 * i], ctx->ev_pool[2 * i + 1]));
        ms[ctx->ev_phase[i]] += t;
        launches[ctx->ev_phase[i]] += (double)ctx->ev_launches[i];
    }
    out_host[0] = ms[0]; out_host[1] = launches[0];
    out_host[2] = ms[1]; out_host[3] = launches[1];
    ctx->ev_used = 0;
    return OV_OK;
}

int ov_set_dslash_variant(ov_ctx* ctx, int variant) {
    if (!ctx) return OV_EINVAL;
    if (variant < 0 || variant > 2) return fail(ctx, OV_EINVAL, "variant must be 0, 1 or 2");
    if (variant == 2 && !tma_usable(ctx))
        return fail(ctx, OV_EINVAL, "the TMA-staged Wilson kernel needs the planes layout and X %% 8 == Y %% 4 == Z %% 4 == 0");
    ctx->dslash_variant = variant;
    return OV_OK;
}

int ov_get_dslash_variant(const ov_ctx* ctx) { return ctx ? effective_variant(ctx) : 0; }

int ov_pack_spinor(ov_ctx* ctx, const void* canonical_dev, void* abi_dev, int nrhs) {
    OV_TRY(check_apply(ctx, canonical_dev, abi_dev, nrhs));
    const size_t n = spinor_elems(ctx);
    for (int r = 0; r < nrhs; r++)
        OV_TRY(launch_pack(ctx, (const double2*)canonical_dev + r * n, (double2*)abi_dev + r * n));
    return OV_OK;
}

int ov_unpack_spinor(ov_ctx* ctx, const void* abi_dev, void* canonical_dev, int nrhs) {
    OV_TRY(check_apply(ctx, abi_dev, canonical_dev, nrhs));
    const size_t n = spinor_elems(ctx);
    for (int r = 0; r < nrhs; r++)
        OV_TRY(launch_unpack(ctx, (const double2*)abi_dev + r * n, (double2*)canonical_dev + r * n));
    return OV_OK;
}

int ov_dslash(ov_ctx* ctx, const void* in, void* out, int nrhs) {
    OV_TRY(check_apply(ctx, in, out, nrhs));
    const size_t n = spinor_elems(ctx);
    Epilogue ep;
    ep.hop_only = 1;
    (void)n;
    return launch_wilson_batch(ctx, (const double2*)in, (double2*)out, ep, nrhs);
}

int ov_apply_hw(ov_ctx* ctx, const void* in, void* out, int nrhs) {
    OV_TRY(check_apply(ctx, in, out, nrhs));
    const size_t n = spinor_elems(ctx);
    Epilogue ep;  // s = 1, gamma5
    (void)n;
    return launch_wilson_batch(ctx, (const double2*)in, (double2*)out, ep, nrhs);
}

}  // extern "C"
