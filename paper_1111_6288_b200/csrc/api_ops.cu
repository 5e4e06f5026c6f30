// C ABI entry points, part 2: polynomial, small space, sign / D_ov, host-buffer variants, BLAS hooks.
#include <cmath>
#include <cstring>

#include "ov_internal.h"

using namespace ov;

static bool overlaps2(const ov_ctx* ctx, const void* a, const void* b, int nrhs) {
    const char* pa = (const char*)a;
    const char* pb = (const char*)b;
    const size_t n = spinor_elems(ctx) * sizeof(double2) * (size_t)nrhs;
    return pa < pb + n && pb < pa + n;
}
static int check2(ov_ctx* ctx, const void* in, void* out, int nrhs) {
    if (!ctx) return OV_EINVAL;
    if (!in || !out || nrhs < 1) return fail(ctx, OV_EINVAL, "null pointer or nrhs < 1");
    if (overlaps2(ctx, in, out, nrhs)) return fail(ctx, OV_EINVAL, "in and out overlap (the operator is a stencil)");
    return OV_OK;
}

extern "C" {

// Chebyshev interpolation of x^(-1/2) on [eps,1] at the order+1 first-kind nodes (O5, reading G4/G5).
int ov_chebyshev_coeffs(int order, double eps, double* coeffs_host) {
    if (order < 0 || !(eps > 0.0) || !(eps < 1.0) || !coeffs_host) return OV_EINVAL;
    const int m = order + 1;
    const long double pi = 3.141592653589793238462643383279502884L;
    std::vector<long double> f(m), th(m);
    for (int k = 0; k < m; k++) {
        th[k] = pi * (k + 0.5L) / m;
        const long double x = 0.5L * ((1.0L - eps) * cosl(th[k]) + 1.0L + eps);
        f[k] = 1.0L / sqrtl(x);
    }
    for (int j = 0; j < m; j++) {
        long double s = 0.0L;
        for (int k = 0; k < m; k++) s += f[k] * cosl(j * th[k]);
        s *= 2.0L / m;
        if (j == 0) s *= 0.5L;
        coeffs_host[j] = (double)s;
    }
    return OV_OK;
}

// the deflation space holds eigenpairs of D_ov^+ D_ov for the sign function in force when they were computed: a new
// polynomial or small space changes that operator, so the (borrowed) space is dropped rather than left to go stale
static void drop_deflation(ov_ctx* ctx) {
    ctx->Wdefl = nullptr;
    ctx->mu_defl.clear();
}

int ov_set_polynomial(ov_ctx* ctx, const double* coeffs_host, int order, double eps, double norm) {
    if (!ctx) return OV_EINVAL;
    if (!coeffs_host || order < 0) return fail(ctx, OV_EINVAL, "null coefficients or negative order");
    if (!(eps > 0.0) || !(eps < 1.0)) return fail(ctx, OV_EINVAL, "eps must lie in (0,1)");
    if (!(norm > 0.0)) return fail(ctx, OV_EINVAL, "norm must be positive");
    for (int j = 0; j <= order; j++)
        if (!std::isfinite(coeffs_host[j])) return fail(ctx, OV_EINVAL, "coefficient %d is not finite", j);
    drop_deflation(ctx);
    ctx->coef.assign(coeffs_host, coeffs_host + order + 1);
    ctx->order = order;
    ctx->eps = eps;
    ctx->norm = norm;
    return OV_OK;
}

int ov_set_smallspace(ov_ctx* ctx, const void* V_dev, const double* lambda_host, int k) {
    if (!ctx) return OV_EINVAL;
    if (k < 0) return fail(ctx, OV_EINVAL, "k < 0");
    if (k == 0) { ctx->k = 0; ctx->Vlow = nullptr; ctx->lambda.clear(); drop_deflation(ctx); return OV_OK; }
    if (!V_dev || !lambda_host) return fail(ctx, OV_EINVAL, "null V or lambda with k > 0");
    if ((size_t)k * 2 * sizeof(double2) > 200 * 1024) return fail(ctx, OV_EINVAL, "k too large (max 6400)");
    std::vector<double> sgn(k);
    for (int i = 0; i < k; i++) {
        if (lambda_host[i] == 0.0 || !std::isfinite(lambda_host[i]))
            return fail(ctx, OV_EINVAL, "lambda[%d] is zero or not finite: sign undefined (reading G8)", i);
        sgn[i] = lambda_host[i] > 0 ? 1.0 : -1.0;
    }
    if (k > ctx->cap_k) {
        OV_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->d_sgn); cudaFree(ctx->d_coef);
        ctx->d_sgn = nullptr; ctx->d_coef = nullptr; ctx->cap_k = 0;
        OV_CUDA(ctx, cudaMalloc(&ctx->d_sgn, (size_t)k * sizeof(double)));
        OV_CUDA(ctx, cudaMalloc(&ctx->d_coef, (size_t)k * 2 * sizeof(double2)));
        ctx->cap_k = k;
    }
    OV_CUDA(ctx, cudaMemcpyAsync(ctx->d_sgn, sgn.data(), (size_t)k * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    OV_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->Vlow = (const double2*)V_dev;
    ctx->lambda.assign(lambda_host, lambda_host + k);
    ctx->k = k;
    drop_deflation(ctx);
    return OV_OK;
}

int ov_project(ov_ctx* ctx, const void* in, void* perp, void* low, double* coef_host) {
    if (!ctx) return OV_EINVAL;
    if (!in || !perp || !low) return fail(ctx, OV_EINVAL, "null pointer");
    if (ctx->k <= 0) return fail(ctx, OV_ESTATE, "no small space set");
    OV_TRY(project(ctx, (const double2*)in, (double2*)perp, (double2*)low));
    if (coef_host) {
        std::vector<double2> c(ctx->k);
        OV_TRY(fetch_results(ctx, ctx->k, c.data()));
        for (int i = 0; i < ctx->k; i++) { coef_host[2 * i] = c[i].x; coef_host[2 * i + 1] = c[i].y; }
    }
    return OV_OK;
}

int ov_apply_sign(ov_ctx* ctx, const void* in, void* out, int nrhs) {
    OV_TRY(check2(ctx, in, out, nrhs));
    const size_t n = spinor_elems(ctx);
    int r = 0;
    for (; nrhs - r >= 2; ) {   // batches of up to kBatch right-hand sides share every Wilson launch
        const int nb = nrhs - r >= kBatch ? kBatch : nrhs - r;
        OV_TRY(apply_batch(ctx, true, 0.0, (const double2*)in + r * n, (double2*)out + r * n, nb));
        r += nb;
    }
    for (; r < nrhs; r++) OV_TRY(apply_sign(ctx, (const double2*)in + r * n, (double2*)out + r * n));
    return OV_OK;
}

int ov_apply_dov(ov_ctx* ctx, double mass, const void* in, void* out, int nrhs) {
    OV_TRY(check2(ctx, in, out, nrhs));
    const size_t n = spinor_elems(ctx);
    int r = 0;
    for (; nrhs - r >= 2; ) {
        const int nb = nrhs - r >= kBatch ? kBatch : nrhs - r;
        OV_TRY(apply_batch(ctx, false, mass, (const double2*)in + r * n, (double2*)out + r * n, nb));
        r += nb;
    }
    for (; r < nrhs; r++) OV_TRY(apply_dov(ctx, mass, (const double2*)in + r * n, (double2*)out + r * n));
    return OV_OK;
}

int ov_apply_dov_reduced(ov_ctx* ctx, double mass, const void* in, void* out, int order, int use_f32) {
    OV_TRY(check2(ctx, in, out, 1));
    return apply_dov_reduced(ctx, mass, (const double2*)in, (double2*)out, order, use_f32 != 0);
}

// test/bench hook for the fp32 instantiation of the Wilson kernel (the adaptive CG's single-precision sweeps):
// in -> fp32, H_w with the fp32 copy of the links, result widened back to fp64.
int ov_apply_hw_f32(ov_ctx* ctx, const void* in, void* out) {
    OV_TRY(check2(ctx, in, out, 1));
    OV_TRY(ensure_gauge_f32(ctx));
    float2 *xf, *yf;
    OV_TRY(workspace_f32(ctx, 0, &xf));
    OV_TRY(workspace_f32(ctx, 1, &yf));
    OV_TRY(launch_scale_to_f32(ctx, 1.0, (const double2*)in, xf));
    EpilogueF ep;  // s = 1, gamma5
    OV_TRY(launch_wilson_gather_f32(ctx, xf, yf, ep));
    return launch_combine_from_f32(ctx, yf, 0.0, nullptr, 0.0, nullptr, 0, (double2*)out);
}

int ov_set_cg_adaptive(ov_ctx* ctx, int mode) {
    if (!ctx) return OV_EINVAL;
    if (mode < 0 || mode > 2) return fail(ctx, OV_EINVAL, "mode must be 0, 1 or 2");
    ctx->cg_adaptive = mode;
    return OV_OK;
}

int ov_cg_orders(const ov_ctx* ctx, int* out_host, int cap) {
    if (!ctx) return 0;
    const int n = (int)ctx->cg_orders.size();
    for (int i = 0; i < n && i < cap && out_host; i++) out_host[i] = ctx->cg_orders[i];
    return n;
}

// host-buffer path: H2D -> pack -> operator -> unpack -> D2H.  With nrhs > 1 the copies run on two copy streams (one per
// direction, double-buffered canonical staging): the H2D of right-hand side r+1 and the D2H of r-1 overlap the operator on r,
// so only the first H2D and the last D2H are exposed.  Host buffers should be pinned for the copies to be asynchronous.
// Staging of the host-buffer path.  Every member is created only if it is still null, so a call that failed half way
// (an allocation that did not fit, say) leaves a state the next call completes instead of overwriting -- nothing leaks,
// and ov_destroy frees whatever exists.  nbuf = 1 (a single right-hand side: nothing to overlap) creates one staging
// buffer and one event set per direction, nbuf = 2 the double-buffered set: 4 resp. 6 spinors of device memory.
static int host_pipe_prepare(ov_ctx* ctx, int nbuf) {
    HostPipe& hp = ctx->host_pipe;
    const size_t bytes = spinor_elems(ctx) * sizeof(double2);
    auto buffer = [&](double2** p) -> int {
        if (*p) return OV_OK;
        const cudaError_t e = cudaMalloc(p, bytes);
        if (e != cudaSuccess) { *p = nullptr; cudaGetLastError(); return cuda_fail(ctx, e, "cudaMalloc (host-path staging)"); }
        return OV_OK;
    };
    auto event = [&](cudaEvent_t* ev) -> int {
        if (*ev) return OV_OK;
        const cudaError_t e = cudaEventCreateWithFlags(ev, cudaEventDisableTiming);
        if (e != cudaSuccess) { *ev = nullptr; return cuda_fail(ctx, e, "cudaEventCreateWithFlags (host path)"); }
        return OV_OK;
    };
    auto stream = [&](cudaStream_t* st) -> int {
        if (*st) return OV_OK;
        const cudaError_t e = cudaStreamCreateWithFlags(st, cudaStreamNonBlocking);
        if (e != cudaSuccess) { *st = nullptr; return cuda_fail(ctx, e, "cudaStreamCreateWithFlags (host path)"); }
        return OV_OK;
    };
    for (int b = 0; b < nbuf; b++) {
        OV_TRY(buffer(&hp.cin[b]));
        OV_TRY(buffer(&hp.cout[b]));
        OV_TRY(event(&hp.in_ready[b]));
        OV_TRY(event(&hp.in_free[b]));
        OV_TRY(event(&hp.out_ready[b]));
        OV_TRY(event(&hp.out_free[b]));
    }
    OV_TRY(buffer(&hp.abi_in));
    OV_TRY(buffer(&hp.abi_out));
    OV_TRY(stream(&hp.h2d));
    OV_TRY(stream(&hp.d2h));
    OV_TRY(event(&hp.start));
    return OV_OK;
}

static int host_apply(ov_ctx* ctx, int which, double mass, const void* in_host, void* out_host, int nrhs) {
    if (!ctx) return OV_EINVAL;
    if (!in_host || !out_host || nrhs < 1) return fail(ctx, OV_EINVAL, "null pointer or nrhs < 1");
    const size_t n = spinor_elems(ctx), bytes = n * sizeof(double2);
    HostPipe& hp = ctx->host_pipe;
    OV_TRY(host_pipe_prepare(ctx, nrhs > 1 ? 2 : 1));
    // the copy streams start after everything the caller enqueued on the context's stream so far
    OV_CUDA(ctx, cudaEventRecord(hp.start, ctx->stream));
    OV_CUDA(ctx, cudaStreamWaitEvent(hp.h2d, hp.start, 0));
    OV_CUDA(ctx, cudaStreamWaitEvent(hp.d2h, hp.start, 0));
    for (int r = 0; r < nrhs; r++) {
        const int b = r & 1;
        if (r >= 2) OV_CUDA(ctx, cudaStreamWaitEvent(hp.h2d, hp.in_free[b], 0));       // pack of r-2 has consumed cin[b]
        OV_CUDA(ctx, cudaMemcpyAsync(hp.cin[b], (const char*)in_host + r * bytes, bytes, cudaMemcpyHostToDevice, hp.h2d));
        OV_CUDA(ctx, cudaEventRecord(hp.in_ready[b], hp.h2d));
        OV_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, hp.in_ready[b], 0));
        OV_TRY(launch_pack(ctx, hp.cin[b], hp.abi_in));
        OV_CUDA(ctx, cudaEventRecord(hp.in_free[b], ctx->stream));
        if (which == 0) {
            Epilogue ep;
            OV_TRY(launch_wilson(ctx, hp.abi_in, hp.abi_out, ep));
        } else {
            OV_TRY(apply_dov(ctx, mass, hp.abi_in, hp.abi_out));
        }
        if (r >= 2) OV_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, hp.out_free[b], 0)); // D2H of r-2 has drained cout[b]
        OV_TRY(launch_unpack(ctx, hp.abi_out, hp.cout[b]));
        OV_CUDA(ctx, cudaEventRecord(hp.out_ready[b], ctx->stream));
        OV_CUDA(ctx, cudaStreamWaitEvent(hp.d2h, hp.out_ready[b], 0));
        OV_CUDA(ctx, cudaMemcpyAsync((char*)out_host + r * bytes, hp.cout[b], bytes, cudaMemcpyDeviceToHost, hp.d2h));
        OV_CUDA(ctx, cudaEventRecord(hp.out_free[b], hp.d2h));
    }
    OV_CUDA(ctx, cudaStreamSynchronize(hp.d2h));
    OV_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return OV_OK;
}

int ov_apply_hw_host(ov_ctx* ctx, const void* in_host, void* out_host, int nrhs) {
    return host_apply(ctx, 0, 0.0, in_host, out_host, nrhs);
}
int ov_apply_dov_host(ov_ctx* ctx, double mass, const void* in_host, void* out_host, int nrhs) {
    return host_apply(ctx, 1, mass, in_host, out_host, nrhs);
}

int ov_blas_axpy(ov_ctx* ctx, double a_re, double a_im, const void* x, void* y) {
    if (!ctx) return OV_EINVAL;
    if (!x || !y) return fail(ctx, OV_EINVAL, "null pointer");
    return launch_axpy(ctx, make_double2(a_re, a_im), (const double2*)x, (double2*)y);
}
int ov_blas_scale(ov_ctx* ctx, double a, void* x) {
    if (!ctx) return OV_EINVAL;
    if (!x) return fail(ctx, OV_EINVAL, "null pointer");
    return launch_scale(ctx, a, (double2*)x);
}
int ov_blas_dot(ov_ctx* ctx, const void* x, const void* y, double* out_host) {
    if (!ctx) return OV_EINVAL;
    if (!x || !y || !out_host) return fail(ctx, OV_EINVAL, "null pointer");
    double2 r;
    OV_TRY(dot_host(ctx, (const double2*)x, (const double2*)y, &r));
    out_host[0] = r.x; out_host[1] = r.y;
    return OV_OK;
}
int ov_blas_norm2(ov_ctx* ctx, const void* x, double* out_host) {
    if (!ctx) return OV_EINVAL;
    if (!x || !out_host) return fail(ctx, OV_EINVAL, "null pointer");
    return norm2_host(ctx, (const double2*)x, out_host);
}

}  // extern "C"
