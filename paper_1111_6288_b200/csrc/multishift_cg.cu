// Multi-shift ("multi-mass") CG on A = D_ov(0)^+ D_ov(0) = gamma5 D_ov gamma5 D_ov (
// PAPER.md:85; O8/G10).  One Krylov space serves all shifts sigma_i = m_i^2/(1 - m_i^2/4).
// Host loop, device vectors; two host synchronisations per iteration (the scalars (p,q) and (r,r)),
// negligible next to the ~2(2n+1) Wilson launches inside each A.
//
// Deflation (SURVEY 8f rank 2; PAPER.md:45 "we use deflation to help speed up the calculation", :81): with orthonormal
// eigenpairs (mu_j, w_j) of A handed over by ov_set_deflation,
//     x_i = sum_j w_j (w_j^+ b) / (mu_j + sigma_i)  +  CG solution for the projected source b - W W^+ b,
// the CG stopping at |r| <= tol |b| (the full source).  The w_j must be eigenvectors of the A this routine applies to
// within tol (include/ov.h): the true residuals returned at the end are computed with the full b and x_i and show it.
#include <algorithm>
#include <cmath>
#include <numeric>

#include "ov_internal.h"

namespace ov {

// out = A in  (tmp: one scratch spinor, none of the three may alias)
static int apply_A(ov_ctx* ctx, const double2* in, double2* tmp, double2* out) {
    OV_TRY(apply_dov(ctx, 0.0, in, tmp));
    OV_TRY(launch_gamma5(ctx, tmp, tmp));
    OV_TRY(apply_dov(ctx, 0.0, tmp, out));
    return launch_gamma5(ctx, out, out);
}

// same at reduced accuracy (adaptive CG): series truncated to `order`, Clenshaw sweeps in fp32 if f32
static int apply_A_reduced(ov_ctx* ctx, const double2* in, double2* tmp, double2* out, int order, bool f32) {
    if (order >= ctx->order && !f32) return apply_A(ctx, in, tmp, out);
    OV_TRY(apply_dov_reduced(ctx, 0.0, in, tmp, order, f32));
    OV_TRY(launch_gamma5(ctx, tmp, tmp));
    OV_TRY(apply_dov_reduced(ctx, 0.0, tmp, out, order, f32));
    return launch_gamma5(ctx, out, out);
}

// Chirally symmetric form (ov_set_cg_operator(1); reading G22): out = A' in = 2 in + gamma5 S in + S gamma5 in.
// A' = gamma5 D gamma5 D + (1 - S^2): the same operator up to the polynomial's error delta, but it commutes with gamma5
// exactly, so (a) the per-sector eigenvectors of ov_lanczos_dov_lowmodes are its exact eigenvectors whatever delta is and
// (b) on a vector of definite chirality s it is 2 in + (s + gamma5) S in: ONE sign instead of two.  chir = the chirality of
// `in` (+-1; the whole Krylov space of a chiral source has it) or 0.  tmp, tmp2: scratch.
static int apply_A_sym(ov_ctx* ctx, const double2* in, double2* tmp, double2* tmp2, double2* out, int chir) {
    OV_TRY(apply_sign(ctx, in, tmp));
    if (chir != 0) return launch_chiral_combine(ctx, 2.0, in, chir, tmp, out);
    OV_TRY(launch_gamma5(ctx, tmp, tmp));
    OV_TRY(launch_axpby(ctx, 2.0, in, 1.0, tmp, out));              // out = 2 in + gamma5 S in
    OV_TRY(launch_gamma5(ctx, in, tmp));
    OV_TRY(apply_sign(ctx, tmp, tmp2));
    return launch_axpy(ctx, make_double2(1.0, 0.0), tmp2, out);     // + S gamma5 in
}

// +1 / -1 if the other chirality half of v is exactly zero, else 0 (tmp: scratch)
static int chirality_of(ov_ctx* ctx, const double2* v, double2* tmp, int* chir) {
    double n[2];
    for (int i = 0; i < 2; i++) {
        OV_TRY(launch_chiral_combine(ctx, 0.0, nullptr, i == 0 ? +1 : -1, v, tmp));   // 2 P_s v
        OV_TRY(norm2_host(ctx, tmp, &n[i]));
    }
    *chir = (n[1] == 0.0 && n[0] > 0.0) ? +1 : (n[0] == 0.0 && n[1] > 0.0) ? -1 : 0;
    return OV_OK;
}

// d[n'] = max over x in [x_lo, 1] of sqrt(x) |P_n(x) - P_n'(x)|: how far the series truncated at n' is from the full
// polynomial, as an operator on the part of the spectrum the polynomial acts on (host, a few hundred grid points)
static std::vector<double> truncation_table(const std::vector<double>& c, double eps, double x_lo) {
    const int n = (int)c.size() - 1, G = 600;
    std::vector<double> d(n + 1, 0.0);
    for (int g = 0; g < G; g++) {
        const double u = (double)g / (G - 1);
        const double x = (g % 2) ? x_lo * std::pow(1.0 / x_lo, u) : x_lo + (1.0 - x_lo) * u;   // log and linear grids
        const double z = (2.0 * x - 1.0 - eps) / (1.0 - eps), sx = std::sqrt(x);
        std::vector<double> T(n + 1);
        T[0] = 1.0;
        if (n >= 1) T[1] = z;
        for (int j = 2; j <= n; j++) T[j] = 2.0 * z * T[j - 1] - T[j - 2];
        double tail = 0.0;
        for (int j = n; j >= 1; j--) {
            tail += c[j] * T[j];
            d[j - 1] = std::max(d[j - 1], sx * std::fabs(tail));
        }
    }
    return d;
}

}  // namespace ov

using namespace ov;

extern "C" int ov_set_cg_operator(ov_ctx* ctx, int mode) {
    if (!ctx) return OV_EINVAL;
    if (mode != 0 && mode != 1) return fail(ctx, OV_EINVAL, "cg operator mode must be 0 or 1");
    ctx->cg_operator = mode;
    return OV_OK;
}
extern "C" int ov_cg_chirality(const ov_ctx* ctx) { return ctx ? ctx->cg_chirality : 0; }

extern "C" int ov_set_deflation(ov_ctx* ctx, const void* W_dev, const double* mu_host, int k) {
    if (!ctx) return OV_EINVAL;
    if (k < 0 || k > 1024 || (k > 0 && (!W_dev || !mu_host))) return fail(ctx, OV_EINVAL, "bad argument to ov_set_deflation");
    for (int i = 0; i < k; i++)
        if (!(mu_host[i] > -1e-6) || !std::isfinite(mu_host[i]))
            return fail(ctx, OV_EINVAL, "deflation eigenvalue %d = %g: A = D^+ D is positive semi-definite", i, mu_host[i]);
    ctx->Wdefl = k > 0 ? (const double2*)W_dev : nullptr;
    ctx->mu_defl.assign(mu_host, mu_host + k);
    return OV_OK;
}

extern "C" int ov_multishift_cg(ov_ctx* ctx, const double* masses_host, int nmass, const void* b_, void* x_,
                                double tol, int maxiter, int* iters_out, double* relres_out) {
    if (!ctx) return OV_EINVAL;
    if (!masses_host || nmass < 1 || nmass > 64 || !b_ || !x_ || !(tol > 0) || maxiter < 1)
        return fail(ctx, OV_EINVAL, "bad argument to ov_multishift_cg");
    if (ctx->order < 0) return fail(ctx, OV_ESTATE, "ov_set_polynomial has not been called");
    if (ctx->cg_operator == 1 && ctx->cg_adaptive)
        return fail(ctx, OV_ESTATE, "the adaptive modes apply to the gamma5 D gamma5 D form only (ov_set_cg_operator(0))");
    if (!ctx->mu_defl.empty() && ctx->cg_adaptive)
        return fail(ctx, OV_ESTATE, "deflation (ov_set_deflation) and the adaptive modes (ov_set_cg_adaptive) cannot be combined: "
                                    "an inexact operator re-populates the deflated directions");
    const size_t n = spinor_elems(ctx), bytes = n * sizeof(double2);
    ctx->cg_orders.clear();
    const double2* b = (const double2*)b_;
    double2* x = (double2*)x_;

    std::vector<double> sig(nmass);
    for (int i = 0; i < nmass; i++) {
        const double m = masses_host[i];
        if (!(m * m < 4.0)) return fail(ctx, OV_EINVAL, "mass %d out of range", i);
        sig[i] = m * m / (1.0 - 0.25 * m * m);
    }
    // the deflated part of x_i divides by mu_j + sigma_i: a zero mode (or rounding noise below zero, which ov_set_deflation
    // lets through) with mass 0 would make the system singular
    for (size_t j = 0; j < ctx->mu_defl.size(); j++)
        for (int i = 0; i < nmass; i++)
            if (!(ctx->mu_defl[j] + sig[i] > 0.0))
                return fail(ctx, OV_EINVAL, "deflation mode %zu (mu = %g) with mass %d (sigma = %g): mu + sigma <= 0, the shifted system is singular",
                            j, ctx->mu_defl[j], i, sig[i]);
    std::vector<int> ord(nmass);
    std::iota(ord.begin(), ord.end(), 0);
    std::sort(ord.begin(), ord.end(), [&](int a, int c) { return sig[a] < sig[c]; });
    const double s0 = sig[ord[0]];

    // device vectors: p_i (nmass), r, q, tmp, tmp2
    double2* pool = nullptr;
    OV_CUDA(ctx, cudaMalloc(&pool, bytes * (size_t)(nmass + 4)));
    struct Free { double2* p; ~Free() { cudaFree(p); } } guard{pool};
    std::vector<double2*> p(nmass);
    for (int i = 0; i < nmass; i++) p[i] = pool + (size_t)i * n;
    double2* r = pool + (size_t)nmass * n;
    double2* q = r + n;
    double2* tmp = q + n;
    double2* tmp2 = tmp + n;
    const bool sym = ctx->cg_operator == 1;
    int chir = 0;   // symmetric form: chirality of the source (and then of every CG vector), 0 = none
    auto apply_op = [&](const double2* in, double2* out) -> int {   // the full-accuracy operator of this solve
        return sym ? apply_A_sym(ctx, in, tmp, tmp2, out, chir) : apply_A(ctx, in, tmp, out);
    };

    double rr;
    OV_TRY(norm2_host(ctx, b, &rr));
    const double bnorm = std::sqrt(rr);   // every tolerance below is relative to the FULL source
    if (bnorm == 0.0) {
        for (int i = 0; i < nmass; i++) OV_TRY(launch_zero(ctx, x + (size_t)i * n));
        if (iters_out) *iters_out = 0;
        if (relres_out) for (int i = 0; i < nmass; i++) relres_out[i] = 0.0;
        return OV_OK;
    }
    // deflation: r = b - W (W^+ b); the deflated part of every solution is added at the end
    const int kd = (int)ctx->mu_defl.size();
    std::vector<double2> cdefl(kd);
    double2* d_cd = nullptr;
    struct FreeC { double2*& p; ~FreeC() { cudaFree(p); } } guard_c{d_cd};
    if (kd > 0) {
        OV_CUDA(ctx, cudaMalloc(&d_cd, (size_t)kd * sizeof(double2)));
        OV_TRY(launch_multi_dot(ctx, ctx->Wdefl, n, kd, b));
        OV_TRY(fetch_results(ctx, kd, cdefl.data()));
        std::vector<double2> neg(kd);
        for (int j = 0; j < kd; j++) neg[j] = make_double2(-cdefl[j].x, -cdefl[j].y);
        OV_CUDA(ctx, cudaMemcpyAsync(d_cd, neg.data(), kd * sizeof(double2), cudaMemcpyHostToDevice, ctx->stream));
        OV_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        MultiAxpyOuts o;
        o.out[0] = r; o.bscale[0] = 1.0;
        OV_TRY(launch_multi_axpy(ctx, ctx->Wdefl, n, kd, 1, d_cd, b, o));
        OV_TRY(norm2_host(ctx, r, &rr));
    } else {
        OV_TRY(launch_copy(ctx, b, r));
    }
    for (int i = 0; i < nmass; i++) {
        OV_TRY(launch_zero(ctx, x + (size_t)i * n));
        OV_TRY(launch_copy(ctx, r, p[i]));
    }
    if (sym) OV_TRY(chirality_of(ctx, r, tmp, &chir));
    ctx->cg_chirality = chir;
    // adaptive accuracy (ov_set_cg_adaptive): the application of A at iteration j may be off by eta_j ~ tol |b| / |r_j|
    std::vector<double> trunc;
    if (ctx->cg_adaptive) {
        double x_lo = ctx->eps;
        // The polynomial only has to be accurate on the spectrum the small space does not cover.  Precondition (include/ov.h,
        // ov_set_cg_adaptive): the caller's small space is COMPLETE below max|lambda_i|, i.e. it holds every mode of Q with
        // |lambda| < max|lambda_i| (what ov_lanczos_lowmodes returns); then x_lo can move up to ~lambda_k^2.
        if (ctx->k > 0) {
            double lmax = 0.0;
            for (double l : ctx->lambda) lmax = std::max(lmax, std::fabs(l));
            x_lo = std::max(ctx->eps, 0.96 * lmax * lmax);
        }
        trunc = truncation_table(ctx->coef, ctx->eps, x_lo);
    }
    // relative error of an fp32 Clenshaw sweep: unit roundoff 6e-8 amplified by sum |c_j| (measured at 24^3x64, order
    // 300, sum |c_j| ~ 100: 1.5e-6)
    double csum = 0.0;
    for (double cj : ctx->coef) csum += std::fabs(cj);
    const double f32_floor = 6e-8 * csum;
    std::vector<double> zeta(nmass, 1.0), zeta_old(nmass, 1.0), zeta_new(nmass);
    std::vector<char> active(nmass, 1);
    double a_old = 1.0, beta_old = 0.0;
    int it = 0;
    bool converged = std::sqrt(rr) <= tol * bnorm;   // e.g. a source inside the deflation space
    while (!converged && it < maxiter) {
        // q = (A + s0) p_0   (position 0 = smallest shift)
        int order = ctx->order;
        bool f32 = false;
        if (ctx->cg_adaptive) {
            const double eta = std::min(0.1, 0.1 * tol * bnorm / std::sqrt(rr));   // allowed relative error of A p
            while (order > 1 && 4.0 * trunc[order - 1] <= eta) order--;
            f32 = ctx->cg_adaptive >= 2 && 4.0 * f32_floor <= eta;
        }
        if (sym) OV_TRY(apply_op(p[0], q));
        else OV_TRY(apply_A_reduced(ctx, p[0], tmp, q, order, f32));
        if (ctx->cg_adaptive) { ctx->cg_orders.push_back(f32 ? -order : order); }
        if (s0 != 0.0) OV_TRY(launch_axpy(ctx, make_double2(s0, 0.0), p[0], q));
        double2 pq;
        OV_TRY(dot_host(ctx, p[0], q, &pq));
        // breakdown guard: (p, (A + s0) p) must be positive and finite for a positive definite A; an inexact (reduced
        // order / fp32) operator or NaN input would otherwise poison every shift silently
        if (!(pq.x > 0.0) || !std::isfinite(pq.x) || !std::isfinite(rr))
            return fail(ctx, OV_ENOCONV, "multi-shift CG breakdown at iteration %d: (p, A p) = %g, |r|^2 = %g", it, pq.x, rr);
        const double a = rr / pq.x;
        for (int j = 0; j < nmass; j++) {
            const double s = sig[ord[j]] - s0;
            zeta_new[j] = zeta[j] * zeta_old[j] * a_old /
                          (a * beta_old * (zeta_old[j] - zeta[j]) + zeta_old[j] * a_old * (1.0 + s * a));
        }
        for (int j = 0; j < nmass; j++)
            if (active[j])
                OV_TRY(launch_axpy(ctx, make_double2(a * zeta_new[j] / zeta[j], 0.0), p[j], x + (size_t)ord[j] * n));
        OV_TRY(launch_axpy(ctx, make_double2(-a, 0.0), q, r));
        double rr_new;
        OV_TRY(norm2_host(ctx, r, &rr_new));
        const double beta = rr_new / rr;
        for (int j = 0; j < nmass; j++)
            if (active[j]) {
                const double ratio = zeta_new[j] / zeta[j];
                OV_TRY(launch_axpby(ctx, zeta_new[j], r, beta * ratio * ratio, p[j], p[j]));
            }
        zeta_old = zeta;
        zeta = zeta_new;
        a_old = a;
        beta_old = beta;
        rr = rr_new;
        it++;
        for (int j = 1; j < nmass; j++)
            if (active[j] && std::fabs(zeta[j]) * std::sqrt(rr) <= tol * bnorm) active[j] = 0;
        if (std::sqrt(rr) <= tol * bnorm) { converged = true; break; }
    }
    if (iters_out) *iters_out = it;
    if (kd > 0) {   // x_i += W (c / (mu + sigma_i))
        std::vector<double2> coef(kd);
        for (int i = 0; i < nmass; i++) {
            for (int j = 0; j < kd; j++) {
                const double d = 1.0 / (ctx->mu_defl[j] + sig[i]);
                coef[j] = make_double2(cdefl[j].x * d, cdefl[j].y * d);
            }
            OV_CUDA(ctx, cudaMemcpyAsync(d_cd, coef.data(), kd * sizeof(double2), cudaMemcpyHostToDevice, ctx->stream));
            OV_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
            MultiAxpyOuts o;
            o.out[0] = x + (size_t)i * n; o.bscale[0] = 1.0;
            OV_TRY(launch_multi_axpy(ctx, ctx->Wdefl, n, kd, 1, d_cd, x + (size_t)i * n, o));
        }
    }
    if (relres_out) {  // true residuals |b - (A + sigma_i) x_i| / |b|
        for (int i = 0; i < nmass; i++) {
            OV_TRY(apply_op(x + (size_t)i * n, q));
            OV_TRY(launch_axpy(ctx, make_double2(sig[i], 0.0), x + (size_t)i * n, q));
            OV_TRY(launch_axpby(ctx, 1.0, b, -1.0, q, q));
            double e;
            OV_TRY(norm2_host(ctx, q, &e));
            relres_out[i] = std::sqrt(e) / bnorm;
        }
    }
    OV_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (!converged) return fail(ctx, OV_ENOCONV, "multi-shift CG: %d iterations without reaching tol", it);
    return OV_OK;
}
