// sign(H_w) and D_ov drivers.
//
//   sign(H_w) x  =  sum_i sign(lambda_i) v_i (v_i^+ x)   +   Q P(Q^2) (1 - V V^+) x
//   P(Q^2) = sum_j c_j T_j(z),  z = (2Q^2 - 1 - eps)/(1 - eps), evaluated by the Clenshaw recurrence with
//   alpha = 4/(1-eps), beta = 2(1+eps)/(1-eps):   b_j = c_j x + alpha Q(Q b_{j+1}) - beta b_{j+1} - b_{j+2}
//   Every Clenshaw order is exactly two launches of the Wilson kernel: the first with epilogue
//   gamma5 * (1/norm), the second with gamma5 * (alpha/norm) plus the three-vector axpy written in place
//   over b_{j+2} -- no separate BLAS-1 pass touches HBM inside the recurrence.
#include "ov_internal.h"

namespace ov {

// C[i*2+0] = -c_i ; C[i*2+1] = sgn_i * c_i     (c = V^+ x sits in d_result after the multi-dot)
__global__ void projector_coef_kernel(const double2* __restrict__ c, const double* __restrict__ sgn, int k,
                                      double2* __restrict__ C) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= k) return;
    const double2 v = c[i];
    const double s = sgn[i];
    C[2 * i + 0] = make_double2(-v.x, -v.y);
    C[2 * i + 1] = make_double2(s * v.x, s * v.y);
}

// c = V^+ x ; perp = x - V c ; low = V (sign(lambda) o c).  Two passes over V ("D_ov requires
// all of the H_w eigenvectors for each matrix multiplication"): 2 k 192 B/site + 4 spinors.
int project(ov_ctx* ctx, const double2* x, double2* perp, double2* low) {
    const size_t stride = spinor_elems(ctx);
    Span span(ctx, 1);
    OV_TRY(launch_multi_dot(ctx, ctx->Vlow, stride, ctx->k, x));
    projector_coef_kernel<<<(ctx->k + 127) / 128, 128, 0, ctx->stream>>>(ctx->d_result, ctx->d_sgn, ctx->k, ctx->d_coef);
    ctx->launches++;
    OV_CUDA(ctx, cudaGetLastError());
    MultiAxpyOuts o;
    o.out[0] = perp; o.bscale[0] = 1.0;
    o.out[1] = low;  o.bscale[1] = 0.0;
    return launch_multi_axpy(ctx, ctx->Vlow, stride, ctx->k, 2, ctx->d_coef, x, o);
}

// C[i*2nb + 2r] = -c_{r,i} ; C[i*2nb + 2r+1] = sgn_i * c_{r,i}   (c_{r,i} = <v_i, x_r> at d_result[r*k + i])
__global__ void projector_coef_batch_kernel(const double2* __restrict__ c, const double* __restrict__ sgn, int k, int nb,
                                            double2* __restrict__ C) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= k * nb) return;
    const int i = q % k, r = q / k;
    const double2 v = c[q];
    const double s = sgn[i];
    C[(size_t)i * 2 * nb + 2 * r + 0] = make_double2(-v.x, -v.y);
    C[(size_t)i * 2 * nb + 2 * r + 1] = make_double2(s * v.x, s * v.y);
}

// Batched projector: for a group of nb = 4 or 2 right-hand sides the eigenvectors
// are streamed once for all V^+ x_r (multi_dot_kernel<nb>) and once for all 2 nb outputs (multi_axpy_kernel<2 nb>), so the
// 2 k 192 B/site of the projector are paid per group, not per right-hand side.
int project_batch(ov_ctx* ctx, const double2* x, double2* perp, double2* low, int nb) {
    const size_t stride = spinor_elems(ctx);
    int r0 = 0;
    while (r0 < nb) {
        // group of 4 or 2 where the batched dot's result block fits in shared memory (k <= 400 / 800), else one at a time
        const int g = (nb - r0 >= 4 && multi_dot_batch_fits(ctx->k, 4)) ? 4
                    : (nb - r0 >= 2 && multi_dot_batch_fits(ctx->k, 2)) ? 2 : 1;
        if (g == 1) {
            OV_TRY(project(ctx, x + r0 * stride, perp + r0 * stride, low + r0 * stride));
        } else {
            Span span(ctx, 1);
            if (ctx->cap_kb < ctx->k * kBatch * 2) {
                if (ctx->d_coefb) cudaFree(ctx->d_coefb);
                ctx->d_coefb = nullptr;
                ctx->cap_kb = 0;
                OV_CUDA(ctx, cudaMalloc(&ctx->d_coefb, (size_t)ctx->k * kBatch * 2 * sizeof(double2)));
                ctx->cap_kb = ctx->k * kBatch * 2;
            }
            OV_TRY(launch_multi_dot_batch(ctx, ctx->Vlow, stride, ctx->k, x + r0 * stride, stride, g));
            projector_coef_batch_kernel<<<(ctx->k * g + 127) / 128, 128, 0, ctx->stream>>>(ctx->d_result, ctx->d_sgn, ctx->k, g, ctx->d_coefb);
            ctx->launches++;
            OV_CUDA(ctx, cudaGetLastError());
            MultiAxpyOuts o;
            for (int r = 0; r < g; r++) {
                o.out[2 * r] = perp + (r0 + r) * stride; o.bscale[2 * r] = 1.0; o.basej[2 * r] = x + (r0 + r) * stride;
                o.out[2 * r + 1] = low + (r0 + r) * stride; o.bscale[2 * r + 1] = 0.0;   // no base: starts from zero
            }
            OV_TRY(launch_multi_axpy(ctx, ctx->Vlow, stride, ctx->k, 2 * g, ctx->d_coefb, nullptr, o));
        }
        r0 += g;
    }
    return OV_OK;
}

// Wilson launch by precision
static int wilson_t(ov_ctx* ctx, const double2* in, double2* out, const Epilogue& ep, int nb) {
    return nb > 1 ? launch_wilson_batch(ctx, in, out, ep, nb) : launch_wilson(ctx, in, out, ep);
}
static int wilson_t(ov_ctx* ctx, const float2* in, float2* out, const EpilogueF& ep, int) { return launch_wilson_gather_f32(ctx, in, out, ep); }

// Clenshaw sweep in precision C over the first n+1 coefficients c[0..n] (a truncation of the caller's series when
// n < ctx->order: the adaptive CG's reduced orders).  b1 must hold c[n]*x on entry; b1, b2, t are scratch.
//   out = (fin.s / norm) * G (y - kappa hop y) + fin.a1 A1 + fin.a2 A2 + fin.a3 A3,   y = P_n(Q^2) x
// with fin.g5 = 1 -> G = gamma5 (plain sign), fin.g5 = 0 -> G = 1 (gamma5 * sign, for D_ov).
template <typename C>
static int clenshaw_t(ov_ctx* ctx, const double* c, int n, const C* x, C* out, const EpilogueT<C>& fin, C* b1, C* b2, C* t,
                      int nb = 1) {
    const double eps = ctx->eps, inv = 1.0 / ctx->norm;
    const double alpha = 4.0 / (1.0 - eps), beta = 2.0 * (1.0 + eps) / (1.0 - eps);
    Span span(ctx, 0);  // every launch in here is the Wilson kernel
    const C* y = b1;
    bool b2_valid = false;
    for (int j = n - 1; j >= 0; j--) {
        EpilogueT<C> e1;  // t = Q b1
        e1.s = inv;
        e1.g5 = 1;
        OV_TRY(wilson_t(ctx, b1, t, e1, nb));
        EpilogueT<C> e2;  // b2 <- f*(alpha Q t - beta b1) + c_j x - b2 ; f = 1 (j >= 1) or 1/2 (j = 0)
        const double f = (j == 0) ? 0.5 : 1.0;
        e2.s = f * alpha * inv;
        e2.g5 = 1;
        e2.A1 = x;  e2.a1 = c[j];
        e2.A2 = b1; e2.a2 = -f * beta;
        if (b2_valid) { e2.A3 = b2; e2.a3 = -1.0; }
        OV_TRY(wilson_t(ctx, t, b2, e2, nb));
        b2_valid = true;
        C* tmp = b1; b1 = b2; b2 = tmp;
        y = b1;  // after the j = 0 step b1 holds y
    }
    EpilogueT<C> ef = fin;
    ef.s = fin.s * inv;
    ef.hop_only = 0;
    return wilson_t(ctx, y, out, ef, nb);
}

int sign_poly(ov_ctx* ctx, const double2* x, double2* out, const Epilogue& fin) {
    if (ctx->order < 0) return fail(ctx, OV_ESTATE, "ov_set_polynomial has not been called");
    const int n = ctx->order;
    double2 *b1, *b2, *t;
    OV_TRY(workspace(ctx, 0, &b1));
    OV_TRY(workspace(ctx, 1, &b2));
    OV_TRY(workspace(ctx, 2, &t));
    OV_TRY(launch_axpby(ctx, ctx->coef[n], x, 0.0, nullptr, b1));   // b_n = c_n x  (b_{n+1} = b_{n+2} = 0)
    return clenshaw_t<double2>(ctx, ctx->coef.data(), n, x, out, fin, b1, b2, t);
}

// nb right-hand sides at once: batched projector, then ONE Clenshaw sweep whose every launch covers the whole batch
// (the links are then read from HBM once per site block and shared through L2/L1 by the right-hand sides).
int apply_batch(ov_ctx* ctx, bool sign_only, double mass, const double2* in, double2* out, int nb) {
    if (ctx->order < 0) return fail(ctx, OV_ESTATE, "ov_set_polynomial has not been called");
    if (nb < 1 || nb > kBatch) return fail(ctx, OV_EINVAL, "batch size out of range");
    const size_t n = spinor_elems(ctx);
    if (!ctx->wsb) OV_CUDA(ctx, cudaMalloc(&ctx->wsb, (size_t)5 * kBatch * n * sizeof(double2)));
    double2 *b1 = ctx->wsb, *b2 = b1 + kBatch * n, *t = b2 + kBatch * n, *perp = t + kBatch * n, *low = perp + kBatch * n;
    const double2* x = in;
    if (ctx->k > 0) {
        OV_TRY(project_batch(ctx, in, perp, low, nb));
        x = perp;
    }
    const int order = ctx->order;
    auto fin_of = [&](int r) {
        Epilogue fin;
        if (sign_only) {
            fin.s = 1.0; fin.g5 = 1;
            if (ctx->k > 0) { fin.A1 = low + r * n; fin.a1 = 1.0; }
        } else {
            fin.s = 1.0 - 0.5 * mass; fin.g5 = 0;
            fin.A1 = in + r * n; fin.a1 = 1.0 + 0.5 * mass;
            if (ctx->k > 0) { fin.A2 = low + r * n; fin.a2 = 1.0 - 0.5 * mass; fin.a_g5 = 2; }
        }
        return fin;
    };
    if (effective_variant(ctx) == 2) {
        // where the TMA-staged kernel runs, one sweep per right-hand side through it (157 us per plain launch) beats the
        // batched gather launch (180 us per right-hand side and launch): only the projector is shared by the batch
        for (int r = 0; r < nb; r++) {
            OV_TRY(launch_axpby(ctx, ctx->coef[order], x + r * n, 0.0, nullptr, b1));
            OV_TRY(clenshaw_t<double2>(ctx, ctx->coef.data(), order, x + r * n, out + r * n, fin_of(r), b1, b2, t));
        }
        return OV_OK;
    }
    OV_TRY(launch_axpby(ctx, ctx->coef[order], x, 0.0, nullptr, b1, nb));
    return clenshaw_t<double2>(ctx, ctx->coef.data(), order, x, out, fin_of(0), b1, b2, t, nb);
}

// D_ov(m) in at reduced accuracy (the adaptive CG): polynomial truncated to order n <= ctx->order and,
// if f32, the Clenshaw sweep in single precision (projector and D_ov assembly stay fp64).
int apply_dov_reduced(ov_ctx* ctx, double mass, const double2* in, double2* out, int n, bool f32) {
    if (ctx->order < 0) return fail(ctx, OV_ESTATE, "ov_set_polynomial has not been called");
    if (n < 0 || n > ctx->order) return fail(ctx, OV_EINVAL, "reduced order out of range");
    const double2* perp = in;
    double2* low = nullptr;
    if (ctx->k > 0) {
        double2* p;
        OV_TRY(workspace(ctx, 3, &p));
        OV_TRY(workspace(ctx, 4, &low));
        OV_TRY(project(ctx, in, p, low));
        perp = p;
    }
    const double sm = 1.0 - 0.5 * mass, sp = 1.0 + 0.5 * mass;
    if (!f32) {
        double2 *b1, *b2, *t;
        OV_TRY(workspace(ctx, 0, &b1));
        OV_TRY(workspace(ctx, 1, &b2));
        OV_TRY(workspace(ctx, 2, &t));
        OV_TRY(launch_axpby(ctx, ctx->coef[n], perp, 0.0, nullptr, b1));
        Epilogue fin;
        fin.s = sm; fin.g5 = 0;
        fin.A1 = in; fin.a1 = sp;
        if (low) { fin.A2 = low; fin.a2 = sm; fin.a_g5 = 2; }
        return clenshaw_t<double2>(ctx, ctx->coef.data(), n, perp, out, fin, b1, b2, t);
    }
    OV_TRY(ensure_gauge_f32(ctx));
    float2 *xf, *b1, *b2, *t;
    OV_TRY(workspace_f32(ctx, 0, &xf));
    OV_TRY(workspace_f32(ctx, 1, &b1));
    OV_TRY(workspace_f32(ctx, 2, &b2));
    OV_TRY(workspace_f32(ctx, 3, &t));
    OV_TRY(launch_scale_to_f32(ctx, 1.0, perp, xf));
    OV_TRY(launch_scale_to_f32(ctx, ctx->coef[n], perp, b1));
    EpilogueF fin;
    fin.s = sm; fin.g5 = 0;
    // the fp32 result r = (1-m/2) D_w y / norm lands in t's partner buffer; b2 or b1 may hold y, so use xf's slot last:
    float2* r = (n % 2 == 0) ? b2 : b1;   // after n swaps y sits in b1 (n even) or b2 (n odd): write to the other one
    OV_TRY(clenshaw_t<float2>(ctx, ctx->coef.data(), n, xf, r, fin, b1, b2, t));
    return launch_combine_from_f32(ctx, r, sp, in, sm, low, 1, out);
}

int apply_sign(ov_ctx* ctx, const double2* in, double2* out) {
    Epilogue fin;
    fin.s = 1.0;
    fin.g5 = 1;
    if (ctx->k > 0) {
        double2 *perp, *low;
        OV_TRY(workspace(ctx, 3, &perp));
        OV_TRY(workspace(ctx, 4, &low));
        OV_TRY(project(ctx, in, perp, low));
        fin.A1 = low; fin.a1 = 1.0;
        return sign_poly(ctx, perp, out, fin);
    }
    return sign_poly(ctx, in, out, fin);
}

// D_ov(m) x = (1 + m/2) x + (1 - m/2) gamma5 sign(H_w) x ; gamma5 * [gamma5 D_w y / norm] = D_w y / norm, so the
// final Wilson launch runs with G = 1 and the x / gamma5 x_low terms ride in its epilogue (row a5).
int apply_dov(ov_ctx* ctx, double mass, const double2* in, double2* out) {
    Epilogue fin;
    fin.s = 1.0 - 0.5 * mass;
    fin.g5 = 0;
    fin.A1 = in; fin.a1 = 1.0 + 0.5 * mass;
    if (ctx->k > 0) {
        double2 *perp, *low;
        OV_TRY(workspace(ctx, 3, &perp));
        OV_TRY(workspace(ctx, 4, &low));
        OV_TRY(project(ctx, in, perp, low));
        fin.A2 = low; fin.a2 = 1.0 - 0.5 * mass; fin.a_g5 = 2;
        return sign_poly(ctx, perp, out, fin);
    }
    return sign_poly(ctx, in, out, fin);
}

}  // namespace ov
