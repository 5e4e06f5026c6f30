// Low modes of Q = H_w/norm (SURVEY 8a row a8; PAPER.md:57 "lowest lying eigenmodes of H_w", :71 "Chebyshev
// acceleration ... polynomial of order 100").  The paper uses implicitly restarted Arnoldi with a 2.5 l
// subspace; H_w is Hermitian, so this is thick-restart Lanczos (the Hermitian form of the same restart)
// on the filtered operator  B = T_d(z(Q^2)),  z(A) = (2A - a - b)/(b - a),  which maps the unwanted part
// [a,b] of the spectrum of Q^2 into [-1,1] and blows the wanted low end up like cosh(d acosh|z|).
// Every filter term is two launches of the Wilson kernel with the three-term axpy in its epilogue, the same
// fused step the Clenshaw recurrence uses.  A final Rayleigh-Ritz in Q itself separates +lambda from -lambda
// and the true residuals |Q v - lambda v| are measured with the kernel (contract: <= tol, G13).
#include <algorithm>
#include <cmath>
#include <numeric>

#include "ov_internal.h"

namespace ov {

__global__ void random_fill_kernel(double2* v, long long n, unsigned long long seed) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    unsigned long long z = seed + 0x9E3779B97F4A7C15ull * (unsigned long long)(e + 1);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    z ^= z >> 31;
    const double a = (double)(z >> 40) / 8388608.0 - 1.0;            // 24 bits -> [-1,1)
    const double b = (double)((z >> 16) & 0xFFFFFF) / 8388608.0 - 1.0;
    v[e] = make_double2(a, b);
}

struct Filter {
    int d;
    double a, b;
};

// out = T_d(z(Q^2)) in ; t1, tq: scratch spinors distinct from in/out.  T_j lives in `out` when j has the parity
// of d and in t1 otherwise; from j = 3 on each T_j is written in place over T_{j-2} (the epilogue reads its
// axpy operands at the output site only).
static int apply_filter(ov_ctx* ctx, const Filter& f, const double2* in, double2* out, double2* /*t0*/, double2* t1,
                        double2* tq) {
    const double inv = 1.0 / ctx->norm, w = f.b - f.a, cs = (f.a + f.b) / w;
    auto buf = [&](int j) { return ((j & 1) == (f.d & 1)) ? out : t1; };
    Epilogue e1; e1.s = inv; e1.g5 = 1;
    OV_TRY(launch_wilson(ctx, in, tq, e1));
    Epilogue e2; e2.s = 2.0 / w * inv; e2.g5 = 1; e2.A1 = in; e2.a1 = -cs;   // T_1 = (2/w) Q Q in - cs in
    OV_TRY(launch_wilson(ctx, tq, buf(1), e2));
    for (int j = 2; j <= f.d; j++) {
        const double2* cur = buf(j - 1);
        const double2* prev = (j == 2) ? in : buf(j - 2);
        OV_TRY(launch_wilson(ctx, cur, tq, e1));
        Epilogue e3; e3.s = 4.0 / w * inv; e3.g5 = 1;                         // T_j = 2 z T_{j-1} - T_{j-2}
        e3.A1 = cur; e3.a1 = -2.0 * cs;
        e3.A2 = prev; e3.a2 = -1.0;
        OV_TRY(launch_wilson(ctx, tq, buf(j), e3));
    }
    return OV_OK;
}

// u -= W[0..nv) (W^+ u), returns the coefficients (host) ; one classical Gram-Schmidt pass
static int cgs_pass(ov_ctx* ctx, const double2* W, size_t stride, int nv, double2* u, double2* d_C,
                    std::vector<double2>& c) {
    OV_TRY(launch_multi_dot(ctx, W, stride, nv, u));
    c.resize(nv);
    OV_TRY(fetch_results(ctx, nv, c.data()));
    std::vector<double2> neg(nv);
    for (int i = 0; i < nv; i++) neg[i] = make_double2(-c[i].x, -c[i].y);
    OV_CUDA(ctx, cudaMemcpyAsync(d_C, neg.data(), nv * sizeof(double2), cudaMemcpyHostToDevice, ctx->stream));
    OV_CUDA(ctx, cudaStreamSynchronize(ctx->stream));  // neg is a stack-owned host buffer
    MultiAxpyOuts o;
    o.out[0] = u; o.bscale[0] = 1.0;
    return launch_multi_axpy(ctx, W, stride, nv, 1, d_C, u, o);
}

// Y[0..ncol) = W[0..m) S[:, cols]  (S row-major m x ldS, host) in blocks of up to 8 columns
static int rotate(ov_ctx* ctx, const double2* W, size_t stride, int m, const std::vector<double2>& S, int ldS,
                  const std::vector<int>& cols, double2* Y, double2* d_C) {
    const int ncol = (int)cols.size();
    int done = 0;
    std::vector<double2> C;
    while (done < ncol) {
        const int rem = ncol - done;
        const int J = rem >= 8 ? 8 : rem >= 4 ? 4 : rem >= 2 ? 2 : 1;
        C.assign((size_t)m * J, make_double2(0, 0));
        for (int i = 0; i < m; i++)
            for (int j = 0; j < J; j++) C[(size_t)i * J + j] = S[(size_t)i * ldS + cols[done + j]];
        OV_CUDA(ctx, cudaMemcpyAsync(d_C, C.data(), C.size() * sizeof(double2), cudaMemcpyHostToDevice, ctx->stream));
        OV_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        MultiAxpyOuts o;
        for (int j = 0; j < J; j++) o.out[j] = Y + (size_t)(done + j) * stride;
        OV_TRY(launch_multi_axpy(ctx, W, stride, m, J, d_C, nullptr, o));
        done += J;
    }
    return OV_OK;
}

static double inverse_filter(const Filter& f, double theta_abs) {
    // x < a with |T_d(z(x))| = theta_abs  ->  |z| = cosh(acosh(theta)/d)
    if (theta_abs <= 1.0) return f.a;
    const double zz = std::cosh(std::acosh(theta_abs) / f.d);
    return 0.5 * (f.a + f.b - zz * (f.b - f.a));
}

}  // namespace ov

using namespace ov;

extern "C" int ov_lanczos_lowmodes(ov_ctx* ctx, int k, double tol, int max_restarts, int cheb_order, int subspace,
                                   void* V_out_dev, double* lambda_out_host, double* resid_out_host) {
    if (!ctx) return OV_EINVAL;
    if (k < 1 || !(tol > 0) || max_restarts < 1 || cheb_order < 1 || !V_out_dev || !lambda_out_host || !resid_out_host)
        return fail(ctx, OV_EINVAL, "bad argument to ov_lanczos_lowmodes");
    if (!(ctx->norm > 0)) return fail(ctx, OV_ESTATE, "ov_set_polynomial (norm) has not been called");
    const size_t n = spinor_elems(ctx), bytes = n * sizeof(double2);
    const long long dim = (long long)n;
    const int keep = k + std::max(8, k / 4);                    // wanted + buffer kept at every restart
    int m = subspace > 0 ? subspace : 2 * k + 16;
    if (m < keep + 8) m = keep + 8;
    if ((long long)m >= dim) return fail(ctx, OV_EINVAL, "subspace %d too large for dimension %lld", m, dim);

    double2* pool = nullptr;  // W[0..m], Y[0..keep), 3 scratch
    const size_t nvec = (size_t)m + 1 + keep + 3;
    OV_CUDA(ctx, cudaMalloc(&pool, bytes * nvec));
    double2* d_C = nullptr;
    if (cudaMalloc(&d_C, (size_t)m * 8 * sizeof(double2)) != cudaSuccess) { cudaFree(pool); return fail(ctx, OV_ENOMEM, "lanczos: out of memory"); }
    struct Free { double2 *a, *b; ~Free() { cudaFree(a); cudaFree(b); } } guard{pool, d_C};
    double2* W = pool;
    double2* Y = pool + (size_t)(m + 1) * n;
    double2* t0 = Y + (size_t)keep * n;
    double2* t1 = t0 + n;
    double2* tq = t1 + n;

    auto normalise = [&](double2* v, double* nrm) -> int {
        double s;
        OV_TRY(norm2_host(ctx, v, &s));
        *nrm = std::sqrt(s);
        return launch_scale(ctx, 1.0 / *nrm, v);
    };

    // ---- phase 0: a few plain Lanczos steps on A = Q^2 for an upper bound on lambda_min^2
    random_fill_kernel<<<(unsigned)((dim + 255) / 256), 256, 0, ctx->stream>>>(W, dim, 0x1111628800ull);
    ctx->launches++;
    double nrm;
    OV_TRY(normalise(W, &nrm));
    double theta_min;
    {
        const int m0 = std::min(m, 40);
        std::vector<double2> T((size_t)m0 * m0, make_double2(0, 0)), S;
        std::vector<double> th;
        std::vector<double2> c;
        const double inv = 1.0 / ctx->norm;
        for (int j = 0; j < m0; j++) {
            double2* u = W + (size_t)(j + 1) * n;
            Epilogue e1; e1.s = inv;
            OV_TRY(launch_wilson(ctx, W + (size_t)j * n, tq, e1));
            OV_TRY(launch_wilson(ctx, tq, u, e1));
            OV_TRY(cgs_pass(ctx, W, n, j + 1, u, d_C, c));
            double alpha = c[j].x;
            OV_TRY(cgs_pass(ctx, W, n, j + 1, u, d_C, c));
            alpha += c[j].x;
            T[(size_t)j * m0 + j].x = alpha;
            OV_TRY(normalise(u, &nrm));
            if (j + 1 < m0) { T[(size_t)j * m0 + j + 1].x = nrm; T[(size_t)(j + 1) * m0 + j].x = nrm; }
        }
        host_eigh(m0, T, th, S);
        theta_min = std::max(th[0], 1e-12);
    }
    Filter f{cheb_order, std::min(4.0 * theta_min, 0.5), 1.0};

    std::vector<double2> T((size_t)m * m), S, c;
    std::vector<double> th;
    int l = 0;            // kept Ritz vectors at the front of W
    double tolB = 0.1 * tol;
    bool refined_filter = false;
    int rc_final = OV_ENOCONV;
    std::fill(T.begin(), T.end(), make_double2(0, 0));
    // start vector: W[0] stays (normalised random)
    for (int restart = 0; restart < max_restarts; restart++) {
        for (int j = l; j < m; j++) {
            double2* u = W + (size_t)(j + 1) * n;
            OV_TRY(apply_filter(ctx, f, W + (size_t)j * n, u, t0, t1, tq));
            OV_TRY(cgs_pass(ctx, W, n, j + 1, u, d_C, c));
            double alpha = c[j].x;
            OV_TRY(cgs_pass(ctx, W, n, j + 1, u, d_C, c));
            alpha += c[j].x;
            T[(size_t)j * m + j] = make_double2(alpha, 0);
            OV_TRY(normalise(u, &nrm));
            if (j + 1 < m) { T[(size_t)j * m + j + 1] = make_double2(nrm, 0); T[(size_t)(j + 1) * m + j] = make_double2(nrm, 0); }
        }
        const double beta_last = nrm;
        std::vector<double2> Tc = T;
        host_eigh(m, Tc, th, S);
        std::vector<int> idx(m);
        std::iota(idx.begin(), idx.end(), 0);
        std::sort(idx.begin(), idx.end(), [&](int a, int b2) { return std::fabs(th[a]) > std::fabs(th[b2]); });
        std::vector<int> kept(idx.begin(), idx.begin() + keep);
        bool conv = true;
        for (int i = 0; i < k; i++) {
            const double2 s = S[(size_t)(m - 1) * m + kept[i]];
            const double res = beta_last * std::hypot(s.x, s.y);
            if (res > tolB * std::fabs(th[kept[i]])) { conv = false; break; }
        }
        // Ritz vectors of the kept set
        OV_TRY(rotate(ctx, W, n, m, S, m, kept, Y, d_C));

        if (!refined_filter) {
            // tighten the filter edge to just above the kept set, restart the Krylov space from the Ritz vectors
            const double xa = inverse_filter(f, std::fabs(th[kept[keep - 1]]));
            refined_filter = true;
            if (xa > 0 && xa < f.a) {
                f.a = std::max(xa, 1.0001 * inverse_filter(f, std::fabs(th[kept[k - 1]])));
                std::vector<double2> ones((size_t)keep, make_double2(1.0, 0.0));
                OV_CUDA(ctx, cudaMemcpyAsync(d_C, ones.data(), keep * sizeof(double2), cudaMemcpyHostToDevice, ctx->stream));
                OV_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
                MultiAxpyOuts o; o.out[0] = W;
                OV_TRY(launch_multi_axpy(ctx, Y, n, keep, 1, d_C, nullptr, o));
                OV_TRY(normalise(W, &nrm));
                std::fill(T.begin(), T.end(), make_double2(0, 0));
                l = 0;
                continue;
            }
        }

        if (conv) {
            // Rayleigh-Ritz in Q on span(Y): M = Y^+ Q Y
            std::vector<double2> M((size_t)keep * keep), SM;
            std::vector<double> mu;
            Epilogue eq; eq.s = 1.0 / ctx->norm;
            for (int j = 0; j < keep; j++) {
                OV_TRY(launch_wilson(ctx, Y + (size_t)j * n, tq, eq));
                OV_TRY(launch_multi_dot(ctx, Y, n, keep, tq));
                c.resize(keep);
                OV_TRY(fetch_results(ctx, keep, c.data()));
                for (int i = 0; i < keep; i++) M[(size_t)i * keep + j] = c[i];
            }
            for (int i = 0; i < keep; i++)
                for (int j = i; j < keep; j++) {  // symmetrise
                    const double2 a = M[(size_t)i * keep + j], b2 = M[(size_t)j * keep + i];
                    const double2 h = make_double2(0.5 * (a.x + b2.x), 0.5 * (a.y - b2.y));
                    M[(size_t)i * keep + j] = h;
                    M[(size_t)j * keep + i] = make_double2(h.x, -h.y);
                }
            host_eigh(keep, M, mu, SM);
            std::vector<int> sel(keep);
            std::iota(sel.begin(), sel.end(), 0);
            std::sort(sel.begin(), sel.end(), [&](int a, int b2) { return std::fabs(mu[a]) < std::fabs(mu[b2]); });
            sel.resize(k);
            double2* Vout = (double2*)V_out_dev;
            OV_TRY(rotate(ctx, Y, n, keep, SM, keep, sel, Vout, d_C));
            double worst = 0.0;
            for (int i = 0; i < k; i++) {
                double2* v = Vout + (size_t)i * n;
                double nv;
                OV_TRY(normalise(v, &nv));
                Epilogue er; er.s = 1.0 / ctx->norm; er.A1 = v; er.a1 = -mu[sel[i]];
                OV_TRY(launch_wilson(ctx, v, tq, er));
                double r2;
                OV_TRY(norm2_host(ctx, tq, &r2));
                lambda_out_host[i] = mu[sel[i]];
                resid_out_host[i] = std::sqrt(r2);
                worst = std::max(worst, resid_out_host[i]);
            }
            if (worst <= tol) { rc_final = OV_OK; break; }
            tolB *= 0.1;  // not there yet: ask more of the Krylov space and go on
        }

        // thick restart: W[0..keep) = Y, W[keep] = W[m], T = diag(theta) + arrow
        OV_CUDA(ctx, cudaMemcpyAsync(W, Y, bytes * (size_t)keep, cudaMemcpyDeviceToDevice, ctx->stream));
        OV_CUDA(ctx, cudaMemcpyAsync(W + (size_t)keep * n, W + (size_t)m * n, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
        std::fill(T.begin(), T.end(), make_double2(0, 0));
        for (int i = 0; i < keep; i++) {
            T[(size_t)i * m + i] = make_double2(th[kept[i]], 0);
            const double2 s = S[(size_t)(m - 1) * m + kept[i]];
            T[(size_t)i * m + keep] = make_double2(beta_last * s.x, -beta_last * s.y);
            T[(size_t)keep * m + i] = make_double2(beta_last * s.x, beta_last * s.y);
        }
        l = keep;
    }
    OV_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (rc_final != OV_OK) return fail(ctx, OV_ENOCONV, "lanczos: residual above tol after %d restarts", max_restarts);
    return OV_OK;
}
