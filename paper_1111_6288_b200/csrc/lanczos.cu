// Low modes of Q = H_w/norm (SURVEY 8a row a8; PAPER.md:57 "lowest lying eigenmodes of H_w", :71 "Chebyshev
// acceleration ... polynomial of order 100").  The paper uses implicitly restarted Arnoldi with a 2.5 l
// subspace; H_w is Hermitian, so this is thick-restart Lanczos (the Hermitian form of the same restart)
// on the filtered operator  B = T_d(z(Q^2)),  z(A) = (2A - a - b)/(b - a),  which maps the unwanted part
// [a,b] of the spectrum of Q^2 into [-1,1] and blows the wanted low end up like cosh(d acosh|z|).
// Every filter term is two launches of the Wilson kernel with the three-term axpy in its epilogue, the same
// fused step the Clenshaw recurrence uses.  A final Rayleigh-Ritz in Q itself separates +lambda from -lambda
// and the true residuals |Q v - lambda v| are measured with the kernel (contract: <= tol, G13).
//
// Memory: the basis W[0..m] is the only large object.  Its first k vectors ARE the caller's output buffer, the rest is a
// pool sized to what is free; restarts and the Rayleigh-Ritz step rotate the basis IN PLACE (rotate_inplace_kernel), so
// k = 200 on 32^3x64 (80.5 GB of eigenvectors) runs in 180 GB with a Krylov space of ~1.5 k instead of needing a second
// copy of the basis (the paper's 2.5 l subspace, would be 201 GB there).
#include <algorithm>
#include <chrono>
#include <cmath>
#include <functional>
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
static int apply_filter(ov_ctx* ctx, const Filter& f, const double2* in, double2* out, double2* t1,
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

// The eigenproblem the driver below works on: the wanted modes are the LOWEST eigenvalues of a Hermitian positive
// semi-definite "base" operator B with spectrum in [0, bmax], found by thick-restart Lanczos on T_d(z(B)); the final
// Rayleigh-Ritz step is done in a Hermitian operator R with R^2 = B (H_w: R = Q, B = Q^2, which separates +lambda from
// -lambda) or R = B (D_ov: one chirality sector of D_ov^+ D_ov).  All callbacks enqueue on ctx->stream.
struct LanczosOp {
    double bmax = 1.0;
    std::function<int(const double2* in, double2* out, double2* scratch)> base;                       // out = B in
    std::function<int(const Filter& f, const double2* in, double2* out, double2* t1, double2* tq)> filter;  // out = T_d(z(B)) in
    std::function<int(const double2* in, double2* out, double2* scratch)> rr;                         // out = R in
    std::function<int(double2* v, double2* scratch)> start;                                           // project the start vector (may be empty)
    std::function<double(double theta_min)> edge0;                                                    // first guess of the filter edge a
};

// out = T_d(z(B)) in for any base operator, three-term recurrence with separate BLAS-1 passes (used where one B costs
// hundreds of Wilson launches, so the two extra streaming passes per term do not matter).  Same buffer rotation as
// apply_filter: T_j lives in `out` when j has the parity of d, else in t1.
static int generic_filter(ov_ctx* ctx, const LanczosOp& op, const Filter& f, const double2* in, double2* out, double2* t1,
                          double2* tq, double2* scratch) {
    const double w = f.b - f.a, cs = (f.a + f.b) / w;
    auto buf = [&](int j) { return ((j & 1) == (f.d & 1)) ? out : t1; };
    OV_TRY(op.base(in, tq, scratch));
    OV_TRY(launch_axpby(ctx, 2.0 / w, tq, -cs, in, buf(1)));                       // T_1 = z(B) in
    for (int j = 2; j <= f.d; j++) {
        const double2* cur = buf(j - 1);
        const double2* prev = (j == 2) ? in : buf(j - 2);
        OV_TRY(op.base(cur, tq, scratch));
        OV_TRY(launch_axpbypcz(ctx, 4.0 / w, tq, -2.0 * cs, cur, -1.0, prev, buf(j)));   // T_j = 2 z T_{j-1} - T_{j-2}
    }
    return OV_OK;
}

// The Lanczos basis in two segments: vectors 0..na-1 in the caller's output buffer, the rest in the pool.
struct Basis {
    double2* a; int na; double2* b; size_t n;
    double2* vec(int i) const { return i < na ? a + (size_t)i * n : b + (size_t)(i - na) * n; }
};

// d_result[0..nv) = W[0..nv)^+ u
static int basis_dots(ov_ctx* ctx, const Basis& W, int nv, const double2* u) {
    const int n1 = std::min(nv, W.na), n2 = nv - n1;
    OV_TRY(launch_multi_dot_at(ctx, W.a, W.n, n1, u, 0, nv));
    if (n2 > 0) OV_TRY(launch_multi_dot_at(ctx, W.b, W.n, n2, u, n1, nv));
    return OV_OK;
}

// u += sum_{first <= i < first+nv} C[i-first] W[i]   (C: nv complex on the device)
static int basis_axpy(ov_ctx* ctx, const Basis& W, int first, int nv, const double2* d_C, double2* u) {
    MultiAxpyOuts o;
    o.out[0] = u; o.bscale[0] = 1.0;
    const int n1 = std::max(0, std::min(first + nv, W.na) - first), n2 = nv - n1;
    if (n1 > 0) OV_TRY(launch_multi_axpy(ctx, W.vec(first), W.n, n1, 1, d_C, u, o));
    if (n2 > 0) OV_TRY(launch_multi_axpy(ctx, W.vec(first + n1), W.n, n2, 1, d_C + n1, u, o));
    return OV_OK;
}

// u -= W[0..nv) (W^+ u), returns the coefficients (host) ; one classical Gram-Schmidt pass
static int cgs_pass(ov_ctx* ctx, const Basis& W, int nv, double2* u, double2* d_C, std::vector<double2>& c) {
    OV_TRY(basis_dots(ctx, W, nv, u));
    c.resize(nv);
    OV_TRY(fetch_results(ctx, nv, c.data()));
    std::vector<double2> neg(nv);
    for (int i = 0; i < nv; i++) neg[i] = make_double2(-c[i].x, -c[i].y);
    OV_CUDA(ctx, cudaMemcpyAsync(d_C, neg.data(), nv * sizeof(double2), cudaMemcpyHostToDevice, ctx->stream));
    OV_CUDA(ctx, cudaStreamSynchronize(ctx->stream));  // neg is a stack-owned host buffer
    return basis_axpy(ctx, W, 0, nv, d_C, u);
}

// W[j] <- sum_{i<m} S[i][cols[j]] W[i], j < cols.size(), in place  (S row-major m x ldS, host)
static int rotate(ov_ctx* ctx, const Basis& W, int m, const std::vector<double2>& S, int ldS, const std::vector<int>& cols,
                  double2* d_St) {
    const int ncol = (int)cols.size();
    std::vector<double2> St((size_t)ncol * m);
    for (int j = 0; j < ncol; j++)
        for (int i = 0; i < m; i++) St[(size_t)j * m + i] = S[(size_t)i * ldS + cols[j]];
    OV_CUDA(ctx, cudaMemcpyAsync(d_St, St.data(), St.size() * sizeof(double2), cudaMemcpyHostToDevice, ctx->stream));
    OV_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return launch_rotate_inplace(ctx, W.a, W.na, W.b, W.n, m, ncol, d_St);
}

// Where the time of a run goes (ov_lanczos_stats): CUDA events on the context's stream mark the start of each device
// phase; flush() synchronises, adds the interval between consecutive marks to the phase of the earlier one and recycles the
// events.  It is called where the driver synchronises anyway (before the host eigensolver, at the end of a run).
struct PhaseClock {
    enum { kFilter = 0, kOrtho = 1, kRotate = 2, kRitz = 3, kPhases = 4 };
    cudaStream_t stream;
    std::vector<cudaEvent_t> pool;
    std::vector<int> phase;
    size_t used = 0;
    double ms[kPhases] = {0, 0, 0, 0};
    explicit PhaseClock(cudaStream_t st) : stream(st) {}
    ~PhaseClock() { for (auto e : pool) cudaEventDestroy(e); }
    void mark(int ph) {   // ph = -1: end of the timed stretch
        if (used == pool.size()) {
            cudaEvent_t e;
            if (cudaEventCreate(&e) != cudaSuccess) return;
            pool.push_back(e);
            phase.push_back(-1);
        }
        phase[used] = ph;
        cudaEventRecord(pool[used++], stream);
    }
    void flush() {
        if (used == 0) return;
        mark(-1);
        cudaStreamSynchronize(stream);
        for (size_t i = 0; i + 1 < used; i++) {
            float t = 0.f;
            if (phase[i] >= 0 && cudaEventElapsedTime(&t, pool[i], pool[i + 1]) == cudaSuccess) ms[phase[i]] += t;
        }
        used = 0;
    }
};

static double inverse_filter(const Filter& f, double theta_abs) {
    // x < a with |T_d(z(x))| = theta_abs  ->  |z| = cosh(acosh(theta)/d)
    if (theta_abs <= 1.0) return f.a;
    const double zz = std::cosh(std::acosh(theta_abs) / f.d);
    return 0.5 * (f.a + f.b - zz * (f.b - f.a));
}

}  // namespace ov

using namespace ov;

extern "C" int ov_lanczos_stats(const ov_ctx* ctx, double* out_host) {
    if (!ctx || !out_host) return OV_EINVAL;
    for (size_t i = 0; i < ctx->lanczos_stats.size(); i++) out_host[i] = ctx->lanczos_stats[i];
    return OV_OK;
}

// Thick-restart Lanczos driver shared by the H_w and the D_ov low-mode routines (see LanczosOp).  nscratch extra spinors
// beyond t1, tq are allocated for the callbacks (op.base / op.rr get the first one).
static int lanczos_driver(ov_ctx* ctx, const LanczosOp& op, int k, double tol, int max_restarts, int cheb_order, int subspace,
                          void* V_out_dev, double* lambda_out_host, double* resid_out_host) {
    const size_t n = spinor_elems(ctx), bytes = n * sizeof(double2);
    const long long dim = (long long)n;
    const int keep = k + std::max(8, k / 4);                    // wanted + buffer kept at every restart
    const int m_min = keep + 8;
    int m = subspace > 0 ? subspace : 2 * k + 16;
    if (m < m_min) m = m_min;
    if ((long long)m >= dim) return fail(ctx, OV_EINVAL, "subspace %d too large for dimension %lld", m, dim);
    if ((size_t)m * kRotTileBytesPerVector > 220 * 1024) m = (int)(220 * 1024 / kRotTileBytesPerVector);
    {   // fit the pool into free memory: vectors k..m of the basis + 3 scratch (+ 2 GB head room for the workspaces)
        size_t free_b = 0, total_b = 0;
        OV_CUDA(ctx, cudaMemGetInfo(&free_b, &total_b));
        const size_t head = (size_t)2 << 30;
        const long long fit = free_b > head ? (long long)((free_b - head) / bytes) - 5 : 0;   // pool vectors available
        if (subspace <= 0 && (long long)(m + 1 - k) > fit) m = (int)(fit + k - 1);
        if (m < m_min) return fail(ctx, OV_ENOMEM, "lanczos: %d basis vectors do not fit in free device memory", m_min + 1);
    }

    double2* pool = nullptr;  // basis vectors k..m, then 3 scratch
    const size_t npool = (size_t)(m + 1 - k) + 3;
    OV_CUDA(ctx, cudaMalloc(&pool, bytes * npool));
    double2 *d_C = nullptr, *d_St = nullptr;
    if (cudaMalloc(&d_C, (size_t)(m + 1) * sizeof(double2)) != cudaSuccess ||
        cudaMalloc(&d_St, (size_t)m * keep * sizeof(double2)) != cudaSuccess) {
        cudaFree(pool); cudaFree(d_C);
        return fail(ctx, OV_ENOMEM, "lanczos: out of memory");
    }
    struct Free { double2 *a, *b, *c; ~Free() { cudaFree(a); cudaFree(b); cudaFree(c); } } guard{pool, d_C, d_St};
    const Basis W{(double2*)V_out_dev, k, pool, n};
    double2* t1 = pool + (size_t)(m + 1 - k) * n;
    double2* tq = t1 + n;
    double2* t2 = tq + n;

    auto normalise = [&](double2* v, double* nrm) -> int {
        double s;
        OV_TRY(norm2_host(ctx, v, &s));
        *nrm = std::sqrt(s);
        return launch_scale(ctx, 1.0 / *nrm, v);
    };

    // ---- phase 0: a few plain Lanczos steps on the base operator B for an upper bound on its lowest eigenvalue
    random_fill_kernel<<<(unsigned)((dim + 255) / 256), 256, 0, ctx->stream>>>(W.vec(0), dim, 0x1111628800ull);
    ctx->launches++;
    if (op.start) OV_TRY(op.start(W.vec(0), t2));
    double nrm;
    OV_TRY(normalise(W.vec(0), &nrm));
    double theta_min;
    {
        const int m0 = std::min(m, 40);
        std::vector<double2> T((size_t)m0 * m0, make_double2(0, 0)), S;
        std::vector<double> th;
        std::vector<double2> c;
        for (int j = 0; j < m0; j++) {
            double2* u = W.vec(j + 1);
            OV_TRY(op.base(W.vec(j), u, t2));
            OV_TRY(cgs_pass(ctx, W, j + 1, u, d_C, c));
            double alpha = c[j].x;
            OV_TRY(cgs_pass(ctx, W, j + 1, u, d_C, c));
            alpha += c[j].x;
            T[(size_t)j * m0 + j].x = alpha;
            OV_TRY(normalise(u, &nrm));
            if (j + 1 < m0) { T[(size_t)j * m0 + j + 1].x = nrm; T[(size_t)(j + 1) * m0 + j].x = nrm; }
        }
        if (!host_eigh(m0, T, th, S)) return fail(ctx, OV_ENOCONV, "dense eigensolver: QR iteration did not converge");
        theta_min = std::max(th[0], 1e-12);
    }
    Filter f{cheb_order, op.edge0(theta_min), op.bmax};

    std::vector<double2> T((size_t)m * m, make_double2(0, 0)), S, c;
    std::vector<double> th;
    int l = 0;            // kept Ritz vectors at the front of W
    double tolB = 0.1 * tol;
    bool refined_filter = false;
    int widenings = 0;
    long long filter_applies = 0;
    const long long launches0 = ctx->launches;
    ctx->lanczos_stats = {};
    int rc_final = OV_ENOCONV;
    PhaseClock clk(ctx->stream);
    double eigh_s = 0.0;
    const auto wall0 = std::chrono::steady_clock::now();
    auto seconds_since = [](std::chrono::steady_clock::time_point t0) {
        return std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    };
    auto timed_eigh = [&](int nn, std::vector<double2>& A, std::vector<double>& w, std::vector<double2>& Z) {
        clk.flush();                                    // the device is idle from here until the decomposition is back
        const auto t0 = std::chrono::steady_clock::now();
        const bool ok = host_eigh(nn, A, w, Z);
        eigh_s += seconds_since(t0);
        return ok;
    };
    auto write_times = [&]() {
        clk.flush();
        ctx->lanczos_stats[6] = eigh_s;
        ctx->lanczos_stats[7] = 1e-3 * clk.ms[PhaseClock::kFilter];
        ctx->lanczos_stats[8] = 1e-3 * clk.ms[PhaseClock::kOrtho];
        ctx->lanczos_stats[9] = 1e-3 * clk.ms[PhaseClock::kRotate];
        ctx->lanczos_stats[10] = 1e-3 * clk.ms[PhaseClock::kRitz];
        ctx->lanczos_stats[11] = seconds_since(wall0);
    };
    // start vector: W[0] stays (normalised random)
    for (int restart = 0; restart < max_restarts; restart++) {
        ctx->lanczos_stats[0] = (double)(restart + 1);
        ctx->lanczos_stats[1] = (double)filter_applies;
        ctx->lanczos_stats[3] = f.a;
        ctx->lanczos_stats[4] = (double)widenings;
        ctx->lanczos_stats[5] = (double)m;
        for (int j = l; j < m; j++) {
            double2* u = W.vec(j + 1);
            clk.mark(PhaseClock::kFilter);
            OV_TRY(op.filter(f, W.vec(j), u, t1, tq));
            filter_applies++;
            clk.mark(PhaseClock::kOrtho);
            OV_TRY(cgs_pass(ctx, W, j + 1, u, d_C, c));
            double alpha = c[j].x;
            OV_TRY(cgs_pass(ctx, W, j + 1, u, d_C, c));
            alpha += c[j].x;
            T[(size_t)j * m + j] = make_double2(alpha, 0);
            OV_TRY(normalise(u, &nrm));
            if (j + 1 < m) { T[(size_t)j * m + j + 1] = make_double2(nrm, 0); T[(size_t)(j + 1) * m + j] = make_double2(nrm, 0); }
        }
        const double beta_last = nrm;
        std::vector<double2> Tc = T;
        if (!timed_eigh(m, Tc, th, S)) return fail(ctx, OV_ENOCONV, "dense eigensolver: QR iteration did not converge");
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
        // Ritz vectors of the kept set, in place: W[0..keep) <- W[0..m) S[:, kept]
        clk.mark(PhaseClock::kRotate);
        OV_TRY(rotate(ctx, W, m, S, m, kept, d_St));
        clk.mark(-1);
        // projected matrix in the rotated basis: diag(theta) + the coupling to the residual vector W[m]
        std::vector<double2> Tk((size_t)keep * keep, make_double2(0, 0)), zk(keep);
        for (int i = 0; i < keep; i++) {
            Tk[(size_t)i * keep + i] = make_double2(th[kept[i]], 0);
            const double2 s = S[(size_t)(m - 1) * m + kept[i]];
            zk[i] = make_double2(beta_last * s.x, -beta_last * s.y);   // T[i][keep]
        }

        // restart the Krylov space from the sum of the kept Ritz vectors with a new filter edge
        auto restart_with_edge = [&](double new_a) -> int {
            f.a = new_a;
            std::vector<double2> ones((size_t)keep, make_double2(1.0, 0.0));
            OV_CUDA(ctx, cudaMemcpyAsync(d_C, ones.data(), keep * sizeof(double2), cudaMemcpyHostToDevice, ctx->stream));
            OV_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
            OV_TRY(basis_axpy(ctx, W, 1, keep - 1, d_C, W.vec(0)));   // W[0] = sum of the kept Ritz vectors
            OV_TRY(normalise(W.vec(0), &nrm));
            std::fill(T.begin(), T.end(), make_double2(0, 0));
            l = 0;
            return OV_OK;
        };
        if (!refined_filter) {
            // completeness guard: the amplified window [0, f.a) of B must hold the whole kept set.  If the keep-th Ritz
            // value is not amplified (|theta| <= 1: it sits in the damped interval, so modes below lambda_k may be hidden
            // there too), the first guess 4 theta_min was too tight -- widen the window and start again.
            if (std::fabs(th[kept[keep - 1]]) <= 1.0 + 1e-6 && f.a < 0.9 * op.bmax && widenings < 12) {
                widenings++;
                OV_TRY(restart_with_edge(std::min(2.0 * f.a, 0.9 * op.bmax)));
                continue;
            }
            // tighten the filter edge to just above the kept set, restart the Krylov space from the Ritz vectors
            const double xa = inverse_filter(f, std::fabs(th[kept[keep - 1]]));
            refined_filter = true;
            if (xa > 0 && xa < f.a) {
                OV_TRY(restart_with_edge(std::max(xa, 1.0001 * inverse_filter(f, std::fabs(th[kept[k - 1]])))));
                continue;
            }
        }
        if (conv) {
            // Rayleigh-Ritz in R on span(W[0..keep)): M = Y^+ R Y
            std::vector<double2> M((size_t)keep * keep), SM;
            std::vector<double> mu;
            clk.mark(PhaseClock::kRitz);
            for (int j = 0; j < keep; j++) {
                OV_TRY(op.rr(W.vec(j), tq, t2));
                OV_TRY(basis_dots(ctx, W, keep, tq));
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
            if (!timed_eigh(keep, M, mu, SM)) return fail(ctx, OV_ENOCONV, "dense eigensolver: QR iteration did not converge");
            std::vector<int> order(keep);
            std::iota(order.begin(), order.end(), 0);
            std::sort(order.begin(), order.end(), [&](int a, int b2) { return std::fabs(mu[a]) < std::fabs(mu[b2]); });
            // rotate the whole kept block by the unitary R = SM[:, order], in place: the wanted k eigenvectors of Q land in
            // W[0..k) = the caller's buffer, and W[0..keep) stays an orthonormal basis of the same space
            clk.mark(PhaseClock::kRotate);
            OV_TRY(rotate(ctx, W, keep, SM, keep, order, d_St));
            clk.mark(PhaseClock::kRitz);
            double worst = 0.0;
            for (int i = 0; i < k; i++) {
                double2* v = W.vec(i);
                double nv;
                OV_TRY(normalise(v, &nv));
                OV_TRY(op.rr(v, tq, t2));
                OV_TRY(launch_axpy(ctx, make_double2(-mu[order[i]], 0.0), v, tq));
                double r2;
                OV_TRY(norm2_host(ctx, tq, &r2));
                lambda_out_host[i] = mu[order[i]];
                resid_out_host[i] = std::sqrt(r2);
                worst = std::max(worst, resid_out_host[i]);
            }
            clk.mark(-1);
            if (worst <= tol) { rc_final = OV_OK; break; }
            tolB *= 0.1;  // not there yet: ask more of the Krylov space and go on, in the rotated basis
            std::vector<double2> R((size_t)keep * keep), tmp((size_t)keep * keep), z2(keep);
            for (int i = 0; i < keep; i++)
                for (int j = 0; j < keep; j++) R[(size_t)i * keep + j] = SM[(size_t)i * keep + order[j]];
            auto mul = [](double2 a, double2 b2) { return make_double2(a.x * b2.x - a.y * b2.y, a.x * b2.y + a.y * b2.x); };
            auto cj = [](double2 a) { return make_double2(a.x, -a.y); };
            for (int i = 0; i < keep; i++)       // tmp = Tk R   (Tk is diagonal here)
                for (int j = 0; j < keep; j++) tmp[(size_t)i * keep + j] = mul(Tk[(size_t)i * keep + i], R[(size_t)i * keep + j]);
            for (int a = 0; a < keep; a++) {     // Tk' = R^+ tmp ; z' = R^+ z
                double2 za = make_double2(0, 0);
                for (int i = 0; i < keep; i++) { const double2 p = mul(cj(R[(size_t)i * keep + a]), zk[i]); za.x += p.x; za.y += p.y; }
                z2[a] = za;
            }
            std::vector<double2> Tn((size_t)keep * keep, make_double2(0, 0));
            for (int a = 0; a < keep; a++)
                for (int i = 0; i < keep; i++) {
                    const double2 ra = cj(R[(size_t)i * keep + a]);
                    for (int b2 = 0; b2 < keep; b2++) {
                        const double2 p = mul(ra, tmp[(size_t)i * keep + b2]);
                        Tn[(size_t)a * keep + b2].x += p.x; Tn[(size_t)a * keep + b2].y += p.y;
                    }
                }
            Tk.swap(Tn);
            zk.swap(z2);
        }

        // thick restart: W[0..keep) holds the kept vectors, W[keep] = W[m], T = [Tk z; z^+ .]
        OV_CUDA(ctx, cudaMemcpyAsync(W.vec(keep), W.vec(m), bytes, cudaMemcpyDeviceToDevice, ctx->stream));
        std::fill(T.begin(), T.end(), make_double2(0, 0));
        for (int i = 0; i < keep; i++) {
            for (int j = 0; j < keep; j++) T[(size_t)i * m + j] = Tk[(size_t)i * keep + j];
            T[(size_t)i * m + keep] = zk[i];
            T[(size_t)keep * m + i] = make_double2(zk[i].x, -zk[i].y);
        }
        l = keep;
    }
    ctx->lanczos_stats[1] = (double)filter_applies;
    ctx->lanczos_stats[2] = (double)(ctx->launches - launches0);
    ctx->lanczos_stats[3] = f.a;
    ctx->lanczos_stats[4] = (double)widenings;
    write_times();
    OV_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (rc_final != OV_OK) return fail(ctx, OV_ENOCONV, "lanczos: residual above tol after %d restarts", max_restarts);
    return OV_OK;
}

extern "C" int ov_lanczos_lowmodes(ov_ctx* ctx, int k, double tol, int max_restarts, int cheb_order, int subspace,
                                   void* V_out_dev, double* lambda_out_host, double* resid_out_host) {
    if (!ctx) return OV_EINVAL;
    if (k < 1 || !(tol > 0) || max_restarts < 1 || cheb_order < 1 || !V_out_dev || !lambda_out_host || !resid_out_host)
        return fail(ctx, OV_EINVAL, "bad argument to ov_lanczos_lowmodes");
    if (!(ctx->norm > 0)) return fail(ctx, OV_ESTATE, "ov_set_polynomial (norm) has not been called");
    LanczosOp op;
    op.bmax = 1.0;                                     // B = Q^2, R = Q
    const double inv = 1.0 / ctx->norm;
    op.base = [ctx, inv](const double2* in, double2* out, double2* scratch) -> int {
        Epilogue e1; e1.s = inv;
        OV_TRY(launch_wilson(ctx, in, scratch, e1));
        return launch_wilson(ctx, scratch, out, e1);
    };
    op.filter = [ctx](const Filter& f, const double2* in, double2* out, double2* t1, double2* tq) -> int {
        return apply_filter(ctx, f, in, out, t1, tq);
    };
    op.rr = [ctx, inv](const double2* in, double2* out, double2*) -> int {
        Epilogue eq; eq.s = inv;
        return launch_wilson(ctx, in, out, eq);
    };
    op.edge0 = [](double theta_min) { return std::min(4.0 * theta_min, 0.5); };
    return lanczos_driver(ctx, op, k, tol, max_restarts, cheb_order, subspace, V_out_dev, lambda_out_host, resid_out_host);
}

// Low modes of the overlap operator ("computing the low lying spectrum of the overlap
// operator", :81 "Arnoldi ... Chebyshev acceleration ... Chebyshev order of 12").  Reading G20: the modes are
// eigenpairs of A = D_ov(0)^+ D_ov(0) = 2 + gamma5 S + S gamma5, computed in ONE chirality sector s, where
//     A_s x = 2 x + (s + gamma5) sign(H_w) x          (one sign per application, spectrum in [0, 4(1+delta)])
// is non-degenerate; the other sector holds the same non-zero levels.  The same thick-restart driver as for H_w, with
// B = R = A_s and the Chebyshev filter built from whole applications of A_s.
extern "C" int ov_lanczos_dov_lowmodes(ov_ctx* ctx, int chirality, int k, double tol, int max_restarts, int cheb_order,
                                       int subspace, void* W_out_dev, double* mu_out_host, double* resid_out_host) {
    if (!ctx) return OV_EINVAL;
    if ((chirality != 1 && chirality != -1) || k < 1 || !(tol > 0) || max_restarts < 1 || cheb_order < 1 || !W_out_dev ||
        !mu_out_host || !resid_out_host)
        return fail(ctx, OV_EINVAL, "bad argument to ov_lanczos_dov_lowmodes");
    if (ctx->order < 0) return fail(ctx, OV_ESTATE, "ov_set_polynomial has not been called");
    for (int i = 0; i <= 5; i++) {                     // the sign's workspaces, before the driver sizes its pool to free memory
        double2* w;
        OV_TRY(workspace(ctx, i, &w));
    }
    LanczosOp op;
    op.bmax = 4.2;                                     // (1 + |S|)^2 with |S| <= 1 + delta, delta < 0.02
    auto sector = [ctx, chirality](const double2* in, double2* out, double2* scratch) -> int {
        OV_TRY(apply_sign(ctx, in, scratch));
        return launch_chiral_combine(ctx, 2.0, in, chirality, scratch, out);
    };
    op.base = sector;
    op.rr = sector;
    // the filter needs one more scratch spinor than the driver hands over: workspace 5 (apply_sign uses 0-4)
    const LanczosOp* self = &op;
    op.filter = [ctx, self](const Filter& f, const double2* in, double2* out, double2* t1, double2* tq) -> int {
        double2* scratch;
        OV_TRY(workspace(ctx, 5, &scratch));
        return generic_filter(ctx, *self, f, in, out, t1, tq, scratch);
    };
    op.start = [ctx, chirality](double2* v, double2* scratch) -> int {            // v <- (1 + s gamma5) v
        OV_TRY(launch_copy(ctx, v, scratch));
        return launch_chiral_combine(ctx, 0.0, nullptr, chirality, scratch, v);
    };
    op.edge0 = [](double theta_min) { return std::max(4.0 * theta_min, 0.2); };
    return lanczos_driver(ctx, op, k, tol, max_restarts, cheb_order, subspace, W_out_dev, mu_out_host, resid_out_host);
}
