// Host-side dense Hermitian eigensolver for the small projected matrices of the Lanczos routine (sizes
// m = 2k + 16 = 116 ... 416).  Pure host code, no device work.  The GPU idles while it runs, once per restart cycle, so it
// has to be quick: Householder reduction to a real symmetric tridiagonal matrix, implicit-shift QR on that with the
// rotations accumulated, back-transformation (~20 n^3 flops): 0.04 s at n = 216 and 0.23 s at n = 416 on one host core,
// where the cyclic Jacobi sweeps of rounds 1-2 took 0.93 s and 8.9 s.
#include <algorithm>
#include <cfloat>
#include <cmath>
#include <numeric>

#include "ov_internal.h"

namespace ov {

static inline double2 hmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

// ---- Householder + implicit-shift QR ------------------------------------------------------------------------------
// A = Q T_c Q^+ with Q = H_0 ... H_{n-3}, H_k = 1 - 2 v_k v_k^+ acting on indices k+1..n-1, T_c Hermitian tridiagonal with
// complex sub-diagonal e_c.  A diagonal unitary D (d_0 = 1, d_{k+1} = d_k e_c[k]/|e_c[k]|) makes it real: T_c = D T_r D^+.
// T_r = R diag(w) R^T by QR sweeps with Wilkinson shifts, deflating from the bottom.  Eigenvectors of A: Z = Q D R.
// Only the lower triangle of A is read and updated.  Returns false if the QR iteration hits its cap (never seen).
// Accuracy is the backward-stable kind, |A Z - Z w| ~ eps |A|: enough for the Ritz values the Lanczos driver keeps (the
// largest of the filtered operator) and for the Rayleigh-Ritz step in Q (|lambda| ~ 1e-2, tolerance 1e-8).
static bool eigh_householder_qr(int n, std::vector<double2>& A, std::vector<double>& w, std::vector<double2>& Z) {
    auto at = [&](int i, int j) -> double2& { return A[(size_t)i * n + j]; };
    std::vector<double2> vs((size_t)n * n, make_double2(0.0, 0.0));   // v_k in row k, entries 0..n-k-2
    std::vector<double2> p(n), q(n), ec(n > 1 ? n - 1 : 0, make_double2(0.0, 0.0));
    for (int k = 0; k + 2 < n; k++) {
        const int m = n - k - 1;              // x = A[k+1.., k], length m
        double2* v = &vs[(size_t)k * n];
        double nx2 = 0.0;
        for (int i = 0; i < m; i++) { v[i] = at(k + 1 + i, k); nx2 += v[i].x * v[i].x + v[i].y * v[i].y; }
        const double nx = std::sqrt(nx2);
        if (nx == 0.0) { for (int i = 0; i < m; i++) v[i] = make_double2(0.0, 0.0); continue; }   // nothing to eliminate
        const double a0 = std::hypot(v[0].x, v[0].y);
        const double2 ph = a0 > 0.0 ? make_double2(v[0].x / a0, v[0].y / a0) : make_double2(1.0, 0.0);
        ec[k] = make_double2(-ph.x * nx, -ph.y * nx);          // H x = alpha e_1, alpha = -phase(x_0) |x|
        v[0].x += ph.x * nx; v[0].y += ph.y * nx;              // v = x - alpha e_1 (no cancellation)
        double nv2 = 0.0;
        for (int i = 0; i < m; i++) nv2 += v[i].x * v[i].x + v[i].y * v[i].y;
        const double inv = 1.0 / std::sqrt(nv2);
        for (int i = 0; i < m; i++) { v[i].x *= inv; v[i].y *= inv; }
        // trailing block B = A[k+1.., k+1..] <- H B H = B - v q^+ - q v^+,  p = B v, K = v^+ p (real), q = 2 (p - K v)
        for (int i = 0; i < m; i++) p[i] = make_double2(0.0, 0.0);
        for (int i = 0; i < m; i++) {
            const double2* row = &at(k + 1 + i, k + 1);
            double2 acc = p[i];
            for (int j = 0; j < i; j++) {
                const double2 b = row[j];
                acc.x += b.x * v[j].x - b.y * v[j].y; acc.y += b.x * v[j].y + b.y * v[j].x;          // B_ij v_j
                p[j].x += b.x * v[i].x + b.y * v[i].y; p[j].y += b.x * v[i].y - b.y * v[i].x;        // conj(B_ij) v_i
            }
            acc.x += row[i].x * v[i].x; acc.y += row[i].x * v[i].y;                                  // real diagonal
            p[i] = acc;
        }
        double K = 0.0;
        for (int i = 0; i < m; i++) K += v[i].x * p[i].x + v[i].y * p[i].y;
        for (int i = 0; i < m; i++) q[i] = make_double2(2.0 * (p[i].x - K * v[i].x), 2.0 * (p[i].y - K * v[i].y));
        for (int i = 0; i < m; i++) {
            double2* row = &at(k + 1 + i, k + 1);
            const double2 vi = v[i], qi = q[i];
            for (int j = 0; j <= i; j++) {     // B_ij -= v_i conj(q_j) + q_i conj(v_j)
                row[j].x -= vi.x * q[j].x + vi.y * q[j].y + qi.x * v[j].x + qi.y * v[j].y;
                row[j].y -= vi.y * q[j].x - vi.x * q[j].y + qi.y * v[j].x - qi.x * v[j].y;
            }
            row[i].y = 0.0;
        }
    }
    if (n >= 2) ec[n - 2] = at(n - 1, n - 2);
    std::vector<double> d(n), e(n > 1 ? n - 1 : 0);
    std::vector<double2> dph(n, make_double2(1.0, 0.0));
    for (int i = 0; i < n; i++) d[i] = at(i, i).x;
    for (int k = 0; k + 1 < n; k++) {
        e[k] = std::hypot(ec[k].x, ec[k].y);
        const double2 u = e[k] > 0.0 ? make_double2(ec[k].x / e[k], ec[k].y / e[k]) : make_double2(1.0, 0.0);
        dph[k + 1] = hmul(dph[k], u);
    }
    // QR sweeps on (d, e); Rt row j = column j of R
    std::vector<double> Rt((size_t)n * n, 0.0);
    for (int i = 0; i < n; i++) Rt[(size_t)i * n + i] = 1.0;
    auto negligible = [&](int k) { return std::fabs(e[k]) <= DBL_EPSILON * (std::fabs(d[k]) + std::fabs(d[k + 1])); };
    int hi = n - 1;
    long long sweeps = 0;
    while (hi > 0) {
        if (negligible(hi - 1)) { e[hi - 1] = 0.0; hi--; continue; }
        int lo = hi - 1;
        while (lo > 0 && !negligible(lo - 1)) lo--;
        if (lo > 0) e[lo - 1] = 0.0;
        if (++sweeps > 60LL * n) return false;
        const double delta = 0.5 * (d[hi - 1] - d[hi]), b2 = e[hi - 1] * e[hi - 1];
        const double mu = d[hi] - b2 / (delta + std::copysign(std::sqrt(delta * delta + b2), delta));   // Wilkinson shift
        double x = d[lo] - mu, z = e[lo];
        for (int k = lo; k < hi; k++) {
            // rotation in the (k, k+1) plane with G (x, z)^T = (r, 0)^T, G = [[c, s], [-s, c]];  T <- G T G^T
            const double r = std::hypot(x, z);
            const double c = r > 0.0 ? x / r : 1.0, s = r > 0.0 ? z / r : 0.0;
            if (k > lo) e[k - 1] = r;
            const double a = d[k], b = e[k], cc = d[k + 1];
            d[k] = c * c * a + 2.0 * c * s * b + s * s * cc;
            d[k + 1] = s * s * a - 2.0 * c * s * b + c * c * cc;
            e[k] = c * s * (cc - a) + (c * c - s * s) * b;
            if (k + 1 < hi) { z = s * e[k + 1]; e[k + 1] = c * e[k + 1]; x = e[k]; }   // the bulge moves down
            double* r0 = &Rt[(size_t)k * n];
            double* r1 = r0 + n;
            for (int i = 0; i < n; i++) {      // R <- R G^T
                const double t0 = r0[i], t1 = r1[i];
                r0[i] = c * t0 + s * t1;
                r1[i] = c * t1 - s * t0;
            }
        }
    }
    // Z = Q D R, one eigenvector (row of Mt) at a time: reflectors in reverse order
    std::vector<double2> Mt((size_t)n * n);
    for (int j = 0; j < n; j++)
        for (int i = 0; i < n; i++) {
            const double rij = Rt[(size_t)j * n + i];
            Mt[(size_t)j * n + i] = make_double2(dph[i].x * rij, dph[i].y * rij);
        }
    for (int k = n - 3; k >= 0; k--) {
        const int m = n - k - 1;
        const double2* v = &vs[(size_t)k * n];
        for (int j = 0; j < n; j++) {
            double2* col = &Mt[(size_t)j * n + k + 1];
            double2 sacc = make_double2(0.0, 0.0);   // v^+ col
            for (int i = 0; i < m; i++) { sacc.x += v[i].x * col[i].x + v[i].y * col[i].y; sacc.y += v[i].x * col[i].y - v[i].y * col[i].x; }
            sacc.x *= 2.0; sacc.y *= 2.0;
            for (int i = 0; i < m; i++) { col[i].x -= sacc.x * v[i].x - sacc.y * v[i].y; col[i].y -= sacc.x * v[i].y + sacc.y * v[i].x; }
        }
    }
    std::vector<int> idx(n);
    std::iota(idx.begin(), idx.end(), 0);
    std::sort(idx.begin(), idx.end(), [&](int a, int b) { return d[a] < d[b]; });
    w.resize(n);
    Z.resize((size_t)n * n);
    for (int j = 0; j < n; j++) {
        w[j] = d[idx[j]];
        for (int i = 0; i < n; i++) Z[(size_t)i * n + j] = Mt[(size_t)idx[j] * n + i];
    }
    return true;
}

// A: n x n Hermitian, row-major, destroyed (only its lower triangle is read).  w: eigenvalues ascending.  Z: row-major,
// eigenvectors as columns.  false: the QR iteration hit its cap of 60 n sweeps (callers report OV_ENOCONV).
bool host_eigh(int n, std::vector<double2>& A, std::vector<double>& w, std::vector<double2>& Z) {
    return eigh_householder_qr(n, A, w, Z);
}

}  // namespace ov

// test hook (host logic only; no device needed): A_host n*n complex row-major (re,im), outputs w[n], Z[n*n]
extern "C" int ov_host_eigh(int n, const double* A_host, double* w_out, double* Z_out) {
    if (n < 1 || !A_host || !w_out || !Z_out) return OV_EINVAL;
    std::vector<double2> A((size_t)n * n), Z;
    std::vector<double> w;
    for (size_t i = 0; i < (size_t)n * n; i++) A[i] = make_double2(A_host[2 * i], A_host[2 * i + 1]);
    if (!ov::host_eigh(n, A, w, Z)) return OV_ENOCONV;
    for (int i = 0; i < n; i++) w_out[i] = w[i];
    for (size_t i = 0; i < (size_t)n * n; i++) { Z_out[2 * i] = Z[i].x; Z_out[2 * i + 1] = Z[i].y; }
    return OV_OK;
}
