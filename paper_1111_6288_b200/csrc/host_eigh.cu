// Host-side dense Hermitian eigensolver for the small projected matrices of the Lanczos routine
// (cyclic complex Jacobi; sizes are a few hundred at most).  Pure host code, no device work.
#include <algorithm>
#include <cmath>
#include <numeric>

#include "ov_internal.h"

namespace ov {

static inline double2 hmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
static inline double2 hconj(double2 a) { return make_double2(a.x, -a.y); }

// A: n x n Hermitian, row-major, destroyed.  w: eigenvalues ascending.  Z: row-major, eigenvectors as columns.
void host_eigh(int n, std::vector<double2>& A, std::vector<double>& w, std::vector<double2>& Z) {
    Z.assign((size_t)n * n, make_double2(0.0, 0.0));
    for (int i = 0; i < n; i++) Z[(size_t)i * n + i].x = 1.0;
    auto at = [&](int i, int j) -> double2& { return A[(size_t)i * n + j]; };
    double total = 0.0;
    for (auto& v : A) total += v.x * v.x + v.y * v.y;
    for (int sweep = 0; sweep < 60; sweep++) {
        double off = 0.0;
        for (int p = 0; p < n; p++)
            for (int q = p + 1; q < n; q++) off += at(p, q).x * at(p, q).x + at(p, q).y * at(p, q).y;
        if (off <= 1e-30 * total || off == 0.0) break;
        for (int p = 0; p < n - 1; p++) {
            for (int q = p + 1; q < n; q++) {
                const double2 apq = at(p, q);
                const double g = std::hypot(apq.x, apq.y);
                if (g < 1e-300) continue;
                const double app = at(p, p).x, aqq = at(q, q).x;
                // unit phase of a_pq, rotation angle from the real 2x2 problem [[app, g],[g, aqq]]
                const double2 ph = make_double2(apq.x / g, apq.y / g);
                const double tau = (aqq - app) / (2.0 * g);
                const double t = (tau >= 0 ? 1.0 : -1.0) / (std::fabs(tau) + std::sqrt(1.0 + tau * tau));
                const double c = 1.0 / std::sqrt(1.0 + t * t), s = t * c;
                // J = [[c, s*ph],[-s*conj(ph), c]] on columns (p,q):  A <- J^+ A J,  Z <- Z J
                const double2 sph = make_double2(s * ph.x, s * ph.y);
                for (int k = 0; k < n; k++) {  // columns: A[:,p], A[:,q]
                    const double2 akp = at(k, p), akq = at(k, q);
                    const double2 m1 = hmul(akq, hconj(sph));
                    const double2 m2 = hmul(akp, sph);
                    at(k, p) = make_double2(c * akp.x - m1.x, c * akp.y - m1.y);
                    at(k, q) = make_double2(c * akq.x + m2.x, c * akq.y + m2.y);
                }
                for (int k = 0; k < n; k++) {  // rows: A[p,:], A[q,:]  (J^+ from the left)
                    const double2 apk = at(p, k), aqk = at(q, k);
                    const double2 m1 = hmul(aqk, sph);
                    const double2 m2 = hmul(apk, hconj(sph));
                    at(p, k) = make_double2(c * apk.x - m1.x, c * apk.y - m1.y);
                    at(q, k) = make_double2(c * aqk.x + m2.x, c * aqk.y + m2.y);
                }
                at(p, q) = make_double2(0.0, 0.0);
                at(q, p) = make_double2(0.0, 0.0);
                at(p, p).y = 0.0;
                at(q, q).y = 0.0;
                for (int k = 0; k < n; k++) {
                    double2& zkp = Z[(size_t)k * n + p];
                    double2& zkq = Z[(size_t)k * n + q];
                    const double2 a = zkp, b = zkq;
                    const double2 m1 = hmul(b, hconj(sph));
                    const double2 m2 = hmul(a, sph);
                    zkp = make_double2(c * a.x - m1.x, c * a.y - m1.y);
                    zkq = make_double2(c * b.x + m2.x, c * b.y + m2.y);
                }
            }
        }
    }
    std::vector<int> idx(n);
    std::iota(idx.begin(), idx.end(), 0);
    std::sort(idx.begin(), idx.end(), [&](int a, int b) { return at(a, a).x < at(b, b).x; });
    w.resize(n);
    std::vector<double2> Zs((size_t)n * n);
    for (int j = 0; j < n; j++) {
        w[j] = at(idx[j], idx[j]).x;
        for (int k = 0; k < n; k++) Zs[(size_t)k * n + j] = Z[(size_t)k * n + idx[j]];
    }
    Z.swap(Zs);
}

}  // namespace ov

// test hook (host logic only; no device needed): A_host n*n complex row-major (re,im), outputs w[n], Z[n*n]
extern "C" int ov_host_eigh(int n, const double* A_host, double* w_out, double* Z_out) {
    if (n < 1 || !A_host || !w_out || !Z_out) return OV_EINVAL;
    std::vector<double2> A((size_t)n * n), Z;
    std::vector<double> w;
    for (size_t i = 0; i < (size_t)n * n; i++) A[i] = make_double2(A_host[2 * i], A_host[2 * i + 1]);
    ov::host_eigh(n, A, w, Z);
    for (int i = 0; i < n; i++) w_out[i] = w[i];
    for (size_t i = 0; i < (size_t)n * n; i++) { Z_out[2 * i] = Z[i].x; Z_out[2 * i + 1] = Z[i].y; }
    return OV_OK;
}
