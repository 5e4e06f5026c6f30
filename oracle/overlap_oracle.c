/*
 * ORACLE -- TEST INFRASTRUCTURE ONLY.  Not part of the product path.
 *
 * Plain, slow, fp64 CPU statement of what the hot path of arXiv 1111.6288 computes, written from the
 * paper and the readings listed in DESIGN.md.  It shares no code, header,
 * table or helper with the CUDA library under paper_1111_6288_b200/csrc.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.
 *
 * Data layout (canonical AoS, the layout workloads/ generates):
 *   gauge   U[site][mu][row][col]      complex double, mu = 0..3 = x,y,z,t ; U_mu(x) links x -> x+mu
 *   spinor  psi[site][spin][colour]    complex double, 4 spins x 3 colours
 *   site    i = x + X*(y + Y*(z + Z*t)),  dims = {X,Y,Z,T}
 *
 * No spin-projection trick, no blocking, no fusion: every hop multiplies by the full 4x4 matrix
 * (1 -+ gamma_mu) and the full 3x3 link, exactly as the operator is written.  The only parallelism is
 * an OpenMP "parallel for" over lattice sites (each site is computed independently in the same
 * arithmetic order, so results do not depend on the thread count).
 *
 * Pins (tests/test_oracle_pins.py): gamma algebra, H_w hermiticity, free-field spectrum in closed form,
 * gauge covariance, dense brute force on 4^4, sign^2 = 1, Ginsparg-Wilson, eq. 2.2, Fig. 1.
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

#define NS 4
#define NC 3
#define SPINOR (NS * NC)

/* ---- gamma matrices: DESIGN.md reading G2 (paper silent, PAPER.md:29-31 only names gamma5) --------
 * Hermitian chiral basis, gamma5 = diag(1,1,-1,-1) = gamma1 gamma2 gamma3 gamma4:
 *   gamma_k = [[0, -i sigma_k],[i sigma_k, 0]] (k=1,2,3),  gamma4 = [[0,1],[1,0]].
 * Index 0..3 = gamma_x, gamma_y, gamma_z, gamma_t ; index 4 = gamma5.                              */
static const cplx GAMMA[5][NS][NS] = {
    {{0, 0, 0, -I}, {0, 0, -I, 0}, {0, I, 0, 0}, {I, 0, 0, 0}},
    {{0, 0, 0, -1}, {0, 0, 1, 0}, {0, 1, 0, 0}, {-1, 0, 0, 0}},
    {{0, 0, -I, 0}, {0, 0, 0, I}, {I, 0, 0, 0}, {0, -I, 0, 0}},
    {{0, 0, 1, 0}, {0, 0, 0, 1}, {1, 0, 0, 0}, {0, 1, 0, 0}},
    {{1, 0, 0, 0}, {0, 1, 0, 0}, {0, 0, -1, 0}, {0, 0, 0, -1}},
};

void orc_gamma(int idx, cplx *out16)
{
    for (int a = 0; a < NS; a++)
        for (int b = 0; b < NS; b++) out16[a * NS + b] = GAMMA[idx][a][b];
}

static long nsites(const int *d) { return (long)d[0] * d[1] * d[2] * d[3]; }

/* Boundary factor of a hop that crosses the lattice boundary in direction mu: +1 periodic, -1 antiperiodic,
 * 0 Dirichlet/open (the hop is removed).  Default = north_star's: periodic in space, antiperiodic in time
 * (reading G11).  PAPER.md:104 "we use Dirichlet boundary conditions both in the direction of the
 * applied electric field and time" is BC = 0 in those two directions (set by orc_set_boundary).             */
static double BC[4] = {1.0, 1.0, 1.0, -1.0};

void orc_set_boundary(const double *bc4)
{
    for (int mu = 0; mu < 4; mu++) BC[mu] = bc4[mu];
}

/* neighbour of site (c[0..3]) one step in direction mu (dir=+1/-1), periodic index; *phase gets the
 * boundary factor BC[mu] when the hop crosses between coordinate d[mu]-1 and 0, +1 otherwise.             */
static long neighbour(const int *d, const int *c, int mu, int dir, double *phase)
{
    int n[4] = {c[0], c[1], c[2], c[3]};
    n[mu] = c[mu] + dir;
    *phase = 1.0;
    if (n[mu] >= d[mu]) {
        n[mu] -= d[mu];
        *phase = BC[mu];
    }
    if (n[mu] < 0) {
        n[mu] += d[mu];
        *phase = BC[mu];
    }
    return n[0] + (long)d[0] * (n[1] + (long)d[1] * (n[2] + (long)d[2] * n[3]));
}

/* Wilson hopping term (the "dslash"):
 *   out(x) = sum_mu [ s+ (1 - gamma_mu) U_mu(x) psi(x+mu) + s- (1 + gamma_mu) U_mu(x-mu)^dagger psi(x-mu) ]
 * (reading G1).                                                                            */
void orc_wilson_hop(const int *dims, const cplx *U, const cplx *psi, cplx *out)
{
    const long V = nsites(dims);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < V; i++) {
        int c[4];
        long r = i;
        c[0] = (int)(r % dims[0]); r /= dims[0];
        c[1] = (int)(r % dims[1]); r /= dims[1];
        c[2] = (int)(r % dims[2]); r /= dims[2];
        c[3] = (int)r;
        cplx acc[NS][NC];
        memset(acc, 0, sizeof acc);
        for (int mu = 0; mu < 4; mu++) {
            double sp, sm;
            const long ip = neighbour(dims, c, mu, +1, &sp);
            const long im = neighbour(dims, c, mu, -1, &sm);
            const cplx *Uf = U + (i * 4 + mu) * 9;  /* U_mu(x)      */
            const cplx *Ub = U + (im * 4 + mu) * 9; /* U_mu(x - mu) */
            const cplx *pf = psi + ip * SPINOR;
            const cplx *pb = psi + im * SPINOR;
            cplx cf[NS][NC], cb[NS][NC]; /* colour-multiplied neighbours */
            for (int s = 0; s < NS; s++)
                for (int a = 0; a < NC; a++) {
                    cplx f = 0, b = 0;
                    for (int bb = 0; bb < NC; bb++) {
                        f += Uf[a * 3 + bb] * pf[s * NC + bb];        /* U psi          */
                        b += conj(Ub[bb * 3 + a]) * pb[s * NC + bb];  /* U^dagger psi   */
                    }
                    cf[s][a] = f;
                    cb[s][a] = b;
                }
            for (int s = 0; s < NS; s++)
                for (int a = 0; a < NC; a++) {
                    cplx f = 0, b = 0;
                    for (int s2 = 0; s2 < NS; s2++) {
                        const cplx one = (s == s2) ? 1.0 : 0.0;
                        f += (one - GAMMA[mu][s][s2]) * cf[s2][a];
                        b += (one + GAMMA[mu][s][s2]) * cb[s2][a];
                    }
                    acc[s][a] += sp * f + sm * b;
                }
        }
        memcpy(out + i * SPINOR, acc, sizeof acc);
    }
}

/* D_w psi = psi - kappa * hop(psi), kappa = 1/(2(m0+4)) ; H_w = gamma5 D_w.          */
void orc_hw(const int *dims, double kappa, const cplx *U, const cplx *in, cplx *out)
{
    const long V = nsites(dims);
    orc_wilson_hop(dims, U, in, out);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < V; i++)
        for (int s = 0; s < NS; s++)
            for (int a = 0; a < NC; a++) {
                const long e = i * SPINOR + s * NC + a;
                out[e] = GAMMA[4][s][s] * (in[e] - kappa * out[e]);
            }
}

/* Q = H_w / norm  (norm is the caller's bound on ||H_w||, reading G3).                  */
static void apply_Q(const int *dims, double kappa, double norm, const cplx *U, const cplx *in, cplx *out)
{
    const long N = nsites(dims) * SPINOR;
    orc_hw(dims, kappa, U, in, out);
#pragma omp parallel for schedule(static)
    for (long e = 0; e < N; e++) out[e] /= norm;
}

/* Large-space polynomial sign ("sign(H_w) ~ Q P(Q^2)"), P = sum_{j=0..n} c_j T_j(z),
 * z = (2 Q^2 - 1 - eps)/(1 - eps), evaluated by the Clenshaw recurrence in the order of DESIGN.md O6:
 *   alpha = 4/(1-eps), beta = 2(1+eps)/(1-eps)   (2z = alpha Q^2 - beta)
 *   b_{n+1} = b_{n+2} = 0
 *   j = n..1:  b_j = c_j x + alpha Q(Q b_{j+1}) - beta b_{j+1} - b_{j+2}
 *   y = c_0 x + (alpha Q(Q b_1) - beta b_1)/2 - b_2 ;  result = Q y
 * c_0 is the true T_0 coefficient (reading G5).                                                      */
void orc_sign_poly(const int *dims, double kappa, const cplx *U, const double *coef, int n, double eps,
                   double norm, const cplx *x, cplx *out)
{
    const long N = nsites(dims) * SPINOR;
    const double alpha = 4.0 / (1.0 - eps), beta = 2.0 * (1.0 + eps) / (1.0 - eps);
    cplx *b1 = calloc(N, sizeof(cplx)), *b2 = calloc(N, sizeof(cplx));
    cplx *t1 = malloc(N * sizeof(cplx)), *t2 = malloc(N * sizeof(cplx)), *bn = malloc(N * sizeof(cplx));
    for (int j = n; j >= 1; j--) {
        apply_Q(dims, kappa, norm, U, b1, t1);
        apply_Q(dims, kappa, norm, U, t1, t2); /* t2 = Q^2 b_{j+1} */
#pragma omp parallel for schedule(static)
        for (long e = 0; e < N; e++) bn[e] = coef[j] * x[e] + alpha * t2[e] - beta * b1[e] - b2[e];
        cplx *tmp = b2; b2 = b1; b1 = bn; bn = tmp;
    }
    apply_Q(dims, kappa, norm, U, b1, t1);
    apply_Q(dims, kappa, norm, U, t1, t2);
#pragma omp parallel for schedule(static)
    for (long e = 0; e < N; e++) bn[e] = coef[0] * x[e] + 0.5 * (alpha * t2[e] - beta * b1[e]) - b2[e];
    apply_Q(dims, kappa, norm, U, bn, out);
    free(b1); free(b2); free(t1); free(t2); free(bn);
}

/* sign(H_w) x with the small space treated exactly (O7, readings G7, G12):
 *   c = V^dagger x ; x_perp = x - V c ; out = sum_i sign(lambda_i) c_i v_i + [Q P(Q^2)] x_perp
 * V: k spinors, contiguous, canonical layout; lambda: eigenvalues of Q. k = 0 -> polynomial only.   */
void orc_sign(const int *dims, double kappa, const cplx *U, const double *coef, int n, double eps, double norm,
              const cplx *V, const double *lambda, int k, const cplx *x, cplx *out)
{
    const long N = nsites(dims) * SPINOR;
    cplx *xp = malloc(N * sizeof(cplx));
    cplx *c = malloc((k > 0 ? k : 1) * sizeof(cplx));
    memcpy(xp, x, N * sizeof(cplx));
    for (int i = 0; i < k; i++) {
        cplx s = 0;
        const cplx *v = V + (long)i * N;
        for (long e = 0; e < N; e++) s += conj(v[e]) * x[e];
        c[i] = s;
    }
    for (int i = 0; i < k; i++) {
        const cplx *v = V + (long)i * N;
#pragma omp parallel for schedule(static)
        for (long e = 0; e < N; e++) xp[e] -= c[i] * v[e];
    }
    orc_sign_poly(dims, kappa, U, coef, n, eps, norm, xp, out);
    for (int i = 0; i < k; i++) {
        const cplx *v = V + (long)i * N;
        const double sg = (lambda[i] > 0) ? 1.0 : -1.0;
#pragma omp parallel for schedule(static)
        for (long e = 0; e < N; e++) out[e] += sg * c[i] * v[e];
    }
    free(xp); free(c);
}

/* D_ov(m) x = (1 + m/2) x + (1 - m/2) gamma5 sign(H_w) x ; m = 0 is eq. 2.1, the mass
 * form is DESIGN.md reading G9.                                                                      */
void orc_dov(const int *dims, double kappa, const cplx *U, const double *coef, int n, double eps, double norm,
             const cplx *V, const double *lambda, int k, double mass, const cplx *x, cplx *out)
{
    const long Vs = nsites(dims);
    orc_sign(dims, kappa, U, coef, n, eps, norm, V, lambda, k, x, out);
    for (long i = 0; i < Vs; i++)
        for (int s = 0; s < NS; s++)
            for (int a = 0; a < NC; a++) {
                const long e = i * SPINOR + s * NC + a;
                out[e] = (1.0 + 0.5 * mass) * x[e] + (1.0 - 0.5 * mass) * GAMMA[4][s][s] * out[e];
            }
}
