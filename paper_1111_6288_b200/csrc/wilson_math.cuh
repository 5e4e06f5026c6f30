// Device-side arithmetic of the Wilson hopping term for the chiral gamma basis of include/ov.h
// (reading G2).  All four gamma_mu are block-off-diagonal, so (1 + sigma*gamma_mu) psi has rank
// 2: its upper two spin components h = (r0, r1) determine the lower two.  A hop therefore costs one
// projection to a half-spinor (6 complex), one SU(3) mat-vec on 2 spin components, and one
// reconstruct-accumulate.  sigma = -1 for the forward hop (1 - gamma_mu), +1 for the backward hop.
#pragma once
#include <cuda_runtime.h>

namespace ov {

__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
// a + i*s*b
__device__ __forceinline__ double2 caddi(double2 a, double2 b, double s) {
    return make_double2(a.x - s * b.y, a.y + s * b.x);
}
// a + s*b (s real)
__device__ __forceinline__ double2 cadds(double2 a, double2 b, double s) {
    return make_double2(a.x + s * b.x, a.y + s * b.y);
}
// acc += a*b
__device__ __forceinline__ void cmadd(double2& acc, double2 a, double2 b) {
    acc.x = fma(a.x, b.x, acc.x);
    acc.x = fma(-a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y);
    acc.y = fma(a.y, b.x, acc.y);
}
// acc += conj(a)*b
__device__ __forceinline__ void cmaddc(double2& acc, double2 a, double2 b) {
    acc.x = fma(a.x, b.x, acc.x);
    acc.x = fma(a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y);
    acc.y = fma(-a.y, b.x, acc.y);
}
__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ double2 cconj(double2 a) { return make_double2(a.x, -a.y); }

// h = upper half of (1 + SIGMA*gamma_MU) psi ; psi[3*spin + colour]
template <int MU, int SIGMA>
__device__ __forceinline__ void project(const double2* __restrict__ psi, double2* __restrict__ h) {
    constexpr double s = (double)SIGMA;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        if (MU == 0) {  // r0 = psi0 - i s psi3 ; r1 = psi1 - i s psi2
            h[c] = caddi(psi[c], psi[9 + c], -s);
            h[3 + c] = caddi(psi[3 + c], psi[6 + c], -s);
        } else if (MU == 1) {  // r0 = psi0 - s psi3 ; r1 = psi1 + s psi2
            h[c] = cadds(psi[c], psi[9 + c], -s);
            h[3 + c] = cadds(psi[3 + c], psi[6 + c], s);
        } else if (MU == 2) {  // r0 = psi0 - i s psi2 ; r1 = psi1 + i s psi3
            h[c] = caddi(psi[c], psi[6 + c], -s);
            h[3 + c] = caddi(psi[3 + c], psi[9 + c], s);
        } else {  // r0 = psi0 + s psi2 ; r1 = psi1 + s psi3
            h[c] = cadds(psi[c], psi[6 + c], s);
            h[3 + c] = cadds(psi[3 + c], psi[9 + c], s);
        }
    }
}

// acc += full (1 + SIGMA*gamma_MU)-spinor whose upper half is g (times the real factor ph = +-1)
template <int MU, int SIGMA>
__device__ __forceinline__ void reconstruct_add(double2* __restrict__ acc, const double2* __restrict__ g,
                                                double ph) {
    const double s = (double)SIGMA * ph;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        acc[c] = cadds(acc[c], g[c], ph);
        acc[3 + c] = cadds(acc[3 + c], g[3 + c], ph);
        if (MU == 0) {  // r2 = i s r1 ; r3 = i s r0
            acc[6 + c] = caddi(acc[6 + c], g[3 + c], s);
            acc[9 + c] = caddi(acc[9 + c], g[c], s);
        } else if (MU == 1) {  // r2 = s r1 ; r3 = -s r0
            acc[6 + c] = cadds(acc[6 + c], g[3 + c], s);
            acc[9 + c] = cadds(acc[9 + c], g[c], -s);
        } else if (MU == 2) {  // r2 = i s r0 ; r3 = -i s r1
            acc[6 + c] = caddi(acc[6 + c], g[c], s);
            acc[9 + c] = caddi(acc[9 + c], g[3 + c], -s);
        } else {  // r2 = s r0 ; r3 = s r1
            acc[6 + c] = cadds(acc[6 + c], g[c], s);
            acc[9 + c] = cadds(acc[9 + c], g[3 + c], s);
        }
    }
}

// third row of an SU(3) matrix from the first two: row2 = conj(row0 x row1)
__device__ __forceinline__ void su3_row2(double2* __restrict__ u) {
    u[6] = cconj(csub(cmul(u[1], u[5]), cmul(u[2], u[4])));
    u[7] = cconj(csub(cmul(u[2], u[3]), cmul(u[0], u[5])));
    u[8] = cconj(csub(cmul(u[0], u[4]), cmul(u[1], u[3])));
}

// g = U h (DAG = false) or U^dagger h (DAG = true) on both spin components of a half-spinor
template <bool DAG>
__device__ __forceinline__ void su3_mul(const double2* __restrict__ u, const double2* __restrict__ h,
                                        double2* __restrict__ g) {
#pragma unroll
    for (int sp = 0; sp < 2; sp++) {
#pragma unroll
        for (int a = 0; a < 3; a++) {
            double2 acc = make_double2(0.0, 0.0);
#pragma unroll
            for (int b = 0; b < 3; b++) {
                if (DAG)
                    cmaddc(acc, u[3 * b + a], h[3 * sp + b]);
                else
                    cmadd(acc, u[3 * a + b], h[3 * sp + b]);
            }
            g[3 * sp + a] = acc;
        }
    }
}

}  // namespace ov
