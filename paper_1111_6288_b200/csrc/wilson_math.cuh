// Device-side arithmetic of the Wilson hopping term for the chiral gamma basis of include/ov.h
// (reading G2).  All four gamma_mu are block-off-diagonal, so (1 + sigma*gamma_mu) psi has rank
// 2: its upper two spin components h = (r0, r1) determine the lower two.  A hop therefore costs one
// projection to a half-spinor (6 complex), one SU(3) mat-vec on 2 spin components, and one
// reconstruct-accumulate.  sigma = -1 for the forward hop (1 - gamma_mu), +1 for the backward hop.
#pragma once
#include <cuda_runtime.h>

namespace ov {

// complex types: double2 (the product path, fp64) and float2 (the reduced-precision tail of the adaptive CG)
template <typename C> struct real_of;
template <> struct real_of<double2> { using type = double; };
template <> struct real_of<float2> { using type = float; };
template <typename C> using real_t = typename real_of<C>::type;
template <typename C> __device__ __forceinline__ C cmake(real_t<C> x, real_t<C> y) { C c; c.x = x; c.y = y; return c; }

template <typename C> __device__ __forceinline__ C cadd(C a, C b) { return cmake<C>(a.x + b.x, a.y + b.y); }
template <typename C> __device__ __forceinline__ C csub(C a, C b) { return cmake<C>(a.x - b.x, a.y - b.y); }
// a + i*s*b
template <typename C> __device__ __forceinline__ C caddi(C a, C b, real_t<C> s) { return cmake<C>(a.x - s * b.y, a.y + s * b.x); }
// a + s*b (s real)
template <typename C> __device__ __forceinline__ C cadds(C a, C b, real_t<C> s) { return cmake<C>(a.x + s * b.x, a.y + s * b.y); }
// acc += a*b
template <typename C> __device__ __forceinline__ void cmadd(C& acc, C a, C b) {
    acc.x = fma(a.x, b.x, acc.x);
    acc.x = fma(-a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y);
    acc.y = fma(a.y, b.x, acc.y);
}
// acc += conj(a)*b
template <typename C> __device__ __forceinline__ void cmaddc(C& acc, C a, C b) {
    acc.x = fma(a.x, b.x, acc.x);
    acc.x = fma(a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y);
    acc.y = fma(-a.y, b.x, acc.y);
}
template <typename C> __device__ __forceinline__ C cmul(C a, C b) { return cmake<C>(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
template <typename C> __device__ __forceinline__ C cconj(C a) { return cmake<C>(a.x, -a.y); }

// h = upper half of (1 + SIGMA*gamma_MU) psi ; psi[3*spin + colour]
template <int MU, int SIGMA, typename C>
__device__ __forceinline__ void project(const C* __restrict__ psi, C* __restrict__ h) {
    constexpr real_t<C> s = (real_t<C>)SIGMA;
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
template <int MU, int SIGMA, typename C>
__device__ __forceinline__ void reconstruct_add(C* __restrict__ acc, const C* __restrict__ g, real_t<C> ph) {
    const real_t<C> s = (real_t<C>)SIGMA * ph;
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
template <typename C>
__device__ __forceinline__ void su3_row2(C* __restrict__ u) {
    u[6] = cconj(csub(cmul(u[1], u[5]), cmul(u[2], u[4])));
    u[7] = cconj(csub(cmul(u[2], u[3]), cmul(u[0], u[5])));
    u[8] = cconj(csub(cmul(u[0], u[4]), cmul(u[1], u[3])));
}

// g = U h (DAG = false) or U^dagger h (DAG = true) on both spin components of a half-spinor
template <bool DAG, typename C>
__device__ __forceinline__ void su3_mul(const C* __restrict__ u, const C* __restrict__ h, C* __restrict__ g) {
#pragma unroll
    for (int sp = 0; sp < 2; sp++) {
#pragma unroll
        for (int a = 0; a < 3; a++) {
            C acc = cmake<C>(0, 0);
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
