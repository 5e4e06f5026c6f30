// Wilson kernel, variant 1 ("gather"): one thread per lattice site, neighbours read straight from
// global memory through L1/L2.  Works for every lattice shape; it is
// the general-shape path and the baseline the tiled kernel (wilson_tiled.cu) is measured against.
//
//   out = s * G (in - kappa * hop(in)) + a1*A1 + a2*A2 + a3*A3        (Epilogue, ov_internal.h)
//   hop(in)(x) = sum_mu [ s+ (1-gamma_mu) U_mu(x) in(x+mu) + s- (1+gamma_mu) U_mu(x-mu)^+ in(x-mu) ]
//
// Layouts: spinor component c of site i at double2 index c*V + i; link entry e (row-major) of U_mu(i) at
// ((mu*NE)+e)*V + i with NE = 9 (recon 18) or 6 (recon 12).  A warp therefore reads 32 consecutive
// double2 (512 B) per component: fully coalesced LDG.128.
#include "ov_internal.h"
#include "wilson_math.cuh"

namespace ov {

struct GatherArgs {
    const double2* gauge;
    const double2* in;
    double2* out;
    int X, Y, Z, T;
    long long V;
    double kappa;
    Epilogue ep;
};

template <int RECON>
__device__ __forceinline__ void load_link(const double2* __restrict__ gauge, long long V, int mu,
                                          long long site, double2* __restrict__ u) {
    constexpr int NE = RECON / 2;
    const double2* p = gauge + ((long long)mu * NE) * V + site;
#pragma unroll
    for (int e = 0; e < NE; e++) u[e] = __ldg(p + (long long)e * V);
    if (RECON == 12) su3_row2(u);
}

template <int MU, int SIGMA, int RECON>
__device__ __forceinline__ void hop(double2* __restrict__ acc, const GatherArgs& a, long long nsite,
                                    long long lsite, double ph) {
    double2 psi[12], h[6], g[6], u[9];
#pragma unroll
    for (int c = 0; c < 12; c++) psi[c] = __ldg(a.in + (long long)c * a.V + nsite);
    project<MU, SIGMA>(psi, h);
    load_link<RECON>(a.gauge, a.V, MU, lsite, u);
    su3_mul<(SIGMA > 0)>(u, h, g);
    reconstruct_add<MU, SIGMA>(acc, g, ph);
}

template <int RECON>
__global__ void __launch_bounds__(128) wilson_gather_kernel(const GatherArgs a) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.V) return;
    long long r = i;
    const int x = (int)(r % a.X); r /= a.X;
    const int y = (int)(r % a.Y); r /= a.Y;
    const int z = (int)(r % a.Z);
    const int t = (int)(r / a.Z);
    const long long sX = 1, sY = a.X, sZ = (long long)a.X * a.Y, sT = (long long)a.X * a.Y * a.Z;

    double2 acc[12];
#pragma unroll
    for (int c = 0; c < 12; c++) acc[c] = make_double2(0.0, 0.0);

    {
        const long long ip = (x + 1 == a.X) ? i - (a.X - 1) * sX : i + sX;
        const long long im = (x == 0) ? i + (a.X - 1) * sX : i - sX;
        hop<0, -1, RECON>(acc, a, ip, i, 1.0);
        hop<0, +1, RECON>(acc, a, im, im, 1.0);
    }
    {
        const long long ip = (y + 1 == a.Y) ? i - (a.Y - 1) * sY : i + sY;
        const long long im = (y == 0) ? i + (a.Y - 1) * sY : i - sY;
        hop<1, -1, RECON>(acc, a, ip, i, 1.0);
        hop<1, +1, RECON>(acc, a, im, im, 1.0);
    }
    {
        const long long ip = (z + 1 == a.Z) ? i - (a.Z - 1) * sZ : i + sZ;
        const long long im = (z == 0) ? i + (a.Z - 1) * sZ : i - sZ;
        hop<2, -1, RECON>(acc, a, ip, i, 1.0);
        hop<2, +1, RECON>(acc, a, im, im, 1.0);
    }
    {
        const bool wp = (t + 1 == a.T), wm = (t == 0);
        const long long ip = wp ? i - (a.T - 1) * sT : i + sT;
        const long long im = wm ? i + (a.T - 1) * sT : i - sT;
        hop<3, -1, RECON>(acc, a, ip, i, wp ? -1.0 : 1.0);  // antiperiodic in time
        hop<3, +1, RECON>(acc, a, im, im, wm ? -1.0 : 1.0);
    }

    const Epilogue& ep = a.ep;
    if (ep.hop_only) {
#pragma unroll
        for (int c = 0; c < 12; c++) a.out[(long long)c * a.V + i] = acc[c];
        return;
    }
    const double slo = ep.g5 ? -ep.s : ep.s;
#pragma unroll
    for (int c = 0; c < 12; c++) {
        const double sc = (c < 6) ? ep.s : slo;
        const double2 own = __ldg(a.in + (long long)c * a.V + i);
        double2 v = make_double2(sc * fma(-a.kappa, acc[c].x, own.x), sc * fma(-a.kappa, acc[c].y, own.y));
        const bool lo = (c >= 6);
        if (ep.A1) { const double2 w = ep.A1[(long long)c * a.V + i]; const double f = (lo && (ep.a_g5 & 1)) ? -ep.a1 : ep.a1; v.x = fma(f, w.x, v.x); v.y = fma(f, w.y, v.y); }
        if (ep.A2) { const double2 w = ep.A2[(long long)c * a.V + i]; const double f = (lo && (ep.a_g5 & 2)) ? -ep.a2 : ep.a2; v.x = fma(f, w.x, v.x); v.y = fma(f, w.y, v.y); }
        if (ep.A3) { const double2 w = ep.A3[(long long)c * a.V + i]; const double f = (lo && (ep.a_g5 & 4)) ? -ep.a3 : ep.a3; v.x = fma(f, w.x, v.x); v.y = fma(f, w.y, v.y); }
        a.out[(long long)c * a.V + i] = v;
    }
}

int launch_wilson_gather(ov_ctx* ctx, const double2* in, double2* out, const Epilogue& ep) {
    GatherArgs a;
    a.gauge = ctx->gauge;
    a.in = in;
    a.out = out;
    a.X = ctx->lat.X; a.Y = ctx->lat.Y; a.Z = ctx->lat.Z; a.T = ctx->lat.T;
    a.V = ctx->lat.V;
    a.kappa = ctx->kappa;
    a.ep = ep;
    const int threads = 128;
    const unsigned blocks = (unsigned)((a.V + threads - 1) / threads);
    if (ctx->recon == 12)
        wilson_gather_kernel<12><<<blocks, threads, 0, ctx->stream>>>(a);
    else
        wilson_gather_kernel<18><<<blocks, threads, 0, ctx->stream>>>(a);
    ctx->launches++;
    OV_CUDA(ctx, cudaGetLastError());
    return OV_OK;
}

}  // namespace ov
