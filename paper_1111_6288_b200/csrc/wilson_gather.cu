// Wilson kernel, variant 1 ("gather"): one thread per lattice site, neighbours read straight from
// global memory through L1/L2.  Works for every lattice shape.
//
//   out = s * G (in - kappa * hop(in)) + a1*A1 + a2*A2 + a3*A3        (Epilogue, ov_internal.h)
//   hop(in)(x) = sum_mu [ s+ (1-gamma_mu) U_mu(x) in(x+mu) + s- (1+gamma_mu) U_mu(x-mu)^+ in(x-mu) ]
//
// Layouts (ov_internal.h: spinor_base / gauge_index; blocked when V % 32 == 0, planes otherwise), NE = 9 link entries
// (recon 18) or 6 (recon 12).  Either way a warp reads 32 consecutive complex values (512 B in fp64: LDG.128; 256 B in fp32: LDG.64) per
// component or link entry, fully coalesced.  The kernel is a template on the complex type: double2 is the product path,
// float2 serves the reduced-precision tail of the adaptive CG.
// Successive launches walk the lattice in opposite block order (GatherArgs::reverse): the spinor one launch wrote last
// is what the next launch reads first, while it is still in the 126 MB L2.
#include "ov_internal.h"
#include "wilson_math.cuh"

namespace ov {

template <typename C>
struct GatherArgs {
    const C* gauge;
    const C* in;
    C* out;
    int X, Y, Z, T;
    long long V;
    double kappa;
    double tphase;         // factor on the hop across the t boundary: -1 antiperiodic, +1 periodic, 0 open
    int field_dir;         // background field (ov_options.field - 1; -1 = none): with 12-real links the rebuilt third row of a
    double field_3qE;      // t link is multiplied by exp(-3 i qE (x_dir - origin)) = det of the U(3) link (phase-tracked recon)
    int field_origin;
    int reverse;
    int nrb;               // rhs groups per site block (batched launch): block id = site_block * nrb + rhs_group
    long long rhs_stride;  // elements between consecutive right-hand sides in in/out/A1..A3
    EpilogueT<C> ep;
};

// fp64: 64-thread blocks at <= 168 registers: 6 blocks = 12 warps per SM.  Measured at 24^3x64 (profiles/): 128 threads
// with no register cap ran at 8 warps/SM and 215 us per apply, this shape at 166 us.
// fp32: half the registers per value: 128-thread blocks at <= 128 registers, 16 warps per SM.
template <typename C> struct GatherShape;
template <> struct GatherShape<double2> { static constexpr int threads = 64, min_blocks = 6; };
template <> struct GatherShape<float2> { static constexpr int threads = 128, min_blocks = 4; };

template <int RECON, bool BL, typename C>
__device__ __forceinline__ void load_link(const C* __restrict__ gauge, long long V, int mu, long long site,
                                          C* __restrict__ u) {
    constexpr int NE = RECON / 2;
    const C* p = gauge + gauge_index<NE, BL>(V, mu, 0, site);
    const long long es = BL ? 32 : V;  // stride between entries
#pragma unroll
    for (int e = 0; e < NE; e++) u[e] = __ldg(p + (long long)e * es);
    if (RECON == 12) su3_row2(u);
}
// 12-real links that carry a U(1) phase (background field): rows 0-1 are stored with the phase, so conj(row0 x row1) is
// the true third row times conj(det U) -- multiply it by det U = w
template <typename C>
__device__ __forceinline__ void row2_phase(C* __restrict__ u, C w) {
#pragma unroll
    for (int e = 6; e < 9; e++) u[e] = cmul(u[e], w);
}

template <int MU, int SIGMA, int RECON, bool BL, typename C>
__device__ __forceinline__ void hop(C* __restrict__ acc, const GatherArgs<C>& a, long long nsite, long long lsite,
                                    real_t<C> ph, const C* det = nullptr) {
    C psi[12], h[6], g[6], u[9];
    const C* pn = a.in + spinor_base<BL>(nsite);
    const long long cs = spinor_stride<BL>(a.V);
#pragma unroll
    for (int c = 0; c < 12; c++) psi[c] = __ldg(pn + c * cs);
    project<MU, SIGMA>(psi, h);
    load_link<RECON, BL>(a.gauge, a.V, MU, lsite, u);
    if (RECON == 12 && MU == 3 && det) row2_phase(u, *det);
    su3_mul<(SIGMA > 0)>(u, h, g);
    reconstruct_add<MU, SIGMA>(acc, g, ph);
}

// NA: number of epilogue operands A1..A_NA (always filled in order); NA = -1: hop only.
// RB: right-hand sides per block (threadIdx.y).  A batched launch puts the rhs groups of one site block on adjacent
// block ids, so they run at the same time: the links are read from HBM once per site block, from L2 by the other
// groups, and from L1 by the second rhs of a block.
template <typename C, int RECON, int NA, bool BL, int RB>
__global__ void __launch_bounds__(GatherShape<C>::threads * RB, GatherShape<C>::min_blocks / RB)
wilson_gather_kernel(GatherArgs<C> a) {
    using R = real_t<C>;
    const unsigned lin = a.reverse ? gridDim.x - 1 - blockIdx.x : blockIdx.x;
    const unsigned blk = lin / a.nrb;
    {
        const long long off = ((long long)(lin % a.nrb) * RB + threadIdx.y) * a.rhs_stride;
        a.in += off; a.out += off;
        if (NA >= 1) a.ep.A1 += off;
        if (NA >= 2) a.ep.A2 += off;
        if (NA >= 3) a.ep.A3 += off;
    }
    const long long i = (long long)blk * blockDim.x + threadIdx.x;
    if (i >= a.V) return;
    long long r = i;
    const int x = (int)(r % a.X); r /= a.X;
    const int y = (int)(r % a.Y); r /= a.Y;
    const int z = (int)(r % a.Z);
    const int t = (int)(r / a.Z);
    const long long sX = 1, sY = a.X, sZ = (long long)a.X * a.Y, sT = (long long)a.X * a.Y * a.Z;

    // out = s G (in - kappa hop) = (-kappa s) G (hop - in/kappa): the site's own spinor goes into the accumulator FIRST, so
    // the +-x hops that follow find its cache lines in L1 instead of the epilogue re-reading them from L2 at the very end
    // (-192 B/site through the SM's L2 port, 2.5-3 % of the launch).
    const long long ib = spinor_base<BL>(i), cs = spinor_stride<BL>(a.V);
    C acc[12];
    if (NA < 0) {
#pragma unroll
        for (int c = 0; c < 12; c++) acc[c] = cmake<C>(0, 0);
    } else {
        const R mik = (R)(-1.0 / a.kappa);
#pragma unroll
        for (int c = 0; c < 12; c++) { const C o = __ldg(a.in + ib + c * cs); acc[c] = cmake<C>(mik * o.x, mik * o.y); }
    }

    {
        const long long ip = (x + 1 == a.X) ? i - (a.X - 1) * sX : i + sX;
        const long long im = (x == 0) ? i + (a.X - 1) * sX : i - sX;
        hop<0, -1, RECON, BL>(acc, a, ip, i, (R)1);
        hop<0, +1, RECON, BL>(acc, a, im, im, (R)1);
    }
    {
        const long long ip = (y + 1 == a.Y) ? i - (a.Y - 1) * sY : i + sY;
        const long long im = (y == 0) ? i + (a.Y - 1) * sY : i - sY;
        hop<1, -1, RECON, BL>(acc, a, ip, i, (R)1);
        hop<1, +1, RECON, BL>(acc, a, im, im, (R)1);
    }
    {
        const long long ip = (z + 1 == a.Z) ? i - (a.Z - 1) * sZ : i + sZ;
        const long long im = (z == 0) ? i + (a.Z - 1) * sZ : i - sZ;
        hop<2, -1, RECON, BL>(acc, a, ip, i, (R)1);
        hop<2, +1, RECON, BL>(acc, a, im, im, (R)1);
    }
    {
        const bool wp = (t + 1 == a.T), wm = (t == 0);
        const long long ip = wp ? i - (a.T - 1) * sT : i + sT;
        const long long im = wm ? i + (a.T - 1) * sT : i - sT;
        C det = cmake<C>(1, 0);   // det of this site's t links (they depend on the space coordinates only)
        const bool field = RECON == 12 && a.field_dir >= 0;
        if (field) {
            const int xd = a.field_dir == 0 ? x : a.field_dir == 1 ? y : z;
            double sn, cs;
            sincos(-a.field_3qE * (double)(xd - a.field_origin), &sn, &cs);
            det = cmake<C>((R)cs, (R)sn);
        }
        hop<3, -1, RECON, BL>(acc, a, ip, i, wp ? (R)a.tphase : (R)1, field ? &det : nullptr);  // boundary in time
        hop<3, +1, RECON, BL>(acc, a, im, im, wm ? (R)a.tphase : (R)1, field ? &det : nullptr);
    }

    const EpilogueT<C>& ep = a.ep;
    if (NA < 0) {
#pragma unroll
        for (int c = 0; c < 12; c++) a.out[ib + c * cs] = acc[c];
        return;
    }
    const R s_up = (R)(-a.kappa * ep.s), s_lo = (R)(ep.g5 ? a.kappa * ep.s : -a.kappa * ep.s);
    // `out` may alias an operand (the Clenshaw step writes b_j over b_{j+2}), so the compiler must keep every operand
    // load behind the previous store: done component by component that is 12 dependent memory round trips.  Load a
    // chunk of components of every operand first (all loads in flight at once), then combine and store the chunk.
    constexpr int CH = 4;
#pragma unroll
    for (int c0 = 0; c0 < 12; c0 += CH) {
        C w1[CH], w2[CH], w3[CH];
#pragma unroll
        for (int k = 0; k < CH; k++) {
            const long long e = ib + (c0 + k) * cs;
            if (NA >= 1) w1[k] = ep.A1[e];
            if (NA >= 2) w2[k] = ep.A2[e];
            if (NA >= 3) w3[k] = ep.A3[e];
        }
#pragma unroll
        for (int k = 0; k < CH; k++) {
            const int c = c0 + k;
            const bool lo = (c >= 6);
            const R sc = lo ? s_lo : s_up;
            C v = cmake<C>(sc * acc[c].x, sc * acc[c].y);
            if (NA >= 1) { const R f = (R)((lo && (ep.a_g5 & 1)) ? -ep.a1 : ep.a1); v.x = fma(f, w1[k].x, v.x); v.y = fma(f, w1[k].y, v.y); }
            if (NA >= 2) { const R f = (R)((lo && (ep.a_g5 & 2)) ? -ep.a2 : ep.a2); v.x = fma(f, w2[k].x, v.x); v.y = fma(f, w2[k].y, v.y); }
            if (NA >= 3) { const R f = (R)((lo && (ep.a_g5 & 4)) ? -ep.a3 : ep.a3); v.x = fma(f, w3[k].x, v.x); v.y = fma(f, w3[k].y, v.y); }
            a.out[ib + c * cs] = v;
        }
    }
}

// nrhs right-hand sides, `stride` elements apart (in, out and every epilogue operand alike)
template <typename C>
static int launch_gather_t(ov_ctx* ctx, const C* gauge, const C* in, C* out, const EpilogueT<C>& ep, int nrhs = 1,
                           long long stride = 0) {
    if (nrhs > 1 && (nrhs & 1)) {   // odd batch: pairs first, then the last one alone
        OV_TRY(launch_gather_t<C>(ctx, gauge, in, out, ep, nrhs - 1, stride));
        EpilogueT<C> e1 = ep;
        const long long off = (long long)(nrhs - 1) * stride;
        if (e1.A1) e1.A1 += off;
        if (e1.A2) e1.A2 += off;
        if (e1.A3) e1.A3 += off;
        return launch_gather_t<C>(ctx, gauge, in + off, out + off, e1, 1, 0);
    }
    const int rb = nrhs > 1 ? 2 : 1;
    GatherArgs<C> a;
    a.nrb = nrhs / rb;
    a.rhs_stride = stride;
    a.gauge = gauge;
    a.in = in;
    a.out = out;
    a.X = ctx->lat.X; a.Y = ctx->lat.Y; a.Z = ctx->lat.Z; a.T = ctx->lat.T;
    a.V = ctx->lat.V;
    a.kappa = ctx->kappa;
    a.tphase = ctx->t_phase;
    a.field_dir = ctx->field_dir;
    a.field_3qE = 3.0 * ctx->field_qE;
    a.field_origin = ctx->field_origin;
    a.ep = ep;
    a.reverse = ctx->flip;
    ctx->flip ^= 1;
    const int threads = GatherShape<C>::threads;
    const long long nblocks = ((a.V + threads - 1) / threads) * (long long)a.nrb;
    if (nblocks > 0x7fffffffLL) return fail(ctx, OV_EINVAL, "too many right-hand sides for one launch (%lld blocks)", nblocks);
    const unsigned blocks = (unsigned)nblocks;
    const dim3 bdim(threads, rb);
    const int na = ep.hop_only ? -1 : (ep.A3 ? 3 : ep.A2 ? 2 : ep.A1 ? 1 : 0);
    if ((ep.A3 && !ep.A2) || (ep.A2 && !ep.A1)) return fail(ctx, OV_EINVAL, "epilogue operands must be filled in order");
#define OV_GATHER_B(R, N, B)                                                                             \
    do {                                                                                                 \
        if (ctx->blocked) wilson_gather_kernel<C, R, N, true, B><<<blocks, bdim, 0, ctx->stream>>>(a);   \
        else wilson_gather_kernel<C, R, N, false, B><<<blocks, bdim, 0, ctx->stream>>>(a);               \
    } while (0)
#define OV_GATHER(R, N)                                        \
    do {                                                       \
        if (rb == 2) OV_GATHER_B(R, N, 2); else OV_GATHER_B(R, N, 1); \
    } while (0)
#define OV_GATHER_NA(R)                                 \
    switch (na) {                                       \
        case -1: OV_GATHER(R, -1); break;               \
        case 0: OV_GATHER(R, 0); break;                 \
        case 1: OV_GATHER(R, 1); break;                 \
        case 2: OV_GATHER(R, 2); break;                 \
        default: OV_GATHER(R, 3); break;                \
    }
    if (ctx->recon == 12) { OV_GATHER_NA(12) } else { OV_GATHER_NA(18) }
#undef OV_GATHER_NA
#undef OV_GATHER
#undef OV_GATHER_B
    ctx->launches++;
    OV_CUDA(ctx, cudaGetLastError());
    return OV_OK;
}

int launch_wilson_gather(ov_ctx* ctx, const double2* in, double2* out, const Epilogue& ep) {
    return launch_gather_t<double2>(ctx, ctx->gauge, in, out, ep);
}
int launch_wilson_batch(ov_ctx* ctx, const double2* in, double2* out, const Epilogue& ep, int nrhs) {
    if (nrhs == 1) return launch_wilson(ctx, in, out, ep);   // single right-hand side: the context's kernel choice
    return launch_gather_t<double2>(ctx, ctx->gauge, in, out, ep, nrhs, (long long)spinor_elems(ctx));
}
int launch_wilson_gather_f32(ov_ctx* ctx, const float2* in, float2* out, const EpilogueF& ep) {
    if (!ctx->gauge_f) return fail(ctx, OV_ESTATE, "fp32 links have not been made");
    return launch_gather_t<float2>(ctx, ctx->gauge_f, in, out, ep);
}

}  // namespace ov
