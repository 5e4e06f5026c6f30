// Wilson kernel, variant 2 ("TMA-staged"): a persistent, warp-specialised kernel for sm_100a (
// PAPER.md:31, :69 "approximately 70 % of the overlap calculation is spent in the dslash routine").
//
//   out = s * G (in - kappa * hop(in)) + a1*A1 + a2*A2 + a3*A3          (Epilogue, ov_internal.h)
//
// Why: the gather kernel (variant 1) pulls 2.2-2.3 kB/site through the SM's L2 port for 960 B/site of HBM traffic and
// sits at the L2 throughput cap.  Here every operand reaches the SM exactly once per tile through the TMA unit:
//   * the lattice is cut into pencils of 8 x 4 x 4 sites in (x,y,z); one CTA marches a pencil along t, one time slice
//     (128 sites) per step;
//   * ONE producer thread issues cp.async.bulk.tensor (5-D boxes over the planes layout [comp][t][z][y][x]) into
//     shared memory: a ring of three interior spinor planes (t, t+1 and one in flight) and one DEDICATED slot per
//     object of a slice -- the x / y / z halo faces (one-site-thick boxes; wrapped coordinates are separate boxes by
//     construction) and the link chunks of the four directions (+ the one-site-thick face of backward links).  Every slot
//     has an mbarrier full/empty pair; the producer polls the empty barriers (test_wait) and refills whichever slot was
//     released first, so no issue order has to be guessed;
//   * EIGHT consumer warps in two groups share the staged data, one site per thread in each group:
//       group A (warps 0-3): own-site term, x and y hops  ->  partial accumulator handed over through shared memory;
//       group B (warps 4-7): starts from A's partial, z and t hops, epilogue, coalesced 16-byte stores.
//     A runs about one slice ahead of B; each object is in use for less than half a slice time and is refilled during the
//     rest, which is why single slots suffice.  The forward t neighbour is the next interior plane (it later becomes the
//     own plane); the backward t hop U_t(x-t)^+ (1+gamma_t) psi(x-t) is carried in B's registers from the previous step.
//     The additions happen in the same order as in the gather kernel, so the two kernels agree to the last bit except
//     where the compiler contracts an FMA differently.
//   * epilogue operands are read by group B from global memory at the output site; the producer prefetches their boxes
//     into L2 (cp.async.bulk.prefetch.tensor) two slices ahead.
// L2->SM traffic per site: 192 (own) + 240 (halo) + 576 (links) + 72 (halo links) = 1080 B instead of ~2200.
//
// Needs the planes layout and X % 8 == 0, Y % 4 == 0, Z % 4 == 0; other shapes use the gather kernel.
#include <cuda.h>

#include <unordered_map>

#include "ov_internal.h"
#include "wilson_math.cuh"

namespace ov {

namespace tma {

constexpr int BX = 8, BY = 4, BZ = 4;           // tile of one time slice
constexpr int SITES = BX * BY * BZ;             // 128 = 4 warps per consumer group
constexpr int NGRP = SITES / 32;                // warps per consumer group
constexpr int NCONS = 2 * NGRP;                 // consumer warps (groups A and B)
constexpr int THREADS = (NCONS + 4) * 32;       // + the producer's warpgroup (one warp issues, three exit at once): three
                                                // aligned warpgroups, so that setmaxnreg can move registers to the consumers
constexpr int REG_CONSUMER = 232, REG_PRODUCER = 40;   // 128 * (2 * 232 + 40) = 64512 <= 65536
constexpr int SI = 3;                           // interior planes in the ring
constexpr int I_BYTES = SITES * 12 * 16;        // 24576
constexpr int FX = BY * BZ, FY = BX * BZ, FZ = BX * BY;   // face sites: 16, 32, 32
constexpr int HX_BYTES = 2 * 12 * FX * 16, HY_BYTES = 2 * 12 * FY * 16, HZ_BYTES = 2 * 12 * FZ * 16;   // minus face, plus face
constexpr int P_BYTES = SITES * 12 * 16;        // group A's partial accumulators
template <int NE> struct LBytes {               // link chunk = the tile's links of one direction + the face of backward links
    static constexpr int x = (SITES + FX) * NE * 16, y = (SITES + FY) * NE * 16, z = (SITES + FZ) * NE * 16, t = SITES * NE * 16;
};
// single-slot objects and their barrier index (full at 2*o, empty at 2*o + 1 after the interior ring's barriers)
enum Obj { HX = 0, HY, HZ, LX, LY, LZ, LT, NOBJ };
constexpr int NBAR = 2 * SI + 2 * NOBJ + 2 * NGRP;
template <int NE> constexpr size_t smem_bytes() {
    return (size_t)SI * I_BYTES + HX_BYTES + HY_BYTES + HZ_BYTES + LBytes<NE>::x + LBytes<NE>::y + LBytes<NE>::z + LBytes<NE>::t +
           P_BYTES + 8 * NBAR;
}

struct Maps {               // tensor maps of one spinor array or of the gauge field (box shapes differ)
    CUtensorMap main, fx, fy, fz;
};

struct Args {
    Maps in;                // spinor: 5-D (2X, Y, Z, T, 12) doubles
    Maps gauge;             // links:  5-D (2X, Y, Z, T, 4*NE) doubles
    CUtensorMap op[3];      // main-box maps of the epilogue operands (L2 prefetch only)
    double2* out;
    const double2* A1;
    const double2* A2;
    const double2* A3;
    double a1, a2, a3;
    int a_g5;
    int X, Y, Z, T;
    long long V;
    double kappa, s;
    int g5;
    int ntx, nty, ntz;      // tiles per direction
    int Lt;                 // slices per work item
    int nitems;
    int reverse;
    double tphase;          // factor on the hop across the t boundary: -1 antiperiodic, +1 periodic, 0 open
};

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ bool mbar_test(unsigned bar, unsigned parity) {
    unsigned ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void tma_load_5d(unsigned dst, const CUtensorMap* map, unsigned bar, int c0, int c1, int c2,
                                            int c3, int c4) {
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4) : "memory");
}
__device__ __forceinline__ void tma_prefetch_5d(const CUtensorMap* map, int c0, int c1, int c2, int c3, int c4) {
    asm volatile("cp.async.bulk.prefetch.tensor.5d.L2.global.tile [%0, {%1, %2, %3, %4, %5}];"
                 ::"l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4) : "memory");
}

struct Item {
    int x0, y0, z0, t0;
};
__device__ __forceinline__ Item decode_item(const Args& a, int it) {
    if (a.reverse) it = a.nitems - 1 - it;
    const int npen = a.ntx * a.nty * a.ntz;
    const int seg = it / npen, pen = it % npen;
    Item r;
    r.x0 = (pen % a.ntx) * BX;
    r.y0 = ((pen / a.ntx) % a.nty) * BY;
    r.z0 = (pen / (a.ntx * a.nty)) * BZ;
    r.t0 = seg * a.Lt;
    return r;
}

// 12 components of one spinor from shared memory: element c at p[c * stride]
__device__ __forceinline__ void lds_spinor(const double2* p, int stride, double2* psi) {
#pragma unroll
    for (int c = 0; c < 12; c++) psi[c] = p[c * stride];
}
template <int RECON>
__device__ __forceinline__ void lds_link(const double2* p, int stride, double2* u) {
    constexpr int NE = RECON / 2;
#pragma unroll
    for (int e = 0; e < NE; e++) u[e] = p[e * stride];
    if (RECON == 12) su3_row2(u);
}

template <int MU, int SIGMA, int RECON>
__device__ __forceinline__ void hop_smem(double2* acc, const double2* pn, int ns, const double2* pl, int ls, double ph) {
    double2 psi[12], h[6], g[6], u[9];
    lds_spinor(pn, ns, psi);
    project<MU, SIGMA>(psi, h);
    lds_link<RECON>(pl, ls, u);
    su3_mul<(SIGMA > 0)>(u, h, g);
    reconstruct_add<MU, SIGMA>(acc, g, ph);
}

// the fill sequence of one staged object as the producer sees it: fill number f belongs to the CTA's j-th work item and
// is the u-th of that item's `per` fills
struct Seq {
    int j = 0, u = 0, per = 0, nitem = 0;
    unsigned f = 0;
    __device__ __forceinline__ bool done() const { return j >= nitem; }
    __device__ __forceinline__ void next() { f++; if (++u == per) { u = 0; j++; } }
};

}  // namespace tma

using namespace tma;

// NA: -1 hop only, 0..3 epilogue operands (read from global memory at the output site)
template <int RECON, int NA>
__global__ void __launch_bounds__(THREADS, 1) wilson_tma_kernel(const __grid_constant__ Args a) {
    constexpr int NE = RECON / 2;
    using LB = LBytes<NE>;
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char* sI = smem;
    unsigned char* sHX = sI + SI * I_BYTES;
    unsigned char* sHY = sHX + HX_BYTES;
    unsigned char* sHZ = sHY + HY_BYTES;
    unsigned char* sLX = sHZ + HZ_BYTES;
    unsigned char* sLY = sLX + LB::x;
    unsigned char* sLZ = sLY + LB::y;
    unsigned char* sLT = sLZ + LB::z;
    unsigned char* sP = sLT + LB::t;
    unsigned long long* bars = (unsigned long long*)(sP + P_BYTES);
    const unsigned bar0 = smem_u32(bars);
    auto fullI = [&](unsigned s) { return bar0 + 8u * s; };
    auto emptyI = [&](unsigned s) { return bar0 + 8u * (SI + s); };
    auto fullO = [&](int o) { return bar0 + 8u * (2 * SI + 2 * o); };
    auto emptyO = [&](int o) { return bar0 + 8u * (2 * SI + 2 * o + 1); };
    auto partFull = [&](int w) { return bar0 + 8u * (2 * SI + 2 * NOBJ + w); };
    auto partEmpty = [&](int w) { return bar0 + 8u * (2 * SI + 2 * NOBJ + NGRP + w); };

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (unsigned s = 0; s < SI; s++) { mbar_init(fullI(s), 1); mbar_init(emptyI(s), NCONS); }
        for (int o = 0; o < NOBJ; o++) { mbar_init(fullO(o), 1); mbar_init(emptyO(o), NGRP); }
        for (int w = 0; w < NGRP; w++) { mbar_init(partFull(w), 1); mbar_init(partEmpty(w), 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int my_items = (a.nitems - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;

    if (warp >= NCONS) {
        // =============================================================== producer: one thread issues every TMA load
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(REG_PRODUCER));
        if (warp != NCONS || lane != 0) return;
        Seq qI, q[NOBJ];
        qI.per = a.Lt + 2; qI.nitem = my_items;                 // planes t0-1, t0 .. t0+Lt-1, t0+Lt
        for (int o = 0; o < NOBJ; o++) { q[o].per = (o == LT) ? a.Lt + 1 : a.Lt; q[o].nitem = my_items; }   // LT: + the slice below
        auto item_of = [&](int j) { return decode_item(a, (int)blockIdx.x + j * (int)gridDim.x); };
        auto wrap = [&](int t) { return t < 0 ? t + a.T : (t >= a.T ? t - a.T : t); };
        int remaining = 1 + NOBJ;
        while (remaining > 0) {
            bool progress = false;
            remaining = 0;
            if (!qI.done()) {
                remaining++;
                const unsigned s = qI.f % SI;
                if (mbar_test(emptyI(s), ((qI.f / SI) & 1u) ^ 1u)) {
                    const Item w = item_of(qI.j);
                    const int t = wrap(w.t0 - 1 + qI.u);
                    mbar_expect_tx(fullI(s), I_BYTES);
                    tma_load_5d(smem_u32(sI + s * I_BYTES), &a.in.main, fullI(s), 2 * w.x0, w.y0, w.z0, t, 0);
                    if (NA >= 1 && qI.u >= 1 && qI.u <= a.Lt) {   // an own plane: pull its epilogue operands into L2
                        tma_prefetch_5d(&a.op[0], 2 * w.x0, w.y0, w.z0, t, 0);
                        if (NA >= 2) tma_prefetch_5d(&a.op[1], 2 * w.x0, w.y0, w.z0, t, 0);
                        if (NA >= 3) tma_prefetch_5d(&a.op[2], 2 * w.x0, w.y0, w.z0, t, 0);
                    }
                    qI.next();
                    progress = true;
                }
            }
#pragma unroll
            for (int o = 0; o < NOBJ; o++) {
                if (q[o].done()) continue;
                remaining++;
                if (!mbar_test(emptyO(o), (q[o].f & 1u) ^ 1u)) continue;
                const Item w = item_of(q[o].j);
                const unsigned fb = fullO(o);
                const int xm = (w.x0 == 0) ? a.X - 1 : w.x0 - 1, xp = (w.x0 + BX == a.X) ? 0 : w.x0 + BX;
                const int ym = (w.y0 == 0) ? a.Y - 1 : w.y0 - 1, yp = (w.y0 + BY == a.Y) ? 0 : w.y0 + BY;
                const int zm = (w.z0 == 0) ? a.Z - 1 : w.z0 - 1, zp = (w.z0 + BZ == a.Z) ? 0 : w.z0 + BZ;
                const int t = (o == LT) ? wrap(w.t0 - 1 + q[o].u) : w.t0 + q[o].u;
                if (o == HX) {
                    mbar_expect_tx(fb, HX_BYTES);
                    tma_load_5d(smem_u32(sHX), &a.in.fx, fb, 2 * xm, w.y0, w.z0, t, 0);
                    tma_load_5d(smem_u32(sHX) + HX_BYTES / 2, &a.in.fx, fb, 2 * xp, w.y0, w.z0, t, 0);
                } else if (o == HY) {
                    mbar_expect_tx(fb, HY_BYTES);
                    tma_load_5d(smem_u32(sHY), &a.in.fy, fb, 2 * w.x0, ym, w.z0, t, 0);
                    tma_load_5d(smem_u32(sHY) + HY_BYTES / 2, &a.in.fy, fb, 2 * w.x0, yp, w.z0, t, 0);
                } else if (o == HZ) {
                    mbar_expect_tx(fb, HZ_BYTES);
                    tma_load_5d(smem_u32(sHZ), &a.in.fz, fb, 2 * w.x0, w.y0, zm, t, 0);
                    tma_load_5d(smem_u32(sHZ) + HZ_BYTES / 2, &a.in.fz, fb, 2 * w.x0, w.y0, zp, t, 0);
                } else if (o == LX) {
                    mbar_expect_tx(fb, LB::x);
                    tma_load_5d(smem_u32(sLX), &a.gauge.main, fb, 2 * w.x0, w.y0, w.z0, t, 0 * NE);
                    tma_load_5d(smem_u32(sLX) + SITES * NE * 16, &a.gauge.fx, fb, 2 * xm, w.y0, w.z0, t, 0 * NE);
                } else if (o == LY) {
                    mbar_expect_tx(fb, LB::y);
                    tma_load_5d(smem_u32(sLY), &a.gauge.main, fb, 2 * w.x0, w.y0, w.z0, t, 1 * NE);
                    tma_load_5d(smem_u32(sLY) + SITES * NE * 16, &a.gauge.fy, fb, 2 * w.x0, ym, w.z0, t, 1 * NE);
                } else if (o == LZ) {
                    mbar_expect_tx(fb, LB::z);
                    tma_load_5d(smem_u32(sLZ), &a.gauge.main, fb, 2 * w.x0, w.y0, w.z0, t, 2 * NE);
                    tma_load_5d(smem_u32(sLZ) + SITES * NE * 16, &a.gauge.fz, fb, 2 * w.x0, w.y0, zm, t, 2 * NE);
                } else {
                    mbar_expect_tx(fb, LB::t);
                    tma_load_5d(smem_u32(sLT), &a.gauge.main, fb, 2 * w.x0, w.y0, w.z0, t, 3 * NE);
                }
                q[o].next();
                progress = true;
            }
            if (!progress) __nanosleep(40);
        }
        return;
    }

    // =================================================================== consumers: one site per thread and group
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(REG_CONSUMER));
    const bool groupA = warp < NGRP;
    const int lz = groupA ? warp : warp - NGRP;
    const int lx = lane & 7, ly = lane >> 3;
    const int sin = lz * 32 + lane;                 // site index inside the tile = element offset inside a plane box
    unsigned nI = 0;                                // interior planes consumed (both groups count every plane)
    unsigned nS = 0;                                // slices done = uses of the per-slice objects and of the hand-over buffer
    unsigned nT = 0;                                // group B: t-link chunks consumed (one extra per work item)
    auto release = [&](unsigned bar) {
        __syncwarp();
        if (lane == 0) mbar_arrive(bar);
    };
    double2* part = (double2*)sP + sin;             // this thread's slot of the hand-over buffer, element c at part[c * SITES]

    if (groupA) {
        // ---------------------------------------------------------------- group A: own term, x and y hops
        for (int j = 0; j < my_items; j++) {
            {   // the plane below the segment is group B's only
                const unsigned s = nI % SI;
                mbar_wait(fullI(s), (nI / SI) & 1u);
                release(emptyI(s));
                nI++;
            }
            for (int dt = 0; dt < a.Lt; dt++) {
                const unsigned s0 = nI % SI;
                mbar_wait(fullI(s0), (nI / SI) & 1u);
                const double2* I0 = (const double2*)(sI + s0 * I_BYTES) + sin;
                double2 acc[12];
                if (NA < 0) {
#pragma unroll
                    for (int c = 0; c < 12; c++) acc[c] = make_double2(0.0, 0.0);
                } else {
                    const double mik = -1.0 / a.kappa;
#pragma unroll
                    for (int c = 0; c < 12; c++) { const double2 o = I0[c * SITES]; acc[c] = make_double2(mik * o.x, mik * o.y); }
                }
                {   // ---- x
                    mbar_wait(fullO(HX), nS & 1u);
                    mbar_wait(fullO(LX), nS & 1u);
                    const double2* Hm = (const double2*)sHX;
                    const double2* Hp = Hm + 12 * FX;
                    const double2* Lb = (const double2*)sLX;
                    const int fi = lz * BY + ly;
                    const bool inp = lx + 1 < BX, inm = lx > 0;
                    hop_smem<0, -1, RECON>(acc, inp ? I0 + 1 : Hp + fi, inp ? SITES : FX, Lb + sin, SITES, 1.0);
                    hop_smem<0, +1, RECON>(acc, inm ? I0 - 1 : Hm + fi, inm ? SITES : FX,
                                           inm ? Lb + sin - 1 : Lb + SITES * NE + fi, inm ? SITES : FX, 1.0);
                    release(emptyO(HX));
                    release(emptyO(LX));
                }
                {   // ---- y
                    mbar_wait(fullO(HY), nS & 1u);
                    mbar_wait(fullO(LY), nS & 1u);
                    const double2* Hm = (const double2*)sHY;
                    const double2* Hp = Hm + 12 * FY;
                    const double2* Lb = (const double2*)sLY;
                    const int fi = lz * BX + lx;
                    const bool inp = ly + 1 < BY, inm = ly > 0;
                    hop_smem<1, -1, RECON>(acc, inp ? I0 + BX : Hp + fi, inp ? SITES : FY, Lb + sin, SITES, 1.0);
                    hop_smem<1, +1, RECON>(acc, inm ? I0 - BX : Hm + fi, inm ? SITES : FY,
                                           inm ? Lb + sin - BX : Lb + SITES * NE + fi, inm ? SITES : FY, 1.0);
                    release(emptyO(HY));
                    release(emptyO(LY));
                }
                release(emptyI(s0));
                nI++;
                // ---- hand the partial sums to group B (warp lz of A feeds warp lz of B)
                mbar_wait(partEmpty(lz), (nS & 1u) ^ 1u);
#pragma unroll
                for (int c = 0; c < 12; c++) part[c * SITES] = acc[c];
                release(partFull(lz));
                nS++;
            }
            {   // the plane above the segment is group B's only
                const unsigned s = nI % SI;
                mbar_wait(fullI(s), (nI / SI) & 1u);
                release(emptyI(s));
                nI++;
            }
        }
        return;
    }

    // -------------------------------------------------------------------- group B: z and t hops, epilogue, stores
    for (int j = 0; j < my_items; j++) {
        const Item w = decode_item(a, (int)blockIdx.x + j * (int)gridDim.x);
        double2 P[6];   // U_t(x, t-1)^+ (1 + gamma_t) psi(x, t-1): the backward-t hop of the next step, before the boundary sign
        {   // ---- prologue: slice t0 - 1
            const unsigned si = nI % SI;
            mbar_wait(fullI(si), (nI / SI) & 1u);
            mbar_wait(fullO(LT), nT & 1u);
            const double2* Ib = (const double2*)(sI + si * I_BYTES) + sin;
            const double2* Lb = (const double2*)sLT + sin;
            double2 psi[12], h[6], u[9];
            lds_spinor(Ib, SITES, psi);
            project<3, +1>(psi, h);
            lds_link<RECON>(Lb, SITES, u);
            su3_mul<true>(u, h, P);
            release(emptyI(si));
            release(emptyO(LT));
            nI++; nT++;
        }
        for (int dt = 0; dt < a.Lt; dt++) {
            const int t = w.t0 + dt;
            const unsigned s0 = nI % SI, s1 = (nI + 1) % SI;
            const long long gsite = (long long)(w.x0 + lx) + (long long)a.X * ((w.y0 + ly) + (long long)a.Y * ((w.z0 + lz) + (long long)a.Z * t));
            double2 acc[12];
            mbar_wait(partFull(lz), nS & 1u);
#pragma unroll
            for (int c = 0; c < 12; c++) acc[c] = part[c * SITES];
            release(partEmpty(lz));
            mbar_wait(fullI(s0), (nI / SI) & 1u);
            const double2* I0 = (const double2*)(sI + s0 * I_BYTES) + sin;
            {   // ---- z
                mbar_wait(fullO(HZ), nS & 1u);
                mbar_wait(fullO(LZ), nS & 1u);
                const double2* Hm = (const double2*)sHZ;
                const double2* Hp = Hm + 12 * FZ;
                const double2* Lb = (const double2*)sLZ;
                const int fi = ly * BX + lx;
                const bool inp = lz + 1 < BZ, inm = lz > 0;
                hop_smem<2, -1, RECON>(acc, inp ? I0 + BX * BY : Hp + fi, inp ? SITES : FZ, Lb + sin, SITES, 1.0);
                hop_smem<2, +1, RECON>(acc, inm ? I0 - BX * BY : Hm + fi, inm ? SITES : FZ,
                                       inm ? Lb + sin - BX * BY : Lb + SITES * NE + fi, inm ? SITES : FZ, 1.0);
                release(emptyO(HZ));
                release(emptyO(LZ));
            }
            {   // ---- t: forward from the next interior plane, backward from the carried product
                mbar_wait(fullO(LT), nT & 1u);
                mbar_wait(fullI(s1), ((nI + 1) / SI) & 1u);
                const double2* Lb = (const double2*)sLT + sin;
                const double2* I1 = (const double2*)(sI + s1 * I_BYTES) + sin;
                hop_smem<3, -1, RECON>(acc, I1, SITES, Lb, SITES, (t + 1 == a.T) ? a.tphase : 1.0);   // boundary in time
                reconstruct_add<3, +1>(acc, P, (t == 0) ? a.tphase : 1.0);
                // the product the next slice needs: U_t(x,t)^+ (1 + gamma_t) psi(x,t)
                double2 psi[12], h[6], u[9];
                lds_spinor(I0, SITES, psi);
                project<3, +1>(psi, h);
                lds_link<RECON>(Lb, SITES, u);
                su3_mul<true>(u, h, P);
                release(emptyO(LT));
                nT++;
            }
            release(emptyI(s0));
            nI++;
            nS++;

            // ---- epilogue (same arithmetic as the gather kernel)
            double2* o = a.out + gsite;
            if (NA < 0) {
#pragma unroll
                for (int c = 0; c < 12; c++) o[c * a.V] = acc[c];
            } else {
                const double s_up = -a.kappa * a.s, s_lo = a.g5 ? a.kappa * a.s : -a.kappa * a.s;
                constexpr int CH = 4;
#pragma unroll
                for (int c0 = 0; c0 < 12; c0 += CH) {
                    double2 w1[CH], w2[CH], w3[CH];
#pragma unroll
                    for (int k = 0; k < CH; k++) {
                        const long long e = gsite + (long long)(c0 + k) * a.V;
                        if (NA >= 1) w1[k] = a.A1[e];
                        if (NA >= 2) w2[k] = a.A2[e];
                        if (NA >= 3) w3[k] = a.A3[e];
                    }
#pragma unroll
                    for (int k = 0; k < CH; k++) {
                        const int c = c0 + k;
                        const bool lo = (c >= 6);
                        const double sc = lo ? s_lo : s_up;
                        double2 v = make_double2(sc * acc[c].x, sc * acc[c].y);
                        if (NA >= 1) { const double f = (lo && (a.a_g5 & 1)) ? -a.a1 : a.a1; v.x = fma(f, w1[k].x, v.x); v.y = fma(f, w1[k].y, v.y); }
                        if (NA >= 2) { const double f = (lo && (a.a_g5 & 2)) ? -a.a2 : a.a2; v.x = fma(f, w2[k].x, v.x); v.y = fma(f, w2[k].y, v.y); }
                        if (NA >= 3) { const double f = (lo && (a.a_g5 & 4)) ? -a.a3 : a.a3; v.x = fma(f, w3[k].x, v.x); v.y = fma(f, w3[k].y, v.y); }
                        o[c * a.V] = v;
                    }
                }
            }
        }
        // the plane above the segment was only the forward-t neighbour of the last slice
        {
            const unsigned s = nI % SI;
            mbar_wait(fullI(s), (nI / SI) & 1u);
            release(emptyI(s));
            nI++;
        }
    }
}

// ------------------------------------------------------------------------------------------------ host side
namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess)
            p = nullptr;
        return (EncodeTiledFn)p;
    }();
    return fn;
}

// 5-D map over a planes array [ncomp][T][Z][Y][X] of complex doubles, box (2*bx, by, bz, 1, nc) doubles
bool make_map(CUtensorMap* m, const void* base, const Lattice& lat, int ncomp, int bx, int by, int bz, int nc) {
    EncodeTiledFn enc = encode_fn();
    if (!enc) return false;
    const cuuint64_t X = lat.X, Y = lat.Y, Z = lat.Z, T = lat.T;
    cuuint64_t gdim[5] = {2 * X, Y, Z, T, (cuuint64_t)ncomp};
    cuuint64_t gstr[4] = {16 * X, 16 * X * Y, 16 * X * Y * Z, 16 * X * Y * Z * T};
    cuuint32_t box[5] = {(cuuint32_t)(2 * bx), (cuuint32_t)by, (cuuint32_t)bz, 1u, (cuuint32_t)nc};
    cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, const_cast<void*>(base), gdim, gstr, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
               bx > 1 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B : CU_TENSOR_MAP_L2_PROMOTION_NONE,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

bool make_maps(Maps* m, const void* base, const Lattice& lat, int ncomp, int nc) {
    return make_map(&m->main, base, lat, ncomp, BX, BY, BZ, nc) && make_map(&m->fx, base, lat, ncomp, 1, BY, BZ, nc) &&
           make_map(&m->fy, base, lat, ncomp, BX, 1, BZ, nc) && make_map(&m->fz, base, lat, ncomp, BX, BY, 1, nc);
}

struct TmaState {
    Maps gauge;
    bool gauge_ok = false;
    std::unordered_map<const void*, Maps> spinor;   // tensor maps by input pointer (a handful of workspaces + caller buffers)
    int sm_count = 0;
    int Lt = 0, nitems = 0;
};

}  // namespace

bool tma_eligible(const Lattice& lat) {
    return lat.X % BX == 0 && lat.Y % BY == 0 && lat.Z % BZ == 0 && lat.T >= 2 && lat.X <= 128 && lat.Y <= 256 &&
           lat.Z <= 256;
}

void tma_state_free(ov_ctx* ctx) {
    delete (TmaState*)ctx->tma_state;
    ctx->tma_state = nullptr;
}

template <int RECON, int NA>
static cudaError_t launch_k(const Args& a, int grid, size_t smem, cudaStream_t st) {
    static bool attr_set = false;   // per instantiation; one device per process (bench.py: one process per GPU)
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(wilson_tma_kernel<RECON, NA>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    wilson_tma_kernel<RECON, NA><<<grid, THREADS, smem, st>>>(a);
    return cudaGetLastError();
}

int launch_wilson_tma(ov_ctx* ctx, const double2* in, double2* out, const Epilogue& ep) {
    if (ctx->blocked || !tma_eligible(ctx->lat))
        return fail(ctx, OV_ESTATE, "the TMA-staged Wilson kernel needs the planes layout and X %% 8 == Y %% 4 == Z %% 4 == 0");
    if (!ctx->tma_state) ctx->tma_state = new TmaState();
    TmaState* st = (TmaState*)ctx->tma_state;
    const Lattice& lat = ctx->lat;
    const int NE = ctx->recon / 2;
    if (!st->gauge_ok) {
        if (!make_maps(&st->gauge, ctx->gauge, lat, 4 * NE, NE))
            return fail(ctx, OV_ECUDA, "cuTensorMapEncodeTiled failed for the gauge field");
        st->gauge_ok = true;
        int dev = 0;
        OV_CUDA(ctx, cudaGetDevice(&dev));
        OV_CUDA(ctx, cudaDeviceGetAttribute(&st->sm_count, cudaDevAttrMultiProcessorCount, dev));
        // slices per work item: the divisor of T that minimises (rounds of items per CTA) x (slices + prologue)
        const int npen = (lat.X / BX) * (lat.Y / BY) * (lat.Z / BZ);
        double best = 1e300;
        for (int L = 1; L <= lat.T; L++) {
            if (lat.T % L) continue;
            const long long items = (long long)npen * (lat.T / L);
            const long long rounds = (items + st->sm_count - 1) / st->sm_count;
            const double cost = (double)rounds * (L + 0.6);
            if (cost < best - 1e-9) { best = cost; st->Lt = L; st->nitems = (int)items; }
        }
    }
    auto map_of = [&](const double2* p, Maps** out) -> bool {   // tensor maps by pointer (a handful of workspaces + caller buffers)
        auto g = st->spinor.find(p);
        if (g == st->spinor.end()) {
            if (st->spinor.size() > 256) st->spinor.clear();
            Maps m;
            if (!make_maps(&m, p, lat, 12, 12)) return false;
            g = st->spinor.emplace(p, m).first;
        }
        *out = &g->second;
        return true;
    };
    Args a;
    {
        Maps* m = nullptr;
        if (!map_of(in, &m)) return fail(ctx, OV_ECUDA, "cuTensorMapEncodeTiled failed for a spinor");
        a.in = *m;
    }
    a.gauge = st->gauge;
    {
        const double2* ops[3] = {ep.hop_only ? nullptr : ep.A1, ep.hop_only ? nullptr : ep.A2, ep.hop_only ? nullptr : ep.A3};
        for (int i = 0; i < 3; i++) {
            Maps* m = nullptr;
            if (ops[i] && !map_of(ops[i], &m)) return fail(ctx, OV_ECUDA, "cuTensorMapEncodeTiled failed for an epilogue operand");
            a.op[i] = m ? m->main : a.in.main;   // unused slots get a valid map (never dereferenced)
        }
    }
    a.out = out;
    a.A1 = ep.A1; a.A2 = ep.A2; a.A3 = ep.A3;
    a.a1 = ep.a1; a.a2 = ep.a2; a.a3 = ep.a3;
    a.a_g5 = ep.a_g5;
    a.X = lat.X; a.Y = lat.Y; a.Z = lat.Z; a.T = lat.T;
    a.V = lat.V;
    a.kappa = ctx->kappa;
    a.s = ep.s;
    a.g5 = ep.g5;
    a.ntx = lat.X / BX; a.nty = lat.Y / BY; a.ntz = lat.Z / BZ;
    a.Lt = st->Lt;
    a.nitems = st->nitems;
    a.reverse = ctx->flip;
    ctx->flip ^= 1;
    a.tphase = ctx->t_phase;
    if ((ep.A3 && !ep.A2) || (ep.A2 && !ep.A1)) return fail(ctx, OV_EINVAL, "epilogue operands must be filled in order");
    const int na = ep.hop_only ? -1 : (ep.A3 ? 3 : ep.A2 ? 2 : ep.A1 ? 1 : 0);
    const int grid = st->nitems < st->sm_count ? st->nitems : st->sm_count;
    const size_t smem = NE == 9 ? smem_bytes<9>() : smem_bytes<6>();
    cudaError_t e;
#define OV_TMA_NA(R)                                                                         \
    switch (na) {                                                                            \
        case -1: e = launch_k<R, -1>(a, grid, smem, ctx->stream); break;           \
        case 0: e = launch_k<R, 0>(a, grid, smem, ctx->stream); break;             \
        case 1: e = launch_k<R, 1>(a, grid, smem, ctx->stream); break;             \
        case 2: e = launch_k<R, 2>(a, grid, smem, ctx->stream); break;             \
        default: e = launch_k<R, 3>(a, grid, smem, ctx->stream); break;            \
    }
    if (ctx->recon == 12) { OV_TMA_NA(12) } else { OV_TMA_NA(18) }
#undef OV_TMA_NA
    ctx->launches++;
    OV_CUDA(ctx, e);
    return OV_OK;
}

}  // namespace ov
