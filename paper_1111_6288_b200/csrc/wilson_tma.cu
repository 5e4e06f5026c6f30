// Wilson kernel, variant 2 ("TMA-staged"): a persistent, warp-specialised kernel for sm_100a (
// PAPER.md:31, :69 "approximately 70 % of the overlap calculation is spent in the dslash routine").
//
//   out = s * G (in - kappa * hop(in)) + a1*A1 + a2*A2 + a3*A3          (Epilogue, ov_internal.h)
//
// Why: the gather kernel (variant 1) pulls 2.2-2.3 kB/site through the SM's L2 port for 960 B/site of HBM traffic and
// is bound there.  Here every operand reaches the SM exactly once per tile through the TMA unit:
//   * the lattice is cut into pencils of 8 x 4 x 4 sites in (x,y,z); one CTA marches a pencil along t, one time slice
//     (128 sites = 4 consumer warps, one site per thread) per step;
//   * ONE producer thread issues cp.async.bulk.tensor (5-D boxes over the planes layout [comp][t][z][y][x]) into three
//     shared-memory rings guarded by mbarrier full/empty pairs: spinor interior planes (3 slots: t, t+1 and one in
//     flight), spinor halo faces of the current slice (6 one-site-thick boxes, wrapped coordinates are separate boxes
//     by construction; 2 slots), and link chunks (one direction of one slice + the one-site-thick halo of backward
//     links; 4 slots).  The producer runs about one slice ahead of the consumers, so ~140 kB are in flight per SM with
//     no register spent on them and no __syncthreads between loading and computing;
//   * consumers read neighbours and links from shared memory only (forward t neighbour = the next interior plane, which
//     later becomes the site's own plane; the backward t hop U_t(x-t)^+ (1+gamma_t) psi(x-t) is carried in registers
//     from the previous step), do the same arithmetic in the same order as the gather kernel (the hop is bit-identical,
//     results with an epilogue agree up to the compiler's FMA contraction) and store with coalesced 16-byte stores;
//   * launches with fused axpy operands (NA >= 1: the second launch of every Clenshaw order, the D_ov assembly) add an
//     EPILOGUE warpgroup: the consumers hand their accumulators over through a 24 KB shared-memory buffer and go on with
//     the next slice, while four epilogue warps -- which hold nothing else in registers -- issue the operand loads of a
//     slice BEFORE its accumulators arrive, so the DRAM latency of those one-touch streams overlaps the hops instead of
//     following them; setmaxnreg moves the registers the producer and the epilogue warps do not need to the consumers.
// L2->SM traffic per site: 192 (own) + 240 (halo) + 576 (links) + 72 (halo links) = 1080 B instead of ~2200.
//
// Needs the planes layout and X % 8 == 0, Y % 4 == 0, Z % 4 == 0; other shapes use the gather kernel.
#include <cuda.h>

#include <cstdlib>
#include <unordered_map>

#include "ov_internal.h"
#include "wilson_math.cuh"

namespace ov {

namespace tma {

constexpr int BX = 8, BY = 4, BZ = 4;           // tile of one time slice
constexpr int SITES = BX * BY * BZ;             // 128 = 4 consumer warps
constexpr int NCONS = SITES / 32;               // consumer warps
constexpr int SI = 3, SH = 2;                   // ring depths: interior planes, halo sets
// per kernel form: without epilogue operands 4 consumer warps + 1 producer warp and 4 link chunks in the ring; with them
// three aligned warpgroups (consumers, epilogue, producer) and 3 link chunks (the 4th slot becomes the hand-over buffer)
template <int NA> struct Form {
    static constexpr bool epi = NA >= 1;
    static constexpr int threads = epi ? 3 * 128 : SITES + 32;
    static constexpr int SL = epi ? 3 : 4;
};
constexpr int P_BYTES = SITES * 12 * 16;        // hand-over buffer: the consumers' accumulators of one slice
constexpr int REG_CONSUMER = 232, REG_PRODUCER = 40;   // epilogue warps keep the compiled 168: 128 * (232 + 168 + 40) <= 65536
constexpr int I_BYTES = SITES * 12 * 16;        // 24576
constexpr int FX = BY * BZ, FY = BX * BZ, FZ = BX * BY;   // face sites: 16, 32, 32
constexpr int H_ELEMS = 12 * (2 * FX + 2 * FY + 2 * FZ);  // 1920 double2
constexpr int H_BYTES = H_ELEMS * 16;           // 30720
// offsets (double2) of the six faces inside a halo slot: x-, x+, y-, y+, z-, z+
constexpr int HOFF_XM = 0, HOFF_XP = 12 * FX, HOFF_YM = 24 * FX, HOFF_YP = 24 * FX + 12 * FY,
              HOFF_ZM = 24 * FX + 24 * FY, HOFF_ZP = 24 * FX + 24 * FY + 12 * FZ;
template <int NE> struct LSlot { static constexpr int bytes = (SITES + 32) * NE * 16; };   // main box + the largest halo face

struct Maps {               // tensor maps of one spinor array or of the gauge field (box shapes differ)
    CUtensorMap main, fx, fy, fz;
};

struct Args {
    Maps in;                // spinor: 5-D (2X, Y, Z, T, 12) doubles
    Maps gauge;             // links:  5-D (2X, Y, Z, T, 4*NE) doubles
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
    int field_dir;          // background field (-1 = none): with 12-real links the rebuilt third row of a t link is multiplied
    double field_3qE;       // by det U = exp(-3 i qE (x_dir - origin))  (phase-tracked reconstruction)
    int field_origin;
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
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n"   // %2: suspend-time hint, the warp sleeps in hardware
        "@p bra WAIT_DONE;\n"                                             // instead of spinning on its scheduler's issue slots
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(bar), "r"(parity), "r"(0x989680u) : "memory");
}
__device__ __forceinline__ void tma_load_5d(unsigned dst, const CUtensorMap* map, unsigned bar, int c0, int c1, int c2,
                                            int c3, int c4) {
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4) : "memory");
}

// ring bookkeeping: fill number n lives in slot n % S and is that slot's (n / S)-th use
template <int S> __device__ __forceinline__ unsigned slot_of(unsigned n) { return n % S; }
template <int S> __device__ __forceinline__ unsigned full_parity(unsigned n) { return (n / S) & 1u; }
template <int S> __device__ __forceinline__ unsigned empty_parity(unsigned n) { return ((n / S) & 1u) ^ 1u; }

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
__device__ __forceinline__ void hop_smem(double2* acc, const double2* pn, int ns, const double2* pl, int ls, double ph,
                                         const double2* det = nullptr) {
    double2 psi[12], h[6], g[6], u[9];
    lds_spinor(pn, ns, psi);
    project<MU, SIGMA>(psi, h);
    lds_link<RECON>(pl, ls, u);
    if (RECON == 12 && det) {
#pragma unroll
        for (int e = 6; e < 9; e++) u[e] = cmul(u[e], *det);
    }
    su3_mul<(SIGMA > 0)>(u, h, g);
    reconstruct_add<MU, SIGMA>(acc, g, ph);
}

}  // namespace tma

using namespace tma;

// NA: -1 hop only, 0..3 epilogue operands (read from global memory at the output site)
template <int RECON, int NA>
__global__ void __launch_bounds__(Form<NA>::threads, 1) wilson_tma_kernel(const __grid_constant__ Args a) {
    constexpr int NE = RECON / 2;
    constexpr int L_BYTES = LSlot<NE>::bytes;
    constexpr bool EPI = Form<NA>::epi;
    constexpr int SL = Form<NA>::SL;
    constexpr int PRODUCER_WARP = EPI ? 8 : NCONS;
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char* sI = smem;
    unsigned char* sH = sI + SI * I_BYTES;
    unsigned char* sL = sH + SH * H_BYTES;
    unsigned char* sP = sL + SL * L_BYTES;          // hand-over buffer (EPI only)
    unsigned long long* bars = (unsigned long long*)(sP + (EPI ? P_BYTES : 0));
    // barrier indices: fullI[SI], emptyI[SI], fullH[SH], emptyH[SH], fullL[SL], emptyL[SL], partFull[NCONS], partEmpty[NCONS]
    const unsigned bar0 = smem_u32(bars);
    auto fullI = [&](unsigned s) { return bar0 + 8u * s; };
    auto emptyI = [&](unsigned s) { return bar0 + 8u * (SI + s); };
    auto fullH = [&](unsigned s) { return bar0 + 8u * (2 * SI + s); };
    auto emptyH = [&](unsigned s) { return bar0 + 8u * (2 * SI + SH + s); };
    auto fullL = [&](unsigned s) { return bar0 + 8u * (2 * SI + 2 * SH + s); };
    auto emptyL = [&](unsigned s) { return bar0 + 8u * (2 * SI + 2 * SH + SL + s); };
    auto partFull = [&](unsigned w) { return bar0 + 8u * (2 * SI + 2 * SH + 2 * SL + w); };
    auto partEmpty = [&](unsigned w) { return bar0 + 8u * (2 * SI + 2 * SH + 2 * SL + NCONS + w); };

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (unsigned s = 0; s < SI; s++) { mbar_init(fullI(s), 1); mbar_init(emptyI(s), NCONS); }
        for (unsigned s = 0; s < SH; s++) { mbar_init(fullH(s), 1); mbar_init(emptyH(s), NCONS); }
        for (unsigned s = 0; s < SL; s++) { mbar_init(fullL(s), 1); mbar_init(emptyL(s), NCONS); }
        if (EPI)
            for (unsigned w = 0; w < NCONS; w++) { mbar_init(partFull(w), 1); mbar_init(partEmpty(w), 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp >= PRODUCER_WARP) {
        // =============================================================== producer: one thread issues every TMA load
        if (EPI) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(REG_PRODUCER));
        if (warp != PRODUCER_WARP || lane != 0) return;
        unsigned nI = 0, nH = 0, nL = 0;
        auto fill_I = [&](const Item& w, int t) {
            const unsigned s = slot_of<SI>(nI);
            mbar_wait(emptyI(s), empty_parity<SI>(nI));
            mbar_expect_tx(fullI(s), I_BYTES);
            tma_load_5d(smem_u32(sI + s * I_BYTES), &a.in.main, fullI(s), 2 * w.x0, w.y0, w.z0, t, 0);
            nI++;
        };
        auto fill_H = [&](const Item& w, int t) {
            const unsigned s = slot_of<SH>(nH);
            mbar_wait(emptyH(s), empty_parity<SH>(nH));
            mbar_expect_tx(fullH(s), H_BYTES);
            const unsigned base = smem_u32(sH + s * H_BYTES);
            const int xm = (w.x0 == 0) ? a.X - 1 : w.x0 - 1, xp = (w.x0 + BX == a.X) ? 0 : w.x0 + BX;
            const int ym = (w.y0 == 0) ? a.Y - 1 : w.y0 - 1, yp = (w.y0 + BY == a.Y) ? 0 : w.y0 + BY;
            const int zm = (w.z0 == 0) ? a.Z - 1 : w.z0 - 1, zp = (w.z0 + BZ == a.Z) ? 0 : w.z0 + BZ;
            tma_load_5d(base + 16 * HOFF_XM, &a.in.fx, fullH(s), 2 * xm, w.y0, w.z0, t, 0);
            tma_load_5d(base + 16 * HOFF_XP, &a.in.fx, fullH(s), 2 * xp, w.y0, w.z0, t, 0);
            tma_load_5d(base + 16 * HOFF_YM, &a.in.fy, fullH(s), 2 * w.x0, ym, w.z0, t, 0);
            tma_load_5d(base + 16 * HOFF_YP, &a.in.fy, fullH(s), 2 * w.x0, yp, w.z0, t, 0);
            tma_load_5d(base + 16 * HOFF_ZM, &a.in.fz, fullH(s), 2 * w.x0, w.y0, zm, t, 0);
            tma_load_5d(base + 16 * HOFF_ZP, &a.in.fz, fullH(s), 2 * w.x0, w.y0, zp, t, 0);
            nH++;
        };
        auto fill_L = [&](const Item& w, int t, int mu) {
            const unsigned s = slot_of<SL>(nL);
            mbar_wait(emptyL(s), empty_parity<SL>(nL));
            const unsigned base = smem_u32(sL + s * L_BYTES);
            const int face = (mu == 0) ? FX : (mu == 1) ? FY : (mu == 2) ? FZ : 0;
            mbar_expect_tx(fullL(s), (SITES + face) * NE * 16);
            tma_load_5d(base, &a.gauge.main, fullL(s), 2 * w.x0, w.y0, w.z0, t, mu * NE);
            if (mu == 0) {
                const int xm = (w.x0 == 0) ? a.X - 1 : w.x0 - 1;
                tma_load_5d(base + SITES * NE * 16, &a.gauge.fx, fullL(s), 2 * xm, w.y0, w.z0, t, mu * NE);
            } else if (mu == 1) {
                const int ym = (w.y0 == 0) ? a.Y - 1 : w.y0 - 1;
                tma_load_5d(base + SITES * NE * 16, &a.gauge.fy, fullL(s), 2 * w.x0, ym, w.z0, t, mu * NE);
            } else if (mu == 2) {
                const int zm = (w.z0 == 0) ? a.Z - 1 : w.z0 - 1;
                tma_load_5d(base + SITES * NE * 16, &a.gauge.fz, fullL(s), 2 * w.x0, w.y0, zm, t, mu * NE);
            }
            nL++;
        };
        for (int it = blockIdx.x; it < a.nitems; it += gridDim.x) {
            const Item w = decode_item(a, it);
            const int tm = (w.t0 == 0) ? a.T - 1 : w.t0 - 1;
            fill_I(w, tm);          // prologue: the slice below the segment, for the carried backward-t product
            fill_L(w, tm, 3);
            fill_I(w, w.t0);
            for (int dt = 0; dt < a.Lt; dt++) {
                const int t = w.t0 + dt, tp = (t + 1 == a.T) ? 0 : t + 1;
                fill_I(w, tp);
                fill_H(w, t);
                fill_L(w, t, 0);
                fill_L(w, t, 1);
                fill_L(w, t, 2);
                fill_L(w, t, 3);
            }
        }
        return;
    }

    if (EPI && warp >= NCONS) {
        // =============================================================== epilogue warps (launches with operands only)
        const int lx = lane & 7, ly = lane >> 3, lz = warp - NCONS;
        const double2* part = (const double2*)sP + lz * 32 + lane;
        const double s_up = -a.kappa * a.s, s_lo = a.g5 ? a.kappa * a.s : -a.kappa * a.s;
        unsigned nS = 0;
        auto rel1 = [&](unsigned bar) {
            __syncwarp();
            if (lane == 0) mbar_arrive(bar);
        };
        // Operand loads run as a two-deep software pipeline of chunks of 3 components (9 loads of 16 B per thread and
        // chunk): the chunk after the one being combined is always in flight, across slice and work-item boundaries, and the
        // first chunk of a slice is issued before its accumulators are waited for.  Larger bursts were slower: with the
        // shared-memory carve-out at its maximum the LSU queue fills up and holds back the consumers' shared-memory loads.
        constexpr int CH = 3;
        auto gsite_of = [&](int it, int dt) -> long long {
            const Item w = decode_item(a, it);
            return (long long)(w.x0 + lx) + (long long)a.X * ((w.y0 + ly) + (long long)a.Y * ((w.z0 + lz) + (long long)a.Z * (w.t0 + dt)));
        };
        auto load_ops = [&](long long gsite, int c0, double2* w1, double2* w2, double2* w3) {
#pragma unroll
            for (int k = 0; k < CH; k++) {
                const long long e = gsite + (long long)(c0 + k) * a.V;
                if (NA >= 1) w1[k] = __ldcs(a.A1 + e);
                if (NA >= 2) w2[k] = __ldcs(a.A2 + e);
                if (NA >= 3) w3[k] = __ldcs(a.A3 + e);
            }
        };
        auto combine_store = [&](long long gsite, int c0, const double2* acc, const double2* w1, const double2* w2, const double2* w3) {
            double2* o = a.out + gsite;
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
        };
        double2 u1[CH], u2[CH], u3[CH], v1[CH], v2[CH], v3[CH], acc[12];   // the two operand buffers
        int it = blockIdx.x, dt = 0;
        if (it < a.nitems) load_ops(gsite_of(it, 0), 0, u1, u2, u3);
        while (it < a.nitems) {
            const long long gsite = gsite_of(it, dt);
            int it_n = it, dt_n = dt + 1;
            if (dt_n == a.Lt) { dt_n = 0; it_n = it + gridDim.x; }
            load_ops(gsite, 3, v1, v2, v3);
            mbar_wait(partFull(lz), nS & 1u);
#pragma unroll
            for (int c = 0; c < 12; c++) acc[c] = part[c * SITES];
            rel1(partEmpty(lz));
            nS++;
            combine_store(gsite, 0, acc, u1, u2, u3);
            load_ops(gsite, 6, u1, u2, u3);
            combine_store(gsite, 3, acc, v1, v2, v3);
            load_ops(gsite, 9, v1, v2, v3);
            combine_store(gsite, 6, acc, u1, u2, u3);
            if (it_n < a.nitems) load_ops(gsite_of(it_n, dt_n), 0, u1, u2, u3);
            combine_store(gsite, 9, acc, v1, v2, v3);
            it = it_n; dt = dt_n;
        }
        return;
    }

    // =================================================================== consumers: one site per thread
    if (EPI) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(REG_CONSUMER));
    const int lx = lane & 7, ly = lane >> 3, lz = warp;
    const int sin = lz * 32 + lane;                 // site index inside the tile = element offset inside a plane box
    unsigned nI = 0, nH = 0, nL = 0, nS = 0;
    auto release = [&](unsigned bar) {
        __syncwarp();
        if (lane == 0) mbar_arrive(bar);
    };

    for (int it = blockIdx.x; it < a.nitems; it += gridDim.x) {
        const Item w = decode_item(a, it);
        double2 P[6];   // U_t(x, t-1)^+ (1 + gamma_t) psi(x, t-1): the backward-t hop of the next step, before the boundary sign
        // 12-real links in a background field: det of this site's t links (it depends on the space coordinates only)
        const bool field = RECON == 12 && a.field_dir >= 0;
        double2 det = make_double2(1.0, 0.0);
        if (field) {
            const int xd = a.field_dir == 0 ? w.x0 + lx : a.field_dir == 1 ? w.y0 + ly : w.z0 + lz;
            sincos(-a.field_3qE * (double)(xd - a.field_origin), &det.y, &det.x);
        }
        auto fix_row2 = [&](double2* u) {
            if (field) {
#pragma unroll
                for (int e = 6; e < 9; e++) u[e] = cmul(u[e], det);
            }
        };
        {   // ---- prologue: slice t0 - 1
            const unsigned si = slot_of<SI>(nI), sl = slot_of<SL>(nL);
            mbar_wait(fullI(si), full_parity<SI>(nI));
            mbar_wait(fullL(sl), full_parity<SL>(nL));
            const double2* Ib = (const double2*)(sI + si * I_BYTES) + sin;
            const double2* Lb = (const double2*)(sL + sl * L_BYTES) + sin;
            double2 psi[12], h[6], u[9];
            lds_spinor(Ib, SITES, psi);
            project<3, +1>(psi, h);
            lds_link<RECON>(Lb, SITES, u);
            fix_row2(u);
            su3_mul<true>(u, h, P);
            release(emptyI(si));
            release(emptyL(sl));
            nI++; nL++;
        }
        for (int dt = 0; dt < a.Lt; dt++) {
            const int t = w.t0 + dt;
            const unsigned s0 = slot_of<SI>(nI), s1 = slot_of<SI>(nI + 1), sh = slot_of<SH>(nH);
            mbar_wait(fullI(s0), full_parity<SI>(nI));
            const double2* I0 = (const double2*)(sI + s0 * I_BYTES) + sin;
            const double2* Hb = (const double2*)(sH + sh * H_BYTES);
            const long long gsite = (long long)(w.x0 + lx) + (long long)a.X * ((w.y0 + ly) + (long long)a.Y * ((w.z0 + lz) + (long long)a.Z * t));

            double2 acc[12];
            if (NA < 0) {
#pragma unroll
                for (int c = 0; c < 12; c++) acc[c] = make_double2(0.0, 0.0);
            } else {
                const double mik = -1.0 / a.kappa;
#pragma unroll
                for (int c = 0; c < 12; c++) { const double2 o = I0[c * SITES]; acc[c] = make_double2(mik * o.x, mik * o.y); }
            }
            mbar_wait(fullH(sh), full_parity<SH>(nH));
            // ---- x
            {
                const unsigned sl = slot_of<SL>(nL);
                mbar_wait(fullL(sl), full_parity<SL>(nL));
                const double2* Lb = (const double2*)(sL + sl * L_BYTES);
                const int fi = lz * BY + ly;
                const bool inp = lx + 1 < BX, inm = lx > 0;
                hop_smem<0, -1, RECON>(acc, inp ? I0 + 1 : Hb + HOFF_XP + fi, inp ? SITES : FX, Lb + sin, SITES, 1.0);
                hop_smem<0, +1, RECON>(acc, inm ? I0 - 1 : Hb + HOFF_XM + fi, inm ? SITES : FX,
                                       inm ? Lb + sin - 1 : Lb + SITES * NE + fi, inm ? SITES : FX, 1.0);
                release(emptyL(sl));
                nL++;
            }
            // ---- y
            {
                const unsigned sl = slot_of<SL>(nL);
                mbar_wait(fullL(sl), full_parity<SL>(nL));
                const double2* Lb = (const double2*)(sL + sl * L_BYTES);
                const int fi = lz * BX + lx;
                const bool inp = ly + 1 < BY, inm = ly > 0;
                hop_smem<1, -1, RECON>(acc, inp ? I0 + BX : Hb + HOFF_YP + fi, inp ? SITES : FY, Lb + sin, SITES, 1.0);
                hop_smem<1, +1, RECON>(acc, inm ? I0 - BX : Hb + HOFF_YM + fi, inm ? SITES : FY,
                                       inm ? Lb + sin - BX : Lb + SITES * NE + fi, inm ? SITES : FY, 1.0);
                release(emptyL(sl));
                nL++;
            }
            // ---- z
            {
                const unsigned sl = slot_of<SL>(nL);
                mbar_wait(fullL(sl), full_parity<SL>(nL));
                const double2* Lb = (const double2*)(sL + sl * L_BYTES);
                const int fi = ly * BX + lx;
                const bool inp = lz + 1 < BZ, inm = lz > 0;
                hop_smem<2, -1, RECON>(acc, inp ? I0 + BX * BY : Hb + HOFF_ZP + fi, inp ? SITES : FZ, Lb + sin, SITES, 1.0);
                hop_smem<2, +1, RECON>(acc, inm ? I0 - BX * BY : Hb + HOFF_ZM + fi, inm ? SITES : FZ,
                                       inm ? Lb + sin - BX * BY : Lb + SITES * NE + fi, inm ? SITES : FZ, 1.0);
                release(emptyL(sl));
                nL++;
            }
            release(emptyH(sh));
            nH++;
            // ---- t: forward from the next interior plane, backward from the carried product
            {
                const unsigned sl = slot_of<SL>(nL);
                mbar_wait(fullL(sl), full_parity<SL>(nL));
                mbar_wait(fullI(s1), full_parity<SI>(nI + 1));
                const double2* Lb = (const double2*)(sL + sl * L_BYTES) + sin;
                const double2* I1 = (const double2*)(sI + s1 * I_BYTES) + sin;
                hop_smem<3, -1, RECON>(acc, I1, SITES, Lb, SITES, (t + 1 == a.T) ? a.tphase : 1.0, field ? &det : nullptr);   // boundary in time
                reconstruct_add<3, +1>(acc, P, (t == 0) ? a.tphase : 1.0);
                // the product the next slice needs: U_t(x,t)^+ (1 + gamma_t) psi(x,t)
                double2 psi[12], h[6], u[9];
                lds_spinor(I0, SITES, psi);
                project<3, +1>(psi, h);
                lds_link<RECON>(Lb, SITES, u);
                fix_row2(u);
                su3_mul<true>(u, h, P);
                release(emptyL(sl));
                nL++;
            }
            release(emptyI(s0));
            nI++;

            if (EPI) {   // ---- hand the accumulators to the epilogue warp of the same sites and go on
                double2* part = (double2*)sP + sin;
                mbar_wait(partEmpty(lz), (nS & 1u) ^ 1u);
#pragma unroll
                for (int c = 0; c < 12; c++) part[c * SITES] = acc[c];
                release(partFull(lz));
                nS++;
                continue;
            }
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
            const unsigned s = slot_of<SI>(nI);
            mbar_wait(fullI(s), full_parity<SI>(nI));
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

// Can this context use the TMA-staged kernel at all?  Asked once, at ov_create_ex, before the layout is fixed: the driver
// entry point cuTensorMapEncodeTiled must resolve and must accept the tensor maps of this lattice (tried on the gauge
// array; only the pointer is used).  The environment variable OV_NO_TMA (set, not "0") answers no: a switch for drivers
// or tools that mishandle tensor maps, and the test hook for the fallback.
bool tma_probe(const ov_ctx* ctx) {
    const char* off = std::getenv("OV_NO_TMA");
    if (off && off[0] && !(off[0] == '0' && !off[1])) return false;
    if (!tma_eligible(ctx->lat) || !encode_fn()) return false;
    Maps m;
    const int NE = ctx->recon / 2;
    return make_maps(&m, ctx->gauge, ctx->lat, 4 * NE, NE);
}

void tma_state_free(ov_ctx* ctx) {
    delete (TmaState*)ctx->tma_state;
    ctx->tma_state = nullptr;
}

template <int RECON, int NA>
static cudaError_t launch_k(const Args& a, int grid, size_t smem, cudaStream_t st) {
    // the opt-in to > 48 KB of dynamic shared memory is a per-device property of the function: remember it per
    // instantiation AND per device ordinal (a process may hold contexts on several GPUs); beyond 64 devices set it each time
    static bool attr_set[64] = {};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64 || !attr_set[dev]) {
        e = cudaFuncSetAttribute(wilson_tma_kernel<RECON, NA>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) attr_set[dev] = true;
    }
    wilson_tma_kernel<RECON, NA><<<grid, Form<NA>::threads, smem, st>>>(a);
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
    auto f = st->spinor.find(in);
    if (f == st->spinor.end()) {
        if (st->spinor.size() > 256) st->spinor.clear();
        Maps m;
        if (!make_maps(&m, in, lat, 12, 12)) return fail(ctx, OV_ECUDA, "cuTensorMapEncodeTiled failed for a spinor");
        f = st->spinor.emplace(in, m).first;
    }
    Args a;
    a.in = f->second;
    a.gauge = st->gauge;
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
    a.field_dir = ctx->field_dir;
    a.field_3qE = 3.0 * ctx->field_qE;
    a.field_origin = ctx->field_origin;
    if ((ep.A3 && !ep.A2) || (ep.A2 && !ep.A1)) return fail(ctx, OV_EINVAL, "epilogue operands must be filled in order");
    const int na = ep.hop_only ? -1 : (ep.A3 ? 3 : ep.A2 ? 2 : ep.A1 ? 1 : 0);
    const int grid = st->nitems < st->sm_count ? st->nitems : st->sm_count;
    const bool epi = na >= 1;
    const int nsl = epi ? Form<1>::SL : Form<0>::SL;
    const size_t smem = (size_t)SI * I_BYTES + (size_t)SH * H_BYTES + (size_t)nsl * (NE == 9 ? LSlot<9>::bytes : LSlot<6>::bytes) +
                        (epi ? P_BYTES : 0) + 8 * (2 * SI + 2 * SH + 2 * nsl + 2 * NCONS);
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
