// Layout conversion and BLAS-1 / reduction kernels on ABI spinors (PAPER.md:75
// "vector additions and scalar products").  Everything here is a pure streaming kernel: the roofline is
// HBM bandwidth, the design rule is 16-byte coalesced accesses and enough loads in flight per thread.
// Reductions are two-stage with a fixed shape (warp shuffle -> per-warp partial in global memory ->
// one block per result summing the partials in a fixed tree), no atomics: bit-reproducible.
#include <algorithm>
#include <cstring>

#include "ov_internal.h"
#include "wilson_math.cuh"

namespace ov {

// ------------------------------------------------------------------------------------------ layout
// canonical gauge [site][mu][9] -> internal layout (gauge_index, ov_internal.h).  MOD: the links are modified on the way
// (ov_options): U_t(x) *= exp(-i qE (x_dir - origin)) (eq. 4.1 with A_t = E (x_dir - origin)) and the
// links across a Dirichlet wall (coordinate d_mu - 1 in a direction of wall_mask) are set to zero.
template <int NE, bool BL, bool MOD>
__global__ void gauge_relayout_kernel(const double2* __restrict__ can, double2* __restrict__ g, long long V, GaugeMods m) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= V) return;
    int c[4];
    double2 ph = make_double2(1.0, 0.0);
    if (MOD) {
        long long r = i;
        c[0] = (int)(r % m.X); r /= m.X;
        c[1] = (int)(r % m.Y); r /= m.Y;
        c[2] = (int)(r % m.Z); r /= m.Z;
        c[3] = (int)r;
        if (m.field_dir >= 0) {
            double sn, cs;
            sincos(-m.qE * (double)(c[m.field_dir] - m.origin), &sn, &cs);
            ph = make_double2(cs, sn);
        }
    }
    const int ext[4] = {m.X, m.Y, m.Z, m.T};
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        const bool wall = MOD && ((m.wall_mask >> mu) & 1) && c[mu] == ext[mu] - 1;
#pragma unroll
        for (int e = 0; e < NE; e++) {
            double2 u = can[(i * 4 + mu) * 9 + e];
            if (MOD && mu == 3 && m.field_dir >= 0) u = make_double2(u.x * ph.x - u.y * ph.y, u.x * ph.y + u.y * ph.x);
            if (wall) u = make_double2(0.0, 0.0);
            g[gauge_index<NE, BL>(V, mu, e, i)] = u;
        }
    }
}

// largest |row2 - conj(row0 x row1)| and |<row_i,row_j> - delta_ij| over all links: recon 12 is only valid for SU(3)
__global__ void su3_defect_kernel(const double2* __restrict__ can, long long nlinks, unsigned long long* worst) {
    const long long l = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= nlinks) return;
    double2 u[9], r[9];
#pragma unroll
    for (int e = 0; e < 9; e++) { u[e] = can[l * 9 + e]; r[e] = u[e]; }
    su3_row2(r);
    double d = 0.0;
#pragma unroll
    for (int e = 6; e < 9; e++) d = fmax(d, fmax(fabs(r[e].x - u[e].x), fabs(r[e].y - u[e].y)));
#pragma unroll
    for (int i = 0; i < 2; i++)
#pragma unroll
        for (int j = i; j < 2; j++) {
            double2 acc = make_double2(0.0, 0.0);
#pragma unroll
            for (int c = 0; c < 3; c++) cmaddc(acc, u[3 * i + c], u[3 * j + c]);
            d = fmax(d, fmax(fabs(acc.x - (i == j ? 1.0 : 0.0)), fabs(acc.y)));
        }
    if (!(d == d) || isinf(d)) d = INFINITY;                          // fmax drops NaN: a non-finite link must fail the check
#pragma unroll
    for (int e = 0; e < 9; e++)
        if (!isfinite(u[e].x) || !isfinite(u[e].y)) d = INFINITY;
    atomicMax(worst, (unsigned long long)__double_as_longlong(d));   // non-negative doubles order like integers
}

int gauge_su3_defect(ov_ctx* ctx, const double2* canonical, double* defect) {
    unsigned long long* d_w = nullptr;
    OV_CUDA(ctx, cudaMalloc(&d_w, sizeof(unsigned long long)));
    OV_CUDA(ctx, cudaMemsetAsync(d_w, 0, sizeof(unsigned long long), ctx->stream));
    const long long nlinks = 4 * ctx->lat.V;
    su3_defect_kernel<<<(unsigned)((nlinks + 127) / 128), 128, 0, ctx->stream>>>(canonical, nlinks, d_w);
    ctx->launches++;
    unsigned long long h = 0;
    cudaError_t e = cudaMemcpyAsync(&h, d_w, sizeof h, cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    cudaFree(d_w);
    OV_CUDA(ctx, e);
    long long bits = (long long)h;
    double v;
    memcpy(&v, &bits, sizeof v);
    *defect = v;
    return OV_OK;
}

int launch_gauge_relayout(ov_ctx* ctx, const double2* canonical, const GaugeMods* mods) {
    const long long V = ctx->lat.V;
    const int threads = 128;
    const unsigned blocks = (unsigned)((V + threads - 1) / threads);
    GaugeMods m{};
    m.field_dir = -1;
    const bool mod = mods && (mods->wall_mask || mods->field_dir >= 0);
    if (mod) m = *mods;
    m.X = ctx->lat.X; m.Y = ctx->lat.Y; m.Z = ctx->lat.Z; m.T = ctx->lat.T;
#define OV_RELAYOUT(NE, BL)                                                                                          \
    do {                                                                                                             \
        if (mod) gauge_relayout_kernel<NE, BL, true><<<blocks, threads, 0, ctx->stream>>>(canonical, ctx->gauge, V, m); \
        else gauge_relayout_kernel<NE, BL, false><<<blocks, threads, 0, ctx->stream>>>(canonical, ctx->gauge, V, m);   \
    } while (0)
    if (ctx->recon == 12) {
        if (ctx->blocked) OV_RELAYOUT(6, true); else OV_RELAYOUT(6, false);
    } else {
        if (ctx->blocked) OV_RELAYOUT(9, true); else OV_RELAYOUT(9, false);
    }
#undef OV_RELAYOUT
    ctx->launches++;
    OV_CUDA(ctx, cudaGetLastError());
    return OV_OK;
}

// canonical spinor [site][12] <-> ABI [12][site], staged through shared memory so both sides coalesce
constexpr int kPackSites = 128;
template <bool PACK, bool BL>
__global__ void __launch_bounds__(kPackSites) pack_kernel(const double2* __restrict__ src,
                                                          double2* __restrict__ dst, long long V) {
    __shared__ double2 tile[kPackSites * 12 + 12];
    const long long base = (long long)blockIdx.x * kPackSites;
    const int n = (int)min((long long)kPackSites, V - base);
    if (PACK) {
        for (int j = threadIdx.x; j < n * 12; j += kPackSites) tile[j] = src[base * 12 + j];
        __syncthreads();
        if ((int)threadIdx.x < n)
#pragma unroll
            for (int c = 0; c < 12; c++) dst[spinor_base<BL>(base + threadIdx.x) + c * spinor_stride<BL>(V)] = tile[threadIdx.x * 12 + c];
    } else {
        if ((int)threadIdx.x < n)
#pragma unroll
            for (int c = 0; c < 12; c++) tile[threadIdx.x * 12 + c] = src[spinor_base<BL>(base + threadIdx.x) + c * spinor_stride<BL>(V)];
        __syncthreads();
        for (int j = threadIdx.x; j < n * 12; j += kPackSites) dst[base * 12 + j] = tile[j];
    }
}

int launch_pack(ov_ctx* ctx, const double2* canonical, double2* abi) {
    const long long V = ctx->lat.V;
    const unsigned blocks = (unsigned)((V + kPackSites - 1) / kPackSites);
    if (ctx->blocked) pack_kernel<true, true><<<blocks, kPackSites, 0, ctx->stream>>>(canonical, abi, V);
    else pack_kernel<true, false><<<blocks, kPackSites, 0, ctx->stream>>>(canonical, abi, V);
    ctx->launches++;
    OV_CUDA(ctx, cudaGetLastError());
    return OV_OK;
}
int launch_unpack(ov_ctx* ctx, const double2* abi, double2* canonical) {
    const long long V = ctx->lat.V;
    const unsigned blocks = (unsigned)((V + kPackSites - 1) / kPackSites);
    if (ctx->blocked) pack_kernel<false, true><<<blocks, kPackSites, 0, ctx->stream>>>(abi, canonical, V);
    else pack_kernel<false, false><<<blocks, kPackSites, 0, ctx->stream>>>(abi, canonical, V);
    ctx->launches++;
    OV_CUDA(ctx, cudaGetLastError());
    return OV_OK;
}

// ------------------------------------------------------------------------------------------ BLAS-1
constexpr int kEw = 4;  // complex elements per thread in elementwise kernels
constexpr int kEwThreads = 256;

__global__ void __launch_bounds__(kEwThreads) axpy_kernel(double2 a, const double2* __restrict__ x,
                                                          double2* __restrict__ y, long long n) {
    const long long base = (long long)blockIdx.x * (kEwThreads * kEw) + threadIdx.x;
    double2 xv[kEw], yv[kEw];
#pragma unroll
    for (int m = 0; m < kEw; m++) {
        const long long e = base + (long long)m * kEwThreads;
        if (e < n) { xv[m] = x[e]; yv[m] = y[e]; }
    }
#pragma unroll
    for (int m = 0; m < kEw; m++) {
        const long long e = base + (long long)m * kEwThreads;
        if (e < n) { cmadd(yv[m], a, xv[m]); y[e] = yv[m]; }
    }
}

// z = a x + b y (a, b real); x or y may be null (treated as zero); z may alias x or y
__global__ void __launch_bounds__(kEwThreads) axpby_kernel(double a, const double2* x, double b,
                                                           const double2* y, double2* z,   // no __restrict__: z may alias x or y
                                                           long long n) {
    const long long base = (long long)blockIdx.x * (kEwThreads * kEw) + threadIdx.x;
#pragma unroll
    for (int m = 0; m < kEw; m++) {
        const long long e = base + (long long)m * kEwThreads;
        if (e < n) {
            double2 v = make_double2(0.0, 0.0);
            if (x) { const double2 w = x[e]; v.x = a * w.x; v.y = a * w.y; }
            if (y) { const double2 w = y[e]; v.x = fma(b, w.x, v.x); v.y = fma(b, w.y, v.y); }
            z[e] = v;
        }
    }
}

// y = gamma5 x : components 6..11 (spins 2,3) change sign.  Element e has component e / V (planes) or (e/32) % 12 (blocked).
__global__ void __launch_bounds__(kEwThreads) gamma5_kernel(const double2* x, double2* y, long long V, int blocked) {
    const long long n = 12 * V;
    const long long base = (long long)blockIdx.x * (kEwThreads * kEw) + threadIdx.x;
#pragma unroll
    for (int m = 0; m < kEw; m++) {
        const long long e = base + (long long)m * kEwThreads;
        if (e < n) {
            double2 v = x[e];
            const bool lower = blocked ? ((e >> 5) % 12) >= 6 : e >= 6 * V;
            if (lower) { v.x = -v.x; v.y = -v.y; }
            y[e] = v;
        }
    }
}

// z = a x + b y + c w (real a, b, c); z may alias any operand (the generic Chebyshev filter of the D_ov eigensolver)
__global__ void __launch_bounds__(kEwThreads) axpbypcz_kernel(double a, const double2* x, double b, const double2* y,
                                                              double c, const double2* w, double2* z, long long n) {
    const long long base = (long long)blockIdx.x * (kEwThreads * kEw) + threadIdx.x;
#pragma unroll
    for (int m = 0; m < kEw; m++) {
        const long long e = base + (long long)m * kEwThreads;
        if (e < n) {
            const double2 xv = x[e], yv = y[e], wv = w[e];
            z[e] = make_double2(fma(c, wv.x, fma(b, yv.x, a * xv.x)), fma(c, wv.y, fma(b, yv.y, a * xv.y)));
        }
    }
}

// out = ax x + (s + gamma5) y : the chirality-sector form of D_ov^+ D_ov (ax = 2, y = sign(H_w) x), or the
// projector 2 P_s y with ax = 0 (x may then be null).  Upper components (spins 0,1) get (s + 1) y, lower ones (s - 1) y.
__global__ void __launch_bounds__(kEwThreads) chiral_combine_kernel(double ax, const double2* x, double s, const double2* y,
                                                                    double2* out, long long V, int blocked) {
    const long long n = 12 * V;
    const long long base = (long long)blockIdx.x * (kEwThreads * kEw) + threadIdx.x;
#pragma unroll
    for (int m = 0; m < kEw; m++) {
        const long long e = base + (long long)m * kEwThreads;
        if (e < n) {
            const bool lower = blocked ? ((e >> 5) % 12) >= 6 : e >= 6 * V;
            const double f = lower ? s - 1.0 : s + 1.0;
            const double2 yv = y[e];
            double2 v = make_double2(f * yv.x, f * yv.y);
            if (x) { const double2 xv = x[e]; v.x = fma(ax, xv.x, v.x); v.y = fma(ax, xv.y, v.y); }
            out[e] = v;
        }
    }
}

static inline unsigned ew_blocks(long long n) { return (unsigned)((n + kEwThreads * kEw - 1) / (kEwThreads * kEw)); }

int launch_axpy(ov_ctx* ctx, double2 a, const double2* x, double2* y) {
    const long long n = (long long)spinor_elems(ctx);
    axpy_kernel<<<ew_blocks(n), kEwThreads, 0, ctx->stream>>>(a, x, y, n);
    ctx->launches++;
    OV_CUDA(ctx, cudaGetLastError());
    return OV_OK;
}
int launch_axpby(ov_ctx* ctx, double a, const double2* x, double b, const double2* y, double2* z, int nrhs) {
    const long long n = (long long)spinor_elems(ctx) * nrhs;
    axpby_kernel<<<ew_blocks(n), kEwThreads, 0, ctx->stream>>>(a, x, b, y, z, n);
    ctx->launches++;
    OV_CUDA(ctx, cudaGetLastError());
    return OV_OK;
}
int launch_axpbypcz(ov_ctx* ctx, double a, const double2* x, double b, const double2* y, double c, const double2* w, double2* z) {
    const long long n = (long long)spinor_elems(ctx);
    axpbypcz_kernel<<<ew_blocks(n), kEwThreads, 0, ctx->stream>>>(a, x, b, y, c, w, z, n);
    ctx->launches++;
    OV_CUDA(ctx, cudaGetLastError());
    return OV_OK;
}
int launch_chiral_combine(ov_ctx* ctx, double ax, const double2* x, int s, const double2* y, double2* out) {
    const long long n = (long long)spinor_elems(ctx);
    chiral_combine_kernel<<<ew_blocks(n), kEwThreads, 0, ctx->stream>>>(ax, x, (double)s, y, out, ctx->lat.V, ctx->blocked ? 1 : 0);
    ctx->launches++;
    OV_CUDA(ctx, cudaGetLastError());
    return OV_OK;
}
int launch_scale(ov_ctx* ctx, double a, double2* x) { return launch_axpby(ctx, a, x, 0.0, nullptr, x); }
int launch_copy(ov_ctx* ctx, const double2* x, double2* y) { return launch_axpby(ctx, 1.0, x, 0.0, nullptr, y); }
int launch_zero(ov_ctx* ctx, double2* x) {
    OV_CUDA(ctx, cudaMemsetAsync(x, 0, spinor_elems(ctx) * sizeof(double2), ctx->stream));
    return OV_OK;
}
int launch_gamma5(ov_ctx* ctx, const double2* x, double2* y) {
    const long long n = (long long)spinor_elems(ctx);
    gamma5_kernel<<<ew_blocks(n), kEwThreads, 0, ctx->stream>>>(x, y, ctx->lat.V, ctx->blocked ? 1 : 0);
    ctx->launches++;
    OV_CUDA(ctx, cudaGetLastError());
    return OV_OK;
}

// ------------------------------------------------------------------------------------------ reductions
// multi-dot: r_j = sum_e conj(x_j[e]) y[e], j < nvec  (the small-space V^+ x of PAPER.md:39/:81 with k = 100-200).
// A warp owns a window of kDotE*32 consecutive elements of y, keeps them in registers and streams the same window of
// every x_j once, so y is read from HBM exactly once.  The vectors are taken four at a time: the loads of the next four
// are issued before the current four are reduced (16 independent 16-byte loads in flight per lane), and the four complex
// partial sums are reduced together by a halving butterfly (18 shuffles per 4 vectors instead of 80).  Warps park their
// sums in shared memory; one fixed-order pass per block writes partial[j][block]: deterministic, no atomics.
constexpr int kDotE = 2;
constexpr int kDotThreads = 256;
constexpr int kDotWarps = kDotThreads / 32;
constexpr int kDotBlockElems = kDotE * kDotThreads;
constexpr int kDotMaxVec = 1024;  // vectors per launch (shared memory: nvec * 8 warps * 16 B)

__device__ __forceinline__ void dot_load4(const double2* __restrict__ xs, size_t stride, int j, int nvec, long long base,
                                          long long n, double2 (&xv)[4][kDotE]) {
#pragma unroll
    for (int u = 0; u < 4; u++)
#pragma unroll
        for (int m = 0; m < kDotE; m++) {
            const long long e = base + m * 32;
            xv[u][m] = (j + u < nvec && e < n) ? __ldcs(xs + (size_t)(j + u) * stride + e) : make_double2(0.0, 0.0);
        }
}

// NB right-hand sides y_r = y + r * ystride at once (the batched small-space projector, "adding a new source
// is relatively inexpensive"): every x_j is still streamed ONCE, its window is reduced against the NB windows of y kept in
// registers.  Results: partial[(r * nvec + j) * nblocks + block].
template <int NB>
__global__ void __launch_bounds__(kDotThreads) multi_dot_kernel(const double2* __restrict__ xs, size_t stride,
                                                                int nvec, const double2* __restrict__ y, size_t ystride,
                                                                long long n, long long nblocks,
                                                                double2* __restrict__ partial) {
    extern __shared__ double2 sacc[];  // [NB][nvec][kDotWarps]
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long base = (long long)blockIdx.x * kDotBlockElems + warp * (kDotE * 32) + lane;
    double2 yv[NB][kDotE];
#pragma unroll
    for (int r = 0; r < NB; r++)
#pragma unroll
        for (int m = 0; m < kDotE; m++) {
            const long long e = base + m * 32;
            yv[r][m] = (e < n) ? y[(size_t)r * ystride + e] : make_double2(0.0, 0.0);
        }
    double2 cur[4][kDotE], nxt[4][kDotE];
    dot_load4(xs, stride, 0, nvec, base, n, cur);
    for (int j = 0; j < nvec; j += 4) {
        dot_load4(xs, stride, j + 4, nvec, base, n, nxt);   // next four in flight while these are reduced
#pragma unroll
      for (int r = 0; r < NB; r++) {
        double v[8];
#pragma unroll
        for (int u = 0; u < 4; u++) {
            double2 acc = make_double2(0.0, 0.0);
#pragma unroll
            for (int m = 0; m < kDotE; m++) cmaddc(acc, cur[u][m], yv[r][m]);
            v[2 * u] = acc.x; v[2 * u + 1] = acc.y;
        }
        // halving butterfly: 8 -> 4 -> 2 -> 1 values per lane, then two plain steps
#pragma unroll
        for (int q = 0; q < 4; q++) {
            const bool up = lane & 16;
            const double send = up ? v[q] : v[q + 4], keep = up ? v[q + 4] : v[q];
            v[q] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
        }
#pragma unroll
        for (int q = 0; q < 2; q++) {
            const bool up = lane & 8;
            const double send = up ? v[q] : v[q + 2], keep = up ? v[q + 2] : v[q];
            v[q] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
        }
        {
            const bool up = lane & 4;
            const double send = up ? v[0] : v[1], keep = up ? v[1] : v[0];
            v[0] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
        }
        v[0] += __shfl_xor_sync(0xffffffffu, v[0], 2);
        v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1);
        // lane l (l % 4 == 0) holds value index 4*bit4 + 2*bit3 + bit2 = (vector j + idx/2, re/im idx%2)
        if ((lane & 3) == 0) {
            const int idx = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);
            const int jj = j + (idx >> 1);
            if (jj < nvec) reinterpret_cast<double*>(sacc + ((size_t)r * nvec + jj) * kDotWarps + warp)[idx & 1] = v[0];
        }
      }
#pragma unroll
        for (int u = 0; u < 4; u++)
#pragma unroll
            for (int m = 0; m < kDotE; m++) cur[u][m] = nxt[u][m];
    }
    __syncthreads();
    for (int jj = threadIdx.x; jj < NB * nvec; jj += kDotThreads) {
        double2 t = sacc[(size_t)jj * kDotWarps];
#pragma unroll
        for (int w = 1; w < kDotWarps; w++) t = cadd(t, sacc[(size_t)jj * kDotWarps + w]);
        partial[(long long)jj * nblocks + blockIdx.x] = t;
    }
}

// one block per result: fixed-order strided accumulation then a fixed shared-memory tree
constexpr int kRedThreads = 256;
__global__ void __launch_bounds__(kRedThreads) reduce_partials_kernel(const double2* __restrict__ partial,
                                                                      long long nwarps, double2* __restrict__ result) {
    __shared__ double2 sh[kRedThreads];
    const double2* p = partial + (long long)blockIdx.x * nwarps;
    double2 acc = make_double2(0.0, 0.0);
    for (long long w = threadIdx.x; w < nwarps; w += kRedThreads) acc = cadd(acc, p[w]);
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int o = kRedThreads / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] = cadd(sh[threadIdx.x], sh[threadIdx.x + o]);
        __syncthreads();
    }
    if (threadIdx.x == 0) result[blockIdx.x] = sh[0];
}

int launch_multi_dot_at(ov_ctx* ctx, const double2* xs, size_t stride, int nvec, const double2* y, int result_offset,
                        int result_total) {
    const long long n = (long long)spinor_elems(ctx);
    const long long nblocks = (n + kDotBlockElems - 1) / kDotBlockElems;
    OV_TRY(ensure_reduction_buffers(ctx, (size_t)nblocks * result_total, (size_t)result_total));
    for (int j0 = 0; j0 < nvec; j0 += kDotMaxVec) {
        const int nv = std::min(kDotMaxVec, nvec - j0);
        const size_t shmem = (size_t)nv * kDotWarps * sizeof(double2);
        if (shmem > 48 * 1024)
            OV_CUDA(ctx, cudaFuncSetAttribute(multi_dot_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shmem));
        double2* partial = ctx->d_partial + (size_t)(result_offset + j0) * nblocks;
        multi_dot_kernel<1><<<(unsigned)nblocks, kDotThreads, shmem, ctx->stream>>>(xs + (size_t)j0 * stride, stride, nv, y, 0, n,
                                                                                     nblocks, partial);
        reduce_partials_kernel<<<nv, kRedThreads, 0, ctx->stream>>>(partial, nblocks, ctx->d_result + result_offset + j0);
        ctx->launches += 2;
    }
    OV_CUDA(ctx, cudaGetLastError());
    return OV_OK;
}

int launch_multi_dot(ov_ctx* ctx, const double2* xs, size_t stride, int nvec, const double2* y) {
    return launch_multi_dot_at(ctx, xs, stride, nvec, y, 0, nvec);
}

// the batched kernel parks all nb * nvec per-warp sums of a block in shared memory (128 B per result): nb = 4 fits up to
// nvec = 400, nb = 2 up to 800; callers (project_batch) take smaller groups beyond that
bool multi_dot_batch_fits(int nvec, int nb) {
    return (size_t)nb * nvec * kDotWarps * sizeof(double2) <= 200 * 1024;
}

// nb in {2, 4} right-hand sides y_r = y + r * ystride in one pass over the x_j: d_result[r * nvec + j] = <x_j, y_r>
int launch_multi_dot_batch(ov_ctx* ctx, const double2* xs, size_t stride, int nvec, const double2* y, size_t ystride, int nb) {
    const long long n = (long long)spinor_elems(ctx);
    const long long nblocks = (n + kDotBlockElems - 1) / kDotBlockElems;
    if (nb != 2 && nb != 4) return fail(ctx, OV_EINVAL, "multi_dot_batch: nb must be 2 or 4");
    const size_t shmem = (size_t)nb * nvec * kDotWarps * sizeof(double2);
    if (!multi_dot_batch_fits(nvec, nb))
        return fail(ctx, OV_EINVAL, "multi_dot_batch: %d x %d results do not fit in shared memory", nb, nvec);
    OV_TRY(ensure_reduction_buffers(ctx, (size_t)nblocks * nb * nvec, (size_t)nb * nvec));
    if (nb == 2) {
        if (shmem > 48 * 1024)
            OV_CUDA(ctx, cudaFuncSetAttribute(multi_dot_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shmem));
        multi_dot_kernel<2><<<(unsigned)nblocks, kDotThreads, shmem, ctx->stream>>>(xs, stride, nvec, y, ystride, n, nblocks, ctx->d_partial);
    } else {
        if (shmem > 48 * 1024)
            OV_CUDA(ctx, cudaFuncSetAttribute(multi_dot_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shmem));
        multi_dot_kernel<4><<<(unsigned)nblocks, kDotThreads, shmem, ctx->stream>>>(xs, stride, nvec, y, ystride, n, nblocks, ctx->d_partial);
    }
    reduce_partials_kernel<<<nb * nvec, kRedThreads, 0, ctx->stream>>>(ctx->d_partial, nblocks, ctx->d_result);
    ctx->launches += 2;
    OV_CUDA(ctx, cudaGetLastError());
    return OV_OK;
}

int fetch_results(ov_ctx* ctx, int n, double2* host_out) {
    OV_CUDA(ctx, cudaMemcpyAsync(ctx->h_result, ctx->d_result, (size_t)n * sizeof(double2),
                                 cudaMemcpyDeviceToHost, ctx->stream));
    OV_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    for (int i = 0; i < n; i++) host_out[i] = ctx->h_result[i];
    return OV_OK;
}

// one plain dot product <x, y>: 8 independent 16-byte loads per thread and pass, fixed-shape reduction
constexpr int kDot1Threads = 256;
constexpr int kDot1E = 4;
__global__ void __launch_bounds__(kDot1Threads) dot1_kernel(const double2* __restrict__ x, const double2* __restrict__ y,
                                                            long long n, double2* __restrict__ partial) {
    __shared__ double2 sh[kDot1Threads];
    const long long base = (long long)blockIdx.x * (kDot1Threads * kDot1E) + threadIdx.x;
    double2 xv[kDot1E], yv[kDot1E];
#pragma unroll
    for (int m = 0; m < kDot1E; m++) {
        const long long e = base + (long long)m * kDot1Threads;
        xv[m] = (e < n) ? x[e] : make_double2(0.0, 0.0);
        yv[m] = (e < n) ? y[e] : make_double2(0.0, 0.0);
    }
    double2 acc = make_double2(0.0, 0.0);
#pragma unroll
    for (int m = 0; m < kDot1E; m++) cmaddc(acc, xv[m], yv[m]);
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int o = kDot1Threads / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] = cadd(sh[threadIdx.x], sh[threadIdx.x + o]);
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}

int dot_host(ov_ctx* ctx, const double2* x, const double2* y, double2* out) {
    const long long n = (long long)spinor_elems(ctx);
    const long long nblocks = (n + kDot1Threads * kDot1E - 1) / (kDot1Threads * kDot1E);
    OV_TRY(ensure_reduction_buffers(ctx, (size_t)nblocks, 1));
    dot1_kernel<<<(unsigned)nblocks, kDot1Threads, 0, ctx->stream>>>(x, y, n, ctx->d_partial);
    reduce_partials_kernel<<<1, kRedThreads, 0, ctx->stream>>>(ctx->d_partial, nblocks, ctx->d_result);
    ctx->launches += 2;
    OV_CUDA(ctx, cudaGetLastError());
    return fetch_results(ctx, 1, out);
}
int norm2_host(ov_ctx* ctx, const double2* x, double* out) {
    double2 r;
    OV_TRY(dot_host(ctx, x, x, &r));
    *out = r.x;
    return OV_OK;
}

// ------------------------------------------------------------------------------------------ multi-axpy
// out_j = bscale_j * base + sum_{i<nvec} C[i*J + j] * x_i   for j < J  (J outputs per pass over the x_i).
// The coefficient block sits in shared memory; every x_i element is read once per pass.
constexpr int kMaThreads = 256;
template <int J>
__global__ void __launch_bounds__(kMaThreads) multi_axpy_kernel(const double2* __restrict__ xs, size_t stride,
                                                                int nvec, const double2* __restrict__ C,
                                                                const double2* base,
                                                                const MultiAxpyOuts o, long long n) {
    extern __shared__ double2 shC[];
    for (int q = threadIdx.x; q < nvec * J; q += kMaThreads) shC[q] = C[q];
    __syncthreads();
    const long long e = (long long)blockIdx.x * kMaThreads + threadIdx.x;
    if (e >= n) return;
    double2 acc[J];
    const double2 b = base ? base[e] : make_double2(0.0, 0.0);
#pragma unroll
    for (int j = 0; j < J; j++) {
        const double2 bj = o.basej[j] ? o.basej[j][e] : b;      // per-output base (batched projector) or the common one
        acc[j] = make_double2(o.bscale[j] * bj.x, o.bscale[j] * bj.y);
    }
    int i = 0;
    for (; i + 4 <= nvec; i += 4) {
        double2 xv[4];
#pragma unroll
        for (int u = 0; u < 4; u++) xv[u] = __ldcs(xs + (size_t)(i + u) * stride + e);
#pragma unroll
        for (int u = 0; u < 4; u++)
#pragma unroll
            for (int j = 0; j < J; j++) cmadd(acc[j], shC[(i + u) * J + j], xv[u]);
    }
    for (; i < nvec; i++) {
        const double2 xv = __ldcs(xs + (size_t)i * stride + e);
#pragma unroll
        for (int j = 0; j < J; j++) cmadd(acc[j], shC[i * J + j], xv);
    }
#pragma unroll
    for (int j = 0; j < J; j++) o.out[j][e] = acc[j];
}

// host wrapper used by the projector and the Lanczos Ritz rotation.
// C_dev: nvec x J complex (row i, column j) on the device; o: J output pointers + base scales (by value).
int launch_multi_axpy(ov_ctx* ctx, const double2* xs, size_t stride, int nvec, int J, const double2* C_dev,
                      const double2* base, const MultiAxpyOuts& o) {
    const long long n = (long long)spinor_elems(ctx);
    const unsigned blocks = (unsigned)((n + kMaThreads - 1) / kMaThreads);
    const size_t shmem = (size_t)nvec * J * sizeof(double2);
    if (shmem > 200 * 1024) return fail(ctx, OV_EINVAL, "multi_axpy: coefficient block too large (%zu B)", shmem);
#define OV_MA_CASE(JJ)                                                                                         \
    case JJ:                                                                                                   \
        if (shmem > 48 * 1024)                                                                                 \
            OV_CUDA(ctx, cudaFuncSetAttribute(multi_axpy_kernel<JJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                                              (int)shmem));                                                    \
        multi_axpy_kernel<JJ><<<blocks, kMaThreads, shmem, ctx->stream>>>(xs, stride, nvec, C_dev, base, o, n); \
        break;
    switch (J) {
        OV_MA_CASE(1)
        OV_MA_CASE(2)
        OV_MA_CASE(4)
        OV_MA_CASE(8)
        default:
            return fail(ctx, OV_EINVAL, "multi_axpy: J must be 1, 2, 4 or 8");
    }
#undef OV_MA_CASE
    ctx->launches++;
    OV_CUDA(ctx, cudaGetLastError());
    return OV_OK;
}

}  // namespace ov

namespace ov {

// ------------------------------------------------------------------------------------------ in-place basis rotation
// W[j] <- sum_{i<m} S[i][j] W[i]  for j < ncol <= m, in place (row a8: the restart and Rayleigh-Ritz rotations of the
// Lanczos basis; at k = 200 on 32^3x64 a second copy of the basis would not fit in HBM).  The basis is two segments:
// vectors 0..na-1 at a + i*stride, vectors na.. at b + (i-na)*stride.  A block stages a tile of kRotE elements of all
// m vectors in shared memory, so every output can overwrite its input.  St is S transposed: St[j*m + i] (device).
constexpr int kRotE = (int)(kRotTileBytesPerVector / sizeof(double2));
constexpr int kRotThreads = 256;
__global__ void __launch_bounds__(kRotThreads) rotate_inplace_kernel(double2* a, int na, double2* b, size_t stride, int m,
                                                                     int ncol, const double2* __restrict__ St, long long n) {
    extern __shared__ double2 tile[];  // [m][kRotE]
    const long long e0 = (long long)blockIdx.x * kRotE;
    const int el = threadIdx.x % kRotE, grp = threadIdx.x / kRotE;
    constexpr int ngrp = kRotThreads / kRotE;
    const bool live = e0 + el < n;
    for (int i = grp; i < m; i += ngrp) {
        const double2* v = (i < na) ? a + (size_t)i * stride : b + (size_t)(i - na) * stride;
        tile[i * kRotE + el] = live ? v[e0 + el] : make_double2(0.0, 0.0);
    }
    __syncthreads();
    for (int j = grp; j < ncol; j += ngrp) {
        const double2* s = St + (size_t)j * m;
        double2 acc0 = make_double2(0.0, 0.0), acc1 = make_double2(0.0, 0.0);
        int i = 0;
        for (; i + 2 <= m; i += 2) {
            cmadd(acc0, __ldg(s + i), tile[i * kRotE + el]);
            cmadd(acc1, __ldg(s + i + 1), tile[(i + 1) * kRotE + el]);
        }
        if (i < m) cmadd(acc0, __ldg(s + i), tile[i * kRotE + el]);
        if (live) {
            double2* v = (j < na) ? a + (size_t)j * stride : b + (size_t)(j - na) * stride;
            v[e0 + el] = cadd(acc0, acc1);
        }
    }
}

int launch_rotate_inplace(ov_ctx* ctx, double2* a, int na, double2* b, size_t stride, int m, int ncol,
                          const double2* St_dev) {
    const long long n = (long long)spinor_elems(ctx);
    const size_t shmem = (size_t)m * kRotE * sizeof(double2);
    if (shmem > 220 * 1024) return fail(ctx, OV_EINVAL, "rotate_inplace: basis too large (%d vectors)", m);
    if (ncol > m) return fail(ctx, OV_EINVAL, "rotate_inplace: ncol > m");
    OV_CUDA(ctx, cudaFuncSetAttribute(rotate_inplace_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shmem));
    const unsigned blocks = (unsigned)((n + kRotE - 1) / kRotE);
    rotate_inplace_kernel<<<blocks, kRotThreads, shmem, ctx->stream>>>(a, na, b, stride, m, ncol, St_dev, n);
    ctx->launches++;
    OV_CUDA(ctx, cudaGetLastError());
    return OV_OK;
}

}  // namespace ov

namespace ov {

// ------------------------------------------------------------------------------------------ fp32 helpers
// The reduced-precision tail of the adaptive CG keeps every CG vector in fp64 and runs only the Clenshaw
// sweep of an operator application in fp32: y32 = (float) a*x on the way in, out = r32 + a1*A1 + a2*[gamma5]A2 on the
// way out (both fp64 operands; the D_ov assembly of row a5).
__global__ void __launch_bounds__(kEwThreads) scale_to_f32_kernel(double a, const double2* __restrict__ x,
                                                                  float2* __restrict__ y, long long n) {
    const long long base = (long long)blockIdx.x * (kEwThreads * kEw) + threadIdx.x;
#pragma unroll
    for (int m = 0; m < kEw; m++) {
        const long long e = base + (long long)m * kEwThreads;
        if (e < n) { const double2 v = x[e]; y[e] = make_float2((float)(a * v.x), (float)(a * v.y)); }
    }
}

__global__ void __launch_bounds__(kEwThreads) combine_from_f32_kernel(const float2* __restrict__ r, double a1,
                                                                      const double2* __restrict__ A1, double a2,
                                                                      const double2* __restrict__ A2, int a2_g5,
                                                                      double2* out, long long V, int blocked) {
    const long long n = 12 * V;
    const long long base = (long long)blockIdx.x * (kEwThreads * kEw) + threadIdx.x;
#pragma unroll
    for (int m = 0; m < kEw; m++) {
        const long long e = base + (long long)m * kEwThreads;
        if (e < n) {
            const float2 rf = r[e];
            double2 v = make_double2((double)rf.x, (double)rf.y);
            if (A1) { const double2 w = A1[e]; v.x = fma(a1, w.x, v.x); v.y = fma(a1, w.y, v.y); }
            if (A2) {
                const bool lower = blocked ? ((e >> 5) % 12) >= 6 : e >= 6 * V;
                const double f = (a2_g5 && lower) ? -a2 : a2;
                const double2 w = A2[e]; v.x = fma(f, w.x, v.x); v.y = fma(f, w.y, v.y);
            }
            out[e] = v;
        }
    }
}

__global__ void __launch_bounds__(kEwThreads) gauge_to_f32_kernel(const double2* __restrict__ g, float2* __restrict__ gf,
                                                                  long long n) {
    const long long e = (long long)blockIdx.x * kEwThreads + threadIdx.x;
    if (e < n) { const double2 v = g[e]; gf[e] = make_float2((float)v.x, (float)v.y); }
}

int launch_scale_to_f32(ov_ctx* ctx, double a, const double2* x, float2* y) {
    const long long n = (long long)spinor_elems(ctx);
    scale_to_f32_kernel<<<ew_blocks(n), kEwThreads, 0, ctx->stream>>>(a, x, y, n);
    ctx->launches++;
    OV_CUDA(ctx, cudaGetLastError());
    return OV_OK;
}
int launch_combine_from_f32(ov_ctx* ctx, const float2* r, double a1, const double2* A1, double a2, const double2* A2,
                            int a2_g5, double2* out) {
    const long long n = (long long)spinor_elems(ctx);
    combine_from_f32_kernel<<<ew_blocks(n), kEwThreads, 0, ctx->stream>>>(r, a1, A1, a2, A2, a2_g5, out, ctx->lat.V,
                                                                          ctx->blocked ? 1 : 0);
    ctx->launches++;
    OV_CUDA(ctx, cudaGetLastError());
    return OV_OK;
}
// fp32 copy of the links (same layout as the fp64 ones), made once on first use
int ensure_gauge_f32(ov_ctx* ctx) {
    if (ctx->gauge_f) return OV_OK;
    const long long n = (long long)gauge_elems(ctx->lat.V, ctx->recon);
    OV_CUDA(ctx, cudaMalloc(&ctx->gauge_f, (size_t)n * sizeof(float2)));
    gauge_to_f32_kernel<<<(unsigned)((n + kEwThreads - 1) / kEwThreads), kEwThreads, 0, ctx->stream>>>(ctx->gauge, ctx->gauge_f, n);
    ctx->launches++;
    OV_CUDA(ctx, cudaGetLastError());
    return OV_OK;
}

}  // namespace ov
