// Internal declarations shared by the translation units of libov.so (CUDA side only).
#pragma once
#include <cuda_runtime.h>

#include <array>
#include <cstdarg>
#include <cstdio>
#include <string>
#include <vector>

#include "ov.h"

namespace ov {

constexpr int kSpinorComplex = 12;  // 4 spins x 3 colours
constexpr size_t kRotTileBytesPerVector = 16 * sizeof(double2);  // rotate_inplace_kernel: kRotE elements per vector

// Layouts.  "Blocked" (BL = true, used whenever V is a multiple of 32): 32 consecutive sites form a block and the
// components of a block are contiguous -- spinor element (comp c, site i) at ((i>>5)*12 + c)*32 + (i&31), link entry
// (mu, e, site i) at ((i>>5)*4*NE + mu*NE + e)*32 + (i&31).  A warp still reads 512 contiguous bytes per component, but
// all components of a site now sit at compile-time offsets (c*512 B) from ONE base address, which removes the 64-bit
// address arithmetic per load (-18 % instructions in the Wilson kernel, +4 % in the power-capped steady state) and
// turns 48 strided planes into one stream.  "Planes" (BL = false, any V): [comp][V] resp. [mu][e][V].
template <bool BL>
__host__ __device__ __forceinline__ long long spinor_base(long long site) {   // index of component 0
    return BL ? ((site >> 5) * (12 * 32) + (site & 31)) : site;
}
template <bool BL>
__host__ __device__ __forceinline__ long long spinor_stride(long long V) { return BL ? 32 : V; }  // between components
template <int NE, bool BL>
__host__ __device__ __forceinline__ long long gauge_index(long long V, int mu, int e, long long site) {
    if (BL) return (((site >> 5) * (4 * NE)) + (mu * NE + e)) * 32 + (site & 31);
    return ((long long)(mu * NE + e)) * V + site;
}
inline size_t gauge_elems(long long V, int recon) { return (size_t)4 * (recon / 2) * (size_t)V; }

struct Lattice {
    int X, Y, Z, T;
    long long V;  // sites
};

// Epilogue of the Wilson kernel:  out = s * G (in - kappa * hop(in)) + a1*A1 + a2*A2 + a3*A3
//   G = gamma5 (g5 = 1) or the identity (g5 = 0);  hop_only: out = hop(in)  (no diagonal term, no axpy)
// A1..A3 are optional ABI spinors read at the output site only, so `out` may alias any of them.
// C = double2 (fp64, the product path) or float2 (the reduced-precision tail of the adaptive CG).
template <typename C>
struct EpilogueT {
    double s = 1.0;
    int g5 = 1;
    int hop_only = 0;
    const C* A1 = nullptr;
    const C* A2 = nullptr;
    const C* A3 = nullptr;
    double a1 = 0.0, a2 = 0.0, a3 = 0.0;
    int a_g5 = 0;  // bit k-1 set: operand A_k enters as gamma5 A_k
};
using Epilogue = EpilogueT<double2>;
using EpilogueF = EpilogueT<float2>;

}  // namespace ov

// staging of the *_host entry points (api_ops.cu::host_apply)
struct HostPipe {   // members are created on demand by api_ops.cu::host_pipe_prepare (null = not created yet)
    double2* cin[2] = {nullptr, nullptr};    // canonical input, double-buffered
    double2* cout[2] = {nullptr, nullptr};   // canonical output, double-buffered
    double2* abi_in = nullptr;
    double2* abi_out = nullptr;
    cudaStream_t h2d = nullptr, d2h = nullptr;
    cudaEvent_t start = nullptr, in_ready[2] = {nullptr, nullptr}, in_free[2] = {nullptr, nullptr},
                out_ready[2] = {nullptr, nullptr}, out_free[2] = {nullptr, nullptr};
};

struct ov_ctx {
    ov::Lattice lat{};
    double kappa = 0.0;
    int recon = 18;
    cudaStream_t stream = nullptr;
    double2* gauge = nullptr;  // see gauge_index()
    float2* gauge_f = nullptr; // fp32 copy of the links, same layout (made on first use by the adaptive CG)
    int dslash_variant = 0;    // ov_set_dslash_variant: 0 automatic, 1 gather, 2 TMA-staged
    double t_phase = -1.0;     // factor on the hop across the t boundary (ov_options::t_boundary)
    int field_dir = -1;        // background field (ov_options::field - 1), its strength q E and origin: the links already carry
    double field_qE = 0.0;     // it; the Wilson kernels need it only to rebuild the third row of 12-real t links
    int field_origin = 0;
    void* tma_state = nullptr; // tensor maps and schedule of the TMA-staged kernel (wilson_tma.cu)
    bool tma_ok = true;        // false: tma_probe failed at ov_create_ex, the context never picks the TMA-staged kernel
    std::vector<int> cg_orders;  // order used at each iteration of the last adaptive CG (negative: fp32 sweep)
    std::array<double, 12> lanczos_stats{};  // last eigensolver run: restarts, filter applies, launches, edge a, widenings, m,
                                             // then seconds: host eigensolver, filter, orthogonalisation, rotations, Rayleigh-Ritz, total
    int cg_adaptive = 0;  // ov_set_cg_adaptive: 0 off, 1 reduced orders, 2 reduced orders + fp32 sweeps
    int cg_operator = 0;  // ov_set_cg_operator: 0 gamma5 D gamma5 D, 1 chirally symmetric form 2 + gamma5 S + S gamma5
    int cg_chirality = 0; // last solve in the symmetric form: chirality of the source the solver detected (0 = none)
    int flip = 0;  // block order of the next Wilson launch (alternates)
    bool blocked = false;  // layout of spinors and links (see spinor_base)
    long long launches = 0;
    mutable std::string err;

    // polynomial
    std::vector<double> coef;
    int order = -1;
    double eps = 0.0, norm = 0.0;

    // small space (borrowed V)
    const double2* Vlow = nullptr;
    std::vector<double> lambda;
    int k = 0;
    double* d_sgn = nullptr;       // k doubles: sign(lambda_i)
    double2* d_coef = nullptr;     // k complex: c = V^+ x
    int cap_k = 0;
    double2* d_coefb = nullptr;    // batched projector: k x 2 kBatch coefficient block
    int cap_kb = 0;

    // deflation space of the multi-shift CG (borrowed W, eigenpairs of A = D_ov^+ D_ov; ov_set_deflation)
    const double2* Wdefl = nullptr;
    std::vector<double> mu_defl;

    // workspaces
    double2* ws[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    float2* wsf[4] = {nullptr, nullptr, nullptr, nullptr};  // fp32 Clenshaw vectors
    double2* wsb = nullptr;  // batched Clenshaw: 5 x kBatch spinors (b1, b2, t, x_perp, x_low)
    double2* d_partial = nullptr;  // reduction partials
    size_t partial_cap = 0;        // in double2
    double2* d_result = nullptr;   // reduced results (device)
    size_t result_cap = 0;
    double2* h_result = nullptr;   // pinned host mirror
    HostPipe host_pipe;

    // live timing (ov_timing_enable): CUDA-event pairs on ctx->stream around the two phases of an apply
    bool timing = false;
    std::vector<cudaEvent_t> ev_pool;   // recorded pairs: [2i] start, [2i+1] stop
    std::vector<int> ev_phase;          // phase of pair i: 0 = Wilson/Clenshaw sweep, 1 = projector
    std::vector<long long> ev_launches; // kernel launches inside pair i
    size_t ev_used = 0;                 // pairs in use
};

namespace ov {

int fail(const ov_ctx* ctx, int code, const char* fmt, ...);
int cuda_fail(const ov_ctx* ctx, cudaError_t e, const char* what);

#define OV_CUDA(ctx, call)                                         \
    do {                                                           \
        cudaError_t e__ = (call);                                  \
        if (e__ != cudaSuccess) return ov::cuda_fail(ctx, e__, #call); \
    } while (0)

#define OV_TRY(call)                 \
    do {                             \
        int rc__ = (call);           \
        if (rc__ != OV_OK) return rc__; \
    } while (0)

inline size_t spinor_elems(const ov_ctx* c) { return (size_t)kSpinorComplex * (size_t)c->lat.V; }

// workspace spinor i (allocated on first use)
int workspace(ov_ctx* ctx, int i, double2** out);
int ensure_reduction_buffers(ov_ctx* ctx, size_t partial_elems, size_t result_elems);

// --- kernels (launchers); all enqueue on ctx->stream and bump ctx->launches ---
// link modifications applied while the gauge field is re-laid out (ov_options: background field, Dirichlet walls)
struct GaugeMods {
    int X, Y, Z, T;
    int wall_mask;   // bit mu: links across the boundary in direction mu are zero
    int field_dir;   // -1 none; 0..2: U_t(x) *= exp(-i qE (x_dir - origin))
    double qE;
    int origin;
};
int launch_gauge_relayout(ov_ctx* ctx, const double2* canonical, const GaugeMods* mods = nullptr);
int gauge_su3_defect(ov_ctx* ctx, const double2* canonical, double* defect);
int launch_pack(ov_ctx* ctx, const double2* canonical, double2* abi);
int launch_unpack(ov_ctx* ctx, const double2* abi, double2* canonical);
int launch_wilson(ov_ctx* ctx, const double2* in, double2* out, const Epilogue& ep);
int effective_variant(const ov_ctx* ctx);  // 1 = gather, 2 = TMA-staged: what launch_wilson picks for this context
int launch_wilson_gather(ov_ctx* ctx, const double2* in, double2* out, const Epilogue& ep);
int launch_wilson_tma(ov_ctx* ctx, const double2* in, double2* out, const Epilogue& ep);   // variant 2 (wilson_tma.cu)
bool tma_eligible(const Lattice& lat);
bool tma_probe(const ov_ctx* ctx);   // tensor maps can be built for this context (needs ctx->gauge allocated); see wilson_tma.cu
void tma_state_free(ov_ctx* ctx);
// batched: nrhs consecutive ABI spinors (stride 12 V) in in/out and in every epilogue operand
int launch_wilson_batch(ov_ctx* ctx, const double2* in, double2* out, const Epilogue& ep, int nrhs);
int launch_wilson_gather_f32(ov_ctx* ctx, const float2* in, float2* out, const EpilogueF& ep);  // needs ctx->gauge_f
// host-side dense Hermitian eigensolver (Householder tridiagonalisation + implicit-shift QR): A (n x n, row-major complex,
// destroyed), w ascending, Z row-major with eigenvectors as COLUMNS; false = no convergence
bool host_eigh(int n, std::vector<double2>& A, std::vector<double>& w, std::vector<double2>& Z);

// BLAS-1 on ABI spinors (n = 12 V complex)
int launch_axpy(ov_ctx* ctx, double2 a, const double2* x, double2* y);                     // y += a x
int launch_axpby(ov_ctx* ctx, double a, const double2* x, double b, const double2* y, double2* z, int nrhs = 1);  // z = a x + b y
int launch_axpbypcz(ov_ctx* ctx, double a, const double2* x, double b, const double2* y, double c, const double2* w, double2* z);
// out = ax x + (s + gamma5) y, s = +-1 (x may be null when ax = 0): chirality-sector algebra of D_ov^+ D_ov
int launch_chiral_combine(ov_ctx* ctx, double ax, const double2* x, int s, const double2* y, double2* out);
int launch_scale(ov_ctx* ctx, double a, double2* x);
int launch_copy(ov_ctx* ctx, const double2* x, double2* y);
int launch_zero(ov_ctx* ctx, double2* x);
int launch_gamma5(ov_ctx* ctx, const double2* x, double2* y);  // y = gamma5 x (may alias)
// nvec dots <x_j, y> for j < nvec, x_j = xs + j*stride (complex results on device in ctx->d_result[0..nvec))
int launch_multi_dot(ov_ctx* ctx, const double2* xs, size_t stride, int nvec, const double2* y);
// same, results written to d_result[result_offset .. result_offset + nvec)
int launch_multi_dot_at(ov_ctx* ctx, const double2* xs, size_t stride, int nvec, const double2* y, int result_offset,
                        int result_total);
// W[j] <- sum_i S[i][j] W[i], j < ncol, in place; basis in two segments (a: na vectors, b: the rest); St = S^T on device
int launch_rotate_inplace(ov_ctx* ctx, double2* a, int na, double2* b, size_t stride, int m, int ncol,
                          const double2* St_dev);
int fetch_results(ov_ctx* ctx, int n, double2* host_out);  // sync + copy d_result[0..n) to host
int dot_host(ov_ctx* ctx, const double2* x, const double2* y, double2* out);
int norm2_host(ov_ctx* ctx, const double2* x, double* out);
// out_j = bscale_j * base + sum_{i<nvec} C[i*J+j] x_i, j < J in {1,2,4,8}; C (nvec x J complex) on the device
struct MultiAxpyOuts {
    double2* out[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    double bscale[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    const double2* basej[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};  // overrides `base` for output j
};
int launch_multi_axpy(ov_ctx* ctx, const double2* xs, size_t stride, int nvec, int J, const double2* C_dev,
                      const double2* base, const MultiAxpyOuts& o);

// fp32 helpers of the adaptive CG (blas.cu)
int launch_scale_to_f32(ov_ctx* ctx, double a, const double2* x, float2* y);   // y = (float)(a x)
int launch_combine_from_f32(ov_ctx* ctx, const float2* r, double a1, const double2* A1, double a2, const double2* A2,
                            int a2_g5, double2* out);                          // out = r + a1 A1 + a2 [gamma5] A2
int ensure_gauge_f32(ov_ctx* ctx);
int workspace_f32(ov_ctx* ctx, int i, float2** out);

int launch_multi_dot_batch(ov_ctx* ctx, const double2* xs, size_t stride, int nvec, const double2* y, size_t ystride, int nb);
bool multi_dot_batch_fits(int nvec, int nb);   // does the nb x nvec result block of launch_multi_dot_batch fit in shared memory
// projector: c = V^+ x (left in ctx->d_result[0..k)); perp = x - V c; low = V (sgn o c)
int project(ov_ctx* ctx, const double2* x, double2* perp, double2* low);
// the same for nb consecutive right-hand sides (stride 12 V) with V streamed once per pass for groups of 4 / 2 of them
int project_batch(ov_ctx* ctx, const double2* x, double2* perp, double2* low, int nb);

// live timing: a Span records an event pair on ctx->stream around a phase when ctx->timing is on
struct Span {
    ov_ctx* ctx;
    int slot = -1;
    long long launches0 = 0;
    Span(ov_ctx* c, int phase);
    ~Span();
};

// operator drivers
int sign_poly(ov_ctx* ctx, const double2* x, double2* out, const Epilogue& fin);
int apply_sign(ov_ctx* ctx, const double2* in, double2* out);
int apply_dov(ov_ctx* ctx, double mass, const double2* in, double2* out);
// nb <= kBatch right-hand sides through one batched Clenshaw sweep (gamma5_out = false: D_ov(mass); true: sign)
constexpr int kBatch = 4;
int apply_batch(ov_ctx* ctx, bool sign_only, double mass, const double2* in, double2* out, int nb);
int apply_dov_reduced(ov_ctx* ctx, double mass, const double2* in, double2* out, int order, bool f32);

}  // namespace ov
