/*
 * ov.h -- C ABI of the B200-native overlap-operator library (libov.so).
 *
 * The hot path of arXiv 1111.6288: applying D_ov = 1 + gamma5 sign(H_w), H_w = gamma5 D_w
 * (eq. 2.1), with sign(H_w) ~ Q P(Q^2), Q = H_w/||H_w|| on the "large space"
 * and the exact sign on the lowest eigenvectors of Q, the "small space".
 * Consumers/producers on the same kernels: a multi-mass CG and an eigensolver for the
 * low modes of H_w.  Readings of points the paper leaves open: DESIGN.md.
 *
 * Conventions
 *   - every call returns an int status: OV_OK or an OV_E* code; nothing throws or aborts across the ABI;
 *     ov_last_error(ctx) gives a NUL-terminated message owned by ctx (valid until the next call).
 *   - "dev" pointers are CUDA device pointers (fp64); "host" pointers are ordinary host memory.
 *   - all device work is enqueued on the cudaStream_t given to ov_create; calls that return host
 *     scalars (dot/norm, CG, Lanczos, *_host variants) synchronise that stream before returning.
 *   - in/out aliasing is forbidden for every apply call (the operator is a stencil) -> OV_EINVAL.
 *   - there is no CPU fallback: without a usable CUDA device every compute call returns OV_ECUDA.
 *
 * Lattice: dims = {X,Y,Z,T}; site index i = x + X*(y + Y*(z + Z*t)); V = X*Y*Z*T sites; directions
 * mu = 0..3 = x,y,z,t; periodic in x,y,z, antiperiodic in t (the hop between t=T-1 and t=0 carries -1).
 * gamma matrices: Hermitian chiral basis, gamma5 = diag(1,1,-1,-1) (reading G2).
 *
 * Layouts
 *   canonical gauge   complex128 [T][Z][Y][X][mu][row][col]   U_mu(x) links x -> x+mu
 *   canonical spinor  complex128 [T][Z][Y][X][spin][colour]   (= [site][12])
 *   ABI spinor        12*V complex128, site-major SoA in one of two forms, fixed per context (ov_spinor_layout):
 *                       1 "blocked" (needs V % 32 == 0): component q = 3*spin+colour of site i at complex
 *                         index ((i/32)*12 + q)*32 + i%32   -- 32-site blocks, components of a block contiguous;
 *                       0 "planes" (any V): component q of site i at q*V + i.
 *                     Which one a context uses is decided at ov_create_ex (ov_options.layout; the automatic rule is
 *                     stated there: planes where the TMA-staged Wilson kernel applies, else blocked when V % 32 == 0).
 *                     (re,im) interleaved; nrhs vectors are consecutive (stride 12*V).  Callers normally never index
 *                     it: ov_pack_spinor / ov_unpack_spinor convert canonical <-> ABI on the device, and every
 *                     BLAS-1 / projector entry point is layout-agnostic.
 */
#ifndef OV_H_
#define OV_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    OV_OK = 0,
    OV_EINVAL = 1,  /* bad argument (null, aliasing, bad dims, lambda == 0, ...)          */
    OV_ENOMEM = 2,  /* device allocation failed                                            */
    OV_ECUDA = 3,   /* CUDA runtime/driver error (message has the CUDA error string)       */
    OV_ESTATE = 4,  /* call order: e.g. ov_apply_sign before ov_set_polynomial             */
    OV_ENOCONV = 5  /* iterative routine hit its iteration limit; outputs hold the last iterate */
};

typedef struct ov_ctx ov_ctx;

/* ---- lifetime ------------------------------------------------------------------------------------
 * ov_create: builds a context for one gauge field.  gauge_dev: canonical gauge on the DEVICE; it is
 * COPIED and re-laid out (site-major SoA, row-major 3x3 per link; recon = 18 keeps all 9 complex
 * entries, recon = 12 keeps rows 0-1 and rebuilds row 2 = conj(row0 x row1) in registers, valid for
 * SU(3) links only: ov_create checks every link and returns OV_EINVAL if one is further than 1e-9 from SU(3); recon = 18
 * takes ANY complex 3x3 links, e.g. U(3) links carrying a U(1) background-field phase, or zero links
 * across a Dirichlet boundary).  The caller may free gauge_dev after the call returns (it synchronises).
 * kappa = 1/(2(m0+4)) is the Wilson hopping parameter (reading G1).
 * cuda_stream: a cudaStream_t (NULL = legacy default stream).                                        */
int ov_create(ov_ctx** out, const int dims[4], double kappa, const void* gauge_dev, int recon,
              void* cuda_stream);
/* ov_create_ex: the same with options (NULL or all-zero = ov_create).
 *   layout      0 automatic (planes when the TMA-staged Wilson kernel applies, i.e. X % 8 == 0, Y % 4 == 0, Z % 4 == 0;
 *                 else blocked when V % 32 == 0; else planes), 1 blocked (needs V % 32 == 0), 2 planes.
 *                 "Applies" is checked, not assumed: ov_create_ex builds the tensor maps of the gauge field once; if
 *                 the driver's cuTensorMapEncodeTiled is missing or refuses them, or the environment variable OV_NO_TMA
 *                 is set (to anything but "0"), the context behaves as on a lattice where the kernel does not apply
 *                 (automatic layout -> blocked when V % 32 == 0, automatic variant -> gather, variant 2 -> OV_EINVAL).
 *   t_boundary  what the hop between t = T-1 and t = 0 is multiplied by: OV_BC_ANTIPERIODIC (-1, the default of this
 *               library: north_star, reading G11), OV_BC_PERIODIC (+1), OV_BC_OPEN (0: no hop across the
 *               boundary, the Dirichlet condition in time of PAPER.md:104).
 *   wall_mask   bit mu (mu = 0, 1, 2 = x, y, z) set: Dirichlet wall in that space direction ("Dirichlet
 *               boundary conditions both in the direction of the applied electric field and time"): the links
 *               U_mu at coordinate d_mu - 1 are zero in the library's copy of the gauge field, so no hop connects
 *               coordinate d_mu - 1 and 0.  (Bit 3 is not used: the time direction is t_boundary.)
 *   field       0 = no background field; 1, 2, 3 = constant electric field along x, y, z (eq. 4.1
 *               "U_mu -> exp(-i q A_mu) U_mu"), in the gauge A_t(x) = E (x_dir - field_origin), other components zero
 *               (reading G19: the paper does not fix the gauge): the library's copy of every t link is
 *               multiplied by exp(-i field_qE (x_dir - field_origin)), field_qE = q E in lattice units.  The links
 *               are then U(3).  recon = 18 stores them whole; recon = 12 keeps rows 0-1 (with the phase) and the kernels
 *               multiply the rebuilt third row by det U = exp(-3 i field_qE (x_dir - field_origin)) (phase-tracked
 *               reconstruction), so the caller's links must be SU(3) as always with recon = 12.                       */
enum { OV_BC_ANTIPERIODIC = 0, OV_BC_PERIODIC = 1, OV_BC_OPEN = 2 };
typedef struct ov_options {
    int layout;
    int t_boundary;
    int wall_mask;
    int field;
    int field_origin;
    int reserved;    /* must be zero */
    double field_qE;
} ov_options;
int ov_create_ex(ov_ctx** out, const int dims[4], double kappa, const void* gauge_dev, int recon,
                 void* cuda_stream, const ov_options* options);
void ov_destroy(ov_ctx* ctx);
const char* ov_last_error(const ov_ctx* ctx);
size_t ov_spinor_bytes(const ov_ctx* ctx); /* 192 * V */
long long ov_volume(const ov_ctx* ctx);
int ov_spinor_layout(const ov_ctx* ctx); /* 1 = blocked, 0 = planes (see Layouts above) */
/* number of CUDA kernels this context has launched since creation (for bench.py's gpu_launches) */
long long ov_launch_count(const ov_ctx* ctx);
/* live timing for bench.py's roofline (CUDA events on the context's stream, recorded inside the calls that
 * follow): ov_timing_enable(ctx, 1) starts accumulating, ov_timing_read synchronises and returns
 * out_host[4] = { ms inside the Wilson/Clenshaw sweeps of ov_apply_sign/dov, kernel launches in them,
 *                 ms inside the small-space projector, kernel launches in it }  and resets the accumulators. */
int ov_timing_enable(ov_ctx* ctx, int on);
int ov_timing_read(ov_ctx* ctx, double* out_host);
/* selects the Wilson kernel of single-right-hand-side launches: 0 = automatic (the TMA-staged kernel where it applies,
 * see DESIGN.md section 10), 1 = gather (one thread per site, operands through L1/L2; every shape and layout),
 * 2 = TMA-staged (persistent warp-specialised kernel: cp.async.bulk.tensor into shared-memory rings, mbarrier
 * producer/consumer, an epilogue warpgroup for launches with fused axpy operands; needs the planes layout and
 * X % 8 == 0, Y % 4 == 0, Z % 4 == 0, else OV_EINVAL).  The two kernels do the same arithmetic in the same order: the
 * hopping term agrees to the last bit, results with an epilogue up to the compiler's FMA contraction (~2e-16 relative).
 * Batched (nrhs > 1) and fp32 launches always use the gather kernel. */
int ov_set_dslash_variant(ov_ctx* ctx, int variant);
/* the variant single-right-hand-side Wilson launches of this context actually use (1 or 2; never 0) */
int ov_get_dslash_variant(const ov_ctx* ctx);

/* ---- layout ------------------------------------------------------------------- */
int ov_pack_spinor(ov_ctx* ctx, const void* canonical_dev, void* abi_dev, int nrhs);
int ov_unpack_spinor(ov_ctx* ctx, const void* abi_dev, void* canonical_dev, int nrhs);

/* ---- Wilson kernel (row a2) -----------------------------------------------------
 * ov_dslash:   out = sum_mu [ s+ (1-gamma_mu) U_mu(x) in(x+mu) + s- (1+gamma_mu) U_mu(x-mu)^+ in(x-mu) ]
 * ov_apply_hw: out = H_w in = gamma5 (in - kappa * dslash(in))      (NOT divided by the norm)
 * in/out: ABI spinors on the device, nrhs of them.  nrhs > 1 here runs batched launches of the gather kernel: two
 * right-hand sides per thread block sharing the link loads.  In ov_apply_sign/ov_apply_dov nrhs > 1 shares the small-space
 * projector (the eigenvectors are streamed once per group of up to four right-hand sides); the Clenshaw
 * sweep then runs batched gather launches (up to four right-hand sides per launch) or, where the TMA-staged kernel is
 * the context's choice, one sweep per right-hand side through it (the faster of the two there).  Every right-hand side
 * gets the result of its nrhs = 1 call (to the last bit with the same kernel).                                       */
int ov_dslash(ov_ctx* ctx, const void* in, void* out, int nrhs);
int ov_apply_hw(ov_ctx* ctx, const void* in, void* out, int nrhs);

/* ---- polynomial (row a3; eq. 2.2) ----------------------------------------------------
 * ov_chebyshev_coeffs: host helper.  Fills coeffs_host[0..order] with the Chebyshev-interpolation
 *   coefficients of x^(-1/2) on [eps,1] in the basis T_j(z), z = (2x-1-eps)/(1-eps); coeffs[0] is the
 *   true T_0 coefficient (P = sum_j c_j T_j, no 1/2 applied anywhere else).
 * ov_set_polynomial: coeffs are COPIED.  order = degree n of P in x = Q^2 (2n+1 H_w applications per
 *   sign).  norm >= ||H_w|| defines Q = H_w/norm; eps > 0: P approximates x^(-1/2) on [eps,1].        */
int ov_chebyshev_coeffs(int order, double eps, double* coeffs_host);
int ov_set_polynomial(ov_ctx* ctx, const double* coeffs_host, int order, double eps, double norm);

/* ---- small space (row a4) -------------------------------------------------------
 * V_dev: k orthonormal ABI spinors, contiguous, on the device: BORROWED, never copied (it is 17-80 GB
 * at the paper's sizes); the caller keeps it alive until it is replaced, k = 0 is set, or the context
 * is destroyed.  lambda_host: the k eigenvalues of Q = H_w/norm (for the norm last set), COPIED;
 * lambda == 0 is rejected (OV_EINVAL).  k = 0 disables the small space.                              */
int ov_set_smallspace(ov_ctx* ctx, const void* V_dev, const double* lambda_host, int k);
/* test/bench hook for the projector alone: c = V^+ in (k complex, to coef_host if non-NULL),
 * perp = in - V c,  low = V (sign(lambda) o c).  perp/low: ABI spinors on the device.                 */
int ov_project(ov_ctx* ctx, const void* in, void* perp, void* low, double* coef_host);

/* ---- the operator (rows a3-a5) ----------------------------------------------------
 * ov_apply_sign: out = sum_i sign(lambda_i) v_i (v_i^+ in) + Q P(Q^2) (1 - V V^+) in
 * ov_apply_dov:  out = (1 + mass/2) in + (1 - mass/2) gamma5 sign(H_w) in     (mass = 0: eq. 2.1)
 * The *_host variants take canonical HOST spinors, copy them to the device, run the same device path
 * and copy the canonical result back (synchronous) -- the end-to-end entry point bench.py times.     */
int ov_apply_sign(ov_ctx* ctx, const void* in, void* out, int nrhs);
int ov_apply_dov(ov_ctx* ctx, double mass, const void* in, void* out, int nrhs);
/* reduced-accuracy D_ov (the building block of the adaptive CG; also a test hook): the polynomial is the
 * caller's Chebyshev series truncated to `order` <= the order set, and with use_f32 != 0 the Clenshaw sweep runs in
 * single precision (links and Clenshaw vectors in fp32; projector, in, out and the D_ov assembly stay fp64).  One RHS. */
int ov_apply_dov_reduced(ov_ctx* ctx, double mass, const void* in, void* out, int order, int use_f32);
/* test/bench hook: out = H_w in computed by the SINGLE-precision instantiation of the Wilson kernel (in is rounded to
 * fp32, the links are the fp32 copy the adaptive CG uses, the result is widened to fp64).  One right-hand side.       */
int ov_apply_hw_f32(ov_ctx* ctx, const void* in, void* out);
/* host-buffer entry points (what bench.py's e2e times): in_host / out_host are nrhs CANONICAL spinors in HOST memory; each
 * right-hand side is copied to the device, re-laid out, run through the operator, re-laid out and copied back.  With
 * nrhs > 1 the copies run on two internal copy streams (double-buffered staging), so the H2D of right-hand side r+1 and
 * the D2H of r-1 overlap the operator on r; pinned host memory is needed for that overlap (pageable memory works, copies
 * then serialise).  The call returns when out_host is complete.                                                       */
int ov_apply_hw_host(ov_ctx* ctx, const void* in_host, void* out_host, int nrhs);
int ov_apply_dov_host(ov_ctx* ctx, double mass, const void* in_host, void* out_host, int nrhs);

/* ---- BLAS-1 hooks (row a6; "vector additions and scalar products") --------------------
 * Vectors are ABI spinors on the device.  Reductions are two-stage with a fixed shape (no atomics), so
 * results are bit-reproducible from run to run.  dot = sum conj(x) y -> out_host[2] = (re, im).       */
int ov_blas_axpy(ov_ctx* ctx, double a_re, double a_im, const void* x, void* y); /* y += a x */
int ov_blas_scale(ov_ctx* ctx, double a, void* x);
int ov_blas_dot(ov_ctx* ctx, const void* x, const void* y, double* out_host);
int ov_blas_norm2(ov_ctx* ctx, const void* x, double* out_host);
/* ov_blas_dot_static: the same scalar product for callers that must not allocate device memory.
 *   Who that is: ov_blas_dot keeps its per-block partial sums in a buffer its ov_ctx gets from cudaMalloc (at ov_create
 *   and again, inside the call, when a longer vector needs a bigger one).  An application that has given all of HBM to
 *   its own pool (eigenvector sets of 17-80 GB leave no slack, so the cudaMalloc fails), or one whose other streams
 *   must not be stalled by the device-wide synchronisation cudaMalloc/cudaFree imply, cannot use that.  This entry
 *   point takes no ov_ctx and calls no cudaMalloc, cudaFree or other allocating routine: its partial sums go to a
 *   fixed 512 KiB array inside libov.so's device image, which every GPU that loads the library holds until the
 *   process exits.
 *   Arguments: x_dev, y_dev: n complex128 (re,im) each on the device, read only, may be the same pointer (norm^2);
 *   out_dev: 2 doubles ON THE DEVICE, receives (re, im) of sum_e conj(x[e]) y[e]; nothing is copied to the host and
 *   the call does not synchronise -- the result is ready when cuda_stream (a cudaStream_t, NULL = legacy default
 *   stream) reaches that point.  The GPU owning the buffers and the stream must be the current device.  n = 0 gives 0.
 *   Limit: n <= ov_blas_dot_static_max() = 33 554 432 (12 components x 2 796 202 sites; 32^3 x 64 fits).  A longer
 *   vector is rejected with OV_EINVAL before anything is launched.  Other errors: OV_EINVAL (null pointer, n < 0),
 *   OV_ECUDA.  ov_blas_dot_static_error() returns the message of the calling thread's last failed call.
 *   Same block shape and summation order as ov_blas_dot: the two agree bit for bit.
 *   First call on each device: looks up the array's device address (cudaGetSymbolAddress) and caches it; make that
 *   call before beginning any stream capture.
 *   Sharing: the one array per GPU serves every call, thread and stream and keeps the previous call's partial sums.
 *   Each call overwrites the entries it later reads, so no clearing is needed; but two calls that can be in flight on
 *   the GPU at once (different streams with no event between them) race on it and both results are undefined.
 *   Calls on one stream are ordered and safe.                                                                      */
int ov_blas_dot_static(const void* x_dev, const void* y_dev, long long n, void* out_dev, void* cuda_stream);
long long ov_blas_dot_static_max(void);
const char* ov_blas_dot_static_error(void);

/* ---- consumers -------------------------------------------------------------------------------------
 * ov_multishift_cg (row a7): solves (A + sigma_i) x_i = b, A = D_ov(0)^+ D_ov(0) applied as
 *   gamma5 D_ov gamma5 D_ov, sigma_i = m_i^2/(1 - m_i^2/4) (reading G10).  b: one ABI spinor; x: nmass
 *   ABI spinors (overwritten, initial guess 0).  Stops when the slowest system has |r| <= tol |b|.
 *   iters_out: iterations; relres_out[nmass]: TRUE relative residuals recomputed with A at the end.
 *   Returns OV_ENOCONV if maxiter was hit.
 * ov_lanczos_lowmodes (row a8): the k eigenpairs of Q = H_w/norm of smallest |lambda|,
 *   by Chebyshev-filtered thick-restart Lanczos on Q^2 followed by Rayleigh-Ritz in Q.  Needs the norm
 *   from ov_set_polynomial.  V_out_dev: k ABI spinors; lambda_out_host, resid_out_host: k values,
 *   resid_i = |Q v_i - lambda_i v_i|.  Returns OV_ENOCONV if some resid_i > tol after max_restarts.
 *   subspace = Krylov dimension m (0 = default: 2k+16, reduced to what fits in free device memory; the paper uses
 *   2.5 k); cheb_order = degree of the filter in Q^2 (paper: 100).
 *   Memory: V_out_dev itself holds the first k basis vectors during the call (its contents are scratch until the
 *   call returns); the library allocates the other m+1-k basis vectors + 2 spinors and frees them before returning.
 *   All basis rotations are done in place, so k = 200 on 32^3x64 (80.5 GB of V) fits in 180 GB.                    */
/* ov_set_cg_adaptive ("adaptive CG": lower polynomial order as the CG converges, then single precision):
 *   mode 0 (default): every operator application at full order in fp64;
 *   mode 1: at iteration j the application of A only needs relative accuracy eta_j ~ tol |b| / |r_j| (inexact-Krylov
 *           relaxation), so the series is truncated to the smallest order whose difference from the full polynomial,
 *           measured on [max(eps, 0.96 max_i lambda_i^2), 1], is below eta_j.  PRECONDITION: the small space set by
 *           ov_set_smallspace is complete below max|lambda_i| (holds every mode of Q with |lambda| < max|lambda_i|, as
 *           ov_lanczos_lowmodes returns); with an incomplete set the reduced sweeps are inaccurate on the missing modes;
 *   mode 2: mode 1, and the Clenshaw sweep runs in fp32 once eta_j is above the fp32 rounding floor.
 * The CG vectors and recurrences stay fp64; the true residuals reported at the end always use the full operator. */
int ov_set_cg_adaptive(ov_ctx* ctx, int mode);
/* the order used at each iteration of the last adaptive solve (negative = fp32 sweep); returns the iteration count */
int ov_cg_orders(const ov_ctx* ctx, int* out_host, int cap);
int ov_multishift_cg(ov_ctx* ctx, const double* masses_host, int nmass, const void* b, void* x, double tol,
                     int maxiter, int* iters_out, double* relres_out);
int ov_lanczos_lowmodes(ov_ctx* ctx, int k, double tol, int max_restarts, int cheb_order, int subspace,
                        void* V_out_dev, double* lambda_out_host, double* resid_out_host);
/* statistics of the last ov_lanczos_lowmodes / ov_lanczos_dov_lowmodes call: out_host[12] = { restart cycles, filter
 * applications (each 2*cheb_order Wilson launches), kernel launches in the call, final lower edge a of the filter window
 * [a,1] of Q^2 (modes with lambda^2 < a are amplified), times the window had to be widened (completeness guard), Krylov
 * dimension m, and where the time went, in seconds: [6] the host eigensolver of the projected matrices (device idle),
 * [7] filter applications, [8] orthogonalisation (two Gram-Schmidt passes + normalisation per step), [9] in-place
 * rotations of the basis, [10] Rayleigh-Ritz in Q and residual checks (CUDA events on the context's stream), [11] wall
 * clock of the whole call (the remainder is allocation, the first-guess Lanczos steps and host bookkeeping) }.   */
int ov_lanczos_stats(const ov_ctx* ctx, double* out_host);

/* ---- low modes of the overlap operator and deflation ("we use deflation to help speed up
 * the calculation.  This consists of computing the low lying spectrum of the overlap operator", :81 "Chebyshev order of
 * 12 ... the 100 lowest eigenmodes for the overlap operator"; reading G20) ------------------------------
 * ov_lanczos_dov_lowmodes: the k lowest eigenpairs (mu_i, w_i) of A = D_ov(0)^+ D_ov(0) in ONE chirality sector
 *   (chirality = +1 or -1, gamma5 w_i = chirality w_i), where A acts as  A_s x = 2 x + (s + gamma5) sign(H_w) x  (one
 *   sign per application; = gamma5 D_ov gamma5 D_ov up to 1 - sign^2 = O(delta)).  A commutes with gamma5 and every
 *   level 0 < mu < 4 occurs once in each sector, so the low modes of A are the union of the two sectors' runs.  Needs
 *   ov_set_polynomial (and ov_set_smallspace where the polynomial needs it).  Same driver, arguments, memory behaviour
 *   and return codes as ov_lanczos_lowmodes; cheb_order = degree of the filter in A_s (paper: 12), each filter term
 *   costs one sign(H_w).  W_out_dev: k ABI spinors; mu_out_host ascending; resid_i = |A_s w_i - mu_i w_i| <= tol.
 * ov_set_deflation: hands k orthonormal eigenpairs of A to ov_multishift_cg (W_dev is BORROWED until replaced or
 *   ov_set_deflation(ctx, NULL, NULL, 0); mu_host is copied).  The solver then returns
 *       x_i = sum_j w_j (w_j^+ b)/(mu_j + sigma_i) + [multi-shift CG on b - W W^+ b],
 *   still stopping at |r| <= tol |b| and reporting true residuals of the full systems.  PRECONDITION: the w_j are
 *   eigenvectors of the operator the CG applies (gamma5 D_ov gamma5 D_ov with the current polynomial) to within tol,
 *   i.e. eigensolver residual and polynomial error delta (the sector form differs from gamma5 D gamma5 D by
 *   1 - sign^2 = O(delta)) both <~ tol (mu_j + sigma_i): the defect of w_j enters x_i amplified by 1/(mu_j + sigma_i);
 *   otherwise the true residuals stall near max(delta, resid) |W^+ b| / min(mu + sigma) and relres_out shows it.
 *   Enforced: with a deflation space set, ov_multishift_cg returns OV_ESTATE under ov_set_cg_adaptive modes 1-2 (an
 *   inexact A re-populates the deflated directions) and OV_EINVAL if some mu_j + sigma_i <= 0 (a zero mode with mass 0:
 *   the shifted system is singular); ov_set_polynomial and ov_set_smallspace change the operator the w_j belong to and
 *   therefore CLEAR the deflation space (call ov_set_deflation again with eigenpairs of the new operator).          */
/* ov_set_cg_operator: which normal operator ov_multishift_cg inverts (reading G22).
 *   0 (default)  A  = gamma5 D_ov gamma5 D_ov, the plain D_ov^+ D_ov of reading G10: two signs per application;
 *   1            A' = 2 + gamma5 S + S gamma5, S = the library's sign(H_w).  A' = A + (1 - S^2): the same operator up to
 *                the polynomial's error delta (they coincide when S^2 = 1), but A' commutes with gamma5 EXACTLY.  So the
 *                eigenvectors ov_lanczos_dov_lowmodes returns are exact eigenvectors of A' and deflate it whatever delta
 *                is (no amplification of 1 - S^2 by 1/(mu + sigma)), and for a source of definite chirality (the other
 *                two spin components exactly zero, e.g. a point source) every CG vector keeps that chirality and one
 *                application costs ONE sign: half the work.  The solver detects the chirality of the (deflated) source
 *                itself; ov_cg_chirality returns what the last solve found (+1, -1 or 0).  True residuals are reported
 *                for A'.  Not combined with the adaptive modes (OV_ESTATE).                                           */
int ov_set_cg_operator(ov_ctx* ctx, int mode);
int ov_cg_chirality(const ov_ctx* ctx);
int ov_lanczos_dov_lowmodes(ov_ctx* ctx, int chirality, int k, double tol, int max_restarts, int cheb_order,
                            int subspace, void* W_out_dev, double* mu_out_host, double* resid_out_host);
int ov_set_deflation(ov_ctx* ctx, const void* W_dev, const double* mu_host, int k);

/* ---- host-logic test hook (no device work): eigen-decomposition of a dense n x n Hermitian matrix by the routine the
 * Lanczos driver uses once per restart cycle (Householder tridiagonalisation + implicit-shift QR, on one host core).
 * A_host: row-major (re,im) pairs, only the lower triangle is read; w_out: n ascending eigenvalues; Z_out: row-major
 * (re,im), eigenvectors as columns.  OV_ENOCONV if the QR iteration does not converge.                          */
int ov_host_eigh(int n, const double* A_host, double* w_out, double* Z_out);

#ifdef __cplusplus
}
#endif
#endif /* OV_H_ */
