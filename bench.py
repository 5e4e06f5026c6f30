"""bench.py -- D_ov applies/s on the headline workload (BASELINE.json configs[3]: 24^3x64, fp64, n = 300,
sqrt(eps) = 0.01, k = 100 low modes, 8 Gaussian sources), one process per GPU.

A "step" is ONE pass of the whole hot path over one source: small-space projector (V^+x, x - Vc, V sgn c),
the Clenshaw polynomial sign (2n+1 = 601 launches of the Wilson kernel with fused epilogues) and the D_ov
assembly (fused into the last launch)  --  `ov_apply_dov` of include/ov.h.

  python bench.py [--gpus N] [--steps K] [--warmup W]          the CUDA library (this repo)
  python bench.py --impl reference ...                          the CPU oracle on the host cores (reference arm)

Multi-GPU: the path does not shard in this build (replicas only), so --gpus N runs N
independent replicas (one per rank, each with its own sources) and reports the aggregate; no collective is on
the data path.  Timing: CUDA events on the library's stream, barrier + synchronize on both sides, max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402

METRIC = "D_ov applies/sec"
UNIT = "applies/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=8)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["b200", "reference"], default="b200")
    ap.add_argument("--config", type=int, default=3, help="index into BASELINE.json configs (3 = headline)")
    ap.add_argument("--order", type=int, default=None, help="override the Chebyshev order (testing only)")
    ap.add_argument("--k", type=int, default=None, help="override the number of low modes (testing only)")
    ap.add_argument("--recon", type=int, default=18, choices=[18, 12])
    ap.add_argument("--variant", type=int, default=0, help="dslash kernel variant (0 = automatic, 1 = gather, 2 = TMA-staged)")
    ap.add_argument("--layout", default="auto", choices=["auto", "blocked", "planes"], help="spinor/link layout (ov_options.layout)")
    ap.add_argument("--modes-file", default=None,
                    help="torch file with the low modes {V, lam}: loaded if present, else written after Lanczos")
    ap.add_argument("--lanczos-order", type=int, default=100, help="Chebyshev filter order (paper: 100)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--ref-budget-s", type=float, default=1500.0,
                    help="--impl reference: wall-clock budget for the measured oracle steps (counts are cut to fit)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cg", action="store_true")
    ap.add_argument("--no-deflation", action="store_true",
                    help="skip the deflated multi-mass CG extra (workloads.DEFLATION, 16^3x32 smooth links, ~1 min)")
    ap.add_argument("--kernels", action="store_true",
                    help="time every kernel class of the path alone (CUDA events) and print a per-kernel roofline table")
    ap.add_argument("--reps", type=int, default=0, help="with --kernels: launches per kernel class (0 = defaults)")
    return ap.parse_args()


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def workload_name(cfg, order, k):
    return (f"configs[{cfg.index}] {cfg.name} fp64, links spread {cfg.spread}, kappa {cfg.kappa}, Chebyshev order "
            f"{order}, sqrt(eps) {cfg.sqrt_eps}, k={k} low modes, {cfg.nsrc} Gaussian sources, one D_ov apply per step")


# ---------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.1)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons)}


# ---------------------------------------------------------------------------------------------- CPU oracle legs
def stand_in_modes(dims, k, seed):
    """k orthonormal stand-in vectors (Gaussian, vector i supported on the sites with index = i mod k) with
    lambda = +-0.05: the oracle cannot compute low modes at this size (O9); for TIMING the projector
    only its shape matters (the oracle loops over every element of every vector)."""
    rng = np.random.default_rng(seed)
    X, Y, Z, T = dims
    nsite = wl.volume(dims)
    V = np.zeros((k, nsite, 12), dtype=np.complex128)
    for i in range(k):
        m = len(range(i, nsite, k))
        V[i, i::k] = rng.standard_normal((m, 12)) + 1j * rng.standard_normal((m, 12))
        V[i] /= np.linalg.norm(V[i])
    lam = 0.05 * np.where(np.arange(k) % 2 == 0, 1.0, -1.0)
    return V.reshape(k, T, Z, Y, X, 4, 3), lam


class OracleRun:
    """The oracle, as it stands, on the workload itself: every step is one FULL-order D_ov apply (2 n + 1 H_w applications
    on the whole lattice + the k-mode projector), timed by the wall clock -- a measurement, not an extrapolation.
    The oracle cannot compute low modes at this size (O9): the reference arm uses k orthonormal stand-in vectors
    (timing depends only on their shape), the b200 arm's cpu_baseline leg is handed the GPU's verified modes."""

    def __init__(self, cfg, order, k, U, V=None, lam=None):
        import oracle
        from oracle import chebyshev as ch
        self.oracle = oracle
        self.cfg, self.order, self.k, self.U = cfg, order, k, U
        self.x = wl.gaussian_source(cfg.dims, wl.source_seed(cfg.index, 0))
        oracle.hw(cfg.dims, cfg.kappa, U, self.x)  # page in, spin up the OpenMP team
        t0 = time.perf_counter()
        oracle.hw(cfg.dims, cfg.kappa, U, self.x)
        self.t_hw = time.perf_counter() - t0
        self.coef = ch.cheb_coeffs(order, cfg.eps)
        self.modes = "none"
        if k > 0 and V is not None:
            self.V, self.lam, self.modes = V, lam, "the GPU Lanczos modes (verified)"
        elif k > 0:
            self.V, self.lam = stand_in_modes(cfg.dims, k, 7)
            self.modes = "orthonormal stand-in vectors (the oracle has no eigensolver at this size; only their shape matters for timing)"
        else:
            self.V, self.lam = None, None
        self.cores = oracle.num_threads()

    def estimate_s(self):
        return (2 * self.order + 1) * self.t_hw * 1.25

    def step(self):
        c = self.cfg
        t0 = time.perf_counter()
        self.oracle.dov(c.dims, c.kappa, self.U, self.coef, c.eps, c.norm, self.V, self.lam, 0.0, self.x)
        return time.perf_counter() - t0  # seconds for one full-order apply, measured

    def hw_one_thread(self):
        """oracle H_w with the OpenMP team cut to one thread (through libgomp, the oracle itself is untouched)."""
        import ctypes
        try:
            gomp = ctypes.CDLL("libgomp.so.1")
            n0 = gomp.omp_get_max_threads()
            gomp.omp_set_num_threads(1)
            t0 = time.perf_counter()
            self.oracle.hw(self.cfg.dims, self.cfg.kappa, self.U, self.x)
            dt = time.perf_counter() - t0
            gomp.omp_set_num_threads(n0)
            return wl.volume(self.cfg.dims) / dt / 1e6
        except Exception:
            return None

    def describe(self, nsteps):
        return (f"{nsteps} measured full-order oracle D_ov applies on the whole {self.cfg.name} lattice: order {self.order} "
                f"({2 * self.order + 1} H_w applies each), k = {self.k} low modes = {self.modes}; no scaling applied; "
                f"oracle H_w alone: {wl.volume(self.cfg.dims) / self.t_hw / 1e6:.2f} Msites/s on {self.cores} threads")


def run_reference(args):
    rank, world, _ = dist_env()
    if rank != 0:
        return 0
    cfg = wl.CONFIGS[args.config]
    order = args.order if args.order is not None else cfg.order
    k = args.k if args.k is not None else cfg.k
    U = wl.su3_links(cfg.dims, cfg.spread, wl.gauge_seed(cfg.index))
    run = OracleRun(cfg, order, k, U)
    # every step is a real full-order apply (~40 s at configs[3] on 16 cores); if warmup + steps would not fit the
    # budget, first the warm-up, then the step count is cut, and the line reports the counts actually run
    est = run.estimate_s()
    fit = max(2, int(args.ref_budget_s / max(est, 1e-9)))
    warmup = min(args.warmup, max(1, fit - args.steps)) if fit < args.warmup + args.steps else args.warmup
    steps = max(1, min(args.steps, fit - warmup))
    for _ in range(warmup):
        run.step()
    times = [run.step() for _ in range(steps)]
    sec = float(np.mean(times))
    value = 1.0 / sec
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": warmup, "ms_per_step": 1e3 * sec, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg, order, k), "note": "CPU oracle on host cores; rank 0 only",
                   "steps_requested": args.steps, "warmup_requested": args.warmup},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": run.cores, "kind": "oracle", "sample": run.describe(steps)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------------------------- replicas (N > 1)
def replica_source_seeds(cfg, rank):
    """Replicas work on independent sources: rank r takes source indices r*nsrc .. (r+1)*nsrc - 1."""
    return [wl.source_seed(cfg.index, rank * cfg.nsrc + j) for j in range(cfg.nsrc)]


def max_over_ranks(ms, world, device):
    """The job's time is the slowest replica's (device-timed) time."""
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(world, steps, ms):
    """Whole-job throughput: every one of the `world` replicas did `steps` applies in `ms` (max over ranks)."""
    return world * steps / (ms * 1e-3)


# ---------------------------------------------------------------------------------------------- the CUDA arm
def algorithmic_bytes_per_sign(order, V, with_low, recon=18):
    """Algorithmic HBM bytes of the 2n+1 Wilson launches of one polynomial sign: every
    launch reads the spinor (192 B/site), the 4 links of the site (576) and writes 192; the second launch of each
    Clenshaw order also reads x, b_{j+1}, b_{j+2} (the first order has no b_{j+2}); the last launch reads x and,
    with a small space, x_low."""
    base = 192 + 4 * (recon // 2) * 16 + 192   # 960 (recon 18) / 768 (recon 12)
    total = 0
    for j in range(order - 1, -1, -1):
        total += base                                   # t = Q b_{j+1}
        total += base + 192 * (2 if j == order - 1 else 3)
    total += base + 192 * (2 if with_low else 1)        # D_ov assembly in the final epilogue
    return total * V


def modes_residual(op, V, lam, norm):
    """max_i |Q v_i - lambda_i v_i|, Q = H_w/norm, recomputed with the context's own kernels."""
    worst = 0.0
    for i in range(V.shape[0]):
        r = op.apply_hw(V[i])
        op.blas_scale(1.0 / norm, r)
        op.blas_axpy(-float(lam[i]), V[i], r)
        worst = max(worst, float(np.sqrt(op.blas_norm2(r))))
    return worst


def get_low_modes(op, cfg, k, args, log):
    """The k low modes of Q: from --modes-file when it fits this context, else from the library's Lanczos.  The file holds
    V in the context's ABI layout, so it records that layout (ov_spinor_layout) beside the dims; a file written under
    another layout (or without the key) is not used.  The residuals of loaded modes are recomputed, never taken from
    the file."""
    import torch
    path = args.modes_file
    if path and os.path.exists(path):
        d = torch.load(path, map_location="cpu", weights_only=True)
        same_dims = tuple(d["dims"].tolist()) == tuple(cfg.dims)
        same_layout = "layout" in d and int(d["layout"]) == op.spinor_layout
        if d["V"].shape[0] >= k and same_dims and same_layout:
            V, lam = d["V"][:k].cuda().contiguous(), d["lam"][:k].numpy()
            resid = modes_residual(op, V, lam, cfg.norm)
            if resid <= 1e-8:
                log(f"low modes: loaded {path} (layout {op.spinor_layout}, residual recomputed: {resid:.2e})")
                return V, lam, resid, 0.0
            log(f"low modes: {path} rejected, recomputed residual {resid:.2e} > 1e-8 (other gauge field or norm?)")
        else:
            log(f"low modes: {path} not usable here (k, dims or spinor layout differ: this context has layout "
                f"{op.spinor_layout}); running Lanczos")
    t0 = time.perf_counter()
    V, lam, res, ok = op.lanczos_lowmodes(k, tol=1e-8, max_restarts=60, cheb_order=args.lanczos_order)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    log(f"low modes: Lanczos k={k} in {dt:.1f} s, max residual {res.max():.2e}, converged={ok}, "
        f"|lambda| in [{np.abs(lam).min():.5f}, {np.abs(lam).max():.5f}]")
    st = op.lanczos_stats()
    args.lanczos_stats = st      # carried to the JSON line (finish)
    log("low modes: where the time went [s]: " + ", ".join(f"{n} {v:.2f}" for n, v in st["seconds"].items())
        + f"; {st['restarts']} restart cycles, {st['filter_applies']} filter applications, Krylov dimension {st['subspace']}")
    if not ok:
        raise RuntimeError(f"Lanczos did not reach 1e-8 (max residual {res.max():.2e})")
    if path:
        torch.save({"V": V.cpu(), "lam": torch.from_numpy(lam), "resid": torch.tensor(float(res.max())),
                    "dims": torch.tensor(cfg.dims), "layout": torch.tensor(op.spinor_layout)}, path)
    return V, lam, float(res.max()), dt


def run_b200(args):
    import torch
    import torch.distributed as dist
    import paper_1111_6288_b200 as ovp
    from paper_1111_6288_b200 import build as ovbuild

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (this library has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        ovbuild.build()
    if world > 1:
        dist.barrier()
    ovp.load_library()
    log = (lambda m: print(f"[bench] {m}", file=sys.stderr, flush=True)) if rank == 0 else (lambda m: None)

    cfg = wl.CONFIGS[args.config]
    order = args.order if args.order is not None else cfg.order
    k = args.k if args.k is not None else cfg.k
    V_sites = wl.volume(cfg.dims)
    t0 = time.perf_counter()
    U = wl.su3_links(cfg.dims, cfg.spread, wl.gauge_seed(cfg.index))
    log(f"links generated in {time.perf_counter() - t0:.1f} s")
    op = ovp.Overlap(cfg.dims, cfg.kappa, U, recon=args.recon, layout=args.layout)
    if args.variant:
        op.set_dslash_variant(args.variant)
    coef = ovp.chebyshev_coeffs(order, cfg.eps)
    op.set_polynomial(coef, cfg.eps, cfg.norm)
    lanczos_s, resid = 0.0, None
    if k > 0:
        Vlow, lam, resid, lanczos_s = get_low_modes(op, cfg, k, args, log)
        op.set_smallspace(Vlow, lam)

    # sources: rank r takes its own seeds (replicas work on independent sources)
    nsrc = cfg.nsrc
    host_src = [torch.from_numpy(wl.gaussian_source(cfg.dims, sd)).pin_memory()
                for sd in replica_source_seeds(cfg, rank)]
    dev_src = [op.pack_spinor(h.cuda(non_blocking=True)) for h in host_src]
    out = op.new_spinor()
    torch.cuda.synchronize()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def timed(fn, nwarm, nstep, sampler=None):
        for i in range(nwarm):
            fn(i)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ctxm = sampler if sampler is not None else _Null()
        with ctxm:
            e0.record(op.stream)
            for i in range(nstep):
                fn(nwarm + i)
            e1.record(op.stream)
            barrier()
        return max_over_ranks(e0.elapsed_time(e1), world, "cuda")

    # ---- device-resident: the headline value
    sampler = ClockSampler(local)
    torch.cuda.cudart().cudaProfilerStart()
    op.timing_enable(False)
    for i in range(args.warmup):
        op.apply_dov(0.0, dev_src[i % nsrc], out)
    op.timing_enable(True)
    l0 = op.launch_count
    ms = timed(lambda i: op.apply_dov(0.0, dev_src[i % nsrc], out), 0, args.steps, sampler)
    launches = op.launch_count - l0
    tim = op.timing_read()
    op.timing_enable(False)
    torch.cuda.cudart().cudaProfilerStop()
    value = aggregate_value(world, args.steps, ms)

    # ---- end to end through the host-buffer entry point (H2D + D2H inside the timed region): one call per step with
    # ne2e sources; the library overlaps the copies of neighbouring sources with the operator (two copy streams)
    e2e = None
    if not args.no_e2e:
        ne2e = min(4, nsrc)
        hin = torch.stack([h for h in host_src[:ne2e]]).contiguous().pin_memory()
        hout = torch.empty_like(hin).pin_memory()
        nst = max(2, min(args.steps, 8))
        ms_e = timed(lambda i: op.apply_dov_host(0.0, hin, hout), 1, nst)
        nbytes = hin.numel() * 16
        e2e = {"value": aggregate_value(world, nst * ne2e, ms_e), "unit": UNIT, "h2d_bytes_per_step": nbytes,
               "d2h_bytes_per_step": nbytes, "steps": nst, "applies_per_step": ne2e,
               "note": f"ov_apply_dov_host(nrhs={ne2e}) from pinned host memory: every source is copied in and its result copied "
                       "out inside the timed region; copies of neighbouring sources overlap the operator"}
        del hin, hout

    # ---- the Wilson kernel alone (ping-pong, working set gauge + 2 spinors > L2), for the extra keys
    a, b = dev_src[0].clone(), op.new_spinor()
    nhw = 100
    ms_hw = timed(lambda i: op.apply_hw(a, b) if i % 2 == 0 else op.apply_hw(b, a), 10, nhw)
    del a, b
    hw_gbs = (384.0 + 32.0 * args.recon) * V_sites * nhw / (ms_hw * 1e-3) / 1e9

    # ---- the same step with 12-real links (row 3 of every SU(3) link rebuilt in registers): reported beside the headline
    recon12 = None
    if args.recon == 18 and not args.no_e2e:
        op12 = ovp.Overlap(cfg.dims, cfg.kappa, U, recon=12)
        op12.set_polynomial(coef, cfg.eps, cfg.norm)
        if k > 0:
            op12.set_smallspace(Vlow, lam)
        ne = max(2, min(args.steps, 4))
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for i in range(2):
            op12.apply_dov(0.0, dev_src[i % nsrc], out)
        barrier()
        e0.record(op12.stream)
        for i in range(ne):
            op12.apply_dov(0.0, dev_src[i % nsrc], out)
        e1.record(op12.stream)
        barrier()
        ms12 = max_over_ranks(e0.elapsed_time(e1), world, "cuda")
        recon12 = {"value": aggregate_value(world, ne, ms12), "unit": UNIT, "bytes_per_site_per_launch": 768,
                   "note": "ov_create(recon=12): 384 B/site of links instead of 576; parity <= 1e-10 (tests)"}
        op12.close()

    # ---- batched right-hand sides (reported separately, G17): 4 sources per Clenshaw sweep
    batched = None
    if not args.no_e2e and nsrc >= 4:
        xb = torch.stack(dev_src[:4]).contiguous()
        yb = torch.empty_like(xb)
        ms_b = timed(lambda i: op.apply_dov(0.0, xb, yb), 1, 2)
        batched = {"nrhs": 4, "value": aggregate_value(world, 2 * 4, ms_b), "unit": UNIT,
                   "note": "ov_apply_dov(nrhs=4): the small-space projector streams the eigenvectors once for the 4 right-hand sides; "
                           "Clenshaw sweeps per right-hand side through the TMA-staged kernel (batched gather launches elsewhere)"}
        del xb, yb

    # ---- multi-mass CG time-to-solution on the same lattice (north_star: reported beside the headline)
    cg = None
    if k > 0 and world == 1 and not args.no_cg:
        masses = wl.CONFIGS[4].masses
        bsrc = op.pack_spinor(torch.from_numpy(wl.point_source(cfg.dims)).cuda())
        cg = {"masses": list(masses), "tol": 1e-8, "source": "point"}
        for mode, name in ((0, "plain"), (2, "adaptive")):
            op.set_cg_adaptive(mode)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            xs, iters, _, okc = op.multishift_cg(masses, bsrc, tol=1e-8, maxiter=200, true_residuals=False)
            torch.cuda.synchronize()
            cg[name] = {"seconds": time.perf_counter() - t0, "iterations": iters, "converged": bool(okc)}
            if mode == 2:
                cg[name]["orders"] = op.cg_orders()
        op.set_cg_adaptive(0)
        # chirally symmetric normal operator (ov_set_cg_operator(1)): the point source is chiral, one sign per step
        op.set_cg_operator(1)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        xs, iters, _, okc = op.multishift_cg(masses, bsrc, tol=1e-8, maxiter=200, true_residuals=False)
        torch.cuda.synchronize()
        cg["symmetric"] = {"seconds": time.perf_counter() - t0, "iterations": iters, "converged": bool(okc),
                           "chirality_detected": op.cg_chirality,
                           "note": "a DIFFERENT operator from 'plain': A' = 2 + gamma5 S + S gamma5 = gamma5 D gamma5 D + (1 - S^2), i.e. O(delta) away from "
                                   "the D_ov^+ D_ov of reading G10 (DESIGN.md reading G22, the builder's option, not the paper's); "
                                   "one sign per application holds for chiral sources only (the point source here is one). "
                                   "Not a speed-up of the 'plain' solve"}
        op.set_cg_operator(0)
        del xs, bsrc
    # ---- deflated multi-mass CG on the workload built for it, reported separately
    deflation = None
    if world == 1 and not args.no_cg and not args.no_deflation and args.config == 3:
        deflation = deflation_extra(ovp, log)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0
    # the cpu_baseline leg gets the GPU's (residual-checked) low modes, copied to the host once, untimed
    modes_host = None
    if k > 0 and world == 1 and not args.no_cpu_baseline:
        X, Y, Z, T = cfg.dims
        Vh = np.empty((k, T, Z, Y, X, 4, 3), dtype=np.complex128)
        for i in range(k):
            Vh[i] = op.unpack_spinor(Vlow[i]).cpu().numpy()
        modes_host = (Vh, np.asarray(lam))
    return finish(args, cfg, order, k, V_sites, world, ms, value, launches, tim, e2e, hw_gbs, ms_hw / nhw,
                  sampler, lanczos_s, resid, U, log, cg, batched, recon12, modes_host, op.dslash_variant, deflation)


def deflation_extra(ovp, log):
    """Low modes of D_ov (per chirality sector) + deflated multi-mass CG on workloads.DEFLATION: 16^3x32, smooth links,
    periodic time (six near-zero modes of D_ov^+ D_ov per sector), 6 masses, point source, tol 1e-8."""
    import torch
    cfg = wl.DEFLATION
    U = wl.su3_links(cfg.dims, cfg.spread, wl.gauge_seed(cfg.index))
    op = ovp.Overlap(cfg.dims, cfg.kappa, U, t_boundary=wl.DEFLATION_T_BOUNDARY)
    op.set_polynomial(ovp.chebyshev_coeffs(10, 0.01), 0.01, cfg.norm)
    t0 = time.perf_counter()
    V, lam, _, ok = op.lanczos_lowmodes(16, tol=1e-9, max_restarts=60, cheb_order=100)
    se = 0.95 * float(np.max(np.abs(lam)))
    n = int(np.ceil(np.log(0.41 / 1e-12) / (2.1 * se)))          # delta ~ 1e-12 (eq. 2.2)
    op.set_polynomial(ovp.chebyshev_coeffs(n, se * se), se * se, cfg.norm)
    op.set_smallspace(V, lam)
    t_hw = time.perf_counter() - t0
    k = 12
    t0 = time.perf_counter()
    Ws, mus = [], []
    for s in (+1, -1):
        W, mu, res, ok2 = op.lanczos_dov_lowmodes(s, k, tol=1e-9, max_restarts=60, cheb_order=12)
        ok = ok and ok2
        Ws.append(W)
        mus.append(mu)
    torch.cuda.synchronize()
    t_modes = time.perf_counter() - t0
    b = op.pack_spinor(torch.from_numpy(wl.point_source(cfg.dims)).cuda())
    out = {"workload": f"{cfg.name}, spread {cfg.spread}, Chebyshev order {n}, sqrt(eps) {se:.4f}, 16 H_w modes",
           "masses": list(cfg.masses), "tol": 1e-8, "source": "point", "modes_per_sector": k, "dov_filter_order": 12,
           "hw_modes_seconds": t_hw, "dov_modes_seconds": t_modes, "modes_converged": bool(ok),
           "mu_min": float(min(m.min() for m in mus)), "mu_max": float(max(m.max() for m in mus))}
    for name, defl, mode in (("plain", False, 0), ("deflated", True, 0), ("deflated_symmetric", True, 1)):
        op.set_cg_operator(mode)
        op.set_deflation(torch.cat(Ws).contiguous() if defl else None, np.concatenate(mus) if defl else None)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        _, iters, relres, okc = op.multishift_cg(list(cfg.masses), b, tol=1e-8, maxiter=5000)
        torch.cuda.synchronize()
        out[name] = {"seconds": time.perf_counter() - t0, "iterations": iters, "converged": bool(okc),
                     "max_true_residual": float(np.max(relres)), "note": "seconds include the true-residual check (12 D_ov applies)"}
    op.set_deflation(None, None)
    op.set_cg_operator(0)
    log(f"deflation extra: {out['plain']['iterations']} -> {out['deflated']['iterations']} iterations, "
        f"{out['plain']['seconds']:.1f} -> {out['deflated']['seconds']:.1f} s ({out['deflated_symmetric']['seconds']:.1f} s in the "
        f"symmetric form), D_ov modes {t_modes:.0f} s")
    op.close()
    return out


class _Null:
    def __enter__(self):
        return self

    def __exit__(self, *a):
        return False


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(config, recon, order, kernel):
    """dram bytes per launch of the Wilson kernel from the committed `ncu --set full` summary -- only if that capture was
    taken on the same workload, link storage and kernel this run launched; otherwise None (a stale or foreign number is
    worse than none)."""
    try:
        import csv
        out = {}
        with open(os.path.join(ROOT, "profiles", "wilson_traffic.csv")) as f:
            for row in list(csv.reader(f))[1:]:
                try:
                    out[row[0]] = float(row[1])
                except ValueError:
                    out[row[0]] = row[1]
        if (int(out.get("config", -1)) != config or int(out.get("recon", -1)) != recon or int(out.get("order", -1)) != order
                or out.get("kernel") != kernel):
            return None
        return out
    except Exception:
        return None


def finish(args, cfg, order, k, V_sites, world, ms, value, launches, tim, e2e, hw_gbs, hw_ms, sampler,
           lanczos_s, resid, U, log, cg=None, batched=None, recon12=None, modes_host=None, variant_used=1, deflation=None):
    peak, peak_src = measured_peak()
    nsign = args.steps
    wl_launches = tim["wilson_launches"]
    alg_bytes = algorithmic_bytes_per_sign(order, V_sites, k > 0, args.recon) * nsign / max(1, wl_launches)  # per launch
    avg_ms = tim["wilson_ms"] / max(1, wl_launches)
    achieved = alg_bytes / (avg_ms * 1e-3) / 1e9
    kernel_name = "wilson_gather_kernel" if variant_used == 1 else "wilson_tma_kernel"
    tr = ncu_traffic(cfg.index, args.recon, order, kernel_name)
    roofline = {
        "bound": "hbm", "kernel": kernel_name + " (Wilson hopping term + fused gamma5/scale/Clenshaw-axpy epilogue)",
        "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
        "traffic": (tr or {}).get("dram_bytes_per_launch"), "peak_source": peak_src,
        "algorithmic_bytes_per_launch": alg_bytes, "avg_launch_ms": avg_ms, "launches_timed": wl_launches,
        "share_of_step": tim["wilson_ms"] / ms,
        "projector": {"ms_per_step": tim["projector_ms"] / nsign,
                      "GB/s": ((2 * k + 4) * 192.0 * V_sites) / max(1e-9, tim["projector_ms"] / nsign * 1e-3) / 1e9},
        "hw_alone": {"GB/s": hw_gbs, "frac": hw_gbs / peak, "ms": hw_ms, "GFLOP/s": 1392.0 * V_sites / (hw_ms * 1e-3) / 1e9,
                     "note": f"100 back-to-back ov_apply_hw, ping-pong, {384 + 32 * args.recon} B/site"},
    }
    cpu = None
    if not args.no_cpu_baseline and world == 1:
        run = OracleRun(cfg, order, k, U, modes_host[0] if modes_host else None, modes_host[1] if modes_host else None)
        sec = run.step()
        one = run.hw_one_thread()
        cpu = {"value": 1.0 / sec, "unit": UNIT, "cores": run.cores, "kind": "oracle", "sample": run.describe(1),
               "seconds_per_apply": sec, "hw_Msites_per_s": wl.volume(cfg.dims) / run.t_hw / 1e6,
               "hw_1thread_Msites_per_s": one}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg, order, k), "recon": args.recon, "parallelism": f"replicas x{world}",
                   "dslash_variant": variant_used, "layout": args.layout,
                   "l2": "inputs larger than L2 (gauge 510 MB + 17 GB of low modes stream every step)",
                   "low_modes": f"GPU Lanczos, max residual {resid:.1e}, {lanczos_s:.0f} s (untimed setup)" if k else "none"},
        "clocks": sampler.summary(), "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu, "lanczos": getattr(args, "lanczos_stats", None), "cg_time_to_solution": cg, "deflated_cg": deflation, "batched": batched, "recon12": recon12,
        "paper_context": "paper: ~30 CPU cores per GPU on unnamed 6 GB GPUs vs Cray XT-5 (PAPER.md:9) - context only",
    }
    print(json.dumps(line), flush=True)
    return 0


def run_kernels(args):
    """Per-kernel table: each entry point that is one kernel class, timed alone with CUDA events on the library's stream,
    algorithmic bytes as in DESIGN.md section 6 (operands of 170 MB each, so nothing lives in L2 between launches)."""
    import torch
    import paper_1111_6288_b200 as ovp
    from paper_1111_6288_b200 import build as ovbuild
    ovbuild.build()
    torch.cuda.set_device(0)
    cfg = wl.CONFIGS[args.config]
    V = wl.volume(cfg.dims)
    U = wl.su3_links(cfg.dims, cfg.spread, wl.gauge_seed(cfg.index))
    op = ovp.Overlap(cfg.dims, cfg.kappa, U, recon=18)              # automatic layout and kernel choice
    op12 = ovp.Overlap(cfg.dims, cfg.kappa, U, recon=12)
    opb = ovp.Overlap(cfg.dims, cfg.kappa, U, recon=18, layout="blocked") if V % 32 == 0 else None   # gather kernel's best layout
    peak, peak_src = measured_peak()
    k = 16  # a small stand-in basis is enough to time the projector kernels per vector
    xs = [op.pack_spinor(torch.from_numpy(wl.gaussian_source(cfg.dims, 100 + j)).cuda()) for j in range(2)]
    x, y = xs
    Vb = torch.stack([x, y] * (k // 2)).contiguous()
    Vb = Vb / torch.linalg.norm(Vb.reshape(k, -1), dim=1).reshape(k, 1, 1)
    op.set_polynomial(ovp.chebyshev_coeffs(8, cfg.eps), cfg.eps, cfg.norm)
    op.set_smallspace(Vb, np.where(np.arange(k) % 2 == 0, 0.05, -0.05))
    x4, y4 = torch.stack([x, y, x, y]).contiguous(), torch.empty(4, *x.shape, dtype=x.dtype, device=x.device)
    can = op.unpack_spinor(x)
    S = 192.0 * V  # bytes of one spinor

    def t(fn, reps):
        for _ in range(3):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(op.stream)
        for _ in range(reps):
            fn()
        e1.record(op.stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    table = {}

    def add(name, nbytes, fn, reps=50):
        ms = t(fn, args.reps if args.reps > 0 else reps)
        table[name] = {"ms": ms, "algorithmic_MB": nbytes / 1e6, "GB/s": nbytes / (ms * 1e-3) / 1e9,
                       "frac_of_measured_hbm": nbytes / (ms * 1e-3) / 1e9 / peak}

    out = torch.empty_like(x)
    torch.cuda.cudart().cudaProfilerStart()
    vname = {1: "wilson_gather", 2: "wilson_tma"}
    for v in ((2, 1) if op.dslash_variant == 2 else (1,)):
        op.set_dslash_variant(v)
        op12.set_dslash_variant(v)
        lay = "blocked" if op.spinor_layout == 1 else "planes"
        add(f"{vname[v]}<18> H_w (ov_apply_hw, {lay} layout)", 960.0 * V, lambda: op.apply_hw(x, out))
        add(f"{vname[v]}<18> hop only (ov_dslash, {lay} layout)", 960.0 * V, lambda: op.dslash(x, out))
        add(f"{vname[v]}<12> H_w (recon 12, {lay} layout)", 768.0 * V, lambda: op12.apply_hw(x, out))
        add(f"{vname[v]}<18> D_ov reduced, order 8, fp64 sweep (17 Wilson launches + projector), {lay} layout", 0.0,
            lambda: op.apply_dov_reduced(0.0, x, 8, False, out), 10)
    op.set_dslash_variant(0)
    op12.set_dslash_variant(0)
    if opb is not None and op.spinor_layout != 1:
        xb_, ob_ = opb.pack_spinor(can), opb.new_spinor()
        add("wilson_gather<18> H_w (ov_apply_hw, blocked layout)", 960.0 * V, lambda: opb.apply_hw(xb_, ob_))
    add("wilson_gather<18> batched, 4 rhs per launch", (4 * 384.0 + 576.0) * V, lambda: op.apply_hw(x4, y4), 20)
    add("axpy (ov_blas_axpy)", 3 * S, lambda: op.blas_axpy(0.5 + 0.25j, x, out))
    add("scale (ov_blas_scale)", 2 * S, lambda: op.blas_scale(1.0, out))
    add("dot1 + reduce_partials (ov_blas_dot, incl. the host synchronisation)", 2 * S, lambda: op.blas_dot(x, y))
    add("pack (ov_pack_spinor)", 2 * S, lambda: op.pack_spinor(can))
    add("unpack (ov_unpack_spinor)", 2 * S, lambda: op.unpack_spinor(x))
    add(f"projector k={k}: multi_dot + coef + multi_axpy<2> (ov_project, incl. host copy of c)", (2 * k + 4) * S,
        lambda: op.project(x), 20)
    add("D_ov reduced, order 8, fp32 sweep (17 fp32 Wilson launches + projector + conversions)", 0.0,
        lambda: op.apply_dov_reduced(0.0, x, 8, True, out), 10)
    torch.cuda.cudart().cudaProfilerStop()
    print(json.dumps({"impl": "kernels", "config": {"workload": f"configs[{cfg.index}] {cfg.name}", "sites": V},
                      "peak_GB/s": peak, "peak_source": peak_src, "kernels": table}), flush=True)
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.kernels:
        return run_kernels(args)
    return run_b200(args)


if __name__ == "__main__":
    sys.exit(main())
