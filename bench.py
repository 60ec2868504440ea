#!/usr/bin/env python
"""bench.py -- throughput of the iterative-PCA hot path on B200 (driver contract).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4] [--impl reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
           --master-port P bench.py --gpus N --steps K --warmup W

One "step" = one pass of the whole hot path over one seeded synthetic problem already resident
in HBM: S0 `pca_center` on a fresh copy of the raw matrix, then `pca_run` (all K components: every
inner pass S2-S8, the fused deflations S9, the epilogue S10).  The default workload is
BASELINE.json configs[3] (M=65536 x N=2048, K=128, GS-PCA, eps=1e-7): the HBM-resident
configuration the metric's HBM roofline -- and the north_star's ">= 70 % of HBM bandwidth"
target -- is quoted on (DESIGN.md section 9 says why not configs[1]); configs[1] is measured in
the same run and reported under "also".

Rank 0 prints ONE JSON line.  `--impl reference` times the CPU oracle (oracle/, as it stands) on
a bounded sample of the same workload instead (this tier's reference arm).

This file may execute oracle/ only in the `cpu_baseline` leg and under `--impl reference`.
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

from paper_0811_1081_b200 import inputs  # noqa: E402  (seeded generators only; no method arithmetic)

METRIC = "PCA components/s"
UNIT = "components/s"
WORKLOADS = {f"cfg{i + 1}": i for i in range(len(inputs.CONFIGS))}
L2_BYTES = 126 * 1024 * 1024


# ------------------------------------------------------------------------------------------------
# algorithmic bytes
# ------------------------------------------------------------------------------------------------
def bytes_per_inner_iteration(M, N, k, gs, reads_of_R=2):
    """`reads_of_R` reads of R, one read of each Gram-Schmidt panel, t and p written once and read once."""
    return 4 * reads_of_R * M * N + (4 * k * (M + N) if gs else 0) + 8 * (M + N)


def algorithmic_bytes(M, N, iters, gs):
    """SURVEY.md section 8(d), the method AS SPECIFIED (two GEMVs per inner pass = two reads of R): the
    inner iterations, + per component the extra WRITE of R of the fused deflation (4MN), + the final
    deflation pass that materialises the residual of eq. (4) (read + write, 8MN)."""
    total = 0
    for k, it in enumerate(iters):
        total += int(it) * bytes_per_inner_iteration(M, N, k, gs) + 4 * M * N
    return total + 8 * M * N


def algorithmic_bytes_single_sweep(M, N, iters, gs):
    """SURVEY.md section 8(d)/(f) F1, the restructured pass the single-sweep kernel runs (t = R p and the
    next R^T t from ONE read of R): per component it_k fused sweeps + the sweep that forms R^T t0 (4MN
    each), the write of R by the deflation fused into that sweep (4MN, k > 0), the panels and vectors as
    above; + the final deflation (8MN).  This is the model `roofline.achieved` uses for that kernel: it is
    what the kernel must move, so achieved / HBM peak stays a fraction."""
    total = 0
    for k, it in enumerate(iters):
        total += (int(it) + 1) * 4 * M * N + int(it) * ((4 * k * (M + N) if gs else 0) + 8 * (M + N))
        total += 4 * M * N if k > 0 else 0
    return total + 8 * M * N


# ------------------------------------------------------------------------------------------------
# clocks during the timed region
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """Samples SM clock and throttle reasons of one GPU through NVML every 100 ms."""

    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown",
               0x4: "sw_power_cap", 0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting"}

    def __init__(self, index):
        self.sm, self.reasons, self.max_mhz, self.power = [], set(), None, 0.0
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception as e:  # noqa: BLE001
            self._nv = None
            self.error = repr(e)

    def _loop(self):
        nv = self._nv
        while not self._stop.is_set():
            try:
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h)) if hasattr(
                    nv, "nvmlDeviceGetCurrentClocksEventReasons") else int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                for bit, name in self.REASONS.items():
                    if mask & bit:
                        self.reasons.add(name)
                self.power = max(self.power, nv.nvmlDeviceGetPowerUsage(self._h) / 1000.0)
            except Exception:  # noqa: BLE001
                pass
            self._stop.wait(0.1)

    def start(self):
        if self._nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()
        if not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "note": "NVML unavailable"}
        return {"sm_mhz": float(np.median(self.sm)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.sm), "power_w_max": round(self.power, 1)}


# ------------------------------------------------------------------------------------------------
# the CUDA arm
# ------------------------------------------------------------------------------------------------
class GpuProblem:
    """Device buffers + context of one workload (torch: memory and streams only)."""

    def __init__(self, cfg, algo, X_np, K=None, eps=None, max_iter=None, options=None):
        import torch
        from paper_0811_1081_b200 import binding
        self.torch, self.binding, self.cfg, self.algo = torch, binding, cfg, algo
        self.M, self.N = cfg.M, cfg.N
        self.K = K or cfg.K
        self.eps = cfg.eps if eps is None else eps
        self.max_iter = max_iter or cfg.max_iter
        self.ctx = binding.PcaContext(self.M, self.N, self.K, self.eps, self.max_iter, algo)
        for opt, val in (options or {}).items():                # plan overrides (--path, --ring-rows, --ring-slots)
            self.ctx.pca_set_option(opt, val)
        self.X_raw = binding.from_colmajor(X_np)
        self.X = torch.empty_like(self.X_raw)
        self.T = torch.empty((self.K, self.M), dtype=torch.float32, device="cuda")
        self.P = torch.empty((self.K, self.N), dtype=torch.float32, device="cuda")
        self.lam = torch.empty(self.K, dtype=torch.float32, device="cuda")
        self.iters = torch.empty(self.K, dtype=torch.int32, device="cuda")
        self.ctx.ensure_workspace()
        self.flush = None
        if 4 * self.M * self.N <= 2 * L2_BYTES:                 # inputs not larger than L2: flush between steps
            self.flush = torch.empty(2 * L2_BYTES, dtype=torch.uint8, device="cuda")

    def step(self):
        """Enqueue one step; returns (event pair of the step, event pair of the solve kernel)."""
        e = [self.torch.cuda.Event(enable_timing=True) for _ in range(4)]
        if self.flush is not None:
            self.flush.fill_(1)
        e[0].record()
        self.X.copy_(self.X_raw)
        self.ctx.pca_center(self.X)
        e[2].record()
        self.ctx.pca_run(self.X, self.T, self.P, self.lam, self.iters)
        e[3].record()
        e[1].record()
        return e

    def launches_per_step(self):
        return 1 + self.ctx.pca_get_info(self.binding.PCA_INFO_LAUNCHES_PER_RUN)   # pca_center + pca_run

    def gs(self):
        return self.algo == inputs.ALGO_GS


def time_steps(prob, steps, warmup):
    torch = prob.torch
    for _ in range(warmup):
        prob.step()
    torch.cuda.synchronize()
    evs = [prob.step() for _ in range(steps)]
    torch.cuda.synchronize()
    step_ms = [e[0].elapsed_time(e[1]) for e in evs]
    run_ms = [e[2].elapsed_time(e[3]) for e in evs]
    return step_ms, run_ms


# ncu --set full captures of full launches, bytes per launch: (config name, K, plan, full solve) -> dram read + write
NCU_TRAFFIC = {("cfg4_65536x2048", 128, "single-sweep streaming", True): 7708773000000 + 109641267000}


def roofline(prob, run_ms_mean, peaks):
    iters = prob.iters.cpu().numpy()
    single = "single-sweep" in prob.ctx.info()["path"]
    two_read = algorithmic_bytes(prob.M, prob.N, iters, prob.gs())
    nbytes = algorithmic_bytes_single_sweep(prob.M, prob.N, iters, prob.gs()) if single else two_read
    achieved = nbytes / (run_ms_mean * 1e-3) / 1e9
    peak = peaks["hbm_gbs"]
    total_iters = int(iters.sum())
    return {
        "bound": "hbm",
        "kernel": (("pca_reg_kernel" if "register" in prob.ctx.info()["path"] else
                    "pca_one_kernel" if "one-CTA" in prob.ctx.info()["path"] else
                    "pca_tma_kernel" if "TMA" in prob.ctx.info()["path"] else "pca_fused_kernel") if single
                   else "pca_solve_kernel") + " (persistent; all passes of all components in one launch)",
        "achieved": round(achieved, 1), "peak": peak, "peak_source": peaks["source"], "unit": "GB/s",
        "frac": round(achieved / peak, 4), "traffic": NCU_TRAFFIC.get((prob.cfg.name, prob.K, prob.ctx.info()["path"], total_iters > 0 and prob.eps > 0)),
        "traffic_note": "dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of this kernel on this workload (same seeded input, same "
                        "plan, full solve to convergence) from `ncu --set full`, profiles/r02b_ncu_full_cfg4_fullsolve.csv: 0.88 x the "
                        "single-sweep algorithmic bytes (alternate sweeps run in opposite row order and re-use the L2-resident tail); "
                        "null for workloads / plans without a capture of the full launch (fixed-work captures: profiles/README.md r02)",
        "algorithmic_bytes_per_launch": int(nbytes), "inner_iterations_per_launch": total_iters,
        "us_per_inner_iteration": round(run_ms_mean * 1e3 / max(total_iters, 1), 3),
        "bytes_model": ("single-sweep (SURVEY 8(f) F1): 4MN + [GS]4k(M+N) + 8(M+N) per inner iteration, + 4MN (R^T t0 sweep) "
                        "+ 4MN (deflation write, k>0) per component, + 8MN final deflation" if single else
                        "8MN + [GS]4k(M+N) + 8(M+N) per inner iteration, + 4MN per component, + 8MN final deflation"),
        "as_specified_two_read_model": {
            "GBps": round(two_read / (run_ms_mean * 1e-3) / 1e9, 1),
            "frac_of_hbm_peak": round(two_read / (run_ms_mean * 1e-3) / 1e9 / peak, 4),
            "note": "SURVEY 8(d) B_iter = 8MN + ...: bytes the paper's two-GEMV pass would move in the same time"},
    }, iters


def max_over_ranks(x, world, device):
    """Replicas only: the job's time is the slowest rank's.  The ONLY collective of the
    benchmark (a scalar), not of the data path; works on any backend (nccl on GPUs, gloo in the CPU tests)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    tt = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def aggregate_value(K, world, ms_per_step):
    """Whole-job throughput of `world` independent replicas of a K-component solve."""
    return world * K / (ms_per_step * 1e-3)


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return {"hbm_gbs": float(d["hbm_gbs"]), "source": "MEASURED_PEAKS.json hbm_gbs (measured copy bandwidth)"}
    return {"hbm_gbs": 6650.0, "source": "fallback 6.65 TB/s (B200_PROFILING.md; MEASURED_PEAKS.json absent)"}


def e2e_leg(prob, X_np, steps):
    """Same metric through the C-ABI call with HOST buffers: H2D of X, centring, solve, D2H of T, P, lambda, iters."""
    torch = prob.torch
    Xh = torch.from_numpy(np.ascontiguousarray(X_np.T)).pin_memory()
    Th = torch.empty((prob.K, prob.M), dtype=torch.float32).pin_memory()
    Ph = torch.empty((prob.K, prob.N), dtype=torch.float32).pin_memory()
    lh = torch.empty(prob.K, dtype=torch.float32).pin_memory()
    ih = torch.empty(prob.K, dtype=torch.int32).pin_memory()
    prob.ctx.pca_fit_host(Xh, Th, Ph, lh, ih)                   # warm-up (allocates the staging buffers)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(steps):
        prob.ctx.pca_fit_host(Xh, Th, Ph, lh, ih)               # synchronises the stream itself
    dt = (time.perf_counter() - t0) / steps
    return dt, 4 * prob.M * prob.N, 4 * prob.K * (prob.M + prob.N) + 8 * prob.K


# The bounded sample of each workload that BOTH oracle legs time (`cpu_baseline` of the CUDA arm and `--impl reference`):
# the first k_s components of the full-size problem, solved to convergence.  Components are extracted one after the
# other, so the first k_s components of the K-component solve ARE the k_s-component solve.
ORACLE_SAMPLE_K = {"cfg1": 8, "cfg2": 32, "cfg3": 2, "cfg4": 8, "cfg5": 8}


def oracle_sample(cfg, wname, algo, Xc, threads=None):
    """Time the oracle as it stands on the sample; returns (k_s, seconds, inner iterations)."""
    import oracle
    ks = min(ORACLE_SAMPLE_K[wname], cfg.K)
    n0 = oracle.num_threads()
    if threads:
        oracle.set_num_threads(threads)
    try:
        t0 = time.perf_counter()
        r = oracle.pca(Xc, ks, cfg.eps, cfg.max_iter, algo, want_residual=False)
        t = time.perf_counter() - t0
    finally:
        oracle.set_num_threads(n0)
    return ks, t, int(r.iters.sum())


def cpu_baseline_leg(cfg, wname, algo, X_np):
    """The oracle as it stands, on this box's host cores, on the bounded sample of the workload (ORACLE_SAMPLE_K): all cores,
    and -- on the first component only, to bound the time -- one thread."""
    import oracle
    Xc = oracle.center(X_np)
    ks, t, its = oracle_sample(cfg, wname, algo, Xc)
    cores = oracle.num_threads()
    oracle.set_num_threads(1)
    try:
        t0 = time.perf_counter()
        r1 = oracle.pca(Xc, 1, cfg.eps, cfg.max_iter, algo, want_residual=False)
        t1 = time.perf_counter() - t0
    finally:
        oracle.set_num_threads(cores)
    return {"value": round(ks / t, 4), "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {ks} of {cfg.K} components of {cfg.name} at full size ({its} inner iterations, "
                      f"{t:.1f} s, float64, eps={cfg.eps:g}); the same sample `--impl reference` times",
            "us_per_inner_iteration": round(t / max(its, 1) * 1e6, 1),
            "one_thread": {"value": round(1 / t1, 4), "unit": UNIT, "cores": 1,
                           "sample": f"first component only ({int(r1.iters[0])} inner iterations, {t1:.1f} s)",
                           "us_per_inner_iteration": round(t1 / max(int(r1.iters[0]), 1) * 1e6, 1)}}


def validity_leg(prob):
    """Sanity of the result of the LAST timed launch (outside the timed region; torch float64 on the device): the
    exchange protocol's status word, orthogonality, ||T_k|| = lambda_k, and the energy identity of eq. (4)."""
    torch, b = prob.torch, prob.binding
    status = prob.ctx.pca_get_info(b.PCA_INFO_RUN_STATUS)
    if status != 0:
        raise SystemExit(f"bench.py: PCA_INFO_RUN_STATUS = {status}: an exchange wait gave up, the timed result is invalid")
    K = prob.K
    I = torch.eye(K, dtype=torch.float64, device="cuda")
    Pd, Td, lam = prob.P.double(), prob.T.double(), prob.lam.double()
    live = lam > 0
    gp = float((Pd @ Pd.T - I)[live][:, live].abs().max())
    tn = Td.norm(dim=1)
    vd = Td / tn.clamp_min(1e-300)[:, None]
    gv = float((vd @ vd.T - I)[live][:, live].abs().max())
    tl = float(((tn - lam).abs() / lam.clamp_min(1e-300))[live].max())
    x2 = float((prob.X.double() ** 2).sum())
    r2 = float((prob.ctx.pca_residual().double() ** 2).sum())
    return {"run_status": status, "max_abs_PtP_minus_I": gp, "max_abs_VtV_minus_I": gv if prob.gs() else None,
            "max_rel_normT_minus_lambda": tl, "energy_identity_defect": abs(r2 - (x2 - float((lam ** 2).sum()))) / x2,
            "degenerate_components": int((~live).sum()),
            "note": "computed from the outputs of the last timed launch, after the timed region (float64 on the device); "
                    "GS-PCA bound of the north_star: max|P^T P - I| <= 1e-5"}


def pick_algo(cfg):
    return inputs.ALGO_GS if inputs.ALGO_GS in cfg.algos else cfg.algos[0]


def run_cuda_arm(args):
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    local = int(os.environ.get("LOCAL_RANK", 0))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the library has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_0811_1081_b200 import binding
    binding.load_library()

    ci = WORKLOADS[args.workload]
    cfg = inputs.config(ci)
    algo = pick_algo(cfg)
    K = args.components or cfg.K
    eps, max_iter = (0.0, args.fixed_iters) if args.fixed_iters else (cfg.eps, cfg.max_iter)
    pr = inputs.generate(cfg)                                   # replicas only: every rank solves the same seeded problem
    from paper_0811_1081_b200 import binding as _b
    plan_opts = {}
    if args.path:
        plan_opts[_b.PCA_OPT_PATH] = args.path
    if args.ring_rows:
        plan_opts[_b.PCA_OPT_RING_ROWS] = args.ring_rows
    if args.ring_slots:
        plan_opts[_b.PCA_OPT_RING_SLOTS] = args.ring_slots
    prob = GpuProblem(cfg, algo, pr.X, K=K, eps=eps, max_iter=max_iter, options=plan_opts)
    peaks = load_peaks()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        prob.step()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    t_wall = time.perf_counter()
    evs = [prob.step() for _ in range(args.steps)]
    barrier()
    t_wall = time.perf_counter() - t_wall
    clocks = sampler.stop()
    step_ms = float(np.sum([e[0].elapsed_time(e[1]) for e in evs]))
    run_ms = float(np.mean([e[2].elapsed_time(e[3]) for e in evs]))
    step_ms = max_over_ranks(step_ms, world, "cuda")
    ms_per_step = step_ms / args.steps
    value = aggregate_value(K, world, ms_per_step)
    roof, iters = roofline(prob, run_ms, peaks)
    validity = validity_leg(prob)
    if prob.gs() and not args.fixed_iters and validity["max_abs_PtP_minus_I"] > 1e-5:
        raise SystemExit(f"bench.py: the timed result is not orthogonal: {validity}")

    out = None
    if rank == 0:
        info = prob.ctx.info()
        out = {
            "metric": METRIC, "value": round(value, 3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": round(ms_per_step, 4), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {
                "workload": f"BASELINE.json configs[{ci}] {cfg.name}: M={cfg.M} N={cfg.N} K={K} "
                            f"{'GS-PCA' if algo == inputs.ALGO_GS else 'NIPALS-PCA'} eps={eps:g} max_iter={max_iter}",
                "recipe": f"{cfg.kind} {cfg.spectrum} noise_std={cfg.noise:g} seed={cfg.seed} ({cfg.note})",
                "parallelism": "replicas only (one independent problem per GPU)" if world > 1 else "single GPU",
                "l2": "input (4MN bytes) larger than L2" if prob.flush is None else "L2 flushed (252 MiB write) between steps",
                "plan": info,
            },
            "gpu_launches": args.steps * prob.launches_per_step(),
            "wall_s_timed_region": round(t_wall, 3),
            "clocks": clocks,
            "roofline": roof,
            "validity": validity,
            "inner_iterations": {"total": int(iters.sum()), "max_per_component": int(iters.max()),
                                 "hit_max_iter": int((iters >= max_iter).sum()) if not args.fixed_iters else None},
        }
    # ---- e2e: host buffers through pca_fit_host (every rank, max over ranks) ----
    if not args.no_e2e:
        dt, h2d, d2h = e2e_leg(prob, pr.X, max(1, min(args.steps, args.e2e_steps)))
        dt = max_over_ranks(dt, world, "cuda")
        if rank == 0:
            out["e2e"] = {"value": round(world * K / dt, 3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                          "d2h_bytes_per_step": d2h, "ms_per_step": round(dt * 1e3, 3),
                          "api": "pca_fit_host (pinned host X in; T, P, lambda, iters out)"}
    # ---- the other BASELINE.json configs measured beside it (seconds each; `--also cfg2` for configs[1] only) ----
    if rank == 0 and not args.no_also and not args.fixed_iters:
        del prob
        torch.cuda.empty_cache()
        out["also"] = []
        names = [w for w in ("cfg2", "cfg1", "cfg5", "cfg3") if w != args.workload and (args.also == "all" or w in args.also.split(","))]
        for wname in names:
            ca = inputs.config(WORKLOADS[wname])
            pa = inputs.generate(ca)
            for al in ca.algos if wname == "cfg3" else (pick_algo(ca),):
                q = GpuProblem(ca, al, pa.X)
                heavy = 4 * ca.M * ca.N * ca.K > (1 << 34)                  # configs 3 and 5: seconds per solve
                s_ms, r_ms = time_steps(q, 2 if heavy else 5, 1 if heavy else 3)
                roofa, ita = roofline(q, float(np.mean(r_ms)), peaks)
                single_stream = "streaming" in q.ctx.info()["path"]
                out["also"].append({
                    "workload": f"BASELINE.json configs[{WORKLOADS[wname]}] {ca.name} K={ca.K} "
                                f"{'GS-PCA' if al == inputs.ALGO_GS else 'NIPALS-PCA'} eps={ca.eps:g}",
                    "value": round(ca.K / (np.mean(s_ms) * 1e-3), 1), "unit": UNIT,
                    "ms_per_step": round(float(np.mean(s_ms)), 4), "plan": q.ctx.info()["path"],
                    "us_per_inner_iteration": roofa["us_per_inner_iteration"],
                    "inner_iterations": int(ita.sum()), "hit_max_iter": int((ita >= ca.max_iter).sum()),
                    "effective_GBps_vs_hbm": roofa["as_specified_two_read_model"]["GBps"],
                    "frac_of_hbm_peak": roofa["as_specified_two_read_model"]["frac_of_hbm_peak"],
                    "bytes_model": "as specified: two reads of R per inner iteration" +
                                   ("" if single_stream else " (R is on chip here: registers)"),
                    "single_sweep_frac_of_hbm_peak": roofa["frac"] if single_stream else None,
                    "l2": "input larger than L2" if q.flush is None else "L2 flushed between steps"})
                del q
                torch.cuda.empty_cache()
            del pa
    # ---- cpu_baseline: the oracle on this box's host cores (rank 0, N = 1 only) ----
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline_leg(cfg, args.workload, algo, pr.X)
    if rank == 0:
        print(json.dumps(out), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------------
# the reference arm (this tier: the CPU oracle, on the host cores)
# ------------------------------------------------------------------------------------------------
def run_reference_arm(args):
    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    if rank != 0:
        return
    import oracle
    ci = WORKLOADS[args.workload]
    cfg = inputs.config(ci)
    algo = pick_algo(cfg)
    pr = inputs.generate(cfg)
    times, its, ks = [], 0, 0
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        Xs = oracle.center(pr.X)                                # the step includes S0, like the CUDA arm's
        ks, _, n_it = oracle_sample(cfg, args.workload, algo, Xs)   # the same sample as the CUDA arm's cpu_baseline
        dt = time.perf_counter() - t0
        if i >= args.warmup:
            times.append(dt)
            its = n_it
    ms = float(np.mean(times)) * 1e3
    value = ks / (ms * 1e-3)
    sample = (f"each step = S0 centring + the first {ks} of {cfg.K} components of {cfg.name} at full size "
              f"({its} inner iterations), float64 oracle as it stands")
    out = {
        "impl": "reference", "metric": METRIC, "value": round(value, 4), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(ms, 3), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{ci}] {cfg.name}: M={cfg.M} N={cfg.N} K={cfg.K} "
                               f"{'GS-PCA' if algo == inputs.ALGO_GS else 'NIPALS-PCA'} eps={cfg.eps:g} max_iter={cfg.max_iter}",
                   "sample": sample},
        "gpu_launches": 0,
        "cpu_baseline": {"value": round(value, 4), "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": round(value, 4), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(out), flush=True)


# ------------------------------------------------------------------------------------------------
# Fig.-1-shaped sweep: the paper's own workload: seeded
# uniform [0,1) X, N = M/2, K = 10, eps = 1e-7, both algorithms.  Reports the GS-PCA overhead over
# NIPALS-PCA (paper: "only about 5-7 % slower") and the per-pass speed-up over the CPU oracle next to the
# paper's "about 12 times" (GTX280 vs one Phenom core, double precision; context, not a target).
# ------------------------------------------------------------------------------------------------
def run_fig1(args):
    import torch
    import oracle
    from paper_0811_1081_b200 import binding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --fig1: no CUDA device -- the library has no CPU fallback")
    torch.cuda.set_device(0)
    sizes = [int(x) for x in args.fig1_sizes.split(",")]
    rows = []
    for i, M in enumerate(sizes):
        N, K = M // 2, 10
        cfg = inputs.Config(f"fig1_{M}x{N}", M, N, K, 1e-7, 10000, (inputs.ALGO_GS, inputs.ALGO_NIPALS), "uniform",
                            seed=inputs.BASE_SEED + 100 + i, note="paper workload: uniform [0,1), N = M/2, K = 10")
        pr = inputs.generate(cfg)
        row = {"M": M, "N": N, "K": K}
        for algo, tag in ((inputs.ALGO_NIPALS, "nipals"), (inputs.ALGO_GS, "gs")):
            prob = GpuProblem(cfg, algo, pr.X)
            step_ms, run_ms = time_steps(prob, 3, 2)
            its = prob.iters.cpu().numpy()
            row[tag] = {"ms_per_solve": round(float(np.mean(step_ms)), 3), "inner_iterations": int(its.sum()),
                        "hit_max_iter": int((its >= cfg.max_iter).sum()), "plan": prob.ctx.info()["path"],
                        "us_per_inner_iteration": round(float(np.mean(run_ms)) * 1e3 / max(int(its.sum()), 1), 3)}
            # oracle: per-pass time on a bounded sample (eps = 0: exactly J passes of the first component)
            Xc = oracle.center(pr.X)
            J = max(2, min(50, int(2e8 / (M * N))))
            t0 = time.perf_counter()
            oracle.pca(Xc, 1, 0.0, J, algo, want_residual=False)
            row[tag]["oracle_us_per_inner_iteration"] = round((time.perf_counter() - t0) / J * 1e6, 1)
            row[tag]["speedup_per_pass_vs_oracle"] = round(row[tag]["oracle_us_per_inner_iteration"] /
                                                           row[tag]["us_per_inner_iteration"], 1)
            del prob
            torch.cuda.empty_cache()
        row["gs_over_nipals_time"] = round(row["gs"]["ms_per_solve"] / row["nipals"]["ms_per_solve"], 4)
        row["gs_over_nipals_per_pass"] = round(row["gs"]["us_per_inner_iteration"] / row["nipals"]["us_per_inner_iteration"], 4)
        rows.append(row)
    print(json.dumps({"fig1": rows, "oracle_cores": oracle.num_threads(), "dtype": "f32 (oracle f64)", "data": "synthetic",
                      "paper": {"speedup": "about 12x at M = 1.5e4 (GTX280 vs Phenom 9950 one core, fp64, whole solve incl. "
                                           "transfers; PAPER.md:188)", "gs_over_nipals": "5-7 % slower (PAPER.md:188)"}}),
          flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="cfg4", choices=sorted(WORKLOADS))
    ap.add_argument("--components", type=int, default=0, help="override K (profiling runs)")
    ap.add_argument("--fixed-iters", type=int, default=0, help="eps=0, max_iter=J: exactly J passes per component")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-also", action="store_true")
    ap.add_argument("--also", default="all", help="other configs measured beside the workload: all | comma list of cfg1,cfg2,cfg3,cfg5")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--path", type=int, default=0, help="PCA_OPT_PATH of the main workload (0 = the library's plan)")
    ap.add_argument("--ring-rows", type=int, default=0, help="path 7: PCA_OPT_RING_ROWS")
    ap.add_argument("--ring-slots", type=int, default=0, help="path 7: PCA_OPT_RING_SLOTS")
    ap.add_argument("--fig1", action="store_true", help="Fig.-1-shaped sweep (paper's workload) instead of the contract line")
    ap.add_argument("--fig1-sizes", default="512,1024,2048,4096,8192,15000")
    args = ap.parse_args()
    if args.fig1:
        return run_fig1(args)
    world = int(os.environ.get("WORLD_SIZE", 1))
    if args.gpus != world and args.impl == "cuda":
        if world == 1 and args.gpus > 1:
            raise SystemExit("bench.py: --gpus N > 1 must be launched with torch.distributed.run (one rank per GPU)")
    if args.impl == "reference":
        run_reference_arm(args)
    else:
        run_cuda_arm(args)


if __name__ == "__main__":
    main()
