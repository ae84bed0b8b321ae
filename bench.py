#!/usr/bin/env python
"""bench.py - energy points/s of the LSE+OBC hot path (S1-S7) on B200.

One "step" = one pass of the whole path (negf_pipeline_device: Sancho-Rubio decimation of both leads ->
retarded RGF -> lesser/greater RGF -> observables) over all energies of one BASELINE.json config, inputs
resident in HBM.  Headline workload: configs[4] (8 energies, n = 20, b = 2048, N = 40960: the largest
single-GPU configuration and the regime BASELINE.json's target ">= 60 % of FP64 tensor peak for block size
>= 1024" is stated on); configs[3], [2], [1] and [0] are measured in the same process and reported under
"other_configs".

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--others 3,2,1,0|none] [--impl reference]

Prints ONE JSON line (see DESIGN.md "Measurement" for every key).  Multi-GPU = energy sharding
("Each E is independent of the other"): every rank runs its own N_E energies of a
grid N times as dense, no data-path collective, weak scaling.  `--impl reference` times the CPU
oracle (oracle/, NumPy) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import gc
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "energy points/sec of RGF G^R+G^<> selected inversion incl. OBC decimation and observables"
UNIT = "energy points/s"
NOMINAL_ITERS = 24           # doublings per lead assumed by SURVEY.md 8(d) when none was measured


# ---------------------------------------------------------------------------------------------
# nominal work: units U = 8 b^3 real flops
# ---------------------------------------------------------------------------------------------
def unit_counts(n, sigma_kind, want_greater, iters_total, n_energy):
    """Returns (gemm_units, inverse_units) for ALL energies of the batch: the SURVEY 8(d) nominal
    count, lowered where the implementation executes fewer products (ballistic Sigma^<>: the
    hoisted S5 needs 3(n-1)+4 products instead of 4n-2).  Never more than nominal.
    iters_total = sum over energies and both leads of the decimation doublings done."""
    gr = 7 * n - 6 + (n - 1)                       # S3 + S4 + corner column
    gr_inv = n
    gx = (11 * n - 9) if sigma_kind == "bt" else (9 * n - 7)
    if sigma_kind == "none":
        gx -= (4 * n - 2) - min(4 * n - 2, 3 * (n - 1) + 4)
    n_x = 2 if want_greater else 1
    obs = 2                                        # Gamma_L G Gamma_R for T(E)
    per_e_gemm = (gr - gr_inv) + n_x * gx + obs
    per_e_inv = gr_inv
    # decimation: 6 products + 1 inversion per doubling, + (1 inversion + 2 products) at the end
    dec_gemm = 6 * iters_total + 2 * 2 * n_energy
    dec_inv = iters_total + 2 * n_energy
    return per_e_gemm * n_energy + dec_gemm, per_e_inv * n_energy + dec_inv


def algorithmic_bytes(wl, n_energy):
    """Algorithmic HBM bytes of one step: every requested output family written once (G^R
    3F + corner, each G^<> 2F), the retained / temporary workspace families (g, X, Y, g^x, Z, Q) written and read
    once, per-energy BT Sigma_S inputs read once; H and S are read once per batch."""
    n, b = wl.n_blocks, wl.block_size
    F = n * b * b * 16.0
    per_e = (3 + 2 + (2 if wl.want_greater else 0)) * F + b * b * 16.0 + 2 * 6 * F
    if wl.sigma_kind == "bt":
        per_e += 7 * F
    return per_e * n_energy + (4 if wl.S_diag is not None else 2) * F


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU every 50 ms through NVML."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop_evt = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
                 nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake"}
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, nm in names.items():
                    if r & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            self._stop_evt.wait(0.05)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# ---------------------------------------------------------------------------------------------
# CPU oracle arm (cpu_baseline leg and --impl reference)
# ---------------------------------------------------------------------------------------------
def _blas_threads():
    try:
        from threadpoolctl import threadpool_info
        return max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        return os.cpu_count()


def oracle_plan(config, flop_budget):
    """A bounded sample of the workload for the oracle (oracle/pipeline.solve_energy as it stands).
    Where whole energies fit the budget the sample is whole energies, evenly spread over the grid.  Where ONE
    energy alone exceeds it (configs[3-4]: 13 and 57 TFLOP per energy) the sample is a SLICE of one energy: the
    same generator at the full block size, truncated to its first n_s blocks and to it_s doublings per lead;
    it is scaled to energy points by the unit count of SURVEY.md 8(d) (every unit is one b x b x b product or
    inversion at the same b, and energies are independent).
    Returns dict(kind, wl, energies or fraction, text)."""
    from paper_2602_03438_b200 import workloads
    wl = workloads.make_workload(config)
    n, b = wl.n_blocks, wl.block_size
    U = 8.0 * b ** 3
    gu, iu = unit_counts(n, wl.sigma_kind, wl.want_greater, 2 * NOMINAL_ITERS, 1)
    per_energy = (gu + iu) * U
    if per_energy <= flop_budget:
        k = int(max(1, min(wl.n_energy, flop_budget // per_energy)))
        stride = max(1, wl.n_energy // k)
        idx = list(range(0, wl.n_energy, stride))[:k]
        return {"kind": "energies", "wl": wl, "idx": idx, "points": float(len(idx)),
                "text": f"{len(idx)} of {wl.n_energy} energies (evenly spread over the grid)"}
    n_s, it_s = 2, 2
    while True:
        gs, is_ = unit_counts(n_s + 1, wl.sigma_kind, wl.want_greater, 2 * (it_s + 1), 1)
        if (gs + is_) * U > flop_budget or n_s + 1 >= n:
            break
        n_s, it_s = n_s + 1, it_s + 1
    gs, is_ = unit_counts(n_s, wl.sigma_kind, wl.want_greater, 2 * it_s, 1)
    sw = workloads.make_workload(config, n_blocks=n_s, n_energy=1)
    sw.max_iter = it_s
    frac = (gs + is_) / (gu + iu)
    return {"kind": "slice", "wl": sw, "idx": [0], "points": frac,
            "text": f"slice of ONE energy point: the config's generator at full block size b = {b} truncated to the first "
                    f"{n_s} of {n} blocks and {it_s} doublings per lead ({gs + is_} of the {gu + iu} units of 8 b^3 flops a "
                    f"full energy point has, SURVEY 8(d), {NOMINAL_ITERS} doublings per lead assumed); scaled to energy points by that ratio"}


def oracle_run(plan):
    """Runs the sample once; returns (energy-point equivalents, seconds)."""
    from oracle import pipeline
    wl = plan["wl"]
    t0 = time.perf_counter()
    for k in plan["idx"]:
        pipeline.solve_energy(wl, k, want_greater=wl.want_greater)
    return plan["points"], time.perf_counter() - t0


def run_reference(args, rank, world):
    if rank != 0:
        return
    plan = oracle_plan(args.config, args.ref_tflop * 1e12)
    wl_name = _config_row(args.config)
    total_p, total_t = 0.0, 0.0
    for i in range(args.warmup + args.steps):
        p, t = oracle_run(plan)
        if i >= args.warmup:
            total_p += p; total_t += t
    threads = _blas_threads()
    v = total_p / total_t
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total_t / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl_name[0], "n_energy": wl_name[1], "n_blocks": wl_name[2], "block_size": wl_name[3],
                   "sample": plan["text"]},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": plan["text"]},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def _config_row(config):
    from paper_2602_03438_b200 import workloads
    return workloads._CONFIG_TABLE[config]


# ---------------------------------------------------------------------------------------------
# GPU arm
# ---------------------------------------------------------------------------------------------
class Resident:
    """One workload resident on one GPU in equal energy batches; step() = one pass of the whole path over all of
    its energies through negf_pipeline_device (runner.DevicePath.run)."""

    def __init__(self, wl, ctx, dev, torch, runner, energy_batch=0):
        self.wl, self.ctx, self.torch = wl, ctx, torch
        free = torch.cuda.mem_get_info(torch.device(dev).index or 0)[0]
        nb = energy_batch or default_energy_batch(wl, free)
        nb = min(nb, wl.n_energy)
        nb = -(-wl.n_energy // -(-wl.n_energy // nb))              # equal batches: ceil(N_E / ceil(N_E / fit))
        self.ne_batch = nb
        self.batches = [(lo, min(lo + nb, wl.n_energy)) for lo in range(0, wl.n_energy, nb)]
        # one resident DevicePath per distinct batch size; Sigma_S of the FIRST batch of that size is reused for
        # the others when it is a per-energy BT family (configs[3]; stated in config.note)
        self.paths = {}
        for lo, hi in self.batches:
            if hi - lo not in self.paths:
                self.paths[hi - lo] = runner.DevicePath(wl, lo, hi, device=dev, ctx=ctx)
        self.energies = {(lo, hi): torch.from_numpy(wl.energies[lo:hi].copy()).to(dev) for lo, hi in self.batches}
        self.weights = {(lo, hi): torch.from_numpy(wl.weights[lo:hi].copy()).to(dev) for lo, hi in self.batches}

    def step(self):
        for lo, hi in self.batches:
            dp = self.paths[hi - lo]
            if len(self.batches) > 1:
                dp.energy.copy_(self.energies[(lo, hi)]); dp.weights.copy_(self.weights[(lo, hi)])
                dp.ctx.set_workspace(dp.workspace)
            dp.run()

    def last(self):
        lo, hi = self.batches[-1]
        return self.paths[hi - lo]

    def release(self):
        self.paths.clear(); self.energies.clear(); self.weights.clear()
        self.ctx.set_workspace(None)
        gc.collect(); self.torch.cuda.empty_cache()


def timed_steps(torch, res, flush, steps, warmup, barrier):
    """W warm-ups, then K steps timed one by one with CUDA events on the current stream (the stream the library
    launches on), an L2 flush (256 MB write) between them outside the event pairs.  Returns (sum of ms, launches)."""
    for _ in range(warmup):
        res.step(); flush.zero_()
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    l0 = res.ctx.launch_count()
    for i in range(steps):
        ev[i][0].record(); res.step(); ev[i][1].record()
        flush.zero_()
    barrier()
    return sum(a.elapsed_time(b) for a, b in ev), res.ctx.launch_count() - l0


def work_accounting(wl, res, steps, launches, gemm_3m, args_groups=0):
    """Decimation iteration statistics of the last step, unit counts and the launch count of one timed region."""
    dp = res.last()
    o = dp.out
    bad = int((o["info_r"] != 0).sum() + (o["info_x"] != 0).sum() + (o["status_L"] != 0).sum() + (o["status_R"] != 0).sum())
    iters_mean = float((o["iters_L"].double().sum() + o["iters_R"].double().sum()) / (2 * dp.ne))
    iters_total = iters_mean * 2 * wl.n_energy
    # The doublings run inside a device-driven WHILE graph (one host launch per group and lead batch), except in the
    # resident regime of NEGF_OPT_FUSED_SMALL: its kernels are counted from the iteration counters, body executions x
    # kernels per body (negf_obc_graph_kernels: 9 for b <= 96 = 2 x [inverse, 2 grouped GEMMs, step] + loop condition;
    # the ~300 launches of two blocked inverses above).  Both leads are one batch up to b = 128, two graph launches above.
    resident = wl.block_size <= 16 or (wl.block_size <= 32 and res.ne_batch <= 148)     # fused_small.cuh:fused_small_regime
    body = 0 if resident else res.ctx.obc_graph_kernels()
    if body > 0:
        itl, itr = int(o["iters_L"].max()), int(o["iters_R"].max())
        execs = -(-max(itl, itr) // 2) if wl.block_size <= 128 else -(-itl // 2) + -(-itr // 2)
        groups = args_groups or (4 if (wl.block_size <= 96 and res.ne_batch >= 32) else 1)
        launches += steps * len(res.batches) * groups * execs * body
    gemm_u, inv_u = unit_counts(wl.n_blocks, wl.sigma_kind, wl.want_greater, iters_total, wl.n_energy)
    if gemm_3m and wl.block_size > 64:
        gemm_u *= 0.75                      # executed DMMA flops of a 3M product: 6 b^3 instead of 8 b^3
    return bad, iters_mean, gemm_u, inv_u, int(launches)


def profile_classes(torch, negf, res, flush, psteps):
    """Per-kernel-class device time of `psteps` passes of the SAME step on the SAME context (negf_profile_*: one
    event per class change on the library's stream; plain launches on the caller's stream)."""
    c = res.ctx
    c.profile_enable(True)
    for k in range(5):
        c.profile_read(k, True)
    for _ in range(psteps):
        res.step(); flush.zero_()
    torch.cuda.synchronize()
    prof = {negf.PROF_NAMES[k]: c.profile_read(k, True) for k in range(5)}
    c.profile_enable(False)
    return prof


def run_gpu(args, rank, local_rank, world):
    import torch
    from paper_2602_03438_b200 import build as _build
    _build.ensure_built()
    from paper_2602_03438_b200 import negf, runner, workloads

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(dev))

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    ctx = negf.Context(local_rank)
    ctx.set_stream(torch.cuda.current_stream().cuda_stream)
    if args.gemm_3m:
        ctx.set_option(negf.OPT_GEMM_3M, 1)
    if args.energy_groups:
        ctx.set_option(negf.OPT_ENERGY_GROUPS, args.energy_groups)
    if args.pdl >= 0:
        ctx.set_option(negf.OPT_PDL, args.pdl)
    if args.graph_loops >= 0:
        ctx.set_option(negf.OPT_GRAPH_LOOPS, args.graph_loops)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2
    peak = ctx.fp64_peak(300.0)
    hbm_peak, hbm_src = measured_hbm_peak()

    wl = workloads.shard_energies(workloads.make_workload(args.config), rank, world)   # grid `world` times as dense
    res = Resident(wl, ctx, dev, torch, runner, args.energy_batch)
    sampler = ClockSampler(local_rank)
    for _ in range(args.warmup):
        res.step(); flush.zero_()
    barrier()
    sampler.start()
    ms, launches = timed_steps(torch, res, flush, args.steps, 0, barrier)
    clocks = sampler.stop()
    if dist is not None:
        t = torch.tensor([ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    value = world * wl.n_energy * args.steps / (ms * 1e-3)
    step_ms = ms / args.steps
    bad, iters_mean, gemm_u, inv_u, launches = work_accounting(wl, res, args.steps, launches, args.gemm_3m, args.energy_groups)
    U = 8.0 * wl.block_size ** 3
    groups = "auto (4 for b <= 96 and N_E >= 32, else 1)" if not args.energy_groups else args.energy_groups
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": wl.name, "n_energy": wl.n_energy, "n_blocks": wl.n_blocks,
                      "block_size": wl.block_size, "energy_batch": res.ne_batch, "sigma_s": wl.sigma_kind,
                      "outputs": "G^R diag/upper/lower/corner, G^< diag/upper" + (", G^> diag/upper" if wl.want_greater else "")
                                 + ", density, LDOS, T(E), bond/contact currents",
                      "l2": "256 MB flush write between timed iterations (outside the event pairs)",
                      "parallelism": f"energy-sharded x{world}, no collective",
                      "api": "negf_pipeline_device, one call per energy batch", "energy_groups": groups,
                      "complex_gemm": "3M" if (args.gemm_3m and wl.block_size > 64) else "4M",
                      "decimation_iters_mean": iters_mean, "numerical_failures": bad},
           "gpu_launches": launches, "clocks": clocks,
           "nominal_tflops": (gemm_u + inv_u) * U / (step_ms * 1e-3) * 1e-12}
    out["frac_of_fp64_peak"] = out["nominal_tflops"] / peak
    if len(res.batches) > 1 and wl.sigma_kind == "bt":
        out["config"]["note"] = "BT Sigma_S arrays of the first energy batch are reused for every batch"

    if rank == 0:
        print(f"[bench] timed region: {step_ms:.3f} ms/step, {value:.4g} {UNIT}, {out['frac_of_fp64_peak']:.3f} of FP64 peak",
              file=sys.stderr, flush=True)
        # ---- roofline of the dominant kernel: profiled passes of the SAME step on the SAME context and stream.
        # At b > 128 the timed region itself is one stream of plain launches, so this IS its launch configuration;
        # in the small-block regime profiling runs the groups one after the other (stated in `measured`).
        psteps = 1 if step_ms > 1500 else max(1, min(3, args.steps))
        prof = profile_classes(torch, negf, res, flush, psteps)
        out["roofline"] = roofline_entry(wl, prof, psteps, step_ms, gemm_u, inv_u, peak, hbm_peak, hbm_src)
        # ---- end to end through the host-buffer C-ABI call (pinned host memory, copies timed)
        res.release()
        if not args.no_e2e:
            out["e2e"] = run_e2e(args, wl, ctx, dev, world, torch, negf)
        # ---- the other configurations, same process, short runs
        others = {}
        if world == 1 and args.others != "none":
            for c in [int(x) for x in args.others.split(",") if x.strip() != ""]:
                if c == args.config:
                    continue
                try:
                    others[f"configs[{c}]"] = run_other(args, c, ctx, dev, torch, negf, runner, workloads, flush, peak,
                                                        hbm_peak, hbm_src)
                except Exception as exc:              # a failing side measurement must not lose the headline
                    others[f"configs[{c}]"] = {"error": repr(exc)[:300]}
        out["other_configs"] = others
        # ---- CPU oracle on a bounded sample of the same workload
        if args.cpu_seconds > 0:
            plan = oracle_plan(args.config, args.ref_tflop * 1e12)
            p, t = oracle_run(plan)
            out["cpu_baseline"] = {"value": p / t, "unit": UNIT, "cores": _blas_threads(), "kind": "oracle",
                                   "sample": plan["text"] + f"; {t:.1f} s, NumPy/OpenBLAS complex128"}
        print(json.dumps(out))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def roofline_entry(wl, prof, psteps, step_ms, gemm_u, inv_u, peak, hbm_peak, hbm_src):
    U = 8.0 * wl.block_size ** 3
    tot = sum(v[0] for v in prof.values()) or 1.0
    gemm_ms, gemm_sites = prof["gemm"]
    fused_ms, fused_sites = prof["fused"]
    if fused_ms > gemm_ms:
        dom, dom_ms, dom_sites, dom_flops = "fused", fused_ms, fused_sites, (gemm_u + inv_u) * U * psteps
    else:
        dom, dom_ms, dom_sites, dom_flops = "gemm", gemm_ms, gemm_sites, gemm_u * U * psteps
    achieved = dom_flops / (dom_ms * 1e-3) * 1e-12 if dom_ms > 0 else 0.0
    r = {"bound": "tensor", "kernel": {"gemm": "zgemm_kernel (DMMA.8x8x4, 4M complex)", "fused": "fused chain kernels"}[dom],
         "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
         "traffic": roofline_traffic(wl.name)[0], "traffic_source": roofline_traffic(wl.name)[1],
         "peak_source": "negf_fp64_peak: DMMA m8n8k4 issue-rate probe run in this process "
                        "(MEASURED_PEAKS.json has no FP64 figure; nominal 37.2 = 148 SM x 1.965 GHz x 128 flop/clk)",
         "flops_per_launch": dom_flops / max(dom_sites, 1),
         "avg_launch_us": 1e3 * dom_ms / max(dom_sites, 1), "launches_per_step": dom_sites / psteps,
         "kernel_ms_per_step": dom_ms / psteps,
         # the dominant kernel's summed time must fit inside the timed step it is said to explain
         "fits_in_step": bool(dom_ms / psteps <= step_ms * 1.02),
         "share_of_step": {k: v[0] / tot for k, v in prof.items()},
         "profiled_ms_per_step": tot / psteps,
         "measured": f"{psteps} profiled pass(es) of the same step on the same context and stream after the timed region"
                     + ("" if wl.block_size > 128 else "; small-block regime: profiling serialises the energy groups, side streams and graphs")}
    # HBM side of the same step (north_star: 'HBM GB/s for the small-block regime')
    nbytes = algorithmic_bytes(wl, wl.n_energy)
    r["hbm_gbs"] = nbytes / (step_ms * 1e-3) * 1e-9
    r["hbm_frac"] = r["hbm_gbs"] / hbm_peak
    r["hbm_peak"] = hbm_peak
    r["hbm_peak_source"] = hbm_src
    r["algorithmic_bytes_per_step"] = nbytes
    return r


def run_other(args, c, ctx, dev, torch, negf, runner, workloads, flush, peak, hbm_peak, hbm_src):
    """Short measurement of another BASELINE.json config in the same process (same timing rules)."""
    wl = workloads.make_workload(c)
    res = Resident(wl, ctx, dev, torch, runner)
    # few steps where a step takes seconds, the requested number where it takes milliseconds
    res.step(); torch.cuda.synchronize()
    t0 = time.perf_counter(); res.step(); torch.cuda.synchronize()
    est = time.perf_counter() - t0
    steps = max(1, min(args.steps, int(20.0 / max(est, 1e-4))))
    warm = 3 if est < 1.0 else 1
    ms, launches = timed_steps(torch, res, flush, steps, warm, torch.cuda.synchronize)
    step_ms = ms / steps
    bad, iters_mean, gemm_u, inv_u, launches = work_accounting(wl, res, steps, launches, args.gemm_3m, args.energy_groups)
    U = 8.0 * wl.block_size ** 3
    nominal = (gemm_u + inv_u) * U / (step_ms * 1e-3) * 1e-12
    prof = profile_classes(torch, negf, res, flush, 1)
    roof = roofline_entry(wl, prof, 1, step_ms, gemm_u, inv_u, peak, hbm_peak, hbm_src)
    res.release()
    return {"workload": wl.name, "n_energy": wl.n_energy, "n_blocks": wl.n_blocks, "block_size": wl.block_size,
            "energy_batch": res.ne_batch, "steps": steps, "warmup": warm + 2, "ms_per_step": step_ms,
            "value": wl.n_energy / (step_ms * 1e-3), "unit": UNIT, "nominal_tflops": nominal,
            "frac_of_fp64_peak": nominal / peak, "gpu_launches_per_step": launches // steps,
            "decimation_iters_mean": iters_mean, "numerical_failures": bad,
            "roofline": {k: roof[k] for k in ("kernel", "achieved", "frac", "avg_launch_us", "launches_per_step",
                                              "fits_in_step", "share_of_step", "hbm_gbs", "hbm_frac")}}


def measured_hbm_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (copy bandwidth, burst)"
    except Exception:
        return 6650.0, "fallback of /opt/skills/guides/B200_PROFILING.md (MEASURED_PEAKS.json absent)"


def roofline_traffic(workload):
    """(DRAM bytes per launch of the dominant kernel, which launch and capture) from the committed ncu capture
    of this workload (profiles/roofline_traffic.csv), or (None, None) when none was taken."""
    import csv
    try:
        with open(os.path.join(ROOT, "profiles", "roofline_traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload:
                    return float(row["bytes_per_launch"]), f'{row["kernel"]}: {row["source"]}'
    except OSError:
        pass
    return None, None


def default_energy_batch(wl, free_bytes):
    """Energies resident at once: outputs (G^R 3F + corner, G^< 2F, G^> 2F) + workspace (g, X, Y, g^x, Z, Q =
    6F, + 2F when the off-diagonal blocks of A are assembled, + 13 scratch blocks + K1 scratch) + BT Sigma_S
    inputs (7F), kept under 85 % of free HBM."""
    n, b = wl.n_blocks, wl.block_size
    blk = b * b * 16
    F = n * blk
    assembled = wl.S_diag is not None or wl.sigma_kind == "bt"
    per_e = (3 + 2 + (2 if wl.want_greater else 0)) * F + 6 * blk          # outputs + boundary blocks
    per_e += (6 + (2 if assembled else 0)) * F + 13 * blk * (2 if b <= 128 else 1) + (128 + 64) * b * 16
    if wl.sigma_kind == "bt":
        per_e += 7 * F
    return max(1, int(0.85 * free_bytes // per_e))


def run_e2e(args, wl, ctx, dev, world, torch, negf):
    """negf_pipeline_host on the first energy batch that fits, HOST (pinned) inputs and outputs."""
    from paper_2602_03438_b200 import runner
    n, b = wl.n_blocks, wl.block_size
    ne = min(wl.n_energy, args.e2e_energies or wl.n_energy)
    F = n * b * b * 16
    cap = 24e9                                # pinned host memory: at most 48 GB and 30 % of what the box has free
    try:
        import psutil
        cap = min(48e9, 0.3 * psutil.virtual_memory().available)
    except Exception:
        pass
    while ne > 1 and ne * F * 12 > cap:
        ne //= 2
    hp = None
    while hp is None:
        try:
            hp = runner.HostPath(wl, ne, device=dev, ctx=ctx)
            up, down = hp.run()
        except (RuntimeError, MemoryError):   # pinned or device allocation refused: fewer energies per call
            hp = None
            gc.collect(); torch.cuda.empty_cache()
            if ne == 1:
                raise
            ne //= 2
    torch.cuda.synchronize()
    t0 = time.perf_counter(); up, down = hp.run(); est = time.perf_counter() - t0
    reps = max(1, min(args.steps, 5, int(15.0 / max(est, 1e-4))))
    t0 = time.perf_counter()
    for _ in range(reps):
        up, down = hp.run()            # synchronises the stream before returning
    dt = time.perf_counter() - t0
    assert int(hp.out["info"].abs().sum()) == 0, "numerical failure flagged in the e2e run"
    # same call with the G block outputs NULL: only density, LDOS, T(E), currents and info cross PCIe on the way back
    del hp                                   # its pinned buffers and device scratch first (configs[3-4] fill the box)
    gc.collect(); torch.cuda.empty_cache()
    ho = runner.HostPath(wl, ne, device=dev, ctx=ctx, blocks=False)
    for _ in range(2):
        up_o, down_o = ho.run()
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    for _ in range(reps):
        up_o, down_o = ho.run()
    dt_o = time.perf_counter() - t1
    del ho
    gc.collect(); torch.cuda.empty_cache()
    obs_only = {"value": world * ne * reps / dt_o, "unit": UNIT, "h2d_bytes_per_step": int(up_o),
                "d2h_bytes_per_step": int(down_o), "ms_per_call": 1e3 * dt_o / reps}
    return {"value": world * ne * reps / dt, "observables_only": obs_only, "unit": UNIT, "h2d_bytes_per_step": int(up), "d2h_bytes_per_step": int(down),
            "energies_per_call": ne, "calls_timed": reps, "ms_per_call": 1e3 * dt / reps,
            "api": "negf_pipeline_host (host pinned buffers in, all selected G blocks + observables out)"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json configs index of the headline workload (default 4)")
    ap.add_argument("--others", default="3,2,1,0", help="configs also measured (short runs) and reported under other_configs; 'none' skips them")
    ap.add_argument("--gemm-3m", action="store_true",
                    help="3M complex products in the compute-bound regime (NEGF_OPT_GEMM_3M); flops are then counted as executed (x 0.75 per product)")
    ap.add_argument("--energy-groups", type=int, default=0, help="NEGF_OPT_ENERGY_GROUPS (0 = the library's automatic choice)")
    ap.add_argument("--graph-loops", type=int, default=-1, help="NEGF_OPT_GRAPH_LOOPS (-1 = the library's default)")
    ap.add_argument("--pdl", type=int, default=-1, help="NEGF_OPT_PDL (-1 = the library's default)")
    ap.add_argument("--energy-batch", type=int, default=0, help="energies resident at once (0 = fit HBM)")
    ap.add_argument("--e2e-energies", type=int, default=0)
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="0 skips the cpu_baseline leg")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg (developer runs)")
    ap.add_argument("--ref-tflop", type=float, default=4.5,
                    help="oracle sample size per step in TFLOP of nominal work (--impl reference and cpu_baseline)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_gpu(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
