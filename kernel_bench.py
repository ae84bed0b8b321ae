"""Micro-benchmarks of the K1/K2 building blocks through the C ABI:

    python kernel_bench.py --kernel zgemm --b 1024 --batch 16 [--opA 0 --opB 1]
    python kernel_bench.py --kernel zinv  --b 1024 --batch 16 [--inv-panel 0]
    python kernel_bench.py --kernel peak
    python kernel_bench.py --kernel chain --b 16 --n-blocks 8 --batch 1 [--fused 0]     # the four C-ABI calls, one by one

Prints one JSON line per run: achieved FP64 TFLOP/s (8 b^3 real flops per complex product or
inversion, the unit U of SURVEY.md 8(d)) and the fraction of the DMMA issue-rate peak probed in
the same process.  Timing: CUDA events on the library's stream, 3 warm-ups, operands rotated over
several buffers so consecutive launches do not reuse L2 lines when the set is larger than L2.
"""
from __future__ import annotations

import argparse
import json

import torch

import os
import sys

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
from paper_2602_03438_b200 import build as _build  # noqa: E402

_build.ensure_built()
from paper_2602_03438_b200 import negf  # noqa: E402


def _rand(shape, gen):
    return torch.complex(torch.randn(shape, dtype=torch.float64, device="cuda", generator=gen),
                         torch.randn(shape, dtype=torch.float64, device="cuda", generator=gen))


def chain(args):
    """Latency of the path's C-ABI calls one by one (CUDA events around each call, median of --reps) on a configs[0]-
    shaped (--batch 1) or configs[1]-shaped workload of block size --b: the view of the resident small-block regime
    (fused_small.cu), where one call is one launch."""
    from paper_2602_03438_b200 import runner, workloads
    wl = workloads.make_workload(0 if args.batch == 1 else 1, n_blocks=args.n_blocks, block_size=args.b,
                                 **({} if args.batch == 1 else {"n_energy": args.batch}))
    dp = runner.DevicePath(wl, want_greater=True)
    dp.ctx.set_option(negf.OPT_FUSED_SMALL, args.fused)
    if args.pdl >= 0:
        dp.ctx.set_option(negf.OPT_PDL, args.pdl)
    if args.energy_groups:
        dp.ctx.set_option(negf.OPT_ENERGY_GROUPS, args.energy_groups)
    calls = [("obc_decimate_pair", dp.obc), ("rgf_retarded", dp.retarded), ("rgf_lesser_greater", dp.lesser_greater),
             ("observables", dp.observables), ("pipeline_device", dp.run)]
    for _ in range(3):
        dp.run_four_calls(); dp.run()
    torch.cuda.synchronize()
    out = {"kernel": "chain", "workload": wl.name if hasattr(wl, "name") else "", "b": args.b, "n_blocks": args.n_blocks,
           "n_energy": wl.n_energy, "fused_small": args.fused, "pdl": args.pdl, "energy_groups": args.energy_groups, "us_median": {}, "launches": {}}
    for name, fn in calls:
        ts = []
        n0 = dp.ctx.launch_count()
        for _ in range(args.reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); fn(); e1.record(); torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e3)
        out["us_median"][name] = round(sorted(ts)[len(ts) // 2], 1)
        out["launches"][name] = (dp.ctx.launch_count() - n0) // args.reps
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--kernel", default="zgemm", choices=["zgemm", "zinv", "peak", "econv", "chain"])
    ap.add_argument("--b", type=int, default=1024)
    ap.add_argument("--batch", type=int, default=16)
    ap.add_argument("--opA", type=int, default=0)
    ap.add_argument("--opB", type=int, default=0)
    ap.add_argument("--reps", type=int, default=10)
    ap.add_argument("--n-blocks", type=int, default=8, help="--kernel chain: blocks of the device")
    ap.add_argument("--fused", type=int, default=1, help="--kernel chain: NEGF_OPT_FUSED_SMALL (0 never, 1 automatic, 2 always for b <= 32)")
    ap.add_argument("--sets", type=int, default=2, help="operand sets rotated between launches")
    ap.add_argument("--inv-panel", type=int, default=1, help="NEGF_OPT_INV_PANEL (1 = row-per-thread Gauss-Jordan panel, 0 = first LU panel kernel)")
    ap.add_argument("--inv-lookahead", type=int, default=1, help="NEGF_OPT_INV_LOOKAHEAD")
    ap.add_argument("--inv-outer", type=int, default=0, help="NEGF_OPT_INV_OUTER (0 = automatic)")
    ap.add_argument("--pdl", type=int, default=-1, help="--kernel chain: NEGF_OPT_PDL (-1 = the library's default)")
    ap.add_argument("--energy-groups", type=int, default=0, help="--kernel chain: NEGF_OPT_ENERGY_GROUPS (0 = automatic)")
    ap.add_argument("--gemm-3m", action="store_true", help="NEGF_OPT_GEMM_3M (tflops still counted as 8 b^3 per product)")
    args = ap.parse_args()
    if args.kernel == "chain":
        return chain(args)
    ctx = negf.Context(0)
    st = torch.cuda.current_stream()
    ctx.set_stream(st.cuda_stream)
    if args.gemm_3m:
        ctx.set_option(negf.OPT_GEMM_3M, 1)
    ctx.set_option(negf.OPT_INV_PANEL, args.inv_panel)
    ctx.set_option(negf.OPT_INV_LOOKAHEAD, args.inv_lookahead)
    ctx.set_option(negf.OPT_INV_OUTER, args.inv_outer)
    peak = ctx.fp64_peak(200.0)
    if args.kernel == "peak":
        print(json.dumps({"kernel": "dmma_peak_probe", "tflops": peak}))
        return
    b, batch = args.b, args.batch
    gen = torch.Generator(device="cuda"); gen.manual_seed(1)
    if args.kernel == "econv":
        # Eq. 3 on a family of selected blocks: --batch energies, --b block size, 63 blocks (configs[1]-like);
        # HBM-bound: (2 N_E + 2 N_E - 1) * 16 bytes per element, against MEASURED_PEAKS.json's copy bandwidth
        ne, M = batch, 63 * b * b
        X1, X2 = _rand((ne, M), gen), _rand((ne, M), gen)
        Y = torch.empty(2 * ne - 1, M, dtype=torch.complex128, device="cuda")
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for _ in range(3):
            ctx.energy_convolve(ne, M, X1, X2, Y, mode=1, transpose_block=b)
        torch.cuda.synchronize()
        times = []
        for _ in range(args.reps):
            e0.record(st); ctx.energy_convolve(ne, M, X1, X2, Y, mode=1, transpose_block=b); e1.record(st)
            torch.cuda.synchronize(); times.append(e0.elapsed_time(e1))
        ms = sorted(times)[len(times) // 2]
        nbytes = (4 * ne - 1) * M * 16.0
        import os
        peak_gbs = None
        try:
            peak_gbs = json.load(open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "MEASURED_PEAKS.json")))["hbm_gbs"]
        except Exception:
            peak_gbs = 6650.0     # fallback of the profiling recipe
        gbs = nbytes / (ms * 1e-3) * 1e-9
        print(json.dumps({"kernel": "econv", "n_energy": ne, "b": b, "elems_per_energy": M, "ms_median": ms,
                          "algorithmic_GBps": gbs, "hbm_peak_GBps": peak_gbs, "frac": gbs / peak_gbs}))
        return
    flops = 8.0 * b ** 3 * batch
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if args.kernel == "zgemm":
        sets = [(_rand((batch, b, b), gen), _rand((batch, b, b), gen), torch.empty(batch, b, b, dtype=torch.complex128, device="cuda"))
                for _ in range(args.sets)]
        run = lambda i: ctx.zgemm_batched(args.opA, args.opB, b, b, b, 1.0, sets[i][0], b, b * b, sets[i][1], b, b * b,
                                          0.0, None, sets[i][2], b, b * b, batch)
    else:
        p = negf.Problem(2, b, batch, None, None, None, None, None, 0.0)
        ws = torch.empty(negf.Context.workspace_bytes(p), dtype=torch.uint8, device="cuda")
        ctx.set_workspace(ws)
        eye = torch.eye(b, dtype=torch.complex128, device="cuda")
        src = [_rand((batch, b, b), gen) / b ** 0.5 + 0.5 * eye for _ in range(args.sets)]
        work = [s.clone() for s in src]
        info = torch.zeros(batch, dtype=torch.int32, device="cuda")
        run = lambda i: ctx.zinverse_batched(b, work[i], b * b, batch, info)
    for i in range(3):
        run(i % args.sets)
    torch.cuda.synchronize()
    times = []
    for r in range(args.reps):
        i = r % args.sets
        if args.kernel == "zinv":
            work[i].copy_(src[i])
        e0.record(st); run(i); e1.record(st)
        torch.cuda.synchronize()
        times.append(e0.elapsed_time(e1))
    ms = sorted(times)[len(times) // 2]
    print(json.dumps({"kernel": args.kernel, "b": b, "batch": batch, "opA": args.opA, "opB": args.opB,
                      "ms_median": ms, "ms_best": min(times), "tflops": flops / (ms * 1e-3) * 1e-12,
                      "peak_tflops": peak, "frac": flops / (ms * 1e-3) * 1e-12 / peak}))


if __name__ == "__main__":
    main()
