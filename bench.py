#!/usr/bin/env python
"""bench.py -- Gibbs sweeps/s of the Horseshoe-Probit sampler at N=1e6, p=1000 (config C3) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C3]

A "step" is one full sweep (every row of SURVEY.md 8(a): fused X pass, reduce, scale conditionals,
Q build, Cholesky, beta draw, auxiliaries, history append) through the C-ABI of include/hsp.h.
Prints ONE JSON line (rank 0).  `value` has X resident in HBM; `e2e` goes through hsp_create_host
(host buffers, uploads inside the timed region) and reads every sweep's draws back to the host.
`roofline` is the fused pass (the dominant kernel) timed with CUDA events inside the timed region.
`cpu_baseline` / `--impl reference` time the oracle (oracle/, plain C++) on the host cores.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

PAPER_SWEEPS_PER_S = 10000.0 / 120.0   # 10,000 iterations in 2 min at (1e6, 1000), Titan X fp32
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the fused pass, from the ncu --set full captures
# summarised in profiles/r01_g_final.md (C3: 4.001072 GB + 4.08 MB) and profiles/r01_h_narrow.md (R1: 732.2 MB read)
NCU_TRAFFIC_BYTES = {"C3": 4005151872, "R1": 732223232}
WORKLOAD_DESC = {
    "C1": "C1 tiny probit: N=1000, p=10, fp64 X iid N(0,1), seed 1",
    "C2": "C2 medium: N=100000, p=100, fp64 X iid N(0,1), 10 nonzeros, seed 2",
    "C3": "C3 paper scale: N=1000000, p=1000, fp32 X iid N(0,1) (4 GB), fp64 state, 20 nonzeros, seed 3",
    "C4": "C4 correlated wide: N=250000, p=4000, fp32 AR(1) rows + intercept, 40 nonzeros, seed 4",
    "C5": "C5 large imbalanced: N=2000000, p=2000, fp32 X iid N(0,1) (16 GB), intercept -2, 50 nonzeros, seed 5",
    "R1": "R1 shape of the paper's real-data run (PAPER.md:309): N=1295848, p=141, fp32, ~0.5 % positives, synthetic, seed 6",
}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled DURING the timed region."""
    FIELDS = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.lines, self.proc = index, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "20"], stdout=subprocess.PIPE, text=True)
            self.thread = threading.Thread(target=lambda: [self.lines.append(l) for l in self.proc.stdout], daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None
        return self

    def __exit__(self, *a):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], 0.0, set()
        for l in self.lines:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0])); mx = max(mx, float(f[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        med = sm[len(sm) // 2] if sm else None
        return {"sm_mhz": med, "sm_max_mhz": mx or None, "reasons": sorted(reasons), "samples": len(sm)}


def oracle_scaled_sweeps_per_s(Xs, ys, seed, N_full, n_sweeps):
    """Oracle sweeps/s for the full workload from n_sweeps oracle sweeps on a row sample: the O(N p)
    row work (steps 1-3) is scaled by N_full/N_sample, the O(p^3)+O(p) rest is taken as measured."""
    import torch
    import oracle
    X64 = torch.from_numpy(Xs).double()
    gram = (X64.T @ X64).numpy()            # library matmul for the sample's X^T X (init, not timed)
    ch = oracle.OracleChain(Xs, ys, seed, gram=gram)
    t0 = time.perf_counter()
    ch.sweep(n_sweeps)
    wall = time.perf_counter() - t0
    t_rows, t_rest = ch.get_timing()
    per_sweep = (t_rows * (N_full / Xs.shape[0]) + t_rest) / n_sweeps
    ch.close()
    return 1.0 / per_sweep, wall


def run_reference(args, rank):
    """--impl reference: the oracle as it stands, on the host cores, rank 0 only."""
    if rank != 0:
        return
    import numpy as np
    import hsp_synth
    cfg = hsp_synth.CONFIGS[args.workload]
    N_full, p = cfg["N"], cfg["p"]
    # per-step budget so that the whole run ends within a few minutes
    per_step = 150.0 / max(1, args.steps + args.warmup)
    est_rest = 0.35 * (p / 1000.0) ** 3 + 1e-4
    rows = int(max(2000, min(N_full, (per_step - est_rest) / (9e-6 + 2.2e-9 * p))))
    wl = hsp_synth.make(args.workload, "cpu", n_rows=rows)
    Xs, ys = wl.host()
    if args.warmup > 0:
        oracle_scaled_sweeps_per_s(Xs, ys, wl.seed, N_full, min(args.warmup, 2))
    value, wall = oracle_scaled_sweeps_per_s(Xs, ys, wl.seed, N_full, args.steps)
    sample = (f"{args.steps} oracle sweeps on the first {rows} rows of the {args.workload} recipe (p={p}); row work "
              f"(eta, z, X^T z) scaled by {N_full}/{rows}, O(p^3)+O(p) work as measured; sample X^T X by a library matmul, untimed")
    line = {"impl": "reference", "metric": "gibbs_sweeps_per_sec", "value": value, "unit": "sweeps/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 / value, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": value / PAPER_SWEEPS_PER_S if args.workload == "C3" else None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD_DESC[args.workload], "wall_s": wall},
            "cpu_baseline": {"value": value, "unit": "sweeps/s", "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": "sweeps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C3", choices=list(WORKLOAD_DESC))
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--paper-design", action="store_true", help="A/B: rows a1-a3 by the paper's own decomposition (two X reads, rejection sampler)")
    ap.add_argument("--sharded", action="store_true", help="N > 1: ONE chain, rows of X sharded over the ranks, one NCCL all-reduce of p doubles per sweep (strong scaling)")
    ap.add_argument("--graph", action="store_true", help="replay the captured CUDA graph in the timed region (no per-kernel events)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import numpy as np
    import torch
    import torch.distributed as dist
    import hsp_synth
    import paper_1608_04329_b200 as hsp
    from paper_1608_04329_b200 import multi

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    elif args.sharded:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1"); os.environ.setdefault("MASTER_PORT", "29533")
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=dev)

    # Multi-GPU: independent chains, one per GPU, same data recipe, seed + rank.
    wl = hsp_synth.make(args.workload, dev)
    seed = multi.chain_seed(wl.seed, rank)
    stream = torch.cuda.Stream(device=dev)
    x_bytes = wl.X.numel() * wl.X.element_size()
    if args.sharded:
        seed = wl.seed                                 # one chain: every rank uses the same Philox key
        r0, r1 = multi.shard_rows(wl.N, rank, world)
        Xl, yl = wl.X[r0:r1].contiguous(), wl.y[r0:r1].contiguous()
        x_bytes = Xl.numel() * Xl.element_size()
    with torch.cuda.stream(stream):
        if args.sharded:
            chain = hsp.HorseshoeProbit(Xl, yl, seed, stream=stream, row_offset=r0)
            chain.set_flags(hsp.HSP_NO_GRAPH)
            multi.sharded_init(chain)
            run_sweeps = lambda n: multi.sharded_sweeps(chain, n)
        else:
            chain = hsp.HorseshoeProbit(wl.X, wl.y, seed, stream=stream)
            chain.set_flags((0 if args.graph else hsp.HSP_NO_GRAPH) | (hsp.HSP_PAPER_DESIGN if args.paper_design else 0))
            run_sweeps = chain.sweep
        run_sweeps(args.warmup)
        chain.sync()
        chain.fused_pass_ms()                     # reset the event accumulator
        k0 = chain.launch_count()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with ClockSampler(local_rank) as clocks:
            ev0.record(stream)
            run_sweeps(args.steps)
            ev1.record(stream)
            chain.sync()
            torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        ms = ev0.elapsed_time(ev1)
        fused_ms, fused_n = chain.fused_pass_ms()
        launches = chain.launch_count() - k0
        variant = chain.fused_variant()
        plan = chain.plan()
        # sanity: the chain is finite and moving
        b, lam, tau = chain.get_draws()
        assert np.all(np.isfinite(b)) and np.all(np.isfinite(lam)) and np.all(tau > 0)
    ms = multi.max_over_ranks(ms, dev)
    value = multi.whole_job_rate(args.steps, ms) if not args.sharded else args.steps / (ms * 1e-3)

    line = None
    if rank == 0:
        peaks, peak_kind = measured_peaks()
        alg_bytes = x_bytes + (wl.N if not args.sharded else (r1 - r0))   # X once + y; z is not stored in the timed run
        roofline = None
        if fused_n > 0 and fused_ms > 0:
            achieved = alg_bytes / (fused_ms * 1e-3) / 1e9
            traffic = NCU_TRAFFIC_BYTES.get(args.workload) if not args.paper_design else None
            roofline = {"bound": "hbm", "kernel": "paper_design(gemv+rejection+gemvT)" if args.paper_design else f"fused_pass_{variant}", "achieved": achieved, "peak": peaks["hbm_gbs"],
                        "peak_kind": f"{peak_kind} copy bandwidth (MEASURED_PEAKS.json hbm_gbs)", "unit": "GB/s",
                        "frac": achieved / peaks["hbm_gbs"], "frac_of_8TBps": achieved / 8000.0, "traffic": traffic,
                        "alg_bytes_per_launch": alg_bytes, "avg_launch_ms": fused_ms, "launches_timed": fused_n,
                        "share_of_step": fused_ms / (ms / args.steps)}
        line = {"metric": "gibbs_sweeps_per_sec", "value": value, "unit": "sweeps/s", "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
                "scaling": "strong" if args.sharded else "weak",
                "vs_baseline": value / PAPER_SWEEPS_PER_S if args.workload == "C3" else None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": WORKLOAD_DESC[args.workload], "x_dtype": str(wl.X.dtype).replace("torch.", ""),
                           "positive_rate": wl.positive_rate, "fused_kernel": variant, "plan": plan,
                           "arithmetic": "state, sampler, Cholesky, beta draw fp64; X fp32: eta in fp32 chains of 4 + fp64 across warps, "
                                         "x*z in fp32 chains of 16 rows + fp64 accumulators (DESIGN.md 5)" if wl.X.dtype == torch.float32
                                         else "fp64 throughout",
                           "l2": "X (%.1f GB) is larger than L2 and is streamed once per step" % (x_bytes / 1e9)
                           if x_bytes > 256e6 else "inputs fit L2: latency-bound config, absolute number only",
                           "launch_mode": "cuda-graph replay" if args.graph else "direct launches, 2 streams",
                           "multi_gpu": ("one chain, rows sharded over %d ranks, one all-reduce of p doubles per sweep" % world) if args.sharded
                           else "independent chains, seed+rank, no collective" if world > 1 else "single chain",
                           "vs_baseline_note": "paper: 83.3 sweeps/s on a Titan X, fp32 (PAPER.md:305); context, not the target"},
                "clocks": clocks.summary(), "gpu_launches": int(launches), "roofline": roofline}

    # ---- e2e: host buffers through the C-ABI, uploads and per-sweep readback inside the timed region
    if not args.no_e2e and not args.sharded:
        Xh = wl.X.cpu().pin_memory()
        yh = wl.y.cpu().pin_memory()
        e2e_steps = args.steps
        hb = torch.empty((1, wl.p), dtype=torch.float64).pin_memory()
        hl = torch.empty((1, wl.p), dtype=torch.float64).pin_memory()
        ht = torch.empty(1, dtype=torch.float64).pin_memory()
        chain.close()
        del chain
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        with torch.cuda.stream(stream):
            c2 = hsp.HorseshoeProbit(Xh, yh, seed, stream=stream, host=True)
            for _ in range(e2e_steps):
                c2.sweep(1)
                c2.get_draws((hb, hl, ht))
            c2.sync()
        torch.cuda.synchronize(dev)
        dt = time.perf_counter() - t0
        c2.close()
        dt = multi.max_over_ranks(dt, dev)
        if rank == 0:
            line["e2e"] = {"value": world * e2e_steps / dt, "unit": "sweeps/s",
                           "h2d_bytes_per_step": (x_bytes + wl.N) / e2e_steps, "d2h_bytes_per_step": (2 * wl.p + 1) * 8,
                           "note": "hsp_create_host (pinned X,y upload + Gram) + %d x [hsp_sweep(1) + hsp_get_draws to pinned host]; "
                                   "the one-off upload is amortised over the steps" % e2e_steps}

    # ---- cpu_baseline: the oracle on a bounded row sample, rank 0, single GPU run only
    if rank == 0 and world == 1 and not args.no_cpu_baseline and not args.sharded:
        n_s = min(wl.N, 60000)
        Xs = wl.X[:n_s].cpu().numpy()
        ys = wl.y[:n_s].cpu().numpy()
        v, wall = oracle_scaled_sweeps_per_s(Xs, ys, wl.seed, wl.N, 3)
        line["cpu_baseline"] = {"value": v, "unit": "sweeps/s", "cores": 1, "kind": "oracle",
                                "sample": f"3 oracle sweeps on the first {n_s} rows (row work scaled by {wl.N}/{n_s}, "
                                          f"p-only work as measured; {wall:.1f} s of CPU); host has {os.cpu_count()} cores"}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if dist.is_initialized():
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
