#!/usr/bin/env python
"""bench.py -- Gibbs sweeps/s of the Horseshoe-Probit sampler at N=1e6, p=1000 (config C3) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C3] [--opt key=value ...]

A "step" is one full sweep (every row of SURVEY.md 8(a): fused X pass, reduce, scale conditionals,
Q build, Cholesky, beta draw, auxiliaries, history append) through the C-ABI of include/hsp.h.
Prints ONE JSON line (rank 0).
  value       X resident in HBM, K sweeps timed with CUDA events on the launching stream
  sustained   the same, over the config's own sweep count (C3: 1000 sweeps), with its own clock record
  e2e         hsp_create_host (host buffers, uploads inside the timed region) + K sweeps whose draws are
              downloaded into a pinned host ring while the chain keeps sweeping (hsp_set_output)
  roofline    the fused pass (the dominant kernel) timed with CUDA events inside the timed region
  cpu_baseline / --impl reference   the oracle (oracle/, plain C++) on the host cores
"""
import argparse
import csv
import hashlib
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

PAPER_SWEEPS_PER_S = 10000.0 / 120.0   # 10,000 iterations in 2 min at (1e6, 1000), Titan X fp32
WORKLOAD_DESC = {
    "C1": "C1 tiny probit: N=1000, p=10, fp64 X iid N(0,1), seed 1",
    "C2": "C2 medium: N=100000, p=100, fp64 X iid N(0,1), 10 nonzeros, seed 2",
    "C3": "C3 paper scale: N=1000000, p=1000, fp32 X iid N(0,1) (4 GB), fp64 state, 20 nonzeros, seed 3",
    "C4": "C4 correlated wide: N=250000, p=4000, fp32 AR(1) rows + intercept, 40 nonzeros, seed 4",
    "C5": "C5 large imbalanced: N=2000000, p=2000, fp32 X iid N(0,1) (16 GB), intercept -2, 50 nonzeros, seed 5",
    "C5b": "C5b: as C5 with intercept -1.645 sqrt(1+|beta|^2) (~5 % positives, DESIGN.md R15), seed 5",
    "R1": "R1 shape of the paper's real-data run (PAPER.md:309): N=1295848, p=141, fp32, ~0.5 % positives, synthetic, seed 6",
}
KERNEL_SOURCES = ("paper_1608_04329_b200/csrc/fused_pass.cu", "paper_1608_04329_b200/csrc/hsp_device.cuh")


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0}, "fallback"


def kernel_source_hash():
    """sha256 (first 12 hex) of the fused-pass sources: an ncu traffic figure is only quoted for the kernel it was
    captured on."""
    h = hashlib.sha256()
    for rel in KERNEL_SOURCES:
        with open(os.path.join(ROOT, rel), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:12]


def ncu_traffic(workload):
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the fused pass from the committed ncu summary
    profiles/ncu_traffic.csv -- or None when the capture was taken on a different version of the kernel source."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if not os.path.exists(path):
        return None, "no profiles/ncu_traffic.csv"
    want = kernel_source_hash()
    with open(path) as f:
        rows = [r for r in csv.DictReader(l for l in f if not l.startswith("#")) if r["workload"] == workload]
    for r in rows:
        if r["kernel_source_sha"] == want:
            return int(r["dram_read_bytes"]) + int(r["dram_write_bytes"]), r["profile"]
    return None, ("capture predates the current kernel source (%s)" % want) if rows else "no capture for this workload"


class ClockSampler:
    """SM clock, power and clock-event reasons sampled DURING a timed region by an NVML thread (every ~5 ms, started
    before the region); falls back to polling nvidia-smi when NVML is unavailable."""
    REASONS = (("hw_slowdown", "nvmlClocksEventReasonHwSlowdown"), ("hw_thermal_slowdown", "nvmlClocksEventReasonHwThermalSlowdown"),
               ("sw_thermal_slowdown", "nvmlClocksEventReasonSwThermalSlowdown"), ("sw_power_cap", "nvmlClocksEventReasonSwPowerCap"),
               ("hw_power_brake", "nvmlClocksEventReasonHwPowerBrakeSlowdown"))

    def __init__(self, index):
        self.index, self.samples, self.stop, self.thread, self.mx, self.source = index, [], threading.Event(), None, None, None
        self.t_begin = self.t_end = None

    def _nvml_loop(self, nv, h):
        masks = [(n, getattr(nv, a, 0)) for n, a in self.REASONS]
        while not self.stop.is_set():
            try:
                sm = nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                try:
                    pw = nv.nvmlDeviceGetPowerUsage(h) / 1000.0
                except Exception:
                    pw = None
                self.samples.append((time.perf_counter(), float(sm), [n for n, m in masks if r & m], pw))
            except Exception:
                pass
            time.sleep(0.005)

    def _smi_loop(self):
        fields = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
                  "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        while not self.stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={fields}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip().split(",")
                f = [x.strip() for x in out]
                self.mx = float(f[1])
                rs = [n for n, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]) if v.lower().startswith("active")]
                self.samples.append((time.perf_counter(), float(f[0]), rs, float(f[2])))
            except Exception:
                time.sleep(0.05)

    def start(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            # NVML enumerates all GPUs of the box; CUDA_VISIBLE_DEVICES may remap index 0
            vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
            ent = vis.split(",")[self.index].strip() if vis else str(self.index)
            h = nv.nvmlDeviceGetHandleByIndex(int(ent)) if ent.isdigit() else nv.nvmlDeviceGetHandleByUUID(ent)
            self.mx = float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            self.source = "nvml"
            self.thread = threading.Thread(target=self._nvml_loop, args=(nv, h), daemon=True)
        except Exception:
            self.source = "nvidia-smi"
            self.thread = threading.Thread(target=self._smi_loop, daemon=True)
        self.thread.start()
        time.sleep(0.25)                  # sampling is running well before the timed region starts
        return self

    def begin(self):
        self.t_begin, self.t_end = time.perf_counter(), None

    def end(self):
        self.t_end = time.perf_counter()

    def finish(self):
        self.stop.set()
        if self.thread:
            self.thread.join(timeout=6)

    def summary(self):
        t0, t1 = self.t_begin, self.t_end if self.t_end is not None else 1e300
        inside = [s for s in self.samples if t0 is not None and t0 <= s[0] <= t1]
        # a region shorter than a few sampling periods: take the samples nearest to it as well
        use = inside if len(inside) >= 3 else [s for s in self.samples if t0 is not None and t0 - 0.03 <= s[0] <= t1 + 0.03]
        sm = sorted(s[1] for s in use)
        reasons = sorted({r for s in use for r in s[2]})
        pw = [s[3] for s in use if s[3] is not None]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_min_mhz": sm[0] if sm else None, "sm_max_mhz": self.mx,
                "reasons": reasons, "samples": len(use), "samples_inside_region": len(inside),
                "power_w_max": max(pw) if pw else None, "source": self.source}


def timed_sweeps(chain, run_sweeps, n, stream, dev, clocks, dist, world):
    """n sweeps bracketed by barrier + synchronize, timed with CUDA events on the launching stream."""
    import torch
    chain.sync()
    chain.fused_pass_ms()                         # reset the event accumulator
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize(dev)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    clocks.begin()
    ev0.record(stream)
    run_sweeps(n)
    ev1.record(stream)
    chain.sync()
    torch.cuda.synchronize(dev)
    clocks.end()
    if world > 1:
        dist.barrier()
    ms = ev0.elapsed_time(ev1)
    fused_ms, fused_n = chain.fused_pass_ms()
    return ms, fused_ms, fused_n


def oracle_scaled_sweeps_per_s(Xs, ys, seed, N_full, n_sweeps, all_cores=False):
    """Oracle sweeps/s for the full workload from n_sweeps oracle sweeps on a row sample: the O(N p)
    row work (steps 1-3) is scaled by N_full/N_sample, the O(p^3)+O(p) rest is taken as measured."""
    import torch
    import oracle
    X64 = torch.from_numpy(Xs).double()
    gram = (X64.T @ X64).numpy()            # library matmul for the sample's X^T X (init, not timed)
    ch = oracle.OracleChain(Xs, ys, seed, gram=gram)
    if all_cores:
        ch.set_flags(oracle.STORE_Z | oracle.ROW_CHUNKS)
    t0 = time.perf_counter()
    ch.sweep(n_sweeps)
    wall = time.perf_counter() - t0
    t_rows, t_rest = ch.get_timing()
    per_sweep = (t_rows * (N_full / Xs.shape[0]) + t_rest) / n_sweeps
    ch.close()
    return 1.0 / per_sweep, wall


def run_reference(args, rank):
    """--impl reference: the oracle as it stands (single thread, the parity configuration), on the host cores, rank 0
    only.  Each step is one oracle sweep on a bounded row sample; the row work is extrapolated to the full N."""
    if rank != 0:
        return
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
    extrapolated = rows < N_full
    sample = (f"{args.steps} oracle sweeps on the first {rows} rows of the {args.workload} recipe (p={p}); row work "
              f"(eta, z, X^T z) scaled by {N_full}/{rows}, O(p^3)+O(p) work as measured; sample X^T X by a library matmul, untimed")
    line = {"impl": "reference", "metric": "gibbs_sweeps_per_sec", "value": value, "unit": "sweeps/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 / value, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": value / PAPER_SWEEPS_PER_S if args.workload == "C3" else None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD_DESC[args.workload], "wall_s": wall, "extrapolated": extrapolated,
                       "rows_run": rows, "rows_full": N_full, "row_fraction": rows / N_full},
            "extrapolated": extrapolated,
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
    ap.add_argument("--no-sustained", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the short side measurements of the other BASELINE.json configs (key other_configs)")
    ap.add_argument("--paper-design", action="store_true", help="A/B: rows a1-a3 by the paper's own decomposition (two X reads, rejection sampler)")
    ap.add_argument("--sharded", action="store_true", help="N > 1: ONE chain, rows of X sharded over the ranks, one NCCL all-reduce of p doubles per sweep (strong scaling)")
    ap.add_argument("--graph", action="store_true", help="replay the captured CUDA graph in the timed region (no per-kernel events)")
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=VALUE", help="plan-time option of libhsp.so (hsp_set_option), e.g. chol_ctas=24")
    ap.add_argument("--create-only", action="store_true", help="time hsp_create (device-resident X; Gram included) --steps times and exit")
    ap.add_argument("--chol-trace", action="store_true", help="per-task device timestamps of the Cholesky task graph (option chol_trace) on a row sample of the workload; prints a summary and exits")
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
    for kv in args.opt:
        k, v = kv.split("=")
        hsp.set_option(k, int(v))
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    elif args.sharded:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1"); os.environ.setdefault("MASTER_PORT", "29533")
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=dev)

    # Multi-GPU: independent chains, one per GPU, same data recipe, seed + rank.
    wl = hsp_synth.make(args.workload, dev)
    seed = multi.chain_seed(wl.seed, rank)
    stream = torch.cuda.Stream(device=dev)

    if args.chol_trace:
        # rows c, d1 alone: per-task timestamps of chol_task_kernel (hsp_dbg_chol_trace) over three direct-launch sweeps
        hsp.set_option("chol_trace", 1)
        wls = hsp_synth.make(args.workload, dev, n_rows=min(wl.N, 8009))
        c = hsp.HorseshoeProbit(wls.X, wls.y, seed)
        c.set_flags(hsp.HSP_NO_GRAPH | hsp.HSP_SERIAL)
        c.sweep(3); c.sync()
        tr = c.chol_trace()
        typ, ke, kb, ts, tk, te = tr[:, 0], tr[:, 4], tr[:, 3], tr[:, 8], tr[:, 9], tr[:, 10]
        out = {"metric": "chol_task_trace", "config": {"workload": WORKLOAD_DESC[args.workload], "p": wl.p, "plan": c.plan()},
               "tasks": int(len(tr)), "makespan_us": float(te.max() - ts.min()) / 1e3, "by_type_mean_us": {}}
        names = {0: "tile L(i,j)", 1: "inverse tile", 2: "POTRF (chain)", 3: "TRSM (chain)", 4: "SYRK (chain)"}
        for t in sorted(set(typ.tolist())):
            m = typ == t
            out["by_type_mean_us"][names[t]] = {"n": int(m.sum()), "mean": float((te[m] - ts[m]).mean()) / 1e3}
        m = (typ == 0) & (ke - kb >= 4)
        if m.any():
            out["kloop_us_per_64x64x64_product"] = {"median": float(np.median((tk[m] - ts[m]) / 1e3 / (ke[m] - kb[m]))),
                                                    "p10": float(np.percentile((tk[m] - ts[m]) / 1e3 / (ke[m] - kb[m]), 10))}
        m2 = typ == 2
        if m2.any():
            po = np.sort(ts[m2])
            out["chain"] = {"potrf_us": float((tk[m2] - ts[m2]).mean()) / 1e3, "inverse_us": float((tr[:, 11][m2] - tk[m2]).mean()) / 1e3,
                            "period_us_per_column": float(np.median(np.diff(po))) / 1e3 if len(po) > 1 else None}
        c.close()
        print(json.dumps(out), flush=True)
        return

    if args.create_only:
        times = []
        with torch.cuda.stream(stream):
            for _ in range(max(2, args.steps)):
                torch.cuda.synchronize(dev)
                t0 = time.perf_counter()
                c = hsp.HorseshoeProbit(wl.X, wl.y, seed, stream=stream)
                c.sync()
                times.append(1e3 * (time.perf_counter() - t0))
                c.close()
        if rank == 0:
            print(json.dumps({"metric": "hsp_create_ms", "value": min(times[1:]), "unit": "ms", "all_ms": times,
                              "config": {"workload": WORKLOAD_DESC[args.workload]}}), flush=True)
        return

    x_bytes = wl.X.numel() * wl.X.element_size()
    if args.sharded:
        seed = wl.seed                                 # one chain: every rank uses the same Philox key
        r0, r1 = multi.shard_rows(wl.N, rank, world)
        Xl, yl = wl.X[r0:r1].contiguous(), wl.y[r0:r1].contiguous()
        x_bytes = Xl.numel() * Xl.element_size()
    clocks = ClockSampler(local_rank).start()
    sustained = None
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
        # history capacity for the longest timed call, allocated now: growing it inside a timed region stalls the GPU
        # behind cudaFree / cudaMalloc (occasionally 0.1 - 1 s on this pool: profiles/r02_d_final.md)
        chain.reserve_history(max(args.steps, wl.n_sweeps))
        run_sweeps(args.warmup)
        k0 = chain.launch_count()
        ms, fused_ms, fused_n = timed_sweeps(chain, run_sweeps, args.steps, stream, dev, clocks, dist, world)
        launches = chain.launch_count() - k0
        clock_summary = clocks.summary()
        variant = chain.fused_variant()
        plan = chain.plan()
        # sanity: the chain is finite and moving
        b, lam, tau = chain.get_draws()
        assert np.all(np.isfinite(b)) and np.all(np.isfinite(lam)) and np.all(tau > 0)
        if not args.no_sustained and not args.paper_design:
            # the config's own sweep count (C3: 1000 sweeps, ~0.6 s): the sustained rate under the board's power management
            n_sus = wl.n_sweeps
            ms_s, fused_ms_s, fused_n_s = timed_sweeps(chain, run_sweeps, n_sus, stream, dev, clocks, dist, world)
            sustained = {"sweeps": n_sus, "ms": ms_s, "fused_ms": fused_ms_s, "fused_n": fused_n_s, "clocks": clocks.summary()}
    clocks.finish()
    ms = multi.max_over_ranks(ms, dev)
    rate = multi.whole_job_rate if not args.sharded else (lambda n, t: n / (t * 1e-3))
    value = rate(args.steps, ms)
    if sustained is not None:
        sustained["ms"] = multi.max_over_ranks(sustained["ms"], dev)

    line = None
    if rank == 0:
        peaks, peak_kind = measured_peaks()
        alg_bytes = x_bytes + (wl.N if not args.sharded else (r1 - r0))   # X once + y; z is not stored in the timed run
        roofline = None
        if fused_n > 0 and fused_ms > 0:
            achieved = alg_bytes / (fused_ms * 1e-3) / 1e9
            traffic, traffic_src = (None, "paper-design A/B") if args.paper_design else ncu_traffic(args.workload)
            roofline = {"bound": "hbm", "kernel": "paper_design(gemv+rejection+gemvT)" if args.paper_design else f"fused_pass_{variant}", "achieved": achieved, "peak": peaks["hbm_gbs"],
                        "peak_kind": f"{peak_kind} copy bandwidth (MEASURED_PEAKS.json hbm_gbs)", "unit": "GB/s",
                        "frac": achieved / peaks["hbm_gbs"], "frac_of_8TBps": achieved / 8000.0, "traffic": traffic,
                        "traffic_source": traffic_src, "kernel_source_sha": kernel_source_hash(),
                        "alg_bytes_per_launch": alg_bytes, "avg_launch_ms": fused_ms, "launches_timed": fused_n,
                        "share_of_step": fused_ms / (ms / args.steps)}
        f32 = wl.X.dtype == torch.float32
        line = {"metric": "gibbs_sweeps_per_sec", "value": value, "unit": "sweeps/s", "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
                "scaling": "strong" if args.sharded else "weak",
                "vs_baseline": value / PAPER_SWEEPS_PER_S if args.workload == "C3" else None,
                "dtype": "f32 X products (fp32 chains) + f64 state/sampler/Cholesky" if f32 else "f64", "x_dtype": "f32" if f32 else "f64",
                "data": "synthetic",
                "config": {"workload": WORKLOAD_DESC[args.workload], "x_dtype": str(wl.X.dtype).replace("torch.", ""),
                           "positive_rate": wl.positive_rate, "fused_kernel": variant, "plan": plan, "options": args.opt,
                           "arithmetic": "state, sampler, Cholesky, beta draw fp64; X fp32: eta in fp32 chains of 4 + fp64 across warps, "
                                         "x*z in fp32 chains of 16 rows + fp64 accumulators (DESIGN.md 5)" if f32
                                         else "fp64 throughout",
                           "l2": "X (%.1f GB) is larger than L2 and is streamed once per step" % (x_bytes / 1e9)
                           if x_bytes > 256e6 else "inputs fit L2: latency-bound config, absolute number only",
                           "launch_mode": "cuda-graph replay" if args.graph else "direct launches, 2 streams",
                           "multi_gpu": ("one chain, rows sharded over %d ranks, one all-reduce of p doubles per sweep" % world) if args.sharded
                           else "independent chains, seed+rank, no collective" if world > 1 else "single chain",
                           "vs_baseline_note": "paper: 83.3 sweeps/s on a Titan X, fp32 (PAPER.md:305); context, not the target"},
                "clocks": clock_summary, "gpu_launches": int(launches), "roofline": roofline}
        if sustained is not None:
            sv = rate(sustained["sweeps"], sustained["ms"])
            line["sustained"] = {"value": sv, "unit": "sweeps/s", "steps": sustained["sweeps"], "ms_per_step": sustained["ms"] / sustained["sweeps"],
                                 "clocks": sustained["clocks"],
                                 "fused_pass_gbs": (alg_bytes / (sustained["fused_ms"] * 1e-3) / 1e9) if sustained["fused_n"] else None,
                                 "note": "the config's own sweep count, timed like `value` right after it"}

    # ---- e2e: host buffers through the C-ABI; upload inside the timed region; every sweep's draws are downloaded
    # into a pinned host ring by the copy stream while the chain keeps sweeping (hsp_set_output)
    if not args.no_e2e and not args.sharded:
        Xh = wl.X.cpu().pin_memory()
        yh = wl.y.cpu().pin_memory()
        e2e_steps = args.steps
        hb = torch.empty((e2e_steps, wl.p), dtype=torch.float64).pin_memory()
        hl = torch.empty((e2e_steps, wl.p), dtype=torch.float64).pin_memory()
        ht = torch.empty(e2e_steps, dtype=torch.float64).pin_memory()
        chain.close()
        del chain
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        with torch.cuda.stream(stream):
            c2 = hsp.HorseshoeProbit(Xh, yh, seed, stream=stream, host=True)
            t_created = time.perf_counter()
            c2.set_output(hb, hl, ht, e2e_steps)
            c2.sweep(e2e_steps)
            landed = c2.output_wait()
        torch.cuda.synchronize(dev)
        dt = time.perf_counter() - t0
        assert landed == e2e_steps and bool(torch.isfinite(hb).all()) and bool((ht > 0).all())
        c2.close()
        dt = multi.max_over_ranks(dt, dev)
        if rank == 0:
            line["e2e"] = {"value": world * e2e_steps / dt, "unit": "sweeps/s",
                           "h2d_bytes_per_step": (x_bytes + wl.N) / e2e_steps, "d2h_bytes_per_step": (2 * wl.p + 1) * 8,
                           "create_s": t_created - t0, "sweeps_s": dt - (t_created - t0),
                           "value_after_create": world * e2e_steps / max(dt - (t_created - t0), 1e-9),
                           "note": "hsp_create_host (pinned X,y upload + Gram) + hsp_set_output + hsp_sweep(%d) + hsp_output_wait: every sweep's "
                                   "draws land in pinned host memory through the copy stream; the one-off upload is amortised over the steps" % e2e_steps}

    # ---- cpu_baseline: the oracle on a bounded row sample, rank 0, single GPU run only: all host cores (fixed row
    # chunks, the analogue of the paper's 16-thread workstation code) and single thread
    if rank == 0 and world == 1 and not args.no_cpu_baseline and not args.sharded:
        import oracle
        n_s = min(wl.N, 60000)
        Xs = wl.X[:n_s].cpu().numpy()
        ys = wl.y[:n_s].cpu().numpy()
        v1, wall1 = oracle_scaled_sweeps_per_s(Xs, ys, wl.seed, wl.N, 3)
        n_a = min(wl.N, 240000)
        Xa = wl.X[:n_a].cpu().numpy()
        ya = wl.y[:n_a].cpu().numpy()
        va, walla = oracle_scaled_sweeps_per_s(Xa, ya, wl.seed, wl.N, 3, all_cores=True)
        line["cpu_baseline"] = {"value": va, "unit": "sweeps/s", "cores": oracle.max_threads(), "kind": "oracle",
                                "single_thread_value": v1,
                                "sample": f"all cores: 3 oracle sweeps on the first {n_a} rows, steps 1-3 over fixed 4096-row chunks with OpenMP "
                                          f"({walla:.1f} s of wall time); single thread: 3 sweeps on the first {n_s} rows ({wall1:.1f} s); row work "
                                          f"scaled to N={wl.N}, p-only work as measured; host has {os.cpu_count()} cores"}
    # ---- the other configs of BASELINE.json (parity-test cases, not the metric): 100 sweeps each, resident X, the same timing,
    # reported under "other_configs" so that their numbers are measured by whoever runs the default command
    if rank == 0 and world == 1 and args.workload == "C3" and not (args.no_other_configs or args.sharded or args.paper_design or args.graph or args.opt):
        try:
            chain.close()
        except Exception:
            pass
        del wl
        torch.cuda.empty_cache()
        others = {}
        for name in ("C1", "C2", "C4", "C5", "C5b", "R1"):
            w2 = hsp_synth.make(name, dev)
            cs = ClockSampler(local_rank).start()
            with torch.cuda.stream(stream):
                c3 = hsp.HorseshoeProbit(w2.X, w2.y, w2.seed, stream=stream)
                c3.set_flags(hsp.HSP_NO_GRAPH)
                c3.reserve_history(100)
                c3.sweep(5)
                ms2, fm2, fn2 = timed_sweeps(c3, c3.sweep, 100, stream, dev, cs, dist, 1)
            cs.finish()
            ck = cs.summary()
            xb = w2.X.numel() * w2.X.element_size() + w2.N
            others[name] = {"value": 100 / (ms2 * 1e-3), "unit": "sweeps/s", "steps": 100, "ms_per_step": ms2 / 100,
                            "fused_kernel": c3.fused_variant(), "fused_pass_ms": fm2, "fused_pass_gbs": xb / (fm2 * 1e-3) / 1e9 if fn2 else None,
                            "plan": c3.plan(), "positive_rate": w2.positive_rate,
                            "clocks": {"sm_mhz": ck["sm_mhz"], "reasons": ck["reasons"], "samples": ck["samples"]}}
            c3.close()
            del c3, w2
            torch.cuda.empty_cache()
        line["other_configs"] = others
    if rank == 0:
        print(json.dumps(line), flush=True)
    if dist.is_initialized():
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
