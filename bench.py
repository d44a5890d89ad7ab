#!/usr/bin/env python
"""bench.py -- causal-set action hot path on B200 (arXiv:1805.04463), BASELINE.json metric.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

A "step" is one pass of the whole hot path -- a1 causal-matrix build, a2 interval abundances,
a3 Benincasa-Dowker action -- over one seeded synthetic sprinkling.  The default workload is
BASELINE.json configs[2] = "config 3": N = 65536 points in the 3+1 flat causal diamond, the
configuration the metric is quoted on.  `value` is interval word-ops per second, with the
word-op count of the paper's Alg. 20, W_alg = sum over related pairs of ((j>>6)-(i>>6)+1) 64-bit
blocks, divided by the time of the whole step.  Inputs are resident in HBM for
`value`; `e2e` goes through cs_action_host with pinned HOST buffers (H2D and D2H inside the timed
region).  With --gpus N > 1 (torchrun) every rank runs an independent replica (the path does not
shard) and the aggregate is units summed / max time over ranks.

--impl reference times the oracle (oracle/, Alg. 20 on the host cores) on a bounded row sample of
the same workload; it is a deliberately plain CPU program, a reported baseline and not the target.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "interval_word_ops_per_s"
UNIT = "word-ops/s"

# ALU roofline of the POPC route: 16 POPC.32 /clk/SM, two per 64-bit word
POPC_PER_CLK_SM = 16.0
# dram__bytes_read.sum + dram__bytes_write.sum of one launch of the a2 kernel at config 3, from the
# `ncu --set full` captures summarised under profiles/ (bytes per launch; None = not captured)
NCU_TRAFFIC = {1: 78.28e9, 2: 51.14e9, 3: 38.12e9, 4: 8.85e9}
# tensor peaks = measured bf16 dense peak x the guide's nominal ratio (bf16 2.25, int8/fp8 4.5, fp4 9 PFLOP/s)
TENSOR_OVER_BF16 = {2: 2.0, 3: 4.0, 4: 4.0}
# dense issue rate of one SM's tensor pipe in op/clk (2 per multiply-add): kind::i8 16384, kind::mxf4 32768
TENSOR_OPS_PER_CLK_SM = {2: 16384.0, 3: 32768.0, 4: 32768.0}
ROUTE_NAME = {1: "popc", 2: "tensor_int8", 3: "tensor_fp4", 4: "tensor_fp4_pair"}
ROUTE_DTYPE = {1: "u64", 2: "int8", 3: "fp4_e2m1", 4: "fp4_e2m1"}
ROUTE_KERNEL = {1: "k_interval_popc", 2: "k_interval_tensor", 3: "k_interval_fp4", 4: "k_interval_pair"}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        d["_source"] = "measured"
        return d
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0,
            "sm_max_mhz": 1965.0, "_source": "fallback"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.perf_counter(), line.strip()))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for t, line in self.lines:
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7 or not (t0 - 0.05 <= t <= t1 + 0.15):
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for n, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def tensor_ops_algorithmic(N: int, tile: int = 128) -> float:
    """Ops (2 per multiply-add) of the 0/1 contraction restricted to K blocks between the
    I block and the J block: sum over tiles I<=J of 2*tile^2*(J-I+1)*tile."""
    nT = (N + tile - 1) // tile
    d = np.arange(nT, dtype=np.float64)
    return float((2.0 * tile ** 3 * (nT - d) * (d + 1)).sum())


def dense_triangular_word_ops(N: int, tile: int = 128) -> float:
    nT = (N + tile - 1) // tile
    d = np.arange(nT, dtype=np.float64)
    return float((tile * tile * (nT - d) * (2 * d + 2)).sum())


def run_reference(args, cfg, rank, world):
    """Oracle (Alg. 20, OpenMP over all host cores) on a bounded strided row sample."""
    if rank != 0:
        return
    import oracle
    from paper_1805_04463_b200 import inputs as inp
    N = args.N or cfg.N
    coords = inp.make_config_coords(cfg, N=N)
    t0 = time.perf_counter()
    bits = oracle.causal_matrix_bits(coords, cfg.geometry)
    t_build = time.perf_counter() - t0
    # calibrate the row stride so that one step is a few seconds of CPU work
    timing = {}
    probe_step = max(1, N // 256)
    _, w, T = oracle.interval_hist_alg20(bits, N, 0, N, row_step=probe_step, timing=timing)
    rate = w / max(timing["loop_seconds"], 1e-9)
    R, W_alg = oracle.count_relations(bits, N)
    target_s = args.ref_seconds
    row_step = max(1, int(round(W_alg / max(rate * target_s, 1.0))))
    times, wops = [], []
    for it in range(args.warmup + args.steps):
        hist, w, T = oracle.interval_hist_alg20(bits, N, it % row_step, N, row_step=row_step, timing=timing)
        oracle.bd_action(hist, N, cfg.dim)
        if it >= args.warmup:
            times.append(timing["loop_seconds"]); wops.append(w)
    value = sum(wops) / sum(times)
    sample = ("Alg. 20 pair loop over rows i = s, s+%d, ... of the N=%d sprinkling (%.3g of W_alg = %.4g "
              "word-ops per step); a1 built once outside the timed region (%.1f s)" %
              (row_step, N, 1.0 / row_step, W_alg, t_build))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
        "config": {"workload": cfg.name, "N": N, "dim": cfg.dim, "geometry": cfg.geometry, "seed": cfg.seed},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": T, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def cpu_baseline(cfg, N, coords, W_alg, seconds):
    """The oracle as it stands, timed on this box's host cores on a bounded sample."""
    import oracle
    t0 = time.perf_counter()
    bits = oracle.causal_matrix_bits(coords, cfg.geometry)
    t_build = time.perf_counter() - t0
    timing = {}
    probe_step = max(1, N // 128)
    _, w, T = oracle.interval_hist_alg20(bits, N, 0, N, row_step=probe_step, timing=timing)
    rate = w / max(timing["loop_seconds"], 1e-9)
    row_step = max(1, int(round(W_alg / max(rate * seconds, 1.0))))
    _, w, T = oracle.interval_hist_alg20(bits, N, 0, N, row_step=row_step, timing=timing)
    return {"value": w / timing["loop_seconds"], "unit": UNIT, "cores": T, "kind": "oracle",
            "sample": "Alg. 20 (oracle tier-1) over every %d-th row of the same N=%d sprinkling: %.4g of "
                      "%.4g word-ops in %.1f s; oracle a1 (all pairs, fp64) took %.1f s" %
                      (row_step, N, w, W_alg, timing["loop_seconds"], t_build)}


def run_ensemble(args, cfg, rank, local_rank, world):
    """Config 5: B independent causets per step through cs_bd_action_batched (one launch per stage).
    Not the headline workload (BASELINE.json's metric is quoted on config 3); same line shape, metric
    causets/s.  Every causet is distinct (own seed); 256 MiB of coordinates + 4 GiB of bit matrices per step,
    all larger than L2."""
    import torch
    from paper_1805_04463_b200 import api, dist as csd, inputs as inp
    torch.cuda.set_device(local_rank)
    csd.init()
    api.load()
    B = args.B or cfg.batch
    N = args.N or cfg.N
    coords = np.ascontiguousarray(np.stack(
        [inp.sprinkle(cfg.geometry, cfg.dim, N, cfg.seed * 4096 + b + 1000003 * rank) for b in range(B)]))
    d_coords = torch.from_numpy(coords).cuda()
    h_coords = torch.from_numpy(coords).pin_memory()
    h_actions = torch.empty(B, dtype=torch.float64).pin_memory()
    ws = torch.empty(api.bd_action_batched_workspace(B, N), dtype=torch.uint8, device="cuda")
    for _ in range(args.warmup):
        actions = api.bd_action_batched(d_coords, cfg.geometry, workspace=ws)
    sampler = ClockSampler(local_rank); sampler.start()
    csd.barrier(); torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = api.launch_count(); t0 = time.perf_counter()
    e0.record()
    for _ in range(args.steps):
        actions = api.bd_action_batched(d_coords, cfg.geometry, workspace=ws)
    e1.record(); torch.cuda.synchronize(); csd.barrier()
    t1 = time.perf_counter()
    launches = api.launch_count() - l0
    clocks = sampler.stop(t0, t1)
    units, secs, value = csd.aggregate(float(B) * args.steps, e0.elapsed_time(e1) / 1e3)
    # e2e: the library's host-buffer entry point (coordinates from pinned host memory chunk by chunk on a copy
    # stream while the kernels run, actions back to the host), every step
    ws_host = torch.empty(int(api.load().cs_bd_action_batched_host_workspace(B, N, cfg.dim)), dtype=torch.uint8, device="cuda")
    for _ in range(2):
        api.bd_action_batched_host(h_coords, cfg.geometry, ws_host, h_actions)
    csd.barrier(); torch.cuda.synchronize()
    e0.record()
    for _ in range(args.steps):
        api.bd_action_batched_host(h_coords, cfg.geometry, ws_host, h_actions)
    e1.record(); torch.cuda.synchronize(); csd.barrier()
    _, e2e_secs, e2e_value = csd.aggregate(float(B) * args.steps, e0.elapsed_time(e1) / 1e3)
    assert np.array_equal(h_actions.numpy(), actions.cpu().numpy())
    if rank == 0:
        print(json.dumps({
            "metric": "ensemble_causets_per_s", "value": value, "unit": "causets/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "fp4_e2m1", "data": "synthetic",
            "config": {"workload": cfg.name, "B": B, "N": N, "dim": cfg.dim, "geometry": cfg.geometry, "kmax": 3,
                       "l2": "inputs larger than L2 (coords %.0f MiB, bit matrices %.0f MiB)" %
                             (coords.nbytes / 2 ** 20, 2.0 * B * N * api.row_stride_words(N) * 8 / 2 ** 20),
                       "parallelism": "replicas x%d" % world, "mean_action": float(actions.mean().item())},
            "e2e": {"value": e2e_value, "unit": "causets/s", "h2d_bytes_per_step": int(coords.nbytes),
                    "d2h_bytes_per_step": int(B * 8), "ms_per_step": 1e3 * e2e_secs / args.steps},
            "gpu_launches": int(launches), "clocks": clocks, "roofline": None, "cpu_baseline": None}))
    csd.shutdown()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json workload 1..5 (default 3: N=65536, 3+1, the headline; 5 = batched ensemble, causets/s)")
    ap.add_argument("--N", type=int, default=0, help="override N (debug only; the line then names it)")
    ap.add_argument("--B", type=int, default=0, help="config 5 only: number of causets per step (default 4096)")
    ap.add_argument("--route", type=int, default=0, help="0 auto, 1 popc, 2 tensor int8, 3 tensor fp4, 4 tensor fp4 on CTA pairs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--ref-seconds", type=float, default=6.0)
    args = ap.parse_args()

    from paper_1805_04463_b200 import dist as csd, inputs as inp
    cfg = inp.CONFIGS[args.config]
    rank, local_rank, world = csd.env_world()

    if args.impl == "reference":
        run_reference(args, cfg, rank, world)
        return

    import torch
    from paper_1805_04463_b200 import api
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    if cfg.batch > 1:
        run_ensemble(args, cfg, rank, local_rank, world)
        return
    torch.cuda.set_device(local_rank)
    csd.init()
    api.load()
    peaks = measured_peaks()

    N = args.N or cfg.N
    seed = csd.replica_seed(cfg.seed, rank)
    coords = inp.sprinkle(cfg.geometry, cfg.dim, N, seed)
    d_coords = torch.from_numpy(coords).cuda()
    h_coords = torch.from_numpy(coords).pin_memory()
    stride = api.row_stride_words(N)
    kmax = api.clamp_kmax(N, cfg.kmax)
    route = args.route or api.default_route(N)

    # persistent device buffers (the library never allocates)
    ws = torch.empty(max(api.interval_hist_workspace(N, kmax, True, route), 256), dtype=torch.uint8, device="cuda")
    ws_host = torch.empty(api.action_host_workspace(N, kmax), dtype=torch.uint8, device="cuda")
    hist_host = torch.empty(kmax + 1, dtype=torch.int64).pin_memory()
    act_host = torch.empty(1, dtype=torch.float64).pin_memory()
    bits = torch.empty((N, stride), dtype=torch.int64, device="cuda")
    bitsT = torch.empty((N, stride), dtype=torch.int64, device="cuda")
    hist = torch.empty(kmax + 1, dtype=torch.int64, device="cuda")
    action = torch.empty(1, dtype=torch.float64, device="cuda")
    lib = api.load()
    st = torch.cuda.current_stream().cuda_stream

    def step(events=None):
        if events is not None: events[0].record()
        api._check(lib.cs_causal_matrix(d_coords.data_ptr(), N, cfg.dim, cfg.geometry, bits.data_ptr(),
                                        bitsT.data_ptr(), st), "cs_causal_matrix")
        if events is not None: events[1].record()
        api._check(lib.cs_interval_hist_ex(bits.data_ptr(), bitsT.data_ptr(), N, kmax, 0, N, route, hist.data_ptr(),
                                           None, ws.data_ptr(), ws.numel(), st), "cs_interval_hist_ex")
        if events is not None: events[2].record()
        api._check(lib.cs_bd_action(hist.data_ptr(), kmax, N, cfg.dim, action.data_ptr(), None, st), "cs_bd_action")
        if events is not None: events[3].record()

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    stats = api.relation_stats(bits, N).cpu().numpy()
    R, W_alg = int(stats[0]), int(stats[1])

    # ---- timed region: exactly K steps, device time, max over ranks -------------------------
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    sampler = ClockSampler(local_rank)
    sampler.start()
    csd.barrier(); torch.cuda.synchronize()
    launches0 = api.launch_count()
    t0 = time.perf_counter()
    for k in range(args.steps):
        step(ev[k])
    torch.cuda.synchronize(); csd.barrier()
    t1 = time.perf_counter()
    launches = api.launch_count() - launches0
    clocks = sampler.stop(t0, t1)
    total_ms = ev[0][0].elapsed_time(ev[-1][3])
    build_ms = [e[0].elapsed_time(e[1]) for e in ev]
    hist_ms = [e[1].elapsed_time(e[2]) for e in ev]
    act_ms = [e[2].elapsed_time(e[3]) for e in ev]
    units, secs, value = csd.aggregate(float(W_alg) * args.steps, total_ms / 1e3)
    ms_per_step = 1e3 * secs / args.steps
    S_dev = float(action.item())

    # ---- e2e: host buffers through cs_action_host, H2D + D2H inside the timed region --------
    for _ in range(2):
        api.action_host(h_coords, cfg.geometry, kmax, ws_host, hist_host, act_host)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    csd.barrier(); torch.cuda.synchronize()
    e0.record()
    for _ in range(args.steps):
        api.action_host(h_coords, cfg.geometry, kmax, ws_host, hist_host, act_host)
    e1.record(); torch.cuda.synchronize(); csd.barrier()
    e2e_units, e2e_secs, e2e_value = csd.aggregate(float(W_alg) * args.steps, e0.elapsed_time(e1) / 1e3)
    assert float(act_host[0]) == S_dev and int(hist_host.sum()) <= R

    if rank != 0:
        csd.shutdown()
        return

    # ---- roofline of the dominant kernel (a2) -----------------------------------------------
    hist_s = statistics.mean(hist_ms) / 1e3
    sm_mhz = clocks.get("sm_mhz") or peaks.get("sm_max_mhz", 1965.0)
    traffic = NCU_TRAFFIC.get(route) if (args.config == 3 and N == cfg.N) else None   # captured at config 3 only
    if route in TENSOR_OVER_BF16:
        ops = tensor_ops_algorithmic(N)
        burst = hist_s < 1.0
        ratio = TENSOR_OVER_BF16[route]
        peak = ratio * (peaks["bf16_tflops"] if burst else peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"]))
        roofline = {"bound": "tensor", "achieved": ops / hist_s / 1e12, "peak": peak, "unit": "TFLOP/s",
                    "frac": ops / hist_s / 1e12 / peak, "traffic": traffic,
                    "kernel": ROUTE_KERNEL[route], "peak_source": "%s bf16 %s x %.0f (%s:bf16 nominal ratio)" %
                    (peaks["_source"], "burst" if burst else "sustained", ratio, ROUTE_DTYPE[route]),
                    "algorithmic_ops": ops}
        # the pipe's own issue rate, for reading frac > 1: the library bf16 GEMM behind `peak` runs power-capped
        # (MEASURED_PEAKS clocks_under_load), this kernel at full clock.  DESIGN.md section 5.
        pipe = 148 * TENSOR_OPS_PER_CLK_SM[route] * peaks.get("sm_max_mhz", 1965.0) * 1e6 / 1e12
        roofline["pipe_peak"] = pipe
        roofline["frac_of_pipe"] = ops / hist_s / 1e12 / pipe
        if route == 4:
            # the pair route does not execute K stages whose 256 x 256 bit block is empty (13.7 % of the stages at
            # config 3, none at configs 2 and 4), so algorithmic ops per second can exceed the pipe's rate
            roofline["note"] = "algorithmic ops (dense-triangular tile set); empty K blocks are skipped, not executed"
    else:
        peak = 148 * POPC_PER_CLK_SM / 2.0 * peaks.get("sm_max_mhz", 1965.0) * 1e6 / 1e12   # T word-ops/s
        executed = dense_triangular_word_ops(N)
        roofline = {"bound": "alu", "achieved": W_alg / hist_s / 1e12, "peak": peak, "unit": "Tword-op/s",
                    "frac": W_alg / hist_s / 1e12 / peak, "traffic": traffic, "kernel": "k_interval_popc",
                    "peak_source": "derived: 148 SM x 16 POPC.32/clk/SM / 2 per 64-bit word x sm_max_mhz (DESIGN.md)",
                    "executed_word_ops": executed, "executed_frac": executed / hist_s / 1e12 / peak}
    build_s = statistics.mean(build_ms) / 1e3
    build_bytes = 2.0 * N * stride * 8 + N * cfg.dim * 8
    stages = {"build_ms": statistics.mean(build_ms), "interval_ms": statistics.mean(hist_ms),
              "action_ms": statistics.mean(act_ms), "interval_ms_min": min(hist_ms),
              "build_hbm_gbs": build_bytes / build_s / 1e9,
              "build_hbm_frac": build_bytes / build_s / 1e9 / peaks["hbm_gbs"],
              "interval_share_of_step": statistics.mean(hist_ms) / (total_ms / args.steps)}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": ROUTE_DTYPE[route], "data": "synthetic",
        "config": {"workload": cfg.name, "N": N, "dim": cfg.dim, "geometry": cfg.geometry, "seed": cfg.seed,
                   "route": ROUTE_NAME[route], "kmax": kmax, "relations": R, "W_alg": W_alg,
                   "l2": "inputs larger than L2 (bits+bitsT = %.0f MiB vs 126 MB)" % (2.0 * N * stride * 8 / 2 ** 20),
                   "parallelism": "replicas x%d" % world, "action": S_dev},
        "action_time_ms": ms_per_step, "stages": stages, "roofline": roofline,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(N * cfg.dim * 8),
                "d2h_bytes_per_step": int((kmax + 1) * 8 + 8), "ms_per_step": 1e3 * e2e_secs / args.steps},
        "gpu_launches": int(launches), "clocks": clocks, "peaks": peaks["_source"],
    }
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(cfg, N, coords, W_alg, args.cpu_seconds)
    elif world == 1:
        line["cpu_baseline"] = None
    print(json.dumps(line))
    csd.shutdown()


if __name__ == "__main__":
    main()
