#!/usr/bin/env python
"""bench.py -- causal-set action hot path on B200 (arXiv:1805.04463), BASELINE.json metric.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

    python bench.py --peaks            # the peak probes alone (cs_peak_probe), one JSON line
    python bench.py --shard --gpus N   # NEXT-4: rows of ONE causet split over N ranks + one histogram all-reduce

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

# ALU roofline of the POPC route: 16 POPC.32 /clk/SM, two per 64-bit word; replaced by the
# rate cs_peak_probe measures on this box when the probe runs
POPC_PER_CLK_SM = 16.0
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the a2 kernel come from the `ncu --set full` captures
# listed in profiles/ncu_traffic.csv (config,route,kernel,dram_bytes_read,dram_bytes_write,source); a workload/route
# with no capture reports "traffic": null
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
STAGE_OPS = 2.0 * 256 ** 3          # tensor ops of one executed (tile, stage) pair of the CTA-pair route
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
    """The oracle as it stands, timed on this box's host cores on a bounded sample.  Returns the line's
    `cpu_baseline` object, the oracle's bit matrix and -- when the sample is the whole workload -- its histogram
    (the parity check below compares the device's with it)."""
    import oracle
    t0 = time.perf_counter()
    bits = oracle.causal_matrix_bits(coords, cfg.geometry)
    t_build = time.perf_counter() - t0
    timing = {}
    probe_step = max(1, N // 128)
    _, w, T = oracle.interval_hist_alg20(bits, N, 0, N, row_step=probe_step, timing=timing)
    rate = w / max(timing["loop_seconds"], 1e-9)
    est_full = W_alg / max(rate, 1.0)
    # the whole workload if it fits twice the budget (config 3 on 16 cores: ~11 s), else every row_step-th row
    row_step = 1 if est_full <= 2.0 * seconds else int(np.ceil(est_full / seconds))
    hist, w, T = oracle.interval_hist_alg20(bits, N, 0, N, row_step=row_step, timing=timing)
    out = {"value": w / timing["loop_seconds"], "unit": UNIT, "cores": T, "kind": "oracle",
           "sample": "Alg. 20 (oracle tier-1) over every %d-th row of the same N=%d sprinkling: %.4g of "
                     "%.4g word-ops in %.1f s; oracle a1 (all pairs, fp64) took %.1f s" %
                     (row_step, N, w, W_alg, timing["loop_seconds"], t_build)}
    return out, bits, (hist if row_step == 1 else None)


def parity_check(api, cfg, N, o_bits, o_hist, d_bits, d_bitsT, d_hist, S_dev):
    """Device results of the timed configuration against the oracle: the bit matrix in full, then the whole
    histogram and the action when the oracle leg produced the whole histogram, else a contiguous row range."""
    import oracle
    bits_ok = bool(np.array_equal(d_bits.cpu().numpy().view(np.uint64), o_bits))
    if o_hist is not None:
        oS, _ = oracle.bd_action(o_hist, N, cfg.dim)
        ok = bits_ok and bool(np.array_equal(d_hist.cpu().numpy(), o_hist)) and float(S_dev) == float(oS)
        return {"ok": ok, "checked": "bits, every bin of N_k (k = 0..N-2) and the action vs the oracle (Alg. 20 over "
                                     "all rows, Eq. 4.10-4.12 on its histogram)", "oracle_action": float(oS)}
    r0, r1 = N // 2, N // 2 + max(32, N // 256)
    part = api.interval_hist(d_bits, d_bitsT, N, row_begin=r0, row_end=r1).cpu().numpy()
    o_part = oracle.interval_hist_alg20(o_bits, N, r0, r1)[0]
    return {"ok": bits_ok and bool(np.array_equal(part, o_part)),
            "checked": "bits in full; N_k of rows [%d, %d) vs the oracle (the whole histogram is compared in "
                       "tests/test_gpu_parity.py::test_config*_full_size)" % (r0, r1)}


def kernel_source_sha256(kernel_file: str) -> str:
    import hashlib
    with open(os.path.join(ROOT, "paper_1805_04463_b200", "csrc", kernel_file), "rb") as f:
        return hashlib.sha256(f.read()).hexdigest()[:16]


def load_traffic(config: int, route: int):
    """dram bytes per launch of the a2 kernel from the ncu captures listed in profiles/ncu_traffic.csv
    (config,route,kernel,dram_bytes_read,dram_bytes_write,kernel_file,kernel_sha256,source).  A capture counts only for
    the kernel source it was taken from: when the file that holds the kernel (tile order included) has changed since,
    the row is stale and `traffic` is null until the capture is repeated."""
    if not os.path.exists(TRAFFIC_CSV):
        return None, None
    with open(TRAFFIC_CSV) as f:
        for line in f:
            p = [x.strip() for x in line.split(",", 7)]
            if len(p) >= 8 and p[0] == str(config) and p[1] == ROUTE_NAME.get(route, ""):
                now = kernel_source_sha256(p[5])
                if now != p[6]:
                    return None, "stale: %s is %s now, the capture in profiles/ncu_traffic.csv was taken at %s" % (p[5], now, p[6])
                return float(p[3]) + float(p[4]), p[7] + " [%s @ %s]" % (p[5], p[6])
    return None, None


def probe(api, kind, iters, ws):
    units, secs, per_clk = api.peak_probe(kind, iters, ws)
    return {"per_s": units / secs if secs > 0 else 0.0, "per_clk_per_sm": per_clk, "ms": secs * 1e3}


def run_peaks(args, local_rank):
    """cs_peak_probe over every kind: the measured denominators quoted in DESIGN.md / profiles/r2_peaks.md."""
    import torch
    from paper_1805_04463_b200 import api
    torch.cuda.set_device(local_rank)
    api.load()
    ws = torch.empty((1 << 30) + 65536, dtype=torch.uint8, device="cuda")
    iters = {"mxf4_pair": 1 << 16, "i8": 1 << 16, "popc": 2048, "dfma": 2048, "ffma": 8192, "ffma2": 8192,
             "hbm_write": 4, "hbm_copy": 4, "tmem_ld4": 1 << 14, "tmem_ld8": 1 << 14, "mxf4_pair_n128": 1 << 16, "mxf4_pair_n128_dep": 1 << 16}
    out = {}
    sampler = ClockSampler(local_rank); sampler.start()
    t0 = time.perf_counter()
    for kind in api.PEAK_KINDS:
        best = None
        for _ in range(3):
            r = probe(api, kind, iters[kind], ws)
            if best is None or r["per_s"] > best["per_s"]:
                best = r
        out[kind] = best
    clocks = sampler.stop(t0, time.perf_counter())
    print(json.dumps({"peaks": out, "clocks": clocks, "given": measured_peaks(),
                      "units": "tensor: op (2 per multiply-add); popc/dfma/ffma: lane-instructions; ffma2: fused "
                               "multiply-adds; hbm: bytes; tmem_ld: bytes"}))


A1_ROUTES = {"auto": 0, "fma": 1, "tensor": 2}


def run_a1_probe(args, local_rank):
    """cs_a1_tensor_probe on seeded sprinklings: what the tensor-core value of the bilinear form is worth (error against the
    fp64 value, the accumulation error alone, error over margin, rows sent to fp64), and the two a1 routes timed side by side."""
    import torch
    from paper_1805_04463_b200 import api, inputs as inp
    torch.cuda.set_device(local_rank)
    api.load()
    out = {}
    cases = [("mink4_N65536", inp.GEOM_MINK_CONE, 4, 65536, inp.CONFIGS[3].seed), ("mink4_N2048", inp.GEOM_MINK_CONE, 4, 2048, 7),
             ("mink5_N16384", inp.GEOM_MINK_CONE, 5, 16384, 7)]
    for name, geom, dim, N, seed in cases:
        d = torch.from_numpy(inp.sprinkle(geom, dim, N, seed)).cuda()
        bits, bitsT, st = api.a1_tensor_probe(d)
        ref, refT = api.causal_matrix(d, geom, route=api.A1_FMA)
        st["equal_to_fma_route"] = bool(torch.equal(bits, ref) and torch.equal(bitsT, refT))
        for rname, route in (("fma", api.A1_FMA), ("tensor", api.A1_TENSOR)):
            ws = torch.empty(max(api.causal_matrix_workspace(1, N, dim, geom, route), 256), dtype=torch.uint8, device="cuda")
            for _ in range(3):
                api.causal_matrix(d, geom, route=route, workspace=ws)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize(); e0.record()
            for _ in range(10):
                api.causal_matrix(d, geom, route=route, workspace=ws)
            e1.record(); torch.cuda.synchronize()
            st["ms_" + rname] = e0.elapsed_time(e1) / 10      # (includes torch.empty of the two outputs: ~10 us)
        out[name] = st
    print(json.dumps({"a1_tensor_probe": out, "units": "max_err_u, max_acc_err_u: 2^-24 C^2; max_err_over_margin: must stay below 1"}))


def time_single(api, cfg, N, route, steps, warmup, seed, local_rank, csd, e2e=True, a1_route=0):
    """K timed steps of a1 -> a2 -> a3 on one seeded sprinkling (inputs resident in HBM), device time per stage,
    then (optionally) the same through cs_action_host with pinned host buffers."""
    import torch
    from paper_1805_04463_b200 import inputs as inp
    coords = inp.sprinkle(cfg.geometry, cfg.dim, N, seed)
    d_coords = torch.from_numpy(coords).cuda()
    stride = api.row_stride_words(N)
    kmax = api.clamp_kmax(N, cfg.kmax)
    # persistent device buffers (the library never allocates)
    ws = torch.empty(max(api.interval_hist_workspace(N, kmax, True, route), 256), dtype=torch.uint8, device="cuda")
    ws1 = torch.empty(max(api.causal_matrix_workspace(1, N, cfg.dim, cfg.geometry, a1_route), 256), dtype=torch.uint8, device="cuda")
    bits = torch.empty((N, stride), dtype=torch.int64, device="cuda")
    bitsT = torch.empty((N, stride), dtype=torch.int64, device="cuda")
    hist = torch.empty(kmax + 1, dtype=torch.int64, device="cuda")
    action = torch.empty(1, dtype=torch.float64, device="cuda")
    lib = api.load()
    st = torch.cuda.current_stream().cuda_stream

    def step(events=None):
        if events is not None: events[0].record()
        api._check(lib.cs_causal_matrix_ex(d_coords.data_ptr(), 1, N, cfg.dim, cfg.geometry, a1_route, bits.data_ptr(),
                                           bitsT.data_ptr(), ws1.data_ptr(), ws1.numel(), st), "cs_causal_matrix_ex")
        if events is not None: events[1].record()
        api._check(lib.cs_interval_hist_ex(bits.data_ptr(), bitsT.data_ptr(), N, kmax, 0, N, route, hist.data_ptr(),
                                           None, ws.data_ptr(), ws.numel(), st), "cs_interval_hist_ex")
        if events is not None: events[2].record()
        api._check(lib.cs_bd_action(hist.data_ptr(), kmax, N, cfg.dim, action.data_ptr(), None, st), "cs_bd_action")
        if events is not None: events[3].record()

    sampler = ClockSampler(local_rank)          # started before the warm-up: nvidia-smi needs ~0.1 s to its first line
    sampler.start()
    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    stats = api.relation_stats(bits, N).cpu().numpy()
    R, W_alg = int(stats[0]), int(stats[1])

    # ---- timed region: exactly K steps, device time, max over ranks -------------------------
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(steps)]
    csd.barrier(); torch.cuda.synchronize()
    launches0 = api.launch_count()
    t0 = time.perf_counter()
    for k in range(steps):
        step(ev[k])
    torch.cuda.synchronize(); csd.barrier()
    t1 = time.perf_counter()
    a1_used = a1_route if a1_route else api.default_a1_route(1, N, cfg.dim, cfg.geometry)
    m = {"coords": coords, "N": N, "kmax": kmax, "stride": stride, "R": R, "W_alg": W_alg, "route": route,
         "a1_route": {1: "fma", 2: "tensor"}[a1_used],
         "launches": api.launch_count() - launches0, "clocks": sampler.stop(t0, t1),
         "total_ms": ev[0][0].elapsed_time(ev[-1][3]),
         "build_ms": [e[0].elapsed_time(e[1]) for e in ev], "hist_ms": [e[1].elapsed_time(e[2]) for e in ev],
         "act_ms": [e[2].elapsed_time(e[3]) for e in ev], "step_ms": [e[0].elapsed_time(e[3]) for e in ev],
         "S": float(action.item()),
         "exec": api.interval_hist_stats(ws), "bits": bits, "bitsT": bitsT, "hist": hist}
    if e2e:
        # host buffers through cs_action_host, H2D + D2H inside the timed region
        h_coords = torch.from_numpy(coords).pin_memory()
        ws_host = torch.empty(api.action_host_workspace(N, kmax), dtype=torch.uint8, device="cuda")
        hist_host = torch.empty(kmax + 1, dtype=torch.int64).pin_memory()
        act_host = torch.empty(1, dtype=torch.float64).pin_memory()
        for _ in range(2):
            api.action_host(h_coords, cfg.geometry, kmax, ws_host, hist_host, act_host)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        csd.barrier(); torch.cuda.synchronize()
        e0.record()
        for _ in range(steps):
            api.action_host(h_coords, cfg.geometry, kmax, ws_host, hist_host, act_host)
        e1.record(); torch.cuda.synchronize(); csd.barrier()
        m["e2e_ms"] = e0.elapsed_time(e1)
        assert float(act_host[0]) == m["S"] and torch.equal(hist_host, hist.cpu())
        del ws_host
    return m


def time_ensemble(api, cfg, B, N, steps, warmup, rank, local_rank, csd, e2e=True, stages=False):
    """Config 5: B independent causets per step through cs_bd_action_batched.  Every causet is distinct (own
    seed); the coordinates (256 MiB) and the bit matrices are larger than L2."""
    import torch
    from paper_1805_04463_b200 import inputs as inp
    coords = np.ascontiguousarray(np.stack(
        [inp.sprinkle(cfg.geometry, cfg.dim, N, cfg.seed * 4096 + b + 1000003 * rank) for b in range(B)]))
    d_coords = torch.from_numpy(coords).cuda()
    ws = torch.empty(api.bd_action_batched_workspace(B, N), dtype=torch.uint8, device="cuda")
    sampler = ClockSampler(local_rank); sampler.start()      # started before the warm-up: nvidia-smi needs ~0.1 s to its first line
    for _ in range(warmup):
        actions = api.bd_action_batched(d_coords, cfg.geometry, workspace=ws)
    csd.barrier(); torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = api.launch_count(); t0 = time.perf_counter()
    e0.record()
    for _ in range(steps):
        actions = api.bd_action_batched(d_coords, cfg.geometry, workspace=ws)
    e1.record(); torch.cuda.synchronize(); csd.barrier()
    t1 = time.perf_counter()
    m = {"B": B, "N": N, "coords_bytes": int(coords.nbytes), "launches": api.launch_count() - l0,
         "clocks": sampler.stop(t0, t1), "total_ms": e0.elapsed_time(e1), "workspace_bytes": int(ws.numel()),
         "mean_action": float(actions.mean().item())}
    if stages:
        # the two batched stages on their own (a1 into materialised matrices, a2 with kmax = 3), for the stage split
        del ws
        bits, bitsT = api.causal_matrix_batched(d_coords, cfg.geometry)
        ws2 = torch.empty(int(api.load().cs_interval_hist_batched_workspace(B, N, 0)), dtype=torch.uint8, device="cuda")
        lib = api.load(); st = torch.cuda.current_stream().cuda_stream
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        a1, a2 = [], []
        for it in range(steps + 1):
            ev[0].record()
            api._check(lib.cs_causal_matrix_batched(d_coords.data_ptr(), B, N, cfg.dim, cfg.geometry, bits.data_ptr(),
                                                    bitsT.data_ptr(), st), "cs_causal_matrix_batched")
            ev[1].record()
            api.interval_hist_batched(bits, bitsT, N, kmax=3, workspace=ws2)
            ev[2].record(); torch.cuda.synchronize()
            if it:
                a1.append(ev[0].elapsed_time(ev[1])); a2.append(ev[1].elapsed_time(ev[2]))
        m["a1_ms"], m["a2_ms"] = statistics.mean(a1), statistics.mean(a2)
        del bits, bitsT, ws2
    if e2e:
        h_coords = torch.from_numpy(coords).pin_memory()
        h_actions = torch.empty(B, dtype=torch.float64).pin_memory()
        ws_host = torch.empty(int(api.load().cs_bd_action_batched_host_workspace(B, N, cfg.dim)), dtype=torch.uint8,
                              device="cuda")
        for _ in range(2):
            api.bd_action_batched_host(h_coords, cfg.geometry, ws_host, h_actions)
        csd.barrier(); torch.cuda.synchronize()
        e0.record()
        for _ in range(steps):
            api.bd_action_batched_host(h_coords, cfg.geometry, ws_host, h_actions)
        e1.record(); torch.cuda.synchronize(); csd.barrier()
        m["e2e_ms"] = e0.elapsed_time(e1)
        assert np.array_equal(h_actions.numpy(), actions.cpu().numpy())
    return m


def run_ensemble(args, cfg, rank, local_rank, world):
    """`--config 5`: same line shape as the headline, metric causets/s (not BASELINE.json's headline workload)."""
    import torch
    from paper_1805_04463_b200 import api, dist as csd
    torch.cuda.set_device(local_rank)
    csd.init()
    api.load()
    B, N = args.B or cfg.batch, args.N or cfg.N
    m = time_ensemble(api, cfg, B, N, args.steps, args.warmup, rank, local_rank, csd, e2e=True, stages=True)
    units, secs, value = csd.aggregate(float(B) * args.steps, m["total_ms"] / 1e3)
    _, e2e_secs, e2e_value = csd.aggregate(float(B) * args.steps, m["e2e_ms"] / 1e3)
    if rank == 0:
        print(json.dumps({
            "metric": "ensemble_causets_per_s", "value": value, "unit": "causets/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "fp4_e2m1", "data": "synthetic",
            "config": {"workload": cfg.name, "B": B, "N": N, "dim": cfg.dim, "geometry": cfg.geometry, "kmax": 3,
                       "l2": "inputs larger than L2 (coords %.0f MiB; workspace %.0f MiB)" %
                             (m["coords_bytes"] / 2 ** 20, m["workspace_bytes"] / 2 ** 20),
                       "parallelism": "replicas x%d" % world, "mean_action": m["mean_action"]},
            "stages": {"build_ms_alone": m["a1_ms"], "interval_ms_alone": m["a2_ms"]},
            "e2e": {"value": e2e_value, "unit": "causets/s", "h2d_bytes_per_step": m["coords_bytes"],
                    "d2h_bytes_per_step": int(B * 8), "ms_per_step": 1e3 * e2e_secs / args.steps},
            "gpu_launches": int(m["launches"]), "clocks": m["clocks"], "roofline": None, "cpu_baseline": None}))
    csd.shutdown()


def run_shard(args, cfg, rank, local_rank, world):
    """NEXT-4 (the paper's MPI scheme PAPER.md:1899-1933 on one node): ONE causet, every rank holds
    the whole bit matrix (it fits: <= 2 GiB at N = 131072), the outer rows of a2 are split over the ranks in
    contiguous blocks of equal tensor work (dist.shard_rows), and the int64 histograms are summed with one
    all-reduce.  Strong scaling: total work fixed."""
    import torch
    from paper_1805_04463_b200 import api, dist as csd, inputs as inp
    torch.cuda.set_device(local_rank)
    csd.init()
    api.load()
    N = args.N or cfg.N
    coords = inp.sprinkle(cfg.geometry, cfg.dim, N, cfg.seed)
    d_coords = torch.from_numpy(coords).cuda()
    kmax = api.clamp_kmax(N, cfg.kmax)
    route = args.route or api.default_route(N)
    r0, r1 = csd.shard_rows(N, world)[rank]
    ws = torch.empty(max(api.interval_hist_workspace(N, kmax, True, route), 256), dtype=torch.uint8, device="cuda")

    def step():
        bits, bitsT = api.causal_matrix(d_coords, cfg.geometry)
        part = api.interval_hist(bits, bitsT, N, kmax=kmax, route=route, row_begin=r0, row_end=r1, workspace=ws)
        hist = csd.all_reduce_sum_(part)
        return bits, hist, api.bd_action(hist, N, cfg.dim)

    for _ in range(args.warmup):
        bits, hist, S = step()
    W_alg = int(api.relation_stats(bits, N).cpu()[1])
    csd.barrier(); torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = api.launch_count()
    e0.record()
    for _ in range(args.steps):
        bits, hist, S = step()
    e1.record(); torch.cuda.synchronize(); csd.barrier()
    secs = csd.reduce_max(e0.elapsed_time(e1) / 1e3)
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": float(W_alg) * args.steps / secs, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps,
            "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": ROUTE_DTYPE[route],
            "data": "synthetic",
            "config": {"workload": cfg.name, "N": N, "dim": cfg.dim, "geometry": cfg.geometry, "seed": cfg.seed,
                       "route": ROUTE_NAME[route], "kmax": kmax, "W_alg": W_alg, "action": float(S.item()),
                       "parallelism": "rows of one causet over %d ranks + 1 all-reduce(sum) of N_k" % world,
                       "rows_rank0": [r0, r1]},
            "gpu_launches": int(api.launch_count() - l0)}))
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
    ap.add_argument("--a1-route", default="auto", choices=sorted(A1_ROUTES), help="a1: auto, FMA pipes, or tensor cores (bilinear predicates)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the short passes over configs 2, 4 and 5")
    ap.add_argument("--peaks", action="store_true", help="run the peak probes only")
    ap.add_argument("--a1-probe", action="store_true", help="run cs_a1_tensor_probe and time the two a1 routes only")
    ap.add_argument("--shard", action="store_true", help="split the rows of one causet over the ranks (NEXT-4)")
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
    if args.peaks:
        if rank == 0:
            run_peaks(args, local_rank)
        return
    if args.a1_probe:
        if rank == 0:
            run_a1_probe(args, local_rank)
        return
    if args.shard:
        run_shard(args, cfg, rank, local_rank, world)
        return
    if cfg.batch > 1:
        run_ensemble(args, cfg, rank, local_rank, world)
        return
    torch.cuda.set_device(local_rank)
    csd.init()
    api.load()
    peaks = measured_peaks()

    N = args.N or cfg.N
    route = args.route or api.default_route(N)
    m = time_single(api, cfg, N, route, args.steps, args.warmup, csd.replica_seed(cfg.seed, rank), local_rank, csd,
                    a1_route=A1_ROUTES[args.a1_route])
    R, W_alg, kmax, stride = m["R"], m["W_alg"], m["kmax"], m["stride"]
    units, secs, value = csd.aggregate(float(W_alg) * args.steps, m["total_ms"] / 1e3)
    ms_per_step = 1e3 * secs / args.steps
    e2e_units, e2e_secs, e2e_value = csd.aggregate(float(W_alg) * args.steps, m["e2e_ms"] / 1e3)

    if rank != 0:
        csd.shutdown()
        return

    # ---- roofline of the dominant kernel (a2), on the work the launch EXECUTED ---------------------
    hist_s = statistics.mean(m["hist_ms"]) / 1e3
    clocks = m["clocks"]
    traffic, traffic_src = load_traffic(args.config, route) if N == cfg.N else (None, None)
    pws = torch.empty(1 << 20, dtype=torch.uint8, device="cuda")
    if route in TENSOR_OVER_BF16:
        ops_alg = tensor_ops_algorithmic(N)
        burst = hist_s < 1.0
        ratio = TENSOR_OVER_BF16[route]
        peak = ratio * (peaks["bf16_tflops"] if burst else peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"]))
        executed_stages, total_stages, blocks_empty, blocks_examined = m["exec"]
        # the pair route reports the stages it issued; the single-CTA tensor routes execute their whole tile set
        ops_exec = executed_stages * STAGE_OPS if route == 4 else ops_alg
        roofline = {"bound": "tensor", "achieved": ops_exec / hist_s / 1e12, "peak": peak, "unit": "TFLOP/s",
                    "frac": ops_exec / hist_s / 1e12 / peak, "traffic": traffic, "traffic_source": traffic_src,
                    "kernel": ROUTE_KERNEL[route], "peak_source": "%s bf16 %s x %.0f (%s:bf16 nominal ratio)" %
                    (peaks["_source"], "burst" if burst else "sustained", ratio, ROUTE_DTYPE[route]),
                    "executed_ops": ops_exec, "algorithmic_ops": ops_alg,
                    "frac_algorithmic": ops_alg / hist_s / 1e12 / peak}
        if route == 4:
            roofline["stages"] = {"executed": executed_stages, "dense_triangular": total_stages,
                                  "blocks_empty": blocks_empty, "blocks_examined": blocks_examined}
            roofline["note"] = ("frac counts only the (tile, stage) pairs whose MMAs were issued (counter of the MMA "
                                "issuer, cs_interval_hist_stats); algorithmic_ops is SURVEY 8(d)'s dense-triangular set")
        # the pipe's own rate measured on this box by cs_peak_probe (same instruction, back to back): `peak` above
        # rests on a cuBLAS bf16 GEMM that runs power-capped near 1.3 GHz, this kernel holds a higher clock
        pk = probe(api, "mxf4_pair" if route >= 3 else "i8", 1 << 15, pws)
        roofline["pipe_peak_measured"] = pk["per_s"] / 1e12
        roofline["pipe_op_per_clk_per_sm"] = pk["per_clk_per_sm"]
        roofline["frac_of_measured_pipe"] = ops_exec / hist_s / max(pk["per_s"], 1.0)
    else:
        pk = probe(api, "popc", 2048, pws)
        per_clk = pk["per_clk_per_sm"] or POPC_PER_CLK_SM
        peak = 148 * per_clk / 2.0 * peaks.get("sm_max_mhz", 1965.0) * 1e6 / 1e12   # T word-ops/s
        executed = dense_triangular_word_ops(N)
        roofline = {"bound": "alu", "achieved": executed / hist_s / 1e12, "peak": peak, "unit": "Tword-op/s",
                    "frac": executed / hist_s / 1e12 / peak, "traffic": traffic, "traffic_source": traffic_src,
                    "kernel": "k_interval_popc",
                    "peak_source": "148 SM x %.2f POPC.32/clk/SM (cs_peak_probe, this run) / 2 per 64-bit word x sm_max_mhz" % per_clk,
                    "executed_word_ops": executed, "algorithmic_word_ops": W_alg,
                    "frac_algorithmic": W_alg / hist_s / 1e12 / peak}
    build_s = statistics.mean(m["build_ms"]) / 1e3
    build_bytes = 2.0 * N * stride * 8 + N * cfg.dim * 8
    stages = {"build_ms": statistics.mean(m["build_ms"]), "interval_ms": statistics.mean(m["hist_ms"]),
              "action_ms": statistics.mean(m["act_ms"]), "interval_ms_min": min(m["hist_ms"]),
              "build_hbm_gbs": build_bytes / build_s / 1e9,
              "build_hbm_frac": build_bytes / build_s / 1e9 / peaks["hbm_gbs"], "build_route": m["a1_route"],
              "interval_share_of_step": statistics.mean(m["hist_ms"]) / (m["total_ms"] / args.steps)}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step,
        # the paper's protocol (warm-ups, then the best of the timed runs), beside the mean the contract asks for
        "ms_per_step_min": min(m["step_ms"]),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": ROUTE_DTYPE[route], "data": "synthetic",
        "config": {"workload": cfg.name, "N": N, "dim": cfg.dim, "geometry": cfg.geometry, "seed": cfg.seed,
                   "route": ROUTE_NAME[route], "kmax": kmax, "relations": R, "W_alg": W_alg,
                   "l2": "inputs larger than L2 (bits+bitsT = %.0f MiB vs 126 MB)" % (2.0 * N * stride * 8 / 2 ** 20),
                   "parallelism": "replicas x%d" % world, "action": m["S"]},
        "action_time_ms": ms_per_step, "stages": stages, "roofline": roofline,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(N * cfg.dim * 8),
                "d2h_bytes_per_step": int((kmax + 1) * 8 + 8), "ms_per_step": 1e3 * e2e_secs / args.steps},
        "gpu_launches": int(m["launches"]), "clocks": clocks, "peaks": peaks["_source"],
    }
    if not args.no_cpu_baseline and world == 1:
        cb, o_bits, o_hist = cpu_baseline(cfg, N, m["coords"], W_alg, args.cpu_seconds)
        line["cpu_baseline"] = cb
        line["parity"] = parity_check(api, cfg, N, o_bits, o_hist, m["bits"], m["bitsT"], m["hist"], m["S"])
        del o_bits
    elif world == 1:
        line["cpu_baseline"] = None
    # ---- the other single-GPU workloads, outside the headline's timed region (short passes) ---------
    if world == 1 and args.config == 3 and not args.N and not args.no_other_configs:
        for k in ("bits", "bitsT", "hist", "coords"):
            m.pop(k, None)
        torch.cuda.empty_cache()
        other = {}
        for c in (2, 4):
            oc = inp.CONFIGS[c]
            om = time_single(api, oc, oc.N, api.default_route(oc.N), 3, 3, oc.seed, local_rank, csd, e2e=False)
            ex = om["exec"]
            other[str(c)] = {"workload": oc.name, "a1_ms": statistics.mean(om["build_ms"]),
                             "a2_ms": statistics.mean(om["hist_ms"]), "step_ms": om["total_ms"] / 3,
                             "a2_executed_ops": ex[0] * STAGE_OPS, "action": om["S"], "clocks": om["clocks"]}
            del om
            torch.cuda.empty_cache()
        oc = inp.CONFIGS[5]
        em = time_ensemble(api, oc, oc.batch, oc.N, 3, 3, 0, local_rank, csd, e2e=True, stages=True)
        other["5"] = {"workload": oc.name, "a1_ms": em["a1_ms"], "a2_ms": em["a2_ms"], "step_ms": em["total_ms"] / 3,
                      "e2e_ms": em["e2e_ms"] / 3, "causets_per_s": oc.batch * 3 / (em["total_ms"] / 1e3),
                      "workspace_mib": em["workspace_bytes"] / 2 ** 20, "clocks": em["clocks"]}
        line["other_configs"] = other
    print(json.dumps(line))
    csd.shutdown()


if __name__ == "__main__":
    main()
