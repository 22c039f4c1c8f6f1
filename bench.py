#!/usr/bin/env python
"""bench.py -- one JSON line: whole-hot-path throughput of libaptsig on a BASELINE.json config.

Default workload = config 4 (the largest single-GPU configuration: 175 616 material points x 40 962 geodesic
directions, B = 1024, ~4.8 M ions, 57.5 GB of signatures); `--config 2|3|5` selects another one.
A "step" = one apx_run (ingest + gather + project/bin + DFT + peak + write-out) over the whole
workload.
  value         device-timed (CUDA events on the launching stream, inputs resident in HBM), L2 flushed between steps
  e2e           the same through apx_run_host with HOST buffers (H2D + D2H inside the timed region)
  roofline      dominant kernel against the MEASURED on-chip peaks of profiles/r2_peaks.json (`--peaks` writes them):
                FP32 pipe and shared-memory atomics; pairs = the (ion, direction) pairs the kernel executes
  cpu_baseline  the oracle as it stands on the host cores (all cores and one core), bounded sample of the same workload
`--impl reference` times the oracle instead (the tier's reference arm).
Multi-GPU (torchrun): the centre list is cut into one slab per rank (parallel.run_sharded), ions replicated, no
collective on the data path: strong scaling of the same workload.  `--replicas` runs the whole workload on every rank.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "direction-histograms/s"
UNIT = "histograms/s"
WORKLOADS = {
    2: "cfg2_single_crystal: fcc Al 20^3 nm (~241k ions), 1000 material points x 10000 Fibonacci directions, "
       "R=2.0 nm, B=1024, window [15,34]",
    3: "cfg3_bicrystal: 30^3 nm fcc Al | bcc W (~832k ions), 27000 material points x 40962 geodesic directions, R=2.0 nm, "
       "B=1024, window [15,34], Al filter run",
    4: "cfg4_nanocrystal: 64 Voronoi grains in 60^3 nm fcc Al (~4.8M ions), 175616 material points x 40962 geodesic "
       "directions, R=2.0 nm, B=1024, window [15,34]",
    5: "cfg5_dilute_alloy: 40^3 nm fcc Al-3%Sc + 5% background (~1.5M ions), 64000 material points x 40962 geodesic "
       "directions, R=3.0 nm, B=2048, window [23,51], Al filter",
}
PAIR_FLOP = 6.0          # FMUL + 2 FFMA + round-down FADD of Eq. 1's projection and floor, per (ion, direction) pair
PEAKS_JSON = os.path.join(ROOT, "profiles", "r2_peaks.json")          # written by `bench.py --peaks`
NCU_JSON = os.path.join(ROOT, "profiles", "r2_ncu_constants.json")    # written by paper_2009_00735_b200/ncu_summary.py
SM_COUNT, SM_MAX_GHZ = 148, 1.965     # B200_PROFILING.md; only used when profiles/r2_peaks.json is missing


def load_peaks():
    """Measured on-chip peaks (profiles/r2_peaks.json), else the derived fallback of DESIGN.md section 6."""
    try:
        pk = json.load(open(PEAKS_JSON))
        t = pk["tests"]
        clk = pk["sm_max_mhz"] * 1e6
        sm = pk["sm_count"]
        # FP32 pipe: the better of plain and packed FFMA (2 / 4 flop per lane and instruction), per clock x max clock
        flop_clk = max(t["ffma"]["warp_inst_per_clk_per_sm"] * 64.0, t["ffma2_packed"]["warp_inst_per_clk_per_sm"] * 128.0)
        atom_clk = max(t["red_shared_conflict_free"]["warp_inst_per_clk_per_sm"],
                       t["red_shared_inc_conflict_free"]["warp_inst_per_clk_per_sm"])
        return {"fp32_tflops": flop_clk * sm * clk / 1e12, "atom_warp_inst_per_s": atom_clk * sm * clk,
                "source": f"measured: profiles/r2_peaks.json (`python bench.py --peaks`, {pk.get('when', '?')}): "
                          f"{flop_clk:.1f} flop/clk/SM, {atom_clk:.3f} conflict-free shared atomics (warp instr)/clk/SM, "
                          f"x {sm} SMs x {pk['sm_max_mhz']:.0f} MHz"}
    except Exception:
        return {"fp32_tflops": SM_COUNT * 128 * 2 * SM_MAX_GHZ * 1e9 / 1e12, "atom_warp_inst_per_s": SM_COUNT * SM_MAX_GHZ * 1e9,
                "source": "fallback (profiles/r2_peaks.json missing): derived 148 SM x 128 FP32 lanes x 2 flop x 1.965 GHz and one "
                          "32-lane shared atomic per SM clock (B200_PROFILING.md unit counts)"}


def ncu_constant(kernel, cfg, key):
    """Per-launch counters of the committed ncu capture of `kernel` on config `cfg` (None when not captured)."""
    try:
        return json.load(open(NCU_JSON))[kernel][str(cfg)][key]
    except Exception:
        return None


class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for t, row in self.rows:
            f = [x.strip() for x in row.split(",")]
            if len(f) < 7:
                continue
            try:
                mx = float(f[1])
                if t0 - 0.05 <= t <= t1 + 0.05:
                    sm.append(float(f[0]))
                    for n, v in zip(names, f[3:7]):
                        if v.lower().startswith("active"):
                            reasons.add(n)
            except ValueError:
                continue
        if not sm and self.rows:
            try:
                sm = [float(self.rows[-1][1].split(",")[0])]
            except ValueError:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def accepted_for(cfg):
    return {0} if cfg in (3, 5) else None        # configs 3 and 5: the Al filter run


def oracle_dirs(w):
    from oracle import oracle as O
    return O.dirs_geodesic(w.grid[1]) if w.grid[0] == "geodesic" else O.dirs_fibonacci(w.D)


def oracle_sample(w, cfg, dirs, idx, nthreads=0):
    """Time the oracle (window mode, identical outputs) on material points `idx` x all directions."""
    from oracle import oracle as O
    t = time.perf_counter()
    O.signatures(w.xyz, w.types, w.centres[idx], dirs, w.R, w.B, k_lo=w.window[0], k_hi=w.window[1],
                 accepted=accepted_for(cfg), nthreads=nthreads)
    dt = time.perf_counter() - t
    return dt, len(idx) * len(dirs), O.num_threads() if nthreads <= 0 else nthreads


def sample_points(M, n, seed):
    return np.sort(np.random.default_rng(seed).choice(M, size=min(n, M), replace=False))


def run_reference(args, rank, world):
    """--impl reference: the oracle on the host cores, bounded sample per step (rank 0 only)."""
    if rank != 0:
        return
    from workloads import make_config
    w = make_config(args.config)
    dirs = oracle_dirs(w)
    n_points = 16
    oracle_sample(w, args.config, dirs, sample_points(len(w.centres), 2, 1))
    for i in range(max(args.warmup - 1, 0)):
        oracle_sample(w, args.config, dirs, sample_points(len(w.centres), 2, 2 + i))
    times, cores = [], 1
    for i in range(args.steps):
        dt, nh, cores = oracle_sample(w, args.config, dirs, sample_points(len(w.centres), n_points, 100 + i))
        times.append(dt)
    v = n_points * w.D * args.steps / sum(times)
    sample = f"{n_points} seeded material points of {len(w.centres)} x {w.D} directions per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / args.steps, "higher_is_better": True,
        "scaling": "strong", "vs_baseline": None, "dtype": "f32 binning, f64 DFT", "data": "synthetic",
        "material_points_per_s": v / w.D,
        "config": {"workload": WORKLOADS[args.config], "sample": sample},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def run_peaks(args):
    """--peaks: the on-chip peak microbenchmarks (include/aptsig_peaks.h) -> profiles/r2_peaks.json + one JSON line."""
    import paper_2009_00735_b200 as apx
    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.2)
    t0 = time.time()
    tests = {}
    n = 0
    while apx.apx_peak_name(n) is not None:
        best = None
        for _ in range(3):                                   # best of three launches of ~10-40 ms each
            r = apx.apx_peak_measure(0, n, args.peak_iters)
            if best is None or r["warp_inst_per_clk_per_sm"] > best["warp_inst_per_clk_per_sm"]:
                best = r
        tests[apx.apx_peak_name(n)] = best
        n += 1
    clocks = sampler.stop(t0, time.time())
    out = {"when": time.strftime("%Y-%m-%dT%H:%M:%SZ", time.gmtime()), "command": "python bench.py --peaks",
           "iters": args.peak_iters, "sm_count": tests["ffma"]["sm_count"], "sm_max_mhz": clocks.get("sm_max_mhz") or 1965.0,
           "clocks": clocks, "tests": tests}
    os.makedirs(os.path.dirname(args.peaks_out), exist_ok=True)
    with open(args.peaks_out, "w") as f:
        json.dump(out, f, indent=1)
    print(json.dumps(out))


def run_ingest(args):
    """--ingest-ions N: step a1 alone (HBM-bound counting sort) on N uniform random ions in config 4's 60^3 nm box;
    not the default bench line -- the roofline evidence for the ingest kernels."""
    import torch
    import paper_2009_00735_b200 as apx
    dev = torch.device("cuda:0")
    N = args.ingest_ions
    rng = np.random.Generator(np.random.PCG64(200900735))
    xyz_np = (rng.random((N, 3), dtype=np.float32) * np.float32(60.0))
    types_np = np.zeros(N, np.uint8)
    plan = apx.Plan(2.0, 1024, apx.apx_dirs_fibonacci(64), k_lo=15, k_hi=34, device=0)
    xyz, types = torch.from_numpy(xyz_np).to(dev), torch.from_numpy(types_np).to(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    for _ in range(max(args.warmup, 3)):
        plan.apx_ingest(xyz, types)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in ev:
        flush.fill_(1)
        a.record(); plan.apx_ingest(xyz, types); b.record()
    torch.cuda.synchronize()
    ms = sum(a.elapsed_time(b) for a, b in ev) / args.steps
    # algorithmic bytes per ion: xyz + type read by k_bounds and k_count (2 x 13), cell id written and read (2 x 4),
    # xyz read again and the 16-byte record written by k_scatter (12 + 16)
    bytes_per_ion = 3 * 13 + 16                     # xyz + type read by the bounds, count and scatter passes; one 16-byte record written
    try:
        peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
        src = "MEASURED_PEAKS.json hbm_gbs"
    except Exception:
        peak, src = 6550.0, "fallback (B200_PROFILING.md)"
    achieved = bytes_per_ion * N / (ms * 1e-3) / 1e9
    print(json.dumps({"metric": "ingested ions/s", "value": N / (ms * 1e-3), "unit": "ions/s", "n_gpus": 1,
                      "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True,
                      "dtype": "f32", "data": "synthetic",
                      "config": {"workload": f"ingest only: {N} uniform random ions in a 60^3 nm box, R = 2.0 (cell edge 1 nm)",
                                 "l2": "flushed between timed steps (256 MiB fill, untimed)"},
                      "gpu_launches": 8 * args.steps,
                      "roofline": {"bound": "hbm", "kernel": "ingest (8 kernels)", "achieved": achieved, "peak": peak,
                                   "unit": "GB/s", "frac": achieved / peak, "traffic": None, "peak_source": src,
                                   "model": f"{bytes_per_ion} B per ion"}}))
    plan.apx_plan_destroy()


def _time_steps(torch, fn, steps, warmup, flush):
    for _ in range(max(warmup, 3)):
        fn()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in ev:
        flush.fill_(1)
        a.record(); fn(); b.record()
    torch.cuda.synchronize()
    return sum(a.elapsed_time(b) for a, b in ev) / steps


def run_index(args):
    """--index: Eq. 3 -- M synthetic normalised images on the paper's 40 962-node mesh against every
    orientation of the stand-in orientation set, N_hat = 1000 strongest nodes (L369, L416).  L2-bound gather: algorithmic
    traffic = 4 B (one fp32 image value) per (material point, orientation, node) triple."""
    import torch
    import paper_2009_00735_b200 as apx
    dev = torch.device("cuda:0")
    rng = np.random.Generator(np.random.PCG64(200900735 + 11))
    dirs = apx.apx_dirs_geodesic(6)
    G = apx.apx_so3_grid_cubic(args.index_spacing)
    D, Ng, n_hat, M, K = len(dirs), len(G), 1000, args.index_points, 4
    # reference: smooth image with <100> poles; measured: the same rotated by random grid orientations + noise
    ref = np.exp(-(1.0 - np.max(np.abs(dirs), axis=1)) / 0.01).astype(np.float32)
    t0 = time.perf_counter()
    ix = apx.Indexer(dirs, G, ref, n_hat, device=0)
    t_pre = time.perf_counter() - t0
    sig = torch.zeros((M, D, 2), dtype=torch.float32, device=dev)
    sig[..., 0] = torch.from_numpy(rng.random((M, D), dtype=np.float32)).to(dev)
    bd = torch.empty((M, K), dtype=torch.float32, device=dev)
    bg = torch.empty((M, K), dtype=torch.int32, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    ms = _time_steps(torch, lambda: ix.apx_index(sig, None, bd, bg), args.steps, args.warmup, flush)
    gathers = float(M) * Ng * n_hat
    try:
        lts = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
    except Exception:
        lts = 6550.0
    # L2 ceiling: ~6300 B/clk full chip (B200_PROFILING.md "LTS throughput cap") at the maximum SM clock
    l2_peak = 6300.0 * SM_MAX_GHZ
    achieved = gathers * 4.0 / (ms * 1e-3) / 1e9
    print(json.dumps({"metric": "indexed (material point, orientation) pairs/s", "value": float(M) * Ng / (ms * 1e-3),
                      "unit": "pairs/s", "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms,
                      "higher_is_better": True, "dtype": "f32", "data": "synthetic",
                      "config": {"workload": f"indexing: {M} images x {Ng} orientations ({args.index_spacing} deg Rodrigues grid, m-3m) x "
                                             f"{n_hat} strongest nodes of {D} (geodesic level 6)", "K": K,
                                 "preprocessing_s": t_pre, "l2": "flushed between timed steps"},
                      "gpu_launches": 3 * args.steps * ((M + 8191) // 8192),
                      "roofline": {"bound": "l2", "kernel": "k_index", "achieved": achieved, "peak": l2_peak, "unit": "GB/s",
                                   "frac": achieved / l2_peak, "traffic": None,
                                   "peak_source": "B200_PROFILING.md LTS throughput cap ~6300 B/clk x 1.965 GHz (HBM copy peak "
                                                  f"{lts:.0f} GB/s for scale)",
                                   "model": "4 B per (material point, orientation, node) gather; one 128-B line serves 32 material points",
                                   "gathers_per_s": gathers / (ms * 1e-3)}}))
    ix.apx_indexer_destroy()


def run_fsp(args):
    """--fsp: Eq. 2 on config 2's cloud: M ROIs x L^3 reciprocal-space points, k_max = 2 pi / nm.
    A dense complex contraction per z-slice on the FP32 pipe: 8 flop per (ion, k point)."""
    import torch
    import paper_2009_00735_b200 as apx
    from workloads import make_config
    dev = torch.device("cuda:0")
    w = make_config(2)
    M, L = args.fsp_points, args.fsp_L
    plan = apx.Plan(w.R, w.B, apx.apx_dirs_fibonacci(64), k_lo=15, k_hi=34, device=0)
    plan.apx_ingest(torch.from_numpy(w.xyz).to(dev), torch.from_numpy(w.types).to(dev))
    centres = torch.from_numpy(np.ascontiguousarray(w.centres[np.arange(M) % len(w.centres)])).to(dev)
    out = torch.empty((M, L, L, L), dtype=torch.float32, device=dev)
    cnt = torch.empty(M, dtype=torch.int32, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    plan.apx_fsp_set_path(args.fsp_path)
    ms = _time_steps(torch, lambda: plan.apx_fsp(centres, 2.0 * np.pi, L, out, cnt), args.steps, args.warmup, flush)
    nw = float(cnt.cpu().numpy().astype(np.int64).sum())
    flops = 8.0 * nw * L ** 3                                  # Eq. 2: one complex multiply-add per (ion, k point)
    pk = load_peaks()
    if args.fsp_path == 1:
        bound, kernel, peak, unit = "alu", "k_fsp", pk["fp32_tflops"], "TFLOP/s"
        achieved, src = flops / (ms * 1e-3) / 1e12, pk["source"]
        model = "8 flop (one complex multiply-add) per (ion, k point) on the FP32 pipe"
    else:
        # tensor-core kernel: the complex contraction as one real GEMM (8 flop per (ion, k point)) executed three times
        # (Ah Bh, Ah Bl, Al Bh of the fp16 hi + lo split): executed tensor flops = 3 x model flops
        try:
            peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["bf16_tflops"]
            src = "MEASURED_PEAKS.json bf16_tflops (burst, kernel timed alone; fp16 has the same nominal rate as bf16)"
        except Exception:
            peak, src = 1600.0, "fallback (B200_PROFILING.md)"
        bound, kernel, unit = "tensor", "k_fsp_mma", "TFLOP/s"
        achieved = 3.0 * flops / (ms * 1e-3) / 1e12
        model = "executed fp16 tensor flops = 3 GEMMs (hi*hi, hi*lo, lo*hi) x 8 flop per (ion, k point)"
    print(json.dumps({"metric": "FSP k-points/s", "value": float(M) * L ** 3 / (ms * 1e-3), "unit": "k-points/s", "n_gpus": 1,
                      "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True,
                      "dtype": "f32" if args.fsp_path == 1 else "f16 hi+lo split operands, f32 accumulate", "data": "synthetic",
                      "config": {"workload": f"FSP (Eq. 2): {M} ROIs of config 2 (R = 2.0 nm, mean {nw / M:.0f} ions) x {L}^3 k points, "
                                             "k_max = 2 pi / nm", "rois_per_s": M / (ms * 1e-3),
                                 "kernel_path": "fp32" if args.fsp_path == 1 else "tensor"},
                      "gpu_launches": (1 if args.fsp_path == 1 else 2) * args.steps,
                      "roofline": {"bound": bound, "kernel": kernel, "achieved": achieved, "peak": peak,
                                   "unit": unit, "frac": achieved / peak, "traffic": None, "peak_source": src, "model": model,
                                   "model_tflops": flops / (ms * 1e-3) / 1e12}}))
    plan.apx_plan_destroy()


def host_buffer(shape, dtype, torch):
    """Pinned host tensor when the box can pin that much, else pageable (said in the line)."""
    t = torch.empty(shape, dtype=dtype)
    try:
        return t.pin_memory(), True
    except RuntimeError:
        return t, False


def mem_available_bytes():
    try:
        for line in open("/proc/meminfo"):
            if line.startswith("MemAvailable:"):
                return int(line.split()[1]) * 1024
    except OSError:
        pass
    return None


def run_ours(args, rank, world, local_rank):
    import torch
    import paper_2009_00735_b200 as apx
    from workloads import make_config

    dist = None
    if world > 1 or os.environ.get("APX_BENCH_DIST") == "1":   # (the variable: exercise the NCCL plumbing with a single rank under torchrun)
        import torch.distributed as dist_mod
        dist = dist_mod
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
    torch.cuda.set_device(local_rank)
    dev = torch.device(f"cuda:{local_rank}")

    cfg = args.config
    w = make_config(cfg)
    dirs = apx.apx_dirs_geodesic(w.grid[1]) if w.grid[0] == "geodesic" else apx.apx_dirs_fibonacci(w.D)   # step a3
    accepted = accepted_for(cfg)
    if args.points:                                            # profiling aid: a leading part of the centre list (said in the line)
        w.centres = np.ascontiguousarray(w.centres[:args.points])
    M_all, D, B = len(w.centres), len(dirs), w.B
    # multi-GPU: strong scaling, rank r owns the contiguous slab shard_range(M, r, world) of the centre list
    # (material points are independent; ions replicated; signatures stay sharded; no collective)
    if args.replicas:
        m_begin, m_end = 0, M_all
    else:
        m_begin, m_end = apx.shard_range(M_all, rank, world)
    M = m_end - m_begin
    plan = apx.Plan(w.R, B, dirs, k_lo=w.window[0], k_hi=w.window[1], accepted_types=accepted, device=local_rank,
                    flags=apx.APX_FLAG_FORCE_FFT if args.path == "fft" else 0)
    plan.apx_plan_reserve(len(w.xyz), M)                       # no allocation (= no device sync) inside the timed steps
    xyz = torch.from_numpy(w.xyz).to(dev)
    types = torch.from_numpy(w.types).to(dev)
    centres = torch.from_numpy(w.centres).to(dev)              # ALL centres; run_sharded slices this rank's slab
    sig = torch.empty((M, D, 2), dtype=torch.float32, device=dev)
    counts = torch.empty(M, dtype=torch.int32, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        if args.replicas:
            plan.apx_run(xyz, types, centres, sig, counts)
        else:
            apx.run_sharded(plan, xyz, types, centres, sig, counts, rank=rank, world=world)

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    # device-timed region: K steps, each bracketed by events on the launching (current) stream; L2 flushed (untimed)
    # between steps; the query (k_signature_*) is bracketed separately for the roofline
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    qev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    local_centres = centres[m_begin:m_end]
    barrier()
    t0 = time.time()
    for i in range(args.steps):
        flush.fill_(i & 0xFF)
        ev[i][0].record()
        plan.apx_ingest(xyz, types)
        qev[i][0].record()
        plan.apx_query(local_centres, sig, counts)
        qev[i][1].record()
        ev[i][1].record()
    barrier()
    t1 = time.time()
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    ms = sum(a.elapsed_time(b) for a, b in ev)
    ms_query = sum(a.elapsed_time(b) for a, b in qev)
    n_c = counts.cpu().numpy().astype(np.int64)

    # ---- end to end through the host-pointer entry: HOST buffers, H2D + D2H inside the timed region ----------------
    sig_bytes = M * D * 8
    avail = mem_available_bytes()
    frac_note = None
    Me = M
    if avail is not None and sig_bytes + (6 << 30) > avail // max(1, min(world, 8)):
        Me = max(1, int((avail // max(1, min(world, 8)) - (6 << 30)) // (D * 8)))          # leading part of the slab that fits
        Me = min(Me, M)
        frac_note = f"host memory holds {Me} of this rank's {M} material points: e2e timed on that leading part"
    e2e_steps = max(1, min(args.steps, 5 if cfg == 2 else 2))
    if args.no_e2e:
        Me = min(Me, 2)
    h_sig, pinned = host_buffer((Me, D, 2), torch.float32, torch)
    h_xyz = torch.from_numpy(w.xyz).pin_memory()
    h_types = torch.from_numpy(w.types).pin_memory()
    h_centres = torch.from_numpy(np.ascontiguousarray(w.centres[m_begin:m_begin + Me])).pin_memory()
    h_counts = torch.empty(Me, dtype=torch.int32).pin_memory()
    plan.apx_run_host(h_xyz, h_types, h_centres, h_sig, h_counts)             # warm-up (grows the staging buffers)
    barrier()
    te = time.perf_counter()
    for _ in range(e2e_steps):
        plan.apx_run_host(h_xyz, h_types, h_centres, h_sig, h_counts)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - te
    # the host-path result is the device-path result (checked on the first and last 64 material points): bit for bit,
    # except that ROIs binned in several passes (> 2048 ions) may differ in the last bits from run to run
    k = min(64, Me)
    for a, b in ((h_sig[:k], sig[:k].cpu()), (h_sig[Me - k:Me], sig[Me - k:Me].cpu())):
        assert torch.allclose(a[..., 0], b[..., 0], rtol=2e-6, atol=1e-3) and float((a[..., 1] == b[..., 1]).float().mean()) > 0.999, \
            "host-path result differs from device-path result"
    del h_sig

    tt = torch.tensor([ms, ms_query, e2e_s], dtype=torch.float64, device=dev)
    sums = torch.tensor([float(M), float(n_c.sum()), float(Me)], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        dist.all_reduce(sums, op=dist.ReduceOp.SUM)
    ms, ms_query, e2e_s = [float(v) for v in tt.cpu()]
    M_tot, nc_tot, Me_tot = [float(v) for v in sums.cpu()]
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    n_hist = M_tot * D                                         # histograms all ranks produced per step
    value = n_hist * args.steps / (ms * 1e-3)
    path = "mma" if plan.apx_plan_path() == 1 else "fft"
    half = bool(plan.apx_plan_paired())
    kname = "k_signature_mma" if path == "mma" else "k_signature_fft"
    # (ion, direction) pairs the kernel EXECUTES: in half-grid mode one direction per antipodal pair is binned (the
    # fix-up groups of flagged pairs, < 1e-4 of the work, are not counted)
    d_exec = D // 2 if half else D
    pairs = nc_tot * d_exec
    q_s = ms_query * 1e-3 / args.steps
    pk = load_peaks()
    fp32_tflops = PAIR_FLOP * pairs / q_s / 1e12
    if path == "fft":
        fp32_tflops += 2.5 * B * np.log2(B) * M_tot * d_exec / q_s / 1e12   # unpruned real FFT of the EXECUTED histograms
    fp32_frac = fp32_tflops / pk["fp32_tflops"]
    atom_rate = pairs / 32.0 / q_s                             # one 32-lane shared atomic per 32 pairs
    atom_frac = atom_rate / pk["atom_warp_inst_per_s"]
    W = w.window[1] - w.window[0] + 1
    nb = 4 if B <= 1024 else 8
    groups = -(-d_exec // (128 // nb))
    tensor_flops = 2.0 * 128 * ((4 * W + 15) // 16 * 16) * (B // nb) * groups * M_tot if path == "mma" else 0.0
    h2d = w.xyz.nbytes + w.types.nbytes + Me * 12
    d2h = Me * D * 8 + Me * 4
    bound_is_atom = atom_frac >= fp32_frac
    # counters of the committed ncu capture, scaled from the material points it ran on to those of this run (DRAM traffic is
    # the 8 B per histogram of output, shared-memory wavefronts follow the pairs: both linear in the material points)
    cap_pts = ncu_constant(kname, cfg, "points") or M_all
    scale = M_tot / world / cap_pts
    traffic = ncu_constant(kname, cfg, "dram_bytes")
    traffic = traffic * scale if traffic else None
    lsu = ncu_constant(kname, cfg, "lsu_wavefronts_shared")
    lsu = lsu * scale * world if lsu else None
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak" if args.replicas else "strong",
        "vs_baseline": None, "dtype": "f32 (DFT operands fp16 hi+lo, fp32 accumulate)" if path == "mma" else "f32",
        "data": "synthetic",
        "material_points_per_s": value / D,
        "config": {"workload": WORKLOADS[cfg] + (f" -- ONLY the first {args.points} material points (--points)" if args.points else ""),
                   "kernel_path": path, "half_grid_mode": half,
                   "l2": "flushed between timed steps (256 MiB fill, untimed)",
                   "ions": int(len(w.xyz)), "mean_ions_per_roi": nc_tot / M_tot,
                   "multi_gpu": ("every rank runs the whole workload (replicas)" if args.replicas else
                                 "centre list cut into one contiguous slab per rank (parallel.run_sharded), ions replicated, "
                                 "no collective on the data path")},
        "clocks": clocks,
        "e2e": {"value": Me_tot * D * e2e_steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                "d2h_bytes_per_step": int(d2h), "entry": "apx_run_host", "steps": e2e_steps, "host_buffers_pinned": pinned,
                "material_points": int(Me_tot), "note": frac_note},
        # 8 ingest kernels (k_reset, k_bounds, k_grid_params, k_zero_cells, k_count, k_scan_local, k_scan_add, k_scatter)
        # + k_signature_mma + k_signature_fft over the deferred list (or k_signature_fft alone) per step and rank
        "gpu_launches": (10 if path == "mma" else 9) * args.steps * world,
        "roofline": {"bound": "alu", "kernel": kname,
                     "achieved": atom_rate / 1e9 if bound_is_atom else fp32_tflops,
                     "peak": pk["atom_warp_inst_per_s"] / 1e9 if bound_is_atom else pk["fp32_tflops"],
                     "unit": "G shared-atomic warp-instr/s" if bound_is_atom else "TFLOP/s",
                     "frac": max(atom_frac, fp32_frac),
                     "traffic": traffic,
                     "fp32": {"achieved_tflops": fp32_tflops, "peak_tflops": pk["fp32_tflops"], "frac": fp32_frac},
                     "shared_atomic": {"achieved_gwarp_inst_s": atom_rate / 1e9, "peak_gwarp_inst_s": pk["atom_warp_inst_per_s"] / 1e9,
                                       "frac": atom_frac},
                     "peak_source": pk["source"],
                     "ms_per_launch": ms_query / args.steps,
                     "model": "per executed (ion,direction) pair: 6 flop (FMUL + 2 FFMA + FADD.RM) and 1/32 of a 32-lane shared "
                              "atomic" + ("" if path == "mma" else "; + 2.5 B log2 B flop per histogram (FFT)"),
                     "pairs_per_launch": pairs, "directions_binned_per_point": d_exec,
                     "lsu_wavefronts_per_pair": (lsu / pairs) if lsu else None,
                     "ncu_capture": ncu_constant(kname, cfg, "capture"),
                     "tensor_tflops": tensor_flops / q_s / 1e12 if path == "mma" else None},
    }
    if path == "mma" and lsu:
        # What the kernel actually keeps busy: the shared-memory arrays, 128 B = one wavefront per clock and
        # SM.  LSU wavefronts from the committed ncu capture (scaled by material points); the tensor core's operand reads and the
        # TMA clears go through the same arrays and are counted from the layout (B <= 1024: double-buffered, TMA clears; B = 2048:
        # the clears are plain stores and already in the LSU figure).  Reported beside the algorithmic fraction.
        K, N = B // nb, (4 * W + 15) // 16 * 16
        sbo = 160 if nb == 4 else 192
        hist_bytes = (K // 8) * 16 * sbo
        n_groups = groups * M_tot
        operand = n_groups * (K // 16) * (128 * 16 * 2 + N * 16 * 2) / 128.0
        clear = n_groups * hist_bytes / 128.0 if nb == 4 else 0.0
        clk = q_s * clocks["sm_mhz"] * 1e6 * SM_COUNT * world
        out["roofline"]["shared_memory_pipe"] = {
            "lsu_busy_frac": lsu / clk, "with_tensor_operands_and_tma_clears_est": (lsu + operand + clear) / clk,
            "lsu_wavefronts": lsu, "tensor_operand_wavefronts": operand, "tma_clear_wavefronts": clear, "sm_clocks": clk,
            "note": "executed shared-memory wavefronts / SM clocks: the resource this design saturates.  The second figure counts "
                    "the tensor core's operand reads and the TMA clears against the same 128 B/clk; it can exceed 1, so they have "
                    "some bandwidth of their own"}
    if not args.no_cpu_baseline:
        # bounded samples of the same workload: all cores until >= 10 s of CPU work, then one core on 2 points
        odirs = np.ascontiguousarray(dirs)
        dt, nh, cores, npts = 0.0, 0, 1, 0
        while dt < 10.0 and npts < M_all:
            d1, n1, cores = oracle_sample(w, cfg, odirs, sample_points(M_all, 32, 7 + npts))
            dt += d1; nh += n1; npts += 32
        d1, n1, _ = oracle_sample(w, cfg, odirs, sample_points(M_all, 2, 5), nthreads=1)
        out["cpu_baseline"] = {"value": nh / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                               "sample": f"{npts} seeded material points of {M_all} x {D} directions, {dt:.1f} s",
                               "single_thread": {"value": n1 / d1, "unit": UNIT, "cores": 1,
                                                 "sample": f"2 material points x {D} directions, {d1:.1f} s"},
                               "paper_context": "0.72 material points/s on 1 Xeon Gold 6138 core (PAPER.md L248)"}
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--path", default="auto", choices=["auto", "fft"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--config", type=int, default=4, choices=[2, 3, 4, 5],
                    help="BASELINE.json config, at full size (default 4 = the largest single-GPU configuration)")
    ap.add_argument("--points", type=int, default=0, help="profiling aid: only the first N material points of the config")
    ap.add_argument("--no-e2e", action="store_true", help="profiling aid: skip the end-to-end leg")
    ap.add_argument("--replicas", action="store_true", help="multi-GPU: every rank runs the whole workload (weak scaling)")
    ap.add_argument("--ingest-ions", type=int, default=0, help="time step a1 (ingest) alone on this many ions")
    ap.add_argument("--index", action="store_true", help="time the indexing step (Eq. 3, NEXT-1)")
    ap.add_argument("--index-points", type=int, default=1024)
    ap.add_argument("--index-spacing", type=float, default=1.0, help="orientation grid spacing in degrees")
    ap.add_argument("--fsp", action="store_true", help="time the reciprocal space method (Eq. 2, NEXT-3)")
    ap.add_argument("--fsp-points", type=int, default=1000)
    ap.add_argument("--fsp-L", type=int, default=64)
    ap.add_argument("--fsp-path", type=int, default=0, choices=[0, 1], help="0 = tensor-core kernel, 1 = FP32-pipe kernel")
    ap.add_argument("--peaks", action="store_true", help="run the on-chip peak microbenchmarks and write --peaks-out")
    ap.add_argument("--peaks-out", default=PEAKS_JSON)
    ap.add_argument("--peak-iters", type=int, default=20000)
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.peaks:
        if rank == 0:
            run_peaks(args)
    elif args.ingest_ions > 0:
        if rank == 0:
            run_ingest(args)
    elif args.index:
        if rank == 0:
            run_index(args)
    elif args.fsp:
        if rank == 0:
            run_fsp(args)
    elif args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    # The contract is ONE JSON line on stdout.  Libraries write there too (NCCL prints its version banner to fd 1 when a
    # communicator is created): everything that is not the result line goes to stderr, the line itself to the real stdout.
    sys.stdout.flush()
    _real_stdout = os.fdopen(os.dup(1), "w")
    os.dup2(2, 1)
    sys.stdout = _real_stdout
    try:
        main()
    finally:
        _real_stdout.flush()
