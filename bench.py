#!/usr/bin/env python
"""bench.py -- one JSON line: whole-hot-path throughput of libaptsig on BASELINE.json config 2.

A "step" = one apx_run (ingest + gather + project/bin + DFT + peak + write-out) over the
whole config-2 workload (1000 material points x 10 000 directions, B = 1024, ~241k ions).
  value     device-timed (CUDA events, inputs resident in HBM), L2 flushed between timed steps
  e2e       the same through apx_run_host with pinned HOST buffers (H2D + D2H inside the timed region)
  roofline  dominant kernel vs the FP32 ALU peak
  cpu_baseline  the oracle as it stands on the host cores, bounded sample of the same workload
`--impl reference` times the oracle instead (the tier's reference arm).
Multi-GPU (torchrun): material points are sharded over ranks, ions replicated, no collective on the data path.
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
WORKLOAD = ("cfg2_single_crystal: fcc Al 20^3 nm (~241k ions), 1000 material points x 10000 Fibonacci directions, "
            "R=2.0 nm, B=1024, window [15,34]")
OTHER_WORKLOADS = {
    3: "cfg3_bicrystal: 30^3 nm fcc Al | bcc W (~832k ions), 27000 material points x 40962 geodesic directions, R=2.0 nm, "
       "B=1024, window [15,34], Al filter run",
    4: "cfg4_nanocrystal: 64 Voronoi grains in 60^3 nm fcc Al (~4.8M ions), 175616 material points x 40962 geodesic "
       "directions, R=2.0 nm, B=1024, window [15,34]",
    5: "cfg5_dilute_alloy: 40^3 nm fcc Al-3%Sc + 5% background (~1.5M ions), 64000 material points x 40962 geodesic "
       "directions, R=3.0 nm, B=2048, window [23,51], Al filter",
}
# nominal FP32 peak used as the "alu" roofline denominator (B200_PROFILING.md: 148 SMs, 1965 MHz max SM clock;
# 128 FP32 lanes per SM, FFMA = 2 flop): derived in DESIGN.md "Roofline".
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12


# issue-slot peak: 148 SMs x 4 schedulers x 32 lanes x 1.965 GHz thread-instructions/s
ISSUE_PEAK_TINST = 148 * 4 * 32 * 1.965e9
PAIR_FLOP = 6.0          # FMUL + 2 FFMA + round-down FADD of Eq. 1's projection and floor, per (ion, direction) pair
# issue slots per pair in the MMA kernel's binning loop: 100 instructions per 8 ions x 2 directions of a lane
# (6 LDS.128, 20 packed FP32x2 for projection / floor / hi3, 32 IMAD, 16 ATOMS, loop control)
PAIR_SLOTS_MMA = 6.25
# shared-memory (LSU data pipe) ceiling: one wavefront per SM and clock
LSU_PEAK_WAVEFRONTS = 148 * 1.965e9
# traffic (dram__bytes_read.sum + dram__bytes_write.sum per launch) of the dominant kernel from the committed
# ncu --set full capture (profiles/), config 2; None for a kernel/config that was not captured
NCU_TRAFFIC = {"k_signature_mma": 180.4e6, "k_signature_fft": 29.7e6}
# shared-memory wavefronts per launch (l1tex__data_pipe_lsu_wavefronts_mem_shared.sum) from the same captures
NCU_LSU_WAVEFRONTS = {"k_signature_mma": 1.0856e9, "k_signature_fft": 3.619e9}


def algorithmic_flops(n_pairs, n_hist, B, path):
    """the FP32-pipe work that the method itself prescribes.  Project-and-bin: 6 flop per
    (ion, direction) pair.  DFT: on the MMA path it runs on the tensor pipe and is NOT counted against the FP32
    peak; on the FFT path the unpruned real FFT's 2.5 B log2 B flop per histogram is added."""
    f = PAIR_FLOP * n_pairs
    if path == "fft":
        f += 2.5 * B * np.log2(B) * n_hist
    return f


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


def oracle_sample(w, dirs, n_points, nthreads=0):
    """Time the oracle on the first `n_points` interior-ish material points x all directions."""
    from oracle import oracle as O
    idx = np.linspace(0, len(w.centres) - 1, n_points).astype(np.int64)
    t = time.perf_counter()
    O.signatures(w.xyz, w.types, w.centres[idx], dirs, w.R, w.B, k_lo=w.window[0], k_hi=w.window[1],
                 nthreads=nthreads)
    dt = time.perf_counter() - t
    return dt, n_points * len(dirs), O.num_threads() if nthreads <= 0 else nthreads


def run_reference(args, rank, world):
    """--impl reference: the oracle on the host cores, bounded sample per step (rank 0 only)."""
    if rank != 0:
        return
    from workloads import make_config
    from oracle import oracle as O
    w = make_config(2)
    dirs = O.dirs_fibonacci(w.D)
    n_points = 16
    for _ in range(args.warmup):
        oracle_sample(w, dirs, 2)
    times = []
    cores = 1
    for _ in range(args.steps):
        dt, nh, cores = oracle_sample(w, dirs, n_points)
        times.append(dt)
    total_h = n_points * w.D * args.steps
    v = total_h / sum(times)
    sample = f"{n_points} of {len(w.centres)} material points x {w.D} directions per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "material_points_per_s": v / w.D,
        "config": {"workload": WORKLOAD, "sample": sample},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


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
    bytes_per_ion = 2 * 13 + 2 * 4 + 12 + 16
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


def run_ours(args, rank, world, local_rank):
    import torch
    import paper_2009_00735_b200 as apx
    from workloads import make_config

    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        dist = dist_mod
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
    torch.cuda.set_device(local_rank)
    dev = torch.device(f"cuda:{local_rank}")

    w = make_config(args.config)
    # step a3 through the library
    dirs = apx.apx_dirs_geodesic(w.grid[1]) if w.grid[0] == "geodesic" else apx.apx_dirs_fibonacci(w.D)
    accepted = {0} if args.config in (3, 5) else None       # configs 3 and 5: the Al filter run
    workload = WORKLOAD if args.config == 2 else OTHER_WORKLOADS[args.config]
    # weak scaling: every rank processes the full config-2 centre list of its own replica shard
    # (material points are independent); ions are replicated, no collective on the data path.
    centres_np = w.centres
    M, D, B = len(centres_np), len(dirs), w.B
    plan = apx.Plan(w.R, B, dirs, k_lo=w.window[0], k_hi=w.window[1], accepted_types=accepted, device=local_rank,
                    flags=apx.APX_FLAG_FORCE_FFT if args.path == "fft" else 0)
    xyz = torch.from_numpy(w.xyz).to(dev)
    types = torch.from_numpy(w.types).to(dev)
    centres = torch.from_numpy(centres_np).to(dev)
    sig = torch.empty((M, D, 2), dtype=torch.float32, device=dev)
    counts = torch.empty(M, dtype=torch.int32, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        plan.apx_run(xyz, types, centres, sig, counts)

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    # device-timed region: K steps, each bracketed by events; L2 flushed (untimed) between steps
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    qev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    t0 = time.time()
    for i in range(args.steps):
        flush.fill_(i & 0xFF)
        ev[i][0].record()
        plan.apx_ingest(xyz, types)
        qev[i][0].record()
        plan.apx_query(centres, sig, counts)
        qev[i][1].record()
        ev[i][1].record()
    barrier()
    t1 = time.time()
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    ms = sum(a.elapsed_time(b) for a, b in ev)
    ms_query = sum(a.elapsed_time(b) for a, b in qev)
    n_c = counts.cpu().numpy().astype(np.int64)

    # end to end through the host-pointer entry (pinned buffers; H2D + D2H inside the timed region); the headline config
    # only: configs 3-5 would pin up to 57 GB of host memory for their signatures
    e2e_s, e2e_steps = 0.0, 0
    if args.config == 2:
        h_xyz = torch.from_numpy(w.xyz).pin_memory()
        h_types = torch.from_numpy(w.types).pin_memory()
        h_centres = torch.from_numpy(centres_np).pin_memory()
        h_sig = torch.empty((M, D, 2), dtype=torch.float32).pin_memory()
        h_counts = torch.empty(M, dtype=torch.int32).pin_memory()
        e2e_steps = max(1, min(args.steps, 5))
        plan.apx_run_host(h_xyz, h_types, h_centres, h_sig, h_counts)
        barrier()
        te = time.perf_counter()
        for _ in range(e2e_steps):
            plan.apx_run_host(h_xyz, h_types, h_centres, h_sig, h_counts)
        torch.cuda.synchronize()
        e2e_s = time.perf_counter() - te
        assert torch.equal(h_sig, sig.cpu()), "host-path result differs from device-path result"

    tt = torch.tensor([ms, ms_query, e2e_s], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    ms, ms_query, e2e_s = [float(v) for v in tt.cpu()]
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    n_hist = M * D * world
    value = n_hist * args.steps / (ms * 1e-3)
    pairs = float(n_c.sum()) * D
    path = "mma" if plan.apx_plan_path() == 1 else "fft"
    kname = "k_signature_mma" if path == "mma" else "k_signature_fft"
    flops = algorithmic_flops(pairs, M * D, B, path)
    q_s = ms_query * 1e-3 / args.steps
    achieved = flops / q_s / 1e12
    W = w.window[1] - w.window[0] + 1
    # executed MMA flops: 2 * 128 * N * K per direction group (N = 4W rounded up to 16, K = B / bin parts, G slots per group;
    # half-grid mode bins one direction per antipodal pair)
    nb, n_slots = (4 if B <= 1024 else 8), (D // 2 if plan.apx_plan_paired() else D)
    groups = -(-n_slots // (128 // nb))
    tensor_flops = 2.0 * 128 * ((4 * W + 15) // 16 * 16) * (B // nb) * groups * M if path == "mma" else 0.0
    h2d = w.xyz.nbytes + w.types.nbytes + centres_np.nbytes
    d2h = M * D * 8 + M * 4
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "material_points_per_s": value / D,
        "config": {"workload": workload,
                   "kernel_path": "mma" if plan.apx_plan_path() == 1 else "fft",
                   "half_grid_mode": bool(plan.apx_plan_paired()),
                   "l2": "flushed between timed steps (256 MiB fill, untimed)",
                   "ions": int(len(w.xyz)), "mean_ions_per_roi": float(n_c.mean()),
                   "multi_gpu": "material points sharded per rank, ions replicated, no collective"},
        "clocks": clocks,
        "e2e": ({"value": n_hist * e2e_steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                 "d2h_bytes_per_step": int(d2h), "entry": "apx_run_host", "steps": e2e_steps} if e2e_steps else None),
        # 8 ingest kernels (k_reset, k_bounds, k_grid_params, k_zero_cells, k_count, k_scan_local, k_scan_add, k_scatter)
        # + k_signature_mma + k_signature_fft over the deferred list (or k_signature_fft alone) per step
        "gpu_launches": (10 if path == "mma" else 9) * args.steps,
        "roofline": {"bound": "alu", "kernel": kname,
                     "achieved": achieved, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s",
                     "frac": achieved / FP32_PEAK_TFLOPS, "traffic": NCU_TRAFFIC.get(kname) if args.config == 2 else None,
                     "peak_source": "derived: 148 SM x 128 FP32 lanes x 2 flop x 1.965 GHz (DESIGN.md); "
                                    "MEASURED_PEAKS.json has no FP32 figure",
                     "ms_per_launch": ms_query / args.steps,
                     "model": "6 flop per (ion,direction) pair" + ("" if path == "mma" else " + 2.5 B log2 B flop per histogram"),
                     "pairs_per_launch": pairs,
                     "issue_slot_frac": (PAIR_SLOTS_MMA * pairs / q_s / ISSUE_PEAK_TINST) if path == "mma" else None,
                     # what actually bounds the binning: the shared-memory data pipe (atomics + ion loads), one
                     # wavefront per SM and clock; wavefronts per launch from the committed ncu capture
                     "lsu_wavefront_frac": (NCU_LSU_WAVEFRONTS[kname] / q_s / LSU_PEAK_WAVEFRONTS)
                     if kname in NCU_LSU_WAVEFRONTS and args.config == 2 else None,
                     "tensor_tflops": tensor_flops / q_s / 1e12 if path == "mma" else None},
    }
    if not args.no_cpu_baseline and args.config == 2:
        # bounded sample: batches of 64 material points until >= 10 s of CPU work
        dt, nh, cores, npts = 0.0, 0, 1, 0
        while dt < 10.0 and npts < M:
            d1, n1, cores = oracle_sample(w, np.ascontiguousarray(dirs), 64)
            dt += d1; nh += n1; npts += 64
        out["cpu_baseline"] = {"value": nh / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                               "sample": f"{npts} of {M} material points x {D} directions, {dt:.1f} s",
                               "paper_context": "0.72 material points/s on 1 Xeon Gold 6138 core (PAPER.md L248)"}
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--path", default="auto", choices=["auto", "fft"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--config", type=int, default=2, choices=[2, 3, 4, 5],
                    help="BASELINE.json config to time at full size (default 2 = the bench line; 3-5: device-timed only)")
    ap.add_argument("--ingest-ions", type=int, default=0, help="time step a1 (ingest) alone on this many ions")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.ingest_ions > 0:
        if rank == 0:
            run_ingest(args)
    elif args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
