#!/usr/bin/env python
"""bench.py -- tau00 inversions/s and FP64 TFLOP/s of the LSMS hot path on B200 (BASELINE.json metric).

A step = one pass of the whole hot path over one batch of synthetic LIZ inputs:
t^-1 from phase shifts -> device assembly of M = t^-1 - g0 (K1) -> blocked LU with DMMA Schur updates
(K2-K4) -> inverse of the final Schur complement (K5).  M is re-assembled every step (the factorisation
is in place).  `value` times the device-resident path (inputs already in HBM); `e2e` times the C-ABI
host entry point lsms_tau00_from_host with pinned HOST buffers (H2D of the inputs and D2H of tau00 inside
the timed region).  Flop convention: 8/3 n^3 per matrix (reading A16).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload T|M|P|C|H] [--impl ours|reference]
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

import synth_liz as sl

METRIC = "tau00_inversions_per_sec"
UNIT = "tau00/s"
# nominal dense tensor peaks used for the dtype ratio (blackwell_cuda_programming.md quick-reference table:
# "FP64 Tensor ... B200's 45" TFLOP/s; bf16 2.25 PFLOP/s): FP64 peak = measured bf16 peak * 45/2250
NOMINAL_FP64_OVER_BF16 = 45.0 / 2250.0
FALLBACK_BF16_TFLOPS = 1590.0          # B200_PROFILING.md fallback (burst); sustained ~1400


def workload_label(cfg) -> str:
    src = "BASELINE.json configs[%d]" % cfg.index if cfg.index < 5 else "SURVEY 8(f) f1, paper shape PAPER.md:104"
    return (f"{cfg.name} LIZ ({src}): {cfg.n_sites} sites, lmax={cfg.lmax}, spin_canted={cfg.spin_canted}, "
            f"n={cfg.n}, k={cfg.k}, batch={cfg.batch} per GPU")


def flops_per_matrix(n: int) -> float:
    return 8.0 / 3.0 * float(n) ** 3


class ClockSampler:
    """nvidia-smi clock / throttle-reason sampling during the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.lines: list[str] = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.gpu)], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._pump, daemon=True).start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        # median of the upper half = clocks under load (idle samples at the edges are dropped)
        sm_sorted = sorted(sm)
        load = sm_sorted[len(sm_sorted) // 2:] if sm_sorted else []
        return {"sm_mhz": float(np.median(load)) if load else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def measured_peaks() -> tuple[dict, str]:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)), "measured"
    return {"bf16_tflops": FALLBACK_BF16_TFLOPS, "bf16_tflops_sustained": 1400.0, "hbm_gbs": 6650.0}, "fallback"


def cpu_sample_items(cfg, cores: int) -> list[int]:
    """Bounded sample for the oracle: one item per host thread, spread over the batch (about 10-30 s)."""
    m = max(1, min(cores, cfg.batch))
    return sorted(set(int(round(i * (cfg.batch - 1) / max(m - 1, 1))) for i in range(m)))


def time_oracle(cfg, items) -> tuple[float, float]:
    import oracle
    batch = sl.make_batch(cfg).select(items)
    oracle.gaunt_table(cfg.lmax)                 # table construction is set-up, not the path
    t0 = time.perf_counter()
    _, info = oracle.tau00_batched(batch, "double")
    dt = time.perf_counter() - t0
    assert not info.any()
    return len(items) / dt, dt


def run_reference(args, cfg) -> None:
    """--impl reference: the CPU oracle, as it stands, on a bounded sample of the same workload per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    cores = oracle.max_threads()
    est = flops_per_matrix(cfg.n) / 1.5e9
    items = cpu_sample_items(cfg, cores)
    if est * (args.steps + args.warmup) > 600:          # keep the whole run within a few minutes
        items = items[:max(1, min(len(items), cores))]
    vals = []
    for i in range(args.warmup + args.steps):
        v, dt = time_oracle(cfg, items)
        if i >= args.warmup:
            vals.append((v, dt))
    value = float(np.mean([v for v, _ in vals]))
    ms = float(np.mean([dt for _, dt in vals])) * 1e3
    sample = f"{len(items)} of {cfg.batch} items of workload {cfg.name} per step (one per host thread), FP64 textbook route"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "c128 (f64)", "data": "synthetic",
        "config": {"workload": workload_label(cfg)},
        "tflops": value * flops_per_matrix(cfg.n) / 1e12,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="P", choices=list(sl.CONFIGS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--nb", type=int, default=0, help="outer panel width override (0 = library default)")
    ap.add_argument("--ib", type=int, default=0, help="inner panel width override")
    ap.add_argument("--no-lookahead", action="store_true", help="factor the next panel in front of, not under, the update")
    ap.add_argument("--panel", type=int, default=1, help="K2 variant: 1 register-blocked 512/256 thr, 0 256 thr, -1 L2-resident")
    ap.add_argument("--no-align", action="store_true", help="every outer panel NB wide (no tile-aligning first panel)")
    ap.add_argument("--shared-g0", action="store_true", help="SURVEY 8(f) f3: assemble with one g0 per energy shared by all atoms")
    ap.add_argument("--panel-cluster", type=int, default=0, help="CTAs per matrix in the panel kernel: 0 auto, 1 never, 2/4/8")
    ap.add_argument("--groups", type=int, default=0, help="batch groups on separate streams (0 = library default)")
    args = ap.parse_args()
    cfg = sl.CONFIGS[args.workload]
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    if args.impl == "reference":
        run_reference(args, cfg)
        return

    import torch
    import torch.distributed as dist
    import paper_2308_16317_b200 as lt

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device(dev))
    lt.lib()
    if args.nb or args.ib:
        lt.lsms_set_blocking(args.nb, args.ib)
    lt.lsms_set_lookahead(not args.no_lookahead)
    lt.lsms_set_groups(args.groups)
    lt.lsms_set_panel_variant(args.panel)
    lt.lsms_set_panel_cluster(args.panel_cluster)
    lt.lsms_set_align_first(not args.no_align)

    # ---- inputs: every rank gets its own central atoms (weak scaling: per-GPU work fixed)
    batch = sl.make_batch(cfg, atom_offset=rank * cfg.n_atoms)
    B, n, k = batch.batch, cfg.n, cfg.k
    delta, species, z, pos, mom = lt.device_inputs(batch, dev)
    nspin = cfg.n_spin
    tinv = torch.empty((B, cfg.n_sites, nspin, cfg.lmax + 1), dtype=torch.complex128, device=dev)
    kappa = torch.empty((B,), dtype=torch.complex128, device=dev)
    M = torch.empty((B, n, n), dtype=torch.complex128, device=dev)
    tau = torch.empty((B, k, k), dtype=torch.complex128, device=dev)
    info = torch.empty((B,), dtype=torch.int32, device=dev)
    ws = torch.empty(lt.lsms_workspace_bytes(cfg.n_sites, cfg.lmax, cfg.spin_canted, B), dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    launches = [0]

    def step():
        lt.lsms_tinv_from_phase_shifts(delta, species, z, cfg.lmax, cfg.n_sites, cfg.spin_canted, 2, B, tinv, kappa, stream)
        c = lt.lsms_last_launch_count()
        if args.shared_g0:
            lt.lsms_build_M_shared_g0_batched(tinv, pos, mom if cfg.spin_canted else None, kappa, cfg.lmax, cfg.n_sites,
                                              cfg.spin_canted, cfg.n_atoms, cfg.n_energies, M, ws, stream)
        else:
            lt.lsms_build_M_batched(tinv, pos, mom if cfg.spin_canted else None, kappa, cfg.lmax, cfg.n_sites, cfg.spin_canted,
                                    B, M, ws, stream)
        c += lt.lsms_last_launch_count()
        lt.lsms_tau00_batched(M, cfg.n_sites, cfg.kmax, cfg.spin_canted, B, tau, info, ws, stream)
        launches[0] = c + lt.lsms_last_launch_count()

    def barrier():
        if world > 1:
            dist.barrier()

    def max_over_ranks(x: float) -> float:
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    assert not info.cpu().numpy().any(), "non-zero info in warm-up"

    # ---- timed region: device-resident path
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    barrier(); torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    torch.cuda.synchronize(); barrier()
    ms_total = max_over_ranks(e0.elapsed_time(e1))
    clocks = sampler.stop() if rank == 0 else None
    assert not info.cpu().numpy().any()
    ms_step = ms_total / args.steps
    launches_timed = launches[0] * args.steps          # counted during the timed region (the breakdown step below runs another schedule)
    value = world * B / (ms_step * 1e-3)
    tflops = value * flops_per_matrix(n) / 1e12

    # ---- per-kernel breakdown of one step + roofline of the Schur update (CUDA events on the launch stream).
    # The breakdown step runs the SERIAL schedule (one batch group, no look-ahead), so that every event pair
    # brackets one kernel running alone; in the timed schedule kernels of two groups and the look-ahead stream overlap.
    lt.lsms_set_groups(1); lt.lsms_set_lookahead(False)
    step(); torch.cuda.synchronize()
    lt.lsms_profile_begin()
    step()
    prof = lt.lsms_profile_end()
    lt.lsms_set_groups(args.groups); lt.lsms_set_lookahead(not args.no_lookahead)
    k4 = prof["K4_schur_gemm"]
    total_prof_ms = sum(v["ms"] for v in prof.values())
    k4_tflops = k4["flops"] / (k4["ms"] * 1e-3) / 1e12 if k4["ms"] > 0 else 0.0
    peaks, peak_src = measured_peaks()
    rule_sustained = peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"]) * NOMINAL_FP64_OVER_BF16
    rule_burst = peaks["bf16_tflops"] * NOMINAL_FP64_OVER_BF16
    probe_dmma = lt.lsms_fp64_peak_probe(0, 4000)
    probe_dfma = lt.lsms_fp64_peak_probe(1, 4000)
    # denominator: the larger (stricter) of the live DMMA probe and the rule-derived figures
    peak_fp64 = max(probe_dmma, rule_sustained, rule_burst)
    # algorithmic bytes of the Schur updates of one step: C read + written once, L21 and U12 read once per launch
    nb = args.nb or 64
    w0 = n % 64 if (not args.no_align and nb % 64 == 0 and n % 64 and n % 64 < min(nb, n - k)) else min(nb, n - k)
    alg_bytes, J, W = 0.0, 0, w0
    while J < n - k:
        mr = n - (J + W)
        alg_bytes += B * 16.0 * (2.0 * mr * mr + 2.0 * mr * W)
        J += W; W = min(nb, n - k - J)
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "k4_traffic.csv")
    if os.path.exists(tpath):
        import csv
        for cap in csv.DictReader(open(tpath)):
            if cap["kernel"] == "k_schur_gemm":   # ncu --set full capture of one launch: measured DRAM bytes / algorithmic bytes
                traffic = float(cap["dram_bytes"]) / float(cap["algorithmic_bytes"]) * alg_bytes / max(k4["launches"], 1)
    roofline = {
        "kernel": "k_schur_gemm (K4, Schur update A22 -= L21*U12, inner dimension NB = 64)",
        "bound": "tensor", "achieved": k4_tflops, "peak": peak_fp64, "unit": "TFLOP/s",
        "frac": k4_tflops / peak_fp64 if peak_fp64 else None, "traffic": traffic,
        "algorithmic_bytes_per_launch": alg_bytes / max(k4["launches"], 1),
        "peak_source": "FP64 tensor peak = max(live register-resident DMMA.8x8x4 probe on all SMs, "
                       f"{peak_src} MEASURED_PEAKS bf16 burst / sustained x nominal FP64:bf16 tensor ratio 45/2250); "
                       "MEASURED_PEAKS.json has no FP64 entry",
        "peak_probe_dmma_tflops": probe_dmma, "peak_probe_dfma_tflops": probe_dfma,
        "peak_rule_bf16_burst_x_ratio": rule_burst, "peak_rule_bf16_sustained_x_ratio": rule_sustained,
        "launches_per_step": k4["launches"], "avg_launch_ms": k4["ms"] / max(k4["launches"], 1),
        "flops_per_launch_avg": k4["flops"] / max(k4["launches"], 1),
        "share_of_step": k4["ms"] / total_prof_ms if total_prof_ms else None,
        "breakdown_schedule": "serial (1 batch group, no look-ahead): each event pair brackets one kernel alone",
        "breakdown_ms": {kname: round(v["ms"], 3) for kname, v in prof.items()},
        "breakdown_total_ms": round(total_prof_ms, 3),
        "k1_assembly_gbs": (16.0 * n * n * B / 1e9) / (prof["K1_assemble"]["ms"] * 1e-3) if prof["K1_assemble"]["ms"] > 0 else None,
        "k1_assembly_frac_of_hbm": ((16.0 * n * n * B / 1e9) / (prof["K1_assemble"]["ms"] * 1e-3) / peaks["hbm_gbs"])
                                   if prof["K1_assemble"]["ms"] > 0 else None,
    }

    # ---- end to end through the C-ABI host entry point (pinned host buffers, copies inside the timed region)
    del M, tau, info, ws
    torch.cuda.empty_cache()
    hc = lt.HostCall(cfg.n_sites, cfg.lmax, cfg.spin_canted, 2, B, dev)
    hc.load(batch)
    for _ in range(2):
        hc.run(stream)
    barrier(); torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        hc.run(stream)
    torch.cuda.synchronize()
    e2e_ms = max_over_ranks((time.perf_counter() - t0) * 1e3) / args.steps
    barrier()
    assert not hc.info.numpy().any()
    e2e = {"value": world * B / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": hc.h2d_bytes,
           "d2h_bytes_per_step": hc.d2h_bytes, "ms_per_step": e2e_ms}

    # ---- CPU baseline: the oracle, as it stands, on a bounded sample (rank 0, N = 1 only)
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        cores = oracle.max_threads()
        est = flops_per_matrix(n) / 1.5e9
        if est <= 60.0:
            items = cpu_sample_items(cfg, cores)
            v, dt = time_oracle(cfg, items)
            cpu_baseline = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                            "sample": f"{len(items)} of {B} items of workload {cfg.name} (one per host thread), "
                                      f"FP64 textbook route, {dt:.1f} s", "gflops": v * flops_per_matrix(n) / 1e9}
        else:
            cpu_baseline = {"value": None, "unit": UNIT, "cores": cores, "kind": "oracle",
                            "sample": f"skipped: one {n}x{n} item needs ~{est:.0f} s per core"}

    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "c128 (f64)", "data": "synthetic",
            "config": {"workload": workload_label(cfg),
                       "l2_policy": f"inputs larger than L2: {16.0 * n * n * B / 1e9:.2f} GB of M re-assembled and streamed per step",
                       "parallelism": f"batch sharded over {world} GPU(s), no data-path collective"},
            "tflops": tflops, "tflops_convention": "8/3 n^3 per matrix",
            "frac_fp64_peak": tflops / peak_fp64 if peak_fp64 else None,
            "schedule": {"groups": args.groups or "auto (2)", "lookahead": not args.no_lookahead, "panel_variant": args.panel,
                         "nb": args.nb or 64, "ib": args.ib or 16, "align_first_panel": not args.no_align,
                         "assembly": "one g0 per energy shared by all atoms (f3)" if args.shared_g0 else "every item assembled independently"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches_timed,
            "roofline": roofline, "cpu_baseline": cpu_baseline,
        }))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
