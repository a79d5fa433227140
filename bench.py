#!/usr/bin/env python
"""bench.py -- tau00 inversions/s and FP64 TFLOP/s of the LSMS hot path on B200 (BASELINE.json metric).

A step = one pass of the whole hot path over one batch of synthetic LIZ inputs:
t^-1 from phase shifts -> device assembly of M = t^-1 - g0 (K1) -> the batch scheduler's elimination (lock-step
blocked LU with DMMA Schur updates K2-K4, or the one-launch small-matrix mode) -> inverse of the final Schur
complement (K5).  M is re-assembled every step (the factorisation is in place).  `value` times the device-resident
path (inputs already in HBM); `e2e` times the C-ABI host entry point lsms_tau00_from_host with pinned HOST buffers
(H2D of the inputs and D2H of tau00 inside the timed region).  Flop convention: 8/3 n^3 per matrix (reading A16).

Several workloads can be timed in one invocation (`--workload P,C,M,T`, the default): the top-level JSON line is the
FIRST one (P = BASELINE.json configs[2], n = 2160, the first size north_star's target names), the others are reported
under "per_workload" with the same keys, so that one driver record covers both target sizes (2160 and 4320) and the
two small-matrix configs.  Every timed run verifies itself ("parity"): after the timed region the tau00 of the timed
schedule is compared with oracle values (the cpu_baseline leg's items and stored values of tests/golden/), and the
residual of the central block column is computed for EVERY item; the process exits non-zero above 1e-10 / 1e-12.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload P,C,M,T] [--impl ours|reference]
"""
from __future__ import annotations

import argparse
import hashlib
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
TAU_TOL, RES_TOL = 1e-10, 1e-12           # north_star: rel. Frobenius error on tau00, normwise residual
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
                                          "-lms", "50", "-i", str(self.gpu)], stdout=subprocess.PIPE, text=True)
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


def time_oracle(cfg, items, atom_offset: int = 0):
    """The oracle as it stands on `items` of the workload: (tau00/s, seconds, tau00 [len(items), k, k])."""
    import oracle
    batch = sl.make_batch(cfg, atom_offset=atom_offset).select(items)
    oracle.gaunt_table(cfg.lmax)                 # table construction is set-up, not the path
    t0 = time.perf_counter()
    tau, info = oracle.tau00_batched(batch, "double")
    dt = time.perf_counter() - t0
    assert not info.any()
    return len(items) / dt, dt, tau


def time_lapack(cfg, items) -> dict:
    """Context beside the oracle: the same items solved by LAPACK (numpy.linalg.solve = zgesv on [M | E], M
    assembled by the oracle), one after the other with the BLAS library's own threading -- what a tuned CPU path
    (the paper's zgetrf/zgetrs on the host) delivers on this box."""
    import oracle
    batch = sl.make_batch(cfg).select(items[:4])
    n, k = cfg.n, cfg.k
    E = np.zeros((n, k), dtype=np.complex128); E[n - k:] = np.eye(k)
    Ms = [oracle.assemble_M(cfg.n_sites, cfg.lmax, cfg.spin_canted, batch.site_pos[b], batch.species[b], batch.delta,
                            batch.moment_dir[b], batch.z[b]) for b in range(batch.batch)]
    t0 = time.perf_counter()
    for M in Ms:
        np.linalg.solve(M, E)
    dt = time.perf_counter() - t0
    v = len(Ms) / dt
    return {"value": v, "unit": UNIT, "gflops": v * flops_per_matrix(n) / 1e9, "kind": "lapack",
            "what": f"numpy.linalg.solve (LAPACK zgesv) on {len(Ms)} oracle-assembled items, BLAS threading as installed"}


def read_golden(key: str, cfg):
    """Stored oracle values of tests/golden/ for this workload: {item: tau00 [k, k]} (written by
    tests/golden/make_golden_full_size.py, which calls only oracle/ and synth_liz/)."""
    out = {}
    gdir = os.path.join(ROOT, "tests", "golden")
    for name in sorted(os.listdir(gdir)) if os.path.isdir(gdir) else []:
        if not name.startswith(f"tau00_full_size_{key}_"):
            continue
        with open(os.path.join(gdir, name)) as f:
            head = f.readline().split()
            if head[1] != key or int(head[3]) != cfg.n or int(head[4]) != cfg.k:
                continue
            ref = np.zeros((cfg.k, cfg.k), dtype=np.complex128)
            for line in f:
                r, c, re, im = line.split()
                ref[int(r), int(c)] = complex(float(re), float(im))
            out[int(head[2])] = ref
    return out


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
        v, dt, _ = time_oracle(cfg, items)
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


def k4_source_hash() -> str:
    """Content hash of the Schur-update kernel's sources: profiles/k4_traffic.csv is stamped with it, so that the
    ncu-measured DRAM traffic is only reported for the kernel it was captured on."""
    h = hashlib.sha256()
    for name in ("gemm.cu", "gemm_body.cuh"):
        with open(os.path.join(ROOT, "paper_2308_16317_b200", "csrc", name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


class Bench:
    def __init__(self, args):
        import torch
        import torch.distributed as dist
        import paper_2308_16317_b200 as lt
        from paper_2308_16317_b200 import shard
        self.torch, self.dist, self.lt, self.shard, self.args = torch, dist, lt, shard, args
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
        # --all-ranks-on-device D: every rank uses cuda:D (one-GPU boxes: the ranks share the GPU by time-slicing, which is
        # fine here because no rank ever waits for another rank's kernel -- the path has no data-path collective); NCCL
        # refuses two ranks on one device, hence gloo for the three small host-side collectives in that case
        self.gpu = args.all_ranks_on_device if args.all_ranks_on_device >= 0 else self.local
        torch.cuda.set_device(self.gpu)
        self.dev = f"cuda:{self.gpu}"
        self.coll_dev = self.dev if args.dist_backend == "nccl" else "cpu"     # where the collectives' tensors live
        if self.world > 1:
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            if args.dist_backend == "nccl":
                dist.init_process_group("nccl", device_id=torch.device(self.dev))
            else:
                dist.init_process_group("gloo")
        lt.lib()
        self.h = lt.lsms_create()
        self.set_schedule(False)
        self.stream = torch.cuda.current_stream()
        self.peaks, self.peak_src = measured_peaks()
        self.probe_dmma = lt.lsms_fp64_peak_probe(self.h, 0, 4000)
        self.probe_dfma = lt.lsms_fp64_peak_probe(self.h, 1, 4000)
        self.rule_sustained = self.peaks.get("bf16_tflops_sustained", self.peaks["bf16_tflops"]) * NOMINAL_FP64_OVER_BF16
        self.rule_burst = self.peaks["bf16_tflops"] * NOMINAL_FP64_OVER_BF16
        # denominator: the larger (stricter) of the live DMMA probe and the rule-derived figures
        self.peak_fp64 = max(self.probe_dmma, self.rule_sustained, self.rule_burst)

    def set_schedule(self, serial: bool):
        a, h = self.args, self.h
        h.set("nb_outer", a.nb).set("ib_inner", a.ib).set("panel_threads", a.panel).set("panel_cluster", a.panel_cluster)
        h.set("align_first", 0 if a.no_align else 1).set("small_mode", a.small_mode)
        h.set("groups", 1 if serial else a.groups).set("lookahead", 0 if (serial or a.no_lookahead) else 1)

    def barrier(self):
        if self.world > 1:
            self.dist.barrier()

    def max_over_ranks(self, x: float) -> float:
        return self.shard.max_over_ranks(x, self.coll_dev)

    # ------------------------------------------------------------------------------------------------
    def run(self, key: str, with_cpu_baseline: bool) -> dict:
        torch, lt, h, args = self.torch, self.lt, self.h, self.args
        cfg = sl.CONFIGS[key]
        world, rank, dev, stream = self.world, self.rank, self.dev, self.stream
        # ---- inputs: every rank gets its own central atoms (weak scaling: per-GPU work fixed)
        atoms = self.shard.shard_atoms(world * cfg.n_atoms, world, rank)
        batch = sl.make_batch(cfg, atom_offset=atoms.start)
        if args.batch_items > 0:                  # the (n, batch) plane: the first K items of the workload, assembled item by item
            batch = batch.select(list(range(min(args.batch_items, batch.batch))))
        B, n, k = batch.batch, cfg.n, cfg.k
        n_species = batch.delta.shape[0]
        delta, species, z, pos, mom = lt.device_inputs(batch, dev)
        momd = mom if cfg.spin_canted else None
        tinv = torch.empty((B, cfg.n_sites, cfg.n_spin, cfg.lmax + 1), dtype=torch.complex128, device=dev)
        kappa = torch.empty((B,), dtype=torch.complex128, device=dev)
        M = torch.empty((B, n, n), dtype=torch.complex128, device=dev)
        tau = torch.empty((B, k, k), dtype=torch.complex128, device=dev)
        info = torch.zeros((3, B), dtype=torch.int32, device=dev)          # one row per stage
        ws = torch.empty(lt.lsms_workspace_bytes(h, cfg.n_sites, cfg.lmax, cfg.spin_canted, B), dtype=torch.uint8, device=dev)
        shared_g0 = not args.per_item_assembly and cfg.n_atoms > 1 and args.batch_items <= 0
        launches = [0]

        def assemble():
            if shared_g0:
                lt.lsms_build_M_shared_g0_batched(h, tinv, pos, momd, kappa, cfg.lmax, cfg.n_sites, cfg.spin_canted,
                                                  cfg.n_atoms, cfg.n_energies, M, info[1], ws, stream)
            else:
                lt.lsms_build_M_batched(h, tinv, pos, momd, kappa, cfg.lmax, cfg.n_sites, cfg.spin_canted, B, M, info[1], ws, stream)

        def step():
            lt.lsms_tinv_from_phase_shifts(h, delta, species, z, cfg.lmax, cfg.n_sites, cfg.spin_canted, n_species, B,
                                           tinv, kappa, info[0], stream)
            c = lt.lsms_last_launch_count(h)
            assemble()
            c += lt.lsms_last_launch_count(h)
            lt.lsms_tau00_batched(h, M, cfg.n_sites, cfg.kmax, cfg.spin_canted, B, tau, info[2], ws, stream)
            launches[0] = c + lt.lsms_last_launch_count(h)

        self.set_schedule(False)
        for _ in range(args.warmup):
            step()
        torch.cuda.synchronize()
        assert not info.cpu().numpy().any(), "non-zero info in warm-up"

        # ---- timed region: device-resident path
        sampler = ClockSampler(self.gpu)
        if rank == 0:
            sampler.start()
            time.sleep(0.25)
        self.barrier(); torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(args.steps):
            step()
        e1.record(stream)
        torch.cuda.synchronize(); self.barrier()
        ms_total = self.max_over_ranks(e0.elapsed_time(e1))
        clocks = sampler.stop() if rank == 0 else None
        assert not info.cpu().numpy().any()
        schedule_used = lt.lsms_last_schedule(h)
        ms_step = ms_total / args.steps
        launches_timed = launches[0] * args.steps      # counted during the timed region (the breakdown step below runs another schedule)
        value = world * B / (ms_step * 1e-3)
        tflops = value * flops_per_matrix(n) / 1e12
        tau_timed = tau.cpu().numpy().transpose(0, 2, 1).copy()          # [b, row, col] of the TIMED schedule's last step
        # N > 1: the k x k outputs of all ranks in global batch order (the only data that crosses GPUs, after the timed region)
        gathered = B
        if world > 1:
            full = self.shard.gather_tau00(tau.to(self.coll_dev), [B] * world)
            gathered = int(full.shape[0])
            if rank == 0 and args.save_gathered:             # [world * B, k, k] as stored (column-major blocks), global batch order
                np.save(args.save_gathered, full.cpu().numpy())

        # ---- per-kernel breakdown of one step + roofline of the dominant kernel (CUDA events on the launch stream).
        # The breakdown step runs the SERIAL schedule (one batch group, no look-ahead), so that every event pair
        # brackets one kernel running alone; in the timed schedule kernels of two groups and the look-ahead stream overlap.
        self.set_schedule(True)
        step(); torch.cuda.synchronize()
        lt.lsms_profile_begin(h)
        step()
        prof = lt.lsms_profile_end(h)
        self.set_schedule(False)
        total_prof_ms = sum(v["ms"] for v in prof.values())
        peaks, peak_fp64 = self.peaks, self.peak_fp64
        peak_note = ("FP64 tensor peak = max(live register-resident DMMA.8x8x4 probe on all SMs, "
                     f"{self.peak_src} MEASURED_PEAKS bf16 burst / sustained x nominal FP64:bf16 tensor ratio 45/2250); "
                     "MEASURED_PEAKS.json has no FP64 entry")
        common = {"peak": peak_fp64, "unit": "TFLOP/s", "bound": "tensor", "peak_source": peak_note,
                  "peak_probe_dmma_tflops": self.probe_dmma, "peak_probe_dfma_tflops": self.probe_dfma,
                  "peak_rule_bf16_burst_x_ratio": self.rule_burst, "peak_rule_bf16_sustained_x_ratio": self.rule_sustained,
                  "breakdown_schedule": "serial (1 batch group, no look-ahead): each event pair brackets one kernel alone",
                  "breakdown_ms": {kname: round(v["ms"], 3) for kname, v in prof.items()},
                  "breakdown_total_ms": round(total_prof_ms, 3),
                  "hidden_ms": round(total_prof_ms - ms_step, 3),
                  "k1_assembly_gbs": (16.0 * n * n * B / 1e9) / (prof["K1_assemble"]["ms"] * 1e-3) if prof["K1_assemble"]["ms"] > 0 else None,
                  "k1_assembly_frac_of_hbm": ((16.0 * n * n * B / 1e9) / (prof["K1_assemble"]["ms"] * 1e-3) / peaks["hbm_gbs"])
                  if prof["K1_assemble"]["ms"] > 0 else None}
        if schedule_used > 0:
            sm = prof["small_mode_lu"]
            ach = sm["flops"] / (sm["ms"] * 1e-3) / 1e12 if sm["ms"] > 0 else 0.0
            kname = (f"k_lu_resident (on-chip small-matrix mode: matrix in the distributed shared memory of a {schedule_used - 100}-CTA "
                     "cluster, whole elimination in one launch; rank-8 DMMA updates from shared memory)" if schedule_used > 100 else
                     f"k_lu_fused (small-matrix mode through L2, {schedule_used} CTA(s) per matrix: whole elimination in one launch; "
                     "DMMA Schur updates inside)")
            roofline = {"kernel": kname,
                        "achieved": ach, "frac": ach / peak_fp64 if peak_fp64 else None, "traffic": None,
                        "launches_per_step": sm["launches"], "avg_launch_ms": sm["ms"] / max(sm["launches"], 1),
                        "flops_per_launch_avg": sm["flops"] / max(sm["launches"], 1),
                        "algorithmic_bytes_per_launch": None,
                        "share_of_step": sm["ms"] / total_prof_ms if total_prof_ms else None, **common}
        else:
            k4 = prof["K4_schur_gemm"]
            k4_tflops = k4["flops"] / (k4["ms"] * 1e-3) / 1e12 if k4["ms"] > 0 else 0.0
            # algorithmic bytes of the Schur updates of one step: C read + written once, L21 and U12 read once per launch
            nb = args.nb or 64
            w0 = n % 64 if (not args.no_align and nb % 64 == 0 and n % 64 and n % 64 < min(nb, n - k)) else min(nb, n - k)
            alg_bytes, J, W = 0.0, 0, w0
            while J < n - k:
                mr = n - (J + W)
                alg_bytes += B * 16.0 * (2.0 * mr * mr + 2.0 * mr * W)
                J += W; W = min(nb, n - k - J)
            traffic, traffic_note = None, "no ncu capture for this kernel version (profiles/k4_traffic.csv is stamped with another source hash)"
            tpath = os.path.join(ROOT, "profiles", "k4_traffic.csv")
            if os.path.exists(tpath):
                import csv
                for cap in csv.DictReader(open(tpath)):
                    if cap["kernel"] == "k_schur_gemm" and cap.get("source_hash", "") == k4_source_hash():
                        # ncu --set full capture of one launch of THIS kernel version: measured DRAM bytes / algorithmic bytes
                        traffic = float(cap["dram_bytes"]) / float(cap["algorithmic_bytes"]) * alg_bytes / max(k4["launches"], 1)
                        traffic_note = "ncu dram__bytes_read+write of one launch (profiles/k4_traffic.csv, same source hash), scaled by algorithmic bytes"
            roofline = {"kernel": "k_schur_gemm (K4, Schur update A22 -= L21*U12, inner dimension NB = 64)",
                        "achieved": k4_tflops, "frac": k4_tflops / peak_fp64 if peak_fp64 else None,
                        "traffic": traffic, "traffic_note": traffic_note,
                        "algorithmic_bytes_per_launch": alg_bytes / max(k4["launches"], 1),
                        "launches_per_step": k4["launches"], "avg_launch_ms": k4["ms"] / max(k4["launches"], 1),
                        "flops_per_launch_avg": k4["flops"] / max(k4["launches"], 1),
                        "share_of_step": k4["ms"] / total_prof_ms if total_prof_ms else None, **common}

        # ---- parity of the timed run, part 1 (untimed): residual of the central block column on EVERY item.
        # M is assembled once more (the elimination overwrote it) and lsms_solve_central_column_batched eliminates a
        # copy of it with the timed schedule; ||M X - E||_F / (||M||_F ||X||_F) is evaluated with torch on the device
        # (verification code, not the product path).
        assemble()
        sws = torch.empty(lt.lsms_solve_workspace_bytes(h, cfg.n_sites, cfg.kmax, cfg.spin_canted, B), dtype=torch.uint8, device=dev)
        X = torch.empty((B, k, n), dtype=torch.complex128, device=dev)
        lt.lsms_solve_central_column_batched(h, M, cfg.n_sites, cfg.kmax, cfg.spin_canted, B, X, info[2], sws, stream)
        torch.cuda.synchronize()
        assert not info.cpu().numpy().any()
        res = []
        for b0 in range(0, B, 8):
            Mm, Xm = M[b0:b0 + 8].transpose(1, 2), X[b0:b0 + 8].transpose(1, 2)
            R = torch.bmm(Mm, Xm)
            R[:, n - k:, :] -= torch.eye(k, dtype=R.dtype, device=dev)
            res.append(torch.linalg.matrix_norm(R) / (torch.linalg.matrix_norm(Mm) * torch.linalg.matrix_norm(Xm)))
            del R
        residual_max = float(torch.cat(res).max())
        x_vs_tau = float(np.abs(X[:, :, n - k:].cpu().numpy().transpose(0, 2, 1) - tau_timed).max())
        del X, sws, M, tau, ws
        torch.cuda.empty_cache()

        # ---- end to end through the C-ABI host entry point (pinned host buffers, copies inside the timed region)
        hc = lt.HostCall(h, cfg.n_sites, cfg.lmax, cfg.spin_canted, n_species, B,
                         n_energies=0 if (args.per_item_assembly or args.batch_items > 0) else cfg.n_energies, device=dev)
        hc.load(batch)
        for _ in range(2):
            hc.run(stream)
        self.barrier(); torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            hc.run(stream)
        torch.cuda.synchronize()
        e2e_ms = self.max_over_ranks((time.perf_counter() - t0) * 1e3) / args.steps
        self.barrier()
        assert not hc.info.numpy().any()
        e2e_equal = bool(np.array_equal(hc.tau00.numpy().transpose(0, 2, 1), tau_timed))
        e2e = {"value": world * B / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": hc.h2d_bytes,
               "d2h_bytes_per_step": hc.d2h_bytes, "ms_per_step": e2e_ms, "bitwise_equal_to_device_path": e2e_equal}
        del hc
        torch.cuda.empty_cache()

        # ---- CPU baseline: the oracle, as it stands, on a bounded sample (rank 0, N = 1 only); its tau00 are the
        # reference values of the parity block
        cpu_baseline, ref_items, ref_tau = None, [], None
        if rank == 0 and world == 1 and with_cpu_baseline:
            import oracle
            cores = oracle.max_threads()
            est = flops_per_matrix(n) / 1.5e9
            if est <= 60.0:
                ref_items = [b for b in cpu_sample_items(cfg, cores) if b < B]
                v, dt, ref_tau = time_oracle(cfg, ref_items)
                cpu_baseline = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"{len(ref_items)} of {B} items of workload {cfg.name} (one per host thread), "
                                          f"FP64 textbook route, {dt:.1f} s", "gflops": v * flops_per_matrix(n) / 1e9,
                                "lapack": time_lapack(cfg, ref_items)}
            else:
                cpu_baseline = {"value": None, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"skipped: one {n}x{n} item needs ~{est:.0f} s per core"}

        # ---- parity of the timed run, part 2: tau00 of the TIMED schedule against oracle values, element by element
        parity = None
        if rank == 0:
            rel_fro, rel_max, items = [], [], []
            refs = [(b, ref_tau[i], "oracle, this run") for i, b in enumerate(ref_items)]
            if world == 1:
                refs += [(b, t, "tests/golden (oracle, stored)") for b, t in read_golden(key, cfg).items() if b < B]
            for b, ref, src in refs:
                d = tau_timed[b] - ref
                rel_fro.append(float(np.linalg.norm(d) / np.linalg.norm(ref)))
                rel_max.append(float(np.abs(d).max() / np.abs(ref).max()))
                items.append({"item": int(b), "source": src})
            parity = {"items": items, "max_rel_fro": max(rel_fro) if rel_fro else None,
                      "max_abs_elem_over_max": max(rel_max) if rel_max else None,
                      "residual_max": residual_max, "residual_items": B,
                      "central_block_of_X_minus_tau00_max_abs": x_vs_tau,
                      "tolerances": {"rel_fro": TAU_TOL, "residual": RES_TOL},
                      "ok": bool(residual_max < RES_TOL and all(v < TAU_TOL for v in rel_fro + rel_max))}

        return {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "c128 (f64)", "data": "synthetic",
            "config": {"workload": workload_label(cfg) + (f"; first {B} items only (--batch-items)" if args.batch_items > 0 else ""),
                       "l2_policy": (f"inputs larger than L2: {16.0 * n * n * B / 1e9:.2f} GB of M re-assembled and streamed per step"
                                     if 16.0 * n * n * B > 200e6 else
                                     f"{16.0 * n * n * B / 1e6:.1f} MB of M per step: L2-resident by design (small-matrix mode); M is re-assembled every step"),
                       "parallelism": f"batch sharded by central atom over {world} GPU(s), no data-path collective; "
                                      f"{gathered} tau00 blocks gathered after the timed region"},
            "n": n, "batch": B, "tflops": tflops, "tflops_convention": "8/3 n^3 per matrix",
            "frac_fp64_peak": tflops / peak_fp64 if peak_fp64 else None,
            "schedule": {"mode": ("on-chip small-matrix mode, cluster of %d CTA(s) (SMs) per matrix, one launch" % (schedule_used - 100)) if schedule_used > 100
                         else ("small-matrix mode through L2, %d CTA(s) per matrix, one launch" % schedule_used) if schedule_used > 0
                         else "lock-step over the batch", "groups": args.groups or "auto", "lookahead": not args.no_lookahead,
                         "panel_threads": args.panel, "nb": args.nb or 64, "ib": args.ib or 16, "align_first_panel": not args.no_align,
                         "assembly": "one g0 per energy shared by all atoms (f3)" if shared_g0 else "every item assembled independently"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches_timed,
            "roofline": roofline, "cpu_baseline": cpu_baseline, "parity": parity,
        }


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="P,C,M,T,H,N,NC",
                    help="comma-separated workloads; the first is the top-level JSON line, the others go under per_workload; "
                         "every one of them appears in the compact `summary` that ends the line")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--batch-items", type=int, default=0, metavar="K",
                    help="time only the first K items of each workload (small batches of large matrices: the paper's one-matrix-per-call pattern, PAPER.md:90-92)")
    ap.add_argument("--dist-backend", default="nccl", choices=["nccl", "gloo"],
                    help="N > 1: backend of the barrier, the MAX over ranks and the gather of the k x k outputs after the timed region")
    ap.add_argument("--all-ranks-on-device", type=int, default=-1, metavar="D",
                    help="N > 1 on a box with fewer GPUs than ranks: every rank uses cuda:D (needs --dist-backend gloo)")
    ap.add_argument("--save-gathered", default="", help="N > 1: rank 0 writes the gathered tau00 blocks of the last step (of the last workload run) to this .npy")
    ap.add_argument("--nb", type=int, default=0, help="outer panel width override (0 = library default)")
    ap.add_argument("--ib", type=int, default=0, help="inner panel width override")
    ap.add_argument("--no-lookahead", action="store_true", help="factor the next panel in front of, not under, the update")
    ap.add_argument("--panel", type=int, default=1, help="K2 footprint: 1 512/256 threads, 0 256 threads")
    ap.add_argument("--no-align", action="store_true", help="every outer panel NB wide (no tile-aligning first panel)")
    ap.add_argument("--per-item-assembly", action="store_true",
                    help="assemble every item independently instead of one g0 per energy shared by all atoms (SURVEY 8(f) f3)")
    ap.add_argument("--panel-cluster", type=int, default=0, help="CTAs per matrix in the panel kernel: 0 auto, 1 never, 2/4/8")
    ap.add_argument("--groups", type=int, default=0, help="batch groups on separate streams (0 = library default)")
    ap.add_argument("--small-mode", type=int, default=0, help="LSMS_OPT_SMALL_MODE: 0 auto, 1 never, 2 when possible, 3..6 forced 1/2/4/8 CTAs")
    args = ap.parse_args()
    keys = [w.strip() for w in args.workload.split(",") if w.strip()]
    for w in keys:
        if w not in sl.CONFIGS:
            raise SystemExit(f"unknown workload {w}")
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.all_ranks_on_device >= 0 and args.dist_backend == "nccl" and int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise SystemExit("--all-ranks-on-device needs --dist-backend gloo (NCCL refuses two ranks on one device)")

    if args.impl == "reference":
        run_reference(args, sl.CONFIGS[keys[0]])
        return

    bench = Bench(args)
    results = {}
    steps = args.steps
    for i, key in enumerate(keys):
        # secondary lines of the tall workloads (H, N, NC: 0.5 - 2 s per step): at most five timed steps each, so that the
        # default run stays within a few minutes; every line states its own "steps"
        args.steps = min(steps, 5) if (i > 0 and sl.CONFIGS[key].n > 5000) else steps
        results[key] = bench.run(key, with_cpu_baseline=not args.no_cpu_baseline)
    args.steps = steps
    if bench.rank == 0:
        line = dict(results[keys[0]])
        if len(keys) > 1:
            line["per_workload"] = {k: results[k] for k in keys[1:]}
        # the LAST key of the line: one compact record per workload (a reader that keeps only the tail of stdout still
        # sees every configuration: ms per step, tau00/s, whole-step and dominant-kernel fractions of the FP64 tensor
        # peak, K1's fraction of the HBM copy rate, end-to-end ms, parity of the timed run)
        def compact(r):
            par, roof = r["parity"] or {}, r["roofline"] or {}
            rnd = lambda v, d: None if v is None else round(v, d)
            sci = lambda v: None if v is None else float(f"{v:.1e}")
            return {"ms": rnd(r["ms_per_step"], 3), "tau00_s": rnd(r["value"], 2),
                    "frac_peak": rnd(r["frac_fp64_peak"], 3), "k_frac": rnd(roof.get("frac"), 3),
                    "k1_hbm": rnd(roof.get("k1_assembly_frac_of_hbm"), 3), "e2e_ms": rnd(r["e2e"]["ms_per_step"], 3),
                    "parity_ok": par.get("ok"), "rel_fro": sci(par.get("max_rel_fro")), "res": sci(par.get("residual_max"))}
        line["summary"] = {k: compact(results[k]) for k in keys}
        print(json.dumps(line))
        bad = [k for k in keys if results[k]["parity"] and not results[k]["parity"]["ok"]]
        if bad:
            print(f"PARITY FAILURE on workload(s) {bad}", file=sys.stderr)
            if bench.world > 1:
                bench.dist.destroy_process_group()
            sys.exit(3)
    if bench.world > 1:
        bench.dist.destroy_process_group()


if __name__ == "__main__":
    main()
