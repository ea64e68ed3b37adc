#!/usr/bin/env python
"""bench.py -- emulated FP64 TFLOPS (2mnk/t) of ozaki2_dgemm on BASELINE.json configs[2] (8192^3, eq. (15) inputs
with phi = 0.5, N = 14..18 moduli, revised fast mode), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--moduli 16] [--mode 2] [--impl reference]

A "step" is one pass of the whole hot path S1..S5 (one ozaki2_dgemm call) over one pair of synthetic matrices.
`value` is measured with A, B, C resident in HBM; `e2e` goes through ozaki2_dgemm_host with pinned HOST buffers
(H2D of A and B and D2H of C inside the timed region).  `roofline` is for the dominant kernel, the batched
tcgen05 INT8 GEMM (S3), timed live with CUDA events that the library records on the launching stream at the
stage boundaries of every timed step; `stages` carries the same for the HBM-bound stages; `path` is the
north-star roofline max(N 2mnk / INT8 peak, bytes / HBM bandwidth) over the whole step.  `cpu_baseline` is the
oracle as it stands, timed on this box's host cores on a bounded slab of the same workload.

Multi-GPU: replicas only -- every rank runs the same-shaped problem on its own GPU, no collective on
the data path; `value` is the aggregate.  `--impl reference` times the CPU oracle (rank 0 only).
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

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

MODE_NAMES = {0: "accurate", 1: "fast", 2: "prop"}
NOMINAL_INT8_TOPS = 4500.0          # P:30 (B200 spec sheet, dense)
INT8_OVER_BF16 = 2.0                # guide's nominal ratio 4.5 / 2.25 PFLOP/s


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--moduli", type=int, default=16, help="number of moduli N (BASELINE configs[2]: 14..18)")
    ap.add_argument("--mode", type=int, default=2, help="0 accurate, 1 original fast, 2 revised fast (headline)")
    ap.add_argument("--size", type=int, default=8192, help="m = n = k (8192 is the BASELINE workload)")
    ap.add_argument("--sgemm", action="store_true", help="SURVEY 8(f) #1: the FP32 in / FP32 out variant (paper: N = 3..12); "
                    "no host-buffer entry point exists for it, so e2e is null")
    ap.add_argument("--skip-e2e", action="store_true", help="profiling runs only: leave out the host-buffer leg")
    ap.add_argument("--skip-cpu-baseline", action="store_true", help="profiling runs only: leave out the oracle leg")
    return ap.parse_args()


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            d = json.load(fh)
        return dict(hbm_gbs=float(d["hbm_gbs"]), bf16=float(d["bf16_tflops"]),
                    bf16_sustained=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), source="measured")
    return dict(hbm_gbs=6650.0, bf16=1590.0, bf16_sustained=1400.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines, self.window = index, None, [], [0.0, float("inf")]

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line))

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.thread.join(timeout=5)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        inside = [ln for ts, ln in self.lines if self.window[0] <= ts <= self.window[1]]
        # a timed region shorter than the sampling period: fall back to every sample taken since start()
        for line in (inside if inside else [ln for _, ln in self.lines]):
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["no samples"])
        return dict(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), power_w_max=max(pw), samples=len(sm),
                    reasons=sorted(reasons))


def profiled_traffic(m, N, mode):
    """DRAM bytes per launch of the dominant kernel from the committed ncu --set full capture (profiles/), only for
    the workload that capture was taken on; None otherwise."""
    path = os.path.join(ROOT, "profiles", "r01c_dram_traffic.csv")
    if not (os.path.exists(path) and m == 8192 and N == 16 and mode == 2):
        return None
    with open(path) as fh:
        for line in fh:
            if line.startswith('"k3_residue_gemm<0>"'):
                return float(line.rsplit(",", 1)[1])
    return None


def cpu_slab_shape(m, n, k):
    """Bounded sample of the workload for the oracle: 512 rows of A against 4096 columns of B at the full k
    (about 15 s on the GPU box's 16 host threads at k = 8192, N = 16)."""
    return min(m, 512), min(n, 4096), k


def time_oracle_slab(A, B, N, mode, shape):
    from oracle import ozaki2_oracle as O
    ms, ns, k = shape
    As, Bs = A[:ms, :], B[:, :ns]
    t0 = time.perf_counter()
    Cs = (O.sgemm if As.dtype == np.float32 else O.dgemm)(As, Bs, N, mode)
    dt = time.perf_counter() - t0
    return Cs, dt, O.num_threads()


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, each step a bounded slab of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import workloads as W
    m = n = k = args.size
    N, mode = args.moduli, args.mode
    ms, ns, _ = cpu_slab_shape(m, n, k)
    # the slab keeps the workload's distribution: same generator, same phi, shape (ms, ns, k)
    A, B = W.config_matrices(2, 0, shape=(ms, ns, k))
    steps, warm = max(1, min(args.steps, 3)), max(0, min(args.warmup, 1))
    threads = 0
    for _ in range(warm):
        time_oracle_slab(A, B, N, mode, (ms, ns, k))
    t = []
    for _ in range(steps):
        _, dt, threads = time_oracle_slab(A, B, N, mode, (ms, ns, k))
        t.append(dt)
    dt = sum(t) / len(t)
    val = 2.0 * ms * ns * k / dt / 1e12
    sample = f"oracle dgemm on a {ms}x{ns}x{k} slab (eq. 15, phi=0.5) per step; steps capped at 3, warmup at 1"
    line = dict(impl="reference", metric="emulated_fp64_tflops", value=val, unit="TFLOPS", n_gpus=args.gpus,
                steps=steps, warmup=warm, ms_per_step=dt * 1e3, higher_is_better=True, scaling="weak",
                vs_baseline=None, dtype="int8xint8->int32 residues, fp64 in/out (CPU: int64 / 256-bit integers)",
                data="synthetic",
                config=dict(workload=f"BASELINE configs[2]: m=n=k={m}, eq.(15) phi=0.5, N={N} moduli, mode={MODE_NAMES[mode]}",
                            moduli=N, scaling_mode=MODE_NAMES[mode], sample=sample),
                cpu_baseline=dict(value=val, unit="TFLOPS", cores=threads, kind="oracle", sample=sample),
                e2e=dict(value=val, unit="TFLOPS", h2d_bytes_per_step=0, d2h_bytes_per_step=0),
                gpu_launches=0)
    print(json.dumps(line))
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import numpy as np
    import torch
    import torch.distributed as dist

    import paper_2606_29129_b200 as pkg
    import workloads as W

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    pkg.lib()
    peaks = measured_peaks()

    m = n = k = args.size
    N, mode = args.moduli, args.mode
    K, Wm = args.steps, max(args.warmup, 3)
    flops = 2.0 * m * n * k

    # ---- inputs: eq. (15), seeded, one variant per rank (replicas)
    A, B = W.config_matrices(2, rank, shape=(m, n, k))
    f32 = bool(args.sgemm)
    npdt, tdt, esz = (np.float32, torch.float32, 4) if f32 else (np.float64, torch.float64, 8)
    if f32:
        A, B = np.asfortranarray(A.astype(np.float32)), np.asfortranarray(B.astype(np.float32))
    Ad, Bd = pkg.colmajor_to_device(A, npdt), pkg.colmajor_to_device(B, npdt)
    Cd = torch.empty((n, m), dtype=tdt, device="cuda")
    pkg.ensure_workspace(m, n, k, N, mode)
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step(events=None):
        if events is None:
            rc = (pkg.ozaki2_sgemm if f32 else pkg.ozaki2_dgemm)(m, n, k, 1.0, Ad, m, Bd, k, 0.0, Cd, m, N, mode, stream)
        else:
            rc = pkg.dgemm_with_stage_events(m, n, k, 1.0, Ad, m, Bd, k, 0.0, Cd, m, N, mode, events, stream, f32=f32)
        if rc:
            raise pkg.Ozaki2Error(rc, "ozaki2_dgemm")

    for _ in range(Wm):
        step()
    # stage events: created by one record each (torch creates lazily), re-recorded by the library
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(K)]
    for row in evs:
        for ev in row:
            ev.record(stream)
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local)
    sampler.start()                       # nvidia-smi takes a moment to come up: started before the last warm-ups
    for _ in range(2):
        step()
    barrier()
    launches0 = pkg.ozaki2_kernel_launches()
    sampler.window[0] = time.time()
    t0.record(stream)
    for s in range(K):
        step(evs[s])
    t1.record(stream)
    barrier()
    sampler.window[1] = time.time()
    launches = pkg.ozaki2_kernel_launches() - launches0
    clocks = sampler.stop()
    total_ms = t0.elapsed_time(t1)
    if world > 1:
        tt = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        total_ms = float(tt.item())
    ms_per_step = total_ms / K
    value = world * flops / (ms_per_step * 1e-3) / 1e12

    stage_ms = [statistics.fmean(evs[s][t].elapsed_time(evs[s][t + 1]) for s in range(K)) for t in range(4)]
    X, Y = float(m) * k + float(k) * n, float(m) * n
    # algorithmic work per launch / stage
    s3_ops = N * flops + (flops if mode == 0 else 0.0)
    int8_peak = INT8_OVER_BF16 * peaks["bf16_sustained"]
    s3_ms = stage_ms[2] if mode != 0 else stage_ms[2]            # mode 0: the auxiliary GEMM sits in S1
    achieved = N * flops / (s3_ms * 1e-3) / 1e12
    roofline = dict(bound="tensor", kernel="k3_residue_gemm<false> (tcgen05.mma kind::i8, batched over N moduli)",
                    achieved=achieved, peak=int8_peak, unit="TFLOP/s", frac=achieved / int8_peak,
                    peak_source=f"2 x bf16_tflops_sustained ({peaks['source']}); INT8 has no measured entry",
                    frac_of_burst=achieved / (INT8_OVER_BF16 * peaks["bf16"]),
                    frac_of_nominal_4500=achieved / NOMINAL_INT8_TOPS, ms_per_launch=s3_ms,
                    traffic=profiled_traffic(m, N, mode), traffic_unit="bytes per launch (ncu dram read + write, profiles/r01c)",
                    algorithmic_bytes=N * X + N * Y)
    stage_bytes = [esz * X if mode != 0 else esz * X + 2 * X, (esz + N) * X, N * X + N * Y, (N + esz) * Y]
    stages = {}
    for nm, ms_, by in zip(("S1_scaling", "S2_conversion", "S3_residue_gemm", "S4S5_crt_unscale"), stage_ms, stage_bytes):
        stages[nm] = dict(ms=ms_, algorithmic_gb=by / 1e9, gbs=by / (ms_ * 1e-3) / 1e9,
                          hbm_frac=by / (ms_ * 1e-3) / 1e9 / peaks["hbm_gbs"])
    stages["S3_residue_gemm"]["int8_tops"] = achieved
    total_bytes = (2 * esz + 2 * N) * X + (2 * N + esz) * Y
    t_roof_ms = max(s3_ops / (int8_peak * 1e12), total_bytes / (peaks["hbm_gbs"] * 1e9)) * 1e3
    t_roof_nominal_ms = max(s3_ops / (NOMINAL_INT8_TOPS * 1e12), total_bytes / (peaks["hbm_gbs"] * 1e9)) * 1e3
    path = dict(roofline_ms=t_roof_ms, frac=t_roof_ms / ms_per_step, roofline_ms_nominal_4500=t_roof_nominal_ms,
                frac_nominal_4500=t_roof_nominal_ms / ms_per_step, total_algorithmic_gb=total_bytes / 1e9,
                int8_ops=s3_ops)

    # ---- e2e: host buffers through ozaki2_dgemm_host (pinned), copies inside the timed region
    e2e = None
    if not args.skip_e2e and not f32:
        Ah = torch.empty((k, m), dtype=torch.float64, pin_memory=True)
        Bh = torch.empty((n, k), dtype=torch.float64, pin_memory=True)
        Ch = torch.empty((n, m), dtype=torch.float64, pin_memory=True)
        Ah.numpy()[...] = A.T
        Bh.numpy()[...] = B.T
        nbytes = pkg.ozaki2_host_scratch_bytes(m, n, k)
        scratch = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        Ke = max(1, min(K, 5))

        def host_step():
            rc = pkg.ozaki2_dgemm_host(m, n, k, 1.0, Ah.data_ptr(), m, Bh.data_ptr(), k, 0.0, Ch.data_ptr(), m, N, mode,
                                       scratch, nbytes, stream)
            if rc:
                raise pkg.Ozaki2Error(rc, "ozaki2_dgemm_host")

        host_step()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(Ke):
            host_step()
        e1.record(stream)
        barrier()
        e_ms = e0.elapsed_time(e1) / Ke
        if world > 1:
            tt = torch.tensor([e_ms], dtype=torch.float64, device="cuda")
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            e_ms = float(tt.item())
        e2e = dict(value=world * flops / (e_ms * 1e-3) / 1e12, unit="TFLOPS", ms_per_step=e_ms, steps=Ke,
                   h2d_bytes_per_step=int(8 * X), d2h_bytes_per_step=int(8 * Y),
                   api="ozaki2_dgemm_host (pinned host A, B, C)")
        # the host-buffer result must be the device-resident one
        same = bool(torch.equal(Ch.cuda(), Cd))
        e2e["matches_device_path"] = same
        del scratch

    # ---- cpu_baseline: the oracle on a slab of the same matrices (rank 0, N = 1 only), compared with the GPU's C
    cpu = None
    if rank == 0 and world == 1 and not args.skip_cpu_baseline:
        ms_, ns_, _ = cpu_slab_shape(m, n, k)
        Cs, dt, threads = time_oracle_slab(A, B, N, mode, (ms_, ns_, k))
        cpu = dict(value=2.0 * ms_ * ns_ * k / dt / 1e12, unit="TFLOPS", cores=threads, kind="oracle", seconds=dt,
                   sample=f"oracle dgemm on rows 0..{ms_ - 1} of A x columns 0..{ns_ - 1} of B, full k={k}, N={N}, "
                          f"mode={MODE_NAMES[mode]}")
        if mode != 0:       # e_i, f_j of modes 1, 2 depend on their own row / column only: the slab of C is comparable
            Cg = Cd[:ns_, :ms_].cpu().numpy().T
            cpu["gpu_slab_bit_exact_vs_oracle"] = bool(np.array_equal(Cg, Cs))

    if rank == 0:
        line = dict(metric="emulated_fp32_tflops" if f32 else "emulated_fp64_tflops", value=value, unit="TFLOPS",
                    n_gpus=world, steps=K, warmup=Wm,
                    ms_per_step=ms_per_step, higher_is_better=True, scaling="weak", vs_baseline=None,
                    dtype="int8xint8->int32 (tcgen05 kind::i8), %s in/out" % ("fp32" if f32 else "fp64"), data="synthetic",
                    config=dict(workload=f"BASELINE configs[2]%s: m=n=k={m}, eq.(15) phi=0.5, N={N} moduli, "
                                         f"mode={MODE_NAMES[mode]}" % (" as SGEMM (SURVEY 8(f) #1)" if f32 else ""),
                                moduli=N, scaling_mode=MODE_NAMES[mode],
                                l2="inputs larger than L2 (A + B = %.2f GB per step, residue planes %.2f GB)" %
                                   (esz * X / 1e9, N * X / 1e9), parallelism="replicas" if world > 1 else "single GPU"),
                    clocks=clocks, e2e=e2e, gpu_launches=int(launches), roofline=roofline, stages=stages, path=path,
                    cpu_baseline=cpu, peaks=dict(hbm_gbs=peaks["hbm_gbs"], bf16_tflops=peaks["bf16"],
                                                 bf16_tflops_sustained=peaks["bf16_sustained"], source=peaks["source"]),
                    context="paper (GH200): cuBLAS DGEMM 60.9 TFLOPS, Ozaki-II DGEMM up to 80.2 TFLOPS (P:48); "
                            "FP64 tensor peak 67 (GH200) / 37 (B200) TFLOPS (P:30)")
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
