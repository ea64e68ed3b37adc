#!/usr/bin/env python
"""bench.py -- emulated FP64 TFLOPS (2mnk/t, eq. (19)) of ozaki2_dgemm on the BASELINE.json workloads, one JSON
line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2|3|4] [--moduli 16] [--mode 2]
                    [--protocol paper] [--impl reference]

Workload (default): BASELINE configs[2], m = n = k = 8192, eq. (15) inputs with phi = 0.5, N = 16 moduli, revised
fast mode.  --config 3: 16384^3, phi = 4 (default N = 20); --config 4: 4096 x 4096 x 65536, phi = 1 (default N = 16).

A "step" is one pass of the whole hot path S1..S5 (one ozaki2_dgemm call) over one pair of synthetic matrices.
Timing follows the paper's protocol: every step is bracketed by CUDA events that the library records on
the launching stream, `ms_per_step` is the MEDIAN over the K timed steps and `value` = 2mnk / that median; the mean
over the whole timed region (one event pair around all K steps, barrier + synchronize on both sides, max over ranks)
is printed beside it.  `--protocol paper` sets the paper's iteration caps (warm-up until 3 s or 100 iterations,
timed until 12 s or 100).  `value` is measured with A, B, C resident in HBM; `e2e` goes through ozaki2_dgemm_host
with pinned HOST buffers (H2D of A and B and D2H of C inside the timed region).

`roofline` is for the dominant kernel, the batched tcgen05 INT8 GEMM (S3): achieved = N 2mnk / its median launch
duration (stage events); peak = 2 x the measured bf16 BURST figure of MEASURED_PEAKS.json (a step is milliseconds
long, not seconds), with the sustained and nominal figures and a ceiling measured in this very process -- the same
kernel with its epilogue reduced to handing the accumulator back, on random and on all-zero residue planes --
beside it.  `stages` carries ms, algorithmic bytes and GB/s against the measured HBM bandwidth for the streaming
stages; `path` is the north-star figure max(N 2mnk / INT8 peak, bytes / HBM bandwidth) / step time with the same peak.
`cpu_baseline` is the oracle as it stands, timed on this box's host cores on a bounded slab of the same workload.

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
DEFAULT_MODULI = {2: 16, 3: 20, 4: 16}
TRAFFIC_CSV = os.path.join("profiles", "r03_dram_traffic.csv")      # ncu dram bytes per launch, see the .md beside it


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, choices=[2, 3, 4], help="BASELINE.json configs[] index")
    ap.add_argument("--moduli", type=int, default=0, help="number of moduli N (default: 16 / 20 / 16 for config 2 / 3 / 4)")
    ap.add_argument("--mode", type=int, default=2, help="0 accurate, 1 original fast, 2 revised fast (headline)")
    ap.add_argument("--size", type=int, default=0, help="m = n = k override (keeps the config's distribution)")
    ap.add_argument("--phi", type=float, default=None, help="spread parameter of eq. (15) override (paper: 0 .. 4)")
    ap.add_argument("--protocol", default="fixed", choices=["fixed", "paper"],
                    help="paper: P:387-392 iteration caps (warm-up 3 s / 100, timed 12 s / 100) instead of --steps / --warmup")
    ap.add_argument("--sgemm", action="store_true", help="SURVEY 8(f) #1: the FP32 in / FP32 out variant (paper: N = 3..12)")
    ap.add_argument("--zgemm", action="store_true", help="SURVEY 8(f) #4: ozaki2_zgemm on complex FP64 matrices of the config's shape "
                    "(emulated complex TFLOPS = 8mnk / t; no e2e, no stage breakdown)")
    ap.add_argument("--cgemm", action="store_true", help="SURVEY 8(f) #4: ozaki2_cgemm (complex FP32; default N = 9)")
    ap.add_argument("--skip-sweep", action="store_true", help="leave out the sweep over the config's other moduli counts")
    ap.add_argument("--skip-e2e", action="store_true", help="profiling runs only: leave out the host-buffer leg")
    ap.add_argument("--skip-cpu-baseline", action="store_true", help="profiling runs only: leave out the oracle leg")
    ap.add_argument("--skip-ceiling", action="store_true", help="profiling runs only: leave out the MMA-only ceiling runs")
    ap.add_argument("--ceiling-reps", type=int, default=20, help="launches per MMA-only ceiling run (200: sustained, under the power cap)")
    ap.add_argument("--accuracy", action="store_true", help="add max relative error vs the double-double reference "
                    "(P:268) on a sampled slab, and max |R_l| on it (INT32 headroom, P:113)")
    a = ap.parse_args()
    a.moduli_defaulted = not a.moduli
    if not a.moduli:
        a.moduli = 9 if a.cgemm else DEFAULT_MODULI[a.config]
    return a


def workload_shape(args):
    import workloads as W
    c = W.CONFIGS[args.config]
    phi = c["phi"] if args.phi is None else args.phi
    if args.size:
        return args.size, args.size, args.size, phi
    return c["m"], c["n"], c["k"], phi


def workload_name(args, m, n, k, phi, N, mode, f32=False):
    shape = f"m=n=k={m}" if m == n == k else f"m={m}, n={n}, k={k}"
    return (f"BASELINE configs[{args.config}]%s: {shape}, eq.(15) phi={phi}, N={N} moduli, mode={MODE_NAMES[mode]}"
            % (" as SGEMM (SURVEY 8(f) #1)" if f32 else ""))


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

    def wait_first_sample(self, timeout=10.0):
        t0 = time.time()
        while self.proc is not None and not self.lines and time.time() - t0 < timeout:
            time.sleep(0.02)

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.thread.join(timeout=5)
        return self.summarize(self.window)

    def summarize(self, window):
        """Clocks over [window[0], window[1]] (host time) from the samples taken so far; the sampler keeps running."""
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        inside = [ln for ts, ln in list(self.lines) if window[0] <= ts <= window[1]]
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
        return dict(sm_mhz=statistics.median(sm), sm_min_mhz=min(sm), sm_max_mhz=max(mx), power_w_max=max(pw),
                    power_w_median=statistics.median(pw), samples=len(sm), samples_in_timed_region=len(inside),
                    reasons=sorted(reasons))


def profiled_traffic(args, m, n, k, N, mode, f32):
    """DRAM bytes per launch of the dominant kernel from the committed `ncu --set full` captures (TRAFFIC_CSV; the .md
    beside it names the commands and the commit they were taken at), for the workloads that were captured; a constant
    from that file, not a measurement of this run (the figure moves from board to board)."""
    path = os.path.join(ROOT, TRAFFIC_CSV)
    if not os.path.exists(path) or f32:
        return None
    key = f"{m}x{n}x{k}_N{N}_mode{mode}"                       # rows: workload,"kernel",bytes
    with open(path) as fh:
        for line in fh:
            if line.startswith(key + ',"k3_residue_gemm'):
                return float(line.rsplit(",", 1)[1])
    return None


NCU_SUMMARY_MD = os.path.join("profiles", "r03_ncu_summary.md")


def profiled_issue_bounds(args, m, n, k, N, mode, f32, sm_count=148, sm_mhz=1965.0):
    """Plain-ALU (instruction issue) bound of the streaming stages: warp instructions per launch from the
    committed `ncu --set full` summary / (SMs x 4 schedulers x max SM clock), in ms per stage; only for the workload of
    that capture (8192^3, N = 16, mode 2, FP64).  DESIGN.md section 6 derives the peak: one warp instruction per scheduler
    and cycle, 4 schedulers per SM."""
    import re
    path = os.path.join(ROOT, NCU_SUMMARY_MD)
    if not (os.path.exists(path) and (m, n, k) == (8192, 8192, 8192) and N == 16 and mode == 2 and not f32):
        return None
    insts = {}
    with open(path) as fh:
        lines = fh.read().splitlines()
    hdr = next((ln for ln in lines if ln.startswith("| kernel |")), None)
    if hdr is None:
        return None
    cols = [c.strip() for c in hdr.strip("|").split("|")]
    if "warp insts" not in cols:
        return None
    iw = cols.index("warp insts")
    for ln in lines:
        mt = re.match(r"\| `(k\d_\w+)", ln)
        if mt:
            cells = [c.strip() for c in ln.strip("|").split("|")]
            insts[mt.group(1)] = insts.get(mt.group(1), 0.0) + float(cells[iw])
    rate = sm_count * 4 * sm_mhz * 1e6                      # warp instructions per second, whole chip
    groups = {"S1_scaling": ("k1_rows", "k1_rows_finalize", "k1_cols"), "S2_conversion": ("k2_tc_rows", "k2_tc_cols"),
              "S4S5_crt_unscale": ("k5_crt_tc",)}
    out = {}
    for st, ks in groups.items():
        w = sum(insts.get(kk, 0.0) for kk in ks)
        if w:
            out[st] = dict(warp_instructions=w, issue_bound_ms=w / rate * 1e3)
    return out or None


def traffic_capture_commit():
    """The commit the ncu capture behind TRAFFIC_CSV was taken at, as the .md beside it states it."""
    import re
    try:
        with open(os.path.join(ROOT, TRAFFIC_CSV[:-4] + ".md")) as fh:
            mt = re.search(r"commit `([0-9a-f]{7,40})`", fh.read())
        return mt.group(1) if mt else "unknown"
    except OSError:
        return "unknown"


def cpu_slab_shape(m, n, k):
    """Bounded sample of the workload for the oracle: about 1.4e11 residue MACs at N = 16, i.e. 512 rows of A against
    4096 columns of B at k = 8192 (about 7 s on the GPU box's 16 host threads), fewer columns at longer k."""
    ns = max(256, min(n, 4096 * 8192 // max(k, 1)))
    return min(m, 512), min(n, ns), k


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
    m, n, k, phi = workload_shape(args)
    N, mode = args.moduli, args.mode
    ms, ns, _ = cpu_slab_shape(m, n, k)
    # the slab keeps the workload's distribution: same generator, same phi, shape (ms, ns, k)
    A, B = W.eq15_matrices(ms, ns, k, phi, W.seed_for(args.config, 0))
    steps, warm = max(1, min(args.steps, 3)), max(0, min(args.warmup, 1))
    threads = 0
    for _ in range(warm):
        time_oracle_slab(A, B, N, mode, (ms, ns, k))
    t = []
    for _ in range(steps):
        _, dt, threads = time_oracle_slab(A, B, N, mode, (ms, ns, k))
        t.append(dt)
    dt = statistics.median(t)
    val = 2.0 * ms * ns * k / dt / 1e12
    sample = f"oracle dgemm on a {ms}x{ns}x{k} slab (eq. 15, phi={phi}) per step; steps capped at 3, warmup at 1"
    line = dict(impl="reference", metric="emulated_fp64_tflops", value=val, unit="TFLOPS", n_gpus=args.gpus,
                steps=steps, warmup=warm, ms_per_step=dt * 1e3, higher_is_better=True, scaling="weak",
                vs_baseline=None, dtype="int8xint8->int32 residues, fp64 in/out (CPU: int64 / 256-bit integers)",
                data="synthetic",
                config=dict(workload=workload_name(args, m, n, k, phi, N, mode), moduli=N, scaling_mode=MODE_NAMES[mode],
                            sample=sample),
                cpu_baseline=dict(value=val, unit="TFLOPS", cores=threads, kind="oracle", sample=sample),
                e2e=dict(value=val, unit="TFLOPS", h2d_bytes_per_step=0, d2h_bytes_per_step=0),
                gpu_launches=0)
    print(json.dumps(line))
    return 0


def measure_int8_ceiling(pkg, torch, m, n, k, N, stream, reps=20):
    """The GEMM kernels with the epilogue reduced to handing the accumulator back (ozaki2_debug_residue_gemm, variants
    4 = CTA pairs, the path's form, and 3 = one CTA per tile), on uniform random symmetric residues and on all-zero
    planes: what this MMA / TMA loop can deliver on this board at the clocks it gets, next to which the mod-p epilogue
    and the real data are judged.  Board power and SM clock are sampled during each run (nvidia-smi, 10 ms)."""
    if k % 128 or m % 16 or k > (1 << 17):
        return None
    out = {}
    RA = torch.empty((N, m, k), dtype=torch.int8, device="cuda")
    RB = torch.empty((N, n, k), dtype=torch.int8, device="cuda")
    U = torch.empty((16,), dtype=torch.uint8, device="cuda")          # untouched by variants 3, 4
    for name in ("random", "zero"):
        if name == "random":
            g = torch.Generator(device="cuda")
            g.manual_seed(29129)
            for t in (RA, RB):
                for l in range(N):                                     # |r| <= 86 is inside every modulus' symmetric range
                    t[l].copy_(torch.randint(-86, 87, t[l].shape, dtype=torch.int8, device="cuda", generator=g))
        else:
            RA.zero_(); RB.zero_()
        for form, variant in (("pair", 4), ("single", 3)):
            for _ in range(3):
                rc = pkg.ozaki2_debug_residue_gemm(N, m, n, k, RA, RB, U, variant, stream)
                if rc:
                    raise pkg.Ozaki2Error(rc, "ozaki2_debug_residue_gemm")
            torch.cuda.synchronize()
            sampler = ClockSampler(torch.cuda.current_device())
            sampler.start()
            sampler.wait_first_sample()
            evs = [torch.cuda.Event(enable_timing=True) for _ in range(reps + 1)]
            sampler.window[0] = time.time()
            evs[0].record(stream)
            for r in range(reps):
                pkg.ozaki2_debug_residue_gemm(N, m, n, k, RA, RB, U, variant, stream)
                evs[r + 1].record(stream)
            torch.cuda.synchronize()
            sampler.window[1] = time.time()
            clk = sampler.stop()
            ms = statistics.median(evs[r].elapsed_time(evs[r + 1]) for r in range(reps))
            entry = dict(tops=N * 2.0 * m * n * k / (ms * 1e-3) / 1e12, ms=ms, reps=reps, sm_mhz=clk.get("sm_mhz"),
                         power_w_max=clk.get("power_w_max"), reasons=clk.get("reasons"))
            if form == "pair":
                out[name] = entry                                     # the path's kernel: roofline.int8_ceiling_tops.{random, zero}
            else:
                out[name + "_single_cta"] = entry
    del RA, RB
    torch.cuda.empty_cache()
    return out


def run_complex(args, pkg, torch, W, local, world, rank, m, n, k, phi, N, mode, K, Wm, peaks):
    """--zgemm / --cgemm: ozaki2_zgemm / ozaki2_cgemm on complex matrices whose real and imaginary parts are
    eq. (15) draws of the config; emulated complex TFLOPS = 8mnk / t (a complex multiply-add = 4 real ones), median of K
    event-bracketed calls.  The call runs the real path on the (2m x 2k)(2k x n) embedding: 4 real products, so the INT8 work
    is N 2 (2m) n (2k) = 4 N 2mnk."""
    import torch.distributed as dist
    cplx = np.complex64 if args.cgemm else np.complex128
    Ar, Br = W.eq15_matrices(m, n, k, phi, W.seed_for(args.config, rank))
    Ai, Bi = W.eq15_matrices(m, n, k, phi, W.seed_for(args.config, rank) + 5)
    Ad = torch.from_numpy(np.ascontiguousarray((Ar + 1j * Ai).astype(cplx).T)).cuda()
    Bd = torch.from_numpy(np.ascontiguousarray((Br + 1j * Bi).astype(cplx).T)).cuda()
    del Ar, Br, Ai, Bi
    Cd = torch.empty((n, m), dtype=Ad.dtype, device="cuda")
    pkg.ensure_zgemm_workspace(m, n, k, N, mode)
    call = pkg.ozaki2_cgemm if args.cgemm else pkg.ozaki2_zgemm
    stream = torch.cuda.current_stream()

    def step():
        rc = call(m, n, k, 1.0, Ad, m, Bd, k, 0.0, Cd, m, N, mode, stream)
        if rc:
            raise pkg.Ozaki2Error(rc, "ozaki2_cgemm" if args.cgemm else "ozaki2_zgemm")

    sampler = ClockSampler(local)
    sampler.start()
    for _ in range(Wm):
        step()
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(K + 1)]
    sampler.wait_first_sample()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    launches0 = pkg.ozaki2_kernel_launches()
    sampler.window[0] = time.time()
    evs[0].record(stream)
    for s_ in range(K):
        step()
        evs[s_ + 1].record(stream)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler.window[1] = time.time()
    launches = pkg.ozaki2_kernel_launches() - launches0
    clocks = sampler.stop()
    step_ms = [evs[s_].elapsed_time(evs[s_ + 1]) for s_ in range(K)]
    med_ms = statistics.median(step_ms)
    if world > 1:
        tt = torch.tensor([med_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        med_ms = float(tt[0].item())
    cflops = 8.0 * m * n * k
    int8_peak = INT8_OVER_BF16 * peaks["bf16"]
    int8_ops = 4.0 * N * 2.0 * m * n * k
    if rank == 0:
        name = "cgemm" if args.cgemm else "zgemm"
        print(json.dumps(dict(
            metric="emulated_complex_fp32_tflops" if args.cgemm else "emulated_complex_fp64_tflops", value=world * cflops / (med_ms * 1e-3) / 1e12,
            unit="TFLOPS", n_gpus=world, steps=K, warmup=Wm, ms_per_step=med_ms, ms_per_step_min=min(step_ms), ms_per_step_max=max(step_ms),
            higher_is_better=True, scaling="weak", vs_baseline=None,
            dtype="int8xint8->int32 (tcgen05 kind::i8), complex %s in/out" % ("fp32" if args.cgemm else "fp64"), data="synthetic",
            config=dict(workload=f"ozaki2_{name} (SURVEY 8(f) #4) on BASELINE configs[{args.config}] shape m={m}, n={n}, k={k}, eq.(15) "
                                 f"phi={phi} real and imaginary parts, N={N} moduli, mode={MODE_NAMES[mode]}", moduli=N,
                        scaling_mode=MODE_NAMES[mode], l2="inputs larger than L2" if 2 * Ad.element_size() * m * k > 126e6 else "inputs fit L2",
                        parallelism="replicas" if world > 1 else "single GPU"),
            clocks=clocks, e2e=None, gpu_launches=int(launches),
            roofline=dict(bound="tensor", kernel="k3_residue_gemm_pair<EPI_MODP> on the real embedding (2m x 2k)(2k x n): 4 real products",
                          achieved=int8_ops / (med_ms * 1e-3) / 1e12, peak=int8_peak, unit="TFLOP/s", frac=int8_ops / (med_ms * 1e-3) / 1e12 / int8_peak,
                          note="achieved = INT8 ops of the embedded product / WHOLE-call time (no stage events on this entry point)", traffic=None),
            cpu_baseline=None, peaks=dict(hbm_gbs=peaks["hbm_gbs"], bf16_tflops=peaks["bf16"], source=peaks["source"]))))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)

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

    m, n, k, phi = workload_shape(args)
    N, mode = args.moduli, args.mode
    K, Wm = args.steps, max(args.warmup, 3)
    flops = 2.0 * m * n * k
    if args.zgemm or args.cgemm:
        return run_complex(args, pkg, torch, W, local, world, rank, m, n, k, phi, N, mode, K, Wm, peaks)

    # ---- inputs: eq. (15), seeded, one variant per rank (replicas)
    A, B = W.eq15_matrices(m, n, k, phi, W.seed_for(args.config, rank))
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

    sampler = ClockSampler(local)
    sampler.start()                       # nvidia-smi takes a moment to come up: started before the warm-up
    for _ in range(3):
        step()
    if args.protocol == "paper":          # warm-up until 3 s or 100 iterations, timed until 12 s or 100 (>= 5)
        t0 = torch.cuda.Event(enable_timing=True); t1 = torch.cuda.Event(enable_timing=True)
        t0.record(stream); step(); t1.record(stream); torch.cuda.synchronize()
        est = max(t0.elapsed_time(t1) * 1e-3, 1e-6)
        Wm = int(max(3, min(100, 3.0 / est)))
        K = int(max(5, min(100, 12.0 / est)))
    for _ in range(max(0, Wm - 3)):
        step()
    # stage events: created by one record each (torch creates lazily), re-recorded by the library
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(K)]
    for row in evs:
        for ev in row:
            ev.record(stream)
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.wait_first_sample()
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
    step_ms = [evs[s][0].elapsed_time(evs[s][4]) for s in range(K)]
    med_ms = statistics.median(step_ms)
    if world > 1:
        tt = torch.tensor([total_ms, med_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        total_ms, med_ms = float(tt[0].item()), float(tt[1].item())
    mean_ms = total_ms / K
    value = world * flops / (med_ms * 1e-3) / 1e12

    stage_ms = [statistics.median(evs[s][t].elapsed_time(evs[s][t + 1]) for s in range(K)) for t in range(4)]
    # the plain call, without the five stage-event records (which cut the programmatic-launch chain at the stage boundaries):
    # K more calls between one event pair; matters below 4096^3, where launch and prologue latencies are a good part of a call
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    p0.record(stream)
    for _ in range(K):
        step()
    p1.record(stream)
    barrier()
    plain_ms = p0.elapsed_time(p1) / K
    if world > 1:
        tp = torch.tensor([plain_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(tp, op=dist.ReduceOp.MAX)
        plain_ms = float(tp[0].item())
    plain_call = dict(ms_per_call=plain_ms, value=world * flops / (plain_ms * 1e-3) / 1e12, unit="TFLOPS", calls=K,
                      what="mean over K back-to-back plain ozaki2_dgemm calls after the timed region (no stage events)")
    X, Y = float(m) * k + float(k) * n, float(m) * n
    # algorithmic work per launch / stage
    s3_ops = N * flops + (flops if mode == 0 else 0.0)          # mode 0: the auxiliary GEMM sits in S1
    int8_peak = INT8_OVER_BF16 * peaks["bf16"]
    s3_ms = stage_ms[2]
    achieved = N * flops / (s3_ms * 1e-3) / 1e12
    ceiling = None
    if not args.skip_ceiling and not f32:
        ceiling = measure_int8_ceiling(pkg, torch, m, n, k, N, stream, reps=args.ceiling_reps)
    # the kernel oz2_launch_gemm_tc picks for this shape: CTA pairs (cta_group::2) for m > 128 and k <= 2^17, else one CTA per tile
    pair = m > 128 and ((k + 127) // 128) * 128 <= (1 << 17) and os.environ.get("OZAKI2_GEMM", "") != "single"
    s3_kernel = "k3_residue_gemm_pair<EPI_MODP> (cta_group::2" if pair else "k3_residue_gemm<EPI_MODP> (cta_group::1"
    roofline = dict(bound="tensor", kernel=s3_kernel + " tcgen05.mma kind::i8, batched over N moduli)",
                    achieved=achieved, peak=int8_peak, unit="TFLOP/s", frac=achieved / int8_peak,
                    peak_source=f"2 x bf16_tflops burst ({peaks['source']}): another dtype's measured peak x the nominal "
                                "ratio 4.5 / 2.25; MEASURED_PEAKS.json has no INT8 entry",
                    frac_of_2x_sustained=achieved / (INT8_OVER_BF16 * peaks["bf16_sustained"]),
                    frac_of_nominal_4500=achieved / NOMINAL_INT8_TOPS, ms_per_launch=s3_ms,
                    int8_ceiling_tops=ceiling,
                    frac_of_ceiling_random=(achieved / ceiling["random"]["tops"]) if ceiling else None,
                    traffic=profiled_traffic(args, m, n, k, N, mode, f32),
                    traffic_unit=f"bytes per launch (ncu dram read + write, {TRAFFIC_CSV}, captured at commit {traffic_capture_commit()})",
                    algorithmic_bytes=N * X + N * Y)
    if roofline["frac"] > 1.0:
        roofline["note"] = "frac > 1: the kernel beats 2 x the cuBLAS bf16 burst figure; see int8_ceiling_tops"
    stage_bytes = [esz * X if mode != 0 else esz * X + 2 * X, (esz + N) * X, N * X + N * Y, (N + esz) * Y]
    stages = {}
    for nm, ms_, by in zip(("S1_scaling", "S2_conversion", "S3_residue_gemm", "S4S5_crt_unscale"), stage_ms, stage_bytes):
        stages[nm] = dict(ms=ms_, algorithmic_gb=by / 1e9, gbs=by / (ms_ * 1e-3) / 1e9,
                          hbm_frac=by / (ms_ * 1e-3) / 1e9 / peaks["hbm_gbs"])
    stages["S3_residue_gemm"]["int8_tops"] = achieved
    alu = profiled_issue_bounds(args, m, n, k, N, mode, f32)
    if alu:
        for nm, v in alu.items():                           # the plain-ALU bound next to the HBM one
            stages[nm].update(alu_bound_ms=v["issue_bound_ms"], alu_warp_instructions=v["warp_instructions"],
                              hbm_bound_ms=stages[nm]["algorithmic_gb"] / peaks["hbm_gbs"] * 1e3,
                              alu_bound_source=f"{NCU_SUMMARY_MD}: warp instructions / (148 SMs x 4 schedulers x 1965 MHz)")
    total_bytes = (2 * esz + 2 * N) * X + (2 * N + esz) * Y
    t_hbm_ms = total_bytes / (peaks["hbm_gbs"] * 1e9) * 1e3
    t_roof_ms = max(s3_ops / (int8_peak * 1e12) * 1e3, t_hbm_ms)
    t_roof_nominal_ms = max(s3_ops / (NOMINAL_INT8_TOPS * 1e12) * 1e3, t_hbm_ms)
    path = dict(roofline_ms=t_roof_ms, frac=t_roof_ms / med_ms, peak_tops=int8_peak, roofline_ms_nominal_4500=t_roof_nominal_ms,
                frac_nominal_4500=t_roof_nominal_ms / med_ms, hbm_ms=t_hbm_ms, total_algorithmic_gb=total_bytes / 1e9,
                int8_ops=s3_ops, stage_sum_ms=sum(stage_ms))

    # ---- sweep over the other moduli counts the config names (BASELINE metric: "TFLOPS ... vs moduli N"; north_star: ">= 70 % of the
    # roofline at 8192^3 with 14-18 moduli"): the same matrices, same mode, 3 warm-up + 10 timed steps per N with stage events
    sweep = None
    if world == 1 and args.moduli_defaulted and not args.skip_sweep and not f32 and not args.size and args.protocol == "fixed":
        sweep = []
        sw = ClockSampler(local)
        sw.start()
        sw.wait_first_sample()
        Ks = 10
        for Ns in W.CONFIGS[args.config]["moduli"]:
            if Ns == N:
                continue
            pkg.ensure_workspace(m, n, k, Ns, mode)
            for _ in range(3):
                rc = pkg.ozaki2_dgemm(m, n, k, 1.0, Ad, m, Bd, k, 0.0, Cd, m, Ns, mode, stream)
                if rc:
                    raise pkg.Ozaki2Error(rc, "ozaki2_dgemm")
            sevs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(Ks)]
            for row in sevs:
                for ev in row:
                    ev.record(stream)
            torch.cuda.synchronize()
            w0 = time.time()
            for r in range(Ks):
                rc = pkg.dgemm_with_stage_events(m, n, k, 1.0, Ad, m, Bd, k, 0.0, Cd, m, Ns, mode, sevs[r], stream)
                if rc:
                    raise pkg.Ozaki2Error(rc, "ozaki2_dgemm_stages")
            torch.cuda.synchronize()
            w1 = time.time()
            ms_n = statistics.median(sevs[r][0].elapsed_time(sevs[r][4]) for r in range(Ks))
            st_n = [statistics.median(sevs[r][t].elapsed_time(sevs[r][t + 1]) for r in range(Ks)) for t in range(4)]
            bytes_n = (2 * esz + 2 * Ns) * X + (2 * Ns + esz) * Y
            roof_n = max(Ns * flops / (int8_peak * 1e12) * 1e3, bytes_n / (peaks["hbm_gbs"] * 1e9) * 1e3)
            ck = sw.summarize((w0, w1))
            sweep.append(dict(moduli=Ns, ms_per_step=ms_n, value=flops / (ms_n * 1e-3) / 1e12, unit="TFLOPS", steps=Ks, warmup=3,
                              stage_ms=dict(S1=st_n[0], S2=st_n[1], S3=st_n[2], S4S5=st_n[3]),
                              k3_tops=Ns * flops / (st_n[2] * 1e-3) / 1e12, roofline_ms=roof_n, path_frac=roof_n / ms_n,
                              clocks=dict(sm_mhz=ck.get("sm_mhz"), power_w_median=ck.get("power_w_median"), samples=ck.get("samples"),
                                          reasons=ck.get("reasons"))))
        sw.stop()
        sweep.append(dict(moduli=N, ms_per_step=med_ms, value=value, unit="TFLOPS", steps=K, warmup=Wm,
                          stage_ms=dict(S1=stage_ms[0], S2=stage_ms[1], S3=stage_ms[2], S4S5=stage_ms[3]), k3_tops=achieved,
                          roofline_ms=t_roof_ms, path_frac=t_roof_ms / med_ms, note="the headline line above"))
        sweep.sort(key=lambda d: d["moduli"])
        pkg.ensure_workspace(m, n, k, N, mode)
        step()                                  # C of the headline N again: the e2e and cpu_baseline legs compare against it
        torch.cuda.synchronize()

    # ---- e2e: host buffers through ozaki2_dgemm_host / ozaki2_sgemm_host (pinned), copies inside the timed region
    e2e = None
    if not args.skip_e2e:
        Ah = torch.empty((k, m), dtype=tdt, pin_memory=True)
        Bh = torch.empty((n, k), dtype=tdt, pin_memory=True)
        Ch = torch.empty((n, m), dtype=tdt, pin_memory=True)
        Ah.numpy()[...] = A.T
        Bh.numpy()[...] = B.T
        nbytes = pkg.ozaki2_host_scratch_bytes(m, n, k)
        scratch = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        Ke = max(1, min(K, 5))
        host_call = pkg.ozaki2_sgemm_host if f32 else pkg.ozaki2_dgemm_host

        def host_step():
            rc = host_call(m, n, k, 1.0, Ah.data_ptr(), m, Bh.data_ptr(), k, 0.0, Ch.data_ptr(), m, N, mode, scratch, nbytes,
                           stream)
            if rc:
                raise pkg.Ozaki2Error(rc, "ozaki2_dgemm_host")

        host_step()
        barrier()
        ee = [torch.cuda.Event(enable_timing=True) for _ in range(Ke + 1)]
        ee[0].record(stream)
        for r in range(Ke):
            host_step()
            ee[r + 1].record(stream)
        barrier()
        e_ms = statistics.median(ee[r].elapsed_time(ee[r + 1]) for r in range(Ke))
        if world > 1:
            tt = torch.tensor([e_ms], dtype=torch.float64, device="cuda")
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            e_ms = float(tt.item())
        e2e = dict(value=world * flops / (e_ms * 1e-3) / 1e12, unit="TFLOPS", ms_per_step=e_ms, steps=Ke,
                   h2d_bytes_per_step=int(esz * X), d2h_bytes_per_step=int(esz * Y),
                   api="ozaki2_%sgemm_host (pinned host A, B, C)" % ("s" if f32 else "d"))
        # the host-buffer result must be the device-resident one
        e2e["matches_device_path"] = bool(torch.equal(Ch.cuda(), Cd))
        del scratch

    # ---- cpu_baseline: the oracle on a slab of the same matrices (rank 0, N = 1 only), compared with the GPU's C
    cpu = None
    accuracy = None
    if rank == 0 and world == 1 and not args.skip_cpu_baseline:
        ms_, ns_, _ = cpu_slab_shape(m, n, k)
        Cs, dt, threads = time_oracle_slab(A, B, N, mode, (ms_, ns_, k))
        cpu = dict(value=2.0 * ms_ * ns_ * k / dt / 1e12, unit="TFLOPS", cores=threads, kind="oracle", seconds=dt,
                   sample=f"oracle dgemm on rows 0..{ms_ - 1} of A x columns 0..{ns_ - 1} of B, full k={k}, N={N}, "
                          f"mode={MODE_NAMES[mode]}")
        if mode != 0:       # e_i, f_j of modes 1, 2 depend on their own row / column only: the slab of C is comparable
            Cg = Cd[:ns_, :ms_].cpu().numpy().T
            cpu["gpu_slab_bit_exact_vs_oracle"] = bool(np.array_equal(Cg, Cs))
    if rank == 0 and world == 1 and args.accuracy:
        # max elementwise relative error against a double-double reference, on a sampled slab of the GPU's C
        # (SGEMM: the reference is the double-double product of the promoted FP32 inputs)
        from oracle import ozaki2_oracle as O
        ra, ca = min(m, 256), min(n, 512)
        hi, lo = O.dd_reference(np.asfortranarray(A[:ra, :].astype(np.float64)), np.asfortranarray(B[:, :ca].astype(np.float64)))
        Cg = Cd[:ca, :ra].cpu().numpy().T.astype(np.float64)
        nz = hi != 0
        accuracy = dict(max_rel_err=float(np.max(np.abs((Cg[nz] - hi[nz]) - lo[nz]) / np.abs(hi[nz]))),
                        sample=f"rows 0..{ra - 1} x columns 0..{ca - 1} of C vs oracle double-double AB",
                        zero_reference_entries=int(np.sum(~nz)))
        if mode != 0 and not f32:
            g = pkg.dgemm_stages(Ad, Bd, N, mode, C_dev=Cd, want=("e", "f"))
            torch.cuda.synchronize()
            e, f = g["e"].cpu().numpy(), g["f"].cpu().numpy()
            rr, cc = min(m, 32), min(n, 64)
            RA = O.residues(0, N, np.asfortranarray(A[:rr, :]), e[:rr])
            RB = O.residues(1, N, np.asfortranarray(B[:, :cc]), f[:cc])
            _, maxR = O.products(N, RA, RB)
            accuracy["max_abs_residue_product"] = int(maxR)
            accuracy["int32_headroom_bits"] = float(31 - np.log2(max(maxR, 1)))

    if rank == 0:
        line = dict(metric="emulated_fp32_tflops" if f32 else "emulated_fp64_tflops", value=value, unit="TFLOPS",
                    n_gpus=world, steps=K, warmup=Wm, ms_per_step=med_ms, ms_per_step_stat="median of the K timed steps "
                    "(P:387-392); ms_per_step_mean = one event pair around all K steps / K", ms_per_step_mean=mean_ms,
                    value_mean=world * flops / (mean_ms * 1e-3) / 1e12, ms_per_step_min=min(step_ms), ms_per_step_max=max(step_ms),
                    higher_is_better=True, scaling="weak", vs_baseline=None,
                    dtype="int8xint8->int32 (tcgen05 kind::i8), %s in/out" % ("fp32" if f32 else "fp64"), data="synthetic",
                    config=dict(workload=workload_name(args, m, n, k, phi, N, mode, f32), moduli=N, scaling_mode=MODE_NAMES[mode],
                                protocol=args.protocol,
                                l2="inputs larger than L2 (A + B = %.2f GB per step, residue planes %.2f GB)" %
                                   (esz * X / 1e9, N * X / 1e9), parallelism="replicas" if world > 1 else "single GPU"),
                    clocks=clocks, e2e=e2e, plain_call=plain_call, gpu_launches=int(launches), roofline=roofline, stages=stages, path=path,
                    cpu_baseline=cpu, accuracy=accuracy, sweep=sweep,
                    peaks=dict(hbm_gbs=peaks["hbm_gbs"], bf16_tflops=peaks["bf16"],
                               bf16_tflops_sustained=peaks["bf16_sustained"], source=peaks["source"]),
                    context="paper (GH200): cuBLAS DGEMM 60.9 TFLOPS, Ozaki-II DGEMM up to 80.2 TFLOPS (P:48); "
                            "FP64 tensor peak 67 (GH200) / 37 (B200) TFLOPS (P:30)")
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
