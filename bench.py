#!/usr/bin/env python
"""bench.py — throughput of the hot path (768-bit Hermitian eigendecomposition) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2] [--impl reference]

One "step" = one pass of the whole hot path (S0 ingest .. S6 export) over one batch of seeded
synthetic input through the C ABI (zkd_diag_herm_ws).  Default workload: BASELINE.json configs[1] = c2, one random
Hermitian N=64 matrix at 768 bit (the paper's random-matrix timing, Fig. 1).  Prints ONE JSON line (rank 0).

Multi-GPU (torchrun): the path does not shard ("replicas only"): every rank runs the same workload on its
own GPU with a different seed stream, no collective on the data path; value = matrices of all ranks / max-over-ranks
time, scaling = "weak".

--impl reference times the CPU oracle (oracle/, MPFR cyclic Jacobi) on the same workload on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "768-bit Hermitian diag matrices/sec"
UNIT = "matrices/s"
WORKLOADS = {
    "c1": "c1: single complex Hermitian N=16, 768-bit, uniform[-1,1] (seed 1001)",
    "c2": "c2: single complex Hermitian N=64, 768-bit, uniform[-1,1] (seed 1002)",
    "c3": "c3: single complex Hermitian N=256, 768-bit, uniform[-1,1] (seed 1003)",
    "c4": "c4: batch of 512 MPS-shaped N=32 PSD trace-1 rank-8 matrices, 768-bit (seed 1004)",
    "c5": "c5: single complex Hermitian N=1024, 64 clusters x 16 spaced 2^-200, 768-bit (seed 1005)",
}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)  # the paper's 10-trial convention
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c2", choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="zkd", choices=["zkd", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the context rows (other configs, saturating batch)")
    return ap.parse_args()


# ---------------------------------------------------------------------------------------------------------------
# clocks
# ---------------------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                       "-i", str(self.idx)], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self) -> dict:
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 9:
                continue
            try:
                sm.append(float(parts[1]))
                mx.append(float(parts[2]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ---------------------------------------------------------------------------------------------------------------
# workloads
# ---------------------------------------------------------------------------------------------------------------
def make_workload(name: str, rank: int, batch: int | None = None):
    import numpy as np

    import zkd_inputs as zi

    if name in ("c1", "c2", "c3"):
        N = {"c1": 16, "c2": 64, "c3": 256}[name]
        b = batch or 1
        # rank r takes seed streams r*b .. r*b+b-1 (rank 0 = the config's own matrix)
        A = np.concatenate([zi.random_hermitian(N, zi.CONFIG_SEEDS[name], rank * b + s) for s in range(b)])
        return N, b, A
    cfg = zi.config(name, batch=batch)
    return cfg["N"], cfg["batch"], cfg["A"]


class Runner:
    """Device-resident buffers for one workload + the call through the C ABI."""

    def __init__(self, z, N, batch, A_np):
        import torch

        self.z, self.N, self.b = z, N, batch
        rb = z.REAL_BYTES
        self.A_host = torch.from_numpy(A_np).pin_memory()
        self.A = self.A_host.cuda()
        self.lam = torch.zeros(batch * N * rb, dtype=torch.uint8, device="cuda")
        self.X = torch.zeros(batch * N * N * 2 * rb, dtype=torch.uint8, device="cuda")
        self.ws = torch.empty(z.diag_herm_bufsize(N, batch), dtype=torch.uint8, device="cuda")
        self.info = torch.zeros(batch * 24, dtype=torch.uint8, device="cuda")
        self.lam_host = torch.zeros(batch * N * rb, dtype=torch.uint8).pin_memory()
        self.X_host = torch.zeros(batch * N * N * 2 * rb, dtype=torch.uint8).pin_memory()

    def step(self):
        self.z.diag_herm_ws(self.N, self.b, self.A, self.lam, self.X, self.ws, self.info)

    def step_e2e(self):
        # HOST buffers in, HOST buffers out, copies inside (zkd_diag_herm_host allocates, copies, runs, copies back)
        self.z.diag_herm_host(self.N, self.b, self.A_host, self.lam_host, self.X_host)

    @property
    def h2d_bytes(self):
        return self.A_host.numel()

    @property
    def d2h_bytes(self):
        return self.lam_host.numel() + self.X_host.numel()


def aggregate(world: int, batch: int, steps: int, seconds: float, device: str = "cuda") -> tuple[float, float]:
    """Whole-job throughput of `world` independent replicas ("replicas only"): every rank processed
    batch*steps matrices in `seconds` of its own device time; the job's time is the MAX over ranks (one all_reduce of a
    scalar, outside the timed region - there is no collective on the data path).  Returns (matrices/s, max seconds)."""
    import torch
    import torch.distributed as dist

    t = torch.tensor([seconds], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    tmax = float(t.item())
    return world * batch * steps / tmax, tmax


def measured_peaks() -> dict:
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except (OSError, ValueError):
        return {}


def roofline_object(gemm_ms, gemm_launches, gemm_macs, i8_ms, i8_launches, i8_macs, imad_peak, steps, total_ms) -> dict:
    """The engine that carries most of the GEMM time.  IMAD path: digit products (IMAD.WIDE) per second against the live
    microbenchmark.  int8 path: s8 x s8 MACs per second, x2 = op/s, against 2 x the measured dense bf16 peak of
    MEASURED_PEAKS.json (int8 is nominally 2 x bf16 on B200; fallback: the profiling guide's nominal 4.5 PFLOP/s int8)."""
    if i8_ms > gemm_ms:
        mp = measured_peaks()
        if "bf16_tflops" in mp:
            peak_tops, src = 2.0 * float(mp["bf16_tflops"]), "2 x MEASURED_PEAKS.json bf16_tflops (burst; kernel timed alone per launch)"
        else:
            peak_tops, src = 4500.0, "fallback: nominal dense int8 4.5 POP/s (B200_PROFILING.md); MEASURED_PEAKS.json absent"
        achieved = 2.0 * i8_macs / (i8_ms * 1e-3) / 1e12
        return {"bound": "tensor", "kernel": "gemm_i8_kernel", "achieved": achieved, "peak": peak_tops, "unit": "TOP/s (int8)",
                "frac": achieved / peak_tops, "traffic": None, "launches": i8_launches, "kernel_ms_per_step": i8_ms / steps,
                "share_of_step": i8_ms / total_ms, "int8_macs_per_step": i8_macs / steps, "peak_source": src,
                "imad_gemm_ms_per_step": gemm_ms / steps}
    achieved = gemm_macs / (gemm_ms * 1e-3) if gemm_ms > 0 else 0.0
    return {"bound": "alu", "kernel": "gemm_digits_kernel", "achieved": achieved / 1e12, "peak": imad_peak / 1e12, "unit": "TIMAD/s",
            "frac": achieved / imad_peak if imad_peak else None, "traffic": None, "launches": gemm_launches,
            "kernel_ms_per_step": gemm_ms / steps, "share_of_step": gemm_ms / total_ms, "digit_macs_per_step": gemm_macs / steps,
            "peak_source": "measured live (zkd_measure_imad_peak): IMAD.WIDE with 64-bit accumulate; nominal 32-bit IMAD rate "
                           "148 SM x 64 lanes/clk x 1.965 GHz = 18.6"}


def timed_steps(torch, runner_step, steps, flush):
    """per-step CUDA-event times (ms) on the current stream; L2 is flushed between steps outside the event pairs"""
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in evs:
        flush.add_(1)  # > L2 size write
        a.record()
        runner_step()
        b.record()
    torch.cuda.synchronize()
    return [a.elapsed_time(b) for a, b in evs]


# ---------------------------------------------------------------------------------------------------------------
# oracle legs (rank 0 only)
# ---------------------------------------------------------------------------------------------------------------
def oracle_sample(name: str):
    """Time the oracle as it stands on a bounded sample of workload `name`.  Returns (matrices/s, cores, sample text)."""
    import oracle
    import zkd_inputs as zi

    cores = oracle.host_threads()
    if name in ("c1", "c2"):
        N, b, A = make_workload(name, 0)
        t0 = time.perf_counter()
        _, _, info = oracle.diag_herm(A, N)  # row-cyclic, 1 thread, full run
        dt = time.perf_counter() - t0
        return 1.0 / dt, 1, f"full run of {name}: {info['sweeps']} sweeps, {info['rotations']} rotations, row-cyclic, 1 thread"
    if name == "c4":
        N, b, A = make_workload(name, 0, batch=2)
        t0 = time.perf_counter()
        for i in range(b):
            oracle.diag_herm(A.reshape(b, -1)[i], N)
        dt = time.perf_counter() - t0
        return b / dt, 1, "first 2 of the 512 matrices, full runs, row-cyclic, 1 thread"
    # c3 / c5: a fixed number of round-robin rounds on all cores, extrapolated to the sweeps a full run needs
    N, b, A = make_workload(name, 0)
    rounds = 8 if name == "c3" else 1
    rot = rounds * (N // 2)
    t0 = time.perf_counter()
    oracle.diag_herm(A, N, ordering="round-robin", threads=cores, max_rotations=rot, want_vectors=True)
    dt = time.perf_counter() - t0
    sweeps = 15 if name == "c3" else 25  # ~15 sweeps random N=256; 25 clustered
    full = dt / rot * (N * (N - 1) // 2) * sweeps
    return 1.0 / full, cores, (f"extrapolated: {rot} rotations of a round-robin sweep on {cores} threads timed, "
                               f"scaled to {sweeps} sweeps x {N * (N - 1) // 2} rotations")


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    vals = []
    cores, sample = 1, ""
    for i in range(args.warmup + args.steps):
        v, cores, sample = oracle_sample(args.workload)
        if i >= args.warmup:
            vals.append(v)
        if sum(1.0 / x for x in vals) > 240:  # keep the whole run within a few minutes
            break
    value = len(vals) / sum(1.0 / v for v in vals)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": len(vals),
        "warmup": args.warmup, "ms_per_step": 1e3 / value, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "mpfr-896bit", "data": "synthetic", "config": {"workload": WORKLOADS[args.workload]},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------------------
# main
# ---------------------------------------------------------------------------------------------------------------
def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return

    import torch
    import torch.distributed as dist

    import paper_2402_11868_b200 as z

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    z.lib()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    N, b, A = make_workload(args.workload, rank)
    run = Runner(z, N, b, A)
    flush = torch.zeros(192 << 20, dtype=torch.uint8, device="cuda")  # 192 MiB > 126 MB L2

    for _ in range(max(args.warmup, 3)):
        run.step()
    torch.cuda.synchronize()

    # ---- timed region: exactly K steps --------------------------------------------------------------------------
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    z.counters_reset()
    z.kernel_timing(True)
    barrier()
    times = timed_steps(torch, run.step, args.steps, flush)
    barrier()
    launches, macs = z.counters()
    gemm_ms, gemm_launches, gemm_macs = z.kernel_timing_read()
    i8_ms, i8_launches, i8_macs = z.kernel_timing_read_i8()
    z.kernel_timing(False)
    clocks = sampler.stop()
    total_ms = sum(times)
    value, tmax = aggregate(world, b, args.steps, total_ms * 1e-3)
    total_ms_max = tmax * 1e3

    # ---- e2e: host buffers through zkd_diag_herm_host -------------------------------------------------------------
    for _ in range(2):
        run.step_e2e()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        run.step_e2e()  # synchronous: returns after the D2H copies completed
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_value, _ = aggregate(world, b, args.steps, e2e_s)

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant GEMM engine: IMAD digit GEMM (integer-multiply pipe) or int8 tcgen05 (tensor pipe) ----
    peak = z.measure_imad_peak(60.0)  # measured, register-only IMAD.WIDE loop on all SMs
    roofline = roofline_object(gemm_ms, gemm_launches, gemm_macs, i8_ms, i8_launches, i8_macs, peak, args.steps, total_ms)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": total_ms_max / args.steps, "ms_per_step_std": statistics.pstdev(times) if len(times) > 1 else 0.0,
        "ms_per_step_all": [round(t, 4) for t in times],
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int32x30 (28-bit digits, 840-bit fixed point)",
        "data": "synthetic",
        "config": {"workload": WORKLOADS[args.workload], "N": N, "batch": b, "prec_bits": 768, "parallelism": "replicas only",
                   "l2": "flushed between steps (192 MiB write)"},
        "eigenpairs_per_s": value * N,
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": run.h2d_bytes, "d2h_bytes_per_step": run.d2h_bytes},
        "gpu_launches": launches,
        "roofline": roofline,
    }

    # ---- context rows: the other configs and a saturating batch (not the headline) --------------------------------
    if not args.no_extra and world == 1:
        extra = {}
        for nm, bb, k in (("c1", 1, 5), ("c2", 1, 5), ("c2", 256, 3), ("c3", 1, 3), ("c4", 512, 2), ("c5", 1, 2)):
            if nm == args.workload and bb == b:
                continue
            try:
                n2, b2, A2 = make_workload(nm, 0, batch=bb)
                r2 = Runner(z, n2, b2, A2)
                r2.step()
                torch.cuda.synchronize()
                z.kernel_timing(True)
                ts = timed_steps(torch, r2.step, k, flush)
                gms, gl, gm = z.kernel_timing_read()
                g8 = z.kernel_timing_read_i8()
                z.kernel_timing(False)
                ms = sum(ts) / len(ts)
                rf = roofline_object(gms, gl, gm, g8[0], g8[1], g8[2], peak, k, sum(ts))
                extra[f"{nm}x{b2}"] = {"matrices_per_s": b2 / (ms * 1e-3), "ms_per_step": ms, "gemm_engine": rf["kernel"],
                                       "gemm_share": rf["share_of_step"], "gemm_frac_of_peak": rf["frac"]}
                del r2
                torch.cuda.empty_cache()
            except Exception as e:  # context only; never fails the bench line
                extra[f"{nm}x{bb}"] = {"error": str(e)[:200]}
        line["other_configs"] = extra

    if not args.no_cpu_baseline:
        v, cores, sample = oracle_sample(args.workload)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}

    print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
