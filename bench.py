"""bench.py -- throughput of the MD4 hot path on B200 (metric of BASELINE.json).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--impl reference]

One "step" = one pass of the whole hot path over one batch of seeded synthetic
shells: md4_build_pairs(bra) + md4_build_pairs(ket) (pair kernel, a1) and md4_compute (fused kernel, a2-a9).
Default workload: BASELINE.json configs[2], uncontracted (ii|ii), 128 x 128 = 16384 shell quartets (the class
the metric is quoted on; it fits one GPU: 3.74 GB of output).  `value` = shell quartets/s with the shells
already resident in HBM; `e2e` = the same through HOST buffers (md4_set_shells + md4_build_pairs +
md4_compute_host, H2D and D2H inside the timed region).  N > 1 (torchrun): every rank runs its own batch
(seed + rank), no data-path collective (quartets are independent); weak scaling.

`--impl reference` times the CPU oracle (oracle/, long-double OS/HGP) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2307_03452_b200 import inputs  # noqa: E402

METRIC = "(ii|ii) shell quartets/s and FP64 TFLOP/s as % of B200 FP64 peak"
UNIT = "quartets/s"
N_SM = 148
FP64_FMA_PER_CLK_PER_SM = 64


def fp64_peak_tflops() -> tuple[float, str]:
    """FP64 peak used as the roofline denominator: 148 SMs x 64 FMA/clk/SM x 2 x max SM
    clock.  The clock is MEASURED_PEAKS.json's sm_max_mhz when the file is there, else the guide's 1965 MHz."""
    mhz, src = 1965.0, "guide clocks.max.sm 1965 MHz"
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            mhz = float(json.load(open(p))["sm_max_mhz"])
            src = "MEASURED_PEAKS.json sm_max_mhz"
        except Exception:
            pass
    return N_SM * FP64_FMA_PER_CLK_PER_SM * 2 * mhz * 1e6 / 1e12, f"148 SM x 64 FP64 FMA/clk x 2 x {mhz:.0f} MHz ({src})"


def workload_by_name(name: str, rank: int = 0):
    if name == "cfg1":
        wl = inputs.config1()
    elif name == "cfg2":
        wl = inputs.config2() if rank == 0 else inputs._perm_config("cfg2 (hh|hh) K=1", 1 + 100 * rank, 64, 5, 10.0, 0.05, 50.0, 64)
    elif name == "cfg3":
        wl = inputs.config3() if rank == 0 else inputs._perm_config("cfg3 (ii|ii) K=1", 2 + 100 * rank, 128, 6, 12.0, 0.05, 50.0, 128)
    elif name == "cfg4":
        wl = inputs.config4() if rank == 0 else inputs._perm_config("cfg4 (ii|ii) K=5/shell", 3 + 100 * rank, 32, 6, 12.0, 0.05, 1.0, 32, K=5)
    else:
        raise SystemExit(f"unknown workload {name}")
    return wl


class ClockSampler:
    """nvidia-smi clocks line of B200_PROFILING.md, sampled every 200 ms while the timed region runs."""

    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.proc = None
        self.path = None

    def start(self):
        try:
            f = tempfile.NamedTemporaryFile("w", suffix=".csv", delete=False)
            self.path = f.name
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.idx}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"], stdout=f,
                                         stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        try:
            for line in open(self.path):
                c = [x.strip() for x in line.split(",")]
                if len(c) < 9:
                    continue
                try:
                    sm.append(float(c[1])); mx.append(float(c[2])); pw.append(float(c[3]))
                except ValueError:
                    continue
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), power_w_max=max(pw), samples=len(sm),
                       reasons=sorted(reasons))
        return out


# ------------------------------------------------------------------------------------------------ oracle leg
def oracle_sample_rate(wl, budget_s: float = 15.0, seed: int = 12345):
    """Times the oracle as it stands (its long-double build, the precision BASELINE.json names; the binary128
    build the parity tests use is ~8x slower) on a seeded sample of wl's quartets, all host cores, one thread
    per quartet.  Returns (quartets/s, cores, n_sampled, seconds)."""
    import oracle

    cores = os.cpu_count() or 1
    sh = oracle.Shells(wl.shells.centers, wl.shells.l, wl.shells.prim_offset, wl.shells.exponents,
                       wl.shells.coefficients)
    rng = np.random.Generator(np.random.PCG64(seed))
    probe = rng.choice(wl.nquartets, size=min(cores, wl.nquartets), replace=False).astype(np.int32)
    t0 = time.perf_counter()
    oracle.compute(sh, wl.bra_ij, wl.ket_ij, subset=probe, nthreads=cores, precision="ld")
    t_probe = max(time.perf_counter() - t0, 1e-6)
    n = int(max(cores, min(wl.nquartets, (budget_s / t_probe) * len(probe))))
    n = min(n, wl.nquartets)
    sub = rng.choice(wl.nquartets, size=n, replace=False).astype(np.int32)
    t0 = time.perf_counter()
    oracle.compute(sh, wl.bra_ij, wl.ket_ij, subset=sub, nthreads=cores, precision="ld")
    dt = time.perf_counter() - t0
    return n / dt, cores, n, dt


def run_reference(args):
    """--impl reference: the CPU oracle on the same config/metric; rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wl = workload_by_name(args.workload)
    per_step_budget = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_sample_rate(wl, budget_s=per_step_budget)
    rates, ns, secs, cores = [], [], [], 1
    for _ in range(args.steps):
        r, cores, n, dt = oracle_sample_rate(wl, budget_s=per_step_budget)
        rates.append(r); ns.append(n); secs.append(dt)
    value = sum(ns) / sum(secs)
    flops = inputs.class_flops(wl.lclass, wl.kclass)
    sample = f"{ns[0]} seeded random quartets of {wl.nquartets} per step, {cores} threads (one quartet per thread at a time)"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * sum(secs) / len(secs), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f80 (x87 long double)", "data": "synthetic",
        "config": {"workload": wl.name, "quartets": wl.nquartets, "lclass": list(wl.lclass), "kclass": list(wl.kclass),
                   "seed": wl.seed},
        "tflops": value * flops / 1e12,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle (long-double build)", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# --------------------------------------------------------------------------------------------------- GPU arm
def reduce_max(x: float, world: int, device: str) -> float:
    """Max over ranks of a host scalar (the only collective of the bench: quartets are independent, S:8(e))."""
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist

    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(world: int, quartets_per_rank: int, ms_per_step: float) -> float:
    """Whole-job quartets/s: every rank processes its own batch of quartets_per_rank in the max-over-ranks time."""
    return world * quartets_per_rank / (ms_per_step * 1e-3)


# ncu --set full capture of the dominant kernel (profiles/r1_eri_kernel_ncu.md): dram read + write bytes per launch
NCU_TRAFFIC_BYTES = {"cfg3": 12.64e9}


def run_gpu(args):
    import torch
    import torch.distributed as dist

    from paper_2307_03452_b200 import build as md4_build
    from paper_2307_03452_b200 import md4

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if local == 0:
        md4_build.ensure_built()   # a checkout has no build artefacts; the kernels themselves have no fallback
    else:
        for _ in range(600):       # the other local ranks wait for rank 0's build
            if os.path.exists(md4_build.LIB):
                break
            time.sleep(0.5)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the MD4 path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    wl = workload_by_name(args.workload, rank)
    s = wl.shells
    eng = md4.Engine(local)
    eng.set_shells(s.centers, s.l, s.prim_offset, s.exponents, s.coefficients)
    stream = torch.cuda.current_stream()
    nq = wl.nquartets
    flops_q = inputs.class_flops(wl.lclass, wl.kclass)
    out_doubles = nq * inputs.class_out_doubles(wl.lclass)
    out = torch.empty(out_doubles, dtype=torch.float64, device=f"cuda:{local}")

    kern_ev = []
    prev = []

    def step(timed: bool):
        # the lists of the step before are released first (md4_free_pairs waits for the work that reads them and
        # hands their buffers to the next md4_build_pairs): the loop a user of the library would write
        while prev:
            b, k = prev.pop()
            b.free(); k.free()
        bra = eng.build_pairs(wl.bra_ij)
        ket = eng.build_pairs(wl.ket_ij)
        if timed:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
        eng.compute(bra, ket, out=out, stream=stream.cuda_stream)
        if timed:
            e1.record(stream)
            kern_ev.append((e0, e1))
        prev.append((bra, ket))

    # ---- device-resident arm: W warm-up steps, then exactly K timed steps
    for _ in range(args.warmup):
        step(False)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    n_launch0 = eng.launch_count()
    barrier()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record(stream)
    for _ in range(args.steps):
        step(True)
    t1.record(stream)
    barrier()
    clocks = sampler.stop() if rank == 0 else {}
    n_launch = eng.launch_count() - n_launch0
    while prev:
        b, k = prev.pop()
        b.free(); k.free()
    ms_total = reduce_max(t0.elapsed_time(t1), world, f"cuda:{local}")
    kern_ms = [a.elapsed_time(b) for a, b in kern_ev]
    ms_step = ms_total / args.steps
    value = whole_job_rate(world, nq, ms_step)

    # ---- end-to-end arm through HOST buffers (same K steps; H2D of shells + pair lists, D2H of all integrals)
    host = torch.empty(out_doubles, dtype=torch.float64, pin_memory=True)
    host_np = host.numpy()
    h2d = int(s.centers.nbytes + s.l.nbytes + s.prim_offset.nbytes + s.exponents.nbytes + s.coefficients.nbytes +
              wl.bra_ij.nbytes + wl.ket_ij.nbytes)
    d2h = int(out_doubles * 8)

    def e2e_step():
        eng.set_shells(s.centers, s.l, s.prim_offset, s.exponents, s.coefficients)
        bra = eng.build_pairs(wl.bra_ij)
        ket = eng.build_pairs(wl.ket_ij)
        eng.compute_host(bra, ket, out=host_np, stream=stream.cuda_stream)
        bra.free(); ket.free()

    e2e_step()
    barrier()
    w0 = time.perf_counter()
    for _ in range(args.steps):
        e2e_step()
    barrier()
    e2e_s = reduce_max(time.perf_counter() - w0, world, f"cuda:{local}")
    e2e_value = whole_job_rate(world, nq, 1e3 * e2e_s / args.steps)

    if rank == 0:
        peak, peak_how = fp64_peak_tflops()
        k_ms = statistics.mean(kern_ms)
        achieved = nq * flops_q / (k_ms * 1e-3) / 1e12
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": wl.name, "quartets_per_gpu": nq, "lclass": list(wl.lclass), "kclass": list(wl.kclass),
                       "seed": wl.seed, "parallelism": f"independent batches x{world}",
                       "l2": "inputs+outputs larger than L2 (H matrices 157 MB, output 3.74 GB for cfg3); no flush"},
            "tflops": value * flops_q / 1e12, "fp64_peak_frac": value * flops_q / 1e12 / (peak * world),
            "flops_per_quartet": flops_q,
            "roofline": {"bound": "tensor", "kernel": "md4::eri_kernel (FP64 DMMA.8x8x4)", "achieved": achieved,
                         "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak, "traffic": NCU_TRAFFIC_BYTES.get(args.workload),
                         "traffic_unit": "bytes per launch (dram read+write, profiles/r1_eri_kernel_ncu.md)",
                         "algorithmic_bytes": out_doubles * 8,
                         "peak_source": peak_how, "kernel_ms": k_ms},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
            "gpu_launches": int(n_launch), "clocks": clocks,
        }
        if world == 1 and not args.no_cpu_baseline:
            r, cores, n, dt = oracle_sample_rate(wl, budget_s=15.0)
            line["cpu_baseline"] = {"value": r, "unit": UNIT, "cores": cores, "kind": "oracle (long-double build)",
                                    "sample": f"{n} seeded random quartets of {nq} in {dt:.1f} s, {cores} threads"}
        print(json.dumps(line), flush=True)
    eng.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg3", choices=["cfg1", "cfg2", "cfg3", "cfg4"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        print("bench.py: note: fewer than 3 warm-up steps", file=sys.stderr)
    return run_reference(args) if args.impl == "reference" else run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
