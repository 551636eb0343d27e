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


def workloads_by_name(name: str, rank: int = 0):
    """The batches of one step: one workload for cfg1-cfg4, the 42 of BASELINE.json config 5 (21 classes x K = 1, 3
    per shell) for cfg5."""
    if name == "cfg5":
        return [inputs.config5(ci, K=K, seed_offset=100 * rank) for K in (1, 3) for ci in range(len(inputs.sweep_classes()))]
    return [workload_by_name(name, rank)]


def config_dict(wls, world: int) -> dict:
    """The `config` object of the JSON line; both arms (ours and --impl reference) print exactly this."""
    l2 = "no flush: inputs+outputs of a step exceed the 126 MB L2 (cfg3: H matrices 330 MB, output 3.74 GB)"
    if len(wls) == 1:
        wl = wls[0]
        if wl.nquartets * inputs.class_out_doubles(wl.lclass) * 8 < (126 << 20):
            l2 = "no flush: the pair lists are rebuilt (rewritten) every step; the output of this small batch fits L2"
        return {"workload": wl.name, "quartets_per_gpu": wl.nquartets, "lclass": list(wl.lclass), "kclass": list(wl.kclass),
                "seed": wl.seed, "parallelism": f"independent batches x{world}", "l2": l2}
    return {"workload": f"cfg5 mixed-class sweep: {len(wls)} batches = 21 classes (l in 4..6) x K = 1, 3 per shell, 64 x 64 quartets each",
            "quartets_per_gpu": sum(w.nquartets for w in wls), "lclass": None, "kclass": None, "seed": wls[0].seed,
            "parallelism": f"independent batches x{world}", "l2": l2}


def ncu_traffic(workload: str):
    """dram read+write bytes per launch of the dominant kernel from the committed ncu capture, keyed by the hash of
    the kernel sources it was taken on (profiles/traffic.json).  None (plus the reason) when the library that runs now
    was built from other sources: a figure from another build is never reported."""
    from paper_2307_03452_b200 import build as md4_build

    path = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        tab = json.load(open(path))
    except Exception as e:
        return None, f"profiles/traffic.json unreadable: {e}"
    h = md4_build.source_hash()
    ent = tab.get("captures", {}).get(h)
    if ent is None:
        return None, f"no ncu capture for source hash {h} (captures: {sorted(tab.get('captures', {}))})"
    w = ent.get(workload)
    if w is None:
        return None, f"capture {h} has no entry for {workload}"
    return float(w["dram_bytes_read"]) + float(w["dram_bytes_write"]), f"profiles/traffic.json[{h}][{workload}] ({ent.get('source', '')})"


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
    build the parity tests use is ~8x slower) on a seeded sample of wl's quartets on all host cores: one thread per
    quartet for uncontracted classes, the primitive loop of one quartet at a time spread over the threads for
    contracted ones.  Returns (quartets/s, cores, n_sampled, seconds)."""
    import oracle

    cores = os.cpu_count() or 1
    sh = oracle.Shells(wl.shells.centers, wl.shells.l, wl.shells.prim_offset, wl.shells.exponents,
                       wl.shells.coefficients)
    rng = np.random.Generator(np.random.PCG64(seed))
    contracted = int(np.prod(wl.kclass)) >= cores
    nslice = cores if contracted else 1
    n0 = 1 if contracted else min(cores, wl.nquartets)
    probe = rng.choice(wl.nquartets, size=n0, replace=False).astype(np.int32)
    t0 = time.perf_counter()
    oracle.compute(sh, wl.bra_ij, wl.ket_ij, subset=probe, nthreads=cores, precision="ld", nslice=nslice)
    t_probe = max(time.perf_counter() - t0, 1e-6)
    n = int(max(n0, min(wl.nquartets, (budget_s / t_probe) * n0)))
    if n == n0:
        return n0 / t_probe, cores, n0, t_probe
    sub = rng.choice(wl.nquartets, size=n, replace=False).astype(np.int32)
    t0 = time.perf_counter()
    oracle.compute(sh, wl.bra_ij, wl.ket_ij, subset=sub, nthreads=cores, precision="ld", nslice=nslice)
    dt = time.perf_counter() - t0
    return n / dt, cores, n, dt


def oracle_step(wls, budget_s: float):
    """One bounded oracle pass over the batches of a step.  Returns (whole-step quartets/s = total quartets / sum over
    batches of quartets_b / rate_b, cores, quartets sampled, seconds spent)."""
    t_full, nsamp, spent, cores = 0.0, 0, 0.0, 1
    for wl in wls:
        r, cores, n, dt = oracle_sample_rate(wl, budget_s=budget_s / len(wls))
        t_full += wl.nquartets / r
        nsamp += n
        spent += dt
    return sum(w.nquartets for w in wls) / t_full, cores, nsamp, spent


def total_flops(wls) -> float:
    return float(sum(w.nquartets * inputs.class_flops(w.lclass, w.kclass) for w in wls))


def run_reference(args):
    """--impl reference: the CPU oracle on the same config/metric; rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wls = workloads_by_name(args.workload)
    nq = sum(w.nquartets for w in wls)
    per_step_budget = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_step(wls, per_step_budget)
    rates, ns, secs, cores = [], [], [], 1
    for _ in range(args.steps):
        r, cores, n, dt = oracle_step(wls, per_step_budget)
        rates.append(r); ns.append(n); secs.append(dt)
    value = len(rates) / sum(1.0 / r for r in rates)     # harmonic mean = total quartets / total (extrapolated) time
    sample = (f"{ns[0]} seeded random quartets of {nq} per step in {secs[0]:.1f} s, {cores} threads; step rate = total quartets / "
              f"sum over batches of (quartets / sampled rate)")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * sum(secs) / len(secs), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f80 (x87 long double)", "data": "synthetic",
        "config": config_dict(wls, max(1, args.gpus)),
        "tflops": value * total_flops(wls) / nq / 1e12,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle (long-double build, as it stands: not a tuned CPU code)",
                         "sample": sample},
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
        md4_build.wait_until_built()   # the other local ranks wait for rank 0's build (atomic rename, never a partial file)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the MD4 path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    wls = workloads_by_name(args.workload, rank)
    multi = len(wls) > 1
    eng = md4.Engine(local)
    stream = torch.cuda.current_stream()
    nq = sum(w.nquartets for w in wls)
    flops_step = total_flops(wls)
    out_doubles = [w.nquartets * inputs.class_out_doubles(w.lclass) for w in wls]
    out = torch.empty(max(out_doubles), dtype=torch.float64, device=f"cuda:{local}")

    def upload(wl):
        s = wl.shells
        eng.set_shells(s.centers, s.l, s.prim_offset, s.exponents, s.coefficients)

    if not multi:
        upload(wls[0])            # shells resident in HBM before the timed region; cfg5 changes the shell set per class
    kern_ev = [[] for _ in wls]
    prev = []

    def step(timed: bool):
        # the lists of the step before are released first (md4_free_pairs hands their memory, with the event of the
        # launch that still reads it, to the next md4_build_pairs): the loop a user of the library would write.
        # Nothing in a step blocks the host: copies, pair kernels and the fused kernel are stream-ordered.
        while prev:
            b, k = prev.pop()
            b.free(); k.free()
        for w, wl in enumerate(wls):
            if multi:
                upload(wl)
            bra = eng.build_pairs(wl.bra_ij)
            ket = eng.build_pairs(wl.ket_ij)
            if timed:
                # the kernel's own duration: the events go behind the (device-side) wait for the two pair kernels
                eng.stream_wait_pairs(bra, stream.cuda_stream)
                eng.stream_wait_pairs(ket, stream.cuda_stream)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
            eng.compute(bra, ket, out=out, stream=stream.cuda_stream)
            if timed:
                e1.record(stream)
                kern_ev[w].append((e0, e1))
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
    kern_ms = [statistics.mean(a.elapsed_time(b) for a, b in evs) for evs in kern_ev]
    ms_step = ms_total / args.steps
    value = whole_job_rate(world, nq, ms_step)

    # ---- end-to-end arm through HOST buffers (same K steps; H2D of shells + pair lists, D2H of all integrals)
    host = torch.empty(max(out_doubles), dtype=torch.float64, pin_memory=True)
    host_np = host.numpy()
    h2d = int(sum(w.shells.centers.nbytes + w.shells.l.nbytes + w.shells.prim_offset.nbytes + w.shells.exponents.nbytes +
                  w.shells.coefficients.nbytes + w.bra_ij.nbytes + w.ket_ij.nbytes for w in wls))
    d2h = int(sum(out_doubles) * 8)

    def e2e_step():
        for wl in wls:
            upload(wl)
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

    # ---- end to end with direct digestion: the same K steps, but the integrals are contracted with
    # an AO density on the device (md4_compute_jk_host: J and K out) instead of being shipped to the host
    dg_rng = np.random.Generator(np.random.PCG64(99))
    dg_bufs, dg_keep = [], []
    for wl in wls:
        nbf = int((2 * wl.shells.l + 1).sum())
        pin = [torch.empty(nbf, nbf, dtype=torch.float64, pin_memory=True) for _ in range(3)]   # D, J, K in pinned host memory
        dg_keep.append(pin)
        D, J, K = (t.numpy() for t in pin)
        D[:] = dg_rng.uniform(-1.0, 1.0, (nbf, nbf)); J[:] = 0.0; K[:] = 0.0
        dg_bufs.append((D, J, K))
    dg_h2d = int(sum(w.shells.centers.nbytes + w.shells.l.nbytes + w.shells.prim_offset.nbytes + w.shells.exponents.nbytes +
                     w.shells.coefficients.nbytes + w.bra_ij.nbytes + w.ket_ij.nbytes + 3 * b[0].nbytes for w, b in zip(wls, dg_bufs)))
    dg_d2h = int(sum(2 * b[0].nbytes for b in dg_bufs))

    def digest_step():
        for wl, (D, J, K) in zip(wls, dg_bufs):
            upload(wl)
            bra = eng.build_pairs(wl.bra_ij)
            ket = eng.build_pairs(wl.ket_ij)
            eng.compute_jk_host(bra, ket, D, J, K, stream=stream.cuda_stream)
            bra.free(); ket.free()

    digest_step()
    barrier()
    w0 = time.perf_counter()
    for _ in range(args.steps):
        digest_step()
    barrier()
    dg_s = reduce_max(time.perf_counter() - w0, world, f"cuda:{local}")
    dg_value = whole_job_rate(world, nq, 1e3 * dg_s / args.steps)

    if rank == 0:
        peak, peak_how = fp64_peak_tflops()
        traffic, traffic_src = ncu_traffic(args.workload)
        k_ms = sum(kern_ms)
        achieved = flops_step / (k_ms * 1e-3) / 1e12
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": config_dict(wls, world),
            "tflops": value * flops_step / nq / 1e12, "fp64_peak_frac": value * flops_step / nq / 1e12 / (peak * world),
            "flops_per_quartet": flops_step / nq,
            "roofline": {"bound": "tensor", "kernel": "md4::eri_kernel (FP64 DMMA.8x8x4)", "achieved": achieved,
                         "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic,
                         "traffic_unit": "bytes per launch (dram read+write)", "traffic_source": traffic_src,
                         "algorithmic_bytes": int(sum(out_doubles) * 8),
                         "peak_source": peak_how, "kernel_ms": k_ms},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
            "e2e_digest": {"value": dg_value, "unit": UNIT, "h2d_bytes_per_step": dg_h2d, "d2h_bytes_per_step": dg_d2h,
                           "what": "md4_set_shells + md4_build_pairs x2 + md4_compute_jk_host: (ab|cd) contracted with an AO density "
                                   "in the kernel epilogue (J and K to the host) instead of 8 Nab Ncd bytes per quartet"},
            "gpu_launches": int(n_launch), "clocks": clocks,
        }
        if multi:
            # BASELINE.json config 5: per-class quartets/s and % of FP64 peak (fused kernel alone, CUDA events)
            line["classes"] = [
                {"name": w.name, "lclass": list(w.lclass), "kclass": list(w.kclass), "quartets": w.nquartets,
                 "kernel_ms": ms, "quartets_per_s": w.nquartets / (ms * 1e-3),
                 "tflops": w.nquartets * inputs.class_flops(w.lclass, w.kclass) / (ms * 1e-3) / 1e12,
                 "frac": w.nquartets * inputs.class_flops(w.lclass, w.kclass) / (ms * 1e-3) / 1e12 / peak}
                for w, ms in zip(wls, kern_ms)]
        if world == 1 and not args.no_cpu_baseline:
            r, cores, n, dt = oracle_step(wls, 15.0)
            line["cpu_baseline"] = {"value": r, "unit": UNIT, "cores": cores,
                                    "kind": "oracle (long-double build, as it stands: not a tuned CPU code)",
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
    ap.add_argument("--workload", default="cfg3", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        print("bench.py: note: fewer than 3 warm-up steps", file=sys.stderr)
    return run_reference(args) if args.impl == "reference" else run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
