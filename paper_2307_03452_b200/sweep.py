"""Per-class throughput report over the BASELINE.json configs (config 5's "per-class quartets/s and % of FP64 peak").

    python -m paper_2307_03452_b200.sweep [--configs cfg1,cfg2,cfg3,cfg4,cfg5,low] [--reps 5] [--out report.md]

For every workload: pair lists are built once (timed separately, the paper excludes H from the quartet loop,
PAPER.md:146, :158), then md4_compute is timed alone with CUDA events on its stream (3 warm-ups, `reps` repetitions,
median and best).  FLOPs are the paper's matrix-only count, bra transformed first.  Prints a
markdown table; needs a CUDA device (no CPU fallback).
"""
from __future__ import annotations

import argparse
import statistics
import sys

from . import inputs


def fp64_peak_tflops(sm_mhz: float = 1965.0) -> float:
    return 148 * 64 * 2 * sm_mhz * 1e6 / 1e12


def workloads(names):
    for n in names:
        if n == "cfg1":
            yield inputs.config1()
        elif n == "cfg2":
            yield inputs.config2()
        elif n == "cfg3":
            yield inputs.config3()
        elif n == "cfg4":
            yield inputs.config4()
        elif n == "low":
            # the remaining classes of the paper's Table 1, same recipe as cfg2
            yield inputs._perm_config("low (dd|dd) K=1", 11, 64, 2, 10.0, 0.05, 50.0, 64)
            yield inputs._perm_config("low (ff|ff) K=1", 12, 64, 3, 10.0, 0.05, 50.0, 64)
        elif n == "cfg5":
            for K in (1, 3):
                for ci in range(len(inputs.sweep_classes())):
                    yield inputs.config5(ci, K=K)
        else:
            raise SystemExit(f"unknown config {n}")


def time_workload(eng, wl, reps: int):
    import torch

    s = wl.shells
    eng.set_shells(s.centers, s.l, s.prim_offset, s.exponents, s.coefficients)
    stream = torch.cuda.current_stream()
    ev = lambda: torch.cuda.Event(enable_timing=True)  # noqa: E731
    # pair build, timed on the second build of the same lists: the first one of a size allocates device memory
    # (cudaMalloc), later ones take their block from the engine's pool (md4_free_pairs) -- the steady state of a batch loop
    bra = eng.build_pairs(wl.bra_ij)
    ket = eng.build_pairs(wl.ket_ij)
    torch.cuda.synchronize()
    bra.free(); ket.free()
    p0, p1 = ev(), ev()
    p0.record(stream)
    bra = eng.build_pairs(wl.bra_ij)
    ket = eng.build_pairs(wl.ket_ij)
    eng.stream_wait_pairs(bra, stream.cuda_stream)   # the pair kernels run on the engine's own stream
    eng.stream_wait_pairs(ket, stream.cuda_stream)
    p1.record(stream)
    torch.cuda.synchronize()
    pair_ms = p0.elapsed_time(p1)
    out = torch.empty(wl.nquartets * inputs.class_out_doubles(wl.lclass), dtype=torch.float64, device="cuda")
    for _ in range(3):
        eng.compute(bra, ket, out=out, stream=stream.cuda_stream)
    torch.cuda.synchronize()
    ms = []
    for _ in range(reps):
        e0, e1 = ev(), ev()
        e0.record(stream)
        eng.compute(bra, ket, out=out, stream=stream.cuda_stream)
        e1.record(stream)
        torch.cuda.synchronize()
        ms.append(e0.elapsed_time(e1))
    bra.free()
    ket.free()
    del out
    return pair_ms, statistics.median(ms), min(ms)


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="cfg1,cfg2,cfg3,cfg4,cfg5")
    ap.add_argument("--reps", type=int, default=5)
    ap.add_argument("--out", default=None)
    args = ap.parse_args(argv)
    import torch

    from . import md4

    if not torch.cuda.is_available():
        raise SystemExit("sweep: no CUDA device -- the MD4 path has no CPU fallback")
    peak = fp64_peak_tflops()
    lines = [f"| workload | quartets | FLOP/quartet | pair build ms | compute ms (median / best) | quartets/s | TFLOP/s | % of {peak:.2f} |",
             "|---|---|---|---|---|---|---|---|"]
    with md4.Engine(0) as eng:
        for wl in workloads(args.configs.split(",")):
            flops = inputs.class_flops(wl.lclass, wl.kclass)
            pair_ms, med, best = time_workload(eng, wl, args.reps)
            qps = wl.nquartets / (med * 1e-3)
            tf = qps * flops / 1e12
            lines.append(f"| {wl.name} | {wl.nquartets} | {flops} | {pair_ms:.2f} | {med:.3f} / {best:.3f} | {qps:.4g} | {tf:.2f} | {100 * tf / peak:.1f} |")
            print(lines[-1], flush=True)
    text = "\n".join(lines) + "\n"
    if args.out:
        with open(args.out, "w") as f:
            f.write(text)
    return 0


if __name__ == "__main__":
    sys.exit(main())
