"""Per-mode timing of the sweep on one config (a measurement helper beside bench.py, which times the fused sweep only).

    python -m paper_2403_09225_b200.bench_modes [--config 3] [--bursts 6]

Each entry point is timed like bench.py times a step: bursts of 3 warm-ups + 20 calls between CUDA events, with a pause
between bursts; the minimum and the median burst are printed with the fraction of the measured HBM peak."""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--bursts", type=int, default=6)
    ap.add_argument("--long", type=int, default=0, help="instead: N fused sweeps back to back, mean time per block of 25")
    args = ap.parse_args()
    import torch
    import paper_2403_09225_b200 as pwa
    import workloads
    cfg = workloads.CONFIGS[args.config]
    dev = torch.device("cuda", 0)
    w = workloads.make_workload(cfg, dev)
    m = pwa.Model(w, device=0, borrow=True)
    th = torch.tensor(workloads.random_start(cfg, 0).numpy(), device=dev)
    v = torch.tensor(workloads.direction(cfg, 0).numpy(), device=dev)
    peak = 6650.0
    pk = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(pk):
        peak = float(json.load(open(pk))["hbm_gbs"])
    nbytes = pwa.pwa_bytes_per_eval(m.h)
    if args.long > 0:
        # the SM clock sags under this FP64 load after some tens of milliseconds: show the time per step along a long run
        torch.cuda.synchronize()
        time.sleep(2.0)
        n = args.long
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(n + 1)]
        ev[0].record()
        for i in range(n):
            pwa.pwa_nll_grad_hvp(m.h, th, v, m.nll_t, m.grad_t, m.hv_t)
            ev[i + 1].record()
        torch.cuda.synchronize()
        ts = [ev[i].elapsed_time(ev[i + 1]) for i in range(n)]
        print(f"config {args.config}: {pwa.pwa_kernel_variant(m.h)}; {n} fused sweeps back to back after a 2 s pause")
        print("| steps | mean ms per step | fraction of the HBM peak |\n|---|---|---|")
        for a in range(0, n, 25):
            blk = ts[a:a + 25]
            ms = sum(blk) / len(blk)
            print(f"| {a}-{a + len(blk) - 1} | {ms:.4f} | {nbytes / ms / 1e6 / peak:.3f} |")
        return
    calls = [("pwa_nll", lambda: pwa.pwa_nll(m.h, th, m.nll_t)),
             ("pwa_nll_grad", lambda: pwa.pwa_nll_grad(m.h, th, m.nll_t, m.grad_t)),
             ("pwa_nll_grad_for_hvp", lambda: pwa.pwa_nll_grad_for_hvp(m.h, th, m.nll_t, m.grad_t)),
             ("pwa_hvp_cached", lambda: pwa.pwa_hvp_cached(m.h, v, m.hv_t)),
             ("pwa_hvp", lambda: pwa.pwa_hvp(m.h, th, v, m.hv_t)),
             ("pwa_nll_grad_hvp", lambda: pwa.pwa_nll_grad_hvp(m.h, th, v, m.nll_t, m.grad_t, m.hv_t))]
    print(f"config {args.config}: {pwa.pwa_kernel_variant(m.h)}; {nbytes} algorithmic bytes per evaluation; peak {peak} GB/s")
    print("| entry point | min ms | median ms | GB/s (min) | fraction of the HBM peak |\n|---|---|---|---|---|")
    for name, fn in calls:
        ts = []
        for _ in range(args.bursts):
            time.sleep(0.5)
            for _ in range(3):
                fn()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(20):
                fn()
            e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1) / 20)
        ts.sort()
        gbs = nbytes / ts[0] / 1e6
        print(f"| `{name}` | {ts[0]:.4f} | {ts[len(ts) // 2]:.4f} | {gbs:.0f} | {gbs / peak:.3f} |")


if __name__ == "__main__":
    main()
