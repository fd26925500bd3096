#!/usr/bin/env python
"""bench.py - the NLL + gradient + HVP sweep of BASELINE.json's target configuration on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

One "step" = one pwa_nll_grad_hvp call = one streaming pass of the whole hot path (propagators, coherent
and incoherent sums, ln I, NLL, gradient, HVP, reduction, Eqs. 4/6/7) over all MC and data events of the
workload.  Prints ONE JSON line (rank 0).  See DESIGN.md §Measurement for every field.

N > 1 (launched with torch.distributed.run): weak scaling over event shards as in PAPER.md:78-98 - every
rank holds its own config-sized shard, runs pwa_raw_sums on it, the raw vectors (4 + 4P doubles) are
all-reduced with NCCL and every rank applies pwa_combine (Eqs. 4, 6, 7).

--impl reference times the CPU oracle (oracle/, test infrastructure) on a bounded sample of the same
workload on this box's host cores; it is a deliberately plain program, not a target.
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

METRIC = "nll_grad_hvp_events_per_s"
UNIT = "events/s"
# entry points a step can call (--mode); the metric's step is the fused sweep
MODES = {"nll_grad_hvp": "pwa_nll_grad_hvp", "nll": "pwa_nll", "nll_grad": "pwa_nll_grad",
         "nll_grad_for_hvp": "pwa_nll_grad_for_hvp", "hvp_cached": "pwa_hvp_cached", "hvp": "pwa_hvp",
         "nll_batch": "pwa_nll_batch", "hvp_cached_batch": "pwa_hvp_cached_batch"}


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """Samples SM clock, power and throttle reasons while a timed region runs: NVML from a thread every ~2 ms
    (so that samples fall inside regions of a few tens of milliseconds), nvidia-smi -lms 20 if NVML is unavailable."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index: int, period_s: float = 0.002):
        self.index, self.period, self.rows, self.proc, self.thread = index, period_s, [], None, None
        self.stop_flag = threading.Event()
        self.source = None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.dev = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_sm = float(pynvml.nvmlDeviceGetMaxClockInfo(self.dev, pynvml.NVML_CLOCK_SM))
            self.source = "nvml"
            self.thread = threading.Thread(target=self._poll_nvml, daemon=True)
            self.thread.start()
            self._wait_first_sample()
            return
        except Exception:
            self.source = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.source = "nvidia-smi -lms 20"
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read_smi, daemon=True)
        self.thread.start()
        self._wait_first_sample()

    def _wait_first_sample(self, timeout_s: float = 3.0):
        """The first NVML query of a process can take tens of milliseconds: a timed region must not start (and end)
        before the sampler has delivered anything."""
        t_end = time.time() + timeout_s
        while not self.rows and time.time() < t_end:
            time.sleep(0.001)

    def _poll_nvml(self):
        nv = self.nv
        bits = [(getattr(nv, "nvmlClocksEventReasonHwSlowdown", getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8)), "hw_slowdown"),
                (getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40)), "hw_thermal_slowdown"),
                (getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20)), "sw_thermal_slowdown"),
                (getattr(nv, "nvmlClocksEventReasonSwPowerCap", getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4)), "sw_power_cap")]
        get_reasons = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or nv.nvmlDeviceGetCurrentClocksThrottleReasons
        while not self.stop_flag.is_set():
            try:
                sm = float(nv.nvmlDeviceGetClockInfo(self.dev, nv.NVML_CLOCK_SM))
                pw = nv.nvmlDeviceGetPowerUsage(self.dev) / 1000.0
                mask = int(get_reasons(self.dev))
                self.rows.append((time.time(), sm, self.max_sm, pw, [n for b, n in bits if mask & b]))
            except Exception:
                pass
            time.sleep(self.period)

    def _read_smi(self):
        for line in self.proc.stdout:
            f = [x.strip() for x in line.strip().split(",")]
            try:
                self.rows.append((time.time(), float(f[0]), float(f[1]), float(f[2]),
                                  [n for n, val in zip(self.NAMES, f[3:7]) if val.lower().startswith("active")]))
            except (ValueError, IndexError):
                continue

    def window(self, t0: float, t1: float):
        """Summary of the samples taken in [t0, t1] (host clock); the sampler keeps running."""
        if self.source is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no clock source (NVML and nvidia-smi unavailable)"]}
        rows = list(self.rows)
        inside = [r for r in rows if t0 <= r[0] <= t1]
        note = None
        if not inside:  # region shorter than the sampling period: the nearest samples on either side
            inside = sorted(rows, key=lambda r: min(abs(r[0] - t0), abs(r[0] - t1)))[:2]
            note = "no sample inside the region; nearest samples reported"
        sm = sorted(r[1] for r in inside)
        reasons = sorted({n for r in inside for n in r[4]})
        out = {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_min_mhz": sm[0] if sm else None,
               "sm_max_mhz": max((r[2] for r in inside), default=None),
               "power_w_max": max((r[3] for r in inside), default=None), "samples": len(sm), "reasons": reasons,
               "source": self.source}
        if note:
            out["note"] = note
        return out

    def stop(self):
        self.stop_flag.set()
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()


def _strip_comments(src: str) -> str:
    """C / C++ source without its comments and with runs of white space collapsed (string and character literals are
    kept as they are): what the compiler sees, so that a comment-only edit does not invalidate a stored capture."""
    out, i, n = [], 0, len(src)
    while i < n:
        c = src[i]
        if c in "\"'":  # literal: copy up to the closing quote
            j = i + 1
            while j < n and src[j] != c:
                j += 2 if src[j] == "\\" else 1
            out.append(src[i:j + 1])
            i = j + 1
        elif src.startswith("//", i):
            j = src.find("\n", i)
            i = n if j < 0 else j
        elif src.startswith("/*", i):
            j = src.find("*/", i + 2)
            i = n if j < 0 else j + 2
            out.append(" ")
        else:
            out.append(c)
            i += 1
    return " ".join("".join(out).split())


def _csrc_digest() -> str:
    """sha256 over the sources (comments and white space aside) of the sweep kernel and its launch configuration: ties a
    stored ncu traffic figure to the code it was captured on."""
    import hashlib
    d = os.path.join(ROOT, "paper_2403_09225_b200", "csrc")
    hsh = hashlib.sha256()
    for name in ("pwa_common.cuh", "pwa_kernels.cuh", "pwa_sweep_lanes.cuh", "pwa_sweep_lanes.cu", "pwa_sweep_pair.cuh"):
        with open(os.path.join(d, name), "r", encoding="utf-8") as f:
            hsh.update(name.encode() + b"\0" + _strip_comments(f.read()).encode())
    return hsh.hexdigest()[:16]


def _stored_traffic(config: int, variant: str):
    """ncu dram__bytes_read.sum + dram__bytes_write.sum per sweep launch from the newest committed --set full capture
    (profiles/r*_traffic.csv: config;kernel_variant;dram_bytes_per_launch;csrc_digest).  Returns (bytes, source) - or
    (None, why) when no row was captured on the kernel sources of this tree, so that a stale figure is never printed."""
    pdir = os.path.join(ROOT, "profiles")
    digest = _csrc_digest()
    stale = None
    for name in sorted((n for n in os.listdir(pdir) if n.endswith("_traffic.csv")), reverse=True):
        try:
            with open(os.path.join(pdir, name)) as f:
                for row in f:
                    parts = [x.strip() for x in row.strip().split(";")]
                    if len(parts) >= 3 and parts[0] == f"config{config}" and parts[1] == variant:
                        if len(parts) >= 4 and parts[3] == digest:
                            return float(parts[2]), f"profiles/{name} (ncu --set full, csrc digest {digest})"
                        stale = stale or f"profiles/{name} was captured on other kernel sources (csrc digest now {digest})"
        except (OSError, ValueError):
            continue
    return None, stale or f"no ncu capture for config{config};{variant};{digest} under profiles/"


_ORACLE_MODELS = {}


def _oracle_sample_time(w, n_mc_s, n_data_s, th, v, threads):
    """Times the CPU oracle (double build, OpenMP) on the first n_mc_s / n_data_s events of the workload
    (the host copy of the sample is made once and is not part of the timed region)."""
    import oracle
    import numpy as np
    key = (id(w), n_mc_s, n_data_s)
    if key in _ORACLE_MODELS:
        m = _ORACLE_MODELS[key]
        t0 = time.perf_counter()
        out = oracle.nll_grad_hvp(m, np.asarray(th), np.asarray(v), "d", threads=threads)
        return time.perf_counter() - t0, out
    to_np = lambda t: None if t is None else t.detach().cpu().numpy()
    data = oracle.Sample(to_np(w.data_mass[:, :n_data_s]), to_np(w.data_amp[:, :, :n_data_s]),
                         to_np(None if w.data_weight is None else w.data_weight[:n_data_s]))
    mc = oracle.Sample(to_np(w.mc_mass[:, :n_mc_s]), to_np(w.mc_amp[:, :, :n_mc_s]), None)
    m = oracle.Model(to_np(w.res_chan), data, mc)
    _ORACLE_MODELS[key] = m
    t0 = time.perf_counter()
    out = oracle.nll_grad_hvp(m, np.asarray(th), np.asarray(v), "d", threads=threads)
    return time.perf_counter() - t0, out


def run_reference(args):
    """--impl reference: the oracle as it stands, on host cores, on a bounded sample of the workload per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import torch
    import oracle
    import workloads
    oracle.build()
    cfg = workloads.CONFIGS[args.config]
    # bounded sample: same model (R, H, C, weights), fewer events, same MC:data ratio
    n_mc_s = min(cfg.n_mc, args.ref_events)
    n_data_s = max(1, n_mc_s * cfg.n_data // cfg.n_mc)
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    w = workloads.make_workload(cfg.scaled(n_mc_s, n_data_s), dev, chunk=1 << 16)
    th = workloads.random_start(cfg, 0).numpy()
    v = workloads.direction(cfg, 0).numpy()
    threads = oracle.max_threads()
    for _ in range(args.warmup):
        _oracle_sample_time(w, n_mc_s, n_data_s, th, v, threads)
    times = [_oracle_sample_time(w, n_mc_s, n_data_s, th, v, threads)[0] for _ in range(args.steps)]
    total = sum(times)
    ev = (n_mc_s + n_data_s) * args.steps / total
    sample = f"first {n_mc_s} MC + {n_data_s} data events of the config-{args.config} recipe per step"
    line = {"impl": "reference", "metric": METRIC, "value": ev, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config {args.config} ({cfg.name}): R={cfg.n_res} H={cfg.n_hel} C={cfg.n_chan}, "
                                   f"bounded sample of {n_mc_s}+{n_data_s} events"},
            "cpu_baseline": {"value": ev, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": ev, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def run_fits(args):
    """--config 5 (BASELINE.json configs[4]): config 2's workload, full truncated Newton-CG fits (<= 50 CG iterations per
    outer step, Armijo line search) from --fits seeded random starts (S16); wall time per fit and the best NLL reached
    against the oracle.  The oracle's side: its reference fit (oracle/fit.py) from theta_true on a bounded sample is far
    too slow at 1.1 M events for 20 random starts, so the comparison is (a) the oracle's NLL and gradient at the point
    the best CUDA fit returned and (b) the oracle's NLL at theta_true, the value every successful fit must beat."""
    import numpy as np
    import torch
    import paper_2403_09225_b200 as pwa
    import workloads
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU path)")
    pwa.load()
    dev = torch.device("cuda", 0)
    base = workloads.CONFIGS[2]
    cfg = base.scaled(args.mc or base.n_mc, args.data or base.n_data)
    w = workloads.make_workload(cfg, dev)
    m = pwa.Model(w, device=0, borrow=True)
    opts = pwa.pwa_fit_opts_default()
    if args.max_seconds > 0:
        opts.max_seconds = args.max_seconds
    th_true = workloads.theta_true(cfg).numpy()
    _, r_true = m.fit(th_true, opts)  # warm-up, and the fit from the generating parameters
    # --concurrent K: K independent fits in flight, each on its own handle and stream over the SAME borrowed event store
    # (one host thread per fit; the kernels of one fit fill the host round trips of the others)
    K = max(1, args.concurrent)
    workers = [m]
    streams = []
    for _ in range(1, K):
        st = torch.cuda.Stream(device=dev)
        streams.append(st)
        workers.append(pwa.Model(w, device=0, borrow=True, stream=st.cuda_stream))
    rows, best = [None] * args.fits, None
    l0 = sum(pwa.pwa_kernel_launches(x.h) for x in workers)

    def one(k):
        mm = workers[k % K]
        th, r = mm.fit(workloads.random_start(cfg, k).numpy(), opts)
        return k, th, r

    torch.cuda.synchronize()
    t_all = time.perf_counter()
    if K == 1:
        results = [one(k) for k in range(args.fits)]
    else:
        import concurrent.futures as cf
        results = []
        with cf.ThreadPoolExecutor(max_workers=K) as ex:
            # start k runs on worker k % K: keep at most one fit per handle in flight
            for base in range(0, args.fits, K):
                results += list(ex.map(one, range(base, min(base + K, args.fits))))
    torch.cuda.synchronize()
    t_all = time.perf_counter() - t_all
    for k, th, r in results:
        rows[k] = {"start": k, "nll": r.nll, "grad_inf": r.grad_inf_norm, "outer": r.outer_iters, "hvp": r.n_hvp,
                   "sweeps": r.n_nll + r.n_grad + r.n_hvp, "stop": r.stop_reason, "status": r.status,
                   "active_bounds": r.n_active, "seconds": r.seconds}
        if r.status == 0 and (best is None or r.nll < best[1].nll):
            best = (th, r)
    m_launches = sum(pwa.pwa_kernel_launches(x.h) for x in workers) - l0
    launches = m_launches
    line = {"metric": "fit_seconds", "value": t_all / max(args.fits, 1), "unit": "s/fit", "n_gpus": 1, "steps": args.fits,
            "warmup": 1, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": f"config 5: Newton-CG fits on config 2's arrays (R={cfg.n_res} H={cfg.n_hel} C={cfg.n_chan}, "
                                   f"N_mc={cfg.n_mc} N_data={cfg.n_data}) from {args.fits} seeded random starts, "
                                   f"{K} fit(s) in flight",
                       "kernel_variant": pwa.pwa_kernel_variant(m.h)},
            "fits_converged": sum(1 for r in rows if r["status"] == 0),
            # roofline-style account of a fit: every sweep (value, gradient or HVP) reads the event store once
            "roofline_fit": (lambda nb, pk: {"bound": "hbm", "unit": "GB/s", "peak": pk[0], "peak_source": pk[1],
                                             "bytes_per_sweep": nb,
                                             "achieved": sum(r["sweeps"] for r in rows) * nb / t_all / 1e9,
                                             "frac": sum(r["sweeps"] for r in rows) * nb / t_all / 1e9 / pk[0],
                                             "us_per_sweep": 1e6 * t_all / max(1, sum(r["sweeps"] for r in rows)),
                                             "what": "algorithmic bytes of all sweeps of all fits / wall time of the fits "
                                                     "(host loop, reductions and CG updates included)"})(
                pwa.pwa_bytes_per_eval(m.h), _peaks()),
            "sweeps_total": sum(r["sweeps"] for r in rows), "gpu_launches": int(launches),
            "fit_from_theta_true": {"nll": r_true.nll, "outer": r_true.outer_iters, "hvp": r_true.n_hvp,
                                    "seconds": r_true.seconds, "status": r_true.status},
            "fits": rows}
    if best is not None and not args.no_cpu_baseline:
        import oracle
        oracle.build()
        om = oracle.model_from_workload(w)
        nt = oracle.max_threads()
        f0, g0, _ = oracle.nll_grad_hvp(om, best[0], None, "d", threads=nt)
        line["best"] = {"nll": best[1].nll, "oracle_nll_at_best_theta": float(f0),
                        "oracle_grad_inf_at_best_theta": float(np.max(np.abs(g0))),
                        "oracle_nll_at_theta_true": float(oracle.nll(om, th_true, "d", threads=nt)),
                        "n_starts_within_1e-6_of_best": sum(1 for r in rows if r["status"] == 0 and
                                                            abs(r["nll"] - best[1].nll) <= 1e-6 * abs(best[1].nll))}
    print(json.dumps(line), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config (1-4, 6: one sweep per step; 5: fits); 3 is the target")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-events", type=int, default=5_000_000, help="MC events in the oracle's bounded sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--mc", type=int, default=0, help="override N_mc (experiments only)")
    ap.add_argument("--data", type=int, default=0, help="override N_data (experiments only)")
    ap.add_argument("--fits", type=int, default=20, help="--config 5: number of seeded random starts")
    ap.add_argument("--max-seconds", type=float, default=0.0, help="--config 5: wall-time cap per fit (0 = off)")
    ap.add_argument("--concurrent", type=int, default=1, help="--config 5: independent fits in flight (handles + streams)")
    ap.add_argument("--mode", default="nll_grad_hvp", choices=list(MODES),
                    help="entry point one step calls (default: the fused sweep, the metric's step)")
    ap.add_argument("--batch", type=int, default=4, help="--mode nll_batch / hvp_cached_batch: evaluations per call (K)")
    ap.add_argument("--sustained-seconds", type=float, default=1.2,
                    help="length of the back-to-back run behind roofline_sustained (0 = skip)")
    ap.add_argument("--shape", default="", help="R,H,C: another model shape on --config's recipe (kernel-shape measurements, "
                    "profiles/r02_shapes.md; with --mc / --data); not a BASELINE.json configuration")
    ap.add_argument("--store", default="auto", choices=["auto", "borrow", "copy"],
                    help="event store of the handle: borrow = the workload's planes in place (zero copy); copy = a library-owned "
                         "copy, which shapes that need 8-event tiles keep TILED (one bulk copy per stage); auto = copy for config 4")
    ap.add_argument("--csrc-digest", action="store_true", help="print the digest a profiles/*_traffic.csv row must carry, and exit")
    args = ap.parse_args()
    if args.csrc_digest:
        print(_csrc_digest())
        return 0
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else max(args.warmup, 1)
    if args.impl == "reference":
        if args.config == 5:
            args.config = 2
        return run_reference(args)
    if args.config == 5:
        return run_fits(args)

    import numpy as np
    import torch
    import paper_2403_09225_b200 as pwa
    import workloads

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU path)")
    pwa.load()  # raises if libpwa_b200.so is missing
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    base = workloads.CONFIGS[args.config]
    if args.shape:
        from dataclasses import replace
        R_, H_, C_ = (int(x) for x in args.shape.split(","))
        base = replace(base, name=f"{base.name}, shape {args.shape}", n_res=R_, n_hel=H_, n_chan=C_, table1=False)
    cfg = base.scaled(args.mc or base.n_mc, args.data or base.n_data)
    if world > 1:  # every rank holds its own shard: same recipe, rank-specific seed
        from dataclasses import replace
        cfg = replace(cfg, index=cfg.index + 1000 * rank)
    t_gen = time.time()
    w = workloads.make_workload(cfg, dev)
    torch.cuda.synchronize()
    t_gen = time.time() - t_gen
    store = args.store if args.store != "auto" else ("copy" if args.config == 4 else "borrow")
    if store == "copy":
        torch.cuda.empty_cache()  # the library's copy is allocated beside the workload (config 4: 2 x 70.7 GB of 180 GB)
    try:
        m = pwa.Model(w, device=local, borrow=store == "borrow")
    except pwa.PwaError as e:  # no room for a second copy beside the workload: time the borrowed planes instead
        if store != "copy" or e.status != pwa.PWA_ERR_OOM:
            raise
        store = "borrow"
        m = pwa.Model(w, device=local, borrow=True)
    P = m.P
    th_np = workloads.random_start(base, 0).numpy()
    v_np = workloads.direction(base, 0).numpy()
    theta = torch.tensor(th_np, device=dev)
    v = torch.tensor(v_np, device=dev)
    raw = torch.zeros(4 + 4 * P, dtype=torch.float64, device=dev)
    events_per_step = cfg.n_mc + cfg.n_data
    bytes_per_step = pwa.pwa_bytes_per_eval(m.h)

    single = {"nll_grad_hvp": lambda: pwa.pwa_nll_grad_hvp(m.h, theta, v, m.nll_t, m.grad_t, m.hv_t),
              "nll": lambda: pwa.pwa_nll(m.h, theta, m.nll_t),
              "nll_grad": lambda: pwa.pwa_nll_grad(m.h, theta, m.nll_t, m.grad_t),
              "nll_grad_for_hvp": lambda: pwa.pwa_nll_grad_for_hvp(m.h, theta, m.nll_t, m.grad_t),
              "hvp_cached": lambda: pwa.pwa_hvp_cached(m.h, v, m.hv_t),
              "hvp": lambda: pwa.pwa_hvp(m.h, theta, v, m.hv_t),
              "nll_batch": lambda: pwa.pwa_nll_batch(m.h, args.batch, theta_k, nll_k),
              "hvp_cached_batch": lambda: pwa.pwa_hvp_cached_batch(m.h, args.batch, v_k, hv_k)}[args.mode]
    evals_per_step = args.batch if args.mode.endswith("_batch") else 1
    if args.mode.endswith("_batch"):  # K parameter sets (seeded random starts) / K directions
        theta_k = torch.tensor(np.stack([workloads.random_start(base, k).numpy() for k in range(args.batch)]), device=dev)
        v_k = torch.tensor(np.stack([workloads.direction(base, k).numpy() for k in range(args.batch)]), device=dev)
        nll_k = torch.zeros(args.batch, dtype=torch.float64, device=dev)
        hv_k = torch.zeros(args.batch, P, dtype=torch.float64, device=dev)
    if args.mode in ("hvp_cached", "hvp_cached_batch"):
        pwa.pwa_nll_grad_for_hvp(m.h, theta, m.nll_t, m.grad_t)
    if world > 1 and args.mode != "nll_grad_hvp":
        raise SystemExit("--mode is a one-GPU measurement")

    def step():
        if world == 1:
            single()
        else:
            pwa.pwa_raw_sums(m.h, theta, v, raw)
            dist.all_reduce(raw)
            pwa.pwa_combine(m.h, raw, v, m.nll_t, m.grad_t, m.hv_t)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.05)
    pwa.pwa_profile_enable(m.h, True)
    pwa.pwa_profile_read(m.h)
    l0 = pwa.pwa_kernel_launches(m.h)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    tw0 = time.time()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    tw1 = time.time()
    ms = e0.elapsed_time(e1)
    sweep_ms, sweep_n = pwa.pwa_profile_read(m.h)
    pwa.pwa_profile_enable(m.h, False)
    launches = pwa.pwa_kernel_launches(m.h) - l0
    clocks = sampler.window(tw0, tw1) if rank == 0 else None
    if world > 1:
        t = torch.tensor([ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    nll_dev = m.nll_t.item()
    ranks_agree = None
    if world > 1:
        # correctness anchor of the sharded path: after the all-reduce of the RAW sums every rank combines the same
        # numbers, so the NLL (and with it theta along a fit) must be the same bits on every rank
        allv = [torch.zeros(1, dtype=torch.float64, device=dev) for _ in range(world)]
        dist.all_gather(allv, m.nll_t)
        ranks_agree = all(x.item() == nll_dev for x in allv)
        assert ranks_agree, "ranks disagree on the NLL after the all-reduce of the raw sums"

    # ---- end to end: H2D of theta, v (pinned) and D2H of nll, grad, hv every step, synchronised ----
    # one GPU: the library's host-buffer entry point; several: the same copies around raw sums -> all-reduce -> combine
    th_h, v_h = np.ascontiguousarray(th_np), np.ascontiguousarray(v_np)
    o_nll, o_g, o_h = np.zeros(1), np.zeros(P), np.zeros(P)
    sharded_e2e = world > 1 or os.environ.get("PWA_BENCH_FORCE_SHARDED_E2E") == "1"
    if sharded_e2e:
        pin_in = torch.empty(2 * P, dtype=torch.float64).pin_memory()
        pin_in[:P] = torch.from_numpy(th_h)
        pin_in[P:] = torch.from_numpy(v_h)
        pin_out = torch.empty(1 + 2 * P, dtype=torch.float64).pin_memory()
        d_in = torch.empty(2 * P, dtype=torch.float64, device=dev)
        d_out = torch.empty(1 + 2 * P, dtype=torch.float64, device=dev)

    def e2e_step():
        if not sharded_e2e:
            pwa.pwa_nll_grad_hvp_host(m.h, th_h, v_h, o_nll, o_g, o_h)
            return
        d_in.copy_(pin_in, non_blocking=True)
        pwa.pwa_raw_sums(m.h, d_in[:P], d_in[P:], raw)
        if world > 1:
            dist.all_reduce(raw)
        pwa.pwa_combine(m.h, raw, d_in[P:], d_out[0:1], d_out[1:1 + P], d_out[1 + P:])
        pin_out.copy_(d_out, non_blocking=True)
        torch.cuda.synchronize()

    for _ in range(2):
        e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        e2e_step()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    if sharded_e2e and world == 1:
        assert abs(float(pin_out[0]) - nll_dev) <= 1e-12 * abs(nll_dev), "sharded e2e path disagrees with the fused call"
    if world > 1:
        t = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())

    # ---- sustained: >= --sustained-seconds of back-to-back steps AFTER the timed region (fits are seconds of
    # back-to-back sweeps; the SM clock sags under the FP64 load after some tens of milliseconds).
    # Per-launch sweep times from the library's CUDA events on the launching stream; the mean of the last half counts.
    sustained = None
    if args.sustained_seconds > 0 and world == 1:
        n_long = int(min(4000, max(50, args.sustained_seconds / (ms / args.steps * 1e-3))))
        pwa.pwa_profile_enable(m.h, True)
        pwa.pwa_profile_read(m.h)
        torch.cuda.synchronize()
        half = n_long // 2
        ts0 = time.time()
        e_a, e_b, e_c = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        e_a.record()
        for _ in range(half):
            step()
        e_b.record()
        torch.cuda.synchronize()
        first_ms, first_n = pwa.pwa_profile_read(m.h)
        ts1 = time.time()
        for _ in range(n_long - half):
            step()
        e_c.record()
        torch.cuda.synchronize()
        ts2 = time.time()
        last_ms, last_n = pwa.pwa_profile_read(m.h)
        pwa.pwa_profile_enable(m.h, False)
        sustained = {"first": (first_ms / max(first_n, 1), e_a.elapsed_time(e_b) / half),
                     "last": (last_ms / max(last_n, 1), e_b.elapsed_time(e_c) / (n_long - half)),
                     "n": n_long, "seconds": ts2 - ts0, "clocks": sampler.window(ts1, ts2)}
    if rank == 0:
        sampler.stop()

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    peak, peak_src = _peaks()
    sweep_avg_s = (sweep_ms / max(sweep_n, 1)) * 1e-3
    achieved = bytes_per_step / sweep_avg_s / 1e9 if sweep_n else None
    traffic, traffic_src = (None, "stored figures are for the fused sweep of the BASELINE.json configurations") \
        if (args.mode != "nll_grad_hvp" or args.shape or args.mc or args.data) else \
        _stored_traffic(args.config, pwa.pwa_kernel_variant(m.h))
    line = {
        "metric": METRIC, "value": world * events_per_step * args.steps / (ms * 1e-3), "unit": UNIT,
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config {args.config} ({cfg.name}): R={cfg.n_res} H={cfg.n_hel} C={cfg.n_chan} "
                               f"P={cfg.n_par}, N_mc={cfg.n_mc} N_data={cfg.n_data} per GPU"
                               f"{', weighted data' if cfg.weighted else ''}",
                   "store": "borrowed planes (zero copy)" if store == "borrow" else "library-owned copy",
                   "l2": f"inputs ({bytes_per_step / 1e6:.0f} MB per step) exceed the 126 MB L2; no flush needed"
                         if bytes_per_step > 2 * 126e6 else "inputs fit in L2 (cache-resident case)",
                   "kernel_variant": pwa.pwa_kernel_variant(m.h), "parallelism": f"event shards x{world}",
                   "entry_point": MODES[args.mode],
                   "workload_gen_s": round(t_gen, 1)},
        "evals_per_s": evals_per_step * args.steps / (ms * 1e-3), "evals_per_step": evals_per_step,
        "nll": nll_dev, "nll_identical_across_ranks": ranks_agree,
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": (achieved / peak) if achieved else None, "traffic": traffic,
                     "traffic_source": traffic_src, "peak_source": peak_src, "kernel": "sweep", "bytes_per_launch": bytes_per_step,
                     "avg_launch_ms": sweep_avg_s * 1e3, "launches_timed": sweep_n},
        "e2e": {"value": world * events_per_step * args.steps / e2e_s, "unit": UNIT,
                "h2d_bytes_per_step": 2 * P * 8, "d2h_bytes_per_step": (1 + 2 * P) * 8,
                "ms_per_step": 1e3 * e2e_s / args.steps},
        "gpu_launches": int(launches),
        "clocks": clocks,
    }
    if sustained is not None:
        k_ms, step_ms = sustained["last"]
        ach = bytes_per_step / (k_ms * 1e-3) / 1e9
        line["roofline_sustained"] = {
            "bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
            "avg_launch_ms": k_ms, "ms_per_step": step_ms, "launches": sustained["n"],
            "seconds": round(sustained["seconds"], 3),
            "first_half": {"avg_launch_ms": sustained["first"][0], "frac": bytes_per_step / (sustained["first"][0] * 1e-3) / 1e9 / peak},
            "what": f"{sustained['n']} back-to-back steps right after the timed region; per-launch CUDA events of the sweep "
                    "kernel; achieved = algorithmic bytes / mean launch time of the LAST half",
            "peak_source": peak_src, "clocks": sustained["clocks"]}
    # the ALU co-limit beside the HBM roofline: FP64 instructions the method needs per event
    # (16 R H + 52 R + 80 DFMA-class) against the FP64 pipe rate measured on this pool
    # (profiles/r01_microbench.md: 17.05 T DFMA/s sustained)
    fp64_per_event = 16 * cfg.n_res * cfg.n_hel + 52 * cfg.n_res + 80
    if sweep_n:
        rate = fp64_per_event * events_per_step / sweep_avg_s / 1e12
        line["fp64_pipe"] = {"dfma_class_per_event_estimate": fp64_per_event, "achieved_estimate": rate, "peak": 17.05,
                             "unit": "T instr/s", "frac_estimate": rate / 17.05,
                             "note": "instruction count is SURVEY 8(d)'s formula 16RH + 52R + 80, not an executed count; "
                                     "the executed FP64-pipe activity is ncu's (profiles/, sweep_full)",
                             "peak_source": "measured (profiles/r01_microbench.md, fp64_peak)"}
    if not args.no_cpu_baseline:
        import oracle
        oracle.build()
        threads = oracle.max_threads()
        n_mc_s = min(cfg.n_mc, args.ref_events)
        n_data_s = max(1, n_mc_s * cfg.n_data // cfg.n_mc)
        # repeat the evaluation until about 10 s of CPU work have been timed (bounded: at most 40 evaluations)
        total, reps = 0.0, 0
        while reps < 40 and (total < 10.0 or reps < 2):
            dt, out = _oracle_sample_time(w, n_mc_s, n_data_s, th_np, v_np, threads)
            total += dt
            reps += 1
        line["cpu_baseline"] = {"value": reps * (n_mc_s + n_data_s) / total, "unit": UNIT, "cores": threads,
                                "kind": "oracle",
                                "note": "the definitional oracle as it stands (gcc -O2, per-parameter derivatives, compensated "
                                        "sums): a deliberately plain program, not a tuned CPU implementation",
                                "sample": f"first {n_mc_s} MC + {n_data_s} data events of the same arrays, {reps} "
                                          f"NLL+grad+HVP evaluations ({total:.1f} s)",
                                "nll_rel_diff_vs_gpu": abs(float(out[0]) - nll_dev) / max(abs(float(out[0])), 1.0)
                                if (n_mc_s == cfg.n_mc and world == 1) else None}
        # the same oracle on ONE thread, on a tenth of the sample ("plus a 1-thread figure")
        n1_mc, n1_d = max(1, n_mc_s // 10), max(1, n_data_s // 10)
        dt1, _ = _oracle_sample_time(w, n1_mc, n1_d, th_np, v_np, 1)
        line["cpu_baseline"]["one_thread"] = {"value": (n1_mc + n1_d) / dt1, "unit": UNIT,
                                              "sample": f"first {n1_mc} MC + {n1_d} data events, one evaluation ({dt1:.1f} s)"}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
