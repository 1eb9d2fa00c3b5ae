#!/usr/bin/env python
"""bench.py -- grid-point updates/s of the Fourier split-operator step on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 5] [--only] [--impl reference]

One bench "step" is one pass of the whole hot path over one batch: a single call of
sso_step(psi, SPLIT_STEPS) that advances the wavefunction by SPLIT_STEPS = 128 split-operator time steps
(the paper's protocol: 128 time steps, one upload before and one download after).

Headline workload at N=1: BASELINE.json's metric is not quoted on one config, so the line's top-level numbers are
for the LARGEST single-GPU configuration, config 5 (3D Dirac, 4 x 256^3 complex128, 1 GiB of psi); the other
workloads (1, 2a, 2b, 3, 4, and the paper's 1D Dirac and 4-component 2D Dirac shapes d1, d2x4, d2A) are timed in the same
run and reported under config.per_workload and, flat, as config.us_<name> / frac8_<name> / fracM_<name>.
  value  device-resident throughput: psi, the potential table and the field table are in HBM before the
         timed region; K calls timed with CUDA events on the launching stream.
  e2e    the same K calls through sso_step_host on a pinned HOST buffer: every call uploads psi, steps and
         downloads it inside the timed region.
  roofline  HBM: algorithmic bytes of one pass-kernel launch (one read + one write of psi, DESIGN.md
         "Rooflines") / average pass-kernel launch duration over the timed region, against MEASURED_PEAKS.json;
         `frac_dominant` = 2 S / mean launch time of the pass kind that takes most of a step / peak;
         `per_pass` = the same for each pass kind of one split step, timed with CUDA events by the library
         (sso_profile_step); `traffic` = ncu DRAM bytes of the dominant kernel from profiles/traffic.json, or
         null when csrc/ has changed since that capture.
  cpu_baseline  the oracle as it stands on the host cores (all cores, and one thread), bounded samples, rank 0
         at N=1 only.
N>1: replicas only: every rank runs the headline workload on its own GPU, no
data-path collective; value = all ranks' updates / max-over-ranks time.
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
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

import workloads as wl  # noqa: E402

METRIC = "grid-point updates/s per split-operator step"
UNIT = "grid-point updates/s"
SPLIT_STEPS = 128  # split-operator steps per sso_step call ("over 128 time steps")
HEADLINE = "5"

# name -> (config number, precision name, passes P per steady-state step)
WORKLOADS = {
    "1": (1, "c128", 1), "2a": (2, "c128", 2), "2b": (2, "c64", 2), "3": (3, "c128", 4), "4": (4, "c128", 2), "5": (5, "c128", 4),
    # the paper's own remaining shapes: 1D Dirac (eq. 35) and 2D Dirac with all four components
    "d1": ("dirac1d", "c128", 1), "d2x4": ("dirac2d4", "c128", 2),
    # the paper's position-space interaction factor (eq. 26): opening, kinetic, closing pass + one rotation kernel per step
    "d2A": ("dirac2dA", "c128", 4),
}
DESCR = {
    "1": "cfg1 1D Schroedinger 4096, harmonic well, complex128",
    "2a": "cfg2 2D Schroedinger 2048x2048, soft-core Coulomb + dipole field E(t), complex128",
    "2b": "cfg2 2D Schroedinger 2048x2048, soft-core Coulomb + dipole field E(t), complex64",
    "3": "cfg3 3D Schroedinger 256^3, 32 random Gaussians, complex128",
    "4": "cfg4 2D Dirac 2 components 1024x1024, soft-core Coulomb + A(t) in the kinetic unitary, complex128",
    "5": "cfg5 3D Dirac 4 components 256^3, soft-core Coulomb, complex128",
    "d1": "1D Dirac 2 components 4096 (PAPER.md:240 eq. 35), soft-core well zeta=1.4133, complex128",
    "d2x4": "2D Dirac 4 components 1024x1024 (the paper's 2D code, PAPER.md:115, 310), harmonic well, complex128",
    "d2A": "2D Dirac 2 components 1024x1024 with A(r) of a magnetic field applied in position space (PAPER.md:198 eq. 26), complex128",
}
# 60 % of the 8 TB/s roofline, us per split step; None where the bar does not apply
OPTIONS = []  # (SSO_OPT_*, value) pairs from --opt, applied to every plan (tuning sweeps)
BAR_US = {"1": None, "2a": 55.9, "2b": 28.0, "3": 447.4, "4": 28.0, "5": 1789.6, "d1": None, "d2x4": 55.9, "d2A": None}


def load_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, device copy)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def csrc_sha() -> str:
    """Hash of the kernel sources: an ncu number is only quoted while the code it was taken from is unchanged."""
    h = hashlib.sha256()
    for p in sorted((ROOT / "paper_1012_3911_b200" / "csrc").glob("*")):
        if p.suffix in (".cu", ".cuh", ".h"):
            h.update(p.name.encode())
            h.update(p.read_bytes())
    return h.hexdigest()[:16]


def ncu_traffic(name: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed capture
    listed in profiles/traffic.json -- or None when there is no capture for this workload or csrc/ has changed."""
    p = ROOT / "profiles" / "traffic.json"
    if not p.exists():
        return None, "no profiles/traffic.json"
    d = json.loads(p.read_text())
    if d.get("csrc_sha16") != csrc_sha():
        return None, f"stale: {d.get('capture')} was taken at csrc {d.get('csrc_sha16')}, csrc is now {csrc_sha()}"
    e = d.get("workloads", {}).get(name)
    if not e:
        return None, "no capture for this workload"
    return float(e["dram_bytes_per_launch"]), f"{d.get('capture')}: {e.get('kernel')}"


def make_workload(name: str, nrows: int):
    cfg, prec, P = WORKLOADS[name]
    if cfg == "dirac1d":
        w = wl.dirac1d(sizes=(4096,), nsteps=nrows, ncomp=2)
    elif cfg == "dirac2d4":
        w = wl.dirac2d4(nsteps=nrows)
    elif cfg == "dirac2dA":
        w = wl.dirac2d_magnetic(nsteps=nrows)
    else:
        w = wl.CONFIGS[cfg](nsteps=nrows)
    return w, prec, P


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled DURING the timed regions (B200_PROFILING.md)."""

    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
            time.sleep(0.15)
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def window(self, t0: float, t1: float):
        """Summary of the samples taken in [t0, t1] (plus one on each side for regions shorter than the period)."""
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        rows = list(self.rows)
        inside = [r for t, r in rows if t0 <= t <= t1] or [r for t, r in rows if t0 - 0.1 <= t <= t1 + 0.1] or [r for _, r in rows[-2:]]
        mhz, mx, reasons = [], None, set()
        for r in inside:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 6:
                continue
            try:
                mhz.append(float(f[0]))
                mx = float(f[1])
            except ValueError:
                continue
            for nm, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(mhz)) if mhz else None, "sm_max_mhz": mx, "reasons": sorted(reasons), "samples": len(mhz)}

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()


def oracle_rate(w, seconds_target: float, threads: int | None = None):
    """The oracle as it stands on a bounded sample of split steps of the same full-size workload."""
    import oracle

    allc = oracle.max_threads()
    if threads:
        oracle.set_threads(threads)
    try:
        o = oracle.Solver(w.sizes, w.dx, w.dt, w.ncomp, w.mass, w.c, w.charge)
        o.set_potential(w.V)
        if w.field_kind:
            o.set_field(w.field_kind, w.step_avg)
        if "A" in w.extra:
            o.set_vector_potential(w.extra["A"])
        psi = w.psi0
        t0 = time.perf_counter()
        psi = o.step(psi, 1)
        one = time.perf_counter() - t0
        n = int(max(1, min(w.step_avg.shape[0] - 1 if w.field_kind else 10**9, (seconds_target - one) / max(one, 1e-6))))
        if seconds_target - one < one:  # the first step already used the budget: it is the sample
            return w.npoints / one, 1, threads or allc, one
        t0 = time.perf_counter()
        o.step(psi, n)
        dt = time.perf_counter() - t0
        return w.npoints * n / dt, n, threads or allc, dt
    finally:
        if threads:
            oracle.set_threads(allc)


def run_reference(args):
    """--impl reference: the oracle on the host cores, same config/metric/unit; each bench step is a bounded
    sample of the workload (REF_SPLIT split-operator steps instead of 128)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle

    name = args.workload
    REF_SPLIT = {"1": 128, "2a": 4, "2b": 4, "3": 1, "4": 8, "5": 1, "d1": 128, "d2x4": 2, "d2A": 4}[name]
    w, prec, P = make_workload(name, REF_SPLIT * (args.steps + args.warmup) + 1)
    o = oracle.Solver(w.sizes, w.dx, w.dt, w.ncomp, w.mass, w.c, w.charge)
    o.set_potential(w.V)
    if w.field_kind:
        o.set_field(w.field_kind, w.step_avg)
    if "A" in w.extra:
        o.set_vector_potential(w.extra["A"])
    psi = w.psi0 if prec == "c128" else w.psi0.astype(np.complex64).astype(np.complex128)
    for _ in range(args.warmup):
        psi = o.step(psi, REF_SPLIT)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        psi = o.step(psi, REF_SPLIT)
    dt = time.perf_counter() - t0
    value = w.npoints * REF_SPLIT * args.steps / dt
    sample = f"{REF_SPLIT} split-operator steps per bench step (of {SPLIT_STEPS}), full grid, fp64"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        # the same descriptive keys and values as the product arm (the workload is the same; that a bench step here is a
        # sample of REF_SPLIT of its 128 split-operator steps is said under cpu_baseline.sample)
        "config": describe_config(name, w, prec, int(os.environ.get("WORLD_SIZE", "1"))),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle", "sample": sample,
                         "split_steps_per_bench_step": REF_SPLIT},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def l2_note(S: float) -> str:
    return ("psi larger than L2: every pass streams it from HBM" if S > 126e6 else
            "psi (%.0f MB) fits L2 (126 MB): consecutive passes of a step sequence re-touch it there; no flush, ncu DRAM bytes are below the algorithmic bytes" % (S / 1e6))


def describe_config(name, w, prec, world):
    """The keys of `config` that name the workload: identical in the product and the reference arm."""
    S = w.npoints * w.ncomp * (16 if prec == "c128" else 8)
    return {"workload": DESCR[name], "split_steps_per_step": SPLIT_STEPS, "grid": list(w.sizes), "ncomp": w.ncomp,
            "parallelism": "replicas" if world > 1 else "single GPU", "l2": l2_note(S)}


def job_throughput(updates_per_rank: float, ms_local: float, world: int, device: str = "cuda"):
    """Replicas-only aggregation: every rank did `updates_per_rank` updates in `ms_local` ms of device
    time; the job's throughput is all ranks' updates over the SLOWEST rank's time.  Returns (updates/s, max ms)."""
    ms = float(ms_local)
    if world > 1:
        import torch
        import torch.distributed as dist

        t = torch.tensor([ms], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    return updates_per_rank * world / (ms * 1e-3), ms


def measure(name, K, W, world, barrier, sampler, want_e2e):
    """Time K calls of sso_step(psi, 128) of one workload.  Returns (record, workload)."""
    import torch

    import paper_1012_3911_b200 as sso

    w, prec, P = make_workload(name, SPLIT_STEPS)  # every call replays field rows 0..127
    precision = sso.C128 if prec == "c128" else sso.C64
    cdt = np.complex128 if prec == "c128" else np.complex64
    esz = 16 if prec == "c128" else 8
    S = w.npoints * w.ncomp * esz
    nd = len(w.sizes)

    plan = sso.Plan(w.sizes, w.dx, w.dt, w.ncomp, precision)
    plan.set_constants(w.mass, w.c, w.charge)
    for opt, val in OPTIONS:
        plan.set_option(opt, val)
    plan.set_potential(w.V)
    if w.field_kind:
        plan.set_field(w.field_kind, np.ascontiguousarray(w.step_avg))
    if "A" in w.extra:
        plan.set_vector_potential(np.ascontiguousarray(w.extra["A"]))
    psi0 = w.psi0.astype(cdt)
    psi = torch.from_numpy(psi0).cuda()
    stream = torch.cuda.current_stream()

    def call():
        plan.set_time_index(0)
        plan.step(psi, SPLIT_STEPS, stream=stream)

    for _ in range(max(W, 3)):
        call()
    launches_per_call = plan.launch_count(SPLIT_STEPS)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.time()
    e0.record(stream)
    for _ in range(K):
        call()
    e1.record(stream)
    barrier()
    t1 = time.time()
    ms_local = e0.elapsed_time(e1)
    norm_after = plan.norm(psi)
    value, ms = job_throughput(float(w.npoints) * SPLIT_STEPS * K, ms_local, world)
    clocks = sampler.window(t0, t1) if sampler else None

    peak, peak_src = load_peaks()
    us_step = ms * 1e3 / (K * SPLIT_STEPS)
    pass_launches = K * (SPLIT_STEPS * P + 1) if nd > 1 else K
    per_launch_s = ms * 1e-3 / pass_launches
    bytes_per_launch = 2.0 * S  # one read + one write of psi
    achieved = bytes_per_launch / per_launch_s / 1e9
    rec = {
        "workload": DESCR[name], "grid": list(w.sizes), "ncomp": w.ncomp, "dtype": "f64" if prec == "c128" else "f32",
        "us_per_split_step": us_step, "updates_per_s": value, "ms_per_call": ms / K, "passes_per_split_step": P if nd > 1 else 0,
        "achieved_GBs": achieved, "frac_of_measured": achieved / peak, "frac_of_8TBs": achieved / 8000.0,
        "bar_us_per_split_step": BAR_US[name], "meets_60pct_of_8TBs": (us_step <= BAR_US[name]) if BAR_US[name] else None,
        "norm_after": norm_after, "clocks": clocks, "gpu_launches": int(launches_per_call * K),
        "l2": l2_note(S),
    }
    if nd == 1:
        rec["note"] = "one persistent CTA, psi stays on the SM for all 128 steps: the HBM figure is 2S per CALL over the call time, not a roofline (SURVEY H5)"
        rec["achieved_GBs"] = rec["frac_of_measured"] = rec["frac_of_8TBs"] = None
    # per pass kind, one profiled split-step sequence (events between the passes: no overlap between passes)
    try:
        plan.set_time_index(0)
        rec["per_pass"] = [{"pass": n_, "launches": c_, "avg_us": t_, "achieved_GBs": (bytes_per_launch / (t_ * 1e-6) / 1e9 if t_ > 0 else None)}
                           for n_, c_, t_ in plan.profile_step(psi, 8, stream=stream)]
    except AttributeError:
        pass
    e2e = None
    if want_e2e:
        host = torch.from_numpy(psi0.copy()).pin_memory()
        for _ in range(2):
            plan.set_time_index(0)
            plan.step_host(host, SPLIT_STEPS)
        host.copy_(torch.from_numpy(psi0))
        barrier()
        h0 = time.perf_counter()
        for _ in range(K):
            plan.set_time_index(0)
            plan.step_host(host, SPLIT_STEPS)  # synchronous: returns after the download
        torch.cuda.synchronize()
        e2e_s = time.perf_counter() - h0
        e2e_value, _ = job_throughput(float(w.npoints) * SPLIT_STEPS * K, e2e_s * 1e3, world)
        e2e_norm = float(np.sum(np.abs(host.numpy().astype(np.complex128)) ** 2) * np.prod(w.dx))
        e2e = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": S, "d2h_bytes_per_step": S, "norm_after": e2e_norm}
        del host
    plan.destroy()
    del psi
    torch.cuda.empty_cache()
    return rec, e2e, w, (ms, bytes_per_launch, per_launch_s, achieved, peak, peak_src)


def run_product(args):
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.gpus != world:
        raise SystemExit(f"bench.py --gpus {args.gpus} but WORLD_SIZE={world}: launch N>1 with torch.distributed.run (one rank per GPU)")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    K, W = args.steps, args.warmup
    head = args.workload
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
    rec, e2e, w, (ms, bytes_per_launch, per_launch_s, achieved, peak, peak_src) = measure(head, K, W, world, barrier, sampler, True)
    per = {head: rec}
    if world == 1 and not args.only:
        for name in WORKLOADS:
            if name != head:
                per[name] = measure(name, min(K, 10), W, world, barrier, sampler, False)[0]
    if sampler:
        sampler.stop()

    if rank == 0:
        traffic, traffic_src = ncu_traffic(head)
        nd = len(w.sizes)
        dominant = max(rec.get("per_pass", []), key=lambda r: r["avg_us"] * r["launches"], default=None)
        # the dominant pass KIND's own fraction: 2 S over its mean launch time (events around each launch of a profiled
        # step sequence), next to the step average `frac`
        dom_gbs = bytes_per_launch / (dominant["avg_us"] * 1e-6) / 1e9 if (dominant and dominant["avg_us"] > 0 and nd > 1) else None
        cfg = describe_config(head, w, "c128" if rec["dtype"] == "f64" else "c64", world)
        cfg.update({"us_per_split_step": rec["us_per_split_step"], "norm_after": rec["norm_after"]})
        # one flat scalar per workload (records that keep only the scalar keys of `config` still carry every workload):
        # us per split step, fraction of the 8 TB/s roofline and of the measured copy bandwidth (None in 1D: psi stays on the SM)
        for nm, r in per.items():
            cfg[f"us_{nm}"] = round(r["us_per_split_step"], 3)
            cfg[f"frac8_{nm}"] = round(r["frac_of_8TBs"], 4) if r["frac_of_8TBs"] is not None else None
            cfg[f"fracM_{nm}"] = round(r["frac_of_measured"], 4) if r["frac_of_measured"] is not None else None
        cfg["per_workload"] = per
        line = {
            "metric": METRIC, "value": rec["updates_per_s"], "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms / K,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": rec["dtype"], "data": "synthetic",
            "config": cfg,
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
                         "traffic_source": traffic_src,
                         "kernel": ("average over the pass launches of a split step (every pass launch moves psi once: sso::ring_kernel on the contiguous axis, sso::sring_kernel on the strided axes); per_pass lists each" if nd > 1 else "sso::pass_kernel (one persistent CTA, psi stays on the SM)"),
                         "dominant_pass": dominant, "dominant_achieved": dom_gbs,
                         "frac_dominant": dom_gbs / peak if dom_gbs else None,
                         "frac_dominant_of_nominal_8TBs": dom_gbs / 8000.0 if dom_gbs else None, "bytes_per_launch": bytes_per_launch, "avg_launch_us": per_launch_s * 1e6,
                         "peak_source": peak_src, "frac_of_nominal_8TBs": achieved / 8000.0},
            "e2e": e2e,
            "gpu_launches": rec["gpu_launches"],
            "clocks": rec["clocks"],
        }
        if world == 1 and not args.no_cpu_baseline:
            v, n, cores, secs = oracle_rate(w, 12.0)
            v1, n1, _, secs1 = oracle_rate(w, 6.0, threads=1)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": f"{n} split-operator steps of the same full-size workload in {secs:.1f} s (fp64)",
                                    "single_thread": {"value": v1, "cores": 1, "sample": f"{n1} split-operator step(s) in {secs1:.1f} s"}}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="sso", choices=["sso", "reference"])
    ap.add_argument("--workload", default=HEADLINE, choices=sorted(WORKLOADS), help="headline workload (top-level numbers)")
    ap.add_argument("--only", action="store_true", help="time the headline workload only (no per_workload sweep)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--opt", default="", help="tuning: comma-separated SSO_OPT_<number>=<value> pairs applied to every plan, e.g. 4=2,5=6")
    args = ap.parse_args()
    for kv in filter(None, args.opt.split(",")):
        k, v = kv.split("=")
        OPTIONS.append((int(k), int(v)))
    if args.impl == "reference":
        return run_reference(args)
    return run_product(args)


if __name__ == "__main__":
    sys.exit(main())
