#!/usr/bin/env python
"""bench.py -- one JSON line for BASELINE.json's metric on BASELINE.json's workload.

A "step" is one pass of the whole hot path: one H_eff + LLG right-hand-side evaluation
(mm_llg_rhs: S1..S6 of DESIGN.md) on config 4 of BASELINE.json, the 512x512x128-cell film
(padded spectrum 1024x1024x256), fp32, seeded random unit vectors.  `value` is cell-updates/s
with m resident in HBM; `e2e` is the same evaluation through the C ABI with HOST buffers, H2D of every
step's m and D2H of its dm/dt inside the timed region: the steps as one mm_llg_rhs_host_batch call
(independent evaluations, copies of neighbouring steps overlapping the kernels) and, under
e2e.serial, one mm_llg_rhs_host call per step.  The line also carries the
same measurement in the other precision (key "f64"), H_demag alone per dtype (`demag_only`), the
per-kernel CUDA-event durations of a second, untimed loop under the kernels' real names, and the
CPU oracle timed on the workload's own mesh (`cpu_baseline`).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

N > 1 (under torch.distributed.run): the path does not shard (replicas
only), so every rank runs an independent replica of the workload; no data-path collective.
--impl reference times the CPU oracle (oracle/) on the host cores, as it stands, on the same
mesh (its tensor table bounded as oracle_rate explains; a sub-mesh only if host memory is short).
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
sys.path.insert(0, ROOT)

import workloads as w  # noqa: E402

METRIC = "H_eff+LLG cell-updates/s (fp32, 512x512x128 film, 1 B200)"
UNIT = "cell-updates/s"
SAMPLE_MESH = (256, 256, 64)   # CPU-oracle fallback sample when host memory is short: 1/8 of the cells
ORACLE_FULL_RAM_GB = 40        # the oracle's FFT path at config 4 holds about 32 GB
ORACLE_TABLE_CUT = (64, 64, 16)  # offsets kept in the oracle's tensor table for TIMING runs (see oracle_rate)


def env_int(name, default):
    return int(os.environ.get(name, default))


# ------------------------------------------------------------------ clocks sampler

class ClockSampler:
    """nvidia-smi sampling every 10 ms in a side process.  Each line carries nvidia-smi's own timestamp
    (the pipe delivers lines in bursts, so the time a line is READ says nothing about when it was taken)."""
    FIELDS = ["timestamp", "clocks.sm", "clocks.max.sm", "power.draw", "clocks_event_reasons.hw_slowdown",
              "clocks_event_reasons.hw_thermal_slowdown", "clocks_event_reasons.sw_thermal_slowdown",
              "clocks_event_reasons.sw_power_cap"]

    def __init__(self, gpu_index, period_ms=10):
        self.samples = []
        self.proc = None
        self.thread = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(gpu_index), "--query-gpu=" + ",".join(self.FIELDS),
                 "--format=csv,noheader,nounits", "-lms", str(period_ms)],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._reader, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    @staticmethod
    def _stamp(text, fallback):
        try:
            import datetime
            return datetime.datetime.strptime(text, "%Y/%m/%d %H:%M:%S.%f").timestamp()
        except ValueError:
            return fallback

    def _reader(self):
        for line in self.proc.stdout:
            parts = [p.strip() for p in line.split(",")]
            if len(parts) == len(self.FIELDS):
                self.samples.append((self._stamp(parts[0], time.time()), parts[1:]))

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()
            if self.thread is not None:
                self.thread.join(timeout=2)

    def summary(self, t0, t1):
        inside = [p for (t, p) in self.samples if t0 <= t <= t1]
        used = inside if len(inside) >= 2 else [p for (_, p) in self.samples]
        sm, smax, reasons = [], [], set()
        for p in used:
            try:
                sm.append(float(p[0]))
                smax.append(float(p[1]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown",
                                  "sw_power_cap"), p[3:]):
                if val == "Active":
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0, "samples_in_timed_region": 0}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(smax), "reasons": sorted(reasons),
                "samples": len(used), "samples_in_timed_region": len(inside)}


# ------------------------------------------------------------------ byte model

def byte_model(n, s, fast=False):
    """Algorithmic bytes per evaluation and per kernel (exact form).
    The half-spectrum axis is z (nz + 1 planes) in the generic passes, x (nx + 1 planes) in the
    x-first fast kernels; the model is the same 84 s B/cell otherwise."""
    nx, ny, nz = n
    ncell = nx * ny * nz
    Kz = 1 if nz == 1 else nz + 1
    Py = 1 if ny == 1 else 2 * ny
    if fast:
        a1 = 3 * (nx + 1) * ny * nz * 2 * s
        a2 = 3 * (nx + 1) * Py * nz * 2 * s
    else:
        a1 = 3 * nx * ny * Kz * 2 * s
        a2 = 3 * nx * Py * Kz * 2 * s
    octant = 6 * (nx + 1) * (ny + 1) * Kz * s
    k = {"S1": 3 * ncell * s + a1, "S2": a1 + a2, "S3": 2 * a2 + octant,
         "S4": a2 + a1, "S5": a1 + 3 * ncell * s, "S6": 9 * ncell * s}
    return k, sum(k.values())


# ------------------------------------------------------------------ rank logic (N > 1: replicas only)

def rank_seed(cfg, rank):
    """Every rank runs an independent replica on its own seeded input."""
    return cfg.seed + 1000 * rank


def max_over_ranks(v, dist=None, device="cuda"):
    """Device time of the job = the slowest rank's (torch.distributed MAX all-reduce)."""
    if dist is None:
        return v
    import torch
    t = torch.tensor([v], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(world, ncell, ms_step):
    """Whole-job cell-updates/s: every rank processed ncell cells per step in ms_step (max over ranks)."""
    return world * ncell / (ms_step / 1e3)


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ------------------------------------------------------------------ CPU oracle leg

def host_mem_available_gb():
    try:
        import psutil
        return psutil.virtual_memory().available / 2 ** 30
    except Exception:
        return 0.0


ORACLE_SAMPLES = [(512, 512, 128), (512, 512, 64), (512, 256, 64), (256, 256, 64)]


def oracle_problem(o, sc):
    """Oracle problem on mesh sc.n with the timing-run table (see oracle_rate); returns (P, setup seconds, cut)."""
    t0 = time.time()
    cut = tuple(min(a, b) for a, b in zip(sc.n, ORACLE_TABLE_CUT))
    N = np.zeros((6,) + tuple(sc.n))
    N[:, :cut[0], :cut[1], :cut[2]] = o.newell_octant(cut, sc.d)
    P = o.Problem(n=sc.n, d=sc.d, Ms=sc.Ms, Aex=sc.Aex, Ku=sc.Ku, axis=sc.axis, alpha=sc.alpha,
                  gamma=sc.gamma, Hext=sc.Hext, terms=sc.terms, N=N).prepare()
    P.N = None
    return P, time.time() - t0, cut


def oracle_rate(cfg, steps, warmup, budget_s=240.0):
    """Times the oracle's own FFT path (O5) + local terms + LLG (orc_llg_rhs, as it stands): `steps`
    evaluations on the workload's own mesh when host memory and the time budget allow, else on the
    largest sub-mesh of ORACLE_SAMPLES (same cell size, material and terms) for which `steps`
    evaluations are estimated to fit `budget_s` (the reason is printed in `sample`).  The estimate
    comes from one evaluation on the smallest sample, scaled by the cell count.

    The Newell table is excluded from the timing (BASELINE.md's plan: "N-hat precomputed and
    excluded"), and at config 4 its quad-precision evaluation alone takes minutes of host time.
    The timed code has no data-dependent branch, so for a TIMING run the table is evaluated only for
    offsets below ORACLE_TABLE_CUT cells and left zero beyond; the transform of the table and every
    timed step run on the full mesh.  (Parity runs always use the full table: tests/.)"""
    from oracle import oracle as o
    o.build()
    avail = host_mem_available_gb()
    small = cfg.with_mesh(ORACLE_SAMPLES[-1])
    why = ""
    if cfg.ncell <= small.ncell:
        sc = cfg
    else:
        Ps, _, _ = oracle_problem(o, small)
        ms_ = w.random_unit_vectors(small.seed, small.n)
        t = time.perf_counter()
        Ps.llg_rhs(ms_)
        per_cell = 1.3 * (time.perf_counter() - t) / small.ncell      # larger meshes run less cache-friendly
        del Ps, ms_
        sc = None
        for n in [tuple(cfg.n)] + [n for n in ORACLE_SAMPLES if n != tuple(cfg.n)]:
            c = cfg.with_mesh(n)
            if c.ncell > cfg.ncell:
                continue
            fits_time = (steps + warmup) * per_cell * c.ncell + 2.0 * per_cell * c.ncell <= budget_s
            fits_mem = avail >= ORACLE_FULL_RAM_GB * c.ncell / (512 * 512 * 128)
            if fits_time and fits_mem:
                sc = c
                break
        if sc is None:
            sc = small
        if sc.n != cfg.n:
            why = (f" -- a sub-mesh because {steps}+{warmup} evaluations of the full mesh were estimated at "
                   f"{(steps + warmup) * per_cell * cfg.ncell:.0f} s (budget {budget_s:.0f} s) with "
                   f"{avail:.0f} GB of host memory available (full size needs ~{ORACLE_FULL_RAM_GB} GB)")
    P, setup, cut = oracle_problem(o, sc)
    m = w.random_unit_vectors(sc.seed, sc.n).astype(np.float32).astype(np.float64)
    for _ in range(warmup):
        P.llg_rhs(m)
    times = []
    for _ in range(steps):
        t = time.perf_counter()
        P.llg_rhs(m)
        times.append(time.perf_counter() - t)
    ms = 1e3 * sum(times) / len(times)
    where = (f"the workload's own {sc.n[0]}x{sc.n[1]}x{sc.n[2]} mesh" if sc.n == cfg.n else
             f"a {sc.n[0]}x{sc.n[1]}x{sc.n[2]} sub-mesh of the workload (same cell size, material and terms)" + why)
    return {"value": sc.ncell / (ms / 1e3), "unit": UNIT, "cores": o.num_threads(), "kind": "oracle",
            "sample": f"{steps} H_eff+LLG evaluation(s) of the oracle FFT path (fp64) on {where}; tensor table "
                      f"evaluated for offsets < {cut[0]}x{cut[1]}x{cut[2]} cells only (timing run: values do not "
                      f"change the time) and its transform ({setup:.0f} s) excluded",
            "mesh": list(sc.n), "ms_per_eval": ms, "best_ms": 1e3 * min(times)}


def run_reference(args, cfg):
    rank = env_int("RANK", 0)
    if rank != 0:
        return 0
    steps = max(1, args.steps)
    cb = oracle_rate(cfg, steps, min(args.warmup, 1))
    line = {"metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": min(args.warmup, 1), "ms_per_step": cb["ms_per_eval"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "impl": "reference",
            "config": {"workload": f"{cfg.name}: one H_eff(demag+exchange+zeeman)+LLG RHS evaluation per step "
                                   f"(oracle, fp64; mesh and bounds in cpu_baseline.sample)",
                       "terms": "demag+exchange+zeeman"},
            "cpu_baseline": cb,
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------ CUDA leg

def measure(args, cfg, dtype, local, rank, dist, with_e2e):
    """One dtype on this rank's replica: timed steps (nothing but mm_llg_rhs launches between the two
    events), then H_demag alone, then an UNTIMED loop with the library's per-kernel CUDA events, then
    (optionally) the end-to-end host-buffer leg."""
    import torch
    from paper_2606_01114_b200 import Context

    tdt = torch.float32 if dtype == "f32" else torch.float64
    ndt = np.float32 if dtype == "f32" else np.float64
    tiles = tuple(int(v) for v in args.tiles.split(",")) if args.tiles else None
    ctx = Context(cfg.n, cfg.d, dtype=tdt, device=f"cuda:{local}", path=args.path, tiles=tiles)
    ctx.set_material(cfg.Ms, cfg.Aex, cfg.Ku, cfg.axis, cfg.alpha, cfg.gamma)
    ctx.set_zeeman(cfg.Hext)
    ctx.set_terms(cfg.terms)
    ctx.demag_init()

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    m_pin = torch.from_numpy(w.random_unit_vectors(rank_seed(cfg, rank), cfg.n).astype(ndt)).pin_memory()
    m = m_pin.cuda()
    out = torch.empty_like(m)
    warm = max(args.warmup, 3)
    for _ in range(warm):
        ctx.llg_rhs(m, out)
    torch.cuda.synchronize()

    sampler = ClockSampler(local) if dtype == "f32" else None
    if sampler:
        time.sleep(0.1)
    l0 = ctx.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t_start = time.time()
    e0.record()
    for _ in range(args.steps):
        ctx.llg_rhs(m, out)
    e1.record()
    barrier()
    t_end = time.time()
    launches = ctx.launch_count - l0
    ms_step = max_over_ranks(e0.elapsed_time(e1) / args.steps, dist)
    clocks = None
    if sampler:
        time.sleep(0.03)          # let the last samples of the timed region reach the pipe
        sampler.stop()
        clocks = sampler.summary(t_start, t_end)

    # demag alone (the other half of BASELINE.json's metric)
    for _ in range(2):
        ctx.demag_field(m, out)
    barrier()
    e0.record()
    for _ in range(args.steps):
        ctx.demag_field(m, out)
    e1.record()
    barrier()
    ms_demag = max_over_ranks(e0.elapsed_time(e1) / args.steps, dist)

    # per-kernel durations: a second, untimed loop with the library's CUDA events around every launch
    ctx.set_profiling(True)
    ctx.kernel_times()
    for _ in range(args.steps):
        ctx.llg_rhs(m, out)
    ktimes = ctx.kernel_times()
    ctx.set_profiling(False)
    names = {k: ctx.kernel_name(i) for i, k in enumerate(ctx.KERNEL_KINDS)}

    ms_e2e = ms_e2e_serial = None
    if with_e2e:   # end to end through the host-buffer ABI calls, copies inside the timed region
        ins = [m_pin, m_pin.clone().pin_memory()]
        outs = [torch.empty_like(m_pin).pin_memory(), torch.empty_like(m_pin).pin_memory()]
        e2e_steps = max(1, min(args.steps, 5))
        m_np, out_np = ins[0].numpy(), outs[0].numpy()
        ctx.llg_rhs_host(m_np, out_np)
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):      # one evaluation per call: upload, kernels, download, one after the other
            ctx.llg_rhs_host(m_np, out_np)
        barrier()
        ms_e2e_serial = max_over_ranks(1e3 * (time.perf_counter() - t0) / e2e_steps, dist)
        # the same steps as ONE batch call: independent evaluations, every step's input uploaded from and result
        # downloaded to pinned host memory, the copies of neighbouring steps overlapping the kernels
        nb = max(2, min(args.steps, 20))
        bi = [ins[i & 1].numpy() for i in range(nb)]
        bo = [outs[i & 1].numpy() for i in range(nb)]
        ctx.llg_rhs_host_batch(bi[:2], bo[:2])
        barrier()
        t0 = time.perf_counter()
        ctx.llg_rhs_host_batch(bi, bo)
        barrier()
        ms_e2e = max_over_ranks(1e3 * (time.perf_counter() - t0) / nb, dist)
    path_name = ctx.path_name
    ctx.close()
    del m, out, ctx
    torch.cuda.empty_cache()
    return {"ms_step": ms_step, "ms_demag": ms_demag, "ms_e2e": ms_e2e, "ms_e2e_serial": ms_e2e_serial, "ktimes": ktimes, "names": names,
            "launches": int(launches), "clocks": clocks, "path": path_name, "warmup": warm}


def traffic_of(kernel, dtype, workload):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` from the committed ncu --set full
    capture (profiles/dominant_kernel_traffic.csv names the capture and the source commit), or None."""
    tp = os.path.join(ROOT, "profiles", "dominant_kernel_traffic.csv")
    try:
        import csv
        for row in csv.DictReader(open(tp)):
            if row["kernel"] == kernel and row["dtype"] == dtype and row["workload"] == workload:
                return int(row["dram_bytes_per_launch"]), row.get("source_commit") or None
    except Exception:
        pass
    return None, None


def report(cfg, dtype, r, world, peak, workload_tag):
    s = 4 if dtype == "f32" else 8
    kbytes, total_bytes = byte_model(cfg.n, s, fast=r["path"] != "generic")
    per_kernel = {}
    for kind, (tot, cnt) in r["ktimes"].items():
        if cnt:
            ms = tot / cnt
            per_kernel[r["names"][kind]] = {"kind": kind, "ms": ms, "algorithmic_GB": kbytes[kind] / 1e9,
                                            "achieved_GBps": kbytes[kind] / ms / 1e6,
                                            "frac": kbytes[kind] / ms / 1e6 / peak}
    dom = max(per_kernel, key=lambda k: per_kernel[k]["ms"])
    traffic, commit = traffic_of(dom, dtype, workload_tag)
    roofline = {"bound": "hbm", "kernel": dom, "kind": per_kernel[dom]["kind"],
                "achieved": per_kernel[dom]["achieved_GBps"], "peak": peak, "unit": "GB/s",
                "frac": per_kernel[dom]["frac"], "traffic": traffic, "traffic_source_commit": commit,
                "algorithmic_bytes_per_launch": kbytes[per_kernel[dom]["kind"]],
                "share_of_step": per_kernel[dom]["ms"] / sum(v["ms"] for v in per_kernel.values())}
    step = {"bound": "hbm", "algorithmic_bytes": total_bytes, "achieved": total_bytes / r["ms_step"] / 1e6,
            "peak": peak, "unit": "GB/s", "frac": total_bytes / r["ms_step"] / 1e6 / peak,
            "frac_of_nominal_8TBps": total_bytes / r["ms_step"] / 1e6 / 8000.0}
    demag_bytes = total_bytes - kbytes["S6"]
    demag = {"value": job_value(world, cfg.ncell, r["ms_demag"]), "unit": UNIT, "ms": r["ms_demag"],
             "frac": demag_bytes / r["ms_demag"] / 1e6 / peak}
    return per_kernel, roofline, step, demag


def run_ours(args, cfg):
    import torch
    from paper_2606_01114_b200 import build

    rank, world, local = env_int("RANK", 0), env_int("WORLD_SIZE", 1), env_int("LOCAL_RANK", 0)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    build.build()
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    r = measure(args, cfg, args.dtype, local, rank, dist, with_e2e=True)
    other = "f64" if args.dtype == "f32" else "f32"
    r2 = None if args.single_dtype else measure(args, cfg, other, local, rank, dist, with_e2e=False)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    ncell = cfg.ncell
    s = 4 if args.dtype == "f32" else 8
    peak, peak_src = measured_peak()
    tag = "cfg4" if not args.mesh else "x".join(str(v) for v in cfg.n)
    per_kernel, roofline, step, demag = report(cfg, args.dtype, r, world, peak, tag)
    roofline["peak_source"] = peak_src
    line = {
        "metric": METRIC, "value": job_value(world, ncell, r["ms_step"]), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": r["warmup"], "ms_per_step": r["ms_step"],
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.dtype,
        "data": "synthetic",
        "config": {"workload": f"{cfg.name}: one H_eff(demag+exchange+zeeman)+LLG RHS evaluation "
                               f"(mm_llg_rhs) per step, {cfg.n[0]}x{cfg.n[1]}x{cfg.n[2]} cells, "
                               f"padded spectrum {2*cfg.n[0]}x{2*cfg.n[1]}x{2*cfg.n[2]}",
                   "l2": "inputs exceed L2 (m 0.4 GB, spectra 2.4 GB, tensor table >= 0.8 GB per step)",
                   "parallelism": "replicas" if world > 1 else "single"},
        "clocks": r["clocks"],
        "e2e": {"value": job_value(world, ncell, r["ms_e2e"]), "unit": UNIT, "ms_per_step": r["ms_e2e"],
                "h2d_bytes_per_step": 3 * ncell * s, "d2h_bytes_per_step": 3 * ncell * s,
                "call": "mm_llg_rhs_host_batch (pinned host buffers; independent evaluations, the upload of step "
                        "i+1 and the download of step i-1 overlap the kernels of step i)",
                "serial": {"value": job_value(world, ncell, r["ms_e2e_serial"]), "ms_per_step": r["ms_e2e_serial"],
                           "call": "mm_llg_rhs_host, one evaluation per call (upload, kernels, download in turn)"}},
        "gpu_launches": r["launches"],
        "roofline": roofline,
        "roofline_step": step,
        "kernels": per_kernel,
        "kernels_note": "per-kernel CUDA events from a second, untimed loop of the same steps",
        "demag_only": demag,
    }
    if r2 is not None:
        pk2, rf2, st2, dm2 = report(cfg, other, r2, world, peak, tag)
        line[other] = {"value": job_value(world, ncell, r2["ms_step"]), "unit": UNIT, "ms_per_step": r2["ms_step"],
                       "dtype": other, "gpu_launches": r2["launches"], "roofline": rf2, "roofline_step": st2,
                       "kernels": pk2, "demag_only": dm2}
    if world == 1 and not args.no_cpu:
        line["cpu_baseline"] = oracle_rate(cfg, 1, 0, budget_s=90.0)   # one evaluation of the workload itself
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


def run_sweep(args):
    """Config 5 of BASELINE.json: H_demag and H_eff+LLG throughput over the sweep meshes, fp32 and
    fp64, one JSON line per (mesh, dtype); the CPU oracle's FFT path is timed at the sizes it
    finishes in about a minute (--no-cpu skips it).  Not the driver's bench line: a report."""
    import torch
    from paper_2606_01114_b200 import Context, build

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    build.build()
    cfg5 = w.get_config(5)
    peak, peak_src = measured_peak()
    steps = max(3, min(args.steps, 30))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def timed(fn):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0.record()
        for _ in range(steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / steps

    meshes = w.PAPER_MESHES if args.paper_meshes else w.SWEEP_MESHES
    for n in meshes:
        cfg = cfg5.with_mesh(n, name=("paper_mesh_%dx%dx%d" if args.paper_meshes else "cfg5_sweep_%dx%dx%d") % n)
        for dt in ("f32", "f64"):
            s = 4 if dt == "f32" else 8
            tdt = torch.float32 if dt == "f32" else torch.float64
            ctx = Context(cfg.n, cfg.d, dtype=tdt, device="cuda:0")
            ctx.set_material(cfg.Ms, cfg.Aex, cfg.Ku, cfg.axis, cfg.alpha, cfg.gamma)
            ctx.set_terms(cfg.terms)
            t0 = time.time()
            ctx.demag_init()
            torch.cuda.synchronize()
            t_init = time.time() - t0
            m = torch.from_numpy(w.random_unit_vectors(cfg.seed, cfg.n).astype(
                np.float32 if dt == "f32" else np.float64)).cuda()
            out = torch.empty_like(m)
            ms_d = timed(lambda: ctx.demag_field(m, out))
            ms_r = timed(lambda: ctx.llg_rhs(m, out))
            kb, total = byte_model(cfg.n, s, fast=ctx.path_name != "generic")
            demag_bytes = total - kb["S6"]
            line = {"sweep": cfg.name, "dtype": dt, "cells": cfg.ncell,
                    "path": {"fast": "fast (x-first)", "mixed": "mixed-radix (x-first)", "generic": "generic (z-first)",
                             "embedded": "fast (x-first) on the enclosing power-of-two mesh"}[ctx.path_name],
                    "demag": {"ms": ms_d, "cell_updates_per_s": cfg.ncell / ms_d * 1e3,
                              "frac_hbm_measured": demag_bytes / ms_d / 1e6 / peak,
                              "frac_hbm_8TBps": demag_bytes / ms_d / 1e6 / 8000.0},
                    "heff_llg": {"ms": ms_r, "cell_updates_per_s": cfg.ncell / ms_r * 1e3,
                                 "frac_hbm_measured": total / ms_r / 1e6 / peak,
                                 "frac_hbm_8TBps": total / ms_r / 1e6 / 8000.0},
                    "init_s": t_init, "peak_GBps": peak}
            if dt == "f64" and tuple(n) in w.PAPER_DEMAG_MS:
                pms, src = w.PAPER_DEMAG_MS[tuple(n)]
                line["paper_context"] = {"demag_ms": pms, "hardware": src, "ratio_demag": pms / ms_d}
            ctx.close()
            del m, out, ctx
            torch.cuda.empty_cache()
            if dt == "f64" and not args.no_cpu and cfg.ncell <= 128 ** 3:
                from oracle import oracle as o
                o.build()
                P = o.Problem(n=cfg.n, d=cfg.d, Ms=cfg.Ms, Aex=cfg.Aex, alpha=cfg.alpha, gamma=cfg.gamma,
                              terms=cfg.terms).prepare()
                mh = w.random_unit_vectors(cfg.seed, cfg.n)
                P.llg_rhs(mh)
                t = time.perf_counter()
                P.llg_rhs(mh)
                dtc = time.perf_counter() - t
                line["cpu_oracle"] = {"cell_updates_per_s": cfg.ncell / dtc, "ms": 1e3 * dtc,
                                      "cores": o.num_threads(), "what": "oracle FFT path, H_eff+LLG, fp64"}
            print(json.dumps(line), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--dtype", default="f32", choices=["f32", "f64"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--path", type=int, default=0, help="0 auto, 1 generic passes, 2 x-first kernels, 3 mixed (experiments)")
    ap.add_argument("--single-dtype", action="store_true", help="skip the other dtype's extra block")
    ap.add_argument("--tiles", default=None, help="generic passes: tile widths bz,by,bk (experiments)")
    ap.add_argument("--mesh", default=None, help="override mesh, e.g. 256x256x64 (experiments)")
    ap.add_argument("--sweep", action="store_true", help="config 5: one line per sweep mesh and dtype")
    ap.add_argument("--paper-meshes", action="store_true",
                    help="with --sweep: the paper's own meshes (N = 100, 350, 400 cubes, 512x512x90)")
    args = ap.parse_args()
    if args.sweep:
        return run_sweep(args)
    cfg = w.get_config(4)
    if args.mesh:
        cfg = cfg.with_mesh(tuple(int(v) for v in args.mesh.split("x")),
                            name="cfg4_material_" + args.mesh)
    if args.impl == "reference":
        return run_reference(args, cfg)
    return run_ours(args, cfg)


if __name__ == "__main__":
    sys.exit(main())
