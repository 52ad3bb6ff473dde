#!/usr/bin/env python
"""bench.py -- one JSON line for BASELINE.json's metric on BASELINE.json's workload.

A "step" is one pass of the whole hot path: one H_eff + LLG right-hand-side evaluation
(mm_llg_rhs: S1..S6 of DESIGN.md) on config 4 of BASELINE.json, the 512x512x128-cell film
(padded spectrum 1024x1024x256), fp32, seeded random unit vectors.  `value` is cell-updates/s
with m resident in HBM; `e2e` is the same call through the C ABI with HOST buffers
(mm_llg_rhs_host: H2D of m and D2H of dm/dt inside the timed region).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

N > 1 (under torch.distributed.run): the path does not shard (replicas
only), so every rank runs an independent replica of the workload; no data-path collective.
--impl reference times the CPU oracle (oracle/) on the host cores, as it stands, on a bounded
sample of the same workload.
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
SAMPLE_MESH = (256, 256, 64)   # CPU-oracle sample: 1/8 of the workload's cells, same cell size


def env_int(name, default):
    return int(os.environ.get(name, default))


# ------------------------------------------------------------------ clocks sampler

class ClockSampler:
    FIELDS = ["clocks.sm", "clocks.max.sm", "power.draw", "clocks_event_reasons.hw_slowdown",
              "clocks_event_reasons.hw_thermal_slowdown", "clocks_event_reasons.sw_thermal_slowdown",
              "clocks_event_reasons.sw_power_cap"]

    def __init__(self, gpu_index, period_ms=50):
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

    def _reader(self):
        for line in self.proc.stdout:
            parts = [p.strip() for p in line.split(",")]
            if len(parts) == len(self.FIELDS):
                self.samples.append((time.time(), parts))

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()

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
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
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
    k = {"S1_zf": 3 * ncell * s + a1, "S2_yf": a1 + a2, "S3_xp": 2 * a2 + octant,
         "S4_yi": a2 + a1, "S5_zi": a1 + 3 * ncell * s, "S6_pointwise": 9 * ncell * s}
    return k, sum(k.values())


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ------------------------------------------------------------------ CPU oracle leg

def oracle_rate(cfg, steps, warmup):
    """Times the oracle's own FFT path (O5) + local terms + LLG on SAMPLE_MESH."""
    from oracle import oracle as o
    o.build()
    sc = cfg.with_mesh(SAMPLE_MESH)
    t0 = time.time()
    P = o.Problem(n=sc.n, d=sc.d, Ms=sc.Ms, Aex=sc.Aex, Ku=sc.Ku, axis=sc.axis, alpha=sc.alpha,
                  gamma=sc.gamma, Hext=sc.Hext, terms=sc.terms).prepare()
    setup = time.time() - t0
    m = w.random_unit_vectors(sc.seed, sc.n).astype(np.float32).astype(np.float64)
    for _ in range(warmup):
        P.llg_rhs(m)
    times = []
    for _ in range(steps):
        t = time.perf_counter()
        P.llg_rhs(m)
        times.append(time.perf_counter() - t)
    ms = 1e3 * sum(times) / len(times)
    return {"value": sc.ncell / (ms / 1e3), "unit": UNIT, "cores": o.num_threads(), "kind": "oracle",
            "sample": f"{steps} H_eff+LLG evaluations of the oracle FFT path (fp64) on a "
                      f"{SAMPLE_MESH[0]}x{SAMPLE_MESH[1]}x{SAMPLE_MESH[2]} sub-mesh of the workload "
                      f"(same cell size, material and terms); Newell table + its FFT "
                      f"({setup:.0f} s) excluded",
            "ms_per_eval": ms, "best_ms": 1e3 * min(times)}


def run_reference(args, cfg):
    rank = env_int("RANK", 0)
    if rank != 0:
        return 0
    steps = max(1, min(args.steps, 8))
    cb = oracle_rate(cfg, steps, min(args.warmup, 1))
    line = {"metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": min(args.warmup, 1), "ms_per_step": cb["ms_per_eval"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "impl": "reference",
            "config": {"workload": cfg.name + " (oracle timed on a bounded sample, see cpu_baseline.sample)",
                       "terms": "demag+exchange+zeeman"},
            "cpu_baseline": cb,
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------ CUDA leg

def run_ours(args, cfg):
    import torch
    from paper_2606_01114_b200 import Context, build

    rank, world, local = env_int("RANK", 0), env_int("WORLD_SIZE", 1), env_int("LOCAL_RANK", 0)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    build.build()
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(v):
        if dist is None:
            return v
        t = torch.tensor([v], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    tdt = torch.float32 if args.dtype == "f32" else torch.float64
    s = 4 if args.dtype == "f32" else 8
    tiles = tuple(int(v) for v in args.tiles.split(",")) if args.tiles else None
    ctx = Context(cfg.n, cfg.d, dtype=tdt, device=f"cuda:{local}", path=args.path, kchunk=args.kchunk, tiles=tiles)
    ctx.set_material(cfg.Ms, cfg.Aex, cfg.Ku, cfg.axis, cfg.alpha, cfg.gamma)
    ctx.set_zeeman(cfg.Hext)
    ctx.set_terms(cfg.terms)
    ctx.demag_init()

    m_host = w.random_unit_vectors(cfg.seed + 1000 * rank, cfg.n).astype(
        np.float32 if args.dtype == "f32" else np.float64)
    m_pin = torch.from_numpy(m_host).pin_memory()
    out_pin = torch.empty_like(m_pin).pin_memory()
    m = m_pin.cuda()
    out = torch.empty_like(m)
    del m_host

    for _ in range(max(args.warmup, 3)):
        ctx.llg_rhs(m, out)
    torch.cuda.synchronize()

    sampler = ClockSampler(local)
    time.sleep(0.15)
    ctx.set_profiling(True)
    ctx.kernel_times()
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
    ms_step = max_over_ranks(e0.elapsed_time(e1) / args.steps)
    ktimes = ctx.kernel_times()
    ctx.set_profiling(False)

    # demag alone (extra line item of BASELINE.json's metric)
    for _ in range(2):
        ctx.demag_field(m, out)
    barrier()
    e0.record()
    for _ in range(args.steps):
        ctx.demag_field(m, out)
    e1.record()
    barrier()
    ms_demag = max_over_ranks(e0.elapsed_time(e1) / args.steps)

    # end to end through the host-buffer ABI call
    e2e_steps = max(1, min(args.steps, 5))
    m_np, out_np = m_pin.numpy(), out_pin.numpy()
    ctx.llg_rhs_host(m_np, out_np)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        ctx.llg_rhs_host(m_np, out_np)
    barrier()
    ms_e2e = max_over_ranks(1e3 * (time.perf_counter() - t0) / e2e_steps)
    sampler.stop()
    clocks = sampler.summary(t_start, t_end)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    ncell = cfg.ncell
    kbytes, total_bytes = byte_model(cfg.n, s, fast=ctx.path_name != "generic")
    peak, peak_src = measured_peak()
    per_kernel = {}
    for k, (tot, cnt) in ktimes.items():
        if cnt:
            ms = tot / cnt
            per_kernel[k] = {"ms": ms, "algorithmic_GB": kbytes[k] / 1e9,
                             "achieved_GBps": kbytes[k] / ms / 1e6, "frac": kbytes[k] / ms / 1e6 / peak}
    dom = max(per_kernel, key=lambda k: per_kernel[k]["ms"])
    traffic = None
    # dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel from the committed ncu --set full
    # capture (profiles/dominant_kernel_traffic.csv; the command is in profiles/r01_v3_fast_path.md)
    tp = os.path.join(ROOT, "profiles", "dominant_kernel_traffic.csv")
    if os.path.exists(tp):
        try:
            import csv
            for row in csv.DictReader(open(tp)):
                if row["kernel"] == dom and row["dtype"] == args.dtype and row["workload"] == "cfg4" and not args.mesh:
                    traffic = int(row["dram_bytes_per_launch"])
        except Exception:
            pass
    roofline = {"bound": "hbm", "kernel": dom, "achieved": per_kernel[dom]["achieved_GBps"],
                "peak": peak, "unit": "GB/s", "frac": per_kernel[dom]["frac"], "traffic": traffic,
                "peak_source": peak_src,
                "algorithmic_bytes_per_launch": kbytes[dom],
                "share_of_step": per_kernel[dom]["ms"] / sum(v["ms"] for v in per_kernel.values())}
    line = {
        "metric": METRIC, "value": world * ncell / (ms_step / 1e3), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.dtype,
        "data": "synthetic",
        "config": {"workload": f"{cfg.name}: one H_eff(demag+exchange+zeeman)+LLG RHS evaluation "
                               f"(mm_llg_rhs) per step, {cfg.n[0]}x{cfg.n[1]}x{cfg.n[2]} cells, "
                               f"padded spectrum {2*cfg.n[0]}x{2*cfg.n[1]}x{2*cfg.n[2]}",
                   "l2": "inputs exceed L2 (m 0.4 GB, spectra 2.4 GB, tensor table >= 0.8 GB per step)",
                   "parallelism": "replicas" if world > 1 else "single"},
        "clocks": clocks,
        "e2e": {"value": world * ncell / (ms_e2e / 1e3), "unit": UNIT, "ms_per_step": ms_e2e,
                "h2d_bytes_per_step": 3 * ncell * s, "d2h_bytes_per_step": 3 * ncell * s,
                "call": "mm_llg_rhs_host (pinned host buffers)"},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "roofline_step": {"bound": "hbm", "algorithmic_bytes": total_bytes,
                          "achieved": total_bytes / ms_step / 1e6, "peak": peak, "unit": "GB/s",
                          "frac": total_bytes / ms_step / 1e6 / peak,
                          "frac_of_nominal_8TBps": total_bytes / ms_step / 1e6 / 8000.0},
        "kernels": per_kernel,
        "demag_only": {"value": world * ncell / (ms_demag / 1e3), "unit": UNIT, "ms": ms_demag},
    }
    if world == 1 and not args.no_cpu:
        line["cpu_baseline"] = oracle_rate(cfg, 4, 1)
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
            demag_bytes = total - kb["S6_pointwise"]
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
    ap.add_argument("--path", type=int, default=0, help="0 auto, 1 generic passes, 2 fast kernels (experiments)")
    ap.add_argument("--kchunk", type=int, default=0, help="kx planes per y/z/y launch group (experiments)")
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
