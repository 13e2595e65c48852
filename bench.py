#!/usr/bin/env python
"""bench.py -- throughput of the B200 UGKS step (fp64 cell x velocity-point updates/s) and its roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C3] [--impl ours|reference] [--no-extra]

A "step" is one pass of the whole hot path (cell moments, face scalars, cell scalars, tables, flux+update) over the
synthetic channel workload; the default workload is C4, the largest single-GPU configuration of BASELINE.json.  N > 1 (under torchrun) runs N independent replicas ("replicas only": the path is
single-GPU by north_star); value = points all ranks processed / max-over-ranks device time.
Prints ONE JSON line on rank 0.  --impl reference times the CPU oracle on a bounded sample instead.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np
import psutil

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "fp64 UGKS cell x velocity-point updates/s"
UNIT = "updates/s"
ALG_BYTES_PER_POINT = 16.0          # read f^n once, write f^{n+1} once
DECLARED_BYTES_PER_POINT = 24.0     # the pass structure built: cell_moments reads f (8 B), flux_update reads + writes f (16 B)
KERNEL_ALG_BYTES = {"cell_moments": 8.0, "flux_update": 16.0}
FP64_PEAK = 148 * 4 * 16 * 1.965e9  # plain FP64 pipe, thread-instructions/s (one warp DFMA per 2 cycles per sub-partition)


COUNTS_FILE = "profiles/r3_counts.json"
_KERNEL_SOURCES = ("ugks_jit_common.cuh", "ugks_jit_moments.cuh", "ugks_jit_update.cuh", "ugks_jit.cu", "ugks_api.cu")


def kernel_source_sha():
    """sha256 over the files that decide the code and the launch geometry of the two f-sized kernels."""
    import hashlib
    h = hashlib.sha256()
    for fn in _KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_1810_08137_b200", "csrc", fn), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def _profile_counts(name):
    """Per-kernel instruction counts and DRAM traffic of workload ``name`` from the committed ncu capture (COUNTS_FILE, written
    from the ncu command named in profiles/r3_kernels.md): FP64 thread instructions (DFMA + DMUL + DADD, predicated on), all
    thread instructions, dram bytes -- per launch of one step.  The counts are static per build: the file records the sha256
    of the kernel sources it was captured from, and (None, note) is returned when the sources here differ (a stale count would
    otherwise be labelled "of this build") or when no capture of that workload is committed."""
    try:
        with open(os.path.join(ROOT, COUNTS_FILE)) as fh:
            d = json.load(fh)
    except Exception:
        return None, f"{COUNTS_FILE} missing"
    if d.get("_meta", {}).get("kernel_source_sha256") != kernel_source_sha():
        return None, f"{COUNTS_FILE} was captured from other kernel sources than this build's: instruction counts not reported"
    return d.get(name), None if d.get(name) else f"no capture of {name} in {COUNTS_FILE}"


def _cpu_model():
    try:
        with open("/proc/cpuinfo") as fh:
            for ln in fh:
                if ln.startswith("model name"):
                    return ln.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def fp64_peak_measured():
    """(pipe rate, three-operand rate): thread-level DFMA/s of the plain FP64 pipe measured by bench_fp64_peak.cu (compiled here
    with nvcc for sm_100a; a bench-side helper library, not part of libugks) -- with two of the three operands reused (the rate
    of the 16-lane pipe itself: the roofline peak) and with three distinct register operands per DFMA (what register-operand
    fetch allows a kernel whose operands all differ; reported beside the peak, not used as the denominator)."""
    import ctypes as C
    src, so = os.path.join(ROOT, "bench_fp64_peak.cu"), os.path.join(ROOT, "libbench_fp64.so")
    if not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = so + f".tmp{os.getpid()}"
        subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-Xcompiler", "-fPIC", "-shared", "-o", tmp, src], check=True)
        os.replace(tmp, so)
    lib = C.CDLL(so)
    out, out3 = C.c_double(0.0), C.c_double(0.0)
    rc = lib.bench_fp64_peak(C.byref(out)) or lib.bench_fp64_peak_3op(C.byref(out3))
    if rc:
        raise RuntimeError(f"bench_fp64_peak -> {rc}")
    return float(out.value), float(out3.value)


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "20"], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            self.t.join(timeout=2)

    def summary(self):
        sm, mx, reasons = [], 0.0, set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = max(mx, float(r[1]))
            except Exception:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx or None, "reasons": sorted(reasons),
                "samples": len(sm)}


def dist_setup(n_gpus, backend=None):
    """(rank, world, dist or None).  One process per GPU under torchrun; plain python for N = 1."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    if world == 1:
        return 0, 1, None
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    if not dist.is_initialized():
        dist.init_process_group(backend=backend or "nccl")
    return rank, world, dist


def dist_max(dist, value, device="cpu"):
    """max over ranks of a python float (identity for a single process)."""
    if dist is None:
        return value
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def dist_sum(dist, value, device="cpu"):
    if dist is None:
        return value
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def oracle_sample(p, seconds_hint=15.0, cores=None):
    """The CPU oracle as it stands on a bounded sample of workload p: same physics and velocity grid, the mesh
    cut to the first rows (J_s rows of I cells, walls kept), enough steps for ~10-30 s of CPU work."""
    from oracle import Oracle
    cores = cores or os.cpu_count() or 1
    est = 1.0e7 * cores * 0.7                                   # updates/s guess, only to size the sample
    pts_target = est * seconds_hint / 3.0
    Js = int(max(4, min(p.J, pts_target / (p.I * p.N))))
    ps = workloads.channel_config(p.name, I=p.I, J=Js)
    W, f, _ = workloads.initial_state(ps)
    o = Oracle(ps, threads=cores)
    o.set_state(W, f)
    o.step(1)                                                   # warm caches / page in
    t0 = time.perf_counter()
    nst = 0
    while True:
        o.step(1); nst += 1
        el = time.perf_counter() - t0
        if el > seconds_hint * 0.6 or nst >= 50:
            break
    return ps.points * nst / el, cores, f"{p.name} physics and {p.Nu}x{p.Nv} velocity grid on a {ps.I}x{ps.J} mesh, {nst} steps, {cores} OpenMP threads", el / nst


def run_reference(args):
    if int(os.environ.get("RANK", "0")) != 0:                    # under torchrun rank 0 alone runs it; no collective
        return
    p = workloads.channel_config(args.config)
    steps = max(1, args.steps)
    from oracle import Oracle
    cores = os.cpu_count() or 1
    Js = int(max(4, min(p.J, 2.5e7 / (p.I * p.N))))
    ps = workloads.channel_config(p.name, I=p.I, J=Js)
    W, f, _ = workloads.initial_state(ps)
    o = Oracle(ps, threads=cores)
    o.set_state(W, f)
    for _ in range(max(1, args.warmup)):
        o.step(1)
    t0 = time.perf_counter()
    for _ in range(steps):
        o.step(1)
    el = time.perf_counter() - t0
    val = ps.points * steps / el
    sample = f"{p.name} physics and {p.Nu}x{p.Nv} velocity grid on a {ps.I}x{ps.J} mesh per step, {cores} OpenMP threads"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * el / steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": _workload_name(p) + f" -- timed on the mesh cut {ps.I}x{ps.J} (first {ps.J} rows, walls kept; throughput per point)",
                       "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "cpu": _cpu_model()},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def _problem(name):
    if name.startswith("M"):
        mesh, nuv = name.split("-")
        return workloads.paper_mesh(mesh, int(nuv))
    return workloads.channel_config(name)


def _summary_row(value, ms_step, hb, clocks):
    return [float("%.4g" % value), round(ms_step, 4), round(hb["step_frac_of_16B_floor"], 4), round(hb["cell_moments"]["frac"], 4),
            round(hb["flux_update"]["frac"], 4), clocks.get("sm_mhz")]


def _workload_name(p):
    return f"{p.name}: channel {p.I}x{p.J} cells, {p.Nu}x{p.Nv} velocity grid, Kn={p.Kn}"


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C4", choices=list(workloads.CONFIGS) + ["M4-29", "M4-69", "M3-49"],
                    help="BASELINE.json config, or one of the paper's own meshes x odd velocity grids (Table 1 / Table 3)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-extra", action="store_true", help="skip the other configs / cpu baseline (N=1 default runs them)")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_1810_08137_b200 import Ugks
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the UGKS path has no CPU fallback")
    rank, world, dist = dist_setup(args.gpus)
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dev = f"cuda:{local}"
    torch.cuda.set_device(local)
    warmup = max(3, args.warmup)
    steps = max(1, args.steps)
    peak, peak_src = _peaks()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def measure(p, steps, warmup, e2e, kernels, tangential=False):
        fh = torch.empty((p.J, p.I, p.Nv, p.Nu), dtype=torch.float64, pin_memory=True)
        W, _, _ = workloads.initial_state(p, out_f=fh.numpy())          # f is drawn straight into pinned memory
        Wh = torch.from_numpy(W).pin_memory()
        del W
        g = Ugks(p, device=dev, tangential=tangential)
        g.set_state(Wh.to(dev), fh.to(dev))
        torch.cuda.empty_cache()
        g.step(warmup); g.sync()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        l0 = g.launch_count
        with ClockSampler(local) as cs:
            e0.record()
            g.step(steps)
            e1.record()
            barrier()
        ms = dist_max(dist, e0.elapsed_time(e1), dev)
        res = {"ms": ms, "launches": g.launch_count - l0, "clocks": cs.summary(), "points": p.points}
        if kernels:
            g.set_option("profile", 1)
            g.step(steps)
            kt = g.kernel_times()
            g.set_option("profile", 0)
            res["kernels"] = {k: {"ms_per_launch": t / max(n, 1), "launches": n} for k, (t, n) in kt.items()}
        if e2e:
            Wo = torch.empty_like(Wh).pin_memory()
            fo = torch.empty_like(fh).pin_memory()
            reps = 3
            for it in range(reps + 1):                       # first pass untimed (page-locks, first-touch)
                if it == 1:
                    barrier(); t0 = time.perf_counter()
                g.set_state(Wh.numpy(), fh.numpy())          # host -> device inside the timed region
                g.step(1)
                g.f(out=fo.numpy()); g.W(out=Wo.numpy())     # device -> host
            barrier()
            el = dist_max(dist, time.perf_counter() - t0, dev)
            res["e2e"] = {"value": world * p.points * reps / el, "unit": UNIT,
                          "h2d_bytes_per_step": int(fh.numel() * 8 + Wh.numel() * 8),
                          "d2h_bytes_per_step": int(fo.numel() * 8 + Wo.numel() * 8), "ms_per_step": 1e3 * el / reps}
        g.close()
        del g, Wh, fh
        torch.cuda.empty_cache()
        return res

    p = _problem(args.config)
    fp64_measured, fp64_3op = fp64_peak_measured()

    def hbm_fracs(q, ms_step, kernel_ms):
        """HBM-roofline fractions of a workload: per f-sized kernel (its algorithmic bytes / its time) and for the step against
        the 16-B floor and against the declared 24-B pass structure."""
        out = {"step_frac_of_16B_floor": ALG_BYTES_PER_POINT * q.points / (ms_step * 1e-3) / 1e9 / peak,
               "step_frac_of_declared_24B": DECLARED_BYTES_PER_POINT * q.points / (ms_step * 1e-3) / 1e9 / peak}
        for k, bpp in KERNEL_ALG_BYTES.items():
            gbs = bpp * q.points / (kernel_ms[k] * 1e-3) / 1e9
            out[k] = {"alg_bytes_per_point": bpp, "achieved_gbs": gbs, "frac": gbs / peak}
        return out

    def alu_fracs(q, kernel_ms, counts):
        """FP64-pipe and issue-slot use of the two f-sized kernels from the committed instruction counts and the live times."""
        if not counts:
            return None
        out = {}
        for k in KERNEL_ALG_BYTES:
            c = counts.get(k)
            if not c:
                continue
            t = kernel_ms[k] * 1e-3
            out[k] = {"fp64_inst_per_point": c["fp64_thread_inst"] / q.points, "inst_per_point": c["thread_inst"] / q.points,
                      "fp64_inst_per_s": c["fp64_thread_inst"] / t, "frac_of_fp64_peak": c["fp64_thread_inst"] / t / fp64_measured,
                      "frac_of_3operand_dfma_rate": c["fp64_thread_inst"] / t / fp64_3op,
                      "dram_bytes": c.get("dram_bytes")}
        return out

    r = measure(p, steps, warmup, e2e=not args.no_e2e, kernels=True)
    value = world * p.points * steps / (r["ms"] * 1e-3)
    kms = {k: v["ms_per_launch"] for k, v in r["kernels"].items()}      # per step (a kernel launched once per step and class)
    tot = sum(kms.values())
    dom = max(KERNEL_ALG_BYTES, key=lambda k: kms[k])
    counts, counts_note = _profile_counts(p.name)
    alu = alu_fracs(p, kms, counts)
    hbm = hbm_fracs(p, r["ms"] / steps, kms)
    # roofline.{achieved, peak, frac}: the dominant kernel's ALGORITHMIC bytes (16 B per point-update for
    # k_flux_update -- f^n read once, f^{n+1} written once) over its CUDA-event time against the measured HBM peak: the number
    # north_star's 60 % bar is read against.  What actually binds the kernel is the plain FP64 pipe: its
    # utilisation (EXECUTED FP64 thread-instructions per second against the measured DFMA rate) is in roofline.pipe_util.
    roof = {"bound": "hbm", "kernel": dom, "achieved": hbm[dom]["achieved_gbs"], "peak": peak, "unit": "GB/s",
            "frac": hbm[dom]["frac"], "traffic": (counts or {}).get(dom, {}).get("dram_bytes"), "peak_source": peak_src,
            "alg_bytes_per_launch": KERNEL_ALG_BYTES[dom] * p.points,
            "step_frac_of_16B_floor": hbm["step_frac_of_16B_floor"], "step_frac_of_declared_24B": hbm["step_frac_of_declared_24B"],
            "binding_roof": "fp64 pipe (see pipe_util): at the executed FP64 instructions per update the pipe alone caps the step below the HBM floor"}
    if alu and dom in alu:
        roof["pipe_util"] = {"kernel": dom, "achieved": alu[dom]["fp64_inst_per_s"] / 1e12, "peak": fp64_measured / 1e12,
                             "unit": "T executed FP64 thread-inst/s", "frac": alu[dom]["frac_of_fp64_peak"],
                             "peak_source": "measured here: bench_fp64_peak.cu, 8 independent DFMA chains per thread (nominal 148 SMs x 4 x 16 lanes x 1.965 GHz = %.3g)" % FP64_PEAK,
                             "peak_3operand": fp64_3op / 1e12, "frac_of_3operand": alu[dom]["fp64_inst_per_s"] / fp64_3op,
                             "counts_source": COUNTS_FILE + " (ncu counters of the kernel sources with the recorded sha256; static per build, times are live)"}
    else:
        roof["pipe_util"] = None
        roof["pipe_util_note"] = counts_note
    roof.update({"hbm": dict(hbm, peak_gbs=peak, peak_source=peak_src), "alu": alu,
                 "kernel_share_of_step": kms[dom] / tot, "kernel_ms": {k: round(v, 5) for k, v in kms.items()}})
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
            "ms_per_step": r["ms"] / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": _workload_name(p), "points_per_step": p.points, "parallelism": f"replicas x{world}",
                       "l2": "inputs larger than L2 (one copy of f = %.0f MB), no flush" % (p.points * 8 / 1e6)
                       if p.points * 8 > 126e6 else "L2-resident workload (f = %.0f MB), no flush" % (p.points * 8 / 1e6)},
            "clocks": r["clocks"], "gpu_launches": r["launches"], "roofline": roof, "e2e": r.get("e2e")}
    if rank == 0 and world == 1 and not args.no_extra:
        v, cores, sample, _ = oracle_sample(p)
        v1, _, sample1, _ = oracle_sample(p, seconds_hint=8.0, cores=1)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "cpu": _cpu_model(),
                                "single_thread": {"value": v1, "unit": UNIT, "cores": 1, "sample": sample1}}
        others = {}
        summary = {p.name: _summary_row(value, r["ms"] / steps, hbm, r["clocks"])}

        def other(q, st, label, tangential=False):
            rr = measure(q, st, 3, e2e=False, kernels=True, tangential=tangential)
            km = {k: v["ms_per_launch"] for k, v in rr["kernels"].items()}
            key = q.name + ("-tangential" if tangential else "")
            hb = hbm_fracs(q, rr["ms"] / st, km)
            others[key] = {"value": q.points * st / (rr["ms"] * 1e-3), "ms_per_step": rr["ms"] / st, "steps": st, "workload": label,
                           "clocks": rr["clocks"], "kernel_ms": {k: round(v, 5) for k, v in km.items()},
                           "hbm": hb, "alu": None if tangential else alu_fracs(q, km, _profile_counts(q.name)[0])}
            summary[key] = _summary_row(others[key]["value"], rr["ms"] / st, hb, rr["clocks"])
        for name in workloads.CONFIGS:
            if name == args.config or name == "C1":
                continue
            q = workloads.channel_config(name)
            if q.points * 8 * 2.2 > psutil.virtual_memory().available:
                others[name] = {"skipped": "host RAM too small to stage the input"}
                continue
            other(q, {"C2": 100, "C3": 40, "C4": 20, "C5": 20}[name], _workload_name(q))
        for mname, nuv, st in (("M4", 29, 100), ("M4", 69, 40), ("M3", 49, 40)):         # the paper's own shapes (Table 1 / Table 3)
            q = workloads.paper_mesh(mname, nuv)
            other(q, st, f"paper mesh {mname} {q.I}x{q.J}, {nuv}x{nuv} velocity grid, Kn=0.1")
        # option "tangential" on the headline workload: its own clocks and kernel fractions
        other(p, max(5, steps // 2), _workload_name(p) + ", option tangential (O3t/O8t)", tangential=True)
        line["other_workloads"] = others
        # one compact row per workload at the END of the line, so that a truncated tail still carries every workload:
        # [updates/s, ms per step, step / 16-B floor, cell_moments HBM frac (8 B/pt), flux_update HBM frac (16 B/pt), median SM MHz]
        line["workload_summary"] = summary
    if rank == 0:
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
