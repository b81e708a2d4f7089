#!/usr/bin/env python
"""bench.py -- the headline measurement of BASELINE.json on one B200 (or N replicas).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

With --gpus N > 1 and no launcher around it (WORLD_SIZE unset) it starts its N ranks itself (launch_ranks); under
torchrun it is one of the ranks.

One STEP = one pass of the whole hot path over one batch of synthetic input: one Navier-Stokes
right-hand-side evaluation psfft_hd_rhs at 512^3 fp64 (spectral curl, 6 inverse + 3 forward 3D
transforms, u x w, 2/3-rule dealias, projection: rows a1-a11 of SURVEY.md §8(a)), input and output
resident in HBM.  `value` = evaluations per second (whole job, all ranks).  The other half of
BASELINE.json's metric -- 512^3 fp64 batch-3 r2c + c2r milliseconds and % of the HBM roofline
(configs[2]) -- is timed in the same run and reported under "fft3d".

Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "fp64 N^3 r2c+c2r 3D FFT ms & % HBM roofline; HD-RHS evals/sec at 512^3"
UNIT = "evals/s"
FALLBACK_HBM_GBS = 6650.0      # /opt/skills/guides/B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


# ---- distributed plumbing (nccl on GPUs; gloo in the CPU tests) ----------------------------------------

def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def dist_init(backend: str):
    import torch.distributed as dist
    rank, _, world = dist_env()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world


def dist_barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def dist_max(x: float, device="cpu") -> float:
    """Max over ranks of a device-measured time (the slowest rank sets the job's time)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate(ms_per_step_max: float, units_per_rank_per_step: float, world: int) -> float:
    """Whole-job throughput: units all ranks processed per second (replicas: weak scaling)."""
    return world * units_per_rank_per_step / (ms_per_step_max * 1e-3)


# ---- clocks ---------------------------------------------------------------------------------------------

class ClockSampler:
    """nvidia-smi sampling DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "100", "-i", str(index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f:
            t = [s.strip() for s in line.split(",")]
            if len(t) < 9:
                continue
            try:
                sm.append(float(t[1])); mx.append(float(t[2])); power.append(float(t[3]))
            except ValueError:
                continue
            for nm, v in zip(names, t[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            sm.sort()
            out.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=max(mx), power_w_max=max(power), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


# ---- peaks ---------------------------------------------------------------------------------------------

def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def kernel_revision() -> str:
    """sha1 (first 12 hex digits) over the DEVICE-code sources: the revision an ncu capture belongs to.  psfft_api.cu
    is left out: it holds the host side of the boundary (argument checks, launch order, copies) and no kernel, so an
    edit there does not change what a capture measured."""
    import hashlib
    d = os.path.join(ROOT, "paper_1808_01309_b200", "csrc")
    h = hashlib.sha1()
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")) and f != "psfft_api.cu":
            h.update(f.encode())
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:12]


def ncu_traffic(kernel: str, workload: str = "512^3 fp64"):
    """(dram bytes (read + write) per launch of `kernel`, source) from the committed ncu --set full captures
    (profiles/traffic.csv: workload,kernel,dram_bytes_per_launch,source,kernel_revision), or (None, why) when
    there is no row or the row was captured on another revision of the kernel sources."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(p):
        return None, "profiles/traffic.csv missing"
    rev = kernel_revision()
    stale = None
    try:
        for line in open(p).read().splitlines()[1:]:
            cols = [c.strip() for c in line.split(",")]
            if len(cols) >= 5 and cols[0] == workload and cols[1] == kernel:
                if cols[4] == rev:
                    return float(cols[2]), cols[3]
                stale = f"capture {cols[3]} is of kernel revision {cols[4]}, the tree is {rev}"
    except Exception as exc:
        return None, str(exc)[:80]
    return None, stale or "no capture for this kernel / workload"


# ---- the oracle as CPU baseline (bench.py is one of the three places allowed to run oracle/) -------------

SAMPLE_N = 256


def work_ratio(N: int, n: int) -> float:
    """N^3 log2 N^3 / n^3 log2 n^3: transform work of the full workload per sample."""
    import math
    return (N ** 3 * 3 * math.log2(N)) / (n ** 3 * 3 * math.log2(n))


def cpu_model() -> str:
    try:
        for l in open("/proc/cpuinfo"):
            if l.startswith("model name"):
                return l.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_hd_rhs_seconds(n: int, threads: int, seed: int = 1234, uh=None):
    """One oracle hd_rhs at n^3 (the metric's field recipe) on `threads` threads; returns (seconds, threads in effect)."""
    import numpy as np
    import oracle
    from paper_1808_01309_b200 import synth
    cores = oracle.set_threads(threads)
    if uh is None:
        uh = synth.solenoidal_spectrum(n, 4.0, min(32, n // 2 - 1), seed)
    t0 = time.perf_counter()
    out = oracle.hd_rhs(uh, 0.0)
    dt = time.perf_counter() - t0
    assert np.isfinite(out[:, :2, :2, :2]).all()
    return dt, cores


def cpu_baseline(N: int) -> dict:
    """The oracle as it stands on the box's host cores (SURVEY.md §8(d) "CPU baseline"): ONE real evaluation of
    the metric's workload (hd_rhs at N^3, O6) on all cores, one r2c3d + c2r3d of one N^3 field (O3 + O4, the
    transform half of the metric), and the single-thread figure measured at 256^3 (a single-thread N = 512
    evaluation takes minutes; the 256^3 time is reported as measured, the scaled figure is labelled as such)."""
    import numpy as np
    import oracle
    from paper_1808_01309_b200 import synth
    ncpu = os.cpu_count() or 1
    dt, cores = oracle_hd_rhs_seconds(N, ncpu)
    x = synth.uniform_field(N, 1, 1234)[0]
    t0 = time.perf_counter()
    X = oracle.r2c3d(x)
    t_f = time.perf_counter() - t0
    t0 = time.perf_counter()
    y = oracle.c2r3d(X)
    t_b = time.perf_counter() - t0
    rt = float(np.abs(y - x).max())
    del X, y, x
    n1 = min(N, SAMPLE_N)
    dt1, c1 = oracle_hd_rhs_seconds(n1, 1)
    oracle.set_threads(ncpu)
    return {"value": 1.0 / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "cpu": cpu_model(),
            "sample": f"one full oracle hd_rhs (O6) at {N}^3, the metric's own workload and field, {dt:.2f} s on {cores} "
                      f"OpenMP threads; no extrapolation",
            "seconds_per_eval": dt,
            "fft3d": {"what": f"oracle r2c3d + c2r3d (O3 + O4) of one {N}^3 fp64 field on {cores} threads",
                      "s_r2c": t_f, "s_c2r": t_b, "ms_r2c_plus_c2r_per_field": (t_f + t_b) * 1e3,
                      "roundtrip_max_abs_err": rt},
            "single_thread": {"N": n1, "cores": c1, "seconds_per_eval": dt1, "evals_per_s_at_that_N": 1.0 / dt1,
                              "scaled_to_metric_N": {"extrapolated": n1 != N, "evals_per_s": 1.0 / (dt1 * work_ratio(N, n1)),
                                                     "how": f"x {work_ratio(N, n1):.2f} (N^3 log2 N^3 work ratio)"}}}


def run_reference(args) -> int:
    """--impl reference: the oracle, as it stands, on the host cores.  Every step is ONE REAL evaluation of the
    metric's workload (oracle hd_rhs at N^3 on all cores, about 15-20 s at 512^3); the number of steps actually run
    is capped so that the arm ends within a few minutes, and `steps` / `ms_per_step` report what was run."""
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    from paper_1808_01309_b200 import synth
    N = args.N
    ncpu = os.cpu_count() or 1
    uh = synth.solenoidal_spectrum(N, 4.0, min(32, N // 2 - 1), 1234)
    t_start = time.perf_counter()
    t_warm, cores = oracle_hd_rhs_seconds(N, ncpu, uh=uh)            # one warm-up evaluation (page faults, thread pool)
    budget = float(args.reference_budget_s)
    steps = max(1, min(args.steps, int((budget - t_warm) / max(t_warm, 1e-3))))
    times = [oracle_hd_rhs_seconds(N, ncpu, uh=uh)[0] for _ in range(steps)]
    dt = sum(times) / len(times)
    value = 1.0 / dt
    sample = (f"each step = one full oracle hd_rhs (O6) at {N}^3 on {cores} threads ({dt:.2f} s); {steps} of the requested "
              f"{args.steps} steps run after 1 warm-up (cap: {budget:.0f} s of oracle time); no extrapolation")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": 1, "steps_requested": args.steps, "warmup_requested": args.warmup,
            "ms_per_step": dt * 1e3, "wall_s": time.perf_counter() - t_start,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(N, world),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                             "cpu": cpu_model()},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def workload_config(N: int, world: int) -> dict:
    return {"workload": f"{N}^3 fp64 HD RHS (the metric's evals/s; field of BASELINE.json configs[1] at N={N}: random-phase "
                        f"solenoidal, E(k)~k^4 exp(-2(k/4)^2), unit energy, seed 1234+rank) + configs[2] {N}^3 fp64 batch-3 "
                        "r2c+c2r under 'fft3d'",
            "N": N, "fields": 3, "transforms_per_step": 9,
            "l2": "no flush needed: every pass streams > 1 GiB per field, far above the 126 MB L2",
            "parallelism": "1 GPU" if world == 1 else f"{world} independent replicas (north_star: no multi-GPU path; no collective)"}


# ---- our arm -------------------------------------------------------------------------------------------

def time_loop(fn, steps: int, stream) -> float:
    import torch
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        fn()
    e1.record(stream)
    e1.synchronize()
    return e0.elapsed_time(e1) / steps


def roofline_of(recs, K: int, ms_step: float, dense_bytes: float, dense_model: str, peak: float, workload: str) -> dict:
    """Roofline object from the per-launch records (kernel name, ms, algorithmic bytes) of K steps.
    Three different questions, kept apart:
      frac                         dominant kernel: its algorithmic bytes (compulsory reads + writes GIVEN the zero
                                   structure of the dealiased spectra) / its launch time / peak
      step_bytes_moved.frac        whole step: sum of all kernels' algorithmic bytes / step time / peak
      step_dense_model.equivalent_frac
                                   whole step against SURVEY.md §8(a)'s DENSE count (42 C HD, 84 C MHD): may exceed 1
                                   because the pruned passes move about half of those bytes -- an equivalent-work
                                   figure, not a bandwidth."""
    tot = {}
    for name, t, b in recs:
        a = tot.setdefault(name, [0.0, 0.0, 0])
        a[0] += t; a[1] += b; a[2] += 1
    dom = max(tot, key=lambda k: tot[k][0])
    achieved = tot[dom][1] / (tot[dom][0] * 1e-3) / 1e9
    moved = sum(v[1] for v in tot.values()) / K
    traffic, traffic_src = ncu_traffic(dom, workload)
    # scalar copies of the nested figures below (a record that keeps only the scalar members of this object still
    # carries the whole-step fractions and every kernel's own fraction): frac_<kernel> = its algorithmic bytes / its
    # time / peak, ms_<kernel> = its time per step
    flat = {"step_bytes_moved_frac": moved / (ms_step * 1e-3) / 1e9 / peak,
            "step_dense_equiv_frac": dense_bytes / (ms_step * 1e-3) / 1e9 / peak}
    for k, v in tot.items():
        short = k[4:] if k.startswith("rhs_") else k
        flat["frac_" + short] = v[1] / (v[0] * 1e-3) / 1e9 / peak
        flat["ms_" + short] = v[0] / K
    return {**flat, "bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
            "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src,
            "launches_timed": tot[dom][2], "avg_launch_ms": tot[dom][0] / tot[dom][2],
            "algorithmic_bytes_per_launch": tot[dom][1] / tot[dom][2],
            "kernel_share_of_step": tot[dom][0] / sum(v[0] for v in tot.values()),
            "per_kernel": {k: {"ms_per_step": v[0] / K, "GBps": v[1] / (v[0] * 1e-3) / 1e9, "frac": v[1] / (v[0] * 1e-3) / 1e9 / peak,
                               "launches_per_step": v[2] / K} for k, v in tot.items()},
            "step_bytes_moved": {"algorithmic_bytes": moved, "GBps": moved / (ms_step * 1e-3) / 1e9,
                                 "frac": moved / (ms_step * 1e-3) / 1e9 / peak},
            "step_dense_model": {"algorithmic_bytes": dense_bytes, "model": dense_model,
                                 "GBps_equivalent": dense_bytes / (ms_step * 1e-3) / 1e9,
                                 "equivalent_frac": dense_bytes / (ms_step * 1e-3) / 1e9 / peak}}


def device_spectrum(torch, synth, N, k0, kcut, seed, tag, cdtype, dev):
    """synth.solenoidal_spectrum built directly on the device: zeros + a scatter of the few thousand modes."""
    iz, iy, ix, v = synth.solenoidal_modes(N, k0, kcut, seed, tag)
    u = torch.zeros((3, N, N, N // 2 + 1), dtype=cdtype, device=dev)
    t = lambda a: torch.from_numpy(a.astype("int64")).to(dev)
    u[:, t(iz), t(iy), t(ix)] = torch.from_numpy(v).to(dev).to(cdtype)
    return u


WORKLOADS = {   # --workload: one right-hand side alone (the command lines of the ncu captures under profiles/)
    "hd512": (512, "float64", "hd", 4.0, 32, 42, "512^3 fp64 HD RHS (the metric's workload)"),
    "hd512f32": (512, "float32", "hd", 4.0, 32, 42, "512^3 fp32 HD RHS"),
    "hd768f32": (768, "float32", "hd", 4.0, 32, 42, "768^3 fp32 HD RHS (BASELINE.json configs[3])"),
    "mhd1024f32": (1024, "float32", "mhd", 3.0, 24, 84, "1024^3 fp32 MHD RHS (BASELINE.json configs[4])"),
}


def rhs_workload(torch, psfft, synth, dev, stream, peak, K, N, rdtype, system, k0, kcut, workload, dense_units, note) -> dict:
    """One right-hand-side workload: plan outside the timed region, 3 warm-up calls, K (<= 10) timed calls between CUDA
    events on device-resident input, then the same calls again with the per-launch events on for the bytes moved."""
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    cdt = torch.complex128 if rdtype == torch.float64 else torch.complex64
    code = psfft.F64 if rdtype == torch.float64 else psfft.F32
    lay = psfft.plan_query(N, code, 1)
    nvec = 2 if system == "mhd" else 1
    need = (lay.work_bytes_mhd if system == "mhd" else lay.work_bytes_hd) + 6 * nvec * lay.spec_bytes
    free = torch.cuda.mem_get_info(dev)[0]
    if free < need + (1 << 30):
        return {"workload": workload, "skipped": f"needs {need / 2**30:.0f} GiB, {free / 2**30:.0f} GiB free"}
    p = psfft.Plan(N, rdtype, 1, device=dev, work=system)
    u = device_spectrum(torch, synth, N, k0, kcut, 1234, 0, cdt, dev)
    ru = torch.empty_like(u)
    wk = p.ensure_work(system)
    if system == "mhd":
        b = device_spectrum(torch, synth, N, k0, kcut, 1234, 1, cdt, dev)
        rb = torch.empty_like(b)
        fn = lambda: psfft.mhd_rhs(p.handle, u, b, ru, rb, 0.0, 0.0, wk)
    else:
        fn = lambda: psfft.hd_rhs(p.handle, u, ru, 0.0, wk)
    n = max(3, min(K, 10))
    for _ in range(3):
        fn()
    torch.cuda.synchronize()
    ms = time_loop(fn, n, stream)
    psfft.profile_reset(p.handle)
    psfft.profile_enable(p.handle, True)
    time_loop(fn, n, stream)
    torch.cuda.synchronize()
    psfft.profile_enable(p.handle, False)
    dt = "fp64" if rdtype == torch.float64 else "fp32"
    rl = roofline_of(psfft.profile_records(p.handle), n, ms, dense_units * lay.spec_bytes,
                     f"fused 3-pass dense count = {dense_units} C (SURVEY.md §8(a))", peak, f"{N}^3 {dt}")
    out = {"workload": workload, "ms": ms, "evals_per_s": 1e3 / ms, "steps": n,
           "frac_bytes_moved": rl["step_bytes_moved"]["frac"],
           "dense_model_equivalent_frac": rl["step_dense_model"]["equivalent_frac"],
           "dominant_kernel": rl["kernel"], "dominant_kernel_frac": rl["frac"],
           "dominant_kernel_traffic": rl["traffic"], "traffic_source": rl["traffic_source"],
           "per_kernel": rl["per_kernel"], "launches_per_eval": psfft.last_launch_count(p.handle), "note": note}
    p.close()
    return out


def other_configs(torch, psfft, synth, dev, stream, peak, K: int) -> dict:
    """BASELINE.json configs 1, 2, 4, 5 (the metric's config 3 / 3b is the headline), same protocol: plan outside
    the timed region, 3 warm-up calls, K timed calls between CUDA events, device-resident inputs; then K more
    calls with the per-launch events on for the bytes actually moved.  Inputs of 768^3 / 1024^3 are far larger
    than L2; 32^3 and 128^3 are (partly) L2-resident and latency-bound -- reported in microseconds, no fraction
    for 32^3 (SURVEY.md §8(d) table "Synthetic inputs")."""
    import gc
    out = {}

    def timed(fn, n):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        return time_loop(fn, n, stream)

    # configs[0]: 32^3 fp64 r2c + c2r, one field
    N = 32
    p = psfft.Plan(N, torch.float64, 1, device=dev)
    x = torch.from_numpy(synth.uniform_field(N, 1, 1234)).to(dev)
    X = torch.empty(p.spec_shape(1), dtype=torch.complex128, device=dev)
    y = torch.empty_like(x)
    w = p.ensure_work("fft")
    t_f = timed(lambda: psfft.fft3d_r2c(p.handle, x, X, w), 200)
    t_b = timed(lambda: psfft.fft3d_c2r(p.handle, X, y, w), 200)
    out["configs[0]"] = {"workload": "32^3 fp64 r2c then c2r, one field, uniform [-1,1) seed 1234", "us_r2c": t_f * 1e3,
                         "us_c2r": t_b * 1e3, "launches": 6, "roundtrip_max_abs_err": float((y - x).abs().max()),
                         "note": "latency-bound (3 launches per direction, 0.5 MB working set in L2): no roofline fraction"}
    p.close()
    del p, x, X, y, w

    def rhs_config(key, N, rdtype, system, k0, kcut, workload, dense_units, note):
        out[key] = rhs_workload(torch, psfft, synth, dev, stream, peak, K, N, rdtype, system, k0, kcut, workload,
                                dense_units, note)

    rhs_config("configs[1]", 128, torch.float64, "hd", 4.0, 32,
               "128^3 fp64 HD RHS, E(k) ~ k^4 exp(-2(k/4)^2), unit energy, seed 1234", 42,
               "working set ~ 0.2 GB against 126 MB of L2: partly L2-resident, fractions may exceed the HBM figure")
    rhs_config("configs[3]", 768, torch.float32, "hd", 4.0, 32,
               "768^3 fp32 HD RHS (radix-3 schedules), same field recipe, k0 = 4", 42, "inputs far larger than L2")
    rhs_config("configs[4]", 1024, torch.float32, "mhd", 3.0, 24,
               "1024^3 fp32 MHD RHS, u and b each E(k) ~ k^4 exp(-2(k/3)^2), 12 inverse + 6 forward transforms", 84,
               "155 GB resident; inputs far larger than L2")
    gc.collect()
    torch.cuda.empty_cache()
    out["flat_box"] = flat_box_rows(torch, psfft, synth, dev, stream, peak, K, timed)
    gc.collect()
    torch.cuda.empty_cache()
    out["slab"] = slab_rows(torch, psfft, dev, stream, K, timed)
    gc.collect()
    torch.cuda.empty_cache()
    return out


def flat_box_rows(torch, psfft, synth, dev, stream, peak, K, timed) -> dict:
    """SURVEY.md §8(f) NEXT-2 at the paper's flat-box size: Boussinesq right-hand side and one RK2
    step on 1024 x 1024 x 256 in the box (2 pi, 2 pi, 2 pi / 4), fp64, device-resident broadband input."""
    import math
    import numpy as np
    shape, box = (1024, 1024, 256), (2 * math.pi, 2 * math.pi, 2 * math.pi / 4)
    p = psfft.Plan(shape, torch.float64, 1, device=dev, work="rk_boussinesq", box=box)
    y = torch.empty(p.spec_shape(4), dtype=torch.complex128, device=dev)
    y[:3].copy_(torch.from_numpy(synth.aniso_spectrum(shape, box, seed=1234, fill=0.2)))
    y[3].copy_(torch.from_numpy(synth.aniso_spectrum(shape, box, seed=1234, tag=7, ncomp=1, fill=0.2)))
    out = torch.empty_like(y)
    wk = p.ensure_work("rk_boussinesq")
    n = max(3, min(K, 10))
    f_rhs = lambda: psfft.boussinesq_rhs(p.handle, y[:3], y[3], out[:3], out[3], 1e-3, 1e-3, 2.0, wk)
    f_rk = lambda: psfft.rk_step(p.handle, psfft.SYS_BOUSSINESQ, y, out, 2, 1e-3, (1e-3, 1e-3, 2.0), wk)
    t_rhs = timed(f_rhs, n)
    psfft.profile_reset(p.handle)
    psfft.profile_enable(p.handle, True)
    time_loop(f_rhs, n, stream)
    torch.cuda.synchronize()
    psfft.profile_enable(p.handle, False)
    rl = roofline_of(psfft.profile_records(p.handle), n, t_rhs, 56.0 * p.layout.spec_bytes,
                     "fused 3-pass dense count = 56 C (9 + 4 transforms + 4 C epilogue reads)", peak, "1024x1024x256 fp64")
    t_rk = timed(f_rk, n)
    p.close()
    del p, y, out, wk
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    big = None
    if torch.cuda.mem_get_info(dev)[0] > 125 * 2**30:   # the paper's largest grid, fp32: 115 GB resident
        shape2 = (2048, 2048, 512)
        bq = torch.cuda.mem_get_info(dev)[0] > 160 * 2**30          # Boussinesq: 150 GB resident; else HD only
        p2 = psfft.Plan(shape2, torch.float32, 1, device=dev, work="boussinesq" if bq else "hd", box=box)
        u2 = torch.zeros(p2.spec_shape(4 if bq else 3), dtype=torch.complex64, device=dev)
        small = synth.aniso_spectrum((256, 256, 64), box, seed=1234, fill=0.4, dtype="complex64")   # modes of the low shells
        idx = lambda n_small, n_big: torch.from_numpy((np.fft.fftfreq(n_small, 1.0 / n_small).astype("int64")) % n_big).to(dev)
        iz, iy = idx(64, 512), idx(256, 2048)
        scale = float(np.prod(shape2)) / (256 * 256 * 64)
        u2[:3, iz[:, None], iy[None, :], :129] = torch.from_numpy(small).to(dev) * scale
        if bq:
            th = synth.aniso_spectrum((256, 256, 64), box, seed=1234, tag=7, ncomp=1, fill=0.4, dtype="complex64")
            u2[3, iz[:, None], iy[None, :], :129] = torch.from_numpy(th).to(dev) * scale
        r2 = torch.empty_like(u2)
        w2 = p2.ensure_work("boussinesq" if bq else "hd")
        nb = max(3, min(K, 5))
        t2 = timed(lambda: psfft.hd_rhs(p2.handle, u2[:3], r2[:3], 1e-3, w2), nb)
        big = {"workload": "2048 x 2048 x 512 fp32 in the box (2 pi, 2 pi, 2 pi/4): the paper's largest grid (PAPER.md:370, "
                           "64 GPUs there) on ONE GPU; band-limited random solenoidal u (+ theta)",
               "hd_rhs": {"ms": t2, "evals_per_s": 1e3 / t2, "resident_GB": 115}}
        if bq:
            t3 = timed(lambda: psfft.boussinesq_rhs(p2.handle, u2[:3], u2[3], r2[:3], r2[3], 1e-3, 1e-3, 2.0, w2), nb)
            big["boussinesq_rhs"] = {"ms": t3, "evals_per_s": 1e3 / t3, "resident_GB": 150}
        p2.close()
        del p2, u2, r2, w2
    res = {"workload": "1024 x 1024 x 256 fp64 Boussinesq in the box (2 pi, 2 pi, 2 pi/4), broadband solenoidal u + theta "
                       "(synth.aniso_spectrum, fill 0.2), nu = kappa = 1e-3, N_bv = 2",
           "boussinesq_rhs": {"ms": t_rhs, "evals_per_s": 1e3 / t_rhs, "frac_bytes_moved": rl["step_bytes_moved"]["frac"],
                              "per_kernel": rl["per_kernel"]},
           "boussinesq_rk2_step": {"ms": t_rk, "steps_per_s": 1e3 / t_rk}, "steps": n, "largest_grid": big}
    return res


def slab_rows(torch, psfft, dev, stream, K, timed) -> dict:
    """what ONE rank of a P = 8 slab decomposition of the 512^3 fp64 transform does
    locally (phase 1: x-pass + y-pass with the all-to-all fused into its stores, packed mode; phase 2: z-pass of its
    x-slab).  The exchange itself needs P GPUs: unmeasured on this box."""
    from paper_1808_01309_b200 import slab
    N, P = 512, 8
    p = psfft.Plan(N, torch.float64, 1, device=dev)
    lay = psfft.slab_query(p.handle, P, 0)
    real = torch.rand((lay.Mz, N, N), dtype=torch.float64, device=dev) * 2 - 1
    zs = torch.empty(lay.zspec_elems, dtype=torch.complex128, device=dev)
    send = torch.empty(lay.zspec_elems, dtype=torch.complex128, device=dev)
    xs = torch.empty(lay.xslab_elems, dtype=torch.complex128, device=dev)
    counts, _ = slab.forward_splits(N, N, p.ldk, P, 0)
    blocks = slab._slice_ptrs(send, counts)
    n = max(3, min(K, 20))
    t1 = timed(lambda: psfft.slab_r2c_xy(p.handle, P, 0, real, zs, blocks, 0), n)
    t2 = timed(lambda: psfft.slab_z(p.handle, P, 0, -1, xs), n)
    res = {"workload": f"rank 0 of P = {P}, {N}^3 fp64, one field: z-slab of {lay.Mz} planes, x-slab of {lay.w} kx columns",
           "ms_phase1_xy_scatter": t1, "ms_phase2_z": t2,
           "bytes_sent_per_rank": (P - 1) * lay.zspec_bytes // P,
           "exchange": "unmeasured on hardware (one GPU per box); at the guide's 770 GB/s per direction the "
                       f"{(P - 1) * lay.zspec_bytes // P / 1e6:.0f} MB take {(P - 1) * lay.zspec_bytes / P / 770e9 * 1e3:.3f} ms",
           "single_gpu_equivalent": "8 virtual ranks reproduce psfft_fft3d_r2c bit for bit (tests/test_gpu_slab.py)"}
    p.close()
    return res


def dist_all_ok(ok: bool, device="cpu") -> bool:
    """True iff EVERY rank says ok (all_reduce MIN of a flag).  Every rank must call it, whether its own set-up worked or
    not: it is how the ranks agree to skip a collective path before any of them has entered it."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return bool(ok)
    t = torch.tensor([1 if ok else 0], dtype=torch.int32, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MIN)
    return bool(int(t.item()))


SLAB_WATCHDOG_S = 180   # seconds the N > 1 slab rows may take before the headline is printed without them
SLAB_RT_TOL = 1e-12     # max |c2r(r2c(x)) - x| of the slab transform on uniform [-1, 1) input (fp64; measured ~4e-16)


def slab_multi(torch, psfft, dev, stream, K: int, N: int = 512) -> dict:
    """N > 1 ranks only: the slab-decomposed N^3 fp64 transform ACROSS the ranks (slab.SlabFFT: y-pass scattering
    into a send buffer, one NCCL all_to_all_single, z-pass of the x-slab), timed like everything else
    (barrier, CUDA events, max over ranks).  Never allowed to take the headline down: the ranks agree (dist_all_ok) that
    every one of them has its plan and buffers before any of them enters the all-to-all -- a rank that failed to set up
    would otherwise leave the others blocked in it -- and run_ours runs this under a watchdog that prints the headline
    without these rows if they do not come back."""
    import torch.distributed as dist
    plan = sf = x = None
    failed = None
    try:
        from paper_1808_01309_b200 import slab
        world, rank = dist.get_world_size(), dist.get_rank()
        plan = psfft.Plan(N, torch.float64, 1, device=dev)
        sf = slab.SlabFFT(plan)
        g = torch.Generator(device=dev).manual_seed(1234 + rank)
        x = torch.rand((sf.lay.Mz, N, N), dtype=torch.float64, device=dev, generator=g) * 2 - 1
    except Exception as exc:     # out of memory, plan refused, ...: decided together below
        failed = f"{type(exc).__name__}: {str(exc)[:200]}"
    if not dist_all_ok(failed is None, dev):
        if plan is not None:
            plan.close()
        return {"failed": failed or "skipped on every rank: another rank could not set up its plan or buffers"}
    try:
        X = sf.r2c(x)
        back = sf.c2r(X.clone())
        err = float((back - x).abs().max())
        n = max(3, min(K, 20))

        def timed(fn):
            for _ in range(3):
                fn()
            torch.cuda.synchronize()
            dist_barrier()
            t = time_loop(fn, n, stream)
            return dist_max(t, dev)

        xbuf = torch.empty(sf.lay.xslab_elems, dtype=torch.complex128, device=dev)     # the time loop allocates nothing
        rbuf = torch.empty_like(x)
        t_f = timed(lambda: sf.r2c(x, out=xbuf))
        Xc = X.clone()
        t_b = timed(lambda: sf.c2r(Xc, out=rbuf))   # overwrites Xc with its own inverse z-pass each call: timing only
        sent = (world - 1) * sf.lay.zspec_bytes // world
        res = {"workload": f"{N}^3 fp64, one field, slab-decomposed over {world} ranks (packed mode, NCCL all_to_all_single)",
               "ms_r2c": t_f, "ms_c2r": t_b, "roundtrip_max_abs_err": err, "bytes_sent_per_rank_per_transform": sent,
               "exchange_GBps_per_rank_if_all_of_r2c_were_exchange": sent / (t_f * 1e-3) / 1e9}
        if not err <= SLAB_RT_TOL:               # also catches NaN
            res["failed"] = f"round trip c2r(r2c(x)) differs from x by {err:.3e} (> {SLAB_RT_TOL:g}) on rank {rank}"
        plan.close()
        return res
    except Exception as exc:     # reported as text; the headline line carries it under slab_multi_failed
        return {"failed": f"{type(exc).__name__}: {str(exc)[:200]}"}


def run_ours(args) -> int:
    import numpy as np
    import torch
    from paper_1808_01309_b200 import build as psbuild
    from paper_1808_01309_b200 import psfft, synth

    rank, local, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libpsfft has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dist_init("nccl")
    psbuild.build_library()
    N, K, W = args.N, args.steps, max(3, args.warmup)
    dev = torch.device("cuda", local)
    stream = torch.cuda.current_stream()
    peak, peak_src = hbm_peak()
    if args.workload != "metric":   # one right-hand side alone: the command line of an ncu capture under profiles/
        Nw, dtw, system, k0, kcut, dense, what = WORKLOADS[args.workload]
        res = rhs_workload(torch, psfft, synth, dev, stream, peak, K, Nw, getattr(torch, dtw), system, k0, kcut, what,
                           dense, "single-workload run (--workload)")
        print(json.dumps({"workload_run": args.workload, **res}), flush=True)
        return 0
    m = metric_parts(torch, psfft, synth, N, K, W, rank, local, world, dev, stream, peak, peak_src)   # its buffers die here

    # ---- the other BASELINE.json configs, after the metric (they need the memory the 512^3 buffers held) ----
    configs = None
    if world == 1 and not args.no_configs:
        configs = other_configs(torch, psfft, synth, dev, stream, peak, K)

    line = {"metric": METRIC, "value": m["value"], "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": m["ms_max"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": workload_config(N, world), "clocks": m["clk"], "e2e": m["e2e"],
            "gpu_launches": m["launches_per_step"] * K, "launches_per_step": m["launches_per_step"],
            "roofline": m["roofline"], "fft3d": m["fft3d"], "next_rows": m["next_rows"], "configs": configs}
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(N)
    if world > 1:
        print_line_with_guarded_rows(line, rank, lambda: slab_multi(torch, psfft, dev, stream, K, N), SLAB_WATCHDOG_S)
    elif rank == 0:
        print(json.dumps(line), flush=True)
    return 0


def print_line_with_guarded_rows(line: dict, rank: int, rows_fn, timeout_s: float) -> None:
    """Print the (already complete) headline line with the N > 1 slab rows added -- or, if rows_fn does not come back
    within timeout_s, without them.  The slab-decomposed transform across the ranks has never met real multi-GPU
    hardware; a collective that hangs must not keep the headline from being printed.  On expiry every rank
    prints-and-exits (code 0) on its own; only rank 0 prints, and always exactly one JSON line."""
    import threading
    lock, state = threading.Lock(), {"printed": False}

    def emit(rows):
        with lock:
            if state["printed"]:
                return
            state["printed"] = True
            line["slab_multi_gpu"] = rows
            line["slab_multi_failed"] = rows.get("failed")     # top-level scalar: null = ran and round-tripped
            if rank == 0:
                print(json.dumps(line), flush=True)

    def expired():
        emit({"failed": f"no result after {timeout_s:g} s (a rank is stuck in the exchange); headline unaffected"})
        os._exit(0)

    dog = threading.Timer(timeout_s, expired)
    dog.daemon = True
    dog.start()
    rows = rows_fn()
    dog.cancel()
    emit(rows)


def metric_parts(torch, psfft, synth, N, K, W, rank, local, world, dev, stream, peak, peak_src) -> dict:
    """The metric's two halves at N^3 fp64 (HD RHS evals/s; batch-3 r2c + c2r) plus e2e and the NEXT rows."""
    # synthetic input (host, pinned) -> device
    kcut = min(32, N // 2 - 1)
    uh_host = torch.from_numpy(synth.solenoidal_spectrum(N, 4.0, kcut, 1234 + rank)).pin_memory()
    rhs_host = torch.empty_like(uh_host).pin_memory()
    plan = psfft.Plan(N, torch.float64, 3, device=dev, work="hd")
    uh = uh_host.to(dev, non_blocking=True)
    rhs = torch.empty_like(uh)
    work = plan.ensure_work("hd")
    h = plan.handle

    def step():
        psfft.hd_rhs(h, uh, rhs, 0.0, work)

    for _ in range(W):
        step()
    torch.cuda.synchronize()
    launches_per_step = psfft.last_launch_count(h)

    # ---- timed region: K steps, device-resident input, measurement hooks OFF -> `value` --------------------
    psfft.profile_enable(h, False)
    clocks = ClockSampler(local)
    dist_barrier()
    torch.cuda.synchronize()
    ms = time_loop(step, K, stream)
    torch.cuda.synchronize()
    dist_barrier()
    ms_max = dist_max(ms, dev)
    value = aggregate(ms_max, 1.0, world)

    # ---- the same K steps again with the per-launch CUDA events of the library ON -> roofline ------------
    psfft.profile_reset(h)
    psfft.profile_enable(h, True)
    torch.cuda.synchronize()
    ms_prof = time_loop(step, K, stream)
    torch.cuda.synchronize()
    psfft.profile_enable(h, False)
    recs = psfft.profile_records(h)
    spec_bytes = plan.layout.spec_bytes
    roofline = roofline_of(recs, K, ms_max, 42.0 * spec_bytes, "fused 3-pass HD RHS = 42 C (SURVEY.md §8(a))", peak,
                           f"{N}^3 fp64")
    roofline["peak_source"] = peak_src
    roofline["ms_per_step_with_event_hooks"] = ms_prof

    # ---- end to end through the C ABI with HOST buffers (H2D + kernels + D2H per step) ----------------
    d_in, d_out = torch.empty_like(uh), torch.empty_like(uh)

    # psfft_hd_rhs_host_box: the call a user with host arrays makes.  Per step it copies the index box around the
    # retained modes host -> device, evaluates, and copies the box of the result back (everything outside the box is
    # ignored on input and an exact zero on output: rhs_host is zeroed once, here, outside the timed region).
    rhs_host.zero_()
    box_bytes = psfft.host_box_bytes(h)

    def step_e2e():
        psfft.hd_rhs_host_box(h, uh_host, rhs_host, 0.0, d_in, d_out, work)

    def step_e2e_dense():      # the round-1/2 number: all 3 dense fields each way
        psfft.hd_rhs_host(h, uh_host, rhs_host, 0.0, d_in, d_out, work)

    step_e2e()
    e2e_equal = bool(torch.equal(rhs_host.to(dev), rhs))     # full host array == device-resident result, bit for bit
    dist_barrier()
    torch.cuda.synchronize()
    ke = min(K, 10)
    ms_e2e = dist_max(time_loop(step_e2e, ke, stream), dev)
    step_e2e_dense()
    ms_dense = dist_max(time_loop(step_e2e_dense, min(K, 3), stream), dev)
    e2e = {"value": aggregate(ms_e2e, 1.0, world), "unit": UNIT, "h2d_bytes_per_step": 3 * box_bytes,
           "d2h_bytes_per_step": 3 * box_bytes, "ms_per_step": ms_e2e, "steps": ke,
           "call": "psfft_hd_rhs_host_box (retained index box only; 12 cudaMemcpy3DAsync each way)",
           "host_result_equals_device_result": e2e_equal,
           "dense_copy_ms_per_step": ms_dense, "dense_copy_bytes_each_way": 3 * spec_bytes,
           "dense_copy_value": aggregate(ms_dense, 1.0, world)}
    clk = clocks.stop()
    del d_in, d_out

    # ---- the other half of the metric: 512^3 fp64 batch-3 r2c + c2r (configs[2]) ----------------------
    fft3d = None
    if rank == 0 or world > 1:
        x = torch.from_numpy(synth.uniform_field(N, 3, 1234 + rank)).to(dev)
        X = torch.empty(plan.spec_shape(3), dtype=torch.complex128, device=dev)
        y = torch.empty_like(x)
        fwork = plan.ensure_work("fft")
        f_fwd = lambda: psfft.fft3d_r2c(h, x, X, fwork)
        f_bwd = lambda: psfft.fft3d_c2r(h, X, y, fwork)
        for _ in range(3):
            f_fwd(); f_bwd()
        torch.cuda.synchronize()
        t_f = dist_max(time_loop(f_fwd, K, stream), dev)
        t_b = dist_max(time_loop(f_bwd, K, stream), dev)
        rt_err = float((y - x).abs().max())
        # side reference only (north_star: cuFFT "may be timed only as a side reference"; never on the product path)
        cufft = None
        try:
            c_f = lambda: torch.fft.rfftn(x, dim=(1, 2, 3))
            c_b = lambda: torch.fft.irfftn(X, s=(N, N, N), dim=(1, 2, 3))
            for _ in range(2):
                c_f(); c_b()
            torch.cuda.synchronize()
            cufft = {"ms_r2c": time_loop(c_f, min(K, 10), stream), "ms_c2r": time_loop(c_b, min(K, 10), stream),
                     "what": "torch.fft.rfftn / irfftn (cuFFT) on the same tensors, allocation of the result included"}
        except Exception as exc:     # out of memory on a busy device: the side reference is optional
            cufft = {"unavailable": str(exc)[:80]}
        fbytes = 3.0 * (plan.layout.real_bytes + 5.0 * spec_bytes)
        fft3d = {"workload": f"{N}^3 fp64 batch 3, uniform [-1,1) seed 1234 (BASELINE.json configs[2])",
                 "ms_r2c": t_f, "ms_c2r": t_b, "ms_r2c_plus_c2r": t_f + t_b, "ms_per_transform_per_field": (t_f + t_b) / 6.0,
                 "algorithmic_bytes_per_direction": fbytes, "GBps_r2c": fbytes / (t_f * 1e-3) / 1e9,
                 "GBps_c2r": fbytes / (t_b * 1e-3) / 1e9, "hbm_frac": 2 * fbytes / ((t_f + t_b) * 1e-3) / 1e9 / peak,
                 "hbm_frac_of_nominal_8TBps": 2 * fbytes / ((t_f + t_b) * 1e-3) / 1e9 / 8000.0,
                 "roundtrip_max_abs_err": rt_err, "side_reference_cufft": cufft}
        del x, X, y

    # ---- the rows SURVEY.md §8(f) marks "next", same size, same protocol (device-resident) --------------
    next_rows = None
    if world == 1:
        th = torch.from_numpy(synth.scalar_spectrum(N, 4.0, kcut, 1234)).to(dev)
        rt = torch.empty_like(th)
        bwork = plan.ensure_work("rk_boussinesq")
        f_b = lambda: psfft.boussinesq_rhs(h, uh, th, rhs, rt, 1e-3, 1e-3, 1.0, bwork)
        f_rk = lambda: psfft.rk_step(h, psfft.SYS_HD, uh, rhs, 2, 1e-3, (1e-3, 0.0, 0.0), bwork)
        f_g = lambda: psfft.gpe_rhs(h, uh, rhs, 0.3, 1.0, bwork)     # the first two fields as (p^, q^)
        for f in (f_b, f_rk, f_g):
            for _ in range(3):
                f()
        torch.cuda.synchronize()
        t_b = time_loop(f_b, K, stream)
        t_rk = time_loop(f_rk, K, stream)
        t_g = time_loop(f_g, K, stream)
        next_rows = {"boussinesq_rhs": {"ms": t_b, "evals_per_s": 1e3 / t_b,
                                        "workload": f"{N}^3 fp64, u as above + random-phase theta, nu = kappa = 1e-3, N_bv = 1"},
                     "hd_rk2_step": {"ms": t_rk, "steps_per_s": 1e3 / t_rk,
                                     "workload": f"{N}^3 fp64, two fused RHS stages, nu = 1e-3, dt = 1e-3"},
                     "gpe_rhs": {"ms": t_g, "evals_per_s": 1e3 / t_g,
                                 "workload": f"{N}^3 fp64, psi = p + i q as two real fields, alpha = 0.3, beta = 1"}}
        del th, rt

    if fft3d is not None:   # the metric's first clause as scalars of the roofline object, next to the kernel's
        roofline["fft3d_ms_r2c_plus_c2r"] = fft3d["ms_r2c_plus_c2r"]
        roofline["fft3d_hbm_frac"] = fft3d["hbm_frac"]
        roofline["fft3d_ms_r2c"] = fft3d["ms_r2c"]
        roofline["fft3d_ms_c2r"] = fft3d["ms_c2r"]
    return {"value": value, "ms_max": ms_max, "clk": clk, "e2e": e2e, "launches_per_step": launches_per_step,
            "roofline": roofline, "fft3d": fft3d, "next_rows": next_rows}


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--N", type=int, default=512, help="grid size (the metric is quoted at 512)")
    ap.add_argument("--workload", default="metric", choices=["metric"] + sorted(WORKLOADS),
                    help="metric: the full bench line (default); otherwise time ONE right-hand-side workload alone")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="skip the other BASELINE.json configs (768^3, 1024^3 ...)")
    ap.add_argument("--reference-budget-s", type=float, default=150.0,
                    help="--impl reference: cap on the oracle time of the whole arm (full-size evaluations)")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return launch_ranks(args.gpus)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


def launch_ranks(n: int) -> int:
    """`bench.py --gpus N` called WITHOUT a launcher (no WORLD_SIZE in the environment): start the N ranks ourselves,
    one process per GPU (one task per GPU, bound by the program, not by the caller), by re-running this
    very command line under torch.distributed.run on 127.0.0.1 with a free port.  Each rank then finds
    RANK / LOCAL_RANK / WORLD_SIZE in its environment and binds to cuda:LOCAL_RANK (run_ours).  Under an external
    launcher (the driver's torchrun line) WORLD_SIZE is set and this function is never reached."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
    return subprocess.call(cmd)


if __name__ == "__main__":
    sys.exit(main())
